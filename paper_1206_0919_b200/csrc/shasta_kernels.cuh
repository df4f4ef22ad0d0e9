// shasta_kernels.cuh -- sm_100a device code of the fused SHASTA sweep.
//
// One sweep along an axis = one kernel launch that reads the five conserved fields once and
// writes them once (80 B/cell in fp64).  Every pencil is processed by a MARCHING thread: it walks
// along the sweep axis with the "front" cell i and keeps a rolling register window, so every
// quantity of eqs. (15)-(22) is computed exactly once per cell / per interface --
// not 5x (U-hat) and 2x (A) per cell as in the paper's Listing 1.
//
// Pipeline of one march step with front cell i (dependency radius 4):
//   S1  (v,p)_i        = cons2prim(U_i)                                  phases 3-4
//   S2  F~_{i-1/2}, U~_{i-1} : half-step predictor, eq. (17) with lambda/2 (flux form, pin P2)
//   S3  (v,p)^{1/2}_{i-1} = cons2prim(U~_{i-1})
//   S4  F_{i-3/2},  U^_{i-2} : full-step transport + diffusion, eqs. (15)-(17), U^n transported
//   S5  D^_{i-3}, A_{i-4}    : phoenical antidiffusion + limiter, eqs. (18)-(21)
//   S6  U^{n+1}_{i-4} = U^_{i-4} - A_{i-4} + A_{i-5}, eq. (22); causality projection Pi
//   S7  (last sweep of a step) primitives of cell i-4
// The fields arrive PERMUTED by the host: slot 0 = E, slot 1 = the momentum PARALLEL to the sweep
// axis (source term lambda*Delta(p)), slots 2,3 = the perpendicular momenta (source
// free), slot 4 = R.  The kernels therefore never branch on the axis.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace shk {

constexpr int NF = 5;       // E, M_par, M_perp1, M_perp2, R
constexpr int GH = 4;       // ghost depth = dependency radius of one sweep
constexpr int EOS_GAMMA = 0;    // p = (Gamma-1) e            (m = 0): closed-form velocity
constexpr int EOS_MASS = 1;     // p = (Gamma-1)(e - m n)     (m > 0): safeguarded Newton

template <typename T>
struct Consts {
    T lam;      // lambda = dt/dx
    T hlam;     // lambda/2 (predictor)
    T gam;      // Gamma
    T gm1;      // Gamma-1
    T g2;       // Gamma^2
    T c4;       // 4 (Gamma-1)
    T hg;       // Gamma/2
    T omd;      // 1 - delta, delta = 1e-12 (reading G7)
    T mass;     // m
};

struct SweepParams {
    const void* in[NF];     // permuted conserved fields of the current buffer
    void* out[NF];          // permuted conserved fields of the other buffer
    void* prim[6];          // e, p, n, v_par, v_perp1, v_perp2 (permuted like the momenta)
    long long stride_axis;  // element stride along the sweep axis
    long long stride_other; // strided kernel: pencil p -> base = (p % nx) + (p / nx) * stride_other
    int nx;                 // extent of the contiguous axis
    int N;                  // extent of the sweep axis
    long long npencil;      // number of pencils (rows for the x sweep)
    int seg;                // cells marched per work item
    int nseg;               // segments per pencil
    int periodic;           // boundary rule (reading G11)
    unsigned long long* counts;   // diagnostics [4]
};

// reading G11: ghost-extend the INPUT of the sweep: outflow = copy of the edge cell, periodic = wrap
__device__ __forceinline__ int ghost_index(int j, int N, int periodic)
{
    if (periodic) { j %= N; return j < 0 ? j + N : j; }
    return min(max(j, 0), N - 1);
}

template <typename T> __device__ __forceinline__ T t_sqrt(T x);
template <> __device__ __forceinline__ double t_sqrt<double>(double x) { return sqrt(x); }
template <> __device__ __forceinline__ float t_sqrt<float>(float x) { return sqrtf(x); }
template <typename T> __device__ __forceinline__ T t_rsqrt(T x);
template <> __device__ __forceinline__ double t_rsqrt<double>(double x) { return rsqrt(x); }
template <> __device__ __forceinline__ float t_rsqrt<float>(float x) { return rsqrtf(x); }
template <typename T> __device__ __forceinline__ T t_fma(T a, T b, T c);
template <> __device__ __forceinline__ double t_fma<double>(double a, double b, double c) { return fma(a, b, c); }
template <> __device__ __forceinline__ float t_fma<float>(float a, float b, float c) { return fmaf(a, b, c); }
template <typename T> __device__ __forceinline__ T t_min(T a, T b) { return a < b ? a : b; }
template <typename T> __device__ __forceinline__ T t_max(T a, T b) { return a > b ? a : b; }
template <typename T> __device__ __forceinline__ T t_abs(T a);
template <> __device__ __forceinline__ double t_abs<double>(double a) { return fabs(a); }
template <> __device__ __forceinline__ float t_abs<float>(float a) { return fabsf(a); }

// ------------------------------------------------------------------------------------------------
// cons2prim: relativistic correction + EOS (phases 3-4; readings G6-G10).
// Solves v (E + P(E - Mc v, R sqrt(1-v^2))) = Mc, Mc = min(|M|, (1-delta) E), on [0,1).
//   EOS_GAMMA: closed form v = 2 Mc / (Gamma E + sqrt(Gamma^2 E^2 - 4 (Gamma-1) Mc^2)) (pin P7 ii).
//   EOS_MASS : Newton with bisection safeguard on the bracket [v(m=0), Mc/E]; the warp leaves the loop
//              together (__all_sync), so there is no intra-warp divergence in the iteration.
// Returns vfac such that v_i = M_i * vfac, plus e, p, and v^2 (for n = R sqrt(1-v^2)).
// The rare clamp branch (|M| > (1-delta) E) is the only data-dependent branch.
template <typename T, int EOS>
__device__ __forceinline__ void cons2prim(const Consts<T>& k, T E, T Ma, T Mb, T Mc, T R,
                                          T& vfac, T& e, T& p, T& v2, int& floored)
{
    const bool vac = !(E > T(0));                   // vacuum (reading G7); also catches NaN
    if (vac) { E = T(1); Ma = Mb = Mc = T(0); }     // keep the arithmetic below finite; result discarded
    floored = 0;
    const T M2 = t_fma(Ma, Ma, t_fma(Mb, Mb, Mc * Mc));
    const T lim = k.omd * E;
    const T lim2 = lim * lim;
    T Mq = M2;          // Mc^2 (clamped)
    T s = T(1);         // Mc / |M|
    if (M2 > lim2) {    // rare: causality clamp, same rule as Pi
        Mq = lim2;
        s = lim * t_rsqrt(M2);
    }
    const T disc = t_fma(k.g2, E * E, -k.c4 * Mq);
    const T sq = t_sqrt(disc);
    const T hden = t_fma(k.hg, E, T(0.5) * sq);     // (Gamma E + sqrt(disc)) / 2
    T inv = T(1) / hden;                            // v = Mc * inv   (m = 0 root)
    if (EOS == EOS_GAMMA) {
        const T eraw = t_fma(-Mq, inv, E);
        if (eraw < T(0)) floored |= 1;
        e = t_max(eraw, T(0));
        p = k.gm1 * e;
        v2 = Mq * inv * inv;
        vfac = s * inv;
    } else {
        const T Mabs = t_sqrt(Mq);
        T lo = Mabs * inv;                          // m = 0 root: lower bound (P_m <= P_0)
        T hi = t_min(Mabs / E, k.omd);              // P = 0 root: upper bound
        lo = t_min(lo, hi);
        const T mR = k.mass * R;
        T v = lo;
        for (int it = 0; it < 48; ++it) {
            const T w2 = t_fma(-v, v, T(1));
            const T w = t_sqrt(w2);
            const T praw = k.gm1 * ((E - Mabs * v) - mR * w);
            const bool pos = praw > T(0);
            const T P = pos ? praw : T(0);
            const T dP = pos ? k.gm1 * (mR * v / w - Mabs) : T(0);
            const T g = t_fma(v, E + P, -Mabs);
            const T dg = t_fma(v, dP, E + P);
            if (g > T(0)) hi = v; else lo = v;
            T vn = v - g / dg;
            if (!(vn >= lo && vn <= hi)) vn = T(0.5) * (lo + hi);
            const T dv = t_abs(vn - v);
            v = vn;
            const T tol = sizeof(T) == 8 ? T(1e-15) : T(2e-7);
            if (__all_sync(__activemask(), dv <= tol)) break;
        }
        v2 = v * v;
        const T eraw = t_fma(-Mabs, v, E);
        if (eraw < T(0)) floored |= 1;
        e = t_max(eraw, T(0));
        const T n = R * t_sqrt(t_fma(-v, v, T(1)));
        const T praw = k.gm1 * (e - k.mass * n);
        if (praw < T(0)) floored |= 2;
        p = t_max(praw, T(0));
        vfac = (M2 > T(0)) ? v * t_rsqrt(M2) : T(0);
    }
    if (vac) { vfac = T(0); e = T(0); p = T(0); v2 = T(0); floored = 0; }
}

// eq. (21) branch-free (reading G12): A = sigma max(0, min(sigma D^_{j+1}, |A^ph|, sigma D^_{j-1}))
template <typename T>
__device__ __forceinline__ T limiter(T aph, T dhp, T dhm)
{
    const T sg = copysign(T(1), aph);
    const T m = t_min(t_min(sg * dhp, t_abs(aph)), sg * dhm);
    return sg * t_max(m, T(0));
}

// ------------------------------------------------------------------------------------------------
// The rolling window of one marching thread.  Index names: member "x<k>" holds the quantity at cell
// (or interface) i-k where i is the front cell of the CURRENT step.
template <typename T, int EOS>
struct Marcher {
    T u1[NF], u2[NF];                       // U^n_{i-1}, U^n_{i-2}
    T dl2[NF], dl3[NF], dl4[NF], dl5[NF];   // Delta_{i-2..i-5}, eq. (16)
    T ft[NF];                               // predictor flux F~ at interface (i-2,i-1)
    T fc[NF];                               // corrector flux F at interface (i-3,i-2)
    T uh3[NF], uh4[NF];                     // U^_{i-3}, U^_{i-4}
    T dh4[NF], dh5[NF];                     // D^_{i-4}, D^_{i-5}, eq. (18)
    T a5[NF];                               // limited antidiffusive flux A_{i-5}
    T eps1, fE1, fE2, fM1, fM2;             // time-n: (lambda/2) v_{i-1}, (p v)_{i-1,i-2}, p_{i-1,i-2}
    T epsh2, gE2, gE3, gM2, gM3;            // half step: lambda v_{i-2}, (p v)_{i-2,i-3}, p_{i-2,i-3}

    __device__ __forceinline__ void init()
    {
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            u1[f] = u2[f] = dl2[f] = dl3[f] = dl4[f] = dl5[f] = ft[f] = fc[f] = T(0);
            uh3[f] = uh4[f] = dh4[f] = dh5[f] = a5[f] = T(0);
        }
        eps1 = fE1 = fE2 = fM1 = fM2 = epsh2 = gE2 = gE3 = gM2 = gM3 = T(0);
    }

    // One march step: consumes U^n at the front cell, produces U^{n+1} of cell i-4 in un[].
    __device__ __forceinline__ void step(const Consts<T>& k, const T (&u0)[NF], T (&un)[NF])
    {
        // S1: time-n primitives of the front cell
        T vf0, e0, p0, v20;
        int fl;
        cons2prim<T, EOS>(k, u0[0], u0[1], u0[2], u0[3], u0[4], vf0, e0, p0, v20, fl);
        const T v0 = u0[1] * vf0;
        const T eps0 = k.hlam * v0;
        const T fE0 = p0 * v0;
        // S2: predictor (half step, no antidiffusion: reading G4), interface (i-1,i), cell i-1
        T ut[NF], dl1[NF];
        {
            const T q = (T(0.5) - eps1) / (T(1) + (eps0 - eps1));   // Q+_{i-1}, eq. (15); Q-_i = 1-q (P1)
            const T a = T(0.5) - q, b = T(0.5) * q * q;
#pragma unroll
            for (int f = 0; f < NF; ++f) {
                dl1[f] = u0[f] - u1[f];                             // eq. (16)
                const T fl = t_fma(a, u1[f], -b * dl1[f]);          // F = (1/2-q) U - 1/2 q^2 Delta (P2)
                ut[f] = (u1[f] - fl) + ft[f];
                ft[f] = fl;
            }
            ut[0] = t_fma(T(-0.5) * k.hlam, fE0 - fE2, ut[0]);      // + (lambda/2) Delta(p v)
            ut[1] = t_fma(T(-0.5) * k.hlam, p0 - fM2, ut[1]);       // + (lambda/2) Delta(p)
        }
        // S3: half-step primitives of cell i-1
        T vfh, eh, ph, v2h;
        cons2prim<T, EOS>(k, ut[0], ut[1], ut[2], ut[3], ut[4], vfh, eh, ph, v2h, fl);
        const T vh1 = ut[1] * vfh;
        const T epsh1 = k.lam * vh1;
        const T gE1 = ph * vh1;
        // S4: corrector transport of U^n, interface (i-2,i-1), cell i-2
        T uh2[NF];
        {
            const T q = (T(0.5) - epsh2) / (T(1) + (epsh1 - epsh2));
            const T a = T(0.5) - q, b = T(0.5) * q * q;
#pragma unroll
            for (int f = 0; f < NF; ++f) {
                const T fl = t_fma(a, u2[f], -b * dl2[f]);
                uh2[f] = (u2[f] - fl) + fc[f];
                fc[f] = fl;
            }
            uh2[0] = t_fma(T(-0.5) * k.lam, gE1 - gE3, uh2[0]);     // + lambda Delta(p v)^{n+1/2}
            uh2[1] = t_fma(T(-0.5) * k.lam, ph - gM3, uh2[1]);      // + lambda Delta(p)^{n+1/2}
        }
        // S5+S6: antidiffusion at interface (i-4,i-3), update of cell i-4
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            const T dh3 = uh2[f] - uh3[f];                                       // eq. (18)
            const T d2 = (dl3[f] + dl5[f]) - T(2) * dl4[f];                      // reading G14
            const T aph = T(0.125) * (dh4[f] - T(0.125) * d2);                   // eq. (19)
            const T a4 = limiter<T>(aph, dh3, dh5[f]);                           // eqs. (20),(21)
            un[f] = (uh4[f] - a4) + a5[f];                                       // eq. (22)
            // shift the window
            a5[f] = a4;
            dh5[f] = dh4[f]; dh4[f] = dh3;
            uh4[f] = uh3[f]; uh3[f] = uh2[f];
            dl5[f] = dl4[f]; dl4[f] = dl3[f]; dl3[f] = dl2[f]; dl2[f] = dl1[f];
            u2[f] = u1[f]; u1[f] = u0[f];
        }
        eps1 = eps0; fE2 = fE1; fE1 = fE0; fM2 = fM1; fM1 = p0;
        epsh2 = epsh1; gE3 = gE2; gE2 = gE1; gM3 = gM2; gM2 = ph;
    }
};

// Pi, readings G6-G8: written back to M at the end of every sweep.  E and R are never modified.
template <typename T>
__device__ __forceinline__ void project(const Consts<T>& k, T (&un)[NF], unsigned long long* counts)
{
    const T E = un[0];
    const T M2 = t_fma(un[1], un[1], t_fma(un[2], un[2], un[3] * un[3]));
    const T lim = k.omd * E;
    if (!(E > T(0))) {
        un[1] = un[2] = un[3] = T(0);
        atomicAdd(counts + 1, 1ULL);
    } else if (M2 > lim * lim) {
        const T s = lim * t_rsqrt(M2);
        un[1] *= s; un[2] *= s; un[3] *= s;
        atomicAdd(counts + 0, 1ULL);
    }
}

// primitives of one cell from its (projected) conserved state, slots permuted like the momenta
template <typename T, int EOS>
__device__ __forceinline__ void primitives(const Consts<T>& k, const T (&u)[NF], T (&pr)[6],
                                           unsigned long long* counts)
{
    T vf, e, p, v2;
    int fl;
    cons2prim<T, EOS>(k, u[0], u[1], u[2], u[3], u[4], vf, e, p, v2, fl);
    pr[0] = e; pr[1] = p;
    pr[2] = u[4] * t_sqrt(t_max(T(1) - v2, T(0)));
    pr[3] = u[1] * vf; pr[4] = u[2] * vf; pr[5] = u[3] * vf;
    if (fl) {                                       // rare: diagnostics [2] e floored, [3] p floored
        if (fl & 1) atomicAdd(counts + 2, 1ULL);
        if (fl & 2) atomicAdd(counts + 3, 1ULL);
    }
}

// ------------------------------------------------------------------------------------------------
// Sweep along y or z: lanes run along the contiguous x axis, so every load and store of a warp is a
// coalesced 256 B (fp64) row piece; no shared memory is needed.  Work item = (pencil, segment).
template <typename T, int EOS, bool EMIT>
__global__ void __launch_bounds__(128) sweep_strided_kernel(SweepParams P, Consts<T> k)
{
    const long long pen = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (pen >= P.npencil) return;
    const int sg = blockIdx.y;
    const int j0 = sg * P.seg;
    const int j1 = min(P.N, j0 + P.seg);
    const long long base = (pen % P.nx) + (pen / P.nx) * P.stride_other;
    const long long sa = P.stride_axis;
    const T* __restrict__ in[NF];
    T* __restrict__ out[NF];
#pragma unroll
    for (int f = 0; f < NF; ++f) { in[f] = (const T*)P.in[f] + base; out[f] = (T*)P.out[f] + base; }

    Marcher<T, EOS> m;
    m.init();
    T nxt[NF];
    {
        const long long o = (long long)ghost_index(j0 - GH, P.N, P.periodic) * sa;
#pragma unroll
        for (int f = 0; f < NF; ++f) nxt[f] = __ldg(in[f] + o);
    }
    for (int i = j0 - GH; i < j1 + GH; ++i) {
        T u0[NF], un[NF];
#pragma unroll
        for (int f = 0; f < NF; ++f) u0[f] = nxt[f];
        if (i + 1 < j1 + GH) {                           // prefetch the next front cell
            const long long o = (long long)ghost_index(i + 1, P.N, P.periodic) * sa;
#pragma unroll
            for (int f = 0; f < NF; ++f) nxt[f] = __ldg(in[f] + o);
        }
        m.step(k, u0, un);
        const int jo = i - GH;
        if (jo >= j0) {
            project<T>(k, un, P.counts);
            const long long o = (long long)jo * sa;
#pragma unroll
            for (int f = 0; f < NF; ++f) out[f][o] = un[f];
            if (EMIT) {
                T pr[6];
                primitives<T, EOS>(k, un, pr, P.counts);
#pragma unroll
                for (int q = 0; q < 6; ++q) ((T*)P.prim[q])[base + o] = pr[q];
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Sweep along x (the contiguous axis): a CTA owns ROWS rows; thread r marches along row r.  The rows
// are staged through shared memory in chunks of CH cells per row (cp.async, double buffered) so that
// global traffic stays coalesced (64 B row pieces) while each thread reads its own row conflict-free
// (row pitch CH+1: odd).  Results go to an output tile and are written back coalesced; the primitives
// of the last sweep are computed element-wise during that write-back.
constexpr int XCH = 8;            // cells per row per chunk
constexpr int XPITCH = XCH + 1;   // odd pitch: conflict-free column access for 8 B elements
constexpr int XNS = 2;            // input stages

template <typename T>
__device__ __forceinline__ void cp_async_elem(T* smem_dst, const T* gsrc)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    if (sizeof(T) == 8)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(d), "l"(gsrc) : "memory");
    else
        asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

template <typename T, int ROWS>
struct XSmem {
    T in[XNS][NF][ROWS * XPITCH];
    T out[NF][ROWS * XPITCH];
};

template <typename T, int EOS, bool EMIT, int ROWS>
__global__ void __launch_bounds__(ROWS) sweep_x_kernel(SweepParams P, Consts<T> k)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    XSmem<T, ROWS>& S = *reinterpret_cast<XSmem<T, ROWS>*>(smem_raw);
    const int t = threadIdx.x;
    const long long row0 = (long long)blockIdx.x * ROWS;
    const int nrows = (int)min((long long)ROWS, P.npencil - row0);
    const int sg = blockIdx.y;
    const int j0 = sg * P.seg;
    const int j1 = min(P.N, j0 + P.seg);
    const int ilo = j0 - GH, ihi = j1 + GH;               // front cells [ilo, ihi)
    const int c_first = (ilo >= 0) ? ilo / XCH : -((-ilo + XCH - 1) / XCH);
    const int c_last = (ihi - 1) / XCH;
    const int N = P.N;

    // cooperative chunk loader: element (row, col) of chunk c <- in[f][(row0+row)*nx + ghost(XCH*c+col)]
    auto load_chunk = [&](int c, int stage) {
        if (c <= c_last) {
            for (int e = t; e < ROWS * XCH; e += ROWS) {
                const int row = e / XCH, col = e % XCH;
                const int i = c * XCH + col;
                if (row < nrows && i >= ilo && i < ihi) {
                    const long long g = (row0 + row) * (long long)N + ghost_index(i, N, P.periodic);
#pragma unroll
                    for (int f = 0; f < NF; ++f)
                        cp_async_elem<T>(&S.in[stage][f][row * XPITCH + col], (const T*)P.in[f] + g);
                }
            }
        }
        cp_async_commit();
    };

    Marcher<T, EOS> m;
    m.init();
    load_chunk(c_first, 0);
    load_chunk(c_first + 1, 1);
    for (int c = c_first; c <= c_last; ++c) {
        const int stage = (c - c_first) % XNS;
        cp_async_wait<XNS - 1>();
        __syncthreads();
        if (t < nrows) {
            for (int s = 0; s < XCH; ++s) {
                const int i = c * XCH + s;
                if (i < ilo || i >= ihi) continue;
                T u0[NF], un[NF];
#pragma unroll
                for (int f = 0; f < NF; ++f) u0[f] = S.in[stage][f][t * XPITCH + s];
                m.step(k, u0, un);
                if (i - GH >= j0) {
                    project<T>(k, un, P.counts);
#pragma unroll
                    for (int f = 0; f < NF; ++f) S.out[f][t * XPITCH + s] = un[f];
                }
            }
        }
        __syncthreads();
        // write-back of output cells [XCH*c - 4, XCH*c + 4) and refill of the stage just consumed
        for (int e = t; e < ROWS * XCH; e += ROWS) {
            const int row = e / XCH, col = e % XCH;
            const int jo = c * XCH - GH + col;
            if (row < nrows && jo >= j0 && jo < j1) {
                const long long g = (row0 + row) * (long long)N + jo;
                T u[NF];
#pragma unroll
                for (int f = 0; f < NF; ++f) {
                    u[f] = S.out[f][row * XPITCH + col];
                    ((T*)P.out[f])[g] = u[f];
                }
                if (EMIT) {
                    T pr[6];
                    primitives<T, EOS>(k, u, pr, P.counts);
#pragma unroll
                    for (int q = 0; q < 6; ++q) ((T*)P.prim[q])[g] = pr[q];
                }
            }
        }
        load_chunk(c + XNS, stage);
    }
    cp_async_wait<0>();
}

}  // namespace shk
