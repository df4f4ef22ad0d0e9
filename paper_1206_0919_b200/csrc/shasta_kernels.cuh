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
//
// The kernel is bound by the fp64 pipe (64 results/clk/SM on B200, measured) about as much as by HBM
// (DESIGN.md 7), so the arithmetic is written for a minimal fp64 instruction count:
//   * no fp64 division or library sqrt on the common path: MUFU.RCP64H / MUFU.RSQ64H seeds (2^-20,
//     measured) + Newton steps written out below;
//   * the flux limiter's min/max/sign run on the integer pipe (sign-magnitude ordering of doubles);
//   * the register window rotates by NAME (march loop unrolled by 4, compile-time slots), not by moves.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace shk {

constexpr int NF = 5;       // E, M_par, M_perp1, M_perp2, R
constexpr int GH = 4;       // ghost depth = dependency radius of one sweep
constexpr int EOS_GAMMA = 0;    // p = (Gamma-1) e            (m = 0): closed-form velocity
constexpr int EOS_MASS = 1;     // p = (Gamma-1)(e - m n)     (m > 0): safeguarded Newton

// EOS / cons2prim constants.  cons2prim, the causality projection and the primitive output ALWAYS run in
// fp64, also on the fp32 storage path (the paper's own plan: "double precision for ... the calculation of
// the boost"): e = E - |M| v cancels gamma^2 digits, which fp32 does not have.
struct EosD {
    double gam;     // Gamma
    double gm1;     // Gamma-1
    double g2;      // Gamma^2
    double c4;      // 4 (Gamma-1)
    double hg;      // Gamma/2
    double omd;     // 1 - delta, delta = 1e-12 (reading G7)
    double omd2;    // (1 - delta)^2
    double mass;    // m
};

template <typename T>
struct Consts {
    T lam;      // lambda = dt/dx
    T hlam;     // lambda/2 (predictor; corrector source factor)
    T qlam;     // lambda/4 (predictor source factor 1/2 * lambda/2)
    EosD d;
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

// Diagnostics are counted per thread in shared memory (or registers) and flushed once per warp at the end of
// the kernel: one global atomic per event on a single address serialises in L2 and cost 60 % of the step
// time once the causality projection fires in ~0.2 % of the cells (profiles/, round 1).
struct Cnt {
    unsigned* p;    // this thread's four counters: p[w * stride]
    int stride;
    __device__ __forceinline__ void add(int w) const { p[w * stride] += 1u; }
    __device__ __forceinline__ void zero() const { p[0] = p[stride] = p[2 * stride] = p[3 * stride] = 0u; }
};
__device__ __forceinline__ void flush_counts(const Cnt& c, unsigned long long* g)
{
    const unsigned mask = __activemask();
    const int leader = __ffs(mask) - 1;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const unsigned v = __reduce_add_sync(mask, c.p[w * c.stride]);
        if ((int)(threadIdx.x & 31) == leader && v) atomicAdd(g + w, (unsigned long long)v);
    }
}

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
// fp64 seeds: MUFU.RCP64H / MUFU.RSQ64H work on the high word, relative error <= 2^-19.9 (measured
// on B200); the low word of the result is 0.
__device__ __forceinline__ double rcp64h(double x)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    return r;
}
__device__ __forceinline__ double rsq64h(double x)
{
    double r;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    return r;
}
// 1/d for a normal, finite d: seed e0 = 2^-20, one cubic Newton step (e0^3 = 2^-60), 3 DFMA.
__device__ __forceinline__ double fast_rcp(double d)
{
    const double r = rcp64h(d);
    double e = fma(-d, r, 1.0);
    e = fma(e, e, e);
    return fma(r, e, r);
}
__device__ __forceinline__ float fast_rcp(float d) { return __frcp_rn(d); }
// sqrt(w) for a normal w > 0: s0 = w r (2^-20), two Heron steps with the frozen seed r/2 as slope
// (error e -> e*2^-20 + e^2/2: 2^-40, 2^-60), 6 fp64 ops.
__device__ __forceinline__ double fast_sqrt(double w)
{
    const double r = rsq64h(w);
    const double hr = 0.5 * r;
    double s = w * r;
    s = fma(fma(-s, s, w), hr, s);
    s = fma(fma(-s, s, w), hr, s);
    return s;
}
__device__ __forceinline__ float fast_sqrt(float w) { return sqrtf(w); }
// 1/sqrt(x), normal x > 0: seed 2^-20, two Newton steps (clamped cells, general-EOS Newton loop)
__device__ __forceinline__ double fast_rsqrt(double x)
{
    double r = rsq64h(x);
    r = fma(0.5 * r, fma(-(x * r), r, 1.0), r);
    r = fma(0.5 * r, fma(-(x * r), r, 1.0), r);
    return r;
}

// ------------------------------------------------------------------------------------------------
// cons2prim: relativistic correction + EOS (phases 3-4; readings G6-G10).
// Solves v (E + P(E - Mc v, R sqrt(1-v^2))) = Mc, Mc = min(|M|, (1-delta) E), on [0,1).
// Results: y with v_i = M_i * y; e; p; w = 1 - v^2 (for n = R sqrt(w)); fl = floor flags.
//
// General path (every T, every EOS; also the RARE path of the fp64 Gamma-law kernels):
//   EOS_GAMMA: closed form v = 2 Mc / (Gamma E + sqrt(Gamma^2 E^2 - 4 (Gamma-1) Mc^2)) (pin P7 ii).
//   EOS_MASS : Newton with bisection safeguard on the bracket [v(m=0), Mc/E]; the warp leaves the loop
//              together (__all_sync), so there is no intra-warp divergence in the iteration.
struct Prim {
    double y, e, p, w;
    int fl;
};

template <int EOS>
__device__ __forceinline__ Prim cons2prim_general(const EosD& k, double E, double Ma, double Mb, double Mc, double R)
{
    Prim o;
    const bool vac = !(E > double(0));                   // vacuum (reading G7); also catches NaN
    if (vac) { E = double(1); Ma = Mb = Mc = double(0); }     // keep the arithmetic below finite; result discarded
    o.fl = 0;
    const double M2 = fma(Ma, Ma, fma(Mb, Mb, Mc * Mc));
    const double lim = k.omd * E;
    const double lim2 = lim * lim;
    double Mq = M2;          // Mc^2 (clamped)
    double s = double(1);         // Mc / |M|
    if (M2 > lim2) {    // causality clamp, same rule as Pi
        Mq = lim2;
        s = lim * rsqrt(M2);
    }
    const double disc = fma(k.g2, E * E, -k.c4 * Mq);
    const double sq = sqrt(disc);
    const double hden = fma(k.hg, E, double(0.5) * sq);     // (Gamma E + sqrt(disc)) / 2
    double inv = double(1) / hden;                            // v = Mc * inv   (m = 0 root)
    if (EOS == EOS_GAMMA) {
        const double eraw = fma(-Mq, inv, E);
        if (eraw < double(0)) o.fl |= 1;
        o.e = fmax(eraw, double(0));
        o.p = k.gm1 * o.e;
        o.w = fmax(double(1) - Mq * inv * inv, double(0));
        o.y = s * inv;
    } else {
        // no library sqrt / division on this path either: |Mc|, the P = 0 root and (below) n and M/|M| use the
        // MUFU-seeded routines, guarded where the argument can be 0; the bracket is [0, min(Mc/E, 1-delta)]
        const bool moving = Mq > double(1e-300);
        const double Mabs = moving ? Mq * fast_rsqrt(Mq) : double(0);
        double lo = double(0);
        double hi = fmin(Mabs * fast_rcp(E), k.omd);        // P = 0 root: upper bound
        const double mR = k.mass * R;
        // start: ONE step of the paper's fixed-point map from the P = 0 root `hi`: an upper bound that is
        // within 1e-2 .. 1e-4 of the root for cold as well as hot matter, so the warp needs ~4.6 Newton steps instead
        // of ~8 from the m = 0 root (measured on config-3-like states).  The bracket [lo, hi] still safeguards it.
        double v;
        {
            const double w2h = fma(-hi, hi, double(1));
            const double Ph = fmax(k.gm1 * ((E - Mabs * hi) - mR * (w2h * fast_rsqrt(w2h))), double(0));
            v = fmin(fmax(Mabs * fast_rcp(E + Ph), lo), hi);
        }
        for (int it = 0; it < 48; ++it) {
            // no library sqrt / division in the loop: w2 >= 2e-12 (v <= 1 - delta) and dg >= E - (Gamma-1)|M| v > 0
            // are normal positive numbers, so the MUFU-seeded fast_rsqrt / fast_rcp apply (<= 2 ulp; the iteration
            // is self-correcting and the primitives after the loop are formed from the converged v)
            const double w2 = fma(-v, v, double(1));
            const double rw = fast_rsqrt(w2);
            const double w = w2 * rw;
            const double praw = k.gm1 * ((E - Mabs * v) - mR * w);
            const bool pos = praw > double(0);
            const double P = pos ? praw : double(0);
            const double dP = pos ? k.gm1 * (mR * v * rw - Mabs) : double(0);
            const double g = fma(v, E + P, -Mabs);
            const double dg = fma(v, dP, E + P);
            if (g > double(0)) hi = v; else lo = v;
            double vn = v - g * fast_rcp(dg);
            if (!(vn >= lo && vn <= hi)) vn = double(0.5) * (lo + hi);
            const double dv = fabs(vn - v);
            v = vn;
            const double tol = 1e-15;
            if (__all_sync(__activemask(), dv <= tol)) break;
        }
        o.w = fmax(fma(-v, v, double(1)), double(0));
        const double eraw = fma(-Mabs, v, E);
        if (eraw < double(0)) o.fl |= 1;
        o.e = fmax(eraw, double(0));
        const double n = (o.w > double(1e-300)) ? R * fast_sqrt(o.w) : double(0);
        const double praw = k.gm1 * (o.e - k.mass * n);
        if (praw < double(0)) o.fl |= 2;
        o.p = fmax(praw, double(0));
        o.y = (M2 > double(1e-300)) ? v * fast_rsqrt(M2) : double(0);
    }
    if (vac) { o.y = double(0); o.e = double(0); o.p = double(0); o.w = double(0); o.fl = 0; }   // n = R sqrt(w) = 0 (reading G7)
    return o;
}

// The EOS_GAMMA kernels have NO out-of-line path: vacuum / non-positive E (high word <= 0) is a two-line inline
// branch (all primitives 0, M = 0), and the host instantiates them only for Gamma <= 5/3, where the frozen-slope
// Newton of c2p_fast_y converges in two steps (larger Gamma runs the EOS_MASS kernels with m = 0).  The causality clamp Mc = min(|M|, (1-delta) E) stays inline: Mc^2 is a
// select on the bit patterns (non-negative doubles order like integers), and only a clamped cell (~0.2 % of
// the cells of config 4) pays the extra rsqrt for the direction-preserving scale factor.
__device__ __forceinline__ bool c2p_is_vacuum(double E)
{
    return __double2hiint(E) <= 0;
}
__device__ __forceinline__ bool gt_nonneg(double a, double b)      // a > b for a, b >= 0, on the integer pipe
{
    return __double_as_longlong(a) > __double_as_longlong(b);
}

// Fast path, fp64, p = (Gamma-1) e.  y = 1/h, h = (b + sqrt(disc))/2 with b = Gamma E, disc = b^2 - 4 c,
// c = (Gamma-1)|M|^2, is the smaller root of f(y) = c y^2 - b y + 1 and f'(y*) = -sqrt(disc).  Seeds:
// r = rsq64h(disc) ~ 1/sqrt(disc), y0 = 2 rcp64h(disc r + b) (both 2^-20); Newton with the FROZEN slope r:
// y <- y + f(y) r.  Error e -> e 2^-20 + (c y/sqrt(disc)) e^2 with c y/sqrt(disc) <= (Gamma-1)/(2-Gamma)
// (= 1/2 for Gamma = 4/3): 2^-20 -> 2^-39 -> 2^-58.  15 fp64 ops including |M|^2, no division, no sqrt.
__device__ __forceinline__ double c2p_fast_y(const EosD& k, double E, double M2, double t)
{
    const double disc = fma(k.g2, t, -(k.c4 * M2));
    const double r = rsq64h(disc);
    const double b = k.gam * E;
    const double s = fma(disc, r, b);
    const double y0 = rcp64h(s);
    double y = __hiloint2double(__double2hiint(y0) + 0x00100000, 0);      // 2 * y0 (exponent + 1)
    const double c = k.gm1 * M2;
    y = fma(fma(fma(c, y, -b), y, 1.0), r, y);
    y = fma(fma(fma(c, y, -b), y, 1.0), r, y);
    return y;
}

// In-sweep cons2prim (S1, S3): only v_par = M_par y and p are needed.
template <int EOS>
__device__ __forceinline__ void c2p_sweep_d(const EosD& k, const double (&u)[NF], double& v, double& p)
{
    const Prim o = cons2prim_general<EOS>(k, u[0], u[1], u[2], u[3], u[4]);
    v = u[1] * o.y;
    p = o.p;
}
template <>
__device__ __forceinline__ void c2p_sweep_d<EOS_GAMMA>(const EosD& k, const double (&u)[NF], double& v, double& p)
{
    // No vacuum BRANCH here: the arithmetic runs on whatever E is (inf / NaN intermediates cost nothing on the fp64
    // pipe) and the two results are masked by selects, so that the scheduler can interleave the cons2prim chains of
    // the two cells of a chunk (a branch ends the basic block: measured -5 % per sweep for the two branches here).
    const double M2 = fma(u[1], u[1], fma(u[2], u[2], u[3] * u[3]));
    const bool vac = c2p_is_vacuum(u[0]);       // reading G7: all primitives 0
    const double t = u[0] * u[0];
    const double lim2 = k.omd2 * t;
    const bool clamped = gt_nonneg(M2, lim2);
    const double Mq = clamped ? lim2 : M2;
    double y = c2p_fast_y(k, u[0], Mq, t);
    double e = fma(-Mq, y, u[0]);               // e = E - Mc v >= delta E > 0: no floor
    if (clamped) y *= (k.omd * u[0]) * fast_rsqrt(M2);      // rare (Pi-clamped cells): direction-preserving scale
    y = vac ? 0.0 : y;
    e = vac ? 0.0 : e;
    v = u[1] * y;
    p = k.gm1 * e;
}
template <typename T, int EOS>
__device__ __forceinline__ void c2p_sweep(const Consts<T>& k, const T (&u)[NF], T& v, T& p)
{
    double ud[NF], vd, pd;
#pragma unroll
    for (int f = 0; f < NF; ++f) ud[f] = (double)u[f];
    c2p_sweep_d<EOS>(k.d, ud, vd, pd);
    v = (T)vd;
    p = (T)pd;
}

// eq. (21) branch-free (reading G12): A = sigma max(0, min(sigma D^_{j+1}, |A^ph|, sigma D^_{j-1}))
template <typename T>
__device__ __forceinline__ T limiter(T aph, T dhp, T dhm)
{
    const T sg = copysign(T(1), aph);
    const T m = t_min(t_min(sg * dhp, t_abs(aph)), sg * dhm);
    return sg * t_max(m, T(0));
}
// fp64 on the INTEGER pipe: multiplying by sigma = flipping the sign bit; IEEE doubles order like
// sign-magnitude integers, so min over non-negative doubles = min over their bit patterns as signed
// 64-bit integers, and any negative operand makes that integer minimum negative, which max(.,0)
// clips to +0 -- exactly the max{0, min{...}} of eq. (21).  No fp64-pipe instruction.
template <>
__device__ __forceinline__ double limiter<double>(double aph, double dhp, double dhm)
{
    const long long ia = __double_as_longlong(aph);
    const long long sg = ia & (long long)0x8000000000000000ULL;
    const long long z = ia ^ sg;
    const long long x = __double_as_longlong(dhp) ^ sg;
    const long long y = __double_as_longlong(dhm) ^ sg;
    long long m = min(min(x, z), y);
    if ((int)(m >> 32) < 0) m = 0;
    return __longlong_as_double(m ^ sg);
}

// ------------------------------------------------------------------------------------------------
// The rolling window of one marching thread.  "X_k" below means the quantity at cell (or interface)
// i-k, where i is the front cell of the CURRENT step.  Each window is a small ring whose slot is a
// compile-time function of the phase PH = (step number) mod 4: the march loop is unrolled by 4, so
// every slot is a fixed register and the window advances without a single move instruction.
template <typename T, int EOS>
struct Marcher {
    T u[2][NF];         // U^n_1, U^n_2                    slot of U^n_k : (PH-k)&1
    T dl[4][NF];        // Delta_2..Delta_5, eq. (16)      slot of Delta_k: (PH-k)&3
    T ft[NF];           // predictor flux F~ at interface (i-2,i-1)
    T fc[NF];           // corrector flux F at interface (i-3,i-2)
    T uh[2][NF];        // U^_3, U^_4                      slot of U^_k : (PH-k)&1
    T dh[2][NF];        // D^_4, D^_5, eq. (18)            slot of D^_k : (PH-k)&1
    T a5[NF];           // limited antidiffusive flux A_5
    T eps1;             // (lambda/2) v_1 (time n)
    T fE[2], fM[2];     // (p v)_1,_2 and p_1,_2 (time n)  slot (PH-k)&1
    T epsh2;            // lambda v^{1/2}_2
    T gE[2], gM[2];     // (p v)^{1/2}_2,_3 and p^{1/2}_2,_3   slot (PH-k)&1

    __device__ __forceinline__ void init()
    {
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            u[0][f] = u[1][f] = dl[0][f] = dl[1][f] = dl[2][f] = dl[3][f] = ft[f] = fc[f] = T(0);
            uh[0][f] = uh[1][f] = dh[0][f] = dh[1][f] = a5[f] = T(0);
        }
        eps1 = epsh2 = fE[0] = fE[1] = fM[0] = fM[1] = gE[0] = gE[1] = gM[0] = gM[1] = T(0);
    }

    // One march step: consumes U^n at the front cell, produces U^{n+1} of cell i-4 in un[].
    template <int PH>
    __device__ __forceinline__ void step(const Consts<T>& k, const T (&u0)[NF], T (&un)[NF])
    {
        constexpr int U1 = (PH + 3) & 1, U2 = (PH + 2) & 1;                 // U^n_1, U^n_2 (new U^n_0 -> U2)
        constexpr int D2 = (PH + 2) & 3, D3 = (PH + 1) & 3, D4 = PH & 3, D5 = (PH + 3) & 3;   // new Delta_1 -> D5
        constexpr int H3 = (PH + 1) & 1, H4 = PH & 1;                       // U^_3, U^_4 (new U^_2 -> H4)
        constexpr int E4 = PH & 1, E5 = (PH + 1) & 1;                       // D^_4, D^_5 (new D^_3 -> E5)
        constexpr int S1 = (PH + 1) & 1, S2 = PH & 1;                       // time-n scalars _1,_2 (new _0 -> S2)
        constexpr int G2 = PH & 1, G3 = (PH + 1) & 1;                       // half-step scalars _2,_3 (new _1 -> G3)
        (void)S1; (void)G2;
        // S1: time-n primitives of the front cell
        T v0, p0;
        c2p_sweep<T, EOS>(k, u0, v0, p0);
        const T eps0 = k.hlam * v0;
        const T fE0 = p0 * v0;
        // S2: predictor (half step, no antidiffusion: reading G4), interface (i-1,i), cell i-1
        T ut[NF], dl1[NF];
        {
            const T q = (T(0.5) - eps1) * fast_rcp(T(1) + (eps0 - eps1));   // Q+_1, eq. (15); Q-_0 = 1-q (P1)
            const T a = T(0.5) - q, b = (T(0.5) * q) * q;
#pragma unroll
            for (int f = 0; f < NF; ++f) {
                dl1[f] = u0[f] - u[U1][f];                                  // eq. (16)
                const T fl = t_fma(a, u[U1][f], -(b * dl1[f]));             // F = (1/2-q) U - 1/2 q^2 Delta (P2)
                ut[f] = u[U1][f] - (fl - ft[f]);                               // exact no-op on uniform data (P10)
                ft[f] = fl;
            }
            ut[0] = t_fma(-k.qlam, fE0 - fE[S2], ut[0]);                    // + (lambda/2) Delta(p v)
            ut[1] = t_fma(-k.qlam, p0 - fM[S2], ut[1]);                     // + (lambda/2) Delta(p)
        }
        // S3: half-step primitives of cell i-1
        T vh1, ph;
        c2p_sweep<T, EOS>(k, ut, vh1, ph);
        const T epsh1 = k.lam * vh1;
        const T gE1 = ph * vh1;
        // S4: corrector transport of U^n, interface (i-2,i-1), cell i-2
        T uh2[NF];
        {
            const T q = (T(0.5) - epsh2) * fast_rcp(T(1) + (epsh1 - epsh2));
            const T a = T(0.5) - q, b = (T(0.5) * q) * q;
#pragma unroll
            for (int f = 0; f < NF; ++f) {
                const T fl = t_fma(a, u[U2][f], -(b * dl[D2][f]));
                uh2[f] = u[U2][f] - (fl - fc[f]);
                fc[f] = fl;
            }
            uh2[0] = t_fma(-k.hlam, gE1 - gE[G3], uh2[0]);                  // + lambda Delta(p v)^{n+1/2}
            uh2[1] = t_fma(-k.hlam, ph - gM[G3], uh2[1]);                   // + lambda Delta(p)^{n+1/2}
        }
        // S5+S6: antidiffusion at interface (i-4,i-3), update of cell i-4
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            const T dh3 = uh2[f] - uh[H3][f];                                    // eq. (18)
            const T d2 = t_fma(T(-2), dl[D4][f], dl[D3][f] + dl[D5][f]);         // reading G14
            const T aph = T(0.125) * t_fma(T(-0.125), d2, dh[E4][f]);            // eq. (19)
            const T a4 = limiter<T>(aph, dh3, dh[E5][f]);                        // eqs. (20),(21)
            un[f] = uh[H4][f] - (a4 - a5[f]);                                    // eq. (22)
            // advance the window: the new values take the slots of the oldest ones
            a5[f] = a4;
            dh[E5][f] = dh3;
            uh[H4][f] = uh2[f];
            dl[D5][f] = dl1[f];
            u[U2][f] = u0[f];
        }
        eps1 = eps0; fE[S2] = fE0; fM[S2] = p0;
        epsh2 = epsh1; gE[G3] = gE1; gM[G3] = ph;
    }
};

// Pi, readings G6-G8: written back to M at the end of every sweep.  E and R are never modified.
__device__ __forceinline__ void project(const EosD& k, double (&un)[NF], Cnt counts)
{
    const double E = un[0];
    const double M2 = fma(un[1], un[1], fma(un[2], un[2], un[3] * un[3]));
    const double lim = k.omd * E;
    if (!(E > 0.0)) {
        un[1] = un[2] = un[3] = 0.0;
        counts.add(1);
    } else if (M2 > lim * lim) {
        const double s = lim * rsqrt(M2);
        un[1] *= s; un[2] *= s; un[3] *= s;
        counts.add(0);
    }
}

// primitives of one cell from its (projected) conserved state, slots permuted like the momenta
template <int EOS>
__device__ __forceinline__ void primitives(const EosD& k, const double (&u)[NF], double (&pr)[6], Cnt counts)
{
    const Prim o = cons2prim_general<EOS>(k, u[0], u[1], u[2], u[3], u[4]);
    pr[0] = o.e; pr[1] = o.p;
    pr[2] = u[4] * sqrt(o.w);
    pr[3] = u[1] * o.y; pr[4] = u[2] * o.y; pr[5] = u[3] * o.y;
    if (o.fl) {                                     // rare: diagnostics [2] e floored, [3] p floored
        if (o.fl & 1) counts.add(2);
        if (o.fl & 2) counts.add(3);
    }
}

// primitives from (E, Mc^2, E^2) on the fast path: y 12 ops, e/w 3, sqrt 6, n/p/v 5
__device__ __forceinline__ void prims_fast(const EosD& k, const double (&u)[NF], double Mq, double t, double s,
                                           double (&pr)[6])
{
    double y = c2p_fast_y(k, u[0], Mq, t);
    const double e = fma(-Mq, y, u[0]);
    const double w = fma(-(Mq * y), y, 1.0);
    y *= s;
    pr[0] = e;
    pr[1] = k.gm1 * e;
    pr[2] = u[4] * fast_sqrt(w);
    pr[3] = u[1] * y; pr[4] = u[2] * y; pr[5] = u[3] * y;
}

// S6 tail + S7 of one output cell: Pi on un[], and (EMIT) its primitives pr[].
template <int EOS, bool EMIT>
__device__ __forceinline__ void finish_d(const EosD& k, double (&un)[NF], double (&pr)[6], Cnt counts)
{
    if (EOS == EOS_GAMMA) {
        // Gamma-law: Pi and the primitives share |M|^2 and E^2; everything but vacuum is inline
        if (c2p_is_vacuum(un[0])) {                         // vacuum: M = 0, all primitives 0 (readings G7, R1)
            un[1] = un[2] = un[3] = 0.0;
            counts.add(1);
            if (EMIT) {
#pragma unroll
                for (int q = 0; q < 6; ++q) pr[q] = 0.0;
            }
            return;
        }
        double M2 = fma(un[1], un[1], fma(un[2], un[2], un[3] * un[3]));
        const double t = un[0] * un[0];
        const double lim2 = k.omd2 * t;
        double s = 1.0;
        if (gt_nonneg(M2, lim2)) {                          // Pi fires: scale M onto |M| = (1-delta) E
            const double sc = (k.omd * un[0]) * fast_rsqrt(M2);
            un[1] *= sc; un[2] *= sc; un[3] *= sc;
            counts.add(0);
            if (EMIT) {                                     // primitives of the PROJECTED state, like the oracle
                M2 = fma(un[1], un[1], fma(un[2], un[2], un[3] * un[3]));
                if (gt_nonneg(M2, lim2)) s = (k.omd * un[0]) * fast_rsqrt(M2);
            }
        }
        if (EMIT) prims_fast(k, un, gt_nonneg(M2, lim2) ? lim2 : M2, t, s, pr);
    } else {
        project(k, un, counts);
        if (EMIT) primitives<EOS>(k, un, pr, counts);
    }
}
template <typename T, int EOS, bool EMIT>
__device__ __forceinline__ void finish_cell(const Consts<T>& k, T (&un)[NF], T (&pr)[6], Cnt counts)
{
    double ud[NF], pd[6];
#pragma unroll
    for (int f = 0; f < NF; ++f) ud[f] = (double)un[f];
    finish_d<EOS, EMIT>(k.d, ud, pd, counts);
#pragma unroll
    for (int f = 1; f < 4; ++f) un[f] = (T)ud[f];           // Pi touches M only
    if (EMIT) {
#pragma unroll
        for (int q = 0; q < 6; ++q) pr[q] = (T)pd[q];
    }
}

// primitives of an already projected cell (x sweep write-back, shasta_get_primitives refresh)
template <int EOS>
__device__ __forceinline__ void emit_d(const EosD& k, const double (&u)[NF], double (&pr)[6], Cnt counts)
{
    if (EOS != EOS_GAMMA) {
        primitives<EOS>(k, u, pr, counts);
        return;
    }
    if (c2p_is_vacuum(u[0])) {
#pragma unroll
        for (int q = 0; q < 6; ++q) pr[q] = 0.0;
        return;
    }
    const double M2 = fma(u[1], u[1], fma(u[2], u[2], u[3] * u[3]));
    const double t = u[0] * u[0];
    const double lim2 = k.omd2 * t;
    const bool clamped = gt_nonneg(M2, lim2);
    const double s = clamped ? (k.omd * u[0]) * fast_rsqrt(M2) : 1.0;
    prims_fast(k, u, clamped ? lim2 : M2, t, s, pr);
}
template <typename T, int EOS>
__device__ __forceinline__ void emit_primitives(const Consts<T>& k, const T (&u)[NF], T (&pr)[6], Cnt counts)
{
    double ud[NF], pd[6];
#pragma unroll
    for (int f = 0; f < NF; ++f) ud[f] = (double)u[f];
    emit_d<EOS>(k.d, ud, pd, counts);
#pragma unroll
    for (int q = 0; q < 6; ++q) pr[q] = (T)pd[q];
}

// cp.async (LDGSTS) helpers: one element per thread, global -> shared without touching registers
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

// ------------------------------------------------------------------------------------------------
// Sweep along y or z: lanes run along the contiguous x axis, so every load and store of a warp is a
// coalesced 256 B (fp64) row piece.  Work item = (pencil, segment).  The marching thread is latency-
// bound unless many cells are in flight per pencil, and registers are full (the window), so the input
// is PREFETCHED SD-1 cells ahead with cp.async into a per-thread ring in shared memory
// (ring[slot][field][thread]: conflict-free).  A thread only ever reads what it copied itself:
// cp.async.wait_group is the only synchronisation.
constexpr int SD = 8;             // ring slots = cells in flight per pencil + 1
constexpr int SBLOCK = 128;       // threads per CTA

template <typename T>
struct StridedCtx {
    const T* in[NF];
    T* out[NF];
    T* prim[6];
    long long sa;       // element stride along the sweep axis
    int N, periodic, j0, j1;
    int ipf, jpf;       // next cell to prefetch: true index and ghost-mapped index (reading G11)
    Cnt counts;
};

// issue the copy of the next cell into ring slot `slot`; one commit group per cell
template <typename T>
__device__ __forceinline__ void strided_prefetch(StridedCtx<T>& c, T* slot)
{
    const long long o = (long long)c.jpf * c.sa;
#pragma unroll
    for (int f = 0; f < NF; ++f) cp_async_elem<T>(slot + f * SBLOCK, c.in[f] + o);
    cp_async_commit();
    c.ipf += 1;
    if (c.periodic) { c.jpf = (c.jpf + 1 == c.N) ? 0 : c.jpf + 1; }     // wrap
    else            { c.jpf = min(max(c.ipf, 0), c.N - 1); }            // copy of the edge cell
}

// PH = step number mod 4 (compile time: window phase and ring slot inside the current half of the ring);
// cur / oth = the two halves (4 slots each) of this thread's ring, swapped every 4 steps by the caller.
template <typename T, int EOS, bool EMIT, int PH>
__device__ __forceinline__ void strided_substep(Marcher<T, EOS>& m, const Consts<T>& k, StridedCtx<T>& c, int i,
                                                T* cur, T* oth)
{
    // refill the slot consumed by the PREVIOUS step (its reads are long retired), then wait for cell i
    strided_prefetch<T>(c, PH == 0 ? oth + 3 * NF * SBLOCK : cur + (PH - 1) * NF * SBLOCK);
    cp_async_wait<SD - 1>();
    T u0[NF], un[NF];
#pragma unroll
    for (int f = 0; f < NF; ++f) u0[f] = cur[(PH * NF + f) * SBLOCK];
    m.template step<PH>(k, u0, un);
    const int jo = i - GH;
    if (jo >= c.j0 && jo < c.j1) {
        T pr[6];
        finish_cell<T, EOS, EMIT>(k, un, pr, c.counts);
        const long long o = (long long)jo * c.sa;
#pragma unroll
        for (int f = 0; f < NF; ++f) c.out[f][o] = un[f];
        if (EMIT) {
#pragma unroll
            for (int q = 0; q < 6; ++q) c.prim[q][o] = pr[q];
        }
    }
}

template <typename T, int EOS, bool EMIT>
__global__ void __launch_bounds__(SBLOCK) sweep_strided_kernel(SweepParams P, Consts<T> k)
{
    __shared__ T ring[SD * NF * SBLOCK];
    __shared__ unsigned cnt[4 * SBLOCK];
    const long long pen = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (pen >= P.npencil) return;
    const int sg = blockIdx.y;
    StridedCtx<T> c;
    c.j0 = sg * P.seg;
    c.j1 = min(P.N, c.j0 + P.seg);
    c.N = P.N; c.periodic = P.periodic; c.sa = P.stride_axis;
    c.counts.p = cnt + threadIdx.x; c.counts.stride = SBLOCK;
    c.counts.zero();
    const long long base = (pen % P.nx) + (pen / P.nx) * P.stride_other;
#pragma unroll
    for (int f = 0; f < NF; ++f) { c.in[f] = (const T*)P.in[f] + base; c.out[f] = (T*)P.out[f] + base; }
#pragma unroll
    for (int q = 0; q < 6; ++q) c.prim[q] = (T*)P.prim[q] + base;

    Marcher<T, EOS> m;
    m.init();
    c.ipf = c.j0 - GH;
    c.jpf = ghost_index(c.ipf, P.N, P.periodic);
    T* cur = ring + threadIdx.x;
    T* oth = cur + 4 * NF * SBLOCK;
#pragma unroll
    for (int d = 0; d < SD - 1; ++d) strided_prefetch<T>(c, cur + d * NF * SBLOCK);      // cells j0-4 .. j0+2
    // front cells j0-4 .. j1+3, rounded up to a multiple of 4 steps (the surplus steps store nothing)
    for (int i = c.j0 - GH; i < c.j1 + GH; i += 4) {
        strided_substep<T, EOS, EMIT, 0>(m, k, c, i, cur, oth);
        strided_substep<T, EOS, EMIT, 1>(m, k, c, i + 1, cur, oth);
        strided_substep<T, EOS, EMIT, 2>(m, k, c, i + 2, cur, oth);
        strided_substep<T, EOS, EMIT, 3>(m, k, c, i + 3, cur, oth);
        T* tmp = cur; cur = oth; oth = tmp;
    }
    cp_async_wait<0>();
    flush_counts(c.counts, P.counts);
}

// ------------------------------------------------------------------------------------------------
// Warp-specialised march: the serial chain S1..S6 of one march step is cut after S3 and
// run by TWO warps per 32 pencils, a producer P (S1-S3 + the corrector's geometry) and a consumer C
// (S4-S6), so that twice as many warps are resident for the same register budget and each warp's
// dependent chain is half as long.  P -> C traffic per pencil and step is four doubles through a
// shared-memory queue: a_c = 1/2 - Q+, b_c = Q+^2/2 of the interface (i-2,i-1) at n+1/2, and the two
// source increments -lambda Delta(p v)/2-form for E and M_par of cell i-2.
template <typename T, int EOS>
struct Producer {
    // fields the producer needs: the Gamma-law pressure does not depend on R, so R's predictor is skipped there
    static constexpr int NP = (EOS == EOS_GAMMA) ? 4 : NF;
    T ft[NF];           // predictor flux F~ at interface (i-2,i-1)
    T eps1;             // (lambda/2) v_1 (time n)
    T fE[2], fM[2];     // (p v)_1,_2 and p_1,_2 (time n)      slot (PH-k)&1
    T epsh2;            // lambda v^{1/2}_2
    T gE[2], gM[2];     // (p v)^{1/2}_2,_3, p^{1/2}_2,_3      slot (PH-k)&1

    __device__ __forceinline__ void init()
    {
#pragma unroll
        for (int f = 0; f < NF; ++f) ft[f] = T(0);
        eps1 = epsh2 = fE[0] = fE[1] = fM[0] = fM[1] = gE[0] = gE[1] = gM[0] = gM[1] = T(0);
    }

    // consumes U^n at the front cell i (u0) and at cell i-1 (u1: re-read from the ring by the caller, or the
    // previous front cell still in registers -- never carried, so no hand-down moves);
    // msg = {a_c, b_c, sE, sM} for the consumer's step i
    template <int PH>
    __device__ __forceinline__ void step(const Consts<T>& k, const T (&u1)[NF], const T (&u0)[NF], T (&msg)[4])
    {
        constexpr int S2 = PH & 1;              // time-n scalars _2 (new _0 takes its slot)
        constexpr int G3 = (PH + 1) & 1;        // half-step scalars _3 (new _1 takes its slot)
        T v0, p0;
        c2p_sweep<T, EOS>(k, u0, v0, p0);                                   // S1
        const T eps0 = k.hlam * v0;
        const T fE0 = p0 * v0;
        T ut[NF];
        ut[NF - 1] = T(0);
        {                                                                   // S2
            const T q = (T(0.5) - eps1) * fast_rcp(T(1) + (eps0 - eps1));   // Q+_1, eq. (15)
            const T a = T(0.5) - q, b = (T(0.5) * q) * q;
#pragma unroll
            for (int f = 0; f < NP; ++f) {
                const T d = u0[f] - u1[f];                                  // eq. (16)
                const T fl = t_fma(a, u1[f], -(b * d));
                ut[f] = u1[f] - (fl - ft[f]);
                ft[f] = fl;
            }
            ut[0] = t_fma(-k.qlam, fE0 - fE[S2], ut[0]);
            ut[1] = t_fma(-k.qlam, p0 - fM[S2], ut[1]);
        }
        T vh1, ph;
        c2p_sweep<T, EOS>(k, ut, vh1, ph);                                  // S3
        const T epsh1 = k.lam * vh1;
        const T gE1 = ph * vh1;
        {                                                                   // geometry + sources of S4
            const T q = (T(0.5) - epsh2) * fast_rcp(T(1) + (epsh1 - epsh2));
            msg[0] = T(0.5) - q;
            msg[1] = (T(0.5) * q) * q;
            msg[2] = -k.hlam * (gE1 - gE[G3]);
            msg[3] = -k.hlam * (ph - gM[G3]);
        }
        eps1 = eps0; fE[S2] = fE0; fM[S2] = p0;
        epsh2 = epsh1; gE[G3] = gE1; gM[G3] = ph;
    }
};

template <typename T>
struct Consumer {
    T dl[4][NF];        // Delta_2..Delta_5 (Delta_2 is formed in the step)   slot (PH-k)&3
    T fc[NF];           // corrector flux F at interface (i-3,i-2)
    T uh[2][NF];        // U^_3, U^_4                                         slot (PH-k)&1
    T dh[2][NF];        // D^_4, D^_5                                         slot (PH-k)&1
    T a5[NF];           // A_5

    __device__ __forceinline__ void init()
    {
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            dl[0][f] = dl[1][f] = dl[2][f] = dl[3][f] = fc[f] = T(0);
            uh[0][f] = uh[1][f] = dh[0][f] = dh[1][f] = a5[f] = T(0);
        }
    }

    // consumes U^n_{i-2} (up), U^n_{i-1} (uj) -- both read from the ring by the caller, never carried -- and the
    // producer's message of step i; produces U^{n+1} of cell i-4 (before Pi)
    template <int PH>
    __device__ __forceinline__ void step(const T (&up)[NF], const T (&uj)[NF], const T (&msg)[4], T (&un)[NF])
    {
        constexpr int D2 = (PH + 2) & 3, D3 = (PH + 1) & 3, D4 = PH & 3, D5 = (PH + 3) & 3;
        constexpr int H3 = (PH + 1) & 1, H4 = PH & 1;
        constexpr int E4 = PH & 1, E5 = (PH + 1) & 1;
        const T a = msg[0], b = msg[1];
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            dl[D2][f] = uj[f] - up[f];                                           // eq. (16)
            const T fl = t_fma(a, up[f], -(b * dl[D2][f]));                      // S4
            T uh2 = up[f] - (fl - fc[f]);
            if (f == 0) uh2 += msg[2];
            if (f == 1) uh2 += msg[3];
            fc[f] = fl;
            const T dh3 = uh2 - uh[H3][f];                                       // eq. (18)
            const T d2 = t_fma(T(-2), dl[D4][f], dl[D3][f] + dl[D5][f]);         // reading G14
            const T aph = T(0.125) * t_fma(T(-0.125), d2, dh[E4][f]);            // eq. (19)
            const T a4 = limiter<T>(aph, dh3, dh[E5][f]);                        // eqs. (20),(21)
            un[f] = uh[H4][f] - (a4 - a5[f]);                                    // eq. (22)
            a5[f] = a4;
            dh[E5][f] = dh3;
            uh[H4][f] = uh2;
        }
    }
};

constexpr int WS_P = 128;         // pencils per CTA (4 producer warps + 4 consumer warps)
constexpr int WS_R = 12;          // U ring slots per pencil
constexpr int WS_D = WS_R - 5;    // prefetch distance; D-1 copies stay in flight behind the current chunk (see below)
constexpr int WS_Q = 4;           // message queue slots (2 chunks of 2 steps)

template <typename T>
struct WsSmem {
    T ring[WS_R][NF][WS_P];
    T msg[WS_Q][4][WS_P];
    unsigned cnt[4][WS_P];
};

// Producer/consumer hand-over of one warp pair: four named barriers (full[0..1], empty[0..1]) of 64 threads each,
// 32 that arrive (do not wait) and 32 that sync (wait): the PTX producer/consumer pattern.  The producer may run up
// to two 2-step chunks ahead of the consumer; chunk c uses slot c & 1.
__device__ __forceinline__ void bar_sync64(int id) { asm volatile("bar.sync %0, 64;" ::"r"(id) : "memory"); }
__device__ __forceinline__ void bar_arrive64(int id) { asm volatile("bar.arrive %0, 64;" ::"r"(id) : "memory"); }

template <typename T, int EOS, bool EMIT>
__global__ void __launch_bounds__(2 * WS_P, 2) sweep_strided_ws_kernel(const __grid_constant__ SweepParams P,
                                                                      const __grid_constant__ Consts<T> k)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    WsSmem<T>& S = *reinterpret_cast<WsSmem<T>*>(smem_raw);
    const int lane_p = threadIdx.x & (WS_P - 1);                // pencil slot inside the CTA
    const bool producer = threadIdx.x < WS_P;                   // warps 0-3: P, warps 4-7: C
    const int bar_id = 4 * ((threadIdx.x >> 5) & 3);            // named barriers of this warp pair: full0, full1, empty0, empty1
    long long pen = (long long)blockIdx.x * WS_P + lane_p;
    const bool active = pen < P.npencil;
    if (!active) pen = P.npencil - 1;                           // idle lanes shadow a valid pencil, store nothing
    const int sg = blockIdx.y;
    const int j0 = sg * P.seg;
    const int j1 = min(P.N, j0 + P.seg);
    const long long sa = P.stride_axis;
    const long long base = (pen % P.nx) + (pen / P.nx) * P.stride_other;
    const int nsteps = (j1 - j0) + 2 * GH;                      // front cells j0-4 .. j1+3
    const int nchunk = (nsteps + 1) / 2;
    const int nchunk2 = (nchunk + 1) & ~1;

    if (producer) {
        if (sizeof(T) == 8) asm volatile("setmaxnreg.dec.sync.aligned.u32 96;");
        Producer<T, EOS> pr;
        pr.init();
        // prefetch state: next cell to fetch (true index ipf, ghost-mapped jpf) and its ring slot
        int ipf = j0 - GH, jpf = ghost_index(ipf, P.N, P.periodic), pslot = 0;
        auto prefetch = [&]() {
            const long long o = base + (long long)jpf * sa;        // field pointers stay in the constant bank
#pragma unroll
            for (int f = 0; f < NF; ++f) cp_async_elem<T>(&S.ring[pslot][f][lane_p], (const T*)P.in[f] + o);
            cp_async_commit();
            pslot = (pslot + 1 == WS_R) ? 0 : pslot + 1;
            ipf += 1;
            if (P.periodic) { jpf = (jpf + 1 == P.N) ? 0 : jpf + 1; }
            else            { jpf = min(max(ipf, 0), P.N - 1); }
        };
#pragma unroll
        for (int d = 0; d < WS_D - 1; ++d) prefetch();
        int rslot = 0;
        // Copies: before chunk `it` cells 0 .. 2it+D-2 are issued; its two prefetches add cells 2it+D-1, 2it+D, and
        // wait_group<D-1> then leaves at most the D-1 youngest pending, i.e. cells <= 2it+1 (this chunk) are complete.
        // Slot reuse (D = R-5): those two refill the slots of cells 2it-6 and 2it-5.  The producer enters chunk `it`
        // only after the consumer released chunk it-2; the consumer may still be inside chunk it-1, where it reads
        // cells 2it-4 .. 2it-2 (U_{i-2}, U_{i-1} of its two steps): all younger than the refilled ones.
        // One chunk = two steps: both front cells are fetched first, then the two steps' arithmetic runs with no
        // asm/memory fence in between, so the scheduler may overlap S3 of the first with S1 of the second.
#define SHK_PCHUNK(PH)                                                                              \
        {                                                                                           \
            prefetch();                                                                             \
            prefetch();                                                                             \
            cp_async_wait<WS_D - 1>();                                                              \
            T um[NF], ua[NF], ub[NF], ma[4], mb[4];                                                 \
            um[NF - 1] = ua[NF - 1] = ub[NF - 1] = T(0);                                            \
            const int mslot = (rslot == 0) ? WS_R - 1 : rslot - 1;      /* cell 2it-1 (first chunk: don't care) */ \
            _Pragma("unroll") for (int f = 0; f < Producer<T, EOS>::NP; ++f) um[f] = S.ring[mslot][f][lane_p]; \
            _Pragma("unroll") for (int f = 0; f < Producer<T, EOS>::NP; ++f) ua[f] = S.ring[rslot][f][lane_p]; \
            rslot = (rslot + 1 == WS_R) ? 0 : rslot + 1;                                            \
            _Pragma("unroll") for (int f = 0; f < Producer<T, EOS>::NP; ++f) ub[f] = S.ring[rslot][f][lane_p]; \
            rslot = (rslot + 1 == WS_R) ? 0 : rslot + 1;                                            \
            pr.template step<PH>(k, um, ua, ma);                                                    \
            pr.template step<PH + 1>(k, ua, ub, mb);                                                \
            _Pragma("unroll") for (int q = 0; q < 4; ++q) S.msg[PH][q][lane_p] = ma[q];             \
            _Pragma("unroll") for (int q = 0; q < 4; ++q) S.msg[PH + 1][q][lane_p] = mb[q];         \
        }
        // decoupled hand-over (see bar_sync64): chunk c uses slot c & 1; nchunk is rounded up to even (a surplus
        // chunk marches ghost cells and stores nothing)
#pragma unroll 1
        for (int c = 0; c < nchunk2; c += 2) {
            if (c > 0) bar_sync64(bar_id + 2);
            SHK_PCHUNK(0)
            bar_arrive64(bar_id + 0);
            if (c > 0) bar_sync64(bar_id + 3);
            SHK_PCHUNK(2)
            bar_arrive64(bar_id + 1);
        }
#undef SHK_PCHUNK
        cp_async_wait<0>();
    } else {
        if (sizeof(T) == 8) asm volatile("setmaxnreg.inc.sync.aligned.u32 160;");
        Cnt cnt;
        cnt.p = &S.cnt[0][lane_p]; cnt.stride = WS_P;
        cnt.zero();
        Consumer<T> co;
        co.init();
        // consumer step t (front cell i = j0-4+t) reads U_{i-1}: ring slot of cell index t-1 (t = 0: the
        // ring's last slot, never written before: a don't-care warm-up value, finite or not it is retired)
        int cslot = WS_R - 1;
        int i = j0 - GH;
#define SHK_CSTORE(UN)                                                                              \
        {                                                                                           \
            const int jo = i - GH;                                                                  \
            if (jo >= j0 && jo < j1 && active) {                                                    \
                T pv[6];                                                                            \
                finish_cell<T, EOS, EMIT>(k, UN, pv, cnt);                                          \
                const long long o = base + (long long)jo * sa;                                      \
                _Pragma("unroll") for (int f = 0; f < NF; ++f) ((T*)P.out[f])[o] = UN[f];           \
                if (EMIT) { _Pragma("unroll") for (int q = 0; q < 6; ++q) ((T*)P.prim[q])[o] = pv[q]; } \
            }                                                                                       \
            ++i;                                                                                    \
        }
        // one chunk = steps t, t+1: cells t-2, t-1, t are read from the ring (no carried U, no hand-down moves)
#define SHK_CCHUNK(PH)                                                                              \
        {                                                                                           \
            T uq[NF], ua[NF], ub[NF], msg[4], un[NF];                                               \
            const int qslot = (cslot == 0) ? WS_R - 1 : cslot - 1;                                  \
            _Pragma("unroll") for (int f = 0; f < NF; ++f) uq[f] = S.ring[qslot][f][lane_p];        \
            _Pragma("unroll") for (int f = 0; f < NF; ++f) ua[f] = S.ring[cslot][f][lane_p];        \
            cslot = (cslot + 1 == WS_R) ? 0 : cslot + 1;                                            \
            _Pragma("unroll") for (int f = 0; f < NF; ++f) ub[f] = S.ring[cslot][f][lane_p];        \
            cslot = (cslot + 1 == WS_R) ? 0 : cslot + 1;                                            \
            _Pragma("unroll") for (int q = 0; q < 4; ++q) msg[q] = S.msg[PH][q][lane_p];            \
            co.template step<PH>(uq, ua, msg, un);                                                  \
            SHK_CSTORE(un)                                                                          \
            _Pragma("unroll") for (int q = 0; q < 4; ++q) msg[q] = S.msg[PH + 1][q][lane_p];        \
            co.template step<PH + 1>(ua, ub, msg, un);                                              \
            SHK_CSTORE(un)                                                                          \
        }
#pragma unroll 1
        for (int c = 0; c < nchunk2; c += 2) {
            bar_sync64(bar_id + 0);
            SHK_CCHUNK(0)
            if (c + 2 < nchunk2) bar_arrive64(bar_id + 2);
            bar_sync64(bar_id + 1);
            SHK_CCHUNK(2)
            if (c + 2 < nchunk2) bar_arrive64(bar_id + 3);
        }
#undef SHK_CCHUNK
#undef SHK_CSTORE
        flush_counts(cnt, P.counts);
    }
}

// ------------------------------------------------------------------------------------------------
// Sweep along x (the contiguous axis): a WARP owns 32 rows; lane r marches along row r.  The rows
// are staged through shared memory in chunks of XCH cells per row (cp.async, double buffered) so that
// global traffic stays coalesced (64 B row pieces) while each thread reads its own row conflict-free
// (row pitch XCH+1: odd).  The result of cell i-4 is written IN PLACE over the slot of the front cell i
// just consumed, so a chunk buffer holds the inputs [8c, 8c+8) before and the outputs [8c-4, 8c+4)
// after its march; the write-back is coalesced (the primitives of the last sweep are computed element-wise there).
constexpr int XCH = 8;            // cells per row per chunk
constexpr int XPITCH = XCH + 1;   // odd pitch: conflict-free column access for 8 B elements
constexpr int XNS = 2;            // stages

constexpr int XW = 32;            // rows per warp: every warp runs its own pipeline, no CTA barrier

template <typename T, int ROWS>
struct XSmem {
    T buf[ROWS / XW][XNS][NF][XW * XPITCH];
    unsigned cnt[4][ROWS];
};

template <typename T, int EOS, int PH>
__device__ __forceinline__ void x_substep(Marcher<T, EOS>& m, const Consts<T>& k, T* sb, int i, int ilo, int ihi,
                                          int j0, Cnt counts)
{
    // sb = &buf[warp][stage][0][lane * XPITCH + 4 h]: column 4 h + PH of the chunk; window phase = PH
    if (i < ilo || i >= ihi) return;
    T u0[NF], un[NF];
#pragma unroll
    for (int f = 0; f < NF; ++f) u0[f] = sb[f * (XW * XPITCH) + PH];
    m.template step<PH>(k, u0, un);
    if (i - GH >= j0) {
        T pr[6];
        finish_cell<T, EOS, false>(k, un, pr, counts);
#pragma unroll
        for (int f = 0; f < NF; ++f) sb[f * (XW * XPITCH) + PH] = un[f];
    }
}

template <typename T, int EOS, bool EMIT, int ROWS>
__global__ void __launch_bounds__(ROWS) sweep_x_kernel(SweepParams P, Consts<T> k)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    XSmem<T, ROWS>& S = *reinterpret_cast<XSmem<T, ROWS>*>(smem_raw);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long row0 = (long long)blockIdx.x * ROWS + warp * XW;
    if (row0 >= P.npencil) return;                        // whole warp idle (no CTA barrier below)
    const int nrows = (int)min((long long)XW, P.npencil - row0);
    const int sg = blockIdx.y;
    const int j0 = sg * P.seg;
    const int j1 = min(P.N, j0 + P.seg);
    const int ilo = j0 - GH, ihi = j1 + GH;               // front cells [ilo, ihi)
    const int c_first = (ilo >= 0) ? ilo / XCH : -((-ilo + XCH - 1) / XCH);
    const int c_last = (ihi - 1) / XCH;
    const int N = P.N;

    // warp-cooperative chunk loader: element (row, col) of chunk c <- in[f][(row0+row)*nx + ghost(XCH*c+col)]
    // (lane -> 8 consecutive lanes cover one 64 B row piece)
    auto load_chunk = [&](int c, int stage) {
        if (c <= c_last) {
#pragma unroll
            for (int e = lane; e < XW * XCH; e += 32) {
                const int row = e / XCH, col = e % XCH;
                const int i = c * XCH + col;
                if (row < nrows && i >= ilo && i < ihi) {
                    const long long g = (row0 + row) * (long long)N + ghost_index(i, N, P.periodic);
#pragma unroll
                    for (int f = 0; f < NF; ++f)
                        cp_async_elem<T>(&S.buf[warp][stage][f][row * XPITCH + col], (const T*)P.in[f] + g);
                }
            }
        }
        cp_async_commit();
    };

    Cnt cnt;
    cnt.p = &S.cnt[0][threadIdx.x]; cnt.stride = ROWS;
    cnt.zero();
    Marcher<T, EOS> m;
    m.init();
    load_chunk(c_first, 0);
    load_chunk(c_first + 1, 1);
    for (int c = c_first; c <= c_last; ++c) {
        const int stage = (c - c_first) % XNS;
        cp_async_wait<XNS - 1>();
        __syncwarp();
        if (lane < nrows) {
#pragma unroll 1
            for (int h = 0; h < XCH / 4; ++h) {
                T* sb = &S.buf[warp][stage][0][lane * XPITCH + 4 * h];
                const int i = c * XCH + 4 * h;
                x_substep<T, EOS, 0>(m, k, sb, i + 0, ilo, ihi, j0, cnt);
                x_substep<T, EOS, 1>(m, k, sb, i + 1, ilo, ihi, j0, cnt);
                x_substep<T, EOS, 2>(m, k, sb, i + 2, ilo, ihi, j0, cnt);
                x_substep<T, EOS, 3>(m, k, sb, i + 3, ilo, ihi, j0, cnt);
            }
        }
        __syncwarp();
        // write-back of output cells [XCH*c - 4, XCH*c + 4), then refill of the same stage.  Every lane
        // refills exactly the elements it has just read (same e -> (row, col) map), so program order
        // (LDS -> STG -> LDGSTS) keeps the refill behind the read.
#pragma unroll
        for (int e = lane; e < XW * XCH; e += 32) {
            const int row = e / XCH, col = e % XCH;
            const int jo = c * XCH - GH + col;
            if (row < nrows && jo >= j0 && jo < j1) {
                const long long g = (row0 + row) * (long long)N + jo;
                T u[NF];
#pragma unroll
                for (int f = 0; f < NF; ++f) {
                    u[f] = S.buf[warp][stage][f][row * XPITCH + col];
                    ((T*)P.out[f])[g] = u[f];
                }
                if (EMIT) {
                    T pr[6];
                    emit_primitives<T, EOS>(k, u, pr, cnt);
#pragma unroll
                    for (int q = 0; q < 6; ++q) ((T*)P.prim[q])[g] = pr[q];
                }
            }
        }
        load_chunk(c + XNS, stage);
    }
    cp_async_wait<0>();
    flush_counts(cnt, P.counts);
}

// ------------------------------------------------------------------------------------------------
// Warp-specialised x sweep: the producer/consumer pair of sweep_strided_ws_kernel, with lane r marching
// along ROW r of a 32-row strip.  Global traffic moves in 4-cell groups = 32 B row pieces (one sector);
// in shared memory a (group, field) TILE is [32 rows][4 cells], dense (1 KB) -- the layout a TMA box
// {4, 32} produces -- with the two 16 B halves of a row swapped when bit 2 of the row is set (the 32 B
// swizzle).  The fill (cp.async, lane -> (row, col) = (lane>>2 + 8k, lane&3)) and the write-back are then
// contiguous 256 B per instruction, the producer reads both cells of a 2-step chunk with one conflict-free
// LDS.128 per field, and the consumer's single-cell accesses are 2-way conflicts at worst.
constexpr int XV_CH = 4;                // cells per group
constexpr int XV_G = 3;                 // ring groups per pair (12 cells)
constexpr int XV_TILE = 32 * XV_CH;     // elements per (group, field) tile

template <typename T>
struct XvPair {
    T ring[XV_G][NF][XV_TILE];          // tiles are 1 KB (fp64): 256 B aligned as the 32 B swizzle needs
    T outb[NF][XV_TILE];
    T msg[WS_Q][4][32];
    unsigned cnt[4][32];
    unsigned long long bar[32];         // bar[0..2]: one mbarrier per ring tile group (TMA completion); rest: padding
};

// tensor maps of the x sweep (permuted field order like SweepParams::in/out): 2-D {nx, ny*nz}, box {4, 32},
// CU_TENSOR_MAP_SWIZZLE_32B.  Only built for fp64 grids with even nx (TMA needs 16 B row strides).
struct XMaps {
    CUtensorMap in[NF];
    CUtensorMap out[NF];
};

// ---- TMA / mbarrier PTX (sm_90+; SASS: UTMALDG / UTMASTG / SYNCS)
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, int c0, int c1, unsigned long long* bar)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* map, int c0, int c1, const void* src)
{
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];"
                 ::"l"(map), "r"(c0), "r"(c1), "r"(smem_u32(src)) : "memory");
}
__device__ __forceinline__ void tma_store_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void tma_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
template <typename T>
struct XvSmem {
    XvPair<T> pair[4];
};

// two adjacent elements with one shared-memory access (LDS.128 for fp64); p is 2-element aligned
__device__ __forceinline__ void load2(const double* p, double& a, double& b)
{
    const double2 v = *reinterpret_cast<const double2*>(p);
    a = v.x; b = v.y;
}
__device__ __forceinline__ void load2(const float* p, float& a, float& b)
{
    const float2 v = *reinterpret_cast<const float2*>(p);
    a = v.x; b = v.y;
}

// element offset of (row, cell c in 0..3) inside a tile
__device__ __forceinline__ int xv_off(int row, int c) { return row * 4 + 2 * ((c >> 1) ^ ((row >> 2) & 1)) + (c & 1); }

template <typename T, int EOS, bool EMIT, bool TMA>
__global__ void __launch_bounds__(256, 2) sweep_x_ws_kernel(const __grid_constant__ SweepParams P,
                                                            const __grid_constant__ Consts<T> k,
                                                            const __grid_constant__ XMaps maps)
{
    extern __shared__ __align__(1024) unsigned char smem_xv[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const bool producer = warp < 4;
    XvPair<T>& S = reinterpret_cast<XvSmem<T>*>(smem_xv)->pair[warp & 3];
    const int bar_id = 4 * (warp & 3);                      // full0, full1, empty0, empty1 of this pair
    const long long row0 = (long long)blockIdx.x * 128 + (warp & 3) * 32;
    const bool idle = row0 >= P.npencil;                    // both warps of the pair leave together (after setmaxnreg)
    const int nrows = (int)min(32LL, P.npencil - row0);
    const int sg = blockIdx.y;
    const int j0 = sg * P.seg;
    const int j1 = min(P.N, j0 + P.seg);
    const int ilo = j0 - GH;
    const int N = P.N;
    const int nsteps = (j1 - j0) + 2 * GH;                  // front cells ilo .. j1+3
    const int nchunk = 2 * ((nsteps + 3) / 4);              // 2-step chunks, rounded to whole 4-cell groups
    // lane -> element map of the group copies: col = lane & 3, rows (lane >> 2) + 8 kk
    const int col = lane & 3, rsub = lane >> 2;

    if (producer) {
        if (sizeof(T) == 8) asm volatile("setmaxnreg.dec.sync.aligned.u32 96;");
        if (idle) return;
        Producer<T, EOS> pr;
        pr.init();
        // group g = cells ilo+4g .. ilo+4g+3 -> ring tile g % 3.  A group that lies inside [0, N) is one TMA box
        // {4 cells, 32 rows} per field (rows beyond the grid are zero-filled, those lanes are idle); a group that
        // touches a boundary needs the ghost map and goes through cp.async, element by element.
        if (TMA) {
            if (lane == 0) {
#pragma unroll
                for (int q = 0; q < XV_G; ++q) mbar_init(&S.bar[q], 1);
            }
            fence_proxy_async();
            __syncwarp();
        }
        unsigned phase = 0;             // bit q: parity to wait for on bar[q]
        auto group_is_tma = [&](int g) { const int x0 = ilo + XV_CH * g; return TMA && x0 >= 0 && x0 + XV_CH <= N && (x0 & 1) == 0; };   // box start 16 B aligned
        auto load_group = [&](int g) {
            const int q = g % XV_G;
            if (2 * g >= nchunk) {      // past the last group: nothing may be left in flight when the CTA exits
                cp_async_commit();
                return;
            }
            if (group_is_tma(g)) {
                if (lane == 0) {
                    mbar_expect_tx(&S.bar[q], NF * XV_TILE * (unsigned)sizeof(T));
#pragma unroll
                    for (int f = 0; f < NF; ++f)
                        tma_load_2d(&S.ring[q][f][0], &maps.in[f], ilo + XV_CH * g, (int)row0, &S.bar[q]);
                }
            } else {
                const int gi = ghost_index(ilo + XV_CH * g + col, N, P.periodic);
                T* dst = &S.ring[q][0][0];
#pragma unroll
                for (int kk = 0; kk < 4; ++kk) {
                    const int row = rsub + 8 * kk;
                    if (row < nrows) {
                        const long long o = (row0 + row) * (long long)N + gi;
                        const int so = xv_off(row, col);
#pragma unroll
                        for (int f = 0; f < NF; ++f) cp_async_elem<T>(dst + f * XV_TILE + so, (const T*)P.in[f] + o);
                    }
                }
            }
            cp_async_commit();          // also for TMA groups (empty): keeps the wait_group arithmetic uniform
        };
        auto wait_group = [&](int g) {
            cp_async_wait<1>();
            if (group_is_tma(g)) {
                const int q = g % XV_G;
                mbar_wait(&S.bar[q], (phase >> q) & 1u);
                phase ^= 1u << q;
            }
            __syncwarp();
        };
        load_group(0);
        int g = 0;
        const int sw = (lane >> 2) & 1;
        // Group g+1 is issued at the start of group g into the tile of group g-2, which the consumer
        // finished (as U_{i-1}) in the iteration before: it runs one 2-step iteration behind this warp.
#define SHK_XPCHUNK(PH, HALF)                                                                        \
        {                                                                                           \
            if (HALF == 0) {                                                                        \
                load_group(g + 1);                                                                  \
                wait_group(g);                                                                      \
            }                                                                                       \
            T um[NF], ua[NF], ub[NF], ma[4], mb[4];                                                 \
            um[NF - 1] = ua[NF - 1] = ub[NF - 1] = T(0);                                            \
            const int tile = g % XV_G;                                                              \
            /* cell before the chunk: cell 1 of this tile (HALF 1) or cell 3 of the previous group's tile (HALF 0) */ \
            const T* srm = HALF ? &S.ring[tile][0][xv_off(lane, 1)]                                 \
                                : &S.ring[(tile + XV_G - 1) % XV_G][0][xv_off(lane, 3)];            \
            const T* src = &S.ring[tile][0][lane * 4 + 2 * (HALF ^ sw)];                            \
            _Pragma("unroll") for (int f = 0; f < Producer<T, EOS>::NP; ++f) {                      \
                um[f] = srm[f * XV_TILE];                                                           \
                load2(src + f * XV_TILE, ua[f], ub[f]);                                             \
            }                                                                                       \
            if (HALF == 1) ++g;                                                                     \
            pr.template step<PH>(k, um, ua, ma);                                                    \
            pr.template step<PH + 1>(k, ua, ub, mb);                                                \
            _Pragma("unroll") for (int q = 0; q < 4; ++q) S.msg[PH][q][lane] = ma[q];               \
            _Pragma("unroll") for (int q = 0; q < 4; ++q) S.msg[PH + 1][q][lane] = mb[q];           \
        }
        for (int c = 0; c < nchunk; c += 2) {                   // nchunk is even here
            if (c >= 2) bar_sync64(bar_id + 2);
            SHK_XPCHUNK(0, 0)
            bar_arrive64(bar_id + 0);
            if (c >= 1) bar_sync64(bar_id + 3);
            SHK_XPCHUNK(2, 1)
            bar_arrive64(bar_id + 1);
        }
#undef SHK_XPCHUNK
        cp_async_wait<0>();
    } else {
        if (sizeof(T) == 8) asm volatile("setmaxnreg.inc.sync.aligned.u32 160;");
        if (idle) return;
        Cnt cnt;
        cnt.p = &S.cnt[0][lane]; cnt.stride = 32;
        cnt.zero();
        Consumer<T> co;
        co.init();
        int t = 0;
        int gprev = XV_G - 1;           // tile of group floor((t-1)/4); t = 0 reads don't-care warm-up values
        const int swc = (lane >> 2) & 1;
#define SHK_XCFIN(UN, PH)                                                                           \
        {                                                                                           \
            T pv[6];                                                                                \
            if (t >= 2 * GH && t < nsteps && lane < nrows) finish_cell<T, EOS, false>(k, UN, pv, cnt); \
            T* dst = &S.outb[0][xv_off(lane, PH)];                                                  \
            _Pragma("unroll") for (int f = 0; f < NF; ++f) dst[f * XV_TILE] = UN[f];                 \
            ++t;                                                                                    \
        }
        // one chunk = steps t, t+1 (t even): cells t-2, t-1 are one aligned pair (LDS.128) of the tile `gprev`,
        // cell t is the first cell of the next pair: of the next tile when t = 0 mod 4 (PH 0), of the same tile
        // when t = 2 mod 4 (PH 2).  Nothing of U is carried in registers.
#define SHK_XCCHUNK(PH)                                                                             \
        {                                                                                           \
            T uq[NF], ua[NF], ub[NF], msg[4], un[NF];                                               \
            const T* s2 = &S.ring[gprev][0][lane * 4 + 2 * ((PH == 0 ? 1 : 0) ^ swc)];              \
            if (PH == 0) gprev = (gprev + 1 == XV_G) ? 0 : gprev + 1;                               \
            const T* s1 = &S.ring[gprev][0][lane * 4 + 2 * ((PH == 0 ? 0 : 1) ^ swc)];              \
            _Pragma("unroll") for (int f = 0; f < NF; ++f) {                                        \
                load2(s2 + f * XV_TILE, uq[f], ua[f]);                                              \
                ub[f] = s1[f * XV_TILE];                                                            \
            }                                                                                       \
            _Pragma("unroll") for (int q = 0; q < 4; ++q) msg[q] = S.msg[PH][q][lane];              \
            co.template step<PH>(uq, ua, msg, un);                                                  \
            SHK_XCFIN(un, PH)                                                                       \
            _Pragma("unroll") for (int q = 0; q < 4; ++q) msg[q] = S.msg[PH + 1][q][lane];          \
            co.template step<PH + 1>(ua, ub, msg, un);                                              \
            SHK_XCFIN(un, PH + 1)                                                                   \
        }
        // write-back of the 4-cell group whose last cell was produced by step t-1: cells j0-8+4m .. +3
        auto write_group = [&]() {
            const int jo = ilo + (t - 4) - GH + col;
            if (jo >= j0 && jo < j1) {
#pragma unroll
                for (int kk = 0; kk < 4; ++kk) {
                    const int row = rsub + 8 * kk;
                    if (row < nrows) {
                        const long long o = (row0 + row) * (long long)N + jo;
                        const int so = xv_off(row, col);
                        T u[NF];
#pragma unroll
                        for (int f = 0; f < NF; ++f) {
                            u[f] = S.outb[f][so];
                            ((T*)P.out[f])[o] = u[f];
                        }
                        if (EMIT) {
                            T pv[6];
                            emit_primitives<T, EOS>(k, u, pv, cnt);
#pragma unroll
                            for (int q = 0; q < 6; ++q) ((T*)P.prim[q])[o] = pv[q];
                        }
                    }
                }
            }
        };
        // a finished group goes out as one TMA box per field when all of its cells are output cells of this
        // segment (or are clipped by the grid edge); otherwise (and for EMIT) through the LSU write-back
        bool store_pending = false;
        for (int c = 0; c < nchunk; c += 2) {                   // nchunk is even here
            bar_sync64(bar_id + 0);
            if (TMA && store_pending) {                     // outb is rewritten below: the TMA must have read it
                if (lane == 0) tma_store_wait_read();
                __syncwarp();
                store_pending = false;
            }
            SHK_XCCHUNK(0)
            if (c + 2 < nchunk) bar_arrive64(bar_id + 2);
            bar_sync64(bar_id + 1);
            SHK_XCCHUNK(2)
            if (c + 3 < nchunk) bar_arrive64(bar_id + 3);
            const int jf = ilo + (t - 4) - GH;              // first cell of the finished group
            if (TMA && !EMIT && (jf & 1) == 0 && jf >= j0 && jf < j1 && (jf + XV_CH <= j1 || j1 == N)) {
                fence_proxy_async();                        // generic-proxy writes of outb -> visible to the TMA engine
                __syncwarp();
                if (lane == 0) {
#pragma unroll
                    for (int f = 0; f < NF; ++f) tma_store_2d(&maps.out[f], jf, (int)row0, &S.outb[f][0]);
                    tma_store_commit();
                }
                store_pending = true;
            } else {
                __syncwarp();
                write_group();
                __syncwarp();
            }
        }
        if (TMA && lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
#undef SHK_XCCHUNK
#undef SHK_XCFIN
        flush_counts(cnt, P.counts);
    }
}

}  // namespace shk
