// shasta_kernels.cuh -- sm_100a device code of the fused SHASTA sweep.
//
// One sweep along an axis = one kernel launch that reads the five conserved fields once and
// writes them once (80 B/cell in fp64).  Every pencil is processed by MARCHING along the sweep axis with
// the "front" cell i and a rolling register window, so every quantity of eqs. (15)-(22)
// is computed exactly once per cell / per interface -- not 5x (U-hat) and 2x (A) per cell as in the
// paper's Listing 1.  The march is run by warp PAIRS (a producer and a consumer
// warp per 32 pencils, setmaxnreg 96/160), in groups of 4 cells fed by TMA: sweep_yz_kernel (y, z) and
// sweep_x2_kernel (x) below; sweep_cell_kernel is the paper's one-thread-per-cell decomposition.
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
// The kernel is bound by the fp64 pipe (63.9 results/clk/SM on B200, measured: tests/probes) about as much
// as by HBM, so the arithmetic is written for a minimal fp64 instruction count:
//   * no fp64 division or library sqrt on the common path: MUFU.RCP64H / MUFU.RSQ64H seeds (2^-20,
//     measured) + Newton steps written out below;
//   * the flux limiter is two DSETP with |.| modifiers + selects (limiter<double>);
//   * vacuum / causality-clamped cells are handled behind one warp vote per four cells (c2p_group);
//   * the register window rotates by NAME (march unrolled by 4, compile-time slots), not by moves.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace shk {

#ifndef SHK_GEOM_C
#define SHK_GEOM_C 0
#endif
constexpr int NF = 5;       // E, M_par, M_perp1, M_perp2, R
constexpr int GH = 4;       // ghost depth = dependency radius of one sweep
constexpr double VAC_E = 0x1p-498;      // reading G7: a cell with !(E >= 2^-498) is vacuum (E^2, |M|^2 not representable below)
// Newton on v stops once a step is below NEWT_DV: the step taken is (to first order) the error BEFORE it, and the error
// after it is 2^-20 of that (slope seeded by rcp64h) plus the quadratic term, i.e. below 1e-16 -- the iterate is converged
// to fp64 without spending one more iteration on confirming it (a step <= 1e-15, the rule of PAPER.md:109's iteration in
// the oracle, bounds the same error from the other side).
#ifndef SHK_NEWT_DV
#define SHK_NEWT_DV 1e-10
#endif
constexpr double NEWT_DV = SHK_NEWT_DV;
constexpr int EOS_GAMMA = 0;    // p = (Gamma-1) e            (m = 0): closed-form velocity
constexpr int EOS_MASS = 1;     // p = (Gamma-1)(e - m n)     (m > 0): safeguarded Newton
constexpr int EOS_TABLE = 2;    // p = bilinear table P(e, n) (reading T1): the same safeguarded Newton

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
    // tabled EOS (EOS_TABLE, reading T1): P at nodes (i de, j dn), i < ne, j < nn, e fastest; device pointer
    const double* tab;
    int ne, nn;
    double ide, idn;    // 1/de, 1/dn
};

// P(e, n) of the table and its two slopes in the cell that holds (e, n): bilinear between nodes, the nearest cell's bilinear
// form outside the table (linear continuation), floored at 0 (then the slopes are 0 too).  Four read-only loads (L1/L2:
// neighbouring cells of the grid hit the same table lines).
__device__ __forceinline__ void eos_table_eval(const EosD& k, double e, double n, double& P, double& Pe, double& Pn)
{
    const double xe = e * k.ide, xn = n * k.idn;
    const int i = min(max(__double2int_rd(xe), 0), k.ne - 2);
    const int j = min(max(__double2int_rd(xn), 0), k.nn - 2);
    const double te = xe - (double)i, tn = xn - (double)j;
    const double* q = k.tab + i + (long long)k.ne * j;
    const double p00 = __ldg(q), p10 = __ldg(q + 1), p01 = __ldg(q + k.ne), p11 = __ldg(q + k.ne + 1);
    const double d0 = p10 - p00, d1 = p11 - p01;
    const double p0 = fma(te, d0, p00), p1 = fma(te, d1, p01);
    const double praw = fma(tn, p1 - p0, p0);
    const bool pos = praw > 0.0;
    P = pos ? praw : 0.0;
    Pe = pos ? fma(tn, d1 - d0, d0) * k.ide : 0.0;
    Pn = pos ? (p1 - p0) * k.idn : 0.0;
}

template <typename T>
struct Consts {
    T lam;      // lambda = dt/dx
    T hlam;     // lambda/2 (predictor; corrector source factor)
    T qlam;     // lambda/4 (predictor source factor 1/2 * lambda/2)
    T aq;       // diff / 8: outer factor of eq. (19) times the paper's `diff`; 1/8 by default
    T ad2;      // factor of the second difference of Delta inside eq. (19): -1/8 = phoenical (default), 0 = explicit
                // antidiffusion A = diff/8 D^ (footnote 1); f2
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
    long long npencil;      // END of the pencil range: pencils (x sweep: rows; y/z: groups of 32 pencils) pbase .. npencil-1
    long long pbase;        // first pencil of the launch: 0, or the start of the active planes (shasta_set_active_planes)
    int seg;                // cells marched per work item
    int nseg;               // segments per pencil
    int periodic;           // boundary rule (reading G11)
    int axis;               // 0 x, 1 y, 2 z
    int odiv;               // y/z kernel, batch of events: `other` index = oy + odiv * event (z sweep: odiv = ny); else INT_MAX
    unsigned long long* counts;   // diagnostics [4]
};

// Diagnostics are counted per thread in REGISTERS and flushed once per warp at the end of the kernel: one global atomic
// per event on a single address serialises in L2 and cost 60 % of the step time once the causality projection fired
// in ~0.2 % of the cells (round 1).
struct Cnt {
    unsigned pv;        // Pi fired (low 16 bits) | vacuum cells (high 16 bits): a thread marches < 65536 cells per launch
    unsigned fl;        // e < 0 floored (low 16) | p < 0 floored (high 16)   (primitive output only)
    __device__ __forceinline__ void zero() { pv = fl = 0u; }
    __device__ __forceinline__ void add(int w) { if (w == 0) pv += 1u; else if (w == 1) pv += 0x10000u; else if (w == 2) fl += 1u; else fl += 0x10000u; }
};
__device__ __forceinline__ void flush_counts(const Cnt& c, unsigned long long* g)
{
    const unsigned mask = __activemask();
    const int leader = __ffs(mask) - 1;
    const unsigned v[4] = {c.pv & 0xffffu, c.pv >> 16, c.fl & 0xffffu, c.fl >> 16};
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const unsigned t = __reduce_add_sync(mask, v[w]);
        if ((int)(threadIdx.x & 31) == leader && t) atomicAdd(g + w, (unsigned long long)t);
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

// 1/sqrt(x), normal x > 0: seed r (2^-20), ONE cubic step r (1 + e/2 + 3 e^2/8), e = 1 - x r^2: truncation 5/16 e^3 = 2^-58.
// 5 fp64 ops (fast_rsqrt: 8); used where the result is needed unconditionally (branch-free causality clamp).
__device__ __forceinline__ double fast_rsqrt3(double x)
{
    const double r = rsq64h(x);
    const double e = fma(-(x * r), r, 1.0);
    const double p = fma(0.375, e, 0.5);
    return fma(r, p * e, r);
}

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

__device__ __forceinline__ void store2(double* p, double a, double b) { *reinterpret_cast<double2*>(p) = make_double2(a, b); }
__device__ __forceinline__ void store2(float* p, float a, float b) { *reinterpret_cast<float2*>(p) = make_float2(a, b); }

// keeps shared-memory loads below this point (registers: a pair of cells is 20 registers)
__device__ __forceinline__ void load_fence() { asm volatile("" ::: "memory"); }

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
    const bool vac = !(E >= VAC_E);                      // vacuum (reading G7); also catches NaN
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
            double Ph;
            if (EOS == EOS_TABLE) {
                double a_, b_;
                eos_table_eval(k, E - Mabs * hi, R * (w2h * fast_rsqrt(w2h)), Ph, a_, b_);
            } else {
                Ph = fmax(k.gm1 * ((E - Mabs * hi) - mR * (w2h * fast_rsqrt(w2h))), double(0));
            }
            v = fmin(fmax(Mabs * fast_rcp(E + Ph), lo), hi);
        }
        bool done = false;
        for (int it = 0; it < 48; ++it) {
            // no library sqrt / division in the loop: w2 >= 2e-12 (v <= 1 - delta) and dg >= E - (Gamma-1)|M| v > 0
            // are normal positive numbers, so the MUFU-seeded fast_rsqrt / fast_rcp apply (<= 2 ulp; the iteration
            // is self-correcting and the primitives after the loop are formed from the converged v)
            const double w2 = fma(-v, v, double(1));
            const double rw = fast_rsqrt(w2);
            const double w = w2 * rw;
            double P, dP;
            if (EOS == EOS_TABLE) {
                // P(e(v), n(v)), e = E - |M| v, n = R sqrt(1 - v^2); dP/dv from the slopes of the table cell (piecewise
                // constant: a kink at a cell border costs the Newton step at most the bisection safeguard below)
                double Pe, Pn;
                eos_table_eval(k, E - Mabs * v, R * w, P, Pe, Pn);
                dP = -(Mabs * Pe) - (R * v * rw) * Pn;
            } else {
                const double praw = k.gm1 * ((E - Mabs * v) - mR * w);
                const bool pos = praw > double(0);
                P = pos ? praw : double(0);
                dP = pos ? k.gm1 * (mR * v * rw - Mabs) : double(0);
            }
            const double g = fma(v, E + P, -Mabs);
            double dg = fma(v, dP, E + P);
            if (EOS == EOS_TABLE) dg = dg > double(0.25) * E ? dg : E;      // a table may be steep: keep the Newton slope sane
            if (g > double(0)) hi = v; else lo = v;
            double vn = v - g * fast_rcp(dg);
            if (!(vn >= lo && vn <= hi)) vn = double(0.5) * (lo + hi);
            // a lane stops moving with its own first converged step: what it returns does not depend on the lanes it shares
            // the loop with (an idle lane may solve for garbage, a partner may need more steps) -- run-to-run reproducible
            const double dv = fabs(vn - v);
            if (!done) v = vn;
            done = done || !(dv > NEWT_DV);      // NaN (idle lane, garbage): done
            if (__all_sync(__activemask(), done)) break;
        }
        o.w = fmax(fma(-v, v, double(1)), double(0));
        const double eraw = fma(-Mabs, v, E);
        if (eraw < double(0)) o.fl |= 1;
        o.e = fmax(eraw, double(0));
        const double n = (o.w > double(1e-300)) ? R * fast_sqrt(o.w) : double(0);
        if (EOS == EOS_TABLE) {
            double a_, b_;
            eos_table_eval(k, o.e, n, o.p, a_, b_);
        } else {
            const double praw = k.gm1 * (o.e - k.mass * n);
            if (praw < double(0)) o.fl |= 2;
            o.p = fmax(praw, double(0));
        }
        o.y = (M2 > double(1e-300)) ? v * fast_rsqrt(M2) : double(0);
    }
    if (vac) { o.y = double(0); o.e = double(0); o.p = double(0); o.w = double(0); o.fl = 0; }   // n = R sqrt(w) = 0 (reading G7)
    return o;
}

// The same solve as the non-Gamma branch of cons2prim_general, cut into init / iter / finish so that the in-sweep cons2prim
// of TWO cells can run as one loop with two independent dependency chains (c2p_group below).  The Newton iteration of one
// cell is a serial chain of ~25 dependent fp64 operations per step; with one cell at a time the producer warp issued an
// instruction every ~7 cycles (round 1: config 3 at a third of the Gamma-law speed).  Same formulas, same bracket, same
// tolerance; a cell that has converged stays where it is while its partner (and the warp) finish.
template <int EOS>
struct Newt {
    double E, Mabs, R, mR, v, lo, hi, M1, M2;
    bool vac, done;
    __device__ __forceinline__ void init(const EosD& k, const double (&u)[NF])
    {
        init_em(k, u[0], u[1], fma(u[1], u[1], fma(u[2], u[2], u[3] * u[3])), u[4]);
    }
    // from E, M_par, |M|^2 and R: all the solve needs (what the producer hands to the consumer for S3)
    __device__ __forceinline__ void init_em(const EosD& k, double E_, double M1_, double M2_, double R_)
    {
        E = E_; M1 = M1_; M2 = M2_; R = R_;
        done = false;
        vac = !(E >= VAC_E);
        if (vac) { E = 1.0; M1 = 0.0; M2 = 0.0; }
        const double lim = k.omd * E;
        const double lim2 = lim * lim;
        const double Mq = M2 > lim2 ? lim2 : M2;
        const bool moving = Mq > 1e-300;
        Mabs = moving ? Mq * fast_rsqrt(Mq) : 0.0;
        lo = 0.0;
        hi = fmin(Mabs * fast_rcp(E), k.omd);
        mR = k.mass * R;
        const double w2h = fma(-hi, hi, 1.0);
        double Ph;
        if (EOS == EOS_TABLE) {
            double a_, b_;
            eos_table_eval(k, E - Mabs * hi, R * (w2h * fast_rsqrt(w2h)), Ph, a_, b_);
        } else {
            Ph = fmax(k.gm1 * ((E - Mabs * hi) - mR * (w2h * fast_rsqrt(w2h))), 0.0);
        }
        v = fmin(fmax(Mabs * fast_rcp(E + Ph), lo), hi);
    }
    __device__ __forceinline__ void iter(const EosD& k)
    {
        const double w2 = fma(-v, v, 1.0);
        const double rw = fast_rsqrt3(w2);              // 2^-58: w enters P, which fixes the root
        const double w = w2 * rw;
        double P, dP;
        if (EOS == EOS_TABLE) {
            double Pe, Pn;
            eos_table_eval(k, E - Mabs * v, R * w, P, Pe, Pn);
            dP = -(Mabs * Pe) - (R * v * rw) * Pn;
        } else {
            const double praw = k.gm1 * ((E - Mabs * v) - mR * w);
            const bool pos = praw > 0.0;
            P = pos ? praw : 0.0;
            dP = pos ? k.gm1 * (mR * v * rw - Mabs) : 0.0;
        }
        const double g = fma(v, E + P, -Mabs);
        double dg = fma(v, dP, E + P);
        if (EOS == EOS_TABLE) dg = dg > 0.25 * E ? dg : E;
        if (g > 0.0) hi = v; else lo = v;
        double vn = v - g * rcp64h(dg);                 // slope to 2^-20 is enough: the step it scales goes to 0
        if (!(vn >= lo && vn <= hi)) vn = 0.5 * (lo + hi);
        // The cell stops moving with its own first converged step: its result does not depend on
        // the cells it shares the loop with (its partner, the other lanes of the vote, an idle lane solving for whatever its
        // shared-memory slot held) -- the same bits from run to run and for any segmentation of the march.  The loops vote on `done`.
        const double dv = fabs(vn - v);
        if (!done) v = vn;
        done = done || !(dv > NEWT_DV);          // a NaN step (an idle lane solving for garbage) counts as done: it must not hold the warp
    }
    // v_par = M_par v / |M| and p of the converged state (vacuum: 0, 0)
    __device__ __forceinline__ void finish(const EosD& k, double& vpar, double& p) const
    {
        const double w = fmax(fma(-v, v, 1.0), 0.0);
        const double e = fmax(fma(-Mabs, v, E), 0.0);
        const double n = (w > 1e-300) ? R * fast_sqrt(w) : 0.0;
        if (EOS == EOS_TABLE) {
            double a_, b_;
            eos_table_eval(k, e, n, p, a_, b_);
        } else {
            p = fmax(k.gm1 * (e - k.mass * n), 0.0);
        }
        const double y = (M2 > 1e-300) ? v * fast_rsqrt(M2) : 0.0;
        vpar = M1 * y;
        if (vac) { vpar = 0.0; p = 0.0; }
    }
};

// The EOS_GAMMA kernels have NO out-of-line path: vacuum / non-positive E (high word <= 0) is a two-line inline
// branch (all primitives 0, M = 0), and the host instantiates them only for Gamma <= 5/3, where the frozen-slope
// Newton of c2p_fast_y converges in two steps (larger Gamma runs the EOS_MASS kernels with m = 0).  The causality clamp Mc = min(|M|, (1-delta) E) stays inline: Mc^2 is a
// select on the bit patterns (non-negative doubles order like integers), and only a clamped cell (~0.2 % of
// the cells of config 4) pays the extra rsqrt for the direction-preserving scale factor.
// Vacuum test of the Gamma-law kernels on the high word: reading G7, !(E >= 2^-498): E <= 0, -0, and every E whose square
// is not representable (exponent field < 0x20D = 1023 - 498); the closed form below would divide by zero there.  NaN with
// a clear sign bit has a large exponent field and propagates instead of being called vacuum (a NaN input is an error).
__device__ __forceinline__ bool c2p_is_vacuum(double E)
{
    return __double2hiint(E) < 0x20D00000;
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
    // No BRANCH here, neither for vacuum nor for the causality clamp: the arithmetic runs on whatever E, M are (inf / NaN
    // intermediates cost nothing on the fp64 pipe) and the results are masked by selects.  A branch ends the basic
    // block, and the producer's cons2prim chains are serial (~20 dependent fp64 operations): only when the whole
    // 4-cell group is ONE basic block can ptxas interleave the chains of its cells (ncu, round 2: with the clamp as a
    // branch the producer issued one instruction every 6.2 cycles, all of it fixed-latency `wait`).  The price is the
    // direction-preserving scale factor Mc/|M| computed for every cell (8 fp64 operations) instead of for the ~0.2 %
    // that are clamped.
    const double M2 = fma(u[1], u[1], fma(u[2], u[2], u[3] * u[3]));
    const bool vac = c2p_is_vacuum(u[0]);       // reading G7: all primitives 0
    const double t = u[0] * u[0];
    const double lim2 = k.omd2 * t;
    const bool clamped = gt_nonneg(M2, lim2);
    const double Mq = clamped ? lim2 : M2;
    double y = c2p_fast_y(k, u[0], Mq, t);
    double e = fma(-Mq, y, u[0]);               // e = E - Mc v >= delta E > 0: no floor
    const double ys = y * ((k.omd * u[0]) * fast_rsqrt3(M2));   // clamped cells: v_i = (Mc y) M_i / |M|
    y = clamped ? ys : y;
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

// In-sweep cons2prim of the FOUR cells of a hand-over group.  Gamma-law: the common case (no vacuum, causality clamp not
// active) is the bare closed form, 19 fp64 operations per cell and no select; whether ANY lane of the warp holds a
// vacuum or clamped cell is decided by one vote per group, and only then is the cell redone by c2p_sweep_d (the
// select form above, identical bits for ordinary cells).  The branch-free select form for every cell (round 2, first
// version) paid the direction-preserving scale factor (8 fp64 operations) and 8 selects per cons2prim for the ~0.2 %
// of the cells that need them; one warp-uniform branch per four cells keeps the four chains in one basic block.
template <typename T, typename CL>
__device__ __forceinline__ void c2p_group(const Consts<T>& k, const T (&c0)[NF], const T (&c1)[NF], const T (&c2)[NF],
                                          const T (&c3)[NF], T (&v)[4], T (&p)[4], const CL& cell, T* out)
{
    // Gamma-law only (the general EOS runs c2p_pairs_general / HalfStep).  `cell(j, u)` re-reads cell j of the group from
    // shared memory, `out + 128 j` is a free 16 B slot of this lane for the redone {v, p} of cell j: the rare path is ONE
    // rolled loop body (its four inlined copies per phase were 5.5 KB of the producer's 17 KB of code; with the emitting
    // consumer the pair no longer fitted the instruction cache: `no_inst` 7-10 % of the stall samples of both roles).
    unsigned rmask = 0u;
#define SHK_C2P_FAST(J, C)                                                                      \
    {                                                                                           \
        const double E = (double)C[0], M1 = (double)C[1];                                       \
        const double M2 = fma(M1, M1, fma((double)C[2], (double)C[2], (double)C[3] * (double)C[3])); \
        const double t = E * E;                                                                 \
        if (gt_nonneg(M2, k.d.omd2 * t) | c2p_is_vacuum(E)) rmask |= 1u << J;                   \
        const double y = c2p_fast_y(k.d, E, M2, t);                                             \
        v[J] = (T)(M1 * y);                                                                     \
        p[J] = (T)(k.d.gm1 * fma(-M2, y, E));                                                   \
    }
    SHK_C2P_FAST(0, c0) SHK_C2P_FAST(1, c1) SHK_C2P_FAST(2, c2) SHK_C2P_FAST(3, c3)
#undef SHK_C2P_FAST
    if (__any_sync(0xffffffffu, rmask != 0u)) {
        unsigned redone = 0u;               // warp-uniform: cells whose {v, p} were redone for the whole warp
#pragma unroll 1
        for (int jj = 0; jj < 4; ++jj) {
            if (__any_sync(0xffffffffu, (rmask >> jj) & 1u)) {
                T u[NF], vv, pp;
                cell(jj, u);
                c2p_sweep<T, EOS_GAMMA>(k, u, vv, pp);          // select form: same bits for ordinary cells
                store2(out + 128 * jj, vv, pp);
                redone |= 1u << jj;
            }
        }
        load_fence();
#pragma unroll
        for (int jj = 0; jj < 4; ++jj)
            if (redone & (1u << jj)) load2(out + 128 * jj, v[jj], p[jj]);
    }
}

// General EOS, S1 of a group: two Newton loops of two cells each (see Newt), written as ONE loop body executed twice
// (#pragma unroll 1): the results go through this lane's scratch slots `scr` (cell j at scr + 128 j) because a rolled
// loop cannot index registers.  Unrolled, the two copies of the solver (with the consumer's two more) made the kernel
// miss the instruction cache: ncu showed `no_inst` as 32 % of the consumer's and 12 % of the producer's stall samples.
// `pairload(pi, a, b)` reads cells 2 pi, 2 pi + 1 of the group from the ring.
template <typename T, int EOS, typename PL>
__device__ __forceinline__ void c2p_pairs_general(const Consts<T>& k, const PL& pairload, T* scr, T (&v)[4], T (&p)[4])
{
#pragma unroll 1
    for (int pi = 0; pi < 2; ++pi) {
        T ca[NF], cb[NF];
        pairload(pi, ca, cb);
        double ua[NF], ub[NF], va, pa, vb, pb;
#pragma unroll
        for (int f = 0; f < NF; ++f) { ua[f] = (double)ca[f]; ub[f] = (double)cb[f]; }
        Newt<EOS> na, nb;
        na.init(k.d, ua); nb.init(k.d, ub);
        for (int it = 0; it < 48; ++it) {
            na.iter(k.d); nb.iter(k.d);
            if (__all_sync(0xffffffffu, na.done && nb.done)) break;
        }
        na.finish(k.d, va, pa); nb.finish(k.d, vb, pb);
        store2(scr + 256 * pi, (T)va, (T)pa);
        store2(scr + 256 * pi + 128, (T)vb, (T)pb);
    }
    load_fence();
#pragma unroll
    for (int j = 0; j < 4; ++j) load2(scr + 128 * j, v[j], p[j]);
}

// eq. (21) branch-free (reading G12): A = sigma max(0, min(sigma D^_{j+1}, |A^ph|, sigma D^_{j-1}))
template <typename T>
__device__ __forceinline__ T limiter(T aph, T dhp, T dhm)
{
    const T sg = copysign(T(1), aph);
    const T m = t_min(t_min(sg * dhp, t_abs(aph)), sg * dhm);
    return sg * t_max(m, T(0));
}
// fp64: the three arguments must agree in sign, else A = 0; if they do, A is the one of smallest magnitude, sign
// included.  Two DSETP with |.| operand modifiers + selects, the sign test is one LOP3 on the high words: 10
// instructions per field (the sign-magnitude integer min of round 1 cost 16, all on the 2-cycle ALU pipe).
template <>
__device__ __forceinline__ double limiter<double>(double aph, double dhp, double dhm)
{
    const int dis = (__double2hiint(aph) ^ __double2hiint(dhp)) | (__double2hiint(aph) ^ __double2hiint(dhm));
    double m = fabs(dhp) < fabs(aph) ? dhp : aph;
    m = fabs(dhm) < fabs(m) ? dhm : m;
    return dis < 0 ? 0.0 : m;
}

// Pi, readings G6-G8: written back to M at the end of every sweep.  E and R are never modified.
__device__ __forceinline__ void project(const EosD& k, double (&un)[NF], Cnt& counts)
{
    const double E = un[0];
    const double M2 = fma(un[1], un[1], fma(un[2], un[2], un[3] * un[3]));
    const double lim = k.omd * E;
    if (!(E >= VAC_E)) {
        un[1] = un[2] = un[3] = 0.0;
        counts.add(1);
    } else if (M2 > lim * lim) {
        const double s = lim * fast_rsqrt(M2);
        un[1] *= s; un[2] *= s; un[3] *= s;
        counts.add(0);
    }
}

// primitives of one cell from its (projected) conserved state, slots permuted like the momenta
template <int EOS>
__device__ __forceinline__ void primitives(const EosD& k, const double (&u)[NF], double (&pr)[6], Cnt& counts)
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
__device__ __forceinline__ void finish_d(const EosD& k, double (&un)[NF], double (&pr)[6], Cnt& counts)
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
__device__ __forceinline__ void finish_cell(const Consts<T>& k, T (&un)[NF], T (&pr)[6], Cnt& counts)
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
__device__ __forceinline__ void emit_d(const EosD& k, const double (&u)[NF], double (&pr)[6], Cnt& counts)
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
__device__ __forceinline__ void emit_primitives(const Consts<T>& k, const T (&u)[NF], T (&pr)[6], Cnt& counts)
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

    // One hand-over group = four march steps with front cells c1..c4 (c0 = the cell before them), arranged in PHASES:
    // S1 of the four cells, S2 of the four cells, S3 of the four cells, geometry -- the same arithmetic as four step<PH>()
    // calls (identical bits), but each cons2prim phase is four INDEPENDENT chains behind one rare-path vote (c2p_group).
    // State slots here: fE[0]/fM[0] = cell -2, [1] = cell -1 (time n); gE/gM likewise for half-step cells -3, -2.
    // `ld` reads cells of the group from the shared-memory ring: ld.first(c0, c1, c2) the cell before the group and its
    // first two cells, ld.second(c3, c4) the last two.  It is called again in every phase that needs U^n (behind a
    // compiler fence), so that U^n is not held in registers across the cons2prim phases (96 registers per thread).
    // `scr` is this lane's slice of the message buffer of the group (16 elements, stride as written by the caller): it
    // holds U~ of the four cells while S3 runs, so that the rare path of S3 can read them back instead of keeping 16
    // values alive in registers.
    template <typename L>
    __device__ __forceinline__ void group(const Consts<T>& k, const L& ld, T* scr, T (&msg)[4][4])
    {
        {
            T v[4], p[4];
            {
                T c0[NF], c1[NF], c2[NF], c3[NF], c4[NF];
                ld.first(c0, c1, c2);
                if constexpr (EOS == EOS_GAMMA) {
                    ld.second(c3, c4);
                    c2p_group<T>(k, c1, c2, c3, c4, v, p, [&](int jj, T (&u)[NF]) { ld.cell(jj, u); }, scr);       // S1
                } else {
                    c2p_pairs_general<T, EOS>(k, [&](int pi, T (&a)[NF], T (&b)[NF]) { ld.pair(pi, a, b); }, scr, v, p);
                }
            }
            T eps[5], pv[6], pp[6];
            eps[0] = eps1; pv[0] = fE[0]; pv[1] = fE[1]; pp[0] = fM[0]; pp[1] = fM[1];
#pragma unroll
            for (int j = 0; j < 4; ++j) { eps[j + 1] = k.hlam * v[j]; pv[j + 2] = p[j] * v[j]; pp[j + 2] = p[j]; }
            T ut[4][NF];
#define SHK_PRED(J, UL, UR)                                                                     \
            {                                                                                   \
                const T q = (T(0.5) - eps[J]) * fast_rcp(T(1) + (eps[J + 1] - eps[J]));         \
                const T a = T(0.5) - q, b = (T(0.5) * q) * q;                                   \
                _Pragma("unroll") for (int f = 0; f < NP; ++f) {                                \
                    const T d = UR[f] - UL[f];                                                  \
                    const T fl = t_fma(a, UL[f], -(b * d));                                     \
                    ut[J][f] = UL[f] - (fl - ft[f]);                                            \
                    ft[f] = fl;                                                                 \
                }                                                                               \
                if (NP < NF) ut[J][NF - 1] = T(0);                                              \
                ut[J][0] = t_fma(-k.qlam, pv[J + 2] - pv[J], ut[J][0]);                         \
                ut[J][1] = t_fma(-k.qlam, pp[J + 2] - pp[J], ut[J][1]);                         \
                if (EOS == EOS_GAMMA) {             /* parked for the rare path of S3 */             \
                    store2(scr + 128 * J, ut[J][0], ut[J][1]);                                  \
                    store2(scr + 128 * J + 64, ut[J][2], ut[J][3]);                             \
                }                                                                               \
            }
            {                                                                                   // S2
                T c0[NF], c1[NF], c2[NF], c3[NF], c4[NF];
                load_fence();
                ld.first(c0, c1, c2);
                SHK_PRED(0, c0, c1) SHK_PRED(1, c1, c2)
                load_fence();
                ld.second(c3, c4);
                SHK_PRED(2, c2, c3) SHK_PRED(3, c3, c4)
            }
#undef SHK_PRED
            eps1 = eps[4]; fE[0] = pv[4]; fE[1] = pv[5]; fM[0] = pp[4]; fM[1] = pp[5];
            if constexpr (EOS != EOS_GAMMA) {
                // general EOS: S3 and the geometry run in the CONSUMER (HalfStep below): the two Newton solves of a cell
                // are split between the two warps of the pair.  The message is what S3 needs: E~, M~_par, |M~|^2, R~.
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    msg[j][0] = ut[j][0];
                    msg[j][1] = ut[j][1];
                    msg[j][2] = (T)fma((double)ut[j][1], (double)ut[j][1], fma((double)ut[j][2], (double)ut[j][2], (double)ut[j][3] * (double)ut[j][3]));
                    msg[j][3] = ut[j][NF - 1];
                }
                return;
            }
            T vh[4], ph[4];
            c2p_group<T>(k, ut[0], ut[1], ut[2], ut[3], vh, ph, [&](int jj, T (&u)[NF]) {      // S3: U~ was parked in scr
                load2(scr + 128 * jj, u[0], u[1]);
                load2(scr + 128 * jj + 64, u[2], u[3]);
                u[NF - 1] = T(0);
            }, scr);
            if (SHK_GEOM_C) {       // A/B: the corrector's geometry in the consumer (HalfStep), the message is {v, p} at n+1/2
#pragma unroll
                for (int j = 0; j < 4; ++j) { msg[j][0] = vh[j]; msg[j][1] = ph[j]; msg[j][2] = T(0); msg[j][3] = T(0); }
                return;
            }
            T eh[5], gv[6], gp[6];
            eh[0] = epsh2; gv[0] = gE[0]; gv[1] = gE[1]; gp[0] = gM[0]; gp[1] = gM[1];
#pragma unroll
            for (int j = 0; j < 4; ++j) { eh[j + 1] = k.lam * vh[j]; gv[j + 2] = ph[j] * vh[j]; gp[j + 2] = ph[j]; }
#pragma unroll
            for (int j = 0; j < 4; ++j) {                                       // geometry + sources of S4
                const T q = (T(0.5) - eh[j]) * fast_rcp(T(1) + (eh[j + 1] - eh[j]));
                msg[j][0] = T(0.5) - q;
                msg[j][1] = (T(0.5) * q) * q;
                msg[j][2] = -k.hlam * (gv[j + 2] - gv[j]);
                msg[j][3] = -k.hlam * (gp[j + 2] - gp[j]);
            }
            epsh2 = eh[4]; gE[0] = gv[4]; gE[1] = gv[5]; gM[0] = gp[4]; gM[1] = gp[5];
        }
    }
};

// General EOS only: S3 (cons2prim of the half-step state) and the corrector's geometry, run by the CONSUMER at the top of a
// group, before its four steps, when only its carried window is alive in registers.  Reads the producer's message
// {E~, M~_par, |M~|^2, R~} of the four cells from this lane's slots of the message buffer and overwrites them with what
// Consumer::step expects: {a_c, b_c, sE, sM}.  State: half-step cells -2 (epsh2, gE[1], gM[1]) and -3 (gE[0], gM[0]).
template <typename T, int EOS>
struct HalfStep {
    T epsh2, gE[2], gM[2];
    __device__ __forceinline__ void init() { epsh2 = gE[0] = gE[1] = gM[0] = gM[1] = T(0); }
    __device__ __forceinline__ void group(const Consts<T>& k, T* mq)
    {
        T vh[4], ph[4];
        if constexpr (EOS == EOS_GAMMA) {
#pragma unroll
            for (int j = 0; j < 4; ++j) load2(mq + 128 * j, vh[j], ph[j]);
        } else {
            // one loop body for both pairs (instruction cache, see c2p_pairs_general): results back through the slots
#pragma unroll 1
            for (int jp = 0; jp < 4; jp += 2) {
                T* ma = mq + 128 * jp;
                T a0, a1, a2, a3, b0, b1, b2, b3;
                load2(ma, a0, a1); load2(ma + 64, a2, a3);
                load2(ma + 128, b0, b1); load2(ma + 192, b2, b3);
                Newt<EOS> na, nb;
                na.init_em(k.d, (double)a0, (double)a1, (double)a2, (double)a3);
                nb.init_em(k.d, (double)b0, (double)b1, (double)b2, (double)b3);
                for (int it = 0; it < 48; ++it) {
                    na.iter(k.d); nb.iter(k.d);
                    if (__all_sync(__activemask(), na.done && nb.done)) break;
                }
                double va, pa, vb, pb;
                na.finish(k.d, va, pa); nb.finish(k.d, vb, pb);
                store2(ma, (T)va, (T)pa);
                store2(ma + 128, (T)vb, (T)pb);
            }
            load_fence();
#pragma unroll
            for (int j = 0; j < 4; ++j) load2(mq + 128 * j, vh[j], ph[j]);
        }
        T eh[5], gv[6], gp[6];
        eh[0] = epsh2; gv[0] = gE[0]; gv[1] = gE[1]; gp[0] = gM[0]; gp[1] = gM[1];
#pragma unroll
        for (int j = 0; j < 4; ++j) { eh[j + 1] = k.lam * vh[j]; gv[j + 2] = ph[j] * vh[j]; gp[j + 2] = ph[j]; }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const T q = (T(0.5) - eh[j]) * fast_rcp(T(1) + (eh[j + 1] - eh[j]));
            store2(mq + 128 * j, T(0.5) - q, (T(0.5) * q) * q);
            store2(mq + 128 * j + 64, -k.hlam * (gv[j + 2] - gv[j]), -k.hlam * (gp[j + 2] - gp[j]));
        }
        epsh2 = eh[4]; gE[0] = gv[4]; gE[1] = gv[5]; gM[0] = gp[4]; gM[1] = gp[5];
        load_fence();
    }
};

template <typename T>
struct Consumer {
    T dl[4][NF];        // Delta_2..Delta_5 (Delta_2 is formed in the step)   slot (PH-k)&3
    T fc[NF];           // corrector flux F at interface (i-3,i-2)
    T uh[2][NF];        // U^_3, U^_4                                         slot (PH-k)&1
    T dh[2][NF];        // D^_4, D^_5                                         slot (PH-k)&1
    T a5[NF];           // A_5
    T aq;               // diff / 8
    T ad2;              // -1/8 (phoenical) | 0 (explicit antidiffusion)

    __device__ __forceinline__ void init(T aq_, T ad2_)
    {
        aq = aq_;
        ad2 = ad2_;
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
            const T aph = aq * t_fma(ad2, d2, dh[E4][f]);                        // eq. (19) (x diff: exact scaling, same bits as the oracle)
            const T a4 = limiter<T>(aph, dh3, dh[E5][f]);                        // eqs. (20),(21)
            un[f] = uh[H4][f] - (a4 - a5[f]);                                    // eq. (22)
            a5[f] = a4;
            dh[E5][f] = dh3;
            uh[H4][f] = uh2;
        }
    }
};

// Producer/consumer hand-over of one warp pair: named barriers of 64 threads each, 32 that arrive (do not wait) and 32
// that sync (wait): the PTX producer/consumer pattern.
__device__ __forceinline__ void bar_sync64(int id) { asm volatile("bar.sync %0, 64;" ::"r"(id) : "memory"); }
__device__ __forceinline__ void bar_arrive64(int id) { asm volatile("bar.arrive %0, 64;" ::"r"(id) : "memory"); }

constexpr int XV_CH = 4;                // cells per group
constexpr int XV_TILE = 32 * XV_CH;     // elements per (group, field) tile

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

// element offset of (row, cell c in 0..3) inside an x-sweep tile [32 rows][4 cells] with the 32 B swizzle
// (fp64: rows of 32 B).  fp32 tiles have 16 B rows, one swizzle atom, so they are dense (TMA: CU_TENSOR_MAP_SWIZZLE_NONE).
template <typename T>
__device__ __forceinline__ int xv_off(int row, int c)
{
    return sizeof(T) == 8 ? row * 4 + 2 * ((c >> 1) ^ ((row >> 2) & 1)) + (c & 1) : row * 4 + c;
}

// ================================================================================================
// Round 2: TMA-fed y/z march, one 4-cell group per hand-over.
// ncu's stall samples of the round-1 kernels say the PRODUCER is the critical warp of a pair (5.8 cycles per issued
// instruction: serial cons2prim chains cut into small basic blocks by the clamp branch; the consumer idles at the
// hand-over 11 % of its time).  So
//   * the producer issues NO per-thread global loads: the five fields of a 4-cell group of its 32 pencils arrive as
//     one TMA box {32 x, 4 cells} per field (3-D tensor map over (x, y, z); ghost groups: four 1-cell boxes with the
//     ghost-mapped coordinate, reading G11), so the ~28 address/LDGSTS/ring-slot instructions per step are gone;
//   * a hand-over chunk is one 4-cell group and the producer's part of it is ONE basic block (no branch in
//     c2p_sweep_d<EOS_GAMMA>), so the four independent cons2prim chains of a group interleave.
constexpr int YZ_G = 4;           // ring tiles (4-cell groups) per warp pair
constexpr int YZ_CH = 4;          // cells per group = steps per hand-over chunk
#ifndef SHK_YZ_PREG
#define SHK_YZ_PREG 96
#endif
constexpr int YZ_PREG = SHK_YZ_PREG;          // registers per producer thread (setmaxnreg); consumer gets 256 - YZ_PREG
constexpr int YZ_CREG = 256 - YZ_PREG;
#ifndef SHK_X_PREG
#define SHK_X_PREG 96
#endif
constexpr int X_PREG = SHK_X_PREG;            // x sweep: its consumer (staging tile addresses) needs the full 160
constexpr int X_CREG = 256 - X_PREG;
// General-EOS kernels (EOS_MASS, EOS_TABLE): SHK_GEN_CTAS = 1 builds them as ONE CTA per SM with a wide register split and
// no spill; measured on B200 (config 3, 128^3) that is slower (3.64 G cell-updates/s) than two CTAs per SM with the
// ~100 B of spills the x kernels and the emitting y/z kernels keep (4.42 G): the Newton chains want the warps more.
#ifndef SHK_GEN_CTAS
#define SHK_GEN_CTAS 2
#endif
constexpr int GEN_CTAS = SHK_GEN_CTAS;
#ifndef SHK_GEN_PREG
#define SHK_GEN_PREG 80
#endif
constexpr int GEN_PREG = GEN_CTAS == 1 ? 168 : SHK_GEN_PREG, GEN_CREG = GEN_CTAS == 1 ? 232 : 256 - SHK_GEN_PREG;

template <typename T>
struct alignas(128) YzPair {      // TMA destinations need 128 B alignment
    T ring[YZ_G][NF][YZ_CH][32];          // tile = what TMA boxes {32, 4} of the five fields produce: [field][cell][lane]
    T msg[2][YZ_CH][2][32][2];            // per step {a_c, b_c} and {sE, sM}: one 16 B access per lane (fp64), conflict-free
    unsigned long long bar[8];            // bar[q]: TMA completion of ring tile q
};                                        // fp64: 28800 B; 4 pairs = 112.5 KB per CTA, two CTAs per SM (diagnostic counters live in registers)
template <typename T>
struct YzSmem {
    YzPair<T> pair[4];
};

// tensor maps of a y or z sweep: 3-D {nx, ny, nz}; in4: box {32, 4, 1} (y) or {32, 1, 4} (z), in1: box {32, 1, 1}.
// The maps live in DEVICE memory (written once at allocation), NF per kind in natural field order; fidx[slot] is the
// natural index of the permuted slot.  A pointer from the constant bank keeps the descriptor address in uniform
// registers: with the maps as __grid_constant__ parameters every UTMALDG paid a 15-instruction ELECT / R2UR loop.
struct YzMaps {
    const CUtensorMap* in4;
    const CUtensorMap* in1;
    int fidx[NF];
};

// one lane of a converged warp: ptxas then knows the region is single-threaded and issues UTMALDG without an ELECT loop
__device__ __forceinline__ bool elect_one()
{
    unsigned pred;
    asm volatile("{\n.reg .pred p;\nelect.sync _|p, 0xffffffff;\nselp.u32 %0, 1, 0, p;\n}" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, int c0, int c1, int c2, unsigned long long* bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}

// P.axis: 1 = y sweep (pencil = (x, z), cell stride nx), 2 = z sweep (pencil = (x, y), cell stride nx ny).
// grid.x = ceil(nxb * n_other / 4) with nxb = ceil(nx / 32) x-blocks per row: warp pair w of CTA b owns the 32 pencils
// x0 .. x0+31 of row `oth`, (xb, oth) = divmod(4 b + w, nxb); grid.y = segments.
// EMIT: 0 = conserved fields only; 1 = also the six primitives of the NEW state (last sweep of a step); 2 = also the six
// primitives of the state this sweep READS (the deferred primitive output of a step whose last sweep ran along x: the
// consumer has U^n of its output cell in the ring tile of the previous group).
template <typename T, int EOS, int EMIT, bool TMA>
__global__ void __launch_bounds__(256, (EOS == EOS_GAMMA) ? 2 : GEN_CTAS) sweep_yz_kernel(const __grid_constant__ SweepParams P,
                                                          const __grid_constant__ Consts<T> k,
                                                          const __grid_constant__ YzMaps maps)
{
    extern __shared__ __align__(1024) unsigned char smem_yz[];
    const int lane = threadIdx.x & 31;
    const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);     // provably warp-uniform: TMA operands stay in uniform registers
    const bool producer = warp < 4;
    YzPair<T>& S = reinterpret_cast<YzSmem<T>*>(smem_yz)->pair[warp & 3];
    const int bar_id = 4 * (warp & 3);                      // full0, full1, empty0, empty1 of this pair
    const int nxb = (P.nx + 31) >> 5;
    const long long pg = P.pbase + (long long)blockIdx.x * 4 + (warp & 3);   // pencil group
    const bool idle = pg >= P.npencil;                      // npencil = nxb * n_other pencil GROUPS for this kernel
    const int oth = (int)(pg / nxb);
    const int x0 = 32 * (int)(pg - (long long)oth * nxb);
    // batch of independent events stacked along z: a y sweep sees nz * B planes, a z sweep B * ny rows of
    // pencils, event `ob` owning the cells [ob * N, (ob + 1) * N) of the stacked z axis
    const int ob = oth / P.odiv, oy = oth - ob * P.odiv;
    const int zoff = ob * P.N;
    const bool active = x0 + lane < P.nx;
    const int xl = active ? x0 + lane : P.nx - 1;           // idle lanes shadow a valid pencil (non-TMA fill), store nothing
    const int j0 = blockIdx.y * P.seg;
    const int j1 = min(P.N, j0 + P.seg);
    const int ilo = j0 - GH;
    const int N = P.N;
    const int nsteps = (j1 - j0) + 2 * GH;                  // front cells ilo .. j1+3
    const int ngroups = (nsteps + YZ_CH - 1) / YZ_CH;
    const long long sa = P.stride_axis;
    const bool ysweep = P.axis == 1;

    if (producer) {
        if (sizeof(T) == 8) {
            if constexpr (EOS == EOS_GAMMA) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(YZ_PREG));
            else asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(GEN_PREG));
        }
        if (idle) return;
        Producer<T, EOS> pr;
        pr.init();
        if (TMA) {
            if (lane == 0) {
#pragma unroll
                for (int q = 0; q < YZ_G; ++q) mbar_init(&S.bar[q], 1);
            }
            fence_proxy_async();
            __syncwarp();
        }
        unsigned phase = 0;             // bit q: parity to wait for on bar[q]
        const long long lbase = (long long)xl + (long long)oy * P.stride_other + (long long)zoff * sa;
        constexpr int NP = Producer<T, EOS>::NP;
        // group g = cells ilo+4g .. ilo+4g+3 -> ring tile g % 4.  Group g+1 is requested at the start of group g into
        // the tile of group g-3, which the consumer finished reading in its group g-2 (the `empty` barrier below).
#pragma unroll 1
        for (int g = -1; g < ngroups; ++g) {
            if (g >= 2) bar_sync64(bar_id + 2 + (g & 1));       // the consumer has finished group g-2
            if (g + 1 < ngroups) {
                const int q = (g + 1) & (YZ_G - 1);
                const int jg = ilo + YZ_CH * (g + 1);
                if (TMA) {
                    if (elect_one()) {
                        mbar_expect_tx(&S.bar[q], NF * YZ_CH * 32 * (unsigned)sizeof(T));
                        if (jg >= 0 && jg + YZ_CH <= N) {
#pragma unroll
                            for (int f = 0; f < NF; ++f)
                                tma_load_3d(&S.ring[q][f][0][0], maps.in4 + maps.fidx[f], x0, ysweep ? jg : oy, ysweep ? oth : zoff + jg, &S.bar[q]);
                        } else {        // ghost group (reading G11): 1-cell boxes at the ghost-mapped coordinate; rare, kept small
#pragma unroll 1
                            for (int c = 0; c < YZ_CH; ++c) {
                                const int jj = ghost_index(jg + c, N, P.periodic);
#pragma unroll 1
                                for (int f = 0; f < NF; ++f)
                                    tma_load_3d(&S.ring[q][f][c][0], maps.in1 + maps.fidx[f], x0, ysweep ? jj : oy, ysweep ? oth : zoff + jj, &S.bar[q]);
                            }
                        }
                    }
                } else {
#pragma unroll 1
                    for (int c = 0; c < YZ_CH; ++c) {
                        const long long o = lbase + (long long)ghost_index(jg + c, N, P.periodic) * sa;
#pragma unroll
                        for (int f = 0; f < NF; ++f) cp_async_elem<T>(&S.ring[q][f][c][lane], (const T*)P.in[f] + o);
                    }
                }
            }
            if (!TMA) cp_async_commit();        // one commit group per iteration (empty past the last group)
            if (g < 0) continue;
            if (TMA) {
                const int q = g & (YZ_G - 1);
                mbar_wait(&S.bar[q], (phase >> q) & 1u);
                phase ^= 1u << q;
            } else {
                cp_async_wait<1>();
            }
            const T* tp = &S.ring[(g + YZ_G - 1) & (YZ_G - 1)][0][YZ_CH - 1][lane];     // last cell of the previous group
            const T* tc = &S.ring[g & (YZ_G - 1)][0][0][lane];
            T mm[4][4];
            struct {
                const T *tp, *tc;
                __device__ __forceinline__ void first(T (&um)[NF], T (&c0)[NF], T (&c1)[NF]) const
                {
                    um[NF - 1] = c0[NF - 1] = c1[NF - 1] = T(0);
#pragma unroll
                    for (int f = 0; f < NP; ++f) {
                        um[f] = tp[f * YZ_CH * 32];
                        c0[f] = tc[f * YZ_CH * 32];
                        c1[f] = tc[f * YZ_CH * 32 + 32];
                    }
                }
                __device__ __forceinline__ void second(T (&c2)[NF], T (&c3)[NF]) const
                {
                    c2[NF - 1] = c3[NF - 1] = T(0);
#pragma unroll
                    for (int f = 0; f < NP; ++f) {
                        c2[f] = tc[f * YZ_CH * 32 + 64];
                        c3[f] = tc[f * YZ_CH * 32 + 96];
                    }
                }
                __device__ __forceinline__ void pair(int pi, T (&a)[NF], T (&b)[NF]) const      // cells 2 pi, 2 pi + 1
                {
                    a[NF - 1] = b[NF - 1] = T(0);
#pragma unroll
                    for (int f = 0; f < NP; ++f) {
                        a[f] = tc[f * YZ_CH * 32 + 64 * pi];
                        b[f] = tc[f * YZ_CH * 32 + 64 * pi + 32];
                    }
                }
                __device__ __forceinline__ void cell(int j, T (&u)[NF]) const                   // cell j of the group
                {
                    u[NF - 1] = T(0);
#pragma unroll
                    for (int f = 0; f < NP; ++f) u[f] = tc[f * YZ_CH * 32 + 32 * j];
                }
            } ld = {tp, tc};
            T* mq = &S.msg[g & 1][0][0][lane][0];
            pr.group(k, ld, mq, mm);
#pragma unroll
            for (int j = 0; j < 4; ++j) { store2(mq + 128 * j, mm[j][0], mm[j][1]); store2(mq + 128 * j + 64, mm[j][2], mm[j][3]); }
            bar_arrive64(bar_id + (g & 1));
        }
        if (!TMA) cp_async_wait<0>();
    } else {
        if (sizeof(T) == 8) {
            if constexpr (EOS == EOS_GAMMA) asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(YZ_CREG));
            else asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(GEN_CREG));
        }
        if (idle) return;
        Cnt cnt;
        cnt.zero();
        Consumer<T> co;
        co.init(k.aq, k.ad2);
        HalfStep<T, EOS> hs;
        hs.init();
        // element offset of the output cell of the NEXT step: cell ilo - 4 (the first two groups store nothing)
        long long o = (long long)(x0 + lane) + (long long)oy * P.stride_other + (long long)(zoff + ilo - GH) * sa;
        int left = active ? (j1 - j0) : 0;      // output cells this lane still has to store
#define SHK_YZ_OUT(UN, S_)                                                                          \
        {                                                                                           \
            if (g >= 2 && (S_) < left) {                                                            \
                T pv[6];                                                                            \
                finish_cell<T, EOS, EMIT == 1 && EOS == EOS_GAMMA>(k, UN, pv, cnt);                 \
                _Pragma("unroll") for (int f = 0; f < NF; ++f) ((T*)P.out[f])[o] = UN[f];           \
                if (EMIT == 1 && EOS == EOS_GAMMA) { _Pragma("unroll") for (int qq = 0; qq < 6; ++qq) ((T*)P.prim[qq])[o] = pv[qq]; } \
            }                                                                                       \
            o += sa;                                                                                \
        }
#pragma unroll 1
        for (int g = 0; g < ngroups; ++g) {
            bar_sync64(bar_id + (g & 1));
            const T* tp = &S.ring[(g + YZ_G - 1) & (YZ_G - 1)][0][0][lane];
            const T* tc = &S.ring[g & (YZ_G - 1)][0][0][lane];
            T* mq = &S.msg[g & 1][0][0][lane][0];
            if constexpr (EOS != EOS_GAMMA || SHK_GEOM_C) hs.group(k, mq);       // S3 + geometry (general EOS)
            T uq[NF], ua[NF], c0[NF], c1[NF], c2[NF], msg[4], un[NF];
#pragma unroll
            for (int f = 0; f < NF; ++f) {
                uq[f] = tp[f * YZ_CH * 32 + 64];
                ua[f] = tp[f * YZ_CH * 32 + 96];
                c0[f] = tc[f * YZ_CH * 32];
            }
            load2(mq, msg[0], msg[1]); load2(mq + 64, msg[2], msg[3]);
            co.template step<0>(uq, ua, msg, un);
            SHK_YZ_OUT(un, 0)
#pragma unroll
            for (int f = 0; f < NF; ++f) c1[f] = tc[f * YZ_CH * 32 + 32];
            load2(mq + 128, msg[0], msg[1]); load2(mq + 192, msg[2], msg[3]);
            co.template step<1>(ua, c0, msg, un);
            SHK_YZ_OUT(un, 1)
#pragma unroll
            for (int f = 0; f < NF; ++f) c2[f] = tc[f * YZ_CH * 32 + 64];
            load2(mq + 256, msg[0], msg[1]); load2(mq + 320, msg[2], msg[3]);
            co.template step<2>(c0, c1, msg, un);
            SHK_YZ_OUT(un, 2)
            load2(mq + 384, msg[0], msg[1]); load2(mq + 448, msg[2], msg[3]);
            co.template step<3>(c1, c2, msg, un);
            SHK_YZ_OUT(un, 3)
            if (EMIT == 1 && EOS != EOS_GAMMA && g >= 2) {
                // general EOS: the primitives of the group's four output cells in ONE rolled loop body (a full Newton solve per
                // cell; inlined into the four steps it made the consumer 47-57 KB of code, far beyond the instruction cache).
                // The cells are read back from global memory: this thread stored them a moment ago.
#pragma unroll 1
                for (int c = 0; c < YZ_CH; ++c) {
                    if (c < left) {
                        const long long oc = o + (long long)(c - YZ_CH) * sa;
                        T uo[NF], pv[6];
#pragma unroll
                        for (int f = 0; f < NF; ++f) uo[f] = ((const T*)P.out[f])[oc];
                        emit_primitives<T, EOS>(k, uo, pv, cnt);
#pragma unroll
                        for (int qq = 0; qq < 6; ++qq) ((T*)P.prim[qq])[oc] = pv[qq];
                    }
                }
            }
            if (EMIT == 2 && g >= 2) {
                // primitives of the INPUT state of this group's output cells = the four cells of the previous group's ring
                // tile; done after the four steps, when only the carried window is alive in registers
                load_fence();
                auto emit_in_cell = [&](int c) {
                    if (c < left) {
                        // momenta in NATURAL order (x, y, z), so that |M|^2 rounds as in the element-wise pass this replaces
                        // (same bits): slots of a y sweep hold (My, Mz, Mx), of a z sweep (Mz, Mx, My)
                        T ui[NF], pv[6];
                        const T m1 = tp[1 * YZ_CH * 32 + 32 * c], m2 = tp[2 * YZ_CH * 32 + 32 * c], m3 = tp[3 * YZ_CH * 32 + 32 * c];
                        ui[0] = tp[32 * c];
                        ui[1] = ysweep ? m3 : m2;
                        ui[2] = ysweep ? m1 : m3;
                        ui[3] = ysweep ? m2 : m1;
                        ui[4] = tp[4 * YZ_CH * 32 + 32 * c];
                        emit_primitives<T, EOS>(k, ui, pv, cnt);
                        const long long oc = o + (long long)(c - YZ_CH) * sa;
#pragma unroll
                        for (int qq = 0; qq < 3; ++qq) ((T*)P.prim[qq])[oc] = pv[qq];
                        ((T*)P.prim[ysweep ? 5 : 4])[oc] = pv[3];
                        ((T*)P.prim[ysweep ? 3 : 5])[oc] = pv[4];
                        ((T*)P.prim[ysweep ? 4 : 3])[oc] = pv[5];
                    }
                };
                if constexpr (EOS == EOS_GAMMA) {
#pragma unroll
                    for (int c = 0; c < YZ_CH; ++c) emit_in_cell(c);       // unrolled: rolled measured 0.449 vs 0.421 ms (four independent chains)
                } else {
#pragma unroll 1
                    for (int c = 0; c < YZ_CH; ++c) emit_in_cell(c);       // general EOS: one copy of the Newton solve (instruction cache)
                }
            }
            if (g >= 2) left -= YZ_CH;
            if (g + 2 < ngroups) bar_arrive64(bar_id + 2 + (g & 1));
        }
#undef SHK_YZ_OUT
        flush_counts(cnt, P.counts);
    }
}


// ------------------------------------------------------------------------------------------------
// x sweep, round 2: the same group-wise producer/consumer pair with lane r marching along ROW r of a 32-row strip.
// A (group, field) tile is [32 rows][4 cells], dense (1 KB in fp64) with the two 16 B halves of a row swapped when bit 2
// of the row is set: what a TMA box {4 cells, 32 rows} with CU_TENSOR_MAP_SWIZZLE_32B produces, so that a lane reads
// an aligned cell pair of its row with one conflict-free LDS.128.  Outputs of a group are staged in `outb` (same
// layout) and leave as one TMA box per field.  Three ring tiles suffice because the consumer releases a tile as soon
// as it has READ it (top of its group), not when it has finished the group.
constexpr int X2_G = 3;

// fp32 storage with TMA ("SUPER" in the kernel): a ring / staging tile holds EIGHT cells of a row, [32 rows][8 cells] = the
// same 32 B rows and 32 B swizzle as an fp64 tile, filled by one TMA box {8, 32}: a 4-cell group of the march is one half
// of it.  With {4, 32} boxes of 16 B rows the fp32 x sweep spent 25 % of its stall samples waiting for TMA data (ncu) and
// ran slower than the fp64 one: the TMA unit works per row piece, and 16 B pieces are the worst case.
template <typename T> struct X2Stride { static constexpr int value = sizeof(T) == 4 ? 2 * XV_TILE : XV_TILE; };

template <typename T>
struct alignas(256) X2Pair {
    T ring[X2_G][NF][X2Stride<T>::value];
    T outb[NF][X2Stride<T>::value];
    T msg[2][YZ_CH][2][32][2];
    unsigned long long bar[4];            // bar[q], q < 3: TMA completion of ring tile q; bar[3]: scratch (early release)
};                                        // fp64: 28928 B; 4 pairs = 113 KB per CTA: two CTAs per SM, exactly
template <typename T>
struct X2Smem {
    X2Pair<T> pair[4];
};

// tensor maps of the x sweep in DEVICE memory (see YzMaps): 2-D {nx, ny*nz}, box {4, 32}, 32 B swizzle
struct X2Maps {
    const CUtensorMap* in;
    const CUtensorMap* out;
    int fidx[NF];
};

template <typename T, int EOS, bool EMIT, bool TMA>
__global__ void __launch_bounds__(256, (EOS == EOS_GAMMA) ? 2 : GEN_CTAS) sweep_x2_kernel(const __grid_constant__ SweepParams P,
                                                          const __grid_constant__ Consts<T> k,
                                                          const __grid_constant__ X2Maps maps)
{
    extern __shared__ __align__(1024) unsigned char smem_x2[];
    const int lane = threadIdx.x & 31;
    const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
    const bool producer = warp < 4;
    X2Pair<T>& S = reinterpret_cast<X2Smem<T>*>(smem_x2)->pair[warp & 3];
    const int bar_id = 4 * (warp & 3);                      // full0, full1, empty0, empty1 of this pair
    const long long row0 = P.pbase + (long long)blockIdx.x * 128 + (warp & 3) * 32;
    const bool idle = row0 >= P.npencil;
    const int nrows = (int)min(32LL, P.npencil - row0);
    const int j0 = blockIdx.y * P.seg;
    const int j1 = min(P.N, j0 + P.seg);
    const int ilo = j0 - GH;
    const int N = P.N;
    const int nsteps = (j1 - j0) + 2 * GH;
    const int ngroups = (nsteps + XV_CH - 1) / XV_CH;
    const int col = lane & 3, rsub = lane >> 2;             // element map of the LSU group copies: col, rows rsub + 8 kk
    constexpr bool SUPER = TMA && sizeof(T) == 4;           // fp32 + TMA: 8-cell tiles, a group is one half (see X2Pair)
    constexpr int FS = X2Stride<T>::value;                // elements between the fields of a tile
    const int sw = (sizeof(T) == 8 || SUPER) ? (lane >> 2) & 1 : 0;    // 32 B swizzle of this lane's row (32 B rows only)
    constexpr int XALIGN = 16 / (int)sizeof(T);             // cells per 16 B: TMA boxes start at 16 B aligned cells
    // SUPER: group G is half (G + 1) & 1 of the 8-cell tile (G + 1) >> 1 of this segment, which starts at cell
    // j0 - 8 + 8 ((G + 1) >> 1) (j0 is a multiple of 8: x segments are); element offset of (row, half h, cell c) in it:
    auto soff = [](int row, int h, int c) { return row * 8 + 4 * (h ^ ((row >> 2) & 1)) + c; };

    if (producer) {
        if (sizeof(T) == 8) {
            if constexpr (EOS == EOS_GAMMA) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(X_PREG));
            else asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(GEN_PREG));
        }
        if (idle) return;
        Producer<T, EOS> pr;
        pr.init();
        if (TMA) {
            if (lane == 0) {
#pragma unroll
                for (int q = 0; q < X2_G; ++q) mbar_init(&S.bar[q], 1);
            }
            fence_proxy_async();
            __syncwarp();
        }
        unsigned phase = 0;
        constexpr int NP = Producer<T, EOS>::NP;
        // a group that lies inside [0, N) and starts at an even cell is one TMA box per field; a group that touches a
        // boundary needs the ghost map (reading G11) and is copied element by element (cp.async)
        auto group_is_tma = [&](int g) { const int xg = ilo + XV_CH * g; return TMA && xg >= 0 && xg + XV_CH <= N && (xg % XALIGN) == 0; };
        int q1 = 0;                     // ring tile of group g+1
#pragma unroll 1
        for (int g = -1; g < ngroups; ++g) {
            if (g >= 1) bar_sync64(bar_id + 2 + ((g - 1) & 1));     // the consumer has read what it needs of group g-2
            const T *tp, *tc;
            if constexpr (SUPER) {
                // fp32: 8-cell tiles.  Group G touches tile (G + 1) >> 1; a tile inside [0, N) is ONE TMA box {8, 32} per
                // field, requested when its first group comes up (two groups ahead of its second half); a tile that touches
                // a boundary is filled half by half through the ghost map (cp.async)
                auto tile_x = [&](int G) { return j0 - 8 + 8 * ((G + 1) >> 1); };
                auto tile_tma = [&](int G) { const int xs = tile_x(G); return xs >= 0 && xs + 8 <= N; };
                auto first_touch = [&](int G) { return G == 0 || ((G + 1) & 1) == 0; };
                const int G = g + 1;
                if (G < ngroups) {
                    const int hh = (G + 1) & 1, qs = ((G + 1) >> 1) % X2_G, xs = tile_x(G);
                    if (tile_tma(G)) {
                        if (first_touch(G) && elect_one()) {
                            mbar_expect_tx(&S.bar[qs], NF * FS * (unsigned)sizeof(T));
#pragma unroll
                            for (int f = 0; f < NF; ++f)
                                tma_load_2d(&S.ring[qs][f][0], maps.in + maps.fidx[f], xs, (int)row0, &S.bar[qs]);
                        }
                    } else {
                        const int gi = ghost_index(xs + 4 * hh + col, N, P.periodic);
                        T* dst = &S.ring[qs][0][0];
#pragma unroll 1
                        for (int kk = 0; kk < 4; ++kk) {
                            const int row = rsub + 8 * kk;
                            if (row < nrows) {
                                const long long o = (row0 + row) * (long long)N + gi;
                                const int so = soff(row, hh, col);
#pragma unroll
                                for (int f = 0; f < NF; ++f) cp_async_elem<T>(dst + f * FS + so, (const T*)P.in[f] + o);
                            }
                        }
                        cp_async_commit();
                    }
                }
                if (g < 0) continue;
                const int hh = (g + 1) & 1, qs = ((g + 1) >> 1) % X2_G;
                if (tile_tma(g)) {
                    if (first_touch(g)) {
                        mbar_wait(&S.bar[qs], (phase >> qs) & 1u);
                        phase ^= 1u << qs;
                    }
                } else {
                    if (G < ngroups && !tile_tma(G)) cp_async_wait<1>(); else cp_async_wait<0>();
                    __syncwarp();
                }
                tc = &S.ring[qs][0][lane * 8 + 4 * (hh ^ sw)];
                tp = hh ? &S.ring[qs][0][lane * 8 + 4 * sw + 3]                                   // cell 3 of half 0, same tile
                        : &S.ring[(qs + X2_G - 1) % X2_G][0][lane * 8 + 4 * (1 ^ sw) + 3];       // cell 3 of half 1, previous tile
            } else {
            if (g + 1 < ngroups) {
                const int xg = ilo + XV_CH * (g + 1);
                if (group_is_tma(g + 1)) {
                    if (elect_one()) {
                        mbar_expect_tx(&S.bar[q1], NF * XV_TILE * (unsigned)sizeof(T));
#pragma unroll
                        for (int f = 0; f < NF; ++f)
                            tma_load_2d(&S.ring[q1][f][0], maps.in + maps.fidx[f], xg, (int)row0, &S.bar[q1]);
                    }
                } else {
                    const int gi = ghost_index(xg + col, N, P.periodic);
                    T* dst = &S.ring[q1][0][0];
#pragma unroll 1
                    for (int kk = 0; kk < 4; ++kk) {
                        const int row = rsub + 8 * kk;
                        if (row < nrows) {
                            const long long o = (row0 + row) * (long long)N + gi;
                            const int so = xv_off<T>(row, col);
#pragma unroll
                            for (int f = 0; f < NF; ++f) cp_async_elem<T>(dst + f * FS + so, (const T*)P.in[f] + o);
                        }
                    }
                    cp_async_commit();
                }
            }
            const int q0 = (q1 == 0) ? X2_G - 1 : q1 - 1;           // tile of group g
            q1 = (q1 + 1 == X2_G) ? 0 : q1 + 1;
            if (g < 0) continue;
            if (group_is_tma(g)) {
                mbar_wait(&S.bar[q0], (phase >> q0) & 1u);
                phase ^= 1u << q0;
            } else {
                // LSU groups are rare and at most two are in flight (g, g+1): wait for all but the youngest
                if (g + 1 < ngroups && !group_is_tma(g + 1)) cp_async_wait<1>(); else cp_async_wait<0>();
                __syncwarp();
            }
            const int qm = (q0 == 0) ? X2_G - 1 : q0 - 1;           // tile of group g-1
            tp = &S.ring[qm][0][xv_off<T>(lane, 3)];
            tc = &S.ring[q0][0][lane * 4];
            }
            T mm[4][4];
            struct {
                const T *tp, *tc;
                int sw;
                // SUPER: tc points at this lane's 16 B half row (four cells): one LDS.128; else at its 4-cell row with the
                // two 16 B halves swizzled (fp64) or dense (fp32 without TMA)
                __device__ __forceinline__ void first(T (&um)[NF], T (&c0)[NF], T (&c1)[NF]) const
                {
                    um[NF - 1] = c0[NF - 1] = c1[NF - 1] = T(0);
#pragma unroll
                    for (int f = 0; f < NP; ++f) {
                        um[f] = tp[f * FS];
                        if constexpr (SUPER) load2(tc + f * FS, c0[f], c1[f]);
                        else load2(tc + f * FS + 2 * sw, c0[f], c1[f]);
                    }
                }
                __device__ __forceinline__ void second(T (&c2)[NF], T (&c3)[NF]) const
                {
                    c2[NF - 1] = c3[NF - 1] = T(0);
#pragma unroll
                    for (int f = 0; f < NP; ++f) {
                        if constexpr (SUPER) load2(tc + f * FS + 2, c2[f], c3[f]);
                        else load2(tc + f * FS + 2 * (1 ^ sw), c2[f], c3[f]);
                    }
                }
                __device__ __forceinline__ void pair(int pi, T (&a)[NF], T (&b)[NF]) const      // cells 2 pi, 2 pi + 1
                {
                    a[NF - 1] = b[NF - 1] = T(0);
#pragma unroll
                    for (int f = 0; f < NP; ++f) {
                        if constexpr (SUPER) load2(tc + f * FS + 2 * pi, a[f], b[f]);
                        else load2(tc + f * FS + 2 * (pi ^ sw), a[f], b[f]);
                    }
                }
                __device__ __forceinline__ void cell(int j, T (&u)[NF]) const                   // cell j of the group
                {
                    u[NF - 1] = T(0);
#pragma unroll
                    for (int f = 0; f < NP; ++f) u[f] = SUPER ? tc[f * FS + j] : tc[f * FS + 2 * ((j >> 1) ^ sw) + (j & 1)];
                }
            } ld = {tp, tc, sw};
            T* mq = &S.msg[g & 1][0][0][lane][0];
            pr.group(k, ld, mq, mm);
#pragma unroll
            for (int j = 0; j < 4; ++j) { store2(mq + 128 * j, mm[j][0], mm[j][1]); store2(mq + 128 * j + 64, mm[j][2], mm[j][3]); }
            bar_arrive64(bar_id + (g & 1));
        }
        cp_async_wait<0>();
    } else {
        if (sizeof(T) == 8) {
            if constexpr (EOS == EOS_GAMMA) asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(X_CREG));
            else asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(GEN_CREG));
        }
        if (idle) return;
        Cnt cnt;
        cnt.zero();
        Consumer<T> co;
        co.init(k.aq, k.ad2);
        HalfStep<T, EOS> hs;
        hs.init();
        int q0 = 0;                     // ring tile of group g
        bool store_pending = false;
#pragma unroll 1
        for (int g = 0; g < ngroups; ++g) {
            bar_sync64(bar_id + (g & 1));
            const T *tp, *tc;
            int ho = 0;                 // SUPER: half of the staging tile that takes this group's outputs (cells of group g-1)
            if constexpr (SUPER) {
                const int hh = (g + 1) & 1, qs = ((g + 1) >> 1) % X2_G;
                tc = &S.ring[qs][0][lane * 8 + 4 * (hh ^ sw)];
                tp = hh ? &S.ring[qs][0][lane * 8 + 4 * sw + 2]                                   // cells 2, 3 of half 0, same tile
                        : &S.ring[(qs + X2_G - 1) % X2_G][0][lane * 8 + 4 * (1 ^ sw) + 2];       // cells 2, 3 of half 1, previous tile
                ho = g & 1;
            } else {
                const int qm = (q0 == 0) ? X2_G - 1 : q0 - 1;
                tp = &S.ring[qm][0][lane * 4 + 2 * (1 ^ sw)];           // cells 2, 3 of group g-1
                tc = &S.ring[q0][0][lane * 4];
            }
            T* mq = &S.msg[g & 1][0][0][lane][0];
            q0 = (q0 + 1 == X2_G) ? 0 : q0 + 1;
            T uq[NF], ua[NF], c0[NF], c1[NF], c2[NF], msg[4], un[NF], uo[NF];
#pragma unroll
            for (int f = 0; f < NF; ++f) load2(tp + f * FS, uq[f], ua[f]);
            // Early release of the tile of group g-1 (the producer's next TMA request refills it).  BAR.ARV does NOT wait
            // for shared-memory loads in flight (measured: issued right behind the LDS, 2.6 % of the cells of a 256^3
            // sweep then differed from run to run), so a 4-byte store whose data depends on all five loads goes first:
            // it cannot issue before uq, ua have arrived, and the barrier stays behind it.
            {
                const unsigned d = (unsigned)(__double2hiint((double)uq[0]) ^ __double2hiint((double)uq[1]) ^ __double2hiint((double)uq[2]) ^
                                              __double2hiint((double)uq[3]) ^ __double2hiint((double)uq[4]));
                *reinterpret_cast<volatile unsigned*>(&S.bar[X2_G]) = d;        // bar[3]: scratch word, never read
                if (g + 1 < ngroups) bar_arrive64(bar_id + 2 + (g & 1));
            }
            const int jf = ilo + XV_CH * g - GH;                            // first output cell of this group
            const bool any_out = g >= 2;                                    // jf >= j0
            if (TMA && store_pending && (!SUPER || ho == 0)) {              // outb is rewritten below: the TMA must have read it
                if (lane == 0) tma_store_wait_read();
                __syncwarp();
                store_pending = false;
            }
            // first and second cell pair of this lane's row in the staging tile
            T* ob = SUPER ? &S.outb[0][lane * 8 + 4 * (ho ^ sw)] : &S.outb[0][lane * 4 + 2 * sw];
            T* ob2 = SUPER ? ob + 2 : &S.outb[0][lane * 4 + 2 * (1 ^ sw)];
            if constexpr (EOS != EOS_GAMMA || SHK_GEOM_C) hs.group(k, mq);       // S3 + geometry (general EOS)
            load2(mq, msg[0], msg[1]); load2(mq + 64, msg[2], msg[3]);
            co.template step<0>(uq, ua, msg, uo);
            if (any_out && jf < j1 && lane < nrows) { T pv[6]; finish_cell<T, EOS, false>(k, uo, pv, cnt); }
            load_fence();
#pragma unroll
            for (int f = 0; f < NF; ++f) load2(tc + f * FS + (SUPER ? 0 : 2 * sw), c0[f], c1[f]);
            load2(mq + 128, msg[0], msg[1]); load2(mq + 192, msg[2], msg[3]);
            co.template step<1>(ua, c0, msg, un);
            if (any_out && jf + 1 < j1 && lane < nrows) { T pv[6]; finish_cell<T, EOS, false>(k, un, pv, cnt); }
#pragma unroll
            for (int f = 0; f < NF; ++f) store2(ob + f * FS, uo[f], un[f]);
            load2(mq + 256, msg[0], msg[1]); load2(mq + 320, msg[2], msg[3]);
            co.template step<2>(c0, c1, msg, uo);
            if (any_out && jf + 2 < j1 && lane < nrows) { T pv[6]; finish_cell<T, EOS, false>(k, uo, pv, cnt); }
            load_fence();
#pragma unroll
            for (int f = 0; f < NF; ++f) c2[f] = tc[f * FS + (SUPER ? 2 : 2 * (1 ^ sw))];
            load2(mq + 384, msg[0], msg[1]); load2(mq + 448, msg[2], msg[3]);
            co.template step<3>(c1, c2, msg, un);
            if (any_out && jf + 3 < j1 && lane < nrows) { T pv[6]; finish_cell<T, EOS, false>(k, un, pv, cnt); }
#pragma unroll
            for (int f = 0; f < NF; ++f) store2(ob2 + f * FS, uo[f], un[f]);
            if (!any_out) continue;
            if constexpr (SUPER && !EMIT) {
                // fp32: the staging tile holds eight cells; it leaves as one TMA box {8, 32} per field when its second half
                // is done (segments are multiples of 8 cells), or after its first half at the ragged end of the grid, where
                // the box is clipped at N (then j1 == N <= jf + 4, so the stale second half lies outside the grid)
                if (ho == 1 || g == ngroups - 1) {
                    fence_proxy_async();
                    __syncwarp();
                    if (lane == 0) {
#pragma unroll
                        for (int f = 0; f < NF; ++f) tma_store_2d(maps.out + maps.fidx[f], jf - 4 * ho, (int)row0, &S.outb[f][0]);
                        tma_store_commit();
                    }
                    store_pending = true;
                }
                continue;
            }
            // the finished group leaves as one TMA box per field when all of its cells are output cells of this segment (or
            // are clipped by the grid edge); otherwise (ragged segment end, odd start, EMIT) through the LSU
            if (TMA && !EMIT && (jf % XALIGN) == 0 && (jf + XV_CH <= j1 || j1 == N)) {
                fence_proxy_async();                        // generic-proxy writes of outb -> visible to the TMA engine
                __syncwarp();
                if (lane == 0) {
#pragma unroll
                    for (int f = 0; f < NF; ++f) tma_store_2d(maps.out + maps.fidx[f], jf, (int)row0, &S.outb[f][0]);
                    tma_store_commit();
                }
                store_pending = true;
            } else {
                __syncwarp();
                const int jo = jf + col;
                if (jo < j1) {
#pragma unroll 1
                    for (int kk = 0; kk < 4; ++kk) {
                        const int row = rsub + 8 * kk;
                        if (row < nrows) {
                            const long long o = (row0 + row) * (long long)N + jo;
                            const int so = SUPER ? soff(row, ho, col) : xv_off<T>(row, col);
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
                                for (int qq = 0; qq < 6; ++qq) ((T*)P.prim[qq])[o] = pv[qq];
                            }
                        }
                    }
                }
                __syncwarp();
            }
        }
        if (TMA && lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
        flush_counts(cnt, P.counts);
    }
}


// ------------------------------------------------------------------------------------------------
// Per-cell path: one thread per cell and sweep, everything recomputed from a window of U^n -- the decomposition of the
// paper's own kernels (one work-item per cell, U-hat recomputed for every neighbour, Listing 1).  It
// exists for the scheme variants the fused kernels do not implement -- the R2 predictor (half step = the complete kernel
// with lambda/2, eqs. (17)-(22); dependency radius 6) -- and as the A/B datapoint "the paper's design
// on this GPU".  It follows the eight steps of DESIGN.md 1 literally on a (2W+1)-cell window; fp64 only.
template <int W>
struct CellWin {
    double u[NF][2 * W + 1];        // U^n at j-W .. j+W (ghost-mapped, reading G11)
    double v[2 * W + 1], p[2 * W + 1];
};

// eq. (17) for one field at window slot m: eps, U at m-1..m+1; src = f_{m+1} - f_{m-1} (0 for source-free fields)
__device__ __forceinline__ double cell_transport(double um, double u0, double up, double em, double e0, double ep,
                                                 double lam, double fm, double fp)
{
    const double Qp = (0.5 - e0) / (1.0 + (ep - e0));            // eq. (15), upper signs (G1)
    const double Qm = (0.5 + e0) / (1.0 - (em - e0));            // lower signs
    const double Dj = up - u0, Djm = u0 - um;                    // eq. (16)
    double uh = 0.5 * Qp * Qp * Dj - 0.5 * Qm * Qm * Djm + (Qp + Qm) * u0;
    uh += lam * (-0.5 * (fp - fm));                              // + lambda Delta(f)
    return uh;
}
// eqs. (18)-(21): limited antidiffusive flux at interface (i, i+1); uh at i-1..i+2, u at i-1..i+2
__device__ __forceinline__ double cell_antiflux(double hm, double h0, double h1, double h2, double um, double u0, double u1,
                                                double u2, double diff, double ad2)
{
    const double Dh = h1 - h0, Dhp = h2 - h1, Dhm = h0 - hm;     // eq. (18)
    const double Di = u1 - u0, Dip = u2 - u1, Dim = u0 - um;
    const double aph = diff * (0.125 * fma(ad2, (Dip + Dim) - 2.0 * Di, Dh));        // eq. (19), G14; ad2 = -1/8 | 0
    const double sg = (aph > 0.0) - (aph < 0.0);                 // eq. (20)
    double m = fmin(fmin(sg * Dhp, fabs(aph)), sg * Dhm);
    return sg * fmax(m, 0.0);                                    // eq. (21)
}

template <int EOS, bool R2>
__global__ void __launch_bounds__(128) sweep_cell_kernel(const __grid_constant__ SweepParams P,
                                                         const __grid_constant__ Consts<double> k, long long ncell,
                                                         double diff, int emit)
{
    constexpr int W = R2 ? 6 : GH;
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= ncell) return;
    const long long sa = P.stride_axis;
    const int N = P.N;
    const int j = (int)((i / sa) % N);
    CellWin<W> w;
    // 1.+2. ghost-extended window and its time-n primitives
#pragma unroll
    for (int m = -W; m <= W; ++m) {
        const long long o = i + (long long)(ghost_index(j + m, N, P.periodic) - j) * sa;
#pragma unroll
        for (int f = 0; f < NF; ++f) w.u[f][m + W] = ((const double*)P.in[f])[o];
        const Prim pr = cons2prim_general<EOS>(k.d, w.u[0][m + W], w.u[1][m + W], w.u[2][m + W], w.u[3][m + W], w.u[4][m + W]);
        w.v[m + W] = w.u[1][m + W] * pr.y;
        w.p[m + W] = pr.p;
    }
    const double lam = k.lam, h = k.hlam;
    // 3. predictor at m = -3..3 (G4: R1 = eq. (17) alone; R2 = eq. (17) then eqs. (18)-(22)), 4. half-step primitives
    double vh[7], ph[7];
    double ut[NF][7];
    if (!R2) {
#pragma unroll
        for (int m = -3; m <= 3; ++m) {
            const int c = m + W;
#pragma unroll
            for (int f = 0; f < NF; ++f) {
                double fm = 0.0, fp = 0.0;
                if (f == 0) { fm = w.p[c - 1] * w.v[c - 1]; fp = w.p[c + 1] * w.v[c + 1]; }
                if (f == 1) { fm = w.p[c - 1]; fp = w.p[c + 1]; }
                ut[f][m + 3] = cell_transport(w.u[f][c - 1], w.u[f][c], w.u[f][c + 1], h * w.v[c - 1], h * w.v[c], h * w.v[c + 1],
                                              h, fm, fp);
            }
        }
    } else {
        double up[NF][11];          // transported half step at m = -5..5
#pragma unroll
        for (int m = -5; m <= 5; ++m) {
            const int c = m + W;
#pragma unroll
            for (int f = 0; f < NF; ++f) {
                double fm = 0.0, fp = 0.0;
                if (f == 0) { fm = w.p[c - 1] * w.v[c - 1]; fp = w.p[c + 1] * w.v[c + 1]; }
                if (f == 1) { fm = w.p[c - 1]; fp = w.p[c + 1]; }
                up[f][m + 5] = cell_transport(w.u[f][c - 1], w.u[f][c], w.u[f][c + 1], h * w.v[c - 1], h * w.v[c], h * w.v[c + 1],
                                              h, fm, fp);
            }
        }
#pragma unroll
        for (int m = -3; m <= 3; ++m) {
            const int c = m + W, q = m + 5;
#pragma unroll
            for (int f = 0; f < NF; ++f) {
                const double a1 = cell_antiflux(up[f][q - 1], up[f][q], up[f][q + 1], up[f][q + 2], w.u[f][c - 1], w.u[f][c],
                                                w.u[f][c + 1], w.u[f][c + 2], diff, k.ad2);
                const double a0 = cell_antiflux(up[f][q - 2], up[f][q - 1], up[f][q], up[f][q + 1], w.u[f][c - 2], w.u[f][c - 1],
                                                w.u[f][c], w.u[f][c + 1], diff, k.ad2);
                ut[f][m + 3] = up[f][q] - a1 + a0;                          // eq. (22)
            }
        }
    }
#pragma unroll
    for (int m = 0; m < 7; ++m) {
        const Prim pr = cons2prim_general<EOS>(k.d, ut[0][m], ut[1][m], ut[2][m], ut[3][m], ut[4][m]);
        vh[m] = ut[1][m] * pr.y;
        ph[m] = pr.p;
    }
    // 5. corrector transport of U^n at m = -2..2, 6.+7. antidiffusion, limiter, update of the centre cell
    double un[NF];
#pragma unroll
    for (int f = 0; f < NF; ++f) {
        double uh[5];
#pragma unroll
        for (int m = -2; m <= 2; ++m) {
            const int c = m + W, q = m + 3;
            double fm = 0.0, fp = 0.0;
            if (f == 0) { fm = ph[q - 1] * vh[q - 1]; fp = ph[q + 1] * vh[q + 1]; }
            if (f == 1) { fm = ph[q - 1]; fp = ph[q + 1]; }
            uh[m + 2] = cell_transport(w.u[f][c - 1], w.u[f][c], w.u[f][c + 1], lam * vh[q - 1], lam * vh[q], lam * vh[q + 1],
                                       lam, fm, fp);
        }
        const double a1 = cell_antiflux(uh[1], uh[2], uh[3], uh[4], w.u[f][W - 1], w.u[f][W], w.u[f][W + 1], w.u[f][W + 2], diff, k.ad2);
        const double a0 = cell_antiflux(uh[0], uh[1], uh[2], uh[3], w.u[f][W - 2], w.u[f][W - 1], w.u[f][W], w.u[f][W + 1], diff, k.ad2);
        un[f] = uh[2] - a1 + a0;                                            // eq. (22)
    }
    // 8. Pi written back (G8), primitives in the last sweep of a step
    Cnt cnt;
    cnt.zero();
    project(k.d, un, cnt);
#pragma unroll
    for (int f = 0; f < NF; ++f) ((double*)P.out[f])[i] = un[f];
    if (emit) {
        double pr[6];
        primitives<EOS>(k.d, un, pr, cnt);
#pragma unroll
        for (int q = 0; q < 6; ++q) ((double*)P.prim[q])[i] = pr[q];
    }
    flush_counts(cnt, P.counts);
}

}  // namespace shk
