/*
 * shasta_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct fp64 CPU implementation of the dimensionally
 * split (3+1)D relativistic SHASTA time step of arXiv:1206.0919,
 * written straight from the paper's equations, in the paper's order and notation.
 * It shares no code with the CUDA path (paper_1206_0919_b200/csrc) and must not:
 * only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may load it.  Build: gcc -O2 -ffp-contract=off -fopenmp -shared.
 * (-ffp-contract=off: no FMA contraction, so the identities the pins test hold as
 * stated.  OpenMP is used ONLY over independent pencils/cells: the result is
 * bitwise identical for any thread count; oracle_set_threads(1) = single thread.)
 *
 * What follows the paper (citations are PAPER.md line numbers):
 *   eqs. (9)-(11)   PAPER.md:58-62    conserved fields from primitives
 *   eq.  (15)       PAPER.md:83       geometric factors Q+-
 *   source term     PAPER.md:88       Delta(f) = -1/2 (f_{j+1} - f_{j-1}), f = p (M par.), p v (E)
 *   eqs. (16),(17)  PAPER.md:90-93    transport + diffusion
 *   eqs. (18)-(22)  PAPER.md:97-107   phoenical antidiffusion, flux limiter, update
 *   four phases     PAPER.md:74-79    transport / antidiffusion / relativistic correction / EOS
 *   half step       PAPER.md:161      "implemented based on a half-step method"
 *   fixed point     PAPER.md:109      velocity by fixed-point root finding
 *   axis table      PAPER.md:295-297  branch[] = {0,1,2,0,2,1,2,0,1,2,1,0,1,2,0,1,0,2}
 *   tabled EOS      PAPER.md:36, 109, 175  "easy implementation of a tabled equation of state": P(e,n) by bilinear
 *                   interpolation in a table; the paper gives no table and no interpolation rule,
 *                   the rule used is stated at eos_table_P below and in DESIGN.md 3 (reading T1)
 *
 * Where the paper is silent the readings G1-G19 of SURVEY.md 8(c.2), restated in
 * DESIGN.md section 3, are used; each is marked "reading Gn" below.
 *
 * PARITY PINS (tests/test_oracle_*.py, -m "not gpu"): P1-P15 of DESIGN.md section 4.  P14 (linear acoustic wave:
 * observed order >= 1.8 only if v and the sources are centred at n+1/2) pins steps 3-5 of oracle_sweep_pencil,
 * P15 (bitwise equality with a hand-extended pencil) pins ghost_index.
 * "parity unpinned" AGAINST THE PAPER'S OWN CODE for the CHOICES the paper leaves open: the predictor
 * without antidiffusion (reading G4; the R2 alternative is oracle_set_option key 4), the causality projection Pi
 * and its write-back (G6-G8) and ghost extension of the sweep input as THE boundary rule (G11): the paper
 * prints no value and no code for them; the arithmetic of each choice is pinned, the choice itself is not.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NF 5          /* E, Mx, My, Mz, R  (R is the paper's N, eq. (9)) */
#define G  4          /* ghost depth of one sweep: dependency radius of the default scheme (R1) */
#define G2 6          /* same for the R2 predictor (half step WITH antidiffusion, reading G4 alternative) */
#define PI_DELTA 1e-12            /* reading G7 */
#define VAC_E    0x1p-498         /* reading G7 (amended in round 2): a cell is vacuum when !(E >= 2^-498 ~ 1.2e-150), i.e. E <= 0,
                                     NaN, or so small that E^2 and |M|^2 are not representable in fp64 -- there |M| =
                                     sqrt(Mx^2+My^2+Mz^2) below is formed from underflowed squares and v = M/(E+P) is rounding
                                     noise in ANY fp64 evaluation.  Such cells arise at a front running into an exact E = 0
                                     exterior (the FCT front is so steep that they touch cells of visible size). */
#define FP_TOL   1e-15            /* reading G9 */
#define FP_MAXIT 200              /* reading G9 */

enum { BC_OUTFLOW = 0, BC_PERIODIC = 1 };

typedef struct eos_table {
    int ne, nn;
    double de, dn;
    const double *p;
} eos_table_t;

typedef struct oracle_shasta {
    int nx, ny, nz;
    double dx, lambda, gamma, mass;
    int bc;
    int predictor;                /* 0 = R1 (reading G4): predictor = eq. (17) alone; 1 = R2: predictor = eqs. (17)-(22) */
    double diff;                  /* Listing 1 'diff': factor on A^ph; 1 = paper default, 0 = "n/af" */
    int adkind;                   /* antidiffusion term: 0 = phoenical (eq. (19), default), 1 = explicit (PAPER.md:123 footnote) */
    long long step_index;
    int table[64];
    int ntable;
    double *U[NF];                /* conserved state, x fastest: ix + nx*(iy + ny*iz) */
    int have_state;
    unsigned long long counts[4]; /* Pi fired, vacuum cells, e<0 floored, p<0 floored */
    eos_table_t tab;              /* tabled EOS (reading T1); have_tab = 0: ideal gas */
    int have_tab;
} oracle_t;

static int g_threads = 1;
void oracle_set_threads(int n) { g_threads = n < 1 ? 1 : n; }
int oracle_get_threads(void) { return g_threads; }

/* ---------------------------------------------------------------- EOS ---- */
/* Tabled EOS (reading T1): pressure at the nodes (e_i, n_j) = (i de, j dn), i < ne, j < nn, stored e fastest:
   p[i + ne*j].  Between nodes bilinear, outside the table the bilinear form of the nearest cell continues
   (linear extrapolation); the result is floored at 0 like the ideal gas. */

double oracle_eos_table_P(const eos_table_t *t, double e, double n)
{
    double xe = e / t->de, xn = n / t->dn;
    int i = (int)floor(xe), j = (int)floor(xn);
    if (i < 0) i = 0;
    if (i > t->ne - 2) i = t->ne - 2;
    if (j < 0) j = 0;
    if (j > t->nn - 2) j = t->nn - 2;
    double te = xe - i, tn = xn - j;
    const double *q = t->p + i + (size_t)t->ne * j;
    double p0 = q[0] + te * (q[1] - q[0]);                      /* along e at n_j */
    double p1 = q[t->ne] + te * (q[t->ne + 1] - q[t->ne]);      /* along e at n_{j+1} */
    double P = p0 + tn * (p1 - p0);
    return P > 0.0 ? P : 0.0;
}

/* ideal gas, reading G10: P(e,n) = max((Gamma-1)(e - m n), 0); with a table: the table */
static double eos_P(double e, double n, double gamma, double mass, const eos_table_t *tab)
{
    if (tab) return oracle_eos_table_P(tab, e, n);
    double p = (gamma - 1.0) * (e - mass * n);
    return p > 0.0 ? p : 0.0;
}

/* --------------------------------------------- eqs. (9)-(11): prim -> cons */
void oracle_prim2cons_eos(double e, double n, double vx, double vy, double vz,
                          double gamma, double mass, const eos_table_t *tab, double out[NF])
{
    double p = eos_P(e, n, gamma, mass, tab);
    double v2 = (vx * vx + vy * vy) + vz * vz;
    double g2 = 1.0 / (1.0 - v2);             /* gamma_L^2 */
    double w = (e + p) * g2;                  /* (eps + p) gamma^2 */
    out[0] = w - p;                           /* eq. (11): (eps + p v^2) gamma^2 = w - p */
    out[1] = w * vx;                          /* eq. (10) */
    out[2] = w * vy;
    out[3] = w * vz;
    out[4] = n * sqrt(g2);                    /* eq. (9) */
}
void oracle_prim2cons(double e, double n, double vx, double vy, double vz,
                      double gamma, double mass, double out[NF])
{
    oracle_prim2cons_eos(e, n, vx, vy, vz, gamma, mass, NULL, out);
}

/* ------------------- phases 3+4: relativistic correction + EOS (cons2prim) */
/* Pi, readings G6-G8: enforce |M| <= (1-delta) E; vacuum if !(E >= VAC_E).
   Returns 1 if the projection fired, 2 if vacuum, 0 otherwise.  E, R untouched. */
int oracle_project(double E, double M[3])
{
    if (!(E >= VAC_E)) { M[0] = M[1] = M[2] = 0.0; return 2; }
    double Mabs = sqrt((M[0] * M[0] + M[1] * M[1]) + M[2] * M[2]);
    double lim = (1.0 - PI_DELTA) * E;
    if (Mabs > lim) {
        double s = lim / Mabs;
        M[0] *= s; M[1] *= s; M[2] *= s;
        return 1;
    }
    return 0;
}

/* out = {e, p, n, vx, vy, vz, |v|}; returns the number of fixed-point iterations.
   flags (may be NULL): flags[0] += e floored, flags[1] += p floored. */
int oracle_cons2prim_eos(double E, double Mx, double My, double Mz, double R,
                         double gamma, double mass, const eos_table_t *tab, double out[7], int flags[2])
{
    double M = sqrt((Mx * Mx + My * My) + Mz * Mz);
    if (!(E >= VAC_E)) {                      /* vacuum, reading G7 */
        for (int i = 0; i < 7; ++i) out[i] = 0.0;
        return 0;
    }
    double lim = (1.0 - PI_DELTA) * E;
    double Mc = M < lim ? M : lim;            /* same rule as Pi */
    double v = 0.0;
    int it = 0;
    for (it = 0; it < FP_MAXIT; ++it) {       /* PAPER.md:109 fixed point, reading G9 */
        double P = eos_P(E - Mc * v, R * sqrt(1.0 - v * v), gamma, mass, tab);
        double vnew = Mc / (E + P);
        double d = fabs(vnew - v);
        v = vnew;
        if (d <= FP_TOL) { ++it; break; }
    }
    double e = E - Mc * v;
    if (e < 0.0) { e = 0.0; if (flags) flags[0]++; }
    double n = R * sqrt(1.0 - v * v);
    double praw = (gamma - 1.0) * (e - mass * n);
    if (!tab && praw < 0.0 && flags) flags[1]++;
    double p = eos_P(e, n, gamma, mass, tab);
    out[0] = e; out[1] = p; out[2] = n;
    if (M > 0.0) { out[3] = v * Mx / M; out[4] = v * My / M; out[5] = v * Mz / M; }
    else         { out[3] = out[4] = out[5] = 0.0; }
    out[6] = v;
    return it;
}
int oracle_cons2prim(double E, double Mx, double My, double Mz, double R,
                     double gamma, double mass, double out[7], int flags[2])
{
    return oracle_cons2prim_eos(E, Mx, My, Mz, R, gamma, mass, NULL, out, flags);
}

/* ------------------------------------------------------------ eq. (15) --- */
/* reading G1: upper signs -> Q+, lower signs -> Q-.  eps = lambda * v. */
double oracle_qplus(double eps_j, double eps_jp1)
{
    return (0.5 - eps_j) / (1.0 + (eps_jp1 - eps_j));
}
double oracle_qminus(double eps_j, double eps_jm1)
{
    return (0.5 + eps_j) / (1.0 - (eps_jm1 - eps_j));
}

/* ------------------------------------------------- eqs. (16),(17) -------- */
/* Transport + diffusion of ONE field on an extended pencil.
   Arrays are indexed 0..n-1; Uhat[j] is written for j = lo..hi-1 and needs
   U, eps, f at j-1..j+1.  f may be NULL (source-free field).  lam multiplies
   Delta(f) = -1/2 (f[j+1] - f[j-1]). */
void oracle_transport(int n, const double *U, const double *eps, const double *f,
                      double lam, double *Uhat, int lo, int hi)
{
    (void)n;
    for (int j = lo; j < hi; ++j) {
        double Qp = oracle_qplus(eps[j], eps[j + 1]);
        double Qm = oracle_qminus(eps[j], eps[j - 1]);
        double Dj = U[j + 1] - U[j];                         /* eq. (16) */
        double Djm = U[j] - U[j - 1];
        double uh = 0.5 * Qp * Qp * Dj - 0.5 * Qm * Qm * Djm + (Qp + Qm) * U[j];
        if (f) uh += lam * (-0.5 * (f[j + 1] - f[j - 1]));   /* + lambda Delta(f) */
        Uhat[j] = uh;                                        /* eq. (17) */
    }
}

/* ------------------------------------------------- eqs. (18)-(22) -------- */
static double sgn(double x) { return (x > 0.0) - (x < 0.0); }
static double min3(double a, double b, double c)
{
    double m = a < b ? a : b;
    return m < c ? m : c;
}
/* Phoenical antidiffusion with flux limiter on ONE field of an extended pencil.
   Unew[j] is written for j = lo..hi-1; needs Uhat at j-2..j+2 and U at j-3..j+3
   (Fig. 3).  diff multiplies A^ph (Listing 1 'diff', reading G13). */
/* kind 0 = the paper's phoenical term, eq. (19); kind 1 = the EXPLICIT antidiffusion of the original SHASTA (Boris & Book:
   A^ex_j = 1/8 Dhat_j), the best known of the "different anti-diffusion terms [that] are possible" of the paper's footnote 1
   (the paper names none of them: SURVEY.md 8(f) f2).  At rest it leaves the residual damping -1/64 delta^4 U
   that the phoenical term removes (pin: tests/test_oracle_variants.py). */
void oracle_antidiffuse_kind(int n, const double *U, const double *Uhat, double diff, int kind,
                             double *Unew, int lo, int hi)
{
    (void)n;
    for (int j = lo; j < hi; ++j) {
        double A[2];                                        /* A_{j-1}, A_j */
        for (int k = 0; k < 2; ++k) {
            int i = j - 1 + k;                              /* interface index */
            double Dh = Uhat[i + 1] - Uhat[i];              /* eq. (18) */
            double Dhp = Uhat[i + 2] - Uhat[i + 1];
            double Dhm = Uhat[i] - Uhat[i - 1];
            double Di = U[i + 1] - U[i];                    /* eq. (16) */
            double Dip = U[i + 2] - U[i + 1];
            double Dim = U[i] - U[i - 1];
            /* eq. (19), evaluation order of reading G14 */
            double Aph = kind == 0 ? diff * (0.125 * (Dh - 0.125 * ((Dip + Dim) - 2.0 * Di)))
                                   : diff * (0.125 * Dh);
            double s = sgn(Aph);                            /* eq. (20) */
            double m = min3(s * Dhp, fabs(Aph), s * Dhm);
            A[k] = s * (m > 0.0 ? m : 0.0);                 /* eq. (21) */
        }
        Unew[j] = Uhat[j] - A[1] + A[0];                    /* eq. (22) */
    }
}

void oracle_antidiffuse(int n, const double *U, const double *Uhat, double diff,
                        double *Unew, int lo, int hi)
{
    oracle_antidiffuse_kind(n, U, Uhat, diff, 0, Unew, lo, hi);
}

/* ------------------------------------------------------------ boundary --- */
/* reading G11: ghost-extend the INPUT of a sweep by G cells per side. */
static int ghost_index(int j, int N, int bc)
{
    if (bc == BC_PERIODIC) { int m = j % N; return m < 0 ? m + N : m; }
    return j < 0 ? 0 : (j >= N ? N - 1 : j);
}

/* ---------------------------------------------------------- one pencil --- */
/* One full sweep (phases 1-4) of one pencil along axis a (0=x,1=y,2=z).
   U[f][0..N-1] is updated in place.  counts (may be NULL): [0] Pi fired, [1] vacuum.
   Scheme variants the paper describes as selectable:
     diff       factor on the antidiffusive flux A^ph ("fine controlled application of numerical viscosity",
                PAPER.md:159; `const float diff = 1.0f`); diff = 0 is the "n/af" mode of Fig. 7
                (no anti-flux);
     predictor  0 = R1 (reading G4, the default): half step = eq. (17) alone with lambda/2;
                1 = R2: half step = the complete kernel with lambda/2, i.e. eq. (17) AND eqs. (18)-(22), which is what
                Listing 2 suggests (the ordinary prop kernels run after half_cfl).  Radius 6. */
void oracle_sweep_pencil_full(int N, double *U[NF], int a, double lambda, double gamma,
                              double mass, int bc, unsigned long long counts[2], double diff, int predictor,
                              const eos_table_t *tab, int adkind)
{
    const int g = predictor ? G2 : G;         /* ghost depth */
    const int NE = N + 2 * g;                 /* extended length, j = -g .. N+g-1 at offset +g */
    double *buf = (double *)malloc(sizeof(double) * (size_t)NE * (5 * NF + 8));
    double *Ue[NF], *Ut[NF], *Uh[NF], *Un[NF], *Up[NF];
    double *p = buf;
    for (int f = 0; f < NF; ++f) { Ue[f] = p; p += NE; }
    for (int f = 0; f < NF; ++f) { Ut[f] = p; p += NE; }
    for (int f = 0; f < NF; ++f) { Uh[f] = p; p += NE; }
    for (int f = 0; f < NF; ++f) { Un[f] = p; p += NE; }
    for (int f = 0; f < NF; ++f) { Up[f] = p; p += NE; }
    double *v = p;  p += NE;  double *pr = p; p += NE;  double *pv = p; p += NE;
    double *eps = p; p += NE; double *vh = p; p += NE;  double *ph = p; p += NE;
    double *pvh = p; p += NE; double *epsh = p; p += NE;
    /* index of cell j in the extended arrays is j + g; lo/hi below are extended indices.  The half-step state is
       needed at j = -3 .. N+2, the corrector transport at j = -2 .. N+1 */
    const int h_lo = g - 3, h_hi = g + N + 3;

    /* 1. extend j = -g .. N+g-1 */
    for (int i = 0; i < NE; ++i) {
        int src = ghost_index(i - g, N, bc);
        for (int f = 0; f < NF; ++f) Ue[f][i] = U[f][src];
    }
    /* 2. time-n primitives on the whole extended pencil */
    for (int i = 0; i < NE; ++i) {
        double o[7];
        oracle_cons2prim_eos(Ue[0][i], Ue[1][i], Ue[2][i], Ue[3][i], Ue[4][i], gamma, mass, tab, o, NULL);
        v[i] = o[3 + a]; pr[i] = o[1]; pv[i] = o[1] * o[3 + a];
    }
    /* 3. predictor (readings G4, G5): eq. (17) with lambda/2, time-n v and p */
    const double h = 0.5 * lambda;
    for (int i = 0; i < NE; ++i) eps[i] = h * v[i];
    for (int f = 0; f < NF; ++f) {
        const double *src = (f == 0) ? pv : (f == 1 + a ? pr : NULL);
        if (!predictor) {
            /* R1: no antidiffusion; j = -3 .. N+2 */
            oracle_transport(NE, Ue[f], eps, src, h, Ut[f], h_lo, h_hi);
        } else {
            /* R2: transport j = -5 .. N+4, then eqs. (18)-(22) j = -3 .. N+2 */
            oracle_transport(NE, Ue[f], eps, src, h, Up[f], h_lo - 2, h_hi + 2);
            oracle_antidiffuse_kind(NE, Ue[f], Up[f], diff, adkind, Ut[f], h_lo, h_hi);
        }
    }
    /* 4. half-step primitives, j = -3 .. N+2 */
    for (int i = h_lo; i < h_hi; ++i) {
        double o[7];
        oracle_cons2prim_eos(Ut[0][i], Ut[1][i], Ut[2][i], Ut[3][i], Ut[4][i], gamma, mass, tab, o, NULL);
        vh[i] = o[3 + a]; ph[i] = o[1]; pvh[i] = o[1] * o[3 + a];
    }
    /* 5. corrector transport: eq. (17) with lambda, half-step v and p, transports U^n;
          j = -2 .. N+1 */
    for (int i = h_lo; i < h_hi; ++i) epsh[i] = lambda * vh[i];
    for (int f = 0; f < NF; ++f) {
        const double *src = (f == 0) ? pvh : (f == 1 + a ? ph : NULL);
        oracle_transport(NE, Ue[f], epsh, src, lambda, Uh[f], h_lo + 1, h_hi - 1);
    }
    /* 6.+7. antidiffusion, limiter, update: j = 0 .. N-1 */
    for (int f = 0; f < NF; ++f)
        oracle_antidiffuse_kind(NE, Ue[f], Uh[f], diff, adkind, Un[f], g, g + N);
    /* 8. relativistic correction Pi written back (reading G8) */
    for (int j = 0; j < N; ++j) {
        double M[3] = { Un[1][g + j], Un[2][g + j], Un[3][g + j] };
        int r = oracle_project(Un[0][g + j], M);
        if (counts) { if (r == 1) counts[0]++; else if (r == 2) counts[1]++; }
        U[0][j] = Un[0][g + j];
        U[1][j] = M[0]; U[2][j] = M[1]; U[3][j] = M[2];
        U[4][j] = Un[4][g + j];
    }
    free(buf);
}

void oracle_sweep_pencil_eos(int N, double *U[NF], int a, double lambda, double gamma,
                             double mass, int bc, unsigned long long counts[2], double diff, int predictor,
                             const eos_table_t *tab)
{
    oracle_sweep_pencil_full(N, U, a, lambda, gamma, mass, bc, counts, diff, predictor, tab, 0);
}

void oracle_sweep_pencil_ex(int N, double *U[NF], int a, double lambda, double gamma,
                            double mass, int bc, unsigned long long counts[2], double diff, int predictor)
{
    oracle_sweep_pencil_eos(N, U, a, lambda, gamma, mass, bc, counts, diff, predictor, NULL);
}

/* the default scheme: diff = 1, predictor R1 */
void oracle_sweep_pencil(int N, double *U[NF], int a, double lambda, double gamma,
                         double mass, int bc, unsigned long long counts[2])
{
    oracle_sweep_pencil_ex(N, U, a, lambda, gamma, mass, bc, counts, 1.0, 0);
}

/* P5 pin helper: advect ONE source-free field with a PRESCRIBED velocity (cons2prim
   bypassed): v_half = v, one step = corrector transport + antidiffusion (eqs. 15-22). */
void oracle_advect_pencil(int N, double *U, const double *vel, double lambda, int bc,
                          int nsteps, double *Uhat_out)
{
    const int NE = N + 2 * G;
    double *Ue = (double *)malloc(sizeof(double) * (size_t)NE * 4);
    double *eps = Ue + NE, *Uh = eps + NE, *Un = Uh + NE;
    for (int s = 0; s < nsteps; ++s) {
        for (int i = 0; i < NE; ++i) {
            int src = ghost_index(i - G, N, bc);
            Ue[i] = U[src]; eps[i] = lambda * vel[src];
        }
        oracle_transport(NE, Ue, eps, NULL, lambda, Uh, 2, NE - 2);
        oracle_antidiffuse(NE, Ue, Uh, 1.0, Un, G, G + N);
        for (int j = 0; j < N; ++j) U[j] = Un[G + j];
        if (Uhat_out) for (int j = 0; j < N; ++j) Uhat_out[j] = Uh[G + j];
    }
    free(Ue);
}

/* ---------------------------------------------------------- the grid ----- */
static const int kBranch[18] = { 0,1,2, 0,2,1, 2,0,1, 2,1,0, 1,2,0, 1,0,2 };

oracle_t *oracle_create(int nx, int ny, int nz, double dx, double lambda, double eos_gamma)
{
    if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0.0) || !(lambda > 0.0) || lambda > 0.5 ||
        !(eos_gamma > 1.0)) return NULL;
    oracle_t *o = (oracle_t *)calloc(1, sizeof(oracle_t));
    o->nx = nx; o->ny = ny; o->nz = nz; o->dx = dx; o->lambda = lambda; o->gamma = eos_gamma;
    o->mass = 0.0; o->bc = BC_OUTFLOW; o->step_index = 0; o->predictor = 0; o->diff = 1.0;
    memcpy(o->table, kBranch, sizeof(kBranch)); o->ntable = 18;
    size_t n = (size_t)nx * ny * nz;
    for (int f = 0; f < NF; ++f) o->U[f] = (double *)calloc(n, sizeof(double));
    return o;
}
void oracle_destroy(oracle_t *o)
{
    if (!o) return;
    for (int f = 0; f < NF; ++f) free(o->U[f]);
    free((void *)o->tab.p);
    free(o);
}
/* Tabled EOS for this grid (copied): p[i + ne*j] at (i e_max/(ne-1), j n_max/(nn-1)); p == NULL: back to the ideal gas */
int oracle_set_eos_table(oracle_t *o, const double *p, int ne, int nn, double e_max, double n_max)
{
    if (!o) return -1;
    free((void *)o->tab.p); o->tab.p = NULL; o->have_tab = 0;
    if (!p) return 0;
    if (ne < 2 || nn < 2 || !(e_max > 0.0) || !(n_max > 0.0)) return -1;
    double *c = (double *)malloc(sizeof(double) * (size_t)ne * nn);
    memcpy(c, p, sizeof(double) * (size_t)ne * nn);
    o->tab.ne = ne; o->tab.nn = nn; o->tab.de = e_max / (ne - 1); o->tab.dn = n_max / (nn - 1); o->tab.p = c;
    o->have_tab = 1;
    return 0;
}
/* keys: 0 boundary (0 outflow, 1 periodic), 1 EOS mass m, 3 step index, 4 predictor (0 = R1, 1 = R2), 5 diff >= 0,
   6 antidiffusion term (0 = phoenical, 1 = explicit) */
int oracle_set_option(oracle_t *o, int key, double value)
{
    if (!o) return -1;
    switch (key) {
    case 0: if (value != 0.0 && value != 1.0) return -1; o->bc = (int)value; return 0;
    case 1: if (value < 0.0) return -1; o->mass = value; return 0;
    case 3: if (value < 0.0) return -1; o->step_index = (long long)value; return 0;
    case 4: if (value != 0.0 && value != 1.0) return -1; o->predictor = (int)value; return 0;
    case 5: if (!(value >= 0.0)) return -1; o->diff = value; return 0;
    case 6: if (value != 0.0 && value != 1.0) return -1; o->adkind = (int)value; return 0;
    default: return -1;
    }
}
int oracle_set_sweep_table(oracle_t *o, const int *axes, int n)
{
    if (!o || !axes || n < 3 || n > 63 || n % 3) return -1;
    for (int i = 0; i < n; ++i) if (axes[i] < 0 || axes[i] > 2) return -1;
    memcpy(o->table, axes, sizeof(int) * (size_t)n); o->ntable = n;
    return 0;
}
int oracle_set_state(oracle_t *o, const double *e, const double *n, const double *vx,
                     const double *vy, const double *vz)
{
    if (!o || !e || !n || !vx || !vy || !vz) return -1;
    long long nc = (long long)o->nx * o->ny * o->nz;
#pragma omp parallel for num_threads(g_threads) schedule(static)
    for (long long i = 0; i < nc; ++i) {
        double c[NF];
        oracle_prim2cons_eos(e[i], n[i], vx[i], vy[i], vz[i], o->gamma, o->mass, o->have_tab ? &o->tab : NULL, c);
        for (int f = 0; f < NF; ++f) o->U[f][i] = c[f];
    }
    o->have_state = 1;
    return 0;
}
int oracle_set_conserved(oracle_t *o, const double *E, const double *Mx, const double *My,
                         const double *Mz, const double *R)
{
    if (!o || !E || !Mx || !My || !Mz || !R) return -1;
    size_t nb = sizeof(double) * (size_t)o->nx * o->ny * o->nz;
    const double *src[NF] = { E, Mx, My, Mz, R };
    for (int f = 0; f < NF; ++f) memcpy(o->U[f], src[f], nb);
    o->have_state = 1;
    return 0;
}
int oracle_get_conserved(oracle_t *o, double *E, double *Mx, double *My, double *Mz, double *R)
{
    if (!o) return -1;
    if (!o->have_state) return -4;
    size_t nb = sizeof(double) * (size_t)o->nx * o->ny * o->nz;
    double *dst[NF] = { E, Mx, My, Mz, R };
    for (int f = 0; f < NF; ++f) if (dst[f]) memcpy(dst[f], o->U[f], nb);
    return 0;
}

/* one sweep of the whole grid along axis a: every pencil independently */
static void sweep_grid(oracle_t *o, int a)
{
    const int n[3] = { o->nx, o->ny, o->nz };
    const long long stride[3] = { 1, o->nx, (long long)o->nx * o->ny };
    const int N = n[a];
    const int b = (a + 1) % 3, c = (a + 2) % 3;      /* the two other axes */
    const long long npencil = (long long)n[b] * n[c];
    unsigned long long c0 = 0, c1 = 0;
#pragma omp parallel for num_threads(g_threads) schedule(static) reduction(+:c0,c1)
    for (long long q = 0; q < npencil; ++q) {
        long long ib = q % n[b], ic = q / n[b];
        long long base = ib * stride[b] + ic * stride[c];
        double *pen = (double *)malloc(sizeof(double) * (size_t)N * NF);
        double *P[NF];
        for (int f = 0; f < NF; ++f) {
            P[f] = pen + (size_t)f * N;
            for (int j = 0; j < N; ++j) P[f][j] = o->U[f][base + j * stride[a]];
        }
        unsigned long long cnt[2] = { 0, 0 };
        oracle_sweep_pencil_full(N, P, a, o->lambda, o->gamma, o->mass, o->bc, cnt, o->diff, o->predictor,
                                 o->have_tab ? &o->tab : NULL, o->adkind);
        for (int f = 0; f < NF; ++f)
            for (int j = 0; j < N; ++j) o->U[f][base + j * stride[a]] = P[f][j];
        c0 += cnt[0]; c1 += cnt[1];
        free(pen);
    }
    o->counts[0] += c0; o->counts[1] += c1;
}

/* one time step dt = lambda dx = three sweeps (reading G3), order from the table */
int oracle_step(oracle_t *o, int nsteps)
{
    if (!o || nsteps < 0) return -1;
    if (!o->have_state) return -4;
    const int n[3] = { o->nx, o->ny, o->nz };
    for (int s = 0; s < nsteps; ++s) {
        for (int k = 0; k < 3; ++k) {
            int a = o->table[(3 * o->step_index + k) % o->ntable];
            if (n[a] == 1) continue;                 /* reading G15 */
            sweep_grid(o, a);
        }
        o->step_index++;
    }
    return 0;
}

int oracle_get_primitives(oracle_t *o, double *e, double *p, double *n, double *vx,
                          double *vy, double *vz)
{
    if (!o) return -1;
    if (!o->have_state) return -4;
    long long nc = (long long)o->nx * o->ny * o->nz;
    unsigned long long f0 = 0, f1 = 0;
#pragma omp parallel for num_threads(g_threads) schedule(static) reduction(+:f0,f1)
    for (long long i = 0; i < nc; ++i) {
        double out[7]; int fl[2] = { 0, 0 };
        oracle_cons2prim_eos(o->U[0][i], o->U[1][i], o->U[2][i], o->U[3][i], o->U[4][i],
                             o->gamma, o->mass, o->have_tab ? &o->tab : NULL, out, fl);
        if (e) e[i] = out[0];
        if (p) p[i] = out[1];
        if (n) n[i] = out[2];
        if (vx) vx[i] = out[3];
        if (vy) vy[i] = out[4];
        if (vz) vz[i] = out[5];
        f0 += (unsigned)fl[0]; f1 += (unsigned)fl[1];
    }
    o->counts[2] += f0; o->counts[3] += f1;
    return 0;
}

/* dx^3 * sum over cells, Neumaier-compensated (eqs. (12)-(14): the totals are conserved) */
int oracle_conserved_totals(oracle_t *o, double totals[NF])
{
    if (!o || !totals) return -1;
    if (!o->have_state) return -4;
    long long nc = (long long)o->nx * o->ny * o->nz;
    double dv = o->dx * o->dx * o->dx;
    for (int f = 0; f < NF; ++f) {
        double s = 0.0, c = 0.0;
        for (long long i = 0; i < nc; ++i) {
            double x = o->U[f][i], t = s + x;
            if (fabs(s) >= fabs(x)) c += (s - t) + x; else c += (x - t) + s;
            s = t;
        }
        totals[f] = dv * (s + c);
    }
    return 0;
}
int oracle_diagnostics(oracle_t *o, unsigned long long counts[4])
{
    if (!o || !counts) return -1;
    for (int i = 0; i < 4; ++i) counts[i] = o->counts[i];
    return 0;
}
long long oracle_step_index(oracle_t *o) { return o ? o->step_index : -1; }
