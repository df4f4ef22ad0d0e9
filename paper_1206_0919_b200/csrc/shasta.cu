// shasta.cu -- host side of libshasta.so: the C ABI of include/shasta.h.
// Orchestration only (Listing 2): axis table, ping-pong buffers, launches.
// Every arithmetic step of the path runs in the kernels of shasta_kernels.cuh.
#include "shasta.h"
#include "shasta_kernels.cuh"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>

using namespace shk;

namespace {

thread_local char g_create_err[256] = "";

const int kBranch[18] = {0, 1, 2, 0, 2, 1, 2, 0, 1, 2, 1, 0, 1, 2, 0, 1, 0, 2};

constexpr int RED_BLOCKS = 592; // 4 per SM
constexpr int RED_THREADS = 256;

}  // namespace

struct shasta {
    int nx, ny, nz;
    long long ncell;        // cells of ALL events of the batch: nbatch * ncell1
    long long ncell1;       // cells of one event, nx * ny * nz
    int nbatch;             // independent events stacked along z (SHASTA_BATCH); 1 by default
    double dx, lambda, gamma, mass;
    double* d_tab;          // tabled EOS (row f1): device copy of P at the nodes, e fastest; NULL = analytic EOS
    int tab_ne, tab_nn;
    double tab_de, tab_dn;
    double diff;            // factor on the antidiffusive flux; 1 by default
    int explicit_ad;        // SHASTA_ANTIDIFFUSION: 0 = phoenical eq. (19) (default), 1 = explicit (PAPER.md:123 footnote 1)
    int cell_path;          // 1 = run the per-cell kernels also for the default scheme (A/B datapoint, tests)
    int predictor;          // 0 = R1 (eq. (17) alone), 1 = R2 (complete kernel at lambda/2): per-cell kernels
    int periodic;
    int az_lo, az_hi;       // shasta_set_active_planes: x and y sweeps update the planes [az_lo, az_hi) only (default all)
    int periodic_z;         // SHASTA_BOUNDARY_Z: -1 = as `periodic`; 0 | 1 = rule of the z sweeps only (z-slab ranks: 0)
    int precision;          // 64 | 32
    int seg_override;
    int no_tma;             // test hook: 1 = x sweep through cp.async even where TMA is possible
    int graph_mode;         // SHASTA_GRAPH: 0 never, 1 always, 2 auto (grids whose sweeps are launch/latency bound)
    struct GraphEntry { int phase, cur, chunk; cudaGraphExec_t exec; long long launches; } graphs[8];
    int ngraphs;
    long long graph_launches;
    cudaStream_t cap_stream;
    int prims_raw;          // test hook: get_primitives copies the primitive fields as stored, without refreshing them
    int no_defer;           // test hook / A-B: 1 = x-last steps write their primitives at once (separate element-wise pass)
    long long step;
    int table[64];
    int ntable;
    void* U[2][NF];         // conserved, ping-pong, natural order E,Mx,My,Mz,R
    CUtensorMap tmap[2][NF]; // TMA maps of U (x sweep), valid when have_tmap
    bool have_tmap;
    CUtensorMap* d_xmaps;   // device copy of tmap: [buffer][field]
    CUtensorMap* d_yzmaps;  // device: [buffer][kind: y4 {32,4,1}, z4 {32,1,4}, c1 {32,1,1}][field], 3-D maps over (x,y,z)
    bool have_yzmap;
    void* prim[6];          // e,p,n,vx,vy,vz
    double* stage;          // fp64 staging (5 fields) for host<->device and fp32 conversion
    int cur;
    bool allocated, have_state, prims_valid;
    unsigned long long* d_counts;
    double* d_partial;      // RED_BLOCKS*NF*2
    double* h_partial;      // pinned
    long long launches;
    int sm_count;
    int device;             // device that was current at create
    char err[256];
};

namespace {

int fail(shasta_t* h, int code, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(h ? h->err : g_create_err, 256, fmt, ap);
    va_end(ap);
    return code;
}

#define CK(call)                                                                              \
    do {                                                                                      \
        cudaError_t e_ = (call);                                                              \
        if (e_ != cudaSuccess)                                                                \
            return fail(h, e_ == cudaErrorMemoryAllocation ? SHASTA_ENOMEM : SHASTA_ECUDA,    \
                        "%s: %s", #call, cudaGetErrorString(e_));                             \
    } while (0)

size_t esize(const shasta_t* h) { return h->precision == 64 ? 8 : 4; }
int axis_periodic(const shasta_t* h, int axis) { return (axis == 2 && h->periodic_z >= 0) ? h->periodic_z : h->periodic; }

int make_tensor_maps(shasta_t* h);
int make_yz_maps(shasta_t* h);

void free_fields(shasta_t* h)
{
    for (int b = 0; b < 2; ++b)
        for (int f = 0; f < NF; ++f) { cudaFree(h->U[b][f]); h->U[b][f] = nullptr; }
    for (int q = 0; q < 6; ++q) { cudaFree(h->prim[q]); h->prim[q] = nullptr; }
    cudaFree(h->d_counts); h->d_counts = nullptr;
    cudaFree(h->d_partial); h->d_partial = nullptr;
    if (h->h_partial) { cudaFreeHost(h->h_partial); h->h_partial = nullptr; }
}

int alloc_fields(shasta_t* h)
{
    const size_t nb = (size_t)h->ncell * esize(h);
    for (int b = 0; b < 2; ++b)
        for (int f = 0; f < NF; ++f) CK(cudaMalloc(&h->U[b][f], nb));
    for (int q = 0; q < 6; ++q) CK(cudaMalloc(&h->prim[q], nb));
    CK(cudaMalloc(&h->d_counts, 4 * sizeof(unsigned long long)));
    CK(cudaMemset(h->d_counts, 0, 4 * sizeof(unsigned long long)));
    CK(cudaMalloc(&h->d_partial, sizeof(double) * RED_BLOCKS * NF * 2));
    CK(cudaMallocHost(&h->h_partial, sizeof(double) * RED_BLOCKS * NF * 2));
    return 0;
}

// the handle belongs to the device that was current at shasta_create
int check_device(shasta_t* h)
{
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (dev != h->device)
        return fail(h, SHASTA_ESTATE, "the handle was created on device %d but device %d is current", h->device, dev);
    return 0;
}

int ensure_alloc(shasta_t* h)
{
    int rc = check_device(h);
    if (rc) return rc;
    if (h->allocated) return 0;
    rc = alloc_fields(h);
    if (rc) { free_fields(h); cudaGetLastError(); return rc; }      // nothing half-allocated is kept
    h->allocated = true;
    make_tensor_maps(h);
    return make_yz_maps(h);
}

// TMA tensor maps of the conserved fields for the x sweep: 2-D {nx, ny*nz*batch}, box {4 cells, 32 rows}; fp64 with the
// 32 B swizzle, fp32 dense (the shared-memory tile layouts of sweep_x2_kernel).  Needs 16 B row strides (fp64: even nx,
// fp32: nx % 4 == 0); otherwise the kernel's cp.async path is used.  The driver entry point is resolved at run time (libshasta.so does not link libcuda).
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int make_tensor_maps(shasta_t* h)
{
    h->have_tmap = false;
    const size_t es = esize(h);
    if (((size_t)h->nx * es) % 16 != 0 || h->nx < 8) return 0;
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
        qres != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return 0;                                   // no TMA: the cp.async path still works
    }
    const cuuint64_t dims[2] = {(cuuint64_t)h->nx, (cuuint64_t)h->ny * (cuuint64_t)h->nz * (cuuint64_t)h->nbatch};
    const cuuint64_t strides[1] = {(cuuint64_t)h->nx * es};
    // 32 B rows with the 32 B swizzle either way: four fp64 cells (one group of the march) or eight fp32 cells (two groups)
    const cuuint32_t box[2] = {(cuuint32_t)(es == 8 ? XV_CH : 2 * XV_CH), 32u};
    const cuuint32_t estr[2] = {1u, 1u};
    const CUtensorMapDataType dt = es == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    const CUtensorMapSwizzle swz = CU_TENSOR_MAP_SWIZZLE_32B;
    for (int b = 0; b < 2; ++b)
        for (int f = 0; f < NF; ++f) {
            CUresult r = ((EncodeTiledFn)fn)(&h->tmap[b][f], dt, 2, h->U[b][f], dims, strides,
                                             box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, swz,
                                             CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (r != CUDA_SUCCESS) return 0;
        }
    if (!h->d_xmaps) CK(cudaMalloc(&h->d_xmaps, sizeof(h->tmap)));
    CK(cudaMemcpy(h->d_xmaps, h->tmap, sizeof(h->tmap), cudaMemcpyHostToDevice));
    h->have_tmap = true;
    return 0;
}

// y/z sweeps (sweep_yz_kernel): 3-D maps {nx, ny, nz}; a warp pair's 4-cell group of 32 pencils is one box {32, 4, 1}
// (y) or {32, 1, 4} (z) per field, ghost groups are four {32, 1, 1} boxes.  Needs 16 B global strides (fp64: even nx,
// fp32: nx % 4 == 0); otherwise the kernel's cp.async fill is used.
int make_yz_maps(shasta_t* h)
{
    h->have_yzmap = false;
    const size_t es = esize(h);
    if (((size_t)h->nx * es) % 16 != 0 || h->nx < 32) return 0;
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
        qres != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return 0;
    }
    const CUtensorMapDataType dt = es == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    const cuuint64_t dims[3] = {(cuuint64_t)h->nx, (cuuint64_t)h->ny, (cuuint64_t)h->nz * (cuuint64_t)h->nbatch};
    const cuuint64_t strides[2] = {(cuuint64_t)h->nx * es, (cuuint64_t)h->nx * (cuuint64_t)h->ny * es};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    const cuuint32_t boxes[3][3] = {{32u, (cuuint32_t)YZ_CH, 1u}, {32u, 1u, (cuuint32_t)YZ_CH}, {32u, 1u, 1u}};
    static CUtensorMap host[2][3][NF];
    memset(host, 0, sizeof(host));
    for (int b = 0; b < 2; ++b)
        for (int m = 0; m < 3; ++m) {
            if (m == 0 && h->ny < YZ_CH) continue;      // that axis falls back to cp.async (see launch)
            if (m == 1 && h->nz < YZ_CH) continue;
            for (int f = 0; f < NF; ++f) {
                CUresult r = ((EncodeTiledFn)fn)(&host[b][m][f], dt, 3, h->U[b][f], dims, strides, boxes[m], estr,
                                                 CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                                 CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
                if (r != CUDA_SUCCESS) return 0;
            }
        }
    if (!h->d_yzmaps) CK(cudaMalloc(&h->d_yzmaps, sizeof(host)));
    CK(cudaMemcpy(h->d_yzmaps, host, sizeof(host), cudaMemcpyHostToDevice));
    h->have_yzmap = true;
    return 0;
}

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) once per kernel and device, not once per launch
int opt_in_smem(shasta_t* h, const void* kern, size_t smem)
{
    struct Key { const void* k; int dev; };
    static Key done[256];
    static int ndone = 0;
    int dev = 0;
    CK(cudaGetDevice(&dev));
    for (int i = 0; i < ndone; ++i)
        if (done[i].k == kern && done[i].dev == dev) return 0;
    CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (ndone < 256) { done[ndone].k = kern; done[ndone].dev = dev; ++ndone; }
    return 0;
}

int ensure_stage(shasta_t* h)
{
    if (!h->stage) CK(cudaMalloc(&h->stage, sizeof(double) * (size_t)h->ncell * 6));
    return 0;
}

// The EOS_GAMMA kernels (closed-form fast cons2prim, shasta_kernels.cuh c2p_fast_y) need m = 0 and Gamma <= 5/3
// (two frozen-slope Newton steps suffice while (Gamma-1)/(2-Gamma) <= 2); everything else runs the EOS_MASS kernels.
bool use_general_eos(const shasta_t* h) { return h->d_tab || h->mass != 0.0 || h->gamma > 5.0 / 3.0 + 1e-12; }
int eos_mode(const shasta_t* h) { return h->d_tab ? EOS_TABLE : (use_general_eos(h) ? EOS_MASS : EOS_GAMMA); }

template <typename T>
Consts<T> make_consts(const shasta_t* h)
{
    Consts<T> k;
    k.lam = (T)h->lambda;
    k.hlam = (T)(0.5 * h->lambda);
    k.qlam = (T)(0.25 * h->lambda);
    k.aq = (T)(0.125 * h->diff);
    k.ad2 = h->explicit_ad ? (T)0 : (T)-0.125;
    k.d.gam = h->gamma;
    k.d.gm1 = h->gamma - 1.0;
    k.d.g2 = h->gamma * h->gamma;
    k.d.c4 = 4.0 * (h->gamma - 1.0);
    k.d.hg = 0.5 * h->gamma;
    k.d.omd = 1.0 - 1e-12;
    k.d.omd2 = (1.0 - 1e-12) * (1.0 - 1e-12);
    k.d.mass = h->mass;
    k.d.tab = h->d_tab;
    k.d.ne = h->tab_ne; k.d.nn = h->tab_nn;
    k.d.ide = h->d_tab ? 1.0 / h->tab_de : 0.0;
    k.d.idn = h->d_tab ? 1.0 / h->tab_dn : 0.0;
    return k;
}

// ---------------------------------------------------------------- elementwise kernels
// eqs. (9)-(11).  Computed in fp64, stored in T.
template <typename T>
__global__ void prim2cons_kernel(long long n, const double* __restrict__ e, const double* __restrict__ nd,
                                 const double* __restrict__ vx, const double* __restrict__ vy,
                                 const double* __restrict__ vz, EosD kd,
                                 T* E, T* Mx, T* My, T* Mz, T* R, T* pe, T* pp, T* pn, T* pvx, T* pvy, T* pvz)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x) {
        const double ee = e[i], nn = nd[i], ax = vx[i], ay = vy[i], az = vz[i];
        double p;
        if (kd.tab) {                                   // tabled EOS (reading T1)
            double a_, b_;
            eos_table_eval(kd, ee, nn, p, a_, b_);
        } else {
            p = kd.gm1 * (ee - kd.mass * nn);
            p = p > 0.0 ? p : 0.0;
        }
        const double v2 = fma(ax, ax, fma(ay, ay, az * az));
        const double g2 = 1.0 / (1.0 - v2);
        const double w = (ee + p) * g2;
        E[i] = (T)(w - p);
        Mx[i] = (T)(w * ax); My[i] = (T)(w * ay); Mz[i] = (T)(w * az);
        R[i] = (T)(nn * sqrt(g2));
        pe[i] = (T)ee; pp[i] = (T)p; pn[i] = (T)nn; pvx[i] = (T)ax; pvy[i] = (T)ay; pvz[i] = (T)az;
    }
}

template <typename T, int EOS>
__global__ void cons2prim_kernel(long long n, Consts<T> k, const T* E, const T* Mx, const T* My, const T* Mz,
                                 const T* R, T* pe, T* pp, T* pn, T* pvx, T* pvy, T* pvz,
                                 unsigned long long* counts)
{
    Cnt cnt;
    cnt.zero();
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x) {
        T u[NF] = {E[i], Mx[i], My[i], Mz[i], R[i]};
        T pr[6];
        emit_primitives<T, EOS>(k, u, pr, cnt);
        pe[i] = pr[0]; pp[i] = pr[1]; pn[i] = pr[2]; pvx[i] = pr[3]; pvy[i] = pr[4]; pvz[i] = pr[5];
    }
    flush_counts(cnt, counts);
}

template <typename A, typename B>
__global__ void convert_kernel(long long n, const A* __restrict__ a, B* __restrict__ b)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x)
        b[i] = (B)a[i];
}

// per-block Neumaier-compensated partial sums of the five fields (sum, compensation)
template <typename T>
__global__ void __launch_bounds__(RED_THREADS) totals_kernel(long long n, const T* f0, const T* f1, const T* f2,
                                                            const T* f3, const T* f4, double* partial)
{
    const T* fld[NF] = {f0, f1, f2, f3, f4};
    __shared__ double sh[RED_THREADS / 32][NF][2];
    double s[NF], c[NF];
#pragma unroll
    for (int f = 0; f < NF; ++f) { s[f] = 0.0; c[f] = 0.0; }
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x) {
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            const double x = (double)fld[f][i];
            const double t = s[f] + x;
            c[f] += (fabs(s[f]) >= fabs(x)) ? ((s[f] - t) + x) : ((x - t) + s[f]);
            s[f] = t;
        }
    }
    // warp tree with two-sum so the compensation survives
#pragma unroll
    for (int f = 0; f < NF; ++f) {
        for (int o = 16; o > 0; o >>= 1) {
            const double so = __shfl_down_sync(0xffffffffu, s[f], o);
            const double co = __shfl_down_sync(0xffffffffu, c[f], o);
            const double t = s[f] + so;
            c[f] += co + ((fabs(s[f]) >= fabs(so)) ? ((s[f] - t) + so) : ((so - t) + s[f]));
            s[f] = t;
        }
        if ((threadIdx.x & 31) == 0) { sh[threadIdx.x >> 5][f][0] = s[f]; sh[threadIdx.x >> 5][f][1] = c[f]; }
    }
    __syncthreads();
    if (threadIdx.x < NF) {
        const int f = threadIdx.x;
        double ss = 0.0, cc = 0.0;
        for (int w = 0; w < RED_THREADS / 32; ++w) {
            const double x = sh[w][f][0];
            const double t = ss + x;
            cc += sh[w][f][1] + ((fabs(ss) >= fabs(x)) ? ((ss - t) + x) : ((x - t) + ss));
            ss = t;
        }
        partial[(blockIdx.x * NF + f) * 2 + 0] = ss;
        partial[(blockIdx.x * NF + f) * 2 + 1] = cc;
    }
}

int ew_grid(const shasta_t* h, int threads)
{
    long long b = (h->ncell + threads - 1) / threads;
    long long cap = (long long)h->sm_count * 16;
    return (int)(b < cap ? (b < 1 ? 1 : b) : cap);
}

// ---------------------------------------------------------------- sweep launch
// Cells marched per work item.  Every segment re-marches 8 halo cells, so long segments are cheap per cell, but
// the grid must fill the machine: a sweep kernel runs 2 CTAs of 128 pencils per SM (`slots` CTAs at once).
// Measured on B200 (segment scan at 64^3 .. 512^3): when one layer of CTAs is already >= 3 waves the
// whole pencil is one segment; large grids want the longest segments that still give ~3 waves (256^3: 2 x 128
// cells); grids that fit into one wave want that wave as full as possible (128^3: 2 x 64, 64^3: 4 x 16).
int auto_segment(const shasta_t* h, int axis, int N, long long base)
{
    if (h->seg_override > 0) return h->seg_override < N ? h->seg_override : N;
    const long long slots = (long long)(eos_mode(h) == EOS_GAMMA ? 2 : GEN_CTAS) * h->sm_count;     // CTAs resident at once
    // base = CTAs per layer of segments
    const long long max_nseg = N / 16 > 1 ? N / 16 : 1;            // segments not shorter than 16 cells
    long long nseg = 1;
    if (base < 3 * slots) {
        const long long one_wave = slots / base;                   // layers that fit one wave (0: none)
        const long long three_waves = (3 * slots + base - 1) / base;
        double best = 1e300;
        const long long cand[2] = {one_wave, three_waves};
        for (int c = 0; c < 2; ++c) {
            long long n = cand[c] < 1 ? 0 : (cand[c] > max_nseg ? max_nseg : cand[c]);
            if (n < 1) continue;
            const double seg = (double)((N + n - 1) / n);
            const double waves = (double)(base * n) / (double)slots;
            const double t = (waves < 1.0 ? 1.0 : waves) * (seg + 8.0);
            if (t < best) { best = t; nseg = n; }
        }
    }
    long long seg = (N + nseg - 1) / nseg;
    if (axis == 0) seg = ((seg + 7) / 8) * 8;             // group-aligned segments for the x sweep (TMA boxes start at 16 B)
    return (int)(seg < N ? seg : N);
}

template <typename T, int EOS, int EMIT>
int launch_sweep_t(shasta_t* h, int axis, cudaStream_t st)
{
    const int n[3] = {h->nx, h->ny, h->nz};
    const long long stride[3] = {1, h->nx, (long long)h->nx * h->ny};
    const int perm[3][3] = {{0, 1, 2}, {1, 2, 0}, {2, 0, 1}};   // parallel, perp1, perp2 momentum components
    SweepParams P;
    const int src = h->cur, dst = 1 - h->cur;
    P.in[0] = h->U[src][0]; P.out[0] = h->U[dst][0];
    for (int c = 0; c < 3; ++c) {
        P.in[1 + c] = h->U[src][1 + perm[axis][c]];
        P.out[1 + c] = h->U[dst][1 + perm[axis][c]];
        P.prim[3 + c] = h->prim[3 + perm[axis][c]];
    }
    P.in[4] = h->U[src][4]; P.out[4] = h->U[dst][4];
    P.prim[0] = h->prim[0]; P.prim[1] = h->prim[1]; P.prim[2] = h->prim[2];
    P.nx = h->nx;
    P.N = n[axis];
    P.stride_axis = stride[axis];
    P.periodic = axis_periodic(h, axis);
    P.axis = axis;
    P.odiv = 0x7fffffff;
    P.counts = h->d_counts;
    const Consts<T> k = make_consts<T>(h);
    const bool zrange = h->az_lo > 0 || h->az_hi < h->nz;      // single event only (checked in shasta_set_active_planes)
    P.pbase = 0;
    if (axis == 0) {
        P.npencil = (long long)h->ny * h->nz * h->nbatch;
        if (zrange) { P.pbase = (long long)h->az_lo * h->ny; P.npencil = (long long)h->az_hi * h->ny; }   // rows y + ny z
        const long long nrow = P.npencil - P.pbase;
        P.stride_other = 0;
        P.seg = auto_segment(h, axis, P.N, (nrow + 127) / 128);
        P.nseg = (P.N + P.seg - 1) / P.seg;
        {
            // producer/consumer warp pairs, 32 rows per pair, 4 pairs per CTA; TMA tiles when possible (fp64, even nx)
            const bool tma = h->have_tmap && !h->no_tma;
            X2Maps maps;
            memset(&maps, 0, sizeof(maps));
            maps.fidx[0] = 0; maps.fidx[4] = 4;
            for (int c = 0; c < 3; ++c) maps.fidx[1 + c] = 1 + perm[axis][c];
            if (tma) { maps.in = h->d_xmaps + src * NF; maps.out = h->d_xmaps + dst * NF; }
            const size_t smem = sizeof(X2Smem<T>);
            dim3 grid((unsigned)((nrow + 127) / 128), (unsigned)P.nseg);
            if (tma) {
                auto kern = sweep_x2_kernel<T, EOS, EMIT == 1, true>;
                int rc = opt_in_smem(h, (const void*)kern, smem);
                if (rc) return rc;
                kern<<<grid, 256, smem, st>>>(P, k, maps);
            } else {
                auto kern = sweep_x2_kernel<T, EOS, EMIT == 1, false>;
                int rc = opt_in_smem(h, (const void*)kern, smem);
                if (rc) return rc;
                kern<<<grid, 256, smem, st>>>(P, k, maps);
            }
        }
    } else {
        // y sweep: pencils (x,z), base = x + z*nx*ny;  z sweep: pencils (x,y), base = x + y*nx = flat
        const int other = axis == 1 ? 2 : 1;
        P.stride_other = stride[other];
        {
            // producer/consumer warp pairs, 32 pencils (one x-block of a row) per pair, 4 pairs per CTA; TMA-fed when possible
            const long long nxb = (h->nx + 31) / 32;
            P.npencil = nxb * n[other] * h->nbatch;                             // pencil GROUPS (all events)
            if (zrange && axis == 1) { P.pbase = nxb * h->az_lo; P.npencil = nxb * h->az_hi; }   // groups xb + nxb z
            P.odiv = (axis == 2 && h->nbatch > 1) ? h->ny : 0x7fffffff;
            const long long ctas = (P.npencil - P.pbase + 3) / 4;
            P.seg = auto_segment(h, axis, P.N, ctas);
            P.nseg = (P.N + P.seg - 1) / P.seg;
            const bool tma = h->have_yzmap && !h->no_tma && P.N >= YZ_CH;
            YzMaps maps;
            memset(&maps, 0, sizeof(maps));
            maps.fidx[0] = 0; maps.fidx[4] = 4;
            for (int c = 0; c < 3; ++c) maps.fidx[1 + c] = 1 + perm[axis][c];
            if (tma) {
                maps.in4 = h->d_yzmaps + (src * 3 + (axis == 1 ? 0 : 1)) * NF;
                maps.in1 = h->d_yzmaps + (src * 3 + 2) * NF;
            }
            const size_t smem = sizeof(YzSmem<T>);
            dim3 grid((unsigned)ctas, (unsigned)P.nseg);
#define SHK_LAUNCH_YZ(TMA_)                                                                        \
            {                                                                                       \
                auto kern = sweep_yz_kernel<T, EOS, EMIT, TMA_>;                                    \
                int rc = opt_in_smem(h, (const void*)kern, smem);                                   \
                if (rc) return rc;                                                                  \
                kern<<<grid, 256, smem, st>>>(P, k, maps);                                          \
            }
            if (tma) SHK_LAUNCH_YZ(true) else SHK_LAUNCH_YZ(false)
#undef SHK_LAUNCH_YZ
        }
    }
    CK(cudaGetLastError());
    h->launches++;
    h->cur = dst;
    return 0;
}

// per-cell kernels (sweep_cell_kernel): the paper's own decomposition, used for the R2 predictor
template <int EOS>
int launch_cell_sweep(shasta_t* h, int axis, bool emit, cudaStream_t st)
{
    const int n[3] = {h->nx, h->ny, h->nz};
    const long long stride[3] = {1, h->nx, (long long)h->nx * h->ny};
    const int perm[3][3] = {{0, 1, 2}, {1, 2, 0}, {2, 0, 1}};
    SweepParams P;
    memset(&P, 0, sizeof(P));
    const int src = h->cur, dst = 1 - h->cur;
    P.in[0] = h->U[src][0]; P.out[0] = h->U[dst][0];
    for (int c = 0; c < 3; ++c) {
        P.in[1 + c] = h->U[src][1 + perm[axis][c]];
        P.out[1 + c] = h->U[dst][1 + perm[axis][c]];
        P.prim[3 + c] = h->prim[3 + perm[axis][c]];
    }
    P.in[4] = h->U[src][4]; P.out[4] = h->U[dst][4];
    P.prim[0] = h->prim[0]; P.prim[1] = h->prim[1]; P.prim[2] = h->prim[2];
    P.nx = h->nx; P.N = n[axis]; P.stride_axis = stride[axis]; P.periodic = axis_periodic(h, axis); P.axis = axis;
    P.counts = h->d_counts;
    const Consts<double> k = make_consts<double>(h);
    const unsigned blocks = (unsigned)((h->ncell + 127) / 128);
    if (h->predictor) sweep_cell_kernel<EOS, true><<<blocks, 128, 0, st>>>(P, k, h->ncell, h->diff, emit ? 1 : 0);
    else              sweep_cell_kernel<EOS, false><<<blocks, 128, 0, st>>>(P, k, h->ncell, h->diff, emit ? 1 : 0);
    CK(cudaGetLastError());
    h->launches++;
    h->cur = dst;
    return 0;
}

// emit: 0 none, 1 primitives of the new state, 2 primitives of the state the sweep reads (y/z fused kernels only)
template <typename T, int EOS>
int launch_sweep_e(shasta_t* h, int axis, int emit, cudaStream_t st)
{
    if (emit == 2 && axis != 0) return launch_sweep_t<T, EOS, 2>(h, axis, st);
    return emit ? launch_sweep_t<T, EOS, 1>(h, axis, st) : launch_sweep_t<T, EOS, 0>(h, axis, st);
}

int launch_sweep_raw(shasta_t* h, int axis, int emit, cudaStream_t st)
{
    const int eos = eos_mode(h);
    if (h->predictor || h->cell_path) {
        if (h->precision != 64) return fail(h, SHASTA_ESTATE, "the per-cell kernels (R2 predictor) run in fp64 only");
        if (eos == EOS_TABLE) return launch_cell_sweep<EOS_TABLE>(h, axis, emit != 0, st);
        return eos == EOS_MASS ? launch_cell_sweep<EOS_MASS>(h, axis, emit != 0, st) : launch_cell_sweep<EOS_GAMMA>(h, axis, emit != 0, st);
    }
    if (h->precision == 64) {
        if (eos == EOS_TABLE) return launch_sweep_e<double, EOS_TABLE>(h, axis, emit, st);
        return eos == EOS_MASS ? launch_sweep_e<double, EOS_MASS>(h, axis, emit, st) : launch_sweep_e<double, EOS_GAMMA>(h, axis, emit, st);
    }
    if (eos == EOS_TABLE) return launch_sweep_e<float, EOS_TABLE>(h, axis, emit, st);
    return eos == EOS_MASS ? launch_sweep_e<float, EOS_MASS>(h, axis, emit, st) : launch_sweep_e<float, EOS_GAMMA>(h, axis, emit, st);
}

template <typename T>
int refresh_prims_t(shasta_t* h, cudaStream_t st)
{
    void** U = h->U[h->cur];
    const int g = ew_grid(h, 256);
    const Consts<T> k = make_consts<T>(h);
    if (eos_mode(h) == EOS_TABLE)
        cons2prim_kernel<T, EOS_TABLE><<<g, 256, 0, st>>>(h->ncell, k, (T*)U[0], (T*)U[1], (T*)U[2], (T*)U[3],
            (T*)U[4], (T*)h->prim[0], (T*)h->prim[1], (T*)h->prim[2], (T*)h->prim[3], (T*)h->prim[4],
            (T*)h->prim[5], h->d_counts);
    else if (use_general_eos(h))
        cons2prim_kernel<T, EOS_MASS><<<g, 256, 0, st>>>(h->ncell, k, (T*)U[0], (T*)U[1], (T*)U[2], (T*)U[3],
            (T*)U[4], (T*)h->prim[0], (T*)h->prim[1], (T*)h->prim[2], (T*)h->prim[3], (T*)h->prim[4],
            (T*)h->prim[5], h->d_counts);
    else
        cons2prim_kernel<T, EOS_GAMMA><<<g, 256, 0, st>>>(h->ncell, k, (T*)U[0], (T*)U[1], (T*)U[2], (T*)U[3],
            (T*)U[4], (T*)h->prim[0], (T*)h->prim[1], (T*)h->prim[2], (T*)h->prim[3], (T*)h->prim[4],
            (T*)h->prim[5], h->d_counts);
    CK(cudaGetLastError());
    h->launches++;
    h->prims_valid = true;
    return 0;
}

bool fused_path(const shasta_t* h) { return !h->predictor && !h->cell_path; }

// One sweep.  emit: 0 none, 1 primitives of the new state, 2 primitives of the state BEFORE the sweep (fused y/z kernels).
// When a sweep along x has to emit (the last sweep of a step), the primitives are written by the element-wise cons2prim
// kernel after it: in the warp-specialised x kernel the consumer warp is the critical one, and six more fields through
// its staging tile cost more than re-reading the five conserved fields once.  shasta_step avoids that pass where it can
// (see there): the NEXT sweep reads those fields anyway and emits their primitives (emit = 2).
int launch_sweep(shasta_t* h, int axis, int emit, cudaStream_t st)
{
    if (emit == 2 && (axis == 0 || !fused_path(h)))
        return fail(h, SHASTA_EINVAL, "emit = 2 (primitives of the input state) exists for the fused y and z sweeps only");
    if (emit == 1 && axis == 0 && fused_path(h)) {
        int rc = launch_sweep_raw(h, axis, 0, st);
        if (rc) return rc;
        return h->precision == 64 ? refresh_prims_t<double>(h, st) : refresh_prims_t<float>(h, st);
    }
    return launch_sweep_raw(h, axis, emit, st);
}

// copy one stored field (T) into a caller fp64 device buffer
int export_field(shasta_t* h, const void* src, double* dst_dev, cudaStream_t st)
{
    if (h->precision == 64) {
        CK(cudaMemcpyAsync(dst_dev, src, sizeof(double) * (size_t)h->ncell, cudaMemcpyDeviceToDevice, st));
    } else {
        convert_kernel<float, double><<<ew_grid(h, 256), 256, 0, st>>>(h->ncell, (const float*)src, dst_dev);
        CK(cudaGetLastError());
        h->launches++;
    }
    return 0;
}

// cached CUDA graphs of whole axis-table cycles (shasta_step): dropped whenever an option or the table changes
void drop_graphs(shasta_t* h)
{
    for (int i = 0; i < h->ngraphs; ++i) cudaGraphExecDestroy(h->graphs[i].exec);
    h->ngraphs = 0;
}

// `nsteps` time steps, launch by launch (step s runs the sweeps branch[3s .. 3s+2]).
int run_steps(shasta_t* h, int nsteps, cudaStream_t st)
{
    const int n[3] = {h->nx, h->ny, h->nz};
    // A step whose last sweep runs along x does not write its primitives at once: the first sweep of the NEXT step reads
    // the same five conserved fields anyway and writes the primitives of its input state beside its own work (emit = 2,
    // +0.14 ms at 256^3 instead of +0.26 ms for the separate element-wise pass).  Every step's primitives are still
    // written exactly once; the deferral never leaves this call (the last step of the call is completed below).
    bool deferred = false;
    for (int s = 0; s < nsteps; ++s) {
        int axes[3], na = 0;
        for (int k = 0; k < 3; ++k) {
            const int a = h->table[(3 * h->step + k) % h->ntable];
            if (n[a] > 1) axes[na++] = a;                 // reading G15: axes of extent 1 are skipped
        }
        for (int k = 0; k < na; ++k) {
            const bool last = k == na - 1;
            int emit = last ? 1 : 0;
            if (deferred) {                               // k == 0
                deferred = false;
                if (!last && axes[k] != 0) emit = 2;
                else {
                    int rc = h->precision == 64 ? refresh_prims_t<double>(h, st) : refresh_prims_t<float>(h, st);
                    if (rc) return rc;
                }
            }
            if (last && axes[k] == 0 && fused_path(h) && !h->no_defer) { emit = 0; deferred = true; }
            int rc = launch_sweep(h, axes[k], emit, st);
            if (rc) return rc;
        }
        if (na > 0) h->prims_valid = true;
        h->step++;
    }
    if (deferred) {
        int rc = h->precision == 64 ? refresh_prims_t<double>(h, st) : refresh_prims_t<float>(h, st);
        if (rc) return rc;
    }
    return 0;
}

// The graph of `chunk` steps starting at table phase `phase` with the state in buffer `cur` (captured on a private
// stream on first use; the capture executes nothing).  PAPER.md:155 names the "orchestration overhead" of many small
// kernels: for grids whose sweeps take ~10 us the launches of a whole cycle (18 sweeps) go to the GPU as one graph.
int get_graph(shasta_t* h, int phase, int chunk, shasta::GraphEntry** out)
{
    *out = nullptr;
    for (int i = 0; i < h->ngraphs; ++i)
        if (h->graphs[i].phase == phase && h->graphs[i].cur == h->cur && h->graphs[i].chunk == chunk) { *out = &h->graphs[i]; return 0; }
    if (h->ngraphs == 8) drop_graphs(h);
    if (!h->cap_stream) CK(cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking));
    const long long step0 = h->step, l0 = h->launches;
    const int cur0 = h->cur;
    const bool pv0 = h->prims_valid;
    CK(cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal));
    const int rc = run_steps(h, chunk, h->cap_stream);
    cudaGraph_t g = nullptr;
    const cudaError_t e = cudaStreamEndCapture(h->cap_stream, &g);
    const long long nl = h->launches - l0;
    const bool same_buffer = h->cur == cur0;
    h->step = step0; h->launches = l0; h->cur = cur0; h->prims_valid = pv0;
    if (rc || e != cudaSuccess || !g || !same_buffer) {
        if (g) cudaGraphDestroy(g);
        cudaGetLastError();
        return rc ? rc : 1;                              // 1 = no graph: the caller launches directly
    }
    cudaGraphExec_t exec = nullptr;
    const cudaError_t e2 = cudaGraphInstantiate(&exec, g, 0);
    cudaGraphDestroy(g);
    if (e2 != cudaSuccess) { cudaGetLastError(); return 1; }
    shasta::GraphEntry& ge = h->graphs[h->ngraphs++];
    ge.phase = phase; ge.cur = cur0; ge.chunk = chunk; ge.exec = exec; ge.launches = nl;
    *out = &ge;
    return 0;
}

}  // namespace

// =========================================================================== C ABI
extern "C" {

int shasta_create(shasta_t** out, int nx, int ny, int nz, double dx, double lambda, double eos_gamma)
{
    shasta_t* h = nullptr;
    if (!out) return fail(h, SHASTA_EINVAL, "shasta_create: out is NULL");
    *out = nullptr;
    if (nx < 1 || ny < 1 || nz < 1) return fail(h, SHASTA_EINVAL, "shasta_create: grid extents must be >= 1");
    if (!(dx > 0.0)) return fail(h, SHASTA_EINVAL, "shasta_create: dx must be > 0");
    if (!(lambda > 0.0) || lambda > 0.5) return fail(h, SHASTA_EINVAL, "shasta_create: need 0 < lambda <= 0.5");
    if (!(eos_gamma > 1.0) || !(eos_gamma < 2.0))
        return fail(h, SHASTA_EINVAL, "shasta_create: need 1 < eos_gamma < 2");
    int dev = 0, ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1)
        return fail(h, SHASTA_ECUDA, "shasta_create: no CUDA device (there is no CPU fallback)");
    if (cudaGetDevice(&dev) != cudaSuccess) return fail(h, SHASTA_ECUDA, "shasta_create: cudaGetDevice failed");
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess)
        return fail(h, SHASTA_ECUDA, "shasta_create: cudaGetDeviceProperties failed");
    if (prop.major < 10)
        return fail(h, SHASTA_ECUDA, "shasta_create: device sm_%d%d is not sm_100 (B200) -- kernels are built for sm_100a only",
                    prop.major, prop.minor);
    h = new (std::nothrow) shasta();
    if (!h) return fail(nullptr, SHASTA_ENOMEM, "shasta_create: host allocation failed");
    memset(h, 0, sizeof(*h));
    h->nx = nx; h->ny = ny; h->nz = nz;
    h->ncell = h->ncell1 = (long long)nx * ny * nz;
    h->nbatch = 1;
    h->dx = dx; h->lambda = lambda; h->gamma = eos_gamma; h->mass = 0.0;
    h->precision = 64;
    h->diff = 1.0;
    h->periodic_z = -1;
    h->az_lo = 0; h->az_hi = nz;
    h->graph_mode = 2;
    memcpy(h->table, kBranch, sizeof(kBranch));
    h->ntable = 18;
    h->sm_count = prop.multiProcessorCount;
    h->device = dev;
    *out = h;
    return 0;
}

void shasta_destroy(shasta_t* h)
{
    if (!h) return;
    drop_graphs(h);
    if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
    free_fields(h);
    cudaFree(h->stage);
    cudaFree(h->d_tab);
    cudaFree(h->d_yzmaps);
    cudaFree(h->d_xmaps);
    delete h;
}

int shasta_set_option(shasta_t* h, int key, double value)
{
    if (!h) return SHASTA_EINVAL;
    drop_graphs(h);                                       // cached graphs bake the options in
    switch (key) {
    case SHASTA_GRAPH:
        if (value != 0.0 && value != 1.0 && value != 2.0) return fail(h, SHASTA_EINVAL, "SHASTA_GRAPH must be 0, 1 or 2");
        h->graph_mode = (int)value;
        return 0;
    case SHASTA_BOUNDARY:
        if (value != 0.0 && value != 1.0) return fail(h, SHASTA_EINVAL, "SHASTA_BOUNDARY must be 0 or 1");
        h->periodic = (int)value;
        return 0;
    case SHASTA_EOS_MASS:
        if (!(value >= 0.0)) return fail(h, SHASTA_EINVAL, "SHASTA_EOS_MASS must be >= 0");
        if (h->have_state && value != h->mass)
            return fail(h, SHASTA_ESTATE, "SHASTA_EOS_MASS must be set before shasta_set_state (the conserved state was built with the old EOS)");
        h->mass = value;
        h->prims_valid = false;
        return 0;
    case SHASTA_PRECISION:
        if (value != 64.0 && value != 32.0) return fail(h, SHASTA_EINVAL, "SHASTA_PRECISION must be 64 or 32");
        if (h->allocated && (int)value != h->precision)
            return fail(h, SHASTA_ESTATE, "SHASTA_PRECISION must be set before the first set_state");
        h->precision = (int)value;
        return 0;
    case SHASTA_STEP_INDEX:
        if (!(value >= 0.0)) return fail(h, SHASTA_EINVAL, "SHASTA_STEP_INDEX must be >= 0");
        h->step = (long long)value;
        return 0;
    case SHASTA_SEGMENT:
        if (!(value >= 0.0)) return fail(h, SHASTA_EINVAL, "SHASTA_SEGMENT must be >= 0");
        h->seg_override = (int)value;
        if (h->seg_override > 0 && h->seg_override < 8) h->seg_override = 8;
        return 0;
    case SHASTA_NO_TMA:
        h->no_tma = value != 0.0;
        return 0;
    case SHASTA_BATCH:
        if (!(value >= 1.0) || value > 65536.0 || value != (double)(int)value)
            return fail(h, SHASTA_EINVAL, "SHASTA_BATCH must be an integer in [1, 65536]");
        if (h->allocated && (int)value != h->nbatch)
            return fail(h, SHASTA_ESTATE, "SHASTA_BATCH must be set before the first set_state");
        if ((double)h->nz * value > 2147483647.0 / 2)
            return fail(h, SHASTA_EINVAL, "SHASTA_BATCH: nz * batch too large");
        if (value != 1.0 && (h->az_lo > 0 || h->az_hi < h->nz))
            return fail(h, SHASTA_ESTATE, "SHASTA_BATCH > 1: not with shasta_set_active_planes");
        h->nbatch = (int)value;
        h->ncell = h->ncell1 * h->nbatch;
        return 0;
    case SHASTA_PRIMS_RAW:
        h->prims_raw = value != 0.0;
        return 0;
    case SHASTA_NO_DEFER:
        h->no_defer = value != 0.0;
        return 0;
    case SHASTA_DIFF:
        if (!(value >= 0.0) || value > 8.0) return fail(h, SHASTA_EINVAL, "SHASTA_DIFF must be in [0, 8]");
        h->diff = value;
        return 0;
    case SHASTA_CELL_PATH:
        h->cell_path = value != 0.0;
        return 0;
    case SHASTA_BOUNDARY_Z:
        if (value != -1.0 && value != 0.0 && value != 1.0)
            return fail(h, SHASTA_EINVAL, "SHASTA_BOUNDARY_Z must be -1 (as SHASTA_BOUNDARY), 0 or 1");
        h->periodic_z = (int)value;
        return 0;
    case SHASTA_ANTIDIFFUSION:
        if (value != 0.0 && value != 1.0)
            return fail(h, SHASTA_EINVAL, "SHASTA_ANTIDIFFUSION must be 0 (phoenical) or 1 (explicit)");
        h->explicit_ad = (int)value;
        return 0;
    case SHASTA_PREDICTOR:
        if (value != 0.0 && value != 1.0) return fail(h, SHASTA_EINVAL, "SHASTA_PREDICTOR must be 0 (R1) or 1 (R2)");
        if (value == 1.0 && h->precision != 64) return fail(h, SHASTA_EINVAL, "SHASTA_PREDICTOR 1 runs in fp64 only");
        h->predictor = (int)value;
        return 0;
    case SHASTA_VARIANT:
        if (value != 0.0) return fail(h, SHASTA_EINVAL, "SHASTA_VARIANT: only 0 exists (the single-role kernels of round 1 were removed)");
        return 0;
    default:
        return fail(h, SHASTA_EINVAL, "shasta_set_option: unknown key %d", key);
    }
}

int shasta_set_eos_table(shasta_t* h, const double* p_host, int ne, int nn, double e_max, double n_max)
{
    if (!h) return SHASTA_EINVAL;
    drop_graphs(h);
    if (!p_host) {                                       // back to the analytic EOS
        if (h->d_tab) { CK(cudaDeviceSynchronize()); cudaFree(h->d_tab); h->d_tab = nullptr; }
        h->prims_valid = false;
        return 0;
    }
    if (ne < 2 || nn < 2 || (long long)ne * nn > (1LL << 26)) return fail(h, SHASTA_EINVAL, "shasta_set_eos_table: need 2 <= ne, nn and ne*nn <= 2^26");
    if (!(e_max > 0.0) || !(n_max > 0.0)) return fail(h, SHASTA_EINVAL, "shasta_set_eos_table: e_max and n_max must be > 0");
    if (h->d_tab) { CK(cudaDeviceSynchronize()); cudaFree(h->d_tab); h->d_tab = nullptr; }
    CK(cudaMalloc(&h->d_tab, sizeof(double) * (size_t)ne * nn));
    CK(cudaMemcpy(h->d_tab, p_host, sizeof(double) * (size_t)ne * nn, cudaMemcpyHostToDevice));
    h->tab_ne = ne; h->tab_nn = nn;
    h->tab_de = e_max / (ne - 1); h->tab_dn = n_max / (nn - 1);
    h->prims_valid = false;
    return 0;
}

int shasta_set_sweep_table(shasta_t* h, const int* axes, int n)
{
    if (!h) return SHASTA_EINVAL;
    if (!axes || n < 3 || n > 63 || n % 3) return fail(h, SHASTA_EINVAL, "sweep table: need n % 3 == 0, 3 <= n <= 63");
    for (int i = 0; i < n; ++i)
        if (axes[i] < 0 || axes[i] > 2) return fail(h, SHASTA_EINVAL, "sweep table: axes must be 0, 1 or 2");
    drop_graphs(h);
    memcpy(h->table, axes, sizeof(int) * (size_t)n);
    h->ntable = n;
    return 0;
}

int shasta_set_state(shasta_t* h, const double* e, const double* n, const double* vx, const double* vy,
                     const double* vz, void* stream)
{
    if (!h) return SHASTA_EINVAL;
    if (!e || !n || !vx || !vy || !vz) return fail(h, SHASTA_EINVAL, "shasta_set_state: NULL field pointer");
    int rc = ensure_alloc(h);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    h->cur = 0;
    void** U = h->U[0];
    const int g = ew_grid(h, 256);
    if (h->precision == 64)
        prim2cons_kernel<double><<<g, 256, 0, st>>>(h->ncell, e, n, vx, vy, vz, make_consts<double>(h).d,
            (double*)U[0], (double*)U[1], (double*)U[2], (double*)U[3], (double*)U[4], (double*)h->prim[0],
            (double*)h->prim[1], (double*)h->prim[2], (double*)h->prim[3], (double*)h->prim[4], (double*)h->prim[5]);
    else
        prim2cons_kernel<float><<<g, 256, 0, st>>>(h->ncell, e, n, vx, vy, vz, make_consts<double>(h).d,
            (float*)U[0], (float*)U[1], (float*)U[2], (float*)U[3], (float*)U[4], (float*)h->prim[0],
            (float*)h->prim[1], (float*)h->prim[2], (float*)h->prim[3], (float*)h->prim[4], (float*)h->prim[5]);
    CK(cudaGetLastError());
    h->launches++;
    h->have_state = true;
    h->prims_valid = true;
    return 0;
}

int shasta_set_state_host(shasta_t* h, const double* e, const double* n, const double* vx, const double* vy,
                          const double* vz, void* stream)
{
    if (!h) return SHASTA_EINVAL;
    if (!e || !n || !vx || !vy || !vz) return fail(h, SHASTA_EINVAL, "shasta_set_state_host: NULL field pointer");
    int rc = ensure_stage(h);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nb = sizeof(double) * (size_t)h->ncell;
    const double* src[5] = {e, n, vx, vy, vz};
    for (int f = 0; f < 5; ++f)
        CK(cudaMemcpyAsync(h->stage + (size_t)f * h->ncell, src[f], nb, cudaMemcpyHostToDevice, st));
    return shasta_set_state(h, h->stage, h->stage + h->ncell, h->stage + 2 * h->ncell, h->stage + 3 * h->ncell,
                            h->stage + 4 * h->ncell, stream);
}

int shasta_set_conserved(shasta_t* h, const double* E, const double* Mx, const double* My, const double* Mz,
                         const double* R, void* stream)
{
    if (!h) return SHASTA_EINVAL;
    if (!E || !Mx || !My || !Mz || !R) return fail(h, SHASTA_EINVAL, "shasta_set_conserved: NULL field pointer");
    int rc = ensure_alloc(h);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const double* src[NF] = {E, Mx, My, Mz, R};
    h->cur = 0;
    for (int f = 0; f < NF; ++f) {
        if (h->precision == 64) {
            CK(cudaMemcpyAsync(h->U[0][f], src[f], sizeof(double) * (size_t)h->ncell, cudaMemcpyDeviceToDevice, st));
        } else {
            convert_kernel<double, float><<<ew_grid(h, 256), 256, 0, st>>>(h->ncell, src[f], (float*)h->U[0][f]);
            CK(cudaGetLastError());
            h->launches++;
        }
    }
    h->have_state = true;
    h->prims_valid = false;
    return 0;
}

int shasta_get_conserved(shasta_t* h, double* E, double* Mx, double* My, double* Mz, double* R, void* stream)
{
    if (!h) return SHASTA_EINVAL;
    if (!h->have_state) return fail(h, SHASTA_ESTATE, "shasta_get_conserved: no state set");
    double* dst[NF] = {E, Mx, My, Mz, R};
    for (int f = 0; f < NF; ++f)
        if (dst[f]) {
            int rc = export_field(h, h->U[h->cur][f], dst[f], (cudaStream_t)stream);
            if (rc) return rc;
        }
    return 0;
}

// planes z0 .. z0+nplanes-1 of the current conserved state (z is the slowest axis: one contiguous block per field)
static int plane_range(shasta_t* h, const char* who, int z0, int nplanes, size_t* off, long long* cnt)
{
    if (!h->have_state) return fail(h, SHASTA_ESTATE, "%s: no state set", who);
    if (h->nbatch != 1) return fail(h, SHASTA_ESTATE, "%s: not with SHASTA_BATCH > 1", who);
    if (z0 < 0 || nplanes < 0 || (long long)z0 + nplanes > h->nz)
        return fail(h, SHASTA_EINVAL, "%s: planes [%d, %d) outside [0, %d)", who, z0, z0 + nplanes, h->nz);
    int rc = check_device(h);
    if (rc) return rc;
    *off = (size_t)z0 * (size_t)h->nx * (size_t)h->ny;
    *cnt = (long long)nplanes * h->nx * h->ny;
    return 0;
}

int shasta_get_planes(shasta_t* h, int z0, int nplanes, double* E, double* Mx, double* My, double* Mz, double* R,
                      void* stream)
{
    if (!h) return SHASTA_EINVAL;
    size_t off; long long cnt;
    int rc = plane_range(h, "shasta_get_planes", z0, nplanes, &off, &cnt);
    if (rc || cnt == 0) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    double* dst[NF] = {E, Mx, My, Mz, R};
    for (int f = 0; f < NF; ++f) {
        if (!dst[f]) continue;
        if (h->precision == 64) {
            CK(cudaMemcpyAsync(dst[f], (const double*)h->U[h->cur][f] + off, sizeof(double) * (size_t)cnt,
                               cudaMemcpyDeviceToDevice, st));
        } else {
            convert_kernel<float, double><<<ew_grid(h, 256), 256, 0, st>>>(cnt, (const float*)h->U[h->cur][f] + off, dst[f]);
            CK(cudaGetLastError());
            h->launches++;
        }
    }
    return 0;
}

int shasta_set_planes(shasta_t* h, int z0, int nplanes, const double* E, const double* Mx, const double* My,
                      const double* Mz, const double* R, void* stream)
{
    if (!h) return SHASTA_EINVAL;
    size_t off; long long cnt;
    int rc = plane_range(h, "shasta_set_planes", z0, nplanes, &off, &cnt);
    if (rc || cnt == 0) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const double* src[NF] = {E, Mx, My, Mz, R};
    for (int f = 0; f < NF; ++f) {
        if (!src[f]) continue;
        if (h->precision == 64) {
            CK(cudaMemcpyAsync((double*)h->U[h->cur][f] + off, src[f], sizeof(double) * (size_t)cnt,
                               cudaMemcpyDeviceToDevice, st));
        } else {
            convert_kernel<double, float><<<ew_grid(h, 256), 256, 0, st>>>(cnt, src[f], (float*)h->U[h->cur][f] + off);
            CK(cudaGetLastError());
            h->launches++;
        }
    }
    h->prims_valid = false;
    return 0;
}

int shasta_set_active_planes(shasta_t* h, int z_lo, int z_hi)
{
    if (!h) return SHASTA_EINVAL;
    if (z_lo < 0 || z_hi > h->nz || z_lo >= z_hi)
        return fail(h, SHASTA_EINVAL, "shasta_set_active_planes: need 0 <= z_lo < z_hi <= nz = %d", h->nz);
    if (h->nbatch != 1 && (z_lo != 0 || z_hi != h->nz))
        return fail(h, SHASTA_ESTATE, "shasta_set_active_planes: not with SHASTA_BATCH > 1");
    drop_graphs(h);
    h->az_lo = z_lo; h->az_hi = z_hi;
    return 0;
}

int shasta_plane_ptr(shasta_t* h, int field, int z0, void** ptr_dev)
{
    if (!h) return SHASTA_EINVAL;
    if (!ptr_dev) return fail(h, SHASTA_EINVAL, "shasta_plane_ptr: NULL output");
    if (field < 0 || field >= NF) return fail(h, SHASTA_EINVAL, "shasta_plane_ptr: field %d outside [0, 5)", field);
    size_t off; long long cnt;
    int rc = plane_range(h, "shasta_plane_ptr", z0, 0, &off, &cnt);
    if (rc) return rc;
    *ptr_dev = (char*)h->U[h->cur][field] + off * esize(h);
    return 0;
}

int shasta_step(shasta_t* h, int nsteps, void* stream)
{
    if (!h) return SHASTA_EINVAL;
    if (nsteps < 0) return fail(h, SHASTA_EINVAL, "shasta_step: nsteps < 0");
    if (!h->have_state) return fail(h, SHASTA_ESTATE, "shasta_step: call shasta_set_state first");
    if (int rc = check_device(h)) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    // whole cycles of the axis table as one CUDA graph each (auto: only where a sweep is short enough for launch gaps to
    // show, < 2^22 cells); the remainder launch by launch
    const bool want_graph = h->graph_mode == 1 || (h->graph_mode == 2 && h->ncell < (1LL << 22));
    if (want_graph && h->ntable % 3 == 0) {
        const int period = h->ntable / 3;
        int na = 0;
        if (h->nx > 1) ++na;
        if (h->ny > 1) ++na;
        if (h->nz > 1) ++na;
        int sweeps = 0;                                   // sweeps of one period (every table entry of an active axis)
        const int n[3] = {h->nx, h->ny, h->nz};
        for (int i = 0; i < h->ntable; ++i) sweeps += n[h->table[i]] > 1;
        const int chunk = (sweeps % 2 == 0) ? period : 2 * period;      // the state must return to the buffer it started in
        while (na > 0 && nsteps >= chunk) {
            shasta::GraphEntry* ge = nullptr;
            const int rc = get_graph(h, (int)(h->step % period), chunk, &ge);
            if (rc < 0) return rc;
            if (!ge) break;
            CK(cudaGraphLaunch(ge->exec, st));
            h->launches += ge->launches;
            h->graph_launches++;
            h->step += chunk;
            h->prims_valid = true;
            nsteps -= chunk;
        }
    }
    return run_steps(h, nsteps, st);
}

int shasta_sweep(shasta_t* h, int axis, int emit_primitives, void* stream)
{
    if (!h) return SHASTA_EINVAL;
    if (axis < 0 || axis > 2) return fail(h, SHASTA_EINVAL, "shasta_sweep: axis must be 0, 1 or 2");
    if (!h->have_state) return fail(h, SHASTA_ESTATE, "shasta_sweep: call shasta_set_state first");
    const int n[3] = {h->nx, h->ny, h->nz};
    if (n[axis] == 1) return 0;
    if (emit_primitives < 0 || emit_primitives > 2) return fail(h, SHASTA_EINVAL, "shasta_sweep: emit_primitives must be 0, 1 or 2");
    int rc = launch_sweep(h, axis, emit_primitives, (cudaStream_t)stream);
    if (rc) return rc;
    h->prims_valid = emit_primitives == 1;
    return 0;
}

int shasta_get_primitives(shasta_t* h, double* e, double* p, double* n, double* vx, double* vy, double* vz,
                          void* stream)
{
    if (!h) return SHASTA_EINVAL;
    if (!h->have_state) return fail(h, SHASTA_ESTATE, "shasta_get_primitives: no state set");
    cudaStream_t st = (cudaStream_t)stream;
    if (!h->prims_valid && !h->prims_raw) {
        int rc = h->precision == 64 ? refresh_prims_t<double>(h, st) : refresh_prims_t<float>(h, st);
        if (rc) return rc;
    }
    double* dst[6] = {e, p, n, vx, vy, vz};
    for (int q = 0; q < 6; ++q)
        if (dst[q]) {
            int rc = export_field(h, h->prim[q], dst[q], st);
            if (rc) return rc;
        }
    return 0;
}

int shasta_get_primitives_host(shasta_t* h, double* e, double* p, double* n, double* vx, double* vy, double* vz,
                               void* stream)
{
    if (!h) return SHASTA_EINVAL;
    if (!h->have_state) return fail(h, SHASTA_ESTATE, "shasta_get_primitives_host: no state set");
    cudaStream_t st = (cudaStream_t)stream;
    if (!h->prims_valid && !h->prims_raw) {
        int rc = h->precision == 64 ? refresh_prims_t<double>(h, st) : refresh_prims_t<float>(h, st);
        if (rc) return rc;
    }
    double* dst[6] = {e, p, n, vx, vy, vz};
    const size_t nb = sizeof(double) * (size_t)h->ncell;
    for (int q = 0; q < 6; ++q) {
        if (!dst[q]) continue;
        if (h->precision == 64) {
            CK(cudaMemcpyAsync(dst[q], h->prim[q], nb, cudaMemcpyDeviceToHost, st));
        } else {
            int rc = ensure_stage(h);
            if (rc) return rc;
            double* tmp = h->stage + (size_t)q * h->ncell;
            rc = export_field(h, h->prim[q], tmp, st);
            if (rc) return rc;
            CK(cudaMemcpyAsync(dst[q], tmp, nb, cudaMemcpyDeviceToHost, st));
        }
    }
    return 0;
}

int shasta_conserved_totals(shasta_t* h, double* totals, void* stream)
{
    if (!h) return SHASTA_EINVAL;
    if (!totals) return fail(h, SHASTA_EINVAL, "shasta_conserved_totals: NULL output");
    if (!h->have_state) return fail(h, SHASTA_ESTATE, "shasta_conserved_totals: no state set");
    cudaStream_t st = (cudaStream_t)stream;
    void** U = h->U[h->cur];
    const double dv = h->dx * h->dx * h->dx;
    for (int b = 0; b < h->nbatch; ++b) {           // one event at a time (totals are per event)
        const size_t off = (size_t)b * (size_t)h->ncell1;
        if (h->precision == 64)
            totals_kernel<double><<<RED_BLOCKS, RED_THREADS, 0, st>>>(h->ncell1, (double*)U[0] + off, (double*)U[1] + off,
                (double*)U[2] + off, (double*)U[3] + off, (double*)U[4] + off, h->d_partial);
        else
            totals_kernel<float><<<RED_BLOCKS, RED_THREADS, 0, st>>>(h->ncell1, (float*)U[0] + off, (float*)U[1] + off,
                (float*)U[2] + off, (float*)U[3] + off, (float*)U[4] + off, h->d_partial);
        CK(cudaGetLastError());
        h->launches++;
        CK(cudaMemcpyAsync(h->h_partial, h->d_partial, sizeof(double) * RED_BLOCKS * NF * 2, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        for (int f = 0; f < NF; ++f) {
            double s = 0.0, c = 0.0;
            for (int k = 0; k < RED_BLOCKS; ++k) {
                const double x = h->h_partial[(k * NF + f) * 2 + 0];
                const double t = s + x;
                c += h->h_partial[(k * NF + f) * 2 + 1] + ((fabs(s) >= fabs(x)) ? ((s - t) + x) : ((x - t) + s));
                s = t;
            }
            totals[b * NF + f] = dv * (s + c);
        }
    }
    return 0;
}

int shasta_diagnostics(shasta_t* h, unsigned long long* counts)
{
    if (!h) return SHASTA_EINVAL;
    if (!counts) return fail(h, SHASTA_EINVAL, "shasta_diagnostics: NULL output");
    if (!h->allocated) { counts[0] = counts[1] = counts[2] = counts[3] = 0; return 0; }
    CK(cudaDeviceSynchronize());
    CK(cudaMemcpy(counts, h->d_counts, 4 * sizeof(unsigned long long), cudaMemcpyDeviceToHost));
    return 0;
}

long long shasta_launch_count(const shasta_t* h) { return h ? h->launches : -1; }
long long shasta_step_index(const shasta_t* h) { return h ? h->step : -1; }
long long shasta_graph_launch_count(const shasta_t* h) { return h ? h->graph_launches : -1; }

const char* shasta_kernel_name(const shasta_t* h, int axis)
{
    if (!h || axis < 0 || axis > 2) return "";
    if (h->predictor || h->cell_path) return "sweep_cell_kernel";
    // "(cp.async)" marks a sweep that cannot (or may not) use its TMA tiles: no 16 B row strides, extent < 4 cells, no
    // driver entry point, SHASTA_NO_TMA.  Before the first set_state the maps do not exist yet: reported as TMA-capable.
    const int n[3] = {h->nx, h->ny, h->nz};
    const bool have = axis == 0 ? h->have_tmap : (h->have_yzmap && n[axis] >= YZ_CH);
    const bool tma = !h->no_tma && (have || !h->allocated);
    if (axis == 0) return tma ? "sweep_x2_kernel" : "sweep_x2_kernel(cp.async)";
    return tma ? "sweep_yz_kernel" : "sweep_yz_kernel(cp.async)";
}

const char* shasta_last_error(const shasta_t* h) { return h ? h->err : g_create_err; }

}  // extern "C"

// ---------------------------------------------------------------- conserved totals without any allocation
// shasta_conserved_totals_static: the block partial sums of totals_kernel go to a file-scope device array instead of
// the handle's cudaMalloc'ed d_partial, and a second small kernel folds them on the device (the handle path folds
// them on the host through pinned memory, also an allocation).  One block per STATIC_CHUNK cells, so the array's
// size bounds the grid: STATIC_MAX_CELLS.
namespace {

constexpr int STATIC_CHUNK = RED_THREADS * 64;                 // cells one block sums (64 per thread)
constexpr int STATIC_MAX_BLOCKS = 4096;
constexpr long long STATIC_MAX_CELLS = (long long)STATIC_CHUNK * STATIC_MAX_BLOCKS;   // 2^26 = 67 108 864 (406^3)

// 4096 * 5 * 2 doubles = 320 KiB on every GPU that loads the library, until exit.  In host code this name is only a
// stand-in for the symbol: kernels get the address cudaGetSymbolAddress returns (static_partial_ptr below).
static __device__ __align__(256) double g_static_partial[STATIC_MAX_BLOCKS * NF * 2];

constexpr int STATIC_MAX_DEVICES = 64;
double* g_static_ptr[STATIC_MAX_DEVICES] = {};                 // device address of g_static_partial, per device
std::mutex g_static_mutex;

// address of the array on the CURRENT device, looked up once per device
int static_partial_ptr(double** out)
{
    shasta_t* h = nullptr;                                      // CK/fail report to shasta_last_error(NULL)
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= STATIC_MAX_DEVICES)
        return fail(h, SHASTA_EINVAL, "shasta_conserved_totals_static: device %d beyond the %d this build tracks", dev,
                    STATIC_MAX_DEVICES);
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {
        double* p = nullptr;
        CK(cudaGetSymbolAddress((void**)&p, g_static_partial));
        if (!p) return fail(h, SHASTA_ECUDA, "cudaGetSymbolAddress(g_static_partial) returned NULL on device %d", dev);
        g_static_ptr[dev] = p;
    }
    *out = g_static_ptr[dev];
    return 0;
}

// fold `nblocks` (sum, compensation) pairs per field: warp f takes field f; out[f] = dv * total
__global__ void __launch_bounds__(32 * NF) totals_fold_kernel(int nblocks, const double* __restrict__ partial, double dv,
                                                              double* __restrict__ out)
{
    const int f = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double s = 0.0, c = 0.0;
    for (int b = lane; b < nblocks; b += 32) {
        const double x = partial[(b * NF + f) * 2 + 0];
        const double t = s + x;
        c += partial[(b * NF + f) * 2 + 1] + ((fabs(s) >= fabs(x)) ? ((s - t) + x) : ((x - t) + s));
        s = t;
    }
    for (int o = 16; o > 0; o >>= 1) {
        const double so = __shfl_down_sync(0xffffffffu, s, o);
        const double co = __shfl_down_sync(0xffffffffu, c, o);
        const double t = s + so;
        c += co + ((fabs(s) >= fabs(so)) ? ((s - t) + so) : ((so - t) + s));
        s = t;
    }
    if (lane == 0) out[f] = dv * (s + c);
}

}  // namespace

extern "C" {

long long shasta_conserved_totals_static_max_cells(void) { return STATIC_MAX_CELLS; }

int shasta_conserved_totals_static(long long ncell, const double* E_dev, const double* Mx_dev, const double* My_dev,
                                   const double* Mz_dev, const double* R_dev, double dv, double* totals_dev, void* stream)
{
    shasta_t* h = nullptr;
    if (ncell < 0) return fail(h, SHASTA_EINVAL, "shasta_conserved_totals_static: ncell = %lld < 0", ncell);
    if (ncell > STATIC_MAX_CELLS)
        return fail(h, SHASTA_EINVAL,
                    "shasta_conserved_totals_static: ncell = %lld exceeds the %lld cells the static scratch array covers "
                    "(use shasta_conserved_totals of a handle)", ncell, STATIC_MAX_CELLS);
    if (!totals_dev) return fail(h, SHASTA_EINVAL, "shasta_conserved_totals_static: NULL output");
    if (ncell > 0 && (!E_dev || !Mx_dev || !My_dev || !Mz_dev || !R_dev))
        return fail(h, SHASTA_EINVAL, "shasta_conserved_totals_static: NULL field");
    double* partial = nullptr;
    int rc = static_partial_ptr(&partial);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const int nblocks = (int)((ncell + STATIC_CHUNK - 1) / STATIC_CHUNK);
    // every slot [0, nblocks) is written by the first kernel before the second reads it (stream order), and no slot
    // beyond is read: nothing in the array has to start at zero, whatever the previous call left there
    if (nblocks > 0) {
        totals_kernel<double><<<nblocks, RED_THREADS, 0, st>>>(ncell, E_dev, Mx_dev, My_dev, Mz_dev, R_dev, partial);
        CK(cudaGetLastError());
    }
    totals_fold_kernel<<<1, 32 * NF, 0, st>>>(nblocks, partial, dv, totals_dev);
    CK(cudaGetLastError());
    return 0;
}

}  // extern "C"
