// fp64_issue_probe.cu -- measures what DESIGN.md 7.1 and bench.py's alu_roofline rest on: the dependent-issue latency of
// DFMA and the fp64 issue rate of one SM sub-partition on the GPU at hand.  Built and run by
// tests/test_gpu_parity.py::test_fp64_issue_rate_probe (nvcc -gencode arch=compute_100a,code=sm_100a); prints one JSON line.
#include <cstdio>
#include <cuda_runtime.h>

template <int ILP>
__global__ void chain(double* out, long long* cyc, double a, double b, int n)
{
    double x[ILP];
#pragma unroll
    for (int i = 0; i < ILP; ++i) x[i] = a + i + threadIdx.x;
    const long long t0 = clock64();
    for (int it = 0; it < n; ++it) {
#pragma unroll
        for (int i = 0; i < ILP; ++i) x[i] = fma(x[i], b, a);
    }
    const long long t1 = clock64();
    double s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s += x[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0 && blockIdx.x == 0) *cyc = t1 - t0;
}

__global__ void mufu_chain(double* out, long long* cyc, double a, int n)
{
    double x = a + threadIdx.x;
    const long long t0 = clock64();
    for (int it = 0; it < n; ++it) {
        double r;
        asm volatile("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
        x = r + 1.0;
    }
    const long long t1 = clock64();
    out[threadIdx.x] = x;
    if (threadIdx.x == 0) *cyc = t1 - t0;
}

int main()
{
    double* o;
    long long* c;
    if (cudaMalloc(&o, 1 << 20) != cudaSuccess || cudaMalloc(&c, 8) != cudaSuccess) return 1;
    long long h = 0;
    const int n = 8192;
    chain<1><<<1, 32>>>(o, c, 1.0, 0.999, n);
    cudaMemcpy(&h, c, 8, cudaMemcpyDeviceToHost);
    const double lat = (double)h / n;                       // cycles per dependent DFMA, one warp
    chain<4><<<1, 32>>>(o, c, 1.0, 0.999, n);
    cudaMemcpy(&h, c, 8, cudaMemcpyDeviceToHost);
    const double one_warp = (double)h / n / 4;              // cycles per warp-instruction, one warp with 4 chains
    chain<4><<<1, 512>>>(o, c, 1.0, 0.999, n);              // 16 warps = 4 per sub-partition
    cudaMemcpy(&h, c, 8, cudaMemcpyDeviceToHost);
    const double full = (double)h / n / 4 / 4;              // cycles per warp-instruction per sub-partition, pipe saturated
    mufu_chain<<<1, 32>>>(o, c, 1.0, n);
    cudaMemcpy(&h, c, 8, cudaMemcpyDeviceToHost);
    const double mufu = (double)h / n - lat;                // MUFU.RCP64H latency (pair minus the dependent DADD)
    if (cudaDeviceSynchronize() != cudaSuccess) return 2;
    printf("{\"dfma_dependent_latency_cycles\": %.2f, \"cycles_per_warp_dfma_one_warp_ilp4\": %.2f, "
           "\"cycles_per_warp_dfma_saturated\": %.3f, \"fp64_results_per_clk_per_sm\": %.1f, \"mufu_rcp64h_latency_cycles\": %.1f}\n",
           lat, one_warp, full, 4 * 32.0 / full, mufu);
    return 0;
}
