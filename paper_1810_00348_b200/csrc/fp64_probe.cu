// fp64_probe.cu - dvm_fp64_peak_probe: what the fp64 pipe of THIS board sustains, measured, for the roofline bench.py reports
// ("fp64 is not in MEASURED_PEAKS - measure it first with a register-resident DFMA microbenchmark").
// Every thread keeps 8 independent chains of fused multiply-adds in registers; no memory traffic, full occupancy, all SMs.
// One DFMA = one lane-operation, the unit the sweep kernel's executed fp64 instructions are counted in.
// Product code (measurement aid): no CPU fallback and nothing shared with oracle/.
#include "../../include/dvm.h"
#include <cuda_runtime.h>

namespace dvm {
int report_error(int code, const char *msg);  // dvm_api.cu
}

namespace {

constexpr int PB = 256, CHAINS = 8;

__global__ void __launch_bounds__(PB) dfma_probe_kernel(double *sink, long long rounds, double a, double b)
{
    double x[CHAINS];
#pragma unroll
    for (int k = 0; k < CHAINS; ++k) x[k] = 1e-3 * (threadIdx.x + 1) + k;
    for (long long r = 0; r < rounds; ++r) {
#pragma unroll
        for (int k = 0; k < CHAINS; ++k) x[k] = fma(x[k], a, b);
    }
    double t = 0.0;
#pragma unroll
    for (int k = 0; k < CHAINS; ++k) t += x[k];
    if (t == 1.2345e300) sink[0] = t;  // never true (the chains converge to b / (1 - a)); keeps the arithmetic alive
}

}  // namespace

extern "C" int dvm_fp64_peak_probe(double *dev_sink, long long rounds, double *host_lane_ops_per_s, double *host_ms)
{
    if (!dev_sink || !host_lane_ops_per_s || rounds <= 0) return dvm::report_error(DVM_EINVAL, "dvm_fp64_peak_probe: bad argument");
    int dev = 0, nsm = 0;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    float ms = 0.f;
    const int grid = nsm * (2048 / PB);  // every SM full: 2048 threads
    if (e == cudaSuccess) {
        dfma_probe_kernel<<<grid, PB>>>(dev_sink, 1024, 0.5, 1.0);  // warm-up: module load, clocks
        cudaEventRecord(e0);
        dfma_probe_kernel<<<grid, PB>>>(dev_sink, rounds, 0.5, 1.0);
        cudaEventRecord(e1);
        e = cudaEventSynchronize(e1);
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (e != cudaSuccess) return dvm::report_error(DVM_ECUDA, cudaGetErrorString(e));
    *host_lane_ops_per_s = (double)grid * PB * CHAINS * (double)rounds / (1e-3 * (double)ms);
    if (host_ms) *host_ms = (double)ms;
    return DVM_OK;
}
