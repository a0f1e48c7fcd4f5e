// residual_noalloc.cu - dvm_residual_noalloc: the convergence residual of PAPER.md:269 between two macroscopic states,
// for callers that must not allocate device memory.
//
// Who needs this.  The residual is a two-level, fixed-order reduction: every block leaves six partial sums in global
// memory and one block adds them up.  Inside a solver those partial sums live in the workspace that dvm_create obtained
// from the allocator.  Some hosts cannot go through dvm_create just to monitor convergence of fields they already hold:
//   * a program that handed the whole of HBM to its own pool at start-up - cudaMalloc then simply fails;
//   * a time-critical loop - cudaMalloc and cudaFree stall every stream of the device while they run;
//   * code that runs where the CUDA allocator may not be entered at all (inside another library's callback, say).
// For them the partial sums below sit in a fixed array that is part of the loaded library image.  The price: each GPU that
// loads libdvm_b200.so gives up 3 MiB until the process exits, the cell count is capped
// (DVM_RESIDUAL_NOALLOC_MAX_CELLS), and all calls share the one array.
//
// Product code: no CPU fallback and nothing shared with oracle/.
#include "../../include/dvm.h"
#include "dvm_dev.cuh"

#include <cstdarg>
#include <cstdio>
#include <mutex>

namespace dvm {
int report_error(int code, const char *msg);  // dvm_api.cu: leaves msg for dvm_last_error()
}

namespace {

constexpr int RB = 256;                                                     // cells per block, one per thread
constexpr long long MAX_CELLS = DVM_RESIDUAL_NOALLOC_MAX_CELLS;
constexpr int MAX_PARTS = (int)((MAX_CELLS + RB - 1) / RB);                 // 65536 blocks at most
constexpr int NSUM = 6;                                                     // num / den of r_rho, r_mom, r_E

// The scratch: partial sum m of block b at [m * MAX_PARTS + b].  6 x 65536 doubles = 3 MiB per device.
// In HOST code this name is only a handle for cudaGetSymbolAddress - it is not a device address (scratch_on_device below).
static __device__ __align__(256) double g_partials[NSUM * MAX_PARTS];

__device__ __forceinline__ double block_total(double v, double *sh)
{
    v = dvm::warp_sum(v);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) sh[wid] = v;
    __syncthreads();
    double r = 0.0;
    if (wid == 0) {
        r = lane < (RB >> 5) ? sh[lane] : 0.0;
        r = dvm::warp_sum(r);
    }
    return r;  // valid in warp 0
}

// level 1: one cell per thread, six sums per block -> part[m * MAX_PARTS + block].  Solid cells hold zeros in both states
// (dvm_moments / dvm_get_state write them so) and therefore add nothing, as in the solver's own reduction.
__global__ void __launch_bounds__(RB) residual_partials_kernel(const double *__restrict__ p0, const double *__restrict__ p1,
                                                               long long n, double *__restrict__ part)
{
    __shared__ double sh[RB / 32];
    const long long c = (long long)blockIdx.x * RB + threadIdx.x;
    double acc[NSUM] = {0, 0, 0, 0, 0, 0};
    if (c < n) {
        const double r1 = p1[c], ux = p1[n + c], uy = p1[2 * n + c], uz = p1[3 * n + c], T1 = p1[4 * n + c];
        const double r0 = p0[c], vx = p0[n + c], vy = p0[2 * n + c], vz = p0[3 * n + c], T0 = p0[4 * n + c];
        const double dmx = r1 * ux - r0 * vx, dmy = r1 * uy - r0 * vy, dmz = r1 * uz - r0 * vz;
        // rho E = 3/4 rho T + 1/2 rho |u|^2 in the units of dvm.h (reading G2)
        const double E1 = 0.75 * r1 * T1 + 0.5 * r1 * (ux * ux + uy * uy + uz * uz);
        const double E0 = 0.75 * r0 * T0 + 0.5 * r0 * (vx * vx + vy * vy + vz * vz);
        acc[0] = (r1 - r0) * (r1 - r0); acc[1] = r1 * r1;
        acc[2] = dmx * dmx + dmy * dmy + dmz * dmz;
        acc[3] = (r1 * ux) * (r1 * ux) + (r1 * uy) * (r1 * uy) + (r1 * uz) * (r1 * uz);
        acc[4] = (E1 - E0) * (E1 - E0); acc[5] = E1 * E1;
    }
    for (int m = 0; m < NSUM; ++m) {
        const double bs = block_total(acc[m], sh);
        if (threadIdx.x == 0) part[(long long)m * MAX_PARTS + blockIdx.x] = bs;
    }
}

// level 2: one block adds the nparts partials of each sum in a fixed order and writes the three ratios
__global__ void __launch_bounds__(RB) residual_total_kernel(const double *__restrict__ part, int nparts, double *__restrict__ out3)
{
    __shared__ double sh[RB / 32];
    __shared__ double tot[NSUM];
    for (int m = 0; m < NSUM; ++m) {
        double v = 0.0;
        for (int t = threadIdx.x; t < nparts; t += RB) v += part[(long long)m * MAX_PARTS + t];
        const double bs = block_total(v, sh);
        if (threadIdx.x == 0) tot[m] = bs;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int m = 0; m < 3; ++m) {
            const double num = tot[2 * m], den = tot[2 * m + 1];
            double r;
            if (den > 0.0) r = sqrt(num / den);
            else r = num > 0.0 ? __longlong_as_double(0x7ff0000000000000LL) : (num == 0.0 ? 0.0 : num);
            out3[m] = r;
        }
    }
}

int fail(int code, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    return dvm::report_error(code, buf);
}

// Device address of g_partials on device `dev`, which must be the current device.  Looked up once per device: the first
// call on a device is the set-up call (it also makes the driver load this module's code onto that device).
constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
double *g_part_addr[MAX_DEVICES] = {};

int scratch_on_device(int dev, double **out)
{
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_part_addr[dev]) {
        double *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void **)&p, g_partials);
        if (e != cudaSuccess || !p)
            return fail(DVM_ECUDA, "dvm_residual_noalloc: cudaGetSymbolAddress on device %d: %s", dev, cudaGetErrorString(e));
        g_part_addr[dev] = p;
    }
    *out = g_part_addr[dev];
    return DVM_OK;
}

// device that owns a caller's buffer, or -1 if it is not device memory
int owner_of(const void *p)
{
    cudaPointerAttributes a{};
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return -1;
    }
    return (a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged) ? a.device : -1;
}

struct CurrentDevice {  // run on `want`, give the caller's device back afterwards
    int prev = -1, want;
    explicit CurrentDevice(int d) : want(d)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        if (prev != want) cudaSetDevice(want);
    }
    ~CurrentDevice()
    {
        if (prev >= 0 && prev != want) cudaSetDevice(prev);
    }
};

}  // namespace

extern "C" int dvm_residual_noalloc(const double *dev_prim_old, const double *dev_prim_new, long long ncell, double *dev_out3,
                                    void *stream)
{
    if (!dev_prim_old || !dev_prim_new || !dev_out3) return fail(DVM_EINVAL, "dvm_residual_noalloc: NULL argument");
    if (ncell <= 0) return fail(DVM_EINVAL, "dvm_residual_noalloc: ncell = %lld, must be positive", ncell);
    if (ncell > MAX_CELLS)
        return fail(DVM_EINVAL,
                    "dvm_residual_noalloc: ncell = %lld is beyond the fixed scratch array, which holds the partial sums of at most "
                    "%lld cells (DVM_RESIDUAL_NOALLOC_MAX_CELLS); use a solver's dvm_residual for larger grids",
                    ncell, MAX_CELLS);
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0) {
        cudaGetLastError();
        return fail(DVM_ECUDA, "dvm_residual_noalloc: no CUDA device (there is no CPU fallback)");
    }
    const int dev = owner_of(dev_out3);
    if (dev < 0 || owner_of(dev_prim_old) != dev || owner_of(dev_prim_new) != dev)
        return fail(DVM_EINVAL, "dvm_residual_noalloc: the three buffers must be device memory of one and the same GPU");
    if (dev >= MAX_DEVICES) return fail(DVM_EINVAL, "dvm_residual_noalloc: device ordinal %d not supported (max %d)", dev, MAX_DEVICES - 1);

    CurrentDevice guard(dev);
    double *part = nullptr;
    if (const int rc = scratch_on_device(dev, &part)) return rc;
    // Nothing in the array has to start at zero: level 2 reads slots [0, nparts) of each sum only, and level 1 of this same
    // call has written every one of them.  Slots beyond nparts keep whatever an earlier, larger call left there.
    const int nparts = (int)((ncell + RB - 1) / RB);
    cudaStream_t st = (cudaStream_t)stream;
    residual_partials_kernel<<<nparts, RB, 0, st>>>(dev_prim_old, dev_prim_new, ncell, part);
    residual_total_kernel<<<1, RB, 0, st>>>(part, nparts, dev_out3);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(DVM_ECUDA, "dvm_residual_noalloc: kernel launch: %s", cudaGetErrorString(e));
    return DVM_OK;
}
