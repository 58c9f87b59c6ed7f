// mc_noalloc.cu -- mc_profile_x_static(): the slice profile of mc_profile_x (Fig. 2) with its scratch in a fixed array of
// the library image instead of the caller's workspace.  For callers that may not allocate or hand over scratch at call time
// (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): the entry point calls no cudaMalloc,
// no cudaFree and no allocating library routine, and allocates nothing on the host either.
//
// The scratch is ONE file-scope array per device that loads the library (192 KB, held until the process exits).  Every call on a
// device shares it and it keeps the last call's contents, so a call clears it first; two calls that overlap on the same GPU
// (two handles on different streams, two host threads) race on it -- serialise them.
//
// In host code the array's NAME is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress(), resolved once per device with that device current.
#include "mc_host.h"

#include <mutex>

namespace {

constexpr int STATIC_MAX_NX = MC_PROFILE_STATIC_MAX_NX;
// 3 sums per x position: int64 fixed point while the pass accumulates, converted in place to the fp64 means that are copied out
static __device__ __align__(256) long long g_profile_scratch[3 * STATIC_MAX_NX];

constexpr int MAX_DEVICES = 64;
long long* g_scratch_addr[MAX_DEVICES];          // device address of g_profile_scratch on device d (nullptr: not resolved yet)
std::mutex g_scratch_mutex;

// device address of the scratch on the CURRENT device (the caller has made the handle's device current)
cudaError_t scratch_address(int device, long long** out)
{
    if (device < 0 || device >= MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_addr[device]) {
        long long* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_profile_scratch);
        if (e != cudaSuccess) return e;
        g_scratch_addr[device] = p;
    }
    *out = g_scratch_addr[device];
    return cudaSuccess;
}

struct DeviceGuard {
    int prev = -1; bool switched = false;
    explicit DeviceGuard(int dev) { if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess; }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

constexpr int ROWS_PER_THREAD = 32;
constexpr int THREADS = 256;

// Variant of profile_x_kernel (mc_util.cuh): sum over (y, z) of the three spin components at every x, exact fixed point.
// One thread = one colour column xh of a chunk of ROWS_PER_THREAD rows; a colour-c site of row (y, z) sits at
// x = 2 xh + ((y + z + c) & 1).  sums[3 x + a] (int64, unit P.fx_inv) must be zero on entry.
__global__ void __launch_bounds__(THREADS) profile_x_static_kernel(const __grid_constant__ mc::Params P, long long* __restrict__ sums)
{
    const uint32_t R = (uint32_t)P.R, rows = (uint32_t)P.ny * (uint32_t)P.nz;
    const uint32_t n_chunks = (rows + ROWS_PER_THREAD - 1) / ROWS_PER_THREAD;
    const uint32_t t = blockIdx.x * THREADS + threadIdx.x;
    if (t >= R * n_chunks) return;
    const uint32_t chunk = t / R, xh = t - chunk * R;
    float acc[2][3] = { { 0.f, 0.f, 0.f }, { 0.f, 0.f, 0.f } };
    const uint32_t r1 = min(rows, (chunk + 1) * ROWS_PER_THREAD);
    for (uint32_t row = chunk * ROWS_PER_THREAD; row < r1; ++row) {
        const uint32_t y = row % (uint32_t)P.ny, z = row / (uint32_t)P.ny;
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const uint32_t p = (y + z + (uint32_t)c) & 1u;
            const float* S = P.S + (long long)c * 3 * P.plane + (long long)row * R + xh;
#pragma unroll
            for (int a = 0; a < 3; ++a) { const float v = S[(long long)a * P.plane]; acc[0][a] += p ? 0.f : v; acc[1][a] += p ? v : 0.f; }
        }
    }
#pragma unroll
    for (int p = 0; p < 2; ++p)
#pragma unroll
        for (int a = 0; a < 3; ++a)
            atomicAdd(reinterpret_cast<unsigned long long*>(sums + 3 * (2 * xh + p) + a), (unsigned long long)__float2ll_rn(acc[p][a] * P.fx_scale));
}

// int64 sums -> fp64 means, in place (both 8 bytes): the host copies the doubles straight into the caller's buffer
__global__ void profile_x_static_finish(long long* __restrict__ sums, int n, double scale)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double v = (double)sums[i] * scale;
    reinterpret_cast<double*>(sums)[i] = v;
}

}  // namespace

extern "C" int mc_profile_x_static(mc_ctx* ctx, double* host_profile)
{
    if (!ctx) return MC_EINVAL;
    if (ctx->sticky) return ctx->sticky;
    ctx->err[0] = 0;
    DeviceGuard guard_(ctx->device);
    if (!host_profile) return mc::fail(ctx, MC_EINVAL, "mc_profile_x_static: null pointer");
    if (ctx->P.sub) return mc::fail(ctx, MC_EINVAL, "mc_profile_x_static: simple cubic lattices only");
    const int nx = ctx->P.nx;
    if (nx > STATIC_MAX_NX) {
        snprintf(ctx->err, sizeof ctx->err, "mc_profile_x_static: nx = %d exceeds the fixed scratch (MC_PROFILE_STATIC_MAX_NX = %d); use mc_profile_x", nx, STATIC_MAX_NX);
        return MC_EINVAL;
    }
    long long* scratch = nullptr;
    MC_CU(scratch_address(ctx->device, &scratch));
    const size_t bytes = (size_t)nx * 3 * sizeof(long long);
    MC_CU(cudaMemsetAsync(scratch, 0, bytes, ctx->stream));                  // the array keeps the last call's contents
    const uint32_t rows = (uint32_t)ctx->P.ny * (uint32_t)ctx->P.nz;
    const uint32_t n_threads = (uint32_t)ctx->P.R * ((rows + ROWS_PER_THREAD - 1) / ROWS_PER_THREAD);
    profile_x_static_kernel<<<(n_threads + THREADS - 1) / THREADS, THREADS, 0, ctx->stream>>>(ctx->P, scratch);
    MC_CU(cudaGetLastError());
    const double scale = ctx->P.fx_inv / ((double)ctx->P.ny * (double)ctx->P.nz);
    profile_x_static_finish<<<(3 * nx + THREADS - 1) / THREADS, THREADS, 0, ctx->stream>>>(scratch, 3 * nx, scale);
    MC_CU(cudaGetLastError());
    ctx->launches += 2;
    MC_CU(cudaMemcpyAsync(host_profile, scratch, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    MC_CU(cudaStreamSynchronize(ctx->stream));
    return MC_OK;
}
