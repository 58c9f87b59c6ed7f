// pipe_rates.cu -- instruction issue rates on sm_100a that the design of the colour pass rests on (DESIGN.md section 8,
// reading C-26, profiles/r01_instruction_throughput.md).  Stand-alone: it shares nothing with the library.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -ftz=true -o pipe_rates pipe_rates.cu && ./pipe_rates
// Every test runs CH independent dependent chains per thread, W warps per SM sub-partition, one CTA per SM, and reports
// cycles per chain step per sub-partition (clock64 of one warp; every warp runs the same loop).
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { fprintf(stderr, "CUDA %s: %s\n", #x, cudaGetErrorString(e_)); return 1; } } while (0)
constexpr int ITER = 2048, CH = 8;

enum Op { FFMA_SCALAR, FFMA_PACKED, FADD_PACKED, FMUL_PACKED, IMAD_LO, IMAD_HI, LOP3_X2, PHILOX_HALF_ROUND, PHILOX_PLUS_FFMA2,
          IMADLO_PLUS_FFMA2, MUFU_RSQ, MUFU_SIN, MUFU_LG2, DADD_F64, I64_ADD };

template <int OP> __global__ void __launch_bounds__(1024) rate_kernel(float* out, float seed, uint32_t useed, long long* cyc)
{
    float2 a[CH]; uint32_t u[CH], v[CH]; float f[CH]; double d[CH]; long long q[CH];
#pragma unroll
    for (int i = 0; i < CH; ++i) {
        a[i] = make_float2(seed + i + threadIdx.x, seed * 0.5f + i); u[i] = useed + i * 77u + threadIdx.x; v[i] = u[i] * 3u;
        f[i] = seed + i * 0.25f + threadIdx.x * 1e-3f; d[i] = (double)f[i]; q[i] = (long long)u[i] << 20;
    }
    const float2 m = make_float2(seed * 0.999f, seed * 0.998f), c = make_float2(seed * 1e-3f, seed * 2e-3f);
    const double dc = (double)seed * 1e-3; const long long qc = (long long)useed << 13;
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < ITER; ++it) {
#pragma unroll
        for (int i = 0; i < CH; ++i) {
            if (OP == FFMA_SCALAR) f[i] = fmaf(f[i], m.x, c.x);
            if (OP == FFMA_PACKED || OP == PHILOX_PLUS_FFMA2 || OP == IMADLO_PLUS_FFMA2) a[i] = __ffma2_rn(a[i], m, c);
            if (OP == FADD_PACKED) a[i] = __fadd2_rn(a[i], c);
            if (OP == FMUL_PACKED) a[i] = __fmul2_rn(a[i], m);
            if (OP == IMAD_LO || OP == IMADLO_PLUS_FFMA2) u[i] = u[i] * 0xD2511F53u;
            if (OP == IMAD_HI) u[i] = __umulhi(u[i], 0xD2511F53u);
            if (OP == LOP3_X2) u[i] = (u[i] ^ useed) & (v[i] | 0x55u);
            if (OP == PHILOX_HALF_ROUND || OP == PHILOX_PLUS_FFMA2) {          // (u,v) <- (hi(M u) ^ v ^ k, lo(M u)): IMAD.WIDE.U32 + LOP3
                const uint64_t p = (uint64_t)0xD2511F53u * u[i];
                u[i] = (uint32_t)(p >> 32) ^ v[i] ^ useed; v[i] = (uint32_t)p;
            }
            if (OP == MUFU_RSQ) f[i] = rsqrtf(f[i]);
            if (OP == MUFU_SIN) f[i] = __sinf(f[i]);
            if (OP == MUFU_LG2) f[i] = __log2f(f[i]);
            if (OP == DADD_F64) d[i] = d[i] + dc;
            if (OP == I64_ADD) q[i] = q[i] + qc;
        }
    }
    const long long t1 = clock64();
    float r = 0;
#pragma unroll
    for (int i = 0; i < CH; ++i) r += a[i].x + a[i].y + (float)u[i] + (float)v[i] + f[i] + (float)d[i] + (float)q[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = r;
    if (threadIdx.x == 0 && blockIdx.x == 0) *cyc = t1 - t0;
}

template <int OP> int run(const char* name, int warps_per_smsp)
{
    float* out; long long* cyc;
    CK(cudaMalloc(&out, 148 * 1024 * 4)); CK(cudaMalloc(&cyc, 8));
    const int threads = 128 * warps_per_smsp;
    for (int r = 0; r < 2; ++r) { rate_kernel<OP><<<148, threads>>>(out, 1.0001f, 12345u, cyc); CK(cudaGetLastError()); CK(cudaDeviceSynchronize()); }
    long long c; CK(cudaMemcpy(&c, cyc, 8, cudaMemcpyDeviceToHost));
    printf("%-46s %d warps/sub-partition: %6.2f cycles per chain step\n", name, warps_per_smsp, (double)c / ((double)ITER * CH * warps_per_smsp));
    cudaFree(out); cudaFree(cyc);
    return 0;
}

int main()
{
    for (int w : { 4, 8 }) {
        run<FFMA_SCALAR>("FFMA", w); run<FFMA_PACKED>("FFMA2 (two fp32 FMAs)", w); run<FADD_PACKED>("FADD2", w); run<FMUL_PACKED>("FMUL2", w);
        run<IMAD_LO>("IMAD (low 32 bits)", w); run<IMAD_HI>("IMAD.HI.U32", w); run<LOP3_X2>("LOP3 x 2", w);
        run<PHILOX_HALF_ROUND>("IMAD.WIDE.U32 + LOP3 (half a Philox round)", w);
        run<PHILOX_PLUS_FFMA2>("IMAD.WIDE.U32 + LOP3 + FFMA2", w); run<IMADLO_PLUS_FFMA2>("IMAD + FFMA2", w);
        run<MUFU_RSQ>("MUFU.RSQ", w); run<MUFU_SIN>("FMUL + MUFU.SIN", w); run<MUFU_LG2>("MUFU.LG2", w);
        run<DADD_F64>("DADD (fp64)", w); run<I64_ADD>("64-bit integer add (IADD3 + IADD3.X)", w);
    }
    return 0;
}
