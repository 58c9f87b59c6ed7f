// mc_util.cuh -- kernels off the timed path: stand-alone finalize, slice profile (f-1), layout conversion, state edits.
// Non-template __global__ functions: include from exactly one translation unit (mc_api.cu).
#pragma once

#include "mc_common.cuh"

namespace mc {

// Stand-alone pass 2 (for sweeps assembled from the half-sweep test hooks): <<<1, BLOCK>>>
__global__ void __launch_bounds__(BLOCK) finalize_kernel(const __grid_constant__ Params P, int mode, int flags)
{
    final_reduce(P, mode, flags);
}

// --------------------------------------------------------------------------------------------------------------
// Slice profile along x (Fig. 2): sum over (y, z) of the three spin components at every x, in exact fixed point.
// One thread = one colour column xh of a chunk of PROFILE_ROWS rows (coalesced along xh); a colour-c site of row (y,z)
// sits at x = 2 xh + ((y + z + c) & 1), so the thread feeds two x positions.  out[3 x + a] (int64, unit P.fx_inv).
// --------------------------------------------------------------------------------------------------------------
constexpr int PROFILE_ROWS = 32;
__global__ void __launch_bounds__(BLOCK) profile_x_kernel(const __grid_constant__ Params P, long long* __restrict__ out)
{
    const uint32_t R = (uint32_t)P.R, rows = (uint32_t)P.ny * (uint32_t)P.nz;
    const uint32_t n_chunks = (rows + PROFILE_ROWS - 1) / PROFILE_ROWS;
    const uint32_t t = blockIdx.x * BLOCK + threadIdx.x;
    if (t >= R * n_chunks) return;
    const uint32_t chunk = t / R, xh = t - chunk * R;
    float acc[2][3] = { { 0.f, 0.f, 0.f }, { 0.f, 0.f, 0.f } };
    const uint32_t r1 = min(rows, (chunk + 1) * PROFILE_ROWS);
    for (uint32_t row = chunk * PROFILE_ROWS; row < r1; ++row) {
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
            atomicAdd(reinterpret_cast<unsigned long long*>(out + 3 * (2 * xh + p) + a), (unsigned long long)__float2ll_rn(acc[p][a] * P.fx_scale));
}

// --------------------------------------------------------------------------------------------------------------
// Layout conversion and state utilities
// --------------------------------------------------------------------------------------------------------------
// lexicographic [N][3] (x fastest) <-> colour-split planes.  to_split normalises every spin (fp32).
__global__ void lex_to_split_kernel(const __grid_constant__ Params P, const float* __restrict__ lex)
{
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= P.N) return;
    const uint32_t x = s % (uint32_t)P.nx, row = s / (uint32_t)P.nx, y = row % (uint32_t)P.ny, z = row / (uint32_t)P.ny;
    uint32_t c = (x + y + z) & 1u, a = row * (uint32_t)P.R + (x >> 1);
    if (P.sub) { c = s / P.Nc; a = s - c * P.Nc; }        // bcc / fcc / basis: site = sublattice * Ncell + cell
    float vx = lex[3ull * s], vy = lex[3ull * s + 1], vz = lex[3ull * s + 2];
    // a spin that is already unit to fp32 rounding (what mc_get_spins returns) is stored as it is: upload(download(state)) is
    // the identity, so a checkpoint restores bit for bit; anything else is normalised
    const float n2 = vx * vx + vy * vy + vz * vz;
    const bool unit = fabsf(n2 - 1.0f) <= 4.0e-7f;
    const float inv = unit ? 1.0f : ((n2 > 0.0f) ? (float)(1.0 / sqrt((double)n2)) : 0.0f);
    float* Sc = P.S + (long long)c * 3 * P.plane;
    Sc[a] = vx * inv; Sc[P.plane + a] = vy * inv; Sc[2 * P.plane + a] = (n2 > 0.0f) ? vz * inv : 1.0f;
}

__global__ void split_to_lex_kernel(const __grid_constant__ Params P, float* __restrict__ lex)
{
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= P.N) return;
    const uint32_t x = s % (uint32_t)P.nx, row = s / (uint32_t)P.nx, y = row % (uint32_t)P.ny, z = row / (uint32_t)P.ny;
    uint32_t c = (x + y + z) & 1u, a = row * (uint32_t)P.R + (x >> 1);
    if (P.sub) { c = s / P.Nc; a = s - c * P.Nc; }
    const float* Sc = P.S + (long long)c * 3 * P.plane;
    lex[3ull * s] = Sc[a]; lex[3ull * s + 1] = Sc[P.plane + a]; lex[3ull * s + 2] = Sc[2 * P.plane + a];
}

__global__ void fill_kernel(const __grid_constant__ Params P, float vx, float vy, float vz)
{
    const uint32_t a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= P.Nc) return;
    for (int c = 0; c < P.ncol; ++c) {
        float* Sc = P.S + (long long)c * 3 * P.plane;
        Sc[a] = vx; Sc[P.plane + a] = vy; Sc[2 * P.plane + a] = vz;
    }
}

// Random start (BASELINE.json configs[2]: "spins start uniformly random on the sphere (seeded)"): the site with lexicographic
// index i takes (r0,r1,..) = Philox(ctr = (i, TAG_INIT, 0, 0), key = seed), z = 2 u(r0) - 1, phi = 2 pi u(r1).
__global__ void init_random_kernel(const __grid_constant__ Params P)
{
    const uint32_t a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= P.Nc) return;
    const uint32_t R = (uint32_t)P.R, row = a / R, xh = a - row * R, y = row % (uint32_t)P.ny, z = row / (uint32_t)P.ny;
    for (uint32_t c = 0; c < (uint32_t)P.ncol; ++c) {
        const uint32_t site = P.sub ? c * P.Nc + a : row * (uint32_t)P.nx + 2u * xh + ((y + z + c) & 1u);
        uint32_t r0, r1, r2, r3;
        philox4x32_10(P.key, site, TAG_INIT, 0u, 0u, r0, r1, r2, r3);
        const float zz = fmaf(2.0f, uniform01(r0), -1.0f);
        float sp, cp; sincospif(2.0f * uniform01(r1), &sp, &cp);
        const float s = sqrtf(fmaxf(0.0f, fmaf(-zz, zz, 1.0f)));
        float vx = s * cp, vy = s * sp, vz = zz;
        const float n = rsqrtf(fmaf(vx, vx, fmaf(vy, vy, vz * vz)));
        float* Sc = P.S + (long long)c * 3 * P.plane;
        Sc[a] = vx * n; Sc[P.plane + a] = vy * n; Sc[2 * P.plane + a] = vz * n;
    }
}

// rigid rotation S <- Rm S of every spin, renormalised (C-12)
struct Mat3 { float m[9]; };
__global__ void rotate_kernel(const __grid_constant__ Params P, const __grid_constant__ Mat3 Rm)
{
    const uint32_t a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= P.Nc) return;
    for (int c = 0; c < P.ncol; ++c) {
        float* Sc = P.S + (long long)c * 3 * P.plane;
        const float x = Sc[a], y = Sc[P.plane + a], z = Sc[2 * P.plane + a];
        const float rx = Rm.m[0] * x + Rm.m[1] * y + Rm.m[2] * z;
        const float ry = Rm.m[3] * x + Rm.m[4] * y + Rm.m[5] * z;
        const float rz = Rm.m[6] * x + Rm.m[7] * y + Rm.m[8] * z;
        const float inv = rsqrtf(rx * rx + ry * ry + rz * rz);
        Sc[a] = rx * inv; Sc[P.plane + a] = ry * inv; Sc[2 * P.plane + a] = rz * inv;
    }
}

// small state edits on the stream (mc_set_cone / mc_set_sweep / mc_reset_accumulators / e_C / M_L)
enum : int { ST_CONE = 0, ST_SWEEP = 1, ST_RESET_ACC = 2, ST_EC = 3, ST_ML = 4, ST_RESET_SWEEP = 5 };
__global__ void state_kernel(DevState* st, int what, double a, double b, double c, unsigned long long u)
{
    if (what == ST_CONE) { st->cone = a; st->one_minus_cos = one_minus_cos_of(a); }
    else if (what == ST_SWEEP) { st->sweep = u; }
    else if (what == ST_RESET_ACC) {
        st->n_samples = 0ull;
        for (int i = 0; i < 4; ++i) { st->sum_m[i] = 0.0; st->sum_m2[i] = 0.0; }
        st->sum_E = 0.0; st->sum_E2 = 0.0;
        for (int i = 0; i < 3; ++i) st->sum_torque[i] = 0.0;
    }
    else if (what == ST_EC) { st->eC[0] = a; st->eC[1] = b; st->eC[2] = c; }
    else if (what == ST_ML) { st->ML = a; }
    else if (what == ST_RESET_SWEEP) { st->count = 0ull; st->ticket = 0u; for (int q = 0; q < NQ; ++q) st->isum[0][q] = 0; }   // discards a sweep in flight
}


}  // namespace mc
