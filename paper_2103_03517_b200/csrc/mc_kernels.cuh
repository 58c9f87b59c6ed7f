// mc_kernels.cuh -- sm_100a kernels of the checkerboard Metropolis path: colour pass (Table A1), constrained pair
// pass (Table A2), fused per-sweep reductions + cone controller, standalone measurement, layout conversion.
//
// Data layout in HBM: colour-split SoA fp32 planes.  For colour c and component k the plane
// S[(3c + k) * plane .. ] holds the sites of colour c in colour-linear order a = (x>>1) + R (y + ny z), R = nx/2.
// With row parity p = (y+z+c)&1 the site is x = 2 (a mod R) + p, and its six neighbours live in the OTHER colour at
//   +-y, +-z : the same a-offset inside the neighbouring row
//   +-x      : xh and xh + (p ? +1 : -1) of the same row  (p=0: +x is xh, -x is xh-1;  p=1: -x is xh, +x is xh+1)
// so one colour pass streams its own colour once (read + write) and the other colour once (read).
#pragma once

#include "mc_device.cuh"

namespace mc {

constexpr int NQ = 9;          // fused sums: Mx My Mz E_exch E_aniso E_zeeman tq_x tq_y tq_z (extensive, fp64)
constexpr int BLOCK = 256;     // threads per CTA of the generic pass kernels
constexpr int MAX_WARPS = 32;  // largest CTA any kernel that reduces uses (1024 threads); block sizes are warp multiples
constexpr int TRACE_CAP = 16384;
constexpr int FLUSH_ITEMS = 8;  // items a thread sums in fp32 before the sums go to 64-bit fixed point

// Controller / reduction state, resident in the workspace (no host round trip per sweep: P:165-171 runs on the device)
struct DevState {
    unsigned long long sweep;        // completed Monte Carlo iterations = Philox counter words 2,3
    double cone;                     // cone half-angle theta (rad)
    float one_minus_cos;             // 1 - cos(theta), what the move kernel needs
    int adaptive;
    unsigned long long count;        // accepted moves of the sweep in flight (integer atomics: order independent)
    unsigned int ticket;             // last-block election
    unsigned int pad4_[4];
    unsigned int pad_;
    double last_acceptance;
    double sums[NQ];                 // fused sums of the last completed sweep
    double meas[NQ];                 // sums written by the standalone measurement
    double ML;                       // M_L = sum_i S_i.e_C of the state; refreshed by finalize and measure
    double eC[3];
    unsigned long long n_samples;
    double sum_m[4], sum_m2[4], sum_E, sum_E2, sum_torque[3];
    unsigned long long trace_rows;   // rows ever written to the trace ring
    long long isum[2][NQ];           // exact fixed-point sums in flight: [0] the sweep (both colour passes), [1] the measurement
};

struct Params {
    int nx, ny, nz, R;               // R = nx/2 sites of one colour per row
    int anti_x;                      // 1: anti-periodic boundary along x (domain-wall box); the wrap bond sees -S_j
    uint32_t Nc;                     // sites per colour
    uint32_t N;
    double invN;                     // 1 / N (host-computed: keeps an fp64 division off the finalising thread)
    long long plane;                 // floats between component planes
    float* S;                        // 6 planes: colour-major, then component
    const uint8_t* mask;   long long mask_plane;     // [2][mask_plane] colour-split bond masks (or null)
    const uint16_t* region; long long region_plane;  // [2][region_plane] colour-split grain ids (or null)
    const float4* axis;              // [n_regions] easy axes
    float J, Ku, Kc;
    float eu[3], B[3];
    uint32_t seed_lo, seed_hi;
    PhiloxKey key;                   // the 10 round keys of (seed_lo, seed_hi), filled by the host: constant-bank operands
    DevState* st;
    float fx_scale;                  // 2^k: fixed-point unit of the fused sums is 2^-k (k chosen by the host so that N * 8 * 2^k < 2^62)
    double fx_inv;                   // 2^-k
    int max_blocks;
    double* trace;                   // [TRACE_CAP][6]
};

struct Geom {                        // per-VEC decomposition of the colour-linear index space into items of VEC sites
    uint32_t n_items, RV;            // RV = items per row
    FastDiv div_rv, div_nz;
    uint32_t yb_shift;               // rows are visited in blocks of 2^yb_shift rows, z fastest between blocks (see locate)
};

enum : int { F_FINALIZE = 1, F_TORQUE = 2, F_SAMPLE_TORQUE = 4 };
enum : int { MODE_SWEEP = 0, MODE_MEASURE = 1 };

// --------------------------------------------------------------------------------------------------------------
template <int VEC> struct Pack { float v[VEC]; };

template <int VEC> __device__ __forceinline__ Pack<VEC> ld_nc(const float* p);
template <> __device__ __forceinline__ Pack<1> ld_nc<1>(const float* p) { Pack<1> r; r.v[0] = __ldg(p); return r; }
template <> __device__ __forceinline__ Pack<4> ld_nc<4>(const float* p)
{
    const float4 t = __ldg(reinterpret_cast<const float4*>(p));
    Pack<4> r; r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w; return r;
}
template <int VEC> __device__ __forceinline__ Pack<VEC> ld_rw(const float* p);
template <> __device__ __forceinline__ Pack<1> ld_rw<1>(const float* p) { Pack<1> r; r.v[0] = *p; return r; }
template <> __device__ __forceinline__ Pack<4> ld_rw<4>(const float* p)
{
    const float4 t = *reinterpret_cast<const float4*>(p);
    Pack<4> r; r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w; return r;
}
template <int VEC> __device__ __forceinline__ void st_rw(float* p, const Pack<VEC>& r);
template <> __device__ __forceinline__ void st_rw<1>(float* p, const Pack<1>& r) { *p = r.v[0]; }
template <> __device__ __forceinline__ void st_rw<4>(float* p, const Pack<4>& r)
{
    *reinterpret_cast<float4*>(p) = make_float4(r.v[0], r.v[1], r.v[2], r.v[3]);
}

// One item = VEC consecutive same-colour sites of one row.  Coordinates + neighbour offsets.
struct ItemPos {
    uint32_t a0;        // colour-linear index of the first site
    uint32_t site0;     // lexicographic index of the first site (next ones are +2)
    uint32_t par;       // (y + z + colour) & 1
    uint32_t o_yp, o_ym, o_zp, o_zm;   // colour-linear index of the same column in the 4 neighbouring rows
    uint32_t o_x;       // colour-linear index of the one extra x-neighbour outside the item's own column range
    uint32_t xh0;       // in-row colour index of the first site (x = 2 xh0 + par)
    float xs;           // -1 if the bond to the extra x-neighbour crosses an anti-periodic x wrap, else +1
};

template <int VEC>
__device__ __forceinline__ ItemPos locate(const Params& P, const Geom& G, uint32_t item, int colour)
{
    // Visiting order of the rows (which thread takes which site; the result does not depend on it): blocks of 2^yb_shift
    // consecutive y-rows, all nz planes of a block before the next block.  The grid-stride window of a pass then holds a
    // site's +-z neighbours together with it, so every other-colour value comes from HBM once; in plain (y, then z) order
    // a thin film (c5: a z-plane is 25 MB per colour) re-read them up to three times.
    uint32_t rowp, xq, t, yb, y, z;
    G.div_rv.divmod(item, rowp, xq);
    t = rowp >> G.yb_shift;
    G.div_nz.divmod(t, yb, z);
    y = (yb << G.yb_shift) + (rowp & ((1u << G.yb_shift) - 1u));
    const uint32_t R = (uint32_t)P.R, ny = (uint32_t)P.ny, nz = (uint32_t)P.nz;
    const uint32_t row = y + ny * z;
    ItemPos q;
    const uint32_t xh0 = xq * VEC;
    q.par = (y + z + (uint32_t)colour) & 1u;
    q.xh0 = xh0;
    q.a0 = row * R + xh0;
    q.site0 = row * (uint32_t)P.nx + 2u * xh0 + q.par;
    const uint32_t yp = (y + 1 == ny) ? 0u : y + 1, ym = (y == 0) ? ny - 1 : y - 1;
    const uint32_t zp = (z + 1 == nz) ? 0u : z + 1, zm = (z == 0) ? nz - 1 : z - 1;
    q.o_yp = (z * ny + yp) * R + xh0;  q.o_ym = (z * ny + ym) * R + xh0;
    q.o_zp = (zp * ny + y) * R + xh0;  q.o_zm = (zm * ny + y) * R + xh0;
    const bool wraps = q.par ? (xh0 + VEC == R) : (xh0 == 0);      // only the item's outermost x-bond can cross the wrap
    const uint32_t xe = q.par ? (wraps ? 0u : xh0 + VEC) : (wraps ? R - 1 : xh0 - 1);
    q.o_x = row * R + xe;
    q.xs = (wraps && P.anti_x) ? -1.0f : 1.0f;
    return q;
}

// Exchange field h = sum_j J_ij S_j of the VEC sites of an item (first term of Eq. 2), WITHOUT the factor J.
// MASKED: bond k of a site contributes only if bit k of its mask is set (grain boundaries P:118, open faces P:116).
template <int VEC, bool MASKED>
__device__ __forceinline__ void exchange_field(const Params& P, const ItemPos& q, int colour, Vec3 (&h)[VEC])
{
    const float* O = P.S + (long long)(1 - colour) * 3 * P.plane;
    uint32_t mbits[VEC];
    if (MASKED) {
        const uint8_t* m = P.mask + (long long)colour * P.mask_plane + q.a0;
        if (VEC == 4) {
            const uint32_t w = __ldg(reinterpret_cast<const uint32_t*>(m));
#pragma unroll
            for (int k = 0; k < VEC; ++k) mbits[k] = (w >> (8 * k)) & 0xFFu;
        } else {
#pragma unroll
            for (int k = 0; k < VEC; ++k) mbits[k] = __ldg(m + k);
        }
    }
    float hc[3][VEC];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float* Oc = O + (long long)c * P.plane;
        const Pack<VEC> o  = ld_nc<VEC>(Oc + q.a0);
        const Pack<VEC> yp = ld_nc<VEC>(Oc + q.o_yp), ym = ld_nc<VEC>(Oc + q.o_ym);
        const Pack<VEC> zp = ld_nc<VEC>(Oc + q.o_zp), zm = ld_nc<VEC>(Oc + q.o_zm);
        const float ex = q.xs * __ldg(Oc + q.o_x);               // the spin across an anti-periodic wrap enters as -S_j
#pragma unroll
        for (int k = 0; k < VEC; ++k) {
            // the second x-neighbour: next column if par = 1, previous column if par = 0
            const float sh = q.par ? ((k + 1 < VEC) ? o.v[(k + 1) % VEC] : ex) : ((k > 0) ? o.v[(k + VEC - 1) % VEC] : ex);
            if (MASKED && VEC != 4) {
                const uint32_t mb = mbits[k];
                // o.v[k] is the +x neighbour when par = 0 and the -x neighbour when par = 1
                const uint32_t bit_o = q.par ? 2u : 1u, bit_s = q.par ? 1u : 2u;
                float s = 0.0f;
                s += (mb & bit_o) ? o.v[k] : 0.0f;
                s += (mb & bit_s) ? sh : 0.0f;
                s += (mb & 4u)  ? yp.v[k] : 0.0f;
                s += (mb & 8u)  ? ym.v[k] : 0.0f;
                s += (mb & 16u) ? zp.v[k] : 0.0f;
                s += (mb & 32u) ? zm.v[k] : 0.0f;
                hc[c][k] = s;
            } else if (VEC != 4) {
                hc[c][k] = ((o.v[k] + sh) + (yp.v[k] + ym.v[k])) + (zp.v[k] + zm.v[k]);
            }
        }
        if (VEC == 4) {
            // the same sums two lanes at a time (the float4 loads are already aligned register pairs); a masked bond is a
            // factor 0 or 1 in an FFMA2 (same value and rounding as adding the neighbour or adding 0)
            const float s0 = q.par ? o.v[1] : ex, s1 = q.par ? o.v[2] : o.v[0], s2 = q.par ? o.v[3] : o.v[1], s3 = q.par ? ex : o.v[2];
#pragma unroll
            for (int h2 = 0; h2 < 2; ++h2) {
                const int a = 2 * h2, b = 2 * h2 + 1;
                const f2 sh2 = h2 ? make_float2(s2, s3) : make_float2(s0, s1);
                f2 r;
                if (MASKED) {
                    const uint32_t bo = q.par ? 1u : 0u, bs = q.par ? 0u : 1u;      // bit index of o's bond / sh's bond
                    auto mf = [&](uint32_t bit) { return make_float2((mbits[a] & (1u << bit)) ? 1.0f : 0.0f, (mbits[b] & (1u << bit)) ? 1.0f : 0.0f); };
                    r = mul2(mf(bo), make_float2(o.v[a], o.v[b]));
                    r = fma2(mf(bs), sh2, r);
                    r = fma2(mf(2u), make_float2(yp.v[a], yp.v[b]), r);
                    r = fma2(mf(3u), make_float2(ym.v[a], ym.v[b]), r);
                    r = fma2(mf(4u), make_float2(zp.v[a], zp.v[b]), r);
                    r = fma2(mf(5u), make_float2(zm.v[a], zm.v[b]), r);
                } else {
                    r = add2(add2(add2(make_float2(o.v[a], o.v[b]), sh2), add2(make_float2(yp.v[a], yp.v[b]), make_float2(ym.v[a], ym.v[b]))),
                             add2(make_float2(zp.v[a], zp.v[b]), make_float2(zm.v[a], zm.v[b])));
                }
                hc[c][a] = r.x; hc[c][b] = r.y;
            }
        }
    }
#pragma unroll
    for (int k = 0; k < VEC; ++k) h[k] = { hc[0][k], hc[1][k], hc[2][k] };
}

// easy axes of the VEC sites of an item: uniform, or per grain through the region table (config c5)
template <int VEC>
__device__ __forceinline__ void easy_axes(const Params& P, const ItemPos& q, int colour, Vec3 (&e)[VEC])
{
    if (P.region) {
        const uint16_t* r = P.region + (long long)colour * P.region_plane + q.a0;
#pragma unroll
        for (int k = 0; k < VEC; ++k) { const float4 a = __ldg(P.axis + __ldg(r + k)); e[k] = { a.x, a.y, a.z }; }
    } else {
#pragma unroll
        for (int k = 0; k < VEC; ++k) e[k] = { P.eu[0], P.eu[1], P.eu[2] };
    }
}

// --------------------------------------------------------------------------------------------------------------
// Fused sums (a-9), pass 1.  A thread carries fp32 partial sums over a small bounded set of sites, converts them ONCE to
// 64-bit fixed point (unit 2^-k) and from there on every addition is an integer addition: exact, hence independent of
// the order (warp shuffles, warps of a block, one 64-bit atomic per block and quantity) and bitwise reproducible.
// fp64 enters in pass 2 only (final_reduce).  Why not fp64 block partials re-read by the last block: their order had to
// be fixed to be reproducible, so they went through an array in HBM that the finalising block re-read behind a chain of
// dependent loads -- 7 us alone on the GPU at the tail of every black pass (224^3).  Exact sums need no order, so one
// atomic per block and quantity replaces the array and the tail is 2.5 us.
// --------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void fx_flush(long long (&acc)[NQ], float (&f)[NQ], float scale)
{
#pragma unroll
    for (int q = 0; q < NQ; ++q) { acc[q] += __float2ll_rn(f[q] * scale); f[q] = 0.0f; }
}

// The generic kernels keep the fixed-point sums of a thread in shared memory (column threadIdx.x of [NQ][BLOCK]: no bank
// conflicts) instead of 18 registers: they are short of registers (spills), and the sums are touched once per
// FLUSH_ITEMS items.
__device__ __forceinline__ void fx_flush_shared(long long (*sacc)[BLOCK], float (&f)[NQ], float scale)
{
#pragma unroll
    for (int q = 0; q < NQ; ++q) { sacc[q][threadIdx.x] += __float2ll_rn(f[q] * scale); f[q] = 0.0f; }
}

__device__ __forceinline__ long long warp_sum_i64(long long v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// mode 0: sums of a sweep in flight; mode 1: standalone measurement
__device__ __forceinline__ void block_reduce(const long long (&acc)[NQ], int cnt, const Params& P, int mode)
{
    __shared__ long long sm[MAX_WARPS][NQ];
    __shared__ int scnt;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = (int)(blockDim.x >> 5);
    if (threadIdx.x == 0) scnt = 0;
    __syncthreads();
    const int wc = __reduce_add_sync(0xffffffffu, cnt);
    if (lane == 0 && wc) atomicAdd(&scnt, wc);
#pragma unroll
    for (int q = 0; q < NQ; ++q) { const long long v = warp_sum_i64(acc[q]); if (lane == 0) sm[warp][q] = v; }
    __syncthreads();
    if (threadIdx.x < NQ) {
        long long v = 0;
        for (int w = 0; w < nwarps; ++w) v += sm[w][threadIdx.x];
        if (v) atomicAdd(reinterpret_cast<unsigned long long*>(&P.st->isum[mode][threadIdx.x]), (unsigned long long)v);
    }
    if (threadIdx.x == 0 && scnt) atomicAdd(&P.st->count, (unsigned long long)scnt);
}

// Pass 2 of the reduction (one block, fixed order) + what follows a sweep: cone controller (P:168-171 read with
// P:205-209; C-2, C-3, C-9), sweep counter, Eq. (6) accumulators, trace row.  mode 0: end of a sweep; 1: measurement.
// Pass 1 left exact fixed-point totals in DevState.isum; here they become fp64.  This block runs alone at the tail of
// the black pass, so its latency is exposed: the controller state is staged through shared memory with one coalesced
// read and one coalesced write (two L2 round trips instead of a chain of dependent ones), thread 0 does the scalar
// work on the shared copy.
static_assert(sizeof(DevState) % 4 == 0, "DevState is staged as 32-bit words");
__device__ void final_reduce(const Params& P, int mode, int flags)
{
    __shared__ double cone_next[2];
    __shared__ float omc_next[2];
    __shared__ DevState sst;
    DevState* st = P.st;
    constexpr int NWORDS = (int)(sizeof(DevState) / 4);
    for (int i = threadIdx.x; i < NWORDS; i += blockDim.x)
        reinterpret_cast<uint32_t*>(&sst)[i] = __ldcg(reinterpret_cast<const uint32_t*>(st) + i);
    __syncthreads();
    // one thread evaluates both possible next cone angles while thread 0 does the rest
    const int cone_thread = blockDim.x > 32 ? 32 : 1;
    if ((int)threadIdx.x == cone_thread && mode == 0) {
        const double deg = 3.14159265358979323846 / 180.0, pi = 3.14159265358979323846;
        double up = sst.cone + deg; if (up > pi) up = pi;
        double dn = sst.cone - deg; if (dn < deg) dn = deg;
        cone_next[0] = up; cone_next[1] = dn;
        omc_next[0] = (float)(1.0 - cos(up)); omc_next[1] = (float)(1.0 - cos(dn));
    }
    double s[NQ];
    if (threadIdx.x == 0) {
        for (int q = 0; q < NQ; ++q) { s[q] = (double)sst.isum[mode][q] * P.fx_inv; sst.isum[mode][q] = 0; }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        DevState& S = sst;
        S.ML = s[0] * S.eC[0] + s[1] * S.eC[1] + s[2] * S.eC[2];
        if (mode == 1) {
            for (int q = 0; q < NQ; ++q) S.meas[q] = s[q];
        } else {
            const double invN = P.invN;
            const unsigned long long cnt = S.count;
            const double cone_used = S.cone;
            S.last_acceptance = (double)cnt * invN;
            if (S.adaptive) {
                const int k = (2ull * cnt > (unsigned long long)P.N) ? 0 : 1;     // C-9: equality decreases
                S.cone = cone_next[k];
                S.one_minus_cos = omc_next[k];
            }
            S.count = 0ull;
            S.sweep += 1ull;
            for (int q = 0; q < NQ; ++q) S.sums[q] = s[q];
            const double mx = s[0] * invN, my = s[1] * invN, mz = s[2] * invN;
            const double ml = sqrt(mx * mx + my * my + mz * mz);
            const double E = (s[3] + s[4] + s[5]) * invN;
            const double mv[4] = { ml, mx, my, mz };
            for (int a = 0; a < 4; ++a) { S.sum_m[a] += mv[a]; S.sum_m2[a] += mv[a] * mv[a]; }
            S.sum_E += E; S.sum_E2 += E * E;
            if (flags & F_SAMPLE_TORQUE) for (int a = 0; a < 3; ++a) S.sum_torque[a] += s[6 + a] * invN;
            S.n_samples += 1ull;
            double* row = P.trace + (S.trace_rows % (unsigned long long)TRACE_CAP) * 6;
            row[0] = S.last_acceptance; row[1] = cone_used; row[2] = mx; row[3] = my; row[4] = mz; row[5] = E;
            S.trace_rows += 1ull;
        }
        S.ticket = 0u;
    }
    __syncthreads();
    for (int i = threadIdx.x; i < NWORDS; i += blockDim.x)
        reinterpret_cast<uint32_t*>(st)[i] = reinterpret_cast<const uint32_t*>(&sst)[i];
}

// Last-block election: returns true in every thread of the block that arrives last.
__device__ __forceinline__ bool last_block_done(DevState* st)
{
    __shared__ bool is_last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) is_last = (atomicAdd(&st->ticket, 1u) == gridDim.x - 1);
    __syncthreads();
    if (is_last) __threadfence();
    return is_last;
}

// --------------------------------------------------------------------------------------------------------------
// Colour pass of Table A1: one item of VEC sites per loop trip, grid-stride.
//   MODE_SWEEP  : propose (a-4), dE (a-5), accept/write (a-6), count (a-7), fused sums of the FINAL spins (a-9).
//   MODE_MEASURE: no move; sums of the current spins (standalone measurement).
// E_exch is accumulated by the BLACK pass only: every bond joins a red and a black site, so
// E_exch = -sum_{i black} S_i.h_i with h already in registers (0 extra bytes).
// --------------------------------------------------------------------------------------------------------------
#ifndef MC_PASS_MIN_BLOCKS
#define MC_PASS_MIN_BLOCKS 3      // <= 80 registers: three CTAs per SM (c5 film: one 354, two 185, three 166 us per sweep)
#endif
template <int VEC, int ANISO, bool MASKED, int MODE>
__global__ void __launch_bounds__(BLOCK, MC_PASS_MIN_BLOCKS)
pass_kernel(const __grid_constant__ Params P, const __grid_constant__ Geom G, int colour, float invT, int flags,
            float* __restrict__ dbg_x, uint8_t* __restrict__ dbg_acc)
{
    DevState* st = P.st;
    grid_dependency_sync();
    const unsigned long long sweep = st->sweep;
    const float omc = st->one_minus_cos;
    const PhiloxKey& key = P.key;
    const uint32_t c1 = TAG_MOVE | ((uint32_t)colour << 8), c2 = (uint32_t)sweep, c3 = (uint32_t)(sweep >> 32);
    float* Sc = P.S + (long long)colour * 3 * P.plane;
    const Vec3 B = { P.B[0], P.B[1], P.B[2] };

    __shared__ long long sacc[NQ][BLOCK];   // exact fixed-point sums of every thread of the block (fx_flush_shared)
    float fs[NQ];                    // fp32 running sums of at most FLUSH_ITEMS items
#pragma unroll
    for (int q = 0; q < NQ; ++q) { sacc[q][threadIdx.x] = 0; fs[q] = 0.0f; }
    int cnt = 0, pending = 0;

    const uint32_t stride = gridDim.x * BLOCK;
    for (uint32_t item = blockIdx.x * BLOCK + threadIdx.x; item < G.n_items; item += stride) {
        const ItemPos q = locate<VEC>(P, G, item, colour);
        const Pack<VEC> sx = ld_rw<VEC>(Sc + q.a0), sy = ld_rw<VEC>(Sc + P.plane + q.a0), sz = ld_rw<VEC>(Sc + 2 * P.plane + q.a0);
        Vec3 h[VEC], e[VEC];
        exchange_field<VEC, MASKED>(P, q, colour, h);
        if (ANISO & 1) easy_axes<VEC>(P, q, colour, e);
        Pack<VEC> nxv = sx, nyv = sy, nzv = sz;
        float f[NQ];
#pragma unroll
        for (int k = 0; k < NQ; ++k) f[k] = 0.0f;
        // random words: one Philox4x32-10 block per pair of x-neighbours (x, x ^ 2) of this colour, two words per site (C-26)
        uint32_t w0[VEC], w1[VEC];
        if (MODE == MODE_SWEEP) {
            if (VEC == 1) {
                const uint32_t half = q.xh0 & 1u;
                uint32_t r0, r1, r2, r3;
                philox4x32_10(key, q.site0 - 2u * half, c1, c2, c3, r0, r1, r2, r3);
                w0[0] = half ? r2 : r0; w1[0] = half ? r3 : r1;
            } else {
#pragma unroll
                for (int k = 0; k + 1 < VEC; k += 2) philox4x32_10(key, q.site0 + 2u * k, c1, c2, c3, w0[k], w1[k], w0[k + 1], w1[k + 1]);
            }
        }
        if (VEC == 4 && MODE == MODE_SWEEP) {
            // ---- two sites at a time in the lanes of FFMA2 / FADD2 / FMUL2 (lane by lane the arithmetic of the scalar loop below)
            const V3p B2 = splat3(B);
            f2 f2s[6];
#pragma unroll
            for (int qq = 0; qq < 6; ++qq) f2s[qq] = splat(0.0f);
#pragma unroll
            for (int kp = 0; kp < 4; kp += 2) {
                V3p S = { make_float2(sx.v[kp], sx.v[kp + 1]), make_float2(sy.v[kp], sy.v[kp + 1]), make_float2(sz.v[kp], sz.v[kp + 1]) };
                const V3p hp = pack3(h[kp], h[kp + 1]);
                const f2 J2 = splat(P.J);
                const V3p hJ = { mul2(J2, hp.x), mul2(J2, hp.y), mul2(J2, hp.z) };
                const V3p ep = (ANISO & 1) ? pack3(e[kp], e[kp + 1]) : B2;
                V3p d, Sn;
                cone_move2(S, omc, make_float2(uniform01(w0[kp]), uniform01(w0[kp + 1])),
                           make_float2(uniform_azimuth(w0[kp], w1[kp]), uniform_azimuth(w0[kp + 1], w1[kp + 1])), d, Sn);
                const V3p hB = { add2(hJ.x, B2.x), add2(hJ.y, B2.y), add2(hJ.z, B2.z) };
                f2 s4S, s4v, euS, euv;
                const f2 dE = delta_energy2_keep<ANISO>(S, d, hB, P.Ku, ep, P.Kc, s4S, s4v, euS, euv);
                const f2 xx = fma2(dE, splat(invT), make_float2(__logf(uniform01(w1[kp])), __logf(uniform01(w1[kp + 1]))));   // P:157-158 in log form (C-8)
                const bool ok0 = xx.x < 0.0f, ok1 = xx.y < 0.0f;
                S.x = make_float2(ok0 ? Sn.x.x : S.x.x, ok1 ? Sn.x.y : S.x.y);
                S.y = make_float2(ok0 ? Sn.y.x : S.y.x, ok1 ? Sn.y.y : S.y.y);
                S.z = make_float2(ok0 ? Sn.z.x : S.z.x, ok1 ? Sn.z.y : S.z.y);
                nxv.v[kp] = S.x.x; nxv.v[kp + 1] = S.x.y; nyv.v[kp] = S.y.x; nyv.v[kp + 1] = S.y.y; nzv.v[kp] = S.z.x; nzv.v[kp + 1] = S.z.y;
                cnt += (int)ok0 + (int)ok1;
                if (dbg_x)   { dbg_x[q.site0 + 2u * kp] = xx.x; dbg_x[q.site0 + 2u * kp + 2u] = xx.y; }
                if (dbg_acc) { dbg_acc[q.site0 + 2u * kp] = (uint8_t)ok0; dbg_acc[q.site0 + 2u * kp + 2u] = (uint8_t)ok1; }
                f2s[0] = add2(f2s[0], S.x); f2s[1] = add2(f2s[1], S.y); f2s[2] = add2(f2s[2], S.z);
                if (colour == 1) f2s[3] = sub2(f2s[3], dot3p(S, hJ));
                if (ANISO) f2s[4] = add2(f2s[4], onsite_from<ANISO>(ok0, ok1, s4S, s4v, euS, euv, P.Ku, P.Kc));
                f2s[5] = sub2(f2s[5], dot3p(S, B2));
            }
#pragma unroll
            for (int qq = 0; qq < 6; ++qq) f[qq] += f2s[qq].x + f2s[qq].y;
        }
#pragma unroll
        for (int k = 0; k < ((VEC == 4 && MODE == MODE_SWEEP) ? 0 : VEC); ++k) {
            Vec3 S = { sx.v[k], sy.v[k], sz.v[k] };
            const Vec3 hJ = { P.J * h[k].x, P.J * h[k].y, P.J * h[k].z };
            if (MODE == MODE_SWEEP) {
                Vec3 d, Sn;
                cone_move(S, omc, uniform01(w0[k]), uniform_azimuth(w0[k], w1[k]), d, Sn);
                const Vec3 hB = { hJ.x + B.x, hJ.y + B.y, hJ.z + B.z };
                const float dE = delta_energy<ANISO>(S, d, hB, P.Ku, e[(ANISO & 1) ? k : 0], P.Kc);
                const float x = fmaf(dE, invT, __logf(uniform01(w1[k])));    // P:157-158 in log form (C-8)
                const bool ok = x < 0.0f;
                if (ok) { S = Sn; nxv.v[k] = Sn.x; nyv.v[k] = Sn.y; nzv.v[k] = Sn.z; }
                cnt += ok;
                if (dbg_x)   dbg_x[q.site0 + 2u * k] = x;
                if (dbg_acc) dbg_acc[q.site0 + 2u * k] = (uint8_t)ok;
            }
            f[0] += S.x; f[1] += S.y; f[2] += S.z;
            if (colour == 1) f[3] -= dot3(S, hJ);
            if (ANISO) f[4] += aniso_energy<ANISO>(S, P.Ku, e[(ANISO & 1) ? k : 0], P.Kc);
            f[5] -= dot3(S, B);
            if (MODE == MODE_MEASURE && (flags & F_TORQUE)) {        // the unconstrained sweep never samples the torque
                const Vec3 t = onsite_torque<ANISO>(S, P.Ku, e[(ANISO & 1) ? k : 0], P.Kc, B);
                f[6] += t.x; f[7] += t.y; f[8] += t.z;
            }
        }
        if (MODE == MODE_SWEEP) {
            st_rw<VEC>(Sc + q.a0, nxv); st_rw<VEC>(Sc + P.plane + q.a0, nyv); st_rw<VEC>(Sc + 2 * P.plane + q.a0, nzv);
        }
#pragma unroll
        for (int k = 0; k < NQ; ++k) fs[k] += f[k];
        if (++pending == FLUSH_ITEMS) { fx_flush_shared(sacc, fs, P.fx_scale); pending = 0; }
    }
    fx_flush_shared(sacc, fs, P.fx_scale);
    long long acc[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) acc[q] = sacc[q][threadIdx.x];

    block_reduce(acc, cnt, P, MODE == MODE_MEASURE ? 1 : 0);
    if (flags & F_FINALIZE) {
        if (last_block_done(st)) final_reduce(P, MODE == MODE_MEASURE ? 1 : 0, flags);
    }
}

// Stand-alone pass 2 (for sweeps assembled from the half-sweep test hooks): <<<1, BLOCK>>>
__global__ void __launch_bounds__(BLOCK) finalize_kernel(const __grid_constant__ Params P, int mode, int flags)
{
    final_reduce(P, mode, flags);
}

// --------------------------------------------------------------------------------------------------------------
// Constrained pair pass of Table A2, one thread per VEC pairs of one colour.
// Pairing (C-11, replaces the shuffled index array of P:38/P:202 by a pure function of (seed, sweep, colour)):
//   the colour-linear index space is cut into H = Nc/B chunks of B consecutive sites, B = largest power of two
//   <= 32 with 2B | Nc, and each chunk into Bh = B/Bl groups of Bl = min(B,4) sites;
//   (r0,r1,r2,.) = Philox(0, TAG_PAIRING | colour<<8, sweep);  m = 2 floor(r0 (H/2) / 2^32) + 1;  sigma = r1 & 1;
//   rot = r2 mod Bl;  q = (r2 >> 2) mod Bh;
//   site (chunk, hi, lo) is a LEADER iff chunk mod 2 == sigma; its follower is ((chunk+m) mod H, (hi+q) mod Bh, (lo+rot) mod Bl).
// With VEC = 4 a thread owns one leader group and one follower group: two aligned float4 per component, the
// lo-rotation is a register permutation -- every access stays a full-sector vector access, no index array (0 bytes).
// --------------------------------------------------------------------------------------------------------------
struct PairGeom {
    uint32_t B, H, Bh, Bl;          // chunk size, chunk count, groups per chunk, sites per group
    uint32_t n_threads;             // = Nc / (2 VEC)
    FastDiv div_r, div_ny;          // colour-linear index -> (row, xh), row -> (z, y)
    uint32_t groups_per_chunk_vec;  // B / VEC  (VEC = 4: = Bh;  VEC = 1: = B)
};

template <int VEC>
__device__ __forceinline__ ItemPos locate_linear(const Params& P, const PairGeom& G, uint32_t a0, int colour)
{
    uint32_t row, xh0, y, z;
    G.div_r.divmod(a0, row, xh0);
    G.div_ny.divmod(row, z, y);
    ItemPos q;
    const uint32_t R = (uint32_t)P.R, ny = (uint32_t)P.ny, nz = (uint32_t)P.nz;
    q.par = (y + z + (uint32_t)colour) & 1u;
    q.xh0 = xh0;
    q.a0 = a0;
    q.site0 = row * (uint32_t)P.nx + 2u * xh0 + q.par;
    const uint32_t yp = (y + 1 == ny) ? 0u : y + 1, ym = (y == 0) ? ny - 1 : y - 1;
    const uint32_t zp = (z + 1 == nz) ? 0u : z + 1, zm = (z == 0) ? nz - 1 : z - 1;
    q.o_yp = (z * ny + yp) * R + xh0;  q.o_ym = (z * ny + ym) * R + xh0;
    q.o_zp = (zp * ny + y) * R + xh0;  q.o_zm = (zm * ny + y) * R + xh0;
    const bool wraps = q.par ? (xh0 + VEC == R) : (xh0 == 0);      // only the item's outermost x-bond can cross the wrap
    const uint32_t xe = q.par ? (wraps ? 0u : xh0 + VEC) : (wraps ? R - 1 : xh0 - 1);
    q.o_x = row * R + xe;
    q.xs = (wraps && P.anti_x) ? -1.0f : 1.0f;
    return q;
}

#ifndef MC_PAIR_MIN_BLOCKS
#define MC_PAIR_MIN_BLOCKS 2      // <= 128 registers: two CTAs per SM
#endif
template <int VEC, int ANISO, bool MASKED>
__global__ void __launch_bounds__(BLOCK, MC_PAIR_MIN_BLOCKS)
pair_kernel(const __grid_constant__ Params P, const __grid_constant__ PairGeom G, int colour, float invT, int flags,
            float* __restrict__ dbg_x, uint8_t* __restrict__ dbg_acc)
{
    DevState* st = P.st;
    grid_dependency_sync();
    const unsigned long long sweep = st->sweep;
    const float omc = st->one_minus_cos;
    const double ML = st->ML;
    const float invML = (float)(1.0 / ML);
    const Vec3 eC = { (float)st->eC[0], (float)st->eC[1], (float)st->eC[2] };
    const PhiloxKey& key = P.key;
    const uint32_t c2 = (uint32_t)sweep, c3 = (uint32_t)(sweep >> 32);
    uint32_t p0, p1, p2, p3;
    philox4x32_10(key, 0u, TAG_PAIRING | ((uint32_t)colour << 8), c2, c3, p0, p1, p2, p3);
    const uint32_t m = 2u * (uint32_t)(((uint64_t)p0 * (uint64_t)(G.H / 2)) >> 32) + 1u;
    const uint32_t sigma = p1 & 1u;
    const uint32_t rot = p2 % G.Bl, qsh = (p2 >> 2) % G.Bh;
    const uint32_t c1 = TAG_PAIR | ((uint32_t)colour << 8);
    float* Sc = P.S + (long long)colour * 3 * P.plane;
    const Vec3 B = { P.B[0], P.B[1], P.B[2] };

    __shared__ long long sacc[NQ][BLOCK];   // exact fixed-point sums of every thread of the block (fx_flush_shared)
    // VEC = 4: the follower group's spins (rows 0..11 = component * 4 + element) and exchange field (rows 12..23) of every
    // thread live in shared memory: the leader's element k pairs with element (k + rot) & 3 of the follower group, which is
    // then one indexed shared-memory access instead of a chain of register selects, and 24 registers less (the kernel spills)
    __shared__ float sF[VEC == 4 ? 24 : 1][BLOCK];
#pragma unroll
    for (int q = 0; q < NQ; ++q) sacc[q][threadIdx.x] = 0;
    int cnt = 0;

    const uint32_t stride = gridDim.x * BLOCK;
    for (uint32_t t = blockIdx.x * BLOCK + threadIdx.x; t < G.n_threads; t += stride) {
        // leader group
        const uint32_t j = t / G.groups_per_chunk_vec, g = t % G.groups_per_chunk_vec;
        const uint32_t chunkL = 2u * j + sigma;
        uint32_t chunkF = chunkL + m; if (chunkF >= G.H) chunkF -= G.H;
        uint32_t aL, aF;
        if (VEC == 4) {
            uint32_t gf = g + qsh; if (gf >= G.Bh) gf -= G.Bh;
            aL = chunkL * G.B + g * 4u; aF = chunkF * G.B + gf * 4u;
        } else {
            const uint32_t hi = g / G.Bl, lo = g % G.Bl;
            uint32_t hf = hi + qsh; if (hf >= G.Bh) hf -= G.Bh;
            uint32_t lf = lo + rot; if (lf >= G.Bl) lf -= G.Bl;
            aL = chunkL * G.B + g; aF = chunkF * G.B + hf * G.Bl + lf;
        }
        const ItemPos qL = locate_linear<VEC>(P, G, aL, colour), qF = locate_linear<VEC>(P, G, aF, colour);
        const Pack<VEC> lx = ld_rw<VEC>(Sc + aL), ly = ld_rw<VEC>(Sc + P.plane + aL), lz = ld_rw<VEC>(Sc + 2 * P.plane + aL);
        const Pack<VEC> fx = ld_rw<VEC>(Sc + aF), fy = ld_rw<VEC>(Sc + P.plane + aF), fz = ld_rw<VEC>(Sc + 2 * P.plane + aF);
        Vec3 hL[VEC], hF[VEC], eL[VEC], eF[VEC];
        exchange_field<VEC, MASKED>(P, qL, colour, hL);
        exchange_field<VEC, MASKED>(P, qF, colour, hF);
        if (ANISO & 1) { easy_axes<VEC>(P, qL, colour, eL); easy_axes<VEC>(P, qF, colour, eF); }
        Pack<VEC> nlx = lx, nly = ly, nlz = lz, nfx = fx, nfy = fy, nfz = fz;
        if (VEC == 4) {
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                sF[e][threadIdx.x] = fx.v[e]; sF[4 + e][threadIdx.x] = fy.v[e]; sF[8 + e][threadIdx.x] = fz.v[e];
                sF[12 + e][threadIdx.x] = hF[e].x; sF[16 + e][threadIdx.x] = hF[e].y; sF[20 + e][threadIdx.x] = hF[e].z;
            }
        }
        float f[NQ];
#pragma unroll
        for (int k = 0; k < NQ; ++k) f[k] = 0.0f;
        if (VEC == 4) {
            // ---- two pairs at a time in the two lanes of FFMA2 / FADD2 / FMUL2: lane x = pair kp, lane y = pair kp + 1.
            // Lane by lane this is the arithmetic of the scalar loop below (VEC = 1), branches turned into selects.
            const V3p eC2 = splat3(eC), B2 = splat3(B);
            f2 f2s[NQ];
#pragma unroll
            for (int q = 0; q < NQ; ++q) f2s[q] = splat(0.0f);
#pragma unroll
            for (int kp = 0; kp < 4; kp += 2) {
                const uint32_t kf0 = (kp + rot) & 3u, kf1 = (kp + 1 + rot) & 3u;
                const uint32_t tx = threadIdx.x;
                V3p Si = { make_float2(lx.v[kp], lx.v[kp + 1]), make_float2(ly.v[kp], ly.v[kp + 1]), make_float2(lz.v[kp], lz.v[kp + 1]) };
                const V3p Sj = { make_float2(sF[kf0][tx], sF[kf1][tx]), make_float2(sF[4 + kf0][tx], sF[4 + kf1][tx]), make_float2(sF[8 + kf0][tx], sF[8 + kf1][tx]) };
                const V3p hj = { make_float2(sF[12 + kf0][tx], sF[12 + kf1][tx]), make_float2(sF[16 + kf0][tx], sF[16 + kf1][tx]), make_float2(sF[20 + kf0][tx], sF[20 + kf1][tx]) };
                const V3p hi = pack3(hL[kp], hL[kp + 1]);
                V3p ei = eC2, ej = eC2;                      // placeholders when ANISO & 1 == 0
                if (ANISO & 1) {
                    ei = pack3(eL[kp], eL[kp + 1]);
                    Vec3 e0 = eF[0], e1 = eF[0];
#pragma unroll
                    for (int s2 = 1; s2 < 4; ++s2) {
                        const bool p0 = kf0 == (uint32_t)s2, p1 = kf1 == (uint32_t)s2;
                        e0.x = p0 ? eF[s2].x : e0.x; e0.y = p0 ? eF[s2].y : e0.y; e0.z = p0 ? eF[s2].z : e0.z;
                        e1.x = p1 ? eF[s2].x : e1.x; e1.y = p1 ? eF[s2].y : e1.y; e1.z = p1 ? eF[s2].z : e1.z;
                    }
                    ej = pack3(e0, e1);
                }
                const uint32_t site_i0 = qL.site0 + 2u * kp, site_i1 = site_i0 + 2u;
                // one Philox block per two pairs: the leaders site_i0 (bit 1 of x clear) and site_i0 + 2 take words (0,1) and (2,3) (C-26)
                uint32_t a0, a1, b0, b1;
                philox4x32_10(key, site_i0, c1, c2, c3, a0, a1, b0, b1);
                V3p di, Sni;
                cone_move2(Si, omc, make_float2(uniform01(a0), uniform01(b0)), make_float2(uniform_azimuth(a0, a1), uniform_azimuth(b0, b1)), di, Sni);
                const f2 pi_ = dot3p(Si, eC2), pj = dot3p(Sj, eC2), pni = dot3p(Sni, eC2);
                const V3p dv = { sub2(Si.x, Sni.x), sub2(Si.y, Sni.y), sub2(Si.z, Sni.z) };
                const f2 dpar = dot3p(dv, eC2), npj = neg2(pj), ndpar = neg2(dpar);
                const V3p pj_perp = { fma2(npj, eC2.x, Sj.x), fma2(npj, eC2.y, Sj.y), fma2(npj, eC2.z, Sj.z) };
                const V3p dl = { fma2(ndpar, eC2.x, dv.x), fma2(ndpar, eC2.y, dv.y), fma2(ndpar, eC2.z, dv.z) };
                const V3p perp = { add2(pj_perp.x, dl.x), add2(pj_perp.y, dl.y), add2(pj_perp.z, dl.z) };
                const V3p tw = { fma2(splat(2.0f), pj_perp.x, dl.x), fma2(splat(2.0f), pj_perp.y, dl.y), fma2(splat(2.0f), pj_perp.z, dl.z) };
                const f2 rho = fma2(pj, pj, neg2(dot3p(dl, tw)));                                   // P:189 radicand, difference form
                const bool v0 = rho.x > 0.0f, v1 = rho.y > 0.0f;                                    // C-13: radicand <= 0 rejects
                const f2 rs = make_float2(v0 ? rho.x : 1.0f, v1 ? rho.y : 1.0f);
                const f2 rt = mul2(rs, make_float2(rsqrtf(rs.x), rsqrtf(rs.y)));
                const f2 pnj = make_float2(copysignf(rt.x, pj.x), copysignf(rt.y, pj.y));           // sign kept
                const V3p v = { fma2(pnj, eC2.x, perp.x), fma2(pnj, eC2.y, perp.y), fma2(pnj, eC2.z, perp.z) };
                const f2 inv = fma2(splat(-0.5f), dot3p(v, v), splat(1.5f));
                const V3p Snj_new = { mul2(v.x, inv), mul2(v.y, inv), mul2(v.z, inv) };
                const f2 yml = mul2(sub2(sub2(add2(pni, pnj), pi_), pj), splat(invML));              // (M_L^ - M_L)/M_L
                const bool w0 = v0 && (1.0f + yml.x > 0.0f), w1 = v1 && (1.0f + yml.y > 0.0f);      // M_L^ > 0 (C-13)
                const f2 poly = mul2(yml, fma2(neg2(yml), fma2(neg2(yml), fma2(splat(-0.25f), yml, splat(0.33333333f)), splat(0.5f)), splat(1.0f)));
                const f2 lg = make_float2(__logf(w0 ? 1.0f + yml.x : 1.0f), __logf(w1 ? 1.0f + yml.y : 1.0f));
                const f2 lr = make_float2(fabsf(yml.x) < 0.03f ? poly.x : lg.x, fabsf(yml.y) < 0.03f ? poly.y : lg.y);
                const V3p dj = { sub2(Snj_new.x, Sj.x), sub2(Snj_new.y, Sj.y), sub2(Snj_new.z, Sj.z) };
                const f2 J2 = splat(P.J);
                const V3p hBi = { fma2(J2, hi.x, B2.x), fma2(J2, hi.y, B2.y), fma2(J2, hi.z, B2.z) };
                const V3p hBj = { fma2(J2, hj.x, B2.x), fma2(J2, hj.y, B2.y), fma2(J2, hj.z, B2.z) };
                const f2 dE = add2(delta_energy2<ANISO>(Si, di, hBi, P.Ku, ei, P.Kc), delta_energy2<ANISO>(Sj, dj, hBj, P.Ku, ej, P.Kc));   // P:193 (C-4)
                const f2 lu = make_float2(__logf(uniform01(a1)), __logf(uniform01(b1)));
                const f2 lq = make_float2(__logf(__fdividef(fabsf(pj.x), fabsf(pnj.x))), __logf(__fdividef(fabsf(pj.y), fabsf(pnj.y))));
                const f2 xr = sub2(sub2(fma2(dE, splat(invT), lu), mul2(splat(2.0f), lr)), lq);     // P:193 in log form
                const float INF = __int_as_float(0x7f800000);
                const float x0 = w0 ? xr.x : INF, x1 = w1 ? xr.y : INF;
                const bool ok0 = x0 < 0.0f, ok1 = x1 < 0.0f;
                // P:194 keep or restore both members
                Si.x = make_float2(ok0 ? Sni.x.x : Si.x.x, ok1 ? Sni.x.y : Si.x.y);
                Si.y = make_float2(ok0 ? Sni.y.x : Si.y.x, ok1 ? Sni.y.y : Si.y.y);
                Si.z = make_float2(ok0 ? Sni.z.x : Si.z.x, ok1 ? Sni.z.y : Si.z.y);
                const V3p Snj = { make_float2(ok0 ? Snj_new.x.x : Sj.x.x, ok1 ? Snj_new.x.y : Sj.x.y),
                                  make_float2(ok0 ? Snj_new.y.x : Sj.y.x, ok1 ? Snj_new.y.y : Sj.y.y),
                                  make_float2(ok0 ? Snj_new.z.x : Sj.z.x, ok1 ? Snj_new.z.y : Sj.z.y) };
                nlx.v[kp] = Si.x.x; nlx.v[kp + 1] = Si.x.y; nly.v[kp] = Si.y.x; nly.v[kp + 1] = Si.y.y; nlz.v[kp] = Si.z.x; nlz.v[kp + 1] = Si.z.y;
                sF[kf0][tx] = Snj.x.x; sF[4 + kf0][tx] = Snj.y.x; sF[8 + kf0][tx] = Snj.z.x;
                sF[kf1][tx] = Snj.x.y; sF[4 + kf1][tx] = Snj.y.y; sF[8 + kf1][tx] = Snj.z.y;
                cnt += (ok0 ? 2 : 0) + (ok1 ? 2 : 0);                                               // P:195 (C-23)
                const uint32_t site_j0 = qF.site0 + 2u * kf0, site_j1 = qF.site0 + 2u * kf1;
                if (dbg_x)   { dbg_x[site_i0] = x0; dbg_x[site_i1] = x1; }
                if (dbg_acc) { dbg_acc[site_i0] = (uint8_t)ok0; dbg_acc[site_j0] = (uint8_t)ok0; dbg_acc[site_i1] = (uint8_t)ok1; dbg_acc[site_j1] = (uint8_t)ok1; }
                // fused sums of the final spins of both members
                f2s[0] = add2(f2s[0], add2(Si.x, Snj.x)); f2s[1] = add2(f2s[1], add2(Si.y, Snj.y)); f2s[2] = add2(f2s[2], add2(Si.z, Snj.z));
                if (colour == 1) {
                    const V3p hJi = { mul2(J2, hi.x), mul2(J2, hi.y), mul2(J2, hi.z) }, hJj = { mul2(J2, hj.x), mul2(J2, hj.y), mul2(J2, hj.z) };
                    f2s[3] = sub2(f2s[3], add2(dot3p(Si, hJi), dot3p(Snj, hJj)));
                }
                if (ANISO) f2s[4] = add2(f2s[4], add2(aniso_energy2<ANISO>(Si, P.Ku, ei, P.Kc), aniso_energy2<ANISO>(Snj, P.Ku, ej, P.Kc)));   // (the pair pass has no registers for the kept-pieces variant)
                f2s[5] = sub2(f2s[5], add2(dot3p(Si, B2), dot3p(Snj, B2)));
                const V3p ti = onsite_torque2<ANISO>(Si, P.Ku, ei, P.Kc, B2), tj = onsite_torque2<ANISO>(Snj, P.Ku, ej, P.Kc, B2);
                f2s[6] = add2(f2s[6], add2(ti.x, tj.x)); f2s[7] = add2(f2s[7], add2(ti.y, tj.y)); f2s[8] = add2(f2s[8], add2(ti.z, tj.z));
            }
#pragma unroll
            for (int q = 0; q < NQ; ++q) f[q] = f2s[q].x + f2s[q].y;
        }
#pragma unroll
        for (int k = 0; k < (VEC == 4 ? 0 : VEC); ++k) {
            // leader element k pairs with follower element kf = (k + rot) mod Bl of the follower group (VEC = 4)
            Vec3 Si = { lx.v[k], ly.v[k], lz.v[k] };
            Vec3 Sj, hj, ej; uint32_t site_j;
            if (VEC == 4) {
                const uint32_t kf = (k + rot) & 3u;
                Sj = { sF[kf][threadIdx.x], sF[4 + kf][threadIdx.x], sF[8 + kf][threadIdx.x] };
                hj = { sF[12 + kf][threadIdx.x], sF[16 + kf][threadIdx.x], sF[20 + kf][threadIdx.x] };
                Vec3 ee = eF[0];
                if (ANISO & 1) {
#pragma unroll
                    for (int s = 1; s < 4; ++s) {
                        const bool pick = kf == (uint32_t)s;
                        ee.x = pick ? eF[s].x : ee.x; ee.y = pick ? eF[s].y : ee.y; ee.z = pick ? eF[s].z : ee.z;
                    }
                }
                ej = ee;
                site_j = qF.site0 + 2u * ((k + rot) & 3u);
            } else {
                Sj = { fx.v[0], fy.v[0], fz.v[0] }; hj = hF[0]; ej = eF[0]; site_j = qF.site0;
            }
            const uint32_t site_i = qL.site0 + 2u * k;
            uint32_t w0, w1;                                                           // the leader's 64 bits (C-26)
            {
                const uint32_t half = (qL.xh0 + (uint32_t)k) & 1u;
                uint32_t r0, r1, r2, r3;
                philox4x32_10(key, site_i - 2u * half, c1, c2, c3, r0, r1, r2, r3);
                w0 = half ? r2 : r0; w1 = half ? r3 : r1;
            }
            Vec3 di, Sni;
            cone_move(Si, omc, uniform01(w0), uniform_azimuth(w0, w1), di, Sni);
            const float pi_ = dot3(Si, eC), pj = dot3(Sj, eC), pni = dot3(Sni, eC);
            const Vec3 dv = { Si.x - Sni.x, Si.y - Sni.y, Si.z - Sni.z };             // stored displacement, exact in fp32
            // transverse parts: S_j,perp and the compensation delta = S_i,perp - S'_i,perp
            const float dpar = dot3(dv, eC);
            const Vec3 pj_perp = { fmaf(-pj, eC.x, Sj.x), fmaf(-pj, eC.y, Sj.y), fmaf(-pj, eC.z, Sj.z) };
            const Vec3 dl = { fmaf(-dpar, eC.x, dv.x), fmaf(-dpar, eC.y, dv.y), fmaf(-dpar, eC.z, dv.z) };
            const Vec3 perp = { pj_perp.x + dl.x, pj_perp.y + dl.y, pj_perp.z + dl.z };
            // P:189 radicand S_j^2 - |S'_j,perp|^2 in difference form: S_j,par^2 - delta.(2 S_j,perp + delta)
            // (no cancellation against 1, so a follower lying almost perpendicular to e_C keeps its relative accuracy)
            const Vec3 tw = { fmaf(2.0f, pj_perp.x, dl.x), fmaf(2.0f, pj_perp.y, dl.y), fmaf(2.0f, pj_perp.z, dl.z) };
            const float rho = fmaf(pj, pj, -dot3(dl, tw));
            float x = __int_as_float(0x7f800000);                                      // +inf: hard rejection (C-13)
            bool ok = false;
            Vec3 Snj = Sj;
            if (rho > 0.0f) {
                const float pnj = copysignf(rho * rsqrtf(rho), pj);                    // sign kept
                Vec3 v = { fmaf(pnj, eC.x, perp.x), fmaf(pnj, eC.y, perp.y), fmaf(pnj, eC.z, perp.z) };
                const float inv = fmaf(-0.5f, dot3(v, v), 1.5f);
                Snj = { v.x * inv, v.y * inv, v.z * inv };
                const float yml = (pni + pnj - pi_ - pj) * invML;                      // (M_L^ - M_L)/M_L
                if (1.0f + yml > 0.0f) {                                               // M_L^ > 0 (C-13)
                    const float lr = (fabsf(yml) < 0.03f) ? yml * (1.0f - yml * (0.5f - yml * (0.33333333f - 0.25f * yml)))
                                                          : __logf(1.0f + yml);
                    const Vec3 dj = { Snj.x - Sj.x, Snj.y - Sj.y, Snj.z - Sj.z };
                    const Vec3 hBi = { fmaf(P.J, hL[k].x, B.x), fmaf(P.J, hL[k].y, B.y), fmaf(P.J, hL[k].z, B.z) };
                    const Vec3 hBj = { fmaf(P.J, hj.x, B.x), fmaf(P.J, hj.y, B.y), fmaf(P.J, hj.z, B.z) };
                    const float dE = delta_energy<ANISO>(Si, di, hBi, P.Ku, eL[(ANISO & 1) ? k : 0], P.Kc)
                                   + delta_energy<ANISO>(Sj, dj, hBj, P.Ku, ej, P.Kc);  // P:193 (C-4)
                    // P:193 in log form: dE/T - 2 ln(M_L^/M_L) - ln|S_j,par / S'_j,par| + ln u2 < 0
                    x = fmaf(dE, invT, __logf(uniform01(w1))) - 2.0f * lr - __logf(__fdividef(fabsf(pj), fabsf(pnj)));
                    ok = x < 0.0f;
                }
            }
            if (ok) {
                Si = Sni; nlx.v[k] = Sni.x; nly.v[k] = Sni.y; nlz.v[k] = Sni.z;
                if (VEC == 4) {
                    const uint32_t kf = (k + rot) & 3u;
                    sF[kf][threadIdx.x] = Snj.x; sF[4 + kf][threadIdx.x] = Snj.y; sF[8 + kf][threadIdx.x] = Snj.z;
                } else { nfx.v[0] = Snj.x; nfy.v[0] = Snj.y; nfz.v[0] = Snj.z; }
            } else {
                Snj = Sj;
            }
            cnt += ok ? 2 : 0;                                                         // P:195 (C-23)
            if (dbg_x)   dbg_x[site_i] = x;
            if (dbg_acc) { dbg_acc[site_i] = (uint8_t)ok; dbg_acc[site_j] = (uint8_t)ok; }
            // fused sums of the final spins of both members
            const Vec3 hJi = { P.J * hL[k].x, P.J * hL[k].y, P.J * hL[k].z }, hJj = { P.J * hj.x, P.J * hj.y, P.J * hj.z };
            f[0] += Si.x + Snj.x; f[1] += Si.y + Snj.y; f[2] += Si.z + Snj.z;
            if (colour == 1) f[3] -= dot3(Si, hJi) + dot3(Snj, hJj);
            if (ANISO) f[4] += aniso_energy<ANISO>(Si, P.Ku, eL[(ANISO & 1) ? k : 0], P.Kc) + aniso_energy<ANISO>(Snj, P.Ku, ej, P.Kc);
            f[5] -= dot3(Si, B) + dot3(Snj, B);
            const Vec3 ti = onsite_torque<ANISO>(Si, P.Ku, eL[(ANISO & 1) ? k : 0], P.Kc, B);
            const Vec3 tj = onsite_torque<ANISO>(Snj, P.Ku, ej, P.Kc, B);
            f[6] += ti.x + tj.x; f[7] += ti.y + tj.y; f[8] += ti.z + tj.z;
        }
        if (VEC == 4) {
#pragma unroll
            for (int e = 0; e < 4; ++e) { nfx.v[e] = sF[e][threadIdx.x]; nfy.v[e] = sF[4 + e][threadIdx.x]; nfz.v[e] = sF[8 + e][threadIdx.x]; }
        }
        st_rw<VEC>(Sc + aL, nlx); st_rw<VEC>(Sc + P.plane + aL, nly); st_rw<VEC>(Sc + 2 * P.plane + aL, nlz);
        st_rw<VEC>(Sc + aF, nfx); st_rw<VEC>(Sc + P.plane + aF, nfy); st_rw<VEC>(Sc + 2 * P.plane + aF, nfz);
        fx_flush_shared(sacc, f, P.fx_scale);        // every item (8 updates): this kernel has no registers to spare for running sums
    }
    long long acc[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) acc[q] = sacc[q][threadIdx.x];

    block_reduce(acc, cnt, P, 0);
    if (flags & F_FINALIZE) {
        if (last_block_done(st)) final_reduce(P, 0, flags);
    }
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
    const uint32_t c = (x + y + z) & 1u, a = row * (uint32_t)P.R + (x >> 1);
    float vx = lex[3ull * s], vy = lex[3ull * s + 1], vz = lex[3ull * s + 2];
    const float n2 = vx * vx + vy * vy + vz * vz;
    const float inv = (n2 > 0.0f) ? (float)(1.0 / sqrt((double)n2)) : 0.0f;
    float* Sc = P.S + (long long)c * 3 * P.plane;
    Sc[a] = vx * inv; Sc[P.plane + a] = vy * inv; Sc[2 * P.plane + a] = (n2 > 0.0f) ? vz * inv : 1.0f;
}

__global__ void split_to_lex_kernel(const __grid_constant__ Params P, float* __restrict__ lex)
{
    const uint32_t s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= P.N) return;
    const uint32_t x = s % (uint32_t)P.nx, row = s / (uint32_t)P.nx, y = row % (uint32_t)P.ny, z = row / (uint32_t)P.ny;
    const uint32_t c = (x + y + z) & 1u, a = row * (uint32_t)P.R + (x >> 1);
    const float* Sc = P.S + (long long)c * 3 * P.plane;
    lex[3ull * s] = Sc[a]; lex[3ull * s + 1] = Sc[P.plane + a]; lex[3ull * s + 2] = Sc[2 * P.plane + a];
}

__global__ void fill_kernel(const __grid_constant__ Params P, float vx, float vy, float vz)
{
    const uint32_t a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= P.Nc) return;
    for (int c = 0; c < 2; ++c) {
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
    for (uint32_t c = 0; c < 2; ++c) {
        const uint32_t site = row * (uint32_t)P.nx + 2u * xh + ((y + z + c) & 1u);
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
    for (int c = 0; c < 2; ++c) {
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
enum : int { ST_CONE = 0, ST_SWEEP = 1, ST_RESET_ACC = 2, ST_EC = 3, ST_ML = 4, ST_RESET_COUNT = 5 };
__global__ void state_kernel(DevState* st, int what, double a, double b, double c, unsigned long long u)
{
    if (what == ST_CONE) { st->cone = a; st->one_minus_cos = (float)(1.0 - cos(a)); }
    else if (what == ST_SWEEP) { st->sweep = u; }
    else if (what == ST_RESET_ACC) {
        st->n_samples = 0ull;
        for (int i = 0; i < 4; ++i) { st->sum_m[i] = 0.0; st->sum_m2[i] = 0.0; }
        st->sum_E = 0.0; st->sum_E2 = 0.0;
        for (int i = 0; i < 3; ++i) st->sum_torque[i] = 0.0;
    }
    else if (what == ST_EC) { st->eC[0] = a; st->eC[1] = b; st->eC[2] = c; }
    else if (what == ST_ML) { st->ML = a; }
    else if (what == ST_RESET_COUNT) { st->count = 0ull; st->ticket = 0u; }
}

}  // namespace mc
