// mc_tile.cuh -- the sm_100a fast path of the colour pass (Table A1) for uniform, fully periodic lattices.
//
// Design:
//   * One CTA owns a y-slab of Ty rows (all of x) and marches through a z-segment of Lz planes.  The three planes
//     z-1, z, z+1 of the OTHER colour that a plane of this colour needs live in a 4-slot shared-memory ring; one warp
//     streams plane z+2 into the free slot with TMA bulk copies (cp.async.bulk, one row per copy, completion on an
//     mbarrier) while all warps update plane z.  Every other-colour value is therefore read from HBM/L2 once per
//     (slab, segment) and then served 6 times from shared memory; the y-halo is 2 rows per slab and the z-halo 2
//     planes per segment.
//   * One thread owns a PAIR of x-adjacent sites of one colour in RP..RP*NPASS rows of the slab for the whole march:
//     all its shared-memory and global offsets are loop invariants, the march only adds constants.
//   * The fp32 arithmetic of the two sites is packed into Blackwell's two-wide FFMA2 / FADD2 / FMUL2 instructions
//     (one issue slot for two sites); Philox, MUFU and the selects stay scalar.
//   * Own colour: LDG.64 / STG.64 straight from/to the colour-split planes (read once, written once).
//   * Fused sums (a-9) are carried per thread in fp32 over its <= 2*NPASS*Lz sites (a bounded, fixed set), converted to
//     64-bit fixed point once, then summed exactly (block_reduce: order-independent, reproducible); fp64 in final_reduce.
// Arithmetic contract: identical to pass_kernel / DESIGN.md section 3 (same Philox stream, same cone construction).
#pragma once

#include "mc_common.cuh"

namespace mc {

constexpr int TILE_NSLOT = 4;
#ifndef MC_TILE_MAX_THREADS
#define MC_TILE_MAX_THREADS 448
#endif
#ifndef MC_TILE_MIN_BLOCKS
#define MC_TILE_MIN_BLOCKS 2
#endif
#ifndef MC_TILE_TY_RT
#define MC_TILE_TY_RT 16
#endif
constexpr int TILE_MAX_THREADS = MC_TILE_MAX_THREADS;   // launch bounds of the tiled pass: threads per CTA ...
constexpr int TILE_MIN_BLOCKS = MC_TILE_MIN_BLOCKS;     // ... and CTAs per SM the register allocation must allow
constexpr int TILE_NPASS_RT = 2;                        // passes (row groups) a thread of a compile-time-R specialisation covers per plane (unrolled)
// CTA shape of a specialisation: threads per CTA, CTAs per SM and the largest slab height.  Default 448 x 2, slabs of 16 rows.
// R = 112 (224^3, the headline lattice): 224 x 4 with slabs of 8 rows -- the same 28 warps per SM in twice as many, smaller CTAs:
// a CTA's per-plane barrier holds up 7 warps instead of 14 (87.7 against 89.9 us per sweep; R = 96 and 32 lose with it: 61.1
// against 57.7 and 12.6 against 11.8 us).
#ifndef MC_TILE_SMALL_CTA_R
#define MC_TILE_SMALL_CTA_R 112
#endif
__host__ __device__ constexpr int tile_threads_rt(int R) { return R == MC_TILE_SMALL_CTA_R ? TILE_MAX_THREADS / 2 : TILE_MAX_THREADS; }
__host__ __device__ constexpr int tile_blocks_rt(int R)  { return R == MC_TILE_SMALL_CTA_R ? 2 * TILE_MIN_BLOCKS : TILE_MIN_BLOCKS; }
__host__ __device__ constexpr int tile_tymax_rt(int R)   { return R == MC_TILE_SMALL_CTA_R ? MC_TILE_TY_RT / 2 : MC_TILE_TY_RT; }
// Slab shape of the specialisation for R colour-sites per row: RP rows per pass = as many as its threads cover
// (one thread = one x-adjacent pair), at most tile_tymax_rt / 2; slab height Ty = 2 RP.  R = 32, 96: 8 x 2 = 16 rows; R = 112: 4 x 2 = 8.
__host__ __device__ constexpr int tile_rp_rt(int R) { return R <= 0 ? 0 : ((tile_threads_rt(R) / (R / 2)) < (tile_tymax_rt(R) / 2) ? (tile_threads_rt(R) / (R / 2)) : (tile_tymax_rt(R) / 2)); }
__host__ __device__ constexpr int tile_ty_rt(int R) { return TILE_NPASS_RT * tile_rp_rt(R); }
// Row lengths R = nx / 2 with a specialised instantiation (every shared-memory offset an immediate, both passes unrolled).
#ifndef MC_TILE_RT_LIST
#define MC_TILE_RT_LIST(X) X(32) X(96) X(112)
#endif
inline bool tile_has_rt(int R)
{
#define MC_TILE_X(r) if (R == r) return true;
    MC_TILE_RT_LIST(MC_TILE_X)
#undef MC_TILE_X
    return false;
}

struct TileGeom {
    int R, PR;                 // colour-sites per row, pairs per row
    int nx, ny, nz;
    int Ty, RP, NPASS;         // rows per slab = RP * NPASS, rows per pass
    int n_slabs, n_segs;       // grid = n_slabs * n_segs
    int Lz, Lz_rem;            // segment s covers Lz + (s < Lz_rem ? 1 : 0) planes
    int slot_floats;           // 3 * (Ty + 2) * R
    int n_active;              // PR * RP working threads (block size is this rounded up to a warp multiple)
    int stream_l2;             // 1: the spin state does not fit the L2 (the specialised instantiations then copy with the evict-first policy)
};

// ---- packed two-wide fp32 helpers (FFMA2 / FADD2 / FMUL2 on sm_100a)
// (f2, add2, mul2, fma2, splat: mc_device.cuh)

// ---- mbarrier / TMA bulk-copy primitives (PTX; CTA-local shared addresses)
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "MC_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra MC_DONE;\n"
        "bra MC_WAIT;\n"
        "MC_DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// L2S: the plane copies carry the evict-first L2 policy.  For lattices whose spin state does not fit the L2: the other colour
// streams through it (each row is wanted again only by the neighbouring slabs and segments, at about the same time), 224^3:
// 86.5 -> 84.9 us per sweep.  A lattice that fits loses with it (192^3: 54.0 -> 57.2: the next pass would have found the rows
// cached), so the choice is a template parameter resolved by the planner, not a run-time branch in the copy.
template <bool L2S>
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar)
{
    if constexpr (L2S) {
        unsigned long long pol;
        asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                     ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(pol) : "memory");
    } else {
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
    }
}

// One plane (Ty + 2 rows x 3 components, periodic wrap in y) of the other colour -> one ring slot, issued by ONE thread.
// Rows that are consecutive in y are consecutive in HBM and in the slot, so a slab in the interior of the lattice
// needs one bulk copy per component; a slab touching y = 0 or y = ny-1 needs one more per wrapped row.
template <bool L2S>
__device__ __forceinline__ void tile_issue_plane(const TileGeom& G, int R, const float* __restrict__ Oth, long long plane, int z, int y0,
                                                 uint32_t slot_addr, uint32_t bar)
{
    const int nrows = G.Ty + 2;
    const uint32_t row_bytes = (uint32_t)R * 4u;
    mbar_arrive_expect_tx(bar, 3u * (uint32_t)nrows * row_bytes);
    const float* zbase = Oth + (long long)z * G.ny * R;
    int ry = 0;
    while (ry < nrows) {
        int y = y0 - 1 + ry;
        if (y < 0) y += G.ny; else if (y >= G.ny) y -= G.ny;
        int run = nrows - ry; if (run > G.ny - y) run = G.ny - y;
#pragma unroll
        for (int comp = 0; comp < 3; ++comp)
            bulk_g2s<L2S>(slot_addr + (uint32_t)(comp * nrows + ry) * row_bytes, zbase + (long long)comp * plane + (long long)y * R,
                     (uint32_t)run * row_bytes, bar);
        ry += run;
    }
}

// u = f - (1 - 2^-24) with f = 1 + (w >> 9) 2^-23 in [1,2): one funnel shift builds f (C-8)
__device__ __forceinline__ float mantissa_1p(uint32_t w) { return __uint_as_float(__funnelshift_r(w, 0x7Fu, 9)); }
// (xor_sign: mc_device.cuh)

// ANISO: bit 0 uniaxial (uniform axis), bit 1 cubic.  FIELD: Zeeman term.  RT: colour-sites per row as a compile-time
// constant (0 = run-time value; the specialisations turn every shared-memory offset into an immediate).
// sum S.h is accumulated by the black pass only (every bond joins a red and a black site, so
// E_exch = -J sum_{i black} S_i.h_i with h already in registers).
// On-site energies of the FINAL spin reuse what dE needs: cubic through s4 = sum_a S_a^4 (on the unit sphere
// Sx^2Sy^2 + Sx^2Sz^2 + Sy^2Sz^2 = (1 - s4)/2, so dE_c = -Kc/2 (s4' - s4) and E_c = Kc/2 (1 - s4)), uniaxial through
// (S.e)^2 and its difference form.
// ANTI: anti-periodic boundary along x (domain-wall box; C-27): the one x-neighbour a pair reads across the row
// end enters with the opposite sign.  Instantiated for the run-time row length only.
template <int ANISO, bool FIELD, int RT, bool DEBUG, bool ANTI = false, bool L2S = false>
__global__ void __launch_bounds__(tile_threads_rt(RT), tile_blocks_rt(RT))
tile_pass_kernel(const __grid_constant__ Params P, const __grid_constant__ TileGeom G, int colour, float invT, int flags,
                  float* __restrict__ dbg_x, uint8_t* __restrict__ dbg_acc)
{
    extern __shared__ __align__(128) float smem[];
    __shared__ __align__(8) unsigned long long bars[TILE_NSLOT];

    DevState* st = P.st;
    grid_dependency_sync();          // nothing a previous pass wrote (spins, controller state) is touched before this point
    const unsigned long long sweep = st->sweep;
    const float omc = st->one_minus_cos;
    const PhiloxKey& key = P.key;
    const uint32_t c1 = TAG_MOVE | ((uint32_t)colour << 8), c2 = (uint32_t)sweep, c3 = (uint32_t)(sweep >> 32);

    const int R = RT ? RT : G.R;
    const int PR = R / 2;
    const int tid = threadIdx.x;
    const int slab = blockIdx.x % G.n_slabs, seg = blockIdx.x / G.n_slabs;
    const int y0 = slab * G.Ty;
    const int Lz = G.Lz + (seg < G.Lz_rem ? 1 : 0);
    const int z0 = seg * G.Lz + (seg < G.Lz_rem ? seg : G.Lz_rem);
    const int nrows = (RT ? tile_ty_rt(RT) : G.Ty) + 2;             // the specialisations fix the slab height ...
    const int NPASS = RT ? TILE_NPASS_RT : G.NPASS, RP = RT ? tile_rp_rt(RT) : G.RP;   // ... and its split into passes
    const int CS = nrows * R;
    const int slot_floats = 3 * CS;

    const float* Oth = P.S + (long long)(1 - colour) * 3 * P.plane;
    float* Sc = P.S + (long long)colour * 3 * P.plane;
    const uint32_t smem_base = smem_u32(smem), bar_base = smem_u32(bars);
    const uint32_t slot_bytes = (uint32_t)slot_floats * 4u;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < TILE_NSLOT; ++s) mbar_init(bar_base + 8u * s, 1u);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        const int nseq = Lz + 2 < TILE_NSLOT ? Lz + 2 : TILE_NSLOT;
        for (int k = 0; k < nseq; ++k) {
            int z = z0 - 1 + k; if (z < 0) z += G.nz; else if (z >= G.nz) z -= G.nz;
            tile_issue_plane<L2S>(G, R, Oth, P.plane, z, y0, smem_base + (uint32_t)k * slot_bytes, bar_base + 8u * k);
        }
    }
    __syncthreads();

    const bool active = tid < G.n_active;
    const int r0 = tid / PR, cp = tid - r0 * PR;
    const int exL = (cp == 0) ? R - 1 : 2 * cp - 1;
    const int exR = (cp == PR - 1) ? 0 : 2 * cp + 2;
    const float sgL = (ANTI && cp == 0) ? -1.0f : 1.0f, sgR = (ANTI && cp == PR - 1) ? -1.0f : 1.0f;   // wrap-bond signs
    const int soff0 = (r0 + 1) * R + 2 * cp;
    const int exo0 = (r0 + 1) * R;
    const int pstride = RP * R;
    const long long zstride = (long long)G.ny * R;
    float* gS = Sc + ((long long)z0 * G.ny + y0 + r0) * R + 2 * cp;
    uint32_t siteb = (uint32_t)(((long long)z0 * G.ny + y0 + r0) * G.nx) + 4u * (uint32_t)cp;
    const uint32_t zsite = (uint32_t)(G.ny * G.nx), psite = (uint32_t)(RP * G.nx);
    int parz = (y0 + r0 + z0 + colour) & 1;

    f2 aMx = splat(0.f), aMy = splat(0.f), aMz = splat(0.f), aEx = splat(0.f), aAn = splat(0.f);
    int cnt = 0;

    const float CU = 0.99999994f;
    const f2 nomc2 = splat(-omc);
    const f2 twopi2 = splat(6.2831853071795865f), angc2 = splat(-9.4247779607693797f);     // phi - pi = 2 pi (f1 - 1) - pi
    const f2 nCU2 = splat(-CU);
    const f2 xscale2 = splat(invT * 1.4426950408889634f);
    const f2 nJ2 = splat(-P.J);
    const f2 e2x = splat(P.eu[0]), e2y = splat(P.eu[1]), e2z = splat(P.eu[2]);
    const f2 B2x = splat(P.B[0]), B2y = splat(P.B[1]), B2z = splat(P.B[2]);
    const f2 nKu2 = splat(-P.Ku), nhKc2 = splat(-0.5f * P.Kc), two = splat(2.0f);

    mbar_wait(bar_base, 0u); mbar_wait(bar_base + 8u, 0u);
    for (int j = 0; j < Lz; ++j, gS += zstride, siteb += zsite, parz ^= 1) {
        { const int k = j + 2; mbar_wait(bar_base + 8u * (k & 3), (uint32_t)(k >> 2) & 1u); }
        const float* sM = smem + ((j) & 3) * slot_floats;
        const float* sC = smem + ((j + 1) & 3) * slot_floats;
        const float* sP = smem + ((j + 2) & 3) * slot_floats;

        if (active) {
            float* g = gS;
            uint32_t sb = siteb;
            int soff = soff0, exo = exo0, parj = parz;
#pragma unroll (RT ? TILE_NPASS_RT : 1)
            for (int pass = 0; pass < NPASS; ++pass, g += pstride, sb += psite, soff += pstride, exo += pstride, parj += RP) {
                const int par = parj & 1;
                const uint32_t site0 = sb + (uint32_t)par;
                const float* pC = sC + soff;
                const float* pP = sP + soff;
                const float* pM = sM + soff;
                const float* pE = sC + exo + (par ? exR : exL);

                const f2 Sx = *reinterpret_cast<const f2*>(g);
                const f2 Sy = *reinterpret_cast<const f2*>(g + P.plane);
                const f2 Sz = *reinterpret_cast<const f2*>(g + 2 * P.plane);

                f2 h[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const f2 o  = *reinterpret_cast<const f2*>(pC + c * CS);
                    const float ex = ANTI ? pE[c * CS] * (par ? sgR : sgL) : pE[c * CS];
                    const f2 yp = *reinterpret_cast<const f2*>(pC + c * CS + R);
                    const f2 ym = *reinterpret_cast<const f2*>(pC + c * CS - R);
                    const f2 zp = *reinterpret_cast<const f2*>(pP + c * CS);
                    const f2 zm = *reinterpret_cast<const f2*>(pM + c * CS);
                    const f2 sh = par ? make_float2(o.y, ex) : make_float2(ex, o.x);
                    h[c] = add2(add2(add2(o, sh), add2(yp, ym)), add2(zp, zm));
                }

                // random numbers (a-2): one Philox4x32-10 block per x-adjacent pair: words 0,1 -> first site, words 2,3 -> second site (C-26)
                uint32_t r0w, r1w, r2w, r3w;
                philox4x32_10(key, site0, c1, c2, c3, r0w, r1w, r2w, r3w);
                const f2 f0 = make_float2(mantissa_1p(r0w), mantissa_1p(r2w));
                const f2 f2u = make_float2(mantissa_1p(r1w), mantissa_1p(r3w));
                const f2 f1 = make_float2(azimuth_1p(r0w, r1w), azimuth_1p(r2w, r3w));

                const f2 nw = mul2(add2(f0, nCU2), nomc2);
                const f2 t  = mul2(nw, fma2(nw, splat(-1.0f), splat(-2.0f)));
                const f2 sa = mul2(t, make_float2(rsqrtf(t.x), rsqrtf(t.y)));
                const f2 ang = fma2(f1, twopi2, angc2);
                const f2 Cc = mul2(sa, make_float2(__cosf(ang.x), __cosf(ang.y)));
                const f2 Ss = mul2(sa, make_float2(__sinf(ang.x), __sinf(ang.y)));
                const f2 sg = make_float2(copysignf(1.0f, Sz.x), copysignf(1.0f, Sz.y));
                const f2 den = add2(sg, Sz);
                const f2 ia = make_float2(__fdividef(1.0f, den.x), __fdividef(1.0f, den.y));
                const f2 uu = mul2(Sx, ia), vv = mul2(Sy, ia);
                const f2 q  = make_float2(xor_sign(Sx.x, Sz.x), xor_sign(Sx.y, Sz.y));      // sg * Sx
                const f2 nt1x = fma2(q, uu, splat(-1.0f));
                const f2 nt1y = mul2(q, vv);
                const f2 nt2x = mul2(Sy, uu);
                const f2 nt2y = fma2(Sy, vv, make_float2(xor_sign(-1.0f, Sz.x), xor_sign(-1.0f, Sz.y)));   // - sg, on the integer pipe
                const f2 dx = fma2(Cc, nt1x, fma2(Ss, nt2x, mul2(nw, Sx)));
                const f2 dy = fma2(Cc, nt1y, fma2(Ss, nt2y, mul2(nw, Sy)));
                const f2 dz = fma2(Cc, q,    fma2(Ss, Sy,   mul2(nw, Sz)));
                const f2 vx = add2(Sx, dx), vy = add2(Sy, dy), vz = add2(Sz, dz);
                const f2 V2x = mul2(vx, vx), V2y = mul2(vy, vy), V2z = mul2(vz, vz);
                const f2 n2 = add2(add2(V2x, V2y), V2z);
                const f2 inv = fma2(n2, splat(-0.5f), splat(1.5f));
                const f2 Nx = mul2(vx, inv), Ny = mul2(vy, inv), Nz = mul2(vz, inv);

                const f2 dh = fma2(dx, h[0], fma2(dy, h[1], mul2(dz, h[2])));
                f2 dE = mul2(nJ2, dh);
                if (FIELD) dE = fma2(splat(-1.0f), fma2(dx, B2x, fma2(dy, B2y, mul2(dz, B2z))), dE);
                f2 eu_old = splat(0.f), eu_new = splat(0.f);
                if (ANISO & 1) {
                    const f2 de = fma2(dx, e2x, fma2(dy, e2y, mul2(dz, e2z)));
                    const f2 se = fma2(Sx, e2x, fma2(Sy, e2y, mul2(Sz, e2z)));
                    const f2 du = mul2(de, fma2(two, se, de));                  // (v.e)^2 - (S.e)^2, difference form
                    dE = fma2(nKu2, du, dE);
                    eu_old = mul2(se, se); eu_new = add2(eu_old, du);
                }
                f2 s4S = splat(0.f), s4v = splat(0.f);
                if (ANISO & 2) {
                    // on the unit sphere Sx^2Sy^2 + Sx^2Sz^2 + Sy^2Sz^2 = (1 - s4)/2 with s4 = sum_a S_a^4
                    const f2 S2x = mul2(Sx, Sx), S2y = mul2(Sy, Sy), S2z = mul2(Sz, Sz);
                    s4S = fma2(S2x, S2x, fma2(S2y, S2y, mul2(S2z, S2z)));
                    s4v = fma2(V2x, V2x, fma2(V2y, V2y, mul2(V2z, V2z)));
                    dE = fma2(nhKc2, sub2(s4v, s4S), dE);
                }

                const f2 u2 = add2(f2u, nCU2);
                const f2 xd = fma2(dE, xscale2, make_float2(__log2f(u2.x), __log2f(u2.y)));
                const bool ok0 = xd.x < 0.0f, ok1 = xd.y < 0.0f;
                f2 Ox, Oy, Oz;
                Ox.x = ok0 ? Nx.x : Sx.x; Oy.x = ok0 ? Ny.x : Sy.x; Oz.x = ok0 ? Nz.x : Sz.x;
                Ox.y = ok1 ? Nx.y : Sx.y; Oy.y = ok1 ? Ny.y : Sy.y; Oz.y = ok1 ? Nz.y : Sz.y;
                cnt += (int)ok0 + (int)ok1;
                // Store policy, measured: a lattice that fits the L2 stores evict-first (192^3: 56.7 -> 54.2 us per sweep); one that
                // does not (L2S: its plane copies already leave the L2 first) stores with the default policy, so that what the L2
                // keeps is the colour just written, which the next pass reads (224^3 with evict-first copies: 84.9 -> 83.1)
                if constexpr (L2S) {
                    *reinterpret_cast<f2*>(g) = Ox; *reinterpret_cast<f2*>(g + P.plane) = Oy; *reinterpret_cast<f2*>(g + 2 * P.plane) = Oz;
                } else {
                    __stcs(reinterpret_cast<f2*>(g), Ox); __stcs(reinterpret_cast<f2*>(g + P.plane), Oy); __stcs(reinterpret_cast<f2*>(g + 2 * P.plane), Oz);
                }
                if (DEBUG) {
                    if (dbg_x)   { dbg_x[site0] = xd.x * 0.69314718055994531f; dbg_x[site0 + 2u] = xd.y * 0.69314718055994531f; }
                    if (dbg_acc) { dbg_acc[site0] = (uint8_t)ok0; dbg_acc[site0 + 2u] = (uint8_t)ok1; }
                }

                // fused sums of the final spins (a-9)
                aMx = add2(aMx, Ox); aMy = add2(aMy, Oy); aMz = add2(aMz, Oz);
                if (colour) aEx = fma2(Ox, h[0], fma2(Oy, h[1], fma2(Oz, h[2], aEx)));
                if (ANISO & 1) aAn = fma2(nKu2, make_float2(ok0 ? eu_new.x : eu_old.x, ok1 ? eu_new.y : eu_old.y), aAn);
                if (ANISO & 2) aAn = fma2(nhKc2, make_float2(ok0 ? s4v.x : s4S.x, ok1 ? s4v.y : s4S.y), aAn);
            }
        }
        __syncthreads();
        if (tid == 0 && j + TILE_NSLOT < Lz + 2) {
            const int k = j + TILE_NSLOT;
            int zn = z0 - 1 + k; if (zn >= G.nz) zn -= G.nz;
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            tile_issue_plane<L2S>(G, R, Oth, P.plane, zn, y0, smem_base + (uint32_t)(k & 3) * slot_bytes, bar_base + 8u * (k & 3));
        }
    }

    // ---- pass 1 of the fused sums: this thread's fp32 sums (<= 2 NPASS Lz sites) -> 64-bit fixed point -> exact block sums
    float f[NQ];
    f[0] = aMx.x + aMx.y; f[1] = aMy.x + aMy.y; f[2] = aMz.x + aMz.y;
    f[3] = colour ? -P.J * (aEx.x + aEx.y) : 0.0f;
    f[4] = aAn.x + aAn.y;
    if ((ANISO & 2) && active) f[4] += 0.5f * P.Kc * (float)(2 * NPASS * Lz);      // the "1" of (1 - s4)/2, once per site
    f[5] = FIELD ? -(f[0] * P.B[0] + f[1] * P.B[1] + f[2] * P.B[2]) : 0.0f;
    f[6] = f[7] = f[8] = 0.0f;
    long long acc[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) acc[q] = 0;
    fx_flush(acc, f, P.fx_scale);
    block_reduce(acc, cnt, P, 0);
    if (flags & F_FINALIZE) {
        if (last_block_done(st)) final_reduce(P, 0, flags);
    }
}
}  // namespace mc
