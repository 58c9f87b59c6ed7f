// mc_pair.cuh -- constrained pair pass of Table A2, generic gather through L1/L2.
#pragma once

#include "mc_common.cuh"

namespace mc {

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

// bcc (C-30): the colour-linear index IS the cell index of the sublattice; rows and the cell outside the item as in bcc_locate
__device__ __forceinline__ BccPos bcc_locate_linear(const Params& P, const PairGeom& G, uint32_t a0, int colour)
{
    uint32_t row, i0, y, z;
    G.div_r.divmod(a0, row, i0);
    G.div_ny.divmod(row, z, y);
    const uint32_t nx = (uint32_t)P.nx, ny = (uint32_t)P.ny, nz = (uint32_t)P.nz;
    BccPos q;
    q.i0 = i0; q.a0 = a0; q.site0 = (uint32_t)colour * P.Nc + a0;
    const uint32_t y2 = colour ? (y + 1 == ny ? 0u : y + 1) : (y == 0 ? ny - 1 : y - 1);
    const uint32_t z2 = colour ? (z + 1 == nz ? 0u : z + 1) : (z == 0 ? nz - 1 : z - 1);
    q.row[0] = (z * ny + y) * nx;  q.row[1] = (z * ny + y2) * nx;
    q.row[2] = (z2 * ny + y) * nx; q.row[3] = (z2 * ny + y2) * nx;
    q.xe = colour ? (i0 + 4 == nx ? 0u : i0 + 4) : (i0 == 0 ? nx - 1 : i0 - 1);
    return q;
}

template <int V> struct IntC { static constexpr int value = V; };

// 128 threads x 4 CTAs per SM (<= 128 registers).  Measured at 224^3, us per constrained sweep: 256 x 2 114.1, 192 x 2 (166
// registers) 115.9, 128 x 3 (166 registers) 112.3, 128 x 4 110.4, 96 x 5 115.9, 64 x 8 118.5
#ifndef MC_PAIR_BLOCK
#define MC_PAIR_BLOCK 128
#endif
#ifndef MC_PAIR_MIN_BLOCKS
#define MC_PAIR_MIN_BLOCKS 4
#endif
// LAT: 0 simple cubic; 1 bcc (VEC = 4 consecutive cells of one sublattice, site-id stride 1, the 8-bond field).
template <int VEC, int ANISO, bool MASKED, int LAT = 0>
__global__ void __launch_bounds__(MC_PAIR_BLOCK, MC_PAIR_MIN_BLOCKS)
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

    __shared__ long long sacc[NQ][MC_PAIR_BLOCK];   // exact fixed-point sums of every thread of the block (fx_flush_shared)
#pragma unroll
    for (int q = 0; q < NQ; ++q) sacc[q][threadIdx.x] = 0;
    int cnt = 0;

    // VEC = 4: the leader's element k pairs with element (k + rot) & 3 of the follower group.  rot is the same for every thread of
    // the launch, so the loop is instantiated for its four values and entered through one uniform switch: the pairing inside a
    // group is then register naming (no select chains, no staging of the follower group in shared memory).
    const uint32_t stride = gridDim.x * MC_PAIR_BLOCK;
    auto run = [&](auto rot_c) {
    constexpr uint32_t ROT = (uint32_t)decltype(rot_c)::value;
    for (uint32_t t = blockIdx.x * MC_PAIR_BLOCK + threadIdx.x; t < G.n_threads; t += stride) {
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
        static_assert(!LAT || (VEC == 4 && !MASKED), "the bcc pair pass is the VEC = 4, unmasked instantiation");
        constexpr uint32_t SS = LAT ? 1u : 2u;                     // site-id stride between the sites of an item
        ItemPos qL, qF;
        Vec3 hL[VEC], hF[VEC], eL[VEC], eF[VEC];
        if (LAT == 1) {
            const BccPos bL = bcc_locate_linear(P, G, aL, colour), bF = bcc_locate_linear(P, G, aF, colour);
            qL.a0 = aL; qL.site0 = bL.site0; qL.xh0 = bL.i0; qL.par = 0u;
            qF.a0 = aF; qF.site0 = bF.site0; qF.xh0 = bF.i0; qF.par = 0u;
            if (VEC == 4) {
                bcc_exchange_field(P, bL, colour, reinterpret_cast<Vec3(&)[4]>(hL));
                bcc_exchange_field(P, bF, colour, reinterpret_cast<Vec3(&)[4]>(hF));
            }
        } else {
            qL = locate_linear<VEC>(P, G, aL, colour); qF = locate_linear<VEC>(P, G, aF, colour);
            exchange_field<VEC, MASKED>(P, qL, colour, hL);
            exchange_field<VEC, MASKED>(P, qF, colour, hF);
        }
        const Pack<VEC> lx = ld_rw<VEC>(Sc + aL), ly = ld_rw<VEC>(Sc + P.plane + aL), lz = ld_rw<VEC>(Sc + 2 * P.plane + aL);
        const Pack<VEC> fx = ld_rw<VEC>(Sc + aF), fy = ld_rw<VEC>(Sc + P.plane + aF), fz = ld_rw<VEC>(Sc + 2 * P.plane + aF);
        if (ANISO & 1) { easy_axes<VEC>(P, qL, colour, eL); easy_axes<VEC>(P, qF, colour, eF); }
        Pack<VEC> nlx = lx, nly = ly, nlz = lz, nfx = fx, nfy = fy, nfz = fz;
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
                const int kf0 = (kp + ROT) & 3, kf1 = (kp + 1 + ROT) & 3;               // compile-time after unrolling
                V3p Si = { make_float2(lx.v[kp], lx.v[kp + 1]), make_float2(ly.v[kp], ly.v[kp + 1]), make_float2(lz.v[kp], lz.v[kp + 1]) };
                const V3p Sj = { make_float2(fx.v[kf0 % VEC], fx.v[kf1 % VEC]), make_float2(fy.v[kf0 % VEC], fy.v[kf1 % VEC]), make_float2(fz.v[kf0 % VEC], fz.v[kf1 % VEC]) };
                const V3p hj = pack3(hF[kf0 % VEC], hF[kf1 % VEC]);
                const V3p hi = pack3(hL[kp], hL[kp + 1]);
                V3p ei = eC2, ej = eC2;                      // placeholders when ANISO & 1 == 0
                if (ANISO & 1) { ei = pack3(eL[kp], eL[kp + 1]); ej = pack3(eF[kf0 % VEC], eF[kf1 % VEC]); }
                const uint32_t site_i0 = qL.site0 + SS * kp, site_i1 = site_i0 + SS;
                // one Philox block per two pairs: the leaders site_i0 (bit 1 of x clear; bcc: even cell) and its same-colour x-neighbour take words (0,1) and (2,3) (C-26, C-30)
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
                nfx.v[kf0 % VEC] = Snj.x.x; nfy.v[kf0 % VEC] = Snj.y.x; nfz.v[kf0 % VEC] = Snj.z.x;
                nfx.v[kf1 % VEC] = Snj.x.y; nfy.v[kf1 % VEC] = Snj.y.y; nfz.v[kf1 % VEC] = Snj.z.y;
                cnt += (ok0 ? 2 : 0) + (ok1 ? 2 : 0);                                               // P:195 (C-23)
                const uint32_t site_j0 = qF.site0 + SS * kf0, site_j1 = qF.site0 + SS * kf1;
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
            // VEC = 1: one pair per thread, the scalar form of the packed arithmetic above (the rotation is in aF)
            Vec3 Si = { lx.v[k], ly.v[k], lz.v[k] };
            const Vec3 Sj = { fx.v[0], fy.v[0], fz.v[0] }, hj = hF[0], ej = eF[0];
            const uint32_t site_j = qF.site0;
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
                nfx.v[0] = Snj.x; nfy.v[0] = Snj.y; nfz.v[0] = Snj.z;
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
        if constexpr (VEC == 4) {                      // evict-first stores (+0.5 %)
            st_rw_streaming(Sc + aL, nlx); st_rw_streaming(Sc + P.plane + aL, nly); st_rw_streaming(Sc + 2 * P.plane + aL, nlz);
            st_rw_streaming(Sc + aF, nfx); st_rw_streaming(Sc + P.plane + aF, nfy); st_rw_streaming(Sc + 2 * P.plane + aF, nfz);
        } else {
        st_rw<VEC>(Sc + aL, nlx); st_rw<VEC>(Sc + P.plane + aL, nly); st_rw<VEC>(Sc + 2 * P.plane + aL, nlz);
        st_rw<VEC>(Sc + aF, nfx); st_rw<VEC>(Sc + P.plane + aF, nfy); st_rw<VEC>(Sc + 2 * P.plane + aF, nfz);
        }
        fx_flush_shared(sacc, f, P.fx_scale);        // every item (8 updates): this kernel has no registers to spare for running sums
    }
    };
    if (VEC == 4) {
        switch (rot) {
            case 0: run(IntC<0>{}); break;  case 1: run(IntC<1>{}); break;
            case 2: run(IntC<2>{}); break;  default: run(IntC<3>{}); break;
        }
    } else {
        run(IntC<0>{});
    }
    long long acc[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) acc[q] = sacc[q][threadIdx.x];

    block_reduce(acc, cnt, P, 0);
    if (flags & F_FINALIZE) {
        if (last_block_done(st)) final_reduce(P, 0, flags);
    }
}


}  // namespace mc
