// mc_pass.cuh -- generic colour pass of Table A1: grid-stride gather through L1/L2, any lattice.
#pragma once

#include "mc_common.cuh"

namespace mc {

// --------------------------------------------------------------------------------------------------------------
// Colour pass of Table A1: one item of VEC sites per loop trip, grid-stride.
//   MODE_SWEEP  : propose (a-4), dE (a-5), accept/write (a-6), count (a-7), fused sums of the FINAL spins (a-9).
//   MODE_MEASURE: no move; sums of the current spins (standalone measurement).
// E_exch is accumulated by the BLACK pass only: every bond joins a red and a black site, so
// E_exch = -sum_{i black} S_i.h_i with h already in registers (0 extra bytes).
// --------------------------------------------------------------------------------------------------------------
// 128 threads x 6 CTAs per SM (<= 80 registers; c5 film with 256-thread CTAs: one per SM 354, two 185, three 166 us per sweep;
// 128 x 6: 160.6 against 162.3 for 256 x 3)
#ifndef MC_PASS_BLOCK
#define MC_PASS_BLOCK 128
#endif
#ifndef MC_PASS_MIN_BLOCKS
#define MC_PASS_MIN_BLOCKS 6
#endif
// the basis-mode instantiation (LAT = 3) holds four rows of the bond table in flight: <= 96 registers, five CTAs per SM
// (176^3 cells of hcp: 1032 against 1083 us per sweep with six)
#ifndef MC_BASIS_MIN_BLOCKS
#define MC_BASIS_MIN_BLOCKS 5
#endif
__host__ __device__ constexpr int pass_min_blocks(int lat) { return lat >= 3 ? MC_BASIS_MIN_BLOCKS : MC_PASS_MIN_BLOCKS; }
// LAT: 0 simple cubic; 1 bcc, 2 fcc, 3 / 4 basis mode (hcp / sc + next-nearest neighbours: eight colours, bond table; with
// COL < 0 the run-time table of either structure under LAT = 3, with COL >= 0 the compile-time table of structure LAT) (mc_common.cuh):
// VEC = 4 consecutive cells of one sublattice, site stride 1 instead of 2;
// fcc: four colours, the exchange energy of a bond is summed in the pass of its higher colour (hl).
// COL >= 0: the colour as a compile-time constant (fcc: which rows and shifts a sublattice reads is then resolved by the compiler).
template <int VEC, int ANISO, bool MASKED, int MODE, int LAT = 0, int COL = -1>
__global__ void __launch_bounds__(MC_PASS_BLOCK, pass_min_blocks(LAT))
pass_kernel(const __grid_constant__ Params P, const __grid_constant__ Geom G, int colour_rt, float invT, int flags,
            float* __restrict__ dbg_x, uint8_t* __restrict__ dbg_acc)
{
    const int colour = COL >= 0 ? COL : colour_rt;
    DevState* st = P.st;
    grid_dependency_sync();
    const unsigned long long sweep = st->sweep;
    const float omc = st->one_minus_cos;
    const PhiloxKey& key = P.key;
    const uint32_t c1 = TAG_MOVE | ((uint32_t)colour << 8), c2 = (uint32_t)sweep, c3 = (uint32_t)(sweep >> 32);
    float* Sc = P.S + (long long)colour * 3 * P.plane;
    const Vec3 B = { P.B[0], P.B[1], P.B[2] };

    __shared__ long long sacc[NQ][MC_PASS_BLOCK];   // exact fixed-point sums of every thread of the block (fx_flush_shared)
    float fs[NQ];                    // fp32 running sums of at most FLUSH_ITEMS items
#pragma unroll
    for (int q = 0; q < NQ; ++q) { sacc[q][threadIdx.x] = 0; fs[q] = 0.0f; }
    int cnt = 0, pending = 0;

    const uint32_t stride = gridDim.x * MC_PASS_BLOCK;
    for (uint32_t item = blockIdx.x * MC_PASS_BLOCK + threadIdx.x; item < G.n_items; item += stride) {
        static_assert(!LAT || (VEC == 4 && !MASKED), "the bcc / fcc passes are VEC = 4, unmasked instantiations");
        constexpr uint32_t SS = LAT ? 1u : 2u;                    // site-id stride between the sites of an item
        ItemPos q;
        Vec3 h[VEC], e[VEC], hl[LAT >= 2 ? VEC : 1];
        const float Jm = LAT >= 3 ? 1.0f : P.J;                   // basis mode: the couplings are already in h, hl
        if (LAT == 1) {
            const BccPos b = bcc_locate(P, G, item, colour);
            q.a0 = b.a0; q.site0 = b.site0; q.xh0 = b.i0; q.par = 0u;
            if (VEC == 4) bcc_exchange_field(P, b, colour, reinterpret_cast<Vec3(&)[4]>(h));
        } else if (LAT == 2) {
            const FccPos b = fcc_locate(P, G, item, colour);
            q.a0 = b.a0; q.site0 = b.site0; q.xh0 = b.i0; q.par = 0u;
            if (VEC == 4) fcc_exchange_field(P, b, colour, reinterpret_cast<Vec3(&)[4]>(h), reinterpret_cast<Vec3(&)[4]>(hl));
        } else if (LAT >= 3) {
            const FccPos b = fcc_locate(P, G, item, colour);
            q.a0 = b.a0; q.site0 = b.site0; q.xh0 = b.i0; q.par = 0u;
            if constexpr (VEC == 4 && LAT >= 3 && COL >= 0)        // structure LAT and sublattice COL fixed at compile time: unrolled table
                basis_exchange_field_ct<LAT, COL>(P, b, reinterpret_cast<Vec3(&)[4]>(h), reinterpret_cast<Vec3(&)[4]>(hl));
            else if (VEC == 4) basis_exchange_field(P, b, colour, reinterpret_cast<Vec3(&)[4]>(h), reinterpret_cast<Vec3(&)[4]>(hl));
        } else {
            q = locate<VEC>(P, G, item, colour);
            exchange_field<VEC, MASKED>(P, q, colour, h);
        }
        const Pack<VEC> sx = ld_rw<VEC>(Sc + q.a0), sy = ld_rw<VEC>(Sc + P.plane + q.a0), sz = ld_rw<VEC>(Sc + 2 * P.plane + q.a0);
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
                for (int k = 0; k + 1 < VEC; k += 2) philox4x32_10(key, q.site0 + SS * k, c1, c2, c3, w0[k], w1[k], w0[k + 1], w1[k + 1]);
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
                const f2 J2 = splat(Jm);
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
                if (dbg_x)   { dbg_x[q.site0 + SS * kp] = xx.x; dbg_x[q.site0 + SS * kp + SS] = xx.y; }
                if (dbg_acc) { dbg_acc[q.site0 + SS * kp] = (uint8_t)ok0; dbg_acc[q.site0 + SS * kp + SS] = (uint8_t)ok1; }
                f2s[0] = add2(f2s[0], S.x); f2s[1] = add2(f2s[1], S.y); f2s[2] = add2(f2s[2], S.z);
                if (LAT >= 2) {
                    const V3p hlp = pack3(hl[LAT >= 2 ? kp : 0], hl[LAT >= 2 ? kp + 1 : 0]);
                    f2s[3] = sub2(f2s[3], dot3p(S, V3p{ mul2(J2, hlp.x), mul2(J2, hlp.y), mul2(J2, hlp.z) }));
                } else if (colour == 1) f2s[3] = sub2(f2s[3], dot3p(S, hJ));
                if (ANISO) f2s[4] = add2(f2s[4], onsite_from<ANISO>(ok0, ok1, s4S, s4v, euS, euv, P.Ku, P.Kc));
                f2s[5] = sub2(f2s[5], dot3p(S, B2));
            }
#pragma unroll
            for (int qq = 0; qq < 6; ++qq) f[qq] += f2s[qq].x + f2s[qq].y;
        }
#pragma unroll
        for (int k = 0; k < ((VEC == 4 && MODE == MODE_SWEEP) ? 0 : VEC); ++k) {
            Vec3 S = { sx.v[k], sy.v[k], sz.v[k] };
            const Vec3 hJ = { Jm * h[k].x, Jm * h[k].y, Jm * h[k].z };
            if (MODE == MODE_SWEEP) {
                Vec3 d, Sn;
                cone_move(S, omc, uniform01(w0[k]), uniform_azimuth(w0[k], w1[k]), d, Sn);
                const Vec3 hB = { hJ.x + B.x, hJ.y + B.y, hJ.z + B.z };
                const float dE = delta_energy<ANISO>(S, d, hB, P.Ku, e[(ANISO & 1) ? k : 0], P.Kc);
                const float x = fmaf(dE, invT, __logf(uniform01(w1[k])));    // P:157-158 in log form (C-8)
                const bool ok = x < 0.0f;
                if (ok) { S = Sn; nxv.v[k] = Sn.x; nyv.v[k] = Sn.y; nzv.v[k] = Sn.z; }
                cnt += ok;
                if (dbg_x)   dbg_x[q.site0 + SS * k] = x;
                if (dbg_acc) dbg_acc[q.site0 + SS * k] = (uint8_t)ok;
            }
            f[0] += S.x; f[1] += S.y; f[2] += S.z;
            if (LAT >= 2) { const Vec3& g = hl[LAT >= 2 ? k : 0]; f[3] -= dot3(S, Vec3{ Jm * g.x, Jm * g.y, Jm * g.z }); }
            else if (colour == 1) f[3] -= dot3(S, hJ);
            if (ANISO) f[4] += aniso_energy<ANISO>(S, P.Ku, e[(ANISO & 1) ? k : 0], P.Kc);
            f[5] -= dot3(S, B);
            if (MODE == MODE_MEASURE && (flags & F_TORQUE)) {        // the unconstrained sweep never samples the torque
                const Vec3 t = onsite_torque<ANISO>(S, P.Ku, e[(ANISO & 1) ? k : 0], P.Kc, B);
                f[6] += t.x; f[7] += t.y; f[8] += t.z;
            }
        }
        if (MODE == MODE_SWEEP) {
            if constexpr ((LAT == 1 || (LAT == 0 && !MASKED)) && VEC == 4) {          // evict-first stores: bcc +4 %, sc 128^3 +2.6 %; masked films lose 11 %
                st_rw_streaming(Sc + q.a0, nxv); st_rw_streaming(Sc + P.plane + q.a0, nyv); st_rw_streaming(Sc + 2 * P.plane + q.a0, nzv);
            } else {
                st_rw<VEC>(Sc + q.a0, nxv); st_rw<VEC>(Sc + P.plane + q.a0, nyv); st_rw<VEC>(Sc + 2 * P.plane + q.a0, nzv);
            }
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


}  // namespace mc
