// mc_march.cuh -- colour pass of Table A1 as a register-carried march: no shared-memory staging, no barrier.
//
// One thread owns an item of 4 consecutive same-colour sites of a row and marches along one lattice axis (z for bulk
// lattices, y for thin films whose z extent is a handful of planes).  Of the six neighbours of a site, the two along the
// march axis are the in-plane values of the previous and the next step at the same column, so a thread carries the other
// colour's steps m-1 and m in registers and loads only step m+1 (its own column), the two side rows of step m and the
// one x-neighbour outside the item: 12 loads of the other colour + 3 of its own per step instead of 18 + 3, and every
// address advances by one constant per step -- the index arithmetic of the grid-stride gather (mc_pass.cuh: two magic
// divisions and seven neighbour addresses per item, ~30 % of its instructions) is gone: 125 instead of 182 instructions per
// update.  The side rows a thread loads are the in-step rows of threads of the same block: L1 serves them.
// Arithmetic: the packed functions of mc_device.cuh in the order of pass_kernel<4,...> and exchange_field<4,...>: the spins
// are bit-identical to the generic pass (the GPU tests check it).  MASKED: bond masks (grain boundaries, open faces) and
// per-grain easy axes (config c5).  x must be periodic (not anti-periodic) with nx % 8 == 0.
#pragma once

#include "mc_common.cuh"

namespace mc {

struct MarchGeom {
    int axis;                  // march axis: 2 = z (threads over (x4, y)), 1 = y (threads over (x4, z))
    int RV;                    // items of 4 sites per row = R / 4
    int XB, SB;                // a block of MARCH_BLOCK threads = XB items x SB side rows (axis 1: SB = nz); axis 2: natural order
    int n_segs, Lm, Lm_rem;    // segments along the march axis: segment s covers Lm + (s < Lm_rem ? 1 : 0) steps
    uint32_t n_threads;
    FastDiv div_rv, div_ns, div_xqb;
};

// 128 threads x 4 CTAs per SM (<= 128 registers): the same 16 warps as 256 x 2, in smaller CTAs (224^3: 90.3 against 91.6 us per sweep)
#ifndef MC_MARCH_BLOCK
#define MC_MARCH_BLOCK 128
#endif
constexpr int MARCH_BLOCK = MC_MARCH_BLOCK;
#ifndef MC_MARCH_MIN_BLOCKS
#define MC_MARCH_MIN_BLOCKS 4
#endif

template <int ANISO, bool MASKED, int AXIS, bool DEBUG>
__global__ void __launch_bounds__(MARCH_BLOCK, MC_MARCH_MIN_BLOCKS)
march_pass_kernel(const __grid_constant__ Params P, const __grid_constant__ MarchGeom G, int colour, float invT, int flags,
                  float* __restrict__ dbg_x, uint8_t* __restrict__ dbg_acc)
{
    DevState* st = P.st;
    grid_dependency_sync();
    const unsigned long long sweep = st->sweep;
    const float omc = st->one_minus_cos;
    const PhiloxKey& key = P.key;
    const uint32_t c1 = TAG_MOVE | ((uint32_t)colour << 8), c2 = (uint32_t)sweep, c3 = (uint32_t)(sweep >> 32);

    f2 aM[3] = { splat(0.f), splat(0.f), splat(0.f) }, aEx = splat(0.f), aAn = splat(0.f), aZe = splat(0.f);
    int cnt = 0;
    const uint32_t t = blockIdx.x * MARCH_BLOCK + threadIdx.x;
    if (t < G.n_threads) {
        const int R = P.R, ny = P.ny, nz = P.nz;
        const int nm = AXIS == 2 ? nz : ny, ns = AXIS == 2 ? ny : nz;     // extents along the march and the side axis
        uint32_t seg, s, xq;
        if (AXIS == 2) {                                                   // t = (seg * ny + y) * RV + xq
            uint32_t rowq; G.div_rv.divmod(t, rowq, xq); G.div_ns.divmod(rowq, seg, s);
        } else {                                                           // block = (seg, x-block); thread = (side row, item of the block)
            uint32_t xqb; G.div_xqb.divmod(blockIdx.x, seg, xqb);
            s = threadIdx.x / (uint32_t)G.XB; xq = xqb * (uint32_t)G.XB + threadIdx.x % (uint32_t)G.XB;
        }
        const int Lm = G.Lm + ((int)seg < G.Lm_rem ? 1 : 0);
        const int m0 = (int)seg * G.Lm + ((int)seg < G.Lm_rem ? (int)seg : G.Lm_rem);
        const int xh0 = 4 * (int)xq;
        const long long ms = AXIS == 2 ? (long long)ny * R : R, ss = AXIS == 2 ? R : (long long)ny * R;   // floats per march / side step
        const int y0 = AXIS == 2 ? (int)s : m0, z0 = AXIS == 2 ? m0 : (int)s;
        const long long a0 = ((long long)z0 * ny + y0) * R + xh0;         // colour-linear index of the item at the first step
        // side rows s+1, s-1: periodic wrap, or (open face: the bond is masked) the row itself
        const bool per_s = P.mask == nullptr || (AXIS == 2 ? (P.per_mask >> 1) & 1 : (P.per_mask >> 2) & 1);
        const bool per_m = P.mask == nullptr || (AXIS == 2 ? (P.per_mask >> 2) & 1 : (P.per_mask >> 1) & 1);
        const long long dsp = (int)s + 1 == ns ? (per_s ? -(long long)(ns - 1) * ss : 0) : ss;
        const long long dsm = s == 0 ? (per_s ? (long long)(ns - 1) * ss : 0) : -ss;
        const float* O = P.S + (long long)(1 - colour) * 3 * P.plane;
        float* pS = P.S + (long long)colour * 3 * P.plane + a0;           // own colour at the current step
        const float* pO = O + a0;                                          // other colour at the current step, this row
        const float* pSp = pO + dsp;                                       // ... side row s+1, side row s-1
        const float* pSm = pO + dsm;
        const uint8_t* pMask = MASKED ? P.mask + (long long)colour * P.mask_plane + a0 : nullptr;
        const uint16_t* pReg = (MASKED && P.region) ? P.region + (long long)colour * P.region_plane + a0 : nullptr;
        // the x-neighbour outside the item, relative to the item: par = 0 -> column xh0 - 1, par = 1 -> column xh0 + 4 (row wrap)
        const int exoff0 = xh0 == 0 ? R - 1 : -1, exoff1 = xh0 + 4 == R ? -xh0 : 4;
        int par = (y0 + z0 + colour) & 1;
        uint32_t site0 = (uint32_t)(((long long)z0 * ny + y0) * P.nx) + 2u * (uint32_t)xh0;      // + par at use
        const uint32_t msite = (uint32_t)(AXIS == 2 ? ny * P.nx : P.nx);
        const Vec3 B = { P.B[0], P.B[1], P.B[2] };
        const V3p B2 = splat3(B);
        const Vec3 eu = { P.eu[0], P.eu[1], P.eu[2] };

        // steps m0 - 1 and m0 of the other colour at this column (m0 - 1 beyond an open face: any valid row, its bond is masked)
        Pack<4> mm[3], oc[3];
        {
            const long long dmm = m0 == 0 ? (per_m ? (long long)(nm - 1) * ms : 0) : -ms;
#pragma unroll
            for (int c = 0; c < 3; ++c) { mm[c] = ld_nc<4>(pO + c * P.plane + dmm); oc[c] = ld_nc<4>(pO + c * P.plane); }
        }
        for (int j = 0; j < Lm; ++j) {
            const int m = m0 + j;
            const long long dmp = m + 1 == nm ? (per_m ? -(long long)(nm - 1) * ms : 0) : ms;
            const int exoff = par ? exoff1 : exoff0;
            Pack<4> mp[3], spv[3], smv[3]; float ex[3];
            Pack<4> sx = ld_rw<4>(pS), sy = ld_rw<4>(pS + P.plane), sz = ld_rw<4>(pS + 2 * P.plane);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                mp[c] = ld_nc<4>(pO + c * P.plane + dmp);
                spv[c] = ld_nc<4>(pSp + c * P.plane);
                smv[c] = ld_nc<4>(pSm + c * P.plane);
                ex[c] = __ldg(pO + c * P.plane + exoff);
            }
            uint32_t mbits[4];
            if (MASKED) {
                const uint32_t w = __ldg(reinterpret_cast<const uint32_t*>(pMask));
#pragma unroll
                for (int k = 0; k < 4; ++k) mbits[k] = (w >> (8 * k)) & 0xFFu;
            }
            // exchange field in the summation order of exchange_field<4, MASKED> (mc_common.cuh): o, x-shift, +y, -y, +z, -z
            const Pack<4>* ypv = AXIS == 2 ? spv : mp;  const Pack<4>* ymv = AXIS == 2 ? smv : mm;
            const Pack<4>* zpv = AXIS == 2 ? mp : spv;  const Pack<4>* zmv = AXIS == 2 ? mm : smv;
            float hc[3][4];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const Pack<4>& o = oc[c];
                const float s0 = par ? o.v[1] : ex[c], s1 = par ? o.v[2] : o.v[0], s2 = par ? o.v[3] : o.v[1], s3 = par ? ex[c] : o.v[2];
#pragma unroll
                for (int h2 = 0; h2 < 2; ++h2) {
                    const int a = 2 * h2, b = 2 * h2 + 1;
                    const f2 sh2 = h2 ? make_float2(s2, s3) : make_float2(s0, s1);
                    f2 r;
                    if (MASKED) {
                        const uint32_t bo = par ? 1u : 0u, bs = par ? 0u : 1u;      // bit index of o's bond / the shifted neighbour's bond
                        auto mf = [&](uint32_t bit) { return make_float2((mbits[a] & (1u << bit)) ? 1.0f : 0.0f, (mbits[b] & (1u << bit)) ? 1.0f : 0.0f); };
                        r = mul2(mf(bo), make_float2(o.v[a], o.v[b]));
                        r = fma2(mf(bs), sh2, r);
                        r = fma2(mf(2u), make_float2(ypv[c].v[a], ypv[c].v[b]), r);
                        r = fma2(mf(3u), make_float2(ymv[c].v[a], ymv[c].v[b]), r);
                        r = fma2(mf(4u), make_float2(zpv[c].v[a], zpv[c].v[b]), r);
                        r = fma2(mf(5u), make_float2(zmv[c].v[a], zmv[c].v[b]), r);
                    } else {
                        r = add2(add2(add2(make_float2(o.v[a], o.v[b]), sh2), add2(make_float2(ypv[c].v[a], ypv[c].v[b]), make_float2(ymv[c].v[a], ymv[c].v[b]))),
                                 add2(make_float2(zpv[c].v[a], zpv[c].v[b]), make_float2(zmv[c].v[a], zmv[c].v[b])));
                    }
                    hc[c][a] = r.x; hc[c][b] = r.y;
                }
            }
            // easy axes: uniform, or per grain through the region table, fetched after the field so that they are not
            // live across it
            Vec3 e[4];
            if (ANISO & 1) {
                if (MASKED && pReg) {
                    const uint2 rr = __ldg(reinterpret_cast<const uint2*>(pReg));
                    const uint32_t id[4] = { rr.x & 0xFFFFu, rr.x >> 16, rr.y & 0xFFFFu, rr.y >> 16 };
#pragma unroll
                    for (int k = 0; k < 4; ++k) { const float4 a = __ldg(P.axis + id[k]); e[k] = { a.x, a.y, a.z }; }
                } else {
#pragma unroll
                    for (int k = 0; k < 4; ++k) e[k] = eu;
                }
            }
            const uint32_t s0id = site0 + (uint32_t)par;
            uint32_t w0[4], w1[4];
#pragma unroll
            for (int k = 0; k < 4; k += 2) philox4x32_10(key, s0id + 2u * k, c1, c2, c3, w0[k], w1[k], w0[k + 1], w1[k + 1]);
            Pack<4> nxv = sx, nyv = sy, nzv = sz;
#pragma unroll
            for (int kp = 0; kp < 4; kp += 2) {
                V3p S = { make_float2(sx.v[kp], sx.v[kp + 1]), make_float2(sy.v[kp], sy.v[kp + 1]), make_float2(sz.v[kp], sz.v[kp + 1]) };
                const V3p hp = { make_float2(hc[0][kp], hc[0][kp + 1]), make_float2(hc[1][kp], hc[1][kp + 1]), make_float2(hc[2][kp], hc[2][kp + 1]) };
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
                if (DEBUG) {
                    if (dbg_x)   { dbg_x[s0id + 2u * kp] = xx.x; dbg_x[s0id + 2u * kp + 2u] = xx.y; }
                    if (dbg_acc) { dbg_acc[s0id + 2u * kp] = (uint8_t)ok0; dbg_acc[s0id + 2u * kp + 2u] = (uint8_t)ok1; }
                }
                aM[0] = add2(aM[0], S.x); aM[1] = add2(aM[1], S.y); aM[2] = add2(aM[2], S.z);
                if (colour == 1) aEx = sub2(aEx, dot3p(S, hJ));
                if (ANISO) aAn = add2(aAn, onsite_from<ANISO>(ok0, ok1, s4S, s4v, euS, euv, P.Ku, P.Kc));
                aZe = sub2(aZe, dot3p(S, B2));
            }
            st_rw<4>(pS, nxv); st_rw<4>(pS + P.plane, nyv); st_rw<4>(pS + 2 * P.plane, nzv);
            // next step: the column's carried steps shift down, every pointer moves one step along the march axis
#pragma unroll
            for (int c = 0; c < 3; ++c) { mm[c] = oc[c]; oc[c] = mp[c]; }
            pS += ms; pO += ms; pSp += ms; pSm += ms; site0 += msite; par ^= 1;
            if (MASKED) { pMask += ms; if (pReg) pReg += ms; }
        }
    }
    // fused sums (a-9): this thread's fp32 sums over its <= 4 Lm sites -> 64-bit fixed point -> exact block sums
    float f[NQ];
    f[0] = aM[0].x + aM[0].y; f[1] = aM[1].x + aM[1].y; f[2] = aM[2].x + aM[2].y;
    f[3] = aEx.x + aEx.y; f[4] = aAn.x + aAn.y; f[5] = aZe.x + aZe.y;
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

// --------------------------------------------------------------------------------------------------------------
// bcc (C-30): the same march for the two-sublattice lattice.  A thread owns 4 consecutive cells of a row of its
// sublattice and marches along k.  Its 8 neighbours per cell are the cells i and i -+ 1 of the rows j, j -+ 1 of the
// planes k and k -+ 1 of the other sublattice (- for sublattice A, + for B): two of the four rows were the in-plane rows
// of the previous step (A: plane k - 1 is the last step's plane k; B: plane k is the last step's plane k + 1), so
// they are carried in registers and a step loads two rows (float4 + the one cell outside the item, per component)
// instead of four.  Summation order of bcc_exchange_field (rows (k,j), (k,j'), (k',j), (k',j')): bit-identical spins.
// --------------------------------------------------------------------------------------------------------------
struct BccRow { Pack<4> o; float ex; };

template <int ANISO, int COLOUR, bool DEBUG>
__global__ void __launch_bounds__(MARCH_BLOCK, MC_MARCH_MIN_BLOCKS)
march_bcc_kernel(const __grid_constant__ Params P, const __grid_constant__ MarchGeom G, int, float invT, int flags,
                 float* __restrict__ dbg_x, uint8_t* __restrict__ dbg_acc)
{
    constexpr int colour = COLOUR;           // the sublattice decides which rows are carried: compile-time, so that they stay registers
    DevState* st = P.st;
    grid_dependency_sync();
    const unsigned long long sweep = st->sweep;
    const float omc = st->one_minus_cos;
    const PhiloxKey& key = P.key;
    const uint32_t c1 = TAG_MOVE | ((uint32_t)colour << 8), c2 = (uint32_t)sweep, c3 = (uint32_t)(sweep >> 32);

    f2 aM[3] = { splat(0.f), splat(0.f), splat(0.f) }, aEx = splat(0.f), aAn = splat(0.f), aZe = splat(0.f);
    int cnt = 0;
    const uint32_t t = blockIdx.x * MARCH_BLOCK + threadIdx.x;
    if (t < G.n_threads) {
        const int nx = P.nx, ny = P.ny, nz = P.nz;
        uint32_t rowq, xq, seg, y;
        G.div_rv.divmod(t, rowq, xq); G.div_ns.divmod(rowq, seg, y);
        const int Lm = G.Lm + ((int)seg < G.Lm_rem ? 1 : 0);
        const int k0 = (int)seg * G.Lm + ((int)seg < G.Lm_rem ? (int)seg : G.Lm_rem);
        const int i0 = 4 * (int)xq;
        const long long ms = (long long)ny * nx;                           // cells per plane
        const int y2 = colour ? ((int)y + 1 == ny ? 0 : (int)y + 1) : (y == 0 ? ny - 1 : (int)y - 1);
        const long long a0 = ((long long)k0 * ny + y) * nx + i0;
        const float* O = P.S + (long long)(1 - colour) * 3 * P.plane;
        float* pS = P.S + (long long)colour * 3 * P.plane + a0;
        const float* pR0 = O + a0;                                          // other sublattice, plane k: row j and row j'
        const float* pR1 = O + ((long long)k0 * ny + y2) * nx + i0;
        const int exoff = colour ? (i0 + 4 == nx ? -i0 : 4) : (i0 == 0 ? nx - 1 : -1);   // the cell outside the item: i0 + 4 (B) or i0 - 1 (A)
        uint32_t site0 = (uint32_t)colour * P.Nc + (uint32_t)a0;
        const Vec3 B = { P.B[0], P.B[1], P.B[2] };
        const V3p B2 = splat3(B);
        const V3p e2 = splat3(Vec3{ P.eu[0], P.eu[1], P.eu[2] });
        auto load_rows = [&](long long d, BccRow (&r0)[3], BccRow (&r1)[3]) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                r0[c].o = ld_nc<4>(pR0 + c * P.plane + d); r0[c].ex = __ldg(pR0 + c * P.plane + d + exoff);
                r1[c].o = ld_nc<4>(pR1 + c * P.plane + d); r1[c].ex = __ldg(pR1 + c * P.plane + d + exoff);
            }
        };
        // carried rows: A carries plane k - 1 (the previous step's plane k), B carries plane k (the previous step's plane k + 1)
        BccRow car0[3], car1[3];
        load_rows(colour ? 0 : (k0 == 0 ? (long long)(nz - 1) * ms : -ms), car0, car1);
        for (int j = 0; j < Lm; ++j) {
            const int k = k0 + j;
            BccRow new0[3], new1[3];
            Pack<4> sx = ld_rw<4>(pS), sy = ld_rw<4>(pS + P.plane), sz = ld_rw<4>(pS + 2 * P.plane);
            load_rows(colour ? (k + 1 == nz ? -(long long)(nz - 1) * ms : ms) : 0, new0, new1);   // B: plane k + 1; A: plane k
            float hc[3][4];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                // rows in the order (k, j), (k, j'), (k', j), (k', j'): plane k is the new load for A and the carried one for B
                const BccRow* rows[4] = { colour ? &car0[c] : &new0[c], colour ? &car1[c] : &new1[c], colour ? &new0[c] : &car0[c], colour ? &new1[c] : &car1[c] };
                f2 lo = splat(0.0f), hi = splat(0.0f);
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    const Pack<4>& o = rows[r]->o; const float ex = rows[r]->ex;
                    const f2 slo = colour ? make_float2(o.v[1], o.v[2]) : make_float2(ex, o.v[0]);
                    const f2 shi = colour ? make_float2(o.v[3], ex) : make_float2(o.v[1], o.v[2]);
                    lo = add2(lo, add2(make_float2(o.v[0], o.v[1]), slo));
                    hi = add2(hi, add2(make_float2(o.v[2], o.v[3]), shi));
                }
                hc[c][0] = lo.x; hc[c][1] = lo.y; hc[c][2] = hi.x; hc[c][3] = hi.y;
            }
            uint32_t w0[4], w1[4];
#pragma unroll
            for (int kk = 0; kk < 4; kk += 2) philox4x32_10(key, site0 + (uint32_t)kk, c1, c2, c3, w0[kk], w1[kk], w0[kk + 1], w1[kk + 1]);
            Pack<4> nxv = sx, nyv = sy, nzv = sz;
#pragma unroll
            for (int kp = 0; kp < 4; kp += 2) {
                V3p S = { make_float2(sx.v[kp], sx.v[kp + 1]), make_float2(sy.v[kp], sy.v[kp + 1]), make_float2(sz.v[kp], sz.v[kp + 1]) };
                const V3p hp = { make_float2(hc[0][kp], hc[0][kp + 1]), make_float2(hc[1][kp], hc[1][kp + 1]), make_float2(hc[2][kp], hc[2][kp + 1]) };
                const f2 J2 = splat(P.J);
                const V3p hJ = { mul2(J2, hp.x), mul2(J2, hp.y), mul2(J2, hp.z) };
                const V3p ep = (ANISO & 1) ? e2 : B2;
                V3p d, Sn;
                cone_move2(S, omc, make_float2(uniform01(w0[kp]), uniform01(w0[kp + 1])),
                           make_float2(uniform_azimuth(w0[kp], w1[kp]), uniform_azimuth(w0[kp + 1], w1[kp + 1])), d, Sn);
                const V3p hB = { add2(hJ.x, B2.x), add2(hJ.y, B2.y), add2(hJ.z, B2.z) };
                f2 s4S, s4v, euS, euv;
                const f2 dE = delta_energy2_keep<ANISO>(S, d, hB, P.Ku, ep, P.Kc, s4S, s4v, euS, euv);
                const f2 xx = fma2(dE, splat(invT), make_float2(__logf(uniform01(w1[kp])), __logf(uniform01(w1[kp + 1]))));
                const bool ok0 = xx.x < 0.0f, ok1 = xx.y < 0.0f;
                S.x = make_float2(ok0 ? Sn.x.x : S.x.x, ok1 ? Sn.x.y : S.x.y);
                S.y = make_float2(ok0 ? Sn.y.x : S.y.x, ok1 ? Sn.y.y : S.y.y);
                S.z = make_float2(ok0 ? Sn.z.x : S.z.x, ok1 ? Sn.z.y : S.z.y);
                nxv.v[kp] = S.x.x; nxv.v[kp + 1] = S.x.y; nyv.v[kp] = S.y.x; nyv.v[kp + 1] = S.y.y; nzv.v[kp] = S.z.x; nzv.v[kp + 1] = S.z.y;
                cnt += (int)ok0 + (int)ok1;
                if (DEBUG) {
                    if (dbg_x)   { dbg_x[site0 + kp] = xx.x; dbg_x[site0 + kp + 1u] = xx.y; }
                    if (dbg_acc) { dbg_acc[site0 + kp] = (uint8_t)ok0; dbg_acc[site0 + kp + 1u] = (uint8_t)ok1; }
                }
                aM[0] = add2(aM[0], S.x); aM[1] = add2(aM[1], S.y); aM[2] = add2(aM[2], S.z);
                if (colour == 1) aEx = sub2(aEx, dot3p(S, hJ));
                if (ANISO) aAn = add2(aAn, onsite_from<ANISO>(ok0, ok1, s4S, s4v, euS, euv, P.Ku, P.Kc));
                aZe = sub2(aZe, dot3p(S, B2));
            }
            st_rw<4>(pS, nxv); st_rw<4>(pS + P.plane, nyv); st_rw<4>(pS + 2 * P.plane, nzv);
#pragma unroll
            for (int c = 0; c < 3; ++c) { car0[c] = new0[c]; car1[c] = new1[c]; }
            pS += ms; pR0 += ms; pR1 += ms; site0 += (uint32_t)ms;
        }
    }
    float f[NQ];
    f[0] = aM[0].x + aM[0].y; f[1] = aM[1].x + aM[1].y; f[2] = aM[2].x + aM[2].y;
    f[3] = aEx.x + aEx.y; f[4] = aAn.x + aAn.y; f[5] = aZe.x + aZe.y;
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
