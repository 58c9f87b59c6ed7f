// mc_common.cuh -- what every kernel of the checkerboard Metropolis path shares: the data layout, the controller /
// reduction state, the colour indexing (a-1), the exchange-field gather (a-3) and the fused per-sweep reductions with the
// cone controller (a-7, a-8, a-9).  The kernels: mc_pass.cuh (Table A1, generic), mc_tile.cuh (Table A1,
// staged), mc_pair.cuh (Table A2), mc_util.cuh (layout conversion, state edits, slice profile).
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

// basis mode (C-32): the bonds of a site of a sublattice, grouped by the ROW of cells they reach = (other sublattice b, cell
// offset dy, dz); xmask: bit 0 / 1 / 2 set <=> the row holds a bond at cell offset dx = -1 / 0 / +1 (same coupling J: b fixes the
// bond length).  Rows into sublattices b < a come first (n_lower of them): their partial field is the part of E_exch this pass owns.
constexpr int MC_MAX_BONDS = 18;
struct BondEntry { signed char b, xmask, dy, dz; float J; };
// The same table before the couplings are filled in, derived from the coordinates -- every (sublattice b, cell offset in {-1,0,1}^3)
// whose separation from a site of sublattice a has a bonding length.  hcp (structure 3): orthohexagonal cell doubled along x,
// units (a/2, sqrt3 a/6, c/2), ideal c/a: |r|^2 = a^2/12 (3 dx^2 + dy^2 + 8 dz^2), nearest neighbours at |r| = a (kind 1).
// sc + next-nearest neighbours (structure 4): the 2 x 2 x 2 block as the cell, |r|^2 = 1 (kind 1: J) and 2 (kind 2: J2).
// constexpr: mc_api.cu evaluates it at run time for the table it uploads, the compile-time instantiations of the pass evaluate it
// in the compiler.  ok = false if a bond stays inside the sublattice or the bond count is not 12 / 18.
struct BondRowCT { int b, xmask, dy, dz, kind; };
struct BondTableCT { BondRowCT row[MC_MAX_BONDS]; int n, nlower; bool ok; };
__host__ __device__ constexpr int hcp_basis_pos(int s, int ax)
{
    // (0,0,0) (1,3,0) (1,1,1) (0,4,1) and the same + (2,0,0)
    const int x = ((s & 3) == 1 || (s & 3) == 2 ? 1 : 0) + (s >= 4 ? 2 : 0);
    const int y = (s & 3) == 0 ? 0 : (s & 3) == 1 ? 3 : (s & 3) == 2 ? 1 : 4;
    const int z = (s & 3) >= 2 ? 1 : 0;
    return ax == 0 ? x : ax == 1 ? y : z;
}
__host__ __device__ constexpr BondTableCT make_bond_table(int structure, int a)
{
    BondTableCT T{};
    const bool hcp = structure == 3;
    const int cell[3] = { hcp ? 4 : 2, hcp ? 6 : 2, 2 }, w[3] = { hcp ? 3 : 1, 1, hcp ? 8 : 1 };
    int rows = 0, bonds = 0, lower = 0;
    bool ok = true;
    for (int pass = 0; pass < 2; ++pass)                                 // rows into lower sublattices first
        for (int b = 0; b < 8; ++b) {
            if ((b < a) != (pass == 0)) continue;
            for (int o = 0; o < 9; ++o) {
                const int dy = o % 3 - 1, dz = o / 3 - 1;
                int mask = 0, kind = 0;
                for (int dx = -1; dx <= 1; ++dx) {
                    const int d[3] = { dx, dy, dz };
                    int q = 0;
                    for (int ax = 0; ax < 3; ++ax) {
                        const int ra = hcp ? hcp_basis_pos(a, ax) : (a >> ax) & 1, rb = hcp ? hcp_basis_pos(b, ax) : (b >> ax) & 1;
                        const int sep = rb + d[ax] * cell[ax] - ra;
                        q += w[ax] * sep * sep;
                    }
                    if (hcp) { if (q != 12) continue; kind = 1; }
                    else if (q == 1) kind = 1; else if (q == 2) kind = 2; else continue;
                    if (b == a) ok = false;
                    mask |= 1 << (dx + 1); ++bonds;
                }
                if (!mask) continue;
                if (rows == MC_MAX_BONDS) { ok = false; continue; }
                T.row[rows].b = b; T.row[rows].xmask = mask; T.row[rows].dy = dy; T.row[rows].dz = dz; T.row[rows].kind = kind;
                ++rows;
                if (b < a) ++lower;
            }
        }
    T.n = rows; T.nlower = lower; T.ok = ok && bonds == (hcp ? 12 : 18);
    return T;
}

struct Params {
    int nx, ny, nz, R;               // R = nx/2 sites of one colour per row
    int anti_x;                      // 1: anti-periodic boundary along x (domain-wall box); the wrap bond sees -S_j
    int per_mask;                    // bit a set: axis a (x, y, z) is periodic (or anti-periodic)
    int fcc;                         // 1: face-centred cubic (C-31): FOUR colours = sublattices, R = nx, 12 neighbours
    int ncol;                        // colours swept per Monte Carlo iteration: 2 (sc, bcc), 4 (fcc)
    int bcc;                         // 1: body-centred cubic (C-30): colour = sublattice, R = nx cells per row, 8 neighbours
    int basis;                       // MC_HCP / MC_SC_NNN (C-32): EIGHT colours = sublattices of an eight-site cell, bonds from the table
    int sub;                         // 1: colours are sublattices stored as full grids of cells (bcc, fcc, basis): site = colour * Nc + cell
    const BondEntry* bonds;          // basis: [8][MC_MAX_BONDS] bonds of a site of every sublattice (device memory in the workspace)
    unsigned char nbonds[8], nlower[8];   // rows of the table per sublattice; how many of them lead into lower sublattices
    uint32_t Nc;                     // sites per colour
    uint32_t N;
    double invN;                     // 1 / N (host-computed: keeps an fp64 division off the finalising thread)
    long long plane;                 // floats between component planes
    float* S;                        // 6 planes: colour-major, then component
    const uint8_t* mask;   long long mask_plane;     // [2][mask_plane] colour-split bond masks (or null)
    const uint16_t* region; long long region_plane;  // [2][region_plane] colour-split grain ids (or null)
    const float4* axis;              // [n_regions] easy axes
    float J, Ku, Kc;
    float J2;                        // next-nearest-neighbour coupling (MC_SC_NNN)
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
template <> __device__ __forceinline__ Pack<2> ld_nc<2>(const float* p)
{
    const float2 t = __ldg(reinterpret_cast<const float2*>(p));
    Pack<2> r; r.v[0] = t.x; r.v[1] = t.y; return r;
}
template <int VEC> __device__ __forceinline__ Pack<VEC> ld_rw(const float* p);
template <> __device__ __forceinline__ Pack<2> ld_rw<2>(const float* p)
{
    const float2 t = *reinterpret_cast<const float2*>(p);
    Pack<2> r; r.v[0] = t.x; r.v[1] = t.y; return r;
}
template <> __device__ __forceinline__ Pack<1> ld_rw<1>(const float* p) { Pack<1> r; r.v[0] = *p; return r; }
template <> __device__ __forceinline__ Pack<4> ld_rw<4>(const float* p)
{
    const float4 t = *reinterpret_cast<const float4*>(p);
    Pack<4> r; r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w; return r;
}
template <int VEC> __device__ __forceinline__ void st_rw(float* p, const Pack<VEC>& r);
template <> __device__ __forceinline__ void st_rw<2>(float* p, const Pack<2>& r) { *reinterpret_cast<float2*>(p) = make_float2(r.v[0], r.v[1]); }
template <> __device__ __forceinline__ void st_rw<1>(float* p, const Pack<1>& r) { *p = r.v[0]; }
template <> __device__ __forceinline__ void st_rw<4>(float* p, const Pack<4>& r)
{
    *reinterpret_cast<float4*>(p) = make_float4(r.v[0], r.v[1], r.v[2], r.v[3]);
}

// the same store with the evict-first ("streaming") policy: the written spins are not read again before the next pass has swept
// the whole other colour.  Pays on the bcc pass only (176^3 cells: 98.6 -> 95.1 us per sweep, 224^3: 187.6 -> 179.5); the film
// (159 -> 178), the march pass (89.4 -> 92.2) and the eight-colour passes (no change) keep the default policy.
__device__ __forceinline__ void st_rw_streaming(float* p, const Pack<4>& r)
{
    __stcs(reinterpret_cast<float4*>(p), make_float4(r.v[0], r.v[1], r.v[2], r.v[3]));
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

// --------------------------------------------------------------------------------------------------------------
// bcc (C-30): the two simple cubic sublattices are the two colours; each is stored as a full nx x ny x nz grid in
// cell order a = i + nx (j + ny k) (R = nx).  The 8 neighbours of A(i,j,k) are B(i-dx, j-dy, k-dz), those of B(i,j,k) are
// A(i+dx, j+dy, k+dz): the cells i and i -+ 1 of four rows of the other sublattice.  An item is 4 consecutive cells of a row:
// per row one float4 plus the one value just outside the item.  Fully periodic lattices only.
// Site ids (Philox counters, debug outputs): sublattice*Ncell + cell; the cells i, i ^ 1 share a Philox block (C-30).
// --------------------------------------------------------------------------------------------------------------
struct BccPos {
    uint32_t a0, site0;              // cell index of the first cell of the item; its site id
    uint32_t row[4];                 // first cell of the rows (j, k), (j', k), (j, k'), (j', k') of the other sublattice; ' = -1 (A) / +1 (B)
    uint32_t xe;                     // in-row cell of the value outside the item: i0 - 1 (A) or i0 + 4 (B), wrapped
    uint32_t i0;
};
__device__ __forceinline__ BccPos bcc_locate(const Params& P, const Geom& G, uint32_t item, int colour)
{
    uint32_t rowp, xq, z, y;
    G.div_rv.divmod(item, rowp, xq);
    const uint32_t nx = (uint32_t)P.nx, ny = (uint32_t)P.ny, nz = (uint32_t)P.nz;
    z = rowp / ny; y = rowp - z * ny;
    BccPos q;
    q.i0 = xq * 4u;
    q.a0 = rowp * nx + q.i0;
    q.site0 = (uint32_t)colour * P.Nc + q.a0;
    const uint32_t y2 = colour ? (y + 1 == ny ? 0u : y + 1) : (y == 0 ? ny - 1 : y - 1);
    const uint32_t z2 = colour ? (z + 1 == nz ? 0u : z + 1) : (z == 0 ? nz - 1 : z - 1);
    q.row[0] = (z * ny + y) * nx;  q.row[1] = (z * ny + y2) * nx;
    q.row[2] = (z2 * ny + y) * nx; q.row[3] = (z2 * ny + y2) * nx;
    q.xe = colour ? (q.i0 + 4 == nx ? 0u : q.i0 + 4) : (q.i0 == 0 ? nx - 1 : q.i0 - 1);
    return q;
}
// h = sum of the 8 neighbours (WITHOUT the factor J), in a fixed order: rows 0..3, in each the cell i then the cell i -+ 1
__device__ __forceinline__ void bcc_exchange_field(const Params& P, const BccPos& q, int colour, Vec3 (&h)[4])
{
    const float* O = P.S + (long long)(1 - colour) * 3 * P.plane;
    float hc[3][4];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float* Oc = O + (long long)c * P.plane;
        f2 lo = splat(0.0f), hi = splat(0.0f);
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const Pack<4> o = ld_nc<4>(Oc + q.row[r] + q.i0);
            const float ex = __ldg(Oc + q.row[r] + q.xe);
            // shifted neighbour: cell i - 1 (sublattice A) or i + 1 (sublattice B)
            const f2 slo = colour ? make_float2(o.v[1], o.v[2]) : make_float2(ex, o.v[0]);
            const f2 shi = colour ? make_float2(o.v[3], ex) : make_float2(o.v[1], o.v[2]);
            lo = add2(lo, add2(make_float2(o.v[0], o.v[1]), slo));
            hi = add2(hi, add2(make_float2(o.v[2], o.v[3]), shi));
        }
        hc[c][0] = lo.x; hc[c][1] = lo.y; hc[c][2] = hi.x; hc[c][3] = hi.y;
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) h[k] = { hc[0][k], hc[1][k], hc[2][k] };
}

// --------------------------------------------------------------------------------------------------------------
// fcc (C-31): four simple cubic sublattices = FOUR colours, each a full nx x ny x nz grid in cell order (R = nx):
// sublattice 0 at the cell corner, 1 at (0,1/2,1/2), 2 at (1/2,0,1/2), 3 at (1/2,1/2,0).  A site has 4 neighbours in each
// OTHER sublattice b: the offsets of a and b differ along two axes; along such an axis the neighbour's cell index is
// {i, i - 1} if a sits at 0 and b at 1/2, {i, i + 1} the other way round.  An item is 4 consecutive cells of a row; if x
// is one of the two axes a sublattice costs 2 rows x (float4 + the one cell outside the item), else 4 rows x float4.
// hl collects the neighbours in sublattices b < a only: E_exch = -J sum_a sum_{i in a} S_i . hl_i counts every bond once,
// in the pass of its higher colour, when both ends are final.
// --------------------------------------------------------------------------------------------------------------
struct FccPos { uint32_t a0, site0, i0, y, z; };
__device__ __forceinline__ FccPos fcc_locate(const Params& P, const Geom& G, uint32_t item, int colour)
{
    uint32_t rowp, xq;
    G.div_rv.divmod(item, rowp, xq);
    FccPos q;
    q.z = rowp / (uint32_t)P.ny; q.y = rowp - q.z * (uint32_t)P.ny;
    q.i0 = xq * 4u;
    q.a0 = rowp * (uint32_t)P.nx + q.i0;
    q.site0 = (uint32_t)colour * P.Nc + q.a0;
    return q;
}
__device__ __forceinline__ void fcc_exchange_field(const Params& P, const FccPos& q, int colour, Vec3 (&h)[4], Vec3 (&hl)[4])
{
    const uint32_t nx = (uint32_t)P.nx, ny = (uint32_t)P.ny, nz = (uint32_t)P.nz;
    const uint32_t offm_tab = 0x3560u;                               // offsets as bit masks (bit 0 x, 1 y, 2 z): sublattice 0: 0, 1: 6, 2: 5, 3: 3
    const uint32_t oa = (offm_tab >> (4 * colour)) & 7u;
    float hc[3][4], hlc[3][4];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int k = 0; k < 4; ++k) { hc[c][k] = 0.0f; hlc[c][k] = 0.0f; }
#pragma unroll
    for (int r = 0; r < 3; ++r) {
        const int b = r + (r >= colour ? 1 : 0);
        const uint32_t ob = (offm_tab >> (4 * b)) & 7u, D = oa ^ ob;
        const float* O = P.S + (long long)b * 3 * P.plane;
        // the second row / plane of the pair along a differing axis: +1 if a sits at 1/2, -1 if at 0
        const uint32_t y2 = (D & 2u) ? ((oa & 2u) ? (q.y + 1 == ny ? 0u : q.y + 1) : (q.y == 0 ? ny - 1 : q.y - 1)) : q.y;
        const uint32_t z2 = (D & 4u) ? ((oa & 4u) ? (q.z + 1 == nz ? 0u : q.z + 1) : (q.z == 0 ? nz - 1 : q.z - 1)) : q.z;
        const bool xs = (D & 1u) != 0, xplus = (oa & 1u) != 0;
        const uint32_t xe = xplus ? (q.i0 + 4 == nx ? 0u : q.i0 + 4) : (q.i0 == 0 ? nx - 1 : q.i0 - 1);
        const uint32_t rows[4] = { (q.z * ny + q.y) * nx, (q.z * ny + y2) * nx, (z2 * ny + q.y) * nx, (z2 * ny + y2) * nx };
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const float* Oc = O + (long long)c * P.plane;
            float s[4] = { 0.f, 0.f, 0.f, 0.f };
            if (xs) {                                                // x and one of y, z differ: rows (y,z) and (y2,z2); cells i and i -+ 1
#pragma unroll
                for (int rr = 0; rr < 4; rr += 3) {
                    const Pack<4> o = ld_nc<4>(Oc + rows[rr] + q.i0);
                    const float ex = __ldg(Oc + rows[rr] + xe);
                    s[0] += o.v[0] + (xplus ? o.v[1] : ex);   s[1] += o.v[1] + (xplus ? o.v[2] : o.v[0]);
                    s[2] += o.v[2] + (xplus ? o.v[3] : o.v[1]); s[3] += o.v[3] + (xplus ? ex : o.v[2]);
                }
            } else {                                                 // y and z differ: the four rows, cell i
#pragma unroll
                for (int rr = 0; rr < 4; ++rr) {
                    const Pack<4> o = ld_nc<4>(Oc + rows[rr] + q.i0);
#pragma unroll
                    for (int k = 0; k < 4; ++k) s[k] += o.v[k];
                }
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) { hc[c][k] += s[k]; if (b < colour) hlc[c][k] += s[k]; }
        }
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) { h[k] = { hc[0][k], hc[1][k], hc[2][k] }; hl[k] = { hlc[0][k], hlc[1][k], hlc[2][k] }; }
}

// --------------------------------------------------------------------------------------------------------------
// basis mode (C-32: hcp, simple cubic with next-nearest neighbours): eight sublattices = EIGHT colours, each a full
// nx x ny x nz grid of cells (R = nx).  The bonds of a site of sublattice a come from a table the host derived from the
// coordinates: (sublattice b, cell offset (dx,dy,dz), coupling J_b).  An item is 4 consecutive cells of a row; a bond with
// dx = 0 costs one float4 per component, dx = +-1 a float4 plus the one cell outside the item.  h INCLUDES the couplings
// (they differ per bond); hl collects the bonds into sublattices b < a (E_exch counts every bond once, as for fcc).
// --------------------------------------------------------------------------------------------------------------
#ifndef MC_BASIS_UNROLL
#define MC_BASIS_UNROLL 4      // rows of the table in flight together (112^3 cells of hcp, us per sweep: 1: 388, 2: 352, 4: 337, 6: 353)
#endif
__device__ __forceinline__ void basis_exchange_field(const Params& P, const FccPos& q, int colour, Vec3 (&h)[4], Vec3 (&hl)[4])
{
    const uint32_t nx = (uint32_t)P.nx, ny = (uint32_t)P.ny, nz = (uint32_t)P.nz;
    float hc[3][4];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int k = 0; k < 4; ++k) hc[c][k] = 0.0f;
    const int2* tab = reinterpret_cast<const int2*>(P.bonds + colour * MC_MAX_BONDS);
    const int n = P.nbonds[colour], nlow = P.nlower[colour];
    const uint32_t xm = q.i0 == 0 ? nx - 1 : q.i0 - 1, xp = q.i0 + 4 == nx ? 0u : q.i0 + 4;      // the cells just outside the item
    auto row = [&](int e) {
        const int2 raw = __ldg(tab + e);
        const int b = raw.x & 0xFF, m = (raw.x >> 8) & 0xFF;
        const int dy = (int)(signed char)((raw.x >> 16) & 0xFF), dz = (int)(signed char)((raw.x >> 24) & 0xFF);
        const float J = __int_as_float(raw.y);
        const float Jm = (m & 1) ? J : 0.0f, J0 = (m & 2) ? J : 0.0f, Jp = (m & 4) ? J : 0.0f;
        const uint32_t y2 = dy > 0 ? (q.y + 1 == ny ? 0u : q.y + 1) : dy < 0 ? (q.y == 0 ? ny - 1 : q.y - 1) : q.y;
        const uint32_t z2 = dz > 0 ? (q.z + 1 == nz ? 0u : q.z + 1) : dz < 0 ? (q.z == 0 ? nz - 1 : q.z - 1) : q.z;
        const float* O = P.S + (long long)b * 3 * P.plane + (z2 * ny + y2) * nx;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const float* Oc = O + (long long)c * P.plane;
            // branch-free: the three candidate cells of every site are always fetched (the two outside the item are L1 hits of the
            // neighbouring items' float4) and weighted with J or 0, so that the loads of several rows can be in flight together
            const Pack<4> o = ld_nc<4>(Oc + q.i0);
            const float em = __ldg(Oc + xm), ep = __ldg(Oc + xp);
            hc[c][0] = fmaf(Jm, em,     fmaf(J0, o.v[0], fmaf(Jp, o.v[1], hc[c][0])));
            hc[c][1] = fmaf(Jm, o.v[0], fmaf(J0, o.v[1], fmaf(Jp, o.v[2], hc[c][1])));
            hc[c][2] = fmaf(Jm, o.v[1], fmaf(J0, o.v[2], fmaf(Jp, o.v[3], hc[c][2])));
            hc[c][3] = fmaf(Jm, o.v[2], fmaf(J0, o.v[3], fmaf(Jp, ep,     hc[c][3])));
        }
    };
    constexpr int UNR = MC_BASIS_UNROLL;
#pragma unroll UNR
    for (int e = 0; e < nlow; ++e) row(e);
#pragma unroll
    for (int k = 0; k < 4; ++k) hl[k] = { hc[0][k], hc[1][k], hc[2][k] };
#pragma unroll UNR
    for (int e = nlow; e < n; ++e) row(e);
#pragma unroll
    for (int k = 0; k < 4; ++k) h[k] = { hc[0][k], hc[1][k], hc[2][k] };
}

// The same field with the table as a compile-time constant (STRUCT 3 hcp / 4 sc + next-nearest neighbours, COL the sublattice):
// the rows are unrolled, the wrapped y / z indices are computed once, a row loads the cells outside the item only where it has a
// bond to them, and the neighbours of a row are summed before ONE multiplication by its coupling.
template <int STRUCT, int COL, int ROW>
__device__ __forceinline__ void basis_rows_ct(const Params& P, const FccPos& q, const uint32_t (&yy)[3], const uint32_t (&zz)[3],
                                              uint32_t xm, uint32_t xp, float (&hc)[3][4], Vec3 (&hl)[4])
{
    constexpr BondTableCT T = make_bond_table(STRUCT, COL);
    static_assert(T.ok, "basis mode: a bond inside a sublattice");
    if constexpr (ROW == T.nlower) {
#pragma unroll
        for (int k = 0; k < 4; ++k) hl[k] = { hc[0][k], hc[1][k], hc[2][k] };
    }
    if constexpr (ROW < T.n) {
        constexpr BondRowCT r = T.row[ROW];
        const float J = r.kind == 1 ? P.J : P.J2;
        const float* O = P.S + (long long)r.b * 3 * P.plane + (zz[r.dz + 1] * (uint32_t)P.ny + yy[r.dy + 1]) * (uint32_t)P.nx;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const float* Oc = O + (long long)c * P.plane;
            const Pack<4> o = ld_nc<4>(Oc + q.i0);
            float s[4] = { 0.f, 0.f, 0.f, 0.f };
            if constexpr ((r.xmask & 2) != 0) { s[0] = o.v[0]; s[1] = o.v[1]; s[2] = o.v[2]; s[3] = o.v[3]; }
            if constexpr ((r.xmask & 1) != 0) { const float em = __ldg(Oc + xm); s[0] += em; s[1] += o.v[0]; s[2] += o.v[1]; s[3] += o.v[2]; }
            if constexpr ((r.xmask & 4) != 0) { const float ep = __ldg(Oc + xp); s[0] += o.v[1]; s[1] += o.v[2]; s[2] += o.v[3]; s[3] += ep; }
#pragma unroll
            for (int k = 0; k < 4; ++k) hc[c][k] = fmaf(J, s[k], hc[c][k]);
        }
        basis_rows_ct<STRUCT, COL, ROW + 1>(P, q, yy, zz, xm, xp, hc, hl);
    }
}
template <int STRUCT, int COL>
__device__ __forceinline__ void basis_exchange_field_ct(const Params& P, const FccPos& q, Vec3 (&h)[4], Vec3 (&hl)[4])
{
    const uint32_t nx = (uint32_t)P.nx, ny = (uint32_t)P.ny, nz = (uint32_t)P.nz;
    const uint32_t yy[3] = { q.y == 0 ? ny - 1 : q.y - 1, q.y, q.y + 1 == ny ? 0u : q.y + 1 };
    const uint32_t zz[3] = { q.z == 0 ? nz - 1 : q.z - 1, q.z, q.z + 1 == nz ? 0u : q.z + 1 };
    const uint32_t xm = q.i0 == 0 ? nx - 1 : q.i0 - 1, xp = q.i0 + 4 == nx ? 0u : q.i0 + 4;
    float hc[3][4];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int k = 0; k < 4; ++k) hc[c][k] = 0.0f;
    basis_rows_ct<STRUCT, COL, 0>(P, q, yy, zz, xm, xp, hc, hl);
#pragma unroll
    for (int k = 0; k < 4; ++k) h[k] = { hc[0][k], hc[1][k], hc[2][k] };
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

// The generic kernels keep the fixed-point sums of a thread in shared memory (column threadIdx.x of [NQ][threads per CTA]: no bank
// conflicts) instead of 18 registers: they are short of registers (spills), and the sums are touched once per
// FLUSH_ITEMS items.
template <int W>
__device__ __forceinline__ void fx_flush_shared(long long (*sacc)[W], float (&f)[NQ], float scale)
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

// 1 - cos(cone) for the cone move (C-6), cone in [0, pi]: 2 sin^2(cone / 2) with sin from its Taylor series to h^17 (h <= pi/2:
// truncation < 5e-14, far below the fp32 it is rounded to).  Straight-line fma code, the same bits on the host (mc_create) and on
// the device (mc_set_cone, end-of-sweep controller): the library routine cos() in fp64 is a call into cold code with table
// look-ups on the one thread the whole grid waits for -- 0.8-2 us per sweep at the tail of the last colour pass.
__host__ __device__ inline float one_minus_cos_of(double cone)
{
    const double h = 0.5 * cone, z = h * h;
    double p = -1.0 / 355687428096000.0;                       // -1/17!
    p = fma(p, z, 1.0 / 1307674368000.0);                       // +1/15!
    p = fma(p, z, -1.0 / 6227020800.0);                         // -1/13!
    p = fma(p, z, 1.0 / 39916800.0);                            // +1/11!
    p = fma(p, z, -1.0 / 362880.0);                             // -1/9!
    p = fma(p, z, 1.0 / 5040.0);                                // +1/7!
    p = fma(p, z, -1.0 / 120.0);                                // -1/5!
    p = fma(p, z, 1.0 / 6.0);                                   // +1/3!  (sign folded below)
    const double s = h * fma(-p, z, 1.0);                       // sin h = h (1 - z/3! + z^2/5! - ...)
    return (float)(2.0 * s * s);
}

// Pass 2 of the reduction (one block, fixed order) + what follows a sweep: cone controller (P:168-171 read with
// P:205-209; C-2, C-3, C-9), sweep counter, Eq. (6) accumulators, trace row.  mode 0: end of a sweep; 1: measurement.
// Pass 1 left exact fixed-point totals in DevState.isum; here they become fp64.  This block runs alone at the tail of
// the black pass, so its latency is exposed: the controller state is staged through shared memory with one coalesced
// read and one coalesced write (two L2 round trips instead of a chain of dependent ones), thread 0 does the scalar
// work on the shared copy.
static_assert(sizeof(DevState) % 4 == 0, "DevState is staged as 32-bit words");
static __device__ __noinline__ void final_reduce(const Params& P, int mode, int flags)
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
        omc_next[0] = one_minus_cos_of(up); omc_next[1] = one_minus_cos_of(dn);
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


}  // namespace mc
