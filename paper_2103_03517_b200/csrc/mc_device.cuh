// mc_device.cuh -- per-update device arithmetic of the checkerboard Metropolis path (sm_100a, fp32).
//
// Every function cites the passage of arXiv 2103.03517 it implements ("P:NN" = line of /root/reference/PAPER.md)
// and the reading in DESIGN.md section 4 ("C-n").  This file shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace mc {

// Programmatic dependent launch (sm_90+): a grid launched with the programmatic-stream-serialization attribute may be
// scheduled while its predecessor drains; griddepcontrol.wait blocks until the predecessor has completed and its writes
// are visible, launch_dependents lets the successor be scheduled in turn.  Both are no-ops in an ordinary launch.
// Every pass kernel calls this before it touches anything a previous kernel wrote.
__device__ __forceinline__ void grid_dependency_sync()
{
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;");
}

// Stream tags (counter word 1, low byte); colour goes to bits 8..
constexpr uint32_t TAG_MOVE = 0u, TAG_PAIR = 1u, TAG_PAIRING = 2u, TAG_INIT = 3u;

// ---------------------------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11): 10 rounds of
//   (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)),  (k0,k1) += (W0,W1) after each round.
// 2 IMAD.WIDE + 2 LOP3 per round; the key schedule is uniform across the grid.
// ---------------------------------------------------------------------------------------------------------------
struct PhiloxKey {            // the 10 round keys, precomputed once per thread from (seed_lo, seed_hi): uniform registers
    uint32_t k0[10], k1[10];
};

__host__ __device__ __forceinline__ PhiloxKey philox_key(uint32_t seed_lo, uint32_t seed_hi)
{
    PhiloxKey k;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        k.k0[r] = seed_lo + 0x9E3779B9u * (uint32_t)r;
        k.k1[r] = seed_hi + 0xBB67AE85u * (uint32_t)r;
    }
    return k;
}

__device__ __forceinline__ void philox4x32_10(const PhiloxKey& k, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k.k0[r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k.k1[r];
        c1 = (uint32_t)p1; c3 = (uint32_t)p0; c0 = n0; c2 = n2;
    }
    r0 = c0; r1 = c1; r2 = c2; r3 = c3;
}

// u = ((r >> 9) + 0.5) * 2^-23 in (0,1), exactly representable in fp32 (C-8).
// Bit trick: (r>>9) | 0x3f800000 is the float 1 + k*2^-23; subtracting (1 - 2^-24) is exact.
__device__ __forceinline__ float uniform01(uint32_t r)
{
    return __uint_as_float((r >> 9) | 0x3f800000u) - 0.99999994f;
}

// ---------------------------------------------------------------------------------------------------------------
// The uniforms of one unconstrained update (C-26).  Two same-colour x-neighbours of a row (x and x ^ 2) share one
// Philox block whose counter word 0 is the lexicographic index of the one with bit 1 of x clear; that site takes
// words (0,1), the other words (2,3).  From its words (w0,w1):
//   u0 = ((w0 >> 9) + 0.5) 2^-23,  u2 = ((w1 >> 9) + 0.5) 2^-23,  u1 = (((w0 & 511) << 9) | (w1 & 511)) 2^-18.
// Why: IMAD.WIDE.U32 issues once per ~6 cycles per SM sub-partition on sm_100a (measured), so the 20 wide multiplies
// of a Philox call cost as much as all the fp32 arithmetic of an update; 64 bits per update halve that.
// ---------------------------------------------------------------------------------------------------------------
// 1 + u1 as a float in [1,2): exponent | 9 low bits of w0 | 9 low bits of w1 | 00000   (one LOP3, one SHF.L, one SHF.R.W)
__device__ __forceinline__ float azimuth_1p(uint32_t w0, uint32_t w1)
{
    return __uint_as_float(__funnelshift_r(w1 << 23, (w0 & 0x1FFu) | 0xFE00u, 18));
}
__device__ __forceinline__ float uniform_azimuth(uint32_t w0, uint32_t w1) { return azimuth_1p(w0, w1) - 1.0f; }

struct Vec3 { float x, y, z; };

__device__ __forceinline__ float dot3(const Vec3& a, const Vec3& b) { return fmaf(a.x, b.x, fmaf(a.y, b.y, a.z * b.z)); }

// ---------------------------------------------------------------------------------------------------------------
// Cone trial move (C-6 half-angle, C-7 uniform in solid angle).
//   w = u0 (1 - cos theta) = 1 - cos(alpha);  sin(alpha) = sqrt(w (2 - w));  phi = 2 pi u1;
//   frame (t1,t2) perpendicular to S: Duff et al. 2017 branch-light construction;
//   d = -w S + sin(alpha) (cos(phi) t1 + sin(phi) t2);   S' = (S + d)/|S + d|.
// Returns d (used for the energy difference) and S' (stored if accepted).
// sin/cos: MUFU on phi - pi in (-pi, pi) where sin.approx / cos.approx are most accurate (abs err ~5e-7);
// sin(phi) = -sin(phi - pi), cos(phi) = -cos(phi - pi).
// |S + d|^2 = 1 + eps with |eps| ~ 1e-6 (rounding only), so 1/|S+d| = 1.5 - 0.5 |S+d|^2 to O(eps^2): one FFMA, no MUFU.
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void cone_move(const Vec3& S, float one_minus_cos, float u0, float u1, Vec3& d, Vec3& Sn)
{
    const float w  = u0 * one_minus_cos;
    const float t  = w * (2.0f - w);
    const float sa = t * rsqrtf(t);                          // sqrt(t), t > 0 always (u0 >= 2^-24, theta >= 1 deg)
    const float ang = fmaf(u1, 6.2831853071795865f, -3.1415926535897932f);
    const float cp = -__cosf(ang), sp = -__sinf(ang);
    const float sg = copysignf(1.0f, S.z);                   // sign BIT of S_z (C-29): -0.0 gives -1, as in the packed paths
    const float a  = __fdividef(-1.0f, sg + S.z);
    const float b  = S.x * S.y * a;
    const Vec3 t1 = { fmaf(sg * S.x * S.x, a, 1.0f), sg * b, -sg * S.x };
    const Vec3 t2 = { b, fmaf(S.y * S.y, a, sg), -S.y };
    const float ca = sa * cp, cb = sa * sp;
    d.x = fmaf(ca, t1.x, fmaf(cb, t2.x, -w * S.x));
    d.y = fmaf(ca, t1.y, fmaf(cb, t2.y, -w * S.y));
    d.z = fmaf(ca, t1.z, fmaf(cb, t2.z, -w * S.z));
    const Vec3 v = { S.x + d.x, S.y + d.y, S.z + d.z };
    const float inv = fmaf(-0.5f, dot3(v, v), 1.5f);
    Sn.x = v.x * inv; Sn.y = v.y * inv; Sn.z = v.z * inv;
}

// ---------------------------------------------------------------------------------------------------------------
// Energy difference E_i(S+d) - E_i(S) of Eq. (2), in DIFFERENCE FORM (no cancellation of O(1) terms):
//   exchange + Zeeman : -d.(h + B),  h = sum_j J_ij S_j (full J per bond, C-1)
//   uniaxial          : -Ku (d.e) ((2S + d).e)
//   cubic             : Sx^2Sy^2 + Sx^2Sz^2 + Sy^2Sz^2 = (1 - sum_a S_a^4)/2 on the unit sphere, so
//                       Kc * ( -1/2 sum_a d_a (2S_a + d_a) (S_a^2 + (S_a+d_a)^2) )
// ANISO: 0 none, 1 uniaxial, 2 cubic, 3 both.
// ---------------------------------------------------------------------------------------------------------------
template <int ANISO>
__device__ __forceinline__ float delta_energy(const Vec3& S, const Vec3& d, const Vec3& hB, float Ku, const Vec3& e, float Kc)
{
    float dE = -dot3(d, hB);
    if (ANISO & 1) {
        const Vec3 s2 = { fmaf(2.0f, S.x, d.x), fmaf(2.0f, S.y, d.y), fmaf(2.0f, S.z, d.z) };
        dE = fmaf(-Ku * dot3(d, e), dot3(s2, e), dE);
    }
    if (ANISO & 2) {
        const float nx = S.x + d.x, ny = S.y + d.y, nz = S.z + d.z;
        const float qx = d.x * (S.x + nx) * fmaf(S.x, S.x, nx * nx);
        const float qy = d.y * (S.y + ny) * fmaf(S.y, S.y, ny * ny);
        const float qz = d.z * (S.z + nz) * fmaf(S.z, S.z, nz * nz);
        dE = fmaf(-0.5f * Kc, qx + qy + qz, dE);
    }
    return dE;
}

// on-site energy terms of the FINAL spin, for the per-sweep reductions (P:52 average anisotropy energy)
template <int ANISO>
__device__ __forceinline__ float aniso_energy(const Vec3& S, float Ku, const Vec3& e, float Kc)
{
    float E = 0.0f;
    if (ANISO & 1) { const float se = dot3(S, e); E = -Ku * se * se; }
    if (ANISO & 2) {
        const float x2 = S.x * S.x, y2 = S.y * S.y, z2 = S.z * S.z;
        E = fmaf(Kc, fmaf(x2, y2, fmaf(x2, z2, y2 * z2)), E);
    }
    return E;
}

// torque S x H with H = -dE_i/dS_i of the on-site terms (anisotropy + Zeeman), P:54 (torque route of Ref.[15])
template <int ANISO>
__device__ __forceinline__ Vec3 onsite_torque(const Vec3& S, float Ku, const Vec3& e, float Kc, const Vec3& B)
{
    Vec3 H = B;
    if (ANISO & 1) { const float f = 2.0f * Ku * dot3(S, e); H.x = fmaf(f, e.x, H.x); H.y = fmaf(f, e.y, H.y); H.z = fmaf(f, e.z, H.z); }
    if (ANISO & 2) {
        const float x2 = S.x * S.x, y2 = S.y * S.y, z2 = S.z * S.z, g = -2.0f * Kc;
        H.x = fmaf(g * S.x, y2 + z2, H.x); H.y = fmaf(g * S.y, x2 + z2, H.y); H.z = fmaf(g * S.z, x2 + y2, H.z);
    }
    return { S.y * H.z - S.z * H.y, S.z * H.x - S.x * H.z, S.x * H.y - S.y * H.x };
}

// ---------------------------------------------------------------------------------------------------------------
// Two-wide fp32 (Blackwell FFMA2 / FADD2 / FMUL2: two independent fp32 operations in one issue slot) and the packed
// twins of the functions above: lane x and lane y are two different sites / pairs, each lane performs exactly the
// scalar function's arithmetic (fmaf <-> fma2 lane by lane).
// ---------------------------------------------------------------------------------------------------------------
typedef float2 f2;
__device__ __forceinline__ f2 add2(f2 a, f2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ f2 splat(float v) { return make_float2(v, v); }
// packed operands take no per-lane negation: a lane-wise minus would be two scalar instructions, so it is a multiply
// by -1 (exact), and a - b is one FFMA2 (-1 * b + a, exact product: the same rounding as a subtraction)
__device__ __forceinline__ f2 neg2(f2 a) { return mul2(a, splat(-1.0f)); }
__device__ __forceinline__ f2 sub2(f2 a, f2 b) { return fma2(splat(-1.0f), b, a); }

struct V3p { f2 x, y, z; };                                  // two 3-vectors, component-wise packed
__device__ __forceinline__ V3p pack3(const Vec3& a, const Vec3& b) { return { make_float2(a.x, b.x), make_float2(a.y, b.y), make_float2(a.z, b.z) }; }
__device__ __forceinline__ V3p splat3(const Vec3& a) { return { splat(a.x), splat(a.y), splat(a.z) }; }
__device__ __forceinline__ Vec3 lane3(const V3p& a, int l) { return l ? Vec3{ a.x.y, a.y.y, a.z.y } : Vec3{ a.x.x, a.y.x, a.z.x }; }
__device__ __forceinline__ f2 dot3p(const V3p& a, const V3p& b) { return fma2(a.x, b.x, fma2(a.y, b.y, mul2(a.z, b.z))); }

__device__ __forceinline__ float xor_sign(float a, float s) { return __uint_as_float(__float_as_uint(a) ^ (__float_as_uint(s) & 0x80000000u)); }   // a * copysign(1, s)

// cone_move for two sites.  Same construction as the scalar function, written with the signs folded in (as the tiled pass
// does): with phi - pi = ang, cos(phi) = -cos(ang), sin(phi) = -sin(ang), so d = sa (cos(ang) (-t1) + sin(ang) (-t2)) - w S,
//   -t1 = (q uu - 1, q vv, q),  -t2 = (Sy uu, Sy vv - sg, Sy),  q = sg Sx,  uu = Sx / (sg + Sz),  vv = Sy / (sg + Sz).
__device__ __forceinline__ void cone_move2(const V3p& S, float one_minus_cos, f2 u0, f2 u1, V3p& d, V3p& Sn)
{
    const f2 nw = mul2(u0, splat(-one_minus_cos));
    const f2 t  = mul2(nw, fma2(nw, splat(-1.0f), splat(-2.0f)));                 // w (2 - w)
    const f2 sa = mul2(t, make_float2(rsqrtf(t.x), rsqrtf(t.y)));
    const f2 ang = fma2(u1, splat(6.2831853071795865f), splat(-3.1415926535897932f));
    const f2 Cc = mul2(sa, make_float2(__cosf(ang.x), __cosf(ang.y)));
    const f2 Ss = mul2(sa, make_float2(__sinf(ang.x), __sinf(ang.y)));
    const f2 sg = make_float2(copysignf(1.0f, S.z.x), copysignf(1.0f, S.z.y));
    const f2 den = add2(sg, S.z);
    const f2 ia = make_float2(__fdividef(1.0f, den.x), __fdividef(1.0f, den.y));
    const f2 uu = mul2(S.x, ia), vv = mul2(S.y, ia);
    const f2 q  = make_float2(xor_sign(S.x.x, S.z.x), xor_sign(S.x.y, S.z.y));    // sg Sx, on the integer pipe
    const f2 nt1x = fma2(q, uu, splat(-1.0f)), nt1y = mul2(q, vv);
    const f2 nt2x = mul2(S.y, uu), nt2y = fma2(S.y, vv, make_float2(xor_sign(-1.0f, S.z.x), xor_sign(-1.0f, S.z.y)));
    d.x = fma2(Cc, nt1x, fma2(Ss, nt2x, mul2(nw, S.x)));
    d.y = fma2(Cc, nt1y, fma2(Ss, nt2y, mul2(nw, S.y)));
    d.z = fma2(Cc, q,    fma2(Ss, S.y,  mul2(nw, S.z)));
    const V3p v = { add2(S.x, d.x), add2(S.y, d.y), add2(S.z, d.z) };
    const f2 inv = fma2(dot3p(v, v), splat(-0.5f), splat(1.5f));
    Sn = { mul2(v.x, inv), mul2(v.y, inv), mul2(v.z, inv) };
}

template <int ANISO>
__device__ __forceinline__ f2 delta_energy2(const V3p& S, const V3p& d, const V3p& hB, float Ku, const V3p& e, float Kc)
{
    f2 dE = neg2(dot3p(d, hB));
    if (ANISO & 1) {
        const V3p s2 = { fma2(splat(2.0f), S.x, d.x), fma2(splat(2.0f), S.y, d.y), fma2(splat(2.0f), S.z, d.z) };
        dE = fma2(mul2(splat(-Ku), dot3p(d, e)), dot3p(s2, e), dE);
    }
    if (ANISO & 2) {
        const f2 nx = add2(S.x, d.x), ny = add2(S.y, d.y), nz = add2(S.z, d.z);
        const f2 qx = mul2(mul2(d.x, add2(S.x, nx)), fma2(S.x, S.x, mul2(nx, nx)));
        const f2 qy = mul2(mul2(d.y, add2(S.y, ny)), fma2(S.y, S.y, mul2(ny, ny)));
        const f2 qz = mul2(mul2(d.z, add2(S.z, nz)), fma2(S.z, S.z, mul2(nz, nz)));
        dE = fma2(splat(-0.5f * Kc), add2(add2(qx, qy), qz), dE);
    }
    return dE;
}

// delta_energy2 that also hands back what the on-site energy of whichever spin is kept needs, so that it is not evaluated
// again: cubic through s4 = sum_a S_a^4 of the old spin (s4S) and of the trial spin S + d (s4v) -- on the unit sphere
// Sx^2Sy^2 + Sx^2Sz^2 + Sy^2Sz^2 = (1 - s4)/2, so dE_c = -Kc/2 (s4v - s4S) and E_c = Kc/2 (1 - s4); uniaxial through
// (S.e)^2 (euS) and ((S+d).e)^2 (euv) with the difference in difference form.  E_onsite(kept) = onsite_from(...).
template <int ANISO>
__device__ __forceinline__ f2 delta_energy2_keep(const V3p& S, const V3p& d, const V3p& hB, float Ku, const V3p& e, float Kc,
                                                 f2& s4S, f2& s4v, f2& euS, f2& euv)
{
    f2 dE = neg2(dot3p(d, hB));
    s4S = s4v = euS = euv = splat(0.0f);
    if (ANISO & 1) {
        const f2 de = dot3p(d, e), se = dot3p(S, e);
        const f2 du = mul2(de, fma2(splat(2.0f), se, de));           // ((S+d).e)^2 - (S.e)^2
        dE = fma2(splat(-Ku), du, dE);
        euS = mul2(se, se); euv = add2(euS, du);
    }
    if (ANISO & 2) {
        const f2 vx = add2(S.x, d.x), vy = add2(S.y, d.y), vz = add2(S.z, d.z);
        const f2 S2x = mul2(S.x, S.x), S2y = mul2(S.y, S.y), S2z = mul2(S.z, S.z);
        const f2 V2x = mul2(vx, vx), V2y = mul2(vy, vy), V2z = mul2(vz, vz);
        s4S = fma2(S2x, S2x, fma2(S2y, S2y, mul2(S2z, S2z)));
        s4v = fma2(V2x, V2x, fma2(V2y, V2y, mul2(V2z, V2z)));
        dE = fma2(splat(-0.5f * Kc), sub2(s4v, s4S), dE);
    }
    return dE;
}
// on-site energy of the kept spins from the pieces above: lane l keeps the trial spin iff ok_l
template <int ANISO>
__device__ __forceinline__ f2 onsite_from(bool ok0, bool ok1, f2 s4S, f2 s4v, f2 euS, f2 euv, float Ku, float Kc)
{
    f2 E = splat(0.0f);
    if (ANISO & 1) E = mul2(splat(-Ku), make_float2(ok0 ? euv.x : euS.x, ok1 ? euv.y : euS.y));
    if (ANISO & 2) E = fma2(splat(-0.5f * Kc), make_float2(ok0 ? s4v.x : s4S.x, ok1 ? s4v.y : s4S.y), add2(E, splat(0.5f * Kc)));
    return E;
}

template <int ANISO>
__device__ __forceinline__ f2 aniso_energy2(const V3p& S, float Ku, const V3p& e, float Kc)
{
    f2 E = splat(0.0f);
    if (ANISO & 1) { const f2 se = dot3p(S, e); E = mul2(mul2(splat(-Ku), se), se); }
    if (ANISO & 2) {
        const f2 x2 = mul2(S.x, S.x), y2 = mul2(S.y, S.y), z2 = mul2(S.z, S.z);
        E = fma2(splat(Kc), fma2(x2, y2, fma2(x2, z2, mul2(y2, z2))), E);
    }
    return E;
}

template <int ANISO>
__device__ __forceinline__ V3p onsite_torque2(const V3p& S, float Ku, const V3p& e, float Kc, const V3p& B)
{
    V3p H = B;
    if (ANISO & 1) { const f2 f = mul2(splat(2.0f * Ku), dot3p(S, e)); H.x = fma2(f, e.x, H.x); H.y = fma2(f, e.y, H.y); H.z = fma2(f, e.z, H.z); }
    if (ANISO & 2) {
        const f2 x2 = mul2(S.x, S.x), y2 = mul2(S.y, S.y), z2 = mul2(S.z, S.z), g = splat(-2.0f * Kc);
        H.x = fma2(mul2(g, S.x), add2(y2, z2), H.x); H.y = fma2(mul2(g, S.y), add2(x2, z2), H.y); H.z = fma2(mul2(g, S.z), add2(x2, y2), H.z);
    }
    return { sub2(mul2(S.y, H.z), mul2(S.z, H.y)), sub2(mul2(S.z, H.x), mul2(S.x, H.z)), sub2(mul2(S.x, H.y), mul2(S.y, H.x)) };
}

// ---------------------------------------------------------------------------------------------------------------
// Division by a run-time constant with a precomputed magic number (host fills it): q = (n * mul) >> (32 + shift).
// Exact for n < 2^31 (round-up method).
// ---------------------------------------------------------------------------------------------------------------
struct FastDiv {
    uint32_t div, mul, shift;
    __device__ __forceinline__ uint32_t quot(uint32_t n) const { return div == 1 ? n : (__umulhi(n, mul) >> shift); }
    __device__ __forceinline__ void divmod(uint32_t n, uint32_t& q, uint32_t& r) const { q = quot(n); r = n - q * div; }
};

}  // namespace mc
