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
    const float sg = (S.z >= 0.0f) ? 1.0f : -1.0f;
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
// Division by a run-time constant with a precomputed magic number (host fills it): q = (n * mul) >> (32 + shift).
// Exact for n < 2^31 (round-up method).
// ---------------------------------------------------------------------------------------------------------------
struct FastDiv {
    uint32_t div, mul, shift;
    __device__ __forceinline__ uint32_t quot(uint32_t n) const { return div == 1 ? n : (__umulhi(n, mul) >> shift); }
    __device__ __forceinline__ void divmod(uint32_t n, uint32_t& q, uint32_t& r) const { q = quot(n); r = n - q * div; }
};

}  // namespace mc
