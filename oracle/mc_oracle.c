/*
 * mc_oracle.c -- plain, slow, fp64, single-threaded ORACLE for the red-black checkerboard Metropolis
 * sweep over unit classical Heisenberg spins (Lepadatu et al., arXiv 2103.03517).
 *
 * TEST INFRASTRUCTURE ONLY (see mc_oracle.h).  Shares no code with the CUDA path.
 * It follows the paper's Tables A1 / A2 step by step, in the paper's order and notation; there is no
 * blocking, fusion or reordering.  "P:NN" = line NN of /root/reference/PAPER.md.  "C-n" = reading n
 * in DESIGN.md section 4 (points where the paper is silent, ambiguous or garbled).
 *
 * Parity status: "parity unpinned" at the bit level (the paper prints no worked numeric example);
 * every function below is pinned by closed forms / invariants / brute force in tests/test_oracle_*.py.
 */
#include "mc_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

#define TAG_MOVE     0u   /* unconstrained trial move, keyed on the site                 */
#define TAG_PAIR     1u   /* constrained pair move, keyed on the leader's site           */
#define TAG_PAIRING  2u   /* pairing parameters of one (sweep, colour); site word = 0    */
#define TAG_INIT     3u   /* random initial state, keyed on the site (sweep words = 0)    */
#define TAG_ORACLE  16u   /* oracle-only cross-check modes (random order, Fisher-Yates)  */

static const double PI = 3.14159265358979323846;

struct orc_ctx {
    int nx, ny, nz, periodic[3];
    int structure;          /* 0 = simple cubic (the paper's lattice); 1 = body-centred cubic, 2 = face-centred cubic, see "bcc / fcc mode";
                               3 = hexagonal close-packed, 4 = simple cubic with next-nearest neighbours: "basis mode" (eight subsets) */
    int n_colours;          /* non-interacting subsets swept one after the other: 2 (sc checkerboard, bcc sublattices), 4 (fcc sublattices)  */
    int64_t Ncell;          /* nx*ny*nz: sc N = Ncell; bcc N = 2 Ncell, fcc N = 4 Ncell (site = sublattice*Ncell + cell)                     */
    /* basis mode: bonds of a site of sublattice a = the sites at the bonding distances, found from the coordinates at creation */
    int n_bonds[8];
    struct { int b, d[3]; double J; } bond[8][24];
    int64_t N;
    double J, Ku, eu[3], Kc, B[3];
    uint8_t* mask;          /* NULL = all bonds allowed by the boundary conditions */
    uint16_t* region;       /* NULL = uniform easy axis eu                         */
    double* region_axis; int n_regions;
    double cone; int adaptive;
    uint64_t seed, sweep;
    double* S;              /* [N][3] lexicographic: site = x + nx*(y + ny*z)       */
    double last_acceptance;
    /* accumulators (Eq. 6) */
    uint64_t n_samples;
    double sum_m[4], sum_m2[4], sum_E, sum_E2, sum_torque[3];
    /* per-sweep trace */
    double* trace; int64_t trace_len, trace_cap;
    /* constrained state */
    int aligned; double eC[3];
    int sampling;           /* 1 = measure + trace + accumulate after every sweep (default) */
    int torque_sampling;    /* 1 only inside orc_constrained_sweep: the torque is the constrained method's observable */
};

/* ------------------------------------------------------------------ Philox4x32-10 (pin P-1) */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* u = ((r>>9) + 0.5) * 2^-23: 24 significant bits, so identical in fp32 and fp64 (pin P-2, reading C-8). */
double orc_uniform(uint32_t r) { return ((double)(r >> 9) + 0.5) * (1.0 / 8388608.0); }

/* Azimuth uniform of the unconstrained move (reading C-26): the 9 low bits of the two words whose 23 high bits
 * make u0 and u2, 18 bits in all, u1 = k 2^-18 in [0,1) (an angle needs no open interval). */
double orc_uniform_azimuth(uint32_t w0, uint32_t w1)
{
    uint32_t k = ((w0 & 0x1FFu) << 9) | (w1 & 0x1FFu);
    return (double)k * (1.0 / 262144.0);
}

static void draw(const orc_ctx* c, uint32_t site, uint32_t tag, int colour, uint64_t sweep, uint32_t r[4])
{
    uint32_t ctr[4] = { site, tag | ((uint32_t)colour << 8), (uint32_t)sweep, (uint32_t)(sweep >> 32) };
    uint32_t key[2] = { (uint32_t)c->seed, (uint32_t)(c->seed >> 32) };
    orc_philox4x32_10(ctr, key, r);
}

/* ------------------------------------------------------------------ cone trial move (C-6, C-7) */
void orc_cone_move(const double S[3], double theta, double u0, double u1, double Sn[3])
{
    /* polar angle alpha from S uniform in solid angle over the cap of half-angle theta: cos(alpha) = 1 - w */
    double w = u0 * (1.0 - cos(theta));
    double sa = sqrt(w * (2.0 - w));
    double phi = 2.0 * PI * u1;
    /* orthonormal frame (t1,t2) perpendicular to S (Duff et al. 2017 construction).  sigma = sign of S_z taken from the
     * SIGN BIT (reading C-29): S_z = -0.0 gives sigma = -1; either frame is a valid frame (sigma + S_z = -1, no
     * singularity), the reading only fixes which one so that every implementation proposes the same trial spin. */
    double sg = signbit(S[2]) ? -1.0 : 1.0;
    double a = -1.0 / (sg + S[2]);
    double b = S[0] * S[1] * a;
    double t1[3] = { 1.0 + sg * S[0] * S[0] * a, sg * b, -sg * S[0] };
    double t2[3] = { b, sg + S[1] * S[1] * a, -S[1] };
    double cp = cos(phi), sp = sin(phi), v[3], n2 = 0.0;
    for (int k = 0; k < 3; ++k) {
        double d = -w * S[k] + sa * (cp * t1[k] + sp * t2[k]);
        v[k] = S[k] + d;
        n2 += v[k] * v[k];
    }
    double inv = 1.0 / sqrt(n2);
    for (int k = 0; k < 3; ++k) Sn[k] = v[k] * inv;
}

/* ------------------------------------------------------------------ lattice helpers */
static inline int64_t site_index(const orc_ctx* c, int x, int y, int z) { return x + (int64_t)c->nx * (y + (int64_t)c->ny * z); }

/* neighbour of (x,y,z) in direction k = (+x,-x,+y,-y,+z,-z); -1 if there is no bond (open face or masked).
 * *sign = -1 when the bond crosses an ANTI-periodic wrap (periodic[axis] == 2): the spin on the other side enters
 * Eq. (2) as -S_j, which is how a domain wall is held in the box ("anti-periodic along x direction"). */
static int64_t neighbour(const orc_ctx* c, int x, int y, int z, int k, double* sign)
{
    int p[3] = { x, y, z }, dim[3] = { c->nx, c->ny, c->nz };
    int axis = k >> 1, step = (k & 1) ? -1 : +1;
    int64_t self = site_index(c, x, y, z);
    *sign = 1.0;
    if (c->mask && !((c->mask[self] >> k) & 1)) return -1;
    p[axis] += step;
    if (p[axis] < 0 || p[axis] >= dim[axis]) {
        if (!c->periodic[axis]) return -1;
        if (c->periodic[axis] == 2) *sign = -1.0;
        p[axis] = (p[axis] + dim[axis]) % dim[axis];
    }
    return site_index(c, p[0], p[1], p[2]);
}

/* exchange field h_i = sum_{j in N_i} J S_j  (first term of Eq. 2; full J per bond, C-1) */
static void exchange_field(const orc_ctx* c, int x, int y, int z, double h[3])
{
    h[0] = h[1] = h[2] = 0.0;
    for (int k = 0; k < 6; ++k) {
        double sg;
        int64_t j = neighbour(c, x, y, z, k, &sg);
        if (j < 0) continue;
        for (int a = 0; a < 3; ++a) h[a] += sg * c->J * c->S[3 * j + a];
    }
}

/* ------------------------------------------------------------------ bcc mode (reading C-30; "this approach can be
 * extended to other crystal structures ... by considering the atomistic lattice as being composed of ... sub-lattices
 * (e.g. 2 simple cubic sub-lattices for bcc ...)").  The conventional cubic cell (i,j,k) holds sublattice A (colour 0) at its
 * corner (i,j,k) and sublattice B (colour 1) at its centre (i+1/2, j+1/2, k+1/2).  The 8 nearest neighbours of a site all lie
 * in the OTHER sublattice, so the two sublattices are the two non-interacting subsets of the checkerboard scheme:
 *   A(i,j,k) -- B(i-dx, j-dy, k-dz),   B(i,j,k) -- A(i+dx, j+dy, k+dz),   dx,dy,dz in {0,1}   (bond index k8 = dx + 2dy + 4dz).
 * Site index = sublattice*Ncell + (i + nx*(j + ny*k)).  Periodic wrap per axis (n = 1: the same neighbour twice, as L = 2
 * does in sc); an open axis drops the bonds that leave the box.  No bond mask, no regions, no anti-periodic wrap here. */
static int64_t bcc_neighbour(const orc_ctx* c, int64_t site, int k8)
{
    int sub = (int)(site / c->Ncell); int64_t cell = site % c->Ncell;
    int p[3] = { (int)(cell % c->nx), (int)((cell / c->nx) % c->ny), (int)(cell / ((int64_t)c->nx * c->ny)) };
    int dim[3] = { c->nx, c->ny, c->nz }, d[3] = { k8 & 1, (k8 >> 1) & 1, (k8 >> 2) & 1 };
    for (int a = 0; a < 3; ++a) {
        p[a] += sub ? d[a] : -d[a];
        if (p[a] < 0 || p[a] >= dim[a]) {
            if (!c->periodic[a]) return -1;
            p[a] = (p[a] + dim[a]) % dim[a];
        }
    }
    return (int64_t)(1 - sub) * c->Ncell + p[0] + (int64_t)c->nx * (p[1] + (int64_t)c->ny * p[2]);
}

/* ------------------------------------------------------------------ fcc mode (reading C-31; "4 simple cubic
 * sub-lattices for fcc").  The conventional cubic cell (i,j,k) holds four sites: sublattice 0 at the corner, 1 at (0,1/2,1/2),
 * 2 at (1/2,0,1/2), 3 at (1/2,1/2,0) from it.  The 12 nearest neighbours (distance a/sqrt 2) of a site are 4 in each of the
 * OTHER three sublattices, none in its own: the four sublattices are four non-interacting subsets, swept as four colours.
 * Towards sublattice b the offsets of a and b differ along exactly two axes; along such an axis the neighbour's cell index is
 * {i-1, i} if a sits at 0 and b at 1/2, {i, i+1} the other way round; along the third axis it is i.
 * Bond index k12 = 4*r + d1 + 2*d2 with r = the rank of b among the other sublattices.  Wrap / open faces as in bcc mode. */
static const int FCC_OFF[4][3] = { { 0, 0, 0 }, { 0, 1, 1 }, { 1, 0, 1 }, { 1, 1, 0 } };   /* in half lattice constants */
static int64_t fcc_neighbour(const orc_ctx* c, int64_t site, int k12, int* b_out)
{
    int a = (int)(site / c->Ncell); int64_t cell = site % c->Ncell;
    int r = k12 >> 2, b = r + (r >= a ? 1 : 0);               /* the r-th sublattice other than a */
    int p[3] = { (int)(cell % c->nx), (int)((cell / c->nx) % c->ny), (int)(cell / ((int64_t)c->nx * c->ny)) };
    int dim[3] = { c->nx, c->ny, c->nz }, d[2] = { k12 & 1, (k12 >> 1) & 1 }, nd = 0;
    for (int ax = 0; ax < 3; ++ax) {
        if (FCC_OFF[a][ax] == FCC_OFF[b][ax]) continue;
        int step = d[nd++];                                   /* 0 or 1 */
        p[ax] += FCC_OFF[a][ax] ? step : -step;               /* a at 1/2: {i, i+1};  a at 0: {i, i-1} */
        if (p[ax] < 0 || p[ax] >= dim[ax]) {
            if (!c->periodic[ax]) return -1;
            p[ax] = (p[ax] + dim[ax]) % dim[ax];
        }
    }
    if (b_out) *b_out = b;
    return (int64_t)b * c->Ncell + p[0] + (int64_t)c->nx * (p[1] + (int64_t)c->ny * p[2]);
}

/* ------------------------------------------------------------------ basis mode (reading C-32; "... 4 simple tetragonal
 * sub-lattices for hcp ... up to 8 non-interacting subsets ... next-nearest neighbours").  A periodic box of nx x ny x nz
 * cells, every cell holding the same basis of EIGHT sites; sublattice s = the s-th basis site of every cell = colour s (eight
 * colour passes per Monte Carlo iteration); site index = s*Ncell + (i + nx*(j + ny*k)).  The bonds are not tabulated by hand:
 * at creation, for every sublattice a, every (sublattice b, cell offset d in {-1,0,1}^3) whose separation
 * r = pos_b + d*cell - pos_a has the bonding length is a bond.  Lengths are compared exactly, in integer units:
 *   hcp (structure 3): orthohexagonal cell of the ideal hcp lattice doubled along x, cell = (2a, sqrt3 a, c), c^2 = 8/3 a^2;
 *       units (a/2, sqrt3 a/6, c/2): cell = (4, 6, 2); basis (0,0,0) (1,3,0) (1,1,1) (0,4,1) and the same + (2,0,0);
 *       |r|^2 = a^2/12 (3 dx^2 + dy^2 + 8 dz^2): nearest neighbours (12 per site, coupling J) have 3 dx^2 + dy^2 + 8 dz^2 = 12;
 *   sc with next-nearest neighbours (structure 4): the 2 x 2 x 2 block of a simple cubic lattice as the cell, units a:
 *       cell = (2,2,2), basis (x,y,z) in {0,1}^3 (s = x + 2y + 4z); |r|^2 = 1: 6 nearest neighbours, coupling J;
 *       |r|^2 = 2: 12 next-nearest neighbours, coupling J2.  The box is a (2nx) x (2ny) x (2nz) simple cubic lattice.
 * In both no bond joins two sites of one sublattice (checked at creation): the eight sublattices are non-interacting subsets.
 * A 1- or 2-cell axis reaches the same site through several offsets and counts it as often (as L = 2 does in sc). */
static const int HCP_POS[8][3] = { { 0, 0, 0 }, { 1, 3, 0 }, { 1, 1, 1 }, { 0, 4, 1 }, { 2, 0, 0 }, { 3, 3, 0 }, { 3, 1, 1 }, { 2, 4, 1 } };
static int build_bonds(orc_ctx* c, double J2)
{
    const int hcp = c->structure == 3;
    const int cell[3] = { hcp ? 4 : 2, hcp ? 6 : 2, 2 }, metric[3] = { hcp ? 3 : 1, 1, hcp ? 8 : 1 };
    for (int a = 0; a < 8; ++a) {
        c->n_bonds[a] = 0;
        for (int b = 0; b < 8; ++b) for (int dz = -1; dz <= 1; ++dz) for (int dy = -1; dy <= 1; ++dy) for (int dx = -1; dx <= 1; ++dx) {
            const int d[3] = { dx, dy, dz };
            int q = 0;
            for (int ax = 0; ax < 3; ++ax) {
                int pa = hcp ? HCP_POS[a][ax] : (a >> ax) & 1, pb = hcp ? HCP_POS[b][ax] : (b >> ax) & 1;
                int r = pb + d[ax] * cell[ax] - pa;
                q += metric[ax] * r * r;
            }
            double J;
            if (hcp) { if (q != 12) continue; J = c->J; }
            else { if (q == 1) J = c->J; else if (q == 2) J = J2; else continue; }
            if (b == a) return -1;                                    /* a bond inside a sublattice: not a non-interacting subset */
            int k = c->n_bonds[a]++;
            c->bond[a][k].b = b; c->bond[a][k].J = J;
            for (int ax = 0; ax < 3; ++ax) c->bond[a][k].d[ax] = d[ax];
        }
        if (c->n_bonds[a] != (hcp ? 12 : 18)) return -1;
    }
    return 0;
}
static int64_t basis_neighbour(const orc_ctx* c, int64_t site, int k, double* J)
{
    int a = (int)(site / c->Ncell); int64_t cellidx = site % c->Ncell;
    int p[3] = { (int)(cellidx % c->nx), (int)((cellidx / c->nx) % c->ny), (int)(cellidx / ((int64_t)c->nx * c->ny)) };
    int dim[3] = { c->nx, c->ny, c->nz };
    for (int ax = 0; ax < 3; ++ax) p[ax] = (p[ax] + c->bond[a][k].d[ax] + dim[ax]) % dim[ax];
    *J = c->bond[a][k].J;
    return (int64_t)c->bond[a][k].b * c->Ncell + p[0] + (int64_t)c->nx * (p[1] + (int64_t)c->ny * p[2]);
}

/* exchange field of ANY site, any structure (sc: decode the site and use the six-direction sum above) */
static void field_at(const orc_ctx* c, int64_t site, double h[3])
{
    if (c->structure == 0) {
        exchange_field(c, (int)(site % c->nx), (int)((site / c->nx) % c->ny), (int)(site / ((int64_t)c->nx * c->ny)), h);
        return;
    }
    h[0] = h[1] = h[2] = 0.0;
    if (c->structure >= 3) {
        for (int k = 0; k < c->n_bonds[site / c->Ncell]; ++k) {
            double J; int64_t j = basis_neighbour(c, site, k, &J);
            for (int a = 0; a < 3; ++a) h[a] += J * c->S[3 * j + a];
        }
        return;
    }
    if (c->structure == 2) {
        for (int k = 0; k < 12; ++k) {
            int64_t j = fcc_neighbour(c, site, k, NULL);
            if (j < 0) continue;
            for (int a = 0; a < 3; ++a) h[a] += c->J * c->S[3 * j + a];
        }
        return;
    }
    for (int k = 0; k < 8; ++k) {
        int64_t j = bcc_neighbour(c, site, k);
        if (j < 0) continue;
        for (int a = 0; a < 3; ++a) h[a] += c->J * c->S[3 * j + a];
    }
}

/* colour of a site: sc (x+y+z) mod 2 with red = even first (C-10); bcc the sublattice */
static int colour_of(const orc_ctx* c, int64_t site)
{
    if (c->structure) return (int)(site / c->Ncell);
    return (int)((site % c->nx + (site / c->nx) % c->ny + site / ((int64_t)c->nx * c->ny)) & 1);
}

static const double* easy_axis(const orc_ctx* c, int64_t site)
{
    return c->region ? &c->region_axis[3 * (int64_t)c->region[site]] : c->eu;
}

/* E_i(S) of Eq. (2), given the exchange field h of site i */
static double site_energy_h(const orc_ctx* c, int64_t site, const double h[3], const double S[3])
{
    const double* e = easy_axis(c, site);
    double se = S[0] * e[0] + S[1] * e[1] + S[2] * e[2];
    double x2 = S[0] * S[0], y2 = S[1] * S[1], z2 = S[2] * S[2];
    return -(S[0] * h[0] + S[1] * h[1] + S[2] * h[2])
           - c->Ku * se * se
           + c->Kc * (x2 * y2 + x2 * z2 + y2 * z2)
           - (S[0] * c->B[0] + S[1] * c->B[1] + S[2] * c->B[2]);
}

double orc_site_energy(const orc_ctx* c, int64_t site, const double S[3])
{
    double h[3];
    field_at(c, site, h);
    return site_energy_h(c, site, h, S);
}

/* extensive H = -J sum_<ij> S_i.S_j + on-site terms, every bond visited ONCE via its + direction (C-1).
 * Independent of exchange_field's 1/2-sum so that it can pin it (pin P-5). */
double orc_total_energy(const orc_ctx* c)
{
    double E = 0.0;
    if (c->structure >= 3) {                 /* basis mode: a bond joins two different sublattices: visit it from the lower one */
        for (int64_t i = 0; i < c->N; ++i) {
            const double* S = &c->S[3 * i];
            int a = (int)(i / c->Ncell);
            for (int k = 0; k < c->n_bonds[a]; ++k) {
                if (c->bond[a][k].b < a) continue;
                double J; int64_t j = basis_neighbour(c, i, k, &J);
                const double* Sj = &c->S[3 * j];
                E -= J * (S[0] * Sj[0] + S[1] * Sj[1] + S[2] * Sj[2]);
            }
            double se = S[0] * c->eu[0] + S[1] * c->eu[1] + S[2] * c->eu[2];
            double x2 = S[0] * S[0], y2 = S[1] * S[1], z2 = S[2] * S[2];
            E += -c->Ku * se * se + c->Kc * (x2 * y2 + x2 * z2 + y2 * z2)
                 - (S[0] * c->B[0] + S[1] * c->B[1] + S[2] * c->B[2]);
        }
        return E;
    }
    if (c->structure == 2) {                 /* fcc: a bond joins two different sublattices: visit it from the lower one */
        for (int64_t i = 0; i < c->N; ++i) {
            const double* S = &c->S[3 * i];
            int a = (int)(i / c->Ncell);
            for (int k = 0; k < 12; ++k) {
                int b; int64_t j = fcc_neighbour(c, i, k, &b);
                if (j < 0 || b < a) continue;
                const double* Sj = &c->S[3 * j];
                E -= c->J * (S[0] * Sj[0] + S[1] * Sj[1] + S[2] * Sj[2]);
            }
            double se = S[0] * c->eu[0] + S[1] * c->eu[1] + S[2] * c->eu[2];
            double x2 = S[0] * S[0], y2 = S[1] * S[1], z2 = S[2] * S[2];
            E += -c->Ku * se * se + c->Kc * (x2 * y2 + x2 * z2 + y2 * z2)
                 - (S[0] * c->B[0] + S[1] * c->B[1] + S[2] * c->B[2]);
        }
        return E;
    }
    if (c->structure) {                      /* bcc: every bond joins an A and a B site: visit the 8 bonds of every A site */
        for (int64_t i = 0; i < c->N; ++i) {
            const double* S = &c->S[3 * i];
            if (i < c->Ncell)
                for (int k = 0; k < 8; ++k) {
                    int64_t j = bcc_neighbour(c, i, k);
                    if (j < 0) continue;
                    const double* Sj = &c->S[3 * j];
                    E -= c->J * (S[0] * Sj[0] + S[1] * Sj[1] + S[2] * Sj[2]);
                }
            double se = S[0] * c->eu[0] + S[1] * c->eu[1] + S[2] * c->eu[2];
            double x2 = S[0] * S[0], y2 = S[1] * S[1], z2 = S[2] * S[2];
            E += -c->Ku * se * se + c->Kc * (x2 * y2 + x2 * z2 + y2 * z2)
                 - (S[0] * c->B[0] + S[1] * c->B[1] + S[2] * c->B[2]);
        }
        return E;
    }
    for (int z = 0; z < c->nz; ++z) for (int y = 0; y < c->ny; ++y) for (int x = 0; x < c->nx; ++x) {
        int64_t i = site_index(c, x, y, z);
        const double* S = &c->S[3 * i];
        for (int k = 0; k < 6; k += 2) {          /* +x, +y, +z only */
            double sg;
            int64_t j = neighbour(c, x, y, z, k, &sg);
            if (j < 0) continue;
            const double* Sj = &c->S[3 * j];
            E -= sg * c->J * (S[0] * Sj[0] + S[1] * Sj[1] + S[2] * Sj[2]);
        }
        const double* e = easy_axis(c, i);
        double se = S[0] * e[0] + S[1] * e[1] + S[2] * e[2];
        double x2 = S[0] * S[0], y2 = S[1] * S[1], z2 = S[2] * S[2];
        E += -c->Ku * se * se + c->Kc * (x2 * y2 + x2 * z2 + y2 * z2)
             - (S[0] * c->B[0] + S[1] * c->B[1] + S[2] * c->B[2]);
    }
    return E;
}

/* ------------------------------------------------------------------ create / state */
orc_ctx* orc_create(int nx, int ny, int nz, const int periodic[3],
                    double J, double Ku, const double eu[3], double Kc, const double B[3],
                    const uint8_t* bond_mask, const uint16_t* region,
                    const double* region_axis, int n_regions,
                    double cone0_rad, int adaptive, uint64_t seed)
{
    if (nx < 1 || ny < 1 || nz < 1) return NULL;
    int dim[3] = { nx, ny, nz };
    for (int a = 0; a < 3; ++a) if (periodic[a] && (dim[a] & 1)) return NULL;   /* two-colouring needs even periodic dims */
    for (int a = 0; a < 3; ++a) if (periodic[a] < 0 || periodic[a] > 2) return NULL;   /* 0 open, 1 periodic, 2 anti-periodic */
    orc_ctx* c = (orc_ctx*)calloc(1, sizeof(orc_ctx));
    c->nx = nx; c->ny = ny; c->nz = nz;
    for (int a = 0; a < 3; ++a) c->periodic[a] = periodic[a];
    c->N = (int64_t)nx * ny * nz; c->Ncell = c->N; c->structure = 0; c->n_colours = 2;
    c->J = J; c->Ku = Ku; c->Kc = Kc;
    double n = sqrt(eu[0] * eu[0] + eu[1] * eu[1] + eu[2] * eu[2]);
    for (int a = 0; a < 3; ++a) { c->eu[a] = (n > 0) ? eu[a] / n : (a == 2); c->B[a] = B[a]; }
    if (bond_mask) { c->mask = (uint8_t*)malloc(c->N); memcpy(c->mask, bond_mask, c->N); }
    if (region) {
        c->region = (uint16_t*)malloc(2 * c->N); memcpy(c->region, region, 2 * c->N);
        c->n_regions = n_regions;
        c->region_axis = (double*)malloc(sizeof(double) * 3 * n_regions);
        for (int r = 0; r < n_regions; ++r) {
            const double* v = &region_axis[3 * r];
            double m = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
            for (int a = 0; a < 3; ++a) c->region_axis[3 * r + a] = v[a] / m;
        }
    }
    c->cone = cone0_rad; c->adaptive = adaptive; c->seed = seed; c->sweep = 0; c->sampling = 1;
    c->S = (double*)malloc(sizeof(double) * 3 * c->N);
    for (int64_t i = 0; i < c->N; ++i) { c->S[3 * i] = 0; c->S[3 * i + 1] = 0; c->S[3 * i + 2] = 1; }
    return c;
}

/* bcc lattice of nx x ny x nz conventional cells, 2 nx ny nz spins (bcc mode above).  Any dimension may be periodic (1) or
 * open (0) and need not be even: the two sublattices are the two colours whatever the size. */
orc_ctx* orc_create_bcc(int nx, int ny, int nz, const int periodic[3],
                        double J, double Ku, const double eu[3], double Kc, const double B[3],
                        double cone0_rad, int adaptive, uint64_t seed)
{
    if (nx < 1 || ny < 1 || nz < 1) return NULL;
    for (int a = 0; a < 3; ++a) if (periodic[a] < 0 || periodic[a] > 1) return NULL;
    orc_ctx* c = (orc_ctx*)calloc(1, sizeof(orc_ctx));
    c->nx = nx; c->ny = ny; c->nz = nz; c->structure = 1; c->n_colours = 2;
    for (int a = 0; a < 3; ++a) c->periodic[a] = periodic[a];
    c->Ncell = (int64_t)nx * ny * nz; c->N = 2 * c->Ncell;
    c->J = J; c->Ku = Ku; c->Kc = Kc;
    double n = sqrt(eu[0] * eu[0] + eu[1] * eu[1] + eu[2] * eu[2]);
    for (int a = 0; a < 3; ++a) { c->eu[a] = (n > 0) ? eu[a] / n : (a == 2); c->B[a] = B[a]; }
    c->cone = cone0_rad; c->adaptive = adaptive; c->seed = seed; c->sweep = 0; c->sampling = 1;
    c->S = (double*)malloc(sizeof(double) * 3 * c->N);
    for (int64_t i = 0; i < c->N; ++i) { c->S[3 * i] = 0; c->S[3 * i + 1] = 0; c->S[3 * i + 2] = 1; }
    return c;
}

/* fcc lattice of nx x ny x nz conventional cells, 4 nx ny nz spins, four colours (fcc mode above) */
orc_ctx* orc_create_fcc(int nx, int ny, int nz, const int periodic[3],
                        double J, double Ku, const double eu[3], double Kc, const double B[3],
                        double cone0_rad, int adaptive, uint64_t seed)
{
    orc_ctx* c = orc_create_bcc(nx, ny, nz, periodic, J, Ku, eu, Kc, B, cone0_rad, adaptive, seed);
    if (!c) return NULL;
    c->structure = 2; c->n_colours = 4; c->N = 4 * c->Ncell;
    free(c->S);
    c->S = (double*)malloc(sizeof(double) * 3 * c->N);
    for (int64_t i = 0; i < c->N; ++i) { c->S[3 * i] = 0; c->S[3 * i + 1] = 0; c->S[3 * i + 2] = 1; }
    return c;
}

/* basis mode above: kind 3 = hcp (J2 ignored), 4 = simple cubic with next-nearest neighbours (J, J2); nx x ny x nz cells of eight
 * sites, 8 nx ny nz spins, every axis periodic, eight colours */
orc_ctx* orc_create_basis(int kind, int nx, int ny, int nz, double J, double J2, double Ku, const double eu[3], double Kc, const double B[3],
                          double cone0_rad, int adaptive, uint64_t seed)
{
    const int periodic[3] = { 1, 1, 1 };
    if (kind != 3 && kind != 4) return NULL;
    orc_ctx* c = orc_create_bcc(nx, ny, nz, periodic, J, Ku, eu, Kc, B, cone0_rad, adaptive, seed);
    if (!c) return NULL;
    c->structure = kind; c->n_colours = 8; c->N = 8 * c->Ncell;
    if (build_bonds(c, J2)) { orc_destroy(c); return NULL; }
    free(c->S);
    c->S = (double*)malloc(sizeof(double) * 3 * c->N);
    for (int64_t i = 0; i < c->N; ++i) { c->S[3 * i] = 0; c->S[3 * i + 1] = 0; c->S[3 * i + 2] = 1; }
    return c;
}

void orc_destroy(orc_ctx* c)
{
    if (!c) return;
    free(c->mask); free(c->region); free(c->region_axis); free(c->S); free(c->trace); free(c);
}

void orc_set_spins(orc_ctx* c, const double* xyz) { memcpy(c->S, xyz, sizeof(double) * 3 * c->N); c->aligned = 0; }
void orc_set_spins_f32(orc_ctx* c, const float* xyz) { for (int64_t i = 0; i < 3 * c->N; ++i) c->S[i] = (double)xyz[i]; c->aligned = 0; }
void orc_get_spins(const orc_ctx* c, double* xyz) { memcpy(xyz, c->S, sizeof(double) * 3 * c->N); }
void orc_init_uniform(orc_ctx* c, const double dir[3])
{
    double n = sqrt(dir[0] * dir[0] + dir[1] * dir[1] + dir[2] * dir[2]);
    for (int64_t i = 0; i < c->N; ++i) for (int a = 0; a < 3; ++a) c->S[3 * i + a] = dir[a] / n;
    c->aligned = 0;
}
/* Random start (BASELINE.json configs[2] "spins start uniformly random on the sphere (seeded)"): site i takes
 * (r0,r1,..) = Philox(ctr = (i, TAG_INIT, 0, 0), key = seed), z = 2 u(r0) - 1, phi = 2 pi u(r1) (Archimedes: z uniform). */
void orc_init_random(orc_ctx* c)
{
    for (int64_t i = 0; i < c->N; ++i) {
        uint32_t r[4];
        draw(c, (uint32_t)i, TAG_INIT, 0, 0, r);
        double z = 2.0 * orc_uniform(r[0]) - 1.0, phi = 2.0 * PI * orc_uniform(r[1]), s = sqrt(1.0 - z * z);
        c->S[3 * i] = s * cos(phi); c->S[3 * i + 1] = s * sin(phi); c->S[3 * i + 2] = z;
    }
    c->aligned = 0;
}
void orc_set_cone(orc_ctx* c, double cone) { c->cone = cone; }
void orc_set_sweep(orc_ctx* c, uint64_t s) { c->sweep = s; }
void orc_set_adaptive(orc_ctx* c, int a) { c->adaptive = a; }
void orc_set_sampling(orc_ctx* c, int on) { c->sampling = on; }

/* ------------------------------------------------------------------ the three uniforms of one unconstrained update
 * Reading C-26: two same-colour sites that are neighbours along x in their colour's row,
 * x and x ^ 2, share ONE Philox4x32-10 block, counter word 0 = lexicographic index of the one with bit 1 of x clear;
 * that site takes words (0,1), the other takes words (2,3).  From its words (w0,w1) a site forms
 *   u0 = ((w0 >> 9) + 0.5) 2^-23   (cone polar draw),     u2 = ((w1 >> 9) + 0.5) 2^-23   (acceptance draw),
 *   u1 = (((w0 & 511) << 9) | (w1 & 511)) 2^-18            (cone azimuth).
 * 64 random bits per update, every bit used once. */
static void site_uniforms_tag(const orc_ctx* c, int x, int y, int z, uint32_t tag, int colour, uint64_t sweep, double* u0, double* u1, double* u2)
{
    int64_t first = site_index(c, x & ~2, y, z);
    int half = (x >> 1) & 1;
    if (c->structure) {      /* bcc (C-30): the same-sublattice x-neighbours i and i ^ 1 share the block; (x,y,z) = cell, colour = sublattice */
        first = (int64_t)colour * c->Ncell + site_index(c, x & ~1, y, z);
        half = x & 1;
    }
    uint32_t r[4];
    draw(c, (uint32_t)first, tag, colour, sweep, r);
    uint32_t w0 = r[2 * half], w1 = r[2 * half + 1];
    *u0 = orc_uniform(w0);
    *u1 = orc_uniform_azimuth(w0, w1);
    *u2 = orc_uniform(w1);
}

void orc_site_uniforms(const orc_ctx* c, int x, int y, int z, int colour, uint64_t sweep, double* u0, double* u1, double* u2)
{
    site_uniforms_tag(c, x, y, z, TAG_MOVE, colour, sweep, u0, u1, u2);
}
/* the same 64 bits per move for the constrained pair move, keyed on the LEADER's site in its own stream (TAG_PAIR) */
void orc_pair_uniforms(const orc_ctx* c, int x, int y, int z, int colour, uint64_t sweep, double* u0, double* u1, double* u2)
{
    site_uniforms_tag(c, x, y, z, TAG_PAIR, colour, sweep, u0, u1, u2);
}

/* ------------------------------------------------------------------ Table A1: one colour pass */
static int metropolis_update(orc_ctx* c, int x, int y, int z, int colour, double T, double* xdec)
{
    int64_t i = site_index(c, x, y, z);                       /* P:155  i = Get_Red(Black)SpinIndex(index) */
    if (c->structure) i += (int64_t)colour * c->Ncell;        /* bcc: (x,y,z) is the cell, colour the sublattice */
    double u0, u1, u2;
    orc_site_uniforms(c, x, y, z, colour, c->sweep, &u0, &u1, &u2);   /* P:156-157 UniformRandom() x 3 (C-8, C-26) */
    double* S = &c->S[3 * i], Sn[3], h[3];
    orc_cone_move(S, c->cone, u0, u1, Sn);                    /* P:156  S_new = UniformRandom_RotateSpin(S_i, theta) */
    field_at(c, i, h);
    double dE = site_energy_h(c, i, h, Sn) - site_energy_h(c, i, h, S);   /* P:158  E(S_new) - E(S_i) */
    double xd = dE / T + log(u2);                             /* P:157-158  P < exp(-dE/kT)  <=>  dE/T + ln P < 0  (C-8) */
    if (xdec) xdec[i] = xd;
    if (xd < 0.0) { S[0] = Sn[0]; S[1] = Sn[1]; S[2] = Sn[2]; return 1; }
    return 0;
}

int64_t orc_half_sweep(orc_ctx* c, double T, int colour, double* xdec, uint8_t* acc)
{
    int64_t count = 0;
    c->aligned = 0;   /* an unconstrained pass moves M off e_C: the next constrained sweep re-aligns (reading C-12) */
    for (int z = 0; z < c->nz; ++z) for (int y = 0; y < c->ny; ++y) for (int x = 0; x < c->nx; ++x) {
        if (!c->structure && ((x + y + z) & 1) != colour) continue;   /* sc: red = even (C-10); bcc: every cell holds one site of each colour */
        int a = metropolis_update(c, x, y, z, colour, T, xdec);
        if (acc) acc[site_index(c, x, y, z) + (c->structure ? (int64_t)colour * c->Ncell : 0)] = (uint8_t)a;
        count += a;
    }
    return count;
}

/* ------------------------------------------------------------------ domain-wall profile (Fig. 2)
 * "the normalized magnetization z component is obtained for each profile point by averaging over the respective
 * cross-section slice": out[3*x + a] = mean over (y,z) of S_a at that x. */
void orc_profile_x(const orc_ctx* c, double* out)
{
    for (int x = 0; x < c->nx; ++x) {
        double s[3] = { 0, 0, 0 };
        for (int z = 0; z < c->nz; ++z) for (int y = 0; y < c->ny; ++y) {
            const double* S = &c->S[3 * site_index(c, x, y, z)];
            s[0] += S[0]; s[1] += S[1]; s[2] += S[2];
        }
        for (int a = 0; a < 3; ++a) out[3 * x + a] = s[a] / ((double)c->ny * c->nz);
    }
}

/* ------------------------------------------------------------------ observables (Eq. 6) */
static void measure(const orc_ctx* c, orc_obs* o)
{
    double M[3] = { 0, 0, 0 }, Eex = 0, Ean = 0, Ez = 0, tq[3] = { 0, 0, 0 };
    for (int64_t i = 0; i < c->N; ++i) {                      /* lexicographic site order (sc: x fastest) */
        const double* S = &c->S[3 * i];
        double h[3];
        field_at(c, i, h);
        for (int a = 0; a < 3; ++a) M[a] += S[a];
        Eex += -0.5 * (S[0] * h[0] + S[1] * h[1] + S[2] * h[2]);          /* every bond once (C-1) */
        const double* e = easy_axis(c, i);
        double se = S[0] * e[0] + S[1] * e[1] + S[2] * e[2];
        double x2 = S[0] * S[0], y2 = S[1] * S[1], z2 = S[2] * S[2];
        Ean += -c->Ku * se * se + c->Kc * (x2 * y2 + x2 * z2 + y2 * z2);
        Ez  += -(S[0] * c->B[0] + S[1] * c->B[1] + S[2] * c->B[2]);
        /* on-site field H = -dE_i/dS_i (anisotropy + Zeeman); torque = S x H */
        double H[3] = {
            2.0 * c->Ku * se * e[0] - 2.0 * c->Kc * S[0] * (y2 + z2) + c->B[0],
            2.0 * c->Ku * se * e[1] - 2.0 * c->Kc * S[1] * (x2 + z2) + c->B[1],
            2.0 * c->Ku * se * e[2] - 2.0 * c->Kc * S[2] * (x2 + y2) + c->B[2] };
        tq[0] += S[1] * H[2] - S[2] * H[1];
        tq[1] += S[2] * H[0] - S[0] * H[2];
        tq[2] += S[0] * H[1] - S[1] * H[0];
    }
    double invN = 1.0 / (double)c->N;
    for (int a = 0; a < 3; ++a) { o->M[a] = M[a] * invN; o->torque[a] = tq[a] * invN; }
    o->m = sqrt(o->M[0] * o->M[0] + o->M[1] * o->M[1] + o->M[2] * o->M[2]);
    o->E_exch = Eex * invN; o->E_aniso = Ean * invN; o->E_zeeman = Ez * invN;
    o->E_total = o->E_exch + o->E_aniso + o->E_zeeman;
}

void orc_end_sweep(orc_ctx* c, int64_t count)
{
    c->last_acceptance = (double)count / (double)c->N;
    double cone_used = c->cone;
    if (c->adaptive) {                                        /* P:168-171 read with P:205-209 (C-2, C-3, C-9) */
        const double deg = PI / 180.0;
        if (2 * count > c->N) { c->cone += deg; if (c->cone > PI) c->cone = PI; }
        else                  { c->cone -= deg; if (c->cone < deg) c->cone = deg; }
    }
    c->sweep += 1;
    if (!c->sampling) return;
    orc_obs o; memset(&o, 0, sizeof o);
    measure(c, &o);
    double mv[4] = { o.m, o.M[0], o.M[1], o.M[2] };
    for (int a = 0; a < 4; ++a) { c->sum_m[a] += mv[a]; c->sum_m2[a] += mv[a] * mv[a]; }
    c->sum_E += o.E_total; c->sum_E2 += o.E_total * o.E_total;
    if (c->torque_sampling) for (int a = 0; a < 3; ++a) c->sum_torque[a] += o.torque[a];   /* constrained sweeps only */
    c->n_samples += 1;
    if (c->trace_len == c->trace_cap) {
        c->trace_cap = c->trace_cap ? 2 * c->trace_cap : 1024;
        c->trace = (double*)realloc(c->trace, sizeof(double) * 6 * c->trace_cap);
    }
    double* row = &c->trace[6 * c->trace_len++];
    row[0] = c->last_acceptance; row[1] = cone_used; row[2] = o.M[0]; row[3] = o.M[1]; row[4] = o.M[2]; row[5] = o.E_total;
}

void orc_sweep(orc_ctx* c, double T, int64_t n)
{
    for (int64_t it = 0; it < n; ++it) {
        int64_t count = orc_half_sweep(c, T, 0, NULL, NULL);
        count += orc_half_sweep(c, T, 1, NULL, NULL);
        for (int col = 2; col < c->n_colours; ++col) count += orc_half_sweep(c, T, col, NULL, NULL);   /* fcc: two more subsets */
        orc_end_sweep(c, count);
    }
}

/* serial Metropolis with a random visiting order -- only for the "serial == parallel" pin */
void orc_sweep_random_order(orc_ctx* c, double T, int64_t n)
{
    int64_t* order = (int64_t*)malloc(sizeof(int64_t) * c->N);
    c->aligned = 0;   /* reading C-12, as in orc_half_sweep */
    for (int64_t it = 0; it < n; ++it) {
        for (int64_t i = 0; i < c->N; ++i) order[i] = i;
        for (int64_t i = c->N - 1; i > 0; --i) {
            uint32_t r[4]; draw(c, (uint32_t)i, TAG_ORACLE, 0, c->sweep, r);
            int64_t j = (int64_t)(((uint64_t)r[0] * (uint64_t)(i + 1)) >> 32);
            int64_t t = order[i]; order[i] = order[j]; order[j] = t;
        }
        int64_t count = 0;
        for (int64_t k = 0; k < c->N; ++k) {
            int64_t s = order[k];
            int64_t cell = s % c->Ncell;
            int x = (int)(cell % c->nx), y = (int)((cell / c->nx) % c->ny), z = (int)(cell / ((int64_t)c->nx * c->ny));
            count += metropolis_update(c, x, y, z, colour_of(c, s), T, NULL);
        }
        orc_end_sweep(c, count);
    }
    free(order);
}

/* ------------------------------------------------------------------ constrained MC (Table A2) */

/* colour-linear index: a = (x>>1) + (nx/2)*(y + ny*z) enumerates the sites of one colour (nx even). */
int64_t orc_site_of(const orc_ctx* c, int colour, int64_t a)
{
    if (c->structure) return (int64_t)colour * c->Ncell + a;   /* bcc: a sublattice is stored contiguously */
    int hx = c->nx / 2;
    int xh = (int)(a % hx); int64_t row = a / hx;
    int y = (int)(row % c->ny), z = (int)(row / c->ny);
    int x = 2 * xh + ((colour + y + z) & 1);
    return site_index(c, x, y, z);
}

/* Pairing of one (sweep, colour): reading C-11.
 *   B = largest power of two <= 32 with 2B | Nc;  H = Nc/B chunks of B consecutive colour-linear indices;
 *   Bl = min(B,4), Bh = B/Bl;
 *   (r0,r1,r2,.) = Philox(ctr = (0, TAG_PAIRING | colour<<8, sweep_lo, sweep_hi));
 *   m = 2*floor(r0*(H/2)/2^32) + 1 (odd);  sigma = r1 & 1;  r = r2 mod Bl;  q = (r2 >> 2) mod Bh;
 *   index a = chunk*B + hi*Bl + lo is a LEADER iff chunk mod 2 == sigma; its follower is
 *   ((chunk+m) mod H)*B + ((hi+q) mod Bh)*Bl + (lo+r) mod Bl.
 * Replaces the paper's shuffled index array; requirements R1-R4 in DESIGN.md. */
int orc_pairing(const orc_ctx* c, uint64_t sweep, int colour, int64_t* partner, uint8_t* is_leader)
{
    if (c->structure >= 2) return -1;                        /* the constrained path sweeps two colours: sc and bcc (not the four of fcc, the eight of basis mode) */
    if (!c->structure && (c->nx & 1)) return -1;
    int64_t Nc = c->N / 2;
    if (Nc & 1) return -1;                                   /* C-15 */
    int64_t B = 32; while (Nc % (2 * B)) B >>= 1;
    int64_t H = Nc / B;
    uint32_t r[4]; draw(c, 0u, TAG_PAIRING, colour, sweep, r);
    int64_t m = 2 * (int64_t)(((uint64_t)r[0] * (uint64_t)(H / 2)) >> 32) + 1;
    int64_t sigma = r[1] & 1u;
    int64_t Bl = B < 4 ? B : 4, Bh = B / Bl;
    int64_t rot = (int64_t)(r[2] % (uint32_t)Bl), q = (int64_t)((r[2] >> 2) % (uint32_t)Bh);
    for (int64_t a = 0; a < Nc; ++a) {
        int64_t chunk = a / B, e = a % B, hi = e / Bl, lo = e % Bl;
        if ((chunk & 1) == sigma) {
            int64_t f = ((chunk + m) % H) * B + ((hi + q) % Bh) * Bl + (lo + rot) % Bl;
            is_leader[a] = 1; partner[a] = f;
            is_leader[f] = 0; partner[f] = a;
        }
    }
    return 0;
}

int orc_align_to(orc_ctx* c, const double eC[3])
{
    double M[3] = { 0, 0, 0 };
    for (int64_t i = 0; i < c->N; ++i) for (int a = 0; a < 3; ++a) M[a] += c->S[3 * i + a];
    double m = sqrt(M[0] * M[0] + M[1] * M[1] + M[2] * M[2]);
    if (m / (double)c->N < 1e-6) return -1;
    double u[3] = { M[0] / m, M[1] / m, M[2] / m };
    /* Rodrigues rotation about k = u x eC by the angle between u and eC */
    double k[3] = { u[1] * eC[2] - u[2] * eC[1], u[2] * eC[0] - u[0] * eC[2], u[0] * eC[1] - u[1] * eC[0] };
    double s = sqrt(k[0] * k[0] + k[1] * k[1] + k[2] * k[2]);
    double co = u[0] * eC[0] + u[1] * eC[1] + u[2] * eC[2];
    if (s < 1e-300) {
        if (co > 0) { c->aligned = 1; memcpy(c->eC, eC, sizeof c->eC); return 0; }   /* already aligned */
        /* antiparallel: rotate by pi about any axis perpendicular to u */
        double t[3] = { 1, 0, 0 }; if (fabs(u[0]) > 0.9) { t[0] = 0; t[1] = 1; }
        k[0] = u[1] * t[2] - u[2] * t[1]; k[1] = u[2] * t[0] - u[0] * t[2]; k[2] = u[0] * t[1] - u[1] * t[0];
        s = sqrt(k[0] * k[0] + k[1] * k[1] + k[2] * k[2]);
        for (int a = 0; a < 3; ++a) k[a] /= s;
        s = 0.0;
    } else {
        for (int a = 0; a < 3; ++a) k[a] /= s;
    }
    for (int64_t i = 0; i < c->N; ++i) {
        double* S = &c->S[3 * i];
        double kxS[3] = { k[1] * S[2] - k[2] * S[1], k[2] * S[0] - k[0] * S[2], k[0] * S[1] - k[1] * S[0] };
        double kS = k[0] * S[0] + k[1] * S[1] + k[2] * S[2];
        double v[3], n2 = 0;
        for (int a = 0; a < 3; ++a) { v[a] = S[a] * co + kxS[a] * s + k[a] * kS * (1.0 - co); n2 += v[a] * v[a]; }
        double inv = 1.0 / sqrt(n2);
        for (int a = 0; a < 3; ++a) S[a] = v[a] * inv;
    }
    c->aligned = 1; memcpy(c->eC, eC, sizeof c->eC);
    return 0;
}

/* one pair move, written frame-free: X_par = X.eC, X_perp = X - X_par eC (C-22). */
static int pair_update(orc_ctx* c, double T, const double e[3], int colour, int64_t si, int64_t sj,
                       double* ML, int ml_mode, double* xdec, int may_be_neighbours)
{
    double u0, u1, u2;                                                    /* P:186, P:193 UniformRandom() x 3 (C-26) */
    const int64_t ci = c->structure ? si % c->Ncell : si;                 /* bcc: the leader's cell (its sublattice is the colour) */
    orc_pair_uniforms(c, (int)(ci % c->nx), (int)((ci / c->nx) % c->ny), (int)(ci / ((int64_t)c->nx * c->ny)), colour, c->sweep, &u0, &u1, &u2);
    double *Si = &c->S[3 * si], *Sj = &c->S[3 * sj], Sni[3], Snj[3];
    orc_cone_move(Si, c->cone, u0, u1, Sni);
    double Si_par = Si[0] * e[0] + Si[1] * e[1] + Si[2] * e[2];
    double Sj_par = Sj[0] * e[0] + Sj[1] * e[1] + Sj[2] * e[2];
    double Sni_par = Sni[0] * e[0] + Sni[1] * e[1] + Sni[2] * e[2];
    double perp[3], p2 = 0;
    for (int a = 0; a < 3; ++a) {                                         /* P:187-188 transverse compensation */
        perp[a] = (Sj[a] - Sj_par * e[a]) + (Si[a] - Si_par * e[a]) - (Sni[a] - Sni_par * e[a]);
        p2 += perp[a] * perp[a];
    }
    double xd = INFINITY;
    int accept = 0;
    double rho = (Sj[0] * Sj[0] + Sj[1] * Sj[1] + Sj[2] * Sj[2]) - p2;    /* P:189 radicand: S_j^2 - y'^2 - z'^2 */
    double MLhat = *ML;
    if (rho > 0.0) {                                                      /* C-13 */
        double Snj_par = ((Sj_par >= 0.0) ? 1.0 : -1.0) * sqrt(rho);      /* P:189 sign kept */
        double n2 = 0;
        for (int a = 0; a < 3; ++a) { Snj[a] = perp[a] + Snj_par * e[a]; n2 += Snj[a] * Snj[a]; }
        double inv = 1.0 / sqrt(n2);
        for (int a = 0; a < 3; ++a) Snj[a] *= inv;
        MLhat = *ML + Sni_par + Snj_par - Si_par - Sj_par;
        if (MLhat > 0.0) {                                                /* C-13 */
            double hi[3], hj[3];
            field_at(c, si, hi);
            field_at(c, sj, hj);
            double dE = site_energy_h(c, si, hi, Sni) + site_energy_h(c, sj, hj, Snj)
                      - site_energy_h(c, si, hi, Si) - site_energy_h(c, sj, hj, Sj);   /* P:193 (C-4) */
            if (may_be_neighbours) {
                /* serial Ref.[15] cross-check only: i and j may share a bond, so the change of the pair energy
                 * is evaluated sequentially (move i in the old field, then j in the field that already holds S'_i) */
                double keep[3] = { Si[0], Si[1], Si[2] };
                double dEi = site_energy_h(c, si, hi, Sni) - site_energy_h(c, si, hi, Si);
                Si[0] = Sni[0]; Si[1] = Sni[1]; Si[2] = Sni[2];
                field_at(c, sj, hj);
                dE = dEi + site_energy_h(c, sj, hj, Snj) - site_energy_h(c, sj, hj, Sj);
                Si[0] = keep[0]; Si[1] = keep[1]; Si[2] = keep[2];
            }
            double ratio = MLhat / *ML;
            /* P < (MLhat/ML)^2 |S_j,par / S'_j,par| exp(-dE/kT), in log form */
            xd = dE / T - 2.0 * log(ratio) - log(fabs(Sj_par / Snj_par)) + log(u2);
            accept = (xd < 0.0);
        }
    }
    if (xdec) xdec[si] = xd;
    if (accept) {
        for (int a = 0; a < 3; ++a) { Si[a] = Sni[a]; Sj[a] = Snj[a]; }
        if (ml_mode == 1) *ML = MLhat;                                    /* serial Ref.[15] variant only */
    }
    return accept;
}

int64_t orc_constrained_half_sweep(orc_ctx* c, double T, const double eC[3], int colour, double* ML,
                                   int ml_mode, int pairing_mode, double* xdec, uint8_t* acc)
{
    int64_t Nc = c->N / 2, count = 0;
    int64_t* partner = (int64_t*)malloc(sizeof(int64_t) * Nc);
    uint8_t* leader = (uint8_t*)calloc(Nc, 1);
    if (pairing_mode == 0) {
        if (orc_pairing(c, c->sweep, colour, partner, leader)) { free(partner); free(leader); return -1; }
    } else {
        /* literal P:38 / P:202: shuffle the indexes of this colour, then pick them sequentially in pairs */
        int64_t* p = (int64_t*)malloc(sizeof(int64_t) * Nc);
        for (int64_t a = 0; a < Nc; ++a) p[a] = a;
        for (int64_t a = Nc - 1; a > 0; --a) {
            uint32_t r[4]; draw(c, (uint32_t)a, TAG_ORACLE, 2 + colour, c->sweep, r);
            int64_t j = (int64_t)(((uint64_t)r[0] * (uint64_t)(a + 1)) >> 32);
            int64_t t = p[a]; p[a] = p[j]; p[j] = t;
        }
        for (int64_t a = 0; a + 1 < Nc; a += 2) { leader[p[a]] = 1; partner[p[a]] = p[a + 1]; leader[p[a + 1]] = 0; partner[p[a + 1]] = p[a]; }
        free(p);
    }
    for (int64_t a = 0; a < Nc; ++a) {                                    /* P:184 for i in 1..N step 2 */
        if (!leader[a]) continue;
        int64_t si = orc_site_of(c, colour, a), sj = orc_site_of(c, colour, partner[a]);
        int ok = pair_update(c, T, eC, colour, si, sj, ML, ml_mode, xdec, 0);
        if (acc) { acc[si] = (uint8_t)ok; acc[sj] = (uint8_t)ok; }
        count += 2 * ok;                                                  /* P:195 (C-23) */
    }
    free(partner); free(leader);
    return count;
}

/* Serial constrained MC of Ref.[15] ("the serial version as introduced in Ref. [15]"): pairs drawn from ALL
 * sites regardless of colour (Fisher-Yates over the whole lattice), exact M_L.  Cross-check mode only: it has
 * neither of the parallel algorithm's approximations (stale M_L, same-colour pairs), so on tiny lattices it must
 * reproduce the unconstrained ensemble's rotation-invariant observables exactly (pin P-17a). */
static int64_t serial_any_pair_sweep(orc_ctx* c, double T, const double e[3], double* ML)
{
    int64_t N = c->N, count = 0;
    int64_t* p = (int64_t*)malloc(sizeof(int64_t) * N);
    for (int64_t a = 0; a < N; ++a) p[a] = a;
    for (int64_t a = N - 1; a > 0; --a) {
        uint32_t r[4]; draw(c, (uint32_t)a, TAG_ORACLE, 4, c->sweep, r);
        int64_t j = (int64_t)(((uint64_t)r[0] * (uint64_t)(a + 1)) >> 32);
        int64_t t = p[a]; p[a] = p[j]; p[j] = t;
    }
    for (int64_t a = 0; a + 1 < N; a += 2) {
        int64_t si = p[a], sj = p[a + 1];
        int x = (int)(si % c->nx), y = (int)((si / c->nx) % c->ny), z = (int)(si / ((int64_t)c->nx * c->ny));
        count += 2 * pair_update(c, T, e, (x + y + z) & 1, si, sj, ML, 1, NULL, 1);
    }
    free(p);
    return count;
}

int orc_constrained_sweep(orc_ctx* c, double T, double theta, double phi, int64_t n, int ml_mode, int pairing_mode)
{
    double e[3] = { sin(theta) * cos(phi), sin(theta) * sin(phi), cos(theta) };
    if (!c->aligned || e[0] != c->eC[0] || e[1] != c->eC[1] || e[2] != c->eC[2])
        if (orc_align_to(c, e)) return -1;                                /* C-12 */
    c->torque_sampling = 1;
    for (int64_t it = 0; it < n; ++it) {
        double ML = 0.0;
        for (int64_t i = 0; i < c->N; ++i) ML += c->S[3 * i] * e[0] + c->S[3 * i + 1] * e[1] + c->S[3 * i + 2] * e[2];
        if (!(ML > 0.0)) { c->torque_sampling = 0; return -1; }
        if (pairing_mode == 2) {
            if (c->structure) return -1;                                      /* the serial cross-check mode is written for the sc lattice */
            orc_end_sweep(c, serial_any_pair_sweep(c, T, e, &ML)); continue;
        }
        int64_t count = orc_constrained_half_sweep(c, T, e, 0, &ML, ml_mode, pairing_mode, NULL, NULL);
        int64_t cb    = orc_constrained_half_sweep(c, T, e, 1, &ML, ml_mode, pairing_mode, NULL, NULL);   /* P:204 (C-5) */
        if (count < 0 || cb < 0) { c->torque_sampling = 0; return -1; }
        orc_end_sweep(c, count + cb);
    }
    c->torque_sampling = 0;
    return 0;
}

/* ------------------------------------------------------------------ read-out */
void orc_observables(orc_ctx* c, orc_obs* o)
{
    memset(o, 0, sizeof *o);
    measure(c, o);
    o->n_sites = (uint64_t)c->N; o->sweep = c->sweep; o->cone_rad = c->cone; o->last_acceptance = c->last_acceptance;
    o->n_samples = c->n_samples;
    for (int a = 0; a < 4; ++a) { o->sum_m[a] = c->sum_m[a]; o->sum_m2[a] = c->sum_m2[a]; }
    o->sum_E = c->sum_E; o->sum_E2 = c->sum_E2;
    for (int a = 0; a < 3; ++a) o->sum_torque[a] = c->sum_torque[a];
}

void orc_reset_accumulators(orc_ctx* c)
{
    c->n_samples = 0;
    memset(c->sum_m, 0, sizeof c->sum_m); memset(c->sum_m2, 0, sizeof c->sum_m2);
    c->sum_E = c->sum_E2 = 0; memset(c->sum_torque, 0, sizeof c->sum_torque);
}

int64_t orc_trace(const orc_ctx* c, int64_t max, double* rows)
{
    int64_t k = c->trace_len < max ? c->trace_len : max;
    memcpy(rows, &c->trace[6 * (c->trace_len - k)], sizeof(double) * 6 * k);
    return k;
}
