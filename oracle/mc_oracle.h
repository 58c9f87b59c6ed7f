/*
 * mc_oracle.h -- C interface of the fp64 serial ORACLE for the checkerboard Metropolis path.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing outside tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may import, call, link or execute anything under oracle/.
 * It shares no code with the CUDA path (paper_2103_03517_b200/csrc/): no headers, helpers,
 * tables or constants.  Both sides restate the same written contract.
 *
 * Citations "P:NN" are line numbers of /root/reference/PAPER.md (Lepadatu et al., arXiv 2103.03517).
 *
 * Parity status: the paper prints no numeric worked example of a single update or sweep, so the
 * bit-level update sequence is "parity unpinned"; every function is pinned by closed forms,
 * invariants and brute force in tests/test_oracle_*.py (orc_align_to:
 * tests/test_oracle_align.py).
 */
#ifndef MC_ORACLE_H
#define MC_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct orc_ctx orc_ctx;

/* Per-sweep observables, all fp64, intensive quantities are per site. */
typedef struct {
    uint64_t n_sites, sweep;
    double cone_rad, last_acceptance;
    double M[3];            /* sum_i S_i / N                                     */
    double m;               /* |M|                                               */
    double E_total, E_exch, E_aniso, E_zeeman;   /* per site, bonds counted once */
    double torque[3];       /* sum_i S_i x (on-site field) / N                   */
    uint64_t n_samples;
    double sum_m[4], sum_m2[4];   /* alpha = l,x,y,z  (Eq. 6)              */
    double sum_E, sum_E2;
    double sum_torque[3];
} orc_obs;

/* Philox4x32-10 (Salmon et al., SC'11), exposed for the known-answer pin. */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* Uniform in (0,1): ((r >> 9) + 0.5) * 2^-23. */
double orc_uniform(uint32_t r);
double orc_uniform_azimuth(uint32_t w0, uint32_t w1);
/* The three uniforms of the unconstrained update of site (x,y,z): one Philox block per pair of x-neighbours of one
 * colour (x, x^2), 64 bits per site (reading C-26 in DESIGN.md section 4). */
void orc_site_uniforms(const orc_ctx* c, int x, int y, int z, int colour, uint64_t sweep, double* u0, double* u1, double* u2);
/* The same for the constrained pair move of the pair whose LEADER is (x,y,z) (stream TAG_PAIR). */
void orc_pair_uniforms(const orc_ctx* c, int x, int y, int z, int colour, uint64_t sweep, double* u0, double* u1, double* u2);
/* Cone trial move: S unit, theta = cone half-angle, u0,u1 in (0,1). */
void orc_cone_move(const double S[3], double theta, double u0, double u1, double Snew[3]);

/* mask: optional [N] bits (+x,-x,+y,-y,+z,-z); region: optional [N]; region_axis: [n_regions][3]. */
orc_ctx* orc_create(int nx, int ny, int nz, const int periodic[3],
                    double J, double Ku, const double eu[3], double Kc, const double B[3],
                    const uint8_t* bond_mask, const uint16_t* region,
                    const double* region_axis, int n_regions,
                    double cone0_rad, int adaptive, uint64_t seed);
/* Body-centred cubic lattice (two simple cubic sublattices = the two colours; reading C-30 in DESIGN.md): nx x ny x nz
 * conventional cells, 2 nx ny nz spins, 8 nearest neighbours, site = sublattice*nx*ny*nz + (i + nx*(j + ny*k)).
 * periodic[a] in {0,1}; no mask / regions.  The constrained calls work as on the sc lattice (two colours, the pairing acts on the
 * cell order of a sublattice; pairing_mode 2 is sc only). */
orc_ctx* orc_create_bcc(int nx, int ny, int nz, const int periodic[3],
                        double J, double Ku, const double eu[3], double Kc, const double B[3],
                        double cone0_rad, int adaptive, uint64_t seed);
/* Face-centred cubic lattice (four simple cubic sublattices = FOUR colours; reading C-31): 4 nx ny nz spins, 12 nearest
 * neighbours, 4 in each other sublattice; site = sublattice*nx*ny*nz + cell; a sweep is four colour passes 0, 1, 2, 3. */
orc_ctx* orc_create_fcc(int nx, int ny, int nz, const int periodic[3],
                        double J, double Ku, const double eu[3], double Kc, const double B[3],
                        double cone0_rad, int adaptive, uint64_t seed);
/* Basis mode ("4 simple tetragonal sub-lattices for hcp ... up to 8 non-interacting subsets ... next-nearest neighbours";
 * reading C-32): nx x ny x nz periodic cells of EIGHT sites, 8 nx ny nz spins, eight colours (a sweep is eight colour passes),
 * site = sublattice*nx*ny*nz + cell.  kind 3: ideal hcp, orthohexagonal cell doubled along x, 12 nearest neighbours (J; J2
 * ignored).  kind 4: simple cubic lattice of (2nx) x (2ny) x (2nz) sites, cell = its 2 x 2 x 2 block (sublattice = x + 2y + 4z of
 * the site in the block), 6 nearest (J) and 12 next-nearest (J2) neighbours.  Unconstrained sweeps only. */
orc_ctx* orc_create_basis(int kind, int nx, int ny, int nz, double J, double J2, double Ku, const double eu[3], double Kc, const double B[3],
                          double cone0_rad, int adaptive, uint64_t seed);
void orc_destroy(orc_ctx*);
/* periodic[a]: 0 open faces, 1 periodic, 2 anti-periodic (the spin across the wrap enters as -S_j). */
/* Slice-averaged magnetisation along x: out[3*x + a], a = x,y,z component. */
void orc_profile_x(const orc_ctx*, double* out);

void orc_set_spins(orc_ctx*, const double* xyz /* [N][3] lexicographic */);
void orc_set_spins_f32(orc_ctx*, const float* xyz);
void orc_get_spins(const orc_ctx*, double* xyz);
void orc_init_uniform(orc_ctx*, const double dir[3]);
void orc_init_random(orc_ctx*);   /* uniform on the sphere, Philox tag 3 keyed on the site */
void orc_set_cone(orc_ctx*, double cone_rad);
void orc_set_sweep(orc_ctx*, uint64_t sweep);
void orc_set_adaptive(orc_ctx*, int adaptive);
/* 0 = skip the per-sweep measurement / trace / accumulators (long equilibrations in the pins). */
void orc_set_sampling(orc_ctx*, int on);

/* One colour pass of Table A1.  Does not advance the sweep counter.
 * xdec[N] (optional): decision variable x = dE/T + ln u2 at the sites of this colour.
 * acc[N]  (optional): 1 where the move was accepted.  Returns the accepted count. */
int64_t orc_half_sweep(orc_ctx*, double T, int colour, double* xdec, uint8_t* acc);
/* Controller + sweep counter + trace + accumulators, count = accepted in both passes. */
void orc_end_sweep(orc_ctx*, int64_t count);
/* n repetitions of: red pass, black pass, end_sweep. */
void orc_sweep(orc_ctx*, double T, int64_t n);
/* Serial Metropolis, random visiting order -- cross-check mode only. */
void orc_sweep_random_order(orc_ctx*, double T, int64_t n);

/* Pairing function of the constrained pass (reading C-11).
 * Writes for every colour-linear index a in [0,Nc): partner[a] (colour-linear) and is_leader[a]. */
int orc_pairing(const orc_ctx*, uint64_t sweep, int colour, int64_t* partner, uint8_t* is_leader);
/* Colour-linear index a <-> lexicographic site. */
int64_t orc_site_of(const orc_ctx*, int colour, int64_t a);

/* Rigid rotation of all spins taking M/|M| onto e_C (reading C-12).  Returns 0, or -1 if |M|/N < 1e-6. */
int orc_align_to(orc_ctx*, const double eC[3]);
/* One colour pass of Table A2 with fixed M_L.
 * mode 0 = stale M_L (the paper's parallel algorithm);  1 = exact M_L updated after every accepted pair (serial, Ref.[15]).
 * pairing_mode 0 = analytic pairing; 1 = Fisher-Yates shuffle of the colour (literal P:38);
 * (orc_constrained_sweep only) 2 = serial Ref.[15]: pairs from all sites regardless of colour, exact M_L. */
int64_t orc_constrained_half_sweep(orc_ctx*, double T, const double eC[3], int colour, double* ML,
                                   int ml_mode, int pairing_mode, double* xdec, uint8_t* acc);
/* n repetitions of P:201-209 with e_C = (sin t cos p, sin t sin p, cos t); aligns on first use / direction change. */
int orc_constrained_sweep(orc_ctx*, double T, double theta, double phi, int64_t n, int ml_mode, int pairing_mode);

void orc_observables(orc_ctx*, orc_obs* out);
void orc_reset_accumulators(orc_ctx*);
/* rows [k][6]: acceptance, cone, mx, my, mz, E_total.  Returns number of rows written (most recent <= max). */
int64_t orc_trace(const orc_ctx*, int64_t max, double* rows);

/* Independent checks used by the pins. */
double orc_site_energy(const orc_ctx*, int64_t site, const double S[3]);   /* E_i of Eq.(2) */
double orc_total_energy(const orc_ctx*);   /* extensive H: every bond once + on-site terms */

#ifdef __cplusplus
}
#endif
#endif
