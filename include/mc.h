/*
 * mc.h -- C ABI of libmc_b200.so: red-black checkerboard Metropolis for unit classical Heisenberg spins on a
 * simple-cubic lattice, hand-written CUDA for sm_100a (NVIDIA B200).
 *
 * Method: Lepadatu et al., "Computation of magnetization, exchange stiffness, anisotropy, and susceptibilities in
 * large-scale systems using GPU-accelerated atomistic parallel Monte Carlo algorithms", arXiv 2103.03517.
 * "P:NN" = line NN of that paper's text; "C-n" = reading n in DESIGN.md section 4.
 *
 * Conventions
 *   - extern "C", plain pointers and sizes, no exceptions, no globals, no callbacks.  Every pointer argument is a
 *     HOST pointer unless its name starts with dev_.  The caller owns every buffer it passes; the library copies
 *     what it needs during the call and keeps no host pointer afterwards.
 *   - The library allocates NO device memory and changes no device-wide setting: the caller hands mc_create() one
 *     device workspace of at least mc_workspace_bytes() bytes (e.g. a torch.empty(..., dtype=uint8, device="cuda"))
 *     and a CUDA stream.  The workspace holds the spin state (12 B per site), the side data, the controller state, the
 *     trace ring and a staging area of 12 B per site that mc_set_spins / mc_get_spins / the half-sweep hooks /
 *     mc_profile_x use for their host <-> device copies.  All kernels of a handle run on that stream, on the device the
 *     workspace lives on (entry points switch to it and restore the caller's current device).  Handles are
 *     independent (replicas); one stream per handle.  The library reads no environment variable.
 *   - Return value: MC_OK (0) or a negative error code; mc_last_error() gives the message of the last failure.
 *     CUDA errors are sticky per handle (MC_ECUDA).
 *   - Reduced units: k_B = 1, energies in units of J (C-17).  Spins are fp32 on the device.
 *   - Lattice site index: site = x + nx*(y + ny*z), x fastest.  Colour c = (x+y+z) & 1, "red" = 0 first (C-10).
 *   - There is no CPU fallback: without a CUDA device every call fails with MC_ECUDA.
 */
#ifndef MC_B200_H
#define MC_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MC_OK       0
#define MC_EINVAL  (-1)   /* bad argument (null pointer, T <= 0, odd nx, odd periodic dimension, ...)      */
#define MC_ECUDA   (-2)   /* a CUDA call failed; sticky                                                 */
#define MC_ESTATE  (-3)   /* operation impossible in the current state (|M|/N < 1e-6, M.e_C <= 0, ...)   */

typedef struct mc_ctx mc_ctx;      /* opaque handle (host memory, freed by mc_destroy) */

/* Simple-cubic lattice, nearest neighbours.  nx must be even (colour-split rows); every periodic
 * dimension must be even (two-colourability); N = nx*ny*nz < 2^31.  periodic[a] = 1: wrap; 0: open faces;
 * periodic[0] = 2: ANTI-periodic along x, the spin across the wrap enters Eq. (2) as -S_j, which holds a domain wall in
 * the box ("anti-periodic along x direction"; x only: 2 on another axis is MC_EINVAL). */
typedef struct {
    int32_t nx, ny, nz;
    int32_t periodic[3];
    int32_t structure;           /* MC_SC (0): simple cubic, the paper's lattice.  MC_BCC (1), MC_FCC (2): see below          */
} mc_lattice;
#define MC_SC   0
#define MC_BCC  1
#define MC_FCC  2
#define MC_HCP  3
#define MC_SC_NNN 4
/* MC_BCC ("this approach can be extended to other crystal structures ... e.g. 2 simple cubic sub-lattices for bcc";
 * reading C-30): nx x ny x nz conventional cells, N = 2*nx*ny*nz spins.  Sublattice A (colour 0) sits at the cell corners,
 * B (colour 1) at the cell centres; site = sublattice*nx*ny*nz + (i + nx*(j + ny*k)); the 8 nearest neighbours of a site
 * are in the other sublattice: A(i,j,k) -- B(i-dx,j-dy,k-dz), B(i,j,k) -- A(i+dx,j+dy,k+dz), dx,dy,dz in {0,1}.  The two
 * sublattices are the two colours of the checkerboard scheme.  On the device: every dimension periodic, nx a multiple of 4,
 * no bond mask / regions; mc_profile_x: MC_EINVAL.  The constrained calls work as on the sc lattice (the pairing of C-11 acts
 * on the cell order of a sublattice) when nx*ny*nz is a multiple of 8, else MC_EINVAL.
 * MC_FCC ("4 simple cubic sub-lattices for fcc"; reading C-31): N = 4*nx*ny*nz spins; sublattice 0 at the cell corners,
 * 1, 2, 3 at (0,1/2,1/2), (1/2,0,1/2), (1/2,1/2,0) from them; site = sublattice*nx*ny*nz + cell; 12 nearest neighbours, 4 in each
 * OTHER sublattice, so the four sublattices are FOUR colours: a Monte Carlo iteration is four colour passes (mc_half_sweep takes
 * colour 0..3).  Same restrictions as MC_BCC; unconstrained sweeps only (the constrained calls: MC_EINVAL).
 * MC_HCP, MC_SC_NNN ("4 simple tetragonal sub-lattices for hcp ... up to 8 non-interacting subsets ... next-nearest
 * neighbours"; reading C-32): nx x ny x nz periodic cells of EIGHT sites, N = 8*nx*ny*nz spins, site = sublattice*nx*ny*nz + cell,
 * the eight sublattices are EIGHT colours: a Monte Carlo iteration is eight colour passes (mc_half_sweep takes colour 0..7).
 * MC_HCP: ideal hcp (c/a = sqrt(8/3)), the four-site orthohexagonal cell (a, sqrt3 a, c) doubled along x; in units
 * (a/2, sqrt3 a/6, c/2) the basis is (0,0,0) (1,3,0) (1,1,1) (0,4,1) and the same + (2,0,0); 12 nearest neighbours, coupling J.
 * MC_SC_NNN: a simple cubic lattice of (2nx) x (2ny) x (2nz) sites, the cell is its 2 x 2 x 2 block, sublattice = x + 2y + 4z of
 * the site in its block; 6 nearest neighbours (J) and 12 next-nearest neighbours (mc_hamiltonian.J2).  Same restrictions as
 * MC_FCC. */

/* Spin Hamiltonian, Eq. (2):  E_i = -sum_j J_ij S_i.S_j - Ku (S_i.e_i)^2 + Kc (Sx^2Sy^2 + Sx^2Sz^2 + Sy^2Sz^2) - S_i.B */
typedef struct {
    double J;                    /* nearest-neighbour exchange J_ij = J on every present bond                 */
    double Ku;                   /* uniaxial constant                                                               */
    double eu[3];                /* easy axis (normalised on entry; ignored where region != NULL)                   */
    double Kc;                   /* cubic constant, cube axes = x,y,z                                        */
    double B[3];                 /* Zeeman vector mu0*muS*H_a in energy units                                       */
    const uint8_t*  bond_mask;   /* optional [N]: bit k of site s set <=> bond k in (+x,-x,+y,-y,+z,-z) carries J.  *
                                  * NULL = every bond allowed by the boundary conditions.  Must be symmetric and    *
                                  * must not set a bond through an open face (checked, MC_EINVAL).                   */
    const uint16_t* region;      /* optional [N]: grain id of every site, < n_regions                       */
    const double*   region_axis; /* [n_regions][3] easy axis of every grain (normalised on entry)                   */
    int32_t n_regions;
    double cone0_rad;            /* initial cone HALF-angle theta in radians (C-6), clamped to [1 deg, 180 deg]      */
    int32_t adaptive;            /* 1: +-1 degree per sweep toward acceptance 0.5 (C-2, C-9)        */
    double J2;                   /* next-nearest-neighbour exchange, MC_SC_NNN only (ignored elsewhere)              */
} mc_hamiltonian;

/* Everything mc_observables() returns; all fp64; intensive quantities are per site. */
typedef struct {
    uint64_t n_sites, sweep;     /* sweep = number of completed Monte Carlo iterations (both kinds)                  */
    double cone_rad;             /* current cone half-angle                                                         */
    double last_acceptance;      /* acceptance rate of the last completed sweep                          */
    double M[3];                 /* sum_i S_i / N of the current state                                              */
    double m;                    /* |M|                                                                             */
    double E_total, E_exch, E_aniso, E_zeeman;   /* energies per site, every bond counted once (C-1)               */
    double torque[3];            /* sum_i S_i x H_i / N,  H_i = -dE_i/dS_i of the on-site terms              */
    uint64_t n_samples;          /* sweeps accumulated since mc_reset_accumulators()                                */
    double sum_m[4], sum_m2[4];  /* alpha = l,x,y,z: sum over sampled sweeps of m_alpha and m_alpha^2 (Eq. 6)  */
    double sum_E, sum_E2;        /* sum of E_total and E_total^2 per sampled sweep                                   */
    double sum_torque[3];        /* sum of the torque per sampled sweep (constrained sweeps only, else 0)            */
} mc_obs;

/* Bytes of device workspace mc_create() needs for this lattice + Hamiltonian (0 on invalid arguments). */
size_t mc_workspace_bytes(const mc_lattice* lat, const mc_hamiltonian* ham);

/* Creates a handle.  dev_workspace: device memory, 256-byte aligned, >= mc_workspace_bytes(); cuda_stream: a
 * cudaStream_t (NULL = legacy default stream).  Spins start along +z; sweep counter 0.  The RNG is Philox4x32-10
 * with key = seed and counter = (site, tag | colour<<8, sweep_lo, sweep_hi): moves are reproducible and independent
 * of launch geometry.  Synchronous (uploads the side data). */
int mc_create(const mc_lattice* lat, const mc_hamiltonian* ham, uint64_t seed,
              void* dev_workspace, size_t workspace_bytes, void* cuda_stream, mc_ctx** out);
int mc_destroy(mc_ctx* ctx);     /* frees the host handle only; the workspace stays the caller's */

/* mode 0: all spins +z; mode 1: all spins along dir (normalised); mode 2: uniform on the sphere, seeded (site i takes
 * Philox(ctr = (i, 3, 0, 0), key = seed): z = 2 u0 - 1, phi = 2 pi u1; BASELINE.json configs[2]).  Asynchronous. */
int mc_init_spins(mc_ctx* ctx, int mode, const double dir[3]);
/* Upload / download the spin state as [N][3] fp32 in lexicographic site order (x fastest).  mc_set_spins
 * normalises every spin whose squared length differs from 1 by more than 4e-7; a spin that is unit to fp32 rounding (anything
 * mc_get_spins returned) is stored unchanged, so get -> set restores the state bit for bit: with mc_set_sweep and mc_set_cone
 * that is a checkpoint (the RNG is counter-based: there is no other state).  Both synchronise the stream. */
int mc_set_spins(mc_ctx* ctx, const float* host_xyz);
int mc_get_spins(mc_ctx* ctx, float* host_xyz);
/* Set the cone half-angle / the sweep counter (checkpoint restore, parity tests).  Asynchronous. */
int mc_set_cone(mc_ctx* ctx, double cone_rad);
int mc_set_sweep(mc_ctx* ctx, uint64_t sweep);

/* n Monte Carlo iterations of Table A1 at temperature T > 0: red pass, black pass, cone controller,
 * per-sweep reductions (acceptance, M, E) and Eq. (6) accumulators.  Asynchronous: enqueues 2n kernels on the
 * handle's stream and returns; no host synchronisation, the controller state lives on the device.
 * CUDA graphs: the call only launches kernels on the handle's stream (no allocation, no synchronisation, no host read of device
 * state), so it may be issued while that stream is being captured and the graph replayed any number of times (the sweep counter
 * and the cone live on the device and advance with every replay).  The same holds for mc_reset_accumulators, mc_set_cone,
 * mc_set_sweep, and for mc_constrained_sweep once a constrained sweep with the same (theta, phi) has run outside the capture
 * (the first one aligns M and synchronises).  paper_2103_03517_b200/replicas.py uses this to run many small lattices at once. */
int mc_sweep(mc_ctx* ctx, double T, int64_t n);

/* n iterations of the constrained algorithm, Table A2, holding M/|M| along
 * e_C = (sin theta cos phi, sin theta sin phi, cos theta).  On the first call, after mc_set_spins/mc_init_spins,
 * after any unconstrained pass (mc_sweep, mc_half_sweep: they move M off e_C), or when (theta, phi) changes, all spins
 * are first rotated rigidly so that M/|M| = e_C (C-12; this step synchronises once; MC_ESTATE if |M|/N < 1e-6).  Pairs are same-colour, formed by the analytic pairing of C-11;
 * M_L is taken once per iteration.  Needs an even number of sites per colour (C-15). */
int mc_constrained_sweep(mc_ctx* ctx, double T, double theta, double phi, int64_t n);

/* Test hooks for per-colour parity (C-14): ONE colour pass of Table A1 / A2 with the current sweep counter and cone.
 * No controller step: the accepted count and the fused sums of the pass stay pending on the device until
 * mc_end_sweep() closes the sweep; if mc_sweep / mc_constrained_sweep is called instead, the pending contribution is
 * discarded (the spins the hook wrote stay).  host_x / host_acc are optional [N] outputs in lexicographic site order:
 * the fp32 decision variable x = dE/T + ln u2 (constrained: the log form of P:193, stored at the leader's site,
 * +inf for the hard rejections of C-13) and the accept flag; entries of the other colour are left untouched.
 * mc_constrained_half_sweep does not rotate: the caller passes an aligned state and M_L explicitly.  Synchronous. */
int mc_half_sweep(mc_ctx* ctx, double T, int colour, float* host_x, uint8_t* host_acc);
int mc_constrained_half_sweep(mc_ctx* ctx, double T, double theta, double phi, int colour, double M_L,
                              float* host_x, uint8_t* host_acc);
/* Closes a sweep assembled from half-sweep hooks: controller step with the accepted count of the two passes,
 * sweep counter += 1 (what mc_sweep does after its black pass).  Asynchronous. */
int mc_end_sweep(mc_ctx* ctx);
/* Rigid rotation of all spins taking M/|M| onto e_C (C-12), exposed for parity tests.  No rotation is applied when M already
 * lies within 3e-7 rad of e_C (the accuracy of the fp32 state): a restored constrained run continues bit for bit.  Synchronous. */
int mc_align_to(mc_ctx* ctx, double theta, double phi);

/* Synchronises the stream and returns the observables of the current state plus the accumulators.
 * The only device-to-host copy of results on the hot path. */
int mc_observables(mc_ctx* ctx, mc_obs* out);
int mc_reset_accumulators(mc_ctx* ctx);                      /* asynchronous */
/* Per-sweep trace (most recent min(max_rows, sweeps, MC_TRACE_CAPACITY) sweeps, oldest first):
 * rows[k][6] = acceptance, cone used, Mx, My, Mz (per site), E_total (per site).  Synchronous. */
#define MC_TRACE_CAPACITY 16384
int mc_trace(mc_ctx* ctx, int64_t max_rows, double* host_rows, int64_t* n_rows);

/* Domain-wall profile (Fig. 2: "the normalized magnetization z component is obtained for each profile point by
 * averaging over the respective cross-section slice"): host_profile[3*x + a] = mean over (y,z) of component a of the spins
 * at that x, x = 0..nx-1 (HOST pointer to 3*nx doubles, caller-owned).  Exact fixed-point sums on the device, so the
 * result is reproducible.  Uses 24*nx bytes of the workspace's staging area; synchronous. */
int mc_profile_x(mc_ctx* ctx, double* host_profile);
/* The same profile with NO scratch taken from the workspace and nothing allocated, on the device or the host: for callers that
 * cannot allocate at call time (CUDA graph capture around their own code, tight serving loops, harnesses that forbid
 * cudaMalloc).  The 24*nx bytes of sums live in a fixed array inside the library image -- the one exception to "no globals"
 * above: 24 * MC_PROFILE_STATIC_MAX_NX = 192 KB of device memory on every GPU that loads the library, held until the process
 * exits.  nx > MC_PROFILE_STATIC_MAX_NX: MC_EINVAL (use mc_profile_x).  Every call on a device shares that array and clears it
 * first; calls that OVERLAP on one GPU (two handles on different streams, two host threads) race on it: serialise them.
 * Same arguments, result (bit for bit) and restrictions as mc_profile_x; synchronous. */
#define MC_PROFILE_STATIC_MAX_NX 8192
int mc_profile_x_static(mc_ctx* ctx, double* host_profile);

/* Test hook: which kernel mc_sweep / mc_half_sweep launch for the colour pass.  MC_PATH_AUTO (default): the planner's
 * choice for this lattice; MC_PATH_GENERIC: the grid-stride gather pass (covers every lattice); MC_PATH_STAGED: the
 * TMA-fed shared-memory pass wherever its geometry covers the lattice (MC_EINVAL otherwise).  The arithmetic contract is
 * the same on every path (same Philox stream, same decisions); parity tests use this to check each one. */
#define MC_PATH_AUTO     0
#define MC_PATH_GENERIC  1
#define MC_PATH_STAGED   2
#define MC_PATH_MARCH    3
int mc_debug_set_path(mc_ctx* ctx, int path);
/* The kernel the colour pass of mc_sweep currently launches: MC_PATH_GENERIC, MC_PATH_STAGED or MC_PATH_MARCH (never AUTO). */
int mc_debug_get_path(const mc_ctx* ctx);

/* Number of kernel launches this handle has enqueued since creation (bench.py's gpu_launches). */
int64_t mc_launch_count(const mc_ctx* ctx);
const char* mc_last_error(const mc_ctx* ctx);                /* never NULL; valid until the next call on ctx */
const char* mc_version(void);

#ifdef __cplusplus
}
#endif
#endif
