// mc_api.cu -- host side of libmc_b200.so: the C ABI declared in include/mc.h.
// Argument marshalling, workspace carving, launch configuration.  Every step of the hot path runs in the kernels
// of mc_kernels.cuh; there is no CPU fallback (without a device every entry point returns MC_ECUDA).
#include "mc_host.h"
#include "mc_util.cuh"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <vector>

using namespace mc;

namespace {

constexpr size_t ALIGN = 256;
inline size_t round_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Layout {            // byte offsets into the caller's workspace
    size_t spins, mask, region, axis, bonds, state, trace, staging, staging_bytes, total;
    long long plane, mask_plane, region_plane;
    int max_blocks;
};

constexpr int MAX_BLOCKS = 148 * 32;     // upper bound on the grid of a pass kernel

bool needs_mask(const mc_lattice* lat, const mc_hamiltonian* ham)
{
    return ham->bond_mask != nullptr || !lat->periodic[0] || !lat->periodic[1] || !lat->periodic[2];
}

int n_sublattices(int structure) { return structure == MC_BCC ? 2 : structure == MC_FCC ? 4 : (structure == MC_HCP || structure == MC_SC_NNN) ? 8 : 0; }

// basis mode (C-32): the run-time copy of the bond table (make_bond_table, mc_common.cuh: derived from the coordinates) with the
// couplings filled in.  Returns false if a bond stays inside a sublattice.
bool build_bond_table(int structure, float J, float J2, mc::BondEntry (*tab)[mc::MC_MAX_BONDS], unsigned char* n, unsigned char* n_lower)
{
    for (int a = 0; a < 8; ++a) {
        const mc::BondTableCT T = mc::make_bond_table(structure, a);
        if (!T.ok) return false;
        for (int r = 0; r < T.n; ++r) {
            tab[a][r].b = (signed char)T.row[r].b; tab[a][r].xmask = (signed char)T.row[r].xmask;
            tab[a][r].dy = (signed char)T.row[r].dy; tab[a][r].dz = (signed char)T.row[r].dz;
            tab[a][r].J = T.row[r].kind == 1 ? J : J2;
        }
        n[a] = (unsigned char)T.n; n_lower[a] = (unsigned char)T.nlower;
    }
    return true;
}

bool valid_lattice(const mc_lattice* lat)
{
    if (!lat) return false;
    const int dim[3] = { lat->nx, lat->ny, lat->nz };
    if (lat->structure == MC_BCC || lat->structure == MC_FCC || lat->structure == MC_HCP || lat->structure == MC_SC_NNN) {
        // P:34, C-30 / C-31 / C-32: sublattices as colours; fully periodic, rows of float4 items
        for (int a = 0; a < 3; ++a) if (dim[a] < 1 || lat->periodic[a] != 1) return false;
        if (lat->nx % 4) return false;
        return (double)n_sublattices(lat->structure) * (double)lat->nx * lat->ny * lat->nz < 2147483648.0;
    }
    if (lat->structure != MC_SC) return false;
    for (int a = 0; a < 3; ++a) {
        if (dim[a] < 1) return false;
        if (lat->periodic[a] && (dim[a] & 1)) return false;
        if (lat->periodic[a] < 0 || lat->periodic[a] > (a == 0 ? 2 : 1)) return false;     // anti-periodic (2) along x only
    }
    if (lat->nx & 1) return false;
    const double N = (double)lat->nx * lat->ny * lat->nz;
    return N < 2147483648.0;
}

Layout make_layout(const mc_lattice* lat, const mc_hamiltonian* ham)
{
    Layout L{};
    const bool sub = n_sublattices(lat->structure) != 0;                        // sublattices as colours, each a full grid of cells
    const size_t ncol = sub ? (size_t)n_sublattices(lat->structure) : 2;
    const size_t Nc = sub ? (size_t)lat->nx * lat->ny * lat->nz : (size_t)lat->nx / 2 * lat->ny * lat->nz;
    L.plane = (long long)round_up(Nc, 64);
    L.mask_plane = (long long)round_up(Nc, 256);
    L.region_plane = (long long)round_up(Nc, 128);
    L.max_blocks = MAX_BLOCKS;
    size_t off = 0;
    L.spins = off;    off += round_up((size_t)3 * ncol * L.plane * sizeof(float), ALIGN);
    L.mask = off;     if (needs_mask(lat, ham)) off += round_up((size_t)2 * L.mask_plane, ALIGN);
    L.region = off;   if (ham->region) off += round_up((size_t)2 * L.region_plane * sizeof(uint16_t), ALIGN);
    L.axis = off;     if (ham->region) off += round_up((size_t)ham->n_regions * sizeof(float4), ALIGN);
    L.bonds = off;    if (lat->structure == MC_HCP || lat->structure == MC_SC_NNN) off += round_up(sizeof(mc::BondEntry) * 8 * mc::MC_MAX_BONDS, ALIGN);
    L.state = off;    off += round_up(sizeof(DevState), ALIGN);
    L.trace = off;    off += round_up((size_t)TRACE_CAP * 6 * sizeof(double), ALIGN);
    // staging: the [N][3] fp32 lexicographic image of the state during mc_set_spins / mc_get_spins, or the [N] fp32 + [N] u8
    // outputs of a half-sweep hook, or the 3 nx int64 sums of mc_profile_x -- the library allocates nothing itself
    const size_t N = ncol * Nc;
    L.staging_bytes = round_up(N * 3 * sizeof(float), ALIGN) + round_up((size_t)lat->nx * 3 * sizeof(long long), ALIGN);
    L.staging = off;  off += L.staging_bytes;
    L.total = off;
    return L;
}

FastDiv make_div(uint32_t d)
{
    FastDiv f{ d, 0u, 0u };
    if (d <= 1) return f;
    uint32_t l = 0; while ((1ull << l) < d) ++l;                       // ceil(log2 d)
    const unsigned __int128 one = 1;
    const unsigned __int128 num = one << (31 + l);
    f.mul = (uint32_t)((num + d - 1) / d);                             // ceil(2^(31+l) / d) < 2^32
    f.shift = l - 1;
    return f;
}

}  // namespace

namespace mc { FastDiv host_make_div(uint32_t d) { return make_div(d); } }

namespace {

#define CU(call) MC_CU(call)
// every entry point runs on the handle's device, whatever the caller's current device is, and restores it on return
struct DeviceGuard {
    int prev = -1; bool switched = false;
    explicit DeviceGuard(int dev) { if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess; }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};
#define CHECK_CTX()                                                                                \
    if (!ctx) return MC_EINVAL; if (ctx->sticky) return ctx->sticky; ctx->err[0] = 0; DeviceGuard guard_(ctx->device)

int launch_pass(mc_ctx* ctx, int mode, int colour, float invT, int flags, float* dx, uint8_t* da)
{
    if (mode == MODE_SWEEP && ctx->tile_ok) return launch_pass_tile(ctx, colour, invT, flags, dx, da);
    if (mode == MODE_SWEEP && ctx->march_ok) return launch_pass_march(ctx, colour, invT, flags, dx, da);
    return launch_pass_generic(ctx, mode, colour, invT, flags, dx, da);
}

int launch_pair(mc_ctx* ctx, int colour, float invT, int flags, float* dx, uint8_t* da)
{
    return launch_pair_generic(ctx, colour, invT, flags, dx, da);
}

int launch_state(mc_ctx* ctx, int what, double a = 0, double b = 0, double c = 0, unsigned long long u = 0)
{
    state_kernel<<<1, 1, 0, ctx->stream>>>(ctx->P.st, what, a, b, c, u);
    ctx->launches += 1;
    CU(cudaGetLastError());
    return MC_OK;
}

// standalone measurement of the current state into st->meas (and st->ML)
int measure(mc_ctx* ctx)
{
    int rc;
    for (int col = 0; col < ctx->P.ncol; ++col)
        if ((rc = launch_pass(ctx, MODE_MEASURE, col, 0.0f, F_TORQUE | (col + 1 == ctx->P.ncol ? F_FINALIZE : 0), nullptr, nullptr))) return rc;
    ctx->ml_valid = true;
    return MC_OK;
}

int read_state(mc_ctx* ctx, DevState* host)
{
    CU(cudaMemcpyAsync(host, ctx->P.st, sizeof(DevState), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return MC_OK;
}

// A half-sweep hook that was not closed by mc_end_sweep() left its accepted count and fused sums in DevState: a following
// mc_sweep / mc_constrained_sweep starts from a clean sweep (the hook's contribution is discarded, the spins it wrote stay).
int discard_pending_hook(mc_ctx* ctx)
{
    if (!ctx->hook_pending) return MC_OK;
    ctx->hook_pending = false;
    return launch_state(ctx, ST_RESET_SWEEP);
}

void direction(double theta, double phi, double e[3])
{
    e[0] = sin(theta) * cos(phi); e[1] = sin(theta) * sin(phi); e[2] = cos(theta);
}

}  // namespace

// =================================================================================================================
extern "C" {

const char* mc_version(void) { return "mc_b200 0.1 (sm_100a)"; }

size_t mc_workspace_bytes(const mc_lattice* lat, const mc_hamiltonian* ham)
{
    if (!valid_lattice(lat) || !ham) return 0;
    if (ham->region && (ham->n_regions < 1 || !ham->region_axis)) return 0;
    return make_layout(lat, ham).total;
}

int mc_create(const mc_lattice* lat, const mc_hamiltonian* ham, uint64_t seed,
              void* dev_workspace, size_t workspace_bytes, void* cuda_stream, mc_ctx** out)
{
    if (!out) return MC_EINVAL;
    *out = nullptr;
    if (!valid_lattice(lat) || !ham || !dev_workspace) return MC_EINVAL;
    if (ham->region && (ham->n_regions < 1 || ham->n_regions > 65536 || !ham->region_axis)) return MC_EINVAL;
    if (lat->structure != MC_SC && (ham->bond_mask || ham->region)) return MC_EINVAL;
    if (((uintptr_t)dev_workspace) % ALIGN) return MC_EINVAL;
    const Layout L = make_layout(lat, ham);
    if (workspace_bytes < L.total) return MC_EINVAL;

    mc_ctx* ctx = new mc_ctx();
    memset(ctx, 0, sizeof *ctx);
    ctx->lat = *lat;
    ctx->J = ham->J; ctx->Ku = ham->Ku; ctx->Kc = ham->Kc; ctx->adaptive = ham->adaptive ? 1 : 0; ctx->seed = seed;
    double n = sqrt(ham->eu[0] * ham->eu[0] + ham->eu[1] * ham->eu[1] + ham->eu[2] * ham->eu[2]);
    for (int a = 0; a < 3; ++a) { ctx->eu[a] = n > 0 ? ham->eu[a] / n : (a == 2 ? 1.0 : 0.0); ctx->B[a] = ham->B[a]; }
    ctx->stream = (cudaStream_t)cuda_stream;

    auto bail = [&](int code, const char* msg) { fprintf(stderr, "mc_create: %s\n", msg); delete ctx; return code; };
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return bail(MC_ECUDA, "no CUDA device");
    {   // the workspace pointer decides the device of the handle (a process may hold handles on several devices)
        cudaPointerAttributes pa;
        if (cudaPointerGetAttributes(&pa, dev_workspace) == cudaSuccess && pa.type == cudaMemoryTypeDevice) dev = pa.device;
        else cudaGetLastError();
    }
    ctx->device = dev;
    DeviceGuard guard_(dev);
    if (cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return bail(MC_ECUDA, "cannot query the device");

    const int nx = lat->nx, ny = lat->ny, nz = lat->nz;
    const bool bcc = lat->structure == MC_BCC, fcc = lat->structure == MC_FCC;
    const bool basis = lat->structure == MC_HCP || lat->structure == MC_SC_NNN, sub = bcc || fcc || basis;
    const uint32_t ncol = sub ? (uint32_t)n_sublattices(lat->structure) : 2u;
    const uint32_t Nc = sub ? (uint32_t)nx * ny * nz : (uint32_t)nx / 2 * ny * nz, N = ncol * Nc, R = sub ? nx : nx / 2;
    char* ws = (char*)dev_workspace;
    Params& P = ctx->P;
    P.nx = nx; P.ny = ny; P.nz = nz; P.R = (int)R; P.Nc = Nc; P.N = N; P.invN = 1.0 / (double)N;
    P.anti_x = lat->periodic[0] == 2 ? 1 : 0;
    P.bcc = bcc ? 1 : 0; P.fcc = fcc ? 1 : 0; P.ncol = (int)ncol;
    P.basis = basis ? lat->structure : 0; P.sub = sub ? 1 : 0; P.bonds = nullptr;
    P.per_mask = (lat->periodic[0] ? 1 : 0) | (lat->periodic[1] ? 2 : 0) | (lat->periodic[2] ? 4 : 0);
    P.plane = L.plane; P.S = (float*)(ws + L.spins);
    P.mask = nullptr; P.mask_plane = L.mask_plane; P.region = nullptr; P.region_plane = L.region_plane; P.axis = nullptr;
    P.J = (float)ham->J; P.Ku = (float)ham->Ku; P.Kc = (float)ham->Kc; P.J2 = (float)ham->J2;
    for (int a = 0; a < 3; ++a) { P.eu[a] = (float)ctx->eu[a]; P.B[a] = (float)ham->B[a]; }
    P.seed_lo = (uint32_t)seed; P.seed_hi = (uint32_t)(seed >> 32);
    P.key = philox_key(P.seed_lo, P.seed_hi);
    P.st = (DevState*)(ws + L.state); P.max_blocks = L.max_blocks;
    {   // fixed-point unit 2^-k of the fused sums: the largest k <= 40 with N * (largest per-site term) * 2^k < 2^61
        const double bmag = sqrt(ham->B[0] * ham->B[0] + ham->B[1] * ham->B[1] + ham->B[2] * ham->B[2]);
        const double zJ = lat->structure == MC_SC_NNN ? 6.0 * fabs(ham->J) + 12.0 * fabs(ham->J2) : (bcc ? 8.0 : (fcc || basis) ? 12.0 : 6.0) * fabs(ham->J);
        const double mag = 1.0 + zJ + 2.0 * fabs(ham->Ku) + 2.0 * fabs(ham->Kc) + bmag;
        int lg = 0; while (ldexp(1.0, lg) < (double)N * mag) ++lg;
        int k = 61 - lg; if (k > 40) k = 40;
        P.fx_scale = (float)ldexp(1.0, k); P.fx_inv = ldexp(1.0, -k);
    }
    P.trace = (double*)(ws + L.trace);
    ctx->staging = ws + L.staging; ctx->staging_bytes = L.staging_bytes;

    ctx->aniso = (ham->Ku != 0.0 ? 1 : 0) | (ham->Kc != 0.0 ? 2 : 0);
    ctx->field = ham->B[0] != 0.0 || ham->B[1] != 0.0 || ham->B[2] != 0.0;
    ctx->masked = needs_mask(lat, ham);
    ctx->vec = (sub || nx % 8 == 0) ? 4 : 1;
    ctx->geom.RV = R / ctx->vec; ctx->geom.n_items = Nc / ctx->vec;
    ctx->geom.div_rv = make_div(ctx->geom.RV); ctx->geom.div_nz = make_div((uint32_t)nz);
    { uint32_t sh = 0; while (sh < 5 && ny % (2 << sh) == 0) ++sh; ctx->geom.yb_shift = sh; }      // up to 32 rows per block

    // pairing geometry (C-11); the constrained path needs an even colour population (C-15)
    ctx->pair_ok = (Nc % 2 == 0) && Nc >= 2 && ncol == 2;      // two-colour lattices (sc, bcc); fcc has four passes per sweep, hcp / sc_nnn eight
    if (ctx->pair_ok) {
        PairGeom& G = ctx->pgeom;
        uint32_t Bc = 32; while (Nc % (2 * Bc)) Bc >>= 1;
        G.B = Bc; G.H = Nc / Bc; G.Bl = Bc < 4 ? Bc : 4; G.Bh = Bc / G.Bl;
        if (ctx->vec == 4 && Bc < 4) ctx->pair_ok = false;      // sc: cannot happen (nx % 8 == 0 implies 8 | Nc); bcc: needs 8 | cells
        G.groups_per_chunk_vec = Bc / ctx->vec;
        G.n_threads = Nc / (2 * ctx->vec);
        G.div_r = make_div(R); G.div_ny = make_div((uint32_t)ny);
    }

    // ---- side data: bond mask (boundary conditions AND the caller's mask) and grain ids, colour-split on the host
    cudaError_t ce = cudaSuccess;
    if (basis) {                                                              // C-32: the bond table of the eight sublattices
        mc::BondEntry tab[8][mc::MC_MAX_BONDS];
        memset(tab, 0, sizeof tab);
        if (!build_bond_table(lat->structure, (float)ham->J, (float)ham->J2, tab, P.nbonds, P.nlower)) return bail(MC_EINVAL, "basis mode: a bond inside a sublattice");
        ce = cudaMemcpyAsync(ws + L.bonds, tab, sizeof tab, cudaMemcpyHostToDevice, ctx->stream);
        if (ce == cudaSuccess) ce = cudaStreamSynchronize(ctx->stream);
        if (ce != cudaSuccess) return bail(MC_ECUDA, cudaGetErrorString(ce));
        P.bonds = (const mc::BondEntry*)(ws + L.bonds);
    }
    if (ctx->masked) {
        std::vector<uint8_t> split((size_t)2 * L.mask_plane, 0);
        const int dim[3] = { nx, ny, nz };
        for (int z = 0; z < nz; ++z) for (int y = 0; y < ny; ++y) for (int x = 0; x < nx; ++x) {
            const size_t s = (size_t)x + (size_t)nx * (y + (size_t)ny * z);
            const int pos[3] = { x, y, z };
            uint8_t bc = 0;
            for (int k = 0; k < 6; ++k) {
                const int axis = k >> 1, q = pos[axis] + ((k & 1) ? -1 : 1);
                if (lat->periodic[axis] || (q >= 0 && q < dim[axis])) bc |= (uint8_t)(1u << k);
            }
            uint8_t m = bc;
            if (ham->bond_mask) {
                m = ham->bond_mask[s];
                if (m & ~bc & 0x3F) return bail(MC_EINVAL, "bond_mask sets a bond through an open face");
                if (m & 0xC0) return bail(MC_EINVAL, "bond_mask has bits above bit 5");
                // symmetry: bit k of s  <=>  bit (k^1) of the neighbour in direction k
                for (int k = 0; k < 6; ++k) {
                    if (!((bc >> k) & 1)) continue;
                    int qv[3] = { x, y, z };
                    const int axis = k >> 1;
                    qv[axis] = (qv[axis] + ((k & 1) ? -1 : 1) + dim[axis]) % dim[axis];
                    const size_t t = (size_t)qv[0] + (size_t)nx * (qv[1] + (size_t)ny * qv[2]);
                    if (((m >> k) & 1) != ((ham->bond_mask[t] >> (k ^ 1)) & 1)) return bail(MC_EINVAL, "bond_mask is not symmetric");
                }
            }
            const int c = (x + y + z) & 1;
            split[(size_t)c * L.mask_plane + ((size_t)(x >> 1) + (size_t)R * (y + (size_t)ny * z))] = m;
        }
        ce = cudaMemcpyAsync(ws + L.mask, split.data(), split.size(), cudaMemcpyHostToDevice, ctx->stream);
        if (ce == cudaSuccess) ce = cudaStreamSynchronize(ctx->stream);
        if (ce != cudaSuccess) return bail(MC_ECUDA, cudaGetErrorString(ce));
        P.mask = (const uint8_t*)(ws + L.mask);
    }
    if (ham->region) {
        if (!(ctx->aniso & 1)) { /* grain axes only matter with Ku != 0; keep the table anyway */ }
        std::vector<uint16_t> split((size_t)2 * L.region_plane, 0);
        for (int z = 0; z < nz; ++z) for (int y = 0; y < ny; ++y) for (int x = 0; x < nx; ++x) {
            const size_t s = (size_t)x + (size_t)nx * (y + (size_t)ny * z);
            if ((int)ham->region[s] >= ham->n_regions) return bail(MC_EINVAL, "region id out of range");
            const int c = (x + y + z) & 1;
            split[(size_t)c * L.region_plane + ((size_t)(x >> 1) + (size_t)R * (y + (size_t)ny * z))] = ham->region[s];
        }
        std::vector<float4> axes((size_t)ham->n_regions);
        for (int r = 0; r < ham->n_regions; ++r) {
            const double* v = ham->region_axis + 3 * (size_t)r;
            const double m = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
            if (!(m > 0)) return bail(MC_EINVAL, "zero region axis");
            axes[r] = make_float4((float)(v[0] / m), (float)(v[1] / m), (float)(v[2] / m), 0.0f);
        }
        ce = cudaMemcpyAsync(ws + L.region, split.data(), split.size() * sizeof(uint16_t), cudaMemcpyHostToDevice, ctx->stream);
        if (ce == cudaSuccess) ce = cudaMemcpyAsync(ws + L.axis, axes.data(), axes.size() * sizeof(float4), cudaMemcpyHostToDevice, ctx->stream);
        if (ce == cudaSuccess) ce = cudaStreamSynchronize(ctx->stream);
        if (ce != cudaSuccess) return bail(MC_ECUDA, cudaGetErrorString(ce));
        P.region = (const uint16_t*)(ws + L.region);
        P.axis = (const float4*)(ws + L.axis);
    }

    plan_tile(ctx);
    plan_march(ctx);

    // ---- device state
    DevState st; memset(&st, 0, sizeof st);
    const double deg = M_PI / 180.0;
    double cone = ham->cone0_rad; if (!(cone >= deg)) cone = deg; if (cone > M_PI) cone = M_PI;
    st.cone = cone; st.one_minus_cos = mc::one_minus_cos_of(cone); st.adaptive = ctx->adaptive;
    st.eC[2] = 1.0;
    ce = cudaMemcpyAsync(P.st, &st, sizeof st, cudaMemcpyHostToDevice, ctx->stream);
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(ctx->stream);
    if (ce != cudaSuccess) return bail(MC_ECUDA, cudaGetErrorString(ce));
    ctx->eC[2] = 1.0;
    *out = ctx;
    const double up[3] = { 0, 0, 1 };
    const int rc = mc_init_spins(ctx, 0, up);
    if (rc) { *out = nullptr; delete ctx; return rc; }
    return MC_OK;
}

int mc_destroy(mc_ctx* ctx) { if (!ctx) return MC_EINVAL; delete ctx; return MC_OK; }

const char* mc_last_error(const mc_ctx* ctx) { return ctx ? ctx->err : "null handle"; }
int64_t mc_launch_count(const mc_ctx* ctx) { return ctx ? ctx->launches : 0; }

int mc_debug_set_path(mc_ctx* ctx, int path)
{
    CHECK_CTX();
    if (path == MC_PATH_AUTO) { const bool keep = ctx->tile_possible; plan_tile(ctx); ctx->tile_possible = keep || ctx->tile_possible; plan_march(ctx); }
    else if (path == MC_PATH_GENERIC) { ctx->tile_ok = false; ctx->march_ok = false; }
    else if (path == MC_PATH_STAGED) {
        if (!ctx->tile_possible) return fail(ctx, MC_EINVAL, "mc_debug_set_path: the staged pass does not cover this lattice / Hamiltonian");
        ctx->tile_ok = true; ctx->march_ok = false;
    } else if (path == MC_PATH_MARCH) {
        if (!ctx->march_possible) return fail(ctx, MC_EINVAL, "mc_debug_set_path: the z-march pass does not cover this lattice / Hamiltonian");
        ctx->march_ok = true; ctx->tile_ok = false;
    } else return fail(ctx, MC_EINVAL, "mc_debug_set_path: unknown path");
    ctx->path = path;
    return MC_OK;
}

int mc_debug_get_path(const mc_ctx* ctx)
{
    if (!ctx) return MC_EINVAL;
    return ctx->tile_ok ? MC_PATH_STAGED : (ctx->march_ok ? MC_PATH_MARCH : MC_PATH_GENERIC);
}

int mc_init_spins(mc_ctx* ctx, int mode, const double dir[3])
{
    CHECK_CTX();
    double d[3] = { 0, 0, 1 };
    if (mode == 1) {
        if (!dir) return fail(ctx, MC_EINVAL, "mc_init_spins: dir is null");
        const double n = sqrt(dir[0] * dir[0] + dir[1] * dir[1] + dir[2] * dir[2]);
        if (!(n > 0)) return fail(ctx, MC_EINVAL, "mc_init_spins: zero direction");
        for (int a = 0; a < 3; ++a) d[a] = dir[a] / n;
    } else if (mode == 2) {
        init_random_kernel<<<(ctx->P.Nc + 255) / 256, 256, 0, ctx->stream>>>(ctx->P);
        ctx->launches += 1;
        CU(cudaGetLastError());
        ctx->ml_valid = false; ctx->aligned = false;
        return MC_OK;
    } else if (mode != 0) return fail(ctx, MC_EINVAL, "mc_init_spins: unknown mode");
    float f[3] = { (float)d[0], (float)d[1], (float)d[2] };
    const double fn = sqrt((double)f[0] * f[0] + (double)f[1] * f[1] + (double)f[2] * f[2]);
    for (int a = 0; a < 3; ++a) f[a] = (float)(f[a] / fn);
    fill_kernel<<<(ctx->P.Nc + 255) / 256, 256, 0, ctx->stream>>>(ctx->P, f[0], f[1], f[2]);
    ctx->launches += 1;
    CU(cudaGetLastError());
    ctx->ml_valid = false; ctx->aligned = false;
    return MC_OK;
}

int mc_set_spins(mc_ctx* ctx, const float* host_xyz)
{
    CHECK_CTX();
    if (!host_xyz) return fail(ctx, MC_EINVAL, "mc_set_spins: null pointer");
    const size_t bytes = (size_t)ctx->P.N * 3 * sizeof(float);
    float* tmp = (float*)ctx->staging;                           // staging area of the caller's workspace
    CU(cudaMemcpyAsync(tmp, host_xyz, bytes, cudaMemcpyHostToDevice, ctx->stream));
    lex_to_split_kernel<<<(ctx->P.N + 255) / 256, 256, 0, ctx->stream>>>(ctx->P, tmp);
    ctx->launches += 1;
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->ml_valid = false; ctx->aligned = false;
    return MC_OK;
}

int mc_get_spins(mc_ctx* ctx, float* host_xyz)
{
    CHECK_CTX();
    if (!host_xyz) return fail(ctx, MC_EINVAL, "mc_get_spins: null pointer");
    const size_t bytes = (size_t)ctx->P.N * 3 * sizeof(float);
    float* tmp = (float*)ctx->staging;
    split_to_lex_kernel<<<(ctx->P.N + 255) / 256, 256, 0, ctx->stream>>>(ctx->P, tmp);
    ctx->launches += 1;
    CU(cudaGetLastError());
    CU(cudaMemcpyAsync(host_xyz, tmp, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return MC_OK;
}

int mc_set_cone(mc_ctx* ctx, double cone_rad)
{
    CHECK_CTX();
    const double deg = M_PI / 180.0;
    if (!(cone_rad >= deg) || cone_rad > M_PI) return fail(ctx, MC_EINVAL, "mc_set_cone: cone must be in [1 deg, 180 deg]");
    return launch_state(ctx, ST_CONE, cone_rad);
}

int mc_set_sweep(mc_ctx* ctx, uint64_t sweep)
{
    CHECK_CTX();
    return launch_state(ctx, ST_SWEEP, 0, 0, 0, (unsigned long long)sweep);
}

int mc_reset_accumulators(mc_ctx* ctx)
{
    CHECK_CTX();
    return launch_state(ctx, ST_RESET_ACC);
}

int mc_sweep(mc_ctx* ctx, double T, int64_t n)
{
    CHECK_CTX();
    if (!(T > 0.0) || n < 0) return fail(ctx, MC_EINVAL, "mc_sweep: need T > 0 and n >= 0");      // C-16
    const float invT = (float)(1.0 / T);
    if (n > 0) {
        int rc;
        if ((rc = discard_pending_hook(ctx))) return rc;
        ctx->aligned = false;             // an unconstrained pass moves M off e_C: the next constrained sweep re-aligns (C-12)
    }
    for (int64_t i = 0; i < n; ++i) {
        int rc;
        for (int col = 0; col + 1 < ctx->P.ncol; ++col)
            if ((rc = launch_pass(ctx, MODE_SWEEP, col, invT, 0, nullptr, nullptr))) return rc;                         // P:166 (fcc: three of four subsets)
        if ((rc = launch_pass(ctx, MODE_SWEEP, ctx->P.ncol - 1, invT, F_FINALIZE, nullptr, nullptr))) return rc;
    }
    if (n > 0) ctx->ml_valid = true;      // finalize refreshed M_L = M.e_C
    return MC_OK;
}

int mc_align_to(mc_ctx* ctx, double theta, double phi)
{
    CHECK_CTX();
    int rc;
    if ((rc = measure(ctx))) return rc;
    DevState st;
    if ((rc = read_state(ctx, &st))) return rc;
    const double M[3] = { st.meas[0], st.meas[1], st.meas[2] };
    const double mlen = sqrt(M[0] * M[0] + M[1] * M[1] + M[2] * M[2]);
    if (mlen / (double)ctx->P.N < 1e-6) return fail(ctx, MC_ESTATE, "cannot align: |M|/N < 1e-6");
    double e[3]; direction(theta, phi, e);
    const double u[3] = { M[0] / mlen, M[1] / mlen, M[2] / mlen };
    // Rodrigues rotation about k = u x e by the angle between u and e:  R = c I + s [k]_x + (1 - c) k k^T
    double k[3] = { u[1] * e[2] - u[2] * e[1], u[2] * e[0] - u[0] * e[2], u[0] * e[1] - u[1] * e[0] };
    double s = sqrt(k[0] * k[0] + k[1] * k[1] + k[2] * k[2]);
    const double c = u[0] * e[0] + u[1] * e[1] + u[2] * e[2];
    double Rm[9] = { 1, 0, 0, 0, 1, 0, 0, 0, 1 };
    bool identity = false;
    // M already along e_C to the accuracy of the fp32 state (e.g. a restored checkpoint of a constrained run): no rotation,
    // so that the restored run continues bit for bit
    if (s < 3e-7 && c > 0) identity = true;
    else if (s < 1e-300) {
        if (c > 0) identity = true;
        else {
            double t[3] = { 1, 0, 0 }; if (fabs(u[0]) > 0.9) { t[0] = 0; t[1] = 1; }
            k[0] = u[1] * t[2] - u[2] * t[1]; k[1] = u[2] * t[0] - u[0] * t[2]; k[2] = u[0] * t[1] - u[1] * t[0];
            const double kn = sqrt(k[0] * k[0] + k[1] * k[1] + k[2] * k[2]);
            for (int a = 0; a < 3; ++a) k[a] /= kn;
            s = 0.0;
        }
    } else { for (int a = 0; a < 3; ++a) k[a] /= s; }
    if (!identity) {
        const double K[9] = { 0, -k[2], k[1], k[2], 0, -k[0], -k[1], k[0], 0 };
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j)
            Rm[3 * i + j] = (i == j ? c : 0.0) + s * K[3 * i + j] + (1.0 - c) * k[i] * k[j];
        Mat3 Rf; for (int i = 0; i < 9; ++i) Rf.m[i] = (float)Rm[i];
        rotate_kernel<<<(ctx->P.Nc + 255) / 256, 256, 0, ctx->stream>>>(ctx->P, Rf);
        ctx->launches += 1;
        CU(cudaGetLastError());
    }
    if ((rc = launch_state(ctx, ST_EC, e[0], e[1], e[2]))) return rc;
    ctx->theta = theta; ctx->phi = phi; for (int a = 0; a < 3; ++a) ctx->eC[a] = e[a];
    ctx->aligned = true; ctx->ml_valid = false;
    return MC_OK;
}

int mc_constrained_sweep(mc_ctx* ctx, double T, double theta, double phi, int64_t n)
{
    CHECK_CTX();
    if (!(T > 0.0) || n < 0) return fail(ctx, MC_EINVAL, "mc_constrained_sweep: need T > 0 and n >= 0");
    if (!ctx->pair_ok) return fail(ctx, MC_EINVAL, "mc_constrained_sweep: needs a two-colour lattice (sc, bcc) with an even number of sites per colour (C-15; bcc: cells a multiple of 8)");
    int rc;
    if (!ctx->aligned || theta != ctx->theta || phi != ctx->phi) { if ((rc = mc_align_to(ctx, theta, phi))) return rc; }
    if (n == 0) return MC_OK;
    if (!ctx->ml_valid) {
        if ((rc = measure(ctx))) return rc;
        DevState st;
        if ((rc = read_state(ctx, &st))) return rc;
        if (!(st.ML > 0.0)) return fail(ctx, MC_ESTATE, "mc_constrained_sweep: M.e_C <= 0");
    }
    if ((rc = discard_pending_hook(ctx))) return rc;
    const float invT = (float)(1.0 / T);
    const int fl = F_TORQUE | F_SAMPLE_TORQUE;
    for (int64_t i = 0; i < n; ++i) {
        if ((rc = launch_pair(ctx, 0, invT, fl, nullptr, nullptr))) return rc;
        if ((rc = launch_pair(ctx, 1, invT, fl | F_FINALIZE, nullptr, nullptr))) return rc;
    }
    ctx->ml_valid = true;
    return MC_OK;
}

// ---- test hooks ---------------------------------------------------------------------------------------------
static int hook_common(mc_ctx* ctx, int colour, float* host_x, uint8_t* host_acc, bool pair, float invT)
{
    const uint32_t N = ctx->P.N;
    // outputs in the staging area of the workspace: [N] fp32 decision variables, then [N] accept flags
    float* dx = host_x ? (float*)ctx->staging : nullptr;
    uint8_t* da = host_acc ? (uint8_t*)ctx->staging + round_up((size_t)N * sizeof(float), ALIGN) : nullptr;
    if (dx) CU(cudaMemsetAsync(dx, 0xFF, (size_t)N * sizeof(float), ctx->stream));
    if (da) CU(cudaMemsetAsync(da, 0, (size_t)N, ctx->stream));
    ctx->hook_pending = true;             // the pass leaves its count and fused sums in DevState until mc_end_sweep()
    int rc = pair ? launch_pair(ctx, colour, invT, F_TORQUE, dx, da) : launch_pass(ctx, MODE_SWEEP, colour, invT, 0, dx, da);
    if (rc) return rc;
    std::vector<float> hx; std::vector<uint8_t> ha;
    if (host_x)   { hx.resize(N); CU(cudaMemcpyAsync(hx.data(), dx, (size_t)N * sizeof(float), cudaMemcpyDeviceToHost, ctx->stream)); }
    if (host_acc) { ha.resize(N); CU(cudaMemcpyAsync(ha.data(), da, (size_t)N, cudaMemcpyDeviceToHost, ctx->stream)); }
    CU(cudaStreamSynchronize(ctx->stream));
    const int nx = ctx->P.nx, ny = ctx->P.ny;
    for (uint32_t s = 0; (host_x || host_acc) && s < N; ++s) {
        const int x = s % nx, y = (s / nx) % ny, z = s / ((uint32_t)nx * ny);
        if ((ctx->P.sub ? (int)(s / ctx->P.Nc) : ((x + y + z) & 1)) != colour) continue;      // bcc / fcc: colour = sublattice
        if (host_x) host_x[s] = hx[s];
        if (host_acc) host_acc[s] = ha[s];
    }
    ctx->ml_valid = false;
    if (!pair) ctx->aligned = false;
    return MC_OK;
}

int mc_half_sweep(mc_ctx* ctx, double T, int colour, float* host_x, uint8_t* host_acc)
{
    CHECK_CTX();
    if (!(T > 0.0) || colour < 0 || colour >= ctx->P.ncol) return fail(ctx, MC_EINVAL, "mc_half_sweep: need T > 0 and a colour of the lattice (0, 1; fcc: 0..3; hcp, sc_nnn: 0..7)");
    return hook_common(ctx, colour, host_x, host_acc, false, (float)(1.0 / T));
}

int mc_constrained_half_sweep(mc_ctx* ctx, double T, double theta, double phi, int colour, double M_L,
                              float* host_x, uint8_t* host_acc)
{
    CHECK_CTX();
    if (!(T > 0.0) || (colour != 0 && colour != 1) || !(M_L > 0.0)) return fail(ctx, MC_EINVAL, "mc_constrained_half_sweep: bad argument");
    if (!ctx->pair_ok) return fail(ctx, MC_EINVAL, "mc_constrained_half_sweep: needs a two-colour lattice with an even number of sites per colour (C-15; bcc: cells a multiple of 8)");
    double e[3]; direction(theta, phi, e);
    int rc;
    if ((rc = launch_state(ctx, ST_EC, e[0], e[1], e[2]))) return rc;
    if ((rc = launch_state(ctx, ST_ML, M_L))) return rc;
    for (int a = 0; a < 3; ++a) ctx->eC[a] = e[a];
    ctx->theta = theta; ctx->phi = phi;
    return hook_common(ctx, colour, host_x, host_acc, true, (float)(1.0 / T));
}

int mc_end_sweep(mc_ctx* ctx)
{
    CHECK_CTX();
    finalize_kernel<<<1, BLOCK, 0, ctx->stream>>>(ctx->P, 0, 0);
    ctx->launches += 1;
    CU(cudaGetLastError());
    ctx->hook_pending = false;
    return MC_OK;
}

// ---- read-out -----------------------------------------------------------------------------------------------
int mc_observables(mc_ctx* ctx, mc_obs* out)
{
    CHECK_CTX();
    if (!out) return fail(ctx, MC_EINVAL, "mc_observables: null pointer");
    int rc;
    const bool keep = ctx->ml_valid;
    if ((rc = measure(ctx))) return rc;
    ctx->ml_valid = keep || ctx->ml_valid;
    DevState st;
    if ((rc = read_state(ctx, &st))) return rc;
    memset(out, 0, sizeof *out);
    const double invN = 1.0 / (double)ctx->P.N;
    out->n_sites = ctx->P.N; out->sweep = st.sweep; out->cone_rad = st.cone; out->last_acceptance = st.last_acceptance;
    for (int a = 0; a < 3; ++a) { out->M[a] = st.meas[a] * invN; out->torque[a] = st.meas[6 + a] * invN; }
    out->m = sqrt(out->M[0] * out->M[0] + out->M[1] * out->M[1] + out->M[2] * out->M[2]);
    out->E_exch = st.meas[3] * invN; out->E_aniso = st.meas[4] * invN; out->E_zeeman = st.meas[5] * invN;
    out->E_total = out->E_exch + out->E_aniso + out->E_zeeman;
    out->n_samples = st.n_samples;
    for (int a = 0; a < 4; ++a) { out->sum_m[a] = st.sum_m[a]; out->sum_m2[a] = st.sum_m2[a]; }
    out->sum_E = st.sum_E; out->sum_E2 = st.sum_E2;
    for (int a = 0; a < 3; ++a) out->sum_torque[a] = st.sum_torque[a];
    return MC_OK;
}

int mc_profile_x(mc_ctx* ctx, double* host_profile)
{
    CHECK_CTX();
    if (!host_profile) return fail(ctx, MC_EINVAL, "mc_profile_x: null pointer");
    if (ctx->P.sub) return fail(ctx, MC_EINVAL, "mc_profile_x: simple cubic lattices only");
    const int nx = ctx->P.nx;
    const size_t bytes = (size_t)nx * 3 * sizeof(long long);
    long long* tmp = (long long*)((char*)ctx->staging + ctx->staging_bytes - round_up(bytes, ALIGN));   // tail of the staging area
    CU(cudaMemsetAsync(tmp, 0, bytes, ctx->stream));
    const uint32_t rows = (uint32_t)ctx->P.ny * (uint32_t)ctx->P.nz;
    const uint32_t n_threads = (uint32_t)ctx->P.R * ((rows + PROFILE_ROWS - 1) / PROFILE_ROWS);
    profile_x_kernel<<<(n_threads + BLOCK - 1) / BLOCK, BLOCK, 0, ctx->stream>>>(ctx->P, tmp);
    ctx->launches += 1;
    CU(cudaGetLastError());
    std::vector<long long> sums((size_t)nx * 3);
    CU(cudaMemcpyAsync(sums.data(), tmp, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    const double scale = ctx->P.fx_inv / ((double)ctx->P.ny * (double)ctx->P.nz);
    for (size_t i = 0; i < sums.size(); ++i) host_profile[i] = (double)sums[i] * scale;
    return MC_OK;
}

int mc_trace(mc_ctx* ctx, int64_t max_rows, double* host_rows, int64_t* n_rows)
{
    CHECK_CTX();
    if (!host_rows || !n_rows || max_rows < 0) return fail(ctx, MC_EINVAL, "mc_trace: bad argument");
    DevState st;
    int rc;
    if ((rc = read_state(ctx, &st))) return rc;
    int64_t have = (int64_t)(st.trace_rows < (unsigned long long)TRACE_CAP ? st.trace_rows : (unsigned long long)TRACE_CAP);
    int64_t k = have < max_rows ? have : max_rows;
    std::vector<double> ring((size_t)TRACE_CAP * 6);
    CU(cudaMemcpyAsync(ring.data(), ctx->P.trace, ring.size() * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    for (int64_t i = 0; i < k; ++i) {
        const unsigned long long row = (st.trace_rows - (unsigned long long)k + (unsigned long long)i) % (unsigned long long)TRACE_CAP;
        memcpy(host_rows + 6 * i, ring.data() + 6 * row, 6 * sizeof(double));
    }
    *n_rows = k;
    return MC_OK;
}

}  // extern "C"
