// mc_march.cu -- instantiations, planner and launcher of the register-carried march colour pass (mc_march.cuh).
#include "mc_host.h"
#include "mc_march.cuh"

namespace mc {
namespace {

typedef void (*MarchFn)(const Params, const MarchGeom, int, float, int, float*, uint8_t*);
template <bool MASKED, int AXIS, bool DEBUG> MarchFn pick_march_a(int aniso)
{
    switch (aniso) {
        case 0: return march_pass_kernel<0, MASKED, AXIS, DEBUG>;  case 1: return march_pass_kernel<1, MASKED, AXIS, DEBUG>;
        case 2: return march_pass_kernel<2, MASKED, AXIS, DEBUG>;  default: return march_pass_kernel<3, MASKED, AXIS, DEBUG>;
    }
}
MarchFn pick_march(int aniso, bool masked, int axis, bool debug)
{
    if (axis == 2) {
        if (masked) return debug ? pick_march_a<true, 2, true>(aniso) : pick_march_a<true, 2, false>(aniso);
        return debug ? pick_march_a<false, 2, true>(aniso) : pick_march_a<false, 2, false>(aniso);
    }
    if (masked) return debug ? pick_march_a<true, 1, true>(aniso) : pick_march_a<true, 1, false>(aniso);
    return debug ? pick_march_a<false, 1, true>(aniso) : pick_march_a<false, 1, false>(aniso);
}

template <int COLOUR, bool DEBUG> MarchFn pick_march_bcc(int aniso)
{
    switch (aniso) {
        case 0: return march_bcc_kernel<0, COLOUR, DEBUG>;  case 1: return march_bcc_kernel<1, COLOUR, DEBUG>;
        case 2: return march_bcc_kernel<2, COLOUR, DEBUG>;  default: return march_bcc_kernel<3, COLOUR, DEBUG>;
    }
}
MarchFn pick_bcc(int aniso, int colour, bool debug)
{
    if (colour) return debug ? pick_march_bcc<1, true>(aniso) : pick_march_bcc<1, false>(aniso);
    return debug ? pick_march_bcc<0, true>(aniso) : pick_march_bcc<0, false>(aniso);
}

}  // namespace

// One resident wave of threads (more waves only to keep a thread's fp32 partial sums short): every thread owns one item
// column of one segment of the march axis.  Bulk lattices march along z; thin films (nz < 16) along y, with the nz planes
// of an x-range in one block so that the side rows come from L1.
bool plan_march(mc_ctx* c)
{
    c->march_ok = c->march_possible = false;
    const mc_lattice& lat = c->lat;
    if (c->P.anti_x || c->P.fcc || c->P.basis) return false;
    if (!c->masked && !(lat.periodic[0] == 1 && lat.periodic[1] == 1 && lat.periodic[2] == 1)) return false;
    if (c->P.bcc ? (lat.nx % 4 != 0 || lat.nz < 8) : (lat.nx % 8 != 0)) return false;     // bcc: 4 cells per item, z-march only
    MarchGeom& G = c->mgeom;
    G.RV = c->P.bcc ? lat.nx / 4 : lat.nx / 8; G.XB = 0; G.SB = 0;
    G.axis = (c->P.bcc || lat.nz >= 16) ? 2 : 1;
    const int nm = G.axis == 2 ? lat.nz : lat.ny, ns = G.axis == 2 ? lat.ny : lat.nz;
    if (nm < 8) return false;
    if (G.axis == 1) {
        if (MARCH_BLOCK % ns) return false;
        G.SB = ns; G.XB = MARCH_BLOCK / ns;
        if (G.RV % G.XB) return false;
    }
    int per_sm = 0;
    const void* probe = c->P.bcc ? (const void*)pick_bcc(c->aniso, 0, false) : (const void*)pick_march(c->aniso, c->masked, G.axis, false);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, probe, MARCH_BLOCK, 0) != cudaSuccess || per_sm < 1) { cudaGetLastError(); return false; }
    const long long resident = (long long)c->sm_count * per_sm * MARCH_BLOCK;
    const long long columns = (long long)ns * G.RV;
    // segments along the march axis: the count that minimises (waves of resident threads) x (steps per thread + the prologue,
    // two loads-only steps counted as half a step); at most 256 steps per thread (1024 sites in its fp32 partial sums), at
    // least 4 (the prologue has to be amortised)
    long long n_lo = (nm + 255) / 256, n_hi = nm / 4 > 0 ? nm / 4 : 1, n_segs = n_lo;
    double best = 1e300;
    for (long long n = n_lo; n <= n_hi; ++n) {
        const double waves = (double)((columns * n + resident - 1) / resident);
        const double cost = waves * ((double)((nm + n - 1) / n) + 0.5);
        if (cost < best) { best = cost; n_segs = n; }
    }
    const double efficiency = (double)nm * (double)columns / (double)resident / best;   // 1 = every slot busy for the whole pass
    G.n_segs = (int)n_segs; G.Lm = nm / G.n_segs; G.Lm_rem = nm % G.n_segs;
    const long long nt = columns * n_segs;
    if (nt > 0x7fffffffLL || (nt + MARCH_BLOCK - 1) / MARCH_BLOCK > 0x7fffffffLL) return false;
    G.n_threads = (uint32_t)nt;
    G.div_rv = host_make_div((uint32_t)G.RV); G.div_ns = host_make_div((uint32_t)ns);
    G.div_xqb = host_make_div((uint32_t)(G.axis == 1 ? G.RV / G.XB : 1));
    c->march_possible = true;
    // default for bulk lattices without side data (measured: +4..9 % over the gather at 128^3 .. 512^3); the staged pass keeps
    // the row lengths it is specialised for; masked lattices stay on the gather (the c5 film: 185 against 163 us per sweep)
    // ... and lattices whose columns fill the machine badly (small ones; sizes that leave a sixth of the slots empty: 320^3)
    // ... and bcc (176^3 cells: 105.6 against 101.8 us per sweep: the gather already serves 60 % of its loads from L1)
    c->march_ok = G.Lm >= 4 && efficiency >= 0.85 && !c->tile_ok && !c->masked && !c->P.bcc;
    return c->march_ok;
}

int launch_pass_march(mc_ctx* ctx, int colour, float invT, int flags, float* dx, uint8_t* da)
{
    MarchFn fn = ctx->P.bcc ? pick_bcc(ctx->aniso, colour, dx || da) : pick_march(ctx->aniso, ctx->masked, ctx->mgeom.axis, dx || da);
    const int grid = (int)((ctx->mgeom.n_threads + MARCH_BLOCK - 1) / MARCH_BLOCK);
    MC_CU(launch_dependent(fn, grid, MARCH_BLOCK, 0, ctx->stream, ctx->P, ctx->mgeom, colour, invT, flags, dx, da));
    ctx->launches += 1;
    return MC_OK;
}

}  // namespace mc
