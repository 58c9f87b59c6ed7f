// mc_tile.cu -- instantiations, planner and launcher of the staged colour pass (mc_tile.cuh).
#include "mc_host.h"

namespace mc {
namespace {

typedef void (*TileFn)(const Params, const TileGeom, int, float, int, float*, uint8_t*);
template <int RT, bool DEBUG, bool ANTI = false, bool L2S = false> TileFn pick_tile_rt(int aniso, bool field)
{
    switch (aniso * 2 + (field ? 1 : 0)) {
        case 0: return tile_pass_kernel<0, false, RT, DEBUG, ANTI, L2S>;  case 1: return tile_pass_kernel<0, true, RT, DEBUG, ANTI, L2S>;
        case 2: return tile_pass_kernel<1, false, RT, DEBUG, ANTI, L2S>;  case 3: return tile_pass_kernel<1, true, RT, DEBUG, ANTI, L2S>;
        case 4: return tile_pass_kernel<2, false, RT, DEBUG, ANTI, L2S>;  case 5: return tile_pass_kernel<2, true, RT, DEBUG, ANTI, L2S>;
        case 6: return tile_pass_kernel<3, false, RT, DEBUG, ANTI, L2S>;  default: return tile_pass_kernel<3, true, RT, DEBUG, ANTI, L2S>;
    }
}
// Row lengths with a specialised instantiation: MC_TILE_RT_LIST (mc_tile.cuh).  Any other R, the anti-periodic wrap and the
// decision-variable debug outputs of the test hooks run the run-time-R instantiation (same arithmetic, same slab shape).
TileFn pick_tile(int R, int Ty, int npass, bool debug, int aniso, bool field, bool anti, bool stream_l2)
{
    if (anti) return debug ? pick_tile_rt<0, true, true>(aniso, field) : pick_tile_rt<0, false, true>(aniso, field);
    if (debug) return pick_tile_rt<0, true>(aniso, field);
    if (!tile_has_rt(R) || Ty != tile_ty_rt(R) || npass != TILE_NPASS_RT) return pick_tile_rt<0, false>(aniso, field);
    switch (R) {
#define MC_TILE_X(r) case r: return stream_l2 ? pick_tile_rt<r, false, false, true>(aniso, field) : pick_tile_rt<r, false>(aniso, field);
        MC_TILE_RT_LIST(MC_TILE_X)
#undef MC_TILE_X
        default: return pick_tile_rt<0, false>(aniso, field);
    }
}

}  // namespace

// Chooses the slab / segment decomposition of the staged colour pass.  Fills ctx->tile_possible
// (the geometry allows the staged pass) and ctx->tile_ok (it is the default for this lattice).
bool plan_tile(mc_ctx* c)
{
    c->tile_ok = c->tile_possible = false;
    const mc_lattice& lat = c->lat;
    if (c->masked || c->P.region || c->P.sub) return false;
    if (!(lat.periodic[0] >= 1 && lat.periodic[1] == 1 && lat.periodic[2] == 1)) return false;   // x may be anti-periodic (ANTI instantiation)
    const int R = lat.nx / 2;
    if (R % 4) return false;                                    // TMA bulk copies move whole rows: 16-byte multiples
    const int PR = R / 2;
    const int max_threads = TILE_MAX_THREADS;
    if (PR > max_threads) return false;
    TileGeom& G = c->tgeom;
    G.R = R; G.PR = PR; G.nx = lat.nx; G.ny = lat.ny; G.nz = lat.nz;
    int RP = 1;
    for (int d = 1; d <= lat.ny; ++d) if (lat.ny % d == 0 && PR * d <= max_threads) RP = d;
    int NP = 1;
    const size_t smem_cap = (size_t)(220 * 1024) / TILE_MIN_BLOCKS - 3 * 1024;   // TILE_MIN_BLOCKS CTAs per SM (run-time-R shape)
    auto slot_bytes = [&](int ty) { return (size_t)3 * (ty + 2) * R * sizeof(float); };
    if (lat.ny % (2 * RP) == 0 && TILE_NSLOT * slot_bytes(2 * RP) <= smem_cap) NP = 2;
    // row lengths with a compile-time specialisation take its slab shape when it tiles ny
    const bool spec = tile_has_rt(R) && tile_rp_rt(R) >= 1 && lat.ny % tile_ty_rt(R) == 0;
    if (spec) { RP = tile_rp_rt(R); NP = TILE_NPASS_RT; }
    G.RP = RP; G.NPASS = NP; G.Ty = RP * NP;
    G.n_slabs = lat.ny / G.Ty;
    G.slot_floats = 3 * (G.Ty + 2) * R;
    G.n_active = PR * RP;
    {   // does the spin state (12 B per site) fit the L2?
        int l2 = 0;
        if (cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, c->device) != cudaSuccess) { cudaGetLastError(); l2 = 0; }
        G.stream_l2 = (12ull * (unsigned long long)c->P.N > (unsigned long long)l2) ? 1 : 0;
    }
    c->tile_threads = (G.n_active + 31) / 32 * 32;
    c->tile_smem = TILE_NSLOT * slot_bytes(G.Ty);
    if (c->tile_smem > 200 * 1024) return false;
    // every instantiation this handle can launch must be allowed its dynamic shared memory
    TileFn fns[2] = { pick_tile(R, G.Ty, G.NPASS, false, c->aniso, c->field, c->P.anti_x != 0, G.stream_l2 != 0), pick_tile(R, G.Ty, G.NPASS, true, c->aniso, c->field, c->P.anti_x != 0, G.stream_l2 != 0) };
    int per_sm = 1;
    for (TileFn f : fns) {
        if (cudaFuncSetAttribute((const void*)f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->tile_smem) != cudaSuccess) { cudaGetLastError(); return false; }
    }
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)fns[0], c->tile_threads, c->tile_smem) != cudaSuccess || per_sm < 1) { cudaGetLastError(); return false; }
    // one wave of CTAs: n_segs z-segments per slab so that n_slabs * n_segs fills sm_count * per_sm slots
    long long slots = (long long)c->sm_count * per_sm;
    int n_segs = (int)(slots / G.n_slabs);
    if (n_segs < 1) n_segs = 1;
    if (n_segs > lat.nz) n_segs = lat.nz;
    G.n_segs = n_segs; G.Lz = lat.nz / n_segs; G.Lz_rem = lat.nz % n_segs;
    if ((long long)G.n_slabs * G.n_segs > c->P.max_blocks) return false;
    c->tile_possible = true;
    const bool specialised = spec && !c->P.anti_x;
    c->tile_ok = specialised && c->P.Nc >= 65536u;             // small lattices are launch-bound: the generic kernel has less prologue
    return c->tile_ok;
}

int launch_pass_tile(mc_ctx* ctx, int colour, float invT, int flags, float* dx, uint8_t* da)
{
    TileFn fn = pick_tile(ctx->tgeom.R, ctx->tgeom.Ty, ctx->tgeom.NPASS, dx || da, ctx->aniso, ctx->field, ctx->P.anti_x != 0, ctx->tgeom.stream_l2 != 0);
    const int grid = ctx->tgeom.n_slabs * ctx->tgeom.n_segs;
    MC_CU(launch_dependent(fn, grid, ctx->tile_threads, ctx->tile_smem, ctx->stream, ctx->P, ctx->tgeom, colour, invT, flags, dx, da));
    ctx->launches += 1;
    return MC_OK;
}

}  // namespace mc
