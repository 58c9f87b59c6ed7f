// mc_pass.cu -- instantiations and launcher of the generic colour pass (mc_pass.cuh).
#include "mc_host.h"
#include "mc_pass.cuh"

namespace mc {
namespace {



template <int VEC, int MODE> PassFn pick_pass(int aniso, bool masked)
{
    switch (aniso * 2 + (masked ? 1 : 0)) {
        case 0: return pass_kernel<VEC, 0, false, MODE>;  case 1: return pass_kernel<VEC, 0, true, MODE>;
        case 2: return pass_kernel<VEC, 1, false, MODE>;  case 3: return pass_kernel<VEC, 1, true, MODE>;
        case 4: return pass_kernel<VEC, 2, false, MODE>;  case 5: return pass_kernel<VEC, 2, true, MODE>;
        case 6: return pass_kernel<VEC, 3, false, MODE>;  default: return pass_kernel<VEC, 3, true, MODE>;
    }
}

template <int MODE, int LAT> PassFn pick_pass_lat(int aniso)
{
    switch (aniso) {
        case 0: return pass_kernel<4, 0, false, MODE, LAT>;  case 1: return pass_kernel<4, 1, false, MODE, LAT>;
        case 2: return pass_kernel<4, 2, false, MODE, LAT>;  default: return pass_kernel<4, 3, false, MODE, LAT>;
    }
}

template <int MODE, int COL> PassFn pick_pass_fcc_c(int aniso)
{
    switch (aniso) {
        case 0: return pass_kernel<4, 0, false, MODE, 2, COL>;  case 1: return pass_kernel<4, 1, false, MODE, 2, COL>;
        case 2: return pass_kernel<4, 2, false, MODE, 2, COL>;  default: return pass_kernel<4, 3, false, MODE, 2, COL>;
    }
}
template <int MODE> PassFn pick_pass_fcc(int aniso, int colour)
{
    switch (colour) {
        case 0: return pick_pass_fcc_c<MODE, 0>(aniso);  case 1: return pick_pass_fcc_c<MODE, 1>(aniso);
        case 2: return pick_pass_fcc_c<MODE, 2>(aniso);  default: return pick_pass_fcc_c<MODE, 3>(aniso);
    }
}

}  // namespace

int launch_pass_generic(mc_ctx* ctx, int mode, int colour, float invT, int flags, float* dx, uint8_t* da)
{
    PassFn fn = (ctx->vec == 4) ? (mode == MODE_SWEEP ? pick_pass<4, MODE_SWEEP>(ctx->aniso, ctx->masked) : pick_pass<4, MODE_MEASURE>(ctx->aniso, ctx->masked))
                                : (mode == MODE_SWEEP ? pick_pass<1, MODE_SWEEP>(ctx->aniso, ctx->masked) : pick_pass<1, MODE_MEASURE>(ctx->aniso, ctx->masked));
    if (ctx->P.bcc) fn = mode == MODE_SWEEP ? pick_pass_lat<MODE_SWEEP, 1>(ctx->aniso) : pick_pass_lat<MODE_MEASURE, 1>(ctx->aniso);
    if (ctx->P.fcc) fn = mode == MODE_SWEEP ? pick_pass_fcc<MODE_SWEEP>(ctx->aniso, colour) : pick_pass_fcc<MODE_MEASURE>(ctx->aniso, colour);
    // eight-colour lattices: sweeps through the compile-time tables, unless the test hook forces the run-time table (MC_PATH_GENERIC);
    // the stand-alone measurement reads the run-time table
    if (ctx->P.basis) fn = mode != MODE_SWEEP ? pick_pass_lat<MODE_MEASURE, 3>(ctx->aniso)
                         : ctx->path == MC_PATH_GENERIC ? pick_pass_lat<MODE_SWEEP, 3>(ctx->aniso)
                         : ctx->P.basis == MC_HCP ? pick_pass_basis_hcp(ctx->aniso, colour) : pick_pass_basis_nnn(ctx->aniso, colour);
    const int grid = grid_for(ctx, ctx->geom.n_items, pass_min_blocks(ctx->P.basis ? 3 : 0), MC_PASS_BLOCK);
    MC_CU(launch_dependent(fn, grid, MC_PASS_BLOCK, 0, ctx->stream, ctx->P, ctx->geom, colour, invT, flags, dx, da));
    ctx->launches += 1;
    return MC_OK;
}

}  // namespace mc
