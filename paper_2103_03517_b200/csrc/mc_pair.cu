// mc_pair.cu -- instantiations and launcher of the constrained pair pass (mc_pair.cuh).
#include "mc_host.h"

namespace mc {
namespace {

typedef void (*PairFn)(const Params, const PairGeom, int, float, int, float*, uint8_t*);

template <int VEC> PairFn pick_pair(int aniso, bool masked)
{
    switch (aniso * 2 + (masked ? 1 : 0)) {
        case 0: return pair_kernel<VEC, 0, false>;  case 1: return pair_kernel<VEC, 0, true>;
        case 2: return pair_kernel<VEC, 1, false>;  case 3: return pair_kernel<VEC, 1, true>;
        case 4: return pair_kernel<VEC, 2, false>;  case 5: return pair_kernel<VEC, 2, true>;
        case 6: return pair_kernel<VEC, 3, false>;  default: return pair_kernel<VEC, 3, true>;
    }
}

PairFn pick_pair_bcc(int aniso)
{
    switch (aniso) {
        case 0: return pair_kernel<4, 0, false, 1>;  case 1: return pair_kernel<4, 1, false, 1>;
        case 2: return pair_kernel<4, 2, false, 1>;  default: return pair_kernel<4, 3, false, 1>;
    }
}

}  // namespace

int launch_pair_generic(mc_ctx* ctx, int colour, float invT, int flags, float* dx, uint8_t* da)
{
    PairFn fn = ctx->P.bcc ? pick_pair_bcc(ctx->aniso) : (ctx->vec == 4) ? pick_pair<4>(ctx->aniso, ctx->masked) : pick_pair<1>(ctx->aniso, ctx->masked);
    const int grid = grid_for(ctx, ctx->pgeom.n_threads, MC_PAIR_MIN_BLOCKS, MC_PAIR_BLOCK);
    MC_CU(launch_dependent(fn, grid, MC_PAIR_BLOCK, 0, ctx->stream, ctx->P, ctx->pgeom, colour, invT, flags, dx, da));
    ctx->launches += 1;
    return MC_OK;
}

}  // namespace mc
