// mc_host.h -- host-side handle of libmc_b200.so and the launchers each kernel translation unit exports to mc_api.cu.
// Nothing here crosses the C ABI (include/mc.h does); no environment variables, no globals, no allocation.
#pragma once

#include "../../include/mc.h"
#include "mc_common.cuh"
#include "mc_pair.cuh"      // PairGeom
#include "mc_tile.cuh"      // TileGeom
#include "mc_march.cuh"     // MarchGeom

#include <cstdio>

struct mc_ctx {
    mc_lattice lat;
    double J, Ku, Kc, eu[3], B[3];
    int adaptive;
    uint64_t seed;
    int device;                       // CUDA device ordinal the workspace lives on; every entry point runs under it
    mc::Params P;
    mc::Geom geom;
    mc::PairGeom pgeom;
    bool pair_ok;
    bool tile_possible, tile_ok; mc::TileGeom tgeom; int tile_threads; size_t tile_smem;   // staged colour pass (mc_tile.cuh)
    bool march_possible, march_ok; mc::MarchGeom mgeom;     // register-carried z-march colour pass (mc_march.cuh)
    int path;                         // MC_PATH_AUTO / GENERIC / STAGED (mc_debug_set_path)
    bool field;
    int vec, aniso;
    bool masked;
    cudaStream_t stream;
    int sm_count;
    bool ml_valid, aligned;
    bool hook_pending;                // a half-sweep hook left its count / fused sums in DevState (closed by mc_end_sweep)
    double theta, phi, eC[3];
    void* staging; size_t staging_bytes;   // scratch inside the caller's workspace: upload / readback / hook outputs
    int64_t launches;
    int sticky;
    char err[512];
};

namespace mc {

inline int fail(mc_ctx* c, int code, const char* fmt, const char* detail = "")
{
    if (c) { snprintf(c->err, sizeof c->err, fmt, detail); if (code == MC_ECUDA) c->sticky = MC_ECUDA; }
    return code;
}

#define MC_CU(call)                                                                                   \
    do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return mc::fail(ctx, MC_ECUDA, "CUDA error: %s", cudaGetErrorString(e_)); } while (0)

// Launch of a pass kernel with programmatic dependent launch: the grid may be scheduled while the previous kernel of the
// stream drains (every pass kernel starts with grid_dependency_sync(), so it reads nothing early).  Hides the launch
// gap between the 2n back-to-back colour passes of mc_sweep(T, n).
template <class Fn, class... Args>
cudaError_t launch_dependent(Fn fn, int grid, int block, size_t smem, cudaStream_t stream, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)block); cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, fn, args...);
}

// grid of a grid-stride kernel: one resident wave (the CTAs per SM its launch bounds allow)
inline int grid_for(const mc_ctx* c, uint32_t n_threads_needed, int resident_per_sm, int block = BLOCK)
{
    const long long need = ((long long)n_threads_needed + block - 1) / block;
    long long cap = (long long)c->sm_count * resident_per_sm;
    if (cap > c->P.max_blocks) cap = c->P.max_blocks;
    long long g = need < cap ? need : cap;
    return (int)(g < 1 ? 1 : g);
}

// ---- mc_pass.cu: generic colour pass / standalone measurement (any lattice)
int launch_pass_generic(mc_ctx* ctx, int mode, int colour, float invT, int flags, float* dx, uint8_t* da);
// ---- mc_basis_hcp.cu / mc_basis_nnn.cu: the sweep passes of the eight-colour lattices with compile-time bond tables
typedef void (*PassFn)(const Params, const Geom, int, float, int, float*, uint8_t*);
PassFn pick_pass_basis_hcp(int aniso, int colour);
PassFn pick_pass_basis_nnn(int aniso, int colour);
// ---- mc_pair.cu: constrained pair pass
int launch_pair_generic(mc_ctx* ctx, int colour, float invT, int flags, float* dx, uint8_t* da);
// ---- mc_march.cu: register-carried z-march colour pass; plan_march fills ctx->march_* at creation
bool plan_march(mc_ctx* ctx);
int launch_pass_march(mc_ctx* ctx, int colour, float invT, int flags, float* dx, uint8_t* da);
// magic-number division for the kernels' FastDiv (mc_api.cu)
FastDiv host_make_div(uint32_t d);
// ---- mc_tile.cu: staged colour pass (TMA-fed shared-memory plane ring); plan_tile fills ctx->tile_* at creation
bool plan_tile(mc_ctx* ctx);
int launch_pass_tile(mc_ctx* ctx, int colour, float invT, int flags, float* dx, uint8_t* da);

}  // namespace mc
