// mc_basis_hcp.cu -- the eight colour passes of the hcp lattice (C-32) with the bond table of every sublattice as a
// compile-time constant: pass_kernel<4, ANISO, false, MODE_SWEEP, 3, colour> (mc_pass.cuh, basis_exchange_field_ct).  A translation
// unit of its own: 32 instantiations with fully unrolled tables.
#include "mc_host.h"
#include "mc_pass.cuh"

namespace mc {
namespace {

template <int COL> PassFn pick_aniso(int aniso)
{
    switch (aniso) {
        case 0: return pass_kernel<4, 0, false, MODE_SWEEP, 3, COL>;  case 1: return pass_kernel<4, 1, false, MODE_SWEEP, 3, COL>;
        case 2: return pass_kernel<4, 2, false, MODE_SWEEP, 3, COL>;  default: return pass_kernel<4, 3, false, MODE_SWEEP, 3, COL>;
    }
}

}  // namespace

PassFn pick_pass_basis_hcp(int aniso, int colour)
{
    switch (colour) {
        case 0: return pick_aniso<0>(aniso);  case 1: return pick_aniso<1>(aniso);  case 2: return pick_aniso<2>(aniso);  case 3: return pick_aniso<3>(aniso);
        case 4: return pick_aniso<4>(aniso);  case 5: return pick_aniso<5>(aniso);  case 6: return pick_aniso<6>(aniso);  default: return pick_aniso<7>(aniso);
    }
}

}  // namespace mc
