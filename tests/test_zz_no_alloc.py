"""mc_profile_x_static: the slice profile with its scratch in a fixed array of the library image (no allocation at call time)
against the existing mc_profile_x (scratch in the caller's workspace) and the oracle's slice average.  Collected last on purpose
(the file name): the suite runs with pytest -x.  Passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-6          # the bar of test_domain_wall_box_profile_and_energy_match_oracle (fp32 state, exact fixed-point sums)


@pytest.fixture(scope="module")
def mods():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    import oracle
    from paper_2103_03517_b200 import binding, build, inputs
    build.build()
    return oracle, binding, inputs


def test_static_scratch_profile_equals_the_workspace_path_on_two_calls_in_a_row(mods):
    import torch
    oracle, binding, inputs = mods
    # first call: a wide lattice fills 3 x 96 sums of the shared array; second call: a narrower one with another state must not see them
    big = binding.Lattice(96, 12, 10, periodic=(2, 1, 1), Ku=0.05, seed=3)
    big.set_spins(inputs.thermal_like_spins(big.N, seed=5, spread=0.6, direction=(0.2, -0.4, 0.9)))
    small = binding.Lattice(20, 6, 4, seed=4)
    small.set_spins(inputs.random_unit_spins(small.N, seed=6))
    ref_big, ref_small = big.profile_x(), small.profile_x()                  # existing path
    out_big = big.profile_x_static()
    out_small = np.full((20, 3), np.nan)
    torch.cuda.synchronize(); free0 = torch.cuda.mem_get_info()[0]
    small.profile_x_static(out_small)                                        # second call in a row, caller-owned output
    torch.cuda.synchronize(); free1 = torch.cuda.mem_get_info()[0]
    assert free1 == free0                                                    # nothing was allocated on the device
    for got, ref, g in ((out_big, ref_big, big), (out_small, ref_small, small)):
        assert got.shape == ref.shape and np.abs(got - ref).max() < TOL
        assert (got == ref).all()                                            # the same exact sums and the same fp64 scaling
        o = oracle.Oracle(*g.shape, periodic=(2, 1, 1) if g is big else (1, 1, 1), Ku=0.05 if g is big else 0.0)
        o.set_spins(g.get_spins())
        assert np.abs(got - o.profile_x()).max() < TOL
    # and again after sweeps changed the state: the array is cleared on every call
    big.sweep(0.8, 3)
    assert (big.profile_x_static() == big.profile_x()).all()
    assert (small.profile_x_static() == ref_small).all()
    big.close(); small.close()


def test_static_scratch_profile_rejects_sizes_beyond_its_fixed_maximum(mods):
    oracle, binding, inputs = mods
    g = binding.Lattice(8192, 2, 2)                                          # the stated maximum: accepted
    assert (g.profile_x_static() == g.profile_x()).all() and np.allclose(g.profile_x_static()[:, 2], 1.0)
    g.close()
    g = binding.Lattice(8194, 2, 2)
    with pytest.raises(binding.McError, match="MC_PROFILE_STATIC_MAX_NX"):
        g.profile_x_static()
    assert g.profile_x().shape == (8194, 3)                                  # the workspace path has no such limit
    g.close()
    b = binding.Lattice(8, 4, 4, structure="bcc")
    with pytest.raises(binding.McError):
        b.profile_x_static()
    b.close()
