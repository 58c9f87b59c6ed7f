"""Many small points at once on one device (replicas.run_points_concurrent): one stream per point, sweeps captured as CUDA graphs and
replayed round robin.  The results must be those of the serial loop bit for bit -- the library's sweep calls allocate nothing and
never synchronise, which is what makes them capturable."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mods():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    from paper_2103_03517_b200 import binding, build, replicas
    build.build()
    return binding, replicas


def _serial(binding, points, constrained):
    out = []
    for k, (T, L, n1, n2) in enumerate(points):
        g = binding.Lattice(L, L, L, Ku=0.05, cone0=0.5, adaptive=True, seed=43 + k)
        if constrained:
            g.constrained_sweep(T, 0.6, 0.2, n1); g.reset_accumulators(); g.constrained_sweep(T, 0.6, 0.2, n2)
        else:
            g.sweep(T, n1); g.reset_accumulators(); g.sweep(T, n2)
        ob = g.observables()
        out.append((g.get_spins(), g.trace(), ob.sum_m[0], ob.sum_E, ob.n_samples, tuple(ob.sum_torque)))
        g.close()
    return out


@pytest.mark.parametrize("constrained", [False, True])
@pytest.mark.parametrize("use_graphs", [True, False])
def test_concurrent_points_equal_the_serial_loop_bit_for_bit(mods, constrained, use_graphs):
    binding, replicas = mods
    points = [(0.4 + 0.3 * k, 32, 170, 131) for k in range(5)]            # chunk 50: 3 chunks + 20, 2 chunks + 31 (constrained: one less)
    ref = _serial(binding, points, constrained)

    def create(point, seed, device, stream):
        return binding.Lattice(point[1], point[1], point[1], Ku=0.05, cone0=0.5, adaptive=True, seed=seed, device=device, stream=stream)

    def phases(point):
        T, L, n1, n2 = point
        if constrained:
            return [("constrained", T, 0.6, 0.2, n1), ("reset",), ("constrained", T, 0.6, 0.2, n2)]
        return [("sweep", T, n1), ("reset",), ("sweep", T, n2)]

    def collect(g, point):
        ob = g.observables()
        r = (g.get_spins(), g.trace(), ob.sum_m[0], ob.sum_E, ob.n_samples, tuple(ob.sum_torque))
        g.close()
        return r

    got = replicas.run_points_concurrent(points, create, phases, collect, base_seed=42, chunk=50, use_graphs=use_graphs, max_concurrent=3)
    assert len(got) == len(ref)
    for a, b in zip(got, ref):
        assert (a[0] == b[0]).all() and (a[1] == b[1]).all() and a[2:] == b[2:]
    with pytest.raises(ValueError):
        replicas.run_points_concurrent(points[:2], create, lambda p: [("sweep", p[0], 10 if p[0] < 0.5 else 20)], collect)
