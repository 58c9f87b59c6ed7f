"""Worker of tests/test_replicas.py: one rank of a world_size-N gloo group on CPU.  The 'Monte Carlo point' is a pure
function of (point, seed): the test is about rank -> points -> seeds -> gather, not about spins."""
import json
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from paper_2103_03517_b200 import replicas


def fake_point(point, seed, device):
    T, theta = point
    return {"T": T, "theta": theta, "seed": seed, "value": (seed * 2654435761 % 1000003) / 1000003.0 + T, "rank": int(os.environ.get("RANK", "0")), "device": device}


def main():
    out_path, use_costs = sys.argv[1], sys.argv[2] == "1"
    points = [(0.1 * (k % 3 + 1), 9.0 * k) for k in range(11)]
    costs = [1 + (k % 4) for k in range(11)] if use_costs else None
    dist = replicas.init_distributed("gloo")
    rank = dist.get_rank() if dist is not None else 0
    res = replicas.run_points(points, fake_point, base_seed=42, costs=costs, dist=dist, device="cpu")
    slowest = replicas.max_over_ranks(10.0 + rank, dist)
    if rank == 0:
        json.dump({"results": res, "slowest": slowest}, open(out_path, "w"))
    else:
        assert res is None
    if dist is not None:
        dist.barrier(); dist.destroy_process_group()


if __name__ == "__main__":
    main()
