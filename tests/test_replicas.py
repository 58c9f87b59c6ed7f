"""Replica scheduler: assignment, seeds, gather and the max-over-ranks time, on CPU with gloo (world_size 2 and 3)."""
import json
import os
import socket
import subprocess
import sys

import pytest

from paper_2103_03517_b200 import replicas

HERE = os.path.dirname(os.path.abspath(__file__))


def test_assignment_is_a_partition_and_balances_costs():
    for n, w in ((16, 1), (16, 2), (33, 4), (5, 8), (0, 3)):
        parts = replicas.assign(n, w)
        assert sorted(k for p in parts for k in p) == list(range(n)) and len(parts) == w
        assert all(p == sorted(p) for p in parts) and max(len(p) for p in parts) - min(len(p) for p in parts) <= 1
    costs = [5, 1, 1, 1, 1, 1, 4, 4, 3, 3]                       # LPT: 24 units over 3 ranks -> 8 each
    parts = replicas.assign(len(costs), 3, costs)
    assert sorted(k for p in parts for k in p) == list(range(len(costs)))
    assert [sum(costs[k] for k in p) for p in parts] == [8, 8, 8]
    assert replicas.assign(len(costs), 3, costs) == parts          # deterministic
    with pytest.raises(ValueError):
        replicas.assign(3, 0)


def test_seed_is_a_function_of_the_point_alone():
    assert [replicas.point_seed(42, k) for k in range(3)] == [43, 44, 45]      # BASELINE.json c2: seed 42 + k, k = 1..


def test_single_process_multi_device_order_and_batches():
    log = []
    def enqueue(point, seed, device): log.append(("enq", point, device)); return (point, seed, device)
    def collect(h): log.append(("col", h[0], h[2])); return {"p": h[0], "seed": h[1], "dev": h[2]}
    res = replicas.run_points_multi_device(list(range(5)), enqueue, collect, ["d0", "d1"], base_seed=7)
    assert [r["p"] for r in res] == list(range(5)) and [r["seed"] for r in res] == [8, 9, 10, 11, 12]
    assert [r["dev"] for r in res] == ["d0", "d1", "d0", "d1", "d0"]
    # a round is fully enqueued before its first read-back (the devices overlap), and rounds do not interleave
    assert [e[0] for e in log] == ["enq", "enq", "col", "col", "enq", "enq", "col", "col", "enq", "col"]


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _run_world(world_size, use_costs, tmp_path):
    out = tmp_path / f"res_{world_size}_{int(use_costs)}.json"
    port = _free_port()
    procs = []
    for r in range(world_size):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world_size), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        if world_size == 1:
            for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"): env.pop(k)
        procs.append(subprocess.Popen([sys.executable, os.path.join(HERE, "replica_worker.py"), str(out), "1" if use_costs else "0"], env=env))
    for p in procs:
        assert p.wait(timeout=240) == 0
    return json.load(open(out))


@pytest.mark.timeout(600)
def test_gloo_world_sizes_give_the_same_answer(tmp_path):
    ref = _run_world(1, False, tmp_path)
    assert [r["seed"] for r in ref["results"]] == [43 + k for k in range(11)] and ref["slowest"] == 10.0
    for ws, use_costs in ((2, False), (2, True), (3, True)):
        got = _run_world(ws, use_costs, tmp_path)
        strip = lambda rs: [{k: v for k, v in r.items() if k != "rank"} for r in rs]
        assert strip(got["results"]) == strip(ref["results"])                   # same values, same seeds, point order
        ranks = [r["rank"] for r in got["results"]]
        assert set(ranks) == set(range(ws))                                      # every rank worked
        if not use_costs:
            assert ranks == [k % ws for k in range(11)]                          # round robin
        assert got["slowest"] == 10.0 + ws - 1                                   # max over ranks


def test_split_chunks():
    assert replicas.split_chunks(170, 50) == (3, 20) and replicas.split_chunks(0, 50) == (0, 0) and replicas.split_chunks(50, 50) == (1, 0)
    with pytest.raises(ValueError):
        replicas.split_chunks(10, 0)
