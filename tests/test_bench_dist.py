"""Host logic of bench.py's N > 1 path (independent replicas, max-over-ranks timing, whole-job value) on CPU with
the gloo backend, world_size 2, plus the golden fixture's internal pins."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert bench.dist_env() == (rank, rank, world)
        local_ms = 10.0 * (rank + 1)                                   # rank 1 is the slow replica
        mx = bench.max_over_ranks(local_ms, torch.device("cpu"))
        val = bench.job_value(2.0e12, mx, world)                       # 2 TFLOP per rank per step
        out.put((rank, mx, val))
    finally:
        dist.destroy_process_group()


def test_replica_aggregation_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for (rank, mx, val) in res:
        assert mx == 20.0                                             # max over ranks, identical on every rank
        assert abs(val - 2 * 2.0e12 / 20e-3 / 1e12) < 1e-9            # all replicas' flops / slowest time


def test_single_process_is_identity():
    import bench
    assert bench.max_over_ranks(3.5, torch.device("cpu")) == 3.5
    assert bench.job_value(1e12, 1000.0, 1) == 1.0


def test_golden_config1_internal_pins():
    """tests/golden/config1_fci.txt (written by make_golden.py from the brute-force FCI): E_total equals the survey's
    independent probe value; the natural occupations pair to 2 (particle-hole symmetry of the half-filled PPP model
    on a bipartite graph - a closed-form property no single mistake in the FCI RDM code would preserve)."""
    vals = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "config1_fci.txt")):
        if line.startswith("#"):
            continue
        key, rest = line.split(None, 1)
        vals[key] = [float(x) for x in rest.split()]
    assert abs(vals["e_el_fci"][0] + vals["e_core"][0] - vals["e_total_fci"][0]) < 2e-10
    assert abs(vals["e_total_fci"][0] - (-0.8822829988)) < 2e-9
    assert abs(vals["e_core"][0] - 8.5092529943) < 1e-9
    occ = np.array(vals["natural_occupations"])
    assert abs(occ.sum() - 10.0) < 1e-6 and abs(vals["trace_gamma"][0] - 10.0) < 1e-9
    assert np.abs(occ + occ[::-1] - 2.0).max() < 1e-6


def test_stored_traffic_is_labelled_and_workload_specific():
    """roofline.traffic comes from the tracked ncu summary (commit + command + number of launches of one step) and only
    for the workload it was captured on."""
    import bench
    t, note = bench.stored_traffic(4, 4096, 26)
    assert t is not None and t > 5.0e10 and "commit" in note and "launches" in note
    assert bench.stored_traffic(4, 2048, 26) == (None, None)
    assert bench.stored_traffic(5, 4096, 40) == (None, None)
