"""World-size-2 checks of the N > 1 host logic (gloo, CPU).  The path is "replicas only"
(DESIGN.md section 8): no data-path collective, the only exchange is the max-over-ranks of the
timed region; `bench.py --impl reference` lets rank 0 alone run the oracle."""
import json
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r "measured" (r + 1) * 10 ms for 5 steps of 1000 units each
    total_ms, value = bench.aggregate_over_ranks(10.0 * (rank + 1), 1000, 5, dist)
    out[rank] = (total_ms, value)
    dist.barrier()
    dist.destroy_process_group()


def test_aggregate_is_max_time_and_sum_of_units():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    for r in range(world):
        total_ms, value = res[r]
        assert total_ms == 20.0                              # max over ranks
        assert abs(value - 2 * 1000 * 5 / 20e-3) < 1e-6      # units of both ranks / slowest rank


def test_single_process_aggregate():
    sys.path.insert(0, ROOT)
    import bench
    total_ms, value = bench.aggregate_over_ranks(4.0, 100, 2, None)
    assert total_ms == 4.0 and abs(value - 100 * 2 / 4e-3) < 1e-9


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"),
           "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "1"]
    res = subprocess.run(cmd, cwd=ROOT, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, timeout=600)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0


def _shard_worker(rank, world, port, out):
    """One rank of a sharded evaluation with the kernels replaced by the oracle (no GPU here): the slab's AEV rows and
    its partial forces (backward with the upstream gradient masked to the slab), exchanged by sharded.py over gloo."""
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import numpy as np
    import oracle
    from gen import make_water_box
    from paper_2310_03121_b200.sharded import central_ranges, gather_rows, sum_partial_forces
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = make_water_box(64, 12.43, 77, "shard")
    first, count = central_ranges(w.n_atoms, world)[rank]
    aev = oracle.aev_forward(w.params, w.pos, w.species, None)
    gm = np.zeros_like(w.grad_aev)
    gm[0, first:first + count] = w.grad_aev[0, first:first + count]
    partial = torch.from_numpy(oracle.aev_backward(w.params, w.pos, w.species, None, gm))
    forces = sum_partial_forces(partial, dist)
    rows = gather_rows(torch.from_numpy(np.ascontiguousarray(aev[0, first:first + count])), w.n_atoms, dist)
    full_f = oracle.aev_backward(w.params, w.pos, w.species, None, w.grad_aev)
    out[rank] = (float(np.abs(forces.numpy() - full_f).max() / np.abs(full_f).max()),
                 float(np.abs(rows.numpy() - aev[0]).max()), tuple(rows.shape), (first, count))
    dist.barrier()
    dist.destroy_process_group()


def test_sharded_exchange_sums_partial_forces_and_gathers_rows():
    """World size 2 (gloo): slabs of central atoms from central_ranges, partial forces all-reduced, AEV rows
    all-gathered (unequal slabs: 192 atoms over 2 ranks is even, so also check 3 ranks' ranges below)."""
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_shard_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0][3] == (0, 96) and res[1][3] == (96, 96)
    for r in range(world):
        f_err, row_err, shape, _ = res[r]
        assert f_err <= 1e-12 and row_err == 0.0 and shape[0] == 192
    sys.path.insert(0, ROOT)
    from paper_2310_03121_b200.sharded import central_ranges
    assert central_ranges(10, 3) == [(0, 4), (4, 3), (7, 3)]
    assert central_ranges(23559, 8)[-1] == (23559 - 2944, 2944) and sum(c for _, c in central_ranges(23559, 8)) == 23559
