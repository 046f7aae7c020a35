#!/usr/bin/env python
"""bench.py -- throughput of the AEV hot path on one B200 (or N independent replicas).

Headline (BASELINE.json:metric): AEV forward+backward atoms/s on the 23,559-atom periodic
water box (config C4, BASELINE.json:configs[3]); a "step" is one pass of
aev_forward (cell-list rebuild + radial + angular AEV, rows A1-A4) + aev_backward (rows
A5-A7) through the C ABI on device-resident inputs.  The JSON line also carries
  roofline      dominant kernel against the FP32-ALU peak,
  cpu_baseline  the fp64 oracle, as it stands, timed on this box's host cores,
  e2e           the same metric through the host-buffer entry point (H2D/D2H inside),
  other         C1/C2/C3 AEV timings and the C5 full energy+forces evaluation (rows A8-A10).
`--impl reference` times the oracle alone (the reference arm of this tier).

Path sharding: independent evaluations, so `--gpus N` runs N replicas
of the same box with no data-path collective ("scaling": "weak").
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "aev_fwd_bwd_atoms_per_s"
UNIT = "atoms/s"
WORKLOAD = "C4: 23,559-atom periodic water box (7,853 H2O, L=61.7 A), cell list rebuilt every evaluation, fp32"

# algorithmic work per unit, SURVEY.md 8(d) / DESIGN.md section 7 (FMA = 2 flops)
FLOP_PAIR_FWD, FLOP_PAIR_BWD = 106.0, 167.0
FLOP_TRIPLET_FWD, FLOP_TRIPLET_BWD = 174.0, 410.0
FLOP_APAIR = 35.0          # directed angular pair set-up (half to each pass)
FLOP_CAND = 20.0           # neighbour candidate test (forward kernel)
# derived ALU peak: 148 SMs x 128 FP32 lanes x 2 flop x 1.965 GHz (B200_PROFILING.md unit counts / clocks)
ALU_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12


def _measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return json.load(fh)
    except Exception:
        return {}


class ClockSampler:
    """Samples SM clocks and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nv = None

    def _run(self):
        nv = self._nv
        names = {
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake_slowdown",
        }
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                try:
                    mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self._h))
                except Exception:
                    mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                for bit, nm in names.items():
                    if mask & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(0.01)

    def start(self):
        if self._nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def _work_counts(counts: np.ndarray, pos: np.ndarray, box, rcr: float):
    """Directed radial pairs, directed angular pairs, triplets, candidate tests of one workload,
    from the library's per-atom neighbour counts and a host histogram of cell occupancy."""
    nA = counts[..., 0].astype(np.int64)
    nB = counts[..., 1].astype(np.int64)
    p_r = int((nA + nB).sum())
    p_a = int(nA.sum())
    trip = int((nA * (nA - 1) // 2).sum())
    if box is None:
        cand = int(pos.shape[0] * pos.shape[1] * pos.shape[1])
    else:
        nc = [max(3, int(np.floor(float(b) / (rcr * 1.0001)))) for b in box]
        w = pos.reshape(-1, 3).astype(np.float64)
        b = np.asarray(box, dtype=np.float64)
        w = w - b * np.floor(w / b)
        idx = [np.minimum((w[:, k] / b[k] * nc[k]).astype(np.int64), nc[k] - 1) for k in range(3)]
        occ = np.zeros(nc, dtype=np.int64)
        np.add.at(occ, (idx[0], idx[1], idx[2]), 1)
        nb = np.zeros_like(occ)
        for dx in (-1, 0, 1):
            for dy in (-1, 0, 1):
                for dz in (-1, 0, 1):
                    nb += np.roll(occ, (dx, dy, dz), axis=(0, 1, 2))
        cand = int((occ * nb).sum())
    return {"radial_pairs_directed": p_r, "angular_pairs_directed": p_a, "triplets": trip, "candidates": cand}


def _ncu_traffic():
    """dram__bytes_read.sum + dram__bytes_write.sum per launch on C4, from the `ncu --set full` capture whose
    summary is tracked as profiles/r3_ncu_traffic.json (written from the .ncu-rep, with the commit it was
    measured at; bench.py never runs under a profiler itself).  ncu's default cache control flushes L2 before
    every kernel, so these are COLD-CACHE bytes: inside a real step the neighbour lists are L2-resident."""
    try:
        with open(os.path.join(ROOT, "profiles", "r3_ncu_traffic.json")) as fh:
            return json.load(fh)
    except Exception:
        return {}


def _flops(wc):
    fwd = FLOP_PAIR_FWD * wc["radial_pairs_directed"] + FLOP_TRIPLET_FWD * wc["triplets"] \
        + 0.5 * FLOP_APAIR * wc["angular_pairs_directed"] + FLOP_CAND * wc["candidates"]
    bwd = FLOP_PAIR_BWD * wc["radial_pairs_directed"] + FLOP_TRIPLET_BWD * wc["triplets"] \
        + 0.5 * FLOP_APAIR * wc["angular_pairs_directed"]
    return fwd, bwd


def _oracle_eval(w, threads=None):
    import oracle
    if threads:
        oracle.set_threads(threads)
    uc = w.box is not None
    oracle.aev_forward(w.params, w.pos, w.species, w.box, use_cells=uc)
    oracle.aev_backward(w.params, w.pos, w.species, w.box, w.grad_aev, use_cells=uc)


def cpu_baseline(budget_s: float = 10.0):
    """The oracle as it stands (fp64 C, OpenMP over central atoms, cell list) on this box's
    host cores, on a bounded sample of the headline workload: full C4 evaluations on all cores, and
    one on a single thread (both numbers and the CPU model are reported)."""
    import oracle
    from oracle.build import cpu_model
    from gen import make_workload
    w = make_workload("C4")
    cores = oracle.max_threads()
    _oracle_eval(w)                       # warm-up (also builds the library)
    n, t0 = 0, time.perf_counter()
    while True:
        _oracle_eval(w)
        n += 1
        dt = time.perf_counter() - t0
        if dt > budget_s or n >= 8:
            break
    t1 = time.perf_counter()
    _oracle_eval(w, threads=1)
    dt1 = time.perf_counter() - t1
    oracle.set_threads(cores)
    return {"value": w.n_atoms * w.batch * n / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "%d full C4 evaluations (fwd+bwd, fp64, cell list) in %.1f s on %d threads; 1 on one thread in %.1f s"
                      % (n, dt, cores, dt1),
            "value_1_thread": w.n_atoms * w.batch / dt1, "cpu_model": cpu_model().split(" [")[0],
            "build": "gcc -O3 -march=native -ffp-contract=off -fopenmp (oracle/build.py)"}


def _config(n_atoms):
    """The `config` object both arms print, key for key (the driver compares them): what the workload is and how
    each arm is timed.  Per-run details (ranks, core count, sample) are in the line's `arm` object."""
    return {"workload": WORKLOAD, "atoms": int(n_atoms),
            "l2": "GPU arm: flushed before every timed step (256 MiB memset outside the event pair); "
                  "reference arm: CPU, not applicable",
            "timing": "GPU arm: per-step CUDA events on the launching stream, summed, max over ranks; "
                      "reference arm: wall clock on rank 0"}


def run_reference(args):
    """Reference arm of this tier: the oracle on the host cores; each step is one full fwd+bwd
    evaluation of the headline workload itself (C4; about 0.7 s on 16 cores, so K <= 200 steps end
    within minutes)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    from oracle.build import cpu_model
    from gen import make_workload
    w = make_workload("C4")
    cores = oracle.max_threads()
    for _ in range(max(1, min(args.warmup, 2))):
        _oracle_eval(w)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _oracle_eval(w)
    dt = time.perf_counter() - t0
    value = w.n_atoms * args.steps / dt
    sample = "each step: one full C4 evaluation (fwd+bwd, fp64, cell list) on %d threads of %s" % (
        cores, cpu_model().split(" [")[0])
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": _config(w.n_atoms), "arm": {"parallelism": "host threads x%d" % cores, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def aggregate_over_ranks(total_ms, units_per_rank, steps, dist, device=None):
    """Whole-job throughput of N independent replicas (replicas only, no
    data-path collective): the timed region of the job is the MAX over ranks, the units are the
    SUM over ranks.  `dist` is torch.distributed (initialised) or None for one process."""
    import torch
    world = 1
    if dist is not None:
        world = dist.get_world_size()
        t = torch.tensor([float(total_ms)], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    return total_ms, world * units_per_rank * steps / (total_ms * 1e-3)


def _time_steps(fn, steps, flush, torch):
    """Per-step CUDA-event timing on the current stream; L2 flushed before every step."""
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for e0, e1 in ev:
        flush()
        e0.record()
        fn()
        e1.record()
    torch.cuda.synchronize()
    return np.array([e0.elapsed_time(e1) for e0, e1 in ev])


def run_quick_c5(args):
    """`--quick --workload C5|C5_ens8|C5_fp32`: only the full energy+forces evaluation (for ncu captures of k_mlp_tc)."""
    import torch
    import paper_2310_03121_b200 as pkg
    from gen import make_ensemble_weights, make_workload
    from gen.workloads import CELU_ALPHA
    dev = torch.device("cuda", 0)
    w5 = make_workload("C5")
    models = {"C5": lambda: make_ensemble_weights(1), "C5_ens8": lambda: make_ensemble_weights(8),
              "C5_fp32": lambda: make_ensemble_weights(1, round_bf16=False)}[args.workload]()
    ctx = pkg.Context(w5.params, max_atoms=w5.n_atoms, device=0)
    ctx.ani_mlp_set_ensemble(len(models))
    for m, nets in enumerate(models):
        for s, (ws, bs) in nets.items():
            ctx.ani_mlp_load_model(m, s, ws, bs, CELU_ALPHA)
    p5, s5 = torch.from_numpy(w5.pos).to(dev), torch.from_numpy(w5.species).to(dev)
    e5 = torch.empty((1,), dtype=torch.float64, device=dev)
    f5 = torch.empty((1, w5.n_atoms, 3), dtype=torch.float32, device=dev)
    flush_buf = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)

    def st5():
        ctx.ani_energy_forces(p5, s5, w5.box, energy_out=e5, forces_out=f5)
    for _ in range(max(args.warmup, 3)):
        st5()
    tt = _time_steps(st5, args.steps, flush_buf.zero_, torch)
    ctx.check_status()
    print(json.dumps({"quick": True, "workload": args.workload, "ms_per_eval": float(tt.mean()),
                      "atoms_per_s": w5.n_atoms / (tt.mean() * 1e-3), "mlp_kernel": ctx.mlp_kernel()}))
    ctx.close()


def run_ours(args):
    import torch
    import paper_2310_03121_b200 as pkg
    from gen import make_c5_weights, make_workload
    from gen.workloads import CELU_ALPHA

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist_
        dist = dist_
        dist.init_process_group("nccl" if torch.cuda.is_available() else "gloo")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)

    w = make_workload("C4")
    n_atoms = w.n_atoms * w.batch
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms, max_batch=w.batch, device=local)
    pos = torch.from_numpy(w.pos).to(dev)
    sp = torch.from_numpy(w.species).to(dev)
    g = torch.from_numpy(w.grad_aev).to(dev)
    aev_out = torch.empty((w.batch, w.n_atoms, ctx.length), dtype=torch.float32, device=dev)
    f_out = torch.empty((w.batch, w.n_atoms, 3), dtype=torch.float32, device=dev)
    flush_buf = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)   # > 126 MB L2

    def flush():
        flush_buf.zero_()

    def step():
        ctx.aev_forward(pos, sp, w.box, aev_out=aev_out)
        ctx.aev_backward(g, forces_out=f_out)

    for _ in range(max(args.warmup, 3)):
        flush()
        step()
    torch.cuda.synchronize()
    ctx.check_status()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    l0 = ctx.launch_count()
    t_ms = _time_steps(step, args.steps, flush, torch)
    launches = ctx.launch_count() - l0
    barrier()
    clocks = sampler.stop()
    total_ms, value = aggregate_over_ranks(float(t_ms.sum()), n_atoms, args.steps, dist, dev)
    ctx.check_status()

    if rank != 0:
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return

    # ---- per-kernel timing (second pass, events around each kernel) -> roofline of the dominant one
    counts = ctx.aev_export_counts(w.batch, w.n_atoms).cpu().numpy()
    wc = _work_counts(counts, w.pos, w.box, float(w.params.rcr))
    flop_fwd, flop_bwd = _flops(wc)
    ctx.aev_set_profiling(True)
    ctx.aev_get_profile()
    for _ in range(args.steps):
        flush()
        step()
    prof = ctx.aev_get_profile()
    ctx.aev_set_profiling(False)
    kern_ms = {k: (v[0] / v[1] if v[1] else 0.0) for k, v in prof.items()}
    flop_nbr = FLOP_CAND * wc["candidates"]
    kflop = {"nbr": flop_nbr, "aev": flop_fwd - flop_nbr, "backward": flop_bwd}
    dom = max(kflop, key=lambda k: kern_ms[k])
    dom_flop = kflop[dom]
    achieved = dom_flop / (kern_ms[dom] * 1e-3) / 1e12
    try:
        probe = pkg.probe_fp32_tflops(local)
    except Exception:
        probe = None
    roofline = {
        "bound": "alu", "kernel": "k_" + dom, "achieved": achieved, "peak": ALU_PEAK_TFLOPS,
        "unit": "TFLOP/s", "frac": achieved / ALU_PEAK_TFLOPS,
        "traffic": (_ncu_traffic().get("k_" + dom) or {}).get("dram_bytes"),
        "traffic_note": "ncu dram__bytes_read+write per launch, COLD cache (L2 flushed by ncu before the kernel); "
                        "profiles/r3_ncu_traffic.json, measured at commit %s" % _ncu_traffic().get("commit"),
        # the AEV / gradient matrix and the per-atom arrays are algorithmic; the neighbour lists are an
        # implementation choice and are listed separately (cold-cache `traffic` contains both)
        "algorithmic_bytes_per_launch": {"nbr": n_atoms * 16, "aev": n_atoms * ctx.length * 4 + n_atoms * 16,
                                         "backward": n_atoms * ctx.length * 4 + n_atoms * 28}[dom],
        "list_bytes_per_launch": wc["radial_pairs_directed"] * 16,
        "frac_vs_probe": (achieved / probe) if probe else None,
        "peak_source": "derived: 148 SM x 128 FP32 lanes x 2 x 1.965 GHz (DESIGN.md section 7)",
        "fma_probe_tflops": probe,
        "algorithmic_flop_per_launch": dom_flop,
        "kernel_ms": kern_ms,
        "step": {"flop": flop_fwd + flop_bwd, "achieved": (flop_fwd + flop_bwd) / (float(t_ms.mean()) * 1e-3) / 1e12,
                 "frac": (flop_fwd + flop_bwd) / (float(t_ms.mean()) * 1e-3) / 1e12 / ALU_PEAK_TFLOPS,
                 "hbm_bytes": 2 * n_atoms * ctx.length * 4 + n_atoms * 28,
                 "hbm_frac": (2 * n_atoms * ctx.length * 4 + n_atoms * 28) / (float(t_ms.mean()) * 1e-3) / 1e9
                 / float(_measured_peaks().get("hbm_gbs", 6650.0))},
        "work": wc,
    }

    if args.quick:
        print(json.dumps({"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                          "ms_per_step": total_ms / args.steps, "quick": True, "roofline": roofline,
                          "gpu_launches": int(launches), "clocks": clocks}))
        ctx.close()
        return

    # ---- end to end through the host-buffer entry point (pinned staging inside the library)
    e2e_steps = max(3, min(args.steps, 20))
    ctx.aev_forward_backward_host(w.pos, w.species, w.box, w.grad_aev)
    # the caller's buffers are page-locked host memory (the library copies from / to them directly)
    pin = lambda a: torch.from_numpy(a).pin_memory().numpy()
    pos_h, sp_h, g_h = pin(w.pos), pin(w.species), pin(w.grad_aev)
    aev_h = torch.empty((w.batch, w.n_atoms, ctx.length), dtype=torch.float32).pin_memory().numpy()
    f_h = torch.empty((w.batch, w.n_atoms, 3), dtype=torch.float32).pin_memory().numpy()
    ctx.aev_forward_backward_host(pos_h, sp_h, w.box, g_h, aev_out=aev_h, forces_out=f_h)
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        ctx.aev_forward_backward_host(pos_h, sp_h, w.box, g_h, aev_out=aev_h, forces_out=f_h)
    dt = time.perf_counter() - t0
    e2e = {"value": n_atoms * e2e_steps / dt, "unit": UNIT, "steps": e2e_steps,
           "h2d_bytes_per_step": int(w.pos.nbytes + w.species.nbytes + w.grad_aev.nbytes),
           "d2h_bytes_per_step": int(aev_h.nbytes + f_h.nbytes),
           "call": "aev_forward_backward_host (pinned host pointers; H2D of grad || forward kernels || D2H of the AEV, then backward + D2H of the forces; synchronous)"}

    # ---- the other configurations (context rows, not the headline)
    other = {}
    for name in ("C1", "C2", "C3"):
        ww = make_workload(name)
        c2 = pkg.Context(ww.params, max_atoms=ww.n_atoms, max_batch=ww.batch, device=local)
        p2, s2, g2 = (torch.from_numpy(x).to(dev) for x in (ww.pos, ww.species, ww.grad_aev))
        a2 = torch.empty_like(g2)
        f2 = torch.empty((ww.batch, ww.n_atoms, 3), dtype=torch.float32, device=dev)

        def st2():
            c2.aev_forward(p2, s2, ww.box, aev_out=a2)
            c2.aev_backward(g2, forces_out=f2)
        for _ in range(3):
            st2()
        tt = _time_steps(st2, min(args.steps, 50), flush, torch)
        other[name] = {"ms_per_eval": float(tt.mean()), "atoms_per_s": ww.batch * ww.n_atoms / (tt.mean() * 1e-3),
                       "evaluations_per_s": ww.batch / (tt.mean() * 1e-3)}
        # the same evaluation captured once in a CUDA graph and replayed (the MD-loop calling pattern)
        try:
            side = torch.cuda.Stream()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                st2()
            torch.cuda.current_stream().wait_stream(side)
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=side):
                st2()
            for _ in range(3):
                graph.replay()
            tg = _time_steps(graph.replay, min(args.steps, 50), flush, torch)
            c2.check_status()
            other[name]["graph_ms_per_eval"] = float(tg.mean())
            other[name]["graph_evaluations_per_s"] = ww.batch / (tg.mean() * 1e-3)
            del graph
        except Exception as exc:      # reported, never fatal for the headline
            other[name]["graph_error"] = repr(exc)[:200]
        c2.close()
    # the headline step in the two optional context modes (same buffers; include/aev.h: flags, skin)
    for tag, kw, what in (("C4_deterministic", {"flags": pkg.AEV_FLAG_DETERMINISTIC},
                           "C4 step with AEV_FLAG_DETERMINISTIC (k_rank + fixed-point force accumulator)"),
                          ("C4_skin", {"skin": 0.5},
                           "C4 step on a Verlet-skin context (skin 0.5), positions unchanged between calls: every timed "
                           "step reuses the lists (k_disp + k_refresh instead of k_bin + k_nbr)")):
        cm = pkg.Context(w.params, max_atoms=w.n_atoms, max_batch=w.batch, device=local, **kw)

        def stm():
            cm.aev_forward(pos, sp, w.box, aev_out=aev_out)
            cm.aev_backward(g, forces_out=f_out)
        for _ in range(3):
            stm()
        tm = _time_steps(stm, min(args.steps, 50), flush, torch)
        cm.check_status()
        other[tag] = {"ms_per_eval": float(tm.mean()), "atoms_per_s": n_atoms / (tm.mean() * 1e-3), "what": what}
        cm.close()
    w5 = make_workload("C5")
    c5 = pkg.Context(w5.params, max_atoms=w5.n_atoms, device=local)
    for s, (ws, bs) in make_c5_weights().items():
        c5.ani_mlp_load(s, ws, bs, CELU_ALPHA)
    p5, s5 = torch.from_numpy(w5.pos).to(dev), torch.from_numpy(w5.species).to(dev)
    e5 = torch.empty((1,), dtype=torch.float64, device=dev)
    f5 = torch.empty((1, w5.n_atoms, 3), dtype=torch.float32, device=dev)

    def st5():
        c5.ani_energy_forces(p5, s5, w5.box, energy_out=e5, forces_out=f5)
    for _ in range(3):
        st5()
    tt = _time_steps(st5, min(args.steps, 50), flush, torch)
    c5.aev_set_profiling(True); c5.aev_get_profile()
    for _ in range(5):
        st5()
    p5prof = c5.aev_get_profile()
    other["C5"] = {"ms_per_eval": float(tt.mean()), "atoms_per_s": w5.n_atoms / (tt.mean() * 1e-3),
                   "what": "ani_energy_forces: AEV + per-species MLP fwd/bwd + AEV backward, 4,500-atom box",
                   "mlp_ms": p5prof["mlp"][0] / max(1, p5prof["mlp"][1]), "mlp_kernel": c5.mlp_kernel()}
    c5.aev_set_profiling(False)
    # the call an MD engine makes: positions in, energy + forces out, host buffers, synchronous
    pin = lambda a: torch.from_numpy(a).pin_memory().numpy()
    p5h, s5h = pin(w5.pos), pin(w5.species)
    for _ in range(3):
        c5.ani_energy_forces_host(p5h, s5h, w5.box)
    t0 = time.perf_counter()
    n5 = 50
    for _ in range(n5):
        c5.ani_energy_forces_host(p5h, s5h, w5.box)
    dt5 = (time.perf_counter() - t0) / n5
    other["C5"]["e2e"] = {"ms_per_eval": dt5 * 1e3, "atoms_per_s": w5.n_atoms / dt5,
                          "h2d_bytes_per_step": int(w5.pos.nbytes + w5.species.nbytes),
                          "d2h_bytes_per_step": int(w5.n_atoms * 12 + 8),
                          "call": "ani_energy_forces_host (wall clock, L2 not flushed)"}
    c5.close()

    def c5_variant(models, tag, what):
        cc = pkg.Context(w5.params, max_atoms=w5.n_atoms, device=local)
        cc.ani_mlp_set_ensemble(len(models))
        for m, nets in enumerate(models):
            for s, (ws, bs) in nets.items():
                cc.ani_mlp_load_model(m, s, ws, bs, CELU_ALPHA)

        def stv():
            cc.ani_energy_forces(p5, s5, w5.box, energy_out=e5, forces_out=f5)
        for _ in range(3):
            stv()
        tv = _time_steps(stv, min(args.steps, 50), flush, torch)
        cc.aev_set_profiling(True); cc.aev_get_profile()
        for _ in range(5):
            stv()
        pv = cc.aev_get_profile()
        other[tag] = {"ms_per_eval": float(tv.mean()), "atoms_per_s": w5.n_atoms / (tv.mean() * 1e-3), "what": what,
                      "mlp_ms": pv["mlp"][0] / max(1, pv["mlp"][1]), "mlp_kernel": cc.mlp_kernel()}
        cc.close()
    # the paper's own ML workload shape: one 60-atom ligand-like region per MD step, host call
    from gen import make_ensemble_weights
    wl = make_workload("C2")
    lig = {}
    for nm in (1, 8):
        cl = pkg.Context(wl.params, max_atoms=wl.n_atoms, device=local)
        cl.ani_mlp_set_ensemble(nm)
        for m, nets in enumerate(make_ensemble_weights(nm, arch={s: [384, 160, 128, 96, 1] for s in range(4)})):
            for s, (ws, bs) in nets.items():
                cl.ani_mlp_load_model(m, s, ws, bs, CELU_ALPHA)
        lp, ls = np.ascontiguousarray(wl.pos[:1]), np.ascontiguousarray(wl.species[:1])
        for _ in range(5):
            cl.ani_energy_forces_host(lp, ls, None)
        t0 = time.perf_counter()
        for _ in range(300):
            cl.ani_energy_forces_host(lp, ls, None)
        lig["models_%d_us_per_call" % nm] = (time.perf_counter() - t0) / 300 * 1e6
        cl.close()
    lig["what"] = "ani_energy_forces_host on one 60-atom conformer of C2 (host positions in, energy + forces out, wall clock)"
    other["ligand_md_step"] = lig
    c5_variant(make_ensemble_weights(8), "C5_ens8",
               "C5 with an ensemble of 8 networks per species (PAPER.md:193), bf16-representable weights")
    c5_variant(make_ensemble_weights(1, round_bf16=False), "C5_fp32_weights",
               "C5 with fp32 (not bf16-representable) weights: weight hi+lo operands on tcgen05")

    cpu = cpu_baseline()

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": _config(n_atoms),
        "arm": {"parallelism": "replicas x%d" % world, "ms_per_step_median": float(np.median(t_ms)),
                "ms_per_step_min": float(t_ms.min())},
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
        "roofline": roofline, "cpu_baseline": cpu, "other": other,
    }
    print(json.dumps(line))
    ctx.close()
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--quick", action="store_true",
                    help="headline loop + per-kernel pass only (for ncu runs): no e2e / other configs / cpu baseline")
    ap.add_argument("--workload", default="C4", choices=["C4", "C5", "C5_ens8", "C5_fp32"],
                    help="with --quick: C4 (headline step) or a C5 variant (full energy+forces evaluation)")
    args = ap.parse_args()
    if args.quick and args.workload != "C4":
        run_quick_c5(args)
        return
    if args.impl == "reference":
        if args.steps > 200:
            args.steps = 200
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
