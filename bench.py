#!/usr/bin/env python
"""bench.py -- libdebye headline benchmark (BASELINE.json metric: G pair.q sinc-terms/s and ms/profile on B200,
fraction of the FP32-issue roofline), with the CPU oracle timed beside it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg2] [--variant auto] [--impl reference]

A "step" is one pass of the whole hot path (type sort + pack + all-pairs kernel + FP64 reduction + epilogue,
SURVEY.md section 8(a) S0-S7) over one synthetic structure: one debye_profile call (one debye_profile_batch call
for cfg4).  Workload at N=1: BASELINE.json configs[1] (cfg2: 10,000-atom globular blob, 101 q on [0, 0.5]).
With N GPUs every rank runs its own structure of the same shape (different seed): the path shards over independent
structures with no data-path collective, so scaling is weak; time = max over ranks.
Prints ONE JSON line (rank 0)."""
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

from paper_1306_2258_b200 import workloads as wl          # noqa: E402  (input generators only, no arithmetic)

METRIC = "pair_q_sinc_terms_per_second"
UNIT = "G pair.q/s"
SM_COUNT, FP32_LANES, MUFU_LANES = 148, 128, 16           # per B200 / per SM per clock (B200_PROFILING.md)
# dram__bytes_read.sum + dram__bytes_write.sum of the pairs kernel, per launch, from the committed ncu --set full captures
# (profiles/r02_ncu_full_pairs_cfg{2,4,5}.txt); None where no capture exists
NCU_TRAFFIC = {("cfg2", "recur"): 239104, ("cfg4", "recur"): 32863232 + 145920, ("cfg5", "recur"): 3322624, ("cfg2", "mufu"): 366336}
NCU_TRAFFIC_SOURCE = ("profiles/r02_ncu_full_pairs_cfg2_v2.txt, r02_ncu_full_pairs_cfg{4,5}_v2.txt, r02_ncu_full_pairs_mufu_cfg2.txt (ncu --set full captures of "
                      "this kernel, commands in profiles/r02_product_form.md and r02_centred_form.md); not measured by this run")


TABLE1 = {f"table1_{n}": n for n in (1000, 2000, 4000, 10000, 20000, 40000, 100000)}       # the paper's Table I rows
# wide grids (more than 256 non-zero q from 0: more than two recurrence chunks, run as contiguous pieces of the centred form)
WIDE = {"wide_1000q": lambda: wl.small_random(5, 30000, 4, 1000, q_max=2.0, box=150.0), "wide_512q": lambda: wl.small_random(4, 3000, 5, 512, q_max=1.5, box=60.0)}


def make_workload(name: str, rank: int = 0, grid: str = "config"):
    if name in TABLE1:
        w = wl.table1(TABLE1[name])
    elif name in WIDE:
        w = WIDE[name]()
    elif name == "cfg2" and rank:
        w = wl.cfg2(seed_off=2 + 1000 * rank, tag=f"cfg2_globular_10k_rank{rank}")
    else:
        w = wl.CONFIGS[name]()
    if grid != "config":                  # the same structure on a grid that is not uniform from 0 or dq (workloads.GRIDS)
        w = wl.with_grid(w, wl.GRIDS[grid](w), grid)
    return w


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return json.load(open(p))
    except Exception:
        return {}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz, self._stop_evt = index, [], set(), None, threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                 "hw_power_brake_slowdown": 0x80, "sync_boost": 0x10, "applications_clocks_setting": 0x2}
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.004)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def cpu_baseline(w, budget_s: float = 15.0):
    """The oracle as it stands (oracle/debye_oracle.c, fp64, OpenMP over rows), timed on this host's cores on a
    bounded sample of the same workload: the first R rows of the symmetric double loop."""
    from oracle import oracle as orc
    xyz = w.xyz[0] if w.xyz.ndim == 3 else w.xyz
    N, M = w.N, w.M
    r_probe = min(N, 64)
    t0 = time.perf_counter()
    _, nthr = orc.debye_sym(xyz, w.type, w.fftab, w.q, rows=(0, r_probe), return_threads=True)
    dt = max(time.perf_counter() - t0, 1e-6)
    pairs = lambda r: r * (N - 1) - r * (r - 1) // 2           # pairs (i<j) with i < r
    rate = pairs(r_probe) * M / dt
    rows = N
    if pairs(N) * M / rate > budget_s:
        rows = r_probe
        while rows < N and pairs(rows) * M / rate < budget_s:
            rows += 64
        rows = min(rows, N)
    t0 = time.perf_counter()
    orc.debye_sym(xyz, w.type, w.fftab, w.q, rows=(0, rows))
    dt = time.perf_counter() - t0
    # the same oracle on ONE thread, on a slab sized for ~4 s from the all-core rate
    rate_all = pairs(rows) * M / dt
    r1 = 1
    while r1 < rows and pairs(r1) * M < rate_all / max(int(nthr), 1) * 4.0:
        r1 += 1
    t0 = time.perf_counter()
    orc.debye_sym(xyz, w.type, w.fftab, w.q, rows=(0, r1), threads=1)
    dt1 = time.perf_counter() - t0
    rate_1 = pairs(r1) * M / dt1
    total = float(w.pair_q)                            # the whole workload (all conformers of a batch)
    return {"value": rate_all / 1e9, "unit": UNIT, "cores": int(nthr), "kind": "oracle",
            "sample": f"rows 0..{rows - 1} of {N} of the i<j double loop ({pairs(rows) * M:.3e} pair.q, {dt:.2f} s)"
                      + (" = the whole profile" if rows == N else ""),
            "seconds": dt,
            "ms_per_step_extrapolated": total / rate_all * 1e3,
            "one_thread": {"value": rate_1 / 1e9, "unit": UNIT, "sample": f"rows 0..{r1 - 1} ({pairs(r1) * M:.3e} pair.q, {dt1:.2f} s)",
                           "ms_per_step_extrapolated": total / rate_1 * 1e3}}


def run_reference(args, rank, world):
    """--impl reference: the oracle itself, each step a bounded row slab of the same workload."""
    if rank != 0:
        return
    from oracle import oracle as orc
    w = make_workload(args.config)
    xyz = w.xyz[0] if w.xyz.ndim == 3 else w.xyz
    N, M = w.N, w.M
    pairs = lambda r: r * (N - 1) - r * (r - 1) // 2
    t0 = time.perf_counter()
    _, nthr = orc.debye_sym(xyz, w.type, w.fftab, w.q, rows=(0, min(N, 64)), return_threads=True)
    rate = pairs(min(N, 64)) * M / max(time.perf_counter() - t0, 1e-6)
    per_step = max(0.2, min(120.0 / (args.steps + args.warmup), 20.0))
    rows = min(N, 64)
    while rows < N and pairs(rows) * M / rate < per_step:
        rows += 64
    rows = min(rows, N)
    for _ in range(args.warmup):
        orc.debye_sym(xyz, w.type, w.fftab, w.q, rows=(0, rows))
    t0 = time.perf_counter()
    for _ in range(args.steps):
        orc.debye_sym(xyz, w.type, w.fftab, w.q, rows=(0, rows))
    dt = time.perf_counter() - t0
    value = pairs(rows) * M * args.steps / dt / 1e9
    sample = f"rows 0..{rows - 1} of {N} per step ({pairs(rows) * M:.3e} pair.q)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "N": N, "T": w.T, "M": M, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": int(nthr), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def respawn_if_needed(args):
    """`python bench.py --gpus N` (N > 1) without a launcher: start N ranks, one per GPU, under torch.distributed.run on
    127.0.0.1 and hand it the same arguments.  Under a launcher (WORLD_SIZE set) the two counts must agree."""
    ws = os.environ.get("WORLD_SIZE")
    if ws is not None:
        if int(ws) != args.gpus:
            raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={ws}: launch with --nproc-per-node {args.gpus}")
        return
    if args.gpus <= 1:
        return
    if args.impl == "reference":
        return          # the oracle arm runs on rank 0's host cores only
    import socket
    import subprocess
    import torch
    have = torch.cuda.device_count()
    if have < args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} needs {args.gpus} CUDA devices, this node has {have}")
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def stored_oracle(name):
    """rows (conformer, k, I) of the oracle's stored whole profile of a full-size config (tests/golden/oracle_full_<name>.txt,
    written by tests/golden/make_golden_full.py from oracle/ alone), or None."""
    path = os.path.join(ROOT, "tests", "golden", f"oracle_full_{name}.txt")
    if not os.path.exists(path):
        return None
    rows = []
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        _, b, k, _, I, _ = line.split()
        rows.append((int(b), int(k), float(I)))
    return rows


def roofline_of(w, variant_ran, pairs_ms, fmax_ghz):
    """Roofline of the pairs kernel.  Algorithmic work per pair.q as SURVEY.md 8(d) counts it for a
    uniform grid: one recurrence FMA + one accumulate = 2 FP32-pipe lane-operations (4 FMA-equivalent flop)."""
    nz = int(np.count_nonzero(w.q))                                             # q = 0 is answered in closed form by the epilogue
    pq_all, pq_nz = float(w.pair_q), float(w.pair_q) / w.M * nz
    if variant_ran in ("recur", "centred"):
        peak = SM_COUNT * FP32_LANES * 2 * fmax_ghz / 1e3                       # TFLOP/s, FMA = 2 flop
        achieved = 4.0 * pq_nz / (pairs_ms * 1e-3) / 1e12
        return {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak, "traffic": None,
                "frac_product_form_1_lane_op": 0.5 * achieved / peak,
                "note": "FP32-pipe roofline with SURVEY 8(d)'s algorithmic count for a uniform grid: 2 lane-ops (recurrence FFMA + "
                        "accumulate = 4 FMA-equivalent flop) per pair.q with q != 0; peak = 148 SM x 128 lanes x 2 x sm_max_mhz "
                        "(MEASURED_PEAKS.json clock; nominal -- bench.py --peaks measures the pipe rates, profiles/r02_pipe_peaks.md). "
                        "The product form of the kernel (DESIGN.md section 5.1) needs ONE FFMA lane per pair.q plus a per-pair "
                        "start-up, so this fraction can exceed 1; frac_product_form_1_lane_op counts 1 lane-op per pair.q instead"}
    peak = SM_COUNT * MUFU_LANES * fmax_ghz / 1e3                               # T MUFU op/s
    achieved = pq_all / (pairs_ms * 1e-3) / 1e12
    return {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "T sin/s", "frac": achieved / peak, "traffic": None,
            "note": "XU (MUFU) roofline: one MUFU.SIN per pair.q, 16 lanes/clk/SM" if variant_ran == "mufu" else
                    "reference variant; XU roofline quoted for scale"}


def measure(db, w, dev, variant, use_hint, steps, warmup, world=1, e2e=True):
    """Times `steps` calls of debye_profile[_batch] on workload w (device-resident inputs, L2 flushed between steps) and,
    separately, the pairs kernel alone and the host-buffer entry.  Returns a dict of raw figures."""
    import torch
    import torch.distributed as dist
    from paper_1306_2258_b200 import sharding
    batch = w.xyz.ndim == 3
    call = db.debye_profile_batch if batch else db.debye_profile
    call_host = db.debye_profile_batch_host if batch else db.debye_profile_host
    x, t, f, q = (torch.from_numpy(a).to(dev) for a in (w.xyz, w.type, w.fftab, w.q))
    out = torch.empty((w.B, w.M) if batch else (w.M,), dtype=torch.float64, device=dev)
    flush = torch.empty(192 * 1024 * 1024, dtype=torch.uint8, device=dev)        # > 126 MB L2
    # the q grid exists on the host (it was generated there), so the caller can tell the library its shape: one pairs launch
    # instead of up to four (include/debye.h, DEBYE_QHINT_*); the device verifies the hint
    hint = db.q_hint(w.q) if use_hint else 0
    if variant == "centred":              # forced centred product form: needs the pieces of the grid whatever its class
        hint = db.q_hint_pieces(w.q)
        if not hint:
            raise SystemExit("bench.py: --variant centred needs a piecewise-uniform grid")
    info = db.launch_info(w.N, w.B, w.T, w.M, variant, with_grid=True, hint=hint)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(warmup):
        call(x, t, f, q, out, variant=variant, hint=hint)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    barrier()
    sampler = ClockSampler(dev.index or 0)
    sampler.start()
    wall0 = time.perf_counter()
    # The host must stay ahead of the device, or the per-step events of a 20 us step measure the Python call overhead: a spin
    # kernel holds the stream while the first steps are enqueued, and again every 25 steps (the launch queue is finite).
    gate = getattr(torch.cuda, "_sleep", None) if w.pair_q < 2e9 else None
    for i, (a, b) in enumerate(ev):
        if gate is not None and i % 25 == 0:
            gate(int(4e6))                      # ~2 ms at 1.9 GHz, outside the per-step events
        flush.fill_(1)                          # L2 flush between steps, outside the per-step events
        a.record()
        call(x, t, f, q, out, variant=variant, hint=hint)
        b.record()
    barrier()
    wall = time.perf_counter() - wall0
    clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = sharding.max_over_ranks(float(np.sum(step_ms)), dev)
    units = sharding.sum_over_ranks(float(w.pair_q), dev)          # pair.q per step over all ranks
    res = {"total_ms": total_ms, "units": units, "wall": wall, "clocks": clocks, "info": info, "hint": hint,
           "value": units * steps / (total_ms * 1e-3) / 1e9}

    # ---- dominant kernel (pairs) timed alone with events recorded by the library around its launch ----------
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(); e1.record(); torch.cuda.synchronize()
    db.set_pairs_events(e0, e1)
    pk = []
    for _ in range(min(steps, 30)):
        if gate is not None:
            gate(int(1e6))
        flush.fill_(1)
        call(x, t, f, q, out, variant=variant, hint=hint)
        torch.cuda.synchronize()
        pk.append(e0.elapsed_time(e1))
    db.set_pairs_events(None, None)
    res["pairs_ms"] = float(np.mean(pk))
    res["result"] = out.cpu().numpy()

    # ---- end to end through the host-buffer C entry (pinned inputs, copies inside the timed region) ----------
    if e2e:
        hx, ht, hf, hq = (torch.from_numpy(a).pin_memory().numpy() for a in (w.xyz, w.type, w.fftab, w.q))
        hout = torch.empty((w.B, w.M) if batch else (w.M,), dtype=torch.float64).pin_memory().numpy()
        for _ in range(3):
            call_host(hx, ht, hf, hq, hout, variant=variant, hint=hint)
        barrier()
        n_e2e = max(5, min(steps, 50))
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            call_host(hx, ht, hf, hq, hout, variant=variant, hint=hint)
        barrier()
        e2e_s = sharding.max_over_ranks(time.perf_counter() - t0, dev)
        assert np.array_equal(res["result"], hout), "host entry and device entry disagree"
        res["e2e"] = {"value": units * n_e2e / e2e_s / 1e9, "unit": UNIT, "h2d_bytes_per_step": int(hx.nbytes + ht.nbytes + hf.nbytes + hq.nbytes),
                      "d2h_bytes_per_step": int(hout.nbytes), "ms_per_step": e2e_s / n_e2e * 1e3, "steps": n_e2e}
    return res


def variant_that_ran(variant, w, use_hint=True):
    """the pairs kernel an automatic call runs: the library's own classification of the grid (debye_q_hint, host copy of q)"""
    if variant != "auto":
        return variant
    from paper_1306_2258_b200 import binding as db
    h = db.q_hint(w.q)
    if use_hint and db.pieces_of(h)[0]:
        return "centred"                  # piecewise uniform / general start, hinted: the centred product form
    if db.pieces_of(h)[0] == 1:           # uniform with a general start, no hint: the device picks the centred launch if one was offered
        return "centred" if w.M <= 32 * 128 else "recur"
    return "recur" if h & (1 << 9) else "mufu"


def kernel_shape(db, w, res, variant_ran):
    """(K, n_chunks) of the pairs launch that did the work."""
    info, hint = res["info"], res["hint"]
    k_ran, chunks_ran = info["q_chunk"], info["n_chunks"]
    if variant_ran == "centred":
        chunks_ran, k_ran = db.pieces_of(db.q_hint_pieces(w.q))
        return k_ran, chunks_ran
    if hint == 0 and variant_ran == "recur" and w.M >= 2 and float(w.q[0]) == 0.0:
        # grid starts at q = 0: the device runs the recurrence launch sized for M - 1 chain indices when the library
        # offered one (it does when that saves accumulators or a chunk)
        alt = db.launch_info(w.N, w.B, w.T, w.M - 1, "recur")
        if alt["n_chunks"] <= 2 and (alt["q_chunk"] < k_ran or alt["n_chunks"] < chunks_ran):
            k_ran, chunks_ran = alt["q_chunk"], alt["n_chunks"]
    return k_ran, chunks_ran


def config_summary(db, name, dev, variant, use_hint, fmax_ghz, grid="config"):
    """One entry of the `configs` object: a full-size BASELINE config measured like the headline (fewer steps) and checked
    against the oracle's stored whole profile (cfg1 / cfg2: the oracle runs live)."""
    from oracle import oracle as orc
    w = make_workload(name, 0, grid)
    steps = {"cfg1": 50, "cfg2": 30, "cfg3": 8, "cfg4": 8, "cfg5": 4}.get(name, 10)
    res = measure(db, w, dev, variant, use_hint, steps, 3, e2e=False)
    vr = variant_that_ran(variant, w, use_hint)
    k_ran, chunks_ran = kernel_shape(db, w, res, vr)
    roof = roofline_of(w, vr, res["pairs_ms"], fmax_ghz)
    rows = stored_oracle(name) if grid == "config" else None
    I = res["result"]
    if rows is None:
        ref = orc.debye_sym(w.xyz, w.type, w.fftab, w.q)
        err, checked, against = float(np.max(np.abs(I - ref) / np.abs(ref))), int(w.M), "oracle run live, every q"
    else:
        err = max(abs((I[b, k] if I.ndim == 2 else I[k]) - ref) / abs(ref) for b, k, ref in rows)
        checked, against = len(rows), f"stored oracle profile tests/golden/oracle_full_{name}.txt (every q" + (", 65 conformers)" if I.ndim == 2 else ")")
    return {"workload": w.name, "N": w.N, "T": w.T, "M": w.M, "B": w.B, "steps": steps, "ms_per_step": res["total_ms"] / steps,
            "T_pair_q_per_s": res["value"] / 1e3, "kernel": f"debye_small_kernel<{k_ran}> (one fused launch)" if res["info"]["n_launches"] == 1 else f"debye_pairs_kernel<{k_ran}, {vr}>", "kernel_ms": res["pairs_ms"],
            "q_chunk": k_ran, "n_chunks": chunks_ran, "pairs_grid": res["info"]["pairs_grid"], "frac": roof["frac"],
            "frac_product_form_1_lane_op": roof.get("frac_product_form_1_lane_op"),
            "pair_q_per_clk_per_sm": float(w.pair_q) / (res["pairs_ms"] * 1e-3) / (SM_COUNT * fmax_ghz * 1e9),
            "clocks": res["clocks"], "max_rel_err": float(err), "values_checked": checked, "checked_against": against}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", default="cfg2", choices=sorted(wl.CONFIGS) + list(TABLE1) + list(WIDE),
                    help="cfg1..cfg5: BASELINE.json's configs; table1_N: the shape of the paper's Table I rows (N atoms, 50 q on (0, 1])")
    ap.add_argument("--variant", default="auto", choices=["auto", "recur", "mufu", "accurate", "fp64", "centred"])
    ap.add_argument("--grid", default="config", choices=["config"] + sorted(wl.GRIDS),
                    help="q grid: the config's own (uniform from 0), or the same number of points as a uniform grid with a general "
                         "start / as two uniform pieces (workloads.GRIDS): these run the centred product form when hinted")
    ap.add_argument("--impl", default="libdebye", choices=["libdebye", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="skip the per-config summary (`configs` object) of the default 1-GPU run")
    ap.add_argument("--split", default="structures", choices=["structures", "tiles"],
                    help="what the headline of a multi-GPU run measures: structures = every rank its own structure (weak scaling, no "
                         "collective; the default, with the tile split of one cfg5 structure reported beside it as `tile_split`); tiles = ONE "
                         "structure (--config) split over the ranks by tiles of the upper triangle, one all-gather of FP64 partials per "
                         "profile (strong scaling; debye_partials_shard + debye_profile_from_partials)")
    ap.add_argument("--path", default="pertype", choices=["pertype", "peratom"],
                    help="pertype: the north_star path (debye_profile, form factors per atom type); peratom: the paper's general "
                         "case (debye_profile_peratom, one form-factor row per atom; NEXT-1)")
    ap.add_argument("--peaks", action="store_true",
                    help="measure what one SM delivers on the instruction mixes of the pairs kernels (debye_pipe_bench) and the MUFU.SIN "
                         "error statistics; prints one JSON object and exits")
    ap.add_argument("--no-hint", action="store_true", help="do not pass the q-grid hint (DEBYE_QHINT_*) computed from the host copy of q")
    args = ap.parse_args()
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    respawn_if_needed(args)
    args.warmup = max(args.warmup, 3) if args.impl == "libdebye" else args.warmup
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        return run_reference(args, rank, world)

    import torch
    import torch.distributed as dist
    from paper_1306_2258_b200 import binding as db
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (libdebye has no CPU fallback)")
    if torch.cuda.device_count() <= local_rank:
        raise SystemExit(f"bench.py: rank {rank} needs CUDA device {local_rank}, this node has {torch.cuda.device_count()}")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    db.lib()

    if args.peaks:
        return run_peaks(dev) if rank == 0 else None
    w = make_workload(args.config, rank, args.grid)
    if args.path == "peratom":
        return run_peratom(args, w, rank, world, dev)
    if args.split == "tiles":
        line = run_tile_split(args, make_workload(args.config, 0), rank, world, dev)
        if rank == 0:
            print(json.dumps(line))
        if world > 1:
            dist.destroy_process_group()
        return
    batch = w.xyz.ndim == 3
    res = measure(db, w, dev, args.variant, not args.no_hint, args.steps, args.warmup, world)
    # multi-GPU: beside the independent structures (weak scaling), ONE cfg5 structure split over the ranks by tiles
    split_line = None
    if world > 1:
        sargs = argparse.Namespace(**vars(args))
        sargs.steps, sargs.warmup = 5, 3
        split_line = run_tile_split(sargs, make_workload("cfg5", 0), rank, world, dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks = measured_peaks()
    fmax_ghz = float(peaks.get("sm_max_mhz", 1965.0)) / 1e3
    variant_ran = variant_that_ran(args.variant, w, not args.no_hint)
    pairs_ms, total_ms, info = res["pairs_ms"], res["total_ms"], res["info"]
    roof = roofline_of(w, variant_ran, pairs_ms, fmax_ghz)
    # dram__bytes_read.sum + dram__bytes_write.sum of the pairs kernel from a committed ncu --set full capture of this command
    # (None where no capture exists): not measured by this run
    roof["traffic"] = NCU_TRAFFIC.get((args.config, variant_ran))
    roof["traffic_source"] = NCU_TRAFFIC_SOURCE if roof["traffic"] is not None else None
    k_ran, chunks_ran = kernel_shape(db, w, res, variant_ran)
    roof["kernel"] = f"debye_small_kernel<{k_ran}>" if info["n_launches"] == 1 else f"debye_pairs_kernel<{k_ran}, {variant_ran}>"
    if variant_ran == "centred":
        roof["note"] = ("FP32-pipe roofline with SURVEY 8(d)'s algorithmic count: 2 lane-ops (4 FMA-equivalent flop) per pair.q with q != 0; the "
                        "centred product form (DESIGN.md section 5.5) executes 1 lane-op per pair.q plus a per-pair, per-piece start-up")
        roof.pop("frac_product_form_1_lane_op", None)
    roof["kernel_ms"] = pairs_ms
    roof["pair_q_per_clk_per_sm"] = float(w.pair_q) / (pairs_ms * 1e-3) / (SM_COUNT * fmax_ghz * 1e9)
    roof["share_of_step"] = pairs_ms / (total_ms / args.steps)

    line = {
        "metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64" if variant_ran == "fp64" else "f32", "data": "synthetic",
        "config": {"workload": w.name, "N": w.N, "T": w.T, "M": w.M, "B": w.B, "variant": variant_ran, "grid": args.grid,
                   "pairs_grid": info["pairs_grid"], "q_chunk": k_ran, "n_chunks": chunks_ran,
                   "q_hint": "passed (grid classified from the host copy of q, verified on the device)" if res["hint"] else "none",
                   "l2": "flushed between steps (192 MiB fill, outside the per-step events)",
                   "parallelism": f"{world} independent structure(s), one per GPU", "wall_s_timed_loop": res["wall"]},
        "clocks": res["clocks"],
        "e2e": res["e2e"],
        "gpu_launches": info["n_launches"] * args.steps,
        "roofline": roof,
    }
    if split_line is not None:
        line["tile_split"] = split_line
    if world == 1 and not args.no_cpu_baseline:
        cb = cpu_baseline(w)
        from oracle import oracle as orc                   # parity of the timed call's output against the oracle
        if not batch:
            ks = list(range(0, w.M, max(1, w.M // 8)))
            ref = orc.debye_sym(w.xyz, w.type, w.fftab[:, ks].copy(), w.q[ks].copy())
            line["parity_max_rel_err"] = float(np.max(np.abs(res["result"][ks] - ref) / np.abs(ref)))
        line["cpu_baseline"] = cb
    if world == 1 and args.config == "cfg2" and args.variant == "auto" and not args.no_configs and not args.no_cpu_baseline:
        # the other BASELINE configs, same launch configuration, fewer steps; each checked against the oracle's whole profile
        line["configs"] = {name: config_summary(db, name, dev, args.variant, not args.no_hint, fmax_ghz) for name in sorted(wl.CONFIGS)}
        # cfg2's structure on grids that are not uniform from 0 (workloads.GRIDS): the centred product form
        line["grids"] = {g: config_summary(db, "cfg2", dev, args.variant, not args.no_hint, fmax_ghz, g) for g in sorted(wl.GRIDS)}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_peaks(dev):
    """--peaks: the measured side of the "alu" roofline.  Rates are per SM clock (clock64 inside the kernels), so they do
    not depend on the clock the part runs at; nominal: 128 FP32 lanes and 16 MUFU lanes per SM and clock."""
    from paper_1306_2258_b200 import binding as db
    L = db.lib()
    sampler = ClockSampler(dev.index or 0)
    sampler.start()
    tests = []
    for t in range(L.debye_pipe_bench_count()):
        row = {"test": t}
        for c in (1, 2, 3, 4):
            r = db.pipe_bench(t, c)
            if r is None:
                continue
            row["name"] = r[0]
            row[f"ctas{c}"] = {"lane_ops_per_clk_per_sm": round(r[1], 2), "sched_cycles_per_instr": round(r[2], 3)}
        tests.append(row)
    mx, rms, mean = db.mufu_sin_error()
    rmx, rrms, rmean = db.mufu_rsq_error()
    print(json.dumps({"pipe_bench": tests, "mufu_rsq_relative_error_log_uniform_1_to_4": {"max": rmx, "rms": rrms, "mean": rmean, "points": 1 << 24}, "nominal": {"fp32_lanes_per_clk_per_sm": FP32_LANES, "mufu_lanes_per_clk_per_sm": MUFU_LANES},
                      "mufu_sin_error_on_0_to_half_turn": {"max_abs": mx, "rms": rms, "mean": mean, "points": 1 << 24},
                      "clocks": sampler.stop()}))


def run_tile_split(args, w, rank, world, dev):
    """--split tiles: one step = one profile of ONE structure on all ranks: debye_partials_shard(rank, world) (setup, pack,
    pairs CTAs c with c % world == rank, final), NCCL all-gather of S[B][T(T+1)/2][M] FP64, debye_profile_from_partials
    (rank-ordered sum + epilogue).  Strong scaling: total work is fixed.  Every rank ends with the full profile."""
    import torch
    import torch.distributed as dist
    from paper_1306_2258_b200 import binding as db, sharding
    x, t, f, q = (torch.from_numpy(a).to(dev) for a in (w.xyz, w.type, w.fftab, w.q))
    hint = 0 if args.no_hint else db.q_hint(w.q)
    flush = torch.empty(192 * 1024 * 1024, dtype=torch.uint8, device=dev)
    info = db.launch_info(w.N, w.B, w.T, w.M, args.variant, with_grid=True, hint=hint)

    sharding.assert_same_schedule(info["pairs_grid"], world, dev)       # CTA c belongs to rank c mod world on EVERY rank

    def step():
        return sharding.profile_tile_split(
            lambda r, wd: db.debye_partials_shard(x, t, q, w.T, r, wd, variant=args.variant, hint=hint),
            db.debye_profile_from_partials, f, rank, world)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        out = step()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    sampler = ClockSampler(dev.index or 0)
    sampler.start()
    for a, b in ev:
        flush.fill_(1)
        a.record()
        out = step()
        b.record()
    barrier()
    clocks = sampler.stop()
    total_ms = sharding.max_over_ranks(float(np.sum([a.elapsed_time(b) for a, b in ev])), dev)
    value = float(w.pair_q) * args.steps / (total_ms * 1e-3) / 1e9              # one structure: the job's units are not multiplied by N
    t0 = time.perf_counter()
    n_e2e = max(5, min(args.steps, 50))
    hx = torch.from_numpy(w.xyz).pin_memory()
    for _ in range(n_e2e):                                                       # coordinates from pinned host memory, profile read back
        x.copy_(hx, non_blocking=True)
        res = step().cpu()
    barrier()
    e2e_s = sharding.max_over_ranks(time.perf_counter() - t0, dev)
    # this rank's pairs kernel alone (events recorded by the library around its launch); max over ranks
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(); e1.record(); torch.cuda.synchronize()
    db.set_pairs_events(e0, e1)
    pk = []
    for _ in range(min(args.steps, 10)):
        flush.fill_(1)
        step()
        torch.cuda.synchronize()
        pk.append(e0.elapsed_time(e1))
    db.set_pairs_events(None, None)
    pairs_ms = sharding.max_over_ranks(float(np.mean(pk)), dev)
    if rank != 0:
        return None
    fmax_ghz = float(measured_peaks().get("sm_max_mhz", 1965.0)) / 1e3
    vr = variant_that_ran(args.variant, w)
    # every rank's pairs kernel does 1/world of the pairs: roofline of ONE GPU's kernel on its share
    roof = roofline_of(w, vr, pairs_ms * world, fmax_ghz)
    roof["kernel_ms"] = pairs_ms
    roof["note"] = f"per GPU: each rank's pairs kernel runs 1/{world} of the CTAs of the single-GPU schedule; " + roof["note"]
    roof["share_of_step"] = pairs_ms / (total_ms / args.steps)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "roofline": roof,
        "dtype": "f64" if args.variant == "fp64" else "f32", "data": "synthetic",
        "config": {"workload": w.name, "N": w.N, "T": w.T, "M": w.M, "B": w.B, "variant": args.variant, "pairs_grid": info["pairs_grid"],
                   "l2": "flushed between steps (192 MiB fill, outside the per-step events)",
                   "parallelism": f"one structure split over {world} rank(s) by tiles; all-gather of {w.B * w.T * (w.T + 1) // 2 * w.M * 8} B per rank"},
        "clocks": clocks,
        "e2e": {"value": float(w.pair_q) * n_e2e / e2e_s / 1e9, "unit": UNIT, "h2d_bytes_per_step": int(hx.numpy().nbytes),
                "d2h_bytes_per_step": int(res.numpy().nbytes), "ms_per_step": e2e_s / n_e2e * 1e3, "steps": n_e2e},
        "gpu_launches": (info["n_launches"] + 1) * args.steps,
    }
    if world == 1 and not args.no_cpu_baseline:
        from oracle import oracle as orc
        if w.xyz.ndim == 2:
            ks = list(range(0, w.M, max(1, w.M // 8)))
            ref = orc.debye_sym(w.xyz, w.type, w.fftab[:, ks].copy(), w.q[ks].copy())
            line["parity_max_rel_err"] = float(np.max(np.abs(out.cpu().numpy()[0][ks] - ref) / np.abs(ref)))
        line["cpu_baseline"] = cpu_baseline(w)
    rows = stored_oracle(args.config if w.name.startswith(args.config) else w.name.split("_")[0])
    if rows is not None and w.xyz.ndim == 2:
        I = out.cpu().numpy()[0]
        line["max_rel_err_vs_stored_oracle"] = float(max(abs(I[k] - ref) / abs(ref) for b, k, ref in rows))
    return line


def run_peratom(args, w, rank, world, dev):
    """--path peratom: one step = one debye_profile_peratom call (self terms, pairs, final: 3 launches) on the same synthetic
    structure with a seeded per-atom table (workloads.peratom_table).  Same JSON contract; roofline = XU pipe (one MUFU.SIN
    per pair.q); fp64 variant quoted against the same roofline for scale."""
    import torch
    import torch.distributed as dist
    from paper_1306_2258_b200 import binding as db, sharding
    batch = w.xyz.ndim == 3            # cfg4: B conformers sharing the table, debye_profile_peratom_batch
    variant = args.variant if args.variant in ("auto", "mufu", "fp64", "recur") else "auto"
    ff = wl.peratom_table(w, rank)
    # with the grid hint (q was generated on the host) a grid q_k = (k + koff) dq runs the recurrence (debye_peratom_recur.cuh)
    hint = 0 if (args.no_hint or variant in ("mufu", "fp64")) else db.q_hint(w.q)
    H, U, Z, D = 1 << 8, 1 << 9, 1 << 10, 1 << 11
    recur = bool(hint & U) and bool(hint & (Z | D)) and (w.M - (1 if hint & Z else 0)) <= 256
    # one small structure on a one-chunk grid: the single fused launch (debye_peratom_small.cuh)
    fused = recur and not batch and w.N <= 2048 and (w.M - (1 if hint & Z else 0)) <= 128
    x, f, q = (torch.from_numpy(a).to(dev) for a in (w.xyz, ff, w.q))
    out = torch.empty((w.B, w.M) if batch else w.M, dtype=torch.float64, device=dev)
    flush = torch.empty(192 * 1024 * 1024, dtype=torch.uint8, device=dev)
    entry = db.debye_profile_peratom_batch if batch else db.debye_profile_peratom

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        entry(x, f, q, out, variant=variant, hint=hint)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    sampler = ClockSampler(dev.index or 0)
    sampler.start()
    wall0 = time.perf_counter()
    # short steps: a spin kernel holds the stream while the steps are enqueued, so the per-step events never include the Python
    # call overhead (as in measure())
    gate = getattr(torch.cuda, "_sleep", None) if w.pair_q < 2e9 else None
    for i, (a, b) in enumerate(ev):
        if gate is not None and i % 25 == 0:
            gate(int(4e6))
        flush.fill_(1)
        a.record()
        entry(x, f, q, out, variant=variant, hint=hint)
        b.record()
    barrier()
    wall = time.perf_counter() - wall0
    clocks = sampler.stop()
    total_ms = sharding.max_over_ranks(float(np.sum([a.elapsed_time(b) for a, b in ev])), dev)
    units = sharding.sum_over_ranks(float(w.pair_q), dev)
    value = units * args.steps / (total_ms * 1e-3) / 1e9
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(); e1.record(); torch.cuda.synchronize()
    db.set_pairs_events(e0, e1)
    pk = []
    for _ in range(min(args.steps, 30)):
        flush.fill_(1)
        entry(x, f, q, out, variant=variant, hint=hint)
        torch.cuda.synchronize()
        pk.append(e0.elapsed_time(e1))
    db.set_pairs_events(None, None)
    pairs_ms = float(np.mean(pk))
    hx, hf, hq = (torch.from_numpy(a).pin_memory().numpy() for a in (w.xyz, ff, w.q))
    hout = torch.empty((w.B, w.M) if batch else w.M, dtype=torch.float64).pin_memory().numpy()
    if batch:       # no host-buffer C entry for batches: pinned host tensors copied in, the device entry, the result copied back
        tx, tf, tq, tout = (torch.from_numpy(a) for a in (hx, hf, hq, hout))

        def host_call():
            x.copy_(tx, non_blocking=True); f.copy_(tf, non_blocking=True); q.copy_(tq, non_blocking=True)
            entry(x, f, q, out, variant=variant, hint=hint)
            tout.copy_(out, non_blocking=True)
            torch.cuda.synchronize()
    else:
        def host_call():
            db.debye_profile_peratom_host(hx, hf, hq, hout, variant=variant, hint=hint)
    for _ in range(3):
        host_call()
    barrier()
    n_e2e = max(5, min(args.steps, 50))
    t0 = time.perf_counter()
    for _ in range(n_e2e):
        host_call()
    barrier()
    e2e_s = sharding.max_over_ranks(time.perf_counter() - t0, dev)
    result_dev = out.cpu().numpy()
    assert np.array_equal(result_dev, hout), "host entry and device entry disagree"
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    fmax_ghz = float(measured_peaks().get("sm_max_mhz", 1965.0)) / 1e3
    peak = SM_COUNT * MUFU_LANES * fmax_ghz / 1e3
    if recur:
        peak = SM_COUNT * FP32_LANES * 2 * fmax_ghz / 1e3                       # TFLOP/s, FMA = 2 flop
    # the library's q-chunk (debye_peratom_kq): the multiple of 4 in [16, 32] with the fewest padded slots, larger on ties
    kq = min(range(32, 12, -4), key=lambda c: ((w.M + c - 1) // c * c, -c))
    n_chunks_label = (w.M + kq - 1) // kq
    if recur:       # the recurrence keeps every chain index of a chunk in registers: K accumulators (a multiple of 8), 1 or 2 chunks
        n_idx = w.M - (1 if float(w.q[0]) == 0.0 else 0)
        n_chunks_label = 1 if n_idx <= 128 else 2
        last = max(n_idx - 1, 0)
        kq = max(8, (8 * (last // (8 * n_chunks_label)) + min(last % (8 * n_chunks_label), 7) + 1 + 7) // 8 * 8)
    achieved = float(w.pair_q) / (pairs_ms * 1e-3) / 1e12
    if recur:       # 2 FP32-pipe lane-operations (chain FFMA + weighted-accumulate FFMA = 4 flop) per pair.q with q != 0
        achieved = 4.0 * float(w.pair_q) / w.M * int(np.count_nonzero(w.q)) / (pairs_ms * 1e-3) / 1e12
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64" if variant == "fp64" else "f32", "data": "synthetic",
        "config": {"workload": w.name + "+peratom_table", "path": "peratom", "N": w.N, "M": w.M, "B": w.B,
                   "variant": "fp64" if variant == "fp64" else ("recur" if recur else "mufu"), "q_chunk": kq, "n_chunks": n_chunks_label,
                   "q_hint": "passed" if hint else "none",
                   "l2": "flushed between steps (192 MiB fill, outside the per-step events)",
                   "parallelism": f"{world} independent structure(s), one per GPU", "wall_s_timed_loop": wall},
        "clocks": clocks,
        "e2e": {"value": units * n_e2e / e2e_s / 1e9, "unit": UNIT, "h2d_bytes_per_step": int(hx.nbytes + hf.nbytes + hq.nbytes),
                "d2h_bytes_per_step": int(hout.nbytes), "ms_per_step": e2e_s / n_e2e * 1e3, "steps": n_e2e},
        "gpu_launches": (1 if fused else (4 if recur else 3 * w.B)) * args.steps,
        "roofline": {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s" if recur else "T sin/s", "frac": achieved / peak,
                     # dram__bytes_read.sum + write.sum of the pairs kernel from the full ncu capture (profiles/r01_v6.md)
                     "traffic": 4248064 if (args.config == "cfg2" and variant != "fp64" and not recur) else None,
                     "note": ("FP32-pipe roofline: 2 lane-ops (chain FFMA + accumulate FFMA against f_j = 4 FMA-equivalent flop) per pair.q "
                              "with q != 0; peak = 148 SM x 128 lanes x 2 x sm_max_mhz") if recur else
                             ("XU (MUFU) roofline: one MUFU.SIN per pair.q, 16 lanes/clk/SM x 148 SM x sm_max_mhz; the q-chunks "
                              "are padded (M = 101 runs 4 x 28 = 112 slots), which the algorithmic count does not credit"),
                     "kernel": "debye_peratom_small_kernel (one fused launch)" if fused else "debye_peratom_recur_kernel" if recur else f"debye_peratom_pairs_kernel<{'fp64' if variant == 'fp64' else 'fp32'}>", "kernel_ms": pairs_ms,
                     "share_of_step": pairs_ms / (total_ms / args.steps)},
    }
    if world == 1 and not args.no_cpu_baseline:
        from oracle import oracle as orc
        ks = list(range(0, w.M, max(1, w.M // 8)))
        if batch:       # first and last conformer
            errs = []
            for bb in (0, w.B - 1):
                ref = orc.debye_peratom(w.xyz[bb], ff[:, ks].copy(), w.q[ks].copy())
                errs.append(float(np.max(np.abs(result_dev[bb][ks] - ref) / np.abs(ref))))
            line["parity_max_rel_err"] = max(errs)
        else:
            ref = orc.debye_peratom(w.xyz, ff[:, ks].copy(), w.q[ks].copy())
            line["parity_max_rel_err"] = float(np.max(np.abs(result_dev[ks] - ref) / np.abs(ref)))
        ns = min(w.N, 6000)
        x0 = w.xyz[0] if batch else w.xyz
        t0 = time.perf_counter()
        orc.debye_peratom(x0[:ns], ff[:ns], w.q)
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": ns * (ns - 1) / 2 * w.M / dt / 1e9, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
                                "sample": f"oracle_debye_peratom on the first {ns} atoms, all {w.M} q ({dt:.2f} s)", "seconds": dt}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
