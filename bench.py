#!/usr/bin/env python
"""bench.py -- GB waveform + delta-lnL evaluations per second on B200 (BASELINE.json metric).

A step = one pass of the whole hot path over BASELINE.json's full ensemble
sweep (config index 4, "config 5"): gb_delta_loglike on 10 temperatures x 36 walkers x 12 000 sources =
4.32 M evaluations against 360 device-resident A/E residuals (10.8 GB), then gb_residual_update of the
seeded 25 % "accepted" rows.  Odd steps scatter with the opposite sign (REMOVE of the same sources), so
every step does identical work and the residuals return to their initial values without any untimed
restore.  Inputs exceed L2 by two orders of magnitude (no flush needed).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

One JSON line on stdout (rank 0).  `value` = evaluations / s over all ranks with inputs resident in HBM;
`e2e` = the same through the *_host C-ABI entry points (pinned host proposal buffers, host<->device copies
in the timed region; residuals and PSDs are the state that lives on the GPU);
`roofline` = the delta-lnL kernels against the FP64 pipe (bound "alu"); `cpu_baseline` = the CPU oracle
timed on a bounded sample.  --impl reference times the oracle itself (no GPU).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from concurrent.futures import ThreadPoolExecutor

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "gb_waveform_dlnL_evals_per_sec"
UNIT = "evals/s"
WORKLOAD = "cfg5_full_ensemble_sweep_10x36x12000"

# ---- algorithmic work per evaluation (frozen in BASELINE.md before optimisation) ----
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12      # 148 SMs x 64 DFMA/clk x 2 flop x 1.965 GHz = 37.2


def median_ms(torch, stream, fn, reps: int = 3, warm: int = 1) -> float:
    """Median over `reps` timed calls of fn() (CUDA events on `stream`, one pair per call) after `warm` untimed ones: the
    side measurements outside the timed step use it so that one disturbed call does not shift the reported figure."""
    for _ in range(warm):
        fn()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
    for a, b in evs:
        a.record(stream)
        fn()
        b.record(stream)
    torch.cuda.synchronize()
    return float(np.median([a.elapsed_time(b) for a, b in evs]))


def ncu_traffic(update: str):
    """DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) of the kernels of one timed step, read from the committed
    summary of the ncu --set full capture under profiles/ (never a literal here).  Returns (bytes or None, provenance)."""
    import csv
    path = os.path.join(ROOT, "profiles", "r2_step_traffic.csv")
    want = {"fused": "r2_step"}.get(update)
    try:
        for row in csv.DictReader(open(path)):
            if row["capture"] == want:
                b = float(row["dram_read_bytes_per_step"]) + float(row["dram_write_bytes_per_step"])
                return b, (f"profiles/r2_step_traffic.csv: capture {row['capture']} at commit {row['commit']}, "
                           f"{row['launches_per_step']} launches of {row['kernels']}")
    except (OSError, KeyError, ValueError):
        pass
    return None, "no committed ncu capture for this step form"


def flops_eval(N):
    N = np.asarray(N, dtype=np.float64)
    return 711.0 * N + 10.0 * N * np.log2(N) + 24.0 * N


def bytes_eval(N):
    return 48.0 * np.asarray(N, dtype=np.float64) + 72.0


def bytes_scatter(N):
    return 64.0 * np.asarray(N, dtype=np.float64)


def shard_info(rank: int, world: int, n_walkers_per_rank: int = 360):
    """Multi-GPU layout: walkers never interact, so each rank owns a whole
    ensemble replica of n_walkers_per_rank residuals; no data-path collective.  Returns the global walker
    ids this rank stands for."""
    lo = rank * n_walkers_per_rank
    return np.arange(lo, lo + n_walkers_per_rank, dtype=np.int64)


def max_over_ranks(ms: float, dist=None) -> float:
    """Step time of the job = max over ranks (device time)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms)
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([ms], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


# ------------------------------------------------------------------------------------------- clocks
_CLK_QUERY = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
              "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")


class ClockSampler:
    def __init__(self, gpu_index: int):
        self.proc = None
        self.lines = []
        self.gpu = gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={_CLK_QUERY}", "--format=csv,noheader,nounits",
                                          "-i", str(self.gpu), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for ln in self.proc.stdout:
            self.lines.append((time.perf_counter(), ln.strip()))

    def stop(self, t0=None, t1=None):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        for ts, ln in self.lines:
            if t0 is not None and not (t0 <= ts <= t1 + 0.1):
                continue
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); smax.append(float(f[2])); power.append(float(f[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples in the timed region"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "power_w_max": float(max(power)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------- oracle timing
def oracle_step(orc, ocfg, odata, sub, sub_w, sign_add: bool, nthreads: int):
    """One oracle step on a sample: delta lnL of every row, then the update of the accepted rows."""
    orc.delta_loglike(ocfg, odata, sub.params_new, None, sub_w, move_all=orc.ADD, n_bins=sub.n_bins, nthreads=nthreads)
    if sign_add:
        orc.residual_update(ocfg, odata, sub.params_new, None, sub_w, move_all=orc.ADD, accepted=sub.accepted,
                            n_bins=sub.n_bins, nthreads=nthreads)
    else:
        orc.residual_update(ocfg, odata, None, sub.params_new, sub_w, move_all=orc.REMOVE, accepted=sub.accepted,
                            n_bins=sub.n_bins, nthreads=nthreads)


ORACLE_WALKERS = 16          # walkers in every oracle sample: gbo_residual_update parallelises over walkers


def cpu_model() -> str:
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_sample(wl, rows_per_walker: int, rows=None, n_walkers_sample: int = ORACLE_WALKERS):
    """The first rows_per_walker sources of each of the first n_walkers_sample walkers of config 5, with those walkers'
    residuals (host).  Both oracle timings (cpu_baseline and --impl reference) draw their rows this way."""
    n_walkers_sample = min(n_walkers_sample, wl.n_walkers)
    per = wl.B // wl.n_walkers
    rows_per_walker = min(rows_per_walker, per)
    idx = (np.arange(n_walkers_sample)[:, None] * per + np.arange(rows_per_walker)[None, :]).reshape(-1)
    sub = wl.subset(idx)
    resid = np.stack([wl.resid_row(w) if rows is None else rows[w] for w in range(n_walkers_sample)])
    sub_w = sub.walker_index.astype(np.int32)
    psd_map = wl.walker_psd[:n_walkers_sample].astype(np.int32)
    return sub, sub_w, resid, psd_map


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the box's host cores (no GPU)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from gb_inputs import make_workload
    from oracle import gb_oracle as orc
    orc.build()
    cores = orc.max_threads()
    wl = make_workload(5, n_walkers=360, per_walker=12000, B=None)
    sub, sub_w, resid, psd_map = oracle_sample(wl, 2048)
    ocfg = orc.Config()
    odata = orc.Data(resid, wl.psd, wl.k_lo, walker_psd=psd_map)
    for i in range(args.warmup):
        oracle_step(orc, ocfg, odata, sub, sub_w, i % 2 == 0, cores)
    t0 = time.perf_counter()
    for i in range(args.steps):
        oracle_step(orc, ocfg, odata, sub, sub_w, (args.warmup + i) % 2 == 0, cores)
    dt = time.perf_counter() - t0
    value = sub.B * args.steps / dt
    sample = (f"{sub.B} rows per step = the first 2048 sources of each of walkers 0..{ORACLE_WALKERS - 1} of config 5 "
              f"(delta lnL of every row + update of the accepted 25 %); {cpu_model()}")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "evals_per_step": int(sub.B), "note": "bounded sample of the workload"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------- our arm
def run_ours(args):
    import torch
    import torch.distributed as dist

    from gb_inputs import make_workload
    from paper_2405_04690_b200 import gbfit

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the GB hot path has no CPU fallback; use --impl reference "
                         "for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    t_setup = time.perf_counter()
    wl = make_workload(5, n_walkers=args.walkers, per_walker=args.per_walker)
    B = wl.B
    full = (args.walkers == 360 and args.per_walker == 12000)
    ctx = gbfit.Context(local)
    stream = torch.cuda.current_stream(dev)

    # ---- residuals: generated row by row on the host (seeded), uploaded once; they live on the GPU
    d_resid = torch.empty((wl.n_walkers, 2, wl.n_f), dtype=torch.complex128, device=dev)
    n_keep = min(ORACLE_WALKERS, wl.n_walkers)      # host copies of the first rows: the oracle sample's residuals
    keep = {}
    stage = [torch.empty((2, wl.n_f), dtype=torch.complex128).pin_memory() for _ in range(2)]
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as pool:
        for i, row in enumerate(pool.map(wl.resid_row, range(wl.n_walkers))):
            buf = stage[i % 2]
            torch.cuda.current_stream().synchronize()
            buf.numpy()[...] = row
            d_resid[i].copy_(buf, non_blocking=True)
            if i < n_keep:
                keep[i] = row
    torch.cuda.synchronize()
    # the noise weights live on the GPU as 1/S_n (formed once when a PSD row is set; the library
    # takes S_n as well and then divides per bin, see gb_data.psd_is_inverse)
    d_psd = torch.from_numpy(1.0 / wl.psd).to(dev)
    d_wpsd = torch.from_numpy(wl.walker_psd).to(dev)
    data = gbfit.Data(d_resid, d_psd, wl.k_lo, walker_psd=d_wpsd, psd_is_inverse=True)

    # ---- proposals: pinned host copies (e2e) and device copies (kernel-only)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_p, h_w, h_nb, h_acc = pin(wl.params_new), pin(wl.walker_index), pin(wl.n_bins), pin(wl.accepted)
    h_out = torch.empty(B, dtype=torch.float64).pin_memory()
    d_p, d_w, d_nb, d_acc = (x.to(dev) for x in (h_p, h_w, h_nb, h_acc))
    d_out = torch.empty(B, dtype=torch.float64, device=dev)
    setup_s = time.perf_counter() - t_setup

    sum_nb = int(wl.n_bins.astype(np.int64).sum())
    fused = args.update == "fused"
    args.kept_update = args.update == "kept"
    # the seeded 25 % "accepted" flags as uniform draws of the accept step: log u = -inf (accepted whatever delta lnL is)
    # or +inf (rejected), so the decisions of gb_delta_loglike_accept are the workload's flags and cannot flip on a threshold
    h_lu = pin(np.where(wl.accepted != 0, -np.inf, np.inf))
    d_lu = h_lu.to(dev)
    d_accout = torch.zeros(B, dtype=torch.uint8, device=dev)
    h_accout = torch.zeros(B, dtype=torch.uint8).pin_memory()
    # store of the accepted windows: 3 % above what this step's decisions need (the library adds its own reservation slack)
    store_bins = int(1.03 * wl.n_bins[wl.accepted != 0].astype(np.int64).sum()) + 1024

    def step_device(i, ev=None):
        if ev:
            ev[0].record(stream)
        if fused:                    # one call: delta lnL of every row, decision, update by the accepted rows underneath
            add = i % 2 == 0
            ctx.delta_loglike_accept(data, d_p if add else None, None if add else d_p, d_w, d_lu,
                                     move_all=gbfit.ADD if add else gbfit.REMOVE, n_bins=d_nb, store_bins=store_bins, apply=1,
                                     out=d_out, accepted_out=d_accout)
            if ev:
                ev[1].record(stream)
                ev[2].record(stream)
            return
        if (not args.kept_update):   # two independent calls: the update regenerates the accepted waveforms
            ctx.delta_loglike(data, d_p, None, d_w, move_all=gbfit.ADD, n_bins=d_nb, out=d_out)
        else:                        # the sweep pair: every window is kept (42 GB of scratch) and scattered from there
            ctx.delta_loglike_keep(data, d_p, None, d_w, move_all=gbfit.ADD, n_bins=d_nb, sum_n_bins=sum_nb, out=d_out)
        if ev:
            ev[1].record(stream)
        if not (not args.kept_update):
            ctx.residual_update_kept(data, d_acc, negate=(i % 2 == 1))
        elif i % 2 == 0:
            ctx.residual_update(data, d_p, None, d_w, move_all=gbfit.ADD, accepted=d_acc, n_bins=d_nb)
        else:
            ctx.residual_update(data, None, d_p, d_w, move_all=gbfit.REMOVE, accepted=d_acc, n_bins=d_nb)
        if ev:
            ev[2].record(stream)

    def step_host(i):
        if fused:
            add = i % 2 == 0
            ctx.delta_loglike_accept_host(data, h_p if add else None, None if add else h_p, h_w, h_lu,
                                          move_all=gbfit.ADD if add else gbfit.REMOVE, n_bins=h_nb, store_bins=store_bins,
                                          apply=1, out=h_out, accepted_out=h_accout)
            return
        ctx.delta_loglike_host(data, h_p, None, h_w, move_all=gbfit.ADD, n_bins=h_nb, out=h_out)
        if i % 2 == 0:
            ctx.residual_update_host(data, h_p, None, h_w, move_all=gbfit.ADD, accepted=h_acc, n_bins=h_nb)
        else:
            ctx.residual_update_host(data, None, h_p, h_w, move_all=gbfit.REMOVE, accepted=h_acc, n_bins=h_nb)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    K, W = args.steps, args.warmup
    # ---- measured DFMA rate of this device (register-only stream; diagnostic entry point of the library)
    dfma_tflops, dfma_lanes = ctx.measure_fp64_peak(clock_mhz=1965.0)
    # ---- kernel-only arm
    for i in range(W):
        step_device(i)
    ctx.check()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(K)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    clk = ClockSampler(local)
    if rank == 0:
        clk.start()
        time.sleep(0.3)
    barrier()
    l0 = ctx.launch_count()
    tw0 = time.perf_counter()
    e0.record(stream)
    for i in range(K):
        step_device(W + i, evs[i])
    e1.record(stream)
    barrier()
    tw1 = time.perf_counter()
    launches = ctx.launch_count() - l0
    scratch_step = ctx.scratch_bytes()   # device scratch of the context after the timed steps (before any other measurement)
    clocks = clk.stop(tw0, tw1) if rank == 0 else None
    ctx.check()
    ms_total = e0.elapsed_time(e1)
    ms_dlnl = float(np.mean([e[0].elapsed_time(e[1]) for e in evs]))
    ms_upd = float(np.mean([e[1].elapsed_time(e[2]) for e in evs]))
    ms_step = max_over_ranks(ms_total / K, dist if world > 1 else None)
    # (W + K) even => residuals are back to the initial values (to rounding); make it so for the e2e arm
    if (W + K) % 2 == 1:
        step_device(W + K)

    # ---- end-to-end arm (host buffers through the C ABI)
    for i in range(min(W, 3)):
        step_host(i)
    if min(W, 3) % 2 == 1:
        step_host(1)
    barrier()
    h0, h1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    h0.record(stream)
    for i in range(K):
        step_host(i)
    h1.record(stream)
    barrier()
    ms_e2e = max_over_ranks(h0.elapsed_time(h1) / K, dist if world > 1 else None)
    ctx.check()
    if K % 2 == 1:
        step_host(1)                      # residuals back to their initial values (to rounding)
    ctx.delta_loglike(data, d_p, None, d_w, move_all=gbfit.ADD, n_bins=d_nb, out=d_out)   # for the spot parity
    spot_out = d_out[:2048].cpu().numpy()
    sanity = float(h_out.numpy()[:1000].std())
    assert np.isfinite(h_out.numpy()).all() and sanity > 0
    if fused:
        assert np.array_equal(h_accout.numpy() != 0, wl.accepted != 0)
        h2d = h_p.numel() * 8 + h_w.numel() * 4 + h_nb.numel() * 4 + h_lu.numel() * 8
        d2h = h_out.numel() * 8 + h_accout.numel()
    else:
        h2d = 2 * (h_p.numel() * 8 + h_w.numel() * 4 + h_nb.numel() * 4) + h_acc.numel()
        d2h = h_out.numel() * 8

    # ---- the plain delta-lnL call on its own and the two-call form (gb_delta_loglike + gb_residual_update, which
    #      regenerates the accepted waveforms), outside the timed step: what the fused call is compared with
    two_call = None
    if fused:
        p0, p1, p2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        t_d, t_u = [], []
        for i in range(6):
            p0.record(stream)
            ctx.delta_loglike(data, d_p, None, d_w, move_all=gbfit.ADD, n_bins=d_nb, out=d_out)
            p1.record(stream)
            if i % 2 == 0:
                ctx.residual_update(data, d_p, None, d_w, move_all=gbfit.ADD, accepted=d_acc, n_bins=d_nb)
            else:
                ctx.residual_update(data, None, d_p, d_w, move_all=gbfit.REMOVE, accepted=d_acc, n_bins=d_nb)
            p2.record(stream)
            torch.cuda.synchronize()
            if i >= 2:
                t_d.append(p0.elapsed_time(p1))
                t_u.append(p1.elapsed_time(p2))
        ctx.check()
        two_call = {"calls": "gb_delta_loglike + gb_residual_update", "ms_dlnl": float(np.mean(t_d)),
                    "ms_update": float(np.mean(t_u)), "ms_per_step": float(np.mean(t_d) + np.mean(t_u)),
                    "evals_per_s": B / ((np.mean(t_d) + np.mean(t_u)) * 1e-3)}

    # ---- SURVEY 8(f) row f1, outside the timed step: Algorithm 1 (gb_band_sweep) on the same residuals --
    # every odd 256-bin sub-band of 1-4 mHz of every walker, 9 sources and 30 sequential proposals per band
    band = None
    if rank == 0 and full and not args.no_band_sweep:
        from gb_inputs import make_band_tasks
        bt = make_band_tasks(wl, 256, 1e-3, n_bands=183, n_src=9, n_prop=30)
        packed = gbfit.pack_band_tasks(**bt.tasks)
        d_tasks = torch.from_numpy(packed.view(np.uint8)).to(dev)
        d_bp0 = torch.from_numpy(bt.params).to(dev)
        d_bp = d_bp0.clone()
        d_bk, d_bq = torch.from_numpy(bt.prop_k).to(dev), torch.from_numpy(bt.prop_params).to(dev)
        d_lq, d_lu = torch.from_numpy(bt.prop_logq).to(dev), torch.from_numpy(bt.prop_logu).to(dev)
        d_acc_b = torch.zeros(bt.prop_k.size, dtype=torch.uint8, device=dev)
        d_dl_b = torch.zeros(bt.prop_k.size, dtype=torch.float64, device=dev)
        def band_call(tasks_dev):            # every call starts from the same parameters (the reset is inside the timing)
            d_bp.copy_(d_bp0)
            ctx.band_sweep(data, tasks_dev, 256, bt.max_stage, d_bp, d_bk, d_bq, d_lq, d_lu, d_acc_b, d_dl_b)
        ms_band = median_ms(torch, stream, lambda: band_call(d_tasks))
        ctx.check()
        # row f3: the same tasks in the odd/even cold-chain buffer mode: residual rows 2w / 2w+1 stand for
        # the even / odd buffer of "walker" w, r' is formed on chip (9 extra waveforms per task), write-back to the odd row
        wv = bt.tasks["walker"]
        packed_oe = gbfit.pack_band_tasks(**dict(bt.tasks, walker=(wv // 2) * 2), subtract_current=np.ones_like(wv),
                                          write_walker=(wv // 2) * 2 + 1)
        d_tasks_oe = torch.from_numpy(packed_oe.view(np.uint8)).to(dev)
        ms_band_oe = median_ms(torch, stream, lambda: band_call(d_tasks_oe))
        ctx.check()
        # row f1 as printed: the proposal step inside the kernel (Philox, randint, group stretch from a
        # 7.1 M-row friends table, Eq. 14), from the current theta_k
        from gb_inputs import make_stretch_inputs
        si = make_stretch_inputs(bt, n_copies=12, n_friends=24)
        sg = gbfit.Stretch(si.seed, si.sweep, torch.from_numpy(si.group).to(dev), si.n_friends, si.lo, si.hi, si.periodic,
                           si.stretch_a)
        g_box = {}

        def gen_call():
            d_bp.copy_(d_bp0)
            g_box["out"] = ctx.band_sweep_generate(data, d_tasks, 256, bt.max_stage, d_bp, sg, bt.prop_k.size)
        ms_band_gen = median_ms(torch, stream, gen_call)
        ctx.check()
        g_out = g_box["out"]
        gen_eval = float(torch.isfinite(g_out[1]).float().mean().item())
        # waveforms actually generated by a call: one per proposal plus the fill of the current-source cache (n_src per task)
        n_wave_band = bt.prop_k.size + int(bt.tasks["n_src"].sum())
        flops_band = n_wave_band * (711.0 * 256 + 10.0 * 256 * 8) + bt.prop_k.size * 60.0 * 256
        band = {"call": "gb_band_sweep (Algorithm 1)", "N": 256, "tasks": int(len(bt.tasks["walker"])),
                "sources_per_band": 9, "proposals_per_band": 30, "proposals": int(bt.prop_k.size),
                "ms_per_call": ms_band, "proposals_per_s": bt.prop_k.size / (ms_band * 1e-3),
                "accepted_fraction_last_call": float(d_acc_b.float().mean().item()),
                "odd_even_buffers": {"ms_per_call": ms_band_oe, "proposals_per_s": bt.prop_k.size / (ms_band_oe * 1e-3),
                                     "note": "GB_BAND_SUBTRACT_CURRENT | GB_BAND_WRITE_OTHER: residual rows needed per "
                                             "walker 2 instead of n_t (72 rows = 2.2 GB instead of 360 = 10.8 GB here)"},
                "generate": {"call": "gb_band_sweep_generate (proposal step inside the kernel: Philox4x32-10, randint, group "
                                     "stretch from the friends table, Eq. 14, prior box)",
                             "ms_per_call": ms_band_gen, "proposals_per_s": bt.prop_k.size / (ms_band_gen * 1e-3),
                             "friends_table_rows": int(si.group.shape[0]), "n_friends": int(si.n_friends),
                             "evaluated_fraction": gen_eval,
                             "accepted_fraction_last_call": float(g_out[0].float().mean().item())},
                # billed by the waveforms a call really generates (the current-source cache makes it one per proposal plus
                # the fill): n_wave (711 N + 10 N log2 N) + 60 N per proposal
                "waveforms_per_call": n_wave_band,
                "alu_frac": flops_band / (ms_band * 1e-3) / 1e12 / FP64_PEAK_TFLOPS,
                "note": "each proposal = 1 new waveform (the old one comes from the L2-resident cache) + Eq. 5 against the staged "
                        "residual + accept/reject + update; includes the device-side reset of the 38 MB parameter array"}

    # ---- the same sweep as the gb_delta_loglike_keep + gb_residual_update_kept pair (outside the timed step unless
    #      --kept-update): the accepted waveforms are not generated a second time
    pair = None
    if rank == 0 and full and not args.no_band_sweep and not args.kept_update:
        k0, k1, k2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        t_d, t_u = [], []
        for i in range(6):
            k0.record(stream)
            ctx.delta_loglike_keep(data, d_p, None, d_w, move_all=gbfit.ADD, n_bins=d_nb, sum_n_bins=sum_nb, out=d_out)
            k1.record(stream)
            ctx.residual_update_kept(data, d_acc, negate=(i % 2 == 1))
            k2.record(stream)
            torch.cuda.synchronize()
            if i >= 2:
                t_d.append(k0.elapsed_time(k1))
                t_u.append(k1.elapsed_time(k2))
        ctx.check()
        ms_pair = float(np.mean(t_d) + np.mean(t_u))
        pair = {"calls": "gb_delta_loglike_keep + gb_residual_update_kept", "ms_per_step": ms_pair,
                "ms_dlnl_keep": float(np.mean(t_d)), "ms_update_kept": float(np.mean(t_u)),
                "evals_per_s": B / (ms_pair * 1e-3), "scratch_bytes": 32.0 * sum_nb,
                "note": "every window is stored by the delta-lnL epilogue (DRAM is at 5 % under that kernel) and the accepted "
                        "rows are scattered from the store: a memory-bound update instead of a second generation"}

    # ---- BASELINE.json configs 1-4 (parity-test cases; each is <= 1 ms of work): latency of one call ----
    small = None
    if rank == 0 and full and not args.no_band_sweep:
        small = {}
        for cfg in (1, 2, 3, 4):
            w2 = make_workload(cfg)
            if cfg == 1:
                r2 = torch.from_numpy(w2.resid()).to(dev)
                dat2 = gbfit.Data(r2, torch.from_numpy(w2.psd).to(dev), w2.k_lo)
            else:   # same band as the sweep: reuse its first residual rows (the values do not matter for timing)
                nw2 = w2.n_walkers
                dat2 = gbfit.Data(d_resid[:nw2], torch.from_numpy(w2.psd).to(dev), w2.k_lo)
            up = lambda x: None if x is None else torch.from_numpy(np.ascontiguousarray(x)).to(dev)
            a_n, a_o, a_w, a_m, a_nb = up(w2.params_new), up(w2.params_old), up(w2.walker_index), up(w2.move), up(w2.n_bins)
            o2 = torch.empty(w2.B, dtype=torch.float64, device=dev)
            call = lambda: ctx.delta_loglike(dat2, a_n, a_o, a_w, move=a_m, move_all=w2.move_all, N=w2.N, n_bins=a_nb, out=o2)
            for _ in range(5):
                call()
            lc0 = ctx.launch_count()
            call()
            lpc = int(ctx.launch_count() - lc0)
            evs2 = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(20)]
            for e_a, e_b in evs2:
                e_a.record(stream)
                call()
                e_b.record(stream)
            torch.cuda.synchronize()
            ctx.check()
            ms2 = float(np.median([e_a.elapsed_time(e_b) for e_a, e_b in evs2]))
            # the same call captured once into a CUDA graph and replayed: no host launch cost between its kernels
            ms2g = None
            try:
                cs = torch.cuda.Stream(dev)
                cs.wait_stream(stream)
                gr = torch.cuda.CUDAGraph()
                with torch.cuda.graph(gr, stream=cs):
                    call()
                for _ in range(3):
                    gr.replay()
                for e_a, e_b in evs2:
                    e_a.record(stream)
                    gr.replay()
                    e_b.record(stream)
                torch.cuda.synchronize()
                ctx.check()
                ms2g = float(np.median([e_a.elapsed_time(e_b) for e_a, e_b in evs2]))
            except Exception as exc:       # capture refused: report the plain number only
                ms2g = None
                small.setdefault("graph_errors", []).append(f"{w2.name}: {exc}")
            small[w2.name] = {"rows": int(w2.B), "ms_per_call_median": ms2, "evals_per_s": w2.B / (ms2 * 1e-3),
                              "ms_per_graph_replay_median": ms2g,
                              "launches_per_call": lpc}

    # ---- SURVEY 8(f) row f2, outside the timed step: Algorithm 2 (gb_temper_sweep), 10-chain ladders ------
    # every odd 256-bin sub-band of 1-4 mHz, 36 ladders per band on disjoint residuals, 9-10 sources per chain
    tmp = None
    if rank == 0 and full and not args.no_band_sweep:
        from gb_inputs import make_temper_tasks
        tt = make_temper_tasks(wl, 256, 1e-3, n_bands=183, n_t=10, n_src=9, n_groups=36)
        d_tt = torch.from_numpy(gbfit.pack_temper_tasks(**tt.tasks).view(np.uint8)).to(dev)
        # the bench residuals hold no signals, so hardly any exchange would pass Eq. D2: force a seeded quarter of the
        # pairs to be accepted (logu = -inf) so that the holder swap and the atomic residual update are in the timing
        lu = tt.chain_logu.copy()
        lu[np.random.Generator(np.random.Philox(key=[5, 77])).random(lu.size) < 0.25] = -np.inf
        targs = [torch.from_numpy(np.ascontiguousarray(x)).to(dev) for x in
                 (tt.params, tt.chain_walker, tt.chain_beta, tt.chain_set_begin, tt.chain_set_n, lu)]
        t_box = {}

        def temper_call():
            t_box["out"] = ctx.temper_sweep(data, d_tt, 256, tt.max_stage, *targs)
        ms_t = median_ms(torch, stream, temper_call)
        ctx.check()
        t_perm, t_acc, t_dl = t_box["out"]
        n_pairs_t = int((tt.tasks["n_t"] - 1).sum())
        n_wave = int(tt.chain_set_n.sum())          # every chain's set is summed once (set-sum cache of gb_temper.cuh)
        tmp = {"call": "gb_temper_sweep (Algorithm 2, Eq. D2)", "N": 256, "ladders": int(len(tt.tasks["n_t"])), "chains": 10,
               "swap_proposals": n_pairs_t, "waveforms_per_call": n_wave, "ms_per_call": ms_t,
               "swap_proposals_per_s": n_pairs_t / (ms_t * 1e-3), "waveforms_per_s": n_wave / (ms_t * 1e-3),
               "alu_frac": n_wave * (711.0 * 256 + 10.0 * 256 * 8) / (ms_t * 1e-3) / 1e12 / FP64_PEAK_TFLOPS,
               "accepted_fraction_last_call": float(t_acc.float().sum().item()) / n_pairs_t}

    # ---- SURVEY 8(f) row f4, outside the timed step: normalised overlaps of 1 M source pairs (gb_overlap) ----
    ovl = None
    if rank == 0 and full and not args.no_band_sweep:
        n_pairs = 1 << 20
        d_pa = d_p[:n_pairs].contiguous()
        jit = torch.zeros((n_pairs, 8), dtype=torch.float64, device=dev)
        jit[:, 1] = 4e-9
        jit[:, 3] = 0.05
        d_pc = d_pa + jit
        d_rows = (torch.arange(n_pairs, device=dev, dtype=torch.int32) % wl.psd.shape[0]).contiguous()
        d_ov = torch.empty(n_pairs, dtype=torch.float64, device=dev)
        view = gbfit.Data.psd_only(d_psd, wl.k_lo, psd_is_inverse=True)
        nb_pairs = d_nb[:n_pairs].contiguous()
        ms_ov = median_ms(torch, stream, lambda: ctx.overlap(view, d_pa, d_pc, psd_row=d_rows, n_bins=nb_pairs, out=d_ov))
        ctx.check()
        ovl = {"call": "gb_overlap", "pairs": n_pairs, "ms_per_call": ms_ov, "pairs_per_s": n_pairs / (ms_ov * 1e-3),
               "mean_N": float(wl.n_bins[:n_pairs].mean()), "median_overlap": float(d_ov.median().item())}

    # ---- SURVEY 8(f) row f4, second half: the search-stage batch shape of App. G: 900 sub-bands x 10
    #      temperatures x 100 walkers, one source per walker, every row against ONE best-fit residual row
    search = None
    if rank == 0 and full and not args.no_band_sweep:
        from gb_inputs import make_search_stage
        ws = make_search_stage()
        dat_s = gbfit.Data(d_resid[:1], torch.from_numpy(1.0 / ws.psd).to(dev), ws.k_lo, psd_is_inverse=True)
        s_p, s_w, s_nb = (torch.from_numpy(np.ascontiguousarray(x)).to(dev) for x in (ws.params_new, ws.walker_index, ws.n_bins))
        s_out = torch.empty(ws.B, dtype=torch.float64, device=dev)
        ms_s = median_ms(torch, stream, lambda: ctx.delta_loglike(dat_s, s_p, None, s_w, move_all=gbfit.ADD, n_bins=s_nb,
                                                                  out=s_out), reps=5)
        ctx.check()
        fl_s = float(flops_eval(ws.n_bins.astype(np.float64)).sum())
        search = {"call": "gb_delta_loglike, search-stage shape (App. G): 900 sub-bands x 10 temperatures x 100 walkers, one "
                          "source per walker, one residual row", "rows": int(ws.B), "ms_per_call": ms_s,
                  "evals_per_s": ws.B / (ms_s * 1e-3), "mean_N": float(ws.n_bins.mean()),
                  "alu_frac": fl_s / (ms_s * 1e-3) / 1e12 / FP64_PEAK_TFLOPS}

    # ---- roofline of the delta-lnL kernels (the dominant launches) and of the scatter
    nb = wl.n_bins.astype(np.float64)
    flops_dlnl = float(flops_eval(nb).sum())
    bytes_dlnl = float(bytes_eval(nb).sum())
    acc_nb = nb[wl.accepted != 0]
    flops_upd = float((711.0 * acc_nb + 10.0 * acc_nb * np.log2(acc_nb)).sum())
    bytes_upd = float(bytes_scatter(acc_nb).sum())
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    hbm_src = "measured" if "hbm_gbs" in peaks else "fallback"
    ach_tf = flops_dlnl / (ms_dlnl * 1e-3) / 1e12
    traffic_bytes, traffic_src = ncu_traffic(args.update)
    roofline = {
        "bound": "alu", "kernel": ("gb_main_kernel<N,0,1,VAR=1> x {1024,512,256,128} x 8 walker chunks (+ 2 gb_prep_kernel passes, "
                                   "gb_pieces_kernel, closing scatter) of gb_delta_loglike_accept: evaluation, decision and the fused update" if fused else
                                   "gb_main_kernel<N,false,true> x {1024,512,256,128} (+ gb_prep_kernel) of gb_delta_loglike"),
        "achieved": ach_tf, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": ach_tf / FP64_PEAK_TFLOPS,
        "peak_source": "derived: 148 SMs x 64 DFMA/clk x 2 x 1.965 GHz (no FP64 figure in MEASURED_PEAKS.json)",
        "peak_measured_dfma": dfma_tflops, "frac_of_measured_dfma": ach_tf / dfma_tflops if dfma_tflops > 0 else None,
        "dfma_lanes_per_clk_sm_at_1965mhz": dfma_lanes,
        "flops_per_launch": flops_dlnl, "ms_per_launch": ms_dlnl,
        # DRAM bytes (read + write) of the kernels of one step, from the committed ncu --set full capture (full workload
        # only); algorithmic bytes are in "hbm"
        "traffic": traffic_bytes if full else None, "traffic_unit": "DRAM bytes per step", "traffic_source": traffic_src,
        "hbm": {"achieved": bytes_dlnl / (ms_dlnl * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                "frac": bytes_dlnl / (ms_dlnl * 1e-3) / 1e9 / hbm_peak, "peak_source": hbm_src,
                "bytes_per_launch": bytes_dlnl},
        "update": ({"call": "inside the same launches (gb_delta_loglike_accept, apply = 1): accepted windows are stored "
                            "once; the CTAs that evaluate walker chunk c+1 move the windows of chunks <= c into the residual "
                            "(cp.async.bulk + cp.reduce.async.bulk add.f64)",
                    "bytes": 1.5 * bytes_upd, "bytes_note": "32 N written + 32 N read + 64 N read-modify-write per accepted row",
                    "store_bytes": 32.0 * store_bins,
                    "scratch_bytes_ctx": scratch_step,
                    "scratch_note": "gb_scratch_bytes after the timed steps: window store incl. reservation slack, source "
                                    "records (192 B/row), work lists, (beta, logq, logu) rows, accepted-row list, pieces"} if fused else
                   {"call": "gb_residual_update (regenerates the accepted waveforms)", "ms_per_launch": ms_upd,
                    "flops": flops_upd, "bytes": bytes_upd,
                    "alu_frac": flops_upd / (ms_upd * 1e-3) / 1e12 / FP64_PEAK_TFLOPS,
                    "hbm_frac": bytes_upd / (ms_upd * 1e-3) / 1e9 / hbm_peak} if (not args.kept_update) else
                   {"call": "gb_residual_update_kept (scatter of the kept windows; bound hbm)", "ms_per_launch": ms_upd,
                    "bytes": 1.5 * bytes_upd, "bytes_note": "32 N read + 64 N read-modify-write per accepted row",
                    "hbm_frac": 1.5 * bytes_upd / (ms_upd * 1e-3) / 1e9 / hbm_peak,
                    "kept_window_store_bytes_in_dlnl_call": 32.0 * float(nb.sum())}),
        "step_frac": (flops_dlnl + (flops_upd if args.update == "regenerate" else 0.0)) / (ms_step * 1e-3) / 1e12
                     / FP64_PEAK_TFLOPS,
    }
    if fused and two_call is not None:
        tf = flops_dlnl / (two_call["ms_dlnl"] * 1e-3) / 1e12
        roofline["plain_dlnl"] = {"call": "gb_delta_loglike alone (no decision, no update), timed after the step loop",
                                  "ms_per_launch": two_call["ms_dlnl"], "achieved": tf, "frac": tf / FP64_PEAK_TFLOPS,
                                  "frac_of_measured_dfma": tf / dfma_tflops if dfma_tflops > 0 else None}


    # ---- CPU baseline: the oracle on a bounded sample (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import gb_oracle as orc
        orc.build()
        cores = orc.max_threads()
        # a 131 072-source subsample (8192 sources of each of 16 walkers), one untimed warm-up step
        sub, sub_w, resid, psd_map = oracle_sample(wl, 8192, keep, n_keep)
        odata = orc.Data(resid, wl.psd, wl.k_lo, walker_psd=psd_map)
        oracle_step(orc, orc.Config(), odata, sub, sub_w, True, cores)
        t0 = time.perf_counter()
        oracle_step(orc, orc.Config(), odata, sub, sub_w, False, cores)
        dt = time.perf_counter() - t0
        # spot parity of the GPU output on the sample (evaluated after the timed loops, on residuals that
        # differ from the initial ones only by the rounding of the +/- scatter pairs)
        ref = orc.delta_loglike(orc.Config(), orc.Data(np.stack([keep[w] for w in range(n_keep)]), wl.psd, wl.k_lo,
                                                       walker_psd=psd_map),
                                wl.params_new[:2048], None, wl.walker_index[:2048].astype(np.int32), n_bins=wl.n_bins[:2048],
                                nthreads=cores)
        spot = float(np.abs(spot_out - ref).max())
        cpu = {"value": sub.B / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "cpu": cpu_model(),
               "sample": f"{sub.B} rows = the first 8192 sources of each of walkers 0..{n_keep - 1} of the same workload, one "
                         f"step (delta lnL + update of accepted rows) after one warm-up step, {dt:.1f} s wall",
               "spot_parity_max_abs_dlnL_err": spot}

    if rank == 0:
        evals = B * world
        line = {
            "metric": METRIC, "value": evals / (ms_step * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K,
            "warmup": W, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD if full else f"cfg5_reduced_{args.walkers}x{args.per_walker}",
                       "evals_per_step_per_gpu": int(B), "n_residuals": int(wl.n_walkers), "n_f": int(wl.n_f),
                       "accepted_fraction": float(wl.accepted.mean()), "mean_N": float(nb.mean()),
                       "l2": "inputs_exceed_l2 (10.8 GB of residuals, no flush)", "psd_layout": "1/S_n rows (psd_is_inverse=1)",
                       "update": {"fused": "fused (gb_delta_loglike_accept, apply = 1)", "regenerate": "regenerate (gb_delta_loglike + "
                                  "gb_residual_update)", "kept": "kept windows (gb_delta_loglike_keep + gb_residual_update_kept)"}[args.update],
                       "parallelism": f"replicas{world}" if world > 1 else "single_gpu",
                       "ms_dlnl": ms_dlnl, "ms_update": ms_upd, "setup_s": setup_s},
            "e2e": {"value": evals / (ms_e2e * 1e-3), "unit": UNIT, "ms_per_step": ms_e2e,
                    "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h)},
            "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu,
            "two_call_form": two_call, "sweep_pair_kept": pair, "band_sweep": band, "temper_sweep": tmp, "overlap": ovl, "search_stage": search, "small_configs_latency": small,
        }
        print(json.dumps(line), flush=True)
    ctx.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=4)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--walkers", type=int, default=360, help="debug: fewer residuals (default = the full config)")
    ap.add_argument("--per-walker", type=int, default=12000, help="debug: fewer sources per walker")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--update", default="fused", choices=["fused", "regenerate", "kept"],
                    help="the timed step: fused = one gb_delta_loglike_accept call (decision in the epilogue, accepted windows "
                         "kept and scattered underneath the evaluation of the remaining walkers); regenerate = "
                         "gb_delta_loglike + gb_residual_update; kept = gb_delta_loglike_keep + gb_residual_update_kept "
                         "(every window kept in 42 GB of scratch)")
    ap.add_argument("--no-band-sweep", action="store_true", help="skip the Algorithm-1 (gb_band_sweep) measurement")
    args = ap.parse_args(argv)
    args.warmup = max(args.warmup, 3)
    args.steps = max(args.steps, 1)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
