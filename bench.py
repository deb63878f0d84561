#!/usr/bin/env python
"""bench.py — full-arc VMAT dose forward + backward on B200 through the pdrt C ABI.

One "step" is one pass of the whole hot path over the workload: pdrt_dose (S1-S6) followed by
pdrt_dose_backward (S7-S10) for every control point of the arc.  Default workload: BASELINE.json
configs[3] ("c4": synthetic prostate CT 200x200x120 @ 2.5 mm, 178 control points, 80 leaf pairs,
k = 21) — the configuration the headline metric "ms per full-arc dose forward+backward" is quoted on.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c3|c4|c5] [--kernel-size k] [--sweep]
  python bench.py --impl reference ...      # the float64 CPU oracle on a bounded sample (context, not a target)

Prints ONE JSON line (rank 0).  Timing: CUDA events on the launch stream, every timed step preceded by an
L2 flush (a 256 MiB memset, outside the timed events); inputs resident in HBM for `value`, host buffers
and copies inside the timed region for `e2e`.  N > 1 shards control points over ranks (one all-reduce of
the dose grid per forward; gradients are disjoint), strong scaling.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "ms per full-arc dose forward+backward"
FP32_LANES_PER_SM = 128
TRAFFIC_RECORD = os.path.join(ROOT, "profiles", "conv_traffic.json")


def kernel_source_sha():
    """sha256 over the CUDA sources and the C header: identifies the build an ncu capture belongs to."""
    import hashlib
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_2512_18863_b200", "csrc")
    for path in sorted(os.path.join(csrc, f) for f in os.listdir(csrc)) + [os.path.join(ROOT, "include", "pdrt.h")]:
        with open(path, "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def recorded_traffic(workload, kernel_size):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of the dominant kernel, from the tracked ncu record
    (profiles/conv_traffic.json) — only when that record was captured on exactly these kernel sources, else None."""
    try:
        with open(TRAFFIC_RECORD) as f:
            rec = json.load(f)
    except (OSError, ValueError):
        return None
    if rec.get("source_sha") != kernel_source_sha() or rec.get("workload") != workload or rec.get("kernel_size") != kernel_size:
        return None
    return float(rec["dram_bytes"])


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return dict(hbm_gbs=float(p["hbm_gbs"]), sm_max_mhz=float(p.get("sm_max_mhz", 1965.0)), source="measured (MEASURED_PEAKS.json)")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback (B200_PROFILING.md)")


class ClockSampler:
    """Samples SM clock, power and throttle reasons through NVML every 20 ms while the load runs."""

    def __init__(self, index=0):
        self.rows, self.index, self.stop, self.thread, self.mark = [], index, False, None, 0
        self.max_mhz = None

    def __enter__(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            # CUDA_VISIBLE_DEVICES may renumber: take the NVML handle of the torch device by PCI bus id when possible
            try:
                import torch
                bus = torch.cuda.get_device_properties(self.index).pci_bus_id
                h = None
                for i in range(nv.nvmlDeviceGetCount()):
                    hi = nv.nvmlDeviceGetHandleByIndex(i)
                    if nv.nvmlDeviceGetPciInfo(hi).bus == bus:
                        h = hi
                h = h or nv.nvmlDeviceGetHandleByIndex(self.index)
            except Exception:
                h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.nv, self.h = nv, h
            self.max_mhz = float(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            self.thread = threading.Thread(target=self._run, daemon=True)
            self.thread.start()
        except Exception:
            self.thread = None
        return self

    def _run(self):
        nv, h = self.nv, self.h
        while not self.stop:
            try:
                self.rows.append((float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)),
                                  int(nv.nvmlDeviceGetCurrentClocksEventReasons(h)) if hasattr(nv, "nvmlDeviceGetCurrentClocksEventReasons")
                                  else int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)),
                                  nv.nvmlDeviceGetPowerUsage(h) / 1e3))
            except Exception:
                pass
            time.sleep(0.02)

    def wait_first(self, timeout=2.0):
        t0 = time.perf_counter()
        while self.thread and not self.rows and time.perf_counter() - t0 < timeout:
            time.sleep(0.01)
        self.mark = len(self.rows)

    def __exit__(self, *exc):
        self.stop = True
        if self.thread:
            self.thread.join(timeout=2)

    def summary(self):
        rows = self.rows[self.mark:] or self.rows       # samples taken while the GPU was under load
        sm = [r[0] for r in rows]
        bits = 0
        for r in rows:
            bits |= r[1]
        names = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
                 0x80: "hw_power_brake_slowdown"}
        reasons = sorted(n for b, n in names.items() if bits & b)
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=self.max_mhz, reasons=reasons, samples=len(sm),
                    power_w_max=max((r[2] for r in rows), default=None),
                    window="NVML every 20 ms from the first warm-up step to the end of the timed steps (same load throughout)")


def make_workload(name, kernel_size, depth_mode="axis"):
    from paper_2512_18863_b200 import workloads as W
    wl = W.config4(kernel_size or 21) if name == "c4" else W.CONFIGS[name]()
    if kernel_size:
        wl.model["kernel_size"] = kernel_size
    wl.model["depth_mode"] = 1 if depth_mode == "fan" else 0
    return wl


def config_dict(wl, n_gpus, extra=None):
    g, m = wl.grid, wl.model
    c = dict(workload=f"{wl.name}: synthetic prostate CT {g['nx']}x{g['ny']}x{g['nz']} @ {g['sx']} mm, "
                      f"{wl.n_cp} control points, {m['n_pairs']} leaf pairs, fluence {m['flu_nu']}x{m['flu_nv']}, "
                      f"kernel {m['kernel_size']}, forward+backward",
             n_cp=wl.n_cp, kernel_size=m["kernel_size"], seed=wl.seed,
             parallelism=f"control points sharded over {n_gpus} GPU(s)" if n_gpus > 1 else "1 GPU",
             depth_mode="fan (one diverging ray per fluence-map pixel)" if m.get("depth_mode") else "axis (central-axis ray, the paper's mode)",
             l2="256 MiB memset between timed steps (L2 flush); compact D_b/G_b blocks exceed L2")
    if extra:
        c.update(extra)
    return c


# ------------------------------------------------------------------------------------------------ the oracle, timed
ORACLE_SAMPLE_CPS = 16


class OracleSample:
    """The float64 oracle, as it stands, on ONE fixed sample of the workload: ORACLE_SAMPLE_CPS evenly spaced control
    points, forward + backward in one call each.  Both the `cpu_baseline` leg of our arm and `--impl reference` time exactly
    this (kernel table built and one small untimed pass run beforehand), so that the two numbers are the same measurement."""

    def __init__(self, wl):
        from oracle.oracle import Oracle
        from paper_2512_18863_b200 import workloads as W
        self.wl = wl
        self.orc = Oracle(wl.grid, wl.model, wl.density)
        self.n_s = max(1, min(ORACLE_SAMPLE_CPS, wl.n_cp))
        idx = np.linspace(0, wl.n_cp - 1, self.n_s).round().astype(int)
        self.args = (wl.leaves[idx], wl.jaws[idx], wl.gantry_deg[idx], wl.mu[idx])
        self.g = W.seeded_dose_gradient(wl, seed=0)
        self.orc._w_tab()                                   # W_tab once, outside the timed region
        one = tuple(a[:1] for a in self.args)
        self.orc.dose(*one)
        self.orc.dose_backward(*one, self.g)                # page in the buffers

    def time_once(self):
        t0 = time.perf_counter()
        self.orc.dose(*self.args)
        self.orc.dose_backward(*self.args, self.g)
        return time.perf_counter() - t0

    def record(self, seconds):
        wl = self.wl
        return dict(value=seconds * 1e3 * wl.n_cp / self.n_s, unit="ms", cores=self.orc.num_threads(), kind="oracle",
                    sample=f"{self.n_s} of {wl.n_cp} control points (evenly spaced), forward+backward in one call each: "
                           f"{seconds:.2f} s measured, scaled by {wl.n_cp}/{self.n_s}",
                    seconds_measured=seconds)


def run_reference(args):
    """--impl reference: each step is one forward+backward of the oracle sample; value = mean step time scaled to the arc."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = make_workload(args.workload, args.kernel_size)
    smp = OracleSample(wl)
    times = []
    for it in range(args.warmup + args.steps):
        dt = smp.time_once()
        if it >= args.warmup:
            times.append(dt)
    rec = smp.record(float(np.mean(times)))
    ms_full = rec["value"]
    line = dict(impl="reference", metric=METRIC, value=ms_full, unit="ms", n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=ms_full, higher_is_better=False, scaling="strong", vs_baseline=None,
                dtype="f64", data="synthetic", config=config_dict(wl, 1), cpu_baseline=rec,
                e2e=dict(value=ms_full, unit="ms", h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))


def cpu_baseline(wl):
    """The `cpu_baseline` leg of our arm (rank 0, N = 1): the same oracle sample, timed once."""
    smp = OracleSample(wl)
    return smp.record(smp.time_once())


def run_c5_loop(args):
    """--workload c5: BASELINE.json configs[4] — the 20-iteration planning loop on the device (PlanLoop: pdrt_validate,
    pdrt_track_jaws, pdrt_dose, pdrt_objective, pdrt_dose_backward, pdrt_validate_backward, pdrt_plan_step).  A step is one
    loop of 20 iterations from the same initial plan; `value` is the mean time of one forward+backward pair inside the
    loop (the 20 library pairs), the update steps are timed separately."""
    import torch
    from paper_2512_18863_b200 import Engine, PdrtLimits, workloads as W
    from paper_2512_18863_b200.planning import PlanLoop
    n_it = 20
    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)
    peaks = load_peaks()
    wl = make_workload("c5", args.kernel_size)
    eng = Engine(wl.grid, wl.model, wl.density, device=str(dev))
    bits, lam, presc = W.structure_bits(wl)
    limits = PdrtLimits(**W.plan_limits(wl))
    loop = PlanLoop(eng, wl.leaves, wl.mu, wl.gantry_deg, limits, bits, lam, presc, power=2)
    l0, m0 = loop.leaves.clone(), loop.mu.clone()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    E = lambda: torch.cuda.Event(enable_timing=True)

    def one_loop(timed):
        """20 iterations; returns per-iteration (pair, other) event triples when timed."""
        loop.leaves.copy_(l0); loop.mu.copy_(m0)
        evs = []
        for _ in range(n_it):
            a, b, c, d = (E(), E(), E(), E()) if timed else (None,) * 4
            if timed: a.record()
            loop.project()
            if timed: b.record()
            eng.dose(loop.p_leaves, loop.jaws, loop.gantry, loop.p_mu, out=loop.dose)
            eng.objective(loop.dose, loop.bits, loop.lam, loop.presc, loop.power, out=(loop.loss, loop.g))
            eng.dose_backward(loop.p_leaves, loop.jaws, loop.gantry, loop.p_mu, loop.g, out=loop.gh)
            if timed: c.record()
            loop.update()
            if timed: d.record()
            evs.append((a, b, c, d))
        return evs

    clk = ClockSampler(0)
    clk.__enter__()
    clk.wait_first()
    for _ in range(max(1, args.warmup // 3)):
        one_loop(False)
    torch.cuda.synchronize()
    steps = max(1, args.steps // 10)                      # a step is a 20-iteration loop: the default 40 steps become 4 loops
    pair_ms, other_ms, loop_ms = [], [], []
    for _ in range(steps):
        flush.zero_()
        evs = one_loop(True)
        torch.cuda.synchronize()
        pair_ms.append(sum(b.elapsed_time(c) for _, b, c, _ in evs))
        other_ms.append(sum(a.elapsed_time(b) + c.elapsed_time(d) for a, b, c, d in evs))
        loop_ms.append(evs[0][0].elapsed_time(evs[-1][3]))
    loss_first = float(loop.loss[0])
    clk.__exit__(None, None, None)
    # the same loop as ONE CUDA graph of an iteration replayed 20 times (no host work between the calls)
    graph_ms = None
    try:
        loop.leaves.copy_(l0); loop.mu.copy_(m0)
        st = torch.cuda.Stream()
        st.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(st):
            loop.iterate()                                # warm the side stream
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=st):
                loop.iterate()
        torch.cuda.current_stream().wait_stream(st)
        ts = []
        for _ in range(steps):
            loop.leaves.copy_(l0); loop.mu.copy_(m0)
            flush.zero_()
            a, b = E(), E()
            a.record()
            for _ in range(n_it):
                g.replay()
            b.record()
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        graph_ms = float(np.mean(ts))
        assert abs(float(loop.loss[0]) - loss_first) <= 1e-6 * abs(loss_first), "graph replay diverged from the eager loop"
    except Exception as exc:                              # noqa: BLE001 — reported, not fatal
        graph_ms = f"capture failed: {type(exc).__name__}: {exc}"
    # stage breakdown and work counters of one forward+backward of the loop's last plan
    eng.set_profiling(True)
    loop.project()
    eng.dose(loop.p_leaves, loop.jaws, loop.gantry, loop.p_mu, out=loop.dose)
    fw_ms, fw_n = eng.get_stage_ms(); wf = eng.get_work()
    eng.dose_backward(loop.p_leaves, loop.jaws, loop.gantry, loop.p_mu, loop.g, out=loop.gh)
    bw_ms, bw_n = eng.get_stage_ms(); wb = eng.get_work()
    eng.set_profiling(False)
    K = wf.kernel_size
    fp32_peak = eng.info.sm_count * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
    achieved = 2.0 * K * K * wf.support_voxels / (fw_ms["conv"] * 1e-3) / 1e12          # on inputs that can be non-zero (see run_ours)
    on_tiles = 2.0 * K * K * wf.footprint_voxels / (fw_ms["conv"] * 1e-3) / 1e12
    executed = 2.0 * wf.conv_macs / (fw_ms["conv"] * 1e-3) / 1e12
    pair = float(np.mean(pair_ms)) / n_it
    line = dict(metric=METRIC, value=pair, unit="ms", n_gpus=1, steps=steps, warmup=max(1, args.warmup // 3), ms_per_step=float(np.mean(loop_ms)),
                higher_is_better=False, scaling="strong", vs_baseline=None, dtype="f32", data="synthetic",
                config=config_dict(wl, 1, dict(loop=f"{n_it} planning iterations per step on the device (PlanLoop); value = mean forward+backward pair "
                                                    "inside the loop; ms_per_step = the whole loop")),
                loop_ms=float(np.mean(loop_ms)), pairs_ms_per_loop=float(np.mean(pair_ms)), update_ms_per_loop=float(np.mean(other_ms)),
                graph_loop_ms=graph_ms, objective_at_iteration_20=loss_first,
                control_points_per_s=wl.n_cp / (pair * 1e-3), clocks=clk.summary(),
                gpu_launches=(sum(fw_n.values()) + sum(bw_n.values()) + 7) * n_it * steps,
                roofline=dict(bound="alu", kernel=("k_conv<K,false,...>", "k_conv_sym<K,false>", "k_conv_fold<K,false>")[wf.conv_symmetric], achieved=achieved, peak=fp32_peak,
                              unit="TFLOP/s", frac=achieved / fp32_peak, achieved_on_footprint_tiles=on_tiles, frac_on_footprint_tiles=on_tiles / fp32_peak,
                              executed=executed, executed_frac=executed / fp32_peak, traffic=recorded_traffic("c5", K),
                              note="algorithmic flops = 2*k^2*|support|; see the c4 line for the other two counts"),
                stages={k: round(fw_ms[k] + bw_ms[k], 4) for k in fw_ms},
                work=dict(support_voxels=wf.support_voxels, footprint_voxels=wf.footprint_voxels, conv_macs_issued_fwd=wf.conv_macs,
                          conv_macs_issued_bwd=wb.conv_macs))
    if not args.no_cpu_baseline:
        smp = OracleSample(wl)
        rec = smp.record(smp.time_once())
        rec["sample"] += f"; one iteration of the loop (x{n_it} for the loop: {rec['value'] * n_it:.0f} ms)"
        line["cpu_baseline"] = rec
    print(json.dumps(line))


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2512_18863_b200 import Engine, STAGES, workloads as W

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if torch.cuda.device_count() < max(world, 1):
        raise SystemExit(f"bench.py: {world} ranks requested but only {torch.cuda.device_count()} CUDA device(s) visible")
    if world > 1:
        os.environ.setdefault("NCCL_DEBUG", "WARN")
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    dev = torch.device(f"cuda:{local}")
    torch.cuda.set_device(dev)
    peaks = load_peaks()
    wl = make_workload(args.workload, args.kernel_size, args.depth_mode)
    eng = Engine(wl.grid, wl.model, wl.density, device=str(dev))

    # shard control points (contiguous blocks); every rank holds the density, tables and dL/dDose
    from paper_2512_18863_b200.shard import ShardedDose
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    sh = ShardedDose(eng, t(wl.leaves), t(wl.jaws), t(wl.gantry_deg), t(wl.mu), eng.dose_shape, rank, world)
    lo, hi, dose, grads = sh.lo, sh.hi, sh.dose, sh.grads
    lv, jw, ga, mu = sh.leaves, sh.jaws, sh.gantry, sh.mu
    # objective gradient (harness): weights and prescriptions of the quadratic target/OAR objective
    wmask = torch.zeros(eng.dose_shape, dtype=torch.float32, device=dev)
    pmask = torch.zeros_like(wmask)
    for mask, weight, presc in wl.masks.values():
        mt = torch.from_numpy(mask).to(dev)
        wmask[mt] += 2.0 * weight / max(int(mask.sum()), 1)
        if presc:
            pmask[mt] = presc
    if not wl.masks:
        wmask.fill_(1.0 / wmask.numel())

    def forward():
        sh.forward()                           # this rank's control points, then the one all-reduce of the dose grid

    def backward():
        sh.backward(g)

    def objective_grad():
        return wmask * (dose - pmask)

    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    forward()
    g = objective_grad().contiguous()          # fixed dL/dDose for the timed steps
    torch.cuda.synchronize()

    def step():
        forward()
        backward()

    clk = ClockSampler(local)
    clk.__enter__()
    clk.wait_first()
    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()

    # timed region: exactly K steps, per-stage profiling events OFF; every step is preceded by an L2 flush that
    # lies outside its events (a -> c)
    ev = [tuple(torch.cuda.Event(enable_timing=True) for _ in range(3)) for _ in range(args.steps)]
    t_wall0 = time.perf_counter()
    try:
        for a, b, c in ev:
            flush.zero_()                      # L2 flush, outside the timed events
            a.record()
            forward()
            b.record()
            backward()
            c.record()
        torch.cuda.synchronize()
    finally:
        clk.__exit__(None, None, None)
    t_wall = time.perf_counter() - t_wall0
    if world > 1:
        dist.barrier()
    # per-stage breakdown: a few extra steps with the engine's stage events ON (not part of `value`)
    stage_ms = {s: 0.0 for s in STAGES}
    launches_per_step = 0
    n_prof = min(args.steps, 5)
    eng.set_profiling(True)
    for _ in range(n_prof):
        flush.zero_()
        if hi <= lo:
            break
        forward()
        fw_ms, fw_n = eng.get_stage_ms()       # read before the backward call resets them
        backward()
        bw_ms, bw_n = eng.get_stage_ms()
        for s in STAGES:
            stage_ms[s] += (bw_ms[s] + fw_ms[s]) / n_prof
        launches_per_step = sum(bw_n.values()) + sum(fw_n.values())
    eng.set_profiling(False)
    launches = launches_per_step * args.steps
    fwd_ms = float(np.mean([a.elapsed_time(b) for a, b, _ in ev]))
    bwd_ms = float(np.mean([b.elapsed_time(c) for _, b, c in ev]))
    step_ms = float(np.mean([a.elapsed_time(c) for a, _, c in ev]))
    if world > 1:
        tt = torch.tensor([step_ms, fwd_ms, bwd_ms], device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        step_ms, fwd_ms, bwd_ms = [float(v) for v in tt]
    # work counters of the forward and the backward call (device-counted from the actual fluence support)
    if hi <= lo:                               # nothing of this rank's to count
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return
    forward(); wf = eng.get_work()
    backward(); wb = eng.get_work()
    K = wf.kernel_size
    fp32_peak = eng.info.sm_count * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12      # TFLOP/s
    conv_flops = 2.0 * K * K * wf.footprint_voxels                 # algorithmic: k^2 MAC per footprint voxel
    conv_adj_flops = 2.0 * K * K * wb.support_voxels
    stages = {}
    if world == 1:
        nvox = eng.info.nx * eng.info.ny * eng.info.nz
        # algorithmic HBM bytes of the dataflow implemented: Phivol over S_k, D_b over F_k, G_b over F_k,
        # H_b over S_k, each written once and read once; dose written once; dL/dDose read once (L2 after)
        sup, fpr = 4.0 * wf.support_voxels, 4.0 * wf.footprint_voxels
        byts = dict(project=sup, conv=sup + fpr, gather=fpr + 4.0 * nvox,
                    transpose=8.0 * nvox, resample_adj=fpr + 4.0 * nvox, conv_adj=fpr + sup, project_adj=sup)
        for s in STAGES:
            stages[s] = dict(ms=round(stage_ms[s], 4))
            if s in byts and stage_ms[s] > 0:
                gbs = byts[s] / (stage_ms[s] * 1e-3) / 1e9
                stages[s].update(algorithmic_gb=round(byts[s] / 1e9, 4), gbs=round(gbs, 1), hbm_frac=round(gbs / peaks["hbm_gbs"], 4))
        if wf.fan_rays:          # divergent-depth mode: the ray marcher (k_fan_depth) dominates the depth stage
            fan_b = 4.0 * nvox + 4.0 * wf.fan_rays * eng.info.beam_nw          # density read once + depth factors written
            ms_d = stage_ms["depth"] / 2.0                                     # forward and backward both trace the rays
            stages["depth"].update(fan_rays=wf.fan_rays, algorithmic_gb=round(fan_b / 1e9, 4), gbs=round(fan_b / (ms_d * 1e-3) / 1e9, 1),
                                   hbm_frac=round(fan_b / (ms_d * 1e-3) / 1e9 / peaks["hbm_gbs"], 4),
                                   note="k_depth + k_fan_depth, per call; bytes = density once + factors written; at most fan_rays x ray_samples trilinear samples")
        stages["conv"].update(tflops=round(conv_flops / (stage_ms["conv"] * 1e-3) / 1e12, 2) if stage_ms["conv"] > 0 else None,
                              issued_tflops=round(2.0 * wf.conv_macs / (stage_ms["conv"] * 1e-3) / 1e12, 2) if stage_ms["conv"] > 0 else None)
        stages["conv_adj"].update(tflops=round(conv_adj_flops / (stage_ms["conv_adj"] * 1e-3) / 1e12, 2) if stage_ms["conv_adj"] > 0 else None,
                                  issued_tflops=round(2.0 * wb.conv_macs / (stage_ms["conv_adj"] * 1e-3) / 1e12, 2) if stage_ms["conv_adj"] > 0 else None)
    # The dominant kernel is the forward convolution.  Algorithmic flops = 2 k^2 |S|: the multiply-adds of Eq. 8 on inputs that can
    # be non-zero (SURVEY.md 8(d) "algorithmic MAC"; products with structurally zero fluence earn nothing).  The symmetric kernels
    # execute about (k+1)/2k of them (k_conv_sym: each row correlation serves two output rows) or ((k+1)/2k)^2 (k_conv_fold: folded
    # columns as well), the output-stationary one more (zeros in the halo): `executed` is what the kernel counted, and executed / peak is the FMA-pipe share of the launch.
    t_conv = stage_ms["conv"] * 1e-3
    achieved = 2.0 * K * K * wf.support_voxels / t_conv / 1e12 if t_conv > 0 else None
    on_tiles = conv_flops / t_conv / 1e12 if t_conv > 0 else None
    executed = 2.0 * wf.conv_macs / t_conv / 1e12 if t_conv > 0 else None
    kname = ("k_conv<K,false,...>", "k_conv_sym<K,false>", "k_conv_fold<K,false>")[wf.conv_symmetric]
    roofline = dict(bound="alu", kernel=f"{kname} (S4+S5: depth-indexed kernel lookup + lateral convolution)",
                    achieved=achieved, peak=fp32_peak, unit="TFLOP/s", frac=(achieved / fp32_peak) if achieved else None,
                    achieved_on_footprint_tiles=on_tiles, frac_on_footprint_tiles=(on_tiles / fp32_peak) if on_tiles else None,
                    executed=executed, executed_frac=(executed / fp32_peak) if executed else None,
                    traffic=recorded_traffic(wl.name, K),
                    note=f"algorithmic flops = 2*k^2*|support| per launch (products with structurally zero fluence not counted); "
                         f"*_on_footprint_tiles uses 2*k^2*|footprint| (SURVEY.md 8(d): the output-tiled count; a kernel that uses the pencil kernel's "
                         f"symmetry executes a half or a quarter of it, so this can exceed the peak); executed = 2 x the multiply-adds the kernel counted; "
                         f"peak = {eng.info.sm_count} SMs x 128 FP32 lanes x 2 x "
                         f"{peaks['sm_max_mhz']:.0f} MHz (plain FP32 FMA pipe; FFMA microbenchmark on this pool: 72.5 TFLOP/s); "
                         f"HBM fractions of the bandwidth-bound stages are under 'stages' against {peaks['hbm_gbs']} GB/s {peaks['source']}")

    # end to end through the host-buffer C-ABI calls: H2D of parameters and dL/dDose, D2H of dose and gradients
    e2e = None
    if world == 1:
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        h_lv, h_jw, h_ga, h_mu = pin(wl.leaves), pin(wl.jaws), pin(wl.gantry_deg), pin(wl.mu)
        h_dose = torch.empty(eng.dose_shape, dtype=torch.float32).pin_memory()
        h_g = g.cpu().pin_memory()
        h_out = (torch.empty(wl.leaves.shape).pin_memory(), torch.empty(wl.jaws.shape).pin_memory(), torch.empty(wl.mu.shape).pin_memory())
        times = []
        for it in range(args.warmup + args.steps):
            flush.zero_()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            eng.dose_host_async(h_lv, h_jw, h_ga, h_mu, h_dose)      # the dose travels to the host while the backward pass runs
            eng.dose_backward_host(h_lv, h_jw, h_ga, h_mu, h_g, *h_out)
            eng.host_wait()
            dt = time.perf_counter() - t0
            if it >= args.warmup:
                times.append(dt)
        par_b = 4 * (h_lv.numel() + h_jw.numel() + h_ga.numel() + h_mu.numel())
        e2e = dict(value=float(np.mean(times)) * 1e3, unit="ms", h2d_bytes_per_step=int(2 * par_b + 4 * h_g.numel()),
                   d2h_bytes_per_step=int(4 * h_dose.numel() + 4 * sum(o.numel() for o in h_out)),
                   note="pdrt_dose_host_async + pdrt_dose_backward_host + pdrt_host_wait with pinned host buffers (the dose download overlaps "
                        "the backward pass, dL/dDose is given); host wall clock around the three calls")

    sweep = None
    if args.sweep and world == 1:
        sweep = {}
        for k in ([int(x) for x in args.sweep_sizes.split(",")] if args.sweep_sizes else wl.kernel_sizes):
            eng.set_kernel_size(k)
            for _ in range(2):
                step()
            torch.cuda.synchronize()
            ts = []
            for _ in range(max(3, args.steps)):
                flush.zero_()
                a, b, c = (torch.cuda.Event(enable_timing=True) for _ in range(3))
                a.record(); forward(); b.record(); backward(); c.record()
                torch.cuda.synchronize()
                ts.append((a.elapsed_time(b), b.elapsed_time(c)))
            sweep[str(k)] = dict(forward_ms=round(float(np.median([x[0] for x in ts])), 4), backward_ms=round(float(np.median([x[1] for x in ts])), 4),
                                 passes=eng.info.kernel_passes, pass_size=eng.info.kernel_size_compiled)
        eng.set_kernel_size(wl.model["kernel_size"])

    if rank == 0:
        clocks = clk.summary()
        line = dict(metric=METRIC, value=step_ms, unit="ms", n_gpus=world, steps=args.steps, warmup=args.warmup,
                    ms_per_step=step_ms, higher_is_better=False, scaling="strong", vs_baseline=None, dtype="f32",
                    data="synthetic", config=config_dict(wl, world),
                    forward_ms=fwd_ms, backward_ms=bwd_ms, control_points_per_s=wl.n_cp / (step_ms * 1e-3),
                    wall_ms_per_step_incl_flush=t_wall / args.steps * 1e3,
                    clocks=clocks, gpu_launches=launches, e2e=e2e, roofline=roofline, stages=stages,
                    work=dict(support_voxels=wf.support_voxels, footprint_voxels=wf.footprint_voxels, region_voxels=wf.region_voxels,
                              conv_items=wf.conv_items, conv_macs_issued_fwd=wf.conv_macs, conv_macs_issued_bwd=wb.conv_macs,
                              kernel_size_compiled=wf.kernel_size_compiled),
                    paper_context="PAPER.md Table 6: 2.051 s forward / 5.102 s forward+backward, 180 CPs, grid 105x224x224, k=55, NVIDIA A40 (other machine, other workload)")
        if sweep:
            line["kernel_size_sweep"] = sweep
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(wl)
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=("ours", "reference"))
    ap.add_argument("--workload", default="c4", choices=("c3", "c4", "c5"))
    ap.add_argument("--kernel-size", type=int, default=0)
    ap.add_argument("--sweep", action="store_true", help="also time the kernel-size sweep of the workload")
    ap.add_argument("--sweep-sizes", default="", help="comma-separated kernel sizes for --sweep (default: the workload's)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--depth-mode", default="axis", choices=("axis", "fan"), help="fan: one diverging ray per fluence-map pixel (NEXT-1)")
    ap.add_argument("--single-pass", action="store_true", help="c5: time one forward+backward instead of the 20-iteration planning loop")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    env_world = os.environ.get("WORLD_SIZE")
    if env_world is not None and int(env_world) != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but the launcher started WORLD_SIZE={env_world} ranks")
    if args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and env_world is None:
        sys.exit(spawn_ranks(args.gpus))
    elif args.workload == "c5" and args.gpus == 1 and not args.single_pass:
        run_c5_loop(args)
    else:
        run_ours(args)


def spawn_ranks(n):
    """`python bench.py --gpus N` without a launcher: re-exec under torch.distributed.run, one rank per GPU."""
    import socket
    import torch
    if torch.cuda.device_count() < n:
        raise SystemExit(f"bench.py: --gpus {n} but only {torch.cuda.device_count()} CUDA device(s) visible")
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
    return subprocess.call(cmd)


if __name__ == "__main__":
    main()
