#!/usr/bin/env python
"""bench.py -- throughput of the batched simulation step (drone-steps/s) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--impl ours|reference] [--no-others]

A "step" is one pass of the whole hot path over one batch of synthetic input: for the planning workload (cfg3) that is
cf_set_state(broadcast) + ONE fused cf_step of 100 sub-steps over 2^20 worlds + the per-world minimum-distance
read-out; for the recording workloads it is one cf_step call (1000 / 2000 / 500 sub-steps) writing its record buffer.
One JSON line is printed by rank 0.  Multi-GPU: one process per GPU (torchrun), worlds
sharded by world_offset with no data-path collective (weak scaling: every rank runs the full per-GPU workload).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC, UNIT = "drone_steps_per_sec", "drone-steps/s"
DEFAULT_WORKLOAD = "cfg3"

# Algorithmic FP32 operations per drone-step: every add / sub / mul / div / sqrt /
# trig / log / min / max / clip of the float64 oracle's formulas counts 1 (an FMA is 2); Philox integer work is not
# counted.  Controller ticks are amortised over their period.
ALGO_FLOPS = {"depth": 4096 * 555,      # per frame: 64 x 64 rays x (16 spheres x 14 + 16 boxes x 19 + plane, direction 27)
               "fp_pos": 720, "fp_rotor": 610, "ab_rk4": 330,      # estimates (cfg2's 689 +- the controller ticks; 4 x Eqs. (7)-(10) + RK4 combine)
               "grad": 2120, "mppi": 161, "cfg1": 214, "cfg2": 689, "cfg3": 182, "cfg3b": 138, "cfg4": 87, "cfg5": 744, "cfg5e": 251}
BOUND = {"fp_pos": "alu", "fp_rotor": "alu", "ab_rk4": "alu", "depth": "alu", "grad": "alu", "mppi": "alu", "cfg1": "alu", "cfg2": "alu", "cfg3": "alu", "cfg3b": "alu", "cfg4": "alu", "cfg5": "alu", "cfg5e": "hbm"}
FP32_LANES = 128          # FP32 lanes per SM (sm_100: 4 sub-partitions x 32)


def under_torchrun() -> bool:
    """Launched by torch.distributed.run (also with a single rank): rendezvous variables are in the environment."""
    return all(k in os.environ for k in ("RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT"))


def device_units():
    """(SM count, max SM clock in MHz) of cuda:<LOCAL_RANK> from the driver (NVML through nvidia-smi for the clock, torch
    for the SM count); None where the query fails -- peaks() then says that it fell back to the B200 data-sheet values."""
    sms = mhz = None
    try:
        import torch
        if torch.cuda.is_available():
            sms = int(torch.cuda.get_device_properties(int(os.environ.get("LOCAL_RANK", "0"))).multi_processor_count)
    except Exception:
        pass
    try:
        out = subprocess.run(["nvidia-smi", "--query-gpu=clocks.max.sm", "--format=csv,noheader,nounits", "-i",
                              os.environ.get("LOCAL_RANK", "0")], capture_output=True, text=True, timeout=20).stdout
        mhz = float(out.strip().splitlines()[0])
    except Exception:
        pass
    return sms, mhz


def ncu_static():
    """Per-workload figures of the dominant kernel from the tracked `ncu --set full` captures (profiles/traffic.json, which
    names the commit and command each figure was captured at): DRAM bytes per launch, FMA-pipe utilisation, SASS flop
    fraction, issue-slot utilisation.  STATIC: ncu never runs inside bench.py; they are printed beside the live numbers."""
    try:
        return json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))
    except Exception:
        return {"workloads": {}}


def peaks():
    """Roofline denominators: measured HBM copy bandwidth from MEASURED_PEAKS.json (else the guide's fallback);
    FP32 ALU peak derived from unit counts and the max SM clock: SMs x 128 lanes x 2 flop x f_max, with the SM
    count and f_max read from the device (f_max: MEASURED_PEAKS.json's if it has one)."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    src, hbm, mhz_file = "fallback", 6650.0, None
    if os.path.exists(path):
        try:
            d = json.load(open(path))
            hbm, src = float(d["hbm_gbs"]), "measured"
            mhz_file = float(d["sm_max_mhz"]) if "sm_max_mhz" in d else None
        except Exception:
            pass
    sms_dev, mhz_dev = device_units()
    sms = sms_dev or 148
    mhz = mhz_file or mhz_dev or 1965.0
    units = (f"{sms} SMs ({'device query' if sms_dev else 'B200 data sheet'}) x {FP32_LANES} lanes x 2 x {mhz:.0f} MHz "
             f"({'MEASURED_PEAKS.json' if mhz_file else 'nvidia-smi clocks.max.sm' if mhz_dev else 'B200 data sheet'})")
    return dict(hbm_gbs=hbm, fp32_tflops=sms * FP32_LANES * 2 * mhz * 1e6 / 1e12, sm_max_mhz=mhz, source=src, sm_count=sms,
                alu_peak_source=units)


def algo_bytes_per_launch(wl) -> int:
    """HBM bytes one cf_step launch must move: command loads + recorded states + state / controller / parameter
    planes in and out once."""
    MN = wl.MN
    cmd = (wl.n_cmds * 16 * MN) if wl.params.get("cmd_source", 0) == 0 else wl.n_cmds * 16
    rec = wl.n_records() * wl.D * 4 * MN
    ctrl_planes = {0: 3 + 4 + 4, 1: 4 + (3 if wl.params.get("iface") == 3 else 0)}[wl.model]
    resident = 2 * (wl.D + ctrl_planes) * 4 * MN + (2 * 8 * 4 * MN if wl.params.get("n_obstacles") else 0)
    wparam = (14 if wl.model == 0 else 11) * 4 * wl.M
    plan = (4 + 2 + 1) * 4 * MN if wl.params.get("cost_on") else 0       # eps, cost (running, total), min distance out
    if wl.name == "depth":    # images out, poses in
        sc = wl.notes["scene"]
        return 4 * MN * sc["width"] * sc["height"] + 7 * 4 * MN
    if wl.name == "grad":     # planes in once, history out and back in, commands in, gradient + loss out
        return (wl.D + 7) * 4 * MN + 2 * wl.n_steps * 18 * 4 * MN + 2 * wl.n_cmds * 16 * MN + 4 * MN    # history: 18 floats / step
    return cmd + rec + resident + wparam + plan


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx, self.rows, self._stop, self._t = gpu_index, [], threading.Event(), None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i", str(self.idx)],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([c.strip() for c in out.split(",")])
            except Exception:
                pass
            self._stop.wait(0.1)

    def __enter__(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=6)

    def summary(self):
        sm, mx, reasons = [], 0.0, set()
        for r in self.rows:
            try:
                sm.append(float(r[1])); mx = max(mx, float(r[2]))
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            except Exception:
                continue
        sm.sort()
        return dict(sm_mhz=sm[len(sm) // 2] if sm else None, sm_max_mhz=mx or None, reasons=sorted(reasons), samples=len(sm))


class Runner:
    """One workload resident on one GPU: device-side step() and host-buffer step_e2e()."""

    def __init__(self, name, device, rank=0, e2e=True):
        import numpy as np
        import torch
        from paper_2606_01478_b200 import cf, workloads as W
        self.torch, self.name = torch, name
        self.rank, self.world = rank, int(os.environ.get("WORLD_SIZE", 1))
        host_cmds = name != "cfg3b"
        if name == "depth":
            return self._init_depth(W.make(name), device, cf, e2e)
        wl = W.make(name, **({} if host_cmds else dict(host_cmds=False)))
        self.wl = wl
        prm = dict(wl.params, world_offset=rank * wl.M)          # disjoint global worlds per rank (weak scaling)
        self.sim = cf.Sim(wl.M, wl.N, wl.model, prm, device=device)
        self.sim.reset(wl.seed)
        if wl.cmds is not None:
            self.cmds_host = torch.from_numpy(np.ascontiguousarray(wl.cmds))
            self.cmds = self.cmds_host.to(device)
        else:   # cfg3b: 1.7 GB of clipped Gaussian command sequences, drawn on the device (input generation only)
            g = torch.Generator(device=device).manual_seed(wl.seed)
            n = wl.notes
            self.cmds = torch.empty((wl.n_steps, wl.MN, 4), dtype=torch.float32, device=device)
            for j in range(4):
                z = torch.randn((wl.n_steps, wl.MN), generator=g, device=device)
                self.cmds[..., j] = (n["nominal"][j] + n["sigma"][j] * z).clamp_(n["lo"][j], n["hi"][j])
            self.cmds_host = None
        self.bstate = None if wl.broadcast_state is None else torch.from_numpy(wl.broadcast_state.astype(np.float32)).to(device)
        n_rec = wl.n_records()
        self.record = torch.empty((n_rec, wl.D, wl.MN), dtype=torch.float32, device=device) if n_rec else None
        self.obst = bool(wl.params.get("n_obstacles"))
        self.min_dist = torch.empty(wl.M, dtype=torch.float32, device=device) if self.obst else None
        # broadcast resets are folded into the rollout launch and the N = 1 minimum distance comes from its epilogue
        self.launches_per_step = 1 + (1 if (self.obst and wl.N > 1) else 0)
        self.planner = name == "mppi"
        self.grad = name == "grad"
        if self.grad:         # one cf_grad launch per step; nothing else moves
            self.loss = torch.empty(wl.MN, dtype=torch.float32, device=device)
            self.gout = torch.empty((wl.n_cmds, wl.MN, 4), dtype=torch.float32, device=device)
            self.kernel = "grad_kernel<FP,INTEG_RK4,IF_ATTITUDE,1|2> (forward + backward launch)"
            self.launches_per_step = 2
            self.block, self.grid = 128, -(-wl.MN // 128)
        if self.planner:      # planning iteration: broadcast reset + fused rollout + update (2 kernels per step)
            n = wl.notes
            self.mpar = self.sim.mppi_params(n["horizon"], wl.cmd_hold, n["n_elite"], n["lam"], n["shift"])
            self.launches_per_step = 2
        # host side buffers for the end-to-end path (pinned)
        self.e2e_ok = e2e and self.cmds_host is not None
        self.sequential_e2e = False
        if self.e2e_ok:
            self.cmds_pin = self.cmds_host.pin_memory()
            self.rec_pin = torch.empty((n_rec, wl.D, wl.MN), dtype=torch.float32, pin_memory=True) if n_rec else None
            self.state_pin = torch.empty((wl.D, wl.MN), dtype=torch.float32, pin_memory=True)
            self.md_pin = torch.empty(wl.M, dtype=torch.float32, pin_memory=True) if self.obst else None
            self.bstate_pin = None if self.bstate is None else self.bstate.cpu().pin_memory()
            if self.planner:
                self.plan_pin = torch.empty((wl.notes["horizon"], 4), dtype=torch.float32, pin_memory=True)
                self.info_pin = torch.empty(4 * wl.notes["n_ctrl"] + 4, dtype=torch.float32, pin_memory=True)
            self.h2d = self.cmds_pin.numel() * 4 + (0 if self.bstate is None else self.bstate.numel() * 4)
            self.d2h = (self.rec_pin.numel() * 4 if n_rec else self.state_pin.numel() * 4) + (wl.M * 4 if self.obst else 0)
            if self.grad:
                self.loss_pin = torch.empty(wl.MN, dtype=torch.float32, pin_memory=True)
                self.gout_pin = torch.empty((wl.n_cmds, wl.MN, 4), dtype=torch.float32, pin_memory=True)
                self.h2d = self.cmds_pin.numel() * 4
                self.d2h = self.loss_pin.numel() * 4 + self.gout_pin.numel() * 4
            if self.planner:
                self.h2d = self.bstate.numel() * 4
                self.d2h = self.plan_pin.numel() * 4 + self.info_pin.numel() * 4

    def _init_depth(self, wl, device, cf, e2e):
        """PAPER.md:L71 workload: one cf_depth launch per step renders every environment's 64 x 64 depth image."""
        torch = self.torch
        self.wl, self.planner, self.grad, self.depth = wl, False, False, True
        self.sim = cf.Sim(wl.M, 1, wl.model, wl.params, device=device)
        self.sim.reset(wl.seed)
        sc = wl.notes["scene"]
        self.dp = self.sim.depth_params(**sc)
        self.img = torch.empty((wl.M, sc["height"], sc["width"]), dtype=torch.float32, device=device)
        self.rays = wl.M * sc["height"] * sc["width"]
        self.kernel, self.block, self.grid = "depth_kernel", 256, wl.M * (-(-sc["height"] // 16)) * (-(-sc["width"] // 16))
        self.launches_per_step, self.record, self.obst, self.bstate = 1, None, False, None
        self.e2e_ok = e2e
        if e2e:
            self.img_pin = torch.empty(self.img.shape, dtype=torch.float32, pin_memory=True)
            self.state_pin = self.sim.get_state().cpu().pin_memory()
            self.h2d, self.d2h = self.state_pin.numel() * 4, self.img_pin.numel() * 4

    depth = False

    def describe(self):
        """Kernel name / geometry of the dominant launch (after at least one step: the record mode is part of the name)."""
        if not (self.grad or self.depth):
            self.kernel, self.grid, self.block = self.sim.describe_launch()
        return self.kernel, self.grid, self.block

    def step(self):
        wl, sim = self.wl, self.sim
        if self.depth:
            sim.depth(self.dp, out=self.img)
            return
        if self.planner:
            out = sim.mppi_iterate(self.mpar, self.bstate, self.cmds)
            if self.world > 1 or under_torchrun():      # the planner's one exchange step: all ranks agree on the best controller's plan
                from paper_2606_01478_b200 import planner
                self.global_plan = planner.select_global_plan(sim, self.mpar, out, self.rank)
            return
        if self.grad:
            sim.grad(self.cmds, wl.n_steps, wl.notes["goal"], cmd_hold=wl.cmd_hold, loss=self.loss, grad=self.gout)
            return
        if self.bstate is not None:
            sim.set_state(self.bstate, broadcast=True)
        sim.step(self.cmds, wl.n_steps, cmd_hold=wl.cmd_hold, record_every=wl.record_every, record=self.record)
        if self.obst:
            sim.min_dist(out=self.min_dist)

    def rollout_only(self):
        wl = self.wl
        if self.grad or self.depth:
            return self.step()
        if self.bstate is not None:
            self.sim.set_state(self.bstate, broadcast=True)      # lazy: folded into the rollout launch
        self.sim.step(self.cmds, wl.n_steps, cmd_hold=wl.cmd_hold, record_every=wl.record_every, record=self.record)

    def step_e2e(self):
        """The same step through the C ABI with HOST buffers: H2D of this step's inputs and D2H of its results
        (records, or final state + min distance when nothing is recorded) inside the call."""
        wl, sim = self.wl, self.sim
        if self.depth:        # poses in (the state planes), images out: cf_depth_host
            sim.depth_host(self.dp, self.img_pin, state_host=self.state_pin)
            return
        if self.grad:         # commands in, loss + gradient out: cf_grad_host
            sim.grad_host(self.cmds_pin, wl.n_steps, wl.notes["goal"], self.loss_pin, self.gout_pin, cmd_hold=wl.cmd_hold)
            return
        if self.planner:      # measured state in (52 B), plan + controller scores out; the nominal stays on the device
            sim.mppi_iterate_host(self.mpar, self.bstate_pin, self.cmds, self.plan_pin, self.info_pin)
            return
        if self.rec_pin is None and not self.sequential_e2e and wl.N == 1:
            # fused rollout: ONE C-ABI call, start state + commands in, final state + minimum distance out, the result
            # copies overlapped with the kernel slice by slice (cf_rollout_host)
            sim.rollout_host(self.cmds_pin, wl.n_steps, self.state_pin, cmd_hold=wl.cmd_hold, x0_host=self.bstate_pin,
                             min_dist_host=self.md_pin, n_slices=8)
            return
        if self.bstate_pin is not None:
            self.bstate.copy_(self.bstate_pin, non_blocking=True)
            sim.set_state(self.bstate, broadcast=True)
        sim.step_host(self.cmds_pin, wl.n_steps, cmd_hold=wl.cmd_hold, record_every=wl.record_every, record_host=self.rec_pin)
        if self.rec_pin is None:
            sim.get_state_host(self.state_pin)
        if self.obst:
            sim.min_dist_host(self.md_pin)


def time_steps(fn, torch, steps, warmup, flush, barrier=None):
    """W untimed warm-ups, then exactly K steps, each bracketed by CUDA events on the launching (current) stream,
    with an L2 flush (a write larger than L2) between timed iterations.  Returns per-step ms list."""
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    if barrier:
        barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in ev:
        if flush is not None:
            flush.fill_(1)
        a.record()
        fn()
        b.record()
    torch.cuda.synchronize()
    if barrier:
        barrier()
    return [a.elapsed_time(b) for a, b in ev]


def time_host_steps(fn, torch, steps, warmup):
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    ts = []
    for _ in range(steps):
        t0 = time.perf_counter()
        fn()                       # synchronous: returns after the D2H copy completed
        ts.append((time.perf_counter() - t0) * 1e3)
    return ts


def time_host_steps_pipelined(make_runner, torch, steps, warmup):
    """Two host threads, each with its own simulator, pinned buffers and CUDA stream, call the synchronous host-buffer
    API back to back: while one call's results cross PCIe the other call's kernel runs.  Every step still moves its
    inputs host->device and its results device->host inside the timed region; returns ms per step (wall / total steps)."""
    import threading
    runners, streams = [], []
    for _ in range(2):
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            R = make_runner()
            R.sim.bind_stream(st)
        runners.append(R); streams.append(st)

    def loop(R, st, n):
        with torch.cuda.stream(st):
            for _ in range(n):
                R.step_e2e()

    for R, st in zip(runners, streams):
        loop(R, st, warmup)
    torch.cuda.synchronize()
    th = [threading.Thread(target=loop, args=(R, st, steps)) for R, st in zip(runners, streams)]
    t0 = time.perf_counter()
    for t in th:
        t.start()
    for t in th:
        t.join()
    torch.cuda.synchronize()
    ms = (time.perf_counter() - t0) * 1e3 / (2 * steps)
    del runners
    return ms


def interactive_mode(device):
    """configs[0] in single-step-per-launch mode (north_star "interactive stepping"): 1000 launches of n_steps = 1,
    plain and as replays of one captured CUDA graph.  Returns microseconds per step (host wall clock around a
    synchronised batch: launch latency is the quantity of interest here)."""
    import torch
    from paper_2606_01478_b200 import cf, workloads as W
    wl = W.cfg1()
    out = {}
    sim = cf.Sim(wl.M, wl.N, wl.model, wl.params, device=device)
    sim.reset(wl.seed)
    cm = torch.from_numpy(wl.cmds).to(device)
    rec = torch.empty((1, wl.D, wl.MN), dtype=torch.float32, device=device)
    for _ in range(50):
        sim.step(cm, 1, record_every=1, record=rec)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(1000):
        sim.step(cm, 1, record_every=1, record=rec)
    torch.cuda.synchronize()
    out["launch_us_per_step"] = (time.perf_counter() - t0) * 1e3
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        sim.bind_stream(side)
        sim.step(cm, 1, record_every=1, record=rec)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            for _ in range(10):
                sim.step(cm, 1, record_every=1, record=rec)
    torch.cuda.current_stream().wait_stream(side)
    for _ in range(5):
        graph.replay()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(100):
        graph.replay()
    torch.cuda.synchronize()
    out["graph_us_per_step"] = (time.perf_counter() - t0) * 1e3
    out["note"] = "1000 single-step launches; graph = 10 captured launches per replay x 100 replays"
    sim.bind_stream()
    return out


def oracle_sample(name, target_seconds=12.0, threads=None):
    """Time the float64 oracle, as it stands, on the host cores, on a bounded sample of the same workload: the same
    recipe at a reduced number of worlds / steps (per-drone work is independent of M)."""
    import numpy as np
    from oracle import cfo
    from paper_2606_01478_b200 import workloads as W
    if threads:
        cfo.set_num_threads(threads)
    if name == "mppi":
        return oracle_sample_mppi(target_seconds)
    if name == "grad":
        return oracle_sample_grad(target_seconds)
    if name == "depth":
        return oracle_sample_depth(target_seconds)
    small = dict(cfg1=dict(M=1, n_steps=1000), cfg2=dict(M=64, n_steps=200), cfg3=dict(M=512, n_steps=100),
                 cfg3b=dict(M=512, n_steps=100), cfg4=dict(M=1, N=512, n_steps=100), cfg5=dict(M=64, n_steps=200),
                 cfg5e=dict(M=64, n_steps=200))[name]

    def run(kw):
        wl = W.make(name, **kw)
        sim = cfo.OracleSim(wl.M, wl.N, wl.model, wl.params)
        sim.reset(wl.seed)
        if wl.broadcast_state is not None:
            sim.set_state(wl.broadcast_state, broadcast=True)
        t0 = time.perf_counter()
        sim.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold, record_every=wl.record_every)
        if wl.params.get("n_obstacles"):
            sim.min_dist()
        return wl.drone_steps / (time.perf_counter() - t0), wl

    rate, _ = run(small)                                     # calibration
    kw = dict(small)
    if name != "cfg1":
        scale = max(1.0, rate * target_seconds / (small.get("M", 1) * small.get("N", 1) * small["n_steps"]))
        kw["M"] = int(min(small["M"] * scale, {"cfg4": 256}.get(name, 1 << 22)))
    rate, wl = run(kw)
    sample = f"{wl.M} worlds x {wl.N} drones x {wl.n_steps} steps of {name} (same recipe; a sample of M worlds sized for ~{target_seconds:.0f} s of CPU work)"
    return rate, cfo.num_threads(), sample, wl


def oracle_sample_depth(target_seconds):
    """The numpy depth oracle as it stands on a reduced number of environments (frames per second)."""
    import numpy as np
    from oracle import cfo, depth as odepth
    from paper_2606_01478_b200 import workloads as W

    def run(M):
        wl = W.depth(M=M)
        sim = cfo.OracleSim(wl.M, 1, wl.model, wl.params)
        sim.reset(wl.seed)
        sc = wl.notes["scene"]
        st = sim.get_state()
        t0 = time.perf_counter()
        odepth.render(st, wl.model, sc["width"], sc["height"], sc["fov_x"], spheres=sc["spheres"], boxes=sc["boxes"],
                      ground_plane=sc["ground_plane"], cam_offset=sc["cam_offset"], t_max=sc["t_max"])
        return wl.M / (time.perf_counter() - t0), wl

    rate, wl = run(8)
    rate, wl = run(int(min(1024, max(8, rate * target_seconds))))
    return rate, 1, f"{wl.M} environments x 64 x 64 rays of depth (same scene, fewer environments; numpy, one thread)", wl


def oracle_sample_grad(target_seconds):
    """The gradient oracle as it stands (161 forward runs of the float64 step per batch) on a reduced number of worlds."""
    from oracle import cfo, grad as ograd
    from paper_2606_01478_b200 import workloads as W

    def run(M):
        wl = W.grad(M=M)
        sim = cfo.OracleSim(wl.M, 1, wl.model, wl.params)
        sim.reset(wl.seed)
        t0 = time.perf_counter()
        ograd.value_and_grad(sim, wl.cmds, wl.n_steps, wl.cmd_hold, wl.notes["goal"])
        return wl.drone_steps / (time.perf_counter() - t0), wl

    rate, wl = run(256)
    M = int(min(1 << 20, max(256, rate * target_seconds / wl.n_steps)))
    rate, wl = run(M)
    return rate, cfo.num_threads(), (f"{wl.M} worlds x {wl.n_steps} steps of grad: value and gradient w.r.t. 40 inputs by "
                                     f"Richardson central differences (same recipe, fewer worlds)"), wl


def oracle_sample_mppi(target_seconds):
    """One planning iteration of the oracle (C rollout + numpy update) at a reduced number of rollouts per controller."""
    import numpy as np
    from oracle import cfo, mppi as omppi
    from paper_2606_01478_b200 import workloads as W

    def run(wpc):
        wl = W.mppi(worlds_per_ctrl=wpc)
        p, n = wl.params, wl.notes
        sim = cfo.OracleSim(wl.M, 1, wl.model, p)
        sim.reset(wl.seed)
        t0 = time.perf_counter()
        sim.set_state(wl.broadcast_state, broadcast=True)
        sim.step(wl.cmds, wl.n_steps, cmd_hold=wl.cmd_hold)
        omppi.update(sim.cost().astype(np.float32), wl.cmds, seed=wl.seed, world_offset=0, worlds_per_ctrl=wpc, s_start=0,
                     cmd_hold=wl.cmd_hold, sigma=p["noise_sigma"], beta=p["noise_beta"], lo=p["cmd_lo"], hi=p["cmd_hi"],
                     n_elite=n["n_elite"], lam=n["lam"], shift=n["shift"])
        return wl.drone_steps / (time.perf_counter() - t0), wl

    rate, wl = run(200)
    wpc = int(min(100_000, max(200, rate * target_seconds / (5 * wl.n_steps))))
    rate, wl = run(wpc)
    return rate, cfo.num_threads(), (f"{wl.M} rollouts ({wpc} per controller) x {wl.n_steps} steps of mppi + the update "
                                     f"(same recipe, fewer rollouts)"), wl


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-others", action="store_true", help="skip the secondary workloads and the CPU baseline")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--sweep", action="store_true",
                    help="Fig. 3B shape (PAPER.md:L63): single drone x 2^k worlds, 50 executions of 50 steps each, "
                         "first-principles model + attitude controller, RK4; prints one JSON line with the table")
    ap.add_argument("--sweep-swarm", action="store_true",
                    help="Fig. 3C shape (PAPER.md:L63, L67): worlds x swarm size with the configs[3] recipe (abstracted model, "
                         "position controller, per-world mass), 20 executions of 50 steps each; one JSON line with the table")
    args = ap.parse_args()
    rank, world = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))
    local = int(os.environ.get("LOCAL_RANK", 0))
    name = args.workload

    if args.impl == "reference":
        # the reference arm of this tier IS the oracle, timed on the host cores; rank 0 only
        if rank != 0:
            return 0
        from paper_2606_01478_b200 import workloads as W
        full = W.make(name) if name != "cfg3b" else W.make(name, host_cmds=False)
        rates = []
        for i in range(args.warmup + args.steps):
            # the whole arm stays within a few minutes whatever K is: ~120 s of oracle time shared by the K + W steps
            budget = min(10.0, max(0.15, 120.0 / max(1, args.steps + args.warmup)))
            r, cores, sample, wl = oracle_sample(name, target_seconds=budget)
            if i >= args.warmup:
                rates.append((r, wl.drone_steps))
        tot = sum(d for _, d in rates)
        secs = sum(d / r for r, d in rates)
        value = tot / secs
        line = dict(metric=METRIC, value=value, unit=UNIT, impl="reference", n_gpus=args.gpus, steps=args.steps,
                    warmup=args.warmup, ms_per_step=1e3 * secs / len(rates), higher_is_better=True, scaling="weak",
                    vs_baseline=None, dtype="f64", data="synthetic",
                    config=dict(workload=name, M=wl.M, N=wl.N, sub_steps=wl.n_steps, full_workload_M=full.M,
                                note="bounded sample of the workload per step: M is the sample's (the last step's)"),
                    cpu_baseline=dict(value=value, unit=UNIT, cores=cores, kind="oracle", sample=sample),
                    e2e=dict(value=value, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
        print(json.dumps(line))
        return 0

    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    from paper_2606_01478_b200 import build
    build.build()
    torch.cuda.set_device(local)
    device = f"cuda:{local}"
    barrier = None
    distributed = world > 1 or under_torchrun()      # torchrun with one rank still runs the NCCL init / barrier / reduce path
    if distributed:
        dist.init_process_group("nccl", device_id=torch.device(device))
        barrier = dist.barrier
    pk = peaks()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=device)     # 256 MiB > 126 MB L2

    def measure(nm, steps, warmup, want_e2e):
        R = Runner(nm, device, rank=rank, e2e=want_e2e)
        wl = R.wl
        with ClockSampler(local) as cs:
            ms = time_steps(R.step, torch, steps, warmup, flush, barrier)
        kms = time_steps(R.rollout_only, torch, max(3, min(steps, 10)), 1, flush)     # dominant kernel alone
        t = torch.tensor([sum(ms)], dtype=torch.float64, device=device)
        if distributed:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
        value = world * wl.drone_steps * steps / (total_ms * 1e-3)
        k_ms = sum(kms) / len(kms)
        if BOUND[nm] == "hbm":
            ach = algo_bytes_per_launch(wl) / (k_ms * 1e-3) / 1e9
            roof = dict(bound="hbm", achieved=ach, peak=pk["hbm_gbs"], unit="GB/s", frac=ach / pk["hbm_gbs"], traffic=None,
                        peak_source=pk["source"])
        else:
            ach = ALGO_FLOPS[nm] * wl.drone_steps / (k_ms * 1e-3) / 1e12
            roof = dict(bound="alu", achieved=ach, peak=pk["fp32_tflops"], unit="TFLOP/s", frac=ach / pk["fp32_tflops"],
                        traffic=None, peak_source=pk["alu_peak_source"])
        if nm == "depth":       # the count is dense (every ray x every primitive) while the kernel culls per tile: not work done
            roof["basis"] = ("dense-equivalent: ALGO_FLOPS counts every ray against every primitive; the kernel skips the "
                             "primitives its tile's cone misses, so frac is a speed-up-inclusive figure -- the executed work "
                             "is ncu_static.sass_flop_frac of peak")
        st = ncu_static()
        sw = st.get("workloads", {}).get(nm, {})
        roof["traffic"] = sw.get("dram_bytes")                      # static, from the tracked ncu capture (see ncu_static)
        roof["ncu_static"] = dict(sw, captured_at=st.get("commit"), source="profiles/traffic.json") if sw else None
        R.describe()
        roof.update(kernel=R.kernel, kernel_ms=k_ms, grid=R.grid, block=R.block,
                    hbm_gbs_algorithmic=algo_bytes_per_launch(wl) / (k_ms * 1e-3) / 1e9,
                    algo_flops_per_drone_step=ALGO_FLOPS[nm], algo_bytes_per_launch=algo_bytes_per_launch(wl))
        out = dict(value=value, ms_per_step=total_ms / steps, roofline=roof, clocks=cs.summary(),
                   gpu_launches=R.launches_per_step * steps, M=wl.M, N=wl.N, sub_steps=wl.n_steps,
                   record_every=wl.record_every, drone_steps_per_step=wl.drone_steps)
        if want_e2e and R.e2e_ok:
            ems = time_host_steps(R.step_e2e, torch, max(3, min(steps, 10)), 2)
            et = torch.tensor([sum(ems) / len(ems)], dtype=torch.float64, device=device)
            if distributed:
                dist.all_reduce(et, op=dist.ReduceOp.MAX)
            out["e2e"] = dict(value=world * wl.drone_steps / (float(et.item()) * 1e-3), unit=UNIT,
                              h2d_bytes_per_step=R.h2d, d2h_bytes_per_step=R.d2h, ms_per_step=float(et.item()))
            if not (R.grad or R.depth or R.planner) and R.rec_pin is None and wl.N == 1:
                R.sequential_e2e = True          # the same through cf_step_host + cf_get_state_host + cf_get_aux_host
                sms = time_host_steps(R.step_e2e, torch, max(3, min(steps, 10)), 2)
                R.sequential_e2e = False
                out["e2e"]["sequential_calls"] = dict(value=wl.drone_steps / (sum(sms) / len(sms) * 1e-3),
                                                      ms_per_step=sum(sms) / len(sms),
                                                      note="cf_step_host, cf_get_state_host, cf_get_aux_host one after the "
                                                           "other (no overlap); value above is cf_rollout_host")
            if world == 1 and nm in ("cfg3", "mppi", "depth"):      # double-buffered host loop (two calls in flight)
                pms = time_host_steps_pipelined(lambda: Runner(nm, device, rank=rank, e2e=True), torch, 10, 2)
                out["e2e"]["pipelined"] = dict(value=wl.drone_steps / (pms * 1e-3), ms_per_step=pms,
                                               note="two host threads, each with its own simulator and stream, same "
                                                    "synchronous host-buffer calls; value above is the single-call figure")
        del R
        torch.cuda.empty_cache()
        return out

    if args.sweep:
        from paper_2606_01478_b200 import cf, workloads as W
        import numpy as np
        rows = []
        for k in range(0, 21, 2):
            wl = W.cfg2(M=1 << k, n_steps=50)
            sim = cf.Sim(wl.M, 1, wl.model, wl.params, device=device)
            sim.reset(wl.seed)
            cm = torch.from_numpy(np.ascontiguousarray(wl.cmds)).to(device)
            ms = time_steps(lambda: sim.step(cm, 50, cmd_hold=wl.cmd_hold), torch, 50, 3, None)
            mean, sd = float(np.mean(ms)), float(np.std(ms))
            rows.append(dict(worlds=wl.M, ms_per_50_steps=mean, sigma_ms=sd, drone_steps_per_sec=wl.M * 50 / (mean * 1e-3)))
            del sim
        if rank == 0:
            print(json.dumps(dict(sweep="FP + attitude controller, RK4 1 kHz, 50 executions x 50 steps (PAPER.md:L63 protocol), "
                                        "state resident, no L2 flush (the paper's loop re-runs the same buffers)", rows=rows)))
        return 0
    if args.sweep_swarm:
        from paper_2606_01478_b200 import cf, workloads as W
        import numpy as np
        rows = []
        for M in (1, 16, 256, 1000, 4096):
            for N in (1, 16, 256, 4000):
                wl = W.cfg4(M=M, N=N, n_steps=50)
                sim = cf.Sim(wl.M, wl.N, wl.model, wl.params, device=device)
                sim.reset(wl.seed)
                cm = torch.from_numpy(np.ascontiguousarray(wl.cmds)).to(device)
                ms = time_steps(lambda: sim.step(cm, 50, cmd_hold=wl.cmd_hold), torch, 20, 3, None)
                mean, sd = float(np.mean(ms)), float(np.std(ms))
                rows.append(dict(worlds=M, drones_per_world=N, drones=M * N, ms_per_50_steps=mean, sigma_ms=sd,
                                 drone_steps_per_sec=M * N * 50 / (mean * 1e-3), world_steps_per_sec=M * 50 / (mean * 1e-3)))
                del sim, cm
                torch.cuda.empty_cache()
        if rank == 0:
            print(json.dumps(dict(sweep_swarm="AB model + position controller 100 Hz, Euler 500 Hz, per-world mass (configs[3] recipe), "
                                              "20 executions x 50 steps, state resident, no record, no L2 flush", rows=rows)))
        return 0
    main_res = measure(name, args.steps, args.warmup, not args.no_e2e)
    others = {}
    if not args.no_others and world == 1:
        for nm in ("depth", "grad", "mppi", "cfg1", "cfg2", "cfg3", "cfg3b", "cfg4", "cfg5", "cfg5e"):
            if nm == name:
                continue
            r = measure(nm, 5, 3, False)
            others[nm] = dict(value=r["value"], ms_per_step=r["ms_per_step"], roofline=r["roofline"], M=r["M"], N=r["N"],
                              sub_steps=r["sub_steps"], record_every=r["record_every"])
    if "cfg1" in others:
        others["cfg1"]["interactive"] = interactive_mode(device)
    cpu = None
    if rank == 0 and world == 1 and not args.no_others:
        rate, cores, sample, _ = oracle_sample(name)
        cpu = dict(value=rate, unit=UNIT, cores=cores, kind="oracle", sample=sample)
    if rank == 0:
        line = dict(metric=METRIC, value=main_res["value"], unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
                    ms_per_step=main_res["ms_per_step"], higher_is_better=True, scaling="weak", vs_baseline=None,
                    dtype="f32", data="synthetic",
                    config=dict(workload=name, M_per_gpu=main_res["M"], N=main_res["N"], sub_steps_per_step=main_res["sub_steps"],
                                record_every=main_res["record_every"], drone_steps_per_step_per_gpu=main_res["drone_steps_per_step"],
                                l2="flushed between timed steps (256 MiB write)", parallelism=f"worlds sharded x{world}, no collective"),
                    roofline=main_res["roofline"], cpu_baseline=cpu, e2e=main_res.get("e2e"), clocks=main_res["clocks"],
                    gpu_launches=main_res["gpu_launches"], workloads=others)
        if name == "grad":      # the paper's unit for Fig. 3D: one gradient = dL/d(all commands) of one world through n steps
            line["config"]["world_gradients_per_sec"] = main_res["value"] / main_res["sub_steps"]
        if name == "depth":     # the paper's unit: frames per second; a "drone-step" here is one frame
            line["metric"], line["unit"] = "depth_frames_per_sec", "frames/s"
            if line.get("e2e"):
                line["e2e"]["unit"] = "frames/s"
            line["config"]["rays_per_sec"] = main_res["value"] * 4096
        if name == "mppi":      # plans per second (the paper's requirement: 50 Hz)
            line["config"]["plans_per_sec"] = 1e3 / main_res["ms_per_step"]
        print(json.dumps(line))
    if distributed:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
