#!/usr/bin/env python
"""bench.py -- one JSON line for the batched rigid-body hot path (FK, Jacobian, RNEA, CRBA) on B200.

A "step" is one pass of the whole hot path over one batch of synthetic states: bard_fk, bard_jacobian,
bard_rnea and bard_crba (four kernel launches through the C ABI) on B environments.  One "env-eval" is all
four operators evaluated for one environment.  Default workload: config 3 (23-DOF humanoid) at B = 65 536,
the point of BASELINE.json's sweep (config 4) from which north_star's roofline target applies.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 0..3] [--B n] [--impl ours|reference]

Multi-GPU (N > 1, under torch.distributed.run): the batch axis shards, every rank evaluates its own B
environments with a replicated model and no data-path collective -> "scaling": "weak".

``--impl reference`` times the fp64 CPU oracle (oracle/, test infrastructure) on a bounded sample of the
same workload on the host cores; rank 0 only.
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

from paper_2605_31481_b200 import roofline as RL            # noqa: E402
from paper_2605_31481_b200 import workloads as W            # noqa: E402

OPS = ("fk", "jacobian", "rnea", "crba")
SPEC_OPS = ("fk", "jacobian", "rnea", "crba", "fused")   # "fused": the one-kernel bard_step (built for small robots)
METRIC = "env_evals_per_s (FK + Jacobian + RNEA + CRBA per environment)"
UNIT = "env-evals/s"
L2_BYTES = 126 * 1024 * 1024


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=3, choices=[0, 1, 2, 3])
    ap.add_argument("--B", type=int, default=65536)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--sweep", action="store_true", help="also time every operator over config 4's batch sweep")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-rollout", action="store_true", help="skip the config-2 24-step rollout section")
    ap.add_argument("--no-specialize", action="store_true",
                    help="skip bard_model_specialize: every operator runs its table-driven team kernel")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU work for the oracle baseline")
    return ap.parse_args()


def workload_name(cfg, B):
    return f"config{cfg}:{W.CONFIG_NAMES[cfg]} B={B} (sweep point of config 4)"


# --------------------------------------------------------------------------------------- oracle timing
def time_oracle(desc, cfg, seconds):
    """The fp64 oracle as it stands, all four operators, OpenMP over environments on the host cores, on a
    bounded sample of the workload's states (same seeded distributions).  Returns env-evals/s and details."""
    import oracle
    o = oracle.Oracle(desc)
    cores = os.cpu_count() or 1
    oracle.set_threads(cores)
    used = oracle.get_threads()

    def one_pass(q, qd, qdd):
        t0 = time.perf_counter()
        o.fk(q)
        o.jacobian(q)
        o.rnea(q, qd, qdd)
        o.crba(q)
        return time.perf_counter() - t0

    n = 16384
    q, qd, qdd = (a.astype(np.float64) for a in W.config_states(cfg, n))
    one_pass(q, qd, qdd)                                  # warm pass (page-in, thread pool)
    t = one_pass(q, qd, qdd)
    passes = int(max(3, min(200, np.ceil(seconds / max(t, 1e-6)))))
    t0 = time.perf_counter()
    for _ in range(passes):
        one_pass(q, qd, qdd)
    total = time.perf_counter() - t0
    return {"value": n * passes / total, "unit": UNIT, "cores": used, "kind": "oracle",
            "sample": f"{passes} passes over {n} environments of the workload's seeded state distribution, all four "
                      f"operators, fp64, OpenMP over environments ({total:.1f} s of CPU work)"}, n, total


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    desc = W.config_robot(args.config)
    import oracle
    o = oracle.Oracle(desc)
    oracle.set_threads(os.cpu_count() or 1)
    n = 8192                                             # bounded sample per step
    q, qd, qdd = (a.astype(np.float64) for a in W.config_states(args.config, n))

    def step():
        o.fk(q); o.jacobian(q); o.rnea(q, qd, qdd); o.crba(q)

    steps = min(args.steps, 20)
    warm = min(args.warmup, 3)
    for _ in range(warm):
        step()
    t0 = time.perf_counter()
    for _ in range(steps):
        step()
    dt = time.perf_counter() - t0
    val = n * steps / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": warm, "ms_per_step": 1e3 * dt / steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args.config, args.B),
                   "note": f"oracle timed on a bounded sample of {n} environments per step (host cores)"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.get_threads(), "kind": "oracle",
                         "sample": f"{n} environments per step x {steps} steps"},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------- clocks sampler
class Clocks(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed regions run."""
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, index):
        super().__init__(daemon=True)
        self.samples, self.reasons, self.max_mhz, self.ok = [], set(), None, False
        self._stop_evt = threading.Event()
        self.active = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        while not self._stop_evt.is_set():
            if self.active.is_set():
                try:
                    self.samples.append(float(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
                    r = int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                    for bit, name in self.REASONS.items():
                        if r & bit:
                            self.reasons.add(name)
                except Exception:
                    pass
            time.sleep(0.005)

    def stop(self):
        self._stop_evt.set()

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# --------------------------------------------------------------------------------------- our arm
class BufferSet:
    """One set of device inputs and outputs (SoA, batch last) for B environments."""

    def __init__(self, torch, m, desc, cfg, B, seed_step, dev):
        q, qd, qdd = W.sample_states(desc, B, seed=2000 + cfg + 100 * seed_step)
        self.q, self.qd, self.qdd = (torch.from_numpy(a).to(dev) for a in (q, qd, qdd))
        self.pose = torch.empty((m.nb, 12, B), device=dev)
        self.J = torch.empty((m.nframes, 6, m.nv, B), device=dev)
        self.tau = torch.empty((m.nv, B), device=dev)
        self.M = torch.empty((m.nv, m.nv, B), device=dev)

    def nbytes(self):
        return sum(t.numel() * 4 for t in (self.q, self.qd, self.qdd, self.pose, self.J, self.tau, self.M))


def op_call(m, op, s, B, stream):
    if op == "fk":
        m.fk(B, s.q, s.pose, stream)
    elif op == "jacobian":
        m.jacobian(B, s.q, s.J, stream)
    elif op == "rnea":
        m.rnea(B, s.q, s.qd, s.qdd, s.tau, stream)
    else:
        m.crba(B, s.q, s.M, stream)


def make_sets(torch, m, desc, cfg, B, dev, min_sets=3, cap_bytes=48 << 30):
    first = BufferSet(torch, m, desc, cfg, B, 0, dev)
    per = first.nbytes()
    n = max(min_sets, -(-3 * L2_BYTES // per))           # rotating sets: total >= 3 x L2
    n = max(1, min(n, cap_bytes // per))
    return [first] + [BufferSet(torch, m, desc, cfg, B, i, dev) for i in range(1, n)], per


def time_op_train(torch, m, op, sets, B, stream, launches, warm=5):
    """Average duration of one launch of `op`, back to back over rotating buffer sets, CUDA events on `stream`."""
    for i in range(warm):
        op_call(m, op, sets[i % len(sets)], B, stream)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for i in range(launches):
        op_call(m, op, sets[i % len(sets)], B, stream)
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) * 1e-3 / launches


def time_op_graph(torch, m, op, sets, B, launches=64, replays=10):
    """Same train captured once into a CUDA graph and replayed: device-side time per launch without the host's
    per-call cost (at B = 4096 a launch through ctypes costs more than the kernel)."""
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        for i in range(4):
            op_call(m, op, sets[i % len(sets)], B, side.cuda_stream)
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        for i in range(launches):
            op_call(m, op, sets[i % len(sets)], B, side.cuda_stream)
    g.replay()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(replays):
        g.replay()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) * 1e-3 / (launches * replays)


def rollout_config2(torch, binding, dev, specialize=True, steps=24, dt=0.005, replays=10):
    """BASELINE.json config 2: the 11-DOF spined quadruped, all four operators per simulated RL step (bard_step)
    over 24 consecutive steps, q advanced on the device by explicit Euler (bard_euler_step) from seeded random qdd.
    The 24-step loop is captured once into a CUDA graph and replayed; reported as env-steps/s."""
    desc = W.config_robot(2)
    m = binding.Model(desc, device=dev.index or 0)
    if specialize:
        m.specialize(SPEC_OPS)
    out = {}
    for B in (4096, 65536):
        q, qd, _ = W.sample_states(desc, B, seed=2002)
        q0, qd0 = torch.from_numpy(q).to(dev), torch.from_numpy(qd).to(dev)
        tq, tqd = q0.clone(), qd0.clone()
        qdds = [torch.from_numpy(np.random.default_rng(2002 + 100 * (k + 1)).normal(size=(desc.nv, B)).astype(np.float32)).to(dev)
                for k in range(steps)]
        outs = [torch.empty(sh, device=dev) for sh in ((m.nb, 12, B), (m.nframes, 6, m.nv, B), (m.nv, B), (m.nv, m.nv, B))]

        def loop(stream):
            for k in range(steps):
                m.step(B, tq, tqd, qdds[k], *outs, stream)
                m.euler_step(B, dt, tq, tqd, qdds[k], stream)

        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            loop(side.cuda_stream)                       # warm-up (also loads every kernel before capture)
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        n0 = binding.launch_count()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            loop(side.cuda_stream)
        per_loop = binding.launch_count() - n0
        tq.copy_(q0); tqd.copy_(qd0)
        g.replay()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ms = []
        for _ in range(replays):
            tq.copy_(q0); tqd.copy_(qd0)                 # every replay integrates the same 24 steps
            e0.record()
            g.replay()
            e1.record()
            torch.cuda.synchronize()
            ms.append(e0.elapsed_time(e1))
        med = float(np.median(ms))
        out[f"B{B}"] = {"env_steps_per_s": B * steps / (med * 1e-3), "us_per_step": med * 1e3 / steps,
                        "ms_per_24_steps": med, "launches_per_24_steps": int(per_loop), "finite": bool(torch.isfinite(outs[3]).all())}
    m.close()
    out["note"] = "CUDA graph of 24 x (bard_step + bard_euler_step), dt 0.005, seeded qdd per step, median of 10 replays"
    return out


def op_report(desc, pk, op, sec, B):
    r = RL.roofline(desc, pk)[op]
    if r["bound"] == "hbm":
        ach, peak, unit = r["bytes"] * B / sec / 1e9, pk["hbm_gbs"], "GB/s"
    else:
        ach, peak, unit = r["flop"] * B / sec / 1e12, pk["fp32_tflops"], "TFLOP/s"
    return {"us": sec * 1e6, "env_evals_per_s": B / sec, "bound": r["bound"], "achieved": ach, "peak": peak,
            "unit": unit, "frac": ach / peak, "bytes_per_env": r["bytes"], "flop_per_env": r["flop"],
            "hbm_gbs": r["bytes"] * B / sec / 1e9, "fp32_tflops": r["flop"] * B / sec / 1e12}


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2605_31481_b200 import binding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg, B, K, Wm = args.config, args.B, args.steps, max(args.warmup, 3)
    desc = W.config_robot(cfg)
    m = binding.Model(desc, device=local)
    if not args.no_specialize:
        m.specialize(SPEC_OPS)          # model-specialised (NVRTC) kernels for the operators that have a generator
    pk = RL.measured_peaks(ROOT)
    sets, per_set = make_sets(torch, m, desc, cfg, B, dev)
    R = len(sets)
    stream = torch.cuda.current_stream().cuda_stream
    clocks = Clocks(local)
    clocks.start()

    def step(i, ev=None):
        s = sets[i % R]
        if ev is None:      # the call a user makes: bard_step = all four operators of one batch (one fused kernel or four)
            m.step(B, s.q, s.qd, s.qdd, s.pose, s.J, s.tau, s.M, stream)
            return
        for k, op in enumerate(OPS):
            if ev is not None:
                ev[k].record()
            op_call(m, op, s, B, stream)
        if ev is not None:
            ev[4].record()

    # ---- device-resident timed region: W warm-up steps, then exactly K steps
    for i in range(Wm):
        step(i)
    # The timed region is K uninstrumented steps between two events: an event record between two launches would
    # end the programmatic overlap of a kernel's prologue with the previous kernel's tail (PDL) and time the
    # events themselves.  Per-operator durations come from a second, identical pass of K steps with an event
    # before every launch (below); its step time is reported next to the headline as ms_per_step_instrumented.
    e_beg, e_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    clocks.active.set()
    n0 = binding.launch_count()
    e_beg.record()
    for i in range(K):
        step(i)
    e_end.record()
    barrier()
    clocks.active.clear()
    launches = binding.launch_count() - n0
    elapsed_ms = e_beg.elapsed_time(e_end)
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(K)]
    barrier()
    clocks.active.set()
    for i in range(K):
        step(i, evs[i])
    barrier()
    clocks.active.clear()
    instrumented_ms = evs[0][0].elapsed_time(evs[-1][4])
    t = torch.tensor([elapsed_ms], device=dev, dtype=torch.float64)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    elapsed_ms = float(t.item())
    value = world * B * K / (elapsed_ms * 1e-3)
    op_sec = {op: float(np.mean([evs[i][k].elapsed_time(evs[i][k + 1]) for i in range(K)])) * 1e-3
              for k, op in enumerate(OPS)}
    ops = {op: op_report(desc, pk, op, op_sec[op], B) for op in OPS}
    for op in OPS:
        ops[op]["share_of_step"] = op_sec[op] / sum(op_sec.values())

    # ---- per-operator back-to-back trains (no events between launches), same rotating buffers
    clocks.active.set()
    for op in OPS:
        sec = time_op_train(torch, m, op, sets, B, stream, launches=max(50, min(K, 500)))
        ops[op]["train"] = {k: v for k, v in op_report(desc, pk, op, sec, B).items()
                            if k in ("us", "env_evals_per_s", "achieved", "frac", "hbm_gbs", "fp32_tflops")}
    # ---- the metric's other batch size: every operator at B = 4096 (latency-bound: roofline times <= 2.2 us)
    small = {}
    if B != 4096:
        sets_s, _ = make_sets(torch, m, desc, cfg, 4096, dev, min_sets=8, cap_bytes=4 << 30)
        for op in OPS:
            sec = time_op_train(torch, m, op, sets_s, 4096, stream, launches=200)
            r = op_report(desc, pk, op, sec, 4096)
            small[op] = {k: r[k] for k in ("us", "env_evals_per_s", "bound", "frac")}
            try:
                secg = time_op_graph(torch, m, op, sets_s, 4096)
                rg = op_report(desc, pk, op, secg, 4096)
                small[op]["cuda_graph"] = {k: rg[k] for k in ("us", "env_evals_per_s", "frac")}
            except Exception as ex:                      # graph capture is a convenience of the bench, not of the path
                small[op]["cuda_graph"] = {"error": str(ex)[:120]}
        # the whole step at B = 4096 through bard_step (fused kernel, or the four operators forked over side streams)
        def steps_4096(n):
            for i in range(n):
                x = sets_s[i % len(sets_s)]
                m.step(4096, x.q, x.qd, x.qdd, x.pose, x.J, x.tau, x.M, stream)
        steps_4096(10)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        n0 = binding.launch_count()
        e0.record()
        steps_4096(200)
        e1.record()
        barrier()
        us = e0.elapsed_time(e1) * 1e3 / 200
        small["step"] = {"us": us, "env_evals_per_s": 4096 / (us * 1e-6), "launches_per_step": (binding.launch_count() - n0) / 200,
                         "sum_of_operator_trains_us": sum(small[op]["us"] for op in OPS)}
        del sets_s
    clocks.active.clear()

    # ---- end to end: pinned host inputs -> device, four launches, every output -> pinned host, per step
    s0 = sets[0]
    h_in = [torch.empty(x.shape, dtype=x.dtype, pin_memory=True).copy_(x.cpu()) for x in (s0.q, s0.qd, s0.qdd)]
    d_out = (s0.pose, s0.J, s0.tau, s0.M)
    h_out = [torch.empty(x.shape, dtype=x.dtype, pin_memory=True) for x in d_out]
    h2d = sum(x.numel() * 4 for x in h_in)
    d2h = sum(x.numel() * 4 for x in h_out)
    Ke = max(3, min(K, 20))

    def e2e_step():
        for h, d in zip(h_in, (s0.q, s0.qd, s0.qdd)):
            d.copy_(h, non_blocking=True)
        m.step(B, s0.q, s0.qd, s0.qdd, s0.pose, s0.J, s0.tau, s0.M, stream)
        for h, d in zip(h_out, d_out):
            h.copy_(d, non_blocking=True)
        torch.cuda.current_stream().synchronize()       # the caller reads the results on the host

    for _ in range(2):
        e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(Ke):
        e2e_step()
    barrier()
    te = torch.tensor([time.perf_counter() - t0], device=dev, dtype=torch.float64)
    if world > 1:
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
    e2e = {"value": world * B * Ke / float(te.item()), "unit": UNIT, "h2d_bytes_per_step": h2d,
           "d2h_bytes_per_step": d2h, "steps": Ke,
           "note": "pinned host q/qd/qdd -> device, 4 launches, pose/J/tau/M -> pinned host, every step"}
    clocks.stop()

    dom = max(OPS, key=lambda o: op_sec[o])
    d = ops[dom]
    spec = (not args.no_specialize) and dom in SPEC_OPS
    fused = launches == K
    roof = {"kernel": f"bard_{dom}_n1 (model-specialised)" if spec else f"{dom}_kernel", "bound": d["bound"], "achieved": d["achieved"], "peak": d["peak"],
            "unit": d["unit"], "frac": d["frac"], "traffic": None,
            "peak_source": ("MEASURED_PEAKS.json hbm_gbs" if d["bound"] == "hbm" else
                            "derived: 148 SM x 128 lanes x 2 x sm_max_mhz") + f" ({pk['source']})",
            "algorithmic_per_launch": (d["bytes_per_env"] if d["bound"] == "hbm" else d["flop_per_env"]) * B,
            "avg_launch_us": d["us"],
            "timing": "CUDA events before every launch, second pass of K steps identical to the timed region"}
    tr = os.path.join(ROOT, "profiles", "traffic.json")   # dram bytes per launch from the committed ncu capture
    if os.path.exists(tr):
        try:
            roof["traffic"] = json.load(open(tr)).get(f"config{cfg}_B{B}", {}).get(dom)
        except Exception:
            pass

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": elapsed_ms / K, "ms_per_step_instrumented": instrumented_ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(cfg, B), "envs_per_gpu": B, "global_envs": world * B,
                   "parallelism": f"batch-sharded x{world}, no collective",
                   "l2": f"{R} rotating buffer sets of {per_set / 1e6:.1f} MB (total {R * per_set / 1e6:.0f} MB > L2 126 MB)",
                   "layout": "SoA batch-fastest",
                   "specialized_ops": [] if args.no_specialize else list(SPEC_OPS),
                   "step_call": "bard_step -> one fused kernel" if fused else "bard_step -> bard_fk, bard_jacobian, bard_rnea, bard_crba"},
        "roofline": roof, "ops": ops, "ops_at_B4096": small, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks.summary(),
    }
    if args.sweep and rank == 0:
        line["sweep"] = sweep(torch, binding, pk, dev, stream, specialize=not args.no_specialize)
    if rank == 0 and world == 1 and not args.no_specialize and not args.no_rollout and m.nv > 0:
        # SURVEY 8(f)2, beyond the four operators of the metric: ABA forward dynamics on the same workload (train timing)
        try:
            m.specialize(("aba",))
            ws = torch.empty(m.aba_workspace_floats(B), device=dev)
            qdd_out = torch.empty((m.nv, B), device=dev)

            def aba_train(n):
                for i in range(n):
                    x = sets[i % R]
                    m.aba(B, x.q, x.qd, x.tau, qdd_out, ws, stream)      # tau of the previous operators as the input torque
            aba_train(5)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            aba_train(50)
            e1.record()
            torch.cuda.synchronize()
            us = e0.elapsed_time(e1) * 1e3 / 50
            io = 4 * (m.nq + 3 * m.nv)
            line["aba"] = {"us": us, "env_evals_per_s": B / (us * 1e-6), "io_bytes_per_env": io, "workspace_bytes_per_env": 40 * m.nv,
                           "hbm_gbs_io_plus_workspace": (io + 80 * m.nv) * B / (us * 1e-6) / 1e9,
                           "note": "generated three-pass articulated-body kernel; not part of the headline metric"}
            del ws, qdd_out
        except Exception as ex:
            line["aba"] = {"error": str(ex)[:200]}
    if rank == 0 and world == 1 and not args.no_rollout:
        try:
            line["config2_rollout"] = rollout_config2(torch, binding, dev, specialize=not args.no_specialize)
        except Exception as ex:                          # graph capture is a convenience of the bench, not of the path
            line["config2_rollout"] = {"error": str(ex)[:200]}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cb, _, _ = time_oracle(desc, cfg, args.cpu_seconds)
        line["cpu_baseline"] = cb
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def sweep(torch, binding, pk, dev, stream, specialize=True):
    """config 4: every operator on the humanoid and the chain at B = 1024 ... 1 048 576 (train timing)."""
    out = {}
    for cfg in (3, 0):
        desc = W.config_robot(cfg)
        m = binding.Model(desc, device=dev.index or 0)
        if specialize:
            m.specialize(SPEC_OPS)
        for B in (1024, 4096, 16384, 65536, 262144, 1048576):
            sets, _ = make_sets(torch, m, desc, cfg, B, dev, cap_bytes=40 << 30)
            row = {}
            for op in OPS:
                sec = time_op_train(torch, m, op, sets, B, stream, launches=100)
                r = op_report(desc, pk, op, sec, B)
                row[op] = {k: r[k] for k in ("us", "env_evals_per_s", "bound", "frac", "hbm_gbs", "fp32_tflops")}
            out[f"{W.CONFIG_NAMES[cfg]}_B{B}"] = row
            del sets
            torch.cuda.empty_cache()
        m.close()
    return out


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
