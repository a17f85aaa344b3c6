#!/usr/bin/env python
"""bench.py -- one JSON line for the batched rigid-body hot path (FK, Jacobian, RNEA, CRBA) on B200.

A "step" is one pass of the whole hot path over one batch of synthetic states: ``bard_step`` = bard_fk, bard_jacobian,
bard_rnea and bard_crba of one (q, qd, qdd) batch through the C ABI.  One "env-eval" is all four operators evaluated
for one environment.  Headline workload: config 3 (23-DOF humanoid) at B = 65 536, the point of BASELINE.json's sweep
(config 4) from which north_star's roofline target applies.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 0..3] [--B n] [--impl ours|reference] [--quick]

Besides the headline the default run (rank 0, one GPU) reports, compactly:
  * ``matrix``: every operator and bard_step on configs 0-3 at B = 4096 and 65 536 (BASELINE.json's metric);
  * ``sweep``: BASELINE.json config 4 -- humanoid and chain-7 at B = 1024 ... 1 048 576: env-evals/s, achieved HBM GB/s
    and FP32 TFLOP/s against the B200 peaks, and the oracle's time on the host cores per B;
  * ``aba`` and ``rnea_vjp`` (generated kernels, each with its roofline; the VJP also table-driven), ``variants``
    (fp64 / AoS), ``config2_rollout``, ``specialize_s``.
Per-operator times are device times of a back-to-back train of launches over rotating buffer sets (> L2 in total)
replayed from a CUDA graph, so that a kernel shorter than the host's launch rate is timed as a kernel.

Multi-GPU (N > 1, under torch.distributed.run): the batch axis shards, every rank evaluates its own B environments with
a replicated model and no data-path collective -> "scaling": "weak"; headline and e2e only.

``--impl reference`` times the fp64 CPU oracle (oracle/, test infrastructure) on a bounded sample of the same workload on
the host cores; rank 0 only.
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

from paper_2605_31481_b200 import dist as D                 # noqa: E402
from paper_2605_31481_b200 import roofline as RL            # noqa: E402
from paper_2605_31481_b200 import workloads as W            # noqa: E402

OPS = ("fk", "jacobian", "rnea", "crba")
SPEC_OPS = ("fk", "jacobian", "rnea", "crba", "fused")   # "fused": the one-kernel forms of bard_step
METRIC = "env_evals_per_s (FK + Jacobian + RNEA + CRBA per environment)"
UNIT = "env-evals/s"
L2_BYTES = 126 * 1024 * 1024
SWEEP_B = (1024, 4096, 16384, 65536, 262144, 1048576)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=3, choices=[0, 1, 2, 3])
    ap.add_argument("--B", type=int, default=65536)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--quick", action="store_true", help="headline, e2e and cpu_baseline only (no matrix / sweep / extras)")
    ap.add_argument("--no-sweep", action="store_true", help="skip BASELINE config 4's batch sweep")
    ap.add_argument("--no-matrix", action="store_true", help="skip configs 0-3 x B in {4096, 65536}")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-rollout", action="store_true", help="skip the config-2 24-step rollout section")
    ap.add_argument("--no-specialize", action="store_true",
                    help="skip bard_model_specialize: every operator runs its table-driven team kernel")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU work for the oracle baseline")
    ap.add_argument("--only", default=None, choices=list(OPS) + ["step", "kin", "aba", "vjp"],
                    help="profiling aid: a short train of ONE operator on --config / --B (rotating buffer sets), then exit")
    ap.add_argument("--option", action="append", default=[], metavar="KEY=VALUE", help="bard_model_set_option before specialising (repeatable)")
    return ap.parse_args()


def workload_name(cfg, B):
    return f"config{cfg}:{W.CONFIG_NAMES[cfg]} B={B} (sweep point of config 4)"


def sig(x, n=4):
    """Round to n significant digits (keeps the JSON line compact)."""
    if x is None or isinstance(x, (str, bool, int)):
        return x
    if isinstance(x, dict):
        return {k: sig(v, n) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [sig(v, n) for v in x]
    x = float(x)
    return x if x == 0 or not np.isfinite(x) else float(f"{x:.{n}g}")


# --------------------------------------------------------------------------------------- oracle timing
def oracle_pass_seconds(o, q, qd, qdd):
    t0 = time.perf_counter()
    o.fk(q)
    o.jacobian(q)
    o.rnea(q, qd, qdd)
    o.crba(q)
    return time.perf_counter() - t0


def time_oracle(desc, cfg, seconds):
    """The fp64 oracle as it stands, all four operators, OpenMP over environments on the host cores, on a bounded sample
    of the workload's states (same seeded distributions).  Returns the cpu_baseline object."""
    import oracle
    o = oracle.Oracle(desc)
    cores = os.cpu_count() or 1
    oracle.set_threads(cores)
    used = oracle.get_threads()
    n = 16384
    q, qd, qdd = (a.astype(np.float64) for a in W.config_states(cfg, n))
    oracle_pass_seconds(o, q, qd, qdd)                    # warm pass (page-in, thread pool)
    t = oracle_pass_seconds(o, q, qd, qdd)
    passes = int(max(3, min(200, np.ceil(seconds / max(t, 1e-6)))))
    t0 = time.perf_counter()
    for _ in range(passes):
        oracle_pass_seconds(o, q, qd, qdd)
    total = time.perf_counter() - t0
    return {"value": n * passes / total, "unit": UNIT, "cores": used, "kind": "oracle",
            "sample": f"{passes} passes over {n} environments of the workload's seeded state distribution, all four "
                      f"operators, fp64, OpenMP over environments ({total:.1f} s of CPU work)"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    desc = W.config_robot(args.config)
    import oracle
    o = oracle.Oracle(desc)
    oracle.set_threads(os.cpu_count() or 1)
    steps, warm = max(1, args.steps), max(0, args.warmup)
    # a bounded sample of the workload per step, sized so that the whole run stays within about a minute of CPU work
    n = int(min(8192, max(256, 8192 * 1500 // max(1, steps + warm))))
    q, qd, qdd = (a.astype(np.float64) for a in W.config_states(args.config, n))
    for _ in range(warm):
        oracle_pass_seconds(o, q, qd, qdd)
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle_pass_seconds(o, q, qd, qdd)
    dt = time.perf_counter() - t0
    val = n * steps / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": warm, "ms_per_step": 1e3 * dt / steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args.config, args.B)},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.get_threads(), "kind": "oracle",
                         "sample": f"the fp64 oracle on the host cores, a bounded sample of {n} environments of the workload per step x {steps} steps"},
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

    def __init__(self, torch, m, ins, shift, dev):
        # the first set holds the seeded states; the others are the same states rolled along the batch axis on the
        # device (same distribution, other addresses and another environment per lane) -- no host RNG per set
        self.q, self.qd, self.qdd = (t if shift == 0 else torch.roll(t, shifts=shift, dims=1) for t in ins)
        B = self.q.shape[1]
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
    elif op == "crba":
        m.crba(B, s.q, s.M, stream)
    elif op == "kin":
        m.kinematics(B, s.q, s.pose, s.J, s.M, stream)
    else:
        m.step(B, s.q, s.qd, s.qdd, s.pose, s.J, s.tau, s.M, stream)


def make_sets(torch, m, desc, cfg, B, dev, min_sets=3, cap_bytes=48 << 30):
    ins = [torch.from_numpy(a).to(dev) for a in W.sample_states(desc, B, seed=2000 + cfg)]
    first = BufferSet(torch, m, ins, 0, dev)
    per = first.nbytes()
    n = max(min_sets, -(-3 * L2_BYTES // per))           # rotating sets: total >= 3 x L2
    n = max(1, min(n, cap_bytes // per, 64))
    return [first] + [BufferSet(torch, m, ins, 17 + 31 * i, dev) for i in range(1, n)], per


def time_graph(torch, m, op, sets, B, launches=None, replays=None):
    """Device time per launch of a back-to-back train of `op` over the rotating buffer sets, captured once into a CUDA
    graph and replayed (no host launch cost inside the timed region): (seconds per launch, launches per replay)."""
    if launches is None:
        launches = max(len(sets), 64 if B <= 65536 else 2 * len(sets))
    if replays is None:
        replays = 10 if B <= 65536 else 4
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        for i in range(min(4, launches)):
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


def time_train(torch, m, op, sets, B, stream, launches, warm=5):
    """Same train through plain host launches (one ctypes call each), CUDA events on `stream`."""
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


def op_report(desc, pk, op, sec, B):
    r = RL.roofline(desc, pk)[op]
    if r["bound"] == "hbm":
        ach, peak, unit = r["bytes"] * B / sec / 1e9, pk["hbm_gbs"], "GB/s"
    else:
        ach, peak, unit = r["flop"] * B / sec / 1e12, pk["fp32_tflops"], "TFLOP/s"
    return {"us": sec * 1e6, "env_evals_per_s": B / sec, "bound": r["bound"], "achieved": ach, "peak": peak,
            "unit": unit, "frac": ach / peak, "bytes_per_env": r["bytes"], "flop_per_env": r["flop"],
            "hbm_gbs": r["bytes"] * B / sec / 1e9, "fp32_tflops": r["flop"] * B / sec / 1e12}


def short(r, keys=("us", "env_evals_per_s", "bound", "frac", "hbm_gbs", "fp32_tflops")):
    return {k: r[k] for k in keys}


def rollout_config2(torch, binding, m, desc, dev, steps=24, dt=0.005, replays=10):
    """BASELINE.json config 2: the 11-DOF spined quadruped, all four operators per simulated RL step (bard_step)
    over 24 consecutive steps, q advanced on the device by explicit Euler from seeded random qdd.  The 24-step loop is
    captured once into a CUDA graph and replayed; reported as env-steps/s.  Two forms: `serial` = bard_step then the
    in-place bard_euler_step on one stream (each step waits for the integrator and the integrator for the step);
    `pipelined` = the out-of-place bard_euler_step_to on a second stream over three rotating state buffers: the next state
    depends on (q, qd, qdd) only, so the integrator runs beside the operators of its own step and leaves the critical path."""
    out = {}
    for B in (4096, 65536):
        q, qd, _ = W.sample_states(desc, B, seed=2002)
        q0, qd0 = torch.from_numpy(q).to(dev), torch.from_numpy(qd).to(dev)
        gen = torch.Generator(device=dev)
        gen.manual_seed(2002)
        qdds = [torch.randn((desc.nv, B), device=dev, generator=gen) for _ in range(steps)]
        outs = [torch.empty(sh, device=dev) for sh in ((m.nb, 12, B), (m.nframes, 6, m.nv, B), (m.nv, B), (m.nv, m.nv, B))]
        tq = [q0.clone() for _ in range(3)]
        tqd = [qd0.clone() for _ in range(3)]
        side, eul = torch.cuda.Stream(), torch.cuda.Stream()

        def serial():
            for k in range(steps):
                m.step(B, tq[0], tqd[0], qdds[k], *outs, side.cuda_stream)
                m.euler_step(B, dt, tq[0], tqd[0], qdds[k], side.cuda_stream)

        def pipelined():
            start = torch.cuda.Event()
            start.record(side)
            eul.wait_event(start)
            step_done, euler_done = [], []
            for k in range(steps):
                s, n = k % 3, (k + 1) % 3
                if k > 0:
                    side.wait_event(euler_done[k - 1])           # (q_k, qd_k) is ready
                m.step(B, tq[s], tqd[s], qdds[k], *outs, side.cuda_stream)
                ev = torch.cuda.Event()
                ev.record(side)
                step_done.append(ev)
                if k >= 2:
                    eul.wait_event(step_done[k - 2])             # buffer n held the state of step k - 2: its operators are done
                m.euler_step_to(B, dt, tq[s], tqd[s], qdds[k], tq[n], tqd[n], eul.cuda_stream)
                ev = torch.cuda.Event()
                ev.record(eul)
                euler_done.append(ev)
            side.wait_event(euler_done[-1])

        res = {}
        for name, loop in (("serial", serial), ("pipelined", pipelined)):
            side.wait_stream(torch.cuda.current_stream())
            eul.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                loop()                                       # warm-up (also loads every kernel before capture)
            torch.cuda.synchronize()
            n0 = binding.launch_count()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=side):
                loop()
            per_loop = binding.launch_count() - n0
            tq[0].copy_(q0); tqd[0].copy_(qd0)
            g.replay()
            torch.cuda.synchronize()
            final = (tq[steps % 3] if name == "pipelined" else tq[0]).clone()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ms = []
            for _ in range(replays):
                tq[0].copy_(q0); tqd[0].copy_(qd0)           # every replay integrates the same 24 steps
                e0.record()
                g.replay()
                e1.record()
                torch.cuda.synchronize()
                ms.append(e0.elapsed_time(e1))
            med = float(np.median(ms))
            res[name] = {"env_steps_per_s": B * steps / (med * 1e-3), "us_per_step": med * 1e3 / steps, "launches_per_24_steps": int(per_loop),
                         "finite": bool(torch.isfinite(outs[3]).all()), "_final": final}
        same = bool(torch.equal(res["serial"].pop("_final"), res["pipelined"].pop("_final")))
        out[f"B{B}"] = dict(res["serial"], pipelined=dict(res["pipelined"], same_final_state_as_serial=same))
    out["note"] = ("CUDA graph of 24 x (bard_step + Euler step), dt 0.005, seeded qdd per step, median of 10 replays; pipelined = "
                   "bard_euler_step_to on a second stream over three rotating state buffers")
    return out


def run_only(args):
    """`--only op`: what the ncu captures under profiles/ run -- `--steps` launches of one operator after `--warmup`."""
    import torch
    from paper_2605_31481_b200 import binding
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    desc = W.config_robot(args.config)
    m = binding.Model(desc, device=0)
    m.set_option("step_calibrate", 0)                   # no calibration launches in front of the kernel an ncu capture is after
    for kv in args.option:
        k, v = kv.split("=")
        m.set_option(k, int(v))
    if not args.no_specialize:
        m.specialize(SPEC_OPS + (("aba",) if args.only == "aba" else ()) + (("rnea_vjp",) if args.only == "vjp" else ()))
    B = args.B
    sets, _ = make_sets(torch, m, desc, args.config, B, dev)
    stream = torch.cuda.current_stream().cuda_stream
    extra = {}
    if args.only == "aba":
        extra = {"ws": torch.empty(m.aba_workspace_floats(B), device=dev), "out": torch.empty((m.nv, B), device=dev)}
    if args.only == "vjp":
        extra = {"ws": torch.empty(max(1, m.rnea_vjp_workspace_floats(B)), device=dev), "out": torch.empty((m.nb, 10), device=dev)}

    def call(i):
        s = sets[i % len(sets)]
        if args.only == "aba":
            m.aba(B, s.q, s.qd, s.qdd, extra["out"], extra["ws"], stream)
        elif args.only == "vjp":
            m.rnea_vjp_params(B, s.q, s.qd, s.qdd, s.qdd, extra["out"], extra["ws"], stream)
        else:
            op_call(m, args.only, s, B, stream)

    for i in range(max(3, args.warmup)):
        call(i)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for i in range(args.steps):
        call(i)
    e1.record()
    torch.cuda.synchronize()
    print(json.dumps({"only": args.only, "config": W.CONFIG_NAMES[args.config], "B": B, "launches": args.steps,
                      "us_per_launch_host_train": e0.elapsed_time(e1) * 1e3 / args.steps}), flush=True)


def run_ours(args):
    import torch
    import torch.distributed as dist
    os.environ.setdefault("BARD_CACHE", "0")      # specialize_s reports NVRTC itself, not a warm on-disk cubin cache
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
        D.barrier()
        torch.cuda.synchronize()

    t_start = time.perf_counter()
    extras = rank == 0 and world == 1 and not args.quick
    cfg, B, K, Wm = args.config, args.B, args.steps, max(args.warmup, 3)
    fp32_meas = None
    try:
        fp32_meas = binding.measure_fp32_peak(local)
    except Exception:
        pass
    pk = RL.measured_peaks(ROOT, fp32_meas)

    models, spec_s = {}, {}

    def model(c):
        """One model per config for the whole run; bard_model_specialize is timed (NVRTC: seconds per robot)."""
        if c not in models:
            d = W.config_robot(c)
            mm = binding.Model(d, device=local)
            for kv in args.option:                      # experiments: bard_model_set_option before specialising
                k, v = kv.split("=")
                mm.set_option(k, int(v))
            if not args.no_specialize:
                t0 = time.perf_counter()
                mm.specialize(SPEC_OPS)
                spec_s[W.CONFIG_NAMES[c]] = time.perf_counter() - t0
            models[c] = (d, mm)
        return models[c]

    desc, m = model(cfg)
    sets, per_set = make_sets(torch, m, desc, cfg, B, dev)
    R = len(sets)
    stream = torch.cuda.current_stream().cuda_stream
    clocks = Clocks(local)
    clocks.start()

    def step(i, ev=None):
        s = sets[i % R]
        if ev is None:      # the call a user makes: bard_step = all four operators of one batch
            m.step(B, s.q, s.qd, s.qdd, s.pose, s.J, s.tau, s.M, stream)
            return
        for k, op in enumerate(OPS):
            ev[k].record()
            op_call(m, op, s, B, stream)
        ev[4].record()

    # ---- device-resident timed region: W warm-up steps, then exactly K steps
    for i in range(Wm):
        step(i)
    # The timed region is K uninstrumented steps between two events: an event record between two launches would
    # end the programmatic overlap of a kernel's prologue with the previous kernel's tail (PDL) and time the
    # events themselves.  Per-operator durations come from a second pass of K steps, the four operators called one by
    # one with an event before every launch; its step time is reported as ms_per_step_instrumented.
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
    elapsed_ms = D.max_over_ranks(e_beg.elapsed_time(e_end), dev)
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(K)]
    for i in range(Wm):
        step(i, evs[0])
    barrier()
    clocks.active.set()
    for i in range(K):
        step(i, evs[i])
    barrier()
    clocks.active.clear()
    instrumented_ms = evs[0][0].elapsed_time(evs[-1][4])
    value = world * B * K / (elapsed_ms * 1e-3)
    op_sec = {op: float(np.mean([evs[i][k].elapsed_time(evs[i][k + 1]) for i in range(K)])) * 1e-3
              for k, op in enumerate(OPS)}
    ops = {}
    for op in OPS:
        r = op_report(desc, pk, op, op_sec[op], B)
        ops[op] = {"in_step": short(r, ("us", "frac", "achieved")), "bound": r["bound"], "unit": r["unit"], "peak": r["peak"],
                   "bytes_per_env": r["bytes_per_env"], "flop_per_env": r["flop_per_env"], "share_of_step": op_sec[op] / sum(op_sec.values())}
    # ---- per-operator back-to-back trains, replayed from a CUDA graph (kernel time without host launch cost)
    clocks.active.set()
    for op in OPS:
        try:
            sec = time_graph(torch, m, op, sets, B)
        except Exception:
            sec = time_train(torch, m, op, sets, B, stream, launches=200)
        ops[op]["train"] = short(op_report(desc, pk, op, sec, B), ("us", "frac", "achieved", "env_evals_per_s"))
    clocks.active.clear()

    # ---- end to end: pinned host inputs -> device, bard_step, every output -> pinned host, per step
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
    te = D.max_over_ranks(time.perf_counter() - t0, dev)
    e2e = {"value": world * B * Ke / te, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": Ke,
           "note": "pinned host q/qd/qdd -> device, bard_step, pose/J/tau/M -> pinned host, every step (PCIe-bound)"}
    del h_in, h_out

    # ---- the roofline object: the dominant kernel of what bard_step ACTUALLY launches on this workload
    per_step = launches / K
    spec = (not args.no_specialize)
    if per_step == 2 and spec:
        # kinematics-fused kernel (FK + Jacobian + CRBA in one walk) + RNEA: a third pass of K steps, the two launches of
        # the step called one after the other (bard_kinematics, bard_rnea) with an event before each
        ev2 = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(K)]

        def step2(i, ev):
            x = sets[i % R]
            ev[0].record()
            m.kinematics(B, x.q, x.pose, x.J, x.M, stream)
            ev[1].record()
            m.rnea(B, x.q, x.qd, x.qdd, x.tau, stream)
            ev[2].record()
        for i in range(Wm):
            step2(i, ev2[0])
        barrier()
        clocks.active.set()
        for i in range(K):
            step2(i, ev2[i])
        barrier()
        clocks.active.clear()
        kin_sec = float(np.mean([ev2[i][0].elapsed_time(ev2[i][1]) for i in range(K)])) * 1e-3
        rd = op_report(desc, pk, "kin", kin_sec, B)
        try:
            train = op_report(desc, pk, "kin", time_graph(torch, m, "kin", sets, B, launches=max(R, 16)), B)["frac"]
        except Exception:
            train = None
        dom, kname = "kin", "bard_kin_n1 (model-specialised: FK + Jacobian + CRBA in one walk; bard_step = this kernel + bard_rnea_n1)"
        timing = "CUDA events before every launch, a third pass of K steps: bard_kinematics then bard_rnea (the two launches of bard_step)"
        ops["kin"] = {"in_step": short(rd, ("us", "frac", "achieved")), "bound": rd["bound"], "bytes_per_env": rd["bytes_per_env"],
                      "rnea_after_kin_us": float(np.mean([ev2[i][1].elapsed_time(ev2[i][2]) for i in range(K)])) * 1e3, "train_frac": train}
    elif per_step == 1 and spec:
        # one fused launch: the step IS the kernel; bytes = every input and output of the four operators once
        c = RL.counts(desc)
        bytes_env = 4 * (m.nq + 2 * m.nv) + sum(c[o]["out"] for o in OPS)
        sec = elapsed_ms * 1e-3 / K
        rd = {"bound": "hbm", "achieved": bytes_env * B / sec / 1e9, "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": bytes_env * B / sec / 1e9 / pk["hbm_gbs"],
              "bytes_per_env": bytes_env, "flop_per_env": sum(c[o]["flop"] for o in OPS), "us": sec * 1e6}
        dom, kname, train = "step", "bard_step_n1 / bard_step4_n1 (model-specialised: the four operators in one launch)", None
        timing = "the timed region itself: K back-to-back bard_step launches between two CUDA events"
    else:
        dom = max(OPS, key=lambda o: op_sec[o])
        rd = op_report(desc, pk, dom, op_sec[dom], B)
        kname = f"bard_{dom}_n1 (model-specialised)" if spec else f"{dom}_kernel"
        train = ops[dom]["train"]["frac"]
        timing = "CUDA events before every launch, a second pass of K steps with the four operators called one by one"
    roof = {"kernel": kname, "bound": rd["bound"], "achieved": rd["achieved"],
            "peak": rd["peak"], "unit": rd["unit"], "frac": rd["frac"], "traffic": None,
            "peak_source": ("MEASURED_PEAKS.json hbm_gbs" if rd["bound"] == "hbm" else
                            "min(measured FFMA chain, 148 SM x 128 lanes x 2 x sm_max_mhz)") + f" ({pk['source']})",
            "algorithmic_per_launch": (rd["bytes_per_env"] if rd["bound"] == "hbm" else rd["flop_per_env"]) * B,
            "avg_launch_us": rd["us"], "frac_back_to_back_train": train, "timing": timing}
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
                   "step_call": f"bard_step -> {launches / K:g} launch(es) per step"},
        "roofline": roof, "ops": sig(ops), "e2e": e2e, "gpu_launches": int(launches),
        "peaks": sig({"hbm_gbs": pk["hbm_gbs"], "fp32_tflops_used": pk["fp32_tflops"], "fp32_tflops_nominal": pk["fp32_tflops_nominal"],
                      "fp32_tflops_measured_ffma_chain": pk["fp32_tflops_measured"], "source": pk["source"]}, 5),
    }
    del sets
    torch.cuda.empty_cache()

    if extras:
        clocks.active.set()
        # ---- BASELINE.json's metric: every operator and the step on configs 0-3 at B = 4096 and 65 536
        if not args.no_matrix:
            matrix = {}
            for c in range(4):
                dc, mc = model(c)
                row = {}
                for Bm in (4096, 65536):
                    ss, _ = make_sets(torch, mc, dc, c, Bm, dev, min_sets=4, cap_bytes=8 << 30)
                    cell = {}
                    for op in OPS:
                        r = op_report(dc, pk, op, time_graph(torch, mc, op, ss, Bm), Bm)
                        cell[op] = short(r, ("us", "env_evals_per_s", "bound", "frac"))
                    n0 = binding.launch_count()
                    op_call(mc, "step", ss[0], Bm, stream)
                    per = binding.launch_count() - n0
                    sec = time_graph(torch, mc, "step", ss, Bm, launches=max(len(ss), 32))
                    roof_us = sum(RL.roofline(dc, pk)[op]["t_env"] for op in OPS) * Bm * 1e6
                    cell["step"] = {"us": sec * 1e6, "env_evals_per_s": Bm / sec, "launches": int(per), "sum_of_rooflines_us": roof_us,
                                    "frac_of_summed_rooflines": roof_us / (sec * 1e6)}
                    row[f"B{Bm}"] = cell
                    del ss
                    torch.cuda.empty_cache()
                matrix[W.CONFIG_NAMES[c]] = row
            line["matrix"] = sig(matrix)
        # ---- BASELINE.json config 4: batch sweep on the humanoid and the chain, with the oracle's time per B
        if not args.no_sweep:
            import oracle
            oracle.set_threads(os.cpu_count() or 1)
            sweep = {}
            for c in (3, 0):
                dc, mc = model(c)
                o = oracle.Oracle(dc)
                n_or = 2048
                oq, oqd, oqdd = (a.astype(np.float64) for a in W.config_states(c, n_or))
                oracle_pass_seconds(o, oq, oqd, oqdd)
                row = {}
                for Bs in SWEEP_B:
                    ss, _ = make_sets(torch, mc, dc, c, Bs, dev, cap_bytes=40 << 30)
                    cell = {}
                    for op in OPS:
                        cell[op] = short(op_report(dc, pk, op, time_graph(torch, mc, op, ss, Bs), Bs))
                    n = min(Bs, n_or)
                    t = min(oracle_pass_seconds(o, oq[:, :n].copy(), oqd[:, :n].copy(), oqdd[:, :n].copy()) for _ in range(2))
                    cell["oracle"] = {"s_for_B_est": t * Bs / n, "env_evals_per_s": n / t, "sample_envs": n}
                    row[f"B{Bs}"] = cell
                    del ss
                    torch.cuda.empty_cache()
                sweep[W.CONFIG_NAMES[c]] = row
            sweep["note"] = (f"per operator: device time of a back-to-back train replayed from a CUDA graph, rotating buffer sets; oracle: fp64, "
                             f"{oracle.get_threads()} host threads, all four operators on min(B, 2048) environments, scaled to B")
            line["sweep"] = sig(sweep)
        # ---- beyond the metric: ABA, RNEA VJP, fp64 / AoS variants, on the headline workload
        if not args.no_specialize and m.nv > 0:
            line.update(extras_section(torch, binding, m, desc, cfg, B, dev, stream, pk, spec_s))
        if not args.no_rollout:
            try:
                d2, m2 = model(2)
                line["config2_rollout"] = sig(rollout_config2(torch, binding, m2, d2, dev))
            except Exception as ex:                      # graph capture is a convenience of the bench, not of the path
                line["config2_rollout"] = {"error": str(ex)[:200]}
        clocks.active.clear()
    clocks.stop()
    line["clocks"] = clocks.summary()
    line["specialize_s"] = sig(spec_s, 3)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = time_oracle(desc, cfg, 4.0 if args.quick else args.cpu_seconds)
    line["bench_wall_s"] = round(time.perf_counter() - t_start, 1)
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def extras_section(torch, binding, m, desc, cfg, B, dev, stream, pk, spec_s):
    out = {}
    sets, _ = make_sets(torch, m, desc, cfg, B, dev)

    def timed(fn, n=30, warm=3):
        for i in range(warm):
            fn(i)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for i in range(n):
            fn(i)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e-3 / n

    try:    # ABA forward dynamics
        t0 = time.perf_counter()
        m.specialize(("aba",))
        spec_s["aba:" + desc.name] = time.perf_counter() - t0
        ws = torch.empty(m.aba_workspace_floats(B), device=dev)
        qdd_out = torch.empty((m.nv, B), device=dev)
        sec = timed(lambda i: m.aba(B, sets[i % len(sets)].q, sets[i % len(sets)].qd, sets[i % len(sets)].qdd, qdd_out, ws, stream))
        r = op_report(desc, pk, "aba", sec, B)
        out["aba"] = {"us": sec * 1e6, "env_evals_per_s": B / sec, "roofline": short(r, ("bound", "achieved", "peak", "unit", "frac")),
                      "bytes_per_env": r["bytes_per_env"], "flop_per_env": r["flop_per_env"],
                      "workspace_bytes_per_env": 4 * m.aba_workspace_floats(B) // B}
        del ws, qdd_out
    except Exception as ex:
        out["aba"] = {"error": str(ex)[:200]}
    try:    # reverse-mode RNEA w.r.t. the inertial parameters: 4 input arrays, one outward pass, the batch sum
        ws = torch.empty(max(1, m.rnea_vjp_workspace_floats(B)), device=dev)
        g = torch.empty((m.nb, 10), device=dev)

        def vjp(i):
            x = sets[i % len(sets)]
            m.rnea_vjp_params(B, x.q, x.qd, x.qdd, x.tau, g, ws, stream)
        m.set_option("spec_vjp_min_b", 1 << 40)
        sec_table = timed(vjp)
        t0 = time.perf_counter()
        m.specialize(("rnea_vjp",))
        spec_s["rnea_vjp:" + desc.name] = time.perf_counter() - t0
        m.set_option("spec_vjp_min_b", -1)
        sec = timed(vjp)
        r = op_report(desc, pk, "rnea_vjp", sec, B)
        out["rnea_vjp"] = {"us": sec * 1e6, "env_evals_per_s": B / sec, "roofline": short(r, ("bound", "achieved", "peak", "unit", "frac")),
                           "bytes_per_env": r["bytes_per_env"], "flop_per_env": r["flop_per_env"], "hbm_gbs": r["hbm_gbs"], "launches": 2,
                           "kernel": "bard_rnea_vjp_n1 (generated) + vjp_reduce_columns_kernel", "table_driven_us": sec_table * 1e6}
        del ws, g
    except Exception as ex:
        out["rnea_vjp"] = {"error": str(ex)[:200]}
    del sets
    torch.cuda.empty_cache()
    # fp64 / AoS variants of the four operators, train timing, own buffers
    var = {}
    try:
        ins32 = W.sample_states(desc, B, seed=2000 + cfg)
        for dtype, layout in (("f32", "aos"), ("f64", "soa")):
            t0 = time.perf_counter()
            m.specialize_variant(OPS, dtype, layout)
            spec_s[f"{dtype}_{layout}:" + desc.name] = time.perf_counter() - t0
            td = torch.float64 if dtype == "f64" else torch.float32
            es = 8 if dtype == "f64" else 4
            tin = [torch.from_numpy(a).to(dev).to(td) for a in ins32]
            shapes = ((m.nb, 12), (m.nframes, 6, m.nv), (m.nv,), (m.nv, m.nv))
            if layout == "aos":
                tin = [t.t().contiguous() for t in tin]
                outs = [torch.empty((B,) + sh, device=dev, dtype=td) for sh in shapes]
            else:
                outs = [torch.empty(sh + (B,), device=dev, dtype=td) for sh in shapes]
            ws = torch.empty(max(m.variant_workspace_bytes(op, dtype, layout, B) for op in OPS) // 4 + 4, device=dev)
            calls = {"fk": lambda i: m.fk_v(dtype, layout, B, tin[0], outs[0], ws, stream),
                     "jacobian": lambda i: m.jacobian_v(dtype, layout, B, tin[0], outs[1], ws, stream),
                     "rnea": lambda i: m.rnea_v(dtype, layout, B, tin[0], tin[1], tin[2], outs[2], ws, stream),
                     "crba": lambda i: m.crba_v(dtype, layout, B, tin[0], outs[3], ws, stream)}
            cell = {}
            for op in OPS:
                sec = timed(calls[op], n=20)
                c = RL.counts(desc)[op]
                cell[op] = {"us": sec * 1e6, "hbm_gbs": c["bytes"] * (es // 4) * B / sec / 1e9, "tflops": c["flop"] * B / sec / 1e12}
            var[f"{dtype}_{layout}"] = cell
            del tin, outs, ws
            torch.cuda.empty_cache()
        out["variants"] = var
    except Exception as ex:
        out["variants"] = {"error": str(ex)[:200]}
    return sig(out)


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    elif a.only:
        run_only(a)
    else:
        run_ours(a)
