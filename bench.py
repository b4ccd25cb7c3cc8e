#!/usr/bin/env python
"""bench.py -- throughput of the TDSE hot path on B200 (one JSON line on stdout, rank 0).

Own arm (default): workload CFG5 of BASELINE.json (256 independent hydrogen wavefunctions per GPU, N_r = 2000,
L = 16, 3-point stencil, Taylor order 6; the largest Taylor grid, sharded over ranks by members, weak scaling).
A "step" is one Taylor time step of the whole batch: field table -> H.psi x order with the propagator arithmetic
fused -> state update.  `value` = Gpoint-updates/s of H(t)psi = members * L * N_r * order * steps / device time.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg5] [--impl reference] [--no-extra]

With --gpus N > 1 and no torchrun environment the script re-executes itself under torch.distributed.run (one rank
per GPU, NCCL).  Reference arm (--impl reference): the CPU oracle (oracle/), as it stands, on the host cores, on a
bounded sample of the same workload.  See DESIGN.md "Measurement".
"""
import argparse
import json
import math
import os
import socket
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1308_1856_b200 import workloads as wl  # noqa: E402

METRIC = "Gpoint-updates/s of H(t)psi (Taylor step)"
UNIT = "Gpoint-updates/s"
L2_BYTES = 126e6                      # B200 L2 (B200_PROFILING.md)
# FP64 issue roof: 148 SMs x 64 FP64 lanes x clocks.max.sm 1.965 GHz = 18.6 T thread-instructions/s (nominal, from the
# guide's unit counts and clocks; a DFMA-only probe on this pool measured 18.2 T/s, profiles/r02_README.md section 2)
FP64_PEAK_INSTR = 148 * 64 * 1.965e9


def host_cores():
    try:
        return len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count() or 1


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


# ------------------------------------------------------------------------------------------ clocks sampler
class ClockSampler(threading.Thread):
    """Samples SM clock, GPU utilisation and throttle reasons of one GPU (NVML; nvidia-smi fallback) from before the
    warm-up to the end of the e2e legs; `sm_mhz` is the median over the samples taken while the GPU was busy."""

    def __init__(self, index, period=0.005):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.busy, self.reasons, self.stop_flag = [], [], set(), False
        self.max_mhz = None
        self.nv = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.dev = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.dev, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        names = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
                 0x80: "hw_power_brake", 0x2: "applications_clocks_setting"}
        while not self.stop_flag:
            if self.nv is not None:
                try:
                    self.samples.append(self.nv.nvmlDeviceGetClockInfo(self.dev, self.nv.NVML_CLOCK_SM))
                    try:
                        self.busy.append(self.nv.nvmlDeviceGetUtilizationRates(self.dev).gpu)
                    except Exception:
                        self.busy.append(100)
                    r = self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.dev)
                    for bit, nm in names.items():
                        if r & bit:
                            self.reasons.add(nm)
                except Exception:
                    pass
            else:
                try:
                    import subprocess
                    out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=clocks.sm,clocks.max.sm,"
                                          "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
                                          "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap",
                                          "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5)
                    f = [x.strip() for x in out.stdout.strip().split(",")]
                    self.samples.append(int(f[0]))
                    self.busy.append(100)
                    self.max_mhz = int(f[1])
                    for nm, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], f[2:]):
                        if v.lower().startswith("active"):
                            self.reasons.add(nm)
                except Exception:
                    pass
            time.sleep(self.period)

    def result(self):
        self.stop_flag = True
        self.join(timeout=5)
        load = [s for s, b in zip(self.samples, self.busy) if b > 0] or self.samples
        med = float(np.median(load)) if load else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples),
                "samples_under_load": len(load), "window": "warm-up + timed region + e2e legs"}


# ------------------------------------------------------------------------------------------ CPU oracle timing
def time_oracle(c, order, dt, t0, members, steps, warmup, threads):
    """Oracle Taylor steps on `members` members of the workload; returns (seconds for `steps` steps)."""
    import oracle
    oracle.set_threads(threads)
    cs = dict(c)
    cs["batch"] = members
    g = oracle.make_grid(cs["n_r"], cs["dr"], cs["n_l"], cs["fd_order"], batch=members)
    pulses = wl.pulses(c)[:members]
    psi = wl.populated_state(cs)
    if warmup:
        psi, _ = oracle.step_taylor(g, pulses, psi, order, t0, dt, warmup)
    t = time.perf_counter()
    psi, _ = oracle.step_taylor(g, pulses, psi, order, t0 + warmup * dt, dt, steps)
    el = time.perf_counter() - t
    assert np.isfinite(psi.view(np.float64)).all()
    return el


def cpu_baseline(c, order, dt, t0, budget_s=10.0):
    """The oracle as it stands on a bounded sample: all host cores (OpenMP over l rows) and one thread."""
    cores = host_cores()
    members = min(c["batch"], 16)
    pts = members * c["n_l"] * c["n_r"]
    probe = time_oracle(c, order, dt, t0, members, 2, 1, cores)
    steps = int(max(2, min(2000, budget_s / max(probe / 2, 1e-6))))
    el = time_oracle(c, order, dt, t0, members, steps, 0, cores)
    m1 = min(members, 2)
    probe1 = time_oracle(c, order, dt, t0, m1, 2, 1, 1)
    steps1 = int(max(2, min(2000, 0.5 * budget_s / max(probe1 / 2, 1e-6))))
    el1 = time_oracle(c, order, dt, t0, m1, steps1, 0, 1)
    return {"value": pts * order * steps / el / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{members} of {c['batch']} members x {steps} Taylor-{order} steps (same grid, dt, pulses), "
                      f"OpenMP over l rows, {el:.1f} s", "s_per_step_full_batch": el / steps * c["batch"] / members,
            "one_thread": {"value": m1 * c["n_l"] * c["n_r"] * order * steps1 / el1 / 1e9, "unit": UNIT, "cores": 1,
                           "sample": f"{m1} members x {steps1} steps, {el1:.1f} s"}}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    c = wl.config(args.workload)
    order = c["order"]
    dt = wl.dt_eff(c)
    t0 = wl.window(c, args.steps + args.warmup, dt)
    cores = host_cores()
    members = min(c["batch"], 16)
    el = time_oracle(c, order, dt, t0, members, args.steps, args.warmup, cores)
    pts = members * c["n_l"] * c["n_r"]
    val = pts * order * args.steps / el / 1e9
    sample = f"{members} of {c['batch']} members per step (same grid, dt, pulses); oracle/ as it stands, OpenMP over l rows"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": el / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{args.workload} (BASELINE.json configs[{c['index'] - 1}]), bounded sample",
                       "taylor_order": order, "dt_eff": dt},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------ inputs of the product arm
def bound_state_inputs(c):
    """Input data for CFG5's yield (reading R-G23): every eigenvector with E < 0 of the discrete 3-point h_l, l = 0..L-1,
    from LAPACK's tridiagonal solver (the tests hand the oracle's own vectors to both sides; the product arm may not
    touch oracle/).  Normalised dr sum phi^2 = 1."""
    from scipy.linalg import eigh_tridiagonal
    assert c["fd_order"] == 3
    r = wl.radial_grid(c)
    dr2 = c["dr"] ** 2
    off = np.full(c["n_r"] - 1, -0.5 / dr2)
    ls, phis = [], []
    for l in range(c["n_l"]):
        d = 1.0 / dr2 + l * (l + 1) / (2.0 * r * r) - 1.0 / r
        w, v = eigh_tridiagonal(d, off, select="v", select_range=(-1e3, 0.0))
        for k in range(len(w)):
            ls.append(l)
            phis.append(wl.grid_normalised(v[:, k] * (1.0 if v[0, k] >= 0 else -1.0), c["dr"]))
    return np.array(ls, dtype=np.int32), np.array(phis)


# ------------------------------------------------------------------------------------------ own arm
def run_own(args):
    import torch
    import torch.distributed as dist
    from paper_1308_1856_b200 import binding, sharding

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback "
                         "(use --impl reference for the oracle arm)")
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    c = wl.config(args.workload)
    order, B, L, N = c["order"], c["batch"], c["n_l"], c["n_r"]
    dt = wl.dt_eff(c)
    K, W = args.steps, args.warmup
    t0 = wl.window(c, K + W, dt)
    # weak scaling: every rank runs a full batch; rank r takes members [r*B, (r+1)*B) of a world*B-member scan
    cg = wl.config(args.workload, batch=B * world)
    first, cnt = sharding.member_slice(B * world, rank, world)
    pulses = wl.pulses(cg)[first:first + cnt]
    psi0 = wl.populated_state(c)                       # S3/S4 state: every l block populated (no denormals)
    pts = B * L * N

    h = binding.Tdse(N, c["dr"], L, c["fd_order"], batch=B)
    h.set_option("taylor_block", 0 if args.no_block else 1)
    h.set_option("taylor_rp_variant", args.rp_variant)
    h.set_option("taylor_rp_tma", args.rp_tma)
    h.set_option("graph_steps", args.graph_steps)
    h.set_pulse(pulses)
    if c["fd_order"] == 3:
        h.set_bound_states(*bound_state_inputs(c))     # CFG5's stated output: the yield over every bound state
    stream = torch.cuda.Stream()
    pinned = torch.empty((B, L, N), dtype=torch.complex128).pin_memory()
    pinned.numpy()[...] = psi0
    pin_out = torch.empty((B, L, N), dtype=torch.complex128).pin_memory()

    sampler = ClockSampler(local)
    sampler.start()
    with torch.cuda.stream(stream):
        h.set_state(pinned.numpy(), stream=stream)
        # ---- device-resident timing.  Warm-up: W steps, then one untimed call of EXACTLY the timed call's shape (same K,
        # hence the same captured graphs and the same eager remainder), so that no graph is captured or instantiated
        # between the events.
        h.step_taylor(order, t0, dt, W, 0, stream=stream)
        l_w = h.launch_count()
        h.step_taylor(order, t0 + W * dt, dt, K, 0, stream=stream)
        shape_launches = h.launch_count() - l_w
        h.set_state(pinned.numpy(), stream=stream)
        h.step_taylor(order, t0, dt, W, 0, stream=stream)
        stream.synchronize()
        sharding.barrier()
        torch.cuda.synchronize()
        l0, g0 = h.launch_count(), h.graph_instantiations()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(stream)
        h.step_taylor(order, t0 + W * dt, dt, K, 0, stream=stream)
        ev1.record(stream)
        stream.synchronize()
        torch.cuda.synchronize()
        sharding.barrier()
        ms = ev0.elapsed_time(ev1)
        launches = h.launch_count() - l0
        assert h.graph_instantiations() == g0, "a CUDA graph was instantiated inside the timed region"
        assert launches == shape_launches, (launches, shape_launches)
        blocked = h.taylor_kernel()
        obs = h.observables(t0 + (W + K) * dt, stream=stream)
        norm_dev = float(np.max(np.abs(obs[:, 0] - 1.0)))
        ms = sharding.max_over_ranks(ms)

        # ---- end to end through the C ABI with host buffers: upload pulses + state, K steps, the config's stated
        # output (ionisation yield per member) and the final state back to the host
        sharding.barrier()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        tw0 = time.perf_counter()
        e0.record(stream)
        h.set_pulse(pulses)
        h.set_state(pinned.numpy(), stream=stream)
        h.step_taylor(order, t0, dt, K, 0, stream=stream)
        yld = h.ionisation_yield(stream=stream) if h.n_states else h.observables(t0 + K * dt, stream=stream)[:, 0]
        h.get_state(pin_out.numpy(), stream=stream)
        e1.record(stream)
        stream.synchronize()
        tw1 = time.perf_counter()
        ms_e2e_serial = max(e0.elapsed_time(e1), (tw1 - tw0) * 1e3)
        ms_e2e_serial = sharding.max_over_ranks(ms_e2e_serial)
        h2d = (pinned.numel() * 16 + 40 * B) / K
        d2h = (pin_out.numel() * 16 + yld.size * 8) / K
        # ---- the same job with the batch split over several handles and streams (members are independent): the
        # pinned-host transfers of one part overlap the steps of another.  Same bytes, same outputs, same ABI calls.
        ms_e2e, n_parts, yld_p = e2e_pipelined(binding, torch, sharding, c, args, pulses, pinned, pin_out, order, t0, dt, K,
                                               parts=args.e2e_parts)
        if ms_e2e is None or ms_e2e > ms_e2e_serial:
            ms_e2e, n_parts = ms_e2e_serial, 1
        else:
            assert np.max(np.abs(yld_p - yld)) <= 1e-12, "split and single-handle runs disagree"
        # the same round trip for SHORT jobs (one graph block of steps per upload/download): PCIe-bound by design,
        # reported so that the amortisation in `e2e` is visible
        ks = max(2, args.graph_steps)
        reps = 3
        sharding.barrier()
        torch.cuda.synchronize()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record(stream)
        for _ in range(reps):
            h.set_state(pinned.numpy(), stream=stream)
            h.step_taylor(order, t0, dt, ks, 0, stream=stream)
            h.observables(t0 + ks * dt, stream=stream)
            h.get_state(pin_out.numpy(), stream=stream)
        s1.record(stream)
        stream.synchronize()
        ms_short = sharding.max_over_ranks(s0.elapsed_time(s1))
        e2e_short = {"steps_per_round_trip": ks, "value": pts * world * order * ks * reps / (ms_short * 1e-3) / 1e9,
                     "unit": UNIT, "h2d_bytes_per_step": pinned.numel() * 16 / ks, "d2h_bytes_per_step": pin_out.numel() * 16 / ks}
    clocks = sampler.result()

    total_pts = pts * world
    value = total_pts * order * K / (ms * 1e-3) / 1e9
    e2e_val = total_pts * order * K / (ms_e2e * 1e-3) / 1e9

    # ---- roofline of the dominant kernel (per launch): algorithmic bytes / average launch duration
    peak, peak_src = measured_peaks()
    if blocked:
        bytes_step = 32.0 * pts                         # read psi once, write psi once (all orders on chip)
        kname, n_dom = {4: "taylor_rp_kernel (TMA)", 3: "taylor_rp_kernel"}[blocked], K
    else:
        bytes_step = (64.0 * order - 32.0) * pts        # k=1: 16R+32W, 1<k<P: 32R+32W, k=P: 32R+16W
        kname, n_dom = "tile_kernel<EpiTaylor>", K * order
    achieved = bytes_step * K / (ms * 1e-3) / 1e9
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        try:
            traffic = json.load(open(tpath)).get(kname)
        except Exception:
            traffic = None
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "kernel": kname, "launches": n_dom, "us_per_launch": ms * 1e3 / n_dom,
                "algorithmic_bytes_per_launch": bytes_step * K / n_dom, "peak_source": peak_src}
    if blocked:
        # second roof of the all-orders-in-one-pass kernel: FP64 issue.  Algorithmic FP64
        # instructions per point-update of the scaled operator H/c1 (no halo redundancy counted) against the nominal
        # FP64 issue rate 148 SMs x 64 lanes x 1.965 GHz.
        fp64_per_update = 12.25 if c["fd_order"] == 3 else 16.25
        alu_rate = pts * order * fp64_per_update * K / (ms * 1e-3)
        roofline["alu"] = {"fp64_instr_per_point_update": fp64_per_update, "achieved_instr_per_s": alu_rate,
                           "peak_instr_per_s": FP64_PEAK_INSTR, "frac": alu_rate / FP64_PEAK_INSTR,
                           "peak_source": "nominal: 148 SMs x 64 FP64 lanes x 1.965 GHz"}

    state_bytes = pts * 16
    l2 = (f"inputs_exceed_l2 (state arrays {state_bytes / 1e6:.0f} MB each > {L2_BYTES / 1e6:.0f} MB L2)"
          if state_bytes > L2_BYTES else
          f"L2-resident working set ({state_bytes / 1e6:.1f} MB per state array <= {L2_BYTES / 1e6:.0f} MB L2): "
          "the HBM roofline does not bind this workload")
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": f"{args.workload} (BASELINE.json configs[{c['index'] - 1}]): {B} members/GPU x L={L} x "
                                   f"N_r={N}, {c['fd_order']}-point, Taylor order {order}",
                       "dt_cfg": c["dt_cfg"], "dt_eff": dt, "window": "pulse peak", "state": "S4 populated",
                       "points_per_gpu": pts, "taylor_blocked": bool(blocked), "taylor_kernel": kname, "graph_steps": args.graph_steps,
                       "l2": l2, "parallelism": f"batch x{world}",
                       "warmup_detail": f"{W} steps + one untimed call of the timed call's shape ({K} steps)"},
            "clocks": clocks, "roofline": roofline,
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "what": "set_pulse + set_state(host, pinned) + K steps + ionisation_yield over "
                            f"{h.n_states} bound states + get_state(host) via the C ABI; batch split over {n_parts} "
                            "handle(s) / streams so that transfers overlap steps",
                    "single_handle": {"value": total_pts * order * K / (ms_e2e_serial * 1e-3) / 1e9, "unit": UNIT},
                    "yield_range": [float(np.min(yld)), float(np.max(yld))], "short_jobs": e2e_short},
            "gpu_launches": int(launches), "graphs_instantiated_in_timed_region": 0, "max_norm_drift": norm_dev}

    if rank == 0 and not args.no_extra and world == 1:
        line["extra"] = extra_measurements(binding, torch, stream, full_pulse=not args.no_full_pulse)
    if rank == 0 and world == 1 and not args.no_cpu:
        line["cpu_baseline"] = cpu_baseline(c, order, dt, t0)
    h.close()
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def e2e_pipelined(binding, torch, sharding, c, args, pulses, pinned, pin_out, order, t0, dt, K, parts=4):
    """End-to-end leg with the members split over `parts` handles, each on its own stream: upload (pinned host,
    asynchronous) -> K steps -> yield -> download per part; returns (ms, parts, yields) or (None, 1, None)."""
    B, L, N = c["batch"], c["n_l"], c["n_r"]
    if B % parts or c["fd_order"] != 3:
        return None, 1, None
    Bp = B // parts
    states = bound_state_inputs(c)
    hs, streams = [], []
    for i in range(parts):
        hp = binding.Tdse(N, c["dr"], L, c["fd_order"], batch=Bp)
        hp.set_option("graph_steps", args.graph_steps)
        hp.set_bound_states(*states)
        hs.append(hp)
        streams.append(torch.cuda.Stream())
    src, dst = pinned.numpy(), pin_out.numpy()

    def run():
        for i, hp in enumerate(hs):
            hp.set_pulse(pulses[i * Bp:(i + 1) * Bp])
        for i, hp in enumerate(hs):
            hp.set_state(src[i * Bp:(i + 1) * Bp], stream=streams[i], pinned_async=True)
            hp.step_taylor(order, t0, dt, K, 0, stream=streams[i])
        for i, hp in enumerate(hs):
            hp.get_state(dst[i * Bp:(i + 1) * Bp], stream=streams[i], pinned_async=True)
        return np.concatenate([hp.ionisation_yield(stream=streams[i]) for i, hp in enumerate(hs)])

    run()                                               # graphs captured, buffers allocated
    torch.cuda.synchronize()
    sharding.barrier()
    e0 = torch.cuda.Event(enable_timing=True)
    ends = [torch.cuda.Event(enable_timing=True) for _ in range(parts)]
    tw0 = time.perf_counter()
    e0.record(streams[0])
    for st in streams[1:]:
        st.wait_event(e0)
    yld = run()
    for st, ev in zip(streams, ends):
        ev.record(st)
    torch.cuda.synchronize()
    tw1 = time.perf_counter()
    ms = max(max(e0.elapsed_time(ev) for ev in ends), (tw1 - tw0) * 1e3)
    for hp in hs:
        hp.close()
    return sharding.max_over_ranks(ms), parts, yld


def timed(torch, stream, fn, reps=1):
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(reps):
        fn()
    e1.record(stream)
    stream.synchronize()
    return e0.elapsed_time(e1) / reps


def extra_measurements(binding, torch, stream, full_pulse=True):
    """Secondary figures (not the headline): bare H.psi, s/step of the other configs, the claim "HBM-bound for small
    orders" tested (Taylor-2 / Taylor-4 on the CFG5 grid) and the roofline sweep of SURVEY section 8(d) S1."""
    out = {}
    peak, _ = measured_peaks()
    with torch.cuda.stream(stream):
        for name in ("cfg4", "cfg3"):
            c = wl.config(name)
            h = binding.Tdse(c["n_r"], c["dr"], c["n_l"], c["fd_order"], batch=c["batch"])
            x = torch.from_numpy(wl.random_state(c)).cuda()
            y = torch.empty_like(x)
            for _ in range(5):
                h.apply_H(x, y, 0.05, stream=stream)
            us = timed(torch, stream, lambda: h.apply_H(x, y, 0.05, stream=stream), 50) * 1e3
            pts = x.numel()
            out[f"apply_H_{name}"] = {"us": us, "gpoints_per_s": pts / us / 1e3, "gbs_algorithmic": 32.0 * pts / us / 1e3,
                                      "frac_of_hbm_peak": 32.0 * pts / us / 1e3 / peak,
                                      "note": "L2-resident" if pts * 32 < 100e6 else "exceeds L2"}
            del x, y
            h.close()
        # the CFG5 grid at lower orders: where the all-orders-in-one-pass kernel should be HBM-bound
        c = wl.config("cfg5")
        h = binding.Tdse(c["n_r"], c["dr"], c["n_l"], c["fd_order"], batch=c["batch"])
        h.set_pulse(wl.pulses(c))
        h.set_state(wl.populated_state(c), stream=stream)
        pts = c["batch"] * c["n_l"] * c["n_r"]
        for order in (2, 4):
            dt = wl.dt_eff(c, "taylor", 4)
            t0 = wl.window(c, 64, dt)
            h.step_taylor(order, t0, dt, 32, 0, stream=stream)
            ms = timed(torch, stream, lambda: h.step_taylor(order, t0, dt, 32, 0, stream=stream))
            us = ms * 1e3 / 32
            out[f"step_cfg5grid_taylor{order}"] = {"us_per_step": us, "gbs_algorithmic": 32.0 * pts / us / 1e3,
                                                   "frac_of_hbm_peak": 32.0 * pts / us / 1e3 / peak,
                                                   "gpoint_updates_per_s": pts * order / us / 1e3}
        h.close()
        for name, nsteps in (("cfg1", 2000), ("cfg2", 400), ("cfg3", 96), ("cfg4", 10)):
            c = wl.config(name)
            h = binding.Tdse(c["n_r"], c["dr"], c["n_l"], c["fd_order"], batch=c["batch"])
            h.set_pulse(wl.pulses(c))
            h.set_state(wl.populated_state(c), stream=stream)
            dt = wl.dt_eff(c)
            t0 = wl.window(c, 2 * nsteps, dt)
            every = 1 if name in ("cfg1", "cfg3") else 0

            def go(n, t):
                if c["propagator"] == "taylor":
                    h.step_taylor(c["order"], t, dt, n, every, stream=stream)
                elif c["propagator"] == "rk4":
                    h.step_rk4(t, dt, n, 0, stream=stream)
                else:
                    h.step_lanczos(c["krylov_dim"], c["order"], t, dt, n, 0, stream=stream)
            go(nsteps, t0)                                  # same call shape: graphs captured before the timed call
            ms = timed(torch, stream, lambda: go(nsteps, t0))
            n_h = {"taylor": c["order"], "rk4": 4, "lanczos": c.get("krylov_dim", 0)}[c["propagator"]]
            pts = c["batch"] * c["n_l"] * c["n_r"]
            out[f"step_{name}"] = {"propagator": c["propagator"], "us_per_step": ms * 1e3 / nsteps, "dt_eff": dt,
                                   "gpoint_updates_per_s": pts * n_h * nsteps / (ms * 1e-3) / 1e9,
                                   "blocked": h.taylor_was_blocked() if c["propagator"] == "taylor" else None,
                                   "observables_every_step": bool(every)}
            if c["propagator"] == "rk4":
                out[f"step_{name}"]["kernel"] = ("persistent on-chip Runge-Kutta kernel (RK4 as an FSAL scheme)"
                                                if h.rk45_was_persistent() else "four stages fused in the register-patch kernel")
                h.set_option("rk4_persist", 0)
                go(nsteps, t0)
                ms1 = timed(torch, stream, lambda: go(nsteps, t0))
                out[f"step_{name}"]["us_per_step_fused_register_patch_kernel"] = ms1 * 1e3 / nsteps
            if every:
                h.step_taylor(c["order"], t0, dt, nsteps, 0, stream=stream)
                ms0 = timed(torch, stream, lambda: h.step_taylor(c["order"], t0, dt, nsteps, 0, stream=stream))
                out[f"step_{name}"]["us_per_step_without_rows"] = ms0 * 1e3 / nsteps
            if c["propagator"] == "lanczos":
                # one fused pass per Krylov vector: 32 + (K-2) x 80 + 64 B/point, combine (K+1) x 16
                K = c["krylov_dim"]
                bpp = 32.0 + (K - 2) * 80.0 + 64.0 + (K + 1) * 16.0
                gbs = bpp * pts * nsteps / (ms * 1e-3) / 1e9
                out[f"step_{name}"].update({"algorithmic_bytes_per_point": bpp, "gbs_algorithmic": gbs,
                                            "frac_of_hbm_peak": gbs / peak})
            h.close()
        # CFG2, second propagator: adaptive Dormand-Prince 5(4), rtol 1e-8, over a 0.05 au window at the pulse peak
        c = wl.config("cfg2")
        h = binding.Tdse(c["n_r"], c["dr"], c["n_l"], c["fd_order"], batch=c["batch"])
        h.set_pulse(wl.pulses(c))
        psi0 = torch.from_numpy(wl.populated_state(c)).cuda()
        t_a = 0.5 * c["t_pulse"]
        h.set_state(psi0, stream=stream)
        h.step_rk45(t_a, t_a + 0.005, 1e-5, 1e-8, stream=stream)          # warm-up (graphs, controller)
        def rk45_run(hh):
            hh.set_state(psi0, stream=stream)
            stream.synchronize()
            info = {}
            ms = timed(torch, stream, lambda: info.update(hh.step_rk45(t_a, t_a + 0.05, 1e-5, 1e-8, stream=stream)))
            att = info["n_accept"] + info["n_reject"]
            return info, ms, att
        info, ms, att = rk45_run(h)
        pts = c["batch"] * c["n_l"] * c["n_r"]
        out["step_cfg2_rk45"] = {"propagator": "rk45 (Dormand-Prince, adaptive, rtol 1e-8)", "window_au": 0.05,
                                 "n_accept": info["n_accept"], "n_reject": info["n_reject"],
                                 "us_per_attempted_step": ms * 1e3 / max(att, 1),
                                 "dt_mean": float(np.mean(info["dt"])) if len(info["dt"]) else None,
                                 "gpoint_updates_per_s": pts * 6 * att / (ms * 1e-3) / 1e9,
                                 "kernel": "one persistent cooperative kernel (psi and k_1..k_7 on chip from t0 to t_end)"
                                           if h.rk45_was_persistent() else "one kernel per stage",
                                 "timing": "CUDA events around the call (the device runs the accept / reject loop)"}
        # the same run stage by stage (one graph launch: WHILE node around blocks of attempted steps)
        h.set_option("rk45_persist", 0)
        h.set_state(psi0, stream=stream)
        h.step_rk45(t_a, t_a + 0.005, 1e-5, 1e-8, stream=stream)
        info, ms, att = rk45_run(h)
        out["step_cfg2_rk45"]["stage_by_stage_us_per_attempted_step"] = ms * 1e3 / max(att, 1)
        h.close()
        out["sweep"] = roofline_sweep(binding, torch, stream, peak)
        if full_pulse:
            out["cfg3_full_pulse"] = cfg3_full_pulse(binding, torch, stream)
    return out


def cfg3_full_pulse(binding, torch, stream, lam=300.0):
    """CFG3 end to end: hydrogen from the (analytic) 1s state through the WHOLE 10-cycle 800 nm pulse at 2e14 W/cm^2,
    Taylor order 10, with the dipole-acceleration expectation logged EVERY step (BASELINE.json configs[2]: "an HHG-shaped
    output").  Feasible only with the centrifugal inner cut-off (an extension beyond the paper, tdse_set_cutoff): at
    Lambda = 300 au the stable step is about 1.4e-3 au (7.9e5 steps) instead of 4.9e-6 (2.2e8 steps)."""
    c = wl.config("cfg3", cutoff_lambda=lam)
    dt = wl.dt_eff(c)
    nsteps = int(round(c["t_pulse"] / dt))
    h = binding.Tdse(c["n_r"], c["dr"], c["n_l"], c["fd_order"])
    h.set_cutoff(lam)
    h.set_pulse(wl.pulses(c))
    h.set_state(wl.ground_state(c), stream=stream)
    h.step_taylor(c["order"], 0.0, dt, 64, 1, stream=stream)            # graphs captured before the timed run
    h.set_state(wl.ground_state(c), stream=stream)
    stream.synchronize()
    tw = time.perf_counter()
    ms = timed(torch, stream, lambda: h.step_taylor(c["order"], 0.0, dt, nsteps, 1, stream=stream))
    rows = h.obs_log()
    wall = time.perf_counter() - tw
    acc = rows[:, 0, 2]
    # harmonic content of <z''>(t): power in windows around odd and even multiples of omega (odd harmonics only)
    spec = np.abs(np.fft.rfft(acc * np.hanning(len(acc)))) ** 2
    freq = 2.0 * np.pi * np.fft.rfftfreq(len(acc), d=dt) / c["omega"]
    def band(k):
        m = (freq > k - 0.25) & (freq < k + 0.25)
        return float(spec[m].sum())
    odd, even = sum(band(k) for k in (3, 5, 7, 9)), sum(band(k) for k in (4, 6, 8, 10))
    h.close()
    return {"cutoff_lambda": lam, "dt": dt, "steps": nsteps, "wall_s": wall, "device_s": ms * 1e-3,
            "us_per_step_with_row": ms * 1e3 / nsteps, "rows_logged": int(rows.shape[0]),
            "max_norm_drift": float(np.max(np.abs(rows[:, 0, 0] - 1.0))),
            "max_abs_accel": float(np.max(np.abs(acc))), "final_dipole": float(rows[-1, 0, 1]),
            "odd_over_even_harmonic_power_3_to_10": odd / max(even, 1e-300),
            "note": "extension beyond the paper (centrifugal inner cut-off); the un-cut operator needs 2.2e8 steps"}


def roofline_sweep(binding, torch, stream, peak):
    """bare H.psi on N_r in 2^14..2^18 x L in {16, 64, 128} (up to 537 MB per array) and one
    Lanczos(8) step on the larger grids; device-generated uniform random states (bandwidth only; parity at the largest
    point is tests/test_gpu_parity.py::test_apply_H_sweep_largest)."""
    rows = []
    for L in (16, 64, 128):
        for e in (14, 15, 16, 17, 18):
            n_r = 1 << e
            pts = n_r * L
            h = binding.Tdse(n_r, 0.1, L, 3)
            x = torch.rand((1, L, n_r), dtype=torch.float64, device="cuda").to(torch.complex128)
            y = torch.empty_like(x)
            for _ in range(3):
                h.apply_H(x, y, 0.05, stream=stream)
            us = timed(torch, stream, lambda: h.apply_H(x, y, 0.05, stream=stream), 20) * 1e3
            row = {"n_r": n_r, "n_l": L, "mb_per_array": pts * 16 / 1e6, "apply_H_us": us,
                   "apply_H_frac_of_hbm": 32.0 * pts / us / 1e3 / peak}
            if pts * 16 > 60e6:
                K = 8
                h.set_pulse((0.05, 0.0, 1.0, 0.0))
                h.set_state(x, stream=stream)
                h.step_lanczos(K, 12, 0.0, 1e-6, 2, 0, stream=stream)
                ms = timed(torch, stream, lambda: h.step_lanczos(K, 12, 0.0, 1e-6, 2, 0, stream=stream))
                bpp = 32.0 + (K - 2) * 80.0 + 64.0 + (K + 1) * 16.0
                row.update({"lanczos8_us_per_step": ms * 1e3 / 2,
                            "lanczos8_frac_of_hbm": bpp * pts * 2 / (ms * 1e-3) / 1e9 / peak})
            rows.append(row)
            del x, y
            h.close()
    return rows


def respawn_under_torchrun(n):
    """`python bench.py --gpus N` without a torchrun environment: launch N ranks (one per GPU) and become them."""
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    os.environ.setdefault("NCCL_DEBUG", "INFO")           # the communicator's log (ring/NVLS choice) goes to stderr
    argv = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr",
            "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
    os.execv(sys.executable, argv)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", default="own", choices=["own", "reference"])
    ap.add_argument("--workload", default="cfg5")
    ap.add_argument("--graph-steps", type=int, default=16)
    ap.add_argument("--no-block", action="store_true", help="one kernel per Taylor order (no temporal blocking)")
    ap.add_argument("--rp-variant", type=int, default=-1, help="instantiation of the register-patch kernel")
    ap.add_argument("--rp-tma", type=int, default=-1, help="register-patch kernel: -1 auto, 0 direct loads, 1 TMA")
    ap.add_argument("--e2e-parts", type=int, default=4, help="handles / streams the end-to-end leg splits the batch over")
    ap.add_argument("--no-extra", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-full-pulse", action="store_true", help="skip the 8e5-step CFG3 run of `extra` (about 70 s)")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        respawn_under_torchrun(args.gpus)
    if args.impl == "reference":
        args.steps = 20 if args.steps is None else args.steps
        args.warmup = 3 if args.warmup is None else max(args.warmup, 0)
        run_reference(args)
    else:
        args.steps = 2000 if args.steps is None else args.steps
        args.warmup = 64 if args.warmup is None else max(args.warmup, 3)
        run_own(args)


if __name__ == "__main__":
    main()
