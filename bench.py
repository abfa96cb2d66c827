#!/usr/bin/env python
"""bench.py -- throughput of the multislice-ptychography hot path on B200.

A "step" is one pass of the whole hot path over one minibatch of synthetic input: pty_forward_loss
followed by pty_backward (object, probe and position gradients; tilt too on config 5).  Metric
(BASELINE.json): diffraction patterns/s per forward+gradient pass, plus the fraction of the
FFT-FLOP roofline of the dominant kernel.  Default workload: config 4 (128^2 detector, 12 probe
modes, 6 slices, 1088^2 object, 128x128 scan), minibatch 1024 -- the headline roofline config.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--batch B] [--impl reference]

N > 1 is launched by torchrun (one rank per GPU); each rank runs its own minibatches (weak scaling)
and the object/probe gradients are all-reduced over NCCL inside the timed step (the one real
exchange of data-parallel ptychography).
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "patterns_per_s_forward_gradient"
UNIT = "patterns/s"
FP32_LANES_PER_SM = 128      # B200: 4 SMSP x 32 FP32 lanes; 2 flops per FMA


def fft_flops_per_pattern(cfg, with_tilt):
    """Nominal 2-D FFT flops: 10 N^2 log2 N each; 4 Nz per (position, mode)."""
    n_fft = 4 * cfg.Nz * cfg.M
    return n_fft * 10.0 * cfg.N * cfg.N * math.log2(cfg.N)


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons of one GPU while the timed region runs."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu = gpu_index
        self.lines = []
        self.proc = None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "reasons": sorted(reasons), "samples": len(sm)}


def fma_peak(device=0, packed=False):
    """FP32 FMA microbenchmark (csrc/pty_bench_util.cu, bench-side helper library): achieved TFLOP/s."""
    import ctypes as C
    lib = C.CDLL(os.path.join(ROOT, "paper_2505_07814_b200", "libpty_benchutil.so"))
    lib.pty_bench_fma_peak.argtypes = [C.c_int32, C.c_int32, C.POINTER(C.c_double)]
    out = C.c_double(0.0)
    rc = lib.pty_bench_fma_peak(int(device), 1 if packed else 0, C.byref(out))
    if rc != 0:
        raise RuntimeError(f"pty_bench_fma_peak failed: {rc}")
    return out.value


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)), "measured"
        except Exception:
            pass
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "sm_max_mhz": 1965.0}, "fallback"


def oracle_per_core(oracle, ev, pos, tilt_e, meas, geom, cores):
    """The oracle on ONE core (workers = 1, a few positions): patterns/s per core and what `cores` perfectly scaling
    workers would give, so that the multi-process figure beside it can be judged."""
    m = max(1, min(3, len(pos)))
    t0 = time.perf_counter()
    oracle.grad_batch(ev["object"], ev["probe"], pos[:m], tilt_e, meas[:m], geom, workers=1)
    per_core = m / (time.perf_counter() - t0)
    return {"per_core": per_core, "positions_timed": m, "ideal_all_cores": per_core * cores}


# ------------------------------------------------------------------------------ reference arm
def run_reference(args, cfg, B):
    """--impl reference: the float64 oracle as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    from paper_2505_07814_b200 import synth
    cores = len(os.sched_getaffinity(0))
    geom = oracle.Geometry(cfg.dz, cfg.lam, cfg.dx)
    tr, ev = synth.truth(cfg), synth.eval_point(cfg, "A")
    # a bounded sample per step: the whole run (steps + warmup) is sized to about two minutes of wall time at the
    # ~4 patterns/s per core the oracle reaches on config 4 (scaled by the per-pattern cost of the other configs)
    per_pattern_s = {1: 0.003, 2: 0.05, 3: 0.11, 4: 0.22, 5: 2.2}[cfg.c]
    n = int(120.0 * cores / per_pattern_s / max(1, args.steps + args.warmup))
    n = max(cores, min(B, n))
    idx = synth.minibatch(cfg, 0, B)[:n]
    tilt_t = tr["tilt"] if cfg.tilt_mode else None
    tilt_e = ev["tilt"] if cfg.tilt_mode else None
    meas = synth.poisson_amplitudes(cfg, oracle.intensity_batch(tr["object"], tr["probe"], tr["positions"][idx],
                                                                tilt_t, geom), idx)
    pos = np.ascontiguousarray(ev["positions"][idx])
    run = lambda: oracle.grad_batch(ev["object"], ev["probe"], pos, tilt_e, meas, geom, workers=cores)
    for _ in range(args.warmup):
        run()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        run()
    dt = time.perf_counter() - t0
    value = n * args.steps / dt
    single = oracle_per_core(oracle, ev, pos, tilt_e, meas, geom, cores)
    sample = f"{n} positions of minibatch 0 of config {cfg.c} per step (of B={B}), float64 numpy, {cores} worker processes"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(cfg, B, extra={"sample": sample}),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                         "single_core": single},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def workload_config(cfg, B, extra=None):
    d = {"workload": f"c{cfg.c}: {cfg.N}x{cfg.N} detector, {cfg.M} probe modes, {cfg.Nz} slices, "
                     f"{cfg.H}x{cfg.W} object, {cfg.ns}x{cfg.ns} scan, minibatch {B}",
         "config_index": cfg.c - 1, "N": cfg.N, "M": cfg.M, "Nz": cfg.Nz, "object": [cfg.Nz, cfg.H, cfg.W],
         "minibatch": B, "n_positions": cfg.n_positions, "dose": cfg.dose, "tilt_mode": cfg.tilt_mode,
         "gradients": "object,probe,positions" + (",tilt" if cfg.tilt_mode else ""),
         "cache": "inputs larger than L2: every step reads a different minibatch and streams its saved waves "
                  "through HBM (>= several GB per step at the default size)"}
    if extra:
        d.update(extra)
    return d


def run_epoch(cfg, B, binding, synth, torch, dev, tr, ev, to):
    """Time full passes over the scan with the paper's minibatch update and constraints (see the call site)."""
    nb = cfg.n_positions // B
    flags = binding.PTY_FLAG_AMP_PHASE | binding.PTY_FLAG_STEP
    plan = binding.plan_for(cfg, Bmax=B, flags=flags, device=dev.index or 0)
    obj_t, probe_t = to(tr["object"]), to(tr["probe"])
    tilt_t = to(tr["tilt"]) if cfg.tilt_mode else None
    inten = torch.empty(B, cfg.N, cfg.N, dtype=torch.float32, device=dev)
    zeros = torch.zeros(B, cfg.N, cfg.N, dtype=torch.float32, device=dev)
    gen = torch.Generator(device=dev)
    pos, meas = [], []
    amp_t, phase_t = obj_t.abs().contiguous(), obj_t.angle().contiguous()
    for j in range(nb):                               # the whole dataset resident on the GPU, as in the paper (:524)
        idx = synth.minibatch(cfg, j, B)
        gen.manual_seed(1000 * cfg.c + 3 + 7919 * j)
        plan.forward_loss_ap(amp_t, phase_t, probe_t, to(tr["positions"][idx]), tilt_t, zeros, intensity=inten)
        meas.append(torch.sqrt(torch.poisson(inten.clamp_min(0), generator=gen)))
        pos.append(to(ev["positions"][idx]))
    del obj_t, amp_t, phase_t, inten, zeros
    obj0 = to(ev["object"])
    amp, phase = obj0.abs().contiguous(), obj0.angle().contiguous()
    probe = to(ev["probe"])
    tilt = to(ev["tilt"]) if cfg.tilt_mode else None
    plan.set_loss(1, 1.0, 0.0, 0.0, 0.1, 1e-6)
    z = lambda t: torch.zeros(t.numel() * (2 if t.is_complex() else 1), device=dev)
    state = {"m_amp": z(amp), "v_amp": z(amp), "m_phase": z(phase), "v_phase": z(phase), "m_probe": z(probe), "v_probe": z(probe)}
    pstate = [(z(p), z(p)) for p in pos]
    if tilt is not None:
        state["m_tilt"], state["v_tilt"] = z(tilt), z(tilt)
    loss = torch.zeros(1, dtype=torch.float64, device=dev)
    losses = []

    def one_epoch(e):
        tot = 0.0
        for j in range(nb):
            hp = binding.pty_adam_ap(5e-4, 5e-4, 1e-4, 5e-4, 1e-5 if tilt is not None else 0.0, 0.9, 0.999, 1e-8, e * nb + j + 1)
            st = dict(state, m_positions=pstate[j][0], v_positions=pstate[j][1])
            plan.step_ap(amp, phase, probe, pos[j], tilt, meas[j], hp, st, loss)
            losses.append(loss.clone())
        plan.constrain(amp=amp, phase=phase, probe=probe, ortho_probe=True, sigma_z=1.0 if cfg.Nz > 1 else 0.0,
                       phase_positive=True, clamp_amp=(0.98, 1.02))

    one_epoch(0)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n_timed = 2
    l0 = plan.launch_count()
    e0.record()
    for e in range(1, 1 + n_timed):
        one_epoch(e)
    e1.record()
    torch.cuda.synchronize()
    rc, _ = plan.status()
    if rc != 0:
        raise SystemExit(f"epoch: pty_status = {rc}: {plan.last_error()}")
    t_iter = e0.elapsed_time(e1) * 1e-3 / n_timed
    per_epoch = [float(torch.stack(losses[k * nb:(k + 1) * nb]).mean()) for k in range(1 + n_timed)]
    out = {"iteration_time_s": t_iter, "patterns": cfg.n_positions, "minibatch": B, "minibatches": nb,
           "patterns_per_s_full_iteration": cfg.n_positions / t_iter, "gpu_launches_per_iteration": (plan.launch_count() - l0) // n_timed,
           "update": "pty_step_ap: Eq. 9 = NRMSE + 0.1 L1 sparsity, Adam lr 5e-4 (probe 1e-4); per iteration: probe "
                     "orthogonalisation, r_z sigma_z=1, phase >= 0, amplitude in [0.98, 1.02] (PAPER.md:539)",
           "mean_loss_per_iteration": per_epoch,
           "paper_context": "PtyRAD 5.69 s per iteration at batch 1024, 12 modes x 6 slices, full A100 80 GB (Table S5, "
                            "PAPER.md:700); another GPU and software stack: context, not a comparison"}
    plan.close()
    return out


# ------------------------------------------------------------------------------ our arm
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--batch", type=int, default=None)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-epoch", action="store_true", help="skip the full-iteration (epoch) timing")
    ap.add_argument("--graph", default="auto", choices=["auto", "on", "off"],
                    help="replay each step (forward + gradient of one minibatch) as one CUDA graph; auto = on for the "
                         "launch-bound small configurations 1 and 2 on one GPU")
    ap.add_argument("--e2e-plans", type=int, default=3, help="plans / streams of the pipelined end-to-end measurement")
    ap.add_argument("--dist-backend", default="nccl", choices=["nccl", "gloo"],
                    help="torch.distributed backend for --gpus > 1; gloo (with ranks wrapping around the visible GPUs) "
                         "only exists to exercise the multi-rank code path on a box with fewer GPUs than ranks")
    ap.add_argument("--plan-flags", type=int, default=0,
                    help="extra pty_dims.flags for the timed plan (16 = PTY_FLAG_TMA_OBJECT, 32 = PTY_FLAG_PAIR_SUM): "
                         "opt-in kernel variants, reported in config.plan_flags")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl != "reference" else args.warmup

    from paper_2505_07814_b200 import synth
    cfg = synth.get_config(args.config)
    B = args.batch or cfg.B
    if args.impl == "reference":
        run_reference(args, cfg, B)
        return

    import torch
    import torch.distributed as dist
    from paper_2505_07814_b200 import build
    build.build()
    from paper_2505_07814_b200 import binding

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device; there is no CPU fallback (use --impl reference for the oracle)")
    if args.dist_backend == "gloo":
        local %= torch.cuda.device_count()
    torch.cuda.set_device(local)
    if world > 1:
        if args.dist_backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group("gloo")
    dev = torch.device("cuda", local)

    # ---- synthetic dataset: truth -> measurements (library forward + Poisson), evaluation point A
    tr, ev = synth.truth(cfg), synth.eval_point(cfg, "A")
    nb_total = max(1, cfg.n_positions // B)
    n_used = min(nb_total, args.steps + args.warmup)
    my_batches = [(rank + world * j) % nb_total for j in range(n_used)]
    want_e2e = not args.no_e2e
    plan = binding.plan_for(cfg, Bmax=B, flags=(binding.PTY_FLAG_HOST if want_e2e else 0) | args.plan_flags, device=local)
    to = lambda x: None if x is None else torch.from_numpy(np.ascontiguousarray(x)).to(dev)
    obj_t, probe_t = to(tr["object"]), to(tr["probe"])
    tilt_t = to(tr["tilt"]) if cfg.tilt_mode else None
    obj, probe = to(ev["object"]), to(ev["probe"])
    tilt = to(ev["tilt"]) if cfg.tilt_mode else None
    pos_batches, meas_batches = [], []
    inten = torch.empty(B, cfg.N, cfg.N, dtype=torch.float32, device=dev)
    gen = torch.Generator(device=dev)
    for j in my_batches:
        idx = synth.minibatch(cfg, j, B)
        gen.manual_seed(1000 * cfg.c + 3 + 7919 * j)
        zeros = torch.zeros(B, cfg.N, cfg.N, dtype=torch.float32, device=dev)
        plan.forward_loss(obj_t, probe_t, to(tr["positions"][idx]), tilt_t, zeros, intensity=inten)
        meas_batches.append(torch.sqrt(torch.poisson(inten.clamp_min(0), generator=gen)))
        pos_batches.append(to(ev["positions"][idx]))
    del obj_t, probe_t, inten, zeros

    g_obj, g_probe = torch.zeros_like(obj), torch.zeros_like(probe)
    # N ranks: one global minibatch of N * B positions per step, rank r owning rows [r B, (r + 1) B) (weak scaling), combined
    # by the library's own data-parallel host logic (parallel.sharded_gradient: one sum all-reduce of the partial
    # object / probe / tilt gradients, the loss and the position-gradient rows)
    g_pos_all = torch.zeros(world * B, 2, device=dev)
    g_pos = g_pos_all[rank * B:(rank + 1) * B]
    g_tilt = torch.zeros(2, device=dev) if cfg.tilt_mode else None
    loss = torch.zeros(1, dtype=torch.float64, device=dev)

    def step_local(i):
        j = i % n_used
        plan.forward_loss(obj, probe, pos_batches[j], tilt, meas_batches[j], loss)
        plan.backward(obj, probe, pos_batches[j], tilt, meas_batches[j], g_obj, g_probe, g_pos, g_tilt,
                      flags=binding.PTY_BWD_REUSE_FORWARD)

    def step(i):
        if world == 1:
            step_local(i)
        else:
            from paper_2505_07814_b200 import parallel
            span = parallel.sharded_gradient(lambda lo, hi: step_local(i), world * B, g_obj, g_probe, g_pos_all, g_tilt, loss)
            assert span == (rank * B, (rank + 1) * B)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    # Launch-bound small configurations: one CUDA graph per minibatch (the calls are enqueue-only, so a step can be
    # captured), replayed in the timed region -- one launch call per step instead of eight.
    use_graph = world == 1 and (args.graph == "on" or (args.graph == "auto" and cfg.c in (1, 2)))
    step_eager, graph_launches = step, 0
    if use_graph:
        step_eager(0)
        torch.cuda.synchronize()
        graphs = []
        for j in range(n_used):
            g = torch.cuda.CUDAGraph()
            lc0 = plan.launch_count()
            with torch.cuda.graph(g):
                step_eager(j)
            graph_launches = plan.launch_count() - lc0
            graphs.append(g)

        def step(i):  # noqa: F811
            graphs[i % n_used].replay()

    for i in range(args.warmup):
        step(i)
    barrier()
    rc, _ = plan.status()
    if rc != 0:
        raise SystemExit(f"pty_status = {rc}: {plan.last_error()}")
    l0 = plan.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clk:
        barrier()
        e0.record()
        for i in range(args.steps):
            step(args.warmup + i)
        e1.record()
        barrier()
        ms_total = e0.elapsed_time(e1)
        launches = graph_launches * args.steps if use_graph else plan.launch_count() - l0
        # per-kernel times for the roofline: the same steps again with the library's per-launch CUDA events on
        # (kept out of the region above: two event records per big launch matter on the launch-bound configs)
        plan.profile(True)
        for i in range(min(args.steps, 20)):
            step_eager(args.warmup + i)
        prof = plan.profile_read()
        plan.profile(False)
    if world > 1:
        t = torch.tensor([ms_total], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = t.item()
    value = world * B * args.steps / (ms_total * 1e-3)
    final_loss = loss.item()

    # ---- end to end through the host-buffer entry point (H2D of every input, D2H of loss + gradients)
    e2e = None
    if want_e2e:
        pin = lambda t: t.cpu().pin_memory()
        h_obj, h_probe = pin(obj), pin(probe)
        h_tilt = pin(tilt) if tilt is not None else None
        h_pos = [pin(p) for p in pos_batches[:3]]
        h_meas = [pin(m) for m in meas_batches[:3]]
        h_loss = torch.zeros(1, dtype=torch.float64).pin_memory()
        h_go, h_gp = torch.zeros_like(h_obj).pin_memory(), torch.zeros_like(h_probe).pin_memory()
        h_gq = torch.zeros(B, 2).pin_memory()
        h_gt = torch.zeros(2).pin_memory() if tilt is not None else None
        k_e2e = max(2, min(args.steps, 12))
        run = lambda i: plan.grad_host(h_obj, h_probe, h_pos[i % len(h_pos)], h_tilt, h_meas[i % len(h_meas)], h_loss,
                                       h_go, h_gp, h_gq, h_gt)
        run(0)
        barrier()
        t0 = time.perf_counter()
        for i in range(k_e2e):
            run(i + 1)
        torch.cuda.synchronize()
        dt_serial = time.perf_counter() - t0
        serial_loss = float(h_loss.item())
        # The same call without its final synchronisation (pty_grad_host_async / pty_grad_host_wait), two plans on two
        # streams fed alternately: the copies of one minibatch overlap the kernels of the other.  Every step still
        # copies all of its inputs host -> device and all of its results device -> host.
        NP = max(2, args.e2e_plans)
        plans = [plan] + [binding.plan_for(cfg, Bmax=B, flags=binding.PTY_FLAG_HOST | args.plan_flags, device=local)
                          for _ in range(NP - 1)]
        streams = [torch.cuda.Stream(device=dev) for _ in range(NP)]
        outs = [(h_loss, h_go, h_gp, h_gq, h_gt)] + [
            (torch.zeros(1, dtype=torch.float64).pin_memory(), torch.zeros_like(h_obj).pin_memory(),
             torch.zeros_like(h_probe).pin_memory(), torch.zeros(B, 2).pin_memory(),
             torch.zeros(2).pin_memory() if tilt is not None else None) for _ in range(NP - 1)]

        def enqueue(i):
            k = i % NP
            with torch.cuda.stream(streams[k]):
                plans[k].grad_host(h_obj, h_probe, h_pos[i % len(h_pos)], h_tilt, h_meas[i % len(h_meas)], *outs[k],
                                   wait=False)

        k_pipe = NP * max(2, min(args.steps, 24) // 2)
        for i in range(NP):
            enqueue(i)
            plans[i].grad_host_wait()
        barrier()
        t0 = time.perf_counter()
        for i in range(k_pipe):
            if i >= NP:
                plans[i % NP].grad_host_wait()        # the step that used this plan NP steps ago
            enqueue(i)
        for k in range(NP):
            plans[k].grad_host_wait()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        pipe_loss = float(outs[(k_pipe - 1) % NP][0].item())
        for q in plans[1:]:
            q.close()
        if world > 1:
            t = torch.tensor([dt, dt_serial], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt, dt_serial = t[0].item(), t[1].item()
        h2d = h_obj.numel() * 8 + h_probe.numel() * 8 + B * 8 + B * cfg.N * cfg.N * 4 + (8 if tilt is not None else 0)
        d2h = 8 + h_go.numel() * 8 + h_gp.numel() * 8 + B * 8 + (8 if tilt is not None else 0)
        e2e = {"value": world * B * k_pipe / dt, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "steps": k_pipe,
               "api": f"pty_grad_host_async + pty_grad_host_wait (pinned host buffers; {NP} plans on {NP} streams fed in "
                      "turn: the copies of one minibatch overlap the kernels of another)",
               "loss": pipe_loss,
               "serial": {"value": world * B * k_e2e / dt_serial, "steps": k_e2e, "loss": serial_loss,
                          "api": "pty_grad_host, one call after the other"}}

    # ---- one full "iteration" in the paper's sense: every pattern of the scan once, minibatch by
    # minibatch, with the paper's update (pty_step_ap: Eq. 9 = NRMSE + 0.1 L1 sparsity, Adam on amplitude, phase,
    # probe, positions with lr 5e-4 / 1e-4 for the probe) and its per-iteration constraints
    # (orthogonalisation, r_z filter sigma_z = 1, phase positivity, amplitude clamp [0.98, 1.02]).  Context for
    # Table S5 (5.69 s per iteration at batch 1024 on an A100), not the headline metric.
    epoch = None
    if world == 1 and not args.no_epoch and cfg.n_positions % B == 0:
        epoch = run_epoch(cfg, B, binding, synth, torch, dev, tr, ev, to)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (FP32 ALU bound)
    peaks, peaks_src = load_peaks()
    clocks = clk.summary()
    sm_max = clocks.get("sm_max_mhz") or peaks.get("sm_max_mhz", 1965.0)
    n_sms = torch.cuda.get_device_properties(local).multi_processor_count
    peak_tf = n_sms * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    flops_launch = 0.5 * fft_flops_per_pattern(cfg, cfg.tilt_mode) * B     # each kernel does 2 Nz M FFTs / pattern
    kern = {}
    for name in ("fwd", "bwd"):
        ms, n = prof[name]
        if n:
            kern[name] = {"avg_ms": ms / n, "launches": n, "tflops": flops_launch / (ms / n * 1e-3) / 1e12}
    dom = max(kern, key=lambda k: kern[k]["avg_ms"]) if kern else None
    roofline = None
    fma_scalar = fma_peak(local, packed=False)     # measured FP32 FMA rate on this GPU, after the timed region
    fma_packed = fma_peak(local, packed=True)
    if dom:
        a = kern[dom]["tflops"]
        roofline = {"bound": "alu", "kernel": (f"pty_{dom}128g2_kernel" if cfg.N == 128 else f"pty_{dom}_kernel<Shape<{cfg.N}>>"), "achieved": a, "peak": peak_tf,
                    "unit": "TFLOP/s", "frac": a / peak_tf, "traffic": None,
                    "peak_source": f"{n_sms} SMs x 128 FP32 lanes x 2 flop x clocks.max.sm {sm_max:.0f} MHz "
                                   "(nominal FP32 FMA peak; HBM is not the bound, DESIGN.md)",
                    "peak_measured_fma": {"scalar_ffma_tflops": fma_scalar, "packed_ffma2_tflops": fma_packed,
                                          "frac_of_measured": a / max(fma_scalar, fma_packed),
                                          "how": "libpty_benchutil.so: independent FFMA / FFMA2 chains on every SM"},
                    "algorithmic_flops_per_launch": flops_launch, "avg_launch_ms": kern[dom]["avg_ms"],
                    "kernels": kern,
                    "whole_step_frac_of_fft_roofline": value * fft_flops_per_pattern(cfg, 0) / world / 1e12 / peak_tf,
                    "hbm_peak_gbs": peaks.get("hbm_gbs"), "peaks": peaks_src}
        tp = os.path.join(ROOT, "profiles", "traffic.json")
        if os.path.exists(tp):
            try:
                roofline["traffic"] = json.load(open(tp)).get(f"c{cfg.c}_B{B}_{dom}")
                if roofline["traffic"] is not None:
                    roofline["traffic_source"] = ("stored figure, not measured by this run: dram__bytes_read.sum + "
                                                  "dram__bytes_write.sum of one `ncu --set full` capture of this kernel "
                                                  "(profiles/traffic.json)")
            except Exception:
                pass

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": workload_config(cfg, B, extra=dict(({"plan_flags": args.plan_flags} if args.plan_flags else {}),
                                                         **({"cuda_graph": "one graph per step (forward + gradient), replayed"} if use_graph else {}))),
           "clocks": clocks, "gpu_launches": int(launches), "roofline": roofline, "loss": final_loss}
    if e2e:
        out["e2e"] = e2e
    if epoch:
        out["epoch"] = epoch

    # ---- the oracle timed on this box's host cores (a reported baseline, not the target)
    if world == 1 and not args.no_cpu_baseline:
        import oracle
        cores = len(os.sched_getaffinity(0))
        geom = oracle.Geometry(cfg.dz, cfg.lam, cfg.dx)
        # ~ 15 s of wall time: measured 0.22 s per pattern per worker on config 4 (16 workers: 4.6 patterns/s)
        per_pattern_s = {1: 0.003, 2: 0.05, 3: 0.11, 4: 0.22, 5: 2.2}[cfg.c]
        n = int(max(cores, min(B, round(15.0 * cores / per_pattern_s))))
        idx = synth.minibatch(cfg, 0, B)[:n]
        tilt_tr = tr["tilt"] if cfg.tilt_mode else None
        tilt_ev = ev["tilt"] if cfg.tilt_mode else None
        meas = synth.poisson_amplitudes(cfg, oracle.intensity_batch(tr["object"], tr["probe"], tr["positions"][idx],
                                                                    tilt_tr, geom), idx)
        pos = np.ascontiguousarray(ev["positions"][idx])
        t0 = time.perf_counter()
        ref = oracle.grad_batch(ev["object"], ev["probe"], pos, tilt_ev, meas, geom, workers=cores)
        dt = time.perf_counter() - t0
        out["cpu_baseline"] = {"value": n / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                               "sample": f"{n} positions of minibatch 0 (of B={B}), forward + all gradients, float64 "
                                         f"numpy, {cores} worker processes, {dt:.1f} s (one cold call incl. process-pool "
                                         "start-up; the --impl reference arm repeats smaller calls)",
                               "single_core": oracle_per_core(oracle, ev, pos, tilt_ev, meas, geom, cores)}
        # parity of the very launch shape that was timed, on the sample the oracle just computed (outside every
        # timed region): loss 1e-4, gradients 1e-3 relative L2 (BASELINE.json north_star)
        dm, dp = to(meas), to(pos)
        gl = plan.forward_loss(obj, probe, dp, tilt, dm).item()
        go, gpr, gq = torch.zeros_like(obj), torch.zeros_like(probe), torch.zeros(n, 2, device=dev)
        gt = torch.zeros(2, device=dev) if cfg.tilt_mode else None
        plan.backward(obj, probe, dp, tilt, dm, go, gpr, gq, gt, flags=binding.PTY_BWD_REUSE_FORWARD)
        rel = lambda x, r: float(np.linalg.norm(np.ravel(x - r)) / max(np.linalg.norm(np.ravel(r)), 1e-300))
        par = {"n": n, "loss_rel": abs(gl - ref["loss"]) / ref["loss"],
               "g_object": rel(go.cpu().numpy(), ref["g_object"]), "g_probe": rel(gpr.cpu().numpy(), ref["g_probe"]),
               "g_positions": rel(gq.cpu().numpy(), ref["g_positions"])}
        if cfg.tilt_mode:
            par["g_tilt"] = rel(gt.cpu().numpy(), ref["g_tilt"].sum(0))
        out["parity_vs_oracle"] = par
        assert par["loss_rel"] <= 1e-4 and all(v <= 1e-3 for k, v in par.items() if k.startswith("g_")), par
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
