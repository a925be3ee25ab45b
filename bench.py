#!/usr/bin/env python
"""bench.py — one JSON line for the batched local-energy path (BASELINE.json metric: local energies/s and
connected-amplitude evaluations/s, with the fraction of the binding roofline).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--impl ours|reference]

A "step" is one pass of the whole hot path (pack, theta contraction, ln psi, fused local energy, statistics) over
one synthetic batch of BASELINE.json configs[--config - 1]; default config 5, the largest single-GPU workload
(65536 samples, N = 1024, chunks of 4096).  Under torchrun (N > 1) every rank processes its own batch (weak
scaling; the only exchange is an all-gather of the 4-double statistics).
"""
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

CONFIG_TEXT = {
    1: "configs[0]: 1D Heisenberg L=10, real RBM alpha=1, 1024 samples",
    2: "configs[1]: 2D Heisenberg 10x10, real RBM alpha=1, 4096 samples",
    3: "configs[2]: 2D TFIM 20x20 h=3, real RBM alpha=2, 8192 samples",
    4: "configs[3]: 2D J1-J2 10x10, complex RBM alpha=4, 16384 samples",
    5: "configs[4]: 2D Heisenberg 32x32, real RBM alpha=2, 65536 samples in chunks of 4096",
    6: "widening case, not a BASELINE.json config: 2D Heisenberg 32x32, real RBM alpha=4 (M = 4096, the width limit), "
       "16384 samples in chunks of 4096",
}

N_SMS = 148


def measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md clocks line): one
    `nvidia-smi -lms` process streaming a line every 20 ms."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.proc = index, [], None

    def run(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                f = [x.strip() for x in line.strip().split(",")]
                if len(f) >= 7:
                    self.rows.append(f)
        except Exception:
            pass

    def summary(self):
        if self.proc is not None:
            self.proc.terminate()
        self.join(timeout=6)
        rows = []
        for r in self.rows:
            try:
                rows.append((float(r[0]), float(r[1]), float(r[2]), r[3:7]))
            except ValueError:
                pass
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        busy = [r for r in rows if r[2] > 0.6 * max(x[2] for x in rows)] or rows     # samples taken under load
        sm = sorted(r[0] for r in busy)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[3][i].lower().startswith("active") for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": rows[0][1], "reasons": reasons, "samples": len(rows),
                "samples_under_load": len(busy), "power_w_max": max(r[2] for r in rows)}


def oracle_rate(p, n_rows, repeat=1):
    """Times the float64 oracle (as it stands) on the first n_rows samples; returns (local energies/s, seconds)."""
    from oracle import nk_oracle as orc
    t0 = time.perf_counter()
    for _ in range(repeat):
        orc.local_energy(p.kind, p.sigma[:n_rows], p.bonds, p.colors, p.J, p.h, p.W, p.a, p.b)
    dt = time.perf_counter() - t0
    return n_rows * repeat / dt, dt


def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [i.get("num_threads", 1) for i in threadpool_info() if i.get("user_api") == "blas"]
        return max(n) if n else 1
    except Exception:
        return os.cpu_count() or 1


ORACLE_ROWS_PER_STEP = {1: 1024, 2: 256, 3: 16, 4: 64, 5: 4, 6: 2}


def run_reference(args):
    """--impl reference: the oracle on the host cores, same config / metric; each step is a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import nk_oracle as orc
    from paper_2112_10526_b200 import inputs as inp
    n = ORACLE_ROWS_PER_STEP[args.config]
    p = inp.make_config(args.config, n_samples=n)
    for _ in range(args.warmup):
        oracle_rate(p, n)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_rate(p, n)
    dt = time.perf_counter() - t0
    rate = n * args.steps / dt
    amps = orc.count_amplitudes(p.kind, p.sigma, p.bonds, p.colors, p.J, p.h) / n
    sample = f"first {n} samples of the batch per step (work is linear in samples)"
    line = {"impl": "reference", "metric": "local_energies_per_sec", "value": rate, "unit": "local energies/s",
            "amplitudes_per_sec": rate * amps, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic (seeded, BASELINE.json recipe)",
            "config": {"workload": CONFIG_TEXT[args.config], "sample": sample},
            "cpu_baseline": {"value": rate, "unit": "local energies/s", "cores": blas_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": rate, "unit": "local energies/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def _time_ms(torch, fn, reps):
    fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


def time_extras(nk, torch, p, op, sigma, W, a, b, dt_code, plan):
    """One Metropolis sweep (N transitions per chain, n_chains = n_samples; exchange rule on the lattice bonds for
    the Heisenberg configs, local rule for TFIM) and one energy-gradient call on the bench batch."""
    from paper_2112_10526_b200 import inputs as inp
    B, N, M = p.n_samples, p.n_sites, p.n_hidden
    lib = nk.load()
    exch = p.kind == inp.KIND_HEISENBERG
    rule = nk.NK_RULE_EXCHANGE if exch else nk.NK_RULE_LOCAL
    clusters = p.bonds if exch else None
    chains = sigma.clone()
    ws = torch.empty(lib.nk_metropolis_workspace_bytes(rule, len(p.bonds) if exch else 0, B, N, M, dt_code, 0),
                     dtype=torch.uint8, device=sigma.device)
    acc = [None]
    sweep = [0]

    def one_sweep():
        acc[0] = nk.metropolis_sample(chains, W, a, b, rule=rule, clusters=clusters, n_steps=N, seed=1,
                                      step_offset=sweep[0] * N, ws=ws)
        sweep[0] += 1

    ms_sweep = _time_ms(torch, one_sweep, 3)
    acceptance = float(acc[0].double().mean().item()) / N
    # a transition that proposes s' = s (exchange of equal spins) evaluates nothing; count the evaluated ones
    if exch:
        anti = (chains[:, torch.from_numpy(p.bonds[:, 0]).to(chains.device).long()] !=
                chains[:, torch.from_numpy(p.bonds[:, 1]).to(chains.device).long()]).double().mean().item()
    else:
        anti = 1.0
    pairs = B * N * anti * M
    eloc, _, stats = plan.run(chains, W, a, b)
    # the contractions over the samples take the whole batch as one chunk (the library default; ~1 GB of workspace at
    # config 5): one launch of each kernel instead of B / chunk_size read-modify-write passes over the accumulator
    gchunk = 0
    gws = torch.empty(lib.nk_energy_gradient_workspace_bytes(B, N, M, dt_code, gchunk), dtype=torch.uint8,
                      device=sigma.device)
    ms_grad = _time_ms(torch, lambda: nk.energy_gradient(chains, W, b, eloc, stats, chunk_size=gchunk, ws=gws), 3)
    ms_eloc = _time_ms(torch, lambda: plan.run(chains, W, a, b), 3)
    # QGT-vector product (one CG iteration of stochastic reconfiguration is this plus 4 vector kernels)
    ga, gb, gW = nk.energy_gradient(chains, W, b, eloc, stats, chunk_size=gchunk, ws=gws)
    qws = torch.empty(lib.nk_qgt_matvec_workspace_bytes(B, N, M, dt_code, gchunk), dtype=torch.uint8,
                      device=sigma.device)
    qout = (torch.empty_like(ga), torch.empty_like(gb), torch.empty_like(gW))
    ms_qgt = _time_ms(torch, lambda: nk.qgt_matvec(chains, W, b, ga, gb, gW, diag_shift=0.01,
                                                   chunk_size=gchunk, ws=qws, out=qout), 3)
    # one conjugate-gradient iteration of the SR solve (theta and the spin conversions are cached across iterations)
    sws = torch.empty(lib.nk_sr_solve_workspace_bytes(B, N, M, dt_code, gchunk), dtype=torch.uint8,
                      device=sigma.device)
    n_cg = 8
    ms_sr = _time_ms(torch, lambda: nk.sr_solve(chains, W, b, ga, gb, gW, diag_shift=0.01, tol=0.0, max_iter=n_cg,
                                                chunk_size=gchunk, ws=sws), 2)
    planes = 2 if p.complex_params else 1
    return {
        "sampler": {"rule": "exchange" if exch else "local", "chains": B, "transitions_per_chain": N,
                    "ms_per_sweep": ms_sweep, "transitions_per_sec": B * N / (ms_sweep * 1e-3), "acceptance": acceptance,
                    "evaluated_fraction_estimate": anti,
                    "roofline": {"bound": "alu", "kernel": "metropolis_kernel", "unit": "Gpair/s",
                                 "achieved": pairs / (ms_sweep * 1e-3) / 1e9}},
        "gradient": {"ms": ms_grad, "chunk_size": "whole batch", "algorithmic_tflops": 2.0 * planes * B * M * N / (ms_grad * 1e-3) / 1e12},
        "qgt_matvec": {"ms": ms_qgt, "n_parameters": N + M + M * N,
                       "algorithmic_tflops": 3 * 2.0 * planes * B * M * N / (ms_qgt * 1e-3) / 1e12,
                       "what": "(G + 0.01) v on the fly, Eq. (75): theta, V_W sigma and J^dagger dw contractions"},
        "sr_solve": {"cg_iterations": n_cg, "ms": ms_sr, "ms_per_cg_iteration": ms_sr / n_cg,
                     "what": "nk_sr_solve with tol = 0: setup (theta of the batch, spin conversions) + 8 CG iterations"},
        "vmc_iteration": {"ms": ms_sweep + ms_eloc + ms_grad, "ms_local_energy_on_sampled_chains": ms_eloc,
                          "what": "one sweep + local energies + energy gradient, same batch, device-resident"},
    }


def time_form(nk, torch, p, op, tensors, dt_code, form_flag, reps):
    """One forced form of the amplitude ratios (nk_local_energy_ex flag) on the bench batch: (ms per step, ms of the
    local-energy phase per step, ms of the series GEMM kernel per step), per-kernel times from the library's brackets."""
    sigma, W, a, b = tensors
    B, N, M = p.n_samples, p.n_sites, p.n_hidden
    plan = nk.LocalEnergyPlan(op, B, N, M, dt_code, p.chunk_size, device=sigma.device, flags=form_flag)
    plan.run(sigma, W, a, b)
    torch.cuda.synchronize()
    nk.profile_enable(True)
    nk.profile_read()
    ms = _time_ms(torch, lambda: plan.run(sigma, W, a, b), reps)
    ph = nk.profile_read()
    nk.profile_enable(False)
    n = reps + 1                                           # _time_ms runs the call 1 + reps times
    return ms, ph["fused"][0] / n, ph["series_gemm"][0] / n


def traffic_record(kernel_key, config):
    """dram bytes per launch of a kernel from its committed `ncu --set full` capture (profiles/r02_traffic.json:
    {kernel: {"cfg<k>": {"bytes": read + write, "capture": tag}}}); None when no capture of this kernel / config exists."""
    try:
        rec = json.load(open(os.path.join(ROOT, "profiles", "r02_traffic.json")))[kernel_key][f"cfg{config}"]
        return float(rec["bytes"]), rec.get("capture")
    except Exception:
        return None, None


def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_2112_10526_b200 as nk
    from paper_2112_10526_b200 import inputs as inp

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit(f"bench.py --gpus {args.gpus} running with WORLD_SIZE={world}: launch one rank per GPU")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback for the product path")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    nk.load()

    p = inp.make_config(args.config, sample_seed_offset=rank)           # weak scaling: own batch per rank
    B, N, M = p.n_samples, p.n_sites, p.n_hidden
    dt_code = nk.NK_C64 if p.complex_params else nk.NK_F32
    op = nk.Operator.from_problem(p)
    sigma_h = torch.from_numpy(p.sigma).pin_memory()
    W_h, a_h, b_h = (torch.from_numpy(x).pin_memory() for x in (p.W, p.a, p.b))
    sigma, W, a, b = (t.to(dev) for t in (sigma_h, W_h, a_h, b_h))
    plan = nk.LocalEnergyPlan(op, B, N, M, dt_code, p.chunk_size, device=dev)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)         # > 126 MB L2
    gathered = [torch.zeros(4, dtype=torch.float64, device=dev) for _ in range(world)]

    # the graded call: nk_local_energy_plan_run — the launches of nk_local_energy captured once into a CUDA graph by the
    # library (nk_local_energy_plan_create) and replayed per step, every kernel of the step included (--call eager times
    # nk_local_energy itself; the other one is reported beside it)
    def call(planned):
        return plan.run_graph(sigma, W, a, b) if planned else plan.run(sigma, W, a, b)

    def step(planned=(args.call == "plan")):
        _, _, stats = call(planned)
        if world > 1:
            dist.all_gather(gathered, stats)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()

    # ---- device-resident timing: K steps, per-step CUDA events, L2 flushed between steps -------------------
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    sampler = ClockSampler(local_rank)
    sampler.start()
    nk.launch_count(reset=True)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    for s in range(args.steps):
        flush.zero_()
        ev[s][0].record()
        step()
        ev[s][1].record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    launches = nk.launch_count(reset=True)
    step_ms = [a_.elapsed_time(b_) for a_, b_ in ev]
    # the other way of making the call, same protocol, fewer steps
    other_planned = args.call != "plan"
    for _ in range(3):
        step(other_planned)
    torch.cuda.synchronize()
    other_ms = 0.0
    n_other = max(3, min(args.steps, 20))
    oe = (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
    for _ in range(n_other):
        flush.zero_()
        oe[0].record()
        step(other_planned)
        oe[1].record()
        torch.cuda.synchronize()
        other_ms += oe[0].elapsed_time(oe[1])
    other_ms /= n_other
    # the same K steps once more with the library's per-kernel CUDA-event brackets on (nk_profile_enable): the kernel
    # durations behind `roofline`.  Kept out of the loop above because the brackets themselves cost timeline (two event
    # records per kernel group and chunk); the clock sampler covers both loops.
    # Two such loops: (a) the call exactly as graded — the preparation of chunk c + 1 overlaps the tensor-core kernel of
    # chunk c on a second stream, so a bracket also spans time in which its kernel shares or waits for SMs;
    # (b) NK_SERIAL_CHUNKS, every kernel alone on the stream: the durations `roofline` divides by.
    nk.profile_enable(True)
    nk.profile_read()
    prof_ev = (torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))

    def profiled_loop(pl):
        total = 0.0
        for _ in range(args.steps):
            flush.zero_()
            prof_ev[0].record()
            pl.run(sigma, W, a, b)
            prof_ev[1].record()
            torch.cuda.synchronize()
            total += prof_ev[0].elapsed_time(prof_ev[1])
        return total, nk.profile_read()

    prof_ms_overlap, phases_overlap = profiled_loop(plan)
    splan = nk.LocalEnergyPlan(op, B, N, M, dt_code, p.chunk_size, device=dev, flags=nk.NK_SERIAL_CHUNKS)
    splan.run(sigma, W, a, b)
    torch.cuda.synchronize()
    nk.profile_read()
    prof_ms, phases = profiled_loop(splan)
    clocks = sampler.summary()
    nk.profile_enable(False)
    total_ms = float(sum(step_ms))
    t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms = float(t.item())
    ms_per_step = total_ms / args.steps

    # ---- end to end through the host-buffer C call (pinned inputs, H2D + D2H inside the timed region) -------
    hplan = nk.HostPlan(op, B, N, M, dt_code, p.chunk_size, device=dev)
    cdt = torch.complex64 if p.complex_params else torch.float32
    out = (torch.empty(B, dtype=cdt).pin_memory().numpy(), torch.empty(B, dtype=cdt).pin_memory().numpy(),
           torch.empty(4, dtype=torch.float64).pin_memory().numpy())
    host_args = (sigma_h.numpy(), W_h.numpy(), a_h.numpy(), b_h.numpy())
    for _ in range(2):
        nk.local_energy_host(op, *host_args, chunk_size=p.chunk_size, plan=hplan, out=out)
    e2e_steps = max(3, min(args.steps, 10))
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(e2e_steps):
        nk.local_energy_host(op, *host_args, chunk_size=p.chunk_size, plan=hplan, out=out)
    e1.record()
    torch.cuda.synchronize()
    t = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    e2e_ms = float(t.item()) / e2e_steps
    esz = 8 if p.complex_params else 4
    h2d = B * N + (M * N + N + M) * esz
    d2h = 2 * B * esz + 32

    # ---- the neighbouring steps of a VMC iteration, timed apart from the step above ----
    extras = None
    if rank == 0 and not args.no_extras:
        extras = time_extras(nk, torch, p, op, sigma, W, a, b, dt_code, plan)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- accounting -----------------------------------------------------------------------------------------
    anti = p.sigma[:, p.bonds[:, 0]] != p.sigma[:, p.bonds[:, 1]]
    if p.kind == inp.KIND_HEISENBERG:
        amps = int(anti[:, p.J[p.colors] != 0].sum())
        n_rows = len(p.bonds)
    else:
        amps = B * N if p.h != 0 else 0
        n_rows = N
    pairs = amps * M                                                     # (amplitude, hidden unit) evaluations
    fused_ms, fused_n = phases["fused"]
    fused_ms_per_step = fused_ms / args.steps
    peaks = measured_peaks()
    sm_max = float(clocks.get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0)
    ghz = sm_max * 1e-3
    cplx = p.complex_params
    # measured pipe peaks of this box (nk_pipe_peaks: MUFU.EX2-only, FFMA-only, LDS.128-only kernels)
    pk = nk.pipe_peaks(dev)
    mufu_lanes, ffma_lanes, lds_bytes = pk["mufu_lanes_per_clk_sm"], pk["ffma_lanes_per_clk_sm"], pk["lds_bytes_per_clk_sm"]
    pair_peak_mufu = N_SMS * mufu_lanes * ghz / (3 if cplx else 1)       # Gpair/s: 1 exponential per real pair (3 complex)
    pair_peak_mufu2 = N_SMS * mufu_lanes * ghz / 2                       # SURVEY.md 8(d)'s denominator: ex2 + lg2 per pair
    pair_peak_fp32 = N_SMS * ffma_lanes * ghz / (8 if cplx else 2)       # product form: 2 FP32 operations per real pair
    pair_peak_smem = N_SMS * lds_bytes * ghz / (8 if cplx else 4)        # product form: 4 B of the table per real pair
    peak_basis = (f"measured on this box by nk_pipe_peaks: MUFU.EX2 {mufu_lanes:.2f} lanes/clk/SM, FFMA {ffma_lanes:.1f} "
                  f"lanes/clk/SM, LDS.128 {lds_bytes:.1f} B/clk/SM; x {N_SMS} SMs x {sm_max:.0f} MHz (clocks.max.sm)")
    form, tau_max = plan.form()
    terms = getattr(plan, "series_terms", 0)
    ach_pairs = pairs / (fused_ms_per_step * 1e-3) / 1e9 if fused_ms_per_step > 0 else 0.0
    bf16_burst = float(peaks.get("bf16_tflops") or 1590.0)
    bf16_sust = float(peaks.get("bf16_tflops_sustained") or 1400.0)
    peak_src = "MEASURED_PEAKS.json (of measured)" if peaks.get("bf16_tflops") else "B200_PROFILING.md fallback (of fallback)"
    common = {"form": {nk.NK_FORM_SERIES: "series", nk.NK_FORM_PRODUCT: "product"}.get(form, "logcosh"),
              "tau_max": tau_max, "pairs_per_step": pairs,
              "pair_rate_gpair_s": ach_pairs, "frac_fp32": ach_pairs / pair_peak_fp32,
              "frac_fp32_basis": "pairs / time of the whole local-energy phase against the FP32-pipe pair roof "
                                 "(2 FP32 operations per (amplitude, hidden unit) pair; SURVEY.md 7 / 8(f)3)",
              "phase_ms_per_step": {k: v[0] / args.steps for k, v in phases.items()},
              "measured_in": f"a loop of {args.steps} steps with the per-kernel event brackets on and NK_SERIAL_CHUNKS (every "
                             f"kernel alone on the stream), {prof_ms / args.steps:.4f} ms per step there; the graded loop "
                             "runs without brackets and overlaps the preparation of the next chunk on a second stream",
              "phase_ms_per_step_overlapped": {k: v[0] / args.steps for k, v in phases_overlap.items()},
              "ms_per_step_overlapped_with_brackets": prof_ms_overlap / args.steps,
              "pipe_peaks": pk}
    if form == nk.NK_FORM_SERIES:
        # tensor-core series form: the dominant kernel is series_gemm_kernel; work = the K + 2 fp16 / bf16 MMA passes of
        # the series over [samples] x [table rows] x [hidden units], peak = measured dense bf16
        g_ms, g_n = phases["series_gemm"]
        flop = 2.0 * B * n_rows * M * (terms + 2)
        ach = flop / (g_ms / args.steps * 1e-3) / 1e12 if g_ms > 0 else 0.0
        traffic, tag = traffic_record("series_gemm_kernel", args.config)
        roofline = {"bound": "tensor", "kernel": "series_gemm_kernel (tcgen05 kind::f16, fp16 hi/lo + bf16 passes)",
                    "series_terms": terms, "mma_passes": terms + 2, "achieved": ach, "peak": bf16_burst,
                    "unit": "TFLOP/s", "frac": ach / bf16_burst, "frac_of_sustained_peak": ach / bf16_sust,
                    "peak_basis": f"{peak_src}: dense bf16 cuBLAS {bf16_burst:.0f} burst / {bf16_sust:.0f} sustained; "
                                  "fp16 and bf16 share the rate",
                    "flop_per_launch": flop / (g_n / args.steps) if g_n else None,
                    "traffic": traffic, "traffic_capture": tag,
                    "ms_per_launch": g_ms / g_n if g_n else None, "launches_per_step": g_n / args.steps}
    elif form == nk.NK_FORM_PRODUCT:
        traffic, tag = traffic_record("fused_eloc_kernel_product", args.config)
        roofline = {"bound": "smem", "kernel": "fused_eloc_kernel<V, CPLX, PROD=true>", "achieved": ach_pairs,
                    "peak": pair_peak_smem, "unit": "Gpair/s", "frac": ach_pairs / pair_peak_smem,
                    "peak_basis": peak_basis + "; 4 B of the tanh(delta) table per pair through LDS.128 (DESIGN.md 13)",
                    "traffic": traffic, "traffic_capture": tag,
                    "ms_per_launch": fused_ms / fused_n if fused_n else None, "launches_per_step": fused_n / args.steps}
    else:
        traffic, tag = traffic_record("fused_eloc_kernel_logcosh", args.config)
        roofline = {"bound": "alu", "kernel": "fused_eloc_kernel<V, CPLX, PROD=false>", "achieved": ach_pairs,
                    "peak": pair_peak_mufu, "unit": "Gpair/s", "frac": ach_pairs / pair_peak_mufu,
                    "peak_basis": peak_basis + f"; {3 if cplx else 1} MUFU per pair (DESIGN.md 6.1)",
                    "traffic": traffic, "traffic_capture": tag,
                    "ms_per_launch": fused_ms / fused_n if fused_n else None, "launches_per_step": fused_n / args.steps}
    roofline.update(common)
    if clocks.get("sm_mhz"):
        roofline["sm_mhz_under_load"] = clocks["sm_mhz"]

    # the kernel BASELINE.json north_star (3) describes — the fused log-cosh kernel — and the SIMT product form, each
    # forced on the same batch (a few steps, after the graded loop): they survive in the driver-parsed line
    tensors = (sigma, W, a, b)
    ms_l, fused_l, _ = time_form(nk, torch, p, op, tensors, dt_code, nk.NK_FORM_LOGCOSH, 3)
    gp = pairs / (fused_l * 1e-3) / 1e9
    roofline["logcosh"] = {"kernel": "fused_eloc_kernel<V, CPLX, PROD=false>", "bound": "alu", "ms_per_step": ms_l,
                           "fused_ms_per_step": fused_l, "local_energies_per_sec": B / (ms_l * 1e-3),
                           "achieved": gp, "unit": "Gpair/s", "peak": pair_peak_mufu, "frac": gp / pair_peak_mufu,
                           "frac_2mufu": gp / pair_peak_mufu2,
                           "peak_basis": f"measured MUFU.EX2 {mufu_lanes:.2f} lanes/clk/SM x {N_SMS} SMs x {sm_max:.0f} MHz; "
                                         f"frac: {3 if cplx else 1} MUFU per pair (what the kernel issues), frac_2mufu: "
                                         "SURVEY.md 8(d)'s 2 MUFU per pair"}
    if not cplx:
        ms_p, fused_p, _ = time_form(nk, torch, p, op, tensors, dt_code, nk.NK_FORM_PRODUCT, 3)
        gp = pairs / (fused_p * 1e-3) / 1e9
        roofline["product_simt"] = {"kernel": "fused_eloc_kernel<V, CPLX, PROD=true>", "bound": "smem", "ms_per_step": ms_p,
                                    "fused_ms_per_step": fused_p, "local_energies_per_sec": B / (ms_p * 1e-3),
                                    "achieved": gp, "unit": "Gpair/s", "peak": pair_peak_smem,
                                    "frac": gp / pair_peak_smem, "frac_fp32": gp / pair_peak_fp32}

    # theta contraction: second roofline, tensor pipe.  Algorithmic work 2 B M N flop per step (x 2
    # planes for complex W); the kernel executes three int8 digit-plane MMAs per product (the exact fixed-point
    # split), so the tensor pipe sees 3 x that in int8 operations.  Peak: measured dense bf16 (burst) x 2 — the nominal
    # fp8 / int8 : bf16 ratio of the 5th-generation tensor cores (4.5 : 2.25 PFLOP/s dense; the guide lists fp8).
    th_ms, th_n = phases["theta"]
    alg_flop = 2.0 * B * M * N * (2 if cplx else 1)
    if th_ms > 0:
        th_s = th_ms / args.steps * 1e-3
        roofline["theta"] = {
            "bound": "tensor", "kernel": "theta_tc_kernel<I8> (tcgen05 kind::i8, 3 digit planes)",
            "achieved": 3.0 * alg_flop / th_s / 1e12, "peak": 2.0 * bf16_burst, "unit": "TOP/s (int8, executed)",
            "frac": 3.0 * alg_flop / th_s / 1e12 / (2.0 * bf16_burst),
            "algorithmic_tflops": alg_flop / th_s / 1e12,
            "frac_of_tf32_peak_algorithmic": alg_flop / th_s / 1e12 / (0.5 * bf16_burst),
            "peak_basis": f"{peak_src} bf16 burst x 2 (nominal fp8 / int8 : bf16 = 4.5 : 2.25 PFLOP/s dense); tf32 = bf16 / 2",
            "ms_per_launch": th_ms / th_n if th_n else None, "launches_per_step": th_n / args.steps}

    # CPU baselines on the box's host cores: (i) the from-scratch oracle as it stands on a bounded sample worth ~12 s
    # (a short probe sizes it); (ii) the separately written incremental float64 route (oracle/nk_incremental.c)
    n0 = min(ORACLE_ROWS_PER_STEP[args.config], B)
    rate0, t0 = oracle_rate(p, n0)
    want = 12.0
    n_or = int(min(B, max(n0, n0 * want / max(t0, 1e-6))))
    rep = int(max(1, min(200, want / max(t0 * n_or / n0, 1e-6)))) if n_or == B else 1
    cpu_rate, cpu_s = oracle_rate(p, n_or, repeat=rep)
    cpu = {"value": cpu_rate, "unit": "local energies/s", "cores": blas_threads(), "kind": "oracle",
           "sample": f"first {n_or} samples of the batch" + (f", {rep} passes" if rep > 1 else "") +
                     f", {cpu_s:.1f} s (work is linear in samples)",
           "host_cpus": os.cpu_count()}
    try:
        from oracle import nk_incremental as inc
        n_in = min(B, 64)
        t1 = time.perf_counter()
        inc.local_energy(p.kind, p.sigma[:n_in], p.bonds, p.colors, p.J, p.h, p.W, p.a, p.b)
        dt1 = max(time.perf_counter() - t1, 1e-6)
        n_in2 = int(min(B, max(n_in, n_in * 8.0 / dt1)))
        t1 = time.perf_counter()
        inc.local_energy(p.kind, p.sigma[:n_in2], p.bonds, p.colors, p.J, p.h, p.W, p.a, p.b)
        dt2 = time.perf_counter() - t1
        cpu["incremental"] = {"value": n_in2 / dt2, "unit": "local energies/s", "cores": inc.num_threads(),
                              "kind": "oracle (incremental float64 route, oracle/nk_incremental.c)",
                              "sample": f"first {n_in2} samples of the batch, {dt2:.1f} s"}
    except Exception as exc:                                              # no C compiler on the box: report, do not fail
        cpu["incremental"] = {"unavailable": str(exc)[:200]}

    value = world * B / (ms_per_step * 1e-3)
    line = {"metric": "local_energies_per_sec", "value": value, "unit": "local energies/s",
            "amplitudes_per_sec": world * amps / (ms_per_step * 1e-3), "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "c64" if cplx else "f32",
            "data": "synthetic (seeded, BASELINE.json recipe)",
            "config": {"workload": CONFIG_TEXT[args.config], "samples_per_gpu": B, "n_sites": N, "n_hidden": M,
                       "call": ("nk_local_energy_plan_run: the step's launches captured once into a CUDA graph by "
                                "nk_local_energy_plan_create and replayed" if args.call == "plan" else "nk_local_energy"),
                       ("ms_per_step_eager_nk_local_energy" if args.call == "plan" else "ms_per_step_planned"): other_ms,
                       "chunk_size": p.chunk_size, "amplitudes_per_step_per_gpu": amps,
                       "l2": "flushed between steps (512 MiB memset outside the per-step CUDA events)",
                       "parallelism": f"samples sharded over {world} rank(s), statistics all-gathered"},
            "clocks": clocks, "e2e": {"value": world * B / (e2e_ms * 1e-3), "unit": "local energies/s",
                                      "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms},
            "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu,
            "step_ms": [round(x, 4) for x in step_ms[:32]], "inputs_sha256": p.sha256()}
    if extras is not None:
        r = extras["sampler"]["roofline"]
        r["peak"] = pair_peak_mufu
        r["frac"] = r["achieved"] / pair_peak_mufu if pair_peak_mufu else None
        line["extras"] = extras
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_peaks(args):
    """--peaks: the pipe-peak microbenchmarks alone (nk_pipe_peaks), one JSON line."""
    import torch

    import paper_2112_10526_b200 as nk
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --peaks needs a CUDA device")
    torch.cuda.set_device(0)
    nk.load()
    out = [nk.pipe_peaks("cuda:0") for _ in range(3)][-1]
    out["what"] = ("MUFU.EX2-only, FFMA-only and LDS.128-only kernels on every SM (4 CTAs x 512 threads per SM, 8 independent "
                   "chains per thread); lanes or bytes per clock per SM at the SM clock measured inside each launch")
    print(json.dumps(out), flush=True)


def spawn_ranks(args):
    """`python bench.py --gpus N` with N > 1 and no torchrun environment: re-run this script under torchrun, one rank per
    GPU (the driver's own launch line), and fail loudly when the node has fewer devices."""
    import torch
    n_dev = torch.cuda.device_count()
    if n_dev < args.gpus:
        raise SystemExit(f"bench.py --gpus {args.gpus}: only {n_dev} CUDA device(s) visible")
    cmd = spawn_command(args)
    raise SystemExit(subprocess.call(cmd))


def spawn_command(args, port=None):
    import socket
    if port is None:
        sock = socket.socket()
        sock.bind(("127.0.0.1", 0))
        port = sock.getsockname()[1]
        sock.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__),
           "--gpus", str(args.gpus), "--steps", str(args.steps), "--warmup", str(args.warmup),
           "--config", str(args.config), "--impl", args.impl, "--call", args.call]
    if args.no_extras:
        cmd.append("--no-extras")
    return cmd


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5, 6])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-extras", action="store_true", help="skip the sampler / gradient timings")
    ap.add_argument("--call", default="plan", choices=["plan", "eager"],
                    help="the graded call: nk_local_energy_plan_run (CUDA-graph replay, default) or nk_local_energy")
    ap.add_argument("--peaks", action="store_true", help="only run the pipe-peak microbenchmarks (nk_pipe_peaks)")
    args = ap.parse_args()
    if args.peaks:
        run_peaks(args)
    elif args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
