#!/usr/bin/env python
"""bench.py - trajectory-steps/s of the whole TA-SC-IVR hot path (all SURVEY.md 8a rows) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--det-stride D] [--impl reference]

A "step" is one sc_ivr_run over the whole workload: propagate (PES, symplectic step, monodromy, action,
Herman-Kluk determinant, overlap, det M flag at every time step) -> z assembly -> Fourier sum -> |.|^2
reduction -> I(E).  Default workload: BASELINE.json config 4 (CH4-like, F = 9, 131072 trajectories,
4000 time steps, 4000 energies), the configuration the north star's target is quoted on.
Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle on a bounded sample instead.
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

from paper_1312_4698_b200 import inputs  # noqa: E402

METRIC = "FP64 trajectory-steps/sec (with monodromy+prefactor)"
UNIT = "trajectory-steps/s"
# FP64 roofline denominator: 148 SMs x 64 FP64 FMA lanes/SM/clk x 2 flop x 1.965 GHz.
# The guides give no FP64 unit count; 64 lanes/SM/clk is what this library's own DFMA/DMMA probe
# measures (37.2 TFLOP/s with mma.sync m8n8k4 f64 at 1965 MHz) - the probe value is reported beside it.
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
# dram__bytes_read.sum + dram__bytes_write.sum per launch of kernel A from one `ncu --set full` capture of the bench command,
# keyed by (workload, ntraj, nsteps, det_stride); the capture is summarised in the profiles/ file named beside it.  Any
# other configuration reports null.
NCU_TRAFFIC_BYTES = {
    ("config4_qff_ch4", 131072, 4000, 1): (16759154000 + 121386496, "profiles/r02_kernelA_ncu_config4.md"),  # write + read
}
CHIRP_L = 8192          # circular convolution length of the chirp-z Fourier stage (csrc/common.cuh SCI_CHIRP_L)
CHIRP_MIN_BLOCK = 1024  # csrc/common.cuh SCI_CHIRP_MIN_BLOCK
CHIRP_MAX_BLOCKS = 16   # csrc/common.cuh SCI_CHIRP_MAX_BLOCKS
# SURVEY.md 8d, complex determinant column (the survey rounds its own count; the formula below is used for other F)
SURVEY_CDET = {1: 10, 3: 95, 6: 615, 9: 1980}


def chirp_blocks(nsteps: int, k: int):
    """Mirror of the library's chirp_plan (csrc/api.cu): number of chirp-z blocks, 0 = direct sum."""
    if nsteps + k <= CHIRP_L:
        return 1
    bsz = CHIRP_L + 1 - k
    if bsz < CHIRP_MIN_BLOCK:
        return 0
    nb = -(-(nsteps + 1) // bsz)
    return nb if nb <= CHIRP_MAX_BLOCKS else 0


def flop_model(F: int, k: int, det_every_step: bool, morse: bool = False, nsteps: int = 4000, nblocks: int = 1):
    """Algorithmic flop per trajectory-step: SURVEY.md 8d's table (1 FMA = 2 flop), column by column; F = 9 QFF gives
    1386 + 150 + 3888 + 486 + 1980 = 7890, + 3570 with the det M check at every step = 11460.  Fourier stage: the direct
    sum of Eq. 11 is 8k per trajectory-step; on an equally spaced grid the library evaluates it as a chirp-z transform
    (two FFTs of length 8192 per trajectory and block), whose own count 2 * 5 L log2 L * nblocks / (nsteps + 1) is what is
    credited; nblocks = 0 means the direct sum.

    Uncoupled Morse oscillators (morse=True) have a DIAGONAL Hessian: each of the 2 F^2 elements of H M_q is one product, not
    an F-term inner product, and that is all the kernels execute (hessian_times in propagate_cml.cu, the tpt kernel likewise).
    The monodromy column is therefore 2 (2 F^2 + 6 F^2) = 16 F^2 for them (SURVEY's F = 1 row, 16, generalised), not the
    dense 2 (2 F^3 + 6 F^2): nothing that is not executed is credited.  The determinant columns stay dense: M_pq, M_qp, 2K and
    M are eliminated as full matrices whatever the surface (their zero pattern is not exploited), so those flop are executed.
    The 60 flop per Morse mode count one exp as the survey does."""
    pes = 60 * F if morse else 2 * (F * F * (F + 1) // 2 + 2 * F * F + F * (F - 1) + 6 * F)
    step = 16 * F + 6
    mono = 16 * F * F if morse else 2 * (2 * F ** 3 + 6 * F ** 2)
    kmat = 6 * F * F
    cdet = SURVEY_CDET.get(F, 8 * (F - 1) * F * (2 * F - 1) // 6 + 6 * F * (F - 1) // 2 + 16 * F)
    # SURVEY's table also lists ~150 flop-equivalents of transcendentals (exp, sincos, sqrt branch of z_c): this build does
    # them in the z assembly kernel, not in kernel A, so they are NOT credited to kernel A's roofline fraction
    a_total = pes + step + mono + kmat + cdet
    n = 2 * F
    check = 2 * ((n - 1) * n * (2 * n - 1) // 6)  # SURVEY 8d "+det M check": the FMAs of the real 2F x 2F elimination
    if det_every_step:
        a_total += check
    fourier = 2 * 5 * CHIRP_L * math.log2(CHIRP_L) * nblocks / (nsteps + 1) if nblocks > 0 else 8 * k
    return dict(propagate=a_total, fourier=fourier)


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.rows, self._stop_ev = index, [], threading.Event()

    def run(self):
        while not self._stop_ev.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.splitlines()[0].split(",")])
            except Exception:
                pass
            self._stop_ev.wait(0.2)

    def stop(self):
        self._stop_ev.set()
        self.join(timeout=6)
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 7 for i in range(4) if r[3 + i].lower().startswith("active")})
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None, reasons=reasons,
                    samples=len(sm))


def cpu_oracle_sample(w, ntraj_sample: int, det_stride: int, integrator: int = 0):
    """The oracle as it stands, on the first ntraj_sample trajectories of the workload (full time and energy grid)."""
    from oracle import capi
    ws = w.prefix(min(ntraj_sample, w.ntraj))
    t0 = time.perf_counter()
    capi.run_workload(ws, det_stride=det_stride, integrator=integrator)
    dt = time.perf_counter() - t0
    return dict(value=ws.ntraj * w.nsteps / dt, unit=UNIT, cores=capi.num_threads(), kind="oracle",
                sample=f"first {ws.ntraj} trajectories of {w.name}, {w.nsteps} steps, {w.k} energies, det_stride={det_stride}: {dt:.1f} s"), dt


def single_thread_oracle(args, ntraj_sample: int):
    """The paper's CPU numbers are single-thread: the same oracle with OMP_NUM_THREADS=1, in a process of its
    own (the OpenMP runtime reads the variable once), on a smaller sample of the same workload."""
    cmd = [sys.executable, os.path.abspath(__file__), "--impl", "reference", "--config", str(args.config), "--steps", "1", "--warmup", "0",
           "--ref-sample", str(ntraj_sample), "--det-stride", str(args.det_stride)]
    for flag, v in (("--ntraj", args.ntraj), ("--nsteps", args.nsteps), ("--k", args.k), ("--morse", args.morse or None),
                    ("--integrator", args.integrator or None)):
        if v is not None:
            cmd += [flag, str(v)]
    try:
        out = subprocess.run(cmd, env=dict(os.environ, OMP_NUM_THREADS="1", RANK="0", WORLD_SIZE="1"), capture_output=True, text=True, timeout=900)
        d = json.loads(out.stdout.strip().splitlines()[-1])
        return dict(value=d["value"], unit=UNIT, cores=d["cpu_baseline"]["cores"], sample=d["cpu_baseline"]["sample"])
    except Exception as ex:  # a reported baseline only
        return dict(error=str(ex)[:200])


def make_workload(config: int, rank: int, ntraj: int | None, nsteps: int | None = None, k: int | None = None, morse: int = 0):
    if morse:  # PAPER.md:204-206, Fig. 6: F uncoupled Morse oscillators, "the same number of trajectories"
        return inputs.make_uncoupled_morse(morse, ntraj or 65536, nsteps or 4000, k or 4000, seed=11 + rank)
    if rank == 0 and config != 5:
        return inputs.make_config(config, ntraj=ntraj, nsteps=nsteps, k=k)
    # rank r > 0 (weak scaling): block r of config 5's 2^20-row draw on config 4's surface, same size as rank 0's
    n = ntraj or inputs._DEFAULTS[4 if config == 5 else config]["ntraj"]
    full = inputs.make_config(5, ntraj=min((rank + 1) * n, 1 << 20), nsteps=nsteps, k=k)
    w = full.prefix(full.ntraj)
    w.p0q0 = np.ascontiguousarray(full.p0q0[:, full.ntraj - n:])
    return w


def run_reference(args, rank):
    if rank != 0:
        return
    w = make_workload(args.config, 0, args.ntraj, args.nsteps, args.k, args.morse)
    times = []
    for i in range(args.warmup + args.steps):
        cb, dt = cpu_oracle_sample(w, args.ref_sample, args.det_stride, args.integrator)
        if i >= args.warmup:
            times.append(dt)
    n = min(args.ref_sample, w.ntraj)
    val = n * w.nsteps / (sum(times) / len(times))
    cb["value"] = val
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "F": w.F, "ntraj_sample": n, "nsteps": w.nsteps, "k": w.k, "det_stride": args.det_stride},
        "cpu_baseline": cb, "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--ntraj", type=int, default=None)
    ap.add_argument("--nsteps", type=int, default=None)
    ap.add_argument("--k", type=int, default=None)
    ap.add_argument("--det-stride", type=int, default=1)
    ap.add_argument("--ref-sample", type=int, default=None,
                    help="trajectories of the oracle sample; default 2048 (BASELINE.md section 3), shrunk in the reference arm so that "
                         "steps + warmup samples end within a few minutes")
    ap.add_argument("--ref-sample-1t", type=int, default=64, help="trajectories of the single-thread oracle sample; 0 = skip")
    ap.add_argument("--integrator", type=int, default=0, choices=[0, 1],
                    help="0 = velocity-Verlet (BASELINE.json), 1 = 4-stage 4th-order symplectic scheme (the paper's, PAPER.md:109; row f2): "
                         "four evaluation points per time step, the flop model is scaled accordingly")
    ap.add_argument("--morse", type=int, default=0, help="F uncoupled Morse oscillators instead of a BASELINE config (row f3)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--nchi", type=int, default=0,
                    help="measure sc_ivr_run_multi with this many reference states (row f4) instead of sc_ivr_run; short JSON line")
    args = ap.parse_args()
    if args.ref_sample is None:
        args.ref_sample = 2048 if args.impl == "ours" else max(256, 2048 // max(1, (args.steps + args.warmup + 5) // 6))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        return run_reference(args, rank)

    import torch
    import torch.distributed as dist
    from paper_1312_4698_b200 import binding as B
    from paper_1312_4698_b200.sharding import combine_spectra

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    B.lib()

    w = make_workload(args.config, rank, args.ntraj, args.nsteps, args.k, args.morse)
    ctx = B.ScIvr.from_workload(w, det_stride=args.det_stride, integrator=args.integrator)
    ctx.set_timing(True)
    d_pq = torch.from_numpy(w.p0q0).cuda()
    ws_bytes = ctx.workspace_bytes(w.ntraj, w.k) + ctx.host_staging_bytes(w.ntraj, w.k)
    wsp = torch.empty(ws_bytes, dtype=torch.uint8, device="cuda")
    I_dev = torch.empty(w.k, dtype=torch.float64, device="cuda")
    h_pq = torch.from_numpy(w.p0q0).pin_memory()
    h_I = torch.empty(w.k, dtype=torch.float64).pin_memory()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        ctx.run(d_pq, w.chi, w.E, I_out=I_dev, workspace=wsp, want_n_good=False)

    if args.nchi > 0:  # row f4: nchi combinations of the states (+-p_eq, q_eq) sharing one propagation
        del wsp
        F = w.F
        chis = np.stack([w.chi, w.chi * np.concatenate([-np.ones(F), np.ones(F)])])
        eps = np.array([[1.0, np.cos(np.pi * n / max(1, args.nchi - 1))] for n in range(args.nchi)])
        wsm = torch.empty(ctx._lib_multi_bytes(w.ntraj, w.k, 2), dtype=torch.uint8, device="cuda")
        for _ in range(args.warmup):
            ctx.run_multi(d_pq, chis, eps, w.E, workspace=wsm)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            ctx.run_multi(d_pq, chis, eps, w.E, workspace=wsm)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / args.steps
        print(json.dumps({"metric": METRIC + ", shared by nchi reference states", "value": w.ntraj * w.nsteps / (ms * 1e-3), "unit": UNIT,
                          "nchi": args.nchi, "ms_per_step": ms, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
                          "config": {"workload": w.name, "F": w.F, "ntraj_per_gpu": w.ntraj, "nsteps": w.nsteps, "k": w.k}}))
        return

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stage = dict(propagate_ms=0.0, zassemble_ms=0.0, twiddle_ms=0.0, fourier_ms=0.0, reduce_ms=0.0)
    launches = 0
    barrier()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    t = ctx.last_timings()  # stage events of the LAST timed step (recorded on the run stream, no sync inside)
    launches = t["launches"] * args.steps
    for key in stage:
        stage[key] = t[key]
    # end to end through the C ABI with HOST buffers: H2D of p0q0, D2H of I(E) inside the timed region
    barrier()
    for _ in range(1):
        ctx.run_host(h_pq, w.chi, w.E, I_out=h_I, workspace=wsp)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _, ng_host, _ = ctx.run_host(h_pq, w.chi, w.E, I_out=h_I, workspace=wsp)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    clocks = sampler.stop()

    tt = torch.tensor([ms, e2e_s * 1e3], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        # the path's only exchange: k + 1 doubles (sharding.combine_spectra)
        I_all, ng_all = combine_spectra(I_dev, ng_host)
    ms, e2e_ms = tt[0].item(), tt[1].item()
    units = w.ntraj * w.nsteps * args.steps * world
    value = units / (ms * 1e-3)
    e2e_value = units / (e2e_ms * 1e-3)

    if rank == 0:
        nblk = chirp_blocks(w.nsteps, w.k)  # inputs.energy_grid is equally spaced: the library takes the chirp-z path when it can
        chirp = nblk > 0
        fm = flop_model(w.F, w.k, args.det_stride == 1, morse=(w.pes_kind != inputs.PES_QFF), nsteps=w.nsteps, nblocks=nblk)
        if args.integrator == 1:  # PES, step and monodromy columns of SURVEY 8d are per evaluation point: four per time step
            f1 = flop_model(w.F, w.k, False, morse=(w.pes_kind != inputs.PES_QFF), nsteps=w.nsteps, nblocks=nblk)["propagate"]
            F_ = w.F
            per_point = f1 - 6 * F_ * F_ - SURVEY_CDET.get(F_, 8 * (F_ - 1) * F_ * (2 * F_ - 1) // 6 + 6 * F_ * (F_ - 1) // 2 + 16 * F_)
            fm["propagate"] += 3 * per_point
        kname = {"propagate": "k_propagate_tpt" if w.F <= 3 else "k_propagate_cml", "fourier": "k_chirp_fft" if chirp else "k_fourier"}
        dom = "fourier" if stage["fourier_ms"] >= stage["propagate_ms"] else "propagate"
        dom_ms = stage[dom + "_ms"]
        flops_per_launch = fm[dom] * w.ntraj * w.nsteps  # one launch per run when the workload is a single batch
        achieved = flops_per_launch / (dom_ms * 1e-3) / 1e12
        other = "propagate" if dom == "fourier" else "fourier"
        other_tf = fm[other] * w.ntraj * w.nsteps / (stage[other + "_ms"] * 1e-3) / 1e12
        try:
            probe = {"dfma_tflops": B.fp64_probe(0, 20000)[0] / 1e12, "dmma_tflops": B.fp64_probe(1, 20000)[0] / 1e12}
        except Exception as ex:  # measurement helper only
            probe = {"error": str(ex)}
        try:
            # issue-budget probes (kernel A "what bounds it"): DFMA rate alone and with a shuffle / LDS after every 4
            # DFMAs or an integer pair after every DFMA, at 16, 2 and 1 warps per scheduler (kernel A runs at 2); only DFMAs count.
            # cycles = SM clock x 4 schedulers x SMs / DFMA warp-instructions per second
            sms = torch.cuda.get_device_properties(local_rank).multi_processor_count
            mhz = clocks.get("sm_mhz") or 1965.0
            issue = {}
            for name, mode in (("dfma_16wps", 0), ("dfma_2wps", 20), ("dfma_shfl_2wps", 22), ("dfma_lds_2wps", 23), ("dfma_int_2wps", 24),
                               ("dfma_1wps", 10), ("dfma_shfl_1wps", 12), ("dfma_lds_1wps", 13), ("dfma_int_1wps", 14)):
                tf = B.fp64_probe(mode, 20000)[0] / 1e12
                issue[name] = {"dfma_tflops": tf, "cycles_per_dfma_per_scheduler": mhz * 1e6 * 4 * sms * 64 / (tf * 1e12)}
            probe["issue"] = issue
        except Exception as ex:  # measurement helper only
            probe["issue"] = {"error": str(ex)}
        cpu = None
        if not args.no_cpu_baseline:
            cpu, _ = cpu_oracle_sample(w, args.ref_sample, args.det_stride, args.integrator)
            if args.ref_sample_1t > 0:
                cpu["single_thread"] = single_thread_oracle(args, args.ref_sample_1t)
        traffic, traffic_src = NCU_TRAFFIC_BYTES.get((w.name, w.ntraj, w.nsteps, args.det_stride), (None, None)) if dom == "propagate" else (None, None)
        dfma = probe.get("dfma_tflops")
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "F": w.F, "ntraj_per_gpu": w.ntraj, "nsteps": w.nsteps, "k": w.k, "dt": w.dt,
                       "det_stride": args.det_stride, "integrator": "velocity-verlet" if args.integrator == 0 else "4-stage 4th-order (McLachlan-Atela)",
                       "l2": "working set per step (raw 32 B + z 16 B per trajectory-step) exceeds L2 by >100x; no flush needed",
                       "parallelism": f"trajectory shards x{world}, one all-reduce of k+1 doubles" if world > 1 else "single GPU"},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(w.p0q0.nbytes + w.E.nbytes),
                    "d2h_bytes_per_step": int(w.k * 8 + 8)},
            "gpu_launches": int(launches),
            "roofline": {"bound": "alu", "kernel": kname[dom], "achieved": achieved, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s",
                         "frac": achieved / FP64_PEAK_TFLOPS, "frac_vs_dfma_probe": (achieved / dfma) if dfma else None,
                         "traffic": traffic, "traffic_source": traffic_src,
                         "peak_source": "nominal: 148 SM x 64 FP64 lanes x 2 x 1.965 GHz (DESIGN.md; MEASURED_PEAKS.json has no FP64 entry); "
                                        "frac_vs_dfma_probe divides by this run's measured DFMA rate instead",
                         "flop_per_trajectory_step": fm[dom], "probe": probe,
                         "other_kernel": {"kernel": kname[other], "achieved": other_tf, "frac": other_tf / FP64_PEAK_TFLOPS,
                                          "flop_per_trajectory_step": fm[other]}},
            "stage_ms_last_step": stage,
            "cpu_baseline": cpu,
        }
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
