#!/usr/bin/env python
"""bench.py -- throughput of the channelised overlap-save dedispersion path on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload gmrt32] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

A "step" is one pass of the whole hot path (corner turn/unpack/framing, forward FFT, chirp,
inverse FFT, discard, detect, integrate) over ONE batch = the whole workload (default: BASELINE.json configs[2], the
32 MHz GMRT mode the metric's real-time factor is quoted on: 512 channels x 62.5 kHz, 16 s, N_fft 4096, n_int 4).

value      device-resident: K dedisp_execute() calls between CUDA events, input already in HBM.
e2e        the same metric through dedisp_stream_push() on pinned HOST buffers in 1 s chunks (H2D, kernels and D2H
           overlapped on three streams), host wall clock around all pushes + the final sync.
roofline   the fused kernel (dominant): nominal flops of its launches / its CUDA-event time (the library's
           dedisp_profile_* events on the launching stream) against the FP32 FMA peak (bound "alu").
cpu_baseline   the fp64 oracle, as it stands, on the host cores, on a bounded leading slice of the same input.
N > 1      every rank runs its own workload-sized batch (its own seed): no data-path collective, "scaling": "weak";
           --shard channels: every rank one channel range of ONE workload (dedisp_plan_shard), "scaling": "strong".
other_workloads   (default run only) step and fused-kernel time of the other four BASELINE.json configs, device-resident,
           so that every roofline fraction DESIGN.md quotes is measured by the driver's own run (wideband on a 1 s cut).
--groups G        per-channel-group framing against the one-framing plan (its own JSON line).
--ubench fp32-issue   cycle cost of the butterfly forms (its own JSON line).
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
from dataclasses import replace

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "complex Msamples/s dedispersed"
UNIT = "Msamples/s"
FP32_LANES_PER_SM = 128   # sm_100: 4 sub-partitions x 32 FP32 lanes per SM; the SM count is read from the device
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "ncu_traffic.csv")


def ncu_traffic(workload: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the fused kernel, from the committed summary of the
    latest `ncu --set full` capture (profiles/ncu_traffic.csv: workload,kernel,dram_read_bytes,dram_write_bytes,capture).
    ncu cannot run inside a timed bench, so this is NOT measured in this run: the line names its source, and it is None
    when no capture of this workload is on file."""
    try:
        with open(TRAFFIC_CSV) as f:
            for ln in f:
                p = [v.strip() for v in ln.split(",")]
                if len(p) >= 5 and p[0] == workload:
                    return float(p[2]) + float(p[3]), f"profiles/ncu_traffic.csv ({p[4]}; not measured in this run)"
    except Exception:
        pass
    return None, "no ncu capture of this workload on file"


def stats(ms):
    """best / median / mean / sigma of per-step times (the paper reports mean +- sigma of 1000 runs)."""
    a = sorted(ms)
    n = len(a)
    mean = sum(a) / n
    return {"best": a[0], "median": a[n // 2] if n % 2 else 0.5 * (a[n // 2 - 1] + a[n // 2]), "mean": mean,
            "std": (sum((v - mean) ** 2 for v in a) / max(n - 1, 1)) ** 0.5, "n": n}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=("ours", "reference"), default="ours")
    ap.add_argument("--workload", default="gmrt32")
    ap.add_argument("--shard", choices=("batches", "channels"), default="batches",
                    help="N > 1: one workload-sized batch per rank (weak scaling, default) or one channel range of ONE "
                         "workload per rank (strong scaling, dedisp_plan_shard; SURVEY 8(e), P:L256-258)")
    ap.add_argument("--fullband", type=int, default=0, metavar="LOG2N",
                    help="time the paper's full-band mode (dedisp_fullband_*) with transforms of 2^LOG2N points, 20 ... 27")
    ap.add_argument("--groups", type=int, default=0,
                    help="G > 1: time the workload as G channel groups, each framed for its own smear "
                         "(dedisp_plan_shard + DEDISP_SHARD_OWN_FRAMING, SURVEY 8(f) NEXT-2), beside the one-framing plan")
    ap.add_argument("--duration", type=float, default=0.0, help="override the workload's seconds of data (debug)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-cufft", action="store_true", help="skip the cuFFT+elementwise reference point")
    ap.add_argument("--no-others", action="store_true",
                    help="skip the short device-resident runs of the other four BASELINE.json workloads (other_workloads)")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target wall time of the cpu_baseline leg")
    ap.add_argument("--ubench", choices=("fp32-issue",), default=None,
                    help="run a micro-benchmark instead of the bench (one JSON line; not the bench contract)")
    return ap.parse_args()


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled every 100 ms while the timed region runs (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.lines, self.proc, self.thr = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            return self
        self.thr = threading.Thread(target=lambda: [self.lines.append(l) for l in self.proc.stdout], daemon=True)
        self.thr.start()
        return self

    def mark(self):
        return len(self.lines)

    def stop(self, lo: int = 0, hi: int | None = None):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()
        rows = []
        for l in self.lines[lo:hi]:
            p = [v.strip() for v in l.split(",")]
            if len(p) >= 7:
                rows.append(p)
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        sm = sorted(float(r[0]) for r in rows)
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        reasons = [n for i, n in enumerate(names) if any(r[3 + i].lower().startswith("active") for r in rows)]
        pw = [float(r[2]) for r in rows if r[2].replace(".", "", 1).isdigit()]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(rows[0][1]), "reasons": reasons,
                "samples": len(rows), "power_w_max": max(pw) if pw else None}


def reduce_max_over_ranks(v: float, world: int, device: str) -> float:
    """Timing rule: a multi-rank time is the MAX over ranks (the only collective bench.py issues besides barriers)."""
    if world == 1:
        return v
    import torch
    import torch.distributed as dist
    t = torch.tensor([v], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(samples_per_rank: int, world: int, seconds_per_step: float) -> float:
    """Msamples/s over all ranks: every rank dedisperses its own batch of `samples_per_rank` valid samples per step."""
    return world * samples_per_rank / seconds_per_step / 1e6


def get_workload(args, rank: int):
    import datagen
    w = datagen.WORKLOADS[args.workload]
    if args.duration > 0:
        w = w.scaled(args.duration)
    if getattr(args, "shard", "batches") == "channels":
        return w                                   # strong scaling: every rank a channel range of the SAME batch
    return replace(w, seed=w.seed + rank)          # weak scaling: every rank its own batch


def channel_shard(n_chan: int, rank: int, world: int):
    """(first channel, number of channels) of rank's contiguous channel range; the ranges tile [0, n_chan)."""
    c0 = rank * n_chan // world
    return c0, (rank + 1) * n_chan // world - c0


def sub_band(w, c0: int, n: int):
    """The workload restricted to channels c0 .. c0+n-1 (same channel width, shifted centre frequency)."""
    dv = w.chan_width_hz
    return replace(w, n_chan=n, bw_hz=n * dv, f_center_hz=w.f_center_hz - 0.5 * w.bw_hz + (c0 + 0.5 * n) * dv)


def framing_counts(head: int, tail: int, L: int, n_samp: int, n_fft: int):
    nb = 0 if n_samp < n_fft else (n_samp - head - tail) // L
    return nb


def nominal_flops_per_unit(n_fft: int, L: int, n_dm: int) -> float:
    """One (channel, block) unit: 5 N log2 N per complex FFT (Eq. 5; one forward shared by the trial DMs + one
    inverse per DM), 6 per chirp multiply (Eq. 5's 3N' term counts a complex multiply on half-length real data), and
    3 (|v|^2) + 1 (integration add) per valid sample."""
    fft = 5.0 * n_fft * math.log2(n_fft)
    return (1 + n_dm) * fft + n_dm * (6.0 * n_fft + 4.0 * L)


def algorithmic_bytes_per_unit(n_fft: int, L: int, n_dm: int, n_int: int) -> float:
    """Fused kernel: reads the block's N samples as int8 pairs (the overlap is re-read: N, not L), writes L/n_int floats
    per DM.  The chirp table (8 B x N per (DM, channel)) is shared by all blocks of a channel and is served by L2."""
    return 2.0 * n_fft + 4.0 * n_dm * L / n_int


def oracle_timed(w, x, n_threads: int, target_s: float):
    """The oracle on a bounded leading slice of x, sized from a short calibration run to take about target_s."""
    import oracle
    cfg = oracle.OracleConfig(w.n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int)
    head, tail, L = oracle.framing(cfg)
    T = x.shape[0]
    n_cal = min(T, 2 * L + head + tail)
    t0 = time.perf_counter()
    oracle.dedisp(cfg, x[:n_cal], n_threads=n_threads)
    t_cal = max(time.perf_counter() - t0, 1e-4)
    nb_cal = (n_cal - head - tail) // L
    nb_all = (T - head - tail) // L
    nb = int(max(1, min(nb_all, nb_cal * target_s / t_cal)))
    n = nb * L + head + tail
    t0 = time.perf_counter()
    out = oracle.dedisp(cfg, x[:n], n_threads=n_threads)
    dt = time.perf_counter() - t0
    assert out.shape[2] == nb * (L // w.n_int)
    samples = w.n_chan * nb * L
    return samples / dt / 1e6, dt, nb, nb_all


def cufft_chain_reference(w, plan, d_in, chirp_host, steps: int = 3):
    """REFERENCE POINT ONLY (BASELINE.json north_star: "cuFFT+elementwise is timed only as a reference point"): the same
    framing computed as an unfused chain of library calls -- unpack, torch.fft.fft (cuFFT), chirp multiply,
    torch.fft.ifft, slice, abs^2, integrate -- each a full HBM round trip.  Nothing of this is in the product."""
    import torch
    N, L, head, n_int = plan.n_fft, plan.L, plan.head, plan.n_int
    T = d_in.shape[0]
    nb = plan.n_blocks(T)
    h = torch.from_numpy(chirp_host).cuda().to(torch.complex64)          # [C][N], includes 1/N; norm="forward" undoes it

    def chain():
        x = torch.view_as_complex(d_in.permute(1, 0, 2).to(torch.float32).contiguous())      # [C][T]
        blocks = x[:, : (nb - 1) * L + N].unfold(1, N, L)                                     # [C][nb][N] view
        spec = torch.fft.fft(blocks, dim=-1)
        spec *= h[:, None, :] * N
        v = torch.fft.ifft(spec, dim=-1)[:, :, head:head + L]
        p = (v.real * v.real + v.imag * v.imag).reshape(w.n_chan, nb * L // n_int, n_int).sum(-1)
        return p

    out = chain()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        out = chain()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    return out, ms


def run_reference(args):
    """--impl reference: the fp64 oracle as it stands on the host cores (this tier's reference arm).  Rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import datagen
    import oracle
    oracle.build()
    w = get_workload(args, 0)
    cores = os.cpu_count() or 1
    # a step = a bounded sample of the workload: the first `per_step_s` seconds of oracle work
    steps_total = args.steps + args.warmup
    per_step_s = min(10.0, 150.0 / max(steps_total, 1))
    # only the leading slice is needed: generate just enough data (full-length generation is for the GPU arm)
    cfg = oracle.OracleConfig(w.n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int)
    head, tail, L = oracle.framing(cfg)
    n_gen = min(w.n_samp, 256 * L + head + tail)
    x = datagen.generate(w, n_samp=n_gen)
    rate, dt, nb, nb_all = oracle_timed(w, x, cores, per_step_s)      # calibration + first warm-up
    n = nb * L + head + tail
    for _ in range(max(args.warmup - 1, 0)):
        oracle.dedisp(cfg, x[:n], n_threads=cores)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.dedisp(cfg, x[:n], n_threads=cores)
    dt = (time.perf_counter() - t0) / max(args.steps, 1)
    value = w.n_chan * nb * L / dt / 1e6
    sample = f"first {nb} of {(w.n_samp - head - tail) // L} blocks of every channel per step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "real_time_factor": value * 1e6 / w.bw_hz,
        "config": {"workload": w.name, "n_chan": w.n_chan, "bw_hz": w.bw_hz, "f_center_hz": w.f_center_hz,
                   "n_fft": w.n_fft, "n_int": w.n_int, "dm": list(w.dm_trials), "duration_s": w.duration_s,
                   "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU path)")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()

    def max_over_ranks(v: float) -> float:
        return reduce_max_over_ranks(v, world, "cuda")

    import datagen
    import paper_1509_00186_b200 as dd          # raises if libdedisp.so is missing: no fallback

    w_band = get_workload(args, rank)
    by_channels = args.shard == "channels"
    if by_channels:
        # rank r holds columns c0 .. c0+n-1 of the band (a host-side slice: here generated directly) and plans them
        # with the WHOLE band's framing, so all ranks share one time axis; no data-path collective in the step
        c0, n_loc = channel_shard(w_band.n_chan, rank, world)
        x = datagen.generate(w_band, chans=range(c0, c0 + n_loc))  # int8 [T][n_loc][2], seeded, host
        plan = dd.dedisp_plan_shard(w_band.n_chan, w_band.bw_hz, w_band.f_center_hz, w_band.dm_trials, w_band.n_fft,
                                    w_band.n_int, c0, n_loc)
        w = sub_band(w_band, c0, n_loc)                           # what this rank processes
    else:
        w = w_band
        x = datagen.generate(w)                                   # int8 [T][C][2], seeded, host
        plan = dd.dedisp_plan(w.n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int)
    T = x.shape[0]
    h_in = torch.from_numpy(x).pin_memory()
    d_in = h_in.cuda(non_blocking=False)
    head, tail, L = plan.head, plan.tail, plan.L
    nb = plan.n_blocks(T)
    n_out = plan.out_samples(T)
    n_units = w.n_chan * nb
    samples = n_units * L                                          # valid complex samples dedispersed per step
    plan.reserve(T)
    d_out = torch.empty((plan.n_dm, w.n_chan, n_out), dtype=torch.float32, device="cuda")

    # ---- device-resident timing -------------------------------------------------------------------------------
    for _ in range(max(args.warmup, 3)):
        plan.execute(d_in, d_out)
    torch.cuda.synchronize()
    sampler = ClockSampler(local).start() if rank == 0 else None
    time.sleep(0.3)
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    plan.profile_enable(True)
    barrier()
    torch.cuda.synchronize()
    mark0 = sampler.mark() if sampler else 0
    evs[0].record()
    for i in range(args.steps):
        plan.execute(d_in, d_out)
        evs[i + 1].record()
    torch.cuda.synchronize()
    barrier()
    mark1 = sampler.mark() if sampler else 0
    ms_total = max_over_ranks(evs[0].elapsed_time(evs[-1]))
    step_stats = stats([evs[i].elapsed_time(evs[i + 1]) for i in range(args.steps)])
    ms_ct, ms_fused, n_prof = plan.profile_read()
    plan.profile_enable(False)
    # keep the load on while the sampler catches at least a few readings (short runs finish between two samples)
    if sampler and mark1 - mark0 < 3:
        t_end = time.time() + 0.6
        while time.time() < t_end:
            plan.execute(d_in, d_out)
        torch.cuda.synchronize()
        mark1 = sampler.mark()
    clocks = sampler.stop(mark0, max(mark1, mark0 + 1)) if sampler else None
    ms_step = ms_total / args.steps
    value = whole_job_value(samples, world, ms_step * 1e-3)
    if by_channels and world > 1:  # channel ranges may differ by one channel: sum the ranks' sample counts
        tot = torch.tensor([float(samples)], dtype=torch.float64, device="cuda")
        dist.all_reduce(tot)
        value = float(tot.item()) / (ms_step * 1e-3) / 1e6
    checksum = float(d_out[:, :, : min(n_out, 1000)].double().mean().item())   # touches the result; sanity only

    # ---- end to end from pinned host memory (config 3: 1 s chunks, double buffered) -------------------------------
    e2e = None
    if not args.no_e2e:
        chunk = int(round((w.chunk_s if w.chunk_s > 0 else 1.0) * w.chan_width_hz))
        chunk = max(min(chunk, T), 1)
        h_out = torch.empty((plan.n_dm, w.n_chan, n_out), dtype=torch.float32).pin_memory()
        plan.stream_begin(chunk)

        def e2e_step():
            plan.stream_begin(chunk)                 # same buffers: resets the carry only
            col, t = 0, 0
            while t < T:
                n = min(chunk, T - t)
                col += plan.stream_push(h_in[t:t + n], h_out, col)
                t += n
            plan.stream_sync()
            return col

        for _ in range(max(args.warmup, 3)):
            assert e2e_step() == n_out
        barrier()
        torch.cuda.synchronize()
        e2e_ms = []
        t0 = time.perf_counter()
        for _ in range(args.steps):
            t1 = time.perf_counter()
            e2e_step()
            e2e_ms.append((time.perf_counter() - t1) * 1e3)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        barrier()
        dt = max_over_ranks(dt) / args.steps
        plan.stream_end()
        same = bool(torch.equal(h_out, d_out.cpu()))
        # the third roofline ("memory transfers turn out to be relatively expensive"): the box's own
        # pinned copy rates, one plain cudaMemcpyAsync of the step's whole input / output through torch, same run
        d_tmp = torch.empty_like(d_in)
        c0, c1, c2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        d_tmp.copy_(h_in, non_blocking=True)
        h_out.copy_(d_out, non_blocking=True)
        torch.cuda.synchronize()
        c0.record()
        d_tmp.copy_(h_in, non_blocking=True)
        c1.record()
        h_out.copy_(d_out, non_blocking=True)
        c2.record()
        torch.cuda.synchronize()
        h2d_gbs = h_in.numel() / (c0.elapsed_time(c1) * 1e-3) / 1e9
        d2h_gbs = h_out.numel() * 4 / (c1.elapsed_time(c2) * 1e-3) / 1e9
        del d_tmp
        e2e = {"value": world * samples / dt / 1e6, "unit": UNIT,
               "h2d_bytes_per_step": int(h_in.numel()), "d2h_bytes_per_step": int(h_out.numel() * 4),
               "ms_per_step": dt * 1e3, "real_time_factor": world * samples / dt / w_band.bw_hz,
               "chunk_samples": chunk, "chunks_per_step": (T + chunk - 1) // chunk,
               "timer": "host wall clock around all pushes + stream_sync",
               "api": "dedisp_stream_push (pinned host int8 in, pinned host fp32 out)",
               "equals_device_resident_output": same, "ms_per_step_stats": stats(e2e_ms),
               "pcie": {"bound": "pcie", "h2d_gbs_measured": h2d_gbs, "d2h_gbs_measured": d2h_gbs,
                        "h2d_gbs_achieved": h_in.numel() / dt / 1e9,
                        "frac_of_pcie": h_in.numel() / dt / 1e9 / h2d_gbs,
                        "how": "one cudaMemcpyAsync of the step's whole pinned input (H2D) and output (D2H), CUDA "
                               "events, same run; H2D is the longer direction and bounds the streamed step"}}
        del h_out

    # ---- cuFFT + elementwise chain on the same framing: a reference point, never part of the product --------------------
    cufft_ref = None
    if not args.no_cufft and rank == 0 and plan.n_dm == 1:
        try:
            import numpy as np
            chirp_host = np.stack([plan.debug_chirp(0, c) for c in range(w.n_chan)]).astype(np.complex64)
            ref_out, ref_ms = cufft_chain_reference(w, plan, d_in, chirp_host)
            rel = float(((ref_out - d_out[0]).norm() / d_out[0].norm()).item())
            cufft_ref = {"ms_per_step": ref_ms, "value": samples / (ref_ms * 1e-3) / 1e6, "unit": UNIT,
                         "speedup_of_fused_path": ref_ms / ms_step, "rel_l2_vs_fused_output": rel,
                         "what": "torch (cuFFT) unpack -> fft -> chirp -> ifft -> slice -> abs^2 -> integrate, unfused"}
            del ref_out
            torch.cuda.empty_cache()
        except Exception as exc:            # the reference point must never take the bench down
            cufft_ref = {"error": repr(exc)[:200]}

    # ---- sub-band alignment + band sum on the step's output (HBM-bound; not part of the step) ------
    band = None
    if rank == 0:
        n_ser = plan.band_samples(n_out)
        if n_ser > 0:
            d_series = torch.empty((plan.n_dm, n_ser), dtype=torch.float32, device="cuda")
            for _ in range(3):
                plan.band_sum(d_out, d_series)
            torch.cuda.synchronize()
            b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            b0.record()
            for _ in range(args.steps):
                plan.band_sum(d_out, d_series)
            b1.record()
            torch.cuda.synchronize()
            b_ms = b0.elapsed_time(b1) / args.steps
            b_bytes = 4.0 * plan.n_dm * n_ser * (w.n_chan + 1)
            band = {"kernel": "band_sum_kernel", "ms_per_launch": b_ms, "n_series": n_ser,
                    "algorithmic_bytes_per_launch": b_bytes, "achieved_gbs": b_bytes / (b_ms * 1e-3) / 1e9,
                    "note": "output of the step is 510 MB: partly L2-resident between launches" if d_out.numel() * 4 < 1e9 else ""}
            del d_series

    # channel shards: the band sum is the one place where ranks exchange data -- every rank sums its own channels on the
    # common time axis (the shard's shifts are the whole band's rows), one all-reduce of n_dm x n_series floats follows
    band_ar = None
    if by_channels and world > 1:
        n_ser = plan.band_samples(n_out)
        if n_ser > 0:
            part = plan.band_sum(d_out)
            torch.cuda.synchronize()
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            dist.barrier()
            a0.record()
            dist.all_reduce(part)
            a1.record()
            torch.cuda.synchronize()
            band_ar = {"collective": "nccl all_reduce(sum)", "floats": int(part.numel()),
                       "ms": max_over_ranks(a0.elapsed_time(a1))}

    # ---- roofline of the dominant (fused) kernel --------------------------------------------------------------------
    peaks, peaks_src = measured_peaks()
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    N_SM = torch.cuda.get_device_properties(local).multi_processor_count
    fp32_peak_tf = N_SM * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    traffic, traffic_source = ncu_traffic(w.name)
    fused_ms = ms_fused / max(n_prof, 1)
    ct_ms = ms_ct / max(n_prof, 1)
    flops = n_units * nominal_flops_per_unit(w.n_fft, L, plan.n_dm)
    abytes = n_units * algorithmic_bytes_per_unit(w.n_fft, L, plan.n_dm, w.n_int)
    achieved_tf = flops / (fused_ms * 1e-3) / 1e12
    roofline = {
        "bound": "alu", "kernel": "fused_aos_kernel", "achieved": achieved_tf, "peak": fp32_peak_tf,
        "unit": "TFLOP/s", "frac": achieved_tf / fp32_peak_tf, "traffic": traffic, "traffic_source": traffic_source,
        "peak_source": f"{N_SM} SM x {FP32_LANES_PER_SM} FP32 lanes x 2 (FMA) x {sm_max:.0f} MHz "
                       f"(sm_max_mhz of MEASURED_PEAKS.json, {peaks_src})",
        "flops_per_launch": flops, "ms_per_launch": fused_ms, "share_of_step": fused_ms / ms_step,
        "hbm": {"algorithmic_bytes_per_launch": abytes, "achieved_gbs": abytes / (fused_ms * 1e-3) / 1e9,
                "peak_gbs": float(peaks.get("hbm_gbs", 6650.0)),
                "frac": abytes / (fused_ms * 1e-3) / 1e9 / float(peaks.get("hbm_gbs", 6650.0))},
        "corner_turn": {"ms_per_launch": ct_ms, "share_of_step": ct_ms / ms_step,
                        "algorithmic_bytes_per_launch": 4.0 * w.n_chan * (nb * L + head + tail),
                        "achieved_gbs": 4.0 * w.n_chan * (nb * L + head + tail) / (ct_ms * 1e-3) / 1e9,
                        "frac_of_hbm_peak": 4.0 * w.n_chan * (nb * L + head + tail) / (ct_ms * 1e-3) / 1e9
                        / float(peaks.get("hbm_gbs", 6650.0))},
    }
    if clocks and clocks.get("sm_mhz"):
        pk = N_SM * FP32_LANES_PER_SM * 2 * clocks["sm_mhz"] * 1e6 / 1e12
        roofline["frac_at_observed_clock"] = achieved_tf / pk

    if rank != 0:
        plan.destroy()
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- CPU baseline: the oracle on the host cores, bounded sample (rank 0, N = 1 only) ----------------------------
    cpu = None
    if not args.no_cpu and world == 1:
        import oracle
        oracle.build()
        cores = os.cpu_count() or 1
        rate, dt, nb_cpu, nb_all = oracle_timed(w, x, cores, args.cpu_seconds)
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"first {nb_cpu} of {nb_all} blocks of every channel ({dt:.1f} s of wall time)",
               "real_time_factor": rate * 1e6 / w.bw_hz}

    others = None
    if world == 1 and not args.no_others and args.workload == "gmrt32" and not by_channels and args.duration == 0:
        try:
            del h_in
            others = measure_other_workloads(max(3, min(args.steps, 10)), fp32_peak_tf)
        except Exception as exc:            # an extra: it must never take the headline down
            others = {"error": repr(exc)[:200]}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "ms_per_step_stats": step_stats, "higher_is_better": True,
        "scaling": "strong" if by_channels else "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "real_time_factor": value * 1e6 / w_band.bw_hz,
        "config": {"workload": w.name, "n_chan": w.n_chan, "bw_hz": w.bw_hz, "f_center_hz": w.f_center_hz,
                   "n_fft": w.n_fft, "n_int": w.n_int, "dm": list(w.dm_trials), "duration_s": w.duration_s,
                   "samples_per_channel": T, "head": head, "tail": tail, "L": L, "blocks_per_channel": nb,
                   "valid_samples_per_step_per_gpu": samples, "input_bytes": int(d_in.numel()),
                   "output_bytes": int(d_out.numel() * 4),
                   "l2": "inputs larger than L2 (no flush needed)" if d_in.numel() > 256e6 else
                         "input smaller than 2x L2: numbers include L2 hits",
                   "sharding": ("one contiguous channel range of ONE workload per rank (dedisp_plan_shard, the whole band's "
                                "framing), no data-path collective in the step; n_chan/bw_hz/f_center_hz above are rank "
                                "0's range") if by_channels else
                               "one workload-sized batch per rank, no data-path collective"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": 2 * args.steps,
        "roofline": roofline, "cpu_baseline": cpu, "cufft_reference_point": cufft_ref, "next_rows": {"band_sum": band, "band_sum_allreduce": band_ar}, "other_workloads": others,
        "checksum_mean_first_1000": checksum,
    }
    print(json.dumps(line), flush=True)
    plan.destroy()
    if world > 1:
        dist.destroy_process_group()


OTHER_WORKLOADS = (("tiny", 0.0), ("gmrt16", 0.0), ("lowfreq", 0.0), ("wideband", 1.0))   # (name, seconds; 0 = full)


def measure_other_workloads(steps: int, fp32_peak_tf: float):
    """Device-resident step and fused-kernel time of the other four BASELINE.json configs, so that their roofline
    fractions are measured by the same run as the headline (wideband on a 1 s cut of its 8 s: 2048 channels x 15
    blocks x 8 DMs, 207 units per SM).  Same method as the headline: CUDA events around `steps` dedisp_execute
    calls, the library's own events around the fused kernel."""
    import torch
    import datagen
    import paper_1509_00186_b200 as dd
    out = {}
    for name, dur in OTHER_WORKLOADS:
        w = datagen.WORKLOADS[name]
        if dur > 0:
            w = w.scaled(dur)
        d_in = torch.from_numpy(datagen.generate(w)).cuda()
        T = d_in.shape[0]
        with dd.dedisp_plan(w.n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int) as plan:
            nb, n_out = plan.n_blocks(T), plan.out_samples(T)
            plan.reserve(T)
            d_out = torch.empty((plan.n_dm, w.n_chan, n_out), dtype=torch.float32, device="cuda")
            for _ in range(3):
                plan.execute(d_in, d_out)
            torch.cuda.synchronize()
            plan.profile_enable(True)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(steps):
                plan.execute(d_in, d_out)
            e1.record()
            torch.cuda.synchronize()
            ms_ct, ms_fused, n_prof = plan.profile_read()
            plan.profile_enable(False)
            ms_step = e0.elapsed_time(e1) / steps
            fused_ms = ms_fused / max(n_prof, 1)
            units = w.n_chan * nb
            tf = units * nominal_flops_per_unit(w.n_fft, plan.L, plan.n_dm) / (fused_ms * 1e-3) / 1e12
            out[name] = {"duration_s": w.duration_s, "n_fft": w.n_fft, "n_dm": plan.n_dm, "n_int": w.n_int,
                         "units": units, "ms_per_step": ms_step, "value": units * plan.L / (ms_step * 1e-3) / 1e6,
                         "real_time_factor": units * plan.L / (ms_step * 1e-3) / w.bw_hz,
                         "fused_ms_per_launch": fused_ms, "fused_frac_of_fp32_peak": tf / fp32_peak_tf,
                         "corner_turn_ms_per_launch": ms_ct / max(n_prof, 1)}
        del d_in, d_out
        torch.cuda.empty_cache()
    return out


def run_fullband(args):
    """--fullband LOG2N: the paper's own mode (dedisp_fullband_*) on synthetic GSB spectra shaped
    like its 32 MHz setting (512 channels, 325 MHz, int8 Gaussian(sigma 20) re/im), one GPU, its own
    JSON line.  DM is the largest that the length rule of P:L139-141 still maps to N = 2^LOG2N.  HBM-bound: a four-step
    transform has to read and write its array once per pass, forward and inverse 2 passes each = 4 x 16 B per complex
    point (two real blocks ride one complex transform) -- the algorithmic figure; this build moves 7 x 16 B
    (4 transposes + 3 row-transform kernels)."""
    import numpy as np
    import torch
    import paper_1509_00186_b200 as dd
    torch.cuda.set_device(0)
    n_chan, bw, f_lo, n_int = 512, 32e6, 309e6, 1024          # 15 us at 64 Msamples/s is ~10^3 samples
    N = 1 << args.fullband
    smear_per_dm = 4.148808e15 * (1.0 / f_lo ** 2 - 1.0 / (f_lo + bw) ** 2) * 2 * bw      # samples per unit DM
    dm = 0.499 * N / smear_per_dm                              # N is the smallest power of 2 > 2 x smear
    plan = dd.FullbandPlan(n_chan, bw, f_lo, (dm,), N, n_int)
    n_blocks = max(2, min(16, (1 << 28) // N))
    n_spec = -(-(n_blocks * plan.L + plan.D) // (2 * n_chan))
    rng = np.random.default_rng(5)
    spec = np.clip(np.rint(rng.normal(0.0, 20.0, size=(n_spec, n_chan, 2))), -127, 127).astype(np.int8)
    d_spec = torch.from_numpy(spec).cuda()
    d_out = torch.empty((1, plan.out_samples(n_spec)), dtype=torch.float32, device="cuda")
    for _ in range(max(args.warmup, 3)):
        plan.execute(d_spec, d_out)
    torch.cuda.synchronize()
    sampler = ClockSampler(0).start()
    time.sleep(0.3)
    mark0 = sampler.mark()
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    evs[0].record()
    for i in range(args.steps):
        plan.execute(d_spec, d_out)
        evs[i + 1].record()
    torch.cuda.synchronize()
    if sampler.mark() - mark0 < 3:          # short runs end between two clock samples: keep the load on a little longer
        t_end = time.time() + 0.6
        while time.time() < t_end:
            plan.execute(d_spec, d_out)
        torch.cuda.synchronize()
    clocks = sampler.stop(mark0, None)
    st = stats([evs[i].elapsed_time(evs[i + 1]) for i in range(args.steps)])
    ms = evs[0].elapsed_time(evs[-1]) / args.steps
    nb = d_out.shape[1] // (plan.L // n_int)
    valid = nb * plan.L                                        # valid real samples dedispersed per step
    pairs = (nb + 1) // 2
    peaks, peaks_src = measured_peaks()
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    alg = pairs * N * 64.0 + n_spec * n_chan * 2.0 + valid * 4.0 / n_int
    line = {"metric": "real Msamples/s dedispersed (full band)", "value": valid / (ms * 1e-3) / 1e6, "unit": "Msamples/s",
            "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "ms_per_step_stats": st,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "real_time_factor": valid / (ms * 1e-3) / (2 * bw),
            "config": {"workload": f"fullband32 (512 ch, 32 MHz at 325 MHz, N = 2^{args.fullband})", "n_chan": n_chan,
                       "bw_hz": bw, "f_lo_hz": f_lo, "dm": [dm], "n_fft": N, "n1": plan.n1, "n2": plan.n2, "n_int": n_int,
                       "D": plan.D, "L": plan.L, "blocks": nb, "n_spec": n_spec},
            "clocks": clocks, "gpu_launches": args.steps * (1 + pairs // max(1, (1 << 27) // N) * 0 + 8),
            "roofline": {"bound": "hbm", "kernel": "whole full-band step (1 c2r + 3 row-transform + 4 transpose + 1 detect kernels)",
                         "achieved": alg / (ms * 1e-3) / 1e9, "peak": hbm, "unit": "GB/s",
                         "frac": alg / (ms * 1e-3) / 1e9 / hbm, "traffic": None,
                         "algorithmic_bytes_per_step": alg, "moved_bytes_per_step_by_design": pairs * N * 112.0,
                         "peak_source": f"hbm_gbs of MEASURED_PEAKS.json ({peaks_src})"},
            "paper_context": "P:L285-287: 1.4x real time at 32 MHz on a Tesla C2075 + Xeon X5550, fp64",
            "checksum_mean": float(d_out.double().mean().item())}
    print(json.dumps(line), flush=True)
    plan.destroy()


def run_groups(args):
    """--groups G: per-channel-group framing (NEXT-2, DESIGN R18) against the one-framing plan on the same input, one GPU.
    Both produce the same dedispersed series on the common time axis (tests/test_gpu_shards.py); what changes is how
    many VALID samples every transform yields, so the comparison is time per step for the same data."""
    import torch
    import datagen
    import paper_1509_00186_b200 as dd
    torch.cuda.set_device(0)
    w = get_workload(args, 0)
    d_in = torch.from_numpy(datagen.generate(w)).cuda()
    T, G = d_in.shape[0], args.groups

    def timed(plans):
        outs = [torch.empty((p.n_dm, p.n_chan, p.out_samples(T)), dtype=torch.float32, device="cuda") for p in plans]
        for p in plans:
            p.reserve(T)
        for _ in range(max(args.warmup, 3)):
            for p, o in zip(plans, outs):
                p.execute(d_in, o)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            for p, o in zip(plans, outs):
                p.execute(d_in, o)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / args.steps

    one = dd.dedisp_plan(w.n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int)
    ms_one = timed([one])
    groups = []
    for g in range(G):
        c0, n = channel_shard(w.n_chan, g, G)
        groups.append(dd.dedisp_plan_shard(w.n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int, c0, n,
                                           full_input=True, own_framing=True))
    ms_grp = timed(groups)
    # the data both cover: the common output range on the whole band's time axis, in input samples per channel
    common = min([one.out_samples(T)] + [p.out_samples(T) - p.time_offset for p in groups]) * w.n_int
    line = {"metric": METRIC, "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3),
            "config": {"workload": w.name, "groups": G, "n_fft": w.n_fft, "n_dm": len(w.dm_trials)},
            "one_framing": {"ms_per_step": ms_one, "L": one.L, "value": w.n_chan * common / (ms_one * 1e-3) / 1e6},
            "group_framing": {"ms_per_step": ms_grp, "L": [p.L for p in groups],
                              "L_mean": sum(p.L * p.n_chan for p in groups) / w.n_chan,
                              "time_offset": [p.time_offset for p in groups],
                              "value": w.n_chan * common / (ms_grp * 1e-3) / 1e6},
            "speedup": ms_one / ms_grp, "higher_is_better": True, "data": "synthetic", "dtype": "f32"}
    print(json.dumps(line), flush=True)


def run_ubench(args):
    """--ubench fp32-issue: SM sub-partition cycles per radix-2 butterfly for every instruction form of
    dedisp_ubench_fp32 (csrc/ubench.cu); the numbers DESIGN.md section 6 quotes come from this command."""
    import torch
    import paper_1509_00186_b200 as dd
    torch.cuda.set_device(0)
    sampler = ClockSampler(0).start()
    time.sleep(0.3)
    rows = []
    for form, name in enumerate(dd.UBENCH_FORMS):
        best = min(dd.dedisp_ubench_fp32(form, 8192) for _ in range(3))
        rows.append({"form": form, "what": name, "cycles_per_butterfly": best[0], "ms": best[1]})
    clocks = sampler.stop()
    print(json.dumps({"ubench": "fp32-issue", "unit": "SM sub-partition cycles per butterfly (8 warps per sub-partition)",
                      "rows": rows, "clocks": clocks}), flush=True)


def main():
    args = parse_args()
    if args.fullband:
        run_fullband(args)
    elif args.groups > 1:
        run_groups(args)
    elif args.ubench:
        run_ubench(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
