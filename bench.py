#!/usr/bin/env python
"""bench.py -- one JSON line for the RUBIX hot path on B200 (contract: task prompt section 4).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload medium]

A "step" is one pass of the whole hot path (rotate, bin, sort, SSP
lookup, Doppler resample, accumulate, PSF, LSF) over one synthetic galaxy.  Default workload:
BASELINE.json configs[2] "medium (headline)": 1 M star particles, SSP 50x7x4300, detector
300x300x3700, PSF 15x15 + LSF 9 taps.  metric = particle*channel samples per second.

  value        device-resident inputs, CUDA events around K steps, max over ranks
  e2e          the same metric through rubix_forward_host: pinned HOST buffers, H2D of the particle
               arrays + SSP grid and D2H of the final cube inside the timed region
  roofline     the dominant kernel (k_accumulate), its time from CUDA event pairs recorded by the
               library on the launching stream inside the timed region
  cpu_baseline the fp64 oracle, as it stands, on this box's host cores, on the WHOLE workload (1 warm-up + 3 timed
               cubes, mean and best; nproc and CPU model; single-thread time of the tiny and small configs)
N > 1 (torchrun): replicas only -- every rank builds its own galaxy (seed + rank); no collective
on the data path; time = max over ranks.
--impl reference times the oracle (this tier's reference arm) on rank 0 only; every step is the whole workload.
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
sys.path.insert(0, ROOT)

METRIC = "particle_channel_samples_per_s"
UNIT = "G particle*channel/s"
# four corner templates x 4 B x (dl_obs / dl_ssp) SSP samples per channel
GATHER_BYTES_PER_SAMPLE = lambda tel, ssp: 16.0 * float(tel.dlambda) / float(ssp.dlambda)
# DRAM bytes of one k_accumulate launch on the medium workload inside rubix_forward, from the committed ncu --set full
# capture (profiles/r02_full_medium.md): 0.0531 GB read + 0.3327 GB written (rows of empty spaxels are not written)
NCU_DRAM_BYTES_K_ACCUMULATE = 0.3858e9
NCU_TRAFFIC_SOURCE = ("STATIC: dram__bytes_read.sum + dram__bytes_write.sum of one k_accumulate launch in the committed "
                      "ncu --set full capture profiles/r02_full_medium.md; not measured in this run")


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="medium", choices=["tiny", "small", "medium", "contention"])
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-adjoint", action="store_true")
    ap.add_argument("--no-batched", action="store_true")
    ap.add_argument("--cell-order", type=int, default=0, choices=[0, 1, 2, 3],
                    help="rubix_telescope.cell_order: 0 auto (the library decides), 1 off, 2 on, 3 on for every spaxel")
    ap.add_argument("--parallelism", default="replicas", choices=["replicas", "sharded"],
                    help="replicas (default, BASELINE.json north_star: one galaxy per GPU, weak scaling) or sharded: ONE galaxy "
                         "over all GPUs by detector rows (paper_2412_08265_b200/sharded.py, SURVEY.md 8(f)-4, strong scaling)")
    return ap.parse_args()


def workload_config(w):
    t, s = w.telescope, w.ssp
    return {"workload": f"{w.name}: {w.particles.n} star particles (disc+bulge), SSP "
                        f"{s.flux.shape[0]}x{s.flux.shape[1]}x{s.flux.shape[2]}, detector "
                        f"{t.n_x}x{t.n_y}x{t.n_channels}, PSF {t.psf_size}x{t.psf_size} + LSF {t.lsf_size} taps"
                        f" (BASELINE.json configs[{['tiny', 'small', 'medium', 'contention'].index(w.name)}])",
            "n_particles": w.particles.n, "n_spaxels": t.n_spaxels, "n_channels": t.n_channels,
            "euler_deg": [round(float(v), 4) for v in w.euler_deg],
            "l2_policy": "cube (%.2f GB) and workspace exceed the 126 MB L2: no flush needed"
                         % (t.n_spaxels * t.n_channels * 4 / 1e9),
            "cell_order": int(getattr(t, "cell_order", 0)),
            "parallelism": "replicas only (one galaxy per GPU, no collective)"}


# ------------------------------------------------------------------------------------- oracle arm
def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_step(w):
    """One step of the oracle (fp64, as it stands) on the WHOLE workload: build + PSF/LSF.  Seconds."""
    import oracle
    t = w.telescope
    t0 = time.perf_counter()
    cube = oracle.build_cube(w.particles, w.rotation, w.ssp, t)
    if t.psf_size > 0 or t.lsf_size > 0:
        cube = oracle.convolve(cube, t.psf_size, t.psf_sigma, t.lsf_size, t.lsf_sigma)
    dt = time.perf_counter() - t0
    del cube
    return dt


def oracle_single_thread(names=("tiny", "small")):
    """Single-thread oracle time of the small parity configs (BASELINE.md "CPU-baseline plan"), in a child process
    because the OpenMP thread count is fixed at library load."""
    import subprocess
    code = ("import sys, json, time; sys.path.insert(0, %r); import oracle; from paper_2412_08265_b200 import synth\n"
            "out = {}\n"
            "for name in %r:\n"
            "    w = synth.make_workload(name); t = w.telescope\n"
            "    oracle.build_cube(w.particles, w.rotation, w.ssp, t)\n"
            "    t0 = time.perf_counter(); oracle.build_cube(w.particles, w.rotation, w.ssp, t)\n"
            "    out[name] = {'seconds_per_cube': time.perf_counter() - t0, 'samples': w.particles.n * t.n_channels}\n"
            "print(json.dumps(out))\n") % (ROOT, tuple(names))
    env = dict(os.environ, OMP_NUM_THREADS="1")
    try:
        r = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, timeout=600)
        res = json.loads(r.stdout.strip().splitlines()[-1])
    except Exception as exc:                                   # reported, never fatal for the bench line
        return {"error": repr(exc)}
    for v in res.values():
        v["value"] = v["samples"] / v["seconds_per_cube"] / 1e9
        v["unit"] = UNIT
    return res


def cpu_baseline_block(w, repeats=3):
    """The oracle timed on this box's host cores on the whole workload: one warm-up, then `repeats` cubes."""
    import oracle
    oracle.build()
    oracle_step(w)
    secs = [oracle_step(w) for _ in range(repeats)]
    n_samples = w.particles.n * w.telescope.n_channels
    best, mean = min(secs), float(np.mean(secs))
    return {"value": n_samples / mean / 1e9, "unit": UNIT, "cores": oracle.n_threads(), "kind": "oracle",
            "sample": f"the WHOLE {w.name} workload (all {w.particles.n} particles, build + PSF/LSF of the full cube), "
                      f"1 warm-up + {repeats} timed cubes, no extrapolation",
            "seconds_per_cube": mean, "seconds_per_cube_best": best, "seconds_per_cube_all": secs,
            "value_best": n_samples / best / 1e9, "nproc": os.cpu_count(), "cpu_model": cpu_model(),
            "single_thread": oracle_single_thread()}


def run_reference(args):
    """--impl reference: the oracle alone, every step the whole workload (no sampling, no scaling)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    from paper_2412_08265_b200 import synth
    oracle.build()
    w = synth.make_workload(args.workload)
    for _ in range(max(args.warmup, 0)):
        oracle_step(w)
    secs = [oracle_step(w) for _ in range(args.steps)]
    t_step = float(np.mean(secs))
    n_samples = w.particles.n * w.telescope.n_channels
    value = n_samples / t_step / 1e9
    cores = oracle.n_threads()
    desc = (f"the WHOLE {w.name} workload per step (all {w.particles.n} particles, build + PSF/LSF of the full cube); "
            f"{args.warmup} warm-up + {args.steps} timed steps, mean {t_step:.2f} s, best {min(secs):.2f} s")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": t_step * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": workload_config(w),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                             "seconds_per_cube": t_step, "seconds_per_cube_best": min(secs),
                             "nproc": os.cpu_count(), "cpu_model": cpu_model()},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------- clocks
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag = index, [], set(), False
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {nv.nvmlClocksEventReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksEventReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksEventReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksEventReasonSwPowerCap: "sw_power_cap"} if hasattr(nv, "nvmlClocksEventReasonHwSlowdown") else \
                {nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap"}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.01)

    def result(self):
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def time_adjoint(B, synth, dev, l2_peak, reps=10):
    """rubix_cube_adjoint on BASELINE.json configs[4]: the config-1 galaxy with
    config-2 PSF/LSF, upstream gradient 2 (cube - target); reported beside the headline step."""
    import torch
    w = synth.make_workload("adjoint")
    other = synth.make_workload("adjoint")
    other.particles = synth.make_particles_for("adjoint", seed=synth.ADJOINT_TARGET_SEED)
    dw, dt = B.DeviceWorkload(w, device=dev), B.DeviceWorkload(other, device=dev)
    grad = (2.0 * (dw.forward() - dt.forward())).contiguous()
    for _ in range(3):
        dw.adjoint(grad)
    torch.cuda.synchronize()
    B.rubix_stage_timing_enable(True)
    B.rubix_stage_timing_read()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        dw.adjoint(grad)
    e1.record()
    torch.cuda.synchronize()
    st = B.rubix_stage_timing_read()
    B.rubix_stage_timing_enable(False)
    adj_ms = e0.elapsed_time(e1) / reps
    t, n = w.telescope, w.particles.n
    k_ms = st["adjoint"]["ms"] / max(st["adjoint"]["calls"], 1)
    n_in = int(dw.sort_artifacts()[2][t.n_spaxels].item())          # in-FoV particles (the others do no work)
    # "as K3 per sample": the four corner rows over the particle's window, read once
    gather_b = GATHER_BYTES_PER_SAMPLE(t, w.ssp) * n_in * t.n_channels
    # fused forward + loss + adjoint (rubix_loss_and_grad): one particle pass, loss reduced on the device
    target = dt.forward()
    for _ in range(3):
        dw.loss_and_grad(target)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(reps):
        loss, _, _ = dw.loss_and_grad(target)
    e1.record()
    torch.cuda.synchronize()
    fused_ms = e0.elapsed_time(e1) / reps
    return {"workload": "adjoint: BASELINE.json configs[4] (100k particles, 25x25x3700, PSF 15x15 + LSF 9)",
            "loss_and_grad_ms_per_call": fused_ms, "loss": float(loss.item()),
            "ms_per_call": adj_ms, "k_adjoint_ms": k_ms,
            "value": n * t.n_channels / (adj_ms * 1e-3) / 1e9, "unit": UNIT,
            "in_fov_particles": n_in,
            "roofline": {"kernel": "k_adjoint_units (step 9)", "bound": "l2", "achieved": gather_b / (k_ms * 1e-3) / 1e9,
                         "peak": l2_peak, "unit": "GB/s", "frac": gather_b / (k_ms * 1e-3) / 1e9 / l2_peak,
                         "algorithmic_bytes_per_launch": gather_b, "kernel_ms": k_ms,
                         "peak_source": "L2->SM read bandwidth measured in this run by rubix_measure_peaks (builder-measured: "
                                        "MEASURED_PEAKS.json has no L2 figure)"}}


def time_batched(B, synth, dev, reps=20):
    """cubes per second for the small cubes (launch-latency bound one at a time) with rubix_forward_batched
    at B = 1, 16, 64 against B looped rubix_forward calls and against B replays of a CUDA graph of one call.  Each element is
    the config's galaxy under its own rotation."""
    import torch
    out = {}
    for name in ("tiny", "small"):
        w = synth.make_workload(name)
        dw = B.DeviceWorkload(w, device=dev)
        t = w.telescope
        res = {}
        for batch in (1, 16, 64):
            R = np.stack([synth.euler_rotation(*synth.random_euler(7000 + b)) for b in range(batch)]).astype(np.float32)
            cubes = torch.empty((batch,) + dw.shape, dtype=torch.float32, device=dev)
            ws = torch.empty(B.rubix_forward_batched_workspace_bytes(w.particles.n, None, batch, dw.ssp, dw.tel),
                             dtype=torch.uint8, device=dev)

            def batched():
                B.rubix_forward_batched(dw.particles, None, batch, dw.ssp, dw.tel, R, cubes, ws)

            def looped():
                for b in range(batch):
                    B.rubix_forward(dw.particles, dw.ssp, dw.tel, R[b], cubes[b], dw.workspace)

            def timed(fn, n):
                for _ in range(3):
                    fn()
                torch.cuda.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                for _ in range(n):
                    fn()
                e1.record()
                torch.cuda.synchronize()
                return e0.elapsed_time(e1) / n

            ms_b = timed(batched, reps)
            launches = B.rubix_last_launch_count()
            ms_l = timed(looped, max(reps // 4, 2))
            res[f"B={batch}"] = {"batched_ms": ms_b, "batched_cubes_per_s": batch / ms_b * 1e3, "launches": launches,
                                 "looped_ms": ms_l, "looped_cubes_per_s": batch / ms_l * 1e3,
                                 "speedup_over_loop": ms_l / ms_b}
        # one captured rubix_forward replayed (the rotation is baked into the graph: a lower bound on the looped cost)
        s = torch.cuda.Stream(device=dev)
        one = torch.empty(dw.shape, dtype=torch.float32, device=dev)
        with torch.cuda.stream(s):
            B.rubix_forward(dw.particles, dw.ssp, dw.tel, dw.R, one, dw.workspace, stream=s.cuda_stream)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            B.rubix_forward(dw.particles, dw.ssp, dw.tel, dw.R, one, dw.workspace, stream=torch.cuda.current_stream().cuda_stream)
        for _ in range(3):
            g.replay()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(64):
            g.replay()
        e1.record()
        torch.cuda.synchronize()
        res["graph_replay_ms_per_cube"] = e0.elapsed_time(e1) / 64
        res["graph_replay_cubes_per_s"] = 64 / e0.elapsed_time(e1) * 1e3
        res["speedup_over_graph_replay_at_B=64"] = res["B=64"]["batched_cubes_per_s"] / res["graph_replay_cubes_per_s"]
        out[name] = res
    # the fused forward + loss + adjoint for 64 concatenated galaxies (rubix_loss_and_grad_batched) against 64 looped calls
    w = synth.make_workload("tiny")
    dw = B.DeviceWorkload(w, device=dev)
    batch, n = 64, w.particles.n
    rep = lambda a: a.repeat(batch, *([1] * (a.dim() - 1))).contiguous()
    arrays = [rep(getattr(dw, f)) for f in ("pos", "vel", "mass", "log_age", "log_z")]
    cp = B.c_particles(*arrays)
    offsets = np.arange(batch + 1, dtype=np.int64) * n
    R = np.stack([synth.euler_rotation(*synth.random_euler(7000 + b)) for b in range(batch)]).astype(np.float32)
    targets = torch.zeros((batch,) + dw.shape, dtype=torch.float32, device=dev)
    loss = torch.zeros(batch, dtype=torch.float64, device=dev)
    g = [torch.empty(batch * n, dtype=torch.float32, device=dev) for _ in range(4)]
    ws = torch.empty(B.rubix_loss_and_grad_batched_workspace_bytes(batch * n, offsets, batch, dw.ssp, dw.tel),
                     dtype=torch.uint8, device=dev)
    g1 = [torch.empty(n, dtype=torch.float32, device=dev) for _ in range(4)]
    ws1 = torch.empty(B.rubix_loss_and_grad_workspace_bytes(n, dw.ssp, dw.tel), dtype=torch.uint8, device=dev)

    def lg_batched():
        B.rubix_loss_and_grad_batched(cp, offsets, batch, dw.ssp, dw.tel, R, targets, loss, None, *g, ws)

    def lg_looped():
        for b in range(batch):
            B.rubix_loss_and_grad(dw.particles, dw.ssp, dw.tel, R[b], targets[b], loss[b:b + 1], None, *g1, ws1)

    def timed2(fn, k):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(k):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / k

    ms_b, ms_l = timed2(lg_batched, reps), timed2(lg_looped, max(reps // 4, 2))
    out["loss_and_grad_tiny_B=64"] = {"batched_ms": ms_b, "batched_galaxies_per_s": batch / ms_b * 1e3, "looped_ms": ms_l,
                                      "looped_galaxies_per_s": batch / ms_l * 1e3, "speedup_over_loop": ms_l / ms_b,
                                      "what": "rubix_loss_and_grad_batched, 64 copies of configs[0] under 64 rotations, zero targets"}
    out["what"] = ("rubix_forward_batched (one launch sequence for B cubes) vs B looped rubix_forward calls vs replays of a CUDA "
                   "graph of one rubix_forward; BASELINE.json configs[0] (tiny) and configs[1] (small), one galaxy under B rotations")
    return out


def run_sharded(args):
    """ONE galaxy over all ranks, sharded by detector rows: all-to-all of particle records, halo
    exchange of raw rows, no cube exchange.  Strong scaling: value = the galaxy's samples / slowest rank's time.  Every rank
    keeps its slice of the particle arrays resident; the step includes the binning, both exchanges and the PSF/LSF."""
    import torch
    import torch.distributed as dist

    from paper_2412_08265_b200 import replicas, sharded, synth

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    own_group = False
    if not dist.is_initialized():
        if world == 1:
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29517")
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=dev)
        own_group = True
    w = synth.make_workload(args.workload)
    t, p = w.telescope, w.particles
    backend = sharded.CudaBackend(dev)
    comm = sharded.DistComm()
    sl = sharded.slice_for_rank(p.n, rank, world)
    rec = sharded.pack_records(p.subset(np.arange(p.n)[sl]), dev)
    flux = backend.upload_flux(w.ssp)

    def step():
        return sharded.forward_sharded(comm, backend, rec, w.rotation, w.ssp, t, flux_dev=flux)

    for _ in range(max(args.warmup, 3)):
        slab = step()
    torch.cuda.synchronize()
    dist.barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        slab = step()
    e1.record()
    torch.cuda.synchronize()
    dist.barrier()
    sampler.stop_flag = True
    sampler.join()
    ms = replicas.max_over_ranks(e0.elapsed_time(e1), dev) / args.steps
    rows = torch.tensor([float(slab.x1 - slab.x0), float(slab.n_received)], dtype=torch.float64, device=dev)
    allr = [torch.zeros_like(rows) for _ in range(world)]
    dist.all_gather(allr, rows)
    if rank == 0:
        line = {"metric": METRIC, "value": p.n * t.n_channels / (ms * 1e-3) / 1e9, "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True,
                "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": dict(workload_config(w), parallelism=f"one galaxy sharded by detector rows over {world} GPUs "
                               "(all-to-all of particle records + halo exchange of raw rows; no cube exchange)"),
                "clocks": sampler.result(),
                "rows_per_rank": [int(v[0].item()) for v in allr], "particles_per_rank": [int(v[1].item()) for v in allr],
                "note": "host-orchestrated steps (routing with torch ops, per-step workspace allocation): a functional "
                        "strong-scaling path, not the tuned single-GPU step of the default run"}
        print(json.dumps(line))
    if own_group:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------- our arm
def run_ours(args):
    import torch
    import torch.distributed as dist

    from paper_2412_08265_b200 import binding as B
    from paper_2412_08265_b200 import replicas, synth

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    B.load()

    # replicas: rank r gets its own galaxy (same recipe, seed + r)
    base = synth.make_workload(args.workload)
    widx = ["tiny", "small", "medium", "contention"].index(args.workload)
    w = base if rank == 0 else synth.make_workload(args.workload, seed=replicas.replica_seed(widx, rank))
    if args.cell_order:
        import dataclasses
        w = dataclasses.replace(w, telescope=dataclasses.replace(w.telescope, cell_order=args.cell_order))
    t, n = w.telescope, w.particles.n
    dw = B.DeviceWorkload(w, device=dev)
    cube = torch.empty(dw.shape, dtype=torch.float32, device=dev)
    final = torch.empty_like(cube)
    has_conv = t.psf_size > 0 or t.lsf_size > 0
    launches_per_step = [0]

    def step():                                               # steps 1-8 in one device call
        B.rubix_forward(dw.particles, dw.ssp, dw.tel, dw.R, final, dw.workspace)
        launches_per_step[0] = B.rubix_last_launch_count()

    def step_two_calls():                                     # the same path as two plain calls (dense raw cube)
        B.rubix_build_cube(dw.particles, dw.ssp, dw.tel, dw.R, cube, dw.workspace)
        if has_conv:
            B.rubix_convolve_psf_lsf(dw.tel, cube, final, dw.workspace)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    B.rubix_stage_timing_enable(True)
    B.rubix_stage_timing_read()
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    sampler.stop_flag = True
    sampler.join()
    elapsed_ms = e0.elapsed_time(e1)
    stages = B.rubix_stage_timing_read()
    B.rubix_stage_timing_enable(False)
    elapsed_ms = replicas.max_over_ranks(elapsed_ms, dev)
    ms_per_step = elapsed_ms / args.steps
    n_in = int(dw.sort_artifacts()[2][t.n_spaxels].item())          # particles inside the field of view
    samples_per_step = float(n) * t.n_channels
    value = replicas.whole_job_value(samples_per_step, world, elapsed_ms, args.steps) / 1e9

    # ---- the same step as rubix_build_cube + rubix_convolve_psf_lsf (no occupancy masks), for comparison
    for _ in range(2):
        step_two_calls()
    torch.cuda.synchronize()
    e0.record()
    for _ in range(5):
        step_two_calls()
    e1.record()
    torch.cuda.synchronize()
    two_call_ms = e0.elapsed_time(e1) / 5
    step()                                                    # `final` holds the fused call's cube again

    # ---- the same step replayed from a CUDA graph (the call is capturable: no launch gaps between its 19 kernels)
    graph_ms = None
    try:
        gs = torch.cuda.Stream(device=dev)
        with torch.cuda.stream(gs):
            B.rubix_forward(dw.particles, dw.ssp, dw.tel, dw.R, final, dw.workspace, stream=gs.cuda_stream)
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=gs):
            B.rubix_forward(dw.particles, dw.ssp, dw.tel, dw.R, final, dw.workspace, stream=torch.cuda.current_stream().cuda_stream)
        for _ in range(3):
            graph.replay()
        torch.cuda.synchronize()
        e0.record()
        for _ in range(10):
            graph.replay()
        e1.record()
        torch.cuda.synchronize()
        graph_ms = e0.elapsed_time(e1) / 10
        del graph
    except Exception as exc:                                  # reported, never fatal for the bench line
        graph_ms = f"failed: {exc}"

    # ---- step 9 on the bench workload itself (outside the timed step): rubix_cube_adjoint with the final cube as the
    #      upstream gradient; the kernel's time per 1e6 in-FoV particles
    adjoint_workload = None
    if has_conv and not args.no_adjoint and rank == 0:
        for _ in range(2):
            dw.adjoint(final)
        torch.cuda.synchronize()
        B.rubix_stage_timing_enable(True)
        B.rubix_stage_timing_read()
        for _ in range(5):
            dw.adjoint(final)
        torch.cuda.synchronize()
        st_a = B.rubix_stage_timing_read()
        B.rubix_stage_timing_enable(False)
        k_ms = st_a["adjoint"]["ms"] / max(st_a["adjoint"]["calls"], 1)
        adjoint_workload = {"what": f"rubix_cube_adjoint on the {w.name} workload (upstream gradient = the final cube)",
                            "k_adjoint_ms": k_ms, "in_fov_particles": n_in, "ms_per_1e6_particles": k_ms * 1e6 / max(n_in, 1),
                            "psf_lsf_transpose_ms": st_a["psf_lsf"]["ms"] / max(st_a["psf_lsf"]["calls"], 1)}

    # ---- end to end through the host-buffer entry point
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    p = w.particles
    hp = [pin(x) for x in (p.pos, p.vel, p.mass, p.log_age, p.log_z)]
    hflux = pin(w.ssp.flux)
    hcube = torch.empty(dw.shape, dtype=torch.float32).pin_memory()
    cp, cs, ct = B.c_particles(*hp), B.c_ssp(w.ssp, hflux), dw.tel
    del cube, final
    scratch = torch.empty(B.rubix_forward_host_pipelined_scratch_bytes(n, cs, ct), dtype=torch.uint8, device=dev)
    h2d = sum(x.numel() * 4 for x in hp) + hflux.numel() * 4
    d2h = hcube.numel() * 4

    def time_e2e(call, drain):
        for _ in range(2):
            call(cp, cs, ct, w.rotation, hcube, scratch)
        drain()
        barrier()
        e0.record()
        for _ in range(args.e2e_steps):
            call(cp, cs, ct, w.rotation, hcube, scratch)
        drain()                                              # the stream waits for every device->host copy
        e1.record()
        barrier()
        ms = replicas.max_over_ranks(e0.elapsed_time(e1), dev)
        return replicas.whole_job_value(samples_per_step, world, ms, args.e2e_steps) / 1e9, ms / args.e2e_steps

    # serial: H2D, compute and D2H of one cube after the other on one stream (rubix_forward_host)
    e2e_serial_value, e2e_serial_ms = time_e2e(B.rubix_forward_host, lambda: None)
    # pipelined: the D2H of cube i overlaps the H2D and compute of cube i + 1 (rubix_forward_host_pipelined)
    e2e_value, e2e_ms = time_e2e(B.rubix_forward_host_pipelined, B.rubix_forward_host_drain)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (k_accumulate), measured on-chip peaks
    peaks_file = os.path.join(ROOT, "MEASURED_PEAKS.json")
    hbm_peak, hbm_src = 6650.0, "fallback (B200_PROFILING.md)"
    if os.path.exists(peaks_file):
        hbm_peak, hbm_src = float(json.load(open(peaks_file))["hbm_gbs"]), "MEASURED_PEAKS.json"
    if scratch.numel() < (1 << 30):                           # the peak micro-benchmarks want >= 64 MiB
        scratch = torch.empty(1 << 30, dtype=torch.uint8, device=dev)
    onchip = B.rubix_measure_peaks(scratch)
    acc_ms = stages["accumulate"]["ms"] / max(stages["accumulate"]["calls"], 1)
    # algorithmic bytes count the in-FoV particles only (the dropped ones sort last and do no work)
    samples_in = float(n_in) * t.n_channels
    gather_b = GATHER_BYTES_PER_SAMPLE(t, w.ssp) * samples_in
    hbm_b = t.n_spaxels * t.n_channels * 4.0 + w.ssp.flux.size * 4.0 + 48.0 * n_in
    achieved = gather_b / (acc_ms * 1e-3) / 1e9
    # L1 data-pipe view (the unit ncu shows saturated, profiles/r01_full_medium.md): bytes the SM's
    # load/store pipe must carry per particle = 4 corner windows (LDG) + table store (STS) + two
    # table reads per channel (LDS); peak = the shared-memory read bandwidth measured in this run
    win = float(t.n_channels) * float(t.dlambda) / float(w.ssp.dlambda)
    l1_b = (16.0 * win + 4.0 * win + 8.0 * t.n_channels) * n_in
    l1_peak = onchip["smem_gbs"]
    roofline = {"kernel": "k_accumulate (steps 4-6)", "bound": "l2", "achieved": achieved,
                "peak": onchip["l2_gbs"], "unit": "GB/s", "frac": achieved / onchip["l2_gbs"],
                "traffic": NCU_DRAM_BYTES_K_ACCUMULATE if args.workload == "medium" else None,
                "traffic_source": NCU_TRAFFIC_SOURCE,
                "in_fov_particles": n_in,
                "l1_view": {"bound": "l1 data pipe", "achieved": l1_b / (acc_ms * 1e-3) / 1e9, "peak": l1_peak,
                            "unit": "GB/s", "frac": l1_b / (acc_ms * 1e-3) / 1e9 / l1_peak,
                            "peak_source": "shared-memory / L1 data-pipe read bandwidth measured in this run by rubix_measure_peaks "
                                           "(nominal 148 SMs x 128 B/clk x 1.965 GHz = 37.2 TB/s)",
                            "algorithmic_bytes_per_launch": l1_b},
                "peak_source": "L2->SM read bandwidth measured in this run by rubix_measure_peaks: BUILDER-measured "
                               "(ld.global.cg over a 32 MiB buffer), not a driver-written figure -- MEASURED_PEAKS.json has "
                               "no L2 entry (SURVEY.md 8(d))",
                "algorithmic_bytes_per_launch": gather_b, "kernel_ms": acc_ms,
                "hbm_view": {"bound": "hbm", "achieved": hbm_b / (acc_ms * 1e-3) / 1e9, "peak": hbm_peak,
                             "unit": "GB/s", "frac": hbm_b / (acc_ms * 1e-3) / 1e9 / hbm_peak,
                             "peak_source": hbm_src, "algorithmic_bytes_per_launch": hbm_b},
                "measured_peaks": onchip}
    stage_ms = {k: (v["ms"] / max(v["calls"], 1) if v["calls"] else 0.0) for k, v in stages.items()}
    # ---- whole-step roofline: t_roof = sum over the stages of max(HBM, on-chip gather, ALU) time
    conv_bytes = 2.0 * t.n_spaxels * t.n_channels * 4.0 if has_conv else 0.0
    pass_bytes = (28.0 + 2 * 16.0 + 48.0 + 16.0) * n + 2.0 * w.ssp.flux.size * 4.0   # arrays in, 2 sort passes, records, grid copy
    terms = {"particle_pass": {"hbm_ms": pass_bytes / hbm_peak / 1e6},
             "accumulate": {"hbm_ms": hbm_b / hbm_peak / 1e6, "l2_gather_ms": gather_b / onchip["l2_gbs"] / 1e6,
                            "alu_ms": 14.0 * samples_in / (onchip["fma_tflops"] * 1e12) * 1e3},
             "psf_lsf": {"hbm_ms": conv_bytes / hbm_peak / 1e6}}
    t_roof = sum(max(v.values()) for v in terms.values())
    whole_step = {"t_roof_ms": t_roof, "ms_per_step": ms_per_step, "frac": t_roof / ms_per_step, "terms": terms,
                  "hbm_only_ms": sum(v["hbm_ms"] for v in terms.values()),
                  "what": "sum over the stages of max(HBM bytes / HBM peak, L2 gather bytes / L2 peak, flops / fp32 peak) "
                          "divided by the measured step (SURVEY.md 8(d); north_star's >= 50 % is judged on this)",
                  "peaks": {"hbm_gbs": hbm_peak, "hbm_source": hbm_src, "l2_gbs": onchip["l2_gbs"],
                            "fma_tflops": onchip["fma_tflops"], "on_chip_source": "builder-measured in this run"}}
    if has_conv:
        conv_b = 2.0 * t.n_spaxels * t.n_channels * 4.0
        roofline["psf_lsf"] = {"bound": "hbm", "achieved": conv_b / (stage_ms["psf_lsf"] * 1e-3) / 1e9,
                               "peak": hbm_peak, "unit": "GB/s",
                               "frac": conv_b / (stage_ms["psf_lsf"] * 1e-3) / 1e9 / hbm_peak,
                               "algorithmic_bytes_per_launch": conv_b, "kernel_ms": stage_ms["psf_lsf"]}

    # ---- SURVEY.md 8(f)-1 variant: the same step with flux-conserving resampling (RUBIX_RESAMPLE_FLUX)
    import dataclasses
    wf = dataclasses.replace(w, telescope=dataclasses.replace(t, resample=1))
    dwf = B.DeviceWorkload(wf, device=dev)
    cube_f = torch.empty(dw.shape, dtype=torch.float32, device=dev)
    final_f = torch.empty_like(cube_f)

    def step_flux():
        B.rubix_build_cube(dwf.particles, dwf.ssp, dwf.tel, dwf.R, cube_f, dwf.workspace)
        if has_conv:
            B.rubix_convolve_psf_lsf(dwf.tel, cube_f, final_f, dwf.workspace)

    for _ in range(3):
        step_flux()
    torch.cuda.synchronize()                              # rank 0 only from here on: no collective
    B.rubix_stage_timing_enable(True)
    B.rubix_stage_timing_read()
    e0.record()
    for _ in range(10):
        step_flux()
    e1.record()
    torch.cuda.synchronize()                              # rank 0 only from here on: no collective
    st_f = B.rubix_stage_timing_read()
    B.rubix_stage_timing_enable(False)
    flux_ms = e0.elapsed_time(e1) / 10
    flux_acc_ms = st_f["accumulate"]["ms"] / max(st_f["accumulate"]["calls"], 1)
    flux_variant = {"what": "same workload with RUBIX_RESAMPLE_FLUX (flux-conserving bin average, SURVEY.md 8(f)-1)",
                    "ms_per_step": flux_ms, "k_accumulate_ms": flux_acc_ms,
                    "value": samples_per_step / (flux_ms * 1e-3) / 1e9, "unit": UNIT,
                    "l2_frac": gather_b / (flux_acc_ms * 1e-3) / 1e9 / onchip["l2_gbs"]}
    del dwf, cube_f, final_f

    # ---- SURVEY.md 8(f)-1 variant: log-sampled SSP grid of the same size (reading R15, table mode)
    table_variant = None
    if args.workload in ("small", "medium", "contention"):
        na, nz, nl = w.ssp.flux.shape
        wl = dataclasses.replace(w, ssp=synth.make_ssp(na, nz, nl, 3000.0, 10000.0, 2101, log_lambda=True))
        dwl = B.DeviceWorkload(wl, device=dev)
        cube_l = torch.empty(dw.shape, dtype=torch.float32, device=dev)
        for _ in range(3):
            dwl.build_cube(out=cube_l)
        torch.cuda.synchronize()
        B.rubix_stage_timing_enable(True)
        B.rubix_stage_timing_read()
        for _ in range(10):
            dwl.build_cube(out=cube_l)
        torch.cuda.synchronize()
        st_l = B.rubix_stage_timing_read()
        B.rubix_stage_timing_enable(False)
        table_variant = {"what": "rubix_build_cube on a log-sampled SSP grid of the same size (table mode, reading R15)",
                         "k_accumulate_ms": st_l["accumulate"]["ms"] / max(st_l["accumulate"]["calls"], 1),
                         "particle_pass_ms": st_l["particle_pass"]["ms"] / max(st_l["particle_pass"]["calls"], 1)}
        del dwl, cube_l

    # ---- general-grid mode (readings R20 / R21): fp64 positions per sample
    gen_variant = None
    if args.workload in ("small", "medium", "contention"):
        na, nz, nl = w.ssp.flux.shape
        gen_variant = {"what": "rubix_build_cube under readings R20 / R21, same particles and detector, k_accumulate ms: the bin average "
                               "on a log-sampled grid (table mode, fixed point) and listed SSP wavelengths (general-grid mode, "
                               "positions per sample in fp64)"}
        cases = {"bin_average_on_log_grid": (synth.make_ssp(na, nz, nl, 3000.0, 10000.0, 2101, log_lambda=True), 1),
                 "listed_ssp_wavelengths_point_rule": (synth.make_ssp(na, nz, nl, 3000.0, 10000.0, 2101, irregular=True), 0),
                 "listed_ssp_wavelengths_bin_average": (synth.make_ssp(na, nz, nl, 3000.0, 10000.0, 2101, irregular=True), 1)}
        for name, (ssp_g, rule) in cases.items():
            wg = dataclasses.replace(w, ssp=ssp_g, telescope=dataclasses.replace(t, resample=rule))
            dwg = B.DeviceWorkload(wg, device=dev)
            cube_g = torch.empty(dw.shape, dtype=torch.float32, device=dev)
            for _ in range(2):
                dwg.build_cube(out=cube_g)
            torch.cuda.synchronize()
            B.rubix_stage_timing_enable(True)
            B.rubix_stage_timing_read()
            for _ in range(5):
                dwg.build_cube(out=cube_g)
            torch.cuda.synchronize()
            st_g = B.rubix_stage_timing_read()
            B.rubix_stage_timing_enable(False)
            gen_variant[name] = {"k_accumulate_ms": st_g["accumulate"]["ms"] / max(st_g["accumulate"]["calls"], 1),
                                 "particle_pass_ms": st_g["particle_pass"]["ms"] / max(st_g["particle_pass"]["calls"], 1)}
            del dwg, cube_g

    # ---- noise stage (reading R17): elementwise, read + write of the cube
    noise_info = None
    if has_conv:
        nz_in = torch.empty(dw.shape, dtype=torch.float32, device=dev).uniform_(0.0, 10.0)
        nz_out = torch.empty_like(nz_in)
        for _ in range(3):
            B.rubix_add_noise(nz_in, nz_out, 1.0, 0.1, 12345)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(10):
            B.rubix_add_noise(nz_in, nz_out, 1.0, 0.1, 12345)
        e1.record()
        torch.cuda.synchronize()
        nz_ms = e0.elapsed_time(e1) / 10
        nz_b = 8.0 * nz_in.numel()
        noise_info = {"what": "rubix_add_noise on a cube of the workload's size (Philox4x32-10 + Box-Muller, read + write)",
                      "ms": nz_ms, "bound": "hbm", "achieved": nz_b / (nz_ms * 1e-3) / 1e9, "peak": hbm_peak,
                      "unit": "GB/s", "frac": nz_b / (nz_ms * 1e-3) / 1e9 / hbm_peak}
        del nz_in, nz_out

    adjoint_info = None
    if not args.no_adjoint:
        del scratch
        adjoint_info = time_adjoint(B, synth, dev, onchip["l2_gbs"])

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": workload_config(w), "clocks": sampler.result(),
            "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": e2e_ms, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h,
                    "api": "rubix_forward_host_pipelined + rubix_forward_host_drain (pinned host buffers; the D2H of cube i "
                           "overlaps the H2D and compute of cube i + 1)",
                    "serial": {"value": e2e_serial_value, "ms_per_step": e2e_serial_ms, "api": "rubix_forward_host"}},
            "gpu_launches": launches_per_step[0] * args.steps, "gpu_launches_per_step": launches_per_step[0],
            "stage_ms": stage_ms, "roofline": roofline,
            "api": "rubix_forward (steps 1-8 in one device call; occupancy-masked PSF/LSF passes)",
            "graph_replay_ms_per_step": graph_ms,
            "two_calls": {"ms_per_step": two_call_ms,
                          "api": "rubix_build_cube + rubix_convolve_psf_lsf (dense raw cube, no masks; 5 steps)"}}
    line["roofline"]["whole_step"] = whole_step
    if not args.no_batched:
        line["batched"] = time_batched(B, synth, dev)
    line["flux_variant"] = flux_variant
    if table_variant is not None:
        line["log_grid_variant"] = table_variant
    if gen_variant is not None:
        line["general_grid_variant"] = gen_variant
    if noise_info is not None:
        line["noise_stage"] = noise_info
    if adjoint_info is not None:
        if adjoint_workload is not None:
            adjoint_info["on_bench_workload"] = adjoint_workload
            gb = GATHER_BYTES_PER_SAMPLE(t, w.ssp) * n_in * t.n_channels
            adjoint_workload["l2_frac"] = gb / (adjoint_workload["k_adjoint_ms"] * 1e-3) / 1e9 / onchip["l2_gbs"]
        line["adjoint"] = adjoint_info

    if not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline_block(base)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    elif a.parallelism == "sharded":
        run_sharded(a)
    else:
        run_ours(a)
