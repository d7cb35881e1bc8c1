#!/usr/bin/env python
"""bench.py -- throughput of the plane-wave H.Psi / Chebyshev-filter / Gram hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--cfg {1..5}] [--impl reference]

One "step" is one pass of the whole hot path over one block of synthetic
wavefunctions of a BASELINE.json config: the scaled Chebyshev filter of the config's degree m on all bands (in the
config's column blocks), followed -- for the configs that name a Gram product -- by H Psi and G = Psi^H (H Psi)
(the Rayleigh-Ritz companion step).  That is (m+1) H applications per band (m without Gram).

    value = band H.psi applications / s = nband * (m [+1]) / step time          (BASELINE.json `metric`)

Timing: W >= 3 warm-up steps, then K steps bracketed by a barrier + torch.cuda.synchronize() and CUDA events on the
launching stream; max over ranks.  The inputs (Psi, P: GBs) are far larger than the 126 MB L2 and every step starts
by restoring Psi from a pristine device copy (inside the timed region), so no step sees a warm cache from the last.
The path does not shard (north_star: one GPU, no collectives): with --gpus N > 1 every rank runs an independent
replica (weak scaling, no data-path collective).

`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "band_Hpsi_applications_per_s"
UNIT = "band-H-applications/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--cfg", type=int, default=int(os.environ.get("PWH_BENCH_CFG", "5")), choices=[1, 2, 3, 4, 5],
                    help="BASELINE.json config; default 5 = the largest single-GPU workload (the metric names no config)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--profile-steps", type=int, default=2, help="steps of the per-kernel event-timed pass (after the timed region)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU seconds of the oracle sample")
    return ap.parse_args()


def workload_name(w):
    s = w.spec
    return (f"cfg{s.cfg_id}: box {s.fft_dims[0]}x{s.fft_dims[1]}x{s.fft_dims[2]}, k={tuple(s.kpt)}, npw={w.npw}, "
            f"nband={s.nband} (blocks of {s.block}), nproj={w.nproj}, Chebyshev degree {s.degree}"
            + (f" + H.Psi + Gram {s.nband}x{s.nband}" if s.with_gram else "") + ", complex128")


def apps_per_band(spec):
    return spec.degree + (1 if spec.with_gram else 0)


# ----------------------------------------------------------------------------------------------------------------
# clocks sampling (B200_PROFILING.md: the clocks line, sampled DURING the timed region)
# ----------------------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx = gpu_index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv", prefix="pwh_clocks_")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.idx), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        try:
            for line in open(self.path):
                f = [x.strip() for x in line.split(",")]
                if len(f) < 9:
                    continue
                try:
                    sm.append(float(f[1])); smax.append(float(f[2])); power.append(float(f[3]))
                except ValueError:
                    continue
                for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"),
                                     f[5:9]):
                    if val.lower().startswith("active"):
                        reasons.add(name)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            sm.sort()
            out.update(sm_mhz=sm[len(sm) // 2], sm_max_mhz=max(smax), reasons=sorted(reasons), samples=len(sm),
                       power_w_max=max(power))
        return out


# ----------------------------------------------------------------------------------------------------------------
# algorithmic work per stage -- per band and per H application
# ----------------------------------------------------------------------------------------------------------------
def fft_flops(n: int) -> float:
    import math
    return 5.0 * n * math.log2(n)


def stage_model(w, info):
    n1, n2, n3 = (int(v) for v in w.fft_dims)
    N, J = w.npw, w.nproj
    ncols, nxl = info["n_zcolumns"], info["n_xlines"]
    return {
        # sphere in + out, pruned column buffer written and read once in each direction
        "local_bytes": 32.0 * N + 64.0 * ncols * n3,
        "local_flops": 2.0 * (ncols * fft_flops(n3) + nxl * n3 * fft_flops(n2) + n2 * n3 * fft_flops(n1)),
        # recurrence fused into the gather: read Y_j, Y_{j-1}, write Y_{j+1}
        "recurrence_bytes": 48.0 * N,
        "zgemm_flops": 16.0 * N * J,          # a7 + a8, 4M convention (8 m n k per complex GEMM)
    }


def oracle_sample(oracle, w, nb: int, light: bool = False):
    """One bounded sample of the step on the CPU oracle, on the first `nb` bands.  Full: a degree-2 Chebyshev filter (2 H
    applications and the three-term recurrence), H.Psi and the Gram product = 3 H applications per band.  Light (the
    --impl reference arm, which repeats it K + W times): a degree-1 filter and the Gram product = 1 H application per
    band.  Returns (seconds, H applications per band)."""
    args = (w.lattice, w.kpt, w.fft_dims, w.gvec, w.vloc, w.proj, w.dij)
    t0 = time.perf_counter()
    if light:
        y = oracle.cheb_filter(*args, w.psi[:nb], 1, w.a, w.b, w.a0)
        oracle.gram(w.psi[:nb], y)
        return time.perf_counter() - t0, 1
    y = oracle.cheb_filter(*args, w.psi[:nb], 2, w.a, w.b, w.a0)
    hy = oracle.apply_h(*args, y)
    oracle.gram(y, hy)
    return time.perf_counter() - t0, 3


def cpu_baseline(w, target_s: float):
    """The oracle as it stands on the host cores, on a bounded sample of the same workload."""
    import oracle
    cores = oracle.n_threads()
    nb = min(w.psi.shape[0], cores)
    t, apps = oracle_sample(oracle, w, nb)
    if t < target_s / 3 and nb < w.psi.shape[0]:
        per = t / max(1, -(-nb // cores))                       # seconds per wave of `cores` bands
        waves = max(1, int(target_s / max(per, 1e-6)))
        nb = min(w.psi.shape[0], waves * cores)
        t, apps = oracle_sample(oracle, w, nb)
    return {"value": nb * apps / t, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"oracle (C, -O2, OpenMP over bands) on the first {nb} bands of the same workload: degree-2 Chebyshev "
                      f"filter + H.Psi + Gram {nb}x{nb} = {apps} H applications per band, {t:.1f} s wall"}


def run_reference(args):
    """--impl reference: the CPU oracle timed on this box's host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    import oracle
    from paper_2604_11139_b200 import synth
    cores = oracle.n_threads()
    spec = synth.CONFIGS[args.cfg]
    nb = min(spec.nband, cores)
    w = synth.make_workload(args.cfg, nband=nb, qr="none")
    w.spec = __import__("dataclasses").replace(w.spec, block=spec.block)
    # bounded: one step = one H application on at most `cores` bands (one band per core), so that the whole
    # --steps K --warmup W run ends within a few minutes even at cfg 5 (about 6 s per step on 16 cores)
    apps = 1
    for _ in range(args.warmup):
        oracle_sample(oracle, w, nb, light=True)
    t = 0.0
    for _ in range(args.steps):
        t += oracle_sample(oracle, w, nb, light=True)[0]
    value = nb * apps * args.steps / t
    sample = (f"each step = the oracle on {nb} bands: degree-1 Chebyshev filter (1 H application + the first recurrence step) "
              f"+ Gram {nb}x{nb} (bounded sample of the config's {spec.nband} bands x {apps_per_band(spec)} applications)")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(w).replace(f"nband={nb}", f"nband={spec.nband}").replace(f"Gram {nb}x{nb}", f"Gram {spec.nband}x{spec.nband}"), "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------------------------------------------
# the CUDA arm
# ----------------------------------------------------------------------------------------------------------------
def max_over_ranks(dist, ms: float, device) -> float:
    """Device-timed milliseconds of the slowest replica (the path has no collective: every rank runs the whole step on its
    own GPU); `dist` is torch.distributed or None for a single process."""
    if dist is None:
        return float(ms)
    import torch
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, nband: int, napps: int, ms_step: float) -> float:
    """band H.psi applications per second of all replicas together (weak scaling: each rank does the full workload)."""
    return world * nband * napps / (ms_step * 1e-3)


def run_ours(args):
    import numpy as np
    import torch

    from paper_2604_11139_b200 import binding, synth

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: CUDA is not available and there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist_
        dist = dist_
        dist.init_process_group("nccl", device_id=dev)
    binding.load_library()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- inputs: seeded synthetic crystal, resident in HBM before any timed region
    t_gen = time.perf_counter()
    w = synth.make_workload(args.cfg, qr="torch-cuda")
    spec = w.spec
    M, N, m, blk = spec.nband, w.npw, spec.degree, spec.block
    ham = binding.ham_setup(w.lattice, w.kpt, w.fft_dims, w.gvec, w.vloc, w.proj, w.dij, device=dev)
    info = ham.info()
    psi0 = torch.from_numpy(w.psi).to(dev)
    psi = torch.empty_like(psi0)
    hpsi = torch.empty_like(psi0) if spec.with_gram else None
    t_gen = time.perf_counter() - t_gen
    napps = apps_per_band(spec)

    filter_events = []

    def step(record=False):
        psi.copy_(psi0)
        if record:
            f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            f0.record()
        for b0 in range(0, M, blk):
            binding.cheb_filter(ham, psi[b0:b0 + blk], m, w.a, w.b, w.a0)
        if record:
            f1.record()
            filter_events.append((f0, f1))
        if spec.with_gram:
            for b0 in range(0, M, blk):
                binding.apply_h(ham, psi[b0:b0 + blk], hpsi[b0:b0 + blk])
            return binding.gram(psi, hpsi, hermitian=True)     # Psi^H (H Psi) is Hermitian
        return None

    for _ in range(max(args.warmup, 0)):
        step()
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    n0 = binding.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        step(record=True)
    e1.record()
    barrier()
    launches = binding.launch_count() - n0
    ms_total = e0.elapsed_time(e1)
    ms_total = max_over_ranks(dist, ms_total, dev)
    clocks = sampler.stop() if rank == 0 else {}
    ms_step = ms_total / args.steps
    nblocks = -(-M // blk)
    filter_ms_block = sum(a.elapsed_time(b) for a, b in filter_events) / (args.steps * nblocks)
    value = whole_job_value(world, M, napps, ms_step)

    if rank != 0:
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return 0

    # ---- per-kernel times: a second pass of the same K steps with one CUDA-event pair around every launch
    psteps = max(1, min(args.steps, args.profile_steps))
    binding.profile_begin()
    pe0, pe1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    pe0.record()
    for _ in range(psteps):
        step()
    pe1.record()
    stages = binding.profile_end()
    ms_step_profiled = pe0.elapsed_time(pe1) / psteps
    peak_dmma = binding.probe_fp64_tensor_peak(20000, dev)

    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    hbm_src = "MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)"

    mod = stage_model(w, info)
    band_apps = M * napps * psteps                       # of the per-kernel pass the stage times come from
    # Gram Psi^H (H Psi): 8 N M^2 flops by definition (4M convention); the Hermitian kernel computes only the 128 x 64 tiles
    # with floor(m/128) <= floor(n/128)
    tiles_m, tiles_n = -(-M // 128), -(-M // 64)
    herm_tiles = sum(min(tiles_m, tn // 2 + 1) for tn in range(tiles_n))
    gram_def = 8.0 * N * M * M * psteps if spec.with_gram else 0.0
    gram_exec = 6.0 * N * herm_tiles * 128 * 64 * psteps if spec.with_gram else 0.0
    zg_ms = stages.get("zgemm_cn", (0.0, 0))[0] + stages.get("zgemm_nn", (0.0, 0))[0]
    zg_n = stages.get("zgemm_cn", (0.0, 0))[1] + stages.get("zgemm_nn", (0.0, 0))[1]
    zg_def = mod["zgemm_flops"] * band_apps + gram_def              # 8 m n k per complex GEMM
    zg_exec = 0.75 * mod["zgemm_flops"] * band_apps + gram_exec     # what the 3M kernels put on the DMMA pipe: 6 m n k
    loc_ms = sum(stages.get(k, (0.0, 0))[0] for k in ("scatter_zinv", "plane", "zfwd_gather"))
    loc_n = sum(stages.get(k, (0.0, 0))[1] for k in ("scatter_zinv", "plane", "zfwd_gather"))
    loc_bytes = (mod["local_bytes"] + mod["recurrence_bytes"]) * band_apps
    loc_flops = mod["local_flops"] * band_apps
    all_ms = sum(v[0] for v in stages.values())
    stage_out = {k: {"ms_per_step": v[0] / psteps, "launches_per_step": v[1] / psteps,
                     "share": v[0] / all_ms if all_ms else None} for k, v in stages.items()}
    fp64_nominal = 148 * 128 * 1.965e9 * 1e-12          # 148 SMs x 64 DFMA/clk x 2 flop x 1.965 GHz = 37.2 TFLOP/s
    traffic = profiled_traffic(args.cfg)
    if zg_ms >= loc_ms and zg_ms > 0:
        ach = zg_exec / (zg_ms * 1e-3) * 1e-12
        n_cn, n_nn = stages.get("zgemm_cn", (0.0, 0))[1], stages.get("zgemm_nn", (0.0, 0))[1]
        t_cn, t_nn = traffic.get("zgemm_cn"), traffic.get("zgemm_nn")
        roofline = {"bound": "tensor", "kernel": "k_zgemm3m_tma (3M complex product on DMMA m8n8k4.f64, TMA-fed; CN + NN instantiations)",
                    "achieved": ach, "peak": peak_dmma, "unit": "TFLOP/s", "frac": ach / peak_dmma,
                    "peak_source": "pwh_probe_fp64_tensor_peak, register-resident DMMA loop measured in this run "
                                   f"(nominal 148 SM x 128 flop/clk x 1.965 GHz = {fp64_nominal:.1f}); MEASURED_PEAKS.json "
                                   "holds no FP64 figure",
                    "frac_of_nominal": ach / fp64_nominal,
                    "flops_per_launch": zg_exec / max(zg_n, 1), "ms_per_launch": zg_ms / max(zg_n, 1),
                    "equiv_8mnk_TFLOPs": zg_def / (zg_ms * 1e-3) * 1e-12,
                    "note": "achieved = flops the kernels execute on the DMMA pipe (3M complex product: 6 m n k; Hermitian "
                            "Gram: computed tiles only) / event time, so frac <= 1; equiv_8mnk_TFLOPs counts the same "
                            "launches as 8 m n k per complex GEMM (SURVEY.md 8d-4) for comparison with 4M libraries",
                    "traffic": ((n_cn * t_cn + n_nn * t_nn) / max(n_cn + n_nn, 1)) if t_cn and t_nn else None,
                    "traffic_source": traffic.get("source")}
    else:
        ach = loc_bytes / (loc_ms * 1e-3) * 1e-9
        roofline = {"bound": "hbm", "kernel": "local-potential kernels (scatter + z, plane, z + gather + recurrence)",
                    "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak, "peak_source": hbm_src,
                    "bytes_per_launch": loc_bytes / max(loc_n, 1), "ms_per_launch": loc_ms / max(loc_n, 1),
                    "traffic": traffic.get("local"), "traffic_source": traffic.get("source")}
    local_roof = {"ms_per_step": loc_ms / psteps, "us_per_band_application": 1e3 * loc_ms / max(band_apps, 1),
                  "alg_GBps": loc_bytes / max(loc_ms, 1e-9) * 1e-6, "hbm_frac": loc_bytes / max(loc_ms, 1e-9) * 1e-6 / hbm_peak,
                  "alg_fp64_TFLOPs": loc_flops / max(loc_ms, 1e-9) * 1e-9,
                  "fp64_frac_of_nominal": loc_flops / max(loc_ms, 1e-9) * 1e-9 / fp64_nominal}
    zgemm_roof = {"ms_per_step": zg_ms / psteps, "executed_TFLOPs": zg_exec / max(zg_ms, 1e-9) * 1e-9,
                  "pipe_frac_of_probe": zg_exec / max(zg_ms, 1e-9) * 1e-9 / peak_dmma,
                  "equiv_8mnk_TFLOPs": zg_def / max(zg_ms, 1e-9) * 1e-9}

    # ---- end to end through the public host-buffer API: pinned host Psi -> device -> path -> host (every step)
    e2e = None
    if args.e2e_steps > 0:
        psi_h = torch.empty((M, N), dtype=torch.complex128).pin_memory()
        src_h = torch.from_numpy(w.psi)
        g_h = torch.empty((M, M), dtype=torch.complex128).pin_memory() if spec.with_gram else None
        del psi, hpsi
        torch.cuda.empty_cache()

        def e2e_step():
            if spec.with_gram:
                binding.sweep_host(ham, psi_h, m, w.a, w.b, w.a0, g_h, block=blk)
            else:
                binding.cheb_filter_host(ham, psi_h, m, w.a, w.b, w.a0, block=blk)

        psi_h.copy_(src_h)
        e2e_step()                                   # warm-up (allocates the staging buffers)
        t_e2e = 0.0
        for _ in range(args.e2e_steps):
            psi_h.copy_(src_h)                       # untimed: restore the host input
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            e2e_step()                               # returns after its final device->host copy has completed
            t_e2e += time.perf_counter() - t0
        h2d = 16 * N * M
        d2h = 16 * N * M + (16 * M * M if spec.with_gram else 0)
        e2e = {"value": M * napps * args.e2e_steps / t_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "ms_per_step": 1e3 * t_e2e / args.e2e_steps,
               "api": "pwh_sweep_host" if spec.with_gram else "pwh_cheb_filter_host"}

    cpu = None
    if not args.no_cpu_baseline:
        cpu = cpu_baseline(w, args.cpu_seconds)

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(w), "band_applications_per_step": M * napps,
                       "filter_ms_per_block": filter_ms_block, "blocks": nblocks, "l2": "inputs (Psi, P) exceed L2; Psi restored from a device copy "
                       "at the start of every step inside the timed region", "parallelism": "replicas only",
                       "setup_s": t_gen},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
            "cpu_baseline": cpu,
            "stages": stage_out, "local_stage": local_roof, "zgemm_stage": zgemm_roof,
            "ms_per_step_profiled_pass": ms_step_profiled, "profiled_steps": psteps, "kernels": ham.kernels()}
    print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def profiled_traffic(cfg: int) -> dict:
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of the dominant kernels, read from the
    committed summary of the `ncu --set full` captures (profiles/ncu_traffic.json; each entry names the capture it was
    taken from).  Empty when no capture exists for this config."""
    try:
        return dict(json.load(open(os.path.join(ROOT, "profiles", "ncu_traffic.json"))).get(f"cfg{cfg}", {}))
    except Exception:
        return {}


def respawn_under_torchrun(args) -> int:
    """`python bench.py --gpus N` with N > 1 and no launcher: start N ranks (one per GPU) the way the driver does."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    args = parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return respawn_under_torchrun(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
