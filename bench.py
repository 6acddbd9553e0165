#!/usr/bin/env python
"""bench.py — MLUPS of the fused D3Q27 Reg-FLBM collide-stream step on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W]            # this repository's CUDA path
    python bench.py --impl reference [--steps K] [--warmup W]      # the CPU oracle, timed as it stands

A "step" is one time step of Eq.24 over the whole lattice: one launch of the fused
pull-stream + collide kernel.  Workload at N=1: BASELINE.json configs[3] — 512^3 periodic, fp64, tau=0.8,
kT=1e-4, seed 11, rho0=1, u=0 (the configuration the MLUPS metric is quoted on; 58 GB A-B workspace).
With --gpus N (torchrun, one rank per GPU) every rank runs an independent replica of that lattice
("replicas only": BASELINE.json fixes one GPU with no sharding and no collectives);
value = sites updated by all ranks / max-over-ranks device time.

One JSON line is printed by rank 0.  value: device-resident throughput (CUDA events on the launching stream
around K steps); sustained: the same measurement over a region of at least 2.5 s with its own clock samples (a short K
is a burst below the 1 kW power cap; the long region is what a production run sees); e2e: the same metric through rflbm_run_host with HOST (pinned) buffers, H2D of (rho,u),
K steps, D2H of the moments all inside the timed region; roofline: algorithmic bytes (2*27*8 B per site)
over the average launch time vs the measured HBM peak; cpu_baseline: the oracle on this box's host cores.
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

METRIC = "MLUPS per B200 (fp64 D3Q27 Reg-FLBM)"
UNIT = "MLUPS"
WORKLOAD = dict(size=512, tau=0.8, kT=1e-4, seed=11, rho0=1.0)
FALLBACK_HBM_GBS = 6650.0      # /opt/skills/guides/B200_PROFILING.md fallback if MEASURED_PEAKS.json is absent


def parse_args():
    p = argparse.ArgumentParser()
    p.add_argument("--gpus", type=int, default=1)
    p.add_argument("--steps", type=int, default=200)
    p.add_argument("--warmup", type=int, default=10)
    p.add_argument("--impl", default="ours", choices=["ours", "reference"])
    # development knobs (the driver does not pass them)
    p.add_argument("--size", type=int, default=WORKLOAD["size"])
    p.add_argument("--shape", default=None, help="nx,ny,nz instead of --size^3")
    p.add_argument("--kT", type=float, default=WORKLOAD["kT"])
    p.add_argument("--precision", default="f64", choices=["f64", "f32"])
    p.add_argument("--variant", default="auto", choices=["auto", "plain", "tma"])
    p.add_argument("--model", default="reg", choices=["reg", "bgk"])
    p.add_argument("--scheme", default="ab", choices=["ab", "aa"])
    p.add_argument("--decomp", default="replicas", choices=["replicas", "slab"],
                   help="N > 1: independent replicas (BASELINE.json: no sharding), or z slabs of ONE lattice of N times the "
                        "height with the faces exchanged every step (paper_2507_08820_b200/slab.py; PAPER.md:292, :300)")
    p.add_argument("--no-e2e", action="store_true")
    p.add_argument("--no-sustained", action="store_true")
    p.add_argument("--aux", action="store_true",
                   help="time the other device calls of the boundary (init, moments, stress, diagnostics, get/set_populations) "
                        "at the bench size instead of the step; one JSON line")
    p.add_argument("--e2e-serial", action="store_true")
    p.add_argument("--no-cpu", action="store_true")
    p.add_argument("--cpu-seconds", type=float, default=12.0)
    return p.parse_args()


# ----------------------------------------------------------------------------- helpers
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [t.strip() for t in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def hbm_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic_bytes(size, precision, scheme, model, kernel):
    """dram bytes per launch of the step kernel from the committed ncu --set full summary of exactly this variant
    (profiles/step_kernel_traffic_<size>_<precision>_<scheme>_<model>.txt, which names the kernel it was captured
    from); None when no capture of the timed variant is committed."""
    path = os.path.join(ROOT, "profiles", f"step_kernel_traffic_{size}_{precision}_{scheme}_{model}.txt")
    val, kern = None, None
    try:
        with open(path) as fh:
            for line in fh:
                if line.startswith("dram_bytes_per_launch="):
                    val = float(line.split("=", 1)[1])
                if line.startswith("kernel="):
                    kern = line.split("=", 1)[1].strip()
    except OSError:
        return None
    return val if (kern is None or kern == kernel) else None


def dist_setup(n_gpus):
    """(rank, world, local_rank); initialises NCCL when launched by torchrun."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        import torch
        backend = "nccl" if torch.cuda.is_available() else "gloo"
        dist.init_process_group(backend, rank=rank, world_size=world)
    return rank, world, local


def barrier_all():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(value, device=None):
    """max over all ranks of a python float (device time in ms): the job finishes when the slowest rank does."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value, device=None):
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


# ----------------------------------------------------------------------------- CPU oracle leg
def time_oracle(steps, warmup, seconds=None, size=64, cores=None):
    """Oracle as it stands on the host cores: `size`^3 sample of the workload, all cores (OpenMP over z) unless
    `cores` is given."""
    import oracle
    cores = oracle.max_threads() if cores is None else cores
    ref = oracle.Ref(size, size, size, WORKLOAD["tau"], WORKLOAD["kT"], WORKLOAD["rho0"], WORKLOAD["seed"],
                     threads=cores)
    ref.init()
    ref.step(max(1, warmup))
    if seconds is not None:                      # bounded: choose the step count for ~`seconds` of CPU work
        t0 = time.perf_counter(); ref.step(2); dt = (time.perf_counter() - t0) / 2
        steps = max(2, min(steps, int(seconds / max(dt, 1e-6))))
    t0 = time.perf_counter()
    ref.step(steps)
    dt = time.perf_counter() - t0
    mlups = size ** 3 * steps / dt / 1e6
    return mlups, cores, steps, dt, f"{size}^3 periodic sub-lattice of the workload (same tau, kT, seed), {steps} steps"


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    size = 64
    mlups, cores, steps, dt, sample = time_oracle(args.steps, args.warmup, seconds=None, size=size)
    line = {
        "impl": "reference", "metric": METRIC, "value": mlups, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": args.warmup, "ms_per_step": dt / steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "512^3 periodic D3Q27 Reg-FLBM fp64, tau=0.8, kT=1e-4, seed 11 (BASELINE configs[3]); "
                               "each step = one oracle time step on a 64^3 sample of it", "l2": "n/a (CPU)"},
        "cpu_baseline": {"value": mlups, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": mlups, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------- CUDA leg
def run_ours(args):
    import torch
    from paper_2507_08820_b200 import binding

    rank, world, local = dist_setup(args.gpus)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: CUDA is not available and the rflbm path has no CPU fallback")
    dev = torch.device(f"cuda:{local}")
    torch.cuda.set_device(dev)
    n = args.size
    nx, ny, nz = (int(v) for v in args.shape.split(",")) if args.shape else (n, n, n)
    prec = binding.F64 if args.precision == "f64" else binding.F32
    es = 8 if prec == binding.F64 else 4
    N = nx * ny * nz
    K, W = args.steps, max(3, args.warmup)

    scheme = binding.SCHEME_AA if args.scheme == "aa" else binding.SCHEME_AB
    lat = None
    if args.decomp == "slab":                       # one lattice nx x ny x (nz * world): every rank owns nz layers of it
        from paper_2507_08820_b200 import slab
        lat = slab.SlabLattice(nx, ny, nz * world, WORKLOAD["tau"], args.kT, WORKLOAD["rho0"], WORKLOAD["seed"], prec,
                               device=dev, scheme=scheme)
        sim, step = lat.sim, lat.step
        args.no_e2e = True                          # rflbm_run_host is the single-handle job
    else:
        sim = binding.Rflbm(nx, ny, nz, WORKLOAD["tau"], args.kT, WORKLOAD["rho0"], WORKLOAD["seed"], prec, device=dev,
                            scheme=scheme)
        step = sim.step
    sim.set_kernel_variant({"auto": binding.KERNEL_AUTO, "plain": binding.KERNEL_PLAIN, "tma": binding.KERNEL_TMA}[args.variant])
    if args.model == "bgk":
        sim.set_model(binding.MODEL_BGK)
    if lat is not None:
        lat.init()
    else:
        sim.init()
    step(W)                                         # warm-up: also thermalises the state
    torch.cuda.synchronize(dev)

    # ---- device-resident timing: K launches of the step kernel, CUDA events on the launching stream
    stream = sim.stream
    vis = [v for v in os.environ.get("CUDA_VISIBLE_DEVICES", "").split(",") if v.strip()]
    smi_index = vis[local] if local < len(vis) else local

    def timed_region(nsteps):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        sampler = ClockSampler(smi_index)
        l0 = sim.launch_count
        barrier_all(); torch.cuda.synchronize(dev)
        if rank == 0:
            sampler.start()
        ev0.record(stream)
        step(nsteps)
        ev1.record(stream)
        torch.cuda.synchronize(dev); barrier_all()
        clk = sampler.stop() if rank == 0 else None
        return ev0.elapsed_time(ev1), sim.launch_count - l0, clk

    ms_local, launches, clocks = timed_region(K)
    ms = max_over_ranks(ms_local, dev)
    value = N * K * world / (ms * 1e-3) / 1e6
    kernel = sim.last_kernel                         # what the library launched (rflbm_last_kernel), not a guess

    # ---- sustained: the same measurement over >= 2.5 s (the part reaches its 1 kW cap after a few hundred ms; a
    # 20-step region is a burst).  Every rank runs the same number of steps.
    sustained = None
    if not args.no_sustained:
        if ms >= 2500.0:
            sustained = {"steps": K, "ms_per_step": ms / K, "value": value, "clocks": clocks, "same_region_as_value": True}
        else:
            Ks = int(max_over_ranks(max(K, 2500.0 / max(ms / K, 1e-3)) + 1, dev))
            ms_s_local, _, clk_s = timed_region(Ks)
            ms_s = max_over_ranks(ms_s_local, dev)
            sustained = {"steps": Ks, "ms_per_step": ms_s / Ks, "value": N * Ks * world / (ms_s * 1e-3) / 1e6,
                         "clocks": clk_s, "same_region_as_value": False}

    # conservation after the run (cheap sanity on the timed state)
    d = sim.diagnostics()
    mass_err = abs(d[0] / N / WORKLOAD["rho0"] - 1.0)

    # ---- end to end through the C-ABI with HOST buffers
    e2e = None
    if not args.no_e2e:
        shape = (nz, ny, nx)
        dt = torch.float64 if prec == binding.F64 else torch.float32
        rho_h = torch.full(shape, WORKLOAD["rho0"], dtype=dt).pin_memory()
        u_h = torch.zeros((3,) + shape, dtype=dt).pin_memory()
        rho_o = torch.empty(shape, dtype=dt).pin_memory()
        u_o = torch.empty((3,) + shape, dtype=dt).pin_memory()
        scratch = torch.empty(4 * N * es, dtype=torch.uint8, device=dev)
        copy_stream = torch.cuda.Stream(device=dev)
        sim.set_copy_stream(None if args.e2e_serial else copy_stream)  # pipelined (time-skewed along z) unless --e2e-serial
        sim.run_host(rho_h, u_h, 2, rho_o, u_o, scratch)              # warm the copy path
        barrier_all(); torch.cuda.synchronize(dev)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        sim.run_host(rho_h, u_h, K, rho_o, u_o, scratch)              # H2D + init + K steps + moments + D2H + sync
        e1.record(stream)
        torch.cuda.synchronize(dev); barrier_all()
        ms_e = max_over_ranks(e0.elapsed_time(e1), dev)
        e2e = {"value": N * K * world / (ms_e * 1e-3) / 1e6, "unit": UNIT,
               "h2d_bytes_per_step": 4 * N * es / K, "d2h_bytes_per_step": 4 * N * es / K,
               "ms_total": ms_e, "pipelined": not args.e2e_serial,
               "what": "rflbm_run_host: pinned host rho,u -> device, init, K steps, moments, device -> pinned host, "
                       "sync; bytes are per job / K; copies on a second stream in bands of z layers, the steps time-skewed behind the upload front, the download behind the last step: all overlapped with the "
                       "kernels (include/rflbm.h)" if not args.e2e_serial else
                       "rflbm_run_host, serial form: pinned host rho,u -> device, init, K steps, moments, device -> "
                       "pinned host, sync; bytes are per job / K"}
        assert abs(float(rho_o.double().mean()) / WORKLOAD["rho0"] - 1.0) < 1e-9
        # what came back to the host is, bit for bit, the moments of the state the job left on the device (the pipelined
        # job assembles them band by band; tests/test_gpu_parity.py ties the serial form to the oracle)
        del scratch
        rho_d, u_d = sim.moments()
        e2e["outputs_equal_device_moments"] = bool(torch.equal(rho_o.to(dev), rho_d)) and all(
            bool(torch.equal(u_o[a].to(dev), u_d[a])) for a in range(3))
        assert e2e["outputs_equal_device_moments"] and sim.step_count == K
        del rho_h, u_h, rho_o, u_o, rho_d, u_d

    if rank != 0:
        return 0

    peak, peak_src = hbm_peak()
    bytes_per_launch = 2 * 27 * es * N
    achieved = bytes_per_launch / (ms_local / K * 1e-3) / 1e9
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": ncu_traffic_bytes(n, args.precision, args.scheme, args.model, kernel) if (args.kT > 0 and not args.shape) else None,
                "peak_source": peak_src, "kernel": kernel,
                "algorithmic_bytes_per_launch": bytes_per_launch,
                "avg_launch_ms": ms_local / K}
    if sustained is not None:
        sustained["hbm_gbs"] = bytes_per_launch * world / (sustained["ms_per_step"] * 1e-3) / 1e9 / world
        sustained["frac"] = sustained["hbm_gbs"] / peak
        # a reader of `roofline` alone must see what the kernel HOLDS under the power cap, not only the burst
        roofline["achieved_sustained"] = sustained["hbm_gbs"]
        roofline["frac_sustained"] = sustained["frac"]
        roofline["sustained_avg_launch_ms"] = sustained["ms_per_step"]
        roofline["sustained_steps"] = sustained["steps"]
        roofline["sustained_clocks"] = sustained["clocks"]
        roofline["frac_is"] = ("the value region itself (>= 2.5 s)" if sustained["same_region_as_value"] else
                               f"a burst: the value region lasts {ms / 1e3:.2f} s; frac_sustained is the same kernel over "
                               f"{sustained['steps']} back-to-back launches (>= 2.5 s, at the clock the part holds under its power cap)")

    cpu = None
    if not args.no_cpu:
        mlups, cores, csteps, cdt, sample = time_oracle(10 ** 6, 1, seconds=args.cpu_seconds, size=64)
        m1, _, s1, dt1, sample1 = time_oracle(10 ** 6, 1, seconds=args.cpu_seconds / 3, size=64, cores=1)
        m128, _, s128, dt128, sample128 = time_oracle(10 ** 6, 1, seconds=args.cpu_seconds / 3, size=128)   # 0.9 GB: far out of cache
        cpu = {"value": mlups, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "seconds": cdt,
               "one_core": {"value": m1, "unit": UNIT, "cores": 1, "sample": sample1, "seconds": dt1},
               "out_of_cache": {"value": m128, "unit": UNIT, "cores": cores, "sample": sample128, "seconds": dt128}}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": args.precision, "data": "synthetic",
        "config": {"workload": f"{nx}x{ny}x{nz} periodic D3Q27 {'BGK-FLBM' if args.model == 'bgk' else 'Reg-FLBM'} {args.precision}, "
                               f"rho0=1, u=0, tau=0.8, kT={args.kT:g}, seed 11"
                               + (" (BASELINE configs[3])" if (nx, ny, nz, args.precision, args.model, args.kT) == (512, 512, 512, "f64", "reg", 1e-4) else "")
                               + (f"; A-B double buffer {2 * 27 * es * N / 1e9:.1f} GB" if args.scheme == "ab"
                                  else f"; in-place AA buffer {27 * es * N / 1e9:.1f} GB"),
                   "scheme": args.scheme, "model": args.model, "kernel_variant": args.variant,
                   "l2": "no flush needed: each step streams 2*27*N*sizeof(real) bytes >> 126 MB L2",
                   "parallelism": ("single GPU" if world == 1 else "replicas only") if lat is None else
                                  f"z slabs: ONE {nx}x{ny}x{nz * world} lattice, {nz} layers per rank, 2 faces of "
                                  f"{lat.face_bytes / 1e6:.1f} MB per rank and step ({lat.transport.backend} send/recv; "
                                  "one rank: device-to-device through the pack/unpack kernels)"},
        "clocks": clocks, "sustained": sustained, "e2e": e2e, "gpu_launches": launches, "roofline": roofline,
        "cpu_baseline": cpu, "hbm_gbs": achieved, "mass_rel_err": mass_err,
    }
    print(json.dumps(line))
    return 0


def run_aux(args):
    """The calls of include/rflbm.h around the step: device time and algorithmic bytes of each at
    the bench size, thermalised state, best of 5 (CUDA events on the handle's stream)."""
    import torch
    from paper_2507_08820_b200 import binding
    dev = torch.device("cuda:0")
    n = args.size
    nx, ny, nz = (int(v) for v in args.shape.split(",")) if args.shape else (n, n, n)
    prec = binding.F64 if args.precision == "f64" else binding.F32
    es = 8 if prec == binding.F64 else 4
    N = nx * ny * nz
    sim = binding.Rflbm(nx, ny, nz, WORKLOAD["tau"], args.kT, WORKLOAD["rho0"], WORKLOAD["seed"], prec, device=dev,
                        scheme=binding.SCHEME_AA if args.scheme == "aa" else binding.SCHEME_AB)
    sim.init()
    sim.step(5)
    dt = sim.dtype
    rho = torch.empty((nz, ny, nx), dtype=dt, device=dev); u = torch.empty((3, nz, ny, nx), dtype=dt, device=dev)
    pi = torch.empty((6, nz, ny, nx), dtype=dt, device=dev)
    f = torch.empty((27, nz, ny, nx), dtype=dt, device=dev)
    sim.get_populations(f)
    # (call, values read per site, values written per site)
    calls = [("rflbm_moments", lambda: sim.moments(rho, u), 27, 4), ("rflbm_stress", lambda: sim.stress(pi), 27, 6),
             ("rflbm_snapshot", lambda: sim.snapshot(rho, u, pi), 27, 10),
             ("rflbm_diagnostics", lambda: sim.diagnostics(), 27, 0), ("rflbm_get_populations", lambda: sim.get_populations(f), 27, 27),
             ("rflbm_set_populations", lambda: sim.set_populations(f, 5), 27, 27),
             ("rflbm_init(rho,u)", lambda: sim.init(rho, u), 4, 27), ("rflbm_init(NULL)", lambda: sim.init(), 0, 27)]
    peak, peak_src = hbm_peak()
    out = {}
    for name, fn, nr, nw in calls:
        best = None
        for _ in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize(dev)
            e0.record(sim.stream); fn(); e1.record(sim.stream)
            torch.cuda.synchronize(dev)
            ms = e0.elapsed_time(e1)
            best = ms if best is None else min(best, ms)
        gbs = (nr + nw) * es * N / (best * 1e-3) / 1e9
        out[name] = {"ms": best, "bytes_per_site": (nr + nw) * es, "gbs": gbs, "frac": gbs / peak}
    print(json.dumps({"aux": out, "config": {"workload": f"{nx}x{ny}x{nz} {args.precision} {args.scheme}"}, "peak_gbs": peak,
                      "peak_source": peak_src, "note": "rflbm_diagnostics includes its host read-back of ten sums"}))
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.aux:
        return run_aux(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
