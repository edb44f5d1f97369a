#!/usr/bin/env python
"""bench.py -- one JSON line for the SPH density + hydro-force hot path on B200.

A *step* is one pass of the whole hot path (DESIGN.md steps a1-a11) over one synthetic particle set:
sph_build_index -> sph_density (smoothing-length iteration to convergence) -> sph_hydro_force.
The default workload is BASELINE.json configs[3], the 10^7-particle clustered set (Wendland C6,
N_ngb = 295) that the metric's roofline target is quoted on; `--workload C1|C2|C3|C5` selects the
others.  `value` = active-particle updates / s with all inputs resident in HBM; `e2e` = the same
through sph_step_host with pinned HOST buffers (copies inside the timed region).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C4] [--n N]

N > 1 (launched by torch.distributed.run): the path does not shard (one GPU, no exchange step --
DESIGN.md "Multi-GPU"), so every rank runs an independent replica of the workload: weak scaling,
value = N x updates / max-over-ranks time.

`--impl reference`: this tier has no reference implementation; the arm times the fp64 CPU oracle
(oracle/, as it stands) on the host cores, on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "active-particle SPH updates/sec (density+force)"
UNIT = "updates/s"

# algorithmic flops per true pair (frozen from the oracle's inner loops)
FLOP_DENSITY_PAIR = {0: 30.0, 1: 40.0}  # cubic spline / Wendland C6
FLOP_FORCE_PAIR = 80.0
# derived FP32 peak: 148 SMs x 128 FP32 lanes x 2 flop/FMA x max SM clock; reported beside
# the measured one (bench_probe.cu), which is the roofline's denominator
FP32_LANES_PER_SM = 128
PROBE_SRC = os.path.join(ROOT, "bench_probe.cu")
PROBE_LIB = os.path.join(ROOT, "bench_probe.so")


def build_probe(force: bool = False) -> str:
    """nvcc -> bench_probe.so (the FP32 FMA issue-rate probe; bench harness only, not part of libsph.so)."""
    if force or not os.path.exists(PROBE_LIB) or os.path.getmtime(PROBE_LIB) < os.path.getmtime(PROBE_SRC):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "--shared",
                               "-Xcompiler", "-fPIC", "-o", PROBE_LIB, PROBE_SRC])
    return PROBE_LIB


def fp32_peak(stream_ptr: int, packed: bool, iters: int = 32) -> float:
    """Measured FP32 FMA rate of this device in TFLOP/s (register-only FMA chains on every SM)."""
    import ctypes as C

    lib = C.CDLL(build_probe())
    lib.bench_fp32_peak.argtypes = [C.c_void_p, C.c_int, C.c_int, C.POINTER(C.c_double)]
    out = C.c_double(0.0)
    rc = lib.bench_fp32_peak(C.c_void_p(stream_ptr), iters, int(packed), C.byref(out))
    if rc:
        raise RuntimeError(f"bench_fp32_peak: cudaError {rc}")
    return float(out.value)


def make_workload(name: str, n: int | None):
    from paper_2003_10850_b200 import inputs as I

    name = name.upper()
    if name == "C1":
        ps = I.config1() if n is None else I.config1(max(2, round(n ** (1 / 3))))
    elif name == "C2":
        ps = I.config2() if n is None else I.config2(max(2, round(n ** (1 / 3))))
    elif name == "C3":
        ps = I.config3() if n is None else I.config3(n, max(2, n // 10000))
    elif name in ("C4", "C5"):
        ps = I.config4() if n is None else I.config4(n, max(2, n // 5000), m_hi=max(2000.0, n / 10.0))
    else:
        raise SystemExit(f"unknown workload {name}")
    return ps


def sfc_order(ps, active_np):
    """--sfc-order: the same particle set handed over in space-filling-curve order of the positions (the paper keeps its
    particles in Hilbert order; here a 3 x 16-bit Morton order), instead of the generator's order.  Only the
    order of the caller's arrays changes: the gathers / scatters between caller order and the library's sorted order
    become nearly sequential."""
    def spread(v):
        v = v.astype(np.uint64)
        v = (v | (v << 32)) & np.uint64(0x1F00000000FFFF)
        v = (v | (v << 16)) & np.uint64(0x1F0000FF0000FF)
        v = (v | (v << 8)) & np.uint64(0x100F00F00F00F00F)
        v = (v | (v << 4)) & np.uint64(0x10C30C30C30C30C3)
        v = (v | (v << 2)) & np.uint64(0x1249249249249249)
        return v
    c = np.minimum((ps.pos.astype(np.float64) / ps.box * 65536.0).astype(np.int64), 65535)
    key = spread(c[:, 0]) | (spread(c[:, 1]) << np.uint64(1)) | (spread(c[:, 2]) << np.uint64(2))
    order = np.argsort(key, kind="stable")
    ps.pos, ps.vel, ps.u, ps.h_guess = ps.pos[order], ps.vel[order], ps.u[order], ps.h_guess[order]
    if active_np is not None:
        inv = np.empty(len(order), np.int64)
        inv[order] = np.arange(len(order))
        active_np = np.sort(inv[active_np]).astype(np.int32)
    return active_np


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={gpu_index}", f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "50"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons, pw = [], [], set(), []
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2])); pw.append(float(c[3]))
            except ValueError:
                continue
            for nm, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons),
                       samples=len(sm), power_w_max=float(max(pw)))
        return out


def oracle_sample_run(ps, active_all, sample: int, seed: int):
    """The oracle, as it stands, on `sample` active particles of the workload: density (h iteration)
    then hydro force.  Neighbours outside the sample enter the force with the generator's state
    (h guess, analytic density, Omega = 1) -- timing only, no value of it is compared.  Returns
    (seconds, updates, threads)."""
    from oracle import sph_oracle as O

    rng = np.random.default_rng(seed)
    pool = np.arange(ps.n, dtype=np.int32) if active_all is None else active_all
    act = np.sort(rng.choice(pool, min(sample, len(pool)), replace=False)).astype(np.int32)
    nd = ps.aux.get("n_density")
    rho = (np.full(ps.n, float(ps.n)) if nd is None else nd) * ps.mass
    rho = rho.astype(np.float32)
    om = np.ones(ps.n, np.float32)
    h = ps.h_guess.copy()
    t0 = time.perf_counter()
    o = O.density(ps.pos, ps.h_guess, kernel=ps.kernel, n_target=ps.n_ngb, n_tol=ps.n_tol, mass_scalar=ps.mass,
                  active=act)
    h[act] = o["H"]; rho[act] = o["rho"]; om[act] = o["omega"]
    O.hydro_force(ps.pos, ps.vel, ps.u, h, rho, om, kernel=ps.kernel, mass_scalar=ps.mass, active=act)
    dt = time.perf_counter() - t0
    return dt, len(act), O.num_threads()


def default_sample(ps) -> int:
    # sized for roughly 10-30 s of oracle work on the box's host cores (measured on 16 cores: ~1.8e4 updates/s
    # at C4; the 64-neighbour configs are several times faster per update)
    return 262144 if ps.kernel == 1 else 1048576


def run_reference(args, rank: int):
    """--impl reference: the oracle timed on the host cores (rank 0 only)."""
    if rank != 0:
        return
    ps = make_workload(args.workload, args.n)
    from paper_2003_10850_b200 import inputs as I
    from oracle import sph_oracle as O

    O.build()
    active = I.config5_active(ps) if args.workload.upper() == "C5" else None
    sample = args.cpu_sample or max(256, default_sample(ps) // 4)
    for w in range(args.warmup):
        oracle_sample_run(ps, active, max(64, sample // 16), 1000 + w)
    tot_t, tot_u, thr = 0.0, 0, 1
    for k in range(args.steps):
        dt, nu, thr = oracle_sample_run(ps, active, sample, 2000 + k)
        tot_t += dt; tot_u += nu
    val = tot_u / tot_t
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(args, ps, active),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": thr, "kind": "oracle",
                         "sample": f"{sample} seeded random active particles of the workload per step (density h-iteration "
                                   "+ hydro force); neighbours keep the generator's state"},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_config(args, ps, active):
    names = {"C1": "configs[0]", "C2": "configs[1]", "C3": "configs[2]", "C4": "configs[3]", "C5": "configs[4]"}
    w = args.workload.upper()
    return {
        "workload": f"{w} = BASELINE.json {names[w]}" + ("" if args.n is None else f" scaled to n={ps.n}")
                    + (" (caller arrays in Morton order: --sfc-order)" if getattr(args, "sfc_order", False) else ""),
        "n_particles": ps.n, "n_active": ps.n if active is None else int(len(active)),
        "kernel": "wendland_c6" if ps.kernel == 1 else "cubic_spline", "n_ngb": ps.n_ngb, "n_tol": ps.n_tol,
        "step": "sph_build_index + sph_density(h iteration) + sph_hydro_force",
        "l2": "inputs larger than L2 (particle state > 126 MB) -- no explicit flush" if ps.n * 76 > 126e6
              else "explicit L2 flush (256 MB write) between timed steps",
        "parallelism": "replicas (path does not shard)" if args.gpus > 1 else "1 GPU",
    }


def max_over_ranks(x: float, world: int, device: str) -> float:
    """Timing rule: every multi-rank number is the MAX over ranks (replicas: the slowest GPU sets the time)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist

    t = torch.tensor([x], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, n_active: int, steps: int, ms: float) -> float:
    """Whole-job throughput: every rank runs one replica of the workload (weak scaling, no exchange step)."""
    return world * n_active * steps / (ms * 1e-3)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C4")
    ap.add_argument("--n", type=int, default=None, help="scale the workload to n particles (development)")
    ap.add_argument("--cpu-sample", type=int, default=None)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extension", action="store_true", help="skip the improved-SPH extension timing")
    ap.add_argument("--kdk-steps", type=int, default=0,
                    help="after the timed region, run this many steps of the kick-drift-kick driver (SURVEY.md 8(f)-3) on the "
                         "workload and report active counts and times per step")
    ap.add_argument("--sfc-order", action="store_true",
                    help="hand the particle set over in Morton order of the positions (variant run; default: generator order)")
    ap.add_argument("--kdk-refresh-max", type=int, default=16,
                    help="sph_kdk_params.refresh_max: steps in a row that refresh the index instead of rebuilding it (0 = never)")
    ap.add_argument("--group-cap", type=int, default=0, help="actives per group (0 = library default)")
    ap.add_argument("--group-node", type=int, default=0, help="group-node capacity (0 = library default)")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2003_10850_b200 import binding as B
    from paper_2003_10850_b200 import inputs as I

    ps = make_workload(args.workload, args.n)
    n = ps.n
    w = args.workload.upper()
    active_np = I.config5_active(ps) if w == "C5" else None
    if args.sfc_order:
        active_np = sfc_order(ps, active_np)
    dev = lambda a, dt=torch.float32: torch.from_numpy(np.ascontiguousarray(a)).to(dt).cuda()
    pos, vel, u, h_guess = dev(ps.pos), dev(ps.vel), dev(ps.u), dev(ps.h_guess)
    active = None if active_np is None else dev(active_np, torch.int32)
    h = h_guess.clone()
    rho, om, du, vs = (torch.zeros(n, device="cuda") for _ in range(4))
    ngb = torch.zeros(n, device="cuda", dtype=torch.int32)
    acc = torch.zeros((n, 3), device="cuda")
    # a stream of its own (the legacy default stream cannot be captured: sph_build_index replays its launches from a CUDA
    # graph from the third identical call on); every torch operation of the bench runs on it as well
    stream = torch.cuda.Stream()
    torch.cuda.set_stream(stream)
    sph = B.Sph(kernel=ps.kernel, stream=stream, group_cap=args.group_cap, group_node=args.group_node)
    n_active = n if active is None else int(active.numel())
    flush = None if n * 76 > 126e6 else torch.empty(64 << 20, device="cuda", dtype=torch.float32)

    if w == "C5":
        # C5 state: the converged (h, rho, Omega) of the whole set, then the active particles' h perturbed
        sph.sph_build_index(pos, None, ps.mass)
        sph.sph_density(h, rho, om, ngb, ps.n_ngb, ps.n_tol)
        hc = h.cpu().numpy()
        h_guess = dev(I.perturb_h(hc, active_np, I.SEED_BASE + 5))
        h.copy_(h_guess)

    def step():
        if active is None:
            h.copy_(h_guess)
        else:
            h.index_copy_(0, active.long(), h_guess.index_select(0, active.long()))
        sph.sph_build_index(pos, None, ps.mass)
        unconv = sph.sph_density(h, rho, om, ngb, ps.n_ngb, ps.n_tol, active=active)
        sph.sph_hydro_force(vel, u, h, rho, om, acc, du, vs, active=active)
        return unconv

    peak_scalar = fp32_peak(stream.cuda_stream, False)
    peak_packed = fp32_peak(stream.cuda_stream, True)
    for _ in range(max(args.warmup, 0)):
        step()
        if flush is not None:
            flush.zero_()
    torch.cuda.synchronize()
    l0 = sph.stats()["launches"]

    sampler = ClockSampler(local)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    per = []
    t_flush = 0.0
    e0.record(stream)
    for _ in range(args.steps):
        unconv = step()
        per.append(sph.stats())  # synchronises; reads the library's own event times of this step's kernels
        per[-1]["unconv"] = unconv
        if flush is not None:
            f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            f0.record(stream); flush.zero_(); f1.record(stream); torch.cuda.synchronize()
            t_flush += f0.elapsed_time(f1)
    e1.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1) - t_flush
    # evaluation histogram of the h iteration (outside the timed region): one more density pass with status
    stt = torch.zeros(n, device="cuda", dtype=torch.int32)
    if active is None:
        h.copy_(h_guess)
    else:
        h.index_copy_(0, active.long(), h_guess.index_select(0, active.long()))
    sph.sph_density(h, rho, om, ngb, ps.n_ngb, ps.n_tol, active=active, status=stt)
    its = (stt & 0xff) if active is None else (stt.index_select(0, active.long()) & 0xff)
    eval_hist = torch.bincount(its.long(), minlength=2).cpu().tolist()
    launches = per[-1]["launches"] - l0
    # active-subset workloads: the same step with sph_refresh_index in place of sph_build_index (what sph_kdk_step does on
    # steps with few active particles), outside the timed region; `value` stays the rebuild step's
    refresh_step = None
    if active is not None:
        k = max(3, min(args.steps, 50))
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for rep in range(2):  # first round warms up
            r0.record(stream)
            for _ in range(k):
                h.index_copy_(0, active.long(), h_guess.index_select(0, active.long()))
                sph.sph_refresh_index(pos)
                sph.sph_density(h, rho, om, ngb, ps.n_ngb, ps.n_tol, active=active)
                sph.sph_hydro_force(vel, u, h, rho, om, acc, du, vs, active=active)
            r1.record(stream)
            torch.cuda.synchronize()
        refresh_step = {"ms_per_step": r0.elapsed_time(r1) / k, "steps": k,
                        "step": "sph_refresh_index + sph_density(h iteration) + sph_hydro_force",
                        "updates_per_s": n_active * k / (r0.elapsed_time(r1) * 1e-3)}
    # improved-SPH extension, outside the timed region: cost of the velocity-gradient pass and of the
    # force pass with per-particle alpha, shear limiter and conduction on the same converged state (CUDA events)
    ext_ms = None
    if not args.no_extension:
        dvv, da = torch.zeros(n, device="cuda"), torch.zeros(n, device="cuda")
        cvv = torch.zeros((n, 3), device="cuda")
        alp = torch.full((n,), 1.0, device="cuda")
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        for rep in range(2):  # first round warms up
            ev[0].record(stream)
            sph.sph_velocity_gradients(vel, h, rho, dvv, cvv, active=active)
            ev[1].record(stream)
            sph.sph_hydro_force_improved(vel, u, h, rho, om, alp, dvv, cvv, acc, du, vs, da, active=active)
            ev[2].record(stream)
            torch.cuda.synchronize()
        ext_ms = {"velocity_gradients": ev[0].elapsed_time(ev[1]), "hydro_force_improved": ev[1].elapsed_time(ev[2]),
                  "note": "whole calls incl. the sorted-state preparation; base sph_hydro_force in phases_ms"}
        # short-range Barnes-Hut gravity with TreePM-like parameters: mesh cell = half the mean particle
        # spacing, r_s = 1.25 cells, r_cut = 4.5 r_s, softening = spacing / 40, opening angle 0.5
        cell = 0.5 / n ** (1.0 / 3.0)
        gk = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        for rep in range(2):
            gk[0].record(stream)
            sph.sph_gravity_short(acc, 1.0, 1.25 * cell, 4.5 * 1.25 * cell, 2.0 * cell / 40.0, 0.5, active=active)
            gk[1].record(stream)
            torch.cuda.synchronize()
        ext_ms["gravity_short_theta0.5"] = gk[0].elapsed_time(gk[1])
    ms = max_over_ranks(ms, world, "cuda")
    value = whole_job_value(world, n_active, args.steps, ms)

    kdk = None
    if args.kdk_steps > 0:
        # the time-bin driver on this set: real active lists step after step; dt_max = 4 x the median
        # Courant step so that several bins are occupied
        vs0 = float(torch.median(vs).item()) if float(vs.max().item()) > 0 else 1.0
        dt_med = 0.3 * float(torch.median(h).item()) / max(vs0, 1e-30)
        stt_ = dict(pos=pos.clone(), vel=vel.clone(), u=u.clone(), h=h.clone(), rho=rho.clone(), omega=om.clone(), ngb=ngb.clone(),
                    acc=torch.zeros((n, 3), device="cuda"), dudt=torch.zeros(n, device="cuda"), vsig=torch.zeros(n, device="cuda"),
                    vpred=torch.zeros((n, 3), device="cuda"), upred=torch.zeros(n, device="cuda"),
                    bin=torch.zeros(n, device="cuda", dtype=torch.int32), tbegin=torch.zeros(n, device="cuda", dtype=torch.int32),
                    active=torch.zeros(n, device="cuda", dtype=torch.int32))
        sph.sph_kdk_init(stt_, ps.mass, 4.0 * dt_med, 12, ps.n_ngb, ps.n_tol, refresh_max=args.kdk_refresh_max)
        torch.cuda.synchronize()
        rows = []
        for _ in range(args.kdk_steps):
            k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            k0.record(stream)
            tick, na = sph.sph_kdk_step(stt_, ps.mass)
            k1.record(stream)
            torch.cuda.synchronize()
            rows.append((tick, na, k0.elapsed_time(k1)))
        tot_a, tot_ms = sum(r[1] for r in rows), sum(r[2] for r in rows)
        kdk = {"steps": len(rows), "dt_max": 4.0 * dt_med, "n_bins": 12, "refresh_max": args.kdk_refresh_max, "active_per_step": [r[1] for r in rows],
               "ms_per_step": [round(r[2], 3) for r in rows], "updates_per_s": tot_a / (tot_ms * 1e-3),
               "bins_occupied": sorted(set(torch.unique(stt_["bin"]).cpu().tolist()))}

    # e2e: the same step through sph_step_host, pinned host buffers, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        hp, hv, hu = pin(ps.pos), pin(ps.vel), pin(ps.u)
        hg_np = h_guess.cpu().numpy()
        hh = pin(hg_np.copy())
        hrho, hom, hdu, hvs = pin(rho.cpu().numpy()), pin(om.cpu().numpy()), pin(np.zeros(n, np.float32)), pin(np.zeros(n, np.float32))
        hngb = pin(np.zeros(n, np.int32))
        hacc = pin(np.zeros((n, 3), np.float32))
        hact = None if active_np is None else pin(active_np)
        hg_pin = pin(hg_np)
        sph2 = B.Sph(kernel=ps.kernel, stream=stream, group_cap=args.group_cap, group_node=args.group_node)
        tt = []
        for k in range(1 + args.steps):
            hh.copy_(hg_pin)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            sph2.sph_step_host(hp, hv, hu, ps.mass, hh, hrho, hom, hngb, hacc, hdu, hvs, ps.n_ngb, ps.n_tol, active=hact)
            tt.append(time.perf_counter() - t0)
        t_e2e = sum(tt[1:])  # first call (allocations) is warm-up
        t_e2e = max_over_ranks(t_e2e, world, "cuda")
        h2d = n * 32 + (0 if hact is None else 4 * len(active_np) + 8 * n)
        d2h = n * 44 if hact is None else 36 * len(active_np)  # an active list: only the actives' results travel back
        e2e = {"value": world * n_active * args.steps / t_e2e, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "ms_per_step": 1e3 * t_e2e / args.steps}
        sph2.close()

    if rank == 0:
        # roofline of the dominant kernel = the gather kernel with the larger event time in this run
        tk = float(np.mean([p["t_density_kernel_ms"] for p in per]))
        tf = float(np.mean([p["t_force_kernel_ms"] for p in per]))
        ti = float(np.mean([p["t_index_ms"] for p in per]))
        tp = float(np.mean([p["t_force_prep_ms"] for p in per]))
        st = per[-1]
        fl_d = FLOP_DENSITY_PAIR[ps.kernel] * st["dens_pairs"]
        fl_f = FLOP_FORCE_PAIR * st["force_pairs"]
        sm_count = torch.cuda.get_device_properties(local).multi_processor_count
        sm_max = clocks.get("sm_max_mhz") or 1965.0
        derived = sm_count * FP32_LANES_PER_SM * 2 * sm_max * 1e6 * 1e-12
        peak = peak_packed  # measured on this device in this run; the derived figure beside it
        hbm_peak, hbm_src = 6650.0, "fallback of B200_PROFILING.md (MEASURED_PEAKS.json absent)"
        try:
            hbm_peak = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"])
            hbm_src = "measured copy bandwidth, MEASURED_PEAKS.json"
        except (OSError, KeyError, ValueError):
            pass
        # DRAM bytes per launch from the committed ncu capture (profiles/traffic.csv), labelled with its commit
        traffic = {}
        tpath = os.path.join(ROOT, "profiles", "traffic.csv")
        if os.path.exists(tpath):
            import csv
            for row in csv.DictReader(open(tpath)):
                if row["workload"] == w:
                    traffic[row["kernel"]] = (int(row["dram_bytes_per_launch"]), row.get("commit", "?"))

        def kroof(name, steps_, flops, t_ms):
            tr = traffic.get(name)
            return {"kernel": f"{name} ({steps_})", "achieved": flops / (t_ms * 1e-3) * 1e-12, "frac": flops / (t_ms * 1e-3) * 1e-12 / peak,
                    "frac_of_derived": flops / (t_ms * 1e-3) * 1e-12 / derived, "kernel_ms": t_ms,
                    "algorithmic_flops_per_launch": flops, "traffic": None if tr is None else tr[0],
                    "traffic_source": None if tr is None else f"ncu dram__bytes_read+write per launch, captured at commit {tr[1]} "
                                                              "(profiles/traffic.csv); not re-measured by this run"}

        rd, rf = kroof("k_density", "a6-a9", fl_d, tk), kroof("k_force", "a10-a11", fl_f, tf)
        dom, other = (rf, rd) if tf >= tk else (rd, rf)
        roof = {"bound": "alu", **dom, "peak": peak, "unit": "TFLOP/s",
                "peak_source": f"measured: packed fma.rn.f32x2 probe on this device in this run (bench_probe.cu); scalar FFMA "
                               f"probe {peak_scalar:.1f}; derived {sm_count} SMs x {FP32_LANES_PER_SM} FP32 lanes x 2 x "
                               f"{sm_max:.0f} MHz = {derived:.1f}",
                "peak_derived": derived, "other_gather_kernel": other,
                "index_build": {"bound": "hbm", "ms": ti, "achieved_GBps": 200.0 * n / (ti * 1e-3) * 1e-9,
                                "algorithmic_bytes": 200.0 * n, "peak_GBps": hbm_peak, "peak_source": hbm_src,
                                "frac": 200.0 * n / (ti * 1e-3) * 1e-9 / hbm_peak}}
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic", "config": workload_config(args, ps, active_np),
            "clocks": {k: clocks.get(k) for k in ("sm_mhz", "sm_max_mhz", "reasons", "samples", "power_w_max")},
            "e2e": e2e, "gpu_launches": int(launches), "roofline": roof,
            "phases_ms": {"index": ti, "density_kernel": tk, "force_prep": tp, "force_kernel": tf},
            "improved_sph_extension_ms": ext_ms, "kdk_driver": kdk, "refresh_step": refresh_step,
            "pairs": {"density_evals_per_particle": st["dens_evals"] / n_active,
                      "density_true_pairs": st["dens_pairs"], "density_candidates": st["dens_candidates"],
                      "force_true_pairs": st["force_pairs"], "force_candidates": st["force_candidates"],
                      "pair_interactions_per_s": (st["dens_pairs"] + st["force_pairs"]) * world / (ms / args.steps * 1e-3),
                      "unconverged": per[-1]["unconv"],
                      "density_eval_histogram": {str(k): int(v) for k, v in enumerate(eval_hist) if v},
                      "updates_per_s_without_index": world * n_active / ((ms / args.steps - ti) * 1e-3)},
        }
        if world == 1 and not args.no_cpu_baseline:
            sample = args.cpu_sample or default_sample(ps)
            dt, nu, thr = oracle_sample_run(ps, active_np, sample, 4242)
            line["cpu_baseline"] = {"value": nu / dt, "unit": UNIT, "cores": thr, "kind": "oracle",
                                    "sample": f"{nu} seeded random active particles of the workload, density h-iteration + "
                                              f"hydro force, {dt:.1f} s"}
        print(json.dumps(line), flush=True)
    sph.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
