#!/usr/bin/env python
"""bench.py -- fp64 projection-step throughput on synthetic fields shaped like the paper's runs.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workloads cfg4,cfg5]

A "step" is one pass of the whole hot path (splitting RHS -> Poisson solve -> correction) over one
batch of synthetic input.  Workloads (BASELINE.json `metric` names both):
  cfg4  512^3 triply periodic, box (2 pi)^3, drops at 5 % volume fraction, rho2/rho1 = 50   [primary line]
  cfg5  1024 x 1024 x 512 wall-bounded, box 4 x 4 x 1, two-layer, rho2/rho1 = 1000          [under "also"]
  cavity 512 x 512 x 256 closed box, walls in x, y, z (cosine expansions; NEXT-2)           [under "also"]
  cfg4ts the cfg4 fields through flutas_time_step (momentum prediction fused in; NEXT-5)    [under "also"]
  cfg4vof the cfg4 colour function through flutas_vof_step (one MTHINC step; NEXT-4)        [under "also"]
  cfg4slab8 the cfg4 step on a z-slab decomposition over 8 ranks, all on one device (NEXT-3) [under "also"]
  cfg4slabN / cfg5slabN: the same on N ranks (experiments)
N > 1 (torchrun): N independent replicas, one per GPU, no data-path collective ("replicas only"); with --slab instead ONE box
decomposed over the N GPUs (paper_2204_08834_b200/slab.py; exercised with N = 1 only in this repository's runs).
Prints ONE JSON line on rank 0.  --impl reference times the CPU oracle (tests' ground truth) on the same workload
(one or two steps of the full 512^3 box); it is a deliberately slow baseline, not a target.
"""
import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fp64 projection-step throughput"
UNIT = "Mpts/s"
WORKLOAD_DESC = {
    "cfg4": "cfg4: 512^3 triply periodic, box (2pi)^3, drops R=16 cells at 5% volume, rho2/rho1=50, dt=1e-3",
    "cfg5": "cfg5: 1024x1024x512 wall-bounded (Neumann p, Thomas in z), box 4x4x1, two-layer, rho2/rho1=1000, dt=1e-3",
    "cavity": "cavity: 512x512x256 closed box, walls (Neumann p, no-slip) in x, y and z: cosine expansions in x, y + Thomas in z "
              "(PAPER.md:287 shape, extruded; SURVEY sec. 8(f) NEXT-2), two-layer, rho2/rho1=5, dt=1e-3",
    "cfg4ts": "cfg4ts: the cfg4 fields (512^3 triply periodic, rho2/rho1=50) through flutas_time_step: momentum prediction "
              "(eq. 15: mu2/mu1=15, surface tension with a synthetic curvature field, gravity) fused with the projection "
              "(SURVEY sec. 8(f) NEXT-5)",
    "cfg4vof": "cfg4vof: the cfg4 colour function and velocity (512^3 triply periodic, 391 drops of radius 16 cells) through "
               "flutas_vof_step: one MTHINC step, beta = 2, CFL 0.3 (SURVEY sec. 8(f) NEXT-4)",
    "cfg4slab8": "cfg4slab8: the cfg4 step (512^3 triply periodic, rho2/rho1=50) on a z-slab decomposition over 8 ranks "
                 "(SURVEY sec. 8(f) NEXT-3: the two all-to-all transposes are the store stages of the y transform and of the z "
                 "stage, written straight into the peers' spectra); all 8 ranks driven phase by phase on ONE device",
    "cfg5slab8": "cfg5slab8: the cfg5 step (1024x1024x512 wall-bounded, rho2/rho1=1000) on a z-slab decomposition over 8 ranks, "
                 "all ranks on ONE device (SURVEY sec. 8(f) NEXT-3)",
    "cfg2": "cfg2: 128^3 triply periodic emulsion-shaped (small case)",
    "cfg3": "cfg3: 256x256x128 wall-bounded two-layer (small case)",
}


def make_workload(name, ratio=None):
    import workloads as wl          # top-level module: loads neither the CUDA library nor the oracle
    if name.startswith("cfg5slab"):
        return wl.config5()
    if name in ("cfg4", "cfg4ts", "cfg4vof") or name.startswith("cfg4slab"):
        return wl.config4(512, 50.0 if ratio is None else ratio)
    if name == "cfg5":
        return wl.config5()
    if name == "cavity":
        return wl.cavity(512, 512, 256, 5.0)
    if name == "cfg2":
        return wl.config2()
    if name == "cfg3":
        return wl.config3()
    raise ValueError(name)


def load_peak():
    """(HBM GB/s, label): the driver-measured copy bandwidth, else the profiling guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def load_ncu_traffic():
    """per-launch DRAM bytes from the committed ncu capture (profiles/ncu_traffic.json), if present"""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.json")) as f:
            return json.load(f)
    except Exception:
        return {}


class ClockSampler(threading.Thread):
    """samples SM clock and throttle reasons through NVML while the timed region runs"""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.mask, self.max_mhz, self.stop_flag = index, [], 0, None, False
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            pass

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        getr = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or nv.nvmlDeviceGetCurrentClocksThrottleReasons
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                self.mask |= int(getr(self.h))
            except Exception:
                pass
            time.sleep(0.004)

    def result(self):
        self.stop_flag = True
        if self.is_alive():
            self.join(timeout=2)
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.max_mhz, "samples": len(self.samples),
                "reasons": sorted(v for k, v in self.REASONS.items() if self.mask & k)}


def visible_gpu_index(local_rank):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


# ------------------------------------------------------------------------------------- our arm
def bench_workload(name, args, rank, local_rank, world, peak_gbs, peak_label, with_e2e, traffic, with_cpu_baseline=False):
    import torch
    import paper_2204_08834_b200 as fl
    from paper_2204_08834_b200 import replicas

    if "slab" in name:      # cfg4slab8 (default list), cfg4slab2, cfg5slab4, ...: the digits are the number of ranks
        return bench_slab(name, args, local_rank, peak_gbs, peak_label, n_ranks=int(name.split("slab")[1]))
    ratio = replicas.replica_density_ratio(rank) if (name == "cfg4" and world > 1) else None
    t0 = time.time()
    W = make_workload(name, ratio)
    gen_s = time.time() - t0
    plan = fl.Plan(W.nx, W.ny, W.nz, *W.box, W.bc_z, W.rho1, W.rho2, bc_x=W.bc_x, bc_y=W.bc_y)
    # experiments only: plan tuning knobs.  A plan refuses options that do not apply to it (e.g. "thomas" on a periodic box);
    # which ones took effect goes into config.options, and run_ours() fails the run if an option was applied nowhere
    opts = {"applied": {}, "rejected": {}}
    for kv in (args.opt or []):
        k_, v_ = kv.split("=")
        try:
            plan.set_option(k_, int(v_))
            opts["applied"][k_] = int(v_)
        except fl.FlutasError as exc:
            opts["rejected"][k_] = str(exc)
            print("bench.py: --opt %s refused by the %s plan: %s" % (kv, name, exc), file=sys.stderr)
    host = list(W.fields())
    dev = [torch.from_numpy(a).cuda() for a in host]
    torch.cuda.synchronize()
    timestep = name.endswith("ts")
    vof = name.endswith("vof")
    if vof:
        # phi^n -> phi^(n+1) out of place on the same resident fields every step (speed depends on the interface area,
        # which the drops of cfg4 fix); dt from CFL 0.3 on the largest velocity component
        cfl_dt = 0.3 / max(float(dev[c].abs().max()) * n_ / l_ for c, n_, l_ in zip(range(3), (W.nx, W.ny, W.nz), W.box))
        phi_next = torch.empty_like(dev[3])

        def one_step():
            plan.vof_step(dev[3], dev[0], dev[1], dev[2], phi_next, 2.0, cfl_dt)
    elif timestep:
        # whole velocity / pressure update: seven more resident fields (curvature, M of two time levels); the velocity
        # stays bounded over the timed steps because every step ends with the projection
        gen = torch.Generator(device="cuda").manual_seed(5)
        kappa = torch.randn(dev[0].shape, dtype=torch.float64, device="cuda", generator=gen)
        kappa *= 0.1
        mbuf = [torch.zeros_like(dev[0]) for _ in range(6)]
        state = {"flip": 0}

        def one_step():
            # a real time loop: M and p ping-pong (p^(n+1) is written over p^(n-1), then the roles swap)
            f = state["flip"]
            a, b = (mbuf[:3], mbuf[3:]) if f == 0 else (mbuf[3:], mbuf[:3])
            pn, po = (dev[4], dev[5]) if f == 0 else (dev[5], dev[4])
            state["flip"] ^= 1
            plan.time_step(dev[0], dev[1], dev[2], dev[3], kappa, pn, po, po, a, b, 0.01, 0.15, 0.05, (0.0, 0.0, -1.0), 1e-4)
    else:
        def one_step():
            plan.projection_step(*dev, W.dt)

    for _ in range(args.warmup):
        one_step()
    torch.cuda.synchronize()
    # ---- the headline: K steps back to back, per-kernel event recording OFF, one event pair around them
    sampler = ClockSampler(visible_gpu_index(local_rank))
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    replicas.barrier()
    torch.cuda.synchronize()
    sampler.start()
    ev0.record()
    for _ in range(args.steps):
        one_step()
    ev1.record()
    torch.cuda.synchronize()
    replicas.barrier()
    clocks = sampler.result()
    ms_local = ev0.elapsed_time(ev1)
    # ---- a second, separately reported loop with the library's per-kernel events on (the roofline table)
    k_steps = max(3, min(args.steps, 10))
    plan.set_timing(True)
    kv0, kv1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    kv0.record()
    for _ in range(k_steps):
        one_step()
    kv1.record()
    torch.cuda.synchronize()
    kms, ksteps = plan.read_timing()
    plan.set_timing(False)
    instrumented_ms = kv0.elapsed_time(kv1) / k_steps
    if vof:
        band = float(((dev[3] > 1e-8) & (dev[3] < 1.0 - 1e-8)).double().mean().item())
        return vof_result(name, W, args, world, units_ms=replicas.aggregate_throughput(float(W.npts) * args.steps, ms_local),
                          clocks=clocks, peak_gbs=peak_gbs, peak_label=peak_label, gen_s=gen_s,
                          finite=bool(torch.isfinite(phi_next).all().item()),
                          drift=float((phi_next.sum() - dev[3].sum()).abs() / dev[3].sum()), plan=plan, band=band,
                          sm_count=torch.cuda.get_device_properties(0).multi_processor_count)
    finite = bool(torch.isfinite(dev[4]).all().item() and torch.isfinite(dev[5]).all().item() and torch.isfinite(dev[0]).all().item())
    units, ms = replicas.aggregate_throughput(float(W.npts) * args.steps, ms_local)

    names, kbytes = plan.kernel_names, plan.kernel_bytes
    if timestep:     # the first kernel is the fused prediction: reads u, v, w, phi, kappa, p, p_old, M_old (3); writes M (3), u', v', w', rhs
        names = ["momentum_rhs"] + names[1:]
        kbytes = [17 * 8.0 * W.npts] + kbytes[1:]
    kernels = []
    for n_, b_, t_ in zip(names, kbytes, kms):
        avg = t_ / max(ksteps, 1)
        kernels.append({"name": n_, "ms": round(avg, 4), "alg_bytes": b_, "gbs": round(b_ / (avg * 1e-3) / 1e9, 1) if avg > 0 else None,
                        "frac": round(b_ / (avg * 1e-3) / 1e9 / peak_gbs, 4) if avg > 0 else None})
    dom = max(kernels, key=lambda k: k["ms"])
    # DRAM bytes of the dominant kernel from the committed ncu capture -- only if that capture is of the kernel
    # that ran here (same device symbol); a stale capture gives null instead of a wrong number
    symbols = dict(zip(names, (["momentum_rhs_kernel"] + plan.kernel_symbols[1:]) if timestep else plan.kernel_symbols))
    tr = traffic.get(name, {}).get(dom["name"])
    if traffic.get("_symbols", {}).get(name, {}).get(dom["name"]) != symbols[dom["name"]]:
        tr = None
    roofline = {"bound": "hbm", "kernel": dom["name"], "achieved": dom["gbs"], "peak": peak_gbs, "unit": "GB/s",
                "frac": dom["frac"], "traffic": tr, "peak_source": peak_label,
                "alg_bytes_per_launch": dom["alg_bytes"], "kernel_ms": dom["ms"], "kernel_symbol": symbols[dom["name"]],
                "traffic_source": (traffic.get("_source") if tr is not None else None),
                "timed_in": "a separate loop of %d steps with per-kernel CUDA events on (%.4f ms/step)" % (k_steps, instrumented_ms)}
    step_ms = ms_local / args.steps
    model_bytes = sum(kbytes)
    step = {"ms": round(step_ms, 4), "model_bytes_per_pt": round(model_bytes / W.npts, 1), "min_bytes_per_pt": 80,
            "min_bytes_note": "80 B/pt = north_star's minimum for the projection step alone" if not timestep else
                              "the whole update reads 10 and writes 7 more fields than that minimum counts",
            "model_gbs": round(model_bytes / (step_ms * 1e-3) / 1e9, 1),
            "frac_of_peak_model_bytes": round(model_bytes / (step_ms * 1e-3) / 1e9 / peak_gbs, 4),
            "frac_of_peak_min_bytes": round(80.0 * W.npts / (step_ms * 1e-3) / 1e9 / peak_gbs, 4),
            "frac_of_8TBs_model_bytes": round(model_bytes / (step_ms * 1e-3) / 1e9 / 8000.0, 4)}

    out = {
        "metric": METRIC, "value": round(units / (ms * 1e-3) / 1e6, 1), "unit": UNIT, "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(ms / args.steps, 4),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD_DESC[name], "grid": [W.nx, W.ny, W.nz], "bc_z": "wall" if W.bc_z else "periodic",
                   "bc_xyz": ["periodic" if b == 0 else "wall" for b in W.bc],
                   "rho2_over_rho1": W.rho2 / W.rho1, "parallelism": f"replicas x{world} (no data-path collective)",
                   "l2": "inputs larger than L2 (6 fields of %.1f GiB each); steps run back to back in place; per-kernel event "
                         "recording off in the timed region" % (W.npts * 8 / 2**30),
                   "input_generation_s": round(gen_s, 1), "options": opts},
        "clocks": clocks, "gpu_launches": args.steps * len(names), "launches_per_step": len(names),
        "roofline": roofline, "step": step, "kernels": kernels, "finite": finite,
        "workspace_gib": round(plan.workspace_bytes / 2**30, 2),
    }

    if not args.no_compare_torch and not args.no_e2e and W.bc_z == 0 and world == 1 and with_e2e:
        fresh = [torch.from_numpy(a).cuda() for a in host]
        plan.projection_step(*fresh, W.dt)
        torch.cuda.synchronize()
        out["comparison"] = torch_comparison(W, [fresh[i] for i in (0, 1, 2, 4)])
        del fresh
        torch.cuda.empty_cache()

    if with_e2e and not timestep:
        # end to end through the host entry point of the C ABI: pinned host buffers, H2D of the six inputs
        # and D2H of u, v, w, p inside the timed region, every step
        e_steps = max(1, min(args.steps, args.e2e_steps))
        pinned = [torch.from_numpy(a).pin_memory() for a in host]
        plan.projection_step_host(*pinned, W.dt)            # warm-up (allocates the staging buffers)
        replicas.barrier()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(e_steps):
            plan.projection_step_host(*pinned, W.dt)
        e1.record()
        torch.cuda.synchronize()
        replicas.barrier()
        eu, ems = replicas.aggregate_throughput(float(W.npts) * e_steps, e0.elapsed_time(e1))
        out["e2e"] = {"value": round(eu / (ems * 1e-3) / 1e6, 1), "unit": UNIT, "h2d_bytes_per_step": 6 * W.npts * 8,
                      "d2h_bytes_per_step": 4 * W.npts * 8, "steps": e_steps, "ms_per_step": round(ems / e_steps, 2),
                      "api": "flutas_projection_step_host (pinned host buffers)"}
        del pinned
    plan.destroy()
    del dev
    torch.cuda.empty_cache()
    if rank == 0 and world == 1 and with_cpu_baseline:
        out["cpu_baseline"] = oracle_full(W)
    return out


def bench_slab(name, args, local_rank, peak_gbs, peak_label, n_ranks=8):
    """NEXT-3 on one device: every rank of the decomposition is a plan of its own with its own buffers; the ranks are
    driven phase by phase on one stream (their kernels never wait for one another), so the time of a step is the SUM of
    the ranks' work -- what one GPU of an n_ranks-GPU node would do is 1 / n_ranks of it, plus the synchronisation and
    the NVLink time of the bytes reported here, which this box cannot measure."""
    import torch
    import workloads as wl
    from paper_2204_08834_b200 import slab
    t0 = time.time()
    W = make_workload(name)
    gen_s = time.time() - t0
    periodic = W.bc_z == 0
    grp = slab.SlabGroup(W.nx, W.ny, W.nz, *W.box, W.bc_z, W.rho1, W.rho2, n_ranks)
    parts = [wl.slab_split(a, n_ranks, periodic) for a in W.fields()]
    dev = [[torch.from_numpy(parts[f][r]).cuda() for f in range(6)] for r in range(n_ranks)]
    del parts
    if not periodic:        # planes beyond a wall are never read; keep them finite for the checks below
        for r in (0, n_ranks - 1):
            for t in dev[r]:
                torch.nan_to_num_(t, nan=0.0)
    torch.cuda.synchronize()

    def one_step(events=None):
        grp.exchange_halos(dev, periodic)       # the step's own velocity is fed back in: plane 0 of w (and phi's halos) from the neighbours
        for phase in range(3):
            for r, pl in enumerate(grp.plans):
                u, v, w, phi, p, po = dev[r]
                pl.step_phase(phase, u, v, w, phi, p, po, p, W.dt, 1.0)
            if events is not None:
                events[phase].record()

    for _ in range(args.warmup):
        one_step()
    torch.cuda.synchronize()
    sampler = ClockSampler(visible_gpu_index(local_rank))
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.start()
    ev0.record()
    for _ in range(args.steps):
        one_step()
    ev1.record()
    torch.cuda.synchronize()
    clocks = sampler.result()
    ms = ev0.elapsed_time(ev1)
    # per phase, in a separate short loop
    k_steps, phase_ms = 3, [0.0, 0.0, 0.0]
    for _ in range(k_steps):
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        evs[0].record()
        one_step(evs[1:])
        torch.cuda.synchronize()
        for i in range(3):
            phase_ms[i] += evs[i].elapsed_time(evs[i + 1]) / k_steps
    finite = all(bool(torch.isfinite(dev[r][f][1:-1]).all().item()) for r in range(n_ranks) for f in (0, 4))
    step_ms = ms / args.steps
    nxh, nzl, rpp = W.nx // 2 + 1, W.nz // n_ranks, W.ny // n_ranks
    # bytes a rank sends to OTHER ranks per step: its share of the spectrum twice (forward rows, backward planes) + halo planes
    fwd = 16.0 * nxh * (W.ny - rpp) * nzl
    bwd = 16.0 * nxh * rpp * (W.nz - nzl) + 16.0 * nxh * rpp * 2
    # algorithmic bytes of all ranks: the one-GPU model (216 / 218 B per point) with nzl + 2 instead of nzl planes in the
    # inverse x, y transforms (the halo planes of p^(n+1))
    model = (216.0 if periodic else 218.0) * W.npts + 2 * n_ranks * (16.0 * 2 + 8.0 + 16.0) * W.nx * W.ny
    for pl in grp.plans:
        pl.destroy()
    return {"metric": METRIC + " (z-slab decomposition, all ranks on one device)", "value": round(W.npts * args.steps / (ms * 1e-3) / 1e6, 1),
            "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(step_ms, 4),
            "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD_DESC.get(name, WORKLOAD_DESC[name.split("slab")[0] + "slab8"]), "grid": [W.nx, W.ny, W.nz],
                       "n_ranks": n_ranks, "planes_per_rank": nzl,
                       "ky_rows_per_rank": rpp, "input_generation_s": round(gen_s, 1)},
            "clocks": clocks, "gpu_launches": args.steps * n_ranks * (7 if periodic else 8), "finite": finite,
            "phase_ms_all_ranks": [round(x, 4) for x in phase_ms],
            "per_rank_ms": round(step_ms / n_ranks, 4),
            "exchange_bytes_per_rank_per_step": {"forward": fwd, "backward": bwd,
                                                 "at_900_GBs_ms": round((fwd + bwd) / 900e9 * 1e3, 4)},
            "step": {"ms": round(step_ms, 4), "model_bytes_per_pt": round(model / W.npts, 1),
                     "model_gbs": round(model / (step_ms * 1e-3) / 1e9, 1),
                     "frac_of_peak_model_bytes": round(model / (step_ms * 1e-3) / 1e9 / peak_gbs, 4)},
            "note": "one device runs all ranks one after the other: no NVLink transfer and no barrier is in this number; every step "
                    "starts with the halo refresh of w and phi (SlabGroup.exchange_halos, device copies of 3 planes per rank)"}


def bench_slab_distributed(name, args, rank, local_rank, world):
    """--slab: ONE box decomposed over the N GPUs (strong scaling), one rank per GPU, exchange buffers in torch symmetric
    memory, an NCCL all-reduce of one element as the barrier between phases.  Exercised in this repository's runs with
    N = 1 only (they have one GPU); the kernels and the index maps are the ones the one-device tests check."""
    import torch
    import torch.distributed as dist
    import workloads as wl
    from paper_2204_08834_b200 import replicas, slab
    if not dist.is_initialized():          # a single process: a group of one rank (the symmetric-memory path needs a group)
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group("nccl", rank=0, world_size=1)
    W = make_workload(name)
    periodic = W.bc_z == 0
    sr = slab.SlabRank(W.nx, W.ny, W.nz, *W.box, W.bc_z, W.rho1, W.rho2)
    dev = [torch.from_numpy(wl.slab_split(a, world, periodic)[rank]).cuda() for a in W.fields()]
    for t in dev:
        torch.nan_to_num_(t, nan=0.0)
    for _ in range(args.warmup):
        sr.step(*dev, W.dt)
    sampler = ClockSampler(visible_gpu_index(local_rank))
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    replicas.barrier()
    torch.cuda.synchronize()
    sampler.start()
    ev0.record()
    for _ in range(args.steps):
        sr.exchange_halos(dev[2], dev[3])       # the loop feeds the corrected velocity back in (NCCL send / recv of 3 planes)
        sr.step(*dev, W.dt)
    ev1.record()
    torch.cuda.synchronize()
    replicas.barrier()
    clocks = sampler.result()
    _, ms = replicas.aggregate_throughput(0.0, ev0.elapsed_time(ev1))
    return {"metric": METRIC, "value": round(W.npts * args.steps / (ms * 1e-3) / 1e6, 1), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(ms / args.steps, 4), "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD_DESC[name], "grid": [W.nx, W.ny, W.nz],
                       "parallelism": f"z-slabs x{world}, transposes fused into the transforms' stores over peer memory"},
            "clocks": clocks, "gpu_launches": args.steps * (7 if periodic else 8),
            "finite": bool(torch.isfinite(dev[4][1:-1]).all().item()),
            "note": "status of this path: run in this repository with N = 1 only (one-GPU boxes). Cross-process mapping of the peers' "
                    "buffers, the all-reduce barrier and write visibility across devices have never run on 2+ GPUs; the index maps, "
                    "the kernels and the halo exchange are covered by one-device (SlabGroup) and gloo tests. The loop is a time loop "
                    "on its own output (halos of w and phi refreshed every step); only finiteness is checked here"}


def vof_result(name, W, args, world, units_ms, clocks, peak_gbs, peak_label, gen_s, finite, drift, plan, band, sm_count):
    """the JSON block of the volume-of-fluid workload.  Seven launches per step (3 x flux + update, the correction).  The
    flux kernels are bound by FP64 arithmetic in the cells that carry a reconstruction: algorithmic work
    = 775 fp64 instructions per such cell and sweep with the algorithm as built (27-point Youngs gradient 230; 8 exponentials
    224 and 1 logarithm 40; 3 divisions, a square root and a reciprocal square root 56; fast reciprocals 32; coefficients of
    the quartic 25; 3.5 Newton iterations of 40; the flux 28); peak = SMs x 64 fp64 lanes x the SM clock."""
    units, ms = units_ms
    step_ms = ms / args.steps
    model_bytes = 28 * 8.0 * W.npts
    ops = 775.0 * 3 * band * W.npts
    sm_ghz = (clocks.get("sm_mhz") or clocks.get("sm_max_mhz") or 1965.0) / 1e3
    peak_ops = sm_count * 64 * sm_ghz            # G fp64 operations (instructions x lanes) per second
    plan.destroy()
    return {"metric": "fp64 volume-of-fluid step throughput", "value": round(units / (ms * 1e-3) / 1e6, 1), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(step_ms, 4), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD_DESC[name], "grid": [W.nx, W.ny, W.nz], "input_generation_s": round(gen_s, 1),
                       "cells_with_a_reconstruction": round(band, 4)},
            "clocks": clocks, "gpu_launches": args.steps * 7, "launches_per_step": 7, "finite": finite,
            "volume_drift_one_step": drift,
            "step": {"ms": round(step_ms, 4), "model_bytes_per_pt": 224.0,
                     "model_gbs": round(model_bytes / (step_ms * 1e-3) / 1e9, 1),
                     "frac_of_peak_model_bytes": round(model_bytes / (step_ms * 1e-3) / 1e9 / peak_gbs, 4)},
            "roofline": {"bound": "alu", "kernel": "vof_flux_kernel (3 launches, ~96 % of the step)",
                         "achieved": round(ops / (step_ms * 1e-3) / 1e9, 1), "peak": round(peak_ops, 1), "unit": "G fp64 op/s",
                         "frac": round(ops / (step_ms * 1e-3) / 1e9 / peak_ops, 4), "traffic": None,
                         "peak_source": "derived: %d SMs x 64 fp64 lanes x %.3f GHz (DESIGN.md sec. 6)" % (sm_count, sm_ghz),
                         "alg_ops_per_launch": ops / 3}}


def torch_cufft_step(u, v, w, phi, p, po, box, rho1, rho2, dt):
    """COMPARISON ONLY (never on the product path, not the oracle): the same triply periodic projection step written
    the obvious way with library calls -- torch.roll stencils + torch.fft.rfftn / irfftn (cuFFT).  Returns u, v, w, p."""
    import math
    import torch
    nz, ny, nx = u.shape
    dx, dy, dz = box[0] / nx, box[1] / ny, box[2] / nz
    rho0 = min(rho1, rho2)
    rc = rho1 * phi + rho2 * (1.0 - phi)
    ph = 2.0 * p - po
    fx = (1.0 - rho0 / (0.5 * (rc + torch.roll(rc, -1, 2)))) * (torch.roll(ph, -1, 2) - ph) / dx
    fy = (1.0 - rho0 / (0.5 * (rc + torch.roll(rc, -1, 1)))) * (torch.roll(ph, -1, 1) - ph) / dy
    fz = (1.0 - rho0 / (0.5 * (rc + torch.roll(rc, -1, 0)))) * (torch.roll(ph, -1, 0) - ph) / dz
    del rc, ph
    up, vp, wp = u + (dt / rho0) * fx, v + (dt / rho0) * fy, w + (dt / rho0) * fz
    del fx, fy, fz
    rhs = (rho0 / dt) * ((up - torch.roll(up, 1, 2)) / dx + (vp - torch.roll(vp, 1, 1)) / dy + (wp - torch.roll(wp, 1, 0)) / dz)
    lam = lambda n, d, m: -2.0 * (1.0 - torch.cos(2.0 * math.pi * torch.arange(m, device=u.device, dtype=torch.float64) / n)) / (d * d)
    den = lam(nz, dz, nz)[:, None, None] + lam(ny, dy, ny)[None, :, None] + lam(nx, dx, nx // 2 + 1)[None, None, :]
    den[0, 0, 0] = 1.0
    spec = torch.fft.rfftn(rhs) / den
    spec[0, 0, 0] = 0.0
    del rhs, den
    pn = torch.fft.irfftn(spec, s=(nz, ny, nx))
    del spec
    c = dt / rho0
    return (up - c * (torch.roll(pn, -1, 2) - pn) / dx, vp - c * (torch.roll(pn, -1, 1) - pn) / dy,
            wp - c * (torch.roll(pn, -1, 0) - pn) / dz, pn)


def torch_comparison(W, ours, steps=5):
    """times torch_cufft_step on the same device-resident inputs and reports how far its result is from ours"""
    import torch
    d = [torch.from_numpy(a).cuda() for a in W.fields()]
    args = (*d, W.box, W.rho1, W.rho2, W.dt)
    ref = torch_cufft_step(*args)
    errs = {n: float((a - b).norm() / b.norm()) for n, a, b in zip("uvwp", ours, ref)}
    del ref
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        out = torch_cufft_step(*args)
        del out
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    # the transforms alone: rfftn + irfftn of one field (our five transform kernels do this plus the division)
    nz, ny, nx = d[0].shape
    e0.record()
    for _ in range(steps):
        sp = torch.fft.rfftn(d[0])
        back = torch.fft.irfftn(sp, s=(nz, ny, nx))
        del sp, back
    e1.record()
    torch.cuda.synchronize()
    ms_fft = e0.elapsed_time(e1) / steps
    return {"cufft_rfftn_irfftn_ms": round(ms_fft, 3), "kind": "COMPARISON ONLY: the same periodic step with torch.roll stencils + torch.fft.rfftn/irfftn (cuFFT), "
                    "inputs resident, out of place", "ms_per_step": round(ms, 3),
            "value": round(W.npts / (ms * 1e-3) / 1e6, 1), "unit": UNIT, "steps": steps,
            "rel_l2_ours_vs_it": {k: float("%.2e" % v) for k, v in errs.items()}}


def naive_dft_flops(W):
    """flop count of the oracle's six naive DFT sweeps (8 flop per term: complex multiply-add on separate re / im arrays;
    n^2 terms per line of length n) -- so that nobody mistakes the CPU baseline for an FFT"""
    nx, ny, nz = W.nx, W.ny, W.nz
    f = 2 * (8.0 * nx * nx * ny * nz + 8.0 * ny * ny * nx * nz)
    if W.bc_z == 0:
        f += 2 * 8.0 * nz * nz * nx * ny
    return f


def oracle_full(W, threads=0):
    """time the CPU oracle, as it stands, on ONE step of the benchmark's own workload (cfg4: the full 512^3 box)"""
    import oracle
    t0 = time.perf_counter()
    oracle.projection_step(*W.fields(), W.box, W.bc_z, W.rho1, W.rho2, W.dt, nthreads=threads)
    dt = time.perf_counter() - t0
    fl = naive_dft_flops(W)
    return {"value": round(W.npts / dt / 1e6, 3), "unit": UNIT, "cores": oracle.threads(threads), "kind": "oracle",
            "sample": "one step of the full workload (%d x %d x %d, all %d points): plain stencils + naive O(n^2) DFT per line"
                      % (W.nx, W.ny, W.nz, W.npts),
            "seconds": round(dt, 2), "naive_dft_flop": fl, "gflops": round(fl / dt / 1e9, 1)}


def run_ours(args):
    import torch
    from paper_2204_08834_b200 import replicas
    rank, local_rank, world = replicas.init_from_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    peak_gbs, peak_label = load_peak()
    traffic = load_ncu_traffic()
    names = [w for w in args.workloads.split(",") if w]
    if world > 1:       # all-ranks-on-one-device workloads are a one-GPU measurement
        names = [n for n in names if "slab" not in n]
    if args.slab:
        out = bench_slab_distributed(names[0], args, rank, local_rank, world)
        if rank == 0:
            print(json.dumps(out), flush=True)
        replicas.barrier()
        return
    results = [bench_workload(n, args, rank, local_rank, world, peak_gbs, peak_label, with_e2e=(not args.no_e2e) and (i == 0 or args.e2e_all),
                              traffic=traffic, with_cpu_baseline=(i == 0 and not args.no_cpu_baseline)) for i, n in enumerate(names)]
    out = results[0]
    if len(results) > 1:
        out["also"] = results[1:]
        # the other workloads in short, inside a key of the base contract (BASELINE.json quotes the metric at 512^3 AND at
        # 1024 x 1024 x 512: cfg5 comes first); the full records stay under "also"
        out["config"]["second_workloads"] = [summary(n, r) for n, r in zip(names[1:], results[1:])]
    # an option that no plan of this run accepted is a typing mistake or a knob that no longer exists: the numbers above
    # would be those of the default configuration, so the run fails instead of printing them
    stale = [kv for kv in (args.opt or [])
             if not any(kv.split("=")[0] in r.get("config", {}).get("options", {}).get("applied", {}) for r in results)]
    if stale:
        raise SystemExit("bench.py: --opt %s was accepted by no plan of this run (unknown name or value); nothing reported" % ", ".join(stale))
    if rank == 0:
        print(json.dumps(out), flush=True)
    replicas.barrier()


def summary(name, r):
    """one workload's record in about 200 bytes"""
    roof, step, clk = r.get("roofline") or {}, r.get("step") or {}, r.get("clocks") or {}
    return {"workload": name, "grid": r.get("config", {}).get("grid"), "ms_per_step": r.get("ms_per_step"), "value": r.get("value"),
            "step_frac_of_peak": step.get("frac_of_peak_model_bytes"), "dominant_kernel": roof.get("kernel"),
            "dominant_frac": roof.get("frac"), "bound": roof.get("bound", "hbm"),
            "clocks": {"sm_mhz": clk.get("sm_mhz"), "reasons": clk.get("reasons")}}


# ------------------------------------------------------------------------------- reference arm
def run_reference(args):
    """the oracle, as it stands, on the host cores, on OUR arm's config (the full primary workload): each timed step is
    one oracle.projection_step of the whole box (about 40 s at 512^3 on 16 cores), so the step count is bounded to keep
    the run within a few minutes.  Imports nothing of the CUDA package."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    t_all = time.perf_counter()
    name = [w for w in args.workloads.split(",") if w][0]
    W = make_workload(name)
    n_warm, n_steps = (1 if args.warmup >= 1 and args.steps <= 1 else 0), max(1, min(args.steps, 2))
    for _ in range(n_warm):
        oracle_full(W)
    samples = [oracle_full(W) for _ in range(n_steps)]
    secs = sum(s_["seconds"] for s_ in samples)
    val = round(W.npts * len(samples) / secs / 1e6, 3)
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": len(samples),
           "warmup": n_warm, "ms_per_step": round(secs / len(samples) * 1e3, 1), "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": WORKLOAD_DESC[name], "grid": [W.nx, W.ny, W.nz], "bc_z": "wall" if W.bc_z else "periodic",
                   "bc_xyz": ["periodic" if b == 0 else "wall" for b in W.bc],
                      "rho2_over_rho1": W.rho2 / W.rho1, "sample": samples[0]["sample"],
                      "steps_note": "bounded to %d step(s) of the full box (requested %d)" % (len(samples), args.steps)},
           "cpu_baseline": dict(samples[0], value=val),
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0, "wall_s": round(time.perf_counter() - t_all, 1)}
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workloads", default="cfg4,cfg5,cavity,cfg4ts,cfg4vof,cfg4slab8")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--e2e-all", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs)")
    ap.add_argument("--no-compare-torch", action="store_true", help="skip the torch/cuFFT statement of the periodic step (comparison only)")
    ap.add_argument("--opt", action="append", help="plan tuning knob name=value (experiments)")
    ap.add_argument("--slab", action="store_true", help="decompose ONE box over the N GPUs (z slabs, SURVEY sec. 8(f) NEXT-3) instead "
                                                        "of running N replicas")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        if args.warmup < 3:
            args.warmup = 3
        run_ours(args)


if __name__ == "__main__":
    main()
