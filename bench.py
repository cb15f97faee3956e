#!/usr/bin/env python
"""bench.py -- MLUPS of the fused LBM stream-and-collide step on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config c2] [--impl ours|reference]

A "step" is one pass of the whole hot path (rows a1-a8 of DESIGN.md; a9-a11 for c5) over the
whole lattice of the config, i.e. one LBM time step.  Default workload: configs[1] = c2, D3Q19
LBGK fp32 256^3 channel with Guo force -- the configuration the metric is quoted on.  Inputs are
seeded synthetic fields (paper_1311_2404_b200/workloads.py) standing in for the paper's duct flow.

The path does not shard (north_star: one GPU, no halo exchange): with --gpus N > 1 every rank runs
an independent replica ("replicas only") and `value` is the sum over ranks.

One JSON line on stdout (rank 0).  --impl reference times the CPU oracle instead.
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

import numpy as np  # noqa: E402

from paper_1311_2404_b200 import workloads as W  # noqa: E402

METRIC = "MLUPS on 1 B200 and achieved HBM GB/s as % of peak (D3Q19 LBGK fp32)"
UNIT = "MLUPS"
# ncu --set full DRAM bytes per step (dram__bytes_read.sum + dram__bytes_write.sum of the step kernel(s)) are
# read from the committed capture summary below, which also records the commit it was taken at.
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "r02_traffic.json")
NCU_DRAM_PEAK_GBS = 8183.8  # ncu's own DRAM peak on this part: 3996 MHz x 2 x 8192 bit / 8 (profiles/)


def ncu_traffic(key: str):
    """(bytes per step, source string) for a config key such as "c2" or "c3_f64"; (None, reason) if absent."""
    try:
        with open(TRAFFIC_FILE) as f:
            t = json.load(f)
        k = t["configs"][key]
        return float(k["dram_bytes_per_step"]), "profiles/r02_traffic.json (ncu --set full at commit %s, kernel %s)" % (k.get("commit", t["commit"]), k["kernel"])
    except Exception as e:  # missing file or key: say so instead of inventing a number
        return None, "no committed capture for %s (%s)" % (key, type(e).__name__)


def algorithmic_bytes_per_site(w) -> float:
    """SURVEY 8(d) / DESIGN.md: (1 - phi_s) * 2*Q*sizeof(real) + 1 mask byte, phi_s = fraction of SOLID sites (they
    move no populations; c3: 145.4 / 289.8); Shan-Chen two-pass floor 472 (fp32)."""
    s = 4 if w.precision == W.F32 else 8
    wet = 1.0 - float((w.mask == W.SOLID).mean())
    if w.model == W.SC2:
        return wet * 3 * (2 * w.Q * s) + 4 * s  # pass 1: read both stores, write psi; pass 2: read both + psi, write both
    return wet * 2 * w.Q * s + 1


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def make_workload(args):
    kw = {} if args.precision is None else {"precision": W.F32 if args.precision == "f32" else W.F64}
    w = W.CONFIGS[args.config](**kw)
    if getattr(args, "model", None) and w.model != W.SC2:
        w.model = {"bgk": W.BGK, "mrt": W.MRT, "reg": W.REG, "les": W.LES}[args.model]
        if w.model == W.MRT and w.rates is None:
            w.rates = W.mrt_rates_d3q19(w.tau[0]) if w.lattice == W.D3Q19 else W.mrt_rates_d2q9(w.tau[0])
        if w.model == W.LES:
            w.smagorinsky_cs = 0.1
        if w.model == W.REG and any(w.force):
            w.force_scheme = W.FORCE_EDM  # reading A23
    return w


def sample_workload(cfg: str):
    """Bounded sample of the config for the CPU oracle: same recipe, same nx*ny cross-section,
    a thin z-slab (the torus closes it), so one oracle step costs ~0.25 s per 2M sites."""
    full = W.CONFIGS[cfg]()
    if full.lattice == W.D2Q9:
        return full, "the full %dx%d lattice" % (full.nx, full.ny)
    nz = max(4, (1 << 21) // (full.nx * full.ny))
    w = W.CONFIGS[cfg](full.nx, full.ny, nz)
    return w, "%dx%dx%d z-slab of the %dx%dx%d workload, same seeded recipe" % (w.nx, w.ny, w.nz, full.nx, full.ny, full.nz)


def time_oracle(cfg: str, steps: int, warmup: int):
    from oracle import oracle
    w, what = sample_workload(cfg)
    ref = oracle.Oracle(**w.params())
    ref.set_geometry(w.mask)
    for s in range(w.ncomp):
        ref.init_equilibrium(w.rho[s], w.u[s], comp=s)
    ref.step(warmup)
    t0 = time.perf_counter()
    ref.step(steps)
    dt = time.perf_counter() - t0
    return dict(value=w.sites * steps / dt / 1e6, unit=UNIT, cores=oracle.num_threads(), kind="oracle",
                sample="%s, %d steps (%.1f s)" % (what, steps, dt)), dt, w


def config_dict(w, cfg, extra=None, store="ab"):
    d = {"workload": "%s: %s %s %s %dx%dx%d" % (cfg, "D2Q9" if w.lattice == W.D2Q9 else "D3Q19",
                                                 ["LBGK", "MRT", "Shan-Chen 2xLBGK", "regularized LBGK", "LBGK+Smagorinsky"][w.model],
                                                 "fp32" if w.precision == W.F32 else "fp64", w.nx, w.ny, w.nz),
         "tau": list(w.tau)[: w.ncomp], "force": list(w.force), "seed": w.seed,
         "solid_fraction": float(w.mask.mean()), "store": ("AA in place" if store == "aa" else "AB double buffer") + ", SoA real[Q][N]",
         "parallelism": "replicas only (path does not shard)"}
    d.update(extra or {})
    return d


def run_reference(args):
    """CPU oracle arm: rank 0 only; each step is one oracle step over the bounded sample."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    if int(os.environ.get("WORLD_SIZE", "1")) > 1 and os.environ.get("OMP_NUM_THREADS") == "1":
        # torchrun pins OMP_NUM_THREADS=1 for its workers; rank 0 alone runs the oracle, on all host cores as at N = 1
        os.environ["OMP_NUM_THREADS"] = str(os.cpu_count() or 1)
    steps = min(args.steps, 60)
    cb, dt, w = time_oracle(args.config, steps, min(args.warmup, 3))
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "warmup": min(args.warmup, 3), "ms_per_step": dt / steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": config_dict(w, args.config, {"sample": cb["sample"]}),
            "cpu_baseline": cb, "gpu_launches": 0,
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def max_over_ranks(value: float, world: int, device) -> float:
    """Slowest rank's time (the contract's max over ranks); identity for one rank."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_mlups(sites: int, steps: int, world: int, seconds: float) -> float:
    """Whole-job throughput of `world` independent replicas (replicas only)."""
    return sites * steps * world / seconds / 1e6


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "20"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        self.p.wait()
        self.f.seek(0)
        rows = [r.split(",") for r in self.f.read().strip().splitlines() if r.count(",") >= 6]
        self.f.close()
        os.unlink(self.f.name)
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm = sorted(float(r[0]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(r[3 + k].strip() == "Active" for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(rows[0][1]), "samples": len(rows),
                "power_w_max": max(float(r[2]) for r in rows), "reasons": reasons}


OTHER_CONFIGS = (("c1", None), ("c3", "f32"), ("c3", "f64"), ("c4", None), ("c5", None), ("ldc", None))


def config_key(cfg, w):
    return cfg + ("_f64" if cfg == "c3" and w.precision == W.F64 else "")


def time_steps(sim, K, repeats, barrier):
    """K steps between CUDA events on the context's stream, `repeats` times; milliseconds per repeat."""
    import torch
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps = []
    for _ in range(repeats):
        barrier()
        e0.record(sim.stream)
        sim.step(K)
        e1.record(sim.stream)
        barrier()
        reps.append(e0.elapsed_time(e1))
    return reps


def roofline_of(w, cfg, ms_per_step):
    peak, which = measured_peak()
    bps = algorithmic_bytes_per_site(w)
    achieved = bps * w.sites / (ms_per_step * 1e-3) / 1e9  # per-launch bytes / per-launch time
    traffic, src = ncu_traffic(config_key(cfg, w))
    kernel = "sc_fields_kernel + sc_step_kernel" if w.model == W.SC2 else "step_kernel"
    r = {"bound": "hbm", "kernel": kernel, "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
         "peak_source": which, "bytes_per_site": bps, "sites_per_launch": w.sites, "traffic": traffic, "traffic_source": src}
    if traffic:  # what the DRAM actually moved (ncu) over this run's time, against ncu's own DRAM peak
        r["dram_gbs"] = traffic / (ms_per_step * 1e-3) / 1e9
        r["frac_of_ncu_dram_peak"] = r["dram_gbs"] / NCU_DRAM_PEAK_GBS
        r["traffic_over_algorithmic"] = traffic / (bps * w.sites)
    return r


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1311_2404_b200 import binding

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    ndev = torch.cuda.device_count()
    if ndev == 0:
        raise RuntimeError("bench.py needs a CUDA device (the CUDA library is the only implementation)")
    dev_index = local % ndev  # one rank per GPU; ranks share a GPU only in the 1-GPU test of this code path
    torch.cuda.set_device(dev_index)
    dev = torch.device("cuda", dev_index)
    if world > 1:
        # NCCL for the barrier and the max-over-ranks reduction; LBM_BENCH_BACKEND=gloo lets the N > 1
        # code path be exercised on a box with fewer GPUs than ranks (NCCL refuses two ranks per GPU)
        backend = os.environ.get("LBM_BENCH_BACKEND", "nccl")
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=dev)
        else:
            dist.init_process_group(backend)
    binding.load()  # no fallback: raises if the CUDA library is missing

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    def prepare(w, store):
        sim = binding.from_workload(w, device=dev, store=binding.LBM_STORE_AA if store == "aa" else binding.LBM_STORE_AB)
        sim.set_geometry(w.mask)
        for s in range(w.ncomp):
            sim.init_equilibrium(w.rho[s], w.u[s], comp=s)
        return sim

    def warm_steps(w):  # small lattices replay 50-step CUDA graphs: capture them before timing
        return max(args.warmup, 3, 128 if w.sites <= (1 << 20) else 0)

    K = args.steps
    w = make_workload(args)
    Wm = warm_steps(w)
    sim = prepare(w, args.store)

    # ---- device-resident: K steps between CUDA events on the context's stream -------------------
    clocks = ClockSampler(dev_index)  # runs through warm-up, the timed steps and the end-to-end call
    sim.step(Wm)
    l0 = sim.counters()[1]
    barrier()
    reps = time_steps(sim, K, args.repeats, barrier)
    launches = (sim.counters()[1] - l0) // args.repeats
    ms = max_over_ranks(float(np.median(reps)), world, dev)
    ms_best = max_over_ranks(float(np.min(reps)), world, dev)
    rho, _ = sim.macro()
    assert bool(torch.isfinite(rho).all()), "state went non-finite during the timed steps"
    dispatch = sim.dispatch()

    # ---- end to end through lbm_run_host: pinned host inputs -> H2D -> init -> K steps -> D2H ------
    tdt = torch.float32 if w.precision == W.F32 else torch.float64
    h_mask = torch.from_numpy(w.mask).pin_memory()
    h_rho = [torch.from_numpy(r).to(tdt).pin_memory() for r in w.rho]
    h_u = [torch.from_numpy(u).to(tdt).pin_memory() for u in w.u]
    o_rho = torch.empty(sim.shape, dtype=tdt).pin_memory()
    o_u = torch.empty((sim.D,) + sim.shape, dtype=tdt).pin_memory()
    sim.run_host(h_mask, h_rho, h_u, Wm, o_rho, o_u)
    barrier()
    t0 = time.perf_counter()
    sim.run_host(h_mask, h_rho, h_u, K, o_rho, o_u)  # synchronises the stream before returning
    e2e_s = time.perf_counter() - t0
    barrier()
    e2e_s = max_over_ranks(e2e_s, world, dev)
    h2d = h_mask.numel() + sum(x.numel() * x.element_size() for x in h_rho + h_u)
    d2h = o_rho.numel() * o_rho.element_size() + o_u.numel() * o_u.element_size()
    assert bool(torch.isfinite(o_rho).all())
    clk = clocks.stop()
    sim.close()
    del sim, h_mask, h_rho, h_u, o_rho, o_u

    # ---- the other configs in the same process (rank 0, one GPU): same protocol, one line carries them all ----
    others = {}
    if rank == 0 and world == 1 and not args.no_other_configs and args.config == "c2" and args.store == "ab" and not args.model:
        for cfg, prec in OTHER_CONFIGS:
            kw = {} if prec is None else {"precision": W.F32 if prec == "f32" else W.F64}
            wo = W.CONFIGS[cfg](**kw)
            so = prepare(wo, "ab")
            so.step(warm_steps(wo))
            r = time_steps(so, K, args.repeats, barrier)
            assert bool(torch.isfinite(so.macro()[0]).all()), cfg
            med = float(np.median(r)) / K
            roof = roofline_of(wo, cfg, med)
            others[config_key(cfg, wo)] = {
                "workload": config_dict(wo, cfg)["workload"], "mlups": wo.sites / (med * 1e-3) / 1e6,
                "mlups_best": wo.sites * K / (min(r) * 1e-3) / 1e6, "ms_per_step": med, "repeats_ms": r,
                "dispatch": so.dispatch(), "bytes_per_site": roof["bytes_per_site"], "achieved_gbs": roof["achieved"],
                "frac": None if wo.sites <= (1 << 20) else roof["frac"],  # c1 is launch-bound, not HBM-bound
                "traffic": roof["traffic"], "frac_of_ncu_dram_peak": roof.get("frac_of_ncu_dram_peak")}
            so.close()
            del so, wo

    if rank == 0:
        cb = None
        if world == 1 and not args.no_cpu_baseline:
            cb, _, _ = time_oracle(args.config, args.cpu_steps, 1)
        line = {"metric": METRIC, "value": aggregate_mlups(w.sites, K, world, ms * 1e-3), "unit": UNIT,
                "n_gpus": world, "steps": K, "warmup": Wm, "ms_per_step": ms / K, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32" if w.precision == W.F32 else "f64",
                "data": "synthetic",
                "best": aggregate_mlups(w.sites, K, world, ms_best * 1e-3), "median": aggregate_mlups(w.sites, K, world, ms * 1e-3),
                "config": config_dict(w, args.config, {
                    "l2": "working set %.2f GB per step >> 126 MB L2 (no flush needed)" % (algorithmic_bytes_per_site(w) * w.sites / 1e9),
                    "timing": "value = median of %d repeats of K steps (best also given), CUDA events on the ctx stream" % args.repeats,
                    "repeats_ms": reps, "dispatch": dispatch}, store=args.store),
                "clocks": clk,
                "e2e": {"value": aggregate_mlups(w.sites, K, world, e2e_s), "unit": UNIT,
                        "h2d_bytes_per_step": h2d / K, "d2h_bytes_per_step": d2h / K,
                        "note": "one lbm_run_host call = H2D(mask, rho0, u0) + init + K steps + macro + D2H(rho, u); bytes amortised over K"},
                "gpu_launches": int(launches),
                "roofline": roofline_of(w, args.config, ms / K),
                "cpu_baseline": cb,
                "other_configs": others}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="c2", choices=sorted(W.CONFIGS))
    ap.add_argument("--repeats", type=int, default=3, help="repeats of the K timed steps; value = median, best also reported")
    ap.add_argument("--no-other-configs", action="store_true", help="skip timing c1, c3, c4, c5 and ldc after the headline")
    ap.add_argument("--cpu-steps", type=int, default=250, help="oracle steps on the bounded sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--precision", default=None, choices=["f32", "f64"], help="override the config's precision (c3 is quoted in both)")
    ap.add_argument("--model", default=None, choices=["bgk", "mrt", "reg", "les"],
                    help="override the collision operator of a single-component config (NEXT-4 variants)")
    ap.add_argument("--store", default="ab", choices=["ab", "aa"], help="AB double buffer (default) or in-place AA")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
