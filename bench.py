#!/usr/bin/env python
"""bench.py -- finite-source magnifications/s of the twk hot path on BASELINE config 3 (Measurement).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl twk|reference] [--workload config3]

A "step" is one pass of the whole hot path (stage 1 -> stage 2 -> stage 3 of twk_magnify, all SURVEY 8(a) rows) over
one batch of synthetic input: config 3 = 4,096 seeded lens models x 1,000 epochs = 4,096,000 source positions at
relative tolerance 1e-4.  `value` = magnifications/s with inputs resident in HBM; `e2e` = the same through
twk_magnify_host with pinned HOST buffers (H2D + D2H inside the timed region).  Rank 0 prints ONE JSON line.
For N > 1 every rank runs its own batch (different seed): independent problems, no collective -> "weak" scaling.
--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
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
sys.path.insert(0, ROOT)

METRIC = "finite-source magnifications/sec at rel. acc 1e-4"
UNIT = "magnifications/s"
# FP64 flop per boundary point (a1-a7: sample, coefficients, solve, lens quantities, ghost filter, its interval's
# link + area + error), the executed-instruction count of the stage-1 kernel on config 3 from the ncu capture in
# profiles/ (2*DFMA + DMUL + DADD thread instructions / boundary points) -- see DESIGN.md "Roofline".
FLOP_PER_POINT = 2155.0
# DRAM bytes of one stage-1 launch on config 3 (dram__bytes_read.sum + dram__bytes_write.sum of the same capture,
# profiles/r01b_ncu_full.csv): 0.10 GB read + 4.05 GB written, of which 4.0 GB is the hand-over arena
STAGE1_DRAM_BYTES_CONFIG3 = 4.147e9
FP64_LANES_PER_SM = 64          # FP64 FMA lanes per SM (derivation of the ALU peak)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="twk", choices=["twk", "reference"])
    ap.add_argument("--workload", default="config3")
    ap.add_argument("--cpu-sample", type=int, default=0, help="sources in the cpu_baseline sample (0 = auto)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def make_workload(name, rank, **size):
    """The batch of rank `rank`: every rank draws its own seeded batch (independent problems, no collective on the
    data path -- P:392 "no communication between devices")."""
    import workloads as W
    if name == "config3":
        return W.config3(seed=250103322 + rank, **size)
    if name == "config5":
        return W.config5(seed=250103323 + rank)
    return W.get(name)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md's clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                       "-i", str(index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1]))
                mx.append(float(c[2]))
                pw.append(float(c[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        os.unlink(self.f.name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


def cpu_baseline(wl, n_sample, tol):
    """The oracle as it stands (paper-style sampler, double) on a bounded seeded sample of the workload."""
    from oracle import api
    n_sample = min(n_sample, wl.n_sources)
    idx = np.sort(np.random.default_rng(12345).choice(wl.n_sources, n_sample, replace=False))
    sub = wl.subset(idx)
    cores = api.num_threads()
    t0 = time.perf_counter()
    r = api.magnify(sub, tol, mode=0, prec=0, nthreads=cores)
    dt = time.perf_counter() - t0
    return {"value": n_sample / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{n_sample} seeded-random sources of {wl.name} (of {wl.n_sources}), oracle paper-style sampler, "
                      f"double, tol {tol:g}, {dt:.1f} s wall, mean {float(r['nsamples'].mean()):.1f} samples/source",
            "seconds": dt}


def max_over_ranks(values, device, world):
    """Timing reduction of the N > 1 run: element-wise MAX over ranks (the only collective of the bench)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores; rank 0 alone works."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import api
    wl = make_workload(args.workload, 0)
    cores = api.num_threads()
    n_sample = args.cpu_sample or min(wl.n_sources, 3000 * cores)
    idx = np.sort(np.random.default_rng(12345).choice(wl.n_sources, n_sample, replace=False))
    sub = wl.subset(idx)
    for _ in range(min(args.warmup, 1)):
        api.magnify(sub.subset(np.arange(min(200, n_sample))), wl.rel_tol, mode=0)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        api.magnify(sub, wl.rel_tol, mode=0, prec=0, nthreads=cores)
    dt = time.perf_counter() - t0
    value = n_sample * args.steps / dt
    sample = f"{n_sample} seeded-random sources of {wl.name} per step (of {wl.n_sources}), oracle paper-style sampler, double"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "rel_tol": wl.rel_tol, "sources_per_step": n_sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    import torch
    import torch.distributed as dist

    import paper_2501_03322_b200 as P

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl twk needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    wl = make_workload(args.workload, rank)
    n = wl.n_sources
    ctx = P.Context(n)
    ctx.twk_enable_stage_timing(True)
    d = ctx.upload(wl, dev)
    out = dict(out_mu=torch.empty(n, dtype=torch.float64, device=dev), out_err=torch.empty(n, dtype=torch.float64, device=dev),
               out_nsamples=torch.empty(n, dtype=torch.int32, device=dev), out_status=torch.empty(n, dtype=torch.int32, device=dev))

    def step():
        ctx.twk_magnify(d["s"], d["q"], d["rho"], d["zeta"], d["model_id"], wl.rel_tol, **out)

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stage_ms = []
    barrier()
    e0.record()
    for _ in range(args.steps):
        step()
        stage_ms.append(ctx.twk_last_stage_ms())      # CUDA events recorded by the library on this stream
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop() if sampler else None
    stats = ctx.twk_last_stats()
    nsamp = out["out_nsamples"].to(torch.int64)
    total_points = int(nsamp.sum().item())
    status = out["out_status"]
    n_conv = int((status & 1).ne(0).sum().item())

    # ---- end to end: pinned host buffers through twk_magnify_host -----------------------------------------------
    hs = {k: torch.from_numpy(np.ascontiguousarray(v)).pin_memory() for k, v in
          dict(s=wl.s, q=wl.q, rho=wl.rho, zeta=wl.zeta, model_id=wl.model_id).items()}
    ho = dict(mu=torch.empty(n, dtype=torch.float64).pin_memory(), err=torch.empty(n, dtype=torch.float64).pin_memory(),
              nsamples=torch.empty(n, dtype=torch.int32).pin_memory(), status=torch.empty(n, dtype=torch.int32).pin_memory())
    h2d = sum(int(t.numel() * t.element_size()) for t in hs.values())
    d2h = sum(int(t.numel() * t.element_size()) for t in ho.values())

    def e2e_step():
        ctx.twk_magnify_host(hs["s"], hs["q"], hs["rho"], hs["zeta"], hs["model_id"], wl.rel_tol, out=ho)

    e2e_step()
    barrier()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record()
    for _ in range(args.steps):
        e2e_step()
    f1.record()
    barrier()
    ms_e2e = f0.elapsed_time(f1)
    assert torch.equal(ho["mu"], out["out_mu"].cpu()), "host-buffer path and device path disagree"

    # ---- for information: the same batch with the optional point-source adequacy tests in front ----------------
    ctx_ps = P.Context(n, point_source_test=1)
    out_ps = {k: torch.empty_like(v) for k, v in out.items()}
    for _ in range(2):
        ctx_ps.twk_magnify(d["s"], d["q"], d["rho"], d["zeta"], d["model_id"], wl.rel_tol, **out_ps)
    barrier()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record()
    for _ in range(args.steps):
        ctx_ps.twk_magnify(d["s"], d["q"], d["rho"], d["zeta"], d["model_id"], wl.rel_tol, **out_ps)
    p1.record()
    barrier()
    ms_ps = p0.elapsed_time(p1)
    ps_fraction = float((out_ps["out_status"] & 64).ne(0).double().mean().item())
    ps_maxdev = float(((out_ps["out_mu"] / out["out_mu"]) - 1).abs().max().item())
    ctx_ps.close()

    ms, ms_e2e, ms_ps = max_over_ranks([ms, ms_e2e, ms_ps], dev, world)

    if rank == 0:
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            pass
        props = torch.cuda.get_device_properties(local)
        sm_max_mhz = float(peaks.get("sm_max_mhz") or (clocks or {}).get("sm_max_mhz") or 1965.0)
        peak_tf = props.multi_processor_count * FP64_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
        probe_tf = P.twk_fp64_peak_probe(1 << 16)
        s1 = float(np.mean([x["stage1"] for x in stage_ms]))
        s2 = float(np.mean([x["stage2"] for x in stage_ms]))
        s3 = float(np.mean([x["stage3"] for x in stage_ms]))
        flop_launch = FLOP_PER_POINT * 64.0 * n                   # stage 1 solves 64 boundary points per source
        achieved = flop_launch / (s1 * 1e-3) / 1e12
        line = {
            "metric": METRIC, "value": world * n * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl.name, "sources_per_step_per_gpu": n, "rel_tol": wl.rel_tol, "n_models": wl.n_models,
                       "seed": wl.meta.get("seed"), "parallelism": f"independent batches x{world}, no collective",
                       "l2": "inputs+outputs per step (~180 MB) exceed the 126 MB L2; no flush needed",
                       "mean_samples_per_source": total_points / n, "converged_fraction": n_conv / n,
                       "sources_to_stage2": stats["n_stage2"], "sources_to_stage3": stats["n_stage3"]},
            "e2e": {"value": world * n * args.steps / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "ms_per_step": ms_e2e / args.steps},
            "with_point_source_test": {"value": world * n * args.steps / (ms_ps * 1e-3), "unit": UNIT,
                                       "ms_per_step": ms_ps / args.steps, "accepted_fraction": ps_fraction,
                                       "max_rel_dev_from_contour": ps_maxdev,
                                       "note": "option point_source_test=1 (SURVEY N1, P:122): sources passing the "
                                               "quadrupole and ghost-image tests skip the contour; NOT the headline"},
            "gpu_launches": stats["n_launches"] * args.steps,
            "clocks": clocks,
            "roofline": {"bound": "alu", "kernel": "stage1_kernel (64 point solves + 64 intervals per source)",
                         "achieved": achieved, "peak": peak_tf, "unit": "TFLOP/s", "frac": achieved / peak_tf,
                         "traffic": STAGE1_DRAM_BYTES_CONFIG3 if wl.name == "config3" else None,
                         "traffic_note": "DRAM bytes per stage-1 launch from profiles/r01b_ncu_full.csv; algorithmic "
                                         "bytes are 45 B/source = 0.18 GB, the rest is the hand-over arena to stage 2",
                         "peak_source": f"derived: {props.multi_processor_count} SMs x {FP64_LANES_PER_SM} FP64 FMA lanes x 2 x "
                                        f"{sm_max_mhz:.0f} MHz (MEASURED_PEAKS.json has no FP64 figure)",
                         "peak_probe_tflops": probe_tf, "frac_of_probe": achieved / probe_tf,
                         "flop_per_point": FLOP_PER_POINT, "points_per_launch": 64 * n,
                         "kernel_ms": {"stage1": s1, "stage2": s2, "stage3": s3},
                         "stage1_share_of_step": s1 / (ms / args.steps),
                         "point_solves_per_s": total_points * args.steps / (ms * 1e-3)},
        }
        if world == 1 and not args.no_cpu_baseline:
            from oracle import api as _api
            ns = args.cpu_sample or min(n, 15000 * _api.num_threads())
            line["cpu_baseline"] = cpu_baseline(wl, ns, wl.rel_tol)
        print(json.dumps(line))
    ctx.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
