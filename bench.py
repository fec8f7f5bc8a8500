#!/usr/bin/env python
"""bench.py -- finite-source magnifications/s of the twk hot path (Measurement).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl twk|reference] [--workload config3]

A "step" is one pass of the whole hot path (stage 0 -> 1 -> 2 -> 3 of twk_magnify, all SURVEY 8(a) rows) over one batch
of synthetic input.  Headline workload: BASELINE config 3 = 4,096 seeded lens models x 1,000 epochs = 4,096,000 source
positions at relative tolerance 1e-4.  `value` = magnifications/s with inputs resident in HBM; `e2e` = the same through
twk_magnify_host with pinned HOST buffers (H2D + D2H inside the timed region).  Rank 0 prints ONE JSON line.  For N > 1
every rank runs its own batch (different seed): independent problems, no collective -> "weak" scaling.
--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.

Roofline inputs are not constants of this file: the executed FP64 instructions (DFMA / DMUL / DADD) and the DRAM bytes of
every kernel launch come from profiles/r02_counts.json, which `--parse-ncu` writes from an ncu pass over
`bench.py --profile-pass` (one step of every workload below) and which carries the hash of the CUDA sources it was
measured on.  When that hash is not the hash compiled into the loaded library (twk_version()), the counts are stale and
`roofline.achieved` is withheld (null) instead of being wrong.

Other modes (not part of the driver's contract):
  --profile-pass         one untimed step of every workload (what the ncu counting pass runs)
  --parse-ncu FILE.csv   turn the ncu --csv log of that pass into profiles/r02_counts.json
  --scaling              time twk_magnify against the number of sources (the paper's Fig.8 question) and
                         write profiles/r02_scaling.csv
"""
from __future__ import annotations

import argparse
import csv
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
FP64_LANES_PER_SM = 64          # FP64 FMA lanes per SM (derivation of the ALU peak)
COUNTS = os.path.join(ROOT, "profiles", "r02_counts.json")
# the workloads of the bench: the headline first, then the ones reported under "other_configs"
OTHER = ["config2", "config4", "config5", "fig5_resonant"]
NCU_METRICS = ("gpu__time_duration.sum,smsp__sass_thread_inst_executed_op_dfma_pred_on.sum,"
               "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum,smsp__sass_thread_inst_executed_op_dadd_pred_on.sum,"
               "dram__bytes_read.sum,dram__bytes_write.sum,sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active,"
               "smsp__issue_active.avg.pct_of_peak_sustained_active")
# launch order inside one twk_magnify, and the stage each launch is counted under (stage 1.5, the first refinement iteration in
# shared memory, belongs to the refinement of stage 2: the library's stage timer brackets the two together)
STAGES = ("seeds_kernel", "stage1_kernel", "refine1_kernel", "adaptive_kernel", "adaptive_kernel")
STAGE_KEY = (0, 1, 2, 2, 3)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="twk", choices=["twk", "reference"])
    ap.add_argument("--workload", default="config3")
    ap.add_argument("--cpu-sample", type=int, default=0, help="sources in the cpu_baseline sample (0 = auto)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true")
    ap.add_argument("--profile-pass", action="store_true")
    ap.add_argument("--pass-workloads", default=None, help="comma list restricting --profile-pass (default: all)")
    ap.add_argument("--parse-ncu", default=None)
    ap.add_argument("--scaling", action="store_true")
    return ap.parse_args()


def make_workload(name, rank=0, **size):
    """The batch of rank `rank`: every rank draws its own seeded batch (independent problems, no collective on the
    data path -- P:392 "no communication between devices")."""
    import workloads as W
    if name == "config3":
        return W.config3(seed=250103322 + rank, **size)
    if name == "config5":
        return W.config5(seed=250103323 + rank)
    if name.startswith("fig5_"):
        return W.fig5_map(name[5:])
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
    """The oracle as it stands (paper-style sampler, double) on a bounded seeded sample of the workload: all host cores,
    and one core on a tenth of that sample."""
    from oracle import api
    n_sample = min(n_sample, wl.n_sources)
    idx = np.sort(np.random.default_rng(12345).choice(wl.n_sources, n_sample, replace=False))
    sub = wl.subset(idx)
    cores = api.num_threads()
    t0 = time.perf_counter()
    r = api.magnify(sub, tol, mode=0, prec=0, nthreads=cores)
    dt = time.perf_counter() - t0
    n1 = max(200, n_sample // (10 * max(cores // 2, 1)))
    sub1 = wl.subset(idx[:: max(1, n_sample // n1)][:n1])
    t0 = time.perf_counter()
    api.magnify(sub1, tol, mode=0, prec=0, nthreads=1)
    dt1 = time.perf_counter() - t0
    return {"value": n_sample / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{n_sample} seeded-random sources of {wl.name} (of {wl.n_sources}), oracle paper-style sampler, "
                      f"double, tol {tol:g}, {dt:.1f} s wall, mean {float(r['nsamples'].mean()):.1f} samples/source",
            "seconds": dt,
            "one_core": {"value": sub1.n_sources / dt1, "unit": UNIT, "cores": 1, "seconds": dt1,
                         "sample": f"{sub1.n_sources} of those sources on one thread"},
            "per_core_of_all_cores": n_sample / dt / cores}


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


# ---------------------------------------------------------------------------------------------------------------------
# executed-instruction counts from ncu (profiles/r02_counts.json)
# ---------------------------------------------------------------------------------------------------------------------
def library_source_hash():
    import paper_2501_03322_b200 as P
    v = P.twk_version()
    return v.split("src:")[1].strip() if "src:" in v else None


def parse_ncu(path):
    """ncu --csv log of `bench.py --profile-pass` -> profiles/r02_counts.json.  The pass launches, for every workload in
    order, the kernels of one twk_magnify call (STAGES); rows are grouped by launch ID."""
    launches = {}
    with open(path, newline="") as f:
        rows = [r for r in csv.reader(f) if len(r) >= 15 and r[0].isdigit()]
    for r in rows:
        lid = int(r[0])
        d = launches.setdefault(lid, {"kernel": r[4]})
        try:
            d[r[12]] = float(r[14].replace(",", ""))
        except ValueError:
            pass
    order = [launches[k] for k in sorted(launches)]
    names = ["config3"] + OTHER
    per = len(STAGES)
    assert len(order) == per * len(names), (len(order), per * len(names))
    out = {"source_hash": library_source_hash(), "workloads": {},
           "command": "ncu --metrics " + NCU_METRICS + " --clock-control none --csv --log-file gpurun_out/r02_counts.csv "
                      "python bench.py --profile-pass ; python bench.py --parse-ncu gpurun_out/r02_counts.csv",
           "note": "per kernel launch of ONE twk_magnify call: executed thread-level FP64 instructions, flop = 2 dfma + "
                   "dmul + dadd, DRAM bytes, duration under ncu (serialised, cold cache), FP64-pipe and issue activity"}
    for w, name in enumerate(names):
        ks = {}
        for s, stage in enumerate(STAGES):
            L = order[w * per + s]
            assert stage in L["kernel"], (stage, L["kernel"])
            dfma = L["smsp__sass_thread_inst_executed_op_dfma_pred_on.sum"]
            dmul = L["smsp__sass_thread_inst_executed_op_dmul_pred_on.sum"]
            dadd = L["smsp__sass_thread_inst_executed_op_dadd_pred_on.sum"]
            one = {"kernel": stage, "dfma": dfma, "dmul": dmul, "dadd": dadd, "flop": 2 * dfma + dmul + dadd,
                   "dram_bytes": L["dram__bytes_read.sum"] + L["dram__bytes_write.sum"],
                   "ncu_ms": L["gpu__time_duration.sum"] * 1e-6,
                   "fp64_pipe_pct": L["sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active"],
                   "issue_active_pct": L["smsp__issue_active.avg.pct_of_peak_sustained_active"]}
            key = f"stage{STAGE_KEY[s]}"
            if key not in ks:
                ks[key] = one
            else:   # two launches under one stage: counts and times add, activities are time-weighted
                o = ks[key]
                tt = o["ncu_ms"] + one["ncu_ms"]
                for a in ("fp64_pipe_pct", "issue_active_pct"):
                    o[a] = (o[a] * o["ncu_ms"] + one[a] * one["ncu_ms"]) / tt if tt > 0 else 0.0
                for a in ("dfma", "dmul", "dadd", "flop", "dram_bytes", "ncu_ms"):
                    o[a] += one[a]
                o["kernel"] = o["kernel"] + " + " + stage
        out["workloads"][name] = ks
    os.makedirs(os.path.dirname(COUNTS), exist_ok=True)
    with open(COUNTS, "w") as f:
        json.dump(out, f, indent=1)
    print("wrote", COUNTS, "source hash", out["source_hash"])


def load_counts():
    try:
        c = json.load(open(COUNTS))
    except Exception:
        return None, "profiles/r02_counts.json missing"
    h = library_source_hash()
    if not h or c.get("source_hash") != h:
        return None, f"profiles/r02_counts.json was measured on sources {c.get('source_hash')}, the library is {h}: stale"
    return c, None


# ---------------------------------------------------------------------------------------------------------------------
def time_workload(P, torch, wl, dev, steps, warmup, barrier, want_e2e=False):
    """Device-resident timing of `steps` twk_magnify calls on `wl` (after `warmup`), then the per-stage durations from
    the library's own CUDA events in a separate pass (no synchronisation inside the timed loop)."""
    n = wl.n_sources
    ctx = P.Context(n)
    d = ctx.upload(wl, dev)
    out = dict(out_mu=torch.empty(n, dtype=torch.float64, device=dev), out_err=torch.empty(n, dtype=torch.float64, device=dev),
               out_nsamples=torch.empty(n, dtype=torch.int32, device=dev), out_status=torch.empty(n, dtype=torch.int32, device=dev))

    def step():
        ctx.twk_magnify(d["s"], d["q"], d["rho"], d["zeta"], d["model_id"], wl.rel_tol, **out)

    for _ in range(max(warmup, 3)):
        step()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        step()
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    ctx.twk_enable_stage_timing(True)
    stage = []
    for _ in range(steps):
        step()
        stage.append(ctx.twk_last_stage_ms())
    ctx.twk_enable_stage_timing(False)
    stats = ctx.twk_last_stats()
    r = {"ms": ms, "stage_ms": {k: float(np.mean([x[k] for x in stage])) for k in ("stage0", "stage1", "stage2", "stage3")},
         "n_stage2": stats["n_stage2"], "n_stage3": stats["n_stage3"], "launches": stats["n_launches"],
         "total_points": int(out["out_nsamples"].to(torch.int64).sum().item()),
         "converged": int((out["out_status"] & 1).ne(0).sum().item()), "ctx": ctx, "d": d, "out": out}
    return r


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    if args.parse_ncu:
        parse_ncu(args.parse_ncu)
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

    if args.profile_pass:                   # what the ncu counting pass runs: one call per workload, nothing else
        for name in (args.pass_workloads.split(",") if args.pass_workloads else ["config3"] + OTHER):
            wl = make_workload(name)
            ctx = P.Context(wl.n_sources)
            d = ctx.upload(wl, dev)
            ctx.twk_magnify(d["s"], d["q"], d["rho"], d["zeta"], d["model_id"], wl.rel_tol)
            torch.cuda.synchronize()
            ctx.close()
        return
    if args.scaling:
        run_scaling(P, torch, dev)
        return

    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    wl = make_workload(args.workload, rank)
    n = wl.n_sources
    sampler = ClockSampler(local) if rank == 0 else None
    barrier()
    R = time_workload(P, torch, wl, dev, args.steps, args.warmup, barrier)
    clocks = sampler.stop() if sampler else None
    ctx, d, out = R["ctx"], R["d"], R["out"]
    ms = R["ms"]

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
    ctx.close()
    # ---- for information: the same batch with the hidden-crossing guard (reading L-4, an extension of Eq.(17)) ----
    ctx_hg = P.Context(n, hidden_crossing_guard=1)
    out_hg = {k: torch.empty_like(v) for k, v in out.items()}
    for _ in range(2):
        ctx_hg.twk_magnify(d["s"], d["q"], d["rho"], d["zeta"], d["model_id"], wl.rel_tol, **out_hg)
    barrier()
    h0, h1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    h0.record()
    for _ in range(args.steps):
        ctx_hg.twk_magnify(d["s"], d["q"], d["rho"], d["zeta"], d["model_id"], wl.rel_tol, **out_hg)
    h1.record()
    barrier()
    ms_hg = h0.elapsed_time(h1)
    hg_dev = ((out_hg["out_mu"] / out["out_mu"]) - 1).abs()
    hg_changed = int((hg_dev > wl.rel_tol).sum().item())
    hg_maxdev = float(hg_dev.max().item())
    ctx_hg.close()

    ms, ms_e2e, ms_ps, ms_hg = max_over_ranks([ms, ms_e2e, ms_ps, ms_hg], dev, world)

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
        counts, stale = load_counts()

        def fracs(name, stage_ms):
            """achieved TFLOP/s and fraction of peak per stage, from the ncu counts of this workload and the live times"""
            if counts is None or name not in counts["workloads"]:
                return None
            o = {}
            for k, c in counts["workloads"][name].items():
                t = stage_ms.get(k, 0.0)
                if t > 0 and c["flop"] > 0:
                    a = c["flop"] / (t * 1e-3) / 1e12
                    inst = c["dfma"] + c["dmul"] + c["dadd"]
                    o[k] = {"achieved_tflops": a, "frac": a / peak_tf, "flop": c["flop"], "dram_bytes": c["dram_bytes"],
                            "fp64_pipe_pct_ncu": c["fp64_pipe_pct"], "issue_active_pct_ncu": c["issue_active_pct"],
                            # what `frac` would read with the FP64 pipe busy every cycle, given this kernel's share of
                            # DFMA (2 flop) among its FP64 instructions
                            "mix_limit": c["flop"] / (2.0 * inst) if inst > 0 else None}
            return o

        sm = R["stage_ms"]
        fr = fracs(wl.name, sm) if world == 1 or True else None
        s1 = sm["stage1"]
        dom = (fr or {}).get("stage1")
        step_flop = sum(v["flop"] for v in fr.values()) if fr else None
        line = {
            "metric": METRIC, "value": world * n * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl.name, "sources_per_step_per_gpu": n, "rel_tol": wl.rel_tol, "n_models": wl.n_models,
                       "seed": wl.meta.get("seed"), "parallelism": f"independent batches x{world}, no collective",
                       "l2": "inputs+outputs per step (~180 MB) and the per-step workspace traffic (seed blocks 1 GB, "
                             "hand-over arena 4 GB) exceed the 126 MB L2; no flush needed",
                       "mean_samples_per_source": R["total_points"] / n, "converged_fraction": R["converged"] / n,
                       "sources_to_stage2": R["n_stage2"], "sources_to_stage3": R["n_stage3"]},
            "e2e": {"value": world * n * args.steps / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "ms_per_step": ms_e2e / args.steps},
            "with_point_source_test": {"value": world * n * args.steps / (ms_ps * 1e-3), "unit": UNIT,
                                       "ms_per_step": ms_ps / args.steps, "accepted_fraction": ps_fraction,
                                       "max_rel_dev_from_contour": ps_maxdev,
                                       "note": "option point_source_test=1 (SURVEY N1, P:122): sources passing the "
                                               "quadrupole and ghost-image tests skip the contour; NOT the headline"},
            "with_hidden_crossing_guard": {"value": world * n * args.steps / (ms_hg * 1e-3), "unit": UNIT,
                                           "ms_per_step": ms_hg / args.steps, "sources_changed_beyond_tol": hg_changed,
                                           "max_rel_change": hg_maxdev,
                                           "note": "option hidden_crossing_guard=1 (DESIGN.md reading L-4: an extension of "
                                                   "Eq.(17) that closes the hidden double crossings the paper's estimate "
                                                   "cannot see; no stage 1.5 with it); NOT the headline"},
            "gpu_launches": R["launches"] * args.steps,
            "clocks": clocks,
            "roofline": {"bound": "alu", "kernel": "stage1_kernel (64 seeded point solves + 64 intervals per source)",
                         "achieved": dom["achieved_tflops"] if dom else None, "peak": peak_tf, "unit": "TFLOP/s",
                         "frac": dom["frac"] if dom else None,
                         "traffic": dom["dram_bytes"] if dom else None,
                         "counts": "profiles/r02_counts.json (ncu, executed DFMA/DMUL/DADD per launch, keyed by the source "
                                   "hash in twk_version())" if dom else stale,
                         "traffic_note": "DRAM bytes of one stage-1 launch (ncu); algorithmic bytes are 45 B/source = "
                                         "0.18 GB, the rest is the seed blocks read (1 GB) and the hand-over arena written",
                         "peak_source": f"derived: {props.multi_processor_count} SMs x {FP64_LANES_PER_SM} FP64 FMA lanes x 2 x "
                                        f"{sm_max_mhz:.0f} MHz (MEASURED_PEAKS.json has no FP64 figure)",
                         "peak_probe_tflops": probe_tf, "frac_of_probe": (dom["achieved_tflops"] / probe_tf) if dom else None,
                         "mix_limit": dom["mix_limit"] if dom else None,
                         "fp64_pipe_active_pct_ncu": dom["fp64_pipe_pct_ncu"] if dom else None,
                         "flop_per_point": (dom["flop"] / (64.0 * n)) if dom else None, "points_per_launch": 64 * n,
                         "kernel_ms": sm, "stage1_share_of_step": s1 / (ms / args.steps),
                         "per_stage": fr,
                         "whole_step_frac": (step_flop / (ms / args.steps * 1e-3) / 1e12 / peak_tf) if step_flop else None,
                         "point_solves_per_s": R["total_points"] * args.steps / (ms * 1e-3)},
        }
        if world == 1 and not args.no_other_configs:
            other = {}
            for name in OTHER:
                w2 = make_workload(name)
                r2 = time_workload(P, torch, w2, dev, max(args.steps, 5), 3, barrier)
                r2["ctx"].close()
                f2 = fracs(name, r2["stage_ms"])
                other[name] = {"value": w2.n_sources * max(args.steps, 5) / (r2["ms"] * 1e-3), "unit": UNIT,
                               "sources": w2.n_sources, "rel_tol": w2.rel_tol, "ms_per_step": r2["ms"] / max(args.steps, 5),
                               "kernel_ms": r2["stage_ms"], "sources_to_stage2": r2["n_stage2"],
                               "sources_to_stage3": r2["n_stage3"], "mean_samples_per_source": r2["total_points"] / w2.n_sources,
                               "converged_fraction": r2["converged"] / w2.n_sources,
                               "stage2_frac": (f2 or {}).get("stage2", {}).get("frac") if f2 else None,
                               "per_stage": f2}
            line["other_configs"] = other
        if world == 1 and not args.no_cpu_baseline:
            from oracle import api as _api
            ns = args.cpu_sample or min(n, 15000 * _api.num_threads())
            line["cpu_baseline"] = cpu_baseline(wl, ns, wl.rel_tol)
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_scaling(P, torch, dev):
    """Time of one twk_magnify call against the number of sources N_source (Fig.8): evenly spaced subsets of
    config 3, device-resident, best of 5 after 2 warm-up calls.  Writes profiles/r02_scaling.csv."""
    full = make_workload("config3")
    sizes = [1, 8, 64, 148, 296, 592, 888, 1184, 2368, 4736, 9472, 18944, 37888, 56832, 113664, 227328, 500000, 1000000, 2000000,
             4096000]
    rows = []
    for ns in sizes:
        idx = np.unique(np.linspace(0, full.n_sources - 1, ns).astype(np.int64))
        wl = full.subset(idx)
        ctx = P.Context(wl.n_sources)
        d = ctx.upload(wl, dev)
        best = 1e30
        for it in range(7):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            ctx.twk_magnify(d["s"], d["q"], d["rho"], d["zeta"], d["model_id"], wl.rel_tol)
            e1.record()
            torch.cuda.synchronize()
            if it >= 2:
                best = min(best, e0.elapsed_time(e1))
        st = ctx.twk_last_stats()
        ctx.close()
        rows.append((wl.n_sources, best, wl.n_sources / (best * 1e-3), st["n_stage2"], st["n_stage3"]))
        print(rows[-1], flush=True)
    path = os.path.join(ROOT, "profiles", "r02_scaling.csv")
    with open(path, "w") as f:
        f.write("# python bench.py --scaling   (one B200; evenly spaced subsets of config 3, tol 1e-4, best of 5 calls)\n")
        f.write("n_sources,ms_per_call,magnifications_per_s,sources_to_stage2,sources_to_stage3\n")
        for r in rows:
            f.write("%d,%.5f,%.4e,%d,%d\n" % r)
    print("wrote", path)


if __name__ == "__main__":
    main()
