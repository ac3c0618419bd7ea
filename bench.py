#!/usr/bin/env python
"""bench.py — the adaptive GROUP BY hot path on B200, one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2|C3|C4|C5:<log2 ndv>:<dense|scattered>|C1|MK:<key cols>:<bits per col>]
                    [--force auto|direct|smem|global|partition] [--impl reference] [--sweep]

A step = one pass of the whole hot path (profile -> select -> init -> aggregate -> compact,
i.e. eiger.groupby with no statistics supplied) over one resident batch of synthetic rows.
`value` = rows/s with the inputs already in HBM; `e2e` = the same through
eiger_groupby_host with pinned HOST buffers (H2D + D2H inside the timed region).
N > 1 (torchrun): independent replicas, one per GPU, different seeds ("replicas only",
DESIGN.md "Multi-GPU"); value = all ranks' rows / max-over-ranks time.
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

METRIC = "groupby_rows_per_s"
UNIT = "rows/s"
VARIANTS = {"auto": 0, "direct": 1, "smem": 2, "global": 3, "partition": 4, "sort": 5}


def parse_args(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C2")
    ap.add_argument("--force", default="auto", choices=list(VARIANTS))
    ap.add_argument("--impl", default="eiger", choices=["eiger", "reference"])
    ap.add_argument("--scale", type=int, default=1, help="divide the row count (development only; prints scale in config)")
    ap.add_argument("--sweep", action="store_true", help="config-5 crossover sweep: every variant at every NDV point")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-curve", action="store_true", help="skip the ndv_curve key (the metric is rows/s vs NDV: C5 points, C3, C4)")
    ap.add_argument("--curve-forced", action="store_true", help="ndv_curve: also time the forced variants (statistics supplied) at every point")
    ap.add_argument("--no-cpu", action="store_true")
    return ap.parse_args(argv)


def build_workload(name: str, device, scale: int = 1, seed_offset: int = 0):
    import datagen
    parts = name.split(":")
    base = parts[0].upper()
    if base == "C1":
        return datagen.config1(device, n=1_000_000 // scale, seed=0 + seed_offset)
    if base == "C2":
        return datagen.config2(device, n=600_000_000 // scale, seed=2 + seed_offset,
                               skewed=len(parts) > 1 and parts[1] == "skewed")
    if base == "C3":
        return datagen.config3(device, n=200_000_000 // scale, seed=3 + seed_offset,
                               dense=len(parts) > 1 and parts[1] == "dense")
    if base == "C4":
        return datagen.config4(device, n=500_000_000 // scale, seed=4 + seed_offset, D=100_000_000 // scale)
    if base == "C5":
        lg = int(parts[1]) if len(parts) > 1 else 16
        n = (1 << 28) // scale
        return datagen.config5(device, n=n, seed=5 + seed_offset, ndv=min(1 << lg, n),
                               scattered=len(parts) > 2 and parts[2] == "scattered")
    if base == "MK":
        # MK[:<key columns>[:<bits per column>]]: multi-key group-by, 2^28 rows of nk int32 key columns
        # (PAPER.md:215-221 smart key fusion; the 4xI32 tables of)
        nk = int(parts[1]) if len(parts) > 1 else 4
        bits = int(parts[2]) if len(parts) > 2 else 4
        return datagen.config_mk(device, n=(1 << 28) // scale, seed=6 + seed_offset, nk=nk, digit_bits=bits)
    raise SystemExit(f"unknown workload {name}")


def workload_label(ds) -> str:
    meta = ",".join(f"{k}={v}" for k, v in ds.meta.items() if k != "seed")
    return f"{ds.name} n={ds.n} row_bytes={ds.row_bytes}" + (f" ({meta})" if meta else "")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            self.t.join(timeout=2)

    def summary(self):
        sm = sorted(int(r[0]) for r in self.rows if r and r[0].isdigit())
        mx = max((int(r[1]) for r in self.rows if len(r) > 1 and r[1].isdigit()), default=None)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 6 for i in range(4) if r[2 + i].lower().startswith("active")})
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": reasons, "samples": len(sm)}


def measured_hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except (OSError, KeyError, ValueError):
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def cpu_baseline(ds_cpu, budget_rows: int):
    """The oracle as it stands, single thread, on a bounded prefix of the same workload."""
    import oracle
    m = min(ds_cpu.n, budget_rows)
    keys = [k[:m].numpy() for k in ds_cpu.keys]
    vals = [v[:m].numpy() for v in ds_cpu.vals]
    res = oracle.groupby(keys, vals, ds_cpu.aggs, exact_f64_sum=ds_cpu.exact_f64_sum)
    return {"value": m / res.seconds, "unit": UNIT, "cores": 1, "host_cores": os.cpu_count(), "kind": "oracle",
            "sample": f"first {m} rows of the workload, one std::unordered_map pass, {res.seconds:.2f} s",
            "n_groups": res.n_groups}


def cpu_sample_rows(name: str) -> int:
    # about 10-30 s of single-thread oracle time (measured rates: ~8 ns/row at 6 groups ... ~250 ns at 10^8)
    base = name.split(":")[0].upper()
    return {"C1": 1_000_000, "C2": 400_000_000, "C3": 100_000_000, "C4": 50_000_000, "C5": 1 << 27, "MK": 1 << 27}.get(base, 1 << 26)


def run_reference(args):
    """--impl reference: the oracle (not tuned) on the host cores; each step = a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    sample = {"C1": 1_000_000, "C2": 1 << 26, "C3": 1 << 24, "C4": 1 << 23, "C5": 1 << 25, "MK": 1 << 25}[args.workload.split(":")[0].upper()]
    ds = build_workload(args.workload, "cpu", scale=max(args.scale, 1))
    m = min(ds.n, sample)
    keys = [k[:m].numpy() for k in ds.keys]
    vals = [v[:m].numpy() for v in ds.vals]
    run = lambda: oracle.groupby(keys, vals, ds.aggs, exact_f64_sum=ds.exact_f64_sum)
    for _ in range(args.warmup):
        run()
    t0 = time.perf_counter()
    secs = 0.0
    for _ in range(args.steps):
        secs += run().seconds
    wall = time.perf_counter() - t0
    value = m * args.steps / secs
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int64", "data": "synthetic",
            "config": {"workload": workload_label(ds), "sample_rows_per_step": m, "wall_s": wall},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "host_cores": os.cpu_count(), "kind": "oracle",
                             "sample": f"first {m} rows per step, std::unordered_map, single thread"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def max_over_ranks(ms: float, dist, device="cuda") -> float:
    """The slowest rank's time, on every rank (replicas only, no data-path collective)."""
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(rows_per_rank: int, world: int, steps: int, ms: float) -> float:
    """rows/s of the whole job: all ranks' rows over the slowest rank's time."""
    return rows_per_rank * world * steps / (ms * 1e-3)


def time_steps(fn, steps, warmup, torch, dist=None):
    for _ in range(warmup):
        fn()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    if dist is not None:
        ms = max_over_ranks(ms, dist)
        dist.barrier()
    return ms


def traffic_from_profiles(workload: str, kernel: str):
    """dram bytes per launch of the dominant kernel from the committed ncu capture, if there is one."""
    try:
        with open(os.path.join(ROOT, "profiles", "r1_traffic.json")) as f:
            d = json.load(f)
        # a capture of exactly this workload, else (C1-C4: one workload per name) of the config
        base = workload.split(":")[0].upper()
        return d.get(f"{workload.upper()}:{kernel}", d.get(f"{base}:{kernel}") if base in ("C1", "C2", "C3", "C4") else None)
    except (OSError, ValueError):
        return None


def main(argv=None):
    args = parse_args(argv)
    if args.impl == "reference":
        return run_reference(args)
    import torch
    import paper_2607_04489_b200 as eiger

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    eiger.lib()
    force = VARIANTS[args.force]

    if args.sweep:
        return sweep(args, eiger, torch, dev)

    ds = build_workload(args.workload, dev, scale=args.scale, seed_offset=rank)
    torch.cuda.synchronize()
    ws = eiger.Workspace(dev)
    last = {}

    def step():
        last["res"] = eiger.groupby(ds.keys, ds.vals, ds.aggs, force=force, workspace=ws)

    # device-resident timing (+ per-kernel events inside the library on the same stream)
    for _ in range(args.warmup):
        step()
    # two back-to-back timed regions of the same K steps: the first without the library's per-kernel
    # event pairs (that is `value`: the events cost ~0.1 ms of host work per call, 15 % of a 0.6 ms
    # call), the second with them (per-kernel times and the roofline line)
    l0 = eiger.launch_count()
    with ClockSampler(local) as clocks:
        ms = time_steps(step, args.steps, 0, torch, dist)
        launches = eiger.launch_count() - l0
        eiger.set_kernel_timing(True)
        for w in range(5):
            eiger.kernel_time_ms(w, True)
        ms_instrumented = time_steps(step, args.steps, 0, torch, dist)
        eiger.set_kernel_timing(False)
    kt = {name: eiger.kernel_time_ms(w, True) for w, name in enumerate(["aggregate", "profile", "partition", "init", "compact"])}
    res = last["res"]
    if ds.ndv is not None:
        assert res.n_groups == ds.ndv, (res.n_groups, ds.ndv)
    cnt_idx = [j for j, (op, _) in enumerate(ds.aggs) if op == eiger.COUNT]
    if cnt_idx:
        assert int(res.aggs[cnt_idx[0]].sum().item()) == ds.n      # sum COUNT = n

    rows_total = ds.n * world * args.steps
    value = whole_job_value(ds.n, world, args.steps, ms)
    in_bytes = ds.n * ds.row_bytes
    peak, peak_src = measured_hbm_peak()
    # dominant kernel and its algorithmic bytes per launch
    dom = max(("aggregate", "partition", "profile"), key=lambda k: kt[k][0])
    key_bytes = sum(k.element_size() for k in ds.keys)
    part_key = res.info["partition_key_bytes"] if res.variant == eiger.PARTITION else 8
    part_row = part_key + 8 * len(ds.vals)   # B': one row of the partitioned copy
    out_row = key_bytes + 8 * len(ds.aggs)
    levels = res.info["partition_levels"] if res.variant == eiger.PARTITION else 0
    # EIGER_AUTO's slice-sketch pass already took the level-1 histogram: no keys-only read in the partition pass
    hist1_bytes = 0 if (res.variant == eiger.PARTITION and res.info["partition_prehist"]) else ds.n * key_bytes
    alg_bytes = {"aggregate": in_bytes if res.variant != eiger.PARTITION else ds.n * part_row + res.n_groups * out_row,
                 "partition": hist1_bytes + ds.n * (ds.row_bytes + part_row) + max(0, levels - 1) * ds.n * (part_row - 8 * len(ds.vals) + 2 * part_row),
                 "profile": ds.n * key_bytes}[dom]
    dom_ms, dom_n = kt[dom]
    achieved = (alg_bytes / ((dom_ms / max(dom_n, 1)) * 1e-3)) / 1e9 if dom_ms > 0 else 0.0
    # the driver's peak is a copy (read + write at once); a pure read stream of this device, measured
    # now by the library's own probe kernels (16-byte loads / bulk copies), is quoted beside it
    try:
        read_peak = max(eiger.probe("read_ldg", 2048), eiger.probe("read_bulk", 2048, 32768))
        eiger.probe("release")
    except eiger.EigerError:
        read_peak = None
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64" if any(v.dtype == torch.float64 for v in ds.vals) else "int64", "data": "synthetic",
        "config": {"workload": workload_label(ds), "force": args.force, "variant": eiger.VARIANT_NAMES[res.variant],
                   "n_groups": res.n_groups, "l2": "inputs larger than L2 (no flush)" if in_bytes > (256 << 20) else "inputs fit L2: warm-L2 number",
                   "parallelism": "replicas only" if world > 1 else "single GPU", "scale": args.scale},
        "input_gb_per_s": value * ds.row_bytes / 1e9 / world,
        "frac_hbm_8tbs": value * ds.row_bytes / 1e9 / world / 8000.0,
        "gpu_launches": launches,
        "kernel_ms_per_step": {k: v[0] / args.steps for k, v in kt.items()},
        "ms_per_step_with_kernel_events": ms_instrumented / args.steps,
        "roofline": {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak if peak else None, "traffic": traffic_from_profiles(args.workload, dom), "peak_source": peak_src,
                     "algorithmic_bytes_per_launch": alg_bytes, "launches_timed": dom_n,
                     "read_only_peak_gbs": read_peak, "frac_of_read_only_peak": (achieved / read_peak) if read_peak else None},
        "clocks": clocks.summary(),
    }

    # end to end: pinned host buffers -> eiger_groupby_host (H2D + compute + D2H per step)
    if not args.no_e2e:
        hk = [k.cpu().pin_memory() for k in ds.keys]
        hv = [v.cpu().pin_memory() for v in ds.vals]
        cap = max(1024, 2 * (ds.ndv or ds.n))
        ok = [torch.empty(cap, dtype=k.dtype).pin_memory() for k in hk]
        oa = [torch.empty(cap, dtype=torch.float64 if (op != eiger.COUNT and hv[c].dtype == torch.float64) else torch.int64).pin_memory()
              for (op, c) in ds.aggs]
        stat = {}

        def e2e_step():
            stat["r"] = eiger.groupby_host(hk, hv, ds.aggs, force=force, out_capacity=cap, out=(ok, oa))
        e2e_ms = time_steps(e2e_step, args.steps, min(args.warmup, 2), torch, dist)
        r, h2d, d2h = stat["r"]
        assert r.n_groups == res.n_groups
        line["e2e"] = {"value": rows_total / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                       "ms_per_step": e2e_ms / args.steps}
        del hk, hv
    if not args.no_cpu and world == 1 and rank == 0:
        line["cpu_baseline"] = cpu_baseline(ds.cpu(), cpu_sample_rows(args.workload) // max(args.scale, 1))
    if not args.no_curve and world == 1:
        del ds, res, ws
        last.clear()
        torch.cuda.empty_cache()
        line["ndv_curve"] = ndv_curve(args, eiger, torch, dev, peak)
    if rank == 0:
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


CURVE_POINTS = [f"C5:{lg}:{lay}" for lay in ("dense", "scattered") for lg in (4, 8, 12, 13, 14, 15, 16, 20, 24, 28)] + ["C3", "C4", "MK:4:2", "MK:4:6"]


def ndv_curve(args, eiger, torch, dev, peak):
    """The metric is "rows/s and input GB/s vs NDV": EIGER_AUTO (statistics gathered inside the timed
    call) at every C5 point (both layouts, 2^13..2^15 included), C3, C4 and two multi-key points (4 x int32 key
    columns, 2^8 and 2^24 groups), each with the per-kernel
    device times of a second, instrumented region.  --curve-forced adds the forced variants with the
    statistics supplied (profile excluded), the reading of "within 10 % of the best single variant"."""
    out = []
    ws = eiger.Workspace(dev)
    names = ["aggregate", "profile", "partition", "init", "compact"]
    for name in CURVE_POINTS:
        try:
            ds = build_workload(name, dev, scale=args.scale)
        except torch.OutOfMemoryError:
            out.append({"workload": name, "error": "oom"})
            continue
        fn = lambda: eiger.groupby(ds.keys, ds.vals, ds.aggs, workspace=ws)
        try:
            r = fn()
            assert ds.ndv is None or r.n_groups == ds.ndv, (name, r.n_groups, ds.ndv)
            est = time_steps(fn, 2, 3, torch) / 2
            k = max(3, min(30, int(40.0 / max(est, 1e-3))))
            ms = time_steps(fn, k, 0, torch) / k
            eiger.set_kernel_timing(True)
            for w in range(5):
                eiger.kernel_time_ms(w, True)
            time_steps(fn, k, 0, torch)
            eiger.set_kernel_timing(False)
            kt = {nm: eiger.kernel_time_ms(w, True)[0] / k for w, nm in enumerate(names)}
            gbs = ds.n * ds.row_bytes / ms / 1e6
            row = {"workload": name, "n": ds.n, "ndv": ds.ndv, "variant": eiger.VARIANT_NAMES[r.variant], "ms": round(ms, 4), "steps": k,
                   "rows_per_s": ds.n / ms * 1e3, "input_gb_per_s": round(gbs, 1), "frac_8tbs": round(gbs / 8000.0, 4),
                   "frac_measured_peak": round(gbs / peak, 4), "kernel_ms": {a: round(b, 4) for a, b in kt.items()}}
            if args.curve_forced:
                st = eiger.profile_keys(ds.keys)
                lg = (ds.ndv or 1).bit_length() - 1
                dense = (not ds.meta.get("scattered", False) and name.startswith("C5")) or (name.startswith("MK") and lg <= 20)
                forced = {}
                for vname, v in VARIANTS.items():
                    if v == 0 or (v == 1 and not dense) or (v == 2 and lg > 16) or (v == 3 and lg > 20):
                        continue      # variants that take tens of milliseconds here (round-1 sweep) are not re-timed
                    try:
                        f2 = lambda: eiger.groupby(ds.keys, ds.vals, ds.aggs, force=v, stats=st, workspace=ws)
                        f2()
                        e2 = time_steps(f2, 2, 2, torch) / 2
                        k2 = max(3, min(30, int(40.0 / max(e2, 1e-3))))
                        forced[vname] = round(time_steps(f2, k2, 0, torch) / k2, 4)
                    except eiger.EigerError as e:
                        forced[vname] = f"error {e.code}"
                row["forced_ms"] = forced
                best = min((x for x in forced.values() if isinstance(x, float)), default=None)
                row["auto_over_best_forced"] = round(ms / best, 3) if best else None
            out.append(row)
        except (eiger.EigerError, AssertionError) as e:
            out.append({"workload": name, "error": str(e)[:200]})
        except torch.OutOfMemoryError:
            out.append({"workload": name, "error": "oom"})
            ws = eiger.Workspace(dev)
        print(json.dumps(out[-1]), file=sys.stderr, flush=True)
        del ds
        torch.cuda.empty_cache()
    return out


def sweep(args, eiger, torch, dev):
    """Config 5: 2^28 rows, NDV = 2^4 .. 2^28, dense and scattered, every variant forced + AUTO.
    Forced-variant time excludes the profile (statistics supplied); AUTO includes it."""
    out = []
    ws = eiger.Workspace(dev)
    n = (1 << 28) // args.scale
    for scattered in (False, True):
        for lg in (4, 8, 12, 16, 20, 24, 28):
            if (1 << lg) > n:
                continue
            import datagen
            ds = datagen.config5(dev, n=n, ndv=1 << lg, scattered=scattered)
            st = [eiger.profile(ds.keys[0])]
            row = {"ndv_log2": lg, "layout": "scattered" if scattered else "dense", "n": n, "ndv_est": st[0].ndv_est}
            for name, v in VARIANTS.items():
                try:
                    fn = (lambda: eiger.groupby(ds.keys, ds.vals, ds.aggs, force=v, workspace=ws)) if v == 0 else \
                         (lambda: eiger.groupby(ds.keys, ds.vals, ds.aggs, force=v, stats=st, workspace=ws))
                    r = fn()
                    assert r.n_groups == ds.ndv
                    # sub-millisecond calls get more timed steps (>= ~30 ms in all): 5 steps of a 0.6 ms
                    # call are 3 ms of timing and moved by +-7 % from run to run
                    est = time_steps(fn, 2, 3, torch) / 2
                    k = max(args.steps, min(50, int(30.0 / max(est, 1e-3))))
                    ms = time_steps(fn, k, 0, torch) / k
                    row[name] = {"ms": ms, "steps": k, "rows_per_s": n / ms * 1e3, "gb_per_s": n * 12 / ms / 1e6,
                                 "variant": eiger.VARIANT_NAMES[r.variant]}
                except eiger.EigerError as e:
                    row[name] = {"error": e.code}
                except torch.OutOfMemoryError:
                    row[name] = {"error": "oom"}
                    ws = eiger.Workspace(dev)
                    torch.cuda.empty_cache()
            t0 = torch.cuda.Event(enable_timing=True); t1 = torch.cuda.Event(enable_timing=True)
            t0.record(); eiger.profile(ds.keys[0]); t1.record(); torch.cuda.synchronize()
            row["profile_ms"] = t0.elapsed_time(t1)
            out.append(row)
            print(json.dumps(row), file=sys.stderr)
            del ds
    print(json.dumps({"metric": "c5_crossover_sweep", "sweep": out}))


if __name__ == "__main__":
    main()
