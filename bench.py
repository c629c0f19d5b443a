#!/usr/bin/env python
"""bench.py — throughput of the TPC cluster finder on synthetic Pb-Pb time frames.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]

A "step" is one pass of the whole hot path (S0..S7 of SURVEY.md §8(a)) over one time frame:
for BASELINE.json:configs[3] that is 14 fragments (13 x 4096 + 3776 bins, 8-bin halo) of
36 sectors, ~4.4e9 digits, resident in HBM when the timed region starts.  Prints ONE JSON
line (rank 0).  Multi-GPU (torchrun): the path does not shard (BASELINE.json:north_star:
"one GPU only, no sharding"), so N ranks run N independent replicas ("replicas only").

--impl reference times the ORACLE (oracle/, plain single-threaded C++ per call, one sector per
host thread) on a bounded sample of the same workload; it is a baseline, not the target.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time
from concurrent.futures import ThreadPoolExecutor

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "tpc_digits_per_sec"
UNIT = "digits/s"
THETA = 64          # peak_min_q16 = 4 ADC (D11 default)


def log(*a):
    print("[bench]", *a, file=sys.stderr, flush=True)


# ----------------------------------------------------------------------------------------------
# distributed plumbing (replicas only): barrier + max over ranks
# ----------------------------------------------------------------------------------------------
def dist_setup(backend=None):
    """Returns (rank, world, local_rank).  Initialises torch.distributed when WORLD_SIZE > 1."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist

        if not dist.is_initialized():
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            dist.init_process_group(backend or "nccl", rank=rank, world_size=world)
    return rank, world, local


def dist_barrier(world, device=None):
    if world > 1:
        import torch.distributed as dist

        if device is not None and dist.get_backend() == "nccl":
            dist.barrier(device_ids=[device])
        else:
            dist.barrier()


def dist_max_sum(ms: float, units: float, world: int, device="cpu"):
    """(max over ranks of the elapsed time, sum over ranks of the units processed)."""
    if world == 1:
        return ms, units
    import torch
    import torch.distributed as dist

    t = torch.tensor([ms], dtype=torch.float64, device=device)
    u = torch.tensor([units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


# ----------------------------------------------------------------------------------------------
# clocks (profiling recipe: sample nvidia-smi DURING the timed region)
# ----------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi sampled every 20 ms from BEFORE the warm-up (the process takes a few hundred ms to start); only
    the samples whose timestamp falls inside the timed region [t0, t1] (host clock) are reported."""
    Q = "timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown," \
        "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown," \
        "clocks_event_reasons.sw_power_cap"
    PERIOD_MS = 20

    def __init__(self, index=0):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", str(self.PERIOD_MS)],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def wait_ready(self, timeout=5.0):
        """nvidia-smi needs a few hundred ms to produce its first sample: do not start a short timed region before."""
        if self.p is None:
            return
        t_end = time.time() + timeout
        while time.time() < t_end and os.path.getsize(self.f.name) == 0:
            time.sleep(0.02)

    def stop(self, t0=None, t1=None):
        import datetime

        out = dict(sm_mhz=None, sm_max_mhz=None, reasons=[], samples=0, period_ms=self.PERIOD_MS)
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 8:
                continue
            try:
                ts = datetime.datetime.strptime(c[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                if t0 is not None and not (t0 <= ts <= t1):
                    continue
                sm.append(float(c[1])); mx.append(float(c[2]))
            except ValueError:
                continue
            for nme, v in zip(names, c[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons),
                       samples=len(sm))
        return out


def kernel_source_sha256():
    """Hash of the CUDA sources: profiles/traffic.json (ncu numbers) is stamped with it, and a bench line whose
    kernels differ from the profiled ones says so instead of quoting stale counters."""
    import hashlib

    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2412_13755_b200", "csrc")
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")):
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def ncu_numbers(cfg_name):
    """profiles/traffic.json: per-launch DRAM bytes and warp instructions per digit from the committed ncu capture,
    keyed by workload; None when there is no entry for this workload."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(p):
        return None
    tj = json.load(open(p))
    ent = tj.get("workloads", {}).get(cfg_name)
    if ent is None:
        return None
    ent = dict(ent)
    ent["stale"] = ent.get("source_sha256") != kernel_source_sha256()
    return ent


def measured_peak_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


# ----------------------------------------------------------------------------------------------
# workload
# ----------------------------------------------------------------------------------------------
def sort_within_sectors(d, offs, order):
    """Digit order inside a sector slice is arbitrary; the configs say "random order".  For the
    sorted-order timings of BASELINE.md §6: re-order every slice by (row,time,pad) or (time,row,pad)."""
    import torch

    w = d.view(torch.int64).view(-1)
    row, pad, tim = w & 0xFF, (w >> 8) & 0xFF, (w >> 16) & 0xFFFF
    key = (row << 24) | (tim << 8) | pad if order == "row_time_pad" else (tim << 16) | (row << 8) | pad
    sec = torch.repeat_interleave(torch.arange(len(offs) - 1, device=d.device),
                                  torch.as_tensor(np.diff(offs).astype(np.int64), device=d.device))
    idx = torch.argsort(key | (sec << 40))
    return w[idx].view(torch.uint8).view(-1, 8)


def make_tf(cfg, device, frags=None, order="shuffled"):
    import gen

    out = []
    t0 = time.time()
    for f, (b, e) in enumerate(cfg.fragments()):
        if frags is not None and f not in frags:
            continue
        d, offs, info = gen.generate_fragment(cfg, f, device=device,
                                              row_chunk=64 if str(device).startswith("cuda") else 16)
        if order != "shuffled":
            d = sort_within_sectors(d, offs, order)
        out.append(dict(f=f, b=b, e=e, base=info["t_time_base"], digits=d, offs=offs, n=int(d.shape[0]),
                        occ=info["occupancy"]))
    log(f"generated {cfg.name}: {len(out)} fragments, {sum(x['n'] for x in out):,} digits, "
        f"mean occupancy {np.mean([x['occ'] for x in out]):.4f}, {time.time() - t0:.1f} s on {device}")
    return out


def oracle_sample(cfg, frag, sectors, threads):
    """Run the oracle on `sectors` of one fragment, one sector per call, `threads` calls in
    parallel.  Returns (seconds, digits processed, {sector: records})."""
    import oracle

    dn = frag["digits_np"]
    offs = frag["offs"]
    npads = cfg.npads_array()

    def one(s):
        a, b_ = int(offs[s]), int(offs[s + 1])
        rec, st = oracle.run(dn[a:b_], np.array([0, b_ - a], dtype=np.uint64), npads, n_sectors=1,
                             tf_time_bins=cfg.tf_time_bins, t_core_begin=frag["b"], t_core_end=frag["e"],
                             halo_bins=cfg.halo_bins, peak_min_q16=THETA, t_time_base=frag.get("base", 0))
        return s, rec

    oracle.build()
    t0 = time.perf_counter()
    with ThreadPoolExecutor(max_workers=threads) as ex:
        res = dict(ex.map(one, sectors))
    dt = time.perf_counter() - t0
    nd = int(sum(int(offs[s + 1]) - int(offs[s]) for s in sectors))
    return dt, nd, res


# ----------------------------------------------------------------------------------------------
def run_reference(args):
    """The oracle as it stands, on the box's host cores, on a bounded sample per step."""
    rank, world, local = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), 0
    if rank != 0:
        return
    import torch
    import gen

    cfg = gen.config(args.config)
    cores = os.cpu_count() or 1
    n_s = min(cfg.n_sectors, cores)
    dev = "cuda:0" if torch.cuda.is_available() else "cpu"
    import gen as _g
    d, offs, info = _g.generate_fragment(cfg, 0, device=dev, sectors=range(n_s),
                                         row_chunk=64 if dev != "cpu" else 16)
    b, e = cfg.fragments()[0]
    frag = dict(b=b, e=e, base=info["t_time_base"], offs=offs, digits_np=_g.as_numpy_digits(d))
    times, nd, ncl = [], 0, 0
    for i in range(args.warmup + args.steps):
        dt, nd, res = oracle_sample(cfg, frag, list(range(n_s)), cores)
        ncl = sum(len(r) for r in res.values())
        if i >= args.warmup:
            times.append(dt)
    ms = 1e3 * float(np.mean(times))
    val = nd / (ms * 1e-3)
    sample = f"{n_s} of {cfg.n_sectors} sectors of fragment 0 ({nd:,} digits), one sector per thread"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "int64/f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "sample": sample},
        "clusters_per_sec": ncl / (ms * 1e-3),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": min(cores, n_s), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }), flush=True)


def workload_name(cfg):
    fr = cfg.fragments()
    return (f"{cfg.name}: {cfg.n_sectors} sectors x {cfg.n_rows} rows x {cfg.tf_time_bins} time bins, "
            f"{len(fr)} fragment(s) of <= {cfg.core_bins} bins, halo {cfg.halo_bins}, seed {cfg.seed}, theta 4 ADC")


def run_ours(args):
    import torch
    import gen
    import paper_2412_13755_b200 as T

    rank, world, local = dist_setup()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    cfg = gen.config(args.config)
    npads = cfg.npads_array()
    tf = make_tf(cfg, dev, order=args.digit_order)
    n_dig = sum(x["n"] for x in tf)
    max_n = max(x["n"] for x in tf)
    stream = torch.cuda.current_stream().cuda_stream

    ctx = T.tpcclus_create(npads, n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins,
                           max_core_bins=cfg.core_bins, halo_bins=cfg.halo_bins, peak_min_q16=THETA,
                           max_digits=max_n, cuda_device=local)
    # count pass (capacity 0): cluster counts per fragment -> exact output sizing
    for x in tf:
        T.tpcclus_run_based(ctx, x["digits"].data_ptr(), x["n"], x["offs"], x["base"], x["b"], x["e"], 0, 0, stream)
    counts = []
    for x in tf:
        st = T.tpcclus_result(ctx, check=False)
        assert st["status"] in (T.TPCCLUS_OK, T.TPCCLUS_ERR_CAPACITY) and st["n_digits_dropped"] == 0, st
        counts.append(int(st["n_clusters"]))
    n_cl = sum(counts)
    starts = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    out = torch.zeros((max(n_cl, 1), 32), dtype=torch.uint8, device=dev)
    ctx_bytes = T.tpcclus_device_bytes(ctx)
    log(f"{n_dig:,} digits -> {n_cl:,} clusters; context holds {ctx_bytes / 1e9:.2f} GB")

    def step():
        for i, x in enumerate(tf):
            T.tpcclus_run_based(ctx, x["digits"].data_ptr(), x["n"], x["offs"], x["base"], x["b"], x["e"],
                                out.data_ptr() + int(starts[i]) * 32, counts[i], stream)
        for i in range(len(tf)):
            st = T.tpcclus_result(ctx)
            assert st["n_clusters"] == counts[i]

    clocks = ClockSampler(local)              # started before the warm-up so that it is sampling by the timed region
    clocks.wait_ready()
    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    dist_barrier(world, local)
    T.tpcclus_set_profiling(ctx, True)
    launches0 = T.tpcclus_launch_count(ctx)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    wall0 = time.time()
    ev0.record()
    for _ in range(args.steps):
        step()
    ev1.record()
    torch.cuda.synchronize()
    wall1 = time.time()
    dist_barrier(world, local)
    ms_total = ev0.elapsed_time(ev1)
    clk = clocks.stop(wall0, wall1)
    if clk["samples"] < 5:
        log(f"only {clk['samples']} clock samples inside the timed region ({ms_total:.1f} ms): raise --steps "
            f"(>= {int(5 * ClockSampler.PERIOD_MS * 1.5 / max(ms_total / args.steps, 1e-3)) + 1} for this config)")
    launches = T.tpcclus_launch_count(ctx) - launches0
    prof, prof_runs = T.tpcclus_get_profile(ctx)
    T.tpcclus_set_profiling(ctx, False)
    ms_step_local = ms_total / args.steps
    ms_step, units = dist_max_sum(ms_step_local, float(n_dig), world, dev)
    value = units / (ms_step * 1e-3)

    if rank != 0:
        T.tpcclus_destroy(ctx)
        return

    # ---- roofline of the dominant kernel (algorithmic bytes per launch / mean launch time) ----
    peak, peak_src = measured_peak_gbs()
    nfr = len(tf)
    # entries appended to the bin lists: every digit once, plus once more when it lies within
    # 5 bins of a 256-bin seam (10/256 of the core bins)
    dup = 1.0 + 10.0 / 256.0
    alg = {   # bytes per launch, DESIGN.md §6
        "k_init": 4.0 * cfg.n_sectors * cfg.n_rows * ((cfg.core_bins + 255) // 256),   # one counter per bin
        "k_bin": (8.0 + 4.0 * dup) * n_dig / nfr,                 # read 8 B/digit, append 4 B per list entry
        "k_tile": (4.0 * dup * n_dig + 32.0 * n_cl) / nfr,        # read every list entry once, write every record
    }
    kern = {}
    for k, ms_sum in prof.items():
        ms_avg = ms_sum / max(prof_runs, 1)
        kern[k] = dict(ms_per_launch=ms_avg, alg_bytes_per_launch=alg[k],
                       achieved_gbs=alg[k] / (ms_avg * 1e-3) / 1e9 if ms_avg > 0 else None,
                       share=ms_sum / max(sum(prof.values()), 1e-9))
    dom = max(kern, key=lambda k: kern[k]["ms_per_launch"])
    # ncu counters of the committed capture of THIS workload (a C3 fragment is a C2 fragment: same generator, same
    # size); null when the capture is of another workload, flagged when the kernels have changed since
    fragment_like = "C2-PbPb-fragment" if cfg.name.startswith(("C3-", "TF-")) else cfg.name
    ncu = ncu_numbers(fragment_like)
    traffic = ncu["dram_bytes_per_launch"].get(dom) if ncu else None
    # secondary, SM-side ceiling: both kernels are bound by instruction issue, not by HBM.
    # Warp instructions per launch come from the same ncu capture as `traffic` (they scale with the digits
    # of a launch); the peak is 4 schedulers x SMs x the SM clock sampled under load.
    issue = None
    if ncu and clk.get("sm_mhz"):
        import torch
        n_sm = torch.cuda.get_device_properties(local).multi_processor_count
        peak_issue = 4.0 * n_sm * clk["sm_mhz"] * 1e6
        issue = {}
        for k in ("k_bin", "k_tile"):
            wi = ncu["warp_inst_per_digit"].get(k)
            if wi and kern[k]["ms_per_launch"] > 0:
                ach = wi * n_dig / nfr / (kern[k]["ms_per_launch"] * 1e-3)
                issue[k] = dict(warp_inst_per_launch=wi * n_dig / nfr, achieved=ach, peak=peak_issue,
                                unit="warp-inst/s", frac=ach / peak_issue)
    roofline = dict(bound="hbm", kernel=dom, achieved=kern[dom]["achieved_gbs"], peak=peak, unit="GB/s",
                    frac=kern[dom]["achieved_gbs"] / peak, traffic=traffic, peak_source=peak_src,
                    traffic_source=(dict(file="profiles/traffic.json", workload=fragment_like,
                                         captured_on_source_sha256=ncu.get("source_sha256"),
                                         this_source_sha256=kernel_source_sha256(), stale=ncu["stale"])
                                    if ncu else None),
                    kernels=kern, issue=issue,
                    whole_step=dict(
                        b_min_bytes=8.0 * n_dig + 32.0 * n_cl,
                        frac_b_min=(8.0 * n_dig + 32.0 * n_cl) / (ms_step_local * 1e-3) / 1e9 / peak,
                        frac_b_min_nominal_8tbs=(8.0 * n_dig + 32.0 * n_cl) / (ms_step_local * 1e-3) / 1e9 / 8000.0,
                        b_alg_bytes=sum(alg.values()) * nfr,
                        frac_b_alg=sum(alg.values()) * nfr / (ms_step_local * 1e-3) / 1e9 / peak))

    # ---- cpu baseline (oracle, bounded sample) + parity check at full size ----
    # Sampled so that the first AND the last fragment and the first AND the last sectors are covered: the lower
    # half of the sectors on fragment 0, the upper half (incl. sectors 32..35: the tail of k_bin's chunk ranges
    # and k_tile's last tickets) on the last fragment (C3: the ragged 3776-bin one at the true TF end).
    cpu, parity = None, None
    if world == 1 and not args.no_cpu:
        cores = os.cpu_count() or 1
        ns = cfg.n_sectors
        half = (ns + 1) // 2
        plan = [(0, list(range(ns)))] if nfr == 1 else [(0, list(range(half))), (nfr - 1, list(range(half, ns)))]
        bad, nrec, parts, t_cpu, nd_cpu = 0, 0, [], 0.0, 0
        single = None
        for fi, secs in plan:
            fx = tf[fi]
            a, b_ = int(fx["offs"][secs[0]]), int(fx["offs"][secs[-1] + 1])
            offs_local = np.asarray(fx["offs"], dtype=np.int64) - a
            frag = dict(b=fx["b"], e=fx["e"], base=fx["base"], offs=offs_local,
                        digits_np=gen.as_numpy_digits(fx["digits"][a:b_]))
            if single is None:      # the same oracle on ONE thread, one sector
                dt1, nd1, _ = oracle_sample(cfg, frag, secs[:1], 1)
                single = dict(value=nd1 / dt1, unit=UNIT, cores=1, seconds=dt1,
                              sample=f"sector {secs[0]} of fragment {fi} ({nd1:,} digits)")
            dt, nd, res = oracle_sample(cfg, frag, secs, cores)
            t_cpu += dt
            nd_cpu += nd
            got = out[int(starts[fi]): int(starts[fi]) + counts[fi]].cpu().numpy().view(T.CLUSTER_DTYPE).reshape(-1)
            for s_, rec in res.items():
                g = got[got["sector"] == s_].copy()
                g["sector"] = 0
                nrec += len(rec)
                bad += (len(g) != len(rec)) or (g.tobytes() != rec.tobytes())
            parts.append(f"fragment {fi} sectors {secs[0]}..{secs[-1]}")
        sample = f"{' + '.join(parts)} of {workload_name(cfg).split(':')[0]} ({nd_cpu:,} digits), one sector per thread"
        cpu = dict(value=nd_cpu / t_cpu, unit=UNIT, cores=min(cores, half if nfr > 1 else ns), kind="oracle", sample=sample,
                   seconds=t_cpu, single_thread=single)
        parity = dict(checked=parts, records=nrec, sectors_not_bit_identical=int(bad))

    # ---- D13 selection pass over the step's cluster list, an HBM-bound kernel of its own ----
    select = None
    if args.select:
        cuts = dict(min_qtot=8.0, reject_single_pad=True, reject_single_time=True)
        sel_out = torch.empty_like(out)
        for _ in range(3):
            T.tpcclus_select(ctx, out.data_ptr(), n_cl, sel_out.data_ptr(), n_cl, stream, **cuts)
            kept = T.tpcclus_select_result(ctx)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 10
        torch.cuda.synchronize()
        e0.record()
        for _ in range(reps):
            T.tpcclus_select(ctx, out.data_ptr(), n_cl, sel_out.data_ptr(), n_cl, stream, **cuts)
            T.tpcclus_select_result(ctx)
        e1.record()
        torch.cuda.synchronize()
        ms_sel = e0.elapsed_time(e1) / reps
        by = 32.0 * n_cl + 32.0 * kept
        select = dict(cuts=cuts, records=n_cl, kept=kept, ms=ms_sel, alg_bytes=by, achieved_gbs=by / (ms_sel * 1e-3) / 1e9,
                      frac_of_hbm_peak=by / (ms_sel * 1e-3) / 1e9 / peak,
                      note="timed with the host wait of tpcclus_select_result inside (one call per repetition)")
        if not args.no_cpu and world == 1:
            got = sel_out[: min(kept, 2_000_000)].cpu().numpy().view(T.CLUSTER_DTYPE).reshape(-1)
            import oracle
            head = out[: min(n_cl, 8_000_000)].cpu().numpy().view(T.CLUSTER_DTYPE).reshape(-1)
            want, _ = oracle.select(head, **cuts)
            m = min(len(want), len(got))
            select["parity_first_records"] = dict(compared=m, identical=bool(got[:m].tobytes() == want[:m].tobytes()))
        del sel_out

    # ---- end to end through the C-ABI with HOST buffers (H2D + kernels + D2H inside the timing) ----
    e2e = None
    if not args.no_e2e:
        try:
            e2e = run_e2e(args, cfg, tf, counts, T, local, world)
        except Exception as ex:  # report, never fake
            log("e2e failed:", repr(ex))
            e2e = dict(value=None, unit=UNIT, error=repr(ex))

    T.tpcclus_destroy(ctx)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u16", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "digits_per_step": n_dig, "clusters_per_step": n_cl,
                   "digit_order": args.digit_order, "fragments": nfr, "context_bytes": int(ctx_bytes), "resident_digit_bytes": int(n_dig * 8),
                   "l2": "inputs larger than L2 (digits %.1f GB per step, %.1f GB per fragment)"
                         % (n_dig * 8 / 1e9, n_dig * 8 / nfr / 1e9),
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "clusters_per_sec": n_cl * world / (ms_step * 1e-3),
        "clocks": clk, "e2e": e2e, "gpu_launches": int(launches),
        "roofline": roofline, "cpu_baseline": cpu, "parity_check": parity,
    }
    if select is not None:
        line["select"] = select
    print(json.dumps(line), flush=True)


def run_e2e(args, cfg, tf, counts, T, local, world):
    import torch

    npads = cfg.npads_array()
    n_dig, n_cl = sum(x["n"] for x in tf), sum(counts)
    ctx = T.tpcclus_create(npads, n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins,
                           max_core_bins=cfg.core_bins, halo_bins=cfg.halo_bins, peak_min_q16=THETA,
                           options=T.TPCCLUS_OPT_HOST_STAGING, max_digits=max(x["n"] for x in tf),
                           max_clusters=max(counts) + 1, cuda_device=local)
    try:
        t0 = time.time()
        hosts = []
        for x in tf:
            h = torch.empty((x["n"], 8), dtype=torch.uint8, pin_memory=True)
            h.copy_(x["digits"])
            hosts.append(h)
        h_out = torch.empty((max(n_cl, 1), 32), dtype=torch.uint8, pin_memory=True)
        torch.cuda.synchronize()
        log(f"e2e: pinned {n_dig * 8 / 1e9:.1f} GB of digits + {n_cl * 32 / 1e9:.1f} GB of records on the host in {time.time() - t0:.1f} s")
        frs = [(h.data_ptr(), x["n"], x["offs"], x["b"], x["e"], x["base"]) for h, x in zip(hosts, tf)]
        n_e2e = max(1, min(args.steps, 3))
        for _ in range(1):
            st = T.tpcclus_run_tf_host(ctx, frs, h_out.data_ptr(), n_cl)
        assert [s["n_clusters"] for s in st] == counts
        dist_barrier(world, local)
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            T.tpcclus_run_tf_host(ctx, frs, h_out.data_ptr(), n_cl)   # returns after the last D2H
        dt = (time.perf_counter() - t0) / n_e2e
        dist_barrier(world, local)
        ms, units = dist_max_sum(dt * 1e3, float(n_dig), world, f"cuda:{local}")
        return dict(value=units / (ms * 1e-3), unit=UNIT, ms_per_step=ms, steps=n_e2e,
                    h2d_bytes_per_step=int(n_dig * 8), d2h_bytes_per_step=int(n_cl * 32),
                    api="tpcclus_run_tf_host, pinned host buffers; H2D, kernels and D2H overlapped across fragments")
    finally:
        T.tpcclus_destroy(ctx)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="3", help="BASELINE.json config index 0..4 (default 3: the full Pb-Pb TF), or "
                    "tf32 | tf128 | tf256: the TF-length sweep of PAPER.md:118 (the C3 generator over 32 / 128 / 256 orbits)")
    ap.add_argument("--digit-order", default="shuffled", choices=["shuffled", "row_time_pad", "time_row_pad"],
                    help="order of the digits inside each sector slice (the configs' 'random order' is the default)")
    ap.add_argument("--select", action="store_true", help="also time tpcclus_select (D13 quality selection) over the step's clusters")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    args = ap.parse_args()
    args.config = int(args.config) if args.config.isdigit() else args.config
    args.warmup = max(args.warmup, 0)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # launched bare: start the N replicas ourselves, one process per GPU, the way the driver would
        # (torch.distributed.run, rendezvous on 127.0.0.1); rank 0 prints the JSON line
        import socket

        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
        sys.exit(subprocess.call(cmd))
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
