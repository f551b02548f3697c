#!/usr/bin/env python
"""bench.py -- SF-TR forward/back projector throughput on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path over one synthetic batch: one ct_fp_sf (y = A x) followed by
one ct_bp_sf (x^ = A^T y) on the headline workload (config 4: 512^3 voxels x 720 views, non-circular
cone beam, flat 768^2 detector).  value = voxel x view updates of both operators / second / 1e9 (GUPS),
inputs resident in HBM; e2e = the same through ct_fp_sf_host / ct_bp_sf_host with pinned HOST buffers.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl reference]

N > 1 (torchrun): every rank runs an independent replica of the workload (the path shards by
batch/volume with no data-path collective), weak scaling, max-over-ranks time.
`--shard views` instead splits the views of ONE workload over the ranks: A on each rank's
shard of views with the volume replicated, A^T on the shard followed by one NCCL sum all-reduce of the volume;
strong scaling.

roofline.peak is MEASURED in the same run (ct_measure_fp32_peak: FMA-only kernel, before the timed region);
roofline.achieved = algorithmic flops (FLOP_PER_UPDATE, a count of the method's arithmetic) /
the dominant kernel's CUDA-event time; the flops the kernels actually execute (ncu op counts, packed forms included),
their DRAM traffic, L2 and shared-memory-pipe utilisation are summed here from the committed ncu capture
profiles/r3_counts_config<C>.csv (measured_counts); `counts_stale` says whether csrc/ has changed since that capture.
"""
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

from paper_2503_16741_b200 import workloads as W  # noqa: E402

METRIC_SHORT = "SF fwd/back GUPS (voxel*view/s)"
METRIC = "SF fwd/back GUPS (voxel*view/s) at 512^3 x 720 views; % of HBM roofline"   # BASELINE.json "metric"


def metric_name(config_index):
    """BASELINE.json's metric string for its headline workload (config 4); the same quantity, named without
    the workload, for the other configs (their workload is in config.workload)."""
    return METRIC if config_index == 4 else METRIC_SHORT
# Algorithmic flop per NOMINAL voxel x view update: live fraction x flop per live
# update (S1-S5 counted from the method at the config's mean footprint size) + dead fraction x 10.
FLOP_PER_UPDATE = {1: 88.0, 2: 46.0, 3: 30.0, 4: 60.0, 5: 10.0}
FP32_LANES_PER_SM, N_SM = 128, 148


def peaks():
    p = {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "src": "fallback"}
    try:
        m = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        p.update(hbm_gbs=float(m["hbm_gbs"]), sm_max_mhz=float(m.get("sm_max_mhz", 1965.0)), src="measured")
    except Exception:
        pass
    p["fp32_tflops_nominal"] = N_SM * FP32_LANES_PER_SM * 2 * p["sm_max_mhz"] * 1e6 / 1e12
    return p


COUNTS_METRICS = (
    "smsp__sass_thread_inst_executed_op_fadd_pred_on.sum,smsp__sass_thread_inst_executed_op_fmul_pred_on.sum,"
    "smsp__sass_thread_inst_executed_op_ffma_pred_on.sum,smsp__sass_thread_inst_executed_op_fadd2_pred_on.sum,"
    "smsp__sass_thread_inst_executed_op_fmul2_pred_on.sum,smsp__sass_thread_inst_executed_op_ffma2_pred_on.sum,"
    "smsp__thread_inst_executed.sum,smsp__inst_executed.sum,dram__bytes_read.sum,dram__bytes_write.sum,"
    "gpu__time_duration.sum,l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum,"
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum,smsp__issue_active.avg.pct_of_peak_sustained_active,"
    "lts__t_sector_hit_rate.pct,lts__t_sectors.avg.pct_of_peak_sustained_elapsed,"
    "l1tex__data_pipe_lsu_wavefronts_mem_shared.avg.pct_of_peak_sustained_elapsed")
COUNTS_CSV = os.path.join(ROOT, "profiles", "r3_counts_config%d.csv")
COUNTS_STAMP = os.path.join(ROOT, "profiles", "r3_counts_stamp.json")
CSRC = os.path.join(ROOT, "paper_2503_16741_b200", "csrc")


def csrc_sha256():
    """One hash over the library's sources: says which build a counts capture belongs to."""
    import hashlib
    h = hashlib.sha256()
    for name in sorted(os.listdir(CSRC)):
        if name.endswith((".cu", ".cuh", ".h", ".cpp")):
            h.update(name.encode())
            h.update(open(os.path.join(CSRC, name), "rb").read())
    return h.hexdigest()[:16]


def measured_counts(config_index, algo, n_updates):
    """Per-operator-call counts of the hot kernels, summed HERE from the committed ncu capture
    profiles/r3_counts_config<C>.csv (one `bench.py --steps 1 --warmup 0` run under
    `ncu --metrics COUNTS_METRICS --clock-control none -k regex:"fp_band|bp_brick|bp_pixel|transpose" --csv`; the full
    command is in profiles/README.md).  Executed flops = FADD + FMUL + 2 FFMA + 2 (FADD2 + FMUL2) + 4 FFMA2 thread
    instructions: the packed forms are counted by their own ncu counters (the scalar ones do not see them).
    Percent-type metrics are time-weighted over the operator's launches.  `stale`: the library's sources differ from
    the ones the capture was stamped with (`bench.py --stamp-counts`, run when the CSVs are committed).
    None when there is no capture for this config / voxel model."""
    import csv
    path = COUNTS_CSV % config_index
    if algo != "SF" or not os.path.exists(path):
        return None
    rows = [l for l in open(path) if l.startswith('"')]
    launches = {}
    for r in csv.DictReader(rows):
        k = launches.setdefault(int(r["ID"]), {"kernel": r["Kernel Name"]})
        k[r["Metric Name"]] = float(r["Metric Value"].replace(",", ""))
    ops = {"ct_fp_sf": ("fp_band", "transpose"), "ct_bp_sf": ("bp_brick", "bp_pixel")}
    out = {}
    for op, tags in ops.items():
        ks = [k for k in launches.values() if any(t in k["kernel"] for t in tags)]
        if not ks:
            continue
        tot = lambda m: sum(k.get(m, 0.0) for k in ks)
        ns = tot("gpu__time_duration.sum")
        wavg = lambda m: (sum(k[m] * k["gpu__time_duration.sum"] for k in ks) / ns) if ns and all(m in k for k in ks) else None
        t = lambda o: tot("smsp__sass_thread_inst_executed_op_%s_pred_on.sum" % o)
        flops = t("fadd") + t("fmul") + 2.0 * t("ffma") + 2.0 * (t("fadd2") + t("fmul2")) + 4.0 * t("ffma2")
        wf = tot("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum")
        out[op] = {
            "launches": len(ks), "ncu_ms": ns / 1e6,
            "flop_per_update": flops / n_updates,
            "packed_share_of_flops": (2.0 * (t("fadd2") + t("fmul2")) + 4.0 * t("ffma2")) / flops if flops else None,
            "thread_inst_per_update": tot("smsp__thread_inst_executed.sum") / n_updates,
            "dram_bytes": tot("dram__bytes_read.sum") + tot("dram__bytes_write.sum"),
            "dram_read_bytes": tot("dram__bytes_read.sum"), "dram_write_bytes": tot("dram__bytes_write.sum"),
            "shared_replay_share": tot("l1tex__data_bank_conflicts_pipe_lsu_mem_shared.sum") / wf if wf else None,
            "issue_active_pct": wavg("smsp__issue_active.avg.pct_of_peak_sustained_active"),
            "l2_hit_rate_pct": wavg("lts__t_sector_hit_rate.pct"),
            "l2_throughput_pct_of_peak": wavg("lts__t_sectors.avg.pct_of_peak_sustained_elapsed"),
            "shared_pipe_pct_of_peak": wavg("l1tex__data_pipe_lsu_wavefronts_mem_shared.avg.pct_of_peak_sustained_elapsed"),
            "src": os.path.relpath(path, ROOT),
        }
    try:
        stamp = json.load(open(COUNTS_STAMP))
    except Exception:
        stamp = {}
    out["_stamp"] = stamp
    out["_stale"] = stamp.get("csrc_sha256") != csrc_sha256()
    return out


class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(", ") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        sm, reasons = [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0]))
                out["sm_max_mhz"] = float(r[1])
                for n, val in zip(names, r[3:7]):
                    if val.strip().lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        if sm:
            busy = sorted(sm)[len(sm) // 2:]          # upper half = samples under load
            out["sm_mhz"] = float(np.median(busy))
            out["samples"] = len(sm)
        out["reasons"] = sorted(reasons)
        return out


def cpu_baseline(c, x, budget_views=12, n_vox=1 << 20):
    """The oracle as it stands, on the host cores, on a bounded sample of the same workload."""
    from oracle.sf_oracle import Oracle
    o = Oracle(W.geom_keys(c))
    rng = np.random.default_rng(7)
    views = np.sort(rng.choice(c["n_views"], size=min(budget_views, c["n_views"]), replace=False))
    t0 = time.perf_counter()
    y = o.fp(x[0], views)
    t_fp = time.perf_counter() - t0
    up_fp = float(c["nx"]) * c["ny"] * c["nz"] * len(views)
    # A^T on sampled voxels over all views, against a synthetic projection set of the right shape
    yfull = np.broadcast_to(y[0].astype(np.float32), (c["n_views"], c["nv"], c["nu"]))
    ijk = np.stack([rng.integers(0, c["nx"], n_vox), rng.integers(0, c["ny"], n_vox),
                    rng.integers(0, c["nz"], n_vox)], axis=1)
    yfull = np.ascontiguousarray(yfull)
    t0 = time.perf_counter()
    o.bp_voxels(yfull, ijk)
    t_bp = time.perf_counter() - t0
    up_bp = float(n_vox) * c["n_views"]
    live = o.live_fraction(16, 8)
    return {"value": (up_fp + up_bp) / (t_fp + t_bp) / 1e9, "unit": "GUPS", "cores": o.threads or o.num_threads(),
            "kind": "oracle",
            "sample": "A on %d of %d views (%.1f s) + A^T on %d random voxels x all views (%.1f s)"
                      % (len(views), c["n_views"], t_fp, n_vox, t_bp),
            "fp_gups": up_fp / t_fp / 1e9, "bp_gups": up_bp / t_bp / 1e9, "live_fraction": live}


def run_reference(args, c):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    x = W.make_phantom(c)
    times, cb = [], None
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        cb = cpu_baseline(c, x, budget_views=2, n_vox=1 << 16)
        if i >= args.warmup:
            times.append(time.perf_counter() - t0)
    val = cb["value"]
    line = {"impl": "reference", "metric": metric_name(c["index"]), "value": val, "unit": "GUPS", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(times)),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": c["name"], "note": "float64 CPU oracle on a bounded sample per step"},
            "cpu_baseline": cb,
            "e2e": {"value": val, "unit": "GUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--impl", default="ctsf")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--stamp-counts", action="store_true",
                    help="write profiles/r3_counts_stamp.json (hash of csrc/ the committed ncu counts belong to) and exit")
    ap.add_argument("--print-counts-metrics", action="store_true", help="print the ncu --metrics list of the counts capture")
    ap.add_argument("--algo", default="SF", choices=["SF", "DD", "SF-TT"],
                    help="voxel model: SF (separable footprint, the headline) or DD (distance-driven, row f4)")
    ap.add_argument("--fbp", action="store_true",
                    help="also time recon mode (row f2): ct_fbp_filter + ct_bp_sf_recon on the step's projections")
    ap.add_argument("--shard", default="replicas", choices=["replicas", "views"],
                    help="N > 1: independent replicas (weak scaling, default) or ONE workload with its views sharded "
                         "over the ranks, A^T followed by one NCCL all-reduce of the volume (strong scaling)")
    ap.add_argument("--view-stride", type=int, default=1,
                    help="profiling aid: use every S-th view only (ordered subset); not a bench value")
    args = ap.parse_args()
    c = W.make_config(args.config)
    if args.impl == "reference":
        return run_reference(args, c)
    if args.print_counts_metrics:
        print(COUNTS_METRICS)
        return
    if args.stamp_counts:
        # run HERE (in the repository, no GPU needed) when profiles/r3_counts_config*.csv are committed
        head = subprocess.run(["git", "-C", ROOT, "rev-parse", "--short=12", "HEAD"], capture_output=True, text=True)
        stamp = {"csrc_sha256": csrc_sha256(), "git_head_at_capture": head.stdout.strip() or None,
                 "files": sorted(f for f in os.listdir(os.path.join(ROOT, "profiles")) if f.startswith("r3_counts_config"))}
        json.dump(stamp, open(COUNTS_STAMP, "w"), indent=1)
        print(json.dumps(stamp))
        return

    import torch
    import torch.distributed as dist
    from paper_2503_16741_b200 import binding as B
    from paper_2503_16741_b200.projector import Geometry

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    B.debug_set("reset")                               # the library's testing switches: every one at its default
    g = dict(W.geom_keys(c), algo=args.algo)
    x_host = W.make_phantom(c)                         # [B, nz, ny, nx] fp32, seeded
    batch = c["batch"]
    geom = Geometry(g)
    x = torch.from_numpy(x_host).cuda()
    vs = max(1, args.view_stride)
    n_sel = (c["n_views"] + vs - 1) // vs
    sel = None if vs == 1 else (0, vs, n_sel)
    if vs > 1:
        args.no_e2e = True
    shard_views = args.shard == "views"
    if shard_views:
        from paper_2503_16741_b200.geometry import shard_views as shard_of
        sel = shard_of(c["n_views"], world, rank)       # this rank's contiguous block of views
        n_sel = sel[2]
        args.no_e2e = True
    y = torch.empty((batch, n_sel, c["nv"], c["nu"]), device="cuda", dtype=torch.float32)
    xb = torch.empty_like(x)
    stream = torch.cuda.current_stream()
    updates = float(W.n_updates(c)) * n_sel / c["n_views"]
    # measured fp32 peak (FMA-only kernel), before the timed region, with the clock it ran at
    peak_sampler = ClockSampler(local) if rank == 0 else None
    peak_flops = [B.ct_measure_fp32_peak(k, stream.cuda_stream)[0] for k in (0, 1, 0, 1)]
    peak_clocks = peak_sampler.stop() if peak_sampler else None
    peak_scalar, peak_packed = max(peak_flops[0::2]) / 1e12, max(peak_flops[1::2]) / 1e12
    mix_ffma2_ffma, mix_ffma2_fmnmx = [B.ct_measure_fp32_peak(k, stream.cuda_stream)[0] / 1e12 for k in (2, 3)]

    def step():
        geom.fp(x, views=sel, out=y)
        n1 = geom.last_launch_count()
        geom.bp(y, views=sel, out=xb)
        if shard_views and world > 1:
            dist.all_reduce(xb)                      # the path's one exchange step
        return n1 + geom.last_launch_count()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(3 * args.steps + 1)]
    sampler = ClockSampler(local) if rank == 0 else None
    launches = 0
    barrier()
    ev[0].record(stream)
    for i in range(args.steps):
        geom.fp(x, views=sel, out=y)
        launches += geom.last_launch_count()
        ev[3 * i + 1].record(stream)
        geom.bp(y, views=sel, out=xb)
        launches += geom.last_launch_count()
        ev[3 * i + 2].record(stream)
        if shard_views and world > 1:
            dist.all_reduce(xb)                      # NCCL, on the current stream
        ev[3 * i + 3].record(stream)
    barrier()
    clocks = sampler.stop() if sampler else None
    total_ms = ev[0].elapsed_time(ev[3 * args.steps])
    fp_ms = float(np.mean([ev[3 * i].elapsed_time(ev[3 * i + 1]) for i in range(args.steps)]))
    bp_ms = float(np.mean([ev[3 * i + 1].elapsed_time(ev[3 * i + 2]) for i in range(args.steps)]))
    t = torch.tensor([total_ms], device="cuda", dtype=torch.float64)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms = t.item()
    ms_per_step = total_ms / args.steps
    ar_ms = float(np.mean([ev[3 * i + 2].elapsed_time(ev[3 * i + 3]) for i in range(args.steps)]))
    if shard_views:
        # one workload over all ranks: whole-job updates / max-over-ranks time
        value = 2.0 * float(W.n_updates(c)) / (ms_per_step * 1e-3) / 1e9
        per_rank = torch.tensor([fp_ms, bp_ms, ar_ms], device="cuda", dtype=torch.float64)
        gathered = [torch.zeros_like(per_rank) for _ in range(world)]
        if world > 1:
            dist.all_gather(gathered, per_rank)
        else:
            gathered = [per_rank]
        per_rank_ms = [[round(v, 3) for v in t.tolist()] for t in gathered]
    else:
        value = world * 2.0 * updates / (ms_per_step * 1e-3) / 1e9

    # ---- recon mode (row f2), reported beside the headline, never part of it -------------------------------
    recon = None
    if args.fbp:
        q = torch.empty_like(y)
        for _ in range(2):
            geom.fbp_filter(y, views=sel, out=q)
            geom.bp_recon(q, views=sel, out=xb)
        barrier()
        e = [torch.cuda.Event(enable_timing=True) for _ in range(2 * args.steps + 1)]
        e[0].record(stream)
        for i in range(args.steps):
            geom.fbp_filter(y, views=sel, out=q)
            e[2 * i + 1].record(stream)
            geom.bp_recon(q, views=sel, out=xb)
            e[2 * i + 2].record(stream)
        barrier()
        f_ms = float(np.mean([e[2 * i].elapsed_time(e[2 * i + 1]) for i in range(args.steps)]))
        r_ms = float(np.mean([e[2 * i + 1].elapsed_time(e[2 * i + 2]) for i in range(args.steps)]))
        taps = float(y.numel()) * c["nu"] / 2.0                      # fp64 multiply-adds of the ramp filter
        recon = {"filter_ms": f_ms, "bp_recon_ms": r_ms, "bp_recon_gups": updates / (r_ms * 1e-3) / 1e9,
                 "filter_fp64_tflops": 2.0 * taps / (f_ms * 1e-3) / 1e12,
                 "fbp_gups": updates / ((f_ms + r_ms) * 1e-3) / 1e9}
        del q

    # ---- end to end through the host-buffer entry points (pinned memory) -----------------------------
    e2e = None
    if not args.no_e2e:
        hx = torch.from_numpy(x_host).pin_memory()
        hy = torch.empty(y.shape, dtype=torch.float32).pin_memory()
        hxb = torch.empty(x.shape, dtype=torch.float32).pin_memory()
        s = stream.cuda_stream

        def e2e_step():
            B.ct_fp_sf_host(geom.handle, hx.data_ptr(), hy.data_ptr(), batch, s)
            B.ct_bp_sf_host(geom.handle, hy.data_ptr(), hxb.data_ptr(), batch, s)
        e2e_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(max(1, args.steps)):
            e2e_step()
        barrier()
        dt = torch.tensor([time.perf_counter() - t0], device="cuda", dtype=torch.float64)
        if world > 1:
            dist.all_reduce(dt, op=dist.ReduceOp.MAX)
        e2e_ms = dt.item() * 1e3 / max(1, args.steps)
        nbytes = 4 * (x.numel() + y.numel())
        e2e = {"value": world * 2.0 * updates / (e2e_ms * 1e-3) / 1e9, "unit": "GUPS", "ms_per_step": e2e_ms,
               "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
               "api": "ct_fp_sf_host + ct_bp_sf_host, pinned host buffers"}
        del hx, hy, hxb

    if rank == 0:
        pk = peaks()
        flop = FLOP_PER_UPDATE[args.config] * updates
        alg_bytes = 4.0 * (x.numel() + y.numel())
        dom, dom_ms = ("ct_fp_sf", fp_ms) if fp_ms >= bp_ms else ("ct_bp_sf", bp_ms)
        mc = (measured_counts(args.config, args.algo, float(W.n_updates(c))) if vs == 1 and not shard_views else None) or {}
        mdom = mc.get(dom, {})
        traffic = mdom.get("dram_bytes") if vs == 1 and not shard_views else None
        achieved = flop / (dom_ms * 1e-3) / 1e12
        peak = max(peak_scalar, peak_packed)
        line = {
            "metric": metric_name(args.config), "value": value, "unit": "GUPS", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "strong" if shard_views else "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": c["name"], "algo": args.algo, "index": args.config, "volume": [c["nz"], c["ny"], c["nx"]],
                       "views": n_sel, "detector": [c["nv"], c["nu"]], "batch": batch,
                       "step": "1 x ct_fp_sf + 1 x ct_bp_sf" + (" + all-reduce(volume)" if shard_views else ""),
                       "updates_per_operator": updates,
                       "l2": "inputs (%.0f MB) exceed the 126 MB L2; no flush" % (alg_bytes / 1e6)
                             if alg_bytes > 126e6 else
                             "inputs (%.1f MB) fit the 126 MB L2 and stay there between steps; no flush (small "
                             "parity-test config, not the headline)" % (alg_bytes / 1e6),
                       "parallelism": ("views sharded over %d ranks + 1 all-reduce" % world) if shard_views
                                      else ("replicas" if world > 1 else "single")},
            "fp_ms": fp_ms, "bp_ms": bp_ms,
            "fp_gups": updates / (fp_ms * 1e-3) / 1e9, "bp_gups": updates / (bp_ms * 1e-3) / 1e9,
            "gpu_launches": launches, "clocks": clocks, "e2e": e2e, "recon": recon,
            "debug_switches": B.debug_state(),       # testing switches off their defaults after the run: {} expected
            "roofline": {"bound": "alu", "kernel": dom, "achieved": achieved, "peak": peak,
                         "unit": "TFLOP/s", "frac": achieved / peak, "traffic": traffic,
                         "peak_src": "measured in this run by ct_measure_fp32_peak (FMA-only kernel, best of 2 x 3): "
                                     "scalar FFMA %.2f, packed FFMA2 %.2f TFLOP/s at %s MHz; nominal 148 SM x 128 lanes x "
                                     "2 x %.0f MHz = %.2f" % (peak_scalar, peak_packed,
                                                              peak_clocks.get("sm_mhz") if peak_clocks else "?",
                                                              pk["sm_max_mhz"], pk["fp32_tflops_nominal"]),
                         "peak_scalar_ffma": peak_scalar, "peak_packed_ffma2": peak_packed,
                         "mix_ffma2_with_ffma_tflops": mix_ffma2_ffma, "mix_ffma2_with_fmnmx_tflops": mix_ffma2_fmnmx,
                         "flop_per_update": FLOP_PER_UPDATE[args.config],
                         "flop_per_update_src": "algorithmic count of S1-S5 per nominal update (DESIGN.md section 7)",
                         "executed_flop_per_update": mdom.get("flop_per_update"),
                         "executed_frac": (mdom["flop_per_update"] * updates / (dom_ms * 1e-3) / 1e12 / peak)
                                          if mdom.get("flop_per_update") else None,
                         "issue_slots_busy_pct": mdom.get("issue_active_pct"),
                         "l2_hit_rate_pct": mdom.get("l2_hit_rate_pct"),
                         "l2_throughput_pct_of_peak": mdom.get("l2_throughput_pct_of_peak"),
                         "shared_pipe_pct_of_peak": mdom.get("shared_pipe_pct_of_peak"),
                         "shared_replay_share": mdom.get("shared_replay_share"),
                         "measured_counts_src": mdom.get("src"),
                         "counts_stale": mc.get("_stale"), "counts_stamp": mc.get("_stamp"),
                         "hbm": {"algorithmic_bytes": alg_bytes, "achieved_gbs": alg_bytes / (dom_ms * 1e-3) / 1e9,
                                 "peak_gbs": pk["hbm_gbs"], "frac": alg_bytes / (dom_ms * 1e-3) / 1e9 / pk["hbm_gbs"],
                                 "note": "algorithmic bytes / kernel time; the path is ALU-bound by >200x "
                                         "(DESIGN.md), so this fraction is small by construction"}},
        }
        if shard_views:
            line["shard"] = {"mode": "views", "per_rank_ms_fp_bp_allreduce": per_rank_ms}
        if world == 1 and not args.no_cpu:
            line["cpu_baseline"] = cpu_baseline(c, x_host)
            lf = line["cpu_baseline"]["live_fraction"]
            line["live_fraction"] = lf
            line["live_gups"] = value * lf
        print(json.dumps(line))
    geom.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
