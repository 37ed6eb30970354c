#!/usr/bin/env python
"""bench.py -- sn-K build benchmark (BASELINE.json metric: "sn-K build wall-time and integrals/s at 1 B200;
fraction of FP64 peak").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

One "step" = one pass of the whole hot path (rows a2-a7 of DESIGN.md plus the density-dependent screening a3;
a0/a1 are per-geometry and reported as ``set_grid_ms``) over the synthetic workload: one ``snk_build_K``.
``value``  = contracted 3c-CP integrals evaluated per second (whole job), inputs resident in HBM.
``e2e``    = the same through ``snk_build_K_host`` (HOST P in, HOST K out; H2D/D2H inside the timed region).
``roofline``: dominant integral-contraction kernel (bound "alu": plain FP64 DFMA pipe) -- algorithmic flops of its
launch (DESIGN.md flop model) / its CUDA-event duration inside the timed region / measured DFMA peak of this GPU.
``cpu_baseline``: the oracle, as it stands, on the host cores, on a bounded, spatially compact sample (whole root cells of
R13 when the budget covers them, else a Morton-order prefix of the first ones); ``--impl reference`` times that same sample.

N > 1 (torchrun): by default every rank builds K for its own density on the whole grid (independent problems, no collective:
weak scaling).  ``--multi shard``: one screening pass gives the primitive pair-points of every batch, root cells are dealt to
ranks by Alg. 2 on them (greedy LPT), every rank builds its partial K and one NCCL all-reduce (Alg. 1 line
13) sums them -- strong scaling of one build.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "sn-K build: contracted 3c-CP integrals per second (snk_build_K wall time also reported as ms_per_step)"
UNIT = "integrals/s"


def _workload_name(cfg, w):
    return "cfg%d %s: %d atoms, %d shells, %d functions, grid %s = %d points, eps=%g" % (
        cfg, w.name, len(w.atoms_z), w.basis.nshells, w.basis.nbf, "x".join(map(str, w.grid_shape)), w.points.shape[0], w.eps)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows = []
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.p = None

    def _read(self):
        for line in self.p.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        sm, mx, reasons = [], [], set()
        for (t, line) in self.rows:
            if t < t0 or t > t1 + 0.2:
                continue
            f = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except Exception:
                continue
            for name, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples in timed region"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons), "samples": len(sm)}


def _morton_order(pts, h0):
    """Order of the points along a Morton (Z-order) curve inside their root cells: a prefix of it is a spatially compact piece of
    the grid, which the oracle's octree turns into batches of the usual size and shape."""
    cell = np.floor(pts / h0)
    q = np.clip(((pts / h0 - cell) * 1024.0).astype(np.int64), 0, 1023)
    key = np.zeros(len(pts), dtype=np.int64)
    for b in range(10):
        for ax in range(3):
            key |= ((q[:, ax] >> b) & 1) << (3 * b + ax)
    ck = (cell[:, 0].astype(np.int64) + (1 << 15)) << 32 | (cell[:, 1].astype(np.int64) + (1 << 15)) << 16 | (cell[:, 2].astype(np.int64) + (1 << 15))
    return np.lexsort((key, ck))


def time_oracle_sample(w, target_s=15.0, first_frac=0.01, return_idx=False):
    """Oracle (as it stands) on a bounded sample sized for ~target_s of host time.  Whole root cells in R13 hash order when the
    budget covers at least the first of them (they hold 5e4-1e5 points each in configs 3-5); otherwise a spatially compact part
    of the first root cells (a Morton-order prefix: whole octree leaves, i.e. batches of the usual size), never scattered
    points -- a batch with a handful of points pays the whole per-batch screening and would make the oracle look 10x slower."""
    from oracle import oracle as orc
    from paper_2303_14280_b200.dist import root_cell_sample
    o = orc.Oracle(w.basis)
    npts = w.points.shape[0]

    def run(idx):
        o.set_grid(w.points[idx], w.weights[idx], eps=w.eps, batch_cell=w.batch_cell, batch_max=w.batch_max)
        t = time.time()
        o.build_K(w.P)
        return time.time() - t, o.stats()

    cells = np.nonzero(root_cell_sample(w.points, w.batch_cell, first_frac))[0] if first_frac < 1.0 else np.arange(npts)
    cells = cells[_morton_order(w.points[cells], w.batch_cell)]
    nprobe = min(len(cells), 256)
    dt0, _ = run(cells[:nprobe])
    want = int(target_s * nprobe / max(dt0, 1e-4))                # points the oracle can do in target_s
    if want >= len(cells):
        how = "whole root cells (R13 hash order)"
        frac = min(1.0, first_frac * want / len(cells))
        idx = np.nonzero(root_cell_sample(w.points, w.batch_cell, frac))[0] if frac < 1.0 else np.arange(npts)
        if len(idx) > 1.3 * want:                                 # the next whole cell overshoots the budget: stay with the first ones
            idx = cells
    else:
        how = "spatially compact part (Morton-order prefix, whole octree leaves) of the first root cells (R13 hash order)"
        idx = cells[:max(want, nprobe)]
    dt, st = run(idx)
    if dt < 0.5 * target_s and len(idx) < npts:                   # the probe's rate was pessimistic: one more pass
        want = int(len(idx) * target_s / max(dt, 1e-3))
        if how.startswith("whole"):
            frac = min(1.0, want / npts)
            idx2 = np.nonzero(root_cell_sample(w.points, w.batch_cell, frac))[0] if frac < 1.0 else np.arange(npts)
        else:
            idx2 = cells[:min(want, len(cells))]
        if len(idx2) > len(idx) and len(idx2) <= 1.5 * want:
            idx = idx2
            dt, st = run(idx)
    extra = {"idx": idx} if return_idx else {}
    nb = len(o.batches()[0]) - 1
    used = int(min(st["threads"], max(nb, 1)))                    # the oracle is parallel over batches: threads that had work
    return dict(extra, value=st["n_int_contracted"] / dt, unit=UNIT, cores=used, kind="oracle",
                sample="%s: %d of %d points (%.3f%%) in %d batches on %d OpenMP threads (parallel over batches: %d had work), "
                       "%.3g contracted integrals, %.2f s; oracle = C++ -O2 -fopenmp McMurchie-Davidson, untuned"
                       % (how, len(idx), npts, 100.0 * len(idx) / npts, nb, st["threads"], used, st["n_int_contracted"], dt),
                seconds=dt, n_int=st["n_int_contracted"])


def oracle_sample_for(w, args):
    """The ONE oracle sample both arms time (the driver passes the same --steps / --warmup to both): sized for a per-step
    budget such that the reference arm's whole run ends within minutes (about 1000 s of oracle time at most), cut back along
    the Morton curve when the sizing pass overshot it.  Returns (point indices, how it was chosen)."""
    budget = min(args.cpu_seconds, 1000.0 / (args.steps + args.warmup + 3))
    first = time_oracle_sample(w, target_s=budget, return_idx=True)
    idx = first.pop("idx")
    if first["seconds"] > 1.25 * budget and first["sample"].startswith("spatially"):
        # the cost per point grows along the Morton curve (towards the nuclei): cut the prefix back to the budget
        idx = idx[:max(256, int(len(idx) * budget / first["seconds"]))]
    return idx, first["sample"].split(":")[0]


def time_oracle_on(w, idx, how, nrep=1, nwarm=0):
    """The oracle's K build on the points idx, nwarm untimed + nrep timed builds -> (rate, seconds per build, cores, sample line)."""
    from oracle import oracle as orc
    o = orc.Oracle(w.basis)
    o.set_grid(w.points[idx], w.weights[idx], eps=w.eps, batch_cell=w.batch_cell, batch_max=w.batch_max)
    res = []
    for i in range(nwarm + nrep):
        t = time.time()
        o.build_K(w.P)
        dt = time.time() - t
        if i >= nwarm:
            res.append(dt)
    st = o.stats()
    n_int = st["n_int_contracted"]
    nb = len(o.batches()[0]) - 1
    used = int(min(st["threads"], max(nb, 1)))
    npts = w.points.shape[0]
    sample = ("%s: %d of %d points (%.3f%%) in %d batches on %d OpenMP threads (parallel over batches: %d had work), %.3g contracted "
              "integrals per build, %.1f s per build; oracle = C++ -O2 -fopenmp McMurchie-Davidson, untuned"
              % (how, len(idx), npts, 100.0 * len(idx) / npts, nb, st["threads"], used, n_int, sum(res) / len(res)))
    return n_int * len(res) / sum(res), sum(res) / len(res), used, sample


def run_reference(args, rank, world):
    """--impl reference: the oracle on the host cores, same config/metric.  Both arms call oracle_sample_for with the same
    flags, so the sample timed here step by step is the one the GPU arm's `cpu_baseline` leg times once; the grid is generated
    on the same device as in the GPU arm (same points and weights)."""
    if rank != 0:
        return
    from paper_2303_14280_b200 import inputs
    w = inputs.make_workload(args.config, grid=args.grid, device=_gen_device(), density=args.density)
    idx, how = oracle_sample_for(w, args)
    val, per_build, used, sample = time_oracle_on(w, idx, how, nrep=args.steps, nwarm=args.warmup)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * per_build, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": _workload_name(args.config, w), "sample": sample, "density": args.density, "batch_cell": w.batch_cell, "batch_max": w.batch_max},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": used, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def _ncu_traffic(cfg, cls_name):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed `ncu --set full`
    summary of this same workload (newest profiles/*_ncu_full_cfg<cfg>.csv); None when no capture of it is committed."""
    import csv
    import glob
    la_lb = {"ss": "0, 0", "ps": "1, 0", "pp": "1, 1", "ds": "2, 0", "dp": "2, 1", "dd": "2, 2", "fs": "3, 0", "fp": "3, 1",
             "fd": "3, 2", "ff": "3, 3"}[cls_name]
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "*_ncu_full_cfg%d.csv" % cfg)), reverse=True):
        try:
            with open(path, newline="") as f:
                rows = list(csv.reader(f))
            hdr = rows[0]
            col = {h.split("[")[0]: (i, (h.split("[")[1][:-1] if "[" in h else "")) for i, h in enumerate(hdr)}
            for r in rows[1:]:
                if "k_integrals<%s>" % la_lb in r[col["kernel"][0]]:
                    v = sum(float(r[col[k][0]]) * scale.get(col[k][1], 1.0) for k in ("dram_read", "dram_write"))
                    return v if v == v else None          # ncu left the section empty for this launch
        except Exception:
            continue
    return None


def _gen_device():
    try:
        import torch
        return "cuda" if torch.cuda.is_available() else "cpu"
    except Exception:
        return "cpu"


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3,
                    help="BASELINE.json config 1..5; default 3 (64 waters, 1 600 functions, 3.9 M points): the largest configuration whose "
                         "build (about 1.5 s) lets the driver's warm-up + timed steps and the e2e leg finish within minutes; config 4 "
                         "(1 029 atoms) takes minutes per build and is run with --config 4 --steps 1")
    ap.add_argument("--grid", type=lambda s: tuple(int(x) for x in s.split(",")), default=None, help="override n_r,n_theta,n_phi")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--density", default="dense", choices=["dense", "decay"],
                    help="'dense' = BASELINE.json's P = C C^T with Gaussian C (no spatial decay: V_j keeps every significant pair); "
                         "'decay' = localised random orbitals, |P| ~ exp(-r / 1.5 bohr) (SURVEY.md section 8(f)-2: sn-LinK deletes work)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=25.0, help="host time the oracle sample of cpu_baseline / --impl reference is sized for")
    ap.add_argument("--workspace-gb", type=float, default=None)
    ap.add_argument("--tile-split", type=int, default=0, help="CTAs per tile in the integral kernel (0 = the library's choice)")
    ap.add_argument("--multi", default="replicas", choices=["replicas", "shard"],
                    help="N>1: 'replicas' = every rank builds K for its own density (independent problems, no collective, weak scaling); "
                         "'shard' = root cells dealt to ranks + NCCL all-reduce of K (Alg. 1/2, strong scaling)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_2303_14280_b200 import inputs, snk
    from paper_2303_14280_b200.dist import all_reduce_K, shard_points

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    snk.load()

    # ---- synthetic workload (seeded, DESIGN.md recipe); the grid generator runs on the GPU for speed ----
    w = inputs.make_workload(args.config, grid=args.grid, device=str(dev), density=args.density)
    shard = world > 1 and args.multi == "shard"
    mine = np.ones(w.points.shape[0], dtype=bool)
    if world > 1 and not shard:       # independent problem per rank: its own density matrix, same molecule and grid
        rng = np.random.Generator(np.random.PCG64(inputs.SEED_BASE + 1000 * rank + args.config))
        C = rng.standard_normal((w.basis.nbf, max(1, w.basis.nbf // 5))) / np.sqrt(max(1, w.basis.nbf // 5))
        w.P = 0.5 * (C @ C.T + (C @ C.T).T)
    pts = torch.as_tensor(np.ascontiguousarray(w.points[mine]), device=dev)
    wts = torch.as_tensor(np.ascontiguousarray(w.weights[mine]), device=dev)
    P = torch.as_tensor(w.P, device=dev)
    K = torch.empty_like(P)
    s = snk.Snk(w.basis)
    s.set_option("eps", w.eps); s.set_option("batch_cell", w.batch_cell); s.set_option("batch_max", w.batch_max)
    if args.workspace_gb:
        s.set_option("workspace_gb", args.workspace_gb)
    if args.tile_split:
        s.set_option("tile_split", args.tile_split)
    dfma_peak, dmma_peak = snk.measure_fp64_peak(5)
    if shard:
        # Alg. 2 on the library's own work model: one screening pass over the whole grid gives the primitive
        # pair-points of every batch; root cells are dealt to ranks by greedy LPT on them (replicated, deterministic)
        from paper_2303_14280_b200.dist import root_cell_costs
        s.set_grid(pts, wts)
        s.screen(P)
        L = s.export_lists(want_V=False)
        cells = root_cell_costs(w.points, w.batch_cell, L["batch_off"], L["perm"], s.batch_costs())
        mine = shard_points(w.points, w.batch_cell, rank, world, cell_costs=cells)
        pts = torch.as_tensor(np.ascontiguousarray(w.points[mine]), device=dev)
        wts = torch.as_tensor(np.ascontiguousarray(w.weights[mine]), device=dev)
    s.set_grid(pts, wts)
    set_grid_ms = s.stats()["ms_set_grid"]

    def step():
        s.build_K(P, K)
        if shard:
            all_reduce_K(K)             # Alg. 1 line 13

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.cudart().cudaProfilerStart()      # `ncu --profile-from-start off` then sees exactly the timed region
    t0 = time.time()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    t1 = time.time()
    torch.cuda.cudart().cudaProfilerStop()
    ms = e0.elapsed_time(e1)
    st = s.stats()            # per-stage CUDA-event times of the LAST timed step (recorded inside the timed region)
    clocks = sampler.stop(t0, t1) if sampler else None

    # ---- e2e: host P -> host K through snk_build_K_host ----
    Ph = torch.as_tensor(w.P).pin_memory()
    Kh = torch.empty_like(Ph).pin_memory()
    s.build_K_host(Ph, Kh)
    barrier()
    te0 = time.time()
    for _ in range(args.steps):
        if world == 1:
            s.build_K_host(Ph, Kh)
        else:
            P.copy_(Ph, non_blocking=True)
            step()
            Kh.copy_(K, non_blocking=True)
            torch.cuda.synchronize(dev)
    barrier()
    e2e_s = time.time() - te0

    # ---- aggregate over ranks: max time, sum of work ----
    n_int = st["n_int_contracted"]
    agg = torch.tensor([ms, e2e_s, n_int, st["n_int_primitive"], st["n_pairpoints"], float(st["n_launches"])], dtype=torch.float64, device=dev)
    if world > 1:
        mx = agg.clone(); dist.all_reduce(mx, op=dist.ReduceOp.MAX)
        sm = agg.clone(); dist.all_reduce(sm, op=dist.ReduceOp.SUM)
        ms, e2e_s = float(mx[0]), float(mx[1])
        n_int, n_prim, n_pp, n_launch = float(sm[2]), float(sm[3]), float(sm[4]), float(sm[5])
    else:
        n_prim, n_pp, n_launch = st["n_int_primitive"], st["n_pairpoints"], float(st["n_launches"])
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    value = n_int * args.steps / (ms * 1e-3)
    nbytes = w.P.nbytes
    # dominant integral kernel of the last timed step
    cls = int(np.argmax(st["ms_G_class"]))
    k_ms = st["ms_G_class"][cls]
    k_flops = st["flops_class"][cls]
    achieved = k_flops / (k_ms * 1e-3) * 1e-12 if k_ms > 0 else 0.0
    all_ms = sum(st["ms_G_class"])
    roofline = {"bound": "alu", "kernel": "k_integrals<%s>" % snk.CLASS_NAMES[cls], "achieved": achieved, "peak": dfma_peak, "unit": "TFLOP/s",
                "frac": achieved / dfma_peak if dfma_peak else None, "traffic": _ncu_traffic(args.config, snk.CLASS_NAMES[cls]),
                "peak_source": "measured on this GPU by snk_measure_fp64_peak (register-resident DFMA loop); nominal 148 SM x 64 DFMA/clk x 2 x 1.965 GHz = 37.2",
                "launches_per_step": int(st["nsuper"]),     # one launch of every class per super-batch
                "flops_per_launch": k_flops / max(1, st["nsuper"]), "ms_per_launch": k_ms / max(1, st["nsuper"]),
                "traffic_note": "dram bytes read + written by the first of these launches in profiles/*_ncu_full_cfg<N>.csv (ncu --set full)",
                "all_integral_kernels": {"achieved": st["flops_integral"] / (all_ms * 1e-3) * 1e-12 if all_ms > 0 else 0.0, "ms": all_ms,
                                         "flops": st["flops_integral"], "share_of_step": all_ms / st["ms_build"] if st["ms_build"] else None},
                "gemm_dmma": {"peak": dmma_peak, "achieved": st["flops_gemm"] / ((st["ms_F"] + st["ms_Kt"] + 1e-12) * 1e-3) * 1e-12,
                              "achieved_algorithmic": st["flops_gemm_alg"] / ((st["ms_F"] + st["ms_Kt"] + 1e-12) * 1e-3) * 1e-12,
                              "flops_executed": st["flops_gemm"], "flops_algorithmic": st["flops_gemm_alg"],
                              "note": "executed = row lists of the chunks padded to the 16 / 32 wide tiles (plus the small screening GEMM); "
                                      "algorithmic = 2 |Q_j| nbf(B_j) nbf per batch for a4 and for a6 (Eq. 48 operand sizes)",
                              "ms_F": st["ms_F"], "ms_Kt": st["ms_Kt"]},
                "per_class": {snk.CLASS_NAMES[c]: {"ms": st["ms_G_class"][c], "achieved": st["flops_class"][c] / (st["ms_G_class"][c] * 1e-3) * 1e-12,
                                                   "frac": st["flops_class"][c] / (st["ms_G_class"][c] * 1e-3) * 1e-12 / dfma_peak if dfma_peak else None}
                              for c in range(len(snk.CLASS_NAMES)) if st["ms_G_class"][c] > 0},
                "flop_model": "far-field (asymptotic Boys) instruction count of the kernel templates, FMA = 2 (DESIGN.md)"}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong" if shard else "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": _workload_name(args.config, w),
                       "why_this_config": "largest single-GPU configuration of BASELINE.json whose K build (seconds) fits warm-up + timed steps + "
                                          "the e2e leg in minutes; configs[3] (343 waters) costs minutes per build: `--config 4 --steps 1`, "
                                          "summary under profiles/",
                       "l2": "working set (Phi, F, G slabs) far larger than the 126 MB L2; no flush needed",
                       "parallelism": "1 GPU" if world == 1 else ("root cells -> %d ranks by Alg. 2 LPT, NCCL all-reduce of K per build" % world if shard else "%d independent replicas (own density each), no collective" % world),
                       "batch_cell": w.batch_cell, "batch_max": w.batch_max, "density": args.density,
                       "pair_survival": (st["sum_V"] / (st["nbatch"] * st["npair_sig"])) if st["nbatch"] and st["npair_sig"] else None,
                       "n_int_per_step": n_int, "n_int_primitive_per_step": n_prim,
                       "n_pairpoints_per_step": n_pp},
            "clocks": clocks,
            "e2e": {"value": n_int * args.steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
                    "ms_per_step": 1e3 * e2e_s / args.steps},
            "gpu_launches": int(n_launch * args.steps),
            "roofline": roofline,
            "build": {"ms_build_last": st["ms_build"], "ms_screen": st["ms_screen"], "ms_colloc": st["ms_colloc"], "ms_F": st["ms_F"],
                      "ms_G": st["ms_G"], "ms_Kt": st["ms_Kt"], "ms_sym": st["ms_sym"], "ms_G_class": dict(zip(snk.CLASS_NAMES, st["ms_G_class"])),
                      "set_grid_ms": set_grid_ms, "nbatch": st["nbatch"], "npair_sig": st["npair_sig"], "sum_V": st["sum_V"],
                      "nsuper": st["nsuper"], "fp64_peak_tflops": {"dfma": dfma_peak, "dmma": dmma_peak},
                      "whole_build_fp64_frac": (st["flops_integral"] + st["flops_gemm"]) / (st["ms_build"] * 1e-3) * 1e-12 / dfma_peak}}
    if not args.no_cpu_baseline:
        idx, how = oracle_sample_for(w, args)                  # the sample `--impl reference` times with the same flags
        val, _, used, sample = time_oracle_on(w, idx, how, nrep=1, nwarm=1)
        line["cpu_baseline"] = {"value": val, "unit": UNIT, "cores": used, "kind": "oracle", "sample": sample}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
