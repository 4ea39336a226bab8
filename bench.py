#!/usr/bin/env python
"""bench.py -- grid points/s of the full E_xc + V_xc + N_el build (fp64) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c5] [--also c4,c3,c2,c1,u2,g1] [--impl reference]

A step = one pass of the whole hot path (weights -> density -> potential -> scatter/finalise) over one
synthetic water-cluster workload (BASELINE.json:configs; generator: workloads/).  Prints ONE JSON line.
The headline workload is c5 (512 waters, 12800 functions, 46.4 M points, PBE): the largest single-GPU
configuration BASELINE.json names; c4 (256 waters) is measured beside it with the same detail (e2e, both
rooflines, clocks, plan seconds); the other workloads are short side entries.
N > 1 (torchrun): the path is not sharded ("replicas only"): every rank runs the same build on
its own GPU, value = N * points / max-over-ranks device time, scaling = "weak".
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "grid points/s for full E_xc+V_xc build (fp64, 1 B200); % of FP64 roofline"
UNIT = "grid points/s"
FP64_NOMINAL_TFLOPS = 37.2   # 148 SM x 64 FP64 FMA/clk x 2 x 1.965 GHz (datasheet-level; the live measurement below is what is used)
FLOP_PER_PAIR = 15.0         # "(a): plain FP64 ALU ...; ~15 flop per evaluated pair; report pairs/point"

DESCR = {
    "c1": "c1: water monomer, 3 atoms, 25 basis functions, 50x194 grid",
    "c2": "c2: 64-water cluster, 192 atoms, 1600 basis functions, 75x302 grid",
    "c3": "c3: 64-water cluster, 192 atoms, 1600 basis functions, 75x302 grid",
    "c4": "c4: 256-water cluster, 768 atoms, 6400 basis functions, 75x302 grid",
    "c5": "c5: 512-water cluster, 1536 atoms, 12800 basis functions, 100x302 grid",
    "u2": "u2: 64-water cluster on a UFG-shaped 99x590 grid (SURVEY 8(f))",
    "s2": "s2: 64-water cluster, 192 atoms, 1600 basis functions, on an SFG-shaped 175x974 grid (SURVEY 8(f))",
    "g1": "g1: irregular 410-water cluster, 1230 atoms, 10250 basis functions, 75x302 grid (SURVEY 8(f))",
}


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            d = json.load(fh)
        return float(d.get("hbm_gbs", 6650.0)), "measured"
    return 6650.0, "fallback"


def _ncu_traffic(workload, kernel):
    """dram bytes per launch of `kernel` from the committed ncu --set full capture of this round (profiles/), or None."""
    p = os.path.join(ROOT, "profiles", "r02_ncu_traffic.txt")
    try:
        with open(p) as fh:
            return json.load(fh).get(workload, {}).get(kernel)
    except Exception:
        return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.thr, self.index = [], None, None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
                for n, v in zip(names, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}


def _hist(a):
    import numpy as np
    a = np.asarray(a, dtype=float)
    return {"mean": float(a.mean()), "p50": float(np.percentile(a, 50)), "p95": float(np.percentile(a, 95)), "max": float(a.max())}


def config_of(name, w, world):
    """The workload as named in the JSON line: derived from the workload alone, so both arms print the same dict."""
    fn = "PBE" if w.functional == 1 else "Slater+VWN5"
    return {"workload": "%s, %s, SSF partition" % (DESCR.get(name, name), fn), "workload_id": name, "functional": fn,
            "n_points": int(len(w.atoms_Z)) * w.n_rad * w.n_ang, "n_basis": int(w.n_basis), "n_atoms": int(len(w.atoms_Z)),
            "partition": "SSF", "parallelism": "replicas only" if world > 1 else "single GPU",
            "l2": "flushed between timed iterations (256 MB fill)", "seed": 200703143}


def run_workload(name, steps, warmup, peaks, do_e2e=True, device=0, sampler=None):
    """Times `steps` full builds of workload `name` on the current GPU. Returns a dict of measurements."""
    import numpy as np
    import torch

    import paper_2007_03143_b200 as xc
    from workloads import make_workload

    w = make_workload(name)
    fn = w.functional
    t0 = time.perf_counter()
    plan = xc.Plan.from_workload(w, spec=xc.grid_spec(w.n_rad, w.n_ang, fn), device=device)
    plan_s = time.perf_counter() - t0
    P = torch.from_numpy(w.P).cuda()
    V = torch.empty_like(P)
    flush = torch.empty(256 * 1024 * 1024 // 8, dtype=torch.float64, device="cuda")  # > 126 MB L2
    ev0 = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
    ev1 = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
    for _ in range(warmup):
        plan.eval(P, V)
    torch.cuda.synchronize()
    stage = {"weights_ms": 0.0, "pack_ms": 0.0, "batch_ms": 0.0, "finalize_ms": 0.0}
    launches = 0
    E = N = 0.0
    ctx = sampler if sampler is not None else ClockSampler(device)
    with ctx:
        for k in range(steps):
            flush.fill_(float(k))           # L2 flush between timed iterations (untimed)
            ev0[k].record()
            E, N, _ = plan.eval(P, V)
            ev1[k].record()
            tm = plan.timings()
            for key in stage:
                stage[key] += tm[key]
            launches += tm["launches"]
        torch.cuda.synchronize()
    total_ms = sum(a.elapsed_time(b) for a, b in zip(ev0, ev1))
    ms = total_ms / steps
    for key in stage:
        stage[key] /= steps
    # cached-weights build (reading A16), reported next to the full build
    t_c = []
    for k in range(min(steps, 5)):
        flush.fill_(1.0)
        plan.eval(P, V, reuse_weights=True)
        t_c.append(plan.timings()["total_ms"])
    # one extra, untimed build that counts the pair factors step (a) evaluates (roofline of the weights kernel)
    plan.eval(P, V, count_pairs=True)
    pairs, nontrivial = plan.counters()
    stats = plan.stats()
    res = dict(workload=name, functional="PBE" if fn == 1 else "Slater+VWN5", n_points=plan.n_points, n_basis=plan.n_basis,
               n_atoms=int(len(w.atoms_Z)), n_batches=plan.n_batches, ms_per_step=ms, stage_ms=stage, launches=launches,
               E_xc=E, N_el=N, N_el_rel_err_vs_trPS=abs(N - 2.0 * w.n_occ) / (2.0 * w.n_occ), plan_seconds=plan_s,
               cached_weights_ms=float(np.median(t_c)), stats=stats, clocks=ctx.summary())
    res["points_per_s"] = plan.n_points / (ms * 1e-3)
    res["builds_per_s"] = 1e3 / ms
    ex = plan.export()
    nq = np.diff(ex.batch_off)
    from workloads import nfun
    foff = np.array([nfun(int(c)) for c in w.shell_L], dtype=np.int64)
    csum = np.concatenate([[0], np.cumsum(foff[ex.shells])])
    nbj = csum[ex.shell_off[1:]] - csum[ex.shell_off[:-1]]
    res["nq_hist"] = _hist(nq)
    res["nb_hist"] = _hist(nbj)
    # the contractions only run over points with w != 0 (exact zeros of the partition add nothing): the algorithmic
    # flop count used for every TFLOP/s and roofline figure is the smaller one, 4 (N_b^j)^2 x (live points of batch j)
    wd = plan.diagnostics(want_points=True)["w"]
    live = np.add.reduceat((wd != 0.0).astype(np.int64), ex.batch_off[:-1]) if len(nq) else np.zeros(0, np.int64)
    # GGA: X GEMM 2 N_b^2 + V^j (SYR2K triangle) 2 N_b^2 per point; LDA: X over the lower triangle of P^j N_b^2 + V^j (SYRK
    # triangle) N_b^2 per point
    per_pt = 4.0 if fn == 1 else 2.0
    res["flops_all_points"] = float(plan.algorithmic_flops) * per_pt / 4.0
    res["flops"] = float(np.sum(per_pt * nbj.astype(np.float64) ** 2 * live))
    res["live_point_fraction"] = float(live.sum() / max(1, plan.n_points))
    res["fp64_tflops"] = res["flops"] / (ms * 1e-3) * 1e-12
    res["fp64_frac"] = res["fp64_tflops"] / peaks["fp64"]
    # rooflines of the two kernels that make up a build
    res["roofline_batch"] = {
        "kernel": "k_xc_batch", "bound": "tensor", "achieved": res["flops"] / (stage["batch_ms"] * 1e-3) * 1e-12, "peak": peaks["fp64"],
        "unit": "TFLOP/s", "peak_source": peaks["fp64_src"], "traffic": _ncu_traffic(name, "k_xc_batch"),
        "ms_per_build": stage["batch_ms"], "algorithmic_flops": res["flops"]}
    res["roofline_batch"]["frac"] = res["roofline_batch"]["achieved"] / peaks["fp64"]
    # step (a): plain FP64 ALU work, FLOP_PER_PAIR flop per evaluated pair factor (counted on the device), against the measured DFMA rate
    wflops = FLOP_PER_PAIR * max(pairs, 0)
    res["roofline_weights"] = {
        "kernel": "k_weights_ssf", "bound": "alu", "achieved": wflops / max(stage["weights_ms"], 1e-9) * 1e-9, "peak": peaks["dfma"],
        "unit": "TFLOP/s", "peak_source": peaks["dfma_src"], "traffic": _ncu_traffic(name, "k_weights_ssf"),
        "ms_per_build": stage["weights_ms"], "pairs_evaluated": pairs, "nontrivial_points": nontrivial,
        "pairs_per_nontrivial_point": pairs / max(1, nontrivial), "pairs_per_point": pairs / max(1, plan.n_points),
        "flop_per_pair": FLOP_PER_PAIR}
    res["roofline_weights"]["frac"] = res["roofline_weights"]["achieved"] / peaks["dfma"]
    if do_e2e:
        # end to end through the C ABI with HOST buffers (pinned): H2D of P and D2H of V inside the timed region
        Ph = torch.from_numpy(w.P).pin_memory()
        Vh = torch.empty_like(Ph).pin_memory()
        plan.eval_host(Ph, Vh)
        t = []
        for k in range(max(3, min(steps, 10))):
            flush.fill_(2.0)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            plan.eval_host(Ph, Vh)
            t.append(time.perf_counter() - t0)
        e2e_s = statistics.mean(t)
        nb2 = plan.n_basis * plan.n_basis * 8
        res["e2e"] = {"value": plan.n_points / e2e_s, "unit": UNIT, "h2d_bytes_per_step": nb2, "d2h_bytes_per_step": nb2 + 16,
                      "ms_per_step": e2e_s * 1e3}
        assert float((Vh - V.cpu()).abs().max()) == 0.0
    plan.close()
    del P, V, flush
    torch.cuda.empty_cache()
    return res, w


def oracle_sample(w, name, target_seconds=15.0, stride=None, fn=None):
    """Times the CPU oracle as it stands (Mode A, its own paper-literal planner, SSF weights with its exact
    pruning) on a bounded sample of the workload: every `stride`-th atom's batches."""
    import numpy as np

    import oracle as orc
    fn = w.functional if fn is None else fn
    basis = (w.shell_atom, w.shell_L, w.shell_nprim, w.shell_prim_off, w.exps, w.coefs)
    na = len(w.atoms_Z)
    if stride is None:
        # calibrated on the GPU box (16 threads): ~0.3 s wall per atom-centred grid at c5 (PBE, 100x302, 1536 atoms); the weights term grows with N_atoms
        per_atom = 0.85 * (1 + na / 800.0) * (1.6 if fn == 1 else 1.0) * (w.n_rad * w.n_ang / 22650.0) / max(1, orc.num_threads())
        stride = max(1, int(round(na * per_atom / target_seconds)))
    atoms = np.arange(0, na, stride)
    t0 = time.perf_counter()
    pts, wq, par = orc.build_grid(w.atoms_xyz, w.n_rad, w.n_ang)
    sel = np.isin(par, atoms)
    pts, wq, par = pts[sel], wq[sel], par[sel]
    rc = orc.rcut(w.shell_nprim, w.shell_prim_off, w.exps)
    plan = orc.plan_paper(w.atoms_xyz, pts, wq, par, w.shell_atom, rc)
    wts = orc.partition_weights(w.atoms_xyz, plan.pts, plan.wq, plan.parent, 0, True)
    r = orc.evaluate(plan, wts, basis, w.atoms_xyz, w.P, fn, want_V=True)
    dt = time.perf_counter() - t0
    return dict(value=len(pts) / dt, unit=UNIT, cores=orc.num_threads(), kind="oracle", seconds=dt,
                sample="atom-centred grids of %d of %d atoms (every %d-th), %d points, %d batches of the oracle's own "
                       "paper-literal planner; grid + SSF weights + Alg. 4 incl. V; %s"
                       % (len(atoms), na, stride, len(pts), plan.n_batches, name), E_sample=r.E_xc)


SIDE_KEYS = ("workload", "functional", "n_points", "n_basis", "n_batches", "ms_per_step", "points_per_s", "builds_per_s", "fp64_tflops",
             "fp64_frac", "live_point_fraction", "stage_ms", "cached_weights_ms", "N_el_rel_err_vs_trPS", "nb_hist", "nq_hist",
             "plan_seconds", "clocks", "roofline_batch", "roofline_weights")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c5")
    ap.add_argument("--also", default="c4,c3,c2,c1,u2,s2,g1", help="comma list of extra workloads reported under other_workloads (or 'none')")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-becke", action="store_true", help="skip the Becke-1988 side measurement (on c2)")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup

    from workloads import make_workload

    if args.impl == "reference":
        # the reference arm of this tier = the CPU oracle, as it stands, on the host cores; rank 0 only
        if rank != 0:
            return
        w = make_workload(args.workload)
        times, last = [], None
        for k in range(args.warmup + args.steps):
            last = oracle_sample(w, args.workload, target_seconds=4.0)
            if k >= args.warmup:
                times.append(last["seconds"])
        npts_sample = last["value"] * last["seconds"]
        val = npts_sample / statistics.mean(times)
        line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": statistics.mean(times) * 1e3, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config_of(args.workload, w, world),
                "cpu_baseline": {"value": val, "unit": UNIT, "cores": last["cores"], "kind": "oracle", "sample": last["sample"]},
                "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
        print(json.dumps(line))
        return

    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        dist.barrier()
    torch.cuda.synchronize()
    # FP64 roofline denominators, measured live on this GPU (MEASURED_PEAKS.json has no FP64 entry): register-resident
    # DMMA (mma.sync m8n8k4 f64) and DFMA chains through the C ABI, burst figure (kernel timed alone)
    import paper_2007_03143_b200 as xc
    dmma_tf, dmma_mhz = xc.measure_fp64_peak(1, local_rank, 5)
    dfma_tf, _ = xc.measure_fp64_peak(0, local_rank, 5)
    how = ("measured live in this run by xc_measure_fp64_peak: DMMA %.2f, DFMA %.2f TFLOP/s (nominal %.1f = 148 SM x 64 FMA/clk x 2 x "
           "1.965 GHz)" % (dmma_tf, dfma_tf, FP64_NOMINAL_TFLOPS))
    peaks = {"fp64": max(dmma_tf, dfma_tf), "fp64_src": "FP64 tensor/FMA pipe " + how, "dfma": dfma_tf, "dfma_src": "FP64 ALU (DFMA) " + how}
    sampler = ClockSampler(local_rank)
    res, w = run_workload(args.workload, args.steps, warmup, peaks, device=local_rank, sampler=sampler)
    ms = res["ms_per_step"]
    if world > 1:
        t = torch.tensor([ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
        e = torch.tensor([res["e2e"]["ms_per_step"]], dtype=torch.float64, device="cuda")
        dist.all_reduce(e, op=dist.ReduceOp.MAX)
        res["e2e"]["value"] = world * res["n_points"] / (float(e.item()) * 1e-3)
        dist.barrier()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    hbm_peak, hbm_src = _peaks()
    value = world * res["n_points"] / (ms * 1e-3)
    st = res["stage_ms"]
    stats = res["stats"]
    # the kernel that takes most of the build comes first; both are reported
    dom, other = ("roofline_weights", "roofline_batch") if st["weights_ms"] >= st["batch_ms"] else ("roofline_batch", "roofline_weights")
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warmup,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": config_of(args.workload, w, world),
            "clocks": res["clocks"], "e2e": {k: res["e2e"][k] for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step")},
            "gpu_launches": res["launches"], "roofline": res[dom], "roofline_second_kernel": res[other],
            "builds_per_s": world * 1e3 / ms, "fp64_tflops": res["flops"] / (ms * 1e-3) * 1e-12,
            "fp64_roofline_frac": res["flops"] / (ms * 1e-3) * 1e-12 / peaks["fp64"],
            "fp64_peak": {"dmma_tflops": dmma_tf, "dfma_tflops": dfma_tf, "implied_sm_mhz": dmma_mhz, "how": "xc_measure_fp64_peak, best of 5"},
            "hbm_peak": {"gbs": hbm_peak, "source": "MEASURED_PEAKS.json hbm_gbs (%s)" % hbm_src,
                         "note": "neither kernel is HBM-bound: see roofline.traffic / profiles/ for the measured DRAM bytes"},
            "stage_ms": st, "cached_weights_ms": res["cached_weights_ms"],
            "cached_weights_points_per_s": res["n_points"] / (res["cached_weights_ms"] * 1e-3),
            "plan": {"seconds": res["plan_seconds"], "n_batches": res["n_batches"], "algorithmic_flops": res["flops"],
                     "algorithmic_flops_all_points": res["flops_all_points"],
                     "live_point_fraction": res["live_point_fraction"], "sum_nb_nq": stats["sum_nb_nq"],
                     "sum_nb2": stats["sum_nb2"], "nq_hist": res["nq_hist"], "nb_hist": res["nb_hist"], "kind": "global k-d bisection"},
            "E_xc": res["E_xc"], "N_el": res["N_el"], "N_el_rel_err_vs_trPS": res["N_el_rel_err_vs_trPS"]}
    # reading A1: the timed path is SSF (the paper's choice); the Becke-1988 partition (no compact support,
    # O(N_A^2) pair terms per point: 13 s per build at c5) is timed beside it on c2, same build otherwise
    if world == 1 and not args.no_becke:
        try:
            wb = make_workload("c2")
            bplan = xc.Plan.from_workload(wb, spec=xc.grid_spec(wb.n_rad, wb.n_ang, wb.functional, partition=1), device=local_rank)
            Pd = torch.from_numpy(wb.P).cuda()
            Vd = torch.empty_like(Pd)
            bplan.eval(Pd, Vd)
            tb = []
            for _ in range(3):
                bplan.eval(Pd, Vd)
                tb.append(bplan.timings())
            line["becke88"] = {"workload": "c2", "ms_per_step": statistics.median(t["total_ms"] for t in tb),
                               "weights_ms": statistics.median(t["weights_ms"] for t in tb),
                               "points_per_s": bplan.n_points / (statistics.median(t["total_ms"] for t in tb) * 1e-3)}
            bplan.close()
            del Pd, Vd
        except Exception as exc:
            line["becke88"] = {"error": repr(exc)[:200]}
    # the spin-unrestricted build (xc_eval_uks: passes of the same kernels) and the meta-GGA
    # intermediate tau (xc_eval_tau), timed on the 64-water PBE workload with P_a = P_b = P/2 (same shapes as c3)
    if world == 1 and not args.no_becke:
        try:
            wu = make_workload("c3")
            uplan = xc.Plan.from_workload(wu, spec=xc.grid_spec(wu.n_rad, wu.n_ang, wu.functional), device=local_rank)
            Ph = torch.from_numpy(0.5 * wu.P).cuda()
            Va, Vb = torch.empty_like(Ph), torch.empty_like(Ph)
            uplan.eval_uks(Ph, Ph, Va, Vb)
            tu = []
            for _ in range(3):
                uplan.eval_uks(Ph, Ph, Va, Vb)
                tu.append(uplan.timings()["total_ms"])
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            uplan.eval_tau(Ph, reuse_weights=True)
            ev0.record()
            uplan.eval_tau(Ph, reuse_weights=True)
            ev1.record()
            torch.cuda.synchronize()
            mplan = xc.Plan.from_workload(wu, spec=xc.grid_spec(wu.n_rad, wu.n_ang, 2), device=local_rank)
            Pf = torch.from_numpy(wu.P).cuda()
            mplan.eval(Pf, Va)
            tm = []
            for _ in range(3):
                mplan.eval(Pf, Va)
                tm.append(mplan.timings()["total_ms"])
            mplan.close()
            line["mgga"] = {"workload": "c3 shapes, MS0 exchange + PBE correlation (functional = 2)", "ms_per_step": statistics.median(tm),
                            "points_per_s": uplan.n_points / (statistics.median(tm) * 1e-3)}
            del Pf
            line["uks"] = {"workload": "c3 (P_a = P_b = P/2)", "ms_per_step": statistics.median(tu),
                           "points_per_s": uplan.n_points / (statistics.median(tu) * 1e-3), "tau_ms_cached_weights": ev0.elapsed_time(ev1)}
            uplan.close()
            del Ph, Va, Vb
        except Exception as exc:
            line["uks"] = {"error": repr(exc)[:200]}
    if not args.no_cpu_baseline:
        cb = oracle_sample(w, args.workload)
        line["cpu_baseline"] = {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample", "seconds")}
    others = []
    if args.also and args.also != "none" and world == 1:
        for nm in args.also.split(","):
            if nm == args.workload:
                continue
            try:
                first_class = nm in ("c4", "c5")
                r2, _ = run_workload(nm, max(3, min(args.steps, 10 if first_class else 5)), 3, peaks, do_e2e=first_class, device=local_rank)
                o = {k: r2[k] for k in SIDE_KEYS}
                if first_class:
                    o["e2e"] = {k: r2["e2e"][k] for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step")}
                others.append(o)
            except Exception as exc:  # an extra workload must never cost the headline line
                others.append({"workload": nm, "error": repr(exc)[:200]})
    line["other_workloads"] = others
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
