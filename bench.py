#!/usr/bin/env python
"""bench.py -- headline benchmark of the matrix-free prism-gravity hot path on B200.

A "step" is ONE data-space CG iteration on a BASELINE.json configuration (default: config 5, the largest,
3.33 M prisms x 178,797 stations): adjoint product G^T p (+ depth weighting W^-2 and the node<->prism
regrouping), forward product G(.), and the fused CG vector updates -- every row of SURVEY.md 8(a) that runs per
iteration.  metric = prism-observation pair evaluations per second (2*N*M pairs per step), FP64.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "prism-obs pair evals/s (matrix-free G*m, G^T*v, FP64)"
UNIT = "pair evals/s"

FP64_LANES_PER_SM = 64          # B200: 148 SMs x 64 FP64 lanes (DGX B200: 37 TFLOP/s FP64 = 148*64*2*1.965e9)
# Measured per-kernel figures come from profiles/kernel_metrics.csv, written by
# `python -m paper_2602_03857_b200.ncu_summary` from an `ncu --set full` capture (the .md beside it names the commands):
# FP64-pipe thread-instructions per node evaluation and DRAM bytes per launch.  Nothing is hard-coded here.
METRICS_CSV = os.path.join(ROOT, "profiles", "kernel_metrics.csv")


def kernel_metrics():
    """{(kernel, config): {column: float}} from profiles/kernel_metrics.csv ({} when the file is absent)."""
    out = {}
    try:
        import csv
        with open(METRICS_CSV) as f:
            for row in csv.DictReader(f):
                vals = {}
                for k, v in row.items():
                    try:
                        vals[k] = float(v)
                    except (TypeError, ValueError):
                        vals[k] = v
                out[(row["kernel"], int(float(row["config"])))] = vals
    except OSError:
        pass
    return out


def metric(kernel, cfg, column, log2d=True):
    """One figure of the capture; fp64_inst_per_eval falls back to the same kernel at any config (the loop body does
    not depend on the config), then to None."""
    km = kernel_metrics()
    row = km.get((kernel, cfg))
    if row is None and column == "fp64_inst_per_eval":
        for (k, _), r in km.items():
            if k == kernel and bool(r.get("log2d", 1.0)) == bool(log2d):
                row = r
                break
    v = None if row is None else row.get(column)
    return v if isinstance(v, float) and v == v else None


def cpu_info():
    """Logical / physical core counts and the CPU model string of this host."""
    model, phys = None, set()
    try:
        pid = cid = None
        for line in open("/proc/cpuinfo"):
            k, _, v = line.partition(":")
            k, v = k.strip(), v.strip()
            if k == "model name" and model is None:
                model = v
            elif k == "physical id":
                pid = v
            elif k == "core id":
                cid = v
            elif not k and pid is not None and cid is not None:
                phys.add((pid, cid))
                pid = cid = None
    except OSError:
        pass
    return {"cpu_model": model, "logical_cores": os.cpu_count(), "physical_cores": len(phys) or None}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--no-paper-shape", action="store_true",
                    help="skip the paper-shaped run (Table 1 shape: Float32 G build + outer inversion loop)")
    ap.add_argument("--paper-shape-matrix-free", action="store_true",
                    help="also run the outer inversion loop matrix-free in FP64 on the paper's shape (~1 min)")
    ap.add_argument("--no-stored", action="store_true", help="skip the stored-G (HBM-bound GEMV) measurement")
    ap.add_argument("--no-fp32", action="store_true", help="skip the Float32 matrix-free leg")
    ap.add_argument("--no-precond", action="store_true", help="skip the plain-vs-Jacobi CG iteration count (config 2)")
    ap.add_argument("--stored-config", type=int, default=3, help="config whose G is tabulated for the stored-G leg")
    return ap.parse_args()


# ---------------------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "200"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            pass

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            t = [x.strip() for x in line.split(",")]
            if len(t) < 8:
                continue
            try:
                sm.append(float(t[0])); mx.append(float(t[1])); pw.append(float(t[2]))
            except ValueError:
                continue
            for nm, val in zip(names, t[4:8]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            # "under load": samples whose power is within 25% of the max seen
            pmax = max(pw)
            load = [s for s, p in zip(sm, pw) if p >= 0.75 * pmax] or sm
            out.update(sm_mhz=statistics.median(load), sm_max_mhz=max(mx), power_w_max=pmax, samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


def cpu_oracle_rate(wl, seconds, sample_note=True):
    """Times the oracle (as it stands) on a bounded sample of the workload: forward on S stations x all prisms."""
    import oracle
    mesh = oracle.Mesh(wl.xn, wl.yn, wl.zn)
    cores = oracle.hardware_threads()
    rng = np.random.default_rng(7)
    u = wl.m_true

    def run(S):
        idx = rng.choice(wl.N, size=min(S, wl.N), replace=False)
        t0 = time.perf_counter()
        oracle.forward(mesh, wl.xo[idx], wl.yo[idx], wl.zo[idx], wl.gamma, u, nthreads=cores)
        return time.perf_counter() - t0, idx.size

    S0 = max(cores, 1)
    t, s = run(S0)
    rate = s * wl.M / t
    S = int(max(S0, min(wl.N, seconds * rate / wl.M)))
    S = max(cores, (S // cores) * cores)
    t, s = run(S)
    return dict(value=s * wl.M / t, unit=UNIT, cores=cores, kind="oracle",
                sample=f"oracle.forward on {s} seeded stations x all {wl.M} prisms ({s * wl.M:.3g} pairs, {t:.1f} s)",
                threads_used=cores, **cpu_info())



def measured_hbm_peak():
    """(GB/s, source): the driver-written copy bandwidth of this pool's B200s, else the profiling guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (copy read+write, burst)"
    except Exception:
        return 6500.0, "fallback (B200_PROFILING.md: ~6.5 TB/s measured copy bandwidth); MEASURED_PEAKS.json absent"


def stored_g_leg(cfg, local, reps=5):
    """BASELINE.json north_star kernel 4: tabulate G once (FP32 storage at config 3, reading C10), then time the
    two HBM-bound mat-vecs d = G u and g = G^T v alone with CUDA events; algorithmic bytes = N*M*sizeof(elem)."""
    import torch
    from paper_2602_03857_b200 import binding, workloads
    wl = workloads.make(cfg)
    fp32 = wl.N * wl.M * 8 > 100e9
    elem = 4 if fp32 else 8
    dev = torch.device("cuda", local)
    ctx = binding.GravContext(wl.xn, wl.yn, wl.zn, wl.xo, wl.yo, wl.zo, wl.gamma, device=local)
    u = torch.as_tensor(np.ascontiguousarray(wl.m_true)).to(dev)
    v = torch.as_tensor(np.random.default_rng(11).standard_normal(wl.N)).to(dev)
    d = torch.empty(wl.N, dtype=torch.float64, device=dev)
    g = torch.empty(wl.M, dtype=torch.float64, device=dev)
    ev = lambda: torch.cuda.Event(enable_timing=True)
    e0, e1 = ev(), ev()
    l0 = ctx.launches
    ctx.store_g(fp32=fp32)                    # untimed first call (one-off shared-memory opt-in of the kernel on the host)
    torch.cuda.synchronize()
    e0.record(); ctx.store_g(fp32=fp32); e1.record(); torch.cuda.synchronize()
    t_tab = e0.elapsed_time(e1)

    def timed(fn):
        fn(); torch.cuda.synchronize()
        ts = []
        for _ in range(reps):            # G (>= 4 GB) is far larger than the 126 MB L2: every pass streams from HBM
            a, b = ev(), ev()
            a.record(); fn(); b.record(); torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        return statistics.median(ts)

    t_mv = timed(lambda: ctx.forward_stored(u, out=d))
    t_mvt = timed(lambda: ctx.adjoint_stored(v, out=g))
    launches = ctx.launches - l0
    dm = ctx.forward(u)
    err = float((d - dm).abs().max() / dm.abs().max())
    nbytes = float(wl.N) * wl.M * elem
    peak, src = measured_hbm_peak()
    dom, t_dom = ("gemv", t_mv) if t_mv >= t_mvt else ("gemvt", t_mvt)
    out = {"workload": wl.name, "elem": "f32" if fp32 else "f64", "g_bytes": nbytes,
           "ms_tabulate": t_tab, "pairs_per_s_tabulate": float(wl.N) * wl.M / (t_tab * 1e-3),
           "ms_gemv": t_mv, "ms_gemvt": t_mvt, "s_per_cg_iter_stored": (t_mv + t_mvt) * 1e-3,
           "max_rel_err_vs_matrix_free_forward": err, "gpu_launches": launches,
           "roofline": {"bound": "hbm", "kernel": dom, "achieved": nbytes / (t_dom * 1e-3) / 1e9, "peak": peak,
                        "unit": "GB/s", "frac": nbytes / (t_dom * 1e-3) / 1e9 / peak,
                        "traffic": metric(dom, cfg, "dram_bytes_per_launch"), "peak_source": src,
                        "frac_of_8TBps_nominal": nbytes / (t_dom * 1e-3) / 1e9 / 8000.0,
                        "gbs_gemv": nbytes / (t_mv * 1e-3) / 1e9, "gbs_gemvt": nbytes / (t_mvt * 1e-3) / 1e9}}
    ctx.close()
    del ctx
    torch.cuda.empty_cache()
    return out


def paper_shape_leg(local, matrix_free=False):
    """the paper's own pipeline on the SHAPE of its largest single-GPU benchmark (Table 1,
    P:168-178: 2,601 stations x 3.28e6 cells, Float32 G = 34.1 GB): build G in Float32, then the outer model-update
    loop (<= 30 updates x <= 20 CG iterations, tolerances 1e-4) with the stored G.  Wall clock around the
    synchronising C-ABI calls.  The paper's 63.88 s (1x A100 40 GB) / 1007.46 s (EPYC 7H12) are quoted as context:
    different hardware, different (unavailable) model and data."""
    import torch
    from paper_2602_03857_b200 import binding, workloads
    wl = workloads.make(6)
    dev = torch.device("cuda", local)
    ctx = binding.GravContext(wl.xn, wl.yn, wl.zn, wl.xo, wl.yo, wl.zo, wl.gamma, device=local)
    w = ctx.depth_weights(wl.beta, wl.z0)
    d_clean = ctx.forward(torch.as_tensor(np.ascontiguousarray(wl.m_true)).to(dev))
    d_obs = d_clean + wl.noise_frac * float(d_clean.abs().max()) * torch.as_tensor(wl.noise()).to(dev)
    lam = wl.lam_factor * float(ctx.gram_diag(w).mean().item())
    ctx.set_mode(binding.STORED_F32)
    torch.cuda.synchronize()
    l0 = ctx.launches
    t0 = time.perf_counter()
    ctx.store_g(fp32=True)
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    out = ctx.invert(d_obs, w, lam, max_outer=30, max_inner=20, tol_outer=1e-4, tol_inner=1e-4,
                     mode=binding.STORED_F32)
    torch.cuda.synchronize()
    t2 = time.perf_counter()
    # fixed work of the paper's schedule: every one of the 30 updates runs its 20 CG iterations, the model recovery
    # and the step product (no early stop) - the adaptive run above stops as soon as an update brings no decrease,
    # which on this ill-conditioned system depends on the last bits of G (3-9 updates observed)
    torch.cuda.synchronize()
    t2b = time.perf_counter()
    dd = torch.empty(wl.N, dtype=torch.float64, device=dev)
    for _ in range(30):
        cg = ctx.dataspace_cg(d_obs, w, lam, 20, mode=binding.STORED_F32)
        ctx.forward_stored(cg["m"], out=dd)
    torch.cuda.synchronize()
    t2c = time.perf_counter()
    res = {"workload": wl.name, "prisms": wl.M, "stations": wl.N, "g_bytes_f32": float(wl.N) * wl.M * 4,
           "build_s": t1 - t0, "fixed_work_inversion_s": t2c - t2b, "total_s": (t1 - t0) + (t2c - t2b),
           "total_note": "FIXED WORK: Float32 G build + 30 updates x (20 CG iterations + model recovery + step product), "
                         "no early stop - the figure to read beside the paper's totals",
           "pairs_per_s_build": float(wl.N) * wl.M / (t1 - t0),
           "adaptive": {"inversion_s": t2 - t1, "outer_updates": out["n_outer"], "stop": out["stop"],
                        "rel_residual": float(out["hist"][-1]),
                        "note": "stopping update not reproducible: with <= 20 CG iterations the inner solves are far "
                                "from converged and which update first brings no decrease depends on the last bits of "
                                "G (DESIGN.md 5.7); not a benchmark figure"},
           "gpu_launches": ctx.launches - l0, "lambda": lam,
           "paper_context": {"total_s_1xA100_f32": 63.88, "total_s_cpu_epyc7h12": 1007.46,
                             "source": "PAPER.md Table 1 (P:168-178), 3.28e6 cells x 2,601 stations"}}
    if matrix_free:
        t3 = time.perf_counter()
        out2 = ctx.invert(d_obs, w, lam, max_outer=30, max_inner=20, tol_outer=1e-4, tol_inner=1e-4)
        torch.cuda.synchronize()
        res["matrix_free_f64_total_s"] = time.perf_counter() - t3
        res["matrix_free_f64_outer_updates"] = out2["n_outer"]
        res["model_diff_f32_vs_f64"] = float((out["m"] - out2["m"]).abs().max() / out2["m"].abs().max())
    ctx.close()
    del ctx
    torch.cuda.empty_cache()
    return res


def fp32_leg(cfgs, local):
    """SURVEY.md 8(f) item 2, second half: the matrix-free products with the Float32 evaluator (the paper's precision,
    P:203; grav_set_precision) on BJ configs and on the paper's Table 1 shape: time per product and the error against the
    FP64 path of the same library (itself within 1e-10 of the oracle), as a fraction of the output's global max."""
    import torch
    from paper_2602_03857_b200 import binding, workloads
    dev = torch.device("cuda", local)
    ev = lambda: torch.cuda.Event(enable_timing=True)
    out = {}
    for cfg in cfgs:
        wl = workloads.make(cfg)
        ctx = binding.GravContext(wl.xn, wl.yn, wl.zn, wl.xo, wl.yo, wl.zo, wl.gamma, device=local)
        u = torch.as_tensor(np.ascontiguousarray(wl.m_true)).to(dev)
        d64 = ctx.forward(u)
        v = d64 + wl.noise_frac * float(d64.abs().max()) * torch.as_tensor(wl.noise()).to(dev)
        g64 = ctx.adjoint(v)
        ctx.set_precision(True)

        def timed(fn):
            fn(); torch.cuda.synchronize()
            a, b = ev(), ev()
            a.record(); r = fn(); b.record(); torch.cuda.synchronize()
            return a.elapsed_time(b), r

        t_f, d32 = timed(lambda: ctx.forward(u))
        t_a, g32 = timed(lambda: ctx.adjoint(v))
        out[wl.name] = {"ms_forward": t_f, "ms_adjoint": t_a,
                        "pairs_per_s_forward": float(wl.N) * wl.M / (t_f * 1e-3),
                        "pairs_per_s_adjoint": float(wl.N) * wl.M / (t_a * 1e-3),
                        "err_of_max_forward": float((d32 - d64).abs().max() / d64.abs().max()),
                        "err_of_max_adjoint": float((g32 - g64).abs().max() / g64.abs().max()),
                        "inputs": "u = true model, v = noisy data"}
        ctx.close()
        del ctx
        torch.cuda.empty_cache()
    out["note"] = ("Float32 Psi (FP64 coordinate differences, cancellation-free R + Y, FP64 accumulation); error vs the "
                   "FP64 path as a fraction of max|output|; not held to the 1e-10 operator tolerance")
    return out


def precond_leg(local, rtol=1e-8, cap=1500):
    """Jacobi-preconditioned CG (M = diag(G W^-2 G^T) + lambda from grav_gram_diag) against plain
    CG on the data-space system: iterations until the recursive residual meets rtol * ||d_obs||, on BJ config 2 (regular
    station grid at one height: a nearly constant Gram diagonal) and on a config-4-like survey small enough to converge
    in seconds (4,096 random stations 2-152 m above a 48 x 48 x 24 mesh: the diagonal varies with the station height)."""
    import torch
    from paper_2602_03857_b200 import binding, workloads
    dev = torch.device("cuda", local)
    res = {"rtol": rtol, "cap": cap}
    for wl in (workloads.make(2),
               workloads.make_custom(48, 48, 24, 50.0, 4096, seed=4, topo_amp=150.0, clearance=2.0, name="topo_48x48x24_4096")):
        ctx = binding.GravContext(wl.xn, wl.yn, wl.zn, wl.xo, wl.yo, wl.zo, wl.gamma, device=local)
        w = ctx.depth_weights(wl.beta, wl.z0)
        d_clean = ctx.forward(torch.as_tensor(np.ascontiguousarray(wl.m_true)).to(dev))
        d_obs = d_clean + wl.noise_frac * float(d_clean.abs().max()) * torch.as_tensor(wl.noise()).to(dev)
        diag = ctx.gram_diag(w)
        lam = wl.lam_factor * float(diag.mean().item())
        one = {"lambda": lam, "gram_diag_max_over_min": float(diag.max() / diag.min())}
        for name, pc in (("plain", None), ("jacobi", diag)):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            out = ctx.dataspace_cg(d_obs, w, lam, cap, rtol=rtol, precond=pc, want_m=False)
            hist = out["hist"].cpu().numpy()
            dt = time.perf_counter() - t0
            below = np.nonzero(hist <= rtol * hist[0])[0]
            one[name] = {"iterations": int(below[0]) if below.size else None,
                         "final_rel_residual": float(hist[-1] / hist[0]), "seconds_for_cap_launches": dt}
        res[wl.name] = one
        ctx.close()
        del ctx
        torch.cuda.empty_cache()
    return res


# ---------------------------------------------------------------------------------------------------------------
def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the host cores.  One step = forward + adjoint restricted
    to a bounded sample of S stations (2*S*M pairs)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    from paper_2602_03857_b200 import workloads
    wl = workloads.make(args.config)
    mesh = oracle.Mesh(wl.xn, wl.yn, wl.zn)
    cores = oracle.hardware_threads()
    S = max(1, min(wl.N, int(round(1.0e8 / (2 * wl.M)))))      # ~1e8 pairs per step: seconds on a multicore host
    S = max(S, min(cores, wl.N))
    rng = np.random.default_rng(7)
    idx = rng.choice(wl.N, size=S, replace=False)
    xo, yo, zo = wl.xo[idx], wl.yo[idx], wl.zo[idx]
    w = oracle.depth_weights(mesh, wl.beta, wl.z0)
    p = rng.standard_normal(S)

    def step():
        g = oracle.adjoint(mesh, xo, yo, zo, wl.gamma, p, nthreads=cores)
        g /= w * w
        return oracle.forward(mesh, xo, yo, zo, wl.gamma, g, nthreads=cores)

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    pairs = 2.0 * S * wl.M * args.steps
    val = pairs / dt
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl.name, "prisms": wl.M, "stations": wl.N,
                       "sample": f"{S} seeded stations x all prisms per step (adjoint + forward)"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"{S} stations x {wl.M} prisms, adjoint+forward per step",
                             "threads_used": cores, **cpu_info()},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    from paper_2602_03857_b200 import binding, workloads
    from paper_2602_03857_b200 import dist as gdist

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        os.environ.setdefault("NCCL_DEBUG", "INFO")       # rank / transport lines ...
        os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")   # ... on stderr (NCCL's default is stdout; the JSON line owns stdout)
    # NCCL, one rank per GPU.  GRAV_DIST_BACKEND=gloo (development only): several ranks share the visible GPUs and the
    # collectives are staged through host memory (dist.Comm.staged) - a functional check of this file's multi-rank logic
    # on a one-GPU box, never a measurement.
    backend = os.environ.get("GRAV_DIST_BACKEND", "nccl")
    rank, world, local = gdist.init_from_env(backend)
    local %= torch.cuda.device_count()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    wl = workloads.make(args.config)
    N, M, Nn = wl.N, wl.M, wl.n_nodes
    # observation-sharded over the ranks; world == 1: the whole station set, no exchange hook
    sh = gdist.ShardedContext(wl, rank, world, local)
    ctx, Nloc = sh.ctx, sh.hi - sh.lo
    to = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64)).to(dev)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            torch.distributed.barrier()
            torch.cuda.synchronize()

    # ---- inputs resident in HBM: d_obs = G m_true + noise (GPU forward, parity-checked in tests/), weights, lambda
    w = ctx.depth_weights(wl.beta, wl.z0)
    d_clean = ctx.forward(to(wl.m_true))
    dmax = d_clean.abs().max().reshape(1)
    if world > 1:
        torch.distributed.all_reduce(dmax, op=torch.distributed.ReduceOp.MAX)
    sigma = wl.noise_frac * float(dmax.item())
    d_obs = d_clean + sigma * sh.local(wl.noise())
    # lambda = 1e-2 * trace(G W^-2 G^T) / N (reading C7) from the full Gram diagonal of this rank's stations (~1.15
    # evaluations per pair with the node-shared per-pair kernel: about one forward product), summed over ranks
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    gdiag = ctx.gram_diag(w)
    ev1.record()
    tr = gdiag.sum().reshape(1)
    if world > 1:
        torch.distributed.all_reduce(tr)
    torch.cuda.synchronize()
    ms_gram = ev0.elapsed_time(ev1)
    lam = wl.lam_factor * float(tr.item()) / N

    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    ev = lambda: torch.cuda.Event(enable_timing=True)
    state = binding.CGState(Nloc, dev)

    def one_step(first):
        state.resume = not first
        ctx.dataspace_cg(d_obs, w, lam, 1, state=state, want_m=False)

    # ---- warm-up, then K timed steps (L2 flushed between steps, CUDA events on the launching stream)
    for k in range(args.warmup):
        one_step(k == 0)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    launches0 = ctx.launches
    total_ms = 0.0
    for k in range(args.steps):
        flush.fill_(k & 0xFF)
        e0, e1 = ev(), ev()
        barrier()
        e0.record()
        one_step(args.warmup == 0 and k == 0)
        e1.record()
        barrier()
        total_ms += gdist.max_over_ranks(e0.elapsed_time(e1), dev)
    launches = ctx.launches - launches0
    pairs_per_step = 2.0 * N * M
    value = pairs_per_step * args.steps / (total_ms * 1e-3)

    # ---- small problems: the same iteration inside ONE multi-iteration call (no per-step Python / set-up launches)
    cg_call = None
    if float(N) * Nn < 1e10:
        its = 20
        state.resume = True
        l0 = ctx.launches
        ctx.dataspace_cg(d_obs, w, lam, its, state=state, want_m=False)
        per_it = (ctx.launches - l0 - 2) / its
        barrier()
        e0, e1 = ev(), ev()
        e0.record()
        ctx.dataspace_cg(d_obs, w, lam, its, state=state, want_m=False)
        e1.record()
        barrier()
        cg_call = {"iters": its, "us_per_iteration": gdist.max_over_ranks(e0.elapsed_time(e1), dev) * 1e3 / its,
                   "launches_per_iteration": per_it,
                   "note": "one grav_dataspace_cg call of 20 iterations resumed from device state, CUDA events around it"}

    # ---- the two dominant kernels timed alone (same launch configuration), for the roofline object
    u_vec = to(wl.m_true)
    dn, gm = torch.empty(Nloc, dtype=torch.float64, device=dev), torch.empty(M, dtype=torch.float64, device=dev)

    def timed(fn, reps):
        fn()
        ts = []
        for _ in range(reps):
            flush.fill_(1)
            e0, e1 = ev(), ev()
            barrier()
            e0.record(); fn(); e1.record()
            barrier()
            ts.append(e0.elapsed_time(e1))
        return statistics.median(ts)

    reps = max(1, min(3, args.steps))
    t_fwd = timed(lambda: ctx.forward(u_vec, out=dn), reps)
    t_adj = timed(lambda: ctx.adjoint(d_obs, out=gm), reps)
    clocks = sampler.stop() if sampler else None

    evals = float(Nloc) * Nn                     # node evaluations one launch of this rank processes
    dom, t_dom = ("forward_nodes", t_fwd) if t_fwd >= t_adj else ("adjoint_nodes", t_adj)
    log2d = ctx.log2d_default
    # FP64-pipe thread-instructions per node evaluation: from the committed ncu capture of each kernel
    # (profiles/kernel_metrics.csv); the SASS census of the z-loop when no capture is committed
    census = 43.0 if log2d else 45.0
    pe_f = metric("forward_nodes", args.config, "fp64_inst_per_eval", log2d) or census
    pe_a = metric("adjoint_nodes", args.config, "fp64_inst_per_eval", log2d) or census
    # algorithmic work = the evaluator's FP64 instructions (census), not what a kernel executes on top of them
    ach_f = census * evals / (t_fwd * 1e-3) / 1e12
    ach_a = census * evals / (t_adj * 1e-3) / 1e12
    achieved = ach_f if dom == "forward_nodes" else ach_a
    peak_nominal = 148 * FP64_LANES_PER_SM * 1.965e9 / 1e12
    probe_rate, _ = binding.fp64_peak_probe(local, 100000)
    clk = (clocks or {}).get("sm_mhz") or 1965.0
    roofline = {
        "bound": "alu", "kernel": dom, "achieved": achieved, "peak": peak_nominal,
        "unit": "T FP64-pipe thread-inst/s", "frac": achieved / peak_nominal,
        "traffic": metric(dom, args.config, "dram_bytes_per_launch"),
        "peak_source": "148 SM x 64 FP64 lanes x 1.965 GHz = 1 DFMA/DMUL/DADD per lane per clock (DESIGN.md 6); "
                       f"DFMA-only probe in this run: {probe_rate / 1e12:.2f} T inst/s",
        "frac_of_probe": achieved / (probe_rate / 1e12),
        "frac_at_held_clock": achieved / (148 * FP64_LANES_PER_SM * clk * 1e6 / 1e12),
        "fp64_inst_per_eval": census, "fp64_inst_per_eval_source": "SASS census of the evaluator (DESIGN.md 6)",
        # round 1's line counted 44 instructions per evaluation; the evaluator has since lost one (and the per-launch time
        # at config 5 is the same to 0.3 %), so the same speed now reads as a lower fraction
        "frac_note": "algorithmic work = 43 FP64 instr / evaluation (round 1: 44); frac with round 1's count = "
                     f"{achieved / peak_nominal * 44.0 / census:.4f}" if log2d else None,
        "fp64_inst_executed_per_eval_ncu": {"forward_nodes": pe_f, "adjoint_nodes": pe_a},
        "log2d_binades": ctx.log2d_binades if log2d else 0, "evals_per_launch": evals,
        "forward_nodes": {"ms": t_fwd, "achieved": ach_f, "frac": ach_f / peak_nominal,
                          "pairs_per_s": float(Nloc) * M / (t_fwd * 1e-3),
                          "traffic": metric("forward_nodes", args.config, "dram_bytes_per_launch")},
        "adjoint_nodes": {"ms": t_adj, "achieved": ach_a, "frac": ach_a / peak_nominal,
                          "pairs_per_s": float(Nloc) * M / (t_adj * 1e-3),
                          "traffic": metric("adjoint_nodes", args.config, "dram_bytes_per_launch")},
        "ms_forward": t_fwd, "ms_adjoint": t_adj,
        "pairs_per_s_forward": float(Nloc) * M / (t_fwd * 1e-3), "pairs_per_s_adjoint": float(Nloc) * M / (t_adj * 1e-3),
    }

    # ---- end to end through the host-buffer C-ABI call: H2D d_obs, weights, 1 CG iteration + model recovery,
    #      D2H alpha and m, every step
    e2e = None
    if not args.no_e2e:
        dh = d_obs.cpu().pin_memory()
        ah = torch.empty(Nloc, dtype=torch.float64).pin_memory()
        mh = torch.empty(M, dtype=torch.float64).pin_memory()
        ctx.dataspace_cg_host(dh, wl.beta, wl.z0, lam, 1, ah, mh)      # warm
        nrep = max(1, min(args.steps, 3))
        barrier()
        t0 = time.perf_counter()
        for _ in range(nrep):
            ctx.dataspace_cg_host(dh, wl.beta, wl.z0, lam, 1, ah, mh)
        barrier()
        dt = gdist.max_over_ranks((time.perf_counter() - t0) * 1e3, dev) * 1e-3
        e2e = {"value": 3.0 * N * M * nrep / dt, "unit": UNIT, "h2d_bytes_per_step": 8 * Nloc,
               "d2h_bytes_per_step": 8 * (Nloc + M), "ms_per_step": 1e3 * dt / nrep,
               "call": "grav_dataspace_cg_host(iters=1): H2D d_obs, depth weights, 1 CG iteration (adjoint+forward) "
                       "+ model recovery (adjoint) = 3*N*M pairs, D2H alpha+m; host wall clock around the "
                       "synchronising call, bytes per rank"}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_oracle_rate(wl, args.cpu_seconds)

    stored = None
    if rank == 0 and world == 1 and not args.no_stored:
        sh.close()
        try:
            stored = stored_g_leg(args.stored_config, local)
        except Exception as ex:          # a secondary leg must never cost the headline line (e.g. not enough free HBM)
            stored = {"error": f"{type(ex).__name__}: {ex}"[:300]}
            torch.cuda.empty_cache()

    paper = None
    if rank == 0 and world == 1 and not args.no_paper_shape:
        sh.close()
        try:
            paper = paper_shape_leg(local, args.paper_shape_matrix_free)
        except Exception as ex:
            paper = {"error": f"{type(ex).__name__}: {ex}"[:300]}
            torch.cuda.empty_cache()

    fp32 = None
    if rank == 0 and world == 1 and not args.no_fp32:
        sh.close()
        try:
            fp32 = fp32_leg(sorted({3, args.config, 6}), local)
        except Exception as ex:
            fp32 = {"error": f"{type(ex).__name__}: {ex}"[:300]}
            torch.cuda.empty_cache()

    precond = None
    if rank == 0 and world == 1 and not args.no_precond:
        sh.close()
        try:
            precond = precond_leg(local)
        except Exception as ex:
            precond = {"error": f"{type(ex).__name__}: {ex}"[:300]}
            torch.cuda.empty_cache()

    # per-rank kernel times (multi-GPU: the driver reads the spread)
    per_rank = None
    if world > 1:
        t = torch.tensor([t_fwd, t_adj], dtype=torch.float64, device=dev if backend == "nccl" else "cpu")
        allt = [torch.empty_like(t) for _ in range(world)]
        torch.distributed.all_gather(allt, t)
        per_rank = [{"rank": r, "stations": gdist.shard_range(N, world, r)[1] - gdist.shard_range(N, world, r)[0],
                     "ms_forward": float(a[0]), "ms_adjoint": float(a[1])} for r, a in enumerate(allt)]

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps,
            "s_per_cg_iter": total_ms / args.steps * 1e-3, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl.name, "prisms": M, "stations": N, "nodes": Nn,
                       "pairs_per_step": pairs_per_step,
                       "step": "one data-space CG iteration (G^T p, W^-2, G(.), fused vector ops)",
                       "parallelism": f"stations sharded over {world} rank(s); all-gather of the (hi, lo) node-sum "
                                      f"planes + all-reduce of the dot partials",
                       "l2": "flushed between steps (256 MiB write)", "lambda": lam,
                       "lambda_note": "1e-2 * trace(G W^-2 G^T) / N from the full Gram diagonal (grav_gram_diag)",
                       "ms_gram_diag": ms_gram, "pairs_per_s_gram_diag": float(Nloc) * M / (ms_gram * 1e-3)},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu,
            "stored_g": stored, "paper_shape": paper, "fp32_matrix_free": fp32, "jacobi_pcg": precond,
            "per_rank": per_rank, "cg_call": cg_call,
        }
        print(json.dumps(line))
    sh.close()
    if world > 1:
        torch.distributed.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
