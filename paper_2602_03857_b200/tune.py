"""A/B timing of the forward / adjoint launch variants (include/grav.h: grav_debug_set_tuning) on one config.

    python -m paper_2602_03857_b200.tune [--config 3] [--reps 3]

Prints one line per variant: milliseconds (best of `reps`, CUDA events), node evaluations per second, scheduler cycles
per warp-evaluation at 1.965 GHz, and the largest difference from variant 0 relative to max|output|.  Variant 0 is
what the library ships; the others exist for this comparison (profiles/r1_tail_and_variants.md)."""
import argparse

import numpy as np
import torch

from . import binding, workloads

FORWARD = {0: "shipped: 2-D log table, 512 thr, unroll 12, if the geometry admits it, else variant 8", 8: "staged z-stream, psi2, 256 thr, unroll 8", 1: "staged, psi2, unroll 4",
           2: "LDG z-stream, psi2, unroll 4", 3: "LDG z-stream, psi2, unroll 8",
           4: "first generation: LDG, psi, 128 thr, unroll 2", 5: "staged, psi2, 512 thr, unroll 8",
           6: "staged, psi2 + 2-D log table, 512 thr, unroll 8", 7: "same, unroll 4"}
ADJOINT = {0: "plan's KC (shipped)", 1: "psi2, 256 thr, KC 4", 2: "psi2, 256 thr, KC 5", 3: "psi2, 128 thr, KC 6",
           4: "first generation: psi, 128 thr, KC 4", 5: "psi2, 128 thr, KC 8",
           6: "psi2 + 2-D log table, 512 thr, KC 4", 7: "psi2 + 2-D log table, 256 thr, KC 8",
           8: "psi2 + 2-D log table, 512 thr, KC 5", 9: "psi2 + 2-D log table, 256 thr, KC 6"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--reps", type=int, default=3)
    args = ap.parse_args()
    wl = workloads.make(args.config)
    ctx = binding.GravContext(wl.xn, wl.yn, wl.zn, wl.xo, wl.yo, wl.zo, wl.gamma, device=0)
    dev = torch.device("cuda", 0)
    u = torch.as_tensor(wl.m_true).to(dev)
    v = torch.as_tensor(np.random.default_rng(1).standard_normal(wl.N)).to(dev)
    d = torch.empty(wl.N, dtype=torch.float64, device=dev)
    g = torch.empty(wl.M, dtype=torch.float64, device=dev)
    evals = wl.N * wl.n_nodes

    def timeit(fn):
        fn()
        torch.cuda.synchronize()
        best = 1e30
        for _ in range(args.reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); fn(); e1.record()
            torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1))
        return best

    print(f"{wl.name}: N={wl.N} M={wl.M} nodes={wl.n_nodes} evaluations per product={evals:.4g}")
    for which, names, run, out in ((0, FORWARD, lambda: ctx.forward(u, out=d), d),
                                   (1, ADJOINT, lambda: ctx.adjoint(v, out=g), g)):
        ctx.set_tuning(which, 0)
        run()
        ref = out.clone()
        for t, label in names.items():
            ctx.set_tuning(which, t)
            ms = timeit(run)
            err = float((out - ref).abs().max() / ref.abs().max())
            cyc = ms * 1e-3 * 1.965e9 * 148 * 4 / (evals / 32)
            print(f"{'forward' if which == 0 else 'adjoint'} {t}: {ms:10.3f} ms  {evals / ms / 1e6:8.2f} Geval/s  "
                  f"{cyc:6.1f} cycles/warp-eval  diff {err:.1e}  {label}")
        ctx.set_tuning(which, 0)
    ctx.close()


if __name__ == "__main__":
    main()
