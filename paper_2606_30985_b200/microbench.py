"""Kernel microbenchmarks of BASELINE config 3:

    python -m paper_2606_30985_b200.microbench [--chi 40] [--what permute,inmethod,qr,gemm] [--json out.json]

* ``permute``: rank-5 fp64 tensor (4,chi,chi,chi,chi) C-order = column-major dims
  (chi,chi,chi,chi,4), iid N(0,1) seed 1, all 120 axis permutations; algorithmic bytes = 2 x 8 x
  elements; three src/dst buffer pairs are rotated so the working set exceeds the L2.
* ``inmethod``: the permutations Algorithm 1 itself issues (cut = U / D / L and their inverses,
  rank 5 / 4 / 3), fused with the diagonal absorb scaling as in the Trotter step.
* ``qr``: Gram / Cholesky-QR of tall-skinny N(0,1) matrices 256000 x 40, 256000 x 160, 64000 x 160.
* ``gemm``: the reconstruction GEMM shape cv (m x n) times W (n x n).

Timing: CUDA events on the launch stream, 3 warm-ups, median of ``--reps`` repetitions.
Peaks: MEASURED_PEAKS.json (hbm_gbs) when present.  This module only calls the C ABI through
``binding``; it holds no arithmetic of the method.
"""
from __future__ import annotations

import argparse
import itertools
import json
import os
import statistics

import torch

from . import binding as B
from . import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f)["hbm_gbs"], "measured"
    return 6650.0, "fallback"


def time_ms(fn, reps, warm=3, inner=6):
    """Median / min milliseconds of one fn(i) call.  `inner` calls are captured into a CUDA graph
    and replayed, so the CPU-side launch cost of the ctypes binding (tens of microseconds, more
    than some of these kernels take) stays out of the measurement."""
    for i in range(warm):
        fn(i)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        for i in range(inner):
            fn(i)
    g.replay()
    torch.cuda.synchronize()
    ts = []
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        g.replay()
        e1.record()
        e1.synchronize()
        ts.append(e0.elapsed_time(e1) / inner)
    return statistics.median(ts), min(ts)


def bench_permute(chi, reps, dev):
    shape = [chi, chi, chi, chi, 4]             # column-major dims of the C-order (4,chi,chi,chi,chi)
    n = 4 * chi ** 4
    host = torch.from_numpy(inputs.normal_tensor(shape, 1))
    nbuf = max(3, int(3 * 130e6 / (16 * n)) + 1)   # rotate: working set > L2 (126 MB)
    srcs = [host.to(dev) for _ in range(nbuf)]
    dsts = [torch.empty(n, dtype=torch.float64, device=dev) for _ in range(nbuf)]
    peak, src_peak = hbm_peak()
    rows = []
    for perm in itertools.permutations(range(5)):
        med, mn = time_ms(lambda i: B.permute(srcs[i % nbuf], shape, perm, dst=dsts[i % nbuf]), reps)
        gbs = 16.0 * n / med * 1e-6
        rows.append({"perm": list(perm), "ms": med, "ms_min": mn, "gbs": gbs, "frac": gbs / peak})
    fr = sorted(r["frac"] for r in rows)
    return {"shape_colmajor": shape, "bytes": 16 * n, "buffers_rotated": nbuf, "peak_gbs": peak, "peak_source": src_peak,
            "n_perms": len(rows), "frac_min": fr[0], "frac_median": fr[len(fr) // 2], "frac_max": fr[-1],
            "n_ge_70pct": sum(f >= 0.7 for f in fr), "rows": rows}


def inmethod_cases(chi):
    """(name, column-major shape, perm) of the a4 permutations and their a11 inverses."""
    out = []
    for deg in (4, 3, 2):
        rank = deg + 1
        shape = [chi] * deg + [4]
        for cut in range(deg - 1):          # cut leg already last -> no permutation
            perm = [l for l in range(deg) if l != cut] + [cut, deg]
            inv = [perm.index(j) for j in range(rank)]
            out.append(("deg%d cut leg %d" % (deg, cut), shape, perm))
            out.append(("deg%d cut leg %d inverse" % (deg, cut), [shape[p] for p in perm], inv))
    return out


def bench_inmethod(chi, reps, dev):
    peak, _ = hbm_peak()
    rows = []
    for name, shape, perm in inmethod_cases(chi):
        n = 1
        for s in shape:
            n *= s
        nbuf = min(8, max(3, int(3 * 130e6 / (16 * n)) + 1))
        srcs = [torch.randn(n, dtype=torch.float64, device=dev) for _ in range(nbuf)]
        dsts = [torch.empty(n, dtype=torch.float64, device=dev) for _ in range(nbuf)]
        scale = [torch.rand(s, dtype=torch.float64, device=dev) + 0.5 if (d < len(shape) - 1) else None
                 for d, s in enumerate(shape)]
        for scaled in (False, True):
            med, mn = time_ms(lambda i: B.permute(srcs[i % nbuf], shape, perm, dst=dsts[i % nbuf],
                                                  scale=scale if scaled else None), reps)
            gbs = 16.0 * n / med * 1e-6
            rows.append({"case": name + (" +absorb" if scaled else ""), "shape": shape, "perm": perm, "ms": med,
                         "gbs": gbs, "frac": gbs / peak})
    return {"chi": chi, "peak_gbs": peak, "rows": rows}


def bench_qr(reps, dev):
    rows = []
    for m, n in ((256000, 40), (256000, 160), (64000, 160), (216000, 240)):
        A = torch.from_numpy(inputs.normal_tensor((m, n), 1)).to(dev)
        ws = B._ws(B._lib.pepo_gram_ws_bytes(m, n), dev)
        med, _ = time_ms(lambda i: B.gram(A, m, n, ws=ws), reps)
        row = {"m": m, "n": n, "gram_ms": med, "gram_tflops_syrk": m * n * (n + 1) / med * 1e-9,
               "gram_gbs": 8.0 * m * n / med * 1e-6}
        Q = torch.empty(m * n, dtype=torch.float64, device=dev)
        ws2 = B._ws(B._lib.pepo_cholqr_ws_bytes(m, n), dev)
        med2, _ = time_ms(lambda i: B.cholqr(A, m, n, Q=Q, ws=ws2), reps)
        row.update({"cholqr_ms": med2, "cholqr_tflops": (m * n * (n + 1) + 2.0 * m * n * n) / med2 * 1e-9})
        rows.append(row)
    return {"rows": rows}


def bench_gemm(reps, dev):
    rows = []
    for m, n, k in ((216000, 240, 240), (3600, 240, 240), (256000, 160, 160)):
        A = torch.randn(m * k, dtype=torch.float64, device=dev)
        W = torch.randn(k * n, dtype=torch.float64, device=dev)
        Cc = torch.empty(m * n, dtype=torch.float64, device=dev)
        med, _ = time_ms(lambda i: B.dgemm(0, 0, m, n, k, A, m, W, k, Cout=Cc, ldc=m), reps)
        rows.append({"M": m, "N": n, "K": k, "ms": med, "tflops": 2.0 * m * n * k / med * 1e-9})
    return {"rows": rows}


def bench_site(chi, reps, dev):
    """The permute-on-load contractions of the bond gate on an interior site tensor (chi^4 x 4), every cut
    leg, next to the plain-layout kernels on the explicit cv of the same size (216000 x 240 at chi = 60)."""
    dims = [chi] * 4
    n, m = 4 * chi, chi ** 3
    nbuf = 3
    psis = [torch.randn(4 * chi ** 4, dtype=torch.float64, device=dev) for _ in range(nbuf)]
    outs = [torch.empty(4 * chi ** 4, dtype=torch.float64, device=dev) for _ in range(nbuf)]
    lam = [torch.rand(chi, dtype=torch.float64, device=dev) + 0.5 for _ in range(4)]
    W = torch.randn(n * n, dtype=torch.float64, device=dev)
    rows = []
    ws = B._ws(B._lib.pepo_gram_ws_bytes(m, n), dev)
    med, _ = time_ms(lambda i: B.gram(psis[i % nbuf], m, n, ws=ws), reps)
    rows.append({"kernel": "gram plain cv", "ms": med, "tflops": m * n * (n + 1) / med * 1e-9})
    med, _ = time_ms(lambda i: B.dgemm(0, 0, m, n, n, psis[i % nbuf], m, W, n, Cout=outs[i % nbuf], ldc=m), reps)
    rows.append({"kernel": "apply plain cv", "ms": med, "tflops": 2.0 * m * n * n / med * 1e-9})
    for cut in range(4):
        med, _ = time_ms(lambda i: B.site_gram(psis[i % nbuf], dims, cut, lam), reps)
        rows.append({"kernel": "site_gram cut leg %d (weighted)" % cut, "ms": med, "tflops": m * n * (n + 1) / med * 1e-9})
        med, _ = time_ms(lambda i: B.site_gram(psis[i % nbuf], dims, cut, None), reps)
        rows.append({"kernel": "site_gram cut leg %d (unweighted)" % cut, "ms": med, "tflops": m * n * (n + 1) / med * 1e-9})
        med, _ = time_ms(lambda i: B.site_apply(psis[i % nbuf], dims, cut, W, chi), reps)
        rows.append({"kernel": "site_apply cut leg %d" % cut, "ms": med, "tflops": 2.0 * m * n * n / med * 1e-9})
    return {"chi": chi, "rows": rows}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--chi", type=int, default=40)
    ap.add_argument("--chi-inmethod", type=int, default=60)
    ap.add_argument("--reps", type=int, default=20)
    ap.add_argument("--what", default="permute,inmethod,qr,gemm")
    ap.add_argument("--json", default=None)
    args = ap.parse_args()
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    out = {}
    what = args.what.split(",")
    if "permute" in what:
        out["permute"] = r = bench_permute(args.chi, args.reps, dev)
        print("permute (4,%d^4): %d perms, fraction of HBM peak %.0f GB/s: min %.2f median %.2f max %.2f, >=70%%: %d"
              % (args.chi, r["n_perms"], r["peak_gbs"], r["frac_min"], r["frac_median"], r["frac_max"], r["n_ge_70pct"]))
        for row in sorted(r["rows"], key=lambda x: x["frac"])[:12]:
            print("   slow: perm %s %.1f us %.0f GB/s (%.2f)" % (row["perm"], row["ms"] * 1e3, row["gbs"], row["frac"]))
    if "inmethod" in what:
        out["inmethod"] = r = bench_inmethod(args.chi_inmethod, args.reps, dev)
        for row in r["rows"]:
            print("in-method chi=%d %-32s perm %s %.1f us %.0f GB/s (%.2f)" % (r["chi"], row["case"], row["perm"],
                                                                            row["ms"] * 1e3, row["gbs"], row["frac"]))
    if "qr" in what:
        out["qr"] = r = bench_qr(args.reps, dev)
        for row in r["rows"]:
            print("gram %dx%d: %.3f ms %.1f TFLOP/s (SYRK count) %.0f GB/s | cholqr %.3f ms %.1f TFLOP/s"
                  % (row["m"], row["n"], row["gram_ms"], row["gram_tflops_syrk"], row["gram_gbs"], row["cholqr_ms"],
                     row["cholqr_tflops"]))
    if "gemm" in what:
        out["gemm"] = r = bench_gemm(args.reps, dev)
        for row in r["rows"]:
            print("dgemm %dx%dx%d: %.3f ms %.1f TFLOP/s" % (row["M"], row["N"], row["K"], row["ms"], row["tflops"]))
    if "site" in what:
        out["site"] = r = bench_site(args.chi_inmethod, args.reps, dev)
        for row in r["rows"]:
            print("site chi=%d %-36s %.3f ms %.1f TFLOP/s" % (r["chi"], row["kernel"], row["ms"], row["tflops"]))
    if args.json:
        with open(args.json, "w") as f:
            json.dump(out, f)


if __name__ == "__main__":
    main()
