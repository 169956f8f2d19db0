#!/usr/bin/env python
"""bench.py - Trotter steps/s of the B200-native PEPO hot path (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload physical|synthetic] [--grid 4] [--chi 60]

One "step" = one pass of the whole hot path:
pepo_trotter_step (field gate + 4 colour classes of bond gates) + pepo_bp_converge +
pepo_correlation.  Workload at N=1: BASELINE configs[1], the 4x4 grid at chi_max = 60 with
every bond saturated.  `--workload physical` (default) reaches that state by running the real
dynamics from the product operator (untimed preparation) and then times the next K steps;
`--workload synthetic` loads the seeded random saturated state of SURVEY.md 8(d)(iii).
Prints ONE JSON line (contract in the task statement).  N > 1: independent replicas, one per
GPU, no collective on the data path ("replicas only").
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

J, H, DT = 1.0, 0.9, 0.05
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the class's main kernel on the 4x4 chi=60
# saturated state, from the `ncu --set full` captures summarised in profiles/r2_ncu_top_kernels.md (bytes; None =
# not captured).  Launch shapes: svd = one core of 240^2; apply_gemm = gathered reconstruction of one interior site
# (216000 x 240 x 240, algorithmic 829.4e6); gram = gathered weighted Gram of one interior site (algorithmic 414.7e6
# + 17 MB of split-K partials); permute = round 1's capture of one 4 x 60^4 interior tensor; bp = partial sweep
# over all 16 pinned slabs (algorithmic 428.4e6).
NCU_TRAFFIC_4x4_CHI60 = {"svd": 0.53e6, "apply_gemm": 792.2e6, "permute": 784.1e6, "bp": 433.7e6, "gram": 434.9e6}
FP64_NOMINAL_RATIO = 45.0 / 2250.0     # B200 fp64 tensor / bf16 tensor, blackwell guide table


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="physical", choices=["physical", "synthetic"])
    ap.add_argument("--grid", type=int, default=4)
    ap.add_argument("--cx", type=int, default=1)
    ap.add_argument("--cy", type=int, default=1)
    ap.add_argument("--chi", type=int, default=60)
    ap.add_argument("--prep-max", type=int, default=60, help="max untimed preparation steps")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-config3", action="store_true", help="skip the BASELINE configs[2] kernel microbenchmarks")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--bp-tol", type=float, default=1e-10)
    ap.add_argument("--bp-damping", type=float, default=0.5)
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=VALUE",
                    help="pepo_set_option tunable (repeatable), e.g. svd_min_cluster=8")
    return ap.parse_args()


# ---------------------------------------------------------------------------------------------
# clocks: sample nvidia-smi DURING the timed region
# ---------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([t.strip() for t in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for k, nm in enumerate(names):
                if len(r) > 3 + k and r[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return {"hbm_gbs": p["hbm_gbs"], "bf16_tflops": p["bf16_tflops"],
                "bf16_tflops_sustained": p.get("bf16_tflops_sustained", p["bf16_tflops"]), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}


# ---------------------------------------------------------------------------------------------
# workload preparation (GPU arm)
# ---------------------------------------------------------------------------------------------
def load_synthetic(sim, L, chi):
    from paper_2606_30985_b200 import inputs
    chis, psi, lam = inputs.synthetic_state(L, L, chi)
    sim.set_bond_dims(chis)
    for e, l in enumerate(lam):
        sim.set_lambda(e, l)
    for v, t in psi.items():
        sim.set_site(v % L, v // L, t)
    return chis, psi, lam


def prepare(sim, args):
    """Bring the context to the saturated state the metric is quoted on.  Returns a dict that
    describes what was done (untimed)."""
    L, chi = args.grid, args.chi
    if args.workload == "synthetic":
        load_synthetic(sim, L, chi)
        return {"prep": "synthetic saturated state (SURVEY 8(d)(iii))"}
    n = 0
    while n < args.prep_max and min(sim.bond_dims()) < chi:
        sim.trotter_step()
        n += 1
    if min(sim.bond_dims()) < chi:
        raise RuntimeError("bonds did not saturate in %d preparation steps: %s" % (n, sim.bond_dims()))
    return {"prep": "%d physical Trotter steps from the product operator (all bonds = %d)" % (n, chi),
            "prep_steps": n}


def fp64_yardsticks(torch, B, dev):
    """fp64 peaks measured in THIS run: (i) a register-only DMMA.8x8x4 loop through the
    library's own pepo_dmma_peak (the instruction every GEMM of the path is built on); (ii) torch.matmul
    fp64 8192^3 (cuBLAS) as an outside yardstick only - nothing on the hot path calls it."""
    sink = torch.zeros(1, dtype=torch.float64, device=dev)
    best = 0.0
    for cps in (1, 2, 4):
        B.dmma_peak(2000, cps, sink)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        fl = B.dmma_peak(20000, cps, sink)
        e1.record()
        e1.synchronize()
        best = max(best, fl / e0.elapsed_time(e1) * 1e-9)
    n = 8192
    a = torch.randn(n, n, dtype=torch.float64, device=dev)
    b = torch.randn(n, n, dtype=torch.float64, device=dev)
    torch.matmul(a, b)
    torch.cuda.synchronize()
    ts = []
    for _ in range(3):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        torch.matmul(a, b)
        e1.record()
        e1.synchronize()
        ts.append(e0.elapsed_time(e1))
    del a, b
    torch.cuda.empty_cache()
    return {"dmma_loop_tflops": best, "torch_matmul_fp64_8192_tflops": 2.0 * n ** 3 / min(ts) * 1e-9}


def config3_numbers(torch, dev, fp64_peak):
    """BASELINE configs[2] (the metric's 'permute GB/s and Gram fp64 TFLOP/s vs peak'): all 120 permutations of
    the (4,40,40,40,40) tensor, Gram / Cholesky-QR of 256000 x 160 and 256000 x 40 (Gram, the triangular
    solve as Q = A R^-1 GEMM, and POTRF + triangular inverse by difference), graph-replayed, rotated buffers."""
    from paper_2606_30985_b200 import microbench as mb
    from paper_2606_30985_b200 import binding as B
    from paper_2606_30985_b200 import inputs
    pm = mb.bench_permute(40, 5, dev)
    slow = sorted(pm["rows"], key=lambda r: r["frac"])[:5]
    out = {"permute_4x40^4": {"bytes_per_permute": pm["bytes"], "peak_gbs": pm["peak_gbs"], "n_perms": pm["n_perms"],
                              "gbs_min": min(r["gbs"] for r in pm["rows"]), "gbs_median": sorted(r["gbs"] for r in pm["rows"])[60],
                              "gbs_max": max(r["gbs"] for r in pm["rows"]), "frac_min": pm["frac_min"],
                              "frac_median": pm["frac_median"], "n_ge_70pct": pm["n_ge_70pct"],
                              "slowest": [{"perm": r["perm"], "frac": r["frac"]} for r in slow]}}
    qr = []
    for m, n in ((256000, 160), (256000, 40)):
        A = torch.from_numpy(inputs.normal_tensor((m, n), 1)).to(dev)
        ws = B._ws(B._lib.pepo_gram_ws_bytes(m, n), dev)
        t_gram, _ = mb.time_ms(lambda i: B.gram(A, m, n, ws=ws), 8)
        Q = torch.empty(m * n, dtype=torch.float64, device=dev)
        ws2 = B._ws(B._lib.pepo_cholqr_ws_bytes(m, n), dev)
        t_qr, _ = mb.time_ms(lambda i: B.cholqr(A, m, n, Q=Q, ws=ws2), 8)
        Rinv = torch.randn(n * n, dtype=torch.float64, device=dev)
        t_trsm, _ = mb.time_ms(lambda i: B.dgemm(0, 0, m, n, n, A, m, Rinv, n, Cout=Q, ldc=m), 8)
        syrk = m * n * (n + 1) / t_gram * 1e-9
        qr.append({"m": m, "n": n, "gram_ms": t_gram, "gram_tflops_syrk": syrk, "gram_frac_of_fp64_peak": syrk / fp64_peak,
                   "gram_gbs": 8.0 * m * n / t_gram * 1e-6, "trsm_as_gemm_ms": t_trsm,
                   "trsm_tflops": 2.0 * m * n * n / t_trsm * 1e-9, "cholqr_ms": t_qr,
                   "potrf_plus_trtri_ms_by_difference": max(t_qr - t_gram - t_trsm, 0.0)})
        del A, Q
    out["cholesky_qr"] = qr
    torch.cuda.empty_cache()
    return out


def one_step(sim):
    sim.trotter_step()
    status, sweeps, delta = sim.bp_converge()
    c = sim.correlation()
    return c, status, sweeps


def run_ours(args):
    import torch
    from paper_2606_30985_b200 import binding as B
    from paper_2606_30985_b200 import replicas as R

    world, rank, local = R.world()
    dev = torch.device("cuda", local)
    torch.cuda.set_device(dev)
    R.init("nccl", dev)
    L, chi = args.grid, args.chi
    yard = fp64_yardsticks(torch, B, dev)
    sim = B.Pepo(L, L, args.cx, args.cy, J, H, DT, chi, args.bp_tol, args.bp_damping, device=str(dev))
    for kv in args.opt:
        k, v = kv.split("=")
        sim.set_option(k, float(v))
    info = prepare(sim, args)

    def barrier():
        R.barrier(dev)

    # ---- device-resident timing ---------------------------------------------------------------
    for _ in range(args.warmup):
        one_step(sim)
    # the timed region runs uninstrumented (what a user of the library gets); the per-kernel CUDA
    # events (two records around every launch group, ~1000 per step) are taken in the same loop run
    # once more right after it (kernels_overlapped) and on the serial schedule (kernels, rooflines)
    launches0 = sim.stats()["kernel_launches"]
    sampler = ClockSampler(local)
    barrier()
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_trot, sweeps_tot, jac = 0.0, 0, 0
    ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    c_last = None
    for _ in range(args.steps):
        ea.record()
        sim.trotter_step()
        eb.record()
        status, sweeps, delta = sim.bp_converge()
        c_last = sim.correlation()
        t_trot += ea.elapsed_time(eb)        # bp_converge synchronised the stream
        sweeps_tot += sweeps
        jac += sim.stats()["jacobi_sweeps"]
    e1.record()
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms = e0.elapsed_time(e1)
    launches = sim.stats()["kernel_launches"] - launches0
    ms = R.max_over_ranks(ms, dev)
    stats = sim.stats()
    sim.set_option("profile", 2)
    ei0, ei1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ei0.record()
    for _ in range(args.steps):
        one_step(sim)
    ei1.record()
    torch.cuda.synchronize()
    ms_instrumented = ei0.elapsed_time(ei1)
    prof_overlapped = sim.profile()
    sim.set_option("profile", 0)
    # per-kernel durations with the GPU to itself: PROF_STEPS more steps on the serial schedule
    # (pipeline = 0) right after the timed region.  In the timed region the default schedule runs
    # the pieces of a colour class on several streams, so a kernel's event-to-event time there
    # includes the SMs it shared with concurrent kernels (reported as kernels_overlapped).
    pipe = 4
    for kv in args.opt:
        if kv.startswith("pipeline="):
            pipe = int(float(kv.split("=")[1]))
    PROF_STEPS = 2
    sim.set_option("pipeline", 0)
    sim.set_option("profile", 2)
    for _ in range(PROF_STEPS):
        one_step(sim)
    prof = sim.profile()
    sim.set_option("profile", 0)
    sim.set_option("pipeline", pipe)

    # ---- end-to-end: host buffers in, host scalar out, copies inside the timed region ----------
    e2e = None
    if not args.no_e2e:
        host = {}
        for y in range(L):
            for x in range(L):
                a = sim.get_site(x, y)
                p = torch.empty(a.size, dtype=torch.float64).pin_memory()
                p.numpy()[:] = a
                host[(x, y)] = p
        lam = [sim.get_lambda(e) for e in range(sim.n_bonds)]
        chis = sim.bond_dims()
        h2d = sum(p.numel() * 8 for p in host.values()) + sum(l.size * 8 for l in lam)

        order = sim.site_order()       # the order in which the step first touches the sites

        def e2e_step():
            sim.set_bond_dims(chis)
            for e, l in enumerate(lam):
                sim.set_lambda(e, l)
            for (x, y) in order:
                sim.set_site_async(x, y, host[(x, y)].numpy())   # pinned -> device on the copy stream
            return one_step(sim)

        for _ in range(max(1, args.warmup // 2)):
            e2e_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            e2e_step()
        barrier()
        dt_e2e = time.perf_counter() - t0
        dt_e2e = R.max_over_ranks(dt_e2e, dev)
        e2e = {"value": world * args.steps / dt_e2e, "unit": "Trotter steps/s",
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": 8 + 8 + 4 * sim.n_bonds,
               "note": "state uploaded from pinned host memory every step (pepo_set_site_async: the step starts on "
                       "the sites that have arrived), C(t) read back"}

    peaks = measured_peaks()
    # dominant kernel class by accumulated device time
    dom = max(prof, key=lambda k: prof[k]["ms"])
    fp64_peak = peaks["bf16_tflops_sustained"] * FP64_NOMINAL_RATIO
    def per_kernel(pr, nsteps):
        out = {}
        tot = sum(v["ms"] for v in pr.values())
        for k, v in pr.items():
            if v["count"] == 0:
                continue
            out[k] = {"ms_per_step": v["ms"] / nsteps, "share": v["ms"] / max(tot, 1e-9),
                      "launch_groups_per_step": v["count"] / nsteps}
            if v["flops"] > 0 and v["ms"] > 0:
                out[k]["tflops"] = v["flops"] / v["ms"] * 1e-9
            if v["bytes"] > 0 and v["ms"] > 0:
                out[k]["gbs"] = v["bytes"] / v["ms"] * 1e-6
        return out

    per = per_kernel(prof, PROF_STEPS)
    per_overlapped = per_kernel(prof_overlapped, args.steps)
    unit_peak = 148 * 64 * 2 * 1.965e9 * 1e-12    # fp64: 148 SMs x 64 FMA/clk x 2 x 1.965 GHz (unit count, context only)
    alu_peak = yard["dmma_loop_tflops"]           # measured in this run: the denominator of every fp64 fraction
    peak_txt = ("fp64 tensor (DMMA.8x8x4) rate measured in this run by a register-only loop (pepo_dmma_peak): %.1f TF/s; "
                "torch.matmul fp64 8192^3 (cuBLAS, yardstick only) in the same run: %.1f TF/s; unit count 148 SMs x 64 "
                "FMA/clk x 2 x 1.965 GHz = %.1f TF/s; MEASURED_PEAKS bf16 sustained %.0f x 45/2250 (guide's nominal ratio) "
                "= %.1f TF/s" % (alu_peak, yard["torch_matmul_fp64_8192_tflops"], unit_peak,
                                 peaks["bf16_tflops_sustained"], fp64_peak))

    def roof_of(k):
        d = prof[k]
        if d["count"] == 0 or d["ms"] <= 0:
            return None
        if k in ("gram", "apply_gemm", "small_gemm"):
            ach = d["flops"] / d["ms"] * 1e-9
            return {"kernel": k, "bound": "tensor", "achieved": ach, "peak": alu_peak, "unit": "TFLOP/s",
                    "frac": ach / alu_peak, "traffic": None, "peak_source": peak_txt}
        if k in ("permute", "field", "bp"):
            ach = d["bytes"] / d["ms"] * 1e-6
            return {"kernel": k, "bound": "hbm", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                    "frac": ach / peaks["hbm_gbs"], "traffic": None, "peak_source": "hbm_gbs of " + peaks["source"]}
        if k == "svd":
            ach = d["flops"] / d["ms"] * 1e-9
            return {"kernel": k, "bound": "alu", "achieved": ach, "peak": alu_peak, "unit": "TFLOP/s",
                    "frac": ach / alu_peak, "traffic": None,
                    "peak_source": "fp64 DFMA rate = the DMMA rate measured in this run (%.1f TF/s; B200 has one fp64 "
                                   "datapath); the Jacobi iteration is latency-bound (one cluster of 8 SMs per core, "
                                   "DESIGN.md 6.3), flops = sweeps x Nc(Nc-1)/2 pairs x 12 L" % alu_peak}
        return None

    rooflines = {k: r for k in prof for r in [roof_of(k)] if r is not None}
    if (L, chi) == (4, 60):
        for k, r in rooflines.items():
            r["traffic"] = NCU_TRAFFIC_4x4_CHI60.get(k)
    roof = dict(rooflines.get(dom) or {"kernel": dom, "bound": "alu", "achieved": None, "peak": alu_peak,
                                       "unit": "TFLOP/s", "frac": None, "traffic": None,
                                       "peak_source": "latency-bound small dense kernel"})
    # classes within 10 % of the dominant one are named beside it (the SVD and the two tall GEMMs are close)
    co = [k for k in prof if k != dom and prof[k]["ms"] >= 0.9 * prof[dom]["ms"] and k in rooflines]
    roof["co_dominant"] = [{"kernel": k, "bound": rooflines[k]["bound"], "achieved": rooflines[k]["achieved"],
                            "peak": rooflines[k]["peak"], "unit": rooflines[k]["unit"], "frac": rooflines[k]["frac"]} for k in co]
    # whole-step view: algorithmic flops of a saturated step (SYRK Gram m n^2 + reconstruction
    # 2 m n^2 per site and gate, n = 4 chi) over the measured Trotter time
    step_flops = 0.0
    for y in range(L):
        for x in range(L):
            deg = (y > 0) + (y < L - 1) + (x > 0) + (x < L - 1)
            step_flops += deg * 3.0 * chi ** (deg - 1) * (4.0 * chi) ** 2
    whole = {"algorithmic_flops_per_step": step_flops, "tflops": step_flops / (t_trot / args.steps) * 1e-9,
             "frac_of_fp64_peak": step_flops / (t_trot / args.steps) * 1e-9 / alu_peak,
             "note": "3 m n^2 per site and gate over the Trotter time of the timed region"}
    line = {
        "metric": "Trotter steps/sec (4x4 chi=60 fp64)" if (L, chi) == (4, 60) else "Trotter steps/sec (%dx%d chi=%d fp64)" % (L, L, chi),
        "value": world * args.steps / (ms * 1e-3), "unit": "Trotter steps/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64",
        "data": ("synthetic (parameter-defined workload: product operator evolved by the method itself, no dataset)"
                 if args.workload == "physical" else "synthetic (seeded random saturated state, SURVEY 8(d)(iii))"),
        "config": {"workload": "BASELINE configs[1]: %dx%d open grid, TFIM J=1 h=0.9 dt=0.05, Z at (%d,%d), chi_max=%d, "
                               "all bonds saturated; step = trotter_step + bp_converge(tol %g, damping %g) + correlation"
                               % (L, L, args.cx, args.cy, chi, args.bp_tol, args.bp_damping),
                   "state": info["prep"], "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": "working set per step (%.1f GB of site tensors) exceeds the 126 MB L2" % (stats["arena_high_water"] / 1e9),
                   "schedule": "pipeline=%d piece streams in the timed region (0 = serial)" % pipe,
                   "rooflines": "per-kernel durations (kernels, roofline, rooflines) from %d extra steps on the serial "
                                "schedule right after the timed region, CUDA events on the launching stream; "
                                "kernels_overlapped = the same event pairs over the timed loop run once more with the "
                                "events on (%.2f ms per step against %.2f uninstrumented), where kernels of different "
                                "streams share the SMs" % (PROF_STEPS, ms_instrumented / args.steps, ms / args.steps)},
        "trotter_only_steps_per_s": world * args.steps / (t_trot * 1e-3),
        "trotter_ms_per_step": t_trot / args.steps,
        "bp_sweeps_per_step": sweeps_tot / args.steps, "jacobi_sweeps_per_step": jac / args.steps,
        "last_C": c_last, "gate_err_last_step": stats["gate_err"],
        "qr": {"cholesky": stats["n_cholesky"], "householder": stats["n_householder"], "chol_rejected": stats["n_chol_failed"]},
        "gpu_launches": int(launches), "clocks": clocks, "roofline": roof, "rooflines": rooflines,
        "whole_step": whole, "fp64_yardsticks": yard, "kernels": per,
        "kernels_overlapped": per_overlapped,
        "arena": {"high_water_bytes": stats["arena_high_water"], "model_bytes": stats["arena_model_bytes"],
                  "inflight_gates": stats["max_inflight_gates"]},
        "e2e": e2e,
    }
    sim.close()
    del sim
    torch.cuda.empty_cache()
    if rank == 0 and world == 1 and not args.no_config3:
        line["config3"] = config3_numbers(torch, dev, alu_peak)
    return line, rank, world


# ---------------------------------------------------------------------------------------------
# CPU oracle arm (cpu_baseline leg and --impl reference): the oracle as it stands, timed on the
# host cores on a bounded sample of the same workload
# ---------------------------------------------------------------------------------------------
def oracle_state(L, chi, cx, cy):
    """Oracle PEPOState holding the seeded synthetic saturated state (same generator as the GPU
    arm's --workload synthetic)."""
    import numpy as np
    from oracle import pepo_oracle as po
    from paper_2606_30985_b200 import inputs
    st = po.PEPOState(L, L, cx, cy, J, H, DT, chi)
    chis, psi, lam = inputs.synthetic_state(L, L, chi)
    for v in range(L * L):
        x, y = v % L, v // L
        dims = [chis[inputs.bond_id(L, L, x, y, d)] for d in inputs.site_legs(L, L, x, y)] + [4]
        st.psi[v] = np.asarray(psi[v]).reshape(dims, order="F").copy()
    st.lam = [np.asarray(l) for l in lam]
    return st


def bond_classes(L):
    """Group the bonds of the LxL grid by the degrees of their two sites; returns
    {(deg1, deg2): [bond ids]} - gates of one class cost the same."""
    from oracle import pepo_oracle as po
    lat = po.Lattice(L, L)
    out = {}
    for e in range(lat.n_bonds):
        v1, _, v2, _ = lat.bond_sites(e)
        key = tuple(sorted((len(lat.legs(v1)), len(lat.legs(v2)))))
        out.setdefault(key, []).append(e)
    return out


def gate_flops(chi, key):
    """6 m n^2 per site (Householder QR + explicit Q + Q M), m = chi^(deg-1), n = 4 chi."""
    return sum(6.0 * chi ** (d - 1) * (4 * chi) ** 2 for d in key)


def oracle_sample(st, L, chi, budget_s, known=None):
    """Time the oracle's field gate and ONE oracle bond gate per bond class, cheapest class first, while
    the projected total stays within budget_s.  `known` = class times MEASURED by an earlier call of this
    function in the same process; a class that does not fit the budget takes its earlier measured time.
    Nothing is extrapolated by a flop model: with known = None every class is timed.
    Returns (seconds per full Trotter step, description, seconds spent, {class: measured seconds})."""
    classes = bond_classes(L)
    order = sorted(classes, key=lambda k: gate_flops(chi, k))
    timed, spent = {}, 0.0
    t0 = time.perf_counter()
    st.apply_field_gate()
    t_field = time.perf_counter() - t0
    spent += t_field
    for key in order:
        if known and key in known and spent + known[key] > budget_s:
            continue
        e = classes[key][0]
        t0 = time.perf_counter()
        st.apply_bond_gate(e)
        timed[key] = time.perf_counter() - t0
        spent += timed[key]
    total = t_field
    reused = []
    for key, bonds in classes.items():
        if key in timed:
            t = timed[key]
        else:
            t = known[key]
            reused.append(key)
        total += t * len(bonds)
    desc = ("field gate on all sites + one oracle bond gate (Algorithm 1, Householder QR, literal 16 chi core) timed for "
            "each of the bond classes %s of the %dx%d chi=%d synthetic saturated state (%.1f s of CPU work), step time = "
            "sum over classes of count x measured gate time%s; BP/Bethe not included"
            % (sorted(timed), L, L, chi, spent,
               ("; classes %s reuse their time measured earlier in this run" % sorted(reused)) if reused else ""))
    allt = dict(known or {})
    allt.update(timed)
    return total, desc, spent, allt


def host_threads():
    try:
        import threadpoolctl
        n = max((p.get("num_threads", 1) for p in threadpoolctl.threadpool_info()), default=1)
        return int(n)
    except Exception:
        return os.cpu_count() or 1


def single_thread_sample(st, L, chi, budget_s, all_thread_times):
    """The same gate timing with the BLAS limited to one thread, on the classes that fit budget_s
    (cheapest first); reports the measured single-thread / all-thread ratio of those classes."""
    try:
        import threadpoolctl
    except Exception:
        return None
    classes = bond_classes(L)
    out, spent = {}, 0.0
    with threadpoolctl.threadpool_limits(limits=1):
        for key in sorted(classes, key=lambda k: gate_flops(chi, k)):
            est = all_thread_times.get(key, 0.0) * 8.0
            if spent + est > budget_s:
                break
            t0 = time.perf_counter()
            st.apply_bond_gate(classes[key][0])
            out[key] = time.perf_counter() - t0
            spent += out[key]
    if not out:
        return None
    return {"classes_timed": [list(k) for k in sorted(out)], "gate_seconds_1_thread": {str(k): v for k, v in out.items()},
            "gate_seconds_all_threads": {str(k): all_thread_times[k] for k in out},
            "ratio_1_thread_over_all": sum(out.values()) / sum(all_thread_times[k] for k in out)}


def run_cpu_baseline(args):
    import numpy  # noqa: F401  (loads the BLAS whose threads are counted)
    st = oracle_state(args.grid, args.chi, args.cx, args.cy)
    total, desc, spent, times = oracle_sample(st, args.grid, args.chi, 1e9)
    one = single_thread_sample(st, args.grid, args.chi, 12.0, times)
    return {"value": 1.0 / total, "unit": "Trotter steps/s", "cores": host_threads(), "kind": "oracle",
            "sample": desc, "extrapolated": False, "single_thread": one}


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores, K timed 'steps' after W warm-ups.  The first
    (warm-up) step times one gate of EVERY bond class; each later step re-times, cheapest first, the
    classes that fit its share of a ~150 s budget and reuses the measured time of the others."""
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if rank != 0:
        return None, rank, world
    L, chi = args.grid, args.chi
    n_runs = max(2, args.steps + max(args.warmup, 1))
    budget = max(2.0, 150.0 / n_runs)
    st = oracle_state(L, chi, args.cx, args.cy)
    totals, desc, known = [], "", None
    n_warm = max(args.warmup, 1)
    for i in range(n_runs):
        total, desc, spent, known = oracle_sample(st, L, chi, 1e9 if known is None else budget, known)
        if i >= n_warm:
            totals.append(total)
    mean = sum(totals) / len(totals)
    val = 1.0 / mean
    line = {
        "impl": "reference",
        "metric": "Trotter steps/sec (4x4 chi=60 fp64)" if (L, chi) == (4, 60) else "Trotter steps/sec (%dx%d chi=%d fp64)" % (L, L, chi),
        "value": val, "unit": "Trotter steps/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": mean * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic (seeded random saturated state, SURVEY 8(d)(iii))",
        "config": {"workload": "BASELINE configs[1]: %dx%d open grid, TFIM J=1 h=0.9 dt=0.05, Z at (%d,%d), chi_max=%d, "
                               "all bonds saturated (seeded synthetic state); Trotter step only" % (L, L, args.cx, args.cy, chi)},
        "cpu_baseline": {"value": val, "unit": "Trotter steps/s", "cores": host_threads(), "kind": "oracle", "sample": desc,
                         "extrapolated": False},
        "e2e": {"value": val, "unit": "Trotter steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    return line, rank, world


def spawn_replicas(args):
    """`python bench.py --gpus N` without torchrun: start the N replica processes ourselves (one per GPU,
    NCCL rendezvous on 127.0.0.1) and pass their output through."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    args = parse()
    if args.impl == "ours" and args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return spawn_replicas(args)
    if args.impl == "reference":
        line, rank, world = run_reference(args)
        if line is not None:
            print(json.dumps(line), flush=True)
        return 0
    line, rank, world = run_ours(args)
    if rank == 0:
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = run_cpu_baseline(args)
        else:
            line["cpu_baseline"] = None
        print(json.dumps(line), flush=True)
    from paper_2606_30985_b200 import replicas as R
    R.finish()
    return 0


if __name__ == "__main__":
    sys.exit(main())
