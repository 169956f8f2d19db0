"""Run one of the BASELINE.json configurations end to end through the C ABI and print C(t):

    python -m paper_2606_30985_b200.run --config 2 [--steps N] [--chi CHI] [--json out.json]

configs (BASELINE.json "configs", 1-based; config 3 is the kernel microbenchmark, see
``python -m paper_2606_30985_b200.microbench``):
  1: 3x3, centre (1,1), chi_max 8, 10 steps, BP tol 1e-10, no damping
  2: 4x4, centre (1,1), chi_max 60, 60 steps, BP tol 1e-10, damping 0.5
  4: 8x8, centre (3,3), chi_max 60, 40 steps, BP tol 1e-9, damping 0.5
  5: 10x10, centre (4,4), chi_max = largest value whose memory model fits the free HBM
     (<= 100), 30 steps, BP tol 1e-8, damping 0.5
TFIM J = 1, h = 0.9, dt = 0.05, first-order Trotter (readings R1, R2).  Every step:
trotter_step, bp_converge, correlation; wall-clock per phase is measured with CUDA events.
"""
from __future__ import annotations

import argparse
import json
import time

import torch

from . import binding as B

CONFIGS = {
    1: dict(L=3, c=(1, 1), chi=8, steps=10, tol=1e-10, damping=0.0),
    2: dict(L=4, c=(1, 1), chi=60, steps=60, tol=1e-10, damping=0.5),
    4: dict(L=8, c=(3, 3), chi=60, steps=40, tol=1e-9, damping=0.5),
    5: dict(L=10, c=(4, 4), chi=100, steps=30, tol=1e-8, damping=0.5),
}


def fit_chi(L, chi_cap, free_bytes, inflight=0):
    """Largest chi_max <= chi_cap whose arena (analytic memory model) fits free_bytes."""
    for chi in range(chi_cap, 0, -1):
        need = B.arena_bytes(L, L, chi, inflight)
        if 0 < need <= free_bytes:
            return chi, need
    raise RuntimeError("no chi_max fits %d bytes" % free_bytes)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=1, choices=sorted(CONFIGS))
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--chi", type=int, default=None)
    ap.add_argument("--inflight", type=int, default=0)
    ap.add_argument("--json", default=None)
    ap.add_argument("--observe", action="store_true",
                    help="use pepo_observe with the alpha ladder (PAPER.md L451-L457) instead of bp_converge + correlation")
    ap.add_argument("--bp-init", type=int, default=None,
                    help="0 = uniform BP init (reading R7), 1 = leading Schmidt vector (R7b); default 0 for configs 1, 2 "
                         "and 1 for configs 4, 5, where the uniform init stops converging from step 22 (DESIGN.md 9.2)")
    ap.add_argument("--md", default=None, help="write the per-step table as markdown (profiles/cfgN_run.md)")
    args = ap.parse_args()
    cfg = dict(CONFIGS[args.config])
    if args.steps is not None:
        cfg["steps"] = args.steps
    if args.chi is not None:
        cfg["chi"] = args.chi
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    L = cfg["L"]
    free, total = torch.cuda.mem_get_info(dev)
    inflight = args.inflight
    if args.config == 5 and inflight == 0:
        inflight = 2
    chi, need = fit_chi(L, cfg["chi"], int(free * 0.985), inflight)
    if chi != cfg["chi"]:
        print("# chi_max %d does not fit %.1f GB free HBM; memory model picks chi_max = %d (%.1f GB)"
              % (cfg["chi"], free / 1e9, chi, need / 1e9), flush=True)
    free0, _ = torch.cuda.mem_get_info(dev)
    sim = B.Pepo(L, L, cfg["c"][0], cfg["c"][1], 1.0, 0.9, 0.05, chi, cfg["tol"], cfg["damping"], device=str(dev),
                 max_inflight=inflight)
    free1, _ = torch.cuda.mem_get_info(dev)
    if args.observe:
        sim.set_option("bp_ladder", 1)
    bp_init = args.bp_init if args.bp_init is not None else (1 if args.config in (4, 5) else 0)
    sim.set_option("bp_init", bp_init)
    rows = []
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    t_start = time.perf_counter()
    for step in range(1, cfg["steps"] + 1):
        ev[0].record()
        sim.trotter_step()
        ev[1].record()
        if args.observe:
            status, c, sweeps, stage = sim.observe()
            delta = sim.stats()["last_bp_delta"]
        else:
            status, sweeps, delta = sim.bp_converge()
            c = sim.correlation()
        ev[2].record()
        ev[2].synchronize()
        st = sim.stats()
        dims = sim.bond_dims()
        row = dict(step=step, C=c, trotter_ms=ev[0].elapsed_time(ev[1]), bp_ms=ev[1].elapsed_time(ev[2]),
                   bp_status=status, bp_sweeps=sweeps, bp_delta=delta, chi_min=min(dims), chi_max=max(dims),
                   gate_err=st["gate_err"], jacobi_sweeps=st["jacobi_sweeps"], n_cholesky=st["n_cholesky"],
                   n_householder=st["n_householder"], n_chol_failed=st["n_chol_failed"])
        rows.append(row)
        print("step %3d  C = % .12f  trotter %9.2f ms  bp %8.2f ms (%4d sweeps, status %d)  chi [%d, %d]  gate_err %.2e"
              % (step, c, row["trotter_ms"], row["bp_ms"], sweeps, status, row["chi_min"], row["chi_max"], st["gate_err"]),
              flush=True)
    wall = time.perf_counter() - t_start
    sim.check_guards()          # raises if any kernel wrote past one of the arena's buffers during the run
    st = sim.stats()
    sat = [r for r in rows if r["chi_min"] == chi]
    summary = dict(config=args.config, L=L, chi_max=chi, steps=cfg["steps"], wall_s=wall,
                   trotter_s=sum(r["trotter_ms"] for r in rows) * 1e-3, bp_s=sum(r["bp_ms"] for r in rows) * 1e-3,
                   steps_per_s_whole_run=cfg["steps"] / (sum(r["trotter_ms"] for r in rows) * 1e-3),
                   steps_per_s_saturated=(len(sat) / (sum(r["trotter_ms"] for r in sat) * 1e-3)) if sat else None,
                   arena_bytes=st["arena_high_water"], arena_model_bytes=st["arena_model_bytes"],
                   arena_tensor_bytes=int(sim.arena.numel()), mem_get_info_delta_bytes=int(free0 - free1),
                   hbm_total_bytes=int(total),
                   inflight_gates=st["max_inflight_gates"], kernel_launches=st["kernel_launches"])
    print("# " + json.dumps(summary), flush=True)
    if args.json:
        with open(args.json, "w") as f:
            json.dump(dict(summary=summary, rows=rows), f)
    if args.md:
        import sys
        with open(args.md, "w") as f:
            f.write("# BASELINE configs[%d] on one B200: %dx%d, chi_max %d, %d steps\n\n" % (args.config - 1, L, L, chi, cfg["steps"]))
            f.write("Command: `python -m paper_2606_30985_b200.run %s`\n\n" % " ".join(sys.argv[1:]))
            f.write("BP init: %s; %s.\n\n" % ("leading Schmidt vector e_0 (reading R7b)" if bp_init else "uniform (reading R7)",
                                             "pepo_observe with the alpha ladder" if args.observe else "pepo_bp_converge + pepo_correlation"))
            f.write("Memory: closed-form model %.3f GB, arena handed out %.3f GB, arena tensor %.3f GB, "
                    "torch.cuda.mem_get_info delta at allocation %.3f GB (of %.1f GB); %d gates in flight.\n\n"
                    % (summary["arena_model_bytes"] / 1e9, summary["arena_bytes"] / 1e9, summary["arena_tensor_bytes"] / 1e9,
                       summary["mem_get_info_delta_bytes"] / 1e9, summary["hbm_total_bytes"] / 1e9, summary["inflight_gates"]))
            f.write("Trotter time %.2f s, BP + Bethe time %.2f s, wall %.2f s; %.2f Trotter steps/s over the whole run%s; "
                    "%d kernel launches; arena guard zones intact after the run (pepo_check_guards).\n\n" % (summary["trotter_s"], summary["bp_s"], summary["wall_s"],
                                                 summary["steps_per_s_whole_run"],
                                                 (", %.2f over the saturated steps" % summary["steps_per_s_saturated"])
                                                 if summary["steps_per_s_saturated"] else "", summary["kernel_launches"]))
            f.write("| step | C(t) | BP status | BP sweeps | BP delta | chi min..max | gate_err | Jacobi sweeps | Cholesky / Householder QRs (cumulative) | rejected | Trotter ms | BP ms |\n")
            f.write("|---|---|---|---|---|---|---|---|---|---|---|---|\n")
            for r in rows:
                f.write("| %d | %.12f | %d | %d | %.2e | %d..%d | %.3e | %d | %d / %d | %d | %.2f | %.2f |\n"
                        % (r["step"], r["C"], r["bp_status"], r["bp_sweeps"], r["bp_delta"], r["chi_min"], r["chi_max"],
                           r["gate_err"], r["jacobi_sweeps"], r["n_cholesky"], r["n_householder"], r["n_chol_failed"],
                           r["trotter_ms"], r["bp_ms"]))
    sim.close()


if __name__ == "__main__":
    main()
