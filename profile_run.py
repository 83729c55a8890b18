"""One call of every timed entry point between cudaProfilerStart/Stop, for ncu captures of single kernels.

    ncu --set full --clock-control none --import-source on --profile-from-start off -o out \\
        python profile_run.py --workload Large

Warm-up steps run first (unprofiled), so the profiled launches see the evolved state `bench.py` times.  The order of
the profiled calls is: lcs_step_fused, lcs_particle_step, lcs_migrate, lcs_step_rk2 (with --rk2), lcs_set_fluid,
lcs_pair_count, lcs_set_particles (with --set-particles).  Nothing here is a measurement: times taken under a
profiler are never bench values.
"""
from __future__ import annotations

import argparse
import os
import sys

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

F8 = ("x", "y", "z", "vx", "vy", "vz", "d", "id")


def main() -> int:
    import numpy as np
    import torch
    from workloads import gen
    from paper_2604_11008_b200 import LCS

    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="Large")
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--rk2", action="store_true")
    ap.add_argument("--set-particles", action="store_true")
    ap.add_argument("--only", default="", help="comma list of: fused,push,migrate,rk2,set_fluid,pair_count,set_particles")
    a = ap.parse_args()
    only = set(x for x in a.only.split(",") if x)
    want = lambda k: not only or k in only
    cfg = gen.get_config(a.workload)
    wl = gen.make_workload(cfg, device="cuda:0")
    lcs = LCS(cfg["N"], *cfg["P"], cfg["capacity"], g=cfg["g"], rk2=a.rk2, device="cuda:0")
    lcs.set_fluid(wl["u"], wl["v"], wl["w"])
    lcs.set_particles(*(wl["particles"][k] for k in F8))
    dt = cfg["dt"]
    for _ in range(a.warmup):
        lcs.step_fused(dt)
    torch.cuda.synchronize()
    torch.cuda.profiler.start()
    if want("fused"):
        lcs.step_fused(dt)
    if want("push") or want("migrate"):
        lcs.particle_step(dt)
        lcs.migrate()
    if a.rk2 and want("rk2"):
        d_min = float(torch.min(wl["particles"]["d"]).item())
        lcs.step_rk2(0.4 * 1000.0 * d_min * d_min / (18.0 * 1.5e-5))
    if want("set_fluid"):
        lcs.set_fluid(wl["u"], wl["v"], wl["w"])
    if want("pair_count"):
        lcs.pair_count(0.0, 2.0 * np.pi / cfg["N"] * 0.25)
    if a.set_particles and want("set_particles"):
        lcs.set_particles(*(wl["particles"][k] for k in F8))
    torch.cuda.synchronize()
    torch.cuda.profiler.stop()
    err, n_tot, n_mig = lcs.get_status()
    print(f"profile_run: {cfg['name']} status {err} total {n_tot} migrants of the last migration {n_mig}")
    lcs.close()
    return 0 if err == 0 else 1


if __name__ == "__main__":
    sys.exit(main())
