"""oracle/calibrate_dt.py -- TEST INFRASTRUCTURE.  Freezes dt of every config in workloads/configs.json.

BASELINE.json fixes dt through the migrant fraction ("dt chosen so that ~5 % of particles cross a
subdomain face per step").  Starting from the closed form of DESIGN.md section 5 (`dt_formula`), dt is
bisected on the ORACLE's first-step migrant fraction until it is within +-0.2 % (absolute) of `target_m`;
the measured fraction, the edge/corner share of the migrants and the sample used are recorded next to dt.
Only oracle/ and the input generators are called (no CUDA-path code).  Large configs use every k-th
particle with the full fluid field (the fraction of a strided sample is an unbiased estimate).

    python -m oracle.calibrate_dt [--configs Tiny Medium ...] [--max-sample 2097152] [--device cuda]
"""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
F8 = ("x", "y", "z", "vx", "vy", "vz", "d", "id")
FACES = (4, 10, 12, 14, 16, 22)


def first_step(cfg, fluid, parts, dt):
    from oracle import oracle as orc
    P = cfg["P"][0] * cfg["P"][1] * cfg["P"][2]
    n = parts["id"].size
    o = orc.Oracle(cfg["N"], *cfg["P"], int(2 * (3 * n // P + 2048)), g=cfg["g"])   # roomy: only the fraction matters
    o.set_fluid(*fluid)
    assert o.set_particles(*(parts[k] for k in F8)) == 0
    rc = o.push(dt)
    tab = o.cnt_table().sum(axis=0)
    o.close()
    mig = tab.copy()
    mig[13] = 0
    m = mig.sum() / n
    edge = (mig.sum() - mig[list(FACES)].sum()) / max(1, mig.sum())
    return rc, float(m), float(edge)


def calibrate(cfg, device, max_sample, tol=0.002):
    from workloads import gen
    wl = gen.make_workload(cfg, device=device)
    fluid = [wl[k].cpu().numpy() for k in "uvw"]
    stride = max(1, cfg["n"] // max_sample)
    parts = {k: wl["particles"][k][::stride].contiguous().cpu().numpy() for k in F8}
    del wl
    dt = cfg["dt_formula"]
    rc, m, edge = first_step(cfg, fluid, parts, dt)
    lo, hi = (dt, None) if m < cfg["target_m"] else (None, dt)
    it = 0
    while abs(m - cfg["target_m"]) > tol and it < 30:
        if lo is None:
            dt = hi * 0.8
        elif hi is None:
            dt = lo * 1.25
        else:
            dt = 0.5 * (lo + hi)
        rc, m, edge = first_step(cfg, fluid, parts, dt)
        if m < cfg["target_m"]:
            lo = dt
        else:
            hi = dt
        it += 1
    return {"dt": float(f"{dt:.6g}"), "measured_m": round(m, 5), "edge_corner_share": round(edge, 4),
            "jump_status": rc, "calibration_sample": f"every {stride}th particle ({parts['id'].size}), full {cfg['N']}^3 field"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", nargs="*", default=None)
    ap.add_argument("--max-sample", type=int, default=1 << 21)
    ap.add_argument("--device", default="cpu")
    ap.add_argument("--out", default=os.path.join(ROOT, "workloads", "configs.json"))
    args = ap.parse_args()
    path = os.path.join(ROOT, "workloads", "configs.json")
    with open(path) as f:
        doc = json.load(f)
    for cfg in doc["configs"]:
        if args.configs and cfg["name"] not in args.configs:
            continue
        res = calibrate(dict(cfg), args.device, args.max_sample)
        print(cfg["name"], res, flush=True)
        cfg.update(res)
    with open(args.out, "w") as f:
        f.write("{\n \"_comment\": " + json.dumps(doc["_comment"]) + ",\n \"configs\": [\n")
        f.write(",\n".join("  " + json.dumps(c) for c in doc["configs"]))
        f.write("\n ]\n}\n")


if __name__ == "__main__":
    main()
