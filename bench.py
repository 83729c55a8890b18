#!/usr/bin/env python
"""bench.py -- particles/s of the fused push + prefix-scan migrate step (BASELINE.json's metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload Large] [--impl reference]

One "step" = one lcs_step_fused over all resident particles of the workload (all of SURVEY.md
section 8(a): gather, advance, classify, count, scan, pack, compaction, unpack).  At N > 1 every
rank owns an independent periodic box of the same workload (weak scaling, no data-path collective;
DESIGN.md section 8).  Prints ONE JSON line on rank 0.

--impl reference times the oracle (oracle/, the plain sequential CPU statement of the same path)
on a bounded sample of the same workload on the host cores.
"""
from __future__ import annotations

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

METRIC = "particles/s (fused push + prefix-scan migrate step)"
F8 = ("x", "y", "z", "vx", "vy", "vz", "d", "id")
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "traffic.json")
KERNEL_SOURCES = [os.path.join(ROOT, "paper_2604_11008_b200", "csrc", f) for f in ("lcs_kernels.cuh", "lcs_api.cu")]


def kernel_source_hash():
    import hashlib
    h = hashlib.sha256()
    for f in KERNEL_SOURCES:
        with open(f, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def ncu_traffic(workload, kernel):
    """DRAM bytes per launch of `kernel` on `workload` from the committed ncu --set full capture listed in
    profiles/traffic.json (dram__bytes_read.sum + dram__bytes_write.sum).  The entry names the capture file and the hash
    of the kernel sources it was taken on; if the sources have changed since, the figure is stale and is NOT reported.
    -> (bytes or None, source string or None, stale flag)"""
    try:
        with open(TRAFFIC_FILE) as f:
            tab = json.load(f)
        e = tab[workload][kernel]
    except Exception:
        return None, None, False
    if e.get("kernel_source_sha256_16") != kernel_source_hash():
        return None, e.get("capture"), True
    return float(e["dram_bytes_read"]) + float(e["dram_bytes_write"]), e.get("capture"), False


def measured_peak_hbm():
    """(GB/s, source): MEASURED_PEAKS.json if present, else the fallback of B200_PROFILING.md."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """SM clock and throttle reasons sampled DURING the timed region: an NVML polling thread (a sample every ~2 ms; the
    timed region of the default run is under 100 ms, too short for nvidia-smi's loop mode), nvidia-smi as the fallback."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index):
        import threading
        self.sm, self.mx, self.reasons = [], [], set()
        self.p = self.f = self.thread = None
        self.stop_flag = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[index]) if vis and all(t.strip().isdigit() for t in vis.split(",")) else index
            h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            mx = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            bits = {"hw_slowdown": pynvml.nvmlClocksThrottleReasonHwSlowdown,
                    "hw_thermal_slowdown": pynvml.nvmlClocksThrottleReasonHwThermalSlowdown,
                    "sw_thermal_slowdown": pynvml.nvmlClocksThrottleReasonSwThermalSlowdown,
                    "sw_power_cap": pynvml.nvmlClocksThrottleReasonSwPowerCap}

            def poll():
                while not self.stop_flag.is_set():
                    try:
                        self.sm.append(float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)))
                        self.mx.append(mx)
                        r = pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                        for nm, bit in bits.items():
                            if r & bit:
                                self.reasons.add(nm)
                    except Exception:
                        pass
                    time.sleep(0.002)

            self.thread = threading.Thread(target=poll, daemon=True)
            self.thread.start()
            return
        except Exception as exc:
            print(f"bench.py: NVML polling unavailable ({exc!r}); falling back to nvidia-smi", file=sys.stderr)
            self.thread = None
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "20"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.thread is not None:
            self.stop_flag.set()
            self.thread.join(timeout=2)
        elif self.p is not None:
            self.p.terminate()
            try:
                self.p.wait(timeout=5)
            except Exception:
                self.p.kill()
            self.f.flush()
            self.f.seek(0)
            for line in self.f:
                t = [c.strip() for c in line.split(",")]
                if len(t) < 7:
                    continue
                try:
                    self.sm.append(float(t[0])); self.mx.append(float(t[1]))
                except ValueError:
                    continue
                for nm, v in zip(self.NAMES, t[3:7]):
                    if v.lower().startswith("active"):
                        self.reasons.add(nm)
            self.f.close()
            os.unlink(self.f.name)
        if self.sm:
            out.update(sm_mhz=float(np.median(self.sm)), sm_max_mhz=float(np.max(self.mx)), samples=len(self.sm))
        out["reasons"] = sorted(self.reasons)
        return out


def max_over_ranks(value, dist, device):
    """MAX of a python float over the ranks of the default process group (identity when dist is None)."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def pick_device():
    import torch
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return torch, rank, world, local


def build_workload(name, device):
    from workloads import gen
    cfg = gen.get_config(name)
    wl = gen.make_workload(cfg, device=device)
    return cfg, wl


def oracle_sample_rate(cfg, wl, stride, steps, torch):
    """Oracle (as it stands, single thread) on every `stride`-th particle of the workload with the
    full fluid field; -> (particles/s, seconds per step, sample size)."""
    from oracle import oracle as orc
    fluid = [wl[k].cpu().numpy() for k in "uvw"]
    parts = {k: wl["particles"][k][::stride].contiguous().cpu().numpy() for k in F8}
    n_s = parts["id"].size
    P = cfg["P"][0] * cfg["P"][1] * cfg["P"][2]
    cap = int(max(64, 2 * np.ceil(1.5 * n_s / P / 2) + 64))
    if cfg.get("clumps"):
        cap = int(max(cap, 2 * np.ceil(cfg["capacity"] / stride * 1.5 / 2) + 64))
    o = orc.Oracle(cfg["N"], *cfg["P"], cap, g=cfg["g"])
    o.set_fluid(*fluid)
    rc = o.set_particles(*(parts[k] for k in F8))
    if rc:
        raise RuntimeError(f"oracle set_particles -> {rc}")
    # one pinned core; push and migrate timed apart: a step is exactly these two calls
    old_aff = None
    try:
        old_aff = os.sched_getaffinity(0)
        os.sched_setaffinity(0, {max(old_aff)})
    except (AttributeError, OSError):
        old_aff = None
    t_push = t_mig = 0.0
    try:
        for _ in range(steps):
            t0 = time.perf_counter()
            rc = o.push(cfg["dt"])
            t1 = time.perf_counter()
            rc = rc or o.migrate()
            t2 = time.perf_counter()
            if rc:
                raise RuntimeError(f"oracle step -> {rc}")
            t_push += t1 - t0
            t_mig += t2 - t1
    finally:
        if old_aff is not None:
            os.sched_setaffinity(0, old_aff)
    dt = t_push + t_mig
    o.close()
    ORACLE_PHASES.update({"push": n_s * steps / t_push, "migrate": n_s * steps / t_mig, "step": n_s * steps / dt,
                          "pinned": old_aff is not None, "core_model": cpu_model(), "nproc": os.cpu_count()})
    return n_s * steps / dt, dt / steps, n_s


ORACLE_PHASES = {}      # filled by the last oracle_sample_rate call: particles/s per phase on the pinned core


def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.lower().startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def bench_config(cfg, args, world):
    """The `config` object of the JSON line: the workload as named, the same keys and values in both arms (the
    reference arm times a bounded sample of it and says which in `sample` / `cpu_baseline.sample`)."""
    return {"workload": cfg["name"], "N": cfg["N"], "P": cfg["P"], "particles_per_gpu": cfg["n"], "capacity": cfg["capacity"],
            "dt": cfg["dt"], "drag_model": args.drag_model, "particle_order": args.order,
            "l2": "inputs larger than L2 (no flush)",
            "parallelism": "independent box per GPU" if world > 1 else "single GPU"}


def run_reference(args):
    torch, rank, world, local = pick_device()
    if rank != 0:
        return 0
    dev = "cuda:0" if torch.cuda.is_available() else "cpu"   # the harness may synthesise inputs on a GPU
    cfg, wl = build_workload(args.workload, dev)
    stride = max(1, cfg["n"] // args.ref_sample)
    # untimed warm-up then K timed steps, each a bounded sample of the workload
    oracle_sample_rate(cfg, wl, stride * 8, max(1, min(args.warmup, 1)), torch)
    rate, sec, n_s = oracle_sample_rate(cfg, wl, stride, args.steps, torch)
    line = {
        "impl": "reference", "metric": METRIC, "value": rate, "unit": "particles/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": bench_config(cfg, args, world),
        "sample": {"particles_timed_per_step": n_s, "stride": stride},
        "cpu_baseline": {"value": rate, "unit": "particles/s", "cores": 1, "kind": "oracle",
                         "sample": f"every {stride}th particle of {cfg['name']} ({n_s} particles, full {cfg['N']}^3 field), "
                                   f"{args.steps} steps, single thread",
                         "phases": dict(ORACLE_PHASES)},
        "e2e": {"value": rate, "unit": "particles/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)
    return 0


def run_cuda(args):
    torch, rank, world, local = pick_device()
    if not torch.cuda.is_available():
        print("bench.py: no CUDA device; the CUDA path has no CPU fallback", file=sys.stderr)
        return 2
    from paper_2604_11008_b200 import LCS
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(dev))
    cfg, wl = build_workload(args.workload, dev)
    n, N = cfg["n"], cfg["N"]
    P = cfg["P"][0] * cfg["P"][1] * cfg["P"][2]
    # the RK2 group is 8 more arrays of P*capacity doubles: 34 GB at Stress, which the box cannot spare beside the inputs
    args.rk2 = bool(args.rk2) and args.phase_steps > 0 and cfg["name"] != "Stress"
    lcs = LCS(N, *cfg["P"], cfg["capacity"], g=cfg["g"], drag_model=args.drag_model, rk2=args.rk2, device=dev)
    lcs.set_fluid(wl["u"], wl["v"], wl["w"])
    parts = wl["particles"]
    if args.order == "morton":
        # labelled variant (never the headline): the same particles, handed over sorted by the Morton key of their cell, so
        # that the particles of a tile gather from neighbouring cells ("may be reported as a labelled variant")
        key = torch.zeros(n, dtype=torch.int64, device=dev)
        cells = [torch.clamp((parts[k] * (N / (2.0 * np.pi))).to(torch.int64), 0, N - 1) for k in "xyz"]
        for b in range(int(N - 1).bit_length()):
            for a in range(3):
                key |= ((cells[a] >> b) & 1) << (3 * b + a)
        perm = torch.argsort(key)
        parts = {k: parts[k][perm].contiguous() for k in F8}
        del key, cells, perm
    lcs.set_particles(*(parts[k] for k in F8))
    err, n_tot, _ = lcs.get_status()
    if (err or n_tot != n):
        print(f"bench.py: set_particles failed: status {err}, total {n_tot}", file=sys.stderr)
        return 3
    dt = cfg["dt"]

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        lcs.step_fused(dt)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    launches0 = lcs.kernel_launches
    lcs.profile_begin(args.steps)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        lcs.step_fused(dt)
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    prof = lcs.profile_end()
    launches = lcs.kernel_launches - launches0
    clocks = sampler.stop() if sampler else None
    err, n_tot, n_mig = lcs.get_status()
    if (err or n_tot != n):
        print(f"bench.py: step failed: sticky status {err}, total {n_tot}", file=sys.stderr)
        return 3
    ms_total = max_over_ranks(ms_total, dist, dev)
    ms_step = ms_total / args.steps
    value = world * n * args.steps / (ms_total * 1e-3)
    m = n_mig / n

    # ---- push and migrate separately (north_star: "for push and migrate separately and together") ---
    # the unfused pair lcs_particle_step + lcs_migrate gives the same result as lcs_step_fused; timed on rank 0's
    # stream with CUDA events, continuing from the state the fused steps left
    phases = None
    if args.phase_steps > 0:
        ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.phase_steps)]
        for k in range(args.phase_steps):
            ev[k][0].record(); lcs.particle_step(dt)
            ev[k][1].record(); lcs.migrate()
            ev[k][2].record()
        torch.cuda.synchronize()
        err_u, n_tot_u, n_mig_u = lcs.get_status()
        if (err_u or n_tot_u != n):
            print(f"bench.py: unfused step failed: sticky status {err_u}, total {n_tot_u}", file=sys.stderr)
            return 3
        # axis-by-axis exchange: lcs_particle_step + lcs_migrate_sweeps, the sweeps timed
        evs = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(3)]
        for k in range(3):
            lcs.particle_step(dt)
            evs[k][0].record(); lcs.migrate_sweeps(); evs[k][1].record()
        torch.cuda.synchronize()
        err_s, n_tot_s, _ = lcs.get_status()
        if (err_s or n_tot_s != n):
            print(f"bench.py: sweep step failed: sticky status {err_s}, total {n_tot_s}", file=sys.stderr)
            return 3
        sweeps_ms = float(np.median([e[0].elapsed_time(e[1]) for e in evs]))
        # the paper's two-stage RK2, in ITS regime: dt = 0.4 tau_p of the smallest droplet (explicit
        # RK2 diverges at the dt of BASELINE.json's configs, R-1), so very few particles migrate per stage
        rk2_ms = None
        if args.rk2:
            d_min = float(torch.min(wl["particles"]["d"]).item())       # the smallest droplet sets the explicit limit
            dt_rk2 = 0.4 * 1000.0 * d_min * d_min / (18.0 * 1.5e-5)
            evr = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(3)]
            for k in range(3):
                evr[k][0].record(); lcs.step_rk2(dt_rk2); evr[k][1].record()
            torch.cuda.synchronize()
            err_r, n_tot_r, n_mig_r = lcs.get_status()
            if (err_r or n_tot_r != n):
                print(f"bench.py: rk2 step failed: sticky status {err_r}, total {n_tot_r}", file=sys.stderr)
                return 3
            rk2_ms = float(np.median([e[0].elapsed_time(e[1]) for e in evr]))
        # per-step fluid refresh (first half): lcs_set_fluid = the repack of the three x-fastest
        # arrays into the internal (u,v,w,0) z-fastest records, as a coupled solver would call it every step
        evf = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(3)]
        for k in range(3):
            evf[k][0].record(); lcs.set_fluid(wl["u"], wl["v"], wl["w"]); evf[k][1].record()
        torch.cuda.synchronize()
        fluid_ms = float(np.median([e[0].elapsed_time(e[1]) for e in evf]))
        # ... and the refresh INSIDE the step, as the paper's coupled run has it (the fluid advances every time step,
        # PAPER.md:41; the particles see the current field, :64): lcs_set_fluid with a field that differs from the one
        # before (negated in place outside the timed region: the reversed flow, still divergence-free, so the slabs keep
        # their occupancy -- a permutation of the components is compressible and overflows them within six steps)
        # + lcs_step_fused, timed together
        evs2 = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(6)]
        for k in range(6):                                                    # an even count: the field ends as it began
            for c in "uvw":
                wl[c].neg_()
            evs2[k][0].record(); lcs.set_fluid(wl["u"], wl["v"], wl["w"]); lcs.step_fused(dt); evs2[k][1].record()
        torch.cuda.synchronize()
        err_f, n_tot_f, n_mig_f = lcs.get_status()
        if (err_f or n_tot_f != n):
            print(f"bench.py: step with fluid refresh failed: sticky status {err_f}, total {n_tot_f}", file=sys.stderr)
            return 3
        refresh_step_ms = float(np.median([e[0].elapsed_time(e[1]) for e in evs2]))
        # statistics hook (second half): the pair count behind g(r), on a thin shell
        r_hi_pc = 2.0 * np.pi / N * 0.25
        evp = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        pc_dev = lcs.pair_count(0.0, r_hi_pc)                                 # warm-up
        evp[0].record(); pc_dev = lcs.pair_count(0.0, r_hi_pc); evp[1].record()
        torch.cuda.synchronize()
        pair_ms = evp[0].elapsed_time(evp[1])
        pairs = int(pc_dev.item())
        g_of_r = pairs / (0.5 * n * (n - 1) * (4.0 / 3.0) * np.pi * r_hi_pc ** 3 / (2.0 * np.pi) ** 3)
        push_ms = float(np.median([e[0].elapsed_time(e[1]) for e in ev]))
        mig_ms = float(np.median([e[1].elapsed_time(e[2]) for e in ev]))
        m_u = n_mig_u / n
        peak_p, _ = measured_peak_hbm()
        push_bytes = 105.0 * n + 24.0 * N ** 3            # R 56 + W 48 + 1 code byte per particle + the grid once
        mig_bytes = n * (129.0 + 128.0 * m_u)             # code byte + stayers R/W 64 + migrants' second hop
        # DRAM bytes per launch from the committed ncu captures (profiles/traffic.json, hash-checked like roofline.traffic)
        tr_push, src_push, stale_push = ncu_traffic(args.workload, "k_push")
        tr_tp, src_tp, stale_tp = ncu_traffic(args.workload, "k_tile_pass<unfused>")
        tr_un, _, _ = ncu_traffic(args.workload, "k_unpack")
        tr_mig = (tr_tp + tr_un) if (tr_tp and tr_un) else None
        phases = {
            "steps": args.phase_steps, "timing": "median of per-call CUDA-event times",
            "push": {"call": "lcs_particle_step", "ms": push_ms, "particles_per_s": n / (push_ms * 1e-3),
                     "algorithmic_GBps": push_bytes / (push_ms * 1e-3) / 1e9,
                     "frac_of_measured_peak": push_bytes / (push_ms * 1e-3) / 1e9 / peak_p,
                     "traffic": tr_push, "traffic_stale": stale_push, "traffic_source": src_push,
                     "traffic_over_algorithmic": (tr_push / push_bytes) if tr_push else None},
            "migrate": {"call": "lcs_migrate", "ms": mig_ms, "particles_per_s": n / (mig_ms * 1e-3),
                        "algorithmic_GBps": mig_bytes / (mig_ms * 1e-3) / 1e9,
                        "frac_of_measured_peak": mig_bytes / (mig_ms * 1e-3) / 1e9 / peak_p,
                        "migrant_fraction": m_u,
                        "traffic": tr_mig, "traffic_stale": stale_tp, "traffic_source": src_tp,
                        "traffic_over_algorithmic": (tr_mig / mig_bytes) if tr_mig else None},
            "migrate_sweeps": {"call": "lcs_migrate_sweeps", "ms": sweeps_ms, "particles_per_s": n / (sweeps_ms * 1e-3),
                               "note": "x, y, z sweeps: three classify + unfused tile pass + scan + table + unpack rounds"},
            "rk2": None if rk2_ms is None else {
                "call": "lcs_step_rk2", "ms": rk2_ms, "particles_per_s": n / (rk2_ms * 1e-3), "dt": dt_rk2,
                "migrant_fraction_second_migration": n_mig_r / n,
                "note": "both stages run inside the tile pass; after stage 1 the slabs (8 arrays) and group B (X0, K1: 6 arrays) migrate in two rounds with the same codes, after stage 2 the slabs"},
            "set_fluid": {"call": "lcs_set_fluid", "ms": fluid_ms,
                          "GBps": (24.0 + 32.0) * N ** 3 / (fluid_ms * 1e-3) / 1e9,
                          "note": "reads 24 B and writes 32 B per cell; timed alone here, inside the step in step_with_refresh"},
            "step_with_refresh": {"call": "lcs_set_fluid + lcs_step_fused", "ms": refresh_step_ms,
                                  "particles_per_s": n / (refresh_step_ms * 1e-3),
                                  "algorithmic_bytes": n * (128.0 + 128.0 * m) + 24.0 * N ** 3 + 24.0 * N ** 3,
                                  "algorithmic_GBps": (n * (128.0 + 128.0 * m) + 48.0 * N ** 3) / (refresh_step_ms * 1e-3) / 1e9,
                                  "migrant_fraction": n_mig_f / n,
                                  "note": "the field changes before every step (PAPER.md:41, :64): repack of a different "
                                          "field + the fused step inside one timed region; bytes = the step's + 24 B per cell "
                                          "read by the repack"},
            "pair_count": {"call": "lcs_pair_count", "ms": pair_ms, "r_lo": 0.0, "r_hi": r_hi_pc, "pairs": pairs, "g": g_of_r,
                           "particles_per_s": n / (pair_ms * 1e-3),
                           "note": "cell list of all particles + 27-cell neighbourhood; g = 1 for a uniform distribution"},
            "fused": {"call": "lcs_step_fused", "ms": ms_total / args.steps,
                      "particles_per_s": n / (ms_total / args.steps * 1e-3)},
        }

    # ---- the state the timed steps left, checked on the device with properties that hold at any size (the element-wise
    # comparison with the oracle is the job of tests/, which runs the same launch configuration): every id exactly once,
    # and every particle inside the subdomain of the slab it sits in
    post = None
    if args.post_check:
        st = lcs.get_particles(n)
        ids = st["id"]
        # every id exactly once: n ids, all in [0, n), and every value of [0, n) hit (a scatter to a bool array)
        ids_ok = ids.numel() == n and int(ids.min()) >= 0 and int(ids.max()) < n
        if ids_ok:
            hit = torch.zeros(n, dtype=torch.bool, device=dev)
            hit[ids] = True
            ids_ok = bool(hit.all())
            del hit
        inv_dx = N / (2.0 * np.pi)
        own = None
        for k, Pk, mul in (("x", cfg["P"][0], 1), ("y", cfg["P"][1], cfg["P"][0]), ("z", cfg["P"][2], cfg["P"][0] * cfg["P"][1])):
            c = torch.clamp(torch.floor(st[k] * inv_dx).to(torch.int64), 0, N - 1) // (N // Pk) * mul
            own = c if own is None else own + c
        slab = torch.repeat_interleave(torch.arange(P, dtype=torch.int64, device=dev), st["counts"])
        misplaced = int((own != slab).sum()) if slab.numel() == n else -1
        post = {"ids_each_once": ids_ok, "particles_outside_their_slab": misplaced, "count_sum": int(st["counts"].sum()),
                "note": "after the timed fused steps and the phase calls; property checks on the device, not an oracle comparison"}
        del st, ids, own, slab
        if not ids_ok or misplaced != 0:
            print(f"bench.py: post-check failed: {post}", file=sys.stderr)
            return 3

    # ---- end to end through the host-buffer entry point (rank-local, then max over ranks) ----------
    e2e = None
    if args.e2e_steps > 0:
        state = lcs.get_particles(n)
        h_in = {k: torch.empty(n, dtype=state[k].dtype, pin_memory=True) for k in F8}
        h_out = {k: torch.empty(n, dtype=state[k].dtype, pin_memory=True) for k in F8}
        h_counts = torch.empty(P, dtype=torch.int64, pin_memory=True)
        for k in F8:
            h_in[k].copy_(state[k])
        del state
        staging = torch.empty(lcs.staging_bytes(n), dtype=torch.uint8, device=dev)
        lcs.step_fused_host(dt, h_in, h_out, h_counts, staging)       # warm-up
        barrier()
        t0 = torch.cuda.Event(enable_timing=True); t1 = torch.cuda.Event(enable_timing=True)
        t0.record()
        src, dst = h_in, h_out
        for _ in range(args.e2e_steps):
            lcs.step_fused_host(dt, src, dst, h_counts, staging)      # synchronises: result is on the host
            src, dst = dst, src
        t1.record()
        barrier()
        ms_e2e = t0.elapsed_time(t1)
        ms_e2e = max_over_ranks(ms_e2e, dist, dev)
        assert int(h_counts.sum()) == n
        # the link itself: one pinned array each way, alone (the floor of this path is 8 arrays in + 8 arrays out)
        one = torch.empty(n, dtype=torch.float64, device=dev)
        lk = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        lk[0].record(); one.copy_(h_in["x"], non_blocking=True); lk[1].record(); h_out["x"].copy_(one, non_blocking=True); lk[2].record()
        torch.cuda.synchronize()
        h2d_gbps = 8.0 * n / (lk[0].elapsed_time(lk[1]) * 1e-3) / 1e9
        d2h_gbps = 8.0 * n / (lk[1].elapsed_time(lk[2]) * 1e-3) / 1e9
        del one
        e2e = {"value": world * n * args.e2e_steps / (ms_e2e * 1e-3), "unit": "particles/s",
               "h2d_GBps_alone": h2d_gbps, "d2h_GBps_alone": d2h_gbps,
               "link_floor_ms_per_step": (64.0 * n / h2d_gbps + 64.0 * n / d2h_gbps) / 1e6,
               "h2d_bytes_per_step": 64 * n, "d2h_bytes_per_step": 64 * n + 8 * P,
               "steps": args.e2e_steps, "ms_per_step": ms_e2e / args.e2e_steps,
               "call": "lcs_step_fused_host (pinned host particle arrays in/out; fluid field resident)"}
        del staging, h_in, h_out

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel (k_tile_pass<fused>) ---------------------------------------
    peak, peak_src = measured_peak_hbm()
    alg_bytes = 128.0 * n + 24.0 * N ** 3            # R64 + W64 per particle + the compulsory grid read
    tile_ms = prof["tile_pass_ms"] / max(prof["steps"], 1)
    achieved = alg_bytes / (tile_ms * 1e-3) / 1e9
    step_bytes = n * (128.0 + 128.0 * m) + 24.0 * N ** 3
    traffic, traffic_src, traffic_stale = ncu_traffic(args.workload, "k_tile_pass<fused>")
    if args.traffic_bytes is not None:
        traffic, traffic_src, traffic_stale = args.traffic_bytes, "--traffic-bytes", False
    roofline = {"bound": "hbm", "kernel": "k_tile_pass<fused>", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic, "traffic_stale": traffic_stale,
                "traffic_source": (f"ncu dram__bytes_read.sum + dram__bytes_write.sum of one launch, {traffic_src}"
                                   if traffic_src else None),
                "traffic_over_algorithmic": (traffic / alg_bytes) if traffic else None,
                "peak_source": peak_src,
                "algorithmic_bytes_per_launch": alg_bytes, "avg_launch_ms": tile_ms,
                "kernel_share_of_step": tile_ms / ms_step,
                "table_ms": prof["table_ms"] / max(prof["steps"], 1),
                "unpack_ms": prof["unpack_ms"] / max(prof["steps"], 1),
                "step_algorithmic_GBps": step_bytes / (ms_step * 1e-3) / 1e9,
                "step_frac_of_measured_peak": step_bytes / (ms_step * 1e-3) / 1e9 / peak,
                "step_frac_of_nominal_8TBps": step_bytes / (ms_step * 1e-3) / 1e9 / 8000.0}

    # ---- what actually bounds the tile pass: the L2 -> SM traffic of the gather ----------------
    # Every particle brings 64 B in by bulk copy and 8 x 32 B record sectors through L1 (random inside the brick of its
    # subdomain, which L2 holds); lcs_probe_gather measures, on the same fluid records and alone on the GPU, what the
    # memory system delivers for that pattern.
    # one brick = the subdomain's cells plus a one-cell halo on both sides: (n + 2) records per axis
    brick_mb = (N // cfg["P"][0] + 2) * (N // cfg["P"][1] + 2) * (N // cfg["P"][2] + 2) * 32 / 1048576.0
    try:
        ceil_l2 = lcs.probe_gather(brick_mb, 200)
        ceil_dram = lcs.probe_gather(N ** 3 * 32 / 1048576.0, 50)
    except Exception as exc:                        # pragma: no cover
        print(f"bench.py: lcs_probe_gather failed: {exc!r}", file=sys.stderr)
        ceil_l2 = ceil_dram = None
    l2_bytes = 320.0 * n
    roofline["l2_to_sm"] = {
        "bytes_per_launch": l2_bytes, "GBps_in_tile_pass": l2_bytes / (tile_ms * 1e-3) / 1e9,
        "gather_ceiling_GBps": ceil_l2, "frac_of_gather_ceiling": (l2_bytes / (tile_ms * 1e-3) / 1e9 / ceil_l2) if ceil_l2 else None,
        "dram_random_sector_GBps": ceil_dram, "brick_MB": brick_mb,
        "note": "64 B bulk copy + 8 record sectors of 32 B per particle; ceiling = lcs_probe_gather on one brick-sized window, "
                "same load instruction, 12 warps per SM, nothing else running"}

    # ---- the oracle on the host cores, bounded sample ---------------------------------------------
    cpu = None
    if args.cpu_sample > 0:
        stride = max(1, n // args.cpu_sample)
        rate, sec, n_s = oracle_sample_rate(cfg, wl, stride, 2, torch)
        cpu = {"value": rate, "unit": "particles/s", "cores": 1, "kind": "oracle",
               "sample": f"every {stride}th particle of {cfg['name']} ({n_s} particles, full {N}^3 field), 2 steps, "
                         f"single thread of {os.cpu_count()} host cores",
               "phases": dict(ORACLE_PHASES)}

    line = {
        "metric": METRIC, "value": value, "unit": "particles/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": bench_config(cfg, args, world), "migrant_fraction_last_step": m,
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "phases": phases, "post_check": post,
        "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="Large")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--phase-steps", type=int, default=5, help="unfused steps timed for the push / migrate split (0 = skip)")
    ap.add_argument("--cpu-sample", type=int, default=1 << 22, help="particles in the oracle's timed sample (0 = skip)")
    ap.add_argument("--ref-sample", type=int, default=1 << 21, help="--impl reference: particles per timed step")
    ap.add_argument("--drag-model", type=int, default=0, choices=[0, 1],
                    help="0: Stokes drag (BASELINE.json's configs); 1: f = 1 + 0.15 Re^0.687 (SURVEY 8(f) NEXT #2)")
    ap.add_argument("--rk2", type=int, default=1, choices=[0, 1],
                    help="1: also time lcs_step_rk2 (SURVEY 8(f) NEXT #1); reserves 8 more arrays of P*capacity doubles")
    ap.add_argument("--order", default="generation", choices=["generation", "morton"],
                    help="order in which the particles are handed to lcs_set_particles: generation order (spatially random, the "
                         "headline) or sorted by the Morton key of their cell (a labelled variant)")
    ap.add_argument("--post-check", type=int, default=1, help="1: check the id multiset and the containment of the final state on the device")
    ap.add_argument("--traffic-bytes", type=float, default=None,
                    help="ncu dram bytes per launch of the dominant kernel (from profiles/), reported as roofline.traffic")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "cuda":
        args.warmup = 3
    return run_reference(args) if args.impl == "reference" else run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
