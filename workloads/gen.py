"""Seeded synthetic inputs shared by the oracle and the CUDA path (identical bytes go to both).

This module holds none of the method's arithmetic (no interpolation, no advance, no classification,
no migration); it only manufactures inputs with the shapes of the paper's workloads
(PAPER.md:47 periodic 2*pi box and N^3 grid, :150/:217 particle counts 0.1-10x the grid count) as
BASELINE.json's five configs describe them.  The recipe is restated in DESIGN.md section 5.

Random draws always come from numpy Generator(PCG64(seed)) on the host so they are the same on every
machine; the heavy evaluations (field synthesis, velocity at the particles) are torch ops on
`device` and may differ in the last bit between a CPU and a GPU run, which is harmless: whatever
bytes come out are handed to both sides.
"""
from __future__ import annotations

import json
import math
import os

import numpy as np
import torch

L_BOX = 6.283185307179586  # 2*pi as the double 0x401921FB54442D18
L_BELOW = float(np.nextafter(L_BOX, 0.0))
N_MODES = 64
NU = 1.5e-5
RHO_RATIO = 1000.0   # BASELINE.json configs (the paper uses 843)

_HERE = os.path.dirname(os.path.abspath(__file__))


def load_configs():
    with open(os.path.join(_HERE, "configs.json")) as f:
        return json.load(f)["configs"]


def get_config(name: str) -> dict:
    for c in load_configs():
        if c["name"].lower() == name.lower():
            return dict(c)
    raise KeyError(name)


def scaled_config(cfg: dict, n: int | None = None, N: int | None = None) -> dict:
    """Same recipe at a smaller particle count / grid (parity-test sizes)."""
    c = dict(cfg)
    if N is not None:
        c["kmax"] = max(2, cfg["kmax"] * N // cfg["N"])
        c["N"] = N
    if n is not None:
        P = c["P"][0] * c["P"][1] * c["P"][2]
        c["capacity"] = max(64, int(math.ceil(cfg["capacity"] * n / cfg["n"] / 2) * 2))
        c["n"] = n
        if n / P < 512:  # small slabs fluctuate more than 1.25x
            c["capacity"] = max(c["capacity"], int(2 * math.ceil(n / P) + 64))
    return c


# ----------------------------------------------------------------------------------------------
# fluid: 64 random divergence-free Fourier modes, E(k) ~ k^-5/3, per-component rms 1
# ----------------------------------------------------------------------------------------------
def make_modes(cfg: dict):
    """-> (k [M,3] float64 integer-valued, a [M,3], b [M,3]) before the rms rescale."""
    rng = np.random.Generator(np.random.PCG64(1000 + cfg["index"]))
    kmax = float(cfg["kmax"])
    ks, As, Bs = [], [], []
    for m in range(N_MODES):
        kappa = kmax ** (m / (N_MODES - 1))
        while True:
            dvec = rng.standard_normal(3)
            dvec /= np.linalg.norm(dvec)
            k = np.rint(dvec * kappa)
            if np.any(k != 0):
                break
        kn = np.linalg.norm(k)
        khat = k / kn
        p = rng.standard_normal(3)
        q = rng.standard_normal(3)
        p -= khat * np.dot(p, khat)      # perpendicular to k: divergence-free
        q -= khat * np.dot(q, khat)
        p /= np.linalg.norm(p)
        q /= np.linalg.norm(q)
        amp = math.sqrt(kn ** (-5.0 / 3.0) * kn)   # shell width ~ kappa for geometric spacing
        ks.append(k)
        As.append(amp * p)
        Bs.append(amp * q)
    return np.array(ks), np.array(As), np.array(Bs)


def _field_slab(k, a, b, N, z0, z1, device):
    """u,v,w on cells k in [z0,z1): tensor [3, z1-z0, N, N] (x fastest)."""
    dt = torch.float64
    kk = torch.as_tensor(k, dtype=dt, device=device)
    A = torch.as_tensor(a, dtype=dt, device=device)
    B = torch.as_tensor(b, dtype=dt, device=device)
    dx = L_BOX / N
    cx = (torch.arange(N, dtype=dt, device=device) + 0.5) * dx
    cz = (torch.arange(z0, z1, dtype=dt, device=device) + 0.5) * dx
    # theta = kx x + ky y + kz z ; cos/sin(theta) via separable tables and one real matmul over modes
    phx = kk[:, 0:1] * cx[None, :]
    phy = kk[:, 1:2] * cx[None, :]
    phz = kk[:, 2:3] * cz[None, :]
    Ex = torch.complex(torch.cos(phx), torch.sin(phx))           # [M, N]
    Eyz = (torch.complex(torch.cos(phz), torch.sin(phz))[:, :, None]
           * torch.complex(torch.cos(phy), torch.sin(phy))[:, None, :])   # [M, Z, N]
    out = torch.empty((3, z1 - z0, N, N), dtype=dt, device=device)
    rhs = torch.cat([Ex.real, Ex.imag], dim=0)                   # [2M, N]
    for c in range(3):
        T = Eyz * torch.complex(A[:, c], -B[:, c])[:, None, None]   # Re(T*Ex) = a cos + b sin
        lhs = torch.cat([T.real, -T.imag], dim=0).reshape(2 * kk.shape[0], -1).t()   # [Z*N, 2M]
        out[c] = (lhs @ rhs).reshape(z1 - z0, N, N)
    return out


def make_fluid(cfg: dict, device="cpu"):
    """-> (u, v, w, modes): flat float64 tensors of N^3 on `device`, index i + N*(j + N*k)."""
    N = cfg["N"]
    k, a, b = make_modes(cfg)
    uvw = [torch.empty(N * N * N, dtype=torch.float64, device=device) for _ in range(3)]
    zchunk = max(1, min(N, (1 << 24) // (N * N)))
    ssq = torch.zeros((), dtype=torch.float64, device=device)
    for z0 in range(0, N, zchunk):
        z1 = min(N, z0 + zchunk)
        slab = _field_slab(k, a, b, N, z0, z1, device)
        ssq += (slab * slab).sum()
        for c in range(3):
            uvw[c][z0 * N * N:z1 * N * N] = slab[c].reshape(-1)
    rms = math.sqrt(float(ssq) / (3.0 * N ** 3))   # "rms u' = 1" read per component
    scale = 1.0 / rms
    for c in range(3):
        uvw[c] *= scale
    modes = {"k": k, "a": a * scale, "b": b * scale}
    return uvw[0], uvw[1], uvw[2], modes


def field_at(modes, x, y, z, device="cpu", chunk=1 << 20):
    """The synthetic field itself (the mode sum, not an interpolant) at points: used only to give
    particles an initial velocity."""
    dt = torch.float64
    kk = torch.as_tensor(modes["k"], dtype=dt, device=device)
    AB = torch.cat([torch.as_tensor(modes["a"], dtype=dt, device=device).t(),
                    torch.as_tensor(modes["b"], dtype=dt, device=device).t()], dim=1)   # [3, 2M]
    n = x.shape[0]
    out = torch.empty((3, n), dtype=dt, device=device)
    for i0 in range(0, n, chunk):
        i1 = min(n, i0 + chunk)
        X = torch.stack([x[i0:i1], y[i0:i1], z[i0:i1]], dim=0)    # [3, c]
        th = kk @ X                                                # [M, c]
        out[:, i0:i1] = AB @ torch.cat([torch.cos(th), torch.sin(th)], dim=0)
    return out[0], out[1], out[2]


# ----------------------------------------------------------------------------------------------
# particles
# ----------------------------------------------------------------------------------------------
def make_particles(cfg: dict, modes, device="cpu"):
    """-> dict of tensors on `device`: x y z vx vy vz d (float64), id (int64); generation order."""
    n = cfg["n"]
    idx = cfg["index"]
    rng = np.random.Generator(np.random.PCG64(2000 + idx))
    if cfg.get("clumps", 0):
        crng = np.random.Generator(np.random.PCG64(4000 + idx))
        centres = crng.random((cfg["clumps"], 3)) * L_BOX
        which = rng.integers(0, cfg["clumps"], size=n)
        sigma = cfg["clump_sigma_cells"] * L_BOX / cfg["N"]
        pos = []
        for a in range(3):
            p = centres[which, a] + sigma * rng.standard_normal(n)
            p = np.mod(p, L_BOX)
            pos.append(np.minimum(p, L_BELOW))
    else:
        pos = [np.minimum(rng.random(n) * L_BOX, L_BELOW) for _ in range(3)]
    rrng = np.random.Generator(np.random.PCG64(3000 + idx))
    radius = cfg["radius_median"] * np.exp(cfg["sigma_ln"] * rrng.standard_normal(n))
    out = {}
    for name, arr in zip(("x", "y", "z"), pos):
        out[name] = torch.from_numpy(arr).to(device)
    out["vx"], out["vy"], out["vz"] = field_at(modes, out["x"], out["y"], out["z"], device)
    out["d"] = torch.from_numpy(2.0 * radius).to(device)
    out["id"] = torch.arange(n, dtype=torch.int64, device=device)
    return out


def make_workload(cfg: dict, device="cpu"):
    u, v, w, modes = make_fluid(cfg, device)
    parts = make_particles(cfg, modes, device)
    return {"cfg": cfg, "u": u, "v": v, "w": w, "modes": modes, "particles": parts}
