"""ctypes binding of include/lcs.h -- argument marshalling only; every step of the path runs in
the CUDA kernels of liblcs_b200.so.  Method names mirror the C entry points."""
from __future__ import annotations

import ctypes as C
import os

LCS_OK, LCS_ERR_INVALID_ARG, LCS_ERR_STATE, LCS_ERR_CUDA = 0, -1, -2, -3
LCS_ERR_CAPACITY, LCS_ERR_JUMP, LCS_ERR_RANGE, LCS_ERR_NOMEM = -4, -5, -6, -7
LCS_ERR_TOO_LARGE = -8
LCS_PAIR_COUNT_STATIC_MAX_SLOTS = 1 << 19

EXPORTED_SYMBOLS = (
    "lcs_workspace_bytes", "lcs_create", "lcs_destroy", "lcs_set_fluid", "lcs_set_particles",
    "lcs_particle_step", "lcs_migrate", "lcs_migrate_sweeps", "lcs_step_rk2", "lcs_step_fused", "lcs_get_counts", "lcs_get_particles",
    "lcs_get_codes", "lcs_get_count_table", "lcs_get_status", "lcs_staging_bytes", "lcs_step_fused_host", "lcs_pair_count", "lcs_pair_count_static", "lcs_probe_gather",
    "lcs_profile_begin", "lcs_profile_end", "lcs_kernel_launches", "lcs_version")

FIELDS = ("x", "y", "z", "vx", "vy", "vz", "d", "id")


class LcsError(RuntimeError):
    def __init__(self, fn, code):
        why = (f": the handle has more than {LCS_PAIR_COUNT_STATIC_MAX_SLOTS} particle slots (P*capacity), the limit of the "
               "library's built-in scratch" if code == LCS_ERR_TOO_LARGE else "")
        super().__init__(f"{fn} returned {code}{why}")
        self.code = code


class LcsParams(C.Structure):
    _fields_ = [("nu", C.c_double), ("rho_ratio", C.c_double), ("g", C.c_double * 3),
                ("send_capacity", C.c_int64), ("drag_model", C.c_int32), ("enable_rk2", C.c_int32)]


def lib_path() -> str:
    return os.path.join(os.path.dirname(os.path.abspath(__file__)), "liblcs_b200.so")


_lib = None


def load_library(build_if_missing: bool = True):
    """dlopen liblcs_b200.so (building it in-tree with nvcc if absent).  Raises if unavailable."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if build_if_missing:
        from . import build as _b
        if _b.stale():
            _b.build()
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: run `python -m paper_2604_11008_b200.build` (needs nvcc)")
    L = C.CDLL(path)
    vp, i64, dbl = C.c_void_p, C.c_int64, C.c_double
    L.lcs_version.restype = C.c_char_p
    L.lcs_workspace_bytes.restype = C.c_size_t
    L.lcs_workspace_bytes.argtypes = [C.c_int] * 4 + [i64, C.POINTER(LcsParams)]
    L.lcs_create.argtypes = [C.c_int] * 4 + [i64, C.POINTER(LcsParams), vp, C.c_size_t, vp, C.POINTER(vp)]
    L.lcs_destroy.argtypes = [vp]
    L.lcs_set_fluid.argtypes = [vp] * 4
    L.lcs_set_particles.argtypes = [vp, i64] + [vp] * 8
    L.lcs_particle_step.argtypes = [vp, dbl]
    L.lcs_migrate.argtypes = [vp]
    L.lcs_migrate_sweeps.argtypes = [vp]
    L.lcs_step_rk2.argtypes = [vp, C.c_double]
    L.lcs_step_fused.argtypes = [vp, dbl]
    L.lcs_get_counts.argtypes = [vp, vp]
    L.lcs_get_particles.argtypes = [vp] * 10
    L.lcs_get_codes.argtypes = [vp, vp]
    L.lcs_get_count_table.argtypes = [vp, vp]
    L.lcs_get_status.argtypes = [vp, C.POINTER(C.c_int), C.POINTER(i64), C.POINTER(i64)]
    L.lcs_pair_count.argtypes = [vp, dbl, dbl, vp]
    L.lcs_pair_count_static.argtypes = [vp, dbl, dbl, vp]
    L.lcs_probe_gather.argtypes = [vp, dbl, C.c_int, C.POINTER(dbl), C.POINTER(dbl)]
    L.lcs_staging_bytes.restype = C.c_size_t
    L.lcs_staging_bytes.argtypes = [i64, C.c_int]
    L.lcs_step_fused_host.argtypes = [vp, dbl, i64, C.POINTER(vp), C.POINTER(vp), vp, vp, C.c_size_t]
    L.lcs_profile_begin.argtypes = [vp, C.c_int]
    L.lcs_profile_end.argtypes = [vp, C.POINTER(dbl), C.POINTER(dbl), C.POINTER(dbl), C.POINTER(C.c_int)]
    L.lcs_kernel_launches.restype = i64
    L.lcs_kernel_launches.argtypes = [vp]
    _lib = L
    return L


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


class LCS:
    """One handle = one periodic box with an N^3 fluid grid and Px*Py*Pz virtual subdomains on one GPU.
    Device tensors in, device tensors out; torch allocates, the library computes."""

    def __init__(self, N, Px, Py, Pz, capacity, nu=1.5e-5, rho_ratio=1000.0, g=(0.0, 0.0, 0.0),
                 send_capacity=0, drag_model=0, rk2=False, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2604_11008_b200 needs a CUDA device (no CPU fallback)")
        self._torch = torch
        self._L = load_library()
        self.device = torch.device(device)
        self.N, self.Px, self.Py, self.Pz, self.capacity = N, Px, Py, Pz, int(capacity)
        self.P = Px * Py * Pz
        self._prm = LcsParams(nu, rho_ratio, (C.c_double * 3)(*g), int(send_capacity), int(drag_model), int(bool(rk2)))
        nbytes = self._L.lcs_workspace_bytes(N, Px, Py, Pz, int(capacity), C.byref(self._prm))
        if nbytes == 0:
            raise LcsError("lcs_workspace_bytes", LCS_ERR_INVALID_ARG)
        self.workspace_bytes = nbytes
        with torch.cuda.device(self.device):
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        base = self._ws.data_ptr()
        self._ws_ptr = (base + 255) // 256 * 256
        h = C.c_void_p()
        rc = self._L.lcs_create(N, Px, Py, Pz, int(capacity), C.byref(self._prm), C.c_void_p(self._ws_ptr),
                                nbytes, C.c_void_p(self.stream.cuda_stream), C.byref(h))
        if rc:
            raise LcsError("lcs_create", rc)
        self._h = h
        self._fluid = None

    def close(self):
        if getattr(self, "_h", None):
            self._L.lcs_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, fn, rc):
        if rc:
            raise LcsError(fn, rc)

    # ---- the C entry points, one method each ------------------------------------------------
    def set_fluid(self, u, v, w):
        for t in (u, v, w):
            assert t.is_cuda and t.dtype == self._torch.float64 and t.is_contiguous() and t.numel() == self.N ** 3
        self._fluid = (u, v, w)   # (the library copies the field at call time, in stream order; kept only so that they outlive the enqueued repack)
        self._chk("lcs_set_fluid", self._L.lcs_set_fluid(self._h, _ptr(u), _ptr(v), _ptr(w)))

    def set_particles(self, x, y, z, vx, vy, vz, d, id):
        n = id.numel()
        if n == 0:                     # zero-size tensors have null data pointers
            x = y = z = vx = vy = vz = d = self._torch.zeros(1, dtype=self._torch.float64, device=self.device)
            id = self._torch.zeros(1, dtype=self._torch.int64, device=self.device)
        ts = (x, y, z, vx, vy, vz, d)
        for t in ts:
            assert t.is_cuda and t.dtype == self._torch.float64 and t.is_contiguous() and t.numel() == max(n, 1)
        assert id.is_cuda and id.dtype == self._torch.int64 and id.is_contiguous()
        self._chk("lcs_set_particles",
                  self._L.lcs_set_particles(self._h, n, *(_ptr(t) for t in ts), _ptr(id)))

    def particle_step(self, dt):
        self._chk("lcs_particle_step", self._L.lcs_particle_step(self._h, float(dt)))

    def migrate(self):
        self._chk("lcs_migrate", self._L.lcs_migrate(self._h))

    def step_rk2(self, dt):
        """The paper's two-stage RK2 with one migration per stage (needs rk2=True at construction; R-25)."""
        self._chk("lcs_step_rk2", self._L.lcs_step_rk2(self._h, float(dt)))

    def migrate_sweeps(self):
        """Axis-by-axis exchange: x, y, z sweeps (R-24)."""
        self._chk("lcs_migrate_sweeps", self._L.lcs_migrate_sweeps(self._h))

    def step_fused(self, dt):
        self._chk("lcs_step_fused", self._L.lcs_step_fused(self._h, float(dt)))

    def get_status(self):
        """-> (sticky_error, n_total, n_migrated_last); synchronises the stream."""
        e, n, m = C.c_int(), C.c_int64(), C.c_int64()
        rc = self._L.lcs_get_status(self._h, C.byref(e), C.byref(n), C.byref(m))
        if rc == LCS_ERR_CUDA or rc == LCS_ERR_INVALID_ARG:
            raise LcsError("lcs_get_status", rc)
        return e.value, n.value, m.value

    def get_counts(self):
        out = self._torch.empty(self.P, dtype=self._torch.int64, device=self.device)
        self._chk("lcs_get_counts", self._L.lcs_get_counts(self._h, _ptr(out)))
        return out

    def get_particles(self, n_total=None):
        """-> dict of packed device tensors (counts, x..id).  n_total defaults to lcs_get_status's."""
        t = self._torch
        if n_total is None:
            _, n_total, _ = self.get_status()
        m = max(int(n_total), 1)       # a zero-size tensor has a null data pointer
        out = {k: t.empty(m, dtype=t.float64, device=self.device) for k in FIELDS[:7]}
        out["id"] = t.empty(m, dtype=t.int64, device=self.device)
        out["counts"] = t.empty(self.P, dtype=t.int64, device=self.device)
        self._chk("lcs_get_particles",
                  self._L.lcs_get_particles(self._h, _ptr(out["counts"]), *(_ptr(out[k]) for k in FIELDS)))
        return {k: (v if k == "counts" else v[:n_total]) for k, v in out.items()}

    def get_codes(self, n_total=None):
        t = self._torch
        if n_total is None:
            _, n_total, _ = self.get_status()
        out = t.empty(max(int(n_total), 1), dtype=t.uint8, device=self.device)
        self._chk("lcs_get_codes", self._L.lcs_get_codes(self._h, _ptr(out)))
        return out[:n_total]

    def get_count_table(self):
        out = self._torch.empty((self.P, 27), dtype=self._torch.int64, device=self.device)
        self._chk("lcs_get_count_table", self._L.lcs_get_count_table(self._h, _ptr(out)))
        return out

    def pair_count(self, r_lo, r_hi):
        """-> device int64 tensor (1 element): unordered pairs with periodic separation in [r_lo, r_hi) (R-26)."""
        out = self._torch.empty(1, dtype=self._torch.int64, device=self.device)
        self._chk("lcs_pair_count", self._L.lcs_pair_count(self._h, float(r_lo), float(r_hi), _ptr(out)))
        return out

    def pair_count_static(self, r_lo, r_hi, out=None):
        """pair_count for a caller that has no device memory to lend and may not allocate any (a diagnostics hook inside
        a time loop whose host application owns all of HBM and bans cudaMalloc there): the scratch is a fixed 17 MiB array
        inside the library instead of the send pool, so P*capacity must not exceed LCS_PAIR_COUNT_STATIC_MAX_SLOTS
        (LcsError with LCS_ERR_TOO_LARGE otherwise).  Pass `out` (1-element int64 device tensor) and the call allocates
        nothing at all; without it the binding asks torch for the 8-byte result.  One shared array per GPU: calls that
        could overlap on the device (two streams) must be serialised by the caller.  include/lcs.h has the details."""
        if out is None:
            out = self._torch.empty(1, dtype=self._torch.int64, device=self.device)
        assert out.is_cuda and out.dtype == self._torch.int64 and out.numel() == 1
        self._chk("lcs_pair_count_static", self._L.lcs_pair_count_static(self._h, float(r_lo), float(r_hi), _ptr(out)))
        return out

    def probe_gather(self, window_mb, iters=200):
        """-> GB/s of 32-byte record loads at random records of the first window_mb MB of the fluid field (measurement aid)."""
        ms, nb = C.c_double(), C.c_double()
        self._chk("lcs_probe_gather", self._L.lcs_probe_gather(self._h, float(window_mb), int(iters), C.byref(ms), C.byref(nb)))
        return nb.value / (ms.value * 1e-3) / 1e9

    def staging_bytes(self, n):
        """Bytes of device scratch lcs_step_fused_host needs for n particles (+ 256 so that the block can be aligned)."""
        return int(self._L.lcs_staging_bytes(int(n), self.P)) + 256

    def step_fused_host(self, dt, h_in, h_out, h_counts, staging):
        """h_in / h_out: dicts of pinned host tensors keyed x..id; h_counts: int64[P] host tensor;
        staging: device uint8 tensor of at least staging_bytes(n) bytes."""
        n = h_in["id"].numel()
        pin = (C.c_void_p * 8)(*(h_in[k].data_ptr() for k in FIELDS))
        pout = (C.c_void_p * 8)(*(h_out[k].data_ptr() for k in FIELDS))
        sp = (staging.data_ptr() + 255) // 256 * 256
        sbytes = staging.numel() - (sp - staging.data_ptr())
        rc = self._L.lcs_step_fused_host(self._h, float(dt), n, pin, pout, C.c_void_p(h_counts.data_ptr()),
                                         C.c_void_p(sp), sbytes)
        self._chk("lcs_step_fused_host", rc)

    def profile_begin(self, max_steps):
        self._chk("lcs_profile_begin", self._L.lcs_profile_begin(self._h, int(max_steps)))

    def profile_end(self):
        """-> dict(tile_pass_ms, table_ms, unpack_ms, steps): summed CUDA-event durations."""
        a, b, c, n = C.c_double(), C.c_double(), C.c_double(), C.c_int()
        self._chk("lcs_profile_end", self._L.lcs_profile_end(self._h, C.byref(a), C.byref(b), C.byref(c), C.byref(n)))
        return {"tile_pass_ms": a.value, "table_ms": b.value, "unpack_ms": c.value, "steps": n.value}

    @property
    def kernel_launches(self):
        return self._L.lcs_kernel_launches(self._h)
