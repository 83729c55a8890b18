"""oracle/oracle.py -- TEST INFRASTRUCTURE, NOT PRODUCT.

ctypes binding of oracle/lcs_oracle.c (the plain sequential fp64 CPU statement of the hot path,
written from PAPER.md and DESIGN.md's readings).  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It imports nothing from
paper_2604_11008_b200/ and the CUDA path imports nothing from here.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lcs_oracle.c")
_LIB = os.path.join(_HERE, "liblcs_oracle.so")
# -ffp-contract=off: fused multiply-adds only where fma() is written (reproducibility rules)
_CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-mfma", "-shared", "-fPIC", "-Wall"]

STAY = 13
OK, ERR_ARG, ERR_CAPACITY, ERR_JUMP, ERR_RANGE, ERR_STATE, ERR_NOMEM = range(7)


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", *_CFLAGS, "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int64)
_bp = C.POINTER(C.c_uint8)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_exp_neg.restype = C.c_double
        L.orc_exp_neg.argtypes = [C.c_double]
        L.orc_pow_0687.restype = C.c_double
        L.orc_pow_0687.argtypes = [C.c_double]
        L.orc_set_drag_model.argtypes = [C.c_void_p, C.c_int]
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int] * 4 + [C.c_int64, C.c_double, C.c_double, _dp]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_destroy.restype = None
        L.orc_cell.restype = C.c_int64
        L.orc_cell.argtypes = [C.c_void_p, C.c_double]
        L.orc_owner.restype = C.c_int64
        L.orc_owner.argtypes = [C.c_void_p] + [C.c_double] * 3
        L.orc_receiver.restype = C.c_int64
        L.orc_receiver.argtypes = [C.c_void_p, C.c_int64, C.c_int]
        L.orc_tau.restype = C.c_double
        L.orc_tau.argtypes = [C.c_void_p, C.c_double]
        L.orc_interp.argtypes = [C.c_void_p, C.c_int64] + [_dp] * 6
        L.orc_set_fluid.argtypes = [C.c_void_p] + [_dp] * 3
        L.orc_set_particles.argtypes = [C.c_void_p, C.c_int64] + [_dp] * 7 + [_ip]
        L.orc_load_packed.argtypes = [C.c_void_p, _ip] + [_dp] * 7 + [_ip, _bp]
        L.orc_push.argtypes = [C.c_void_p, C.c_double]
        L.orc_migrate.argtypes = [C.c_void_p]
        L.orc_classify_axis.argtypes = [C.c_void_p, C.c_int]
        L.orc_rk2_stage1.argtypes = [C.c_void_p, C.c_double]
        L.orc_rk2_stage2.argtypes = [C.c_void_p, C.c_double]
        L.orc_total.restype = C.c_int64
        L.orc_total.argtypes = [C.c_void_p]
        L.orc_status.argtypes = [C.c_void_p]
        L.orc_n_migrated_last.restype = C.c_int64
        L.orc_n_migrated_last.argtypes = [C.c_void_p]
        L.orc_get_counts.argtypes = [C.c_void_p, _ip]
        L.orc_get_counts.restype = None
        L.orc_get_cnt_table.argtypes = [C.c_void_p, _ip]
        L.orc_get_cnt_table.restype = None
        L.orc_get_particles.argtypes = [C.c_void_p, _ip] + [_dp] * 7 + [_ip, _bp]
        L.orc_get_particles.restype = None
        L.orc_get_last_send_slots.argtypes = [C.c_void_p, C.c_int64, C.c_int64, _ip]
        L.orc_get_last_send_slots.restype = None
        L.orc_pair_count.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.orc_pair_count.restype = C.c_int64
        _lib = L
    return _lib


def _d(a):
    return a.ctypes.data_as(_dp)


def _i(a):
    return a.ctypes.data_as(_ip)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def exp_neg(z: float) -> float:
    return lib().orc_exp_neg(float(z))


def pow_0687(R: float) -> float:
    """R^0.687 as specified in DESIGN.md R-23 (the drag factor of PAPER.md:59 is 1 + 0.15 * this)."""
    return lib().orc_pow_0687(float(R))


FIELDS = ("x", "y", "z", "vx", "vy", "vz", "d", "id")


class Oracle:
    """One periodic box [0, 2*pi)^3 with an N^3 fluid grid and Px*Py*Pz virtual subdomains."""

    def __init__(self, N, Px, Py, Pz, capacity, nu=1.5e-5, rho_ratio=1000.0, g=(0.0, 0.0, 0.0), drag_model=0):
        self.N, self.Px, self.Py, self.Pz, self.cap = N, Px, Py, Pz, int(capacity)
        self.P = Px * Py * Pz
        gv = (C.c_double * 3)(*g)
        self._h = lib().orc_create(N, Px, Py, Pz, int(capacity), float(nu), float(rho_ratio), gv)
        if not self._h:
            raise ValueError("orc_create: invalid arguments")
        if lib().orc_set_drag_model(self._h, int(drag_model)):
            raise ValueError("drag_model must be 0 (Stokes) or 1 (1 + 0.15 Re^0.687)")
        self._fluid = None

    def close(self):
        if getattr(self, "_h", None):
            lib().orc_destroy(self._h)
            self._h = None

    __del__ = close

    # --- single-function views used by the pins -------------------------------------------
    def cell(self, a):
        return lib().orc_cell(self._h, float(a))

    def owner(self, x, y, z):
        return lib().orc_owner(self._h, float(x), float(y), float(z))

    def receiver(self, s, c):
        return lib().orc_receiver(self._h, int(s), int(c))

    def tau(self, d):
        return lib().orc_tau(self._h, float(d))

    def interp(self, x, y, z):
        x, y, z = _f64(x), _f64(y), _f64(z)
        ou, ov, ow = (np.empty_like(x) for _ in range(3))
        rc = lib().orc_interp(self._h, x.size, _d(x), _d(y), _d(z), _d(ou), _d(ov), _d(ow))
        if rc:
            raise RuntimeError(f"orc_interp -> {rc}")
        return ou, ov, ow

    # --- the path ------------------------------------------------------------------------
    def set_fluid(self, u, v, w):
        """u, v, w: N^3 float64 each, x fastest (flat index i + N*(j + N*k)); borrowed."""
        self._fluid = tuple(_f64(a).reshape(-1) for a in (u, v, w))
        for a in self._fluid:
            assert a.size == self.N ** 3
        return lib().orc_set_fluid(self._h, *(_d(a) for a in self._fluid))

    def set_particles(self, x, y, z, vx, vy, vz, d, id):
        arrs = [_f64(a) for a in (x, y, z, vx, vy, vz, d)]
        ids = np.ascontiguousarray(id, dtype=np.int64)
        return lib().orc_set_particles(self._h, ids.size, *(_d(a) for a in arrs), _i(ids))

    def load_packed(self, counts, x, y, z, vx, vy, vz, d, id, code=None):
        counts = np.ascontiguousarray(counts, dtype=np.int64)
        arrs = [_f64(a) for a in (x, y, z, vx, vy, vz, d)]
        ids = np.ascontiguousarray(id, dtype=np.int64)
        cp = None
        if code is not None:
            code = np.ascontiguousarray(code, dtype=np.uint8)
            cp = code.ctypes.data_as(_bp)
        return lib().orc_load_packed(self._h, _i(counts), *(_d(a) for a in arrs), _i(ids), cp)

    def push(self, dt):
        return lib().orc_push(self._h, float(dt))

    def migrate(self):
        return lib().orc_migrate(self._h)

    def step(self, dt):
        rc = self.push(dt)
        return rc if rc else self.migrate()

    def rk2_stage1(self, dt):
        return lib().orc_rk2_stage1(self._h, float(dt))

    def rk2_stage2(self, dt):
        return lib().orc_rk2_stage2(self._h, float(dt))

    def step_rk2(self, dt):
        """The paper's two-stage RK2 (Heun) with one migration per stage (R-25)."""
        for stage in (self.rk2_stage1, self.rk2_stage2):
            rc = stage(dt)
            rc = rc if rc else self.migrate()
            if rc:
                return rc
        return 0

    def classify_axis(self, axis):
        """Codes of ONE axis (0: x, 1: y, 2: z) from the current positions, relative to the slab each particle sits in."""
        return lib().orc_classify_axis(self._h, int(axis))

    def migrate_sweeps(self):
        """Axis-by-axis exchange (R-24): x, then y, then z; -> (rc, migrants moved in each sweep)."""
        moved = []
        for axis in range(3):
            rc = self.classify_axis(axis)
            rc = rc if rc else self.migrate()
            if rc:
                return rc, moved
            moved.append(self.n_migrated_last)
        return 0, moved

    @property
    def status(self):
        return lib().orc_status(self._h)

    @property
    def total(self):
        return lib().orc_total(self._h)

    @property
    def n_migrated_last(self):
        return lib().orc_n_migrated_last(self._h)

    def counts(self):
        c = np.empty(self.P, dtype=np.int64)
        lib().orc_get_counts(self._h, _i(c))
        return c

    def cnt_table(self):
        c = np.empty((self.P, 27), dtype=np.int64)
        lib().orc_get_cnt_table(self._h, _i(c))
        return c

    def get_particles(self):
        """-> dict(counts, x, y, z, vx, vy, vz, d, id, code), packed subdomain by subdomain."""
        n = self.total
        out = {k: np.empty(n, dtype=np.float64) for k in FIELDS[:7]}
        out["id"] = np.empty(n, dtype=np.int64)
        out["code"] = np.empty(n, dtype=np.uint8)
        out["counts"] = np.empty(self.P, dtype=np.int64)
        lib().orc_get_particles(self._h, _i(out["counts"]), *(_d(out[k]) for k in FIELDS[:7]),
                                _i(out["id"]), out["code"].ctypes.data_as(_bp))
        return out

    def pair_count(self, r_lo, r_hi):
        """Unordered pairs of all particles with periodic separation in [r_lo, r_hi) (O(n^2); R-26)."""
        c = lib().orc_pair_count(self._h, float(r_lo), float(r_hi))
        if c < 0:
            raise ValueError("orc_pair_count: need 0 <= r_lo < r_hi")
        return c

    def last_send_slots(self, s, n):
        o = np.empty(n, dtype=np.int64)
        lib().orc_get_last_send_slots(self._h, int(s), int(n), _i(o))
        return o
