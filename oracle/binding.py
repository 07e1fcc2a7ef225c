"""ctypes wrapper around oracle/liboracle_mpc.so (TEST INFRASTRUCTURE, not the product).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import
this module. It shares nothing with paper_2406_15236_b200 (the parameter struct is re-typed).
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_f32p = np.ctypeslib.ndpointer(dtype=np.float32, flags="C_CONTIGUOUS")
_u32p = np.ctypeslib.ndpointer(dtype=np.uint32, flags="C_CONTIGUOUS")
_f64p = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_i32p = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")


class OracleParams(C.Structure):
    _fields_ = [("collision", C.c_int), ("conserve_L", C.c_int), ("thermostat", C.c_int),
                ("alpha", C.c_float), ("dt", C.c_float), ("kT", C.c_float), ("mass", C.c_float),
                ("g", C.c_float * 3), ("bc", C.c_int * 3), ("grid_shift", C.c_int),
                ("rebin_every", C.c_int), ("brick", C.c_int * 3), ("shear_rate", C.c_float),
                ("phantoms", C.c_int), ("solute_id0", C.c_uint), ("solute_mass", C.c_float), ("wall_velocity", C.c_float)]


class OracleObs(C.Structure):
    _fields_ = [("n", C.c_ulonglong), ("P", C.c_double * 3), ("E_kin", C.c_double),
                ("kT_est", C.c_double), ("kT_cell", C.c_double), ("max_cell_count", C.c_uint),
                ("n_singular_cells", C.c_ulonglong), ("step", C.c_ulonglong)]


_lib = None
_lib_path = None     # set before the first call to load another build of the oracle (the sanitizer build: tests/test_oracle_sanitize.py)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_lib_path or _build.build())
        _lib.oracle_create.argtypes = [C.POINTER(C.c_void_p), C.POINTER(C.c_float), C.POINTER(C.c_int), C.c_float,
                                       C.POINTER(OracleParams), C.c_ulonglong]
        _lib.oracle_destroy.argtypes = [C.c_void_p]
        _lib.oracle_num_keys.argtypes = [C.c_void_p, C.POINTER(C.c_ulonglong)]
        _lib.oracle_set_state.argtypes = [C.c_void_p, C.c_ulonglong] + [_f32p] * 6 + [C.c_void_p, C.c_uint]
        _lib.oracle_step.argtypes = [C.c_void_p, C.c_int]
        _lib.oracle_get_state.argtypes = [C.c_void_p] + [_f32p] * 6 + [_u32p]
        _lib.oracle_get_cells.argtypes = [C.c_void_p, _u32p, _f64p, _f64p, _f64p, _f64p, _u32p]
        _lib.oracle_observables.argtypes = [C.c_void_p, C.POINTER(OracleObs), C.c_void_p]
        _lib.oracle_philox4x32_10.argtypes = [_u32p, _u32p, _u32p]
        _lib.oracle_philox4x32_10.restype = None
        _lib.oracle_grid_shift.argtypes = [C.c_void_p, C.c_uint, _f32p]
        _lib.oracle_srd_axis.argtypes = [C.c_void_p, C.c_uint, C.c_uint, _f64p]
        _lib.oracle_mbs_energy.argtypes = [C.c_void_p, C.c_uint, C.c_uint, C.c_uint, C.POINTER(C.c_double)]
        _lib.oracle_normals.argtypes = [C.c_void_p, C.c_uint, C.c_uint, C.c_uint, C.c_uint, _f64p]
        _lib.oracle_cell_of.argtypes = [C.c_void_p, _f32p, _f32p, _i32p, C.POINTER(C.c_uint), C.POINTER(C.c_uint), _f32p]
        _lib.oracle_stream_one.argtypes = [C.c_void_p, _f32p, _f32p]
        _lib.oracle_collide_one_cell.argtypes = [C.c_void_p, C.c_uint, C.c_uint, C.c_void_p, C.c_void_p]
        _lib.oracle_stream_one_at.argtypes = [C.c_void_p, C.c_uint, _f32p, _f32p]
        _lib.oracle_cell_of_le.argtypes = [C.c_void_p, C.c_uint, _f32p, _f32p, _i32p, C.POINTER(C.c_uint), C.POINTER(C.c_uint),
                                           C.POINTER(C.c_int)]
        _lib.oracle_phantoms.argtypes = [C.c_void_p, _i32p, _f32p, C.c_uint, C.c_int, _f64p, _f64p, C.POINTER(C.c_int)]
        _lib.oracle_le_offset.argtypes = [C.c_void_p, C.c_uint, C.POINTER(C.c_float), C.POINTER(C.c_float)]
    return _lib


def philox(ctr, key):
    out = np.zeros(4, np.uint32)
    lib().oracle_philox4x32_10(np.asarray(ctr, np.uint32), np.asarray(key, np.uint32), out)
    return out


def make_params(collision=0, conserve_L=0, thermostat=0, alpha_deg=130.0, dt=0.1, kT=1.0, mass=1.0,
                g=(0.0, 0.0, 0.0), bc=(0, 0, 0), grid_shift=1, rebin_every=1, brick=1, shear_rate=0.0,
                phantoms=0, solute_id0=0, solute_mass=0.0, wall_velocity=0.0):
    p = OracleParams()
    p.phantoms, p.solute_id0, p.solute_mass, p.wall_velocity = phantoms, solute_id0, solute_mass, wall_velocity
    p.shear_rate = shear_rate
    p.collision, p.conserve_L, p.thermostat = collision, conserve_L, thermostat
    p.alpha = np.float32(np.deg2rad(alpha_deg))
    p.dt, p.kT, p.mass = dt, kT, mass
    p.g[:] = g
    p.bc[:] = bc
    p.grid_shift, p.rebin_every = grid_shift, rebin_every
    p.brick[:] = (brick,) * 3 if isinstance(brick, int) else tuple(brick)
    return p


class Oracle:
    """One MPC system advanced by the CPU oracle. Arrays are host numpy arrays."""

    def __init__(self, box, cells, n_per_cell, seed, **kw):
        self.params = make_params(**kw)
        self._h = C.c_void_p()
        b = (C.c_float * 3)(*box)
        c = (C.c_int * 3)(*cells)
        rc = lib().oracle_create(C.byref(self._h), b, c, n_per_cell, C.byref(self.params), seed)
        if rc != 0:
            raise ValueError(f"oracle_create failed: {rc}")
        nk = C.c_ulonglong()
        lib().oracle_num_keys(self._h, C.byref(nk))
        self.nkeys = nk.value
        self.cells = tuple(cells)
        self.box = tuple(box)
        self.n = 0

    def __del__(self):
        if getattr(self, "_h", None):
            lib().oracle_destroy(self._h)
            self._h = None

    def set_state(self, x, y, z, vx, vy, vz, id=None, step=0):
        arrs = [np.ascontiguousarray(a, np.float32) for a in (x, y, z, vx, vy, vz)]
        self.n = arrs[0].size
        idp = None
        if id is not None:
            self._id = np.ascontiguousarray(id, np.uint32)
            idp = self._id.ctypes.data_as(C.c_void_p)
        rc = lib().oracle_set_state(self._h, self.n, *arrs, idp, step)
        if rc != 0:
            raise RuntimeError(f"oracle_set_state failed: {rc}")

    def step(self, nsteps=1):
        rc = lib().oracle_step(self._h, nsteps)
        if rc != 0:
            raise RuntimeError(f"oracle_step failed: {rc}")

    def get_state(self):
        out = [np.empty(self.n, np.float32) for _ in range(6)]
        ids = np.empty(self.n, np.uint32)
        rc = lib().oracle_get_state(self._h, *out, ids)
        if rc != 0:
            raise RuntimeError(f"oracle_get_state failed: {rc}")
        return (*out, ids)

    def get_cells(self):
        cnt = np.empty(self.nkeys, np.uint32)
        p = [np.empty(self.nkeys, np.float64) for _ in range(4)]
        key = np.empty(self.n, np.uint32)
        rc = lib().oracle_get_cells(self._h, cnt, *p, key)
        if rc != 0:
            raise RuntimeError(f"oracle_get_cells failed: {rc}")
        return cnt, p[0], p[1], p[2], p[3], key

    def observables(self, profile_bins=0):
        o = OracleObs()
        prof = np.zeros(max(profile_bins, 1), np.float32)
        rc = lib().oracle_observables(self._h, C.byref(o), prof.ctypes.data_as(C.c_void_p) if profile_bins else None)
        if rc != 0:
            raise RuntimeError(f"oracle_observables failed: {rc}")
        d = dict(n=o.n, P=np.array(o.P[:]), E_kin=o.E_kin, kT_est=o.kT_est, kT_cell=o.kT_cell,
                 max_cell_count=o.max_cell_count, n_singular_cells=o.n_singular_cells, step=o.step)
        if profile_bins:
            d["profile"] = prof
        return d

    # hooks
    def grid_shift(self, t):
        s = np.zeros(3, np.float32)
        lib().oracle_grid_shift(self._h, t, s)
        return s

    def srd_axis(self, cid, t):
        n = np.zeros(3, np.float64)
        lib().oracle_srd_axis(self._h, cid, t, n)
        return n

    def mbs_energy(self, cid, t, Nc):
        e = C.c_double()
        lib().oracle_mbs_energy(self._h, cid, t, Nc, C.byref(e))
        return e.value

    def normals(self, index, sub, t, tag):
        g = np.zeros(4, np.float64)
        lib().oracle_normals(self._h, index, sub, t, tag, g)
        return g

    def cell_of(self, r, s):
        ijk = np.zeros(3, np.int32)
        rho = np.zeros(3, np.float32)
        cid, key = C.c_uint(), C.c_uint()
        lib().oracle_cell_of(self._h, np.asarray(r, np.float32), np.asarray(s, np.float32), ijk, C.byref(cid),
                             C.byref(key), rho)
        return ijk, cid.value, key.value, rho

    def stream_one(self, r, v):
        r = np.array(r, np.float32)
        v = np.array(v, np.float32)
        lib().oracle_stream_one(self._h, r, v)
        return r, v

    def stream_one_at(self, t, r, v):
        r = np.array(r, np.float32)
        v = np.array(v, np.float32)
        lib().oracle_stream_one_at(self._h, t, r, v)
        return r, v

    def cell_of_le(self, t, r, s):
        ijk = np.zeros(3, np.int32)
        cid, key, im = C.c_uint(), C.c_uint(), C.c_int()
        lib().oracle_cell_of_le(self._h, t, np.asarray(r, np.float32), np.asarray(s, np.float32), ijk, C.byref(cid),
                                C.byref(key), C.byref(im))
        return ijk, cid.value, key.value, im.value

    def phantoms(self, ijk, s, t, cap=256):
        """Explicit phantom particles (reading U22) of cell ijk: (rho[n,3] cell-local coordinates, v[n,3])."""
        rho, v, n = np.zeros(3 * cap), np.zeros(3 * cap), C.c_int()
        rc = lib().oracle_phantoms(self._h, np.asarray(ijk, np.int32), np.asarray(s, np.float32), t, cap, rho, v, C.byref(n))
        if rc != 0:
            raise RuntimeError(f"oracle_phantoms failed: {rc}")
        return rho[:3 * n.value].reshape(-1, 3), v[:3 * n.value].reshape(-1, 3)

    def le_offset(self, t):
        d, u = C.c_float(), C.c_float()
        lib().oracle_le_offset(self._h, t, C.byref(d), C.byref(u))
        return d.value, u.value

    def collide_one_cell(self, cid=0, t=0, axis=None, kappa=None):
        ax = np.asarray(axis, np.float64) if axis is not None else None
        kp = C.c_double(kappa) if kappa is not None else None
        rc = lib().oracle_collide_one_cell(self._h, cid, t, ax.ctypes.data_as(C.c_void_p) if ax is not None else None,
                                           C.byref(kp) if kp is not None else None)
        if rc != 0:
            raise RuntimeError(f"oracle_collide_one_cell failed: {rc}")
