"""Thin Python binding of the C ABI in include/mpc_b200.h: argument marshalling only.

Every step of the MPC path runs in the CUDA kernels of libmpc_b200.so. PyTorch supplies device
memory (the workspace and the I/O tensors) and the CUDA stream, nothing else. There is no CPU
fallback: if the library is missing it must be built (paper_2406_15236_b200.build), and every
compute call needs a CUDA device."""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libmpc_b200.so")

MPC_OK, MPC_EINVAL, MPC_ESTATE, MPC_ENOMEM, MPC_ECUDA, MPC_ERANGE = 0, -1, -2, -3, -4, -5
PROFILE_NOALLOC_MAX_LAYERS = 2048
DEBUG_NO_FUSE_GATHER, DEBUG_EAGER_CANONICAL, DEBUG_ATOMIC_SCATTER, DEBUG_EAGER_COLLIDE, DEBUG_NO_LANE_SPREAD = 1, 2, 4, 8, 16

# every symbol include/mpc_b200.h declares
SYMBOLS = ["mpc_create", "mpc_num_keys", "mpc_num_particles", "mpc_workspace_bytes", "mpc_bind", "mpc_set_state", "mpc_set_state_host",
           "mpc_step", "mpc_set_debug", "mpc_get_state", "mpc_get_state_host", "mpc_observables", "mpc_get_cells",
           "mpc_philox4x32_10", "mpc_launch_count", "mpc_profile_enable", "mpc_profile_read", "mpc_last_error",
           "mpc_destroy", "mpc_sub_export", "mpc_sub_connect", "mpc_sub_begin", "mpc_sub_end", "mpc_sub_pack",
           "mpc_velocity_profile_noalloc"]


class mpc_params(C.Structure):
    _fields_ = [("collision", C.c_int), ("conserve_L", C.c_int), ("thermostat", C.c_int),
                ("alpha", C.c_float), ("dt", C.c_float), ("kT", C.c_float), ("mass", C.c_float),
                ("g", C.c_float * 3), ("bc", C.c_int * 3), ("grid_shift", C.c_int),
                ("rebin_every", C.c_int), ("brick", C.c_int * 3), ("shear_rate", C.c_float),
                ("phantoms", C.c_int), ("solute_id0", C.c_uint), ("solute_mass", C.c_float), ("wall_velocity", C.c_float),
                ("sub_z0", C.c_int), ("sub_nz", C.c_int)]


class mpc_obs(C.Structure):
    _fields_ = [("n", C.c_ulonglong), ("P", C.c_double * 3), ("E_kin", C.c_double),
                ("kT_est", C.c_double), ("kT_cell", C.c_double), ("max_cell_count", C.c_uint),
                ("n_singular_cells", C.c_ulonglong), ("step", C.c_ulonglong), ("n_range_overflows", C.c_ulonglong)]


class MPCError(RuntimeError):
    pass


_lib = None


def load():
    """dlopen libmpc_b200.so and declare the prototypes. Fails loudly if the library is not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise MPCError(f"{LIB_PATH} is missing: run `python -m paper_2406_15236_b200.build` "
                       "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, ull, fp, up = C.c_void_p, C.c_ulonglong, C.c_void_p, C.c_void_p
    L.mpc_create.argtypes = [C.POINTER(vp), C.POINTER(C.c_float), C.POINTER(C.c_int), C.c_float,
                             C.POINTER(mpc_params), ull]
    L.mpc_num_keys.argtypes = [vp, C.POINTER(ull)]
    L.mpc_num_particles.argtypes = [vp, C.POINTER(ull)]
    L.mpc_workspace_bytes.argtypes = [vp, ull, C.c_int, C.POINTER(C.c_size_t)]
    L.mpc_bind.argtypes = [vp, vp, C.c_size_t, ull, vp]
    L.mpc_set_state.argtypes = [vp, ull, fp, fp, fp, fp, fp, fp, up, C.c_uint]
    L.mpc_set_state_host.argtypes = L.mpc_set_state.argtypes
    L.mpc_step.argtypes = [vp, C.c_int]
    L.mpc_set_debug.argtypes = [vp, C.c_uint]
    L.mpc_get_state.argtypes = [vp, fp, fp, fp, fp, fp, fp, up]
    L.mpc_get_state_host.argtypes = L.mpc_get_state.argtypes
    L.mpc_observables.argtypes = [vp, C.POINTER(mpc_obs), vp, C.c_int]
    L.mpc_get_cells.argtypes = [vp, up, fp, fp, fp, fp, up]
    L.mpc_philox4x32_10.argtypes = [C.POINTER(C.c_uint), C.POINTER(C.c_uint), C.POINTER(C.c_uint)]
    L.mpc_philox4x32_10.restype = None
    L.mpc_launch_count.argtypes = [vp]
    L.mpc_launch_count.restype = ull
    L.mpc_profile_enable.argtypes = [vp, C.c_int]
    L.mpc_profile_read.argtypes = [vp, C.POINTER(C.c_int), C.POINTER(C.c_char_p), C.POINTER(C.c_double), C.POINTER(ull)]
    L.mpc_last_error.argtypes = [vp]
    L.mpc_last_error.restype = C.c_char_p
    L.mpc_destroy.argtypes = [vp]
    L.mpc_sub_export.argtypes = [vp, C.POINTER(vp), C.POINTER(C.c_int)]
    L.mpc_sub_connect.argtypes = [vp, C.POINTER(vp), C.c_int, C.POINTER(vp), C.c_int]
    L.mpc_sub_begin.argtypes = [vp, C.c_int]
    L.mpc_sub_end.argtypes = [vp]
    L.mpc_sub_pack.argtypes = [vp, fp, fp, fp, fp, fp, fp, up, C.POINTER(ull)]
    L.mpc_velocity_profile_noalloc.argtypes = [vp, ull, fp, fp, C.c_int, fp, up, vp]
    for s in SYMBOLS:
        getattr(L, s)
    _lib = L
    return L


def philox4x32_10(ctr, key):
    c = (C.c_uint * 4)(*[int(v) for v in ctr])
    k = (C.c_uint * 2)(*[int(v) for v in key])
    o = (C.c_uint * 4)()
    load().mpc_philox4x32_10(c, k, o)
    return np.array(o[:], np.uint32)


def make_params(collision=0, conserve_L=0, thermostat=0, alpha_deg=130.0, dt=0.1, kT=1.0, mass=1.0,
                g=(0.0, 0.0, 0.0), bc=(0, 0, 0), grid_shift=1, rebin_every=1, brick=1, shear_rate=0.0,
                phantoms=0, solute_id0=0, solute_mass=0.0, wall_velocity=0.0, sub=(0, 0)):
    p = mpc_params()
    p.sub_z0, p.sub_nz = sub
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


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


class MPC:
    """One MPC system on one GPU. Tensors passed in/out are torch CUDA tensors (device API) or
    pinned/pageable host tensors / numpy arrays (the *_host API)."""

    def __init__(self, box, cells, n_per_cell, seed, n_max, device="cuda:0", compact=False, stream=None, workspace_alloc=None, **kw):
        """workspace_alloc: optional callable bytes -> device pointer (int) for a workspace the caller owns (e.g. memory that
        can be shared with other processes: slab_run.py); default: a torch uint8 tensor"""
        import torch

        self._torch = torch
        self.lib = load()
        self.params = make_params(**kw)
        self._h = C.c_void_p()
        rc = self.lib.mpc_create(C.byref(self._h), (C.c_float * 3)(*box), (C.c_int * 3)(*cells),
                                 float(n_per_cell), C.byref(self.params), int(seed))
        if rc != MPC_OK:
            self._h = None
            raise MPCError(f"mpc_create failed: {rc}")
        nk = C.c_ulonglong()
        self._check(self.lib.mpc_num_keys(self._h, C.byref(nk)))
        self.nkeys = nk.value
        self.box, self.cells, self.n_max = tuple(box), tuple(cells), int(n_max)
        self.device = torch.device(device)
        nbytes = C.c_size_t()
        self._check(self.lib.mpc_workspace_bytes(self._h, self.n_max, 1 if compact else 0, C.byref(nbytes)))
        self.workspace_bytes = nbytes.value
        with torch.cuda.device(self.device):      # mpc_bind records the current device; later calls switch to it themselves
            if workspace_alloc is None:
                self.workspace = torch.empty(nbytes.value, dtype=torch.uint8, device=self.device)
                self.workspace_ptr = self.workspace.data_ptr()
            else:
                self.workspace = None
                self.workspace_ptr = int(workspace_alloc(nbytes.value))
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self._check(self.lib.mpc_bind(self._h, C.c_void_p(self.workspace_ptr), nbytes.value, self.n_max,
                                          C.c_void_p(self.stream.cuda_stream)))

    @property
    def n(self):
        """current number of particles (a slab subdomain's changes when a reorder hands particles over)"""
        v = C.c_ulonglong()
        self._check(self.lib.mpc_num_particles(self._h, C.byref(v)))
        return int(v.value)

    def _check(self, rc):
        if rc != MPC_OK:
            msg = self.lib.mpc_last_error(self._h).decode() if self._h else ""
            raise MPCError(f"mpc error {rc}: {msg}")

    # ---- slab subdomains of a multi-GPU run (include/mpc_b200.h "slab subdomains") ----
    def sub_export(self):
        """([cell sums, cell offsets, staging buffer] device pointers, local brick layers) of this rank, to hand to its neighbours"""
        p, nb = (C.c_void_p * 3)(), C.c_int()
        self._check(self.lib.mpc_sub_export(self._h, p, C.byref(nb)))
        return [int(v or 0) for v in p], nb.value

    def sub_connect(self, below, above):
        """below / above = sub_export() of the neighbours towards smaller / larger z (peer memory reachable from this device)"""
        pb, pa = (C.c_void_p * 3)(*below[0]), (C.c_void_p * 3)(*above[0])
        self._check(self.lib.mpc_sub_connect(self._h, pb, below[1], pa, above[1]))

    def sub_begin(self, steps_ahead=0):
        self._check(self.lib.mpc_sub_begin(self._h, int(steps_ahead)))

    def sub_end(self):
        self._check(self.lib.mpc_sub_end(self._h))

    def sub_pack(self):
        """the state class by class: ([x, y, z, vx, vy, vz, id] device tensors of the current length, (n_stay, n_below, n_above))"""
        torch = self._torch
        n = max(self.n, 1)
        with torch.cuda.device(self.device):
            out = [torch.empty(n, dtype=torch.float32, device=self.device) for _ in range(6)] + [torch.empty(n, dtype=torch.int32, device=self.device)]
        cnt = (C.c_ulonglong * 3)()
        self._check(self.lib.mpc_sub_pack(self._h, *[_ptr(t) for t in out], cnt))
        return [t[:self.n] for t in out], tuple(int(v) for v in cnt)

    def close(self):
        if getattr(self, "_h", None):
            self.lib.mpc_destroy(self._h)
            self._h = None

    def __del__(self):
        self.close()

    # ---- state ----
    def set_state(self, x, y, z, vx, vy, vz, id=None, step=0):
        ts = [x, y, z, vx, vy, vz]
        for t in ts:
            assert t.is_cuda and t.dtype == self._torch.float32 and t.is_contiguous()
        self._check(self.lib.mpc_set_state(self._h, ts[0].numel(), *[_ptr(t) for t in ts], _ptr(id), step))

    def set_state_host(self, x, y, z, vx, vy, vz, id=None, step=0):
        """Host arrays: numpy arrays or CPU torch tensors (pinned makes the copies asynchronous)."""
        torch = self._torch
        ts = [torch.as_tensor(a) for a in (x, y, z, vx, vy, vz)]
        for t in ts:
            assert (not t.is_cuda) and t.dtype == torch.float32 and t.is_contiguous()
        idt = None if id is None else torch.as_tensor(id)
        self._keep = (ts, idt)
        self._check(self.lib.mpc_set_state_host(self._h, ts[0].numel(), *[_ptr(t) for t in ts], _ptr(idt), step))

    def step(self, nsteps=1):
        self._check(self.lib.mpc_step(self._h, int(nsteps)))

    def get_state(self):
        torch = self._torch
        out = [torch.empty(self.n, dtype=torch.float32, device=self.device) for _ in range(6)]
        ids = torch.empty(self.n, dtype=torch.int32, device=self.device)
        self._check(self.lib.mpc_get_state(self._h, *[_ptr(t) for t in out], _ptr(ids)))
        return (*out, ids)

    def canonicalise(self):
        """Bring the state into the form mpc_get_state returns (last collision applied, (key, id) order inside every
        cell) without copying anything out: indices into the internal order stay valid until the next step."""
        self._check(self.lib.mpc_get_state(self._h, *([None] * 7)))

    def get_state_at(self, index):
        """Particles `index` (a device int64 tensor of positions in the current internal order) as seven host numpy
        arrays (x,y,z,vx,vy,vz,id). Pulls one full array at a time through mpc_get_state (NULL = skipped), so it needs
        4 n bytes of device memory beside the workspace instead of 28 n."""
        torch = self._torch
        res = []
        for a in range(7):
            buf = torch.empty(self.n, dtype=torch.float32 if a < 6 else torch.int32, device=self.device)
            ptrs = [None] * 7
            ptrs[a] = C.c_void_p(buf.data_ptr())
            self._check(self.lib.mpc_get_state(self._h, *ptrs))
            res.append(buf[index].cpu().numpy())
            del buf
        res[6] = res[6].view(np.uint32)
        return tuple(res)

    def get_state_host(self, out=None):
        """Returns numpy arrays (x,y,z,vx,vy,vz,id); `out` may supply 7 pre-allocated host tensors."""
        torch = self._torch
        if out is None:
            out = [torch.empty(self.n, dtype=torch.float32) for _ in range(6)] + [torch.empty(self.n, dtype=torch.int32)]
        self._check(self.lib.mpc_get_state_host(self._h, *[_ptr(t) for t in out]))
        res = [t.numpy() for t in out]
        res[6] = res[6].view(np.uint32)
        return tuple(res)

    def get_cells(self):
        torch = self._torch
        cnt = torch.empty(self.nkeys, dtype=torch.int32, device=self.device)
        p = [torch.empty(self.nkeys, dtype=torch.float32, device=self.device) for _ in range(4)]
        key = torch.empty(self.n, dtype=torch.int32, device=self.device)
        self._check(self.lib.mpc_get_cells(self._h, _ptr(cnt), *[_ptr(t) for t in p], _ptr(key)))
        return cnt, p[0], p[1], p[2], p[3], key

    def set_debug(self, flags):
        self._check(self.lib.mpc_set_debug(self._h, int(flags)))

    @property
    def profile_layers(self):
        """Number of entries of the velocity profile: the fluid cells along the wall axis (z without walls)."""
        bc = tuple(self.params.bc)
        axis = max((d for d in range(3) if bc[d] != 0), default=2)
        return self.cells[axis]

    def observables(self, profile=False):
        """System observables as a dict; profile=True adds the layer-averaged velocity profile (profile_layers floats).
        A range overflow of the fixed-point sums (MPC_ERANGE) is reported as d["n_range_overflows"] != 0, not raised."""
        o = mpc_obs()
        nb = self.profile_layers
        prof = np.zeros(nb, np.float32)            # sized by the library's own rule, never by the caller
        rc = self.lib.mpc_observables(self._h, C.byref(o), prof.ctypes.data_as(C.c_void_p) if profile else None, nb)
        if rc != MPC_ERANGE:
            self._check(rc)
        d = dict(n=o.n, P=np.array(o.P[:]), E_kin=o.E_kin, kT_est=o.kT_est, kT_cell=o.kT_cell,
                 max_cell_count=o.max_cell_count, n_singular_cells=o.n_singular_cells, step=o.step,
                 n_range_overflows=o.n_range_overflows)
        if profile:
            d["profile"] = prof
        return d

    def velocity_profile_noalloc(self, r_w, v_f, profile, counts=None, stream=None):
        """mpc_velocity_profile_noalloc: the layer averages of v_f over the layers floor(r_w / a), written into the caller's
        float32 device tensor `profile` (its length is the number of layers, at most PROFILE_NOALLOC_MAX_LAYERS); `counts`:
        optional int64 device tensor of the same length for the particles per layer. For callers that cannot allocate device
        memory: the library's scratch for this call is a fixed array inside its own image, so nothing is allocated here either
        (all four tensors are the caller's) and no workspace is touched. Enqueues on `stream` (default: the current stream
        of the tensors' device, which must be the current device) and does not synchronise. Calls that may overlap on the
        GPU share that one array and race; see include/mpc_b200.h."""
        torch = self._torch
        for t in (r_w, v_f, profile):
            assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
        assert r_w.numel() == v_f.numel()
        assert counts is None or (counts.is_cuda and counts.dtype == torch.int64 and counts.is_contiguous() and counts.numel() == profile.numel())
        s = stream if stream is not None else torch.cuda.current_stream(profile.device)
        self._check(self.lib.mpc_velocity_profile_noalloc(self._h, r_w.numel(), _ptr(r_w), _ptr(v_f), profile.numel(), _ptr(profile),
                                                          _ptr(counts), C.c_void_p(s.cuda_stream)))

    def profile_enable(self, on=True):
        self._check(self.lib.mpc_profile_enable(self._h, 1 if on else 0))

    def profile_read(self):
        """{family: (total_ms, timed_sections)} since the last read; synchronises the stream."""
        n = C.c_int()
        names = (C.c_char_p * 16)()
        ms = (C.c_double * 16)()
        cnt = (C.c_ulonglong * 16)()
        self._check(self.lib.mpc_profile_read(self._h, C.byref(n), names, ms, cnt))
        return {names[i].decode(): (ms[i], cnt[i]) for i in range(n.value)}

    @property
    def launch_count(self):
        return int(self.lib.mpc_launch_count(self._h))
