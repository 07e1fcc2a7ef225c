"""CPU-side checks of the boundary: the C-ABI library loads, exports every symbol include/mpc_b200.h
declares, validates arguments, and its host-side Philox agrees with the known-answer vectors.
No compute call is made (no GPU here)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_2406_15236_b200 as pkg
from paper_2406_15236_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def test_header_symbols_are_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "mpc_b200.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(mpc_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(binding.SYMBOLS)
    for s in declared:
        assert hasattr(lib, s)


def test_library_philox_known_answers(lib, golden):
    for r in golden("philox_kat.txt"):
        v = [int(t, 16) for t in r]
        assert [int(o) for o in pkg.philox4x32_10(v[0:4], v[4:6])] == v[6:10]


def _create(lib, box=(8, 8, 8), cells=(8, 8, 8), npc=10.0, **kw):
    h = C.c_void_p()
    p = binding.make_params(**kw)
    rc = lib.mpc_create(C.byref(h), (C.c_float * 3)(*box), (C.c_int * 3)(*cells), npc, C.byref(p), 1)
    return rc, h


def test_create_validates_arguments(lib):
    rc, h = _create(lib)
    assert rc == 0
    nk = C.c_ulonglong()
    assert lib.mpc_num_keys(h, C.byref(nk)) == 0 and nk.value == 512
    assert lib.mpc_step(h, 1) == binding.MPC_ESTATE          # not bound
    assert b"mpc_bind" in lib.mpc_last_error(h)
    nb = C.c_size_t()
    assert lib.mpc_workspace_bytes(h, 5120, 0, C.byref(nb)) == 0
    nb2 = C.c_size_t()
    assert lib.mpc_workspace_bytes(h, 5120, 1, C.byref(nb2)) == 0
    assert 0 < nb2.value < nb.value
    assert lib.mpc_destroy(h) == 0
    assert _create(lib, box=(8, 8, 9))[0] == binding.MPC_EINVAL
    assert _create(lib, cells=(8, 8, 0))[0] == binding.MPC_EINVAL
    assert _create(lib, box=(8, 8, 2), cells=(8, 8, 2))[0] == binding.MPC_EINVAL
    assert _create(lib, rebin_every=0)[0] == binding.MPC_EINVAL
    assert _create(lib, brick=3)[0] == binding.MPC_EINVAL
    assert _create(lib, bc=(1, 0, 1))[0] == binding.MPC_EINVAL
    assert _create(lib, bc=(0, 0, 1), g=(0, 0, 0.1))[0] == binding.MPC_EINVAL
    assert _create(lib, collision=1, rebin_every=2)[0] == binding.MPC_EINVAL
    assert _create(lib, conserve_L=1, thermostat=1)[0] == binding.MPC_EINVAL
    # Lees-Edwards shear (U21): periodic SRD without +a only
    rc, h = _create(lib, shear_rate=0.05, thermostat=1)
    assert rc == 0
    lib.mpc_destroy(h)
    assert _create(lib, shear_rate=0.05, bc=(0, 0, 1))[0] == binding.MPC_EINVAL
    assert _create(lib, shear_rate=0.05, collision=1)[0] == binding.MPC_EINVAL
    assert _create(lib, shear_rate=0.05, conserve_L=1)[0] == binding.MPC_EINVAL
    rc, h = _create(lib, cells=(8, 8, 8), bc=(0, 0, 1), thermostat=1, brick=4)
    assert rc == 0
    assert lib.mpc_num_keys(h, C.byref(nk)) == 0 and nk.value == 8 * 8 * 12     # 10 layers padded to 3 bricks of 4
    lib.mpc_destroy(h)


def test_no_cpu_fallback_without_library(monkeypatch):
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", "/nonexistent/libmpc_b200.so")
    with pytest.raises(binding.MPCError):
        binding.load()


def test_wall_kinds_are_validated(lib):
    # bc: 0 periodic, 1 no-slip, 2 slip (reading U20); anything else, two wall axes, a force along the wall normal,
    # or walls with MPC-AT / +a (would need explicit phantom sets, U8) are rejected
    for bc, extra, ok in (((0, 0, 2), {}, True), ((2, 0, 0), {}, True), ((0, 0, 3), {}, False), ((0, 1, 2), {}, False),
                          ((0, 0, 2), dict(g=(0.0, 0.0, 0.1)), False), ((0, 0, 2), dict(collision=1), False),
                          ((0, 0, 2), dict(conserve_L=1), False)):
        rc, h = _create(lib, bc=bc, **extra)
        assert (rc == 0) == ok, (bc, extra, rc)
        if rc == 0:
            nk = C.c_ulonglong()
            assert lib.mpc_num_keys(h, C.byref(nk)) == 0 and nk.value == 8 * 8 * 10      # two extra layers on the wall axis
            lib.mpc_destroy(h)


def test_workspace_sizes(lib):
    # the compact workspace has no second copy of the particle arrays; both grow linearly with n_max
    rc, h = _create(lib)
    assert rc == 0
    full, comp, full2 = C.c_size_t(), C.c_size_t(), C.c_size_t()
    assert lib.mpc_workspace_bytes(h, 1 << 20, 0, C.byref(full)) == 0
    assert lib.mpc_workspace_bytes(h, 1 << 20, 1, C.byref(comp)) == 0
    assert lib.mpc_workspace_bytes(h, 1 << 21, 0, C.byref(full2)) == 0
    n = 1 << 20
    assert comp.value < full.value
    assert 17 * 4 * n <= full.value <= 17 * 4 * n + (1 << 20)        # 7 + 7 arrays, slot, key, perm, + cell data
    assert 12 * 4 * n <= comp.value <= 12 * 4 * n + (1 << 20)        # 7 arrays, 8-byte slots, spare, key, perm
    assert full2.value - full.value == 17 * 4 * n
    lib.mpc_destroy(h)
