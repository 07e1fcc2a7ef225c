"""mpc_velocity_profile_noalloc: the one entry point for callers that cannot allocate device memory.

Who that is: a monitoring / in-situ analysis hook called from inside another program's time loop, where that program's
caching allocator already holds nearly the whole GPU (a direct cudaMalloc fails, or stalls every stream while it runs),
code that must not allocate after start-up, or a caller that only has pointers handed to it by another runtime. The
library's usual contract (the caller allocates a workspace for mpc_bind) is no help to them, so this call keeps its
accumulation buffer in a fixed 32 KiB array inside the library image and needs a context from mpc_create only.

Checked here, on the GPU: its output against the existing path (the profile of mpc_observables, which works in the bound
workspace) for the same particles, at the tolerance the profile comparisons of the other tests use (1e-5 absolute;
the fixed-point sums in fact make the two equal), on calls made one after the other: the built-in array is shared by all
calls and keeps the last call's sums, so a call that did not clear it would fail the second comparison. The context given
to the new call is a fresh, unbound one: no workspace exists for it.

The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here must not hide the parity
tests. It runs on its own (`pytest tests/test_zz_no_alloc.py -m gpu`) as well as after the others."""
import ctypes as C

import numpy as np
import pytest

from paper_2406_15236_b200 import binding, build

PROFILE_TOL = 1e-5      # tests/test_parity_gpu.py::test_observables_match_oracle


def _unbound_context(lib, box, cells, nbar, **kw):
    """mpc_create only: host memory, no mpc_bind, no workspace"""
    h = C.c_void_p()
    p = binding.make_params(**kw)
    assert lib.mpc_create(C.byref(h), (C.c_float * 3)(*box), (C.c_int * 3)(*cells), float(nbar), C.byref(p), 1) == binding.MPC_OK
    return h


def test_more_layers_than_the_builtin_array_holds_are_refused():
    # no GPU needed: the size check comes before any CUDA call
    build.build()
    lib = binding.load()
    h = _unbound_context(lib, (8.0, 8.0, 8.0), (8, 8, 8), 10)
    one = C.c_void_p(256)      # never dereferenced: the call returns before it touches the device
    too_many = binding.PROFILE_NOALLOC_MAX_LAYERS + 1
    assert lib.mpc_velocity_profile_noalloc(h, 0, None, None, too_many, one, None, None) == binding.MPC_EINVAL
    msg = lib.mpc_last_error(h).decode()
    assert "MPC_PROFILE_NOALLOC_MAX_LAYERS" in msg and "2048" in msg
    assert lib.mpc_velocity_profile_noalloc(h, 0, None, None, 0, one, None, None) == binding.MPC_EINVAL
    assert lib.mpc_velocity_profile_noalloc(h, 0, None, None, 8, None, None, None) == binding.MPC_EINVAL
    assert lib.mpc_velocity_profile_noalloc(h, 5, None, None, 8, one, None, None) == binding.MPC_EINVAL
    assert lib.mpc_velocity_profile_noalloc(None, 0, None, None, 8, one, None, None) == binding.MPC_EINVAL
    lib.mpc_destroy(h)


@pytest.mark.gpu
def test_noalloc_profile_equals_the_workspace_path_on_calls_in_a_row():
    torch = pytest.importorskip("torch")
    from paper_2406_15236_b200 import MPC
    from paper_2406_15236_b200.inputs import uniform_maxwell

    lib = binding.load()
    # a slit along z with a driven flow along x (the kind of run the profile is for), several warps per layer and a ragged tail
    cells, nbar = (12, 8, 10), 10
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar + 37
    kw = dict(thermostat=1, bc=(0, 0, 1), g=(0.05, 0.0, 0.0), rebin_every=4, brick=4)
    g = MPC(box, cells, nbar, 99, n_max=n, **kw)
    st = uniform_maxwell(box, n, 5)
    g.set_state(*[torch.from_numpy(a).cuda() for a in st[:6]])
    h = _unbound_context(lib, box, cells, nbar, **kw)
    nb = cells[2]
    # the caller's own buffers, made once, before the calls (the entry point itself allocates nothing)
    prof = torch.full((nb,), float("nan"), dtype=torch.float32, device="cuda")
    cnt = torch.full((nb,), -1, dtype=torch.int64, device="cuda")
    stream = torch.cuda.current_stream()

    def both(steps):
        g.step(steps)
        ref = g.observables(profile=True)["profile"]                    # existing path: scratch in the bound workspace
        x, y, z, vx, vy, vz, ids = g.get_state()
        rc = lib.mpc_velocity_profile_noalloc(h, n, C.c_void_p(z.data_ptr()), C.c_void_p(vx.data_ptr()), nb, C.c_void_p(prof.data_ptr()),
                                              C.c_void_p(cnt.data_ptr()), C.c_void_p(stream.cuda_stream))
        assert rc == binding.MPC_OK, lib.mpc_last_error(h).decode()
        torch.cuda.synchronize()
        layer = np.clip(np.floor(z.cpu().numpy()).astype(np.int64), 0, nb - 1)      # a = 1
        return ref, prof.cpu().numpy().copy(), cnt.cpu().numpy().copy(), np.bincount(layer, minlength=nb)

    ref1, out1, cnt1, lay1 = both(3)
    assert np.abs(ref1).max() > 0.05                                    # a real flow, not a row of zeros
    assert np.allclose(out1, ref1, rtol=0, atol=PROFILE_TOL)
    assert np.array_equal(cnt1, lay1) and cnt1.sum() == n
    # second call straight after the first, other velocities: the array still holds the first call's sums when it starts
    ref2, out2, cnt2, lay2 = both(6)
    assert np.abs(ref2 - ref1).max() > 1e-3
    assert np.allclose(out2, ref2, rtol=0, atol=PROFILE_TOL)
    assert np.array_equal(cnt2, lay2) and cnt2.sum() == n
    # third and fourth: fewer layers than before (the words beyond them keep old sums, which must not matter), then
    # no particles at all; through the binding's method this time, on the bound context
    x, y, z, vx, vy, vz, ids = g.get_state()
    half = torch.empty(nb // 2, dtype=torch.float32, device="cuda")
    g.velocity_profile_noalloc(z, vx, half)
    torch.cuda.synchronize()
    zz, vv = z.cpu().numpy().astype(np.float64), vx.cpu().numpy().astype(np.float64)
    lay = np.clip(np.floor(zz).astype(np.int64), 0, nb // 2 - 1)
    want = np.bincount(lay, weights=vv, minlength=nb // 2) / np.bincount(lay, minlength=nb // 2)
    assert np.allclose(half.cpu().numpy(), want, rtol=0, atol=PROFILE_TOL)
    g.velocity_profile_noalloc(z[:0], vx[:0], prof, counts=cnt)
    torch.cuda.synchronize()
    assert np.all(prof.cpu().numpy() == 0.0) and np.all(cnt.cpu().numpy() == 0)
    lib.mpc_destroy(h)
    g.close()
