"""GPU parity for the angular-momentum-conserving variants SRD+a (Eqs. 3-4) and
MPC-AT+a (U5). Tolerance = SURVEY.md 8(c) reading U10: 2e-5 sqrt(kT/m) for particles of cells whose inertia
tensor has condition number <= 10^2, 1e-3 otherwise (omega = I^-1 dL amplifies fp32 rounding of the per-particle
omega x r_c by the conditioning); the fraction of loosely compared particles is printed. No cell is exempt: the
rejection rule of U10 is evaluated in double on both sides, so both must reject the same cells (equal counts)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle.binding import Oracle  # noqa: E402
from paper_2406_15236_b200 import MPC  # noqa: E402
from paper_2406_15236_b200.inputs import uniform_maxwell  # noqa: E402
from test_parity_gpu import gpu_get, gpu_set  # noqa: E402


def lambda_min_per_particle(o, so, key, step):
    """Per particle: smallest eigenvalue of its cell's inertia tensor / (m a^2) (N=2: sum |r|^2), the cell's occupancy,
    and the condition number of the tensor (1 for N <= 2, where U10 does not invert a tensor)."""
    s = o.grid_shift(step).astype(np.float32)
    q = np.stack(so[0:3], 1) + s
    rho = (q - np.floor(q)).astype(np.float64)
    nk = o.nkeys
    key = key.astype(np.int64)
    N = np.bincount(key, minlength=nk).astype(float)
    rcm = np.stack([np.bincount(key, weights=rho[:, d], minlength=nk) / np.maximum(N, 1) for d in range(3)], 1)
    r = rho - rcm[key]
    r2 = (r**2).sum(1)
    I = np.zeros((nk, 3, 3))
    for a in range(3):
        for b in range(3):
            I[:, a, b] = np.bincount(key, weights=(r2 if a == b else 0) - r[:, a] * r[:, b], minlength=nk)
    ev = np.linalg.eigvalsh(I)
    lam = np.where(N == 2, np.bincount(key, weights=r2, minlength=nk), ev[:, 0])
    with np.errstate(invalid="ignore", divide="ignore"):
        cond = np.where(N >= 3, ev[:, 2] / np.maximum(ev[:, 0], 1e-300), 1.0)
    return lam[key], N[key], cond[key]


def check_plus_a_velocities(so, sg, cond, label=""):
    """U10 tolerance: 2e-5 where cond(I_c) <= 1e2, 1e-3 elsewhere; returns the fraction compared loosely."""
    err = np.max(np.abs(np.stack(so[3:6]).astype(np.float64) - np.stack(sg[3:6])), axis=0)
    loose = cond > 1e2
    tol = np.where(loose, 1e-3, 2e-5)
    worst = int(np.argmax(err / tol))
    assert (err <= tol).all(), f"{label}: err {err[worst]:.3g} > tol {tol[worst]:.3g} at cond {cond[worst]:.3g}"
    print(f"{label}: max err strict {err[~loose].max(initial=0):.3g}, loose {err[loose].max(initial=0):.3g}, "
          f"loosely compared fraction {loose.mean():.4f}")
    return loose.mean()


@pytest.mark.parametrize("collision,nbar,every,brick", [(0, 10, 1, 4), (0, 10, 3, (16, 16, 8)), (0, 3, 1, 1),
                                                         (1, 10, 1, 4), (1, 3, 1, (4, 2, 1))])
def test_plus_a_parity(collision, nbar, every, brick):
    cells = (16, 16, 8)
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar + 11
    st = uniform_maxwell(box, n, 5)
    kw = dict(collision=collision, conserve_L=1, dt=0.05, brick=brick, rebin_every=every)
    o = Oracle(box, cells, nbar, 77, **kw)
    g = MPC(box, cells, nbar, 77, n_max=n, **kw)
    o.set_state(*st)
    for t in range(every + 1):
        gpu_set(g, o.get_state(), step=t)
        o.step(1)
        g.step(1)
        so, sg = o.get_state(), gpu_get(g)
        assert np.array_equal(so[6], sg[6])                                   # sort order
        for d in range(3):
            assert np.max(np.abs(so[d] - sg[d])) <= 1e-5
        cnt_o, px, py, pz, _e, key_o = o.get_cells()
        cnt_g, gx, gy, gz, _ge, key_g = [a.cpu().numpy() for a in g.get_cells()]
        assert np.array_equal(key_o, key_g.view(np.uint32))
        assert np.array_equal(cnt_o, cnt_g.view(np.uint32))
        _lam, _N, cond = lambda_min_per_particle(o, so, key_o, t)
        frac = check_plus_a_velocities(so, sg, cond, f"collision={collision} nbar={nbar} t={t}")
        if nbar == 10:
            assert frac < 0.05
        assert int(o.observables()["n_singular_cells"]) == int(g.observables()["n_singular_cells"])


@pytest.mark.parametrize("collision", [0, 1])
def test_plus_a_conserves_angular_momentum_on_gpu(collision):
    # the invariant itself, measured on the GPU output (not only agreement with the oracle)
    cells, nbar = (12, 12, 12), 10
    box = (12.0, 12.0, 12.0)
    n = 12**3 * nbar
    st = uniform_maxwell(box, n, 9)
    kw = dict(collision=collision, conserve_L=1, dt=0.05, brick=4)
    g = MPC(box, cells, nbar, 5, n_max=n, **kw)
    gpu_set(g, st)
    g.step(1)
    x, y, z, vx, vy, vz, ids = gpu_get(g)
    key = g.get_cells()[5].cpu().numpy().view(np.uint32).astype(np.int64)
    order = np.argsort(ids)
    o = Oracle(box, cells, nbar, 5, **kw)
    s = o.grid_shift(0).astype(np.float32)
    q = np.stack([x, y, z], 1)[order] + s
    rho = (q - np.floor(q)).astype(np.float64)
    key = key[order]
    nk = g.nkeys
    N = np.bincount(key, minlength=nk).astype(float)
    rcm = np.stack([np.bincount(key, weights=rho[:, d], minlength=nk) / np.maximum(N, 1) for d in range(3)], 1)
    r = rho - rcm[key]
    pre = np.stack(st[3:6], 1).astype(np.float64)
    post = np.stack([vx, vy, vz], 1).astype(np.float64)[order]
    L0 = np.stack([np.bincount(key, weights=np.cross(r, pre)[:, d], minlength=nk) for d in range(3)], 1)
    L1 = np.stack([np.bincount(key, weights=np.cross(r, post)[:, d], minlength=nk) for d in range(3)], 1)
    scale = np.bincount(key, weights=np.abs(pre).sum(1), minlength=nk) + 1e-30
    rel = np.abs(L1 - L0).max(1) / scale
    assert np.quantile(rel, 0.999) < 1e-5
    P0 = np.stack([np.bincount(key, weights=pre[:, d], minlength=nk) for d in range(3)], 1)
    P1 = np.stack([np.bincount(key, weights=post[:, d], minlength=nk) for d in range(3)], 1)
    assert (np.abs(P1 - P0).max(1) / scale).max() < 1e-5
    assert np.mean(np.abs(post - pre).max(1) > 1e-3) > 0.9


def test_at_plus_a_multi_step_call_equals_single_steps():
    cells, nbar = (16, 16, 8), 10
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar
    st = uniform_maxwell(box, n, 3)
    res = []
    for calls in ((5,), (1,) * 5, (2, 3)):
        g = MPC(box, cells, nbar, 17, n_max=n, collision=1, conserve_L=1, dt=0.02, brick=(16, 16, 8))
        gpu_set(g, st)
        for k in calls:
            g.step(k)
        res.append(gpu_get(g))
    for r in res[1:]:
        for a, b in zip(res[0], r):
            assert np.array_equal(a, b)
