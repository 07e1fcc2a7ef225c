"""GPU parity for the extensions beyond the pure fluid: explicit phantom particles in wall-cut cells (U22;
+a and MPC-AT at walls), embedded solutes with their own mass (U23), moving no-slip walls (U24). Lock-step against
the oracle from the same fp32 state; tolerances as everywhere else: keys / counts / order bit-exact, positions 1e-5 a,
velocities 2e-5 sqrt(kT/m) (+a: 1e-3 for particles of cells with cond(I_c) > 10^2, with the phantoms and
the masses entering I_c)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle.binding import Oracle  # noqa: E402
from paper_2406_15236_b200 import MPC  # noqa: E402
from paper_2406_15236_b200.inputs import uniform_maxwell  # noqa: E402
from test_parity_gpu import gpu_get, gpu_set  # noqa: E402


def cond_per_particle(o, so, key, step, kw, n_fluid_ids):
    """Condition number of every particle's cell inertia tensor (members = real particles with their masses + the
    oracle's phantoms of wall-cut cells); 1 where the cell has <= 2 members."""
    s = o.grid_shift(step).astype(np.float32)
    q = np.stack(so[0:3], 1) + s
    rho = (q - np.floor(q)).astype(np.float64)
    m = np.where(so[6] >= kw.get("solute_id0", 0), kw["solute_mass"], 1.0) if kw.get("solute_mass", 0) > 0 else np.ones(len(key))
    members = {}
    for i, k in enumerate(key):
        members.setdefault(int(k), []).append((m[i], rho[i]))
    cond_cell = {}
    wall = kw.get("phantoms", 0)
    w = [d for d in range(3) if kw.get("bc", (0, 0, 0))[d] == 1][0] if wall else 2
    nz = o.cells[w]
    lo, hi = ((1, nz + 1) if s[w] > 0 else (0, nz)) if wall else (-1, -1)
    for k, mem in members.items():
        if wall:
            ijk = np.zeros(3, np.int32)
            r0 = so[0][key == k][0], so[1][key == k][0], so[2][key == k][0]
            ijk, _cid, _key, _rho = o.cell_of(np.array(r0, np.float32), s)
            if ijk[w] in (lo, hi):
                prho, _pv = o.phantoms(ijk, s, step)
                mem = mem + [(1.0, p) for p in prho]
        if len(mem) <= 2:
            cond_cell[k] = 1.0
            continue
        wt = np.array([a for a, _ in mem])
        r = np.array([b for _, b in mem])
        rc = r - (wt[:, None] * r).sum(0) / wt.sum()
        I = sum(wi * ((x @ x) * np.eye(3) - np.outer(x, x)) for wi, x in zip(wt, rc))
        ev = np.linalg.eigvalsh(I)
        cond_cell[k] = ev[2] / max(ev[0], 1e-300)
    return np.array([cond_cell[int(k)] for k in key])


CASES = [
    ("SRD+a, walls, phantoms", dict(conserve_L=1, bc=(0, 0, 1), phantoms=1)),
    ("MPC-AT, walls, phantoms, gravity", dict(collision=1, bc=(0, 0, 1), phantoms=1, g=(0.02, 0, 0))),
    ("MPC-AT+a, walls, phantoms", dict(collision=1, conserve_L=1, bc=(0, 0, 1), phantoms=1)),
    ("SRD-a + thermostat, walls, phantoms", dict(thermostat=1, bc=(0, 0, 1), phantoms=1)),
    ("SRD+a, moving walls, phantoms", dict(conserve_L=1, bc=(0, 0, 1), phantoms=1, wall_velocity=0.4)),
    ("MPC-AT+a, walls on y, phantoms", dict(collision=1, conserve_L=1, bc=(0, 1, 0), phantoms=1)),
    ("SRD-a, solutes", dict(solute_mass=5.0)),
    ("SRD-a + thermostat, solutes", dict(thermostat=1, solute_mass=5.0)),
    ("SRD+a, solutes", dict(conserve_L=1, solute_mass=3.0)),
    ("MPC-AT, solutes", dict(collision=1, solute_mass=5.0)),
    ("MPC-AT+a, solutes, walls, phantoms", dict(collision=1, conserve_L=1, solute_mass=4.0, bc=(0, 0, 1), phantoms=1)),
]


@pytest.mark.parametrize("name,kw", CASES, ids=[c[0] for c in CASES])
def test_ext_lockstep_parity(name, kw):
    cells, nbar = (16, 8, 8), 8
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar + 7
    st = uniform_maxwell(box, n, 5)
    kw = dict(kw, dt=0.1, brick=4, rebin_every=1)
    if kw.get("solute_mass", 0) > 0:
        kw["solute_id0"] = n - n // 8
    o = Oracle(box, cells, nbar, 77, **kw)
    g = MPC(box, cells, nbar, 77, n_max=n, **kw)
    o.set_state(*st)
    plus_a = bool(kw.get("conserve_L"))
    for t in range(3):
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
        # per-cell momentum of the real particles, mass-weighted (U13: relative to the L1 scale of the summands)
        mw = np.where(so[6] >= kw["solute_id0"], kw["solute_mass"], 1.0) if kw.get("solute_mass", 0) > 0 else np.ones(n)
        for a, b in ((px, gx), (py, gy), (pz, gz)):
            scale = np.bincount(key_o, weights=mw * 1.0, minlength=o.nkeys) * 4.0 + 1e-30
            assert np.max(np.abs(a - b) / scale) <= 1e-5
        err = np.max(np.abs(np.stack(so[3:6]).astype(np.float64) - np.stack(sg[3:6])), axis=0)
        if plus_a:
            cond = cond_per_particle(o, so, key_o, t, kw, n)
            loose = cond > 1e2
            tol = np.where(loose, 1e-3, 2e-5)
            worst = int(np.argmax(err / tol))
            assert (err <= tol).all(), f"{name} t={t}: err {err[worst]:.3g} > tol {tol[worst]:.3g} at cond {cond[worst]:.3g}"
            print(f"{name} t={t}: max err strict {err[~loose].max(initial=0):.3g}, loose {err[loose].max(initial=0):.3g}, loose fraction {loose.mean():.4f}")
            assert loose.mean() < 0.05
            assert int(o.observables()["n_singular_cells"]) == int(g.observables()["n_singular_cells"])
        else:
            assert err.max() <= 2e-5, f"{name} t={t}: {err.max():.3g}"
        oo, og = o.observables(), g.observables()
        assert np.allclose(oo["P"], og["P"], atol=2e-3 * np.sqrt(n)) and og["E_kin"] == pytest.approx(oo["E_kin"], rel=1e-5)
        assert og["kT_est"] == pytest.approx(oo["kT_est"], rel=1e-5)


@pytest.mark.parametrize("kw", [dict(thermostat=1, bc=(0, 0, 1), wall_velocity=0.3, rebin_every=1),
                                dict(thermostat=1, bc=(0, 0, 1), wall_velocity=0.3, g=(0.01, 0, 0), rebin_every=3, brick=(16, 16, 8))])
def test_moving_walls_on_the_srd_hot_path_lockstep(kw):
    # U24 with the velocity-only virtual particles of U8: the fused SRD sweep's bounce-back and k_cell's virtual particles
    cells, nbar = (32, 16, 8), 10
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar - 5
    st = uniform_maxwell(box, n, 8)
    kw = dict(dict(brick=4), **kw)
    o = Oracle(box, cells, nbar, 31, **kw)
    g = MPC(box, cells, nbar, 31, n_max=n, **kw)
    o.set_state(*st)
    for t in range(4):
        gpu_set(g, o.get_state(), step=t)
        o.step(1)
        g.step(1)
        so, sg = o.get_state(), gpu_get(g)
        assert np.array_equal(so[6], sg[6])
        for d in range(3):
            assert np.array_equal(so[d], sg[d])
        for d in range(3, 6):
            assert np.max(np.abs(so[d] - sg[d])) <= 2e-5


def test_moving_walls_fused_path_directly_against_oracle():
    # the multi-step call (collision of step t-1 inside the sweep of step t, staged reorder) with moving walls: a twin
    # context advances k-1 steps in one call, the oracle takes its state and advances one step
    cells, nbar, k = (32, 16, 16), 10, 5
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar
    st = uniform_maxwell(box, n, 12)
    kw = dict(thermostat=1, bc=(0, 0, 1), wall_velocity=0.5, g=(0.01, 0, 0), rebin_every=3, brick=(16, 16, 8))
    a = MPC(box, cells, nbar, 3, n_max=n, **kw)
    b = MPC(box, cells, nbar, 3, n_max=n, **kw)
    gpu_set(a, st); gpu_set(b, st)
    a.step(k)
    b.step(k - 1)
    o = Oracle(box, cells, nbar, 3, **kw)
    sb = gpu_get(b)
    o.set_state(*sb[:6], id=sb[6], step=k - 1)
    o.step(1)
    so, sa = o.get_state(), gpu_get(a)
    io, ia = np.argsort(so[6]), np.argsort(sa[6])
    for d in range(3):
        assert np.array_equal(so[d][io], sa[d][ia])
    for d in range(3, 6):
        assert np.max(np.abs(so[d][io] - sa[d][ia])) <= 2e-5


def test_couette_flow_on_gpu():
    # steady plane Couette flow between walls moving with -+uw on the fused SRD path: linear profile, little slip
    cells, nbar, uw = (32, 32, 16), 10, 0.3
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar
    st = uniform_maxwell(box, n, 5)
    g = MPC(box, cells, nbar, 99, n_max=n, thermostat=1, bc=(0, 0, 1), wall_velocity=uw, rebin_every=10, brick=(16, 16, 8))
    gpu_set(g, st)
    g.step(1500)                                   # relaxation time L^2 / (pi^2 nu) = 30 = 300 steps
    prof, nav = np.zeros(16), 0
    for _ in range(100):
        g.step(5)
        prof += g.observables(profile=True)["profile"]
        nav += 1
    prof /= nav
    zc = np.arange(16) + 0.5
    A = np.stack([2 * zc / 16 - 1, np.ones(16)], 1)
    coef, *_ = np.linalg.lstsq(A, prof, rcond=None)
    assert coef[0] == pytest.approx(uw, rel=0.05) and abs(coef[1]) < 0.01
    assert np.abs(prof - A @ coef).max() < 0.012
    ob = g.observables()
    assert ob["kT_cell"] == pytest.approx(1.0, rel=0.02) and ob["n_range_overflows"] == 0


@pytest.mark.parametrize("kw", [dict(collision=1, conserve_L=1), dict(thermostat=1)])
def test_solutes_equilibrate_on_gpu(kw):
    cells, nbar, M = (16, 16, 16), 10, 5.0
    box = tuple(float(c) for c in cells)
    n = 16**3 * nbar
    nsol = 4096
    st = uniform_maxwell(box, n, 2)
    g = MPC(box, cells, nbar, 3, n_max=n, solute_id0=n - nsol, solute_mass=M, rebin_every=1, brick=4, **kw)
    gpu_set(g, st)
    p0 = g.observables()["P"]
    g.step(100)
    acc, k = 0.0, 0
    for _ in range(20):
        g.step(5)
        *_p, vx, vy, vz, ids = gpu_get(g)
        sel = ids >= n - nsol
        acc += (vx[sel].astype(np.float64) ** 2 + vy[sel].astype(np.float64) ** 2 + vz[sel].astype(np.float64) ** 2).mean() / 3
        k += 1
    assert acc / k == pytest.approx(1.0 / M, rel=0.03)
    ob = g.observables()
    assert ob["kT_est"] == pytest.approx(1.0, rel=0.02)
    assert np.allclose(ob["P"], p0, atol=0.05)      # mass-weighted momentum is conserved


def test_ext_parameter_validation():
    from paper_2406_15236_b200.binding import MPCError
    box, cells = (8.0, 8.0, 8.0), (8, 8, 8)
    bad = [(dict(conserve_L=1, bc=(0, 0, 1)), True),                          # +a at walls needs phantoms
           (dict(phantoms=1), True),                                           # phantoms need a wall
           (dict(phantoms=1, bc=(0, 0, 2)), True),                             # ... a no-slip one
           (dict(phantoms=1, bc=(0, 0, 1), rebin_every=2), False),             # the CUDA path needs the fresh order every step
           (dict(solute_mass=2.0, rebin_every=5), False),
           (dict(solute_mass=-1.0), True),
           (dict(wall_velocity=0.1), True),                                    # no wall
           (dict(wall_velocity=0.1, bc=(1, 0, 0)), True),                      # flow axis is x
           (dict(wall_velocity=0.1, bc=(0, 0, 2)), True)]
    for kw, oracle_too in bad:
        kw = dict(dict(rebin_every=1), **kw)
        with pytest.raises(MPCError):
            MPC(box, cells, 10, 1, n_max=100, **kw)
        if oracle_too:
            with pytest.raises(ValueError):
                Oracle(box, cells, 10, 1, **kw)
    MPC(box, cells, 10, 1, n_max=100, conserve_L=1, bc=(0, 0, 1), phantoms=1, rebin_every=1)
