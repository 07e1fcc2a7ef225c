"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.
Tolerances are BASELINE.json north_star's: keys / counts / sort order bit-exact, positions <= 1e-5 a,
velocities <= 2e-5 sqrt(kT/m) absolute, per-cell momentum sums <= 1e-5 relative (L1 scale, U13)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle.binding import Oracle  # noqa: E402
from paper_2406_15236_b200 import MPC  # noqa: E402
from paper_2406_15236_b200.inputs import uniform_maxwell  # noqa: E402

POS_TOL, VEL_TOL, MOM_TOL = 1e-5, 2e-5, 1e-5


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_set(g, st, step=0):
    x, y, z, vx, vy, vz, ids = st
    g.set_state(*[dev(a) for a in (x, y, z, vx, vy, vz)], id=dev(ids.view(np.int32)), step=step)


def gpu_get(g):
    out = g.get_state()
    torch.cuda.synchronize()
    arrs = [t.cpu().numpy() for t in out]
    arrs[6] = arrs[6].view(np.uint32)
    return arrs


def compare_step(o, g, kT=1.0, mass=1.0, a=1.0, check_order=True, vel_tol=VEL_TOL):
    """Compare the states and the last step's cell data of oracle `o` and GPU system `g`."""
    so, sg = o.get_state(), gpu_get(g)
    if check_order:
        assert np.array_equal(so[6], sg[6]), "particle order (ids) differs"
        oo = og = slice(None)
    else:
        oo, og = np.argsort(so[6]), np.argsort(sg[6])
        assert np.array_equal(so[6][oo], sg[6][og])
    for d in range(3):
        assert np.max(np.abs(so[d][oo].astype(np.float64) - sg[d][og]), initial=0) <= POS_TOL * a
    sc = np.sqrt(kT / mass)
    for d in range(3, 6):
        err = np.max(np.abs(so[d][oo].astype(np.float64) - sg[d][og]), initial=0)
        assert err <= vel_tol * sc, f"velocity component {d - 3}: {err}"
    cnt_o, px, py, pz, e2, key_o = o.get_cells()
    cnt_g, gx, gy, gz, ge, key_g = [t.cpu().numpy() for t in g.get_cells()]
    assert np.array_equal(key_o[oo], key_g.view(np.uint32)[og]), "cell keys differ"
    assert np.array_equal(cnt_o, cnt_g.view(np.uint32)), "cell counts differ"
    # U13: relative to the L1 scale of the summands, m * sum |v_i| ~ count * mean|v|; use e2-based bound
    l1 = mass * np.sqrt(np.maximum(e2, 1e-30) * np.maximum(cnt_o, 1))     # >= m * sum |v| / sqrt(3) by Cauchy-Schwarz
    for po, pg in ((px, gx), (py, gy), (pz, gz)):
        rel = np.abs(po - pg) / np.maximum(l1, 1e-30)
        assert np.max(rel[cnt_o > 0], initial=0) <= MOM_TOL
    return so, sg


def make_pair(box, cells, nbar, seed, n, **kw):
    o = Oracle(box, cells, nbar, seed, **kw)
    g = MPC(box, cells, nbar, seed, n_max=max(n, 1), **kw)
    return o, g


CASES = {
    # BASELINE.json config 1 shape: 16^3 cells, 10/cell, SRD, no thermostat
    "cfg1_srd": dict(cells=(16, 16, 16), nbar=10, kw=dict()),
    "srd_mbs_brick4": dict(cells=(16, 12, 8), nbar=10, kw=dict(thermostat=1, brick=4)),
    "srd_mbs_low_density": dict(cells=(12, 12, 12), nbar=3, kw=dict(thermostat=1)),
    # thermostat draw (U6) outside the table of (c, k) pairs the kernel reads for N_c < 64, and with a wall fill of 80
    "srd_mbs_high_density": dict(cells=(6, 6, 6), nbar=80, kw=dict(thermostat=1, brick=2)),
    "walls_high_density": dict(cells=(6, 6, 6), nbar=80, kw=dict(thermostat=1, bc=(0, 0, 1), g=(0.001, 0, 0))),
    "srd_a2": dict(cells=(8, 8, 8), nbar=10, kw=dict(thermostat=1), a=2.0),
    "at": dict(cells=(12, 12, 12), nbar=10, kw=dict(collision=1, dt=0.02)),
    "at_brick2": dict(cells=(10, 12, 6), nbar=5, kw=dict(collision=1, dt=0.02, brick=2)),
    "walls_gravity": dict(cells=(16, 8, 8), nbar=10, kw=dict(thermostat=1, bc=(0, 0, 1), g=(0.001, 0, 0))),
    "walls_x_brick4": dict(cells=(8, 8, 16), nbar=10, kw=dict(thermostat=1, bc=(1, 0, 0), g=(0, 0.01, 0), brick=4)),
    "noshift": dict(cells=(8, 8, 8), nbar=10, kw=dict(grid_shift=0)),
    "srd_mbs_brick16x16x8": dict(cells=(32, 16, 24), nbar=10, kw=dict(thermostat=1, brick=(16, 16, 8))),
    "srd_brick_4x2x1_ragged": dict(cells=(10, 7, 5), nbar=6, kw=dict(thermostat=1, brick=(4, 2, 1))),
    "walls_gravity_brick16x16x8": dict(cells=(16, 16, 16), nbar=10,
                                       kw=dict(thermostat=1, bc=(0, 0, 1), g=(0.001, 0, 0), brick=(16, 16, 8))),
    # slip walls (specular reflection, no virtual particles; U20)
    "slip_walls_gravity": dict(cells=(16, 8, 8), nbar=10, kw=dict(thermostat=1, bc=(0, 0, 2), g=(0.01, 0, 0))),
    "slip_walls_y_brick16x16x8": dict(cells=(16, 16, 16), nbar=10, kw=dict(bc=(0, 2, 0), dt=0.3, brick=(16, 16, 8))),
    # Lees-Edwards shear (U21): strong shear and a long step so that many particles cross the sheared face
    "shear": dict(cells=(12, 12, 12), nbar=10, kw=dict(thermostat=1, shear_rate=0.05, dt=0.3)),
    "shear_brick16x16x8": dict(cells=(32, 16, 16), nbar=10, kw=dict(shear_rate=0.11, brick=(16, 16, 8))),
    "shear_negative_brick4": dict(cells=(8, 12, 8), nbar=5, kw=dict(thermostat=1, shear_rate=-0.07, brick=4)),
}


@pytest.mark.parametrize("name", list(CASES))
def test_single_step_parity(name):
    c = CASES[name]
    a = c.get("a", 1.0)
    cells = c["cells"]
    box = tuple(float(n) * a for n in cells)
    n = int(np.prod(cells)) * c["nbar"] + 37                   # ragged tail: not a multiple of any block size
    st = uniform_maxwell(box, n, 100 + len(name))
    o, g = make_pair(box, cells, c["nbar"], 1234, n, **c["kw"])
    o.set_state(*st)
    gpu_set(g, st)
    o.step(1)
    g.step(1)
    compare_step(o, g, a=a)


@pytest.mark.parametrize("name", ["cfg1_srd", "srd_mbs_brick4", "at", "walls_gravity", "slip_walls_gravity", "shear",
                                  "shear_brick16x16x8"])
def test_lockstep_parity_many_steps(name):
    # U15: after every step the oracle state is copied to the GPU, then both advance one step
    c = CASES[name]
    cells = c["cells"]
    box = tuple(float(n) for n in cells)
    n = int(np.prod(cells)) * c["nbar"]
    st = uniform_maxwell(box, n, 7)
    o, g = make_pair(box, cells, c["nbar"], 99, n, **c["kw"])
    o.set_state(*st)
    for t in range(12):
        gpu_set(g, o.get_state(), step=t)
        o.step(1)
        g.step(1)
        compare_step(o, g)


@pytest.mark.parametrize("every", [3, 10])
def test_stale_order_parity(every):
    # reorder only every `every` steps: between reorders both keep the stale order (U3)
    cells, nbar = (12, 12, 12), 10
    box = tuple(float(n) for n in cells)
    n = int(np.prod(cells)) * nbar
    st = uniform_maxwell(box, n, 8)
    kw = dict(thermostat=1, rebin_every=every, brick=4)
    o, g = make_pair(box, cells, nbar, 5, n, **kw)
    o.set_state(*st)
    for t in range(every + 2):
        gpu_set(g, o.get_state(), step=t)
        o.step(1)
        g.step(1)
        compare_step(o, g)


def test_gpu_is_bit_reproducible_and_order_independent():
    # fixed-point cell sums: the trajectory does not depend on the memory order,
    # the reorder interval, the key layout, or the run
    cells, nbar = (16, 16, 16), 10
    box = (16.0, 16.0, 16.0)
    n = 16**3 * nbar
    st = uniform_maxwell(box, n, 3)
    res = []
    for kw in (dict(), dict(), dict(rebin_every=7), dict(brick=8), dict(brick=4, rebin_every=1000),
               dict(brick=(16, 16, 8), rebin_every=10), dict(brick=(4, 2, 1), rebin_every=3)):
        g = MPC(box, cells, nbar, 42, n_max=n, thermostat=1, **kw)
        gpu_set(g, st)
        g.step(25)
        s = gpu_get(g)
        order = np.argsort(s[6])
        res.append(np.stack([s[d][order] for d in range(6)]))
    for r in res[1:]:
        assert np.array_equal(r, res[0])


@pytest.mark.parametrize("kw", [dict(thermostat=1, brick=(16, 16, 8), rebin_every=4),
                                dict(thermostat=1, bc=(0, 0, 1), g=(0.01, 0, 0), brick=4, rebin_every=3),
                                dict(collision=1, dt=0.02)])
def test_one_call_of_k_steps_equals_k_calls(kw):
    # mpc_step(k) runs the fused sweep (collision of step t-1 inside the streaming pass of step t);
    # k calls of mpc_step(1) never do. Same arithmetic per particle -> bit-identical states. Together with
    # the lock-step parity tests (which use mpc_step(1)) this carries parity over to the fused path.
    cells, nbar = (32, 16, 16), 10
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar
    st = uniform_maxwell(box, n, 31)
    res = []
    for calls in ((9,), (1,) * 9, (4, 5), (2, 3, 4)):
        g = MPC(box, cells, nbar, 17, n_max=n, **kw)
        gpu_set(g, st)
        for k in calls:
            g.step(k)
        res.append(gpu_get(g) + [t.cpu().numpy() for t in g.get_cells()])
    for r in res[1:]:
        for a, b in zip(res[0], r):
            assert np.array_equal(a, b)


def test_free_running_conservation_cfg1():
    # BASELINE.json config 1: 100 steps, no thermostat: momentum and kinetic energy conserved
    cells, nbar = (16, 16, 16), 10
    box = (16.0, 16.0, 16.0)
    n = 16**3 * nbar
    st = uniform_maxwell(box, n, 1)
    g = MPC(box, cells, nbar, 1234, n_max=n)
    gpu_set(g, st)
    ob0 = g.observables()
    g.step(100)
    ob = g.observables()
    assert ob["step"] == 100 and ob["n"] == n
    assert abs(ob["E_kin"] - ob0["E_kin"]) / ob0["E_kin"] < 1e-5
    assert np.all(np.abs(ob["P"] - ob0["P"]) < 0.05)           # sum of 40960 fp32-rounded updates x 100 steps
    assert ob["kT_est"] == pytest.approx(1.0, rel=0.02)
    # same run on the oracle agrees statistically (free-running trajectories diverge, U15)
    o = Oracle(box, cells, nbar, 1234)
    o.set_state(*st)
    o.step(100)
    oo = o.observables()
    assert ob["E_kin"] == pytest.approx(oo["E_kin"], rel=1e-5)
    assert abs(ob["max_cell_count"] - oo["max_cell_count"]) <= 6


def test_observables_match_oracle():
    cells, nbar = (12, 8, 10), 10
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar
    st = uniform_maxwell(box, n, 12)
    kw = dict(thermostat=1, bc=(0, 0, 1), g=(0.01, 0, 0))
    o, g = make_pair(box, cells, nbar, 77, n, **kw)
    o.set_state(*st)
    gpu_set(g, st)
    o.step(1)
    g.step(1)
    a, b = o.observables(10), g.observables(profile=True)
    assert a["n"] == b["n"] and a["step"] == b["step"] and a["max_cell_count"] == b["max_cell_count"]
    assert np.allclose(a["P"], b["P"], atol=2e-2)
    assert b["E_kin"] == pytest.approx(a["E_kin"], rel=1e-6)
    assert b["kT_est"] == pytest.approx(a["kT_est"], rel=1e-6)
    assert b["kT_cell"] == pytest.approx(a["kT_cell"], rel=1e-5)
    assert np.allclose(a["profile"], b["profile"], atol=1e-5)


def test_edge_cases():
    box, cells = (4.0, 4.0, 4.0), (4, 4, 4)
    # empty system
    g = MPC(box, cells, 10, 1, n_max=16)
    e = torch.empty(0, dtype=torch.float32, device="cuda")
    g.set_state(e, e, e, e, e, e)
    g.step(3)
    ob = g.observables()
    assert ob["n"] == 0 and ob["step"] == 3
    # one particle: collision with itself leaves it unchanged; streaming wraps
    o, g = make_pair(box, cells, 10, 1, 1)
    st = [np.array([v], np.float32) for v in (3.95, 0.0, 2.0, 1.0, -1.0, 0.5)] + [np.array([0], np.uint32)]
    o.set_state(*st)
    gpu_set(g, st)
    o.step(2)
    g.step(2)
    so, sg = compare_step(o, g)
    assert sg[3][0] == np.float32(1.0) and sg[4][0] == np.float32(-1.0)
    # particles exactly on cell faces and box faces, zero velocity, no shift: keys are floor(r)
    o, g = make_pair(box, cells, 10, 1, 64, grid_shift=0)
    gx, gy, gz = np.meshgrid(np.arange(4.0), np.arange(4.0), np.arange(4.0), indexing="ij")
    z = np.zeros(64, np.float32)
    st = [gx.ravel().astype(np.float32), gy.ravel().astype(np.float32), gz.ravel().astype(np.float32), z, z, z,
          np.arange(64, dtype=np.uint32)]
    o.set_state(*st)
    gpu_set(g, st)
    o.step(1)
    g.step(1)
    compare_step(o, g)
    cnt = g.get_cells()[0].cpu().numpy()
    assert np.all(cnt == 1)
    # all particles in one cell (maximum occupancy, heavy atomic contention)
    n = 1500
    o, g = make_pair(box, cells, 10, 1, n, thermostat=1, dt=0.01)
    rng = np.random.default_rng(0)
    st = [np.full(n, 1.5, np.float32) + rng.uniform(-0.2, 0.2, n).astype(np.float32) for _ in range(3)]
    st += [rng.normal(0, 1, n).astype(np.float32) for _ in range(3)] + [np.arange(n, dtype=np.uint32)]
    o.set_state(*st)
    gpu_set(g, st)
    o.step(1)
    g.step(1)
    compare_step(o, g)
    assert g.observables()["max_cell_count"] >= n // 8


def test_precision_is_relative_to_thermal_velocity():
    # same system in units where kT = 1e-4 (velocities 100x smaller): tolerance scales with sqrt(kT/m)
    cells, nbar, kT = (10, 10, 10), 10, 1e-4
    box = (10.0, 10.0, 10.0)
    n = 10**3 * nbar
    st = uniform_maxwell(box, n, 5, kT=kT)
    o, g = make_pair(box, cells, nbar, 3, n, thermostat=1, kT=kT, dt=10.0)
    o.set_state(*st)
    gpu_set(g, st)
    o.step(1)
    g.step(1)
    compare_step(o, g, kT=kT)


def test_host_api_roundtrip_and_errors():
    box, cells = (8.0, 8.0, 8.0), (8, 8, 8)
    n = 5120
    st = uniform_maxwell(box, n, 2)
    g = MPC(box, cells, 10, 9, n_max=n, thermostat=1)
    g.set_state_host(*st[:6], id=st[6].view(np.int32), step=5)
    back = g.get_state_host()
    for a, b in zip(st, back):
        assert np.array_equal(a, b)
    g.step(2)
    g2 = MPC(box, cells, 10, 9, n_max=n, thermostat=1)
    gpu_set(g2, st, step=5)
    g2.step(2)
    for a, b in zip(g.get_state_host(), gpu_get(g2)):
        assert np.array_equal(a, b)
    # errors
    from paper_2406_15236_b200 import MPCError
    with pytest.raises(MPCError):
        big = uniform_maxwell(box, n + 1, 2)
        g.set_state_host(*big[:6])
    g3 = MPC(box, cells, 10, 9, n_max=n)
    with pytest.raises(MPCError):
        g3.step(1)                     # no state yet
    with pytest.raises(MPCError):
        g3.get_cells()


def test_compact_workspace_gives_identical_results():
    cells, nbar = (12, 12, 12), 10
    box = (12.0, 12.0, 12.0)
    n = 12**3 * nbar
    st = uniform_maxwell(box, n, 4)
    res = []
    for compact in (False, True):
        g = MPC(box, cells, nbar, 6, n_max=n, compact=compact, thermostat=1, rebin_every=2, brick=4)
        gpu_set(g, st)
        g.step(5)
        res.append(gpu_get(g))
    for a, b in zip(*res):
        assert np.array_equal(a, b)


@pytest.mark.gpu
@pytest.mark.parametrize("kw", [dict(thermostat=1, brick=(16, 16, 8), rebin_every=2),
                                dict(thermostat=1, bc=(0, 0, 1), g=(0.01, 0, 0), brick=4, rebin_every=3),
                                dict(brick=(4, 2, 1), rebin_every=5),
                                dict(thermostat=1, shear_rate=0.05, brick=(16, 16, 8), rebin_every=3)])
def test_reorder_code_paths_agree(kw):
    # Ways to apply a reorder inside a multi-step call (rebin_every >= 3 and two further steps in the call, else the unfolded
    # reorder runs in every variant): (a) default: folded into three sweeps: arrival ranks from the sweep of the reorder step,
    # 32-byte records written at their slots of the new order by the next sweep (no atomics), read back by the one after;
    # particles grouped by key only, canonical (key, id) order restored when the state is read; (b) separate gather kernel; (c) eager canonical order
    # (scatter + rank by id + gather), the path the lock-step parity tests exercise with mpc_step(1); (d) cursor
    # atomics in the scatter; (e) the last collision of a call applied at once instead of staying pending; (f) plain cell
    # order in memory between reads instead of the lane-spread order of every group of 32 cells.
    # State AND memory order must be identical.
    from paper_2406_15236_b200 import binding as B
    cells, nbar = (32, 16, 16), 10
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar - 13          # ragged tail: not a multiple of 32
    st = uniform_maxwell(box, n, 77)
    res = []
    for flags in (0, B.DEBUG_NO_FUSE_GATHER, B.DEBUG_EAGER_CANONICAL, B.DEBUG_ATOMIC_SCATTER, B.DEBUG_EAGER_COLLIDE, B.DEBUG_NO_LANE_SPREAD,
                  B.DEBUG_NO_LANE_SPREAD | B.DEBUG_ATOMIC_SCATTER, B.DEBUG_NO_FUSE_GATHER | B.DEBUG_ATOMIC_SCATTER):
        g = MPC(box, cells, nbar, 23, n_max=n, **kw)
        g.set_debug(flags)
        gpu_set(g, st)
        g.step(7)
        a = gpu_get(g)
        b = gpu_get(g)                             # reading twice does not change anything
        for x, y in zip(a, b):
            assert np.array_equal(x, y)
        g.step(4)
        res.append(gpu_get(g) + [t.cpu().numpy() for t in g.get_cells()])
    for r in res[1:]:
        for x, y in zip(res[0], r):
            assert np.array_equal(x, y)


@pytest.mark.parametrize("kw,nbar", [(dict(thermostat=1, brick=(16, 16, 8), rebin_every=3), 10),
                                     (dict(thermostat=1, brick=(16, 16, 8), rebin_every=2), 20),      # window = half a brick
                                     (dict(thermostat=1, bc=(0, 0, 1), g=(0.01, 0, 0), brick=4, rebin_every=3), 10),
                                     (dict(brick=(4, 2, 1), rebin_every=2), 10)])                     # bricks below 32 cells: no windows
def test_compact_workspace_gathers_agree(kw, nbar):
    # compact workspace (property-wise reorder through one spare array): from the second reorder on the
    # gather goes through shared-memory windows over the previous order's ranges (k_gather_win); with
    # MPC_DEBUG_NO_FUSE_GATHER it is the plain element-wise gather; and the workspace with the second particle copy moves
    # records instead. State AND memory order must be identical in all three, after several reorders and a long step that
    # carries a good part of the particles out of their window.
    from paper_2406_15236_b200 import binding as B
    cells = (32, 16, 16)
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar - 13
    st = uniform_maxwell(box, n, 78)
    res = []
    for compact, flags in ((True, 0), (True, B.DEBUG_NO_FUSE_GATHER), (False, 0)):
        g = MPC(box, cells, nbar, 24, n_max=n, compact=compact, dt=0.5, **kw)
        g.set_debug(flags)
        gpu_set(g, st)
        g.profile_enable()
        g.step(7)
        fam = g.profile_read()
        g.step(4)
        res.append(gpu_get(g) + [t.cpu().numpy() for t in g.get_cells()])
        if compact:
            assert fam["gather"][1] >= 2 and fam["sweep_gather"][1] == 0, fam    # property-wise reorders, nothing folded
    for r in res[1:]:
        for x, y in zip(res[0], r):
            assert np.array_equal(x, y)


_FOLD = dict(thermostat=1, brick=(16, 16, 8), rebin_every=4)
_FOLD_WALL = dict(thermostat=1, bc=(0, 0, 1), g=(0.01, 0, 0), brick=4, rebin_every=4)
_FOLD_LE = dict(thermostat=1, shear_rate=0.08, brick=(16, 16, 8), rebin_every=4)


@pytest.mark.parametrize("name,kw,t0,k,folded", [
    ("plain fused step", dict(thermostat=1, brick=(16, 16, 8), rebin_every=10), 1, 3, False),
    ("step after an unfolded reorder", dict(thermostat=1, brick=(16, 16, 8), rebin_every=4), 2, 4, False),
    ("second step after an unfolded reorder", dict(thermostat=1, brick=(16, 16, 8), rebin_every=4), 2, 5, False),
    ("walls + gravity, unfolded reorder", dict(thermostat=1, bc=(0, 0, 1), g=(0.01, 0, 0), brick=4, rebin_every=3), 1, 4, False),
    ("no thermostat, small bricks", dict(brick=(4, 2, 1), rebin_every=5), 3, 4, False),
    ("Lees-Edwards shear, unfolded reorder", dict(thermostat=1, shear_rate=0.08, brick=(16, 16, 8), rebin_every=3), 1, 4, False),
    ("Lees-Edwards shear, plain fused step", dict(shear_rate=0.08, dt=0.3, brick=4, rebin_every=10), 5, 3, False),
    # the reorder folded into three sweeps (the path bench.py times): from t = 0 the reorder at t = 0 is unfolded (no order
    # yet), the one at t = 4 is folded when two more steps follow in the call: rank pass at t = 4, scatter pass at t = 5,
    # read-back pass at t = 6 (the last step for k = 7), first plain sweep on the new lane-spread order at t = 7 (k = 8)
    ("folded reorder: read-back pass", _FOLD, 0, 7, True),
    ("folded reorder: first plain sweep on the new order", _FOLD, 0, 8, True),
    ("folded reorder, walls + gravity: read-back pass", _FOLD_WALL, 0, 7, True),
    ("folded reorder, walls + gravity: first plain sweep on the new order", _FOLD_WALL, 0, 8, True),
    ("folded reorder, Lees-Edwards shear: read-back pass", _FOLD_LE, 0, 7, True),
    ("folded reorder, Lees-Edwards shear: first plain sweep on the new order", _FOLD_LE, 0, 8, True),
])
def test_fused_path_directly_against_oracle(name, kw, t0, k, folded):
    # The multi-step call runs code no single-step call runs: the collision of step t-1 inside the sweep of step t, and
    # the reorder folded into three consecutive sweeps (arrival ranks written by the sweep of the reorder step, 32-byte
    # records written at their slots of the new order by the next sweep, read back by the one after). Direct check
    # with no single-step call in the chain: a twin context advances k-1 steps in ONE call, the oracle takes the
    # twin's state and advances ONE step; the first context advances k steps in ONE call. Element-by-element parity
    # of the k-th step, which ran entirely inside the fused path. (The twin's shorter call cannot fold the reorder at
    # t = 4 - too few steps left - so the state the oracle starts from has come through the unfolded reorder.)
    # The kernel-family counters say which path the first context took: the test fails if the folded reorder did not run
    # where the case says it does.
    cells, nbar = (32, 16, 16), 10
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar - 5
    st = uniform_maxwell(box, n, 101)             # thermal start: the fixed-point sums are sized for thermal velocities (U19)
    g, twin = MPC(box, cells, nbar, 29, n_max=n, **kw), MPC(box, cells, nbar, 29, n_max=n, **kw)
    gpu_set(g, st, step=t0)
    gpu_set(twin, st, step=t0)
    twin.step(k - 1)
    g.profile_enable()
    g.step(k)
    fam = g.profile_read()
    g.profile_enable(False)
    assert fam["sweep_gather"][1] == (3 if folded else 0), fam    # rank, scatter and read-back passes of ONE folded reorder
    assert fam["sweep"][1] + fam["sweep_gather"][1] == k
    o = Oracle(box, cells, nbar, 29, **kw)
    o.set_state(*gpu_get(twin), step=t0 + k - 1)
    o.step(1)
    # the oracle reorders by (key, id) only on reorder steps, like the library: same memory order unless the last
    # step reordered (then both are in the fresh canonical order)
    compare_step(o, g)
    assert g.observables()["n_range_overflows"] == 0


def test_range_overflow_is_reported():
    # fixed-point sums have a finite range ("overflows may occur ... invalidating the results"): the
    # library must say so. Velocities of 10^3 thermal velocities are far outside it; ordinary runs report 0.
    from paper_2406_15236_b200 import binding as B
    cells, nbar = (8, 8, 8), 10
    box = (8.0, 8.0, 8.0)
    n = 8**3 * nbar
    st = list(uniform_maxwell(box, n, 4))
    for kw in (dict(thermostat=1, dt=1e-4), dict(collision=1, dt=1e-4)):
        g = MPC(box, cells, nbar, 5, n_max=n, **kw)
        gpu_set(g, st)
        g.step(3)
        assert g.observables()["n_range_overflows"] == 0
        hot = [a.copy() for a in st]
        hot[3][:7] *= 1e3
        gpu_set(g, hot)
        assert g.observables()["n_range_overflows"] == 0            # nothing summed yet
        g.step(1)
        ob = g.observables()
        assert ob["n_range_overflows"] >= 7
        o = B.mpc_obs()
        assert g.lib.mpc_observables(g._h, B.C.byref(o), None, 0) == B.MPC_ERANGE
        gpu_set(g, st)                                              # a new state resets the counter
        g.step(1)
        assert g.observables()["n_range_overflows"] == 0


def test_crowded_cell_two_steps_with_reorder():
    # 450 thermal particles in ONE cell, handled by one CTA once the order is known (step 0 reorders): the 32-bit
    # energy word of the shared-memory tile wraps (450 * 3 u^2 * 2^22 > 2^32); the carry must reach the 48-bit
    # global field. Two lock-steps, the second on the fresh order.
    box, cells = (4.0, 4.0, 4.0), (4, 4, 4)
    n = 450
    rng = np.random.default_rng(1)
    st = [np.full(n, 1.5, np.float32) + rng.uniform(-0.3, 0.3, n).astype(np.float32) for _ in range(3)]
    st += [(1.3 * rng.normal(0, 1, n)).astype(np.float32) for _ in range(3)] + [np.arange(n, dtype=np.uint32)]
    o, g = make_pair(box, cells, 10, 1, n, thermostat=1, dt=0.01, rebin_every=1, brick=4, grid_shift=0)
    o.set_state(*st)
    gpu_set(g, st)
    o.step(1)
    g.step(1)
    compare_step(o, g)
    g2 = MPC(box, cells, 10, 1, n_max=n, thermostat=1, dt=0.01, rebin_every=10, brick=4, grid_shift=0)
    gpu_set(g2, st)
    g2.step(2)                                   # step 1 runs on the order of step 0: all 450 in one tile cell
    o.step(1)
    so, sg = o.get_state(), gpu_get(g2)
    oo, og = np.argsort(so[6]), np.argsort(sg[6])
    for d in range(3, 6):
        # the two runs are free-running for two steps: velocities differ by accumulated rounding only
        assert np.max(np.abs(so[d][oo].astype(np.float64) - sg[d][og])) <= 1e-4
    ob = g2.observables()
    assert ob["max_cell_count"] >= 440 and ob["n_range_overflows"] == 0
    assert ob["kT_cell"] == pytest.approx(o.observables()["kT_cell"], rel=1e-5)


def test_slip_walls_plug_flow_on_gpu():
    # frictionless walls: under a body force the fluid accelerates as one, P_x(t) = N m g t to rounding, in a
    # multi-step call (fused sweep, staged reorder) as well; the same law pins the oracle (test_oracle_walls.py)
    cells, nbar = (32, 16, 16), 10
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar
    gx, h, steps = 0.01, 0.1, 200
    st = uniform_maxwell(box, n, 12)
    g = MPC(box, cells, nbar, 9, n_max=n, thermostat=1, bc=(0, 0, 2), g=(gx, 0, 0), rebin_every=10, brick=(16, 16, 8))
    gpu_set(g, st)
    p0 = g.observables()["P"][0]
    g.step(steps)
    ob = g.observables(profile=True)
    assert ob["P"][0] - p0 == pytest.approx(n * gx * steps * h, rel=2e-5)
    assert np.abs(ob["profile"] - gx * steps * h).max() < 0.06          # flat profile (5,120 particles per layer: 4 sigma)
    assert ob["kT_cell"] == pytest.approx(1.0, rel=1e-2)


def test_shear_flow_on_gpu_keeps_the_linear_profile():
    # Lees-Edwards shear (U21) in one fused multi-step call on the GPU: started on the steady profile
    # v_x = gamma (z - L_z/2), the fluid must stay on it (a wrong image displacement or velocity jump at the sheared
    # face shows up as a kink or a drift within a few hundred steps), and the thermostat must hold k_BT.
    cells, nbar, gam = (32, 16, 16), 10, 0.02
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar
    st = list(uniform_maxwell(box, n, 5))
    st[3] = (st[3] + gam * (st[2] - box[2] / 2)).astype(np.float32)
    g = MPC(box, cells, nbar, 3, n_max=n, thermostat=1, shear_rate=gam, rebin_every=10, brick=(16, 16, 8))
    gpu_set(g, st)
    prof = np.zeros(16)
    for _ in range(10):
        g.step(60)
        ob = g.observables(profile=True)
        prof += ob["profile"] / 10
    zmid = np.arange(16) + 0.5
    assert np.polyfit(zmid, prof, 1)[0] == pytest.approx(gam, rel=0.04)
    assert np.abs(prof - gam * (zmid - 8.0)).max() < 0.02              # 5,120 particles per layer, 10 samples
    assert ob["kT_cell"] == pytest.approx(1.0, rel=1e-2) and ob["n_range_overflows"] == 0
