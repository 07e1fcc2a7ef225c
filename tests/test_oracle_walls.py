"""Pins for the oracle's wall / gravity path: bounce-back (reading U7), virtual wall
particles (reading U8), Poiseuille flow against the analytic SRD viscosity
(closed forms of refs [31],[32] checked against the paper's printed eta = 111.3)."""
import numpy as np
import pytest

from oracle.binding import Oracle
from paper_2406_15236_b200.inputs import uniform_maxwell
from util import srd_viscosity


def test_viscosity_closed_form_reproduces_printed_value(golden):
    (row,) = golden("viscosity.txt")
    assert row[0] == "srd+a"
    nbar, h, alpha, eta = (float(t) for t in row[1:])
    k, c = srd_viscosity(nbar, h, alpha, conserve_L=True)
    assert nbar * (k + c) == pytest.approx(eta, abs=0.05)       # 111.29 vs printed 111.3
    k, c = srd_viscosity(10, 0.1, 130)
    assert k + c == pytest.approx(0.870025, abs=1e-5)


def test_bounce_back_hand_cases():
    o = Oracle((8, 8, 8), (8, 8, 8), 10, 1, bc=(0, 0, 1), dt=0.1, thermostat=1)
    # hits z = 0 after half the step, comes back along the same line with reversed velocity
    r, v = o.stream_one([3.0, 4.0, 0.05], [0.5, -0.25, -1.0])
    assert np.allclose(r, [3.0, 4.0, 0.05], atol=2e-7)
    assert np.array_equal(v, np.array([-0.5, 0.25, 1.0], np.float32))
    # upper wall
    r, v = o.stream_one([3.0, 4.0, 7.98], [0.0, 0.0, 1.0])
    assert r[2] == pytest.approx(7.92, abs=1e-6) and v[2] == -1.0    # wall at t=0.02, 0.08 back
    # no crossing: plain streaming; a particle sitting on the wall moving inwards is not bounced
    r, v = o.stream_one([3.0, 4.0, 0.0], [0.0, 0.0, 1.0])
    assert r[2] == pytest.approx(0.1, abs=1e-7) and v[2] == 1.0
    r, v = o.stream_one([3.0, 4.0, 8.0], [0.0, 0.0, -1.0])
    assert r[2] == pytest.approx(7.9, abs=1e-6) and v[2] == -1.0
    # x stays periodic
    r, v = o.stream_one([7.99, 4.0, 4.0], [1.0, 0.0, 0.0])
    assert 0.0 <= r[0] < 0.1


def test_bounce_back_with_gravity_keeps_particles_inside():
    box = (8.0, 8.0, 8.0)
    st = uniform_maxwell(box, 4000, 7)
    o = Oracle(box, (8, 8, 8), 8, 3, bc=(0, 0, 1), g=(0.01, 0, 0), thermostat=1)
    o.set_state(*st)
    o.step(20)
    x, y, z, *_ = o.get_state()
    assert z.min() >= 0.0 and z.max() <= 8.0
    assert x.min() >= 0.0 and x.max() < 8.0
    cnt = o.get_cells()[0]
    assert cnt.sum() == 4000


def test_wall_layers_and_cut_cells():
    # wall axis has n+2 layers; which layers hold particles depends on the sign of the shift (U8)
    box = (4.0, 4.0, 4.0)
    st = uniform_maxwell(box, 4**3 * 10, 7)
    o = Oracle(box, (4, 4, 4), 10, 3, bc=(0, 0, 1), thermostat=1, dt=1e-30)
    assert o.nkeys == 4 * 4 * 6
    seen = set()
    for t in range(12):
        o.set_state(*st, step=t)
        o.step(1)
        cnt = o.get_cells()[0].reshape(6, 4, 4).sum(axis=(1, 2))
        sz = o.grid_shift(t)[2]
        seen.add(sz > 0)
        if sz > 0:
            assert cnt[0] == 0 and cnt[1] > 0 and cnt[5] > 0
            assert cnt[1] < cnt[2] and cnt[5] < cnt[4]       # cut layers are partially filled
        else:
            assert cnt[5] == 0 and cnt[0] > 0 and cnt[4] > 0
    assert seen == {True, False}


def test_virtual_wall_particles_recomputed_by_hand():
    # one real particle in a wall-cut cell: the collision partner is nbar-1 virtual particles whose
    # velocities come from the (cell, k, t, TAG_WALL) stream. Recompute Eq. (2) in numpy.
    nbar = 5
    o = Oracle((2.0, 2.0, 2.0), (2, 2, 2), nbar, 11, bc=(0, 0, 1), dt=1e-30, kT=1.0)
    t = 0
    while o.grid_shift(t)[2] <= 0:
        t += 1
    s = o.grid_shift(t)
    r = np.array([0.7, 1.2, 0.05], np.float32)
    v = np.array([0.3, -0.4, 0.5], np.float32)
    ijk, cid, key, _ = o.cell_of(r, s)
    assert ijk[2] == 1                                        # cut layer at the lower wall for s_z > 0
    o.set_state([r[0]], [r[1]], [r[2]], [v[0]], [v[1]], [v[2]], step=t)
    o.step(1)
    *_p, vx, vy, vz, _ = o.get_state()
    virt = np.array([o.normals(cid, k, t, 4)[:3] for k in range(nbar - 1)])
    vcm = (v.astype(np.float64) + virt.sum(0)) / nbar
    ax = o.srd_axis(cid, t)
    w = v - vcm
    a = np.deg2rad(np.float32(130.0)).astype(np.float32).astype(np.float64)
    wr = w * np.cos(a) + np.cross(ax, w) * np.sin(a) + ax * (ax @ w) * (1 - np.cos(a))
    assert np.allclose([vx[0], vy[0], vz[0]], vcm + wr, atol=3e-7)
    # an interior cell gets no virtual particles: a lone particle keeps its velocity
    o.set_state([0.7], [1.2], [1.0], [0.3], [-0.4], [0.5], step=t)
    o.step(1)
    *_p, vx, vy, vz, _ = o.get_state()
    assert (vx[0], vy[0], vz[0]) == (np.float32(0.3), np.float32(-0.4), np.float32(0.5))


def test_kappa_in_a_wall_cut_cell_counts_virtual_particles():
    # PAPER.md:54-68 (Eqs. 5-7 + "Boundary conditions"), reading U8: in a wall-cut cell the thermostat sees the
    # virtual particles too: v_cm, sum |v - v_cm|^2 and f = 3(N_c - 1) are taken over real + virtual particles
    # (N_c = nbar). One real particle + nbar-1 virtual ones, thermostat ON; everything recomputed in numpy from
    # the RNG hooks. Dropping the virtual terms from W2, or using the real count in f, fails this.
    nbar, kT = 6, 0.7
    o = Oracle((2.0, 2.0, 2.0), (2, 2, 2), nbar, 19, bc=(0, 0, 1), dt=1e-30, kT=kT, thermostat=1)
    t = 0
    while o.grid_shift(t)[2] <= 0:
        t += 1
    s = o.grid_shift(t)
    r = np.array([1.3, 0.4, 0.07], np.float32)
    v = np.array([-0.6, 0.2, 0.9], np.float32)
    ijk, cid, _key, _ = o.cell_of(r, s)
    assert ijk[2] == 1
    o.set_state([r[0]], [r[1]], [r[2]], [v[0]], [v[1]], [v[2]], step=t)
    o.step(1)
    *_p, vx, vy, vz, _ = o.get_state()
    sig = np.sqrt(kT)
    virt = sig * np.array([o.normals(cid, k, t, 4)[:3] for k in range(nbar - 1)])
    allv = np.vstack([v.astype(np.float64), virt])
    vcm = allv.mean(0)
    W2 = ((allv - vcm) ** 2).sum()                             # real + virtual
    Ek = kT * o.mbs_energy(cid, t, nbar)                       # Gamma(3(nbar-1)/2) draw for N_c = nbar
    kappa = np.sqrt(2.0 * Ek / W2)                             # Eq. (6), m = 1
    ax = o.srd_axis(cid, t)
    w = v - vcm
    a = np.deg2rad(np.float32(130.0)).astype(np.float32).astype(np.float64)
    wr = w * np.cos(a) + np.cross(ax, w) * np.sin(a) + ax * (ax @ w) * (1 - np.cos(a))
    want = vcm + kappa * wr
    assert np.allclose([vx[0], vy[0], vz[0]], want, atol=3e-7)
    # the two plausible misreadings give measurably different answers for this case
    W2_real = ((v - vcm) ** 2).sum()
    assert abs(np.sqrt(2.0 * Ek / W2_real) - kappa) > 1e-2
    assert abs(o.mbs_energy(cid, t, 1 + 1) - o.mbs_energy(cid, t, nbar)) > 1e-2


@pytest.mark.parametrize("bc", [1, 2])
def test_wall_hit_with_gravity_closed_form(bc):
    # PAPER.md:68 (bounce-back / specular reflection) with PAPER.md:70 (constant acceleration), readings U7/U20:
    # the particle flies ballistically under g for t_c, is reflected AT the wall, and flies for h - t_c.
    # x0 = 3, v = (0.5, -0.25, -1), z0 = 0.03 -> t_c = 0.03 of h = 0.1; g = 2 along x.
    g, h = 2.0, 0.1
    o = Oracle((8, 8, 8), (8, 8, 8), 10, 1, bc=(0, 0, bc), dt=h, g=(g, 0, 0), thermostat=1)
    r0 = np.array([3.0, 4.0, 0.03])
    v0 = np.array([0.5, -0.25, -1.0])
    r, v = o.stream_one(r0, v0)
    tc, tr = 0.03, 0.07
    x1 = r0[0] + v0[0] * tc + 0.5 * g * tc * tc
    vx1 = v0[0] + g * tc
    y1 = r0[1] + v0[1] * tc
    if bc == 1:      # bounce-back: every component reverses at the wall
        want_r = [x1 - vx1 * tr + 0.5 * g * tr * tr, y1 - v0[1] * tr, 1.0 * tr]
        want_v = [-vx1 + g * tr, -v0[1], 1.0]
    else:            # specular: only the normal component reverses; the tangential flight is the free one
        want_r = [r0[0] + v0[0] * h + 0.5 * g * h * h, r0[1] + v0[1] * h, 1.0 * tr]
        want_v = [v0[0] + g * h, v0[1], 1.0]
    assert np.allclose(r, want_r, atol=1e-6)
    assert np.allclose(v, want_v, atol=1e-6)
    # and without a wall hit: plain ballistic flight with the half-step velocity
    r, v = o.stream_one([3.0, 4.0, 4.0], v0)
    assert np.allclose(r, [3.0 + 0.5 * h + 0.5 * g * h * h, 4.0 - 0.25 * h, 4.0 - h], atol=1e-6)
    assert np.allclose(v, [0.5 + g * h, -0.25, -1.0], atol=1e-6)


@pytest.mark.slow
def test_poiseuille_profile_matches_analytic_viscosity():
    # gravity + two walls -> parabola; nu = 0.870 for <N_c>=10, h=0.1, alpha=130 deg.
    # Thin box (L_z = 16, relaxation time L_z^2/(pi^2 nu) = 30 = 300 steps).
    box, cells = (16.0, 8.0, 16.0), (16, 8, 16)
    st = uniform_maxwell(box, 16 * 8 * 16 * 10, 5)
    g = 0.005
    zc = np.arange(16) + 0.5
    A = np.stack([zc * (16 - zc), np.ones(16)], 1)

    def steady_flow(fill):
        # fill = the number the virtual wall particles top a wall-cut cell up to (U8): 10 = <N_c>, the method; 1 = a cell
        # that holds a particle at all gets none, i.e. bounce-back walls WITHOUT virtual particles, the comparison case
        o = Oracle(box, cells, fill, 321, thermostat=1, g=(g, 0, 0), bc=(0, 0, 1))
        o.set_state(*st)
        o.step(1200)
        prof = np.zeros(16)
        nav = 0
        for _ in range(440):
            o.step(5)
            prof += o.observables(16)["profile"]
            nav += 1
        prof /= nav
        coef, *_ = np.linalg.lstsq(A, prof, rcond=None)
        return o, prof, g / (2 * coef[0]), coef[1]

    o, prof, nu_fit, slip = steady_flow(10)
    nu = sum(srd_viscosity(10, 0.1, 130))
    assert nu_fit == pytest.approx(nu, rel=0.06)
    # the virtual wall particles "reduce boundary slip"; they do not remove it, and the paper gives no number.
    # The pin is therefore the statement itself: the fitted velocity at the wall (the intercept of the parabola) against
    # the same flow without virtual particles. Measured over two seeds: 4-7 % of v_max with them (standard error of one
    # fitted intercept ~1.5 % of v_max; a slip length of about a quarter of a cell), 21 % without. A fill that did
    # nothing, or a wrong sign or scale of the virtual momentum, lands at or beyond the second number.
    _, prof_bare, _, slip_bare = steady_flow(1)
    assert slip_bare > 0.15 * prof_bare.max()                  # without virtual particles the fluid slips markedly
    assert abs(slip) / prof.max() < 0.5 * slip_bare / prof_bare.max()
    assert abs(slip) < 0.10 * prof.max()                       # (loose absolute bound, three standard errors above the measured value)
    assert abs(prof - prof[::-1]).max() < 0.02                 # symmetric
    ob = o.observables()
    assert ob["kT_cell"] == pytest.approx(1.0, rel=0.03)        # thermostat holds k_BT under forcing


# ---- slip walls: specular reflection, no virtual wall particles (reading U20) ----------

def test_specular_reflection_hand_cases():
    o = Oracle((8, 8, 8), (8, 8, 8), 10, 1, bc=(0, 0, 2), dt=0.1, thermostat=1)
    # hits z = 0 after half the step: only the normal component is reversed, the tangential motion goes on
    r, v = o.stream_one([3.0, 4.0, 0.05], [0.5, -0.25, -1.0])
    assert np.allclose(r, [3.05, 3.975, 0.05], atol=3e-7)
    assert np.array_equal(v, np.array([0.5, -0.25, 1.0], np.float32))
    # upper wall: wall at t = 0.02, 0.08 back
    r, v = o.stream_one([3.0, 4.0, 7.98], [1.0, 0.0, 1.0])
    assert r[2] == pytest.approx(7.92, abs=1e-6) and v[2] == -1.0 and v[0] == 1.0
    assert r[0] == pytest.approx(3.1, abs=1e-6)
    # no crossing: plain streaming
    r, v = o.stream_one([3.0, 4.0, 4.0], [0.0, 0.0, 1.0])
    assert r[2] == pytest.approx(4.1, abs=1e-6) and v[2] == 1.0


def test_slip_walls_are_frictionless():
    # Between slip walls nothing exchanges tangential momentum with the walls (specular reflection keeps the
    # tangential components, there are no virtual wall particles, collisions conserve momentum per cell), so
    # (1) without force and thermostat: tangential momentum and kinetic energy are conserved to rounding, the
    #     wall-normal momentum is not;
    # (2) with a body force g along x the whole fluid accelerates as one: P_x(t) = N m g t exactly (to rounding),
    #     and the profile stays flat (plug flow), unlike the no-slip parabola.
    box, cells, nbar = (8.0, 8.0, 8.0), (8, 8, 8), 10
    n = 8 * 8 * 8 * nbar
    st = uniform_maxwell(box, n, 11)
    o = Oracle(box, cells, nbar, 5, bc=(0, 0, 2))
    o.set_state(*st)
    a = o.observables()
    o.step(40)
    b = o.observables()
    assert abs(b["P"][0] - a["P"][0]) < 2e-3 and abs(b["P"][1] - a["P"][1]) < 2e-3
    assert abs(b["P"][2] - a["P"][2]) > 1.0                           # the walls do take normal momentum
    assert b["E_kin"] == pytest.approx(a["E_kin"], rel=2e-6)
    assert b["n"] == n

    g, h, steps = 0.01, 0.1, 200
    o = Oracle(box, cells, nbar, 5, bc=(0, 0, 2), g=(g, 0, 0), thermostat=1)
    o.set_state(*st)
    p0 = o.observables()["P"][0]
    o.step(steps)
    ob = o.observables(8)
    assert ob["P"][0] - p0 == pytest.approx(n * g * steps * h, rel=1e-5)
    prof = ob["profile"]
    assert np.abs(prof - g * steps * h).max() < 0.08                  # flat: thermal noise of 640 particles per layer
    assert abs(prof[:2].mean() - prof[3:5].mean()) < 0.08             # no wall layer lagging behind


def test_slip_wall_cells_get_no_virtual_particles():
    # one particle alone in a wall-cut cell: with no-slip walls it collides with nbar-1 virtual particles
    # (test above), with slip walls it is alone and keeps its velocity
    o = Oracle((8, 8, 8), (8, 8, 8), 10, 1, bc=(0, 0, 2), thermostat=1)
    o.set_state([0.7], [1.2], [0.02], [0.3], [-0.4], [0.5], step=0)
    o.step(1)
    *_p, vx, vy, vz, _ = o.get_state()
    assert (vx[0], vy[0], vz[0]) == (np.float32(0.3), np.float32(-0.4), np.float32(0.5))
