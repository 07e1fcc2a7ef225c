"""Pins for the oracle's extensions beyond the pure fluid (SURVEY.md 8(f) rank 4 and the rest of rank 2):
explicit phantom-particle sets in wall-cut cells (reading U22), embedded point-particle solutes
with their own mass (reading U23), moving no-slip walls (reading U24)."""
import numpy as np
import pytest

from oracle.binding import Oracle, philox
from paper_2406_15236_b200.inputs import uniform_maxwell
from util import srd_viscosity

TAG_AT, TAG_PHANTOM = 3, 5
F24 = np.float32(2.0**-24)


def rodrigues(ax, w, alpha_deg=130.0):
    a = np.deg2rad(np.float32(alpha_deg)).astype(np.float32).astype(np.float64)
    return w * np.cos(a) + np.cross(ax, w) * np.sin(a) + ax * (ax @ w) * (1 - np.cos(a))


def find_step(o, positive):
    t = 0
    while (o.grid_shift(t)[2] > 0) != positive or o.grid_shift(t)[2] == 0:
        t += 1
    return t


# ---------------------------------------------------------------------------------------------------------------
# explicit phantom particles (U22)
# ---------------------------------------------------------------------------------------------------------------

@pytest.mark.parametrize("positive", [True, False])
def test_phantom_stream_layout_from_raw_philox_words(positive):
    # count = floorf(fmaf(nbar, phi, u)) with u = word 0 of block (cell, 0, t, TAG_PHANTOM); phantom k: words 0,1,2 of
    # block (cell, 1+2k) -> rho_x, rho_y, zeta, normals of block (cell, 2+2k) -> velocity. phi = wall fraction.
    nbar, kT, seed = 9, 0.8, 77
    o = Oracle((4.0, 4.0, 4.0), (4, 4, 4), nbar, seed, bc=(0, 0, 1), phantoms=1, kT=kT, thermostat=1)
    t = find_step(o, positive)
    s = o.grid_shift(t)
    sp = np.float32(s[2]) if positive else np.float32(1.0) + np.float32(s[2])
    lo, hi = (1, 5) if positive else (0, 4)
    for iz, top in ((lo, False), (hi, True)):
        ijk = np.array([2, 1, iz], np.int32)
        cid = 2 + 4 * (1 + 4 * iz)
        phi = np.float32(1.0) - sp if top else sp
        w = philox([cid, 0, t, TAG_PHANTOM], [seed, 0])
        u = np.float32(w[0] >> 8) * F24
        nph = int(np.floor(np.float32(np.float64(np.float32(nbar)) * np.float64(phi) + np.float64(u))))   # fmaf: one rounding
        rho, v = o.phantoms(ijk, s, t)
        assert len(rho) == nph and nph >= 0
        for k in range(nph):
            P = philox([cid, 1 + 2 * k, t, TAG_PHANTOM], [seed, 0])
            ua, ub, zeta = (np.float32(P[j] >> 8) * F24 for j in range(3))
            rw = np.float32(np.float64(zeta) * np.float64(phi) + np.float64(sp)) if top else zeta * phi
            assert np.array_equal(rho[k], np.array([ua, ub, rw], np.float64))
            g = o.normals(cid, 2 + 2 * k, t, TAG_PHANTOM)[:3]
            assert np.allclose(v[k], np.sqrt(kT) * g, atol=1e-14)
            # the phantom lies in the wall: its z coordinate, (layer - 1 + rho_w) a - s_z, is outside [0, L]
            z = (iz - 1 + rho[k, 2]) * 1.0 - float(s[2])
            assert (z > 4.0 - 1e-6) if top else (z < 1e-6)
    # cells that are not cut get none
    assert len(o.phantoms(np.array([2, 1, 2], np.int32), s, t)[0]) == 0


def test_phantoms_fill_cut_cells_to_the_mean_density():
    # "... such that the whole collision cell contains the same average number <N_c> of fluid particles":
    # over many shifts, real + phantom particles per cut cell average to <N_c>, and the phantoms' wall-normal
    # coordinate is uniform over the wall part of the cell.
    nbar, cells = 10, (6, 6, 6)
    box = tuple(float(c) for c in cells)
    n = 6**3 * nbar
    st = uniform_maxwell(box, n, 3)
    o = Oracle(box, cells, nbar, 5, bc=(0, 0, 1), phantoms=1, dt=1e-30, thermostat=1)
    tot, ncell, zs = 0.0, 0, []
    for t in range(60):
        o.set_state(*st, step=t)
        o.step(1)
        s = o.grid_shift(t)
        cnt = o.get_cells()[0].reshape(8, 6, 6)
        lo, hi = (1, 7) if s[2] > 0 else (0, 6)
        sp = s[2] if s[2] > 0 else 1.0 + s[2]
        for iz, top in ((lo, False), (hi, True)):
            for iy in range(6):
                for ix in range(6):
                    rho, _ = o.phantoms(np.array([ix, iy, iz], np.int32), s, t)
                    tot += cnt[iz, iy, ix] + len(rho)
                    ncell += 1
                    phi = (1.0 - sp) if top else sp
                    if len(rho):
                        zs.extend((((rho[:, 2] - sp) if top else rho[:, 2]) / phi).tolist())
    assert tot / ncell == pytest.approx(nbar, rel=0.02)            # 4320 cells x 10: sigma of the mean ~ 0.4 %
    zs = np.array(zs)
    assert zs.min() >= 0.0 and zs.max() <= 1.0
    assert zs.mean() == pytest.approx(0.5, abs=0.01) and zs.var() == pytest.approx(1 / 12, rel=0.05)


@pytest.mark.parametrize("collision", [0, 1])
def test_phantoms_take_part_in_plus_a_collision_recomputed_by_hand(collision):
    # two real particles in a wall-cut cell, SRD+a or MPC-AT+a with explicit phantoms: the members of the cell are the
    # real particles (ascending id) followed by the phantoms; Eqs. (2)-(4) / reading U5 recomputed in numpy.
    nbar, seed, kT = 6, 41, 1.3
    o = Oracle((3.0, 3.0, 3.0), (3, 3, 3), nbar, seed, bc=(0, 0, 1), phantoms=1, conserve_L=1, collision=collision, dt=1e-30, kT=kT)
    t = find_step(o, True)
    s = o.grid_shift(t)
    r = np.array([[1.2, 0.3, 0.04], [1.6, 0.7, 0.10]], np.float32)
    v = np.array([[0.3, -0.4, 0.5], [-0.8, 0.1, 0.2]], np.float32)
    cells = [o.cell_of(r[i], s) for i in range(2)]
    assert cells[0][1] == cells[1][1] and cells[0][0][2] == 1
    ijk, cid = cells[0][0], cells[0][1]
    o.set_state(r[:, 0], r[:, 1], r[:, 2], v[:, 0], v[:, 1], v[:, 2], step=t)
    o.step(1)
    got = np.stack(o.get_state()[3:6], 1)[np.argsort(o.get_state()[6])]
    prho, pv = o.phantoms(ijk, s, t)
    assert len(prho) >= 1
    rho = np.vstack([np.stack([cells[i][3] for i in range(2)]).astype(np.float64), prho])
    vel = np.vstack([v.astype(np.float64), pv])
    N = len(rho)
    vcm, rcm = vel.mean(0), rho.mean(0)
    rc = rho - rcm
    if collision == 0:
        ax = o.srd_axis(cid, t)
        vnew = np.array([rodrigues(ax, w) for w in vel - vcm])
    else:
        vr = np.sqrt(kT) * np.array([o.normals(cid, k, t, TAG_AT)[:3] for k in range(N)])
        vnew = vr - vr.mean(0)
    dL = np.cross(rc, (vel - vcm) - vnew).sum(0)
    I = sum((x @ x) * np.eye(3) - np.outer(x, x) for x in rc)
    om = np.linalg.solve(I, dL)
    want = vcm + vnew + np.cross(om, rc)
    assert np.allclose(got, want[:2], atol=5e-7)
    # angular momentum about the centre of mass and momentum of ALL members are conserved by the rule
    assert np.allclose(np.cross(rc, want).sum(0), np.cross(rc, vel).sum(0), atol=1e-12)
    assert np.allclose(want.sum(0), vel.sum(0), atol=1e-12)


@pytest.mark.slow
def test_poiseuille_with_phantoms_and_mpc_at_matches_analytic_viscosity():
    # MPC-AT-a between no-slip walls with explicit phantoms, body force along x: parabola with the closed-form MPC-AT
    # viscosity (Noguchi, Kikuchi, Gompper 2007; ref. [70] of the paper): nu_kin = (kT h/m) (N/(N-1+e^-N) - 1/2),
    # nu_col = a^2 (N-1+e^-N) / (12 h N). <N_c> = 10, h = 0.1: nu = 0.0611 + 0.7500 = 0.8111.
    box, cells, nbar, h, g = (12.0, 8.0, 12.0), (12, 8, 12), 10, 0.1, 0.005
    st = uniform_maxwell(box, 12 * 8 * 12 * nbar, 5)
    o = Oracle(box, cells, nbar, 321, collision=1, g=(g, 0, 0), bc=(0, 0, 1), phantoms=1, dt=h)
    o.set_state(*st)
    o.step(800)
    prof, nav = np.zeros(12), 0
    for _ in range(500):
        o.step(4)
        prof += o.observables(12)["profile"]
        nav += 1
    prof /= nav
    zc = np.arange(12) + 0.5
    A = np.stack([zc * (12 - zc), np.ones(12)], 1)
    coef, *_ = np.linalg.lstsq(A, prof, rcond=None)
    fac = nbar - 1 + np.exp(-nbar)
    nu = h * (nbar / fac - 0.5) + fac / (12 * h * nbar)
    assert g / (2 * coef[0]) == pytest.approx(nu, rel=0.07)
    assert abs(coef[1]) < 0.08 * prof.max()                        # near no-slip
    assert o.observables()["kT_est"] == pytest.approx(1.0, rel=0.03)


# ---------------------------------------------------------------------------------------------------------------
# embedded solutes (U23)
# ---------------------------------------------------------------------------------------------------------------

def test_solute_hand_cell():
    # masses 1 and 3, v1 = (1,0,0), v2 = (-1,2,0): v_cm = (-0.5, 1.5, 0); rotation by 90 deg about z:
    # w1 = (1.5,-1.5,0) -> (1.5,1.5,0), w2 = (-0.5,0.5,0) -> (-0.5,-0.5,0)  =>  v1' = (1,3,0), v2' = (-1,1,0).
    # Momentum (-2,6,0) and kinetic energy 8 unchanged.
    o = Oracle((3.0, 3.0, 3.0), (3, 3, 3), 2, 1, alpha_deg=90.0, solute_id0=1, solute_mass=3.0)
    o.set_state([0.2, 0.6], [0.3, 0.5], [0.5, 0.5], [1.0, -1.0], [0.0, 2.0], [0.0, 0.0])
    o.collide_one_cell(axis=[0.0, 0.0, 1.0])
    *_p, vx, vy, vz, ids = o.get_state()
    assert np.array_equal(ids, [0, 1])
    assert np.allclose([vx[0], vy[0], vz[0]], [1.0, 3.0, 0.0], atol=3e-7)
    assert np.allclose([vx[1], vy[1], vz[1]], [-1.0, 1.0, 0.0], atol=3e-7)
    ob = o.observables()
    assert np.allclose(ob["P"], [-2.0, 6.0, 0.0], atol=1e-6) and ob["E_kin"] == pytest.approx(8.0, abs=1e-6)


def _per_cell(key, nkeys, w):
    return np.bincount(key, weights=w, minlength=nkeys)


@pytest.mark.parametrize("kw", [dict(), dict(conserve_L=1), dict(collision=1), dict(collision=1, conserve_L=1), dict(thermostat=1)])
def test_solute_collisions_conserve_mass_weighted_momentum(kw):
    # per cell: sum m_i v_i unchanged by the collision for every variant; SRD-a without thermostat: sum m_i v_i^2 too;
    # +a: sum m_i r_i x v_i about any fixed point of the cell too (dt ~ 0: positions do not move).
    cells, nbar, M = (6, 6, 6), 8, 4.0
    box = tuple(float(c) for c in cells)
    n = 6**3 * nbar
    st = uniform_maxwell(box, n, 9)
    nsol = n // 10
    o = Oracle(box, cells, nbar, 17, dt=1e-30, solute_id0=n - nsol, solute_mass=M, **kw)
    o.set_state(*st)
    o.step(1)
    x, y, z, vx, vy, vz, ids = o.get_state()
    key = o.get_cells()[5]
    order = np.argsort(ids)
    inv = np.empty(n, np.int64); inv[ids] = np.arange(n)
    m = np.where(ids >= n - nsol, M, 1.0)
    v0 = np.stack(st[3:6], 1).astype(np.float64)[ids]            # velocities before, in the order after
    v1 = np.stack([vx, vy, vz], 1).astype(np.float64)
    for d in range(3):
        a, b = _per_cell(key, o.nkeys, m * v0[:, d]), _per_cell(key, o.nkeys, m * v1[:, d])
        assert np.abs(a - b).max() < 2e-5
    if not kw:
        e0, e1 = _per_cell(key, o.nkeys, m * (v0**2).sum(1)), _per_cell(key, o.nkeys, m * (v1**2).sum(1))
        assert np.abs(e0 - e1).max() < 1e-4
    if kw.get("conserve_L"):
        s = o.grid_shift(0)
        r = np.stack([x, y, z], 1).astype(np.float64) + s
        rho = r - np.floor(r)
        L0, L1 = np.cross(rho, v0) * m[:, None], np.cross(rho, v1) * m[:, None]
        for d in range(3):
            assert np.abs(_per_cell(key, o.nkeys, L0[:, d]) - _per_cell(key, o.nkeys, L1[:, d])).max() < 3e-5
        assert o.observables()["n_singular_cells"] < 5


def test_solute_kappa_and_andersen_draws_use_the_particle_mass():
    # Eq. (6) with sum m_i v_ic^2; MPC-AT: v_ran,i = sqrt(kT/m_i) g_i, centred with mass weights. Recomputed in numpy.
    M, kT = 5.0, 0.6
    r = np.array([[0.2, 0.3, 0.4], [0.6, 0.5, 0.5], [0.8, 0.1, 0.7]], np.float32)
    v = np.array([[1.0, 0.2, -0.3], [-0.5, 0.4, 0.1], [0.3, -0.6, 0.8]], np.float32)
    m = np.array([1.0, 1.0, M])
    for collision in (0, 1):
        o = Oracle((3.0, 3.0, 3.0), (3, 3, 3), 3, 23, thermostat=1, collision=collision, kT=kT, solute_id0=2, solute_mass=M)
        o.set_state(r[:, 0], r[:, 1], r[:, 2], v[:, 0], v[:, 1], v[:, 2])
        o.collide_one_cell(cid=7, t=4)
        got = np.stack(o.get_state()[3:6], 1)
        vd = v.astype(np.float64)
        vcm = (m[:, None] * vd).sum(0) / m.sum()
        if collision == 0:
            W2 = (m[:, None] * (vd - vcm) ** 2).sum()
            kappa = np.sqrt(2.0 * kT * o.mbs_energy(7, 4, 3) / W2)
            ax = o.srd_axis(7, 4)
            want = vcm + kappa * np.array([rodrigues(ax, w) for w in vd - vcm])
        else:
            vr = np.array([np.sqrt(kT / m[k]) * o.normals(7, k, 4, TAG_AT)[:3] for k in range(3)])
            want = vcm + vr - (m[:, None] * vr).sum(0) / m.sum()
        assert np.allclose(got, want, atol=5e-7)


@pytest.mark.parametrize("kw", [dict(collision=1), dict(thermostat=1)])
def test_solutes_equilibrate_to_kT_over_their_mass(kw):
    # equipartition: <v_d^2> of a solute of mass M is kT / M (MPC-AT by construction, SRD through the collisions with
    # the thermostatted solvent)
    cells, nbar, M = (8, 8, 8), 10, 5.0
    box = tuple(float(c) for c in cells)
    n = 8**3 * nbar
    st = uniform_maxwell(box, n, 2)
    nsol = 512
    o = Oracle(box, cells, nbar, 3, solute_id0=n - nsol, solute_mass=M, **kw)
    o.set_state(*st)
    o.step(60)
    acc, k = 0.0, 0
    for _ in range(40):
        o.step(5)
        *_p, vx, vy, vz, ids = o.get_state()
        sel = ids >= n - nsol
        acc += (vx[sel].astype(np.float64) ** 2 + vy[sel].astype(np.float64) ** 2 + vz[sel].astype(np.float64) ** 2).mean() / 3
        k += 1
    assert acc / k == pytest.approx(1.0 / M, rel=0.04)
    assert o.observables()["kT_est"] == pytest.approx(1.0, rel=0.02)


# ---------------------------------------------------------------------------------------------------------------
# moving no-slip walls (U24)
# ---------------------------------------------------------------------------------------------------------------

def test_moving_wall_bounce_back_hand_cases():
    uw = 0.4
    o = Oracle((8, 8, 8), (8, 8, 8), 10, 1, bc=(0, 0, 1), dt=0.1, thermostat=1, wall_velocity=uw)
    # upper wall (moves with +uw): hit at t = 0.02; in the wall frame v -> -v, i.e. v' = 2 u_wall - v
    r, v = o.stream_one([3.0, 4.0, 7.98], [0.5, 0.25, 1.0])
    assert np.allclose(v, [2 * uw - 0.5, -0.25, -1.0], atol=1e-7)
    assert np.allclose(r, [3.0 + 0.5 * 0.02 + (2 * uw - 0.5) * 0.08, 4.0 + 0.25 * 0.02 - 0.25 * 0.08, 7.92], atol=1e-6)
    # lower wall (moves with -uw)
    r, v = o.stream_one([3.0, 4.0, 0.05], [0.5, -0.25, -1.0])
    assert np.allclose(v, [-2 * uw - 0.5, 0.25, 1.0], atol=1e-7)
    assert np.allclose(r, [3.0 + 0.5 * 0.05 + (-2 * uw - 0.5) * 0.05, 4.0, 0.05], atol=1e-6)
    # no hit: untouched
    r, v = o.stream_one([3.0, 4.0, 4.0], [0.5, -0.25, -1.0])
    assert np.array_equal(v, np.array([0.5, -0.25, -1.0], np.float32))


@pytest.mark.parametrize("phantoms", [0, 1])
def test_moving_wall_particles_are_thermal_about_the_wall_velocity(phantoms):
    # virtual (U8) and phantom (U22) particles of a moving wall: Gaussian about the wall velocity, -uw at the wall at 0,
    # +uw at the wall at L. One real particle in a cut cell at each wall; Eq. (2) recomputed in numpy.
    nbar, uw, seed = 5, 0.7, 13
    o = Oracle((2.0, 2.0, 2.0), (2, 2, 2), nbar, seed, bc=(0, 0, 1), dt=1e-30, wall_velocity=uw, phantoms=phantoms)
    t = find_step(o, True)
    s = o.grid_shift(t)
    for r, sign in (([0.7, 1.2, 0.03], -1.0), ([0.7, 1.2, 1.99], +1.0)):
        r = np.array(r, np.float32)
        v = np.array([0.3, -0.4, 0.5], np.float32)
        ijk, cid, _k, _rho = o.cell_of(r, s)
        assert ijk[2] == (1 if sign < 0 else 3)
        o.set_state([r[0]], [r[1]], [r[2]], [v[0]], [v[1]], [v[2]], step=t)
        o.step(1)
        got = np.array([a[0] for a in o.get_state()[3:6]])
        if phantoms:
            _rho, virt = o.phantoms(ijk, s, t)
            raw = np.array([o.normals(cid, 2 + 2 * k, t, TAG_PHANTOM)[:3] for k in range(len(virt))])
        else:
            raw = np.array([o.normals(cid, k, t, 4)[:3] for k in range(nbar - 1)])
            virt = raw + np.array([sign * uw, 0.0, 0.0])
        assert np.allclose(virt - raw, [sign * uw, 0.0, 0.0], atol=1e-12)
        if len(virt) == 0:
            assert np.array_equal(got, v)
            continue
        allv = np.vstack([v.astype(np.float64), virt])
        vcm = allv.mean(0)
        want = vcm + rodrigues(o.srd_axis(cid, t), v - vcm)
        assert np.allclose(got, want, atol=3e-7)


@pytest.mark.slow
def test_couette_profile_is_linear_with_little_slip():
    # steady plane Couette flow between walls moving with -+uw: v_x(z) = uw (2 z / L - 1); relaxation time
    # L^2/(pi^2 nu) = 7.5 (75 steps) for L = 8, nu = 0.87
    box, cells, nbar, uw = (8.0, 8.0, 8.0), (8, 8, 8), 10, 0.3
    st = uniform_maxwell(box, 8**3 * nbar, 5)
    o = Oracle(box, cells, nbar, 99, thermostat=1, bc=(0, 0, 1), wall_velocity=uw)
    o.set_state(*st)
    o.step(400)
    prof, nav = np.zeros(8), 0
    for _ in range(400):
        o.step(3)
        prof += o.observables(8)["profile"]
        nav += 1
    prof /= nav
    zc = np.arange(8) + 0.5
    A = np.stack([2 * zc / 8 - 1, np.ones(8)], 1)
    coef, res, *_ = np.linalg.lstsq(A, prof, rcond=None)
    assert coef[0] == pytest.approx(uw, rel=0.06)                  # slope: no more than a few per cent of slip
    assert abs(coef[1]) < 0.01
    assert np.abs(prof - A @ coef).max() < 0.012                    # linear
    assert o.observables()["kT_cell"] == pytest.approx(1.0, rel=0.03)


def test_kappa_counts_the_phantoms():
    # thermostat on, explicit phantoms: N_c, v_cm and sum m |v - v_cm|^2 of Eqs. (5)-(7) run over real + phantom
    # particles (they "participate in the collision step as all other fluid particles")
    nbar, kT, seed = 7, 0.9, 29
    o = Oracle((2.0, 2.0, 2.0), (2, 2, 2), nbar, seed, bc=(0, 0, 1), dt=1e-30, kT=kT, thermostat=1, phantoms=1)
    t = find_step(o, False)
    s = o.grid_shift(t)
    r = np.array([1.3, 0.4, 0.02], np.float32)
    v = np.array([-0.6, 0.2, 0.9], np.float32)
    ijk, cid, _k, _rho = o.cell_of(r, s)
    assert ijk[2] == 0                                             # cut layer at the wall at 0 for s_z < 0
    o.set_state([r[0]], [r[1]], [r[2]], [v[0]], [v[1]], [v[2]], step=t)
    o.step(1)
    got = np.array([a[0] for a in o.get_state()[3:6]])
    _rho, pv = o.phantoms(ijk, s, t)
    assert len(pv) >= 2
    allv = np.vstack([v.astype(np.float64), pv])
    vcm = allv.mean(0)
    kappa = np.sqrt(2.0 * kT * o.mbs_energy(cid, t, len(allv)) / ((allv - vcm) ** 2).sum())
    want = vcm + kappa * rodrigues(o.srd_axis(cid, t), v - vcm)
    assert np.allclose(got, want, atol=3e-7)
    assert abs(np.sqrt(2.0 * kT * o.mbs_energy(cid, t, 2) / ((allv - vcm) ** 2).sum()) - kappa) > 1e-2
