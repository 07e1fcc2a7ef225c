"""Pins for the oracle's Lees-Edwards shear boundary ("Optionally, shear flow can also be added",
PAPER.md:350 "periodic, no-slip (both also supporting shear flow)"; reading U21 in DESIGN.md): the periodic images
above / below the box along z are displaced by +-D(t) = +-gamma L_z t along x and move with +-U = +-gamma L_z.

Hand cases for the crossing and for a collision across the sheared face, then the two physics pins: the steady profile
v_x(z) = gamma (z - L_z/2) and the shear viscosity from the measured shear stress (momentum flux through planes),
which must equal the closed form nu = 0.8700 that the Poiseuille test (test_oracle_walls.py) pins independently."""
import numpy as np
import pytest

from oracle.binding import Oracle
from paper_2406_15236_b200.inputs import uniform_maxwell
from util import srd_viscosity


def test_crossing_the_sheared_face_hand_case():
    g, Lz, h = 0.05, 8.0, 0.1
    o = Oracle((8, 8, 8), (8, 8, 8), 10, 1, shear_rate=g, dt=h)
    U = g * Lz
    for t in (0, 7, 123):
        D, Uo = o.le_offset(t)
        assert Uo == pytest.approx(U, rel=1e-7)
        assert D == pytest.approx((U * h * (t + 1)) % 8.0, abs=1e-6)
        # leaves through the top: re-enters at the bottom of the image above, which is ahead by D and faster by U
        r, v = o.stream_one_at(t, [3.0, 4.0, 7.95], [0.5, 0.25, 1.0])
        assert np.allclose(r, [(3.0 + 0.05 - D) % 8.0, 4.025, 0.05], atol=2e-6)
        assert np.allclose(v, [0.5 - U, 0.25, 1.0], atol=1e-7)
        # leaves through the bottom
        r, v = o.stream_one_at(t, [3.0, 4.0, 0.02], [0.5, 0.25, -1.0])
        assert np.allclose(r, [(3.0 + 0.05 + D) % 8.0, 4.025, 7.92], atol=2e-6)
        assert np.allclose(v, [0.5 + U, 0.25, -1.0], atol=1e-7)
        # no crossing: nothing changes, x stays periodic
        r, v = o.stream_one_at(t, [7.99, 4.0, 4.0], [1.0, 0.0, 0.5])
        assert np.allclose(r, [0.09, 4.0, 4.05], atol=2e-6) and np.allclose(v, [1.0, 0.0, 0.5])
    # gamma = 0 is the plain periodic box
    o0 = Oracle((8, 8, 8), (8, 8, 8), 10, 1, dt=h)
    r, v = o0.stream_one_at(5, [3.0, 4.0, 7.95], [0.5, 0.25, 1.0])
    assert np.allclose(r, [3.05, 4.025, 0.05], atol=2e-6) and np.allclose(v, [0.5, 0.25, 1.0])


def test_collision_across_the_sheared_face_recomputed_by_hand():
    # Two particles that share a collision cell only through the sheared image: one just below the top face whose
    # shifted z leaves the box (it collides as its image: x - D, v_x - U), one just above the bottom face.
    g, L, h, nbar = 0.25, 4.0, 0.1, 10
    o = Oracle((L, L, L), (4, 4, 4), nbar, 5, shear_rate=g, dt=h)
    U = g * L
    t = 0
    while o.grid_shift(t)[2] < 0.2:
        t += 1
    s = o.grid_shift(t)
    D, _ = o.le_offset(t)
    assert 0.05 < D < L - 0.05
    # positions AFTER the move of step t (velocities chosen first, start positions = end - v h)
    vt, vb = np.array([0.7, -0.3, 0.2]), np.array([-0.4, 0.6, -0.1])
    top_end = np.array([2.3, 1.4, L - 0.1])                           # z + s_z >= L: image frame
    xb = (top_end[0] - D) % L                                          # same column in the image frame
    bot_end = np.array([xb, 1.4, 0.05])
    start = [top_end - vt * h, bot_end - vb * h]
    st = np.array(start, np.float32)
    vel = np.array([vt, vb], np.float32)
    o.set_state(st[:, 0], st[:, 1], st[:, 2], vel[:, 0], vel[:, 1], vel[:, 2], step=t)
    o.step(1)
    x, y, z, vx, vy, vz, ids = o.get_state()
    order = np.argsort(ids)
    cnt, *_r, key = o.get_cells()
    assert key[order][0] == key[order][1] and cnt[key[0]] == 2         # one cell, two members
    ijk, cid, k, im = o.cell_of_le(t, [x[order][0], y[order][0], z[order][0]], s)
    assert im == -1 and k == key[order][0]
    ijk_b, _cid, kb, imb = o.cell_of_le(t, [x[order][1], y[order][1], z[order][1]], s)
    assert imb == 0 and kb == k
    # Eq. (2) in the frame of the image: the top particle enters with v_x - U and gets U back afterwards
    v_in = np.array([vel[0].astype(np.float64) - [U, 0, 0], vel[1].astype(np.float64)])
    vcm = v_in.mean(0)
    ax = o.srd_axis(cid, t)
    a = np.deg2rad(np.float32(130.0)).astype(np.float32).astype(np.float64)
    out = []
    for w in v_in - vcm:
        out.append(vcm + w * np.cos(a) + np.cross(ax, w) * np.sin(a) + ax * (ax @ w) * (1 - np.cos(a)))
    out = np.array(out)
    out[0, 0] += U
    got = np.stack([vx, vy, vz], 1)[order]
    assert np.allclose(got, out, atol=5e-7)
    # momentum is conserved; kinetic energy is conserved in the image frame, NOT in the laboratory frame
    assert np.allclose(got.sum(0), vel.sum(0), atol=1e-6)
    e_img = lambda v: ((v[0] - [U, 0, 0]) ** 2).sum() + (v[1] ** 2).sum()
    assert e_img(got.astype(np.float64)) == pytest.approx(e_img(vel.astype(np.float64)), abs=2e-6)
    assert abs((got.astype(np.float64) ** 2).sum() - (vel.astype(np.float64) ** 2).sum()) > 1e-2


@pytest.mark.slow
def test_shear_profile_and_viscosity_from_shear_stress():
    # Steady simple shear: v_x(z) = gamma (z - L_z/2), and the shear stress sigma_xz = eta gamma with
    # eta = rho nu = 10 * 0.8700 (SRD closed form, kinetic + collisional; pinned to the paper's printed 111.3 in
    # test_oracle_walls.py). The stress is measured as the flux of x-momentum through the interior planes z = 1..L-1:
    # particles carrying m v_x across a plane while streaming (kinetic part) and the momentum handed from the members
    # of a collision cell below the plane to those above it (collisional part).
    L, nbar, g, h = 16, 10, 0.02, 0.1
    box, cells = (float(L),) * 3, (L, L, L)
    n = L**3 * nbar
    st = list(uniform_maxwell(box, n, 21))
    st[3] = (st[3] + g * (st[2] - L / 2)).astype(np.float32)           # start on the steady profile: short transient
    o = Oracle(box, cells, nbar, 77, thermostat=1, shear_rate=g, dt=h)
    o.set_state(*st)
    o.step(300)
    nplanes = L - 1                                                    # the interior planes z = 1 .. L-1
    kin = col = kin_all = 0.0
    prof = np.zeros(L)
    nsamp = 2400
    U = g * L
    x0, y0, z0, vx0, vy0, vz0, id0 = o.get_state()
    for it in range(nsamp):
        t = int(o.observables()["step"])
        o.step(1)
        x1, y1, z1, vx1, vy1, vz1, id1 = o.get_state()                # rebin_every = 1: order changes, match by id
        a0, a1 = np.argsort(id0), np.argsort(id1)
        zb, vzb, vxb = z0[a0].astype(np.float64), vz0[a0].astype(np.float64), vx0[a0].astype(np.float64)
        za = zb + vzb * h                                              # unwrapped end of the move
        # a particle going from zb to za crosses the interior planes p with zb < p <= za upwards (or za < p <= zb downwards):
        # their number, signed, is the difference of the two layer indices clipped to the box
        crossed = np.clip(np.floor(za), 0, L - 1) - np.clip(np.floor(zb), 0, L - 1)
        kin += (vxb * crossed).sum()
        # the same flux averaged over ALL plane heights in (0, L) instead of the 15 integer ones: v_x times the stretch of z
        # the particle covers (every particle contributes at every step, so the thermal noise is far smaller); the part of
        # the stretch beyond the sheared face is covered in the image, where the particle's velocity is v_x -+ U
        kin_all += (vxb * (np.clip(za, 0.0, L) - zb)).sum() + ((vxb - U) * np.maximum(za - L, 0.0)).sum() + ((vxb + U) * np.minimum(za, 0.0)).sum()
        # collision of step t: members of the cell layer that straddles a plane, by the side of the plane they are on
        s = o.grid_shift(t)
        zc = z1[a1].astype(np.float64)                                 # positions at the collision
        dvx = vx1[a1].astype(np.float64) - vxb
        # particles that crossed the sheared face while streaming changed v_x by -+U outside the collision: undo
        dvx += U * ((za >= L).astype(float) - (za < 0).astype(float))
        lay = np.floor(zc + s[2]).astype(int)                          # cell layer (unwrapped) of every particle
        p = lay if s[2] > 0 else lay + 1                               # the plane inside the layer [lay - s_z, lay + 1 - s_z)
        col += dvx[(p >= 1) & (p <= L - 1) & (zc >= p)].sum()          # handed to the members above the plane
        prof += o.observables(L)["profile"]
        x0, y0, z0, vx0, vy0, vz0, id0 = x1, y1, z1, vx1, vy1, vz1, id1
    prof /= nsamp
    zmid = np.arange(L) + 0.5
    slope = np.polyfit(zmid, prof, 1)[0]
    assert slope == pytest.approx(g, rel=0.03)
    assert np.abs(prof - g * (zmid - L / 2)).max() < 0.015             # linear through the sheared face, no slip
    flux = (kin + col) / (nsamp * nplanes * L * L * h)                 # x-momentum per area and time, upwards (m = 1)
    eta = -flux / g
    nu_kin, nu_col = srd_viscosity(nbar, h, 130)
    assert eta == pytest.approx(nbar * (nu_kin + nu_col), rel=0.04)    # 8.70
    # kinetic part alone: eta_kin = rho nu_kin = 0.486, from the all-heights estimator: a sum of n = 40,960 terms v_x v_z h per
    # step with variance (kT/m)^2 h^2 each, so its standard error is sqrt(n / nsamp) / (L^3 g) = 0.050. Checked at 3 standard
    # errors, |eta_kin - 0.486| < 0.15: a missing kinetic part (0) and a doubled one (0.97) both fail. (The 15-plane
    # estimator that the total uses has a standard error of 0.15 here on its kinetic part alone; in the total that noise
    # cancels, because the thermal v_x a particle carries across a plane is handed back by the collisions.)
    eta_kin = -kin_all / (nsamp * L * L * L * h * g)
    se = np.sqrt(n / nsamp) / (L**3 * g)
    assert se < 0.052
    assert abs(eta_kin - nbar * nu_kin) < 3 * se, eta_kin
    assert abs(-kin / (nsamp * nplanes * L * L * h * g) - eta_kin) < 3 * 0.15   # the two estimators agree
    assert o.observables()["kT_cell"] == pytest.approx(1.0, rel=0.02)
