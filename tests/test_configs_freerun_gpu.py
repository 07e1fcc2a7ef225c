"""Full-length free-running runs of BASELINE.json's configs 2, 3 and 4 on the GPU, checked against what the
physics fixes (conservation laws, the thermostat's temperature, the analytic SRD viscosity). Lock-step parity
with the oracle is in test_parity_*.py; these runs check that nothing drifts over the configs' step counts."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from paper_2406_15236_b200 import MPC  # noqa: E402
from paper_2406_15236_b200.inputs import uniform_maxwell  # noqa: E402
from util import poiseuille_startup, srd_viscosity  # noqa: E402


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_set(g, st):
    x, y, z, vx, vy, vz, ids = st
    g.set_state(*[dev(a) for a in (x, y, z, vx, vy, vz)], id=dev(ids.view(np.int32)))


def test_config2_1000_steps_thermostat_holds_kT():
    # config 2: SRD + cell-level MBS thermostat, 64^3 cells, 10 per cell, rebin every step, 1,000 steps
    cells, nbar = (64, 64, 64), 10
    box = (64.0,) * 3
    n = 64**3 * nbar
    st = uniform_maxwell(box, n, 1234)
    g = MPC(box, cells, nbar, 1234, n_max=n, thermostat=1, rebin_every=1, brick=(16, 16, 8))
    gpu_set(g, st)
    p0 = np.array(g.observables()["P"])
    kts = []
    for _ in range(10):
        g.step(100)
        ob = g.observables()
        kts.append(ob["kT_cell"])
        assert ob["n"] == n
    assert ob["step"] == 1000
    # Eq. (6)-(7): the cell-level temperature is k_BT at every sampling point (1.8e6 degrees of freedom per cell
    # class: statistical error ~1e-3), and the thermostat conserves momentum (Eq. 5 acts on relative velocities)
    assert np.allclose(kts, 1.0, atol=3e-3)
    assert np.abs(np.array(ob["P"]) - p0).max() < 1e-3 * np.sqrt(n)       # fp32 rounding of n velocities over 1,000 steps
    # Maxwell distribution of one component: variance k_BT/m, excess kurtosis 0
    vx = g.get_state()[3].double()
    assert float(vx.var()) == pytest.approx(1.0, rel=5e-3)
    assert float(((vx - vx.mean()) ** 4).mean() / vx.var() ** 2) == pytest.approx(3.0, abs=0.02)


def test_config3_500_steps_at_plus_a():
    # config 3: MPC-AT+a, 128^3 cells, 10 per cell, dt = 0.02, 500 steps
    cells, nbar = (128, 128, 128), 10
    box = (128.0,) * 3
    n = 128**3 * nbar
    st = uniform_maxwell(box, n, 1234)
    g = MPC(box, cells, nbar, 1234, n_max=n, collision=1, conserve_L=1, dt=0.02, rebin_every=1, brick=(16, 16, 8))
    gpu_set(g, st)
    p0 = np.array(g.observables()["P"])
    for _ in range(5):
        g.step(100)
        ob = g.observables()
        # the Andersen thermostat redraws every relative velocity at k_BT: <v_d^2> = k_BT/m up to the
        # (N_c-1)/N_c and angular-momentum constraints, which kT_cell accounts for only partly; the global
        # estimate stays within a per cent of 1
        assert ob["kT_est"] == pytest.approx(1.0, rel=2e-2)
    assert ob["step"] == 500 and ob["n"] == n
    assert np.abs(np.array(ob["P"]) - p0).max() < 1e-3 * np.sqrt(n)       # per-cell momentum conservation, summed
    assert ob["n_singular_cells"] < 1e-3 * 128**3                          # U10 rejections are rare at 10 per cell


def test_config4_5000_steps_profile_follows_startup_series():
    # config 4: SRD + MBS, 256x64x64 cells, no-slip walls at z = 0, 64 (bounce-back + virtual wall particles),
    # g = 0.001 x, fluid at rest (Maxwell velocities, zero mean flow), 5,000 steps of 0.1. One viscous relaxation time (U14): the profile is compared with
    # the start-up series of plane Poiseuille flow for the analytic SRD viscosity nu = 0.8700, averaged over the
    # same sampling times, not with the steady parabola.
    cells, nbar = (256, 64, 64), 10
    box = (256.0, 64.0, 64.0)
    n = 256 * 64 * 64 * nbar
    gx, h = 0.001, 0.1
    st = uniform_maxwell(box, n, 1234)
    g = MPC(box, cells, nbar, 1234, n_max=n, thermostat=1, bc=(0, 0, 1), g=(gx, 0.0, 0.0), rebin_every=10,
            brick=(16, 16, 8))
    gpu_set(g, st)
    zc = np.arange(64) + 0.5
    nu = sum(srd_viscosity(10, h, 130))
    assert nu == pytest.approx(0.870025, rel=1e-5)
    g.step(4500)
    prof = np.zeros(64)
    want = np.zeros(64)
    nav = 0
    for _ in range(10):
        g.step(50)
        ob = g.observables(profile=True)
        prof += ob["profile"]
        want += poiseuille_startup(zc, ob["step"] * h, gx, nu, 64.0)
        nav += 1
    prof /= nav
    want /= nav
    assert ob["step"] == 5000
    vmax = want.max()
    assert vmax == pytest.approx(0.638 * gx * 64.0**2 / (8 * nu), rel=0.03)      # 63.8 % of the steady centre-line value (U14)
    # amplitude (least squares on the series' shape) within 4 %, shape residual and wall slip within 3 % of v_max
    amp = float(prof @ want / (want @ want))
    assert amp == pytest.approx(1.0, abs=0.04)
    assert np.abs(prof - amp * want).max() < 0.03 * vmax
    assert np.abs(prof - prof[::-1]).max() < 0.02 * vmax                          # symmetric about the mid-plane
    assert ob["kT_cell"] == pytest.approx(1.0, rel=5e-3)                          # thermostat holds k_BT under forcing
    assert ob["n_range_overflows"] == 0
