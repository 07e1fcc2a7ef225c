"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times
(brick = {16,16,8}; config 5 with rebin_every = 10).

configs 2-4 are compared element by element against the oracle (one step costs the oracle seconds).
config 5 (1.34e9 particles) is checked on sampled outputs the oracle computes one by one: for a random
sample of collision cells ALL member particles are pulled from the GPU, and the oracle's stream / cell
index / collision hooks are applied to exactly those particles; plus properties that hold at any size."""
import gc

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle.binding import Oracle  # noqa: E402
from paper_2406_15236_b200 import MPC  # noqa: E402
from paper_2406_15236_b200.inputs import uniform_maxwell, uniform_maxwell_cuda  # noqa: E402
from test_parity_gpu import compare_step, gpu_get, gpu_set  # noqa: E402
from test_parity_plus_a_gpu import check_plus_a_velocities, lambda_min_per_particle  # noqa: E402

BRICK = (16, 16, 8)


def test_config2_srd_mbs_64cubed():
    cells, nbar = (64, 64, 64), 10
    box = (64.0, 64.0, 64.0)
    n = 64**3 * nbar
    st = uniform_maxwell(box, n, 1234)
    kw = dict(thermostat=1, rebin_every=1, brick=BRICK)
    o = Oracle(box, cells, nbar, 1234, **kw)
    g = MPC(box, cells, nbar, 1234, n_max=n, **kw)
    o.set_state(*st)
    for t in range(2):
        gpu_set(g, o.get_state(), step=t)
        o.step(1)
        g.step(1)
        compare_step(o, g)
    # free running from here: equilibrium temperature and conservation on the GPU (config 2: thermostat on)
    g.step(50)
    ob = g.observables()
    assert ob["kT_cell"] == pytest.approx(1.0, rel=5e-3)
    assert np.all(np.abs(ob["P"]) < 1.0)


def test_config3_at_plus_a_128cubed():
    cells, nbar = (128, 128, 128), 10
    box = (128.0,) * 3
    n = 128**3 * nbar
    st = uniform_maxwell(box, n, 1234)
    kw = dict(collision=1, conserve_L=1, dt=0.02, brick=BRICK)
    o = Oracle(box, cells, nbar, 1234, **kw)
    g = MPC(box, cells, nbar, 1234, n_max=n, **kw)
    o.set_state(*st)
    gpu_set(g, st)
    o.step(1)
    g.step(1)
    so, sg = o.get_state(), gpu_get(g)
    assert np.array_equal(so[6], sg[6])
    for d in range(3):
        assert np.max(np.abs(so[d] - sg[d])) <= 1e-5
    cnt_o, *_r, key_o = o.get_cells()
    cnt_g, *_q, key_g = [a.cpu().numpy() for a in g.get_cells()]
    assert np.array_equal(key_o, key_g.view(np.uint32)) and np.array_equal(cnt_o, cnt_g.view(np.uint32))
    _lam, _N, cond = lambda_min_per_particle(o, so, key_o, 0)
    assert check_plus_a_velocities(so, sg, cond, "config 3") < 0.05     # U10 tolerance, fraction of loose particles
    assert int(o.observables()["n_singular_cells"]) == int(g.observables()["n_singular_cells"])
    g.step(20)
    ob = g.observables()
    assert ob["kT_est"] == pytest.approx(1.0, rel=5e-3)      # Andersen thermostat holds k_BT


def test_config4_walls_gravity_256x64x64():
    cells, nbar = (256, 64, 64), 10
    box = (256.0, 64.0, 64.0)
    n = 256 * 64 * 64 * nbar
    st = uniform_maxwell(box, n, 1234)
    kw = dict(thermostat=1, bc=(0, 0, 1), g=(0.001, 0.0, 0.0), rebin_every=1, brick=BRICK)
    o = Oracle(box, cells, nbar, 1234, **kw)
    g = MPC(box, cells, nbar, 1234, n_max=n, **kw)
    o.set_state(*st)
    gpu_set(g, st)
    o.step(1)
    g.step(1)
    compare_step(o, g)
    a, b = o.observables(64), g.observables(profile=True)
    assert np.allclose(a["profile"], b["profile"], atol=2e-5)
    assert b["kT_cell"] == pytest.approx(a["kT_cell"], rel=1e-5)


def members_of(key, sample_keys, nkeys):
    """Indices (device int64) of the particles whose key is in sample_keys, found chunk by chunk through a bitmap over
    the key space (torch.isin would sort 2.7e9 keys)."""
    bitmap = torch.zeros(nkeys, dtype=torch.bool, device=key.device)
    bitmap[sample_keys.long()] = True
    out = []
    for lo in range(0, key.numel(), 1 << 28):
        c = key[lo:lo + (1 << 28)]
        out.append(torch.nonzero(bitmap[c.long()]).squeeze(1) + lo)
    return torch.cat(out)


@pytest.mark.parametrize("nbar", [5, 10, 20])
def test_config5_sampled_cells_512cubed(nbar):
    # BASELINE.json configs[4], all three densities of its sweep, in the launch configuration bench.py times.
    # <N_c> = 20: 2,684,354,560 particles (> 2^31: unsigned 32-bit indices), compact workspace (property-wise reorder,
    # PAPER.md:156-162), state handed over through the host-pointer ABI as bench.py does.
    # One call of 13 steps from t = 0: reorder of an unordered state at t = 0 (unfolded), nine fused steps on a stale order,
    # the reorder at t = 10, which is folded into the sweeps of t = 10, 11, 12 where the second particle copy exists (arrival
    # ranks, 32-byte records written at their slots of the new order, records read back) and property-wise
    # otherwise (compact workspace, 20 per cell), and t = 12, the step checked here against the oracle: with the second copy
    # it IS the read-back pass of the folded reorder, so every sampled particle has gone through all three passes (the
    # kernel-family counters are asserted, the test cannot fall back to the unfolded path unnoticed). No single-step call
    # in the chain: the state before the last step comes from a run of 12 steps in one call, which cannot fold the reorder
    # at t = 10 (too few steps left) and so takes the unfolded one (the GPU path is bit-reproducible, and independent of how
    # steps are split over calls: test_config5_fused_call_equals_single_steps_512cubed).
    gc.collect()
    torch.cuda.empty_cache()                     # blocks cached by earlier tests count as used
    free, _total = torch.cuda.mem_get_info()
    if free < 165e9:
        pytest.skip("needs ~165 GB of device memory")
    cells, seed = (512, 512, 512), 1234
    box = (512.0,) * 3
    n = 512**3 * nbar
    compact = nbar == 20
    kw = dict(thermostat=1, rebin_every=10, brick=BRICK)
    nsteps = 13
    g = MPC(box, cells, nbar, seed, n_max=n, compact=compact, **kw)
    nkeys = g.nkeys

    def fresh_state():
        if compact:                              # 64 GB of inputs do not fit beside the 138 GB workspace
            st = uniform_maxwell_cuda(box, n, seed, to_host=True)
            g.set_state_host(*st)
        else:
            st = uniform_maxwell_cuda(box, n, seed)
            g.set_state(*st)
        torch.cuda.synchronize()
        del st
        g._keep = None
        torch.cuda.empty_cache()

    # run 1: the full call; sample cells and their members from the keys of the last step
    fresh_state()
    g.profile_enable()
    g.step(nsteps)
    fam = g.profile_read()
    g.profile_enable(False)
    assert fam["sweep_gather"][1] == (0 if compact else 3), fam   # rank, scatter and read-back passes of the reorder at t = 10
    g.canonicalise()                             # keys below are per particle of the CURRENT order: fix it first
    cnt, px, py, pz, e2, key = g.get_cells()
    assert int(cnt.sum(dtype=torch.int64)) == n
    ob = g.observables()
    assert ob["n"] == n and ob["step"] == nsteps and ob["n_range_overflows"] == 0
    assert ob["kT_cell"] == pytest.approx(1.0, rel=2e-3)
    assert np.all(np.abs(ob["P"]) < 100.0)                       # zero net momentum up to fp32 rounding of 1e9 terms
    assert ob["max_cell_count"] < {5: 30, 10: 45, 20: 70}[nbar]   # Poisson(<N_c>) over 1.3e8 cells
    rng = np.random.default_rng(7)
    sample = torch.from_numpy(np.unique(rng.integers(0, nkeys, 300)).astype(np.int32)).cuda()
    idx = members_of(key, sample, nkeys)
    k = key[idx].cpu().numpy().view(np.uint32)
    cnt_h = cnt[sample.long()].cpu().numpy().view(np.uint32)
    psum = [t[sample.long()].cpu().numpy() for t in (px, py, pz)]
    del cnt, px, py, pz, e2, key
    torch.cuda.empty_cache()
    Q = g.get_state_at(idx)                                      # post-collision state of the members, canonical order
    # run 2: the same trajectory stopped one step earlier (12 steps in one call) -> state before the last step
    fresh_state()
    g.step(nsteps - 1)
    g.canonicalise()
    P = g.get_state_at(idx)
    assert np.array_equal(P[6], Q[6])                            # t = 12 does not reorder: same memory order
    if nbar == 20:
        assert int(idx.max()) > 2**31                            # indices beyond 2^31 are exercised
    o = Oracle(box, cells, nbar, seed, **kw)
    t = nsteps - 1
    s = o.grid_shift(t)
    tested = 0
    for j, c in enumerate(sample.cpu().numpy()):
        m = k == np.uint32(c)
        assert m.sum() == cnt_h[j]                               # membership is complete
        if m.sum() == 0:
            continue
        ids = P[6][m]
        r0 = np.stack([P[0][m], P[1][m], P[2][m]], 1)
        v0 = np.stack([P[3][m], P[4][m], P[5][m]], 1)
        r1 = np.stack([Q[0][m], Q[1][m], Q[2][m]], 1)
        v1 = np.stack([Q[3][m], Q[4][m], Q[5][m]], 1)
        cid = None
        for i in range(len(ids)):                                # MOVE and cell index, particle by particle
            rr, vv = o.stream_one(r0[i], v0[i])
            assert np.array_equal(rr, r1[i])
            _ijk, cj, kj, _rho = o.cell_of(rr, s)
            assert kj == c
            cid = cj
        o.set_state(r1[:, 0], r1[:, 1], r1[:, 2], v0[:, 0], v0[:, 1], v0[:, 2], id=ids, step=t)
        o.collide_one_cell(cid=cid, t=t)                          # Eq. (2),(5)-(7) on exactly these particles
        *_p, ox, oy, oz, oid = o.get_state()
        want = np.stack([ox, oy, oz], 1)
        assert np.array_equal(oid, ids)
        assert np.max(np.abs(want.astype(np.float64) - v1)) <= 2e-5
        # cell momentum: GPU sums vs the members' velocities
        want_p = v0.astype(np.float64).sum(0)
        l1 = np.abs(v0).sum() + 1e-30
        got = np.array([psum[0][j], psum[1][j], psum[2][j]])
        assert np.max(np.abs(got - want_p)) / l1 <= 1e-5
        tested += 1
    assert tested > 250
    g.close()


def test_config5_fused_call_equals_single_steps_512cubed():
    # At config 5's full size, in the launch configuration bench.py times: one call of 13 steps from t = 0 (first-step sweep,
    # unfolded reorder of the unordered state at t = 0, the steady-state 3-CTA sweep with the collision of the previous step
    # fused in, the reorder at t = 10 folded into the sweeps of t = 10, 11, 12: asserted from the kernel-family counters)
    # must leave bit for bit the state that 13 calls of one step leave (unfused: sweep, cell, trailing collide each, every
    # reorder unfolded; that path is the one checked against the oracle in lock-step at small sizes).
    gc.collect()
    torch.cuda.empty_cache()                     # blocks cached by earlier tests count as used
    free, _total = torch.cuda.mem_get_info()
    if free < 150e9:
        pytest.skip("needs ~150 GB of device memory")
    cells, nbar, seed = (512, 512, 512), 10, 1234
    box = (512.0,) * 3
    n = 512**3 * nbar
    kw = dict(thermostat=1, rebin_every=10, brick=BRICK)
    g = MPC(box, cells, nbar, seed, n_max=n, **kw)

    def fresh_state():
        st = uniform_maxwell_cuda(box, n, seed)  # the same seeded state both times
        g.set_state(*st, step=0)
        torch.cuda.synchronize()
        del st
        torch.cuda.empty_cache()

    fresh_state()
    for _ in range(13):
        g.step(1)                                # t = 0 .. 12, one call each
    ref = [t.cpu() for t in g.get_state()]
    torch.cuda.empty_cache()
    fresh_state()
    g.profile_enable()
    g.step(13)                                   # the same thirteen steps in one call
    fam = g.profile_read()
    g.profile_enable(False)
    assert fam["sweep_gather"][1] == 3 and fam["sweep"][1] == 10, fam
    got = g.get_state()
    for a, b in zip(ref, got):
        assert torch.equal(a, b.cpu())
    assert g.observables()["step"] == 13
