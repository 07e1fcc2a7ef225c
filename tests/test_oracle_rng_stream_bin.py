"""Pins for the oracle: Philox stream, streaming (Eq. 1), grid shift, binning and reorder.
CPU only. Citations: PAPER.md:29-37 (Sec. II), 152-154 (III.B.3); readings U1-U4, U12."""
import numpy as np
import pytest

from oracle.binding import Oracle, philox
from paper_2406_15236_b200.inputs import uniform_maxwell


def test_philox_known_answers(golden):
    rows = golden("philox_kat.txt")
    assert len(rows) == 3
    for r in rows:
        v = [int(t, 16) for t in r]
        out = philox(v[0:4], v[4:6])
        assert [int(o) for o in out] == v[6:10]


def test_philox_counter_and_key_sensitivity():
    # every counter word and key word changes the block (guards against a dropped word)
    base = philox([1, 2, 3, 4], [5, 6])
    for w in range(4):
        c = [1, 2, 3, 4]
        c[w] ^= 1
        assert not np.array_equal(philox(c, [5, 6]), base)
    assert not np.array_equal(philox([1, 2, 3, 4], [4, 6]), base)
    assert not np.array_equal(philox([1, 2, 3, 4], [5, 7]), base)


def test_philox_uniformity():
    outs = np.array([philox([i, 0, 7, 1], [1234, 0]) for i in range(4000)], dtype=np.uint64)
    u = (outs >> 8).astype(np.float64) / 2**24
    assert abs(u.mean() - 0.5) < 0.01
    assert abs(u.var() - 1 / 12) < 0.005
    # bits are balanced
    bits = ((outs[:, :, None] >> np.arange(32, dtype=np.uint64)) & 1).mean(axis=(0, 1))
    assert np.all(np.abs(bits - 0.5) < 0.03)


def test_stream_is_fmaf_closed_form():
    o = Oracle((16, 16, 16), (16, 16, 16), 10, 1, dt=0.1)
    rng = np.random.default_rng(0)
    for _ in range(200):
        r = rng.uniform(1, 15, 3).astype(np.float32)
        v = rng.normal(0, 1, 3).astype(np.float32)
        r1, v1 = o.stream_one(r, v)
        # fmaf(v,h,r) == the correctly rounded value of v*h + r, which float64 reproduces exactly here
        exact = (v.astype(np.float64) * np.float64(np.float32(0.1)) + r.astype(np.float64)).astype(np.float32)
        assert np.array_equal(r1, exact)
        assert np.array_equal(v1, v)


def test_periodic_wrap_edges():
    L = 16.0
    o = Oracle((L, L, L), (16, 16, 16), 10, 1, dt=0.1)
    tiny = np.float32(1e-9)
    # r = 0, v*h = -tiny: r + L rounds to exactly L, which must map to 0 (reading U2)
    r1, _ = o.stream_one([0.0, 0.0, 0.0], [-tiny * 10, 0.0, 0.0])
    assert r1[0] == 0.0
    # just below L stays
    below = np.nextafter(np.float32(L), np.float32(0))
    r1, _ = o.stream_one([below, 1.0, 1.0], [0.0, 0.0, 0.0])
    assert r1[0] == below
    # crossing the upper face comes back near 0
    r1, _ = o.stream_one([below, 1.0, 1.0], [1.0, 0.0, 0.0])
    assert 0.0 <= r1[0] < 0.11
    # crossing the lower face comes back near L
    r1, _ = o.stream_one([0.05, 1.0, 1.0], [-1.0, 0.0, 0.0])
    assert L - 0.06 < r1[0] < L
    # exactly 0 stays 0
    r1, _ = o.stream_one([0.0, 0.0, 0.0], [0.0, 0.0, 0.0])
    assert np.all(r1 == 0.0)


def test_gravity_update_closed_form():
    g = 0.25
    o = Oracle((16, 16, 16), (16, 16, 16), 10, 1, dt=0.1, g=(g, 0, 0), thermostat=1)
    r1, v1 = o.stream_one([3.0, 4.0, 5.0], [0.5, -0.25, 0.125])
    h = 0.1
    assert r1[0] == pytest.approx(3.0 + 0.5 * h + 0.5 * g * h * h, abs=1e-6)
    assert v1[0] == pytest.approx(0.5 + g * h, abs=1e-7)
    assert r1[1] == pytest.approx(4.0 - 0.025, abs=1e-6) and v1[1] == np.float32(-0.25)


def test_shift_range_and_moments():
    o = Oracle((8, 8, 8), (8, 8, 8), 10, 99)
    s = np.array([o.grid_shift(t) for t in range(6000)], dtype=np.float64)
    assert s.min() >= -0.5 and s.max() < 0.5
    assert np.all(np.abs(s.mean(axis=0)) < 0.02)
    assert np.all(np.abs(s.var(axis=0) - 1 / 12) < 0.006)
    # independent axes, and steps differ
    assert abs(np.corrcoef(s[:, 0], s[:, 1])[0, 1]) < 0.05
    assert len({tuple(r) for r in s}) == len(s)
    # scales with a
    o2 = Oracle((16, 16, 16), (8, 8, 8), 10, 99)
    assert np.allclose(o2.grid_shift(5), 2.0 * o.grid_shift(5))
    # switched off
    o3 = Oracle((8, 8, 8), (8, 8, 8), 10, 99, grid_shift=0)
    assert np.all(o3.grid_shift(3) == 0)


def test_keys_without_shift_equal_floor():
    box, cells = (12.0, 8.0, 10.0), (12, 8, 10)
    st = uniform_maxwell(box, 5000, 3)
    o = Oracle(box, cells, 10, 5, grid_shift=0, dt=1e-30)
    o.set_state(*st)
    o.step(1)
    x, y, z, *_rest, ids = o.get_state()
    cnt, *_s, key = o.get_cells()
    expect = np.floor(x).astype(np.int64) + 12 * (np.floor(y).astype(np.int64) + 8 * np.floor(z).astype(np.int64))
    assert np.array_equal(key.astype(np.int64), expect)
    assert cnt.sum() == 5000
    assert np.array_equal(cnt, np.bincount(key, minlength=o.nkeys))


@pytest.mark.parametrize("brick", [1, 4, (4, 2, 8)])
def test_binning_bruteforce_with_shift(brick):
    box, cells = (8.0, 12.0, 16.0), (8, 12, 16)
    n = 8 * 12 * 16 * 10
    st = uniform_maxwell(box, n, 11)
    o = Oracle(box, cells, 10, 77, brick=brick)
    o.set_state(*st)
    o.step(1)
    x, y, z, vx, vy, vz, ids = o.get_state()
    cnt, px, py, pz, e2, key = o.get_cells()
    s = o.grid_shift(0).astype(np.float64)
    # brute force in float64: where the shifted position is not within 1e-5 of a cell face the index is unambiguous
    q = np.stack([x, y, z], 1).astype(np.float64) + s
    frac = q - np.floor(q)
    safe = np.all((frac > 1e-5) & (frac < 1 - 1e-5), axis=1)
    assert safe.mean() > 0.999
    ijk = np.floor(q).astype(np.int64) % np.array(cells)
    if brick == 1:
        expect = ijk[:, 0] + 8 * (ijk[:, 1] + 12 * ijk[:, 2])
    else:
        B = np.array((brick,) * 3 if isinstance(brick, int) else brick)
        mb = [int(np.ceil(c / bb)) for c, bb in zip(cells, B)]
        b = ijk // B
        l = ijk % B
        expect = ((b[:, 2] * mb[1] + b[:, 1]) * mb[0] + b[:, 0]) * int(np.prod(B)) + (l[:, 2] * B[1] + l[:, 1]) * B[0] + l[:, 0]
    assert np.array_equal(key[safe].astype(np.int64), expect[safe])
    # the oracle's own cell_of hook agrees for every particle (also the unsafe ones)
    for i in np.flatnonzero(~safe)[:20]:
        _, _, k, _ = o.cell_of([x[i], y[i], z[i]], o.grid_shift(0))
        assert k == key[i]
    # sorted by (key, id), strictly ascending
    kk = key.astype(np.int64) * 2**32 + ids.astype(np.int64)
    assert np.all(np.diff(kk) > 0)
    assert cnt.sum() == n
    # occupancy is Poisson(10) for uniform positions
    assert o.nkeys == 8 * 12 * 16          # all three layouts tile this box exactly
    occ = cnt
    assert abs(occ.mean() - 10) < 1e-9
    assert abs(occ.var() - 10) < 1.5


def test_physics_independent_of_key_layout_and_rebin_interval():
    box, cells = (8.0, 8.0, 8.0), (8, 8, 8)
    st = uniform_maxwell(box, 5120, 21)
    res = []
    for brick, every in [(1, 1), (4, 1), (2, 3), (1, 1000), ((16, 16, 8), 2), ((4, 2, 1), 1)]:
        o = Oracle(box, cells, 10, 4242, brick=brick, rebin_every=every, thermostat=1)
        o.set_state(*st)
        o.step(7)
        x, y, z, vx, vy, vz, ids = o.get_state()
        order = np.argsort(ids)
        res.append(np.stack([a[order] for a in (x, y, z, vx, vy, vz)]))
    for r in res[1:]:
        assert np.array_equal(r, res[0])   # sums are taken in ascending id: bit-identical


def test_create_rejects_bad_arguments():
    with pytest.raises(ValueError):
        Oracle((8, 8, 9), (8, 8, 8), 10, 1)                      # non-cubic cells
    with pytest.raises(ValueError):
        Oracle((8, 8, 8), (8, 8, 0), 10, 1)
    with pytest.raises(ValueError):
        Oracle((8, 8, 8), (8, 8, 8), 10, 1, conserve_L=1, thermostat=1)   # SRD+a with MBS (U6)
    with pytest.raises(ValueError):
        Oracle((8, 8, 8), (8, 8, 8), 10, 1, bc=(1, 0, 1))        # more than one wall axis
    with pytest.raises(ValueError):
        Oracle((8, 8, 8), (8, 8, 8), 10, 1, bc=(0, 0, 1), g=(0, 0, 0.1))
    with pytest.raises(ValueError):
        Oracle((8, 8, 8), (8, 8, 8), 10, 1, rebin_every=0)
