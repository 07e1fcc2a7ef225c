"""Slab subdomains (multi-GPU domain decomposition) on ONE GPU: R
subdomain contexts in one process, run one after the other (nothing waits on anything: a barrier of the ranks is the
end of a Python loop here), each adding the sums of its shared cells into its neighbours' arrays (device pointers: on
several GPUs the same pointers are peer mappings). Integer sums commute and every cell draws its random numbers by its
id in the whole box, so the decomposed trajectory must equal the single-domain one BIT FOR BIT."""
import numpy as np
import pytest
import torch

from paper_2406_15236_b200 import MPC
from paper_2406_15236_b200.binding import MPCError
from paper_2406_15236_b200.inputs import uniform_maxwell
from paper_2406_15236_b200.slab import slab_neighbours, slab_owner, slab_partition

pytestmark = pytest.mark.gpu


def to_dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def by_id(state):
    s = [t.cpu().numpy() for t in state]
    order = np.argsort(s[6].view(np.uint32))
    return [a[order] for a in s]


def make_ranks(box, cells, nbar, seed, st, world, brick, n_max_of=None, **kw):
    parts = slab_partition(cells[2], world, brick[2])
    a = box[2] / cells[2]
    owner = slab_owner(st[2], a, parts)
    ranks = []
    for r, (z0, nz) in enumerate(parts):
        sel = np.nonzero(owner == r)[0]
        n_max = max(2 * len(sel), 1) if n_max_of is None else n_max_of(r, len(sel))
        g = MPC(box, cells, nbar, seed, n_max=n_max, brick=brick, sub=(z0, nz), **kw)
        ranks.append((g, sel))
    exports = [g.sub_export() for g, _ in ranks]
    if not all(e[0][2] for e in exports):                         # staging buffers on all ranks or on none (mpc_sub_connect)
        exports = [([e[0][0], e[0][1], 0], e[1]) for e in exports]
    for r, (g, _) in enumerate(ranks):
        below, above = slab_neighbours(r, world)
        g.sub_connect(exports[below], exports[above])
    for g, sel in ranks:
        g.set_state(*[to_dev(st[d][sel]) for d in range(6)], id=to_dev(st[6][sel].view(np.int32)))
    return ranks


def step_all(ranks, n, ahead=None):
    """n steps of all ranks; ahead: the steps promised to the library after each one (default: the rest of this call)"""
    for i in range(n):
        for g, _ in ranks:
            g.sub_begin(n - 1 - i if ahead is None else ahead)
        torch.cuda.synchronize()          # barrier of the ranks
        for g, _ in ranks:
            g.sub_end()
        torch.cuda.synchronize()          # barrier of the ranks


@pytest.mark.parametrize("world,cells,brick,kw", [
    (2, (32, 16, 64), (16, 16, 8), dict(thermostat=1, rebin_every=5)),
    (4, (32, 16, 64), (16, 16, 8), dict(thermostat=1, rebin_every=4)),
    (3, (16, 16, 48), (16, 16, 8), dict(rebin_every=3)),
    (3, (16, 16, 56), (16, 16, 8), dict(thermostat=1, rebin_every=4)),    # uneven slabs: 3, 2, 2 brick layers
    (2, (12, 10, 24), (4, 2, 4), dict(thermostat=1, rebin_every=2)),      # generic bricks, ragged x / y
    (2, (32, 16, 32), (16, 16, 8), dict(thermostat=1, rebin_every=1)),    # every layer of the box is held by both ranks
])
def test_slabs_equal_the_single_domain_run_bit_for_bit(world, cells, brick, kw):
    nbar = 10
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar - 7
    st = uniform_maxwell(box, n, 11)
    steps = 12
    ref = MPC(box, cells, nbar, 77, n_max=n, brick=brick, **kw)
    ref.set_state(*[to_dev(st[d]) for d in range(6)], id=to_dev(st[6].view(np.int32)))
    ref.step(steps)
    want = by_id(ref.get_state())
    ranks = make_ranks(box, cells, nbar, 77, st, world, brick, **kw)
    step_all(ranks, steps)
    parts = [g.get_state() for g, _ in ranks]
    got = by_id([torch.cat([p[d] for p in parts]) for d in range(7)])
    assert np.array_equal(got[6], want[6])                       # nobody lost, nobody doubled
    for d in range(6):
        assert np.array_equal(got[d], want[d]), d                # positions and velocities: bit for bit
    for g, _ in ranks:
        ob = g.observables()
        assert ob["n_range_overflows"] == 0 and ob["step"] == steps


def test_particles_change_owner_inside_the_reorder():
    # PAPER.md:152, in the kernels: with a long step the particles cross the slab faces quickly; every folded reorder
    # (t = 4, 8, ..., each with two further steps promised) writes the particles of the halo layers into the new owner's
    # staging buffer. No call of the test moves a particle, and the run still equals the single-domain one bit for bit.
    world, cells, brick, nbar = 3, (16, 16, 72), (16, 16, 8), 10
    kw = dict(thermostat=1, rebin_every=4, dt=0.5)
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar
    st = uniform_maxwell(box, n, 14)
    ref = MPC(box, cells, nbar, 6, n_max=n, brick=brick, **kw)
    ref.set_state(*[to_dev(st[d]) for d in range(6)], id=to_dev(st[6].view(np.int32)))
    ref.step(31)
    want = by_id(ref.get_state())
    ranks = make_ranks(box, cells, nbar, 6, st, world, brick, **kw)
    first = [set(st[6][sel].tolist()) for _, sel in ranks]
    step_all(ranks, 31)
    parts = slab_partition(cells[2], world, brick[2])
    states = [[a.cpu().numpy() for a in g.get_state()] for g, _ in ranks]
    changed = 0
    for r, s in enumerate(states):
        ids = set(s[6].view(np.uint32).tolist())
        changed += len(ids - first[r])
        # every particle sits in its rank's own layers or has drifted there since the last hand-over (t = 28): within the halo
        layer = np.floor(s[2]).astype(int)
        z0, nz = parts[r]
        up = (layer - z0) % cells[2]
        assert np.all((up < nz + 8) | (up >= cells[2] - 8))
        assert np.mean(up < nz) > 0.9
    assert changed > 0.05 * n                                     # a good part of the particles has changed owner
    got = by_id([np.concatenate([s[d] for s in states]) for d in range(7)])
    for d in range(7):
        assert np.array_equal(got[d], want[d]), d
    for g, _ in ranks:
        assert g.observables()["n_range_overflows"] == 0
    # a reorder step without two further steps promised stays local; reading the state in the middle of a folded reorder is refused
    step_all(ranks, 1, ahead=3)                                   # t = 31
    step_all(ranks, 1, ahead=2)                                   # t = 32: reorder step, folded
    with pytest.raises(MPCError):
        ranks[0][0].get_state()
    step_all(ranks, 2, ahead=0)
    ranks[0][0].get_state()


def by_id(state):
    s = [t.cpu().numpy() if hasattr(t, "cpu") else t for t in state]
    order = np.argsort(s[6].view(np.uint32))
    return [a[order] for a in s]


def test_particles_handed_to_their_owners_between_steps():
    # the caller's part of PAPER.md:152 ("particles that have left the subdomain are sent to the new one when the particles
    # are sorted"): read the states, deal the particles to their owners, set the states; the run continues bit for bit
    world, cells, brick, nbar = 2, (16, 16, 48), (16, 16, 8), 10
    kw = dict(thermostat=1, rebin_every=5, dt=0.5)              # a long step: particles cross the slab faces quickly
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar
    st = uniform_maxwell(box, n, 12)
    ref = MPC(box, cells, nbar, 5, n_max=n, brick=brick, **kw)
    ref.set_state(*[to_dev(st[d]) for d in range(6)], id=to_dev(st[6].view(np.int32)))
    ranks = make_ranks(box, cells, nbar, 5, st, world, brick, **kw)
    parts = slab_partition(cells[2], world, brick[2])
    t = 0
    for leg in range(4):
        ref.step(5)
        step_all(ranks, 5)
        t += 5
        states = [[a.cpu().numpy() for a in g.get_state()] for g, _ in ranks]
        allp = [np.concatenate([s[d] for s in states]) for d in range(7)]
        owner = slab_owner(allp[2], 1.0, parts)
        moved = 0
        for r, (g, _) in enumerate(ranks):
            sel = np.nonzero(owner == r)[0]
            moved += int((owner[:len(states[0][0])] != 0).sum()) if r == 0 else 0
            g.set_state(*[to_dev(allp[d][sel]) for d in range(6)], id=to_dev(allp[6][sel].view(np.int32)), step=t)
        assert moved > 0                                          # the test does exercise the hand-over
    want = by_id(ref.get_state())
    got = by_id([torch.cat([g.get_state()[d] for g, _ in ranks]) for d in range(7)])
    for d in range(7):
        assert np.array_equal(got[d], want[d]), d


@pytest.mark.parametrize("world", [2, 3])
def test_slab_step_with_hand_over_against_the_oracle(world):
    # The decomposed path in front of the ORACLE (not only of the single-domain GPU run): the whole-box oracle takes the
    # state before the last step and advances one step; the slab ranks advance 7 steps from t = 0, the last of which (t = 6)
    # is the read-back pass of the reorder folded into t = 4, 5, 6, with the particles of the halo layers written into their
    # new owners' staging buffers at t = 5. The state before the last step comes from a second set of ranks that runs 6 steps
    # (too few to fold: its reorder at t = 4 stays local and hands nothing over). Element by element, matched by id, at the
    # tolerances of tests/test_parity_gpu.py.
    from oracle.binding import Oracle
    cells, brick, nbar = (16, 16, 24 * world), (16, 16, 8), 10
    kw = dict(thermostat=1, rebin_every=4, dt=0.5)
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar - 3
    st = uniform_maxwell(box, n, 31)
    twin = make_ranks(box, cells, nbar, 8, st, world, brick, **kw)
    step_all(twin, 6)
    before = by_id([torch.cat([g.get_state()[d] for g, _ in twin]) for d in range(7)])
    assert all(g.n == len(sel) for g, sel in twin)                # nothing handed over there
    ranks = make_ranks(box, cells, nbar, 8, st, world, brick, **kw)
    for g, _ in ranks:
        g.profile_enable()
    step_all(ranks, 7)
    for g, _ in ranks:
        assert g.profile_read()["sweep_gather"][1] == 3           # rank, scatter and read-back pass of the folded reorder
    assert sum(abs(g.n - len(sel)) for g, sel in ranks) > 0       # particles have changed owner
    got = by_id([torch.cat([g.get_state()[d] for g, _ in ranks]) for d in range(7)])
    o = Oracle(box, cells, nbar, 8, brick=brick, **kw)
    o.set_state(*before[:6], before[6].view(np.uint32), step=6)
    o.step(1)
    want = by_id(o.get_state())
    assert np.array_equal(got[6].view(np.uint32), want[6].view(np.uint32))
    for d in range(3):
        assert np.max(np.abs(want[d].astype(np.float64) - got[d])) <= 1e-5
    for d in range(3, 6):
        assert np.max(np.abs(want[d].astype(np.float64) - got[d])) <= 2e-5
    for g, _ in ranks:
        assert g.observables()["n_range_overflows"] == 0


def test_an_empty_slab_takes_part_and_is_handed_particles():
    # rank 1 of 3 starts without a single particle. It must still scan its (complete) cell counts at every reorder, fold the
    # reorder like its neighbours and read back what they hand over; the particles it receives still owe the collision of the
    # step before. Bit for bit against the single-domain run of the same state.
    world, cells, brick, nbar = 3, (16, 16, 72), (16, 16, 8), 10
    kw = dict(thermostat=1, rebin_every=4, dt=0.1)              # (short step: particles fly freely through the empty part, and must
    box = tuple(float(c) for c in cells)                        # not get further than the halo between two hand-overs)
    n = int(np.prod(cells)) * nbar
    st = uniform_maxwell(box, n, 23)
    parts = slab_partition(cells[2], world, brick[2])
    keep = slab_owner(st[2], 1.0, parts) != 1
    st = [a[keep] for a in st]
    ref = MPC(box, cells, nbar, 4, n_max=len(st[0]), brick=brick, **kw)
    ref.set_state(*[to_dev(st[d]) for d in range(6)], id=to_dev(st[6].view(np.int32)))
    ref.step(15)
    want = by_id(ref.get_state())
    ranks = make_ranks(box, cells, nbar, 4, st, world, brick, n_max_of=lambda r, m: 2 * m + 30000, **kw)
    assert ranks[1][0].n == 0
    step_all(ranks, 15)                                           # folded reorders with hand-over at t = 4, 8 (12: not enough steps left)
    assert ranks[1][0].n > 1000                                   # particles have arrived in the empty slab
    for g, _ in ranks:
        assert g.observables()["n_range_overflows"] == 0
    states = [[a.cpu().numpy() for a in g.get_state()] for g, _ in ranks]
    got = by_id([np.concatenate([s[d] for s in states]) for d in range(7)])
    for d in range(7):
        assert np.array_equal(got[d], want[d]), d
    for g, _ in ranks:
        assert g.observables()["n_range_overflows"] == 0


def test_hand_over_beyond_n_max_is_refused_before_anything_is_written():
    # Rank 0 starts thin (40 % of the density) beside a full rank 1 and has room for 16 particles more than it holds: the
    # first folded reorder (t = 4) would hand it far more. The rank's mpc_sub_end of that step must refuse (MPC_ENOMEM),
    # i.e. BEFORE the next step, whose scatter passes (its own and its neighbours') write the arrivals into its staging
    # buffer of n_max records; the context is dead afterwards, the neighbour's is untouched and still readable.
    world, cells, brick, nbar = 2, (16, 16, 48), (16, 16, 8), 10
    kw = dict(thermostat=1, rebin_every=4, dt=0.5)
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar
    st = uniform_maxwell(box, n, 21)
    parts = slab_partition(cells[2], world, brick[2])
    thin = (slab_owner(st[2], 1.0, parts) == 0) & (np.arange(n) % 5 >= 2)
    st = [a[~thin] for a in st]
    ranks = make_ranks(box, cells, nbar, 9, st, world, brick, n_max_of=lambda r, m: m + 16 if r == 0 else 2 * m, **kw)
    n0 = ranks[0][0].n
    step_all(ranks, 4, ahead=8)                                   # t = 0 (local reorder) .. 3
    for g, _ in ranks:
        g.sub_begin(8)                                            # t = 4: rank pass of a folded reorder
    torch.cuda.synchronize()
    with pytest.raises(MPCError, match="n_max"):
        ranks[0][0].sub_end()
    ranks[1][0].sub_end()                                         # the neighbour has room
    torch.cuda.synchronize()
    assert ranks[0][0].n == n0                                    # nothing was handed over
    with pytest.raises(MPCError):
        ranks[0][0].sub_begin(7)                                  # dead for good
    with pytest.raises(MPCError):
        ranks[0][0].get_state()


def test_set_state_is_refused_in_the_middle_of_a_step():
    world, cells, brick, nbar = 2, (16, 16, 48), (16, 16, 8), 10
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar
    st = uniform_maxwell(box, n, 22)
    ranks = make_ranks(box, cells, nbar, 9, st, world, brick, thermostat=1, rebin_every=4)
    g, sel = ranks[0]
    args = [to_dev(st[d][sel]) for d in range(6)]
    step_all(ranks, 4, ahead=8)
    for h, _ in ranks:
        h.sub_begin(8)
    with pytest.raises(MPCError):
        g.set_state(*args)                                        # between mpc_sub_begin and mpc_sub_end
    torch.cuda.synchronize()
    for h, _ in ranks:
        h.sub_end()
    torch.cuda.synchronize()
    with pytest.raises(MPCError):
        g.set_state(*args)                                        # folded reorder in flight (t = 4 was its first step)
    step_all(ranks, 2, ahead=0)
    g.set_state(*args)                                            # between steps, nothing in flight: fine


def test_a_particle_outside_its_slab_is_reported():
    world, cells, brick, nbar = 2, (16, 16, 48), (16, 16, 8), 10
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar
    st = list(uniform_maxwell(box, n, 13))
    ranks = make_ranks(box, cells, nbar, 5, st, world, brick, thermostat=1, rebin_every=5)
    g, sel = ranks[0]
    z = st[2][sel].copy()
    z[0] = 40.5                                                   # rank 0 holds the layers 40..47 and 0..31: 40.5 is in its halo
    z[1] = 36.0                                                   # ... but layer 36 is not held by rank 0
    g.set_state(*[to_dev(a) for a in (st[0][sel], st[1][sel], z, st[3][sel], st[4][sel], st[5][sel])], id=to_dev(st[6][sel].view(np.int32)))
    step_all(ranks, 1)
    assert g.observables()["n_range_overflows"] == 1              # mpc_observables returns MPC_ERANGE: the run is invalid
    assert ranks[1][0].observables()["n_range_overflows"] == 0


def test_subdomain_rules():
    box, cells = (32.0, 16.0, 64.0), (32, 16, 64)
    for bad in (dict(sub=(0, 8)), dict(sub=(4, 32)), dict(sub=(0, 56)), dict(sub=(0, 32), bc=(0, 1, 0)), dict(sub=(0, 32), collision=1),
                dict(sub=(0, 32), g=(0.01, 0, 0)), dict(sub=(0, 32), shear_rate=0.1)):
        with pytest.raises(MPCError):
            MPC(box, cells, 10, 1, n_max=100, brick=(16, 16, 8), **bad)
    g = MPC(box, cells, 10, 1, n_max=100, brick=(16, 16, 8), sub=(0, 32))
    with pytest.raises(MPCError):
        g.sub_begin()                                             # not connected, no state
    h = MPC(box, cells, 10, 1, n_max=100, brick=(16, 16, 8), sub=(32, 32))
    g.sub_connect(h.sub_export(), h.sub_export())
    z = torch.zeros(4, device="cuda")
    g.set_state(z, z, z, z, z, z)
    with pytest.raises(MPCError):
        g.step(1)                                                 # mpc_step is for whole boxes
    with pytest.raises(MPCError):
        g.sub_end()                                               # begin first


WORKER = r"""
import os, sys
import numpy as np
import torch, torch.distributed as dist
sys.path.insert(0, sys.argv[1])
from paper_2406_15236_b200 import MPC
from paper_2406_15236_b200.inputs import uniform_maxwell
from paper_2406_15236_b200.slab_run import SlabRank
rank, world = int(sys.argv[3]), int(sys.argv[4])
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:" + sys.argv[2], rank=rank, world_size=world)
cells, nbar, brick = (16, 16, 64), 10, (16, 16, 8)
box = tuple(float(c) for c in cells)
n = int(np.prod(cells)) * nbar
st = uniform_maxwell(box, n, 21)
kw = dict(thermostat=1, rebin_every=5, dt=0.4)
r = SlabRank(box, cells, nbar, 9, brick, n_max=n, device="cuda:0", **kw)
r.set_global_state(st)
r.step(17)                                 # hand-overs at t = 5, 10, 15
got = r.gather_state()
moved = r.migrate()
if rank == 0:
    ref = MPC(box, cells, nbar, 9, n_max=n, brick=brick, **kw)
    ref.set_state(*[torch.from_numpy(st[d]).cuda() for d in range(6)], id=torch.from_numpy(st[6].view(np.int32)).cuda())
    ref.step(17)
    want = [t.cpu().numpy() for t in ref.get_state()]
    order = np.argsort(want[6].view(np.uint32))
    for d in range(7):
        assert np.array_equal(got[d], want[d][order]), d
assert r.range_overflows() == 0
r.close()
print("ok", rank, moved)
"""


@pytest.mark.parametrize("world", [2, 3])
def test_one_process_per_rank_with_ipc_mappings(world, tmp_path):
    # the deployment path: one process per rank, the neighbours' workspaces mapped with CUDA IPC, a process group for the
    # barriers and the hand-over of particles. All ranks share this box's one GPU (their kernels never wait on one
    # another: the barriers are host-side), which exercises every line of the plumbing but measures nothing.
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = str(29700 + os.getpid() % 200 + world)
    procs = [subprocess.Popen([sys.executable, str(script), root, port, str(r), str(world)], stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
             for r in range(world)]
    outs = [p.communicate(timeout=600)[0] for p in procs]
    for r, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0 and f"ok {r}" in o, o[-3000:]
