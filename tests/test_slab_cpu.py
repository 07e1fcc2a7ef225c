"""Host-side logic of the slab decomposition (paper_2406_15236_b200/slab.py): partition, neighbours, ownership; and the
agreement of the ranks on it through a process group (gloo, world size 2)."""
import os
import subprocess
import sys

import numpy as np
import pytest

from paper_2406_15236_b200.slab import slab_neighbours, slab_owner, slab_partition

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_partition_covers_the_box_in_whole_brick_layers():
    for nz, world, bz in [(64, 2, 8), (64, 4, 8), (512, 8, 8), (72, 3, 8), (40, 2, 4), (48, 3, 8)]:
        parts = slab_partition(nz, world, bz)
        assert parts[0][0] == 0 and sum(n for _, n in parts) == nz
        for (z0, n), (z1, _) in zip(parts, parts[1:] + [(nz, 0)]):
            assert z0 + n == z1 and z0 % bz == 0 and n % bz == 0 and n >= 2 * bz and n + 2 * bz <= nz
        assert max(n for _, n in parts) - min(n for _, n in parts) <= bz


@pytest.mark.parametrize("args", [(60, 2, 8), (64, 1, 8), (64, 5, 8), (16, 2, 8)])
def test_partition_rejects_what_the_kernels_cannot_hold(args):
    with pytest.raises(ValueError):
        slab_partition(*args)


def test_neighbours_and_owner():
    assert slab_neighbours(0, 4) == (3, 1) and slab_neighbours(3, 4) == (2, 0) and slab_neighbours(1, 2) == (0, 0)
    parts = slab_partition(64, 4, 8)
    z = np.array([0.0, 15.999, 16.0, 31.5, 32.0, 63.999])
    assert list(slab_owner(z, 1.0, parts)) == [0, 0, 1, 1, 2, 3]
    assert list(slab_owner(2.0 * z, 2.0, parts)) == [0, 0, 1, 1, 2, 3]


WORKER = r"""
import os, sys
import numpy as np
import torch, torch.distributed as dist
sys.path.insert(0, sys.argv[1])
from paper_2406_15236_b200.slab import slab_partition, slab_neighbours, slab_owner
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:" + sys.argv[2], rank=int(sys.argv[3]), world_size=2)
rank, world = dist.get_rank(), dist.get_world_size()
parts = slab_partition(64, world, 8)
below, above = slab_neighbours(rank, world)
# every rank hands its (pointer, brick layers) pair to its neighbours: here the pair is (rank tag, layers)
mine = torch.tensor([1000 + rank, parts[rank][1] // 8 + 2], dtype=torch.int64)
got = [torch.zeros(2, dtype=torch.int64) for _ in range(world)]
dist.all_gather(got, mine)
assert got[below][0].item() == 1000 + below and got[above][1].item() == parts[above][1] // 8 + 2
# particles are dealt to their owners; nobody is lost or doubled
rng = np.random.default_rng(5)
z = rng.uniform(0, 64, 1000)
own = slab_owner(z, 1.0, parts)
n = torch.tensor([int((own == rank).sum())])
dist.all_reduce(n)
assert n.item() == 1000
dist.barrier()
print("ok", rank)
"""


def test_two_ranks_agree_on_the_decomposition(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = str(29600 + os.getpid() % 300)
    procs = [subprocess.Popen([sys.executable, str(script), ROOT, port, str(r)], stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
             for r in range(2)]
    outs = [p.communicate(timeout=120)[0] for p in procs]
    for r, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0 and f"ok {r}" in o, o
