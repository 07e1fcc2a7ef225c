"""Seeded synthetic input generators shared by the tests, bench.py and the oracle checks.

Holds none of the method's arithmetic: only uniform positions and Maxwell velocities with the
shapes of the paper's benchmark workloads (uniform-density boxes, <N_c> = 5..50, PAPER.md:274-276;
configs in BASELINE.json). Host arrays come from numpy's PCG64; device arrays (config 5, 1.3e9
particles) from torch's CUDA generator. Recipe: DESIGN.md "Input recipe".
"""
import numpy as np


def uniform_maxwell(box, n, seed, kT=1.0, mass=1.0, zero_momentum=True, rest=False):
    """Positions i.i.d. uniform in [0,L_d); velocities i.i.d. N(0, kT/m) per component with the mean
    removed (double sum, cast). Returns six float32 arrays and ids 0..n-1."""
    rng = np.random.Generator(np.random.PCG64(seed))
    pos = []
    for d in range(3):
        u = rng.random(n, dtype=np.float32)            # [0,1) in fp32
        r = (u * np.float32(box[d])).astype(np.float32)
        r[r >= np.float32(box[d])] = np.float32(0.0)   # u*L can round up to L
        pos.append(r)
    vel = []
    for d in range(3):
        if rest:
            vel.append(np.zeros(n, np.float32))
            continue
        v = rng.standard_normal(n) * np.sqrt(kT / mass)
        if zero_momentum:
            v -= v.mean()
        vel.append(v.astype(np.float32))
    ids = np.arange(n, dtype=np.uint32)
    return (*pos, *vel, ids)


def uniform_maxwell_cuda(box, n, seed, kT=1.0, mass=1.0, device="cuda:0", to_host=False):
    """Device twin for sizes the host cannot hold comfortably: same distributions from torch's
    CUDA generator. Returns six float32 device tensors (ids are implied 0..n-1); with to_host=True each
    array is moved to pinned host memory as soon as it is made (for states that do not fit beside the
    library's workspace: config 5 at 20 particles per cell)."""
    import torch

    g = torch.Generator(device=device)
    g.manual_seed(seed)
    out = []
    for d in range(3):
        r = torch.rand(n, device=device, dtype=torch.float32, generator=g)
        r.mul_(float(box[d]))
        r.masked_fill_(r >= float(box[d]), 0.0)
        out.append(_park(r, to_host))
    for d in range(3):
        v = torch.randn(n, device=device, dtype=torch.float32, generator=g)
        v.mul_(float(np.sqrt(kT / mass)))
        tot = 0.0                       # mean in float64, chunk by chunk (no second full-size array)
        for c in v.split(1 << 28):
            tot += float(c.sum(dtype=torch.float64))
        v.sub_(tot / n)
        out.append(_park(v, to_host))
    return tuple(out)


def _park(t, to_host):
    if not to_host:
        return t
    import torch

    h = torch.empty(t.shape, dtype=t.dtype, pin_memory=True)
    h.copy_(t)
    return h
