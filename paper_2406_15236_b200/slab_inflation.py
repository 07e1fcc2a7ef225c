"""Work inflation of the slab decomposition, measured on ONE GPU.

    python -m paper_2406_15236_b200.slab_inflation --ranks 2 [--cells 512,512,256] [--nbar 10] [--steps 20] [--warmup 12] [--rebin-every 10]

prints one JSON line. Not a benchmark of the product and not a scaling number (see measure_slabs)."""
import argparse
import json

import numpy as np


def measure_slabs(cells, nbar, world_sub, steps, warmup, rebin_every):
    """Work inflation of the slab decomposition on ONE GPU: the box once as a whole and once as `world_sub`
    slab subdomain contexts run one after the other (a barrier of the ranks = the end of a Python loop here), same seeded
    input, same number of steps; both timed with CUDA events. Not a scaling number: nothing runs in parallel, there is no
    NVLink in it. It says how much more work the ranks do together than the single-domain run (halo cells finalised twice,
    shared sums added twice, hand-over records)."""
    import torch

    from paper_2406_15236_b200 import MPC
    from paper_2406_15236_b200.inputs import uniform_maxwell_cuda
    from paper_2406_15236_b200.slab import slab_neighbours, slab_partition

    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * nbar
    brick = (16, 16, 8)
    kw = dict(thermostat=1, rebin_every=rebin_every, brick=brick)
    st = list(uniform_maxwell_cuda(box, n, 4321, device="cuda:0", to_host=False))
    out = {}
    whole = MPC(box, cells, nbar, 99, n_max=n, **kw)
    whole.set_state(*st)
    whole.step(warmup)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(whole.stream); whole.step(steps); e1.record(whole.stream)
    torch.cuda.synchronize()
    out["whole_ms_per_step"] = e0.elapsed_time(e1) / steps
    whole.close()
    del whole
    torch.cuda.empty_cache()
    parts = slab_partition(cells[2], world_sub, brick[2])
    layer = torch.floor(st[2]).to(torch.int64)                      # a = 1 in the bench boxes
    ranks = []
    for z0, nz in parts:
        sel = torch.nonzero((layer >= z0) & (layer < z0 + nz)).flatten()
        g = MPC(box, cells, nbar, 99, n_max=int(1.1 * sel.numel()) + 1024, sub=(z0, nz), **kw)
        ranks.append((g, sel))
    for r, (g, _) in enumerate(ranks):
        below, above = slab_neighbours(r, world_sub)
        g.sub_connect(ranks[below][0].sub_export(), ranks[above][0].sub_export())
    for g, sel in ranks:
        g.set_state(*[a[sel].contiguous() for a in st[:6]], id=sel.to(torch.int32))      # ids = index in the whole box
    del st, layer
    torch.cuda.empty_cache()

    def run(k):
        for i in range(k):
            for g, _ in ranks:
                g.sub_begin(k - 1 - i)
            for g, _ in ranks:
                g.sub_end()

    run(warmup)
    torch.cuda.synchronize()
    s = ranks[0][0].stream
    e0.record(s); run(steps); e1.record(s)
    torch.cuda.synchronize()
    out["slabs_ms_per_step_summed_over_ranks"] = e0.elapsed_time(e1) / steps
    out["ranks"] = world_sub
    out["inflation"] = out["slabs_ms_per_step_summed_over_ranks"] / out["whole_ms_per_step"]
    out["range_overflows"] = sum(int(g.observables()["n_range_overflows"]) for g, _ in ranks)
    out["config"] = {"cells": list(cells), "n_per_cell": nbar, "particles": n, "rebin_every": rebin_every, "steps": steps, "warmup": warmup,
                     "note": "one GPU, ranks run one after the other; the reorders of the subdomains are the folded ones and hand particles over inside their kernels"}
    for g, _ in ranks:
        g.close()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--ranks", type=int, default=2)
    ap.add_argument("--cells", default="512,512,256")
    ap.add_argument("--nbar", type=int, default=10)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=12)
    ap.add_argument("--rebin-every", type=int, default=10)
    a = ap.parse_args()
    cells = tuple(int(t) for t in a.cells.split(","))
    print(json.dumps({"slab_work_inflation": measure_slabs(cells, a.nbar, a.ranks, a.steps, a.warmup, a.rebin_every)}), flush=True)


if __name__ == "__main__":
    main()
