"""One process per GPU: slab subdomains of one box over a torch.distributed process group.

Plumbing only. The kernels of libmpc_b200.so do the work, including the halo exchange: a rank's sweep adds the sums of
the cells it shares with a neighbour straight into the neighbour's workspace, which this module maps into the process
with CUDA IPC (cuda-python) after the ranks have traded handles through the process group. The group is otherwise used
for the two barriers of a step and for handing particles to their new owners between steps.

    python -m torch.distributed.run --nproc-per-node R -m paper_2406_15236_b200.slab_run --cells 64,64,128 --steps 20

runs a seeded box and prints the global observables; tests/test_slab_gpu.py runs two such processes on one GPU against the
single-domain result."""
import argparse
import os

import numpy as np

from .binding import MPC, MPCError
from .slab import slab_neighbours, slab_owner, slab_partition


def _cudart():
    from cuda.bindings import runtime as cudart
    return cudart


def _ok(res):
    err = res[0]
    if int(err) != 0:
        raise RuntimeError(f"CUDA runtime error {err}")
    return res[1] if len(res) == 2 else res[1:]


class SlabRank:
    """This process's slab of the box. `group`: an initialised torch.distributed process group (any backend: device
    tensors go through it directly with NCCL, through pinned host copies otherwise)."""

    def __init__(self, box, cells, n_per_cell, seed, brick, n_max, device="cuda:0", group=None, **kw):
        import torch
        import torch.distributed as dist

        self.torch, self.dist, self.group = torch, dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.parts = slab_partition(cells[2], self.world, brick[2])
        self.a = box[2] / cells[2]
        self.device = torch.device(device)
        cudart = _cudart()
        torch.cuda.set_device(self.device)
        self._allocs = []

        def alloc(nbytes):
            p = _ok(cudart.cudaMalloc(nbytes))
            self._allocs.append(p)
            self._ws_bytes = nbytes
            return p

        self.sim = MPC(box, cells, n_per_cell, seed, n_max=n_max, device=device, brick=brick, sub=self.parts[self.rank],
                       workspace_alloc=alloc, **kw)
        # trade (IPC handle of the workspace, offsets of the exported arrays in it, local brick layers) with the neighbours
        ptrs, layers = self.sim.sub_export()
        handle = _ok(cudart.cudaIpcGetMemHandle(self.sim.workspace_ptr))
        mine = dict(rank=self.rank, pid=os.getpid(), handle=bytes(handle.reserved),
                    offsets=[(p - self.sim.workspace_ptr) if p else None for p in ptrs], layers=layers)
        everyone = [None] * self.world
        dist.all_gather_object(everyone, mine, group=group)
        # the folded reorder (with its hand-over) must be on for every rank or for none: one rank without a staging buffer
        # (compact workspace) turns it off everywhere
        fold = all(e["offsets"][2] is not None for e in everyone)
        self._opened = {}
        ends = []
        for nb in slab_neighbours(self.rank, self.world):
            info = everyone[nb]
            if info["pid"] == os.getpid():                                   # (a single-rank group cannot be partitioned; kept for symmetry)
                base = self.sim.workspace_ptr
            elif nb in self._opened:
                base = self._opened[nb]
            else:
                h = cudart.cudaIpcMemHandle_t()
                h.reserved = info["handle"]
                base = _ok(cudart.cudaIpcOpenMemHandle(h, cudart.cudaIpcMemLazyEnablePeerAccess))
                self._opened[nb] = base
            ptrs_nb = [(int(base) + o) if o is not None else 0 for o in info["offsets"]]
            if not fold:
                ptrs_nb[2] = 0
            ends.append((ptrs_nb, info["layers"]))
        self.sim.sub_connect(ends[0], ends[1])
        self.t = 0
        self._overflows = 0          # range overflows counted before earlier hand-overs (mpc_set_state restarts the library's count)
        self.barrier()

    # ---- plumbing ----
    def barrier(self):
        self.torch.cuda.synchronize(self.device)
        self.dist.barrier(group=self.group)

    def _barrier_with_status(self, err):
        """the barrier that ends a step, carrying each rank's status: if mpc_sub_end failed on ANY rank (a hand-over beyond
        that rank's n_max), every rank raises here, before any of them starts the step whose kernels would write the arrivals"""
        torch, dist = self.torch, self.dist
        torch.cuda.synchronize(self.device)
        nccl = dist.get_backend(self.group) == "nccl"
        flag = torch.tensor([1 if err is not None else 0], dtype=torch.int32, device=self.device if nccl else "cpu")
        dist.all_reduce(flag, op=dist.ReduceOp.MAX, group=self.group)
        if err is not None:
            raise err
        if int(flag.item()):
            raise MPCError("another rank's mpc_sub_end failed (hand-over beyond its n_max): the run stops on every rank")

    def _exchange(self, send_below, send_above):
        """rows of 7 columns (float32 bit patterns) to the two neighbours; returns what they sent here"""
        torch, dist = self.torch, self.dist
        below, above = slab_neighbours(self.rank, self.world)
        nccl = dist.get_backend(self.group) == "nccl"
        outs = [send_below.contiguous(), send_above.contiguous()]
        counts = torch.tensor([outs[0].shape[0], outs[1].shape[0]], dtype=torch.int64)
        allc = [torch.zeros(2, dtype=torch.int64) for _ in range(self.world)]
        if nccl:
            counts = counts.to(self.device)
            allc = [c.to(self.device) for c in allc]
        dist.all_gather(allc, counts, group=self.group)
        n_from_below, n_from_above = int(allc[below][1]), int(allc[above][0])     # what below sends up, what above sends down
        dev = self.device if nccl else "cpu"
        recv = [torch.empty((n_from_below, 7), dtype=torch.float32, device=dev), torch.empty((n_from_above, 7), dtype=torch.float32, device=dev)]
        send = [o if nccl else o.cpu() for o in outs]
        ops = []
        if self.world == 2:      # both neighbours are the same rank: two messages each way, told apart by their tags
            ops += [dist.P2POp(dist.isend, send[0], below, group=self.group, tag=1), dist.P2POp(dist.isend, send[1], above, group=self.group, tag=2)]
            ops += [dist.P2POp(dist.irecv, recv[0], below, group=self.group, tag=2), dist.P2POp(dist.irecv, recv[1], above, group=self.group, tag=1)]
        else:
            ops += [dist.P2POp(dist.isend, send[0], below, group=self.group), dist.P2POp(dist.isend, send[1], above, group=self.group)]
            ops += [dist.P2POp(dist.irecv, recv[0], below, group=self.group), dist.P2POp(dist.irecv, recv[1], above, group=self.group)]
        for w in dist.batch_isend_irecv(ops):
            w.wait()
        return [r.to(self.device) for r in recv]

    # ---- the run ----
    def set_global_state(self, st):
        """st = (x, y, z, vx, vy, vz, id) numpy arrays of the WHOLE box (every rank passes the same); keeps its own particles"""
        torch = self.torch
        sel = np.nonzero(slab_owner(st[2], self.a, self.parts) == self.rank)[0]
        self.sim.set_state(*[torch.from_numpy(np.ascontiguousarray(st[d][sel])).to(self.device) for d in range(6)],
                           id=torch.from_numpy(np.ascontiguousarray(st[6][sel].view(np.int32))).to(self.device), step=self.t)
        self.barrier()

    def migrate(self):
        """particles that have left the rank's layers go to their new owner"""
        torch = self.torch
        self._overflows += int(self.sim.observables()["n_range_overflows"])
        arrs, (n_stay, n_below, n_above) = self.sim.sub_pack()
        rows = torch.stack([a.view(torch.float32) for a in arrs], dim=1)          # (n, 7) bit patterns
        got = self._exchange(rows[n_stay:n_stay + n_below], rows[n_stay + n_below:n_stay + n_below + n_above])
        new = torch.cat([rows[:n_stay]] + got, dim=0)
        cols = [new[:, d].contiguous() for d in range(7)]
        self.sim.set_state(*cols[:6], id=cols[6].view(torch.int32), step=self.t)
        self.barrier()
        return n_below + n_above

    def step(self, nsteps, migrate_every=None):
        """advance nsteps. Particles change owner inside the reorder's kernels (the library is told how many steps follow, so
        that a reorder can fold its passes into them); migrate_every = m additionally hands them over explicitly
        (mpc_sub_pack + the process group) before every m-th step"""
        i = 0
        while i < nsteps:
            run = nsteps - i
            if migrate_every:
                if self.t > 0 and self.t % migrate_every == 0:
                    self.migrate()
                run = min(run, migrate_every - self.t % migrate_every)
            for j in range(run):
                self.sim.sub_begin(run - 1 - j)
                self.barrier()
                err = None
                try:
                    self.sim.sub_end()
                except MPCError as e:
                    err = e
                self._barrier_with_status(err)
                self.t += 1
            i += run

    def range_overflows(self):
        """events in which a particle was outside the layers this rank holds (or a velocity outside the range of the
        fixed-point sums) since the start of the run, on this rank; non-zero: the run is invalid (MPC_ERANGE)"""
        return self._overflows + int(self.sim.observables()["n_range_overflows"])

    def gather_state(self):
        """the whole box on every rank, ordered by id (tests, output): [x, y, z, vx, vy, vz, id] numpy arrays"""
        st = [t.cpu().numpy() for t in self.sim.get_state()]
        everyone = [None] * self.world
        self.dist.all_gather_object(everyone, st, group=self.group)
        cat = [np.concatenate([e[d] for e in everyone]) for d in range(7)]
        order = np.argsort(cat[6].view(np.uint32), kind="stable")
        return [c[order] for c in cat]

    def close(self):
        cudart = _cudart()
        self.barrier()
        self.sim.close()
        for base in self._opened.values():
            cudart.cudaIpcCloseMemHandle(base)
        self.barrier()
        for p in self._allocs:
            cudart.cudaFree(p)


def main():
    import torch
    import torch.distributed as dist

    from .inputs import uniform_maxwell

    ap = argparse.ArgumentParser()
    ap.add_argument("--cells", default="64,64,128")
    ap.add_argument("--nbar", type=int, default=10)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--rebin-every", type=int, default=10)
    ap.add_argument("--backend", default=None, help="default: nccl if every rank has its own GPU, else gloo")
    ap.add_argument("--one-gpu", action="store_true", help="all ranks on cuda:0 (functional test of the plumbing)")
    a = ap.parse_args()
    rank, world = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))
    local = 0 if a.one_gpu else int(os.environ.get("LOCAL_RANK", 0))
    backend = a.backend or ("gloo" if a.one_gpu else "nccl")
    torch.cuda.set_device(local)
    dist.init_process_group(backend, device_id=torch.device(f"cuda:{local}") if backend == "nccl" else None)
    cells = tuple(int(v) for v in a.cells.split(","))
    box = tuple(float(c) for c in cells)
    n = int(np.prod(cells)) * a.nbar
    st = uniform_maxwell(box, n, 1234)
    r = SlabRank(box, cells, a.nbar, 1234, (16, 16, 8), n_max=int(2.5 * n / world) + 1024, device=f"cuda:{local}", thermostat=1, rebin_every=a.rebin_every)
    r.set_global_state(st)
    r.step(a.warmup)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    r.barrier()
    e0.record(r.sim.stream)
    r.step(a.steps)
    e1.record(r.sim.stream)
    r.barrier()
    ms = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64)
    if backend == "nccl":
        ms = ms.cuda()
    dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    ob = r.sim.observables()
    tot = torch.tensor([ob["n"], ob["E_kin"], r.range_overflows()], dtype=torch.float64)
    if backend == "nccl":
        tot = tot.cuda()
    dist.all_reduce(tot)
    if rank == 0:
        print(f"slab run: {world} ranks, {int(tot[0])} particles, {a.steps} timed steps after {a.warmup}: {float(ms) / a.steps:.3f} ms per step = "
              f"{float(tot[0]) * a.steps / (float(ms) * 1e-3):.4g} particle-updates/s (device time of the slowest rank, host barriers included), "
              f"kT = {2 * float(tot[1]) / (3 * float(tot[0])):.5f}, range overflows = {int(tot[2])}")
    r.close()
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
