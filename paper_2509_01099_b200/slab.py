"""One-rank-per-GPU slab decomposition of the cavity along its slowest axis (y in 2-D, z in 3-D).

Plumbing only: it splits the coordinate array, creates the local `islbm_create_slab` handle, and moves the halo
layers between neighbouring ranks with `torch.distributed` point-to-point operations (NCCL over NVLink on GPUs).
Every step of the method runs in the kernels of libislbm.so; the per-step exchange is one layer of the planes
whose velocity has a component along the slab axis (12 of 26 in 3-D, 8 of 14 in 2-D; `islbm_halo`), and the
diagnostics are partial sums added over the ranks (`islbm_diag_sums` / `islbm_diag_from_sums`).

This module imports the CUDA binding lazily, so that the decomposition arithmetic and the exchange schedule can be
tested on CPU (gloo) with plain tensors.
"""
from __future__ import annotations

import numpy as np


def split(n: int, world: int):
    """Owned index ranges [(lo, hi)] of `n` layers over `world` ranks, as even as possible, every rank >= 1 layer."""
    if world < 1 or n < world:
        raise ValueError(f"cannot split {n} layers over {world} ranks")
    base, rem = divmod(n, world)
    out, lo = [], 0
    for r in range(world):
        hi = lo + base + (1 if r < rem else 0)
        out.append((lo, hi))
        lo = hi
    return out


def slab_inputs(coords, delta, rank: int, world: int):
    """Local coordinates (owned layers + one ghost layer at each non-wall end), the islbm_slab description, and the
    (ghost_lo, ghost_hi) counts, for `rank` of `world`."""
    coords = [np.ascontiguousarray(c, dtype=np.float64) for c in coords]
    axis = len(coords) - 1
    n = len(coords[axis])
    lo, hi = split(n, world)[rank]
    glo, ghi = (0 if rank == 0 else 1), (0 if rank == world - 1 else 1)
    local = list(coords)
    local[axis] = coords[axis][lo - glo: hi + ghi].copy()
    if len(local[axis]) < 3:
        raise ValueError(f"rank {rank}: a slab needs at least 3 layers including its ghost layers "
                         f"(got {len(local[axis])}); use fewer ranks")
    layer_nodes = 1
    for a in range(axis):
        layer_nodes *= len(coords[a])
    slab = dict(lo_is_wall=rank == 0, hi_is_wall=rank == world - 1,
                L_eff_global=float(coords[axis][-1] - coords[axis][0] + delta),
                node_offset=(lo - glo) * layer_nodes)
    return local, slab, (lo, hi), (glo, ghi)


def exchange_p2p(send_lo, recv_lo, send_hi, recv_hi, rank: int, world: int, dist=None):
    """Exchange halo layers with rank-1 (low side) and rank+1 (high side): lists of tensors, same length and order
    on every rank.  Batched isend/irecv; returns after the receives have completed on the current stream."""
    import torch.distributed as td
    dist = dist or td
    ops = []
    if rank > 0:
        ops += [dist.P2POp(dist.isend, t, rank - 1) for t in send_lo]
        ops += [dist.P2POp(dist.irecv, t, rank - 1) for t in recv_lo]
    if rank < world - 1:
        ops += [dist.P2POp(dist.isend, t, rank + 1) for t in send_hi]
        ops += [dist.P2POp(dist.irecv, t, rank + 1) for t in recv_hi]
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()


class SlabCavity:
    """The cavity of `coords` decomposed over `world` ranks; this object is rank `rank`'s slab.

    Two ways to move the halo: (default) after every step, batched isend/irecv of the halo layers
    (`exchange_p2p`); or, after `connect_ipc()` / `connect_local()`, FUSED: each rank's step kernel stores its
    boundary layers straight into the neighbour's ghost layers through peer-mapped memory (NVLink) while it emits
    them, and the only thing left between two steps is a barrier."""

    def __init__(self, coords, delta, Ra, Pr, Ma, rank, world, precision=0, device="cuda", exchange=None):
        from . import islbm
        self.rank, self.world = rank, world
        local, slab, self.own, self.ghosts = slab_inputs(coords, delta, rank, world)
        self.sim = islbm.Islbm(local, delta, Ra, Pr, Ma, precision=precision, device=device, slab=slab)
        self._exchange = exchange or self._exchange_dist
        self._fused = False
        self._peers = []          # keeps the IPC mappings of the neighbours' workspaces alive

    # -- fused halo exchange ----------------------------------------------------------------------------------
    def connect_ipc(self, host_barrier=None):
        """One process per rank on one node: map the neighbours' workspaces with CUDA IPC (torch's tensor sharing),
        hand them and the neighbours' halo layouts (ghost layers, step flags, buffer parity, step count) to the
        library, and switch to the fused exchange.  Collective over the default process group.

        From then on a step is ONE kernel per rank: boundary layers go into the neighbours' ghost layers by peer
        stores, and neighbours order their steps through flags in each other's memory (st.release.sys by the last
        boundary CTA of a step, ld.acquire.sys by the boundary CTAs of the next) — no collective between steps.
        host_barrier: order the steps on the host instead (device synchronise + barrier after every step), so that no
        kernel ever has to WAIT for another rank; required when several ranks share one GPU (kernels of different
        ranks are then not guaranteed to run at the same time: the tests), default when the backend is not NCCL."""
        import torch
        import torch.distributed as dist
        from torch.multiprocessing.reductions import reduce_tensor
        mine = dict(tensor=reduce_tensor(self.sim.workspace), lo=self.sim.halo_layout(0), hi=self.sim.halo_layout(1))
        everyone = [None] * self.world
        dist.all_gather_object(everyone, mine)
        for side, nb in ((0, self.rank - 1), (1, self.rank + 1)):
            if 0 <= nb < self.world:
                fn, args = everyone[nb]["tensor"]
                t = fn(*args)                                   # the neighbour's workspace, mapped here
                self._peers.append(t)
                self.sim.set_peer(side, t.data_ptr(), everyone[nb]["hi" if side == 0 else "lo"])
        torch.cuda.synchronize(self.sim.device)
        dist.barrier()                                          # every rank has initialised its flags before any step
        if host_barrier is None:
            host_barrier = dist.get_backend() != "nccl"
        self._fused = True
        if host_barrier:
            def barrier():
                torch.cuda.synchronize(self.sim.device)
                dist.barrier()
            self._exchange = barrier
        else:
            self._exchange = None                               # nothing between steps: islbm_step(n) runs n kernels

    # -- halo -------------------------------------------------------------------------------------------------
    def halo_views(self):
        _, s_lo, r_lo = self.sim.halo(0)
        _, s_hi, r_hi = self.sim.halo(1)
        return s_lo, r_lo, s_hi, r_hi

    def _exchange_dist(self):
        s_lo, r_lo, s_hi, r_hi = self.halo_views()
        exchange_p2p(s_lo, r_lo, s_hi, r_hi, self.rank, self.world)

    # -- the path ---------------------------------------------------------------------------------------------
    def init(self, seed=0, noise_amp=1e-3):
        self.sim.init(seed, noise_amp)          # noise is drawn by GLOBAL node index: ghost layers come out right

    def step(self, n=1):
        if self._exchange is None:              # fused exchange with device-side neighbour flags
            self.sim.step(n)
            return
        for _ in range(n):
            self.sim.step(1)
            self._exchange()

    def diagnostics(self):
        """Nu_hot, Nu_cold, Re, u2, Nu_vol, Nu_middle of the WHOLE cavity (all-reduce of 8 doubles)."""
        import torch
        import torch.distributed as dist
        s = torch.tensor(self.sim.diag_sums(), dtype=torch.float64)
        if dist.is_available() and dist.is_initialized() and self.world > 1:
            s = s.to(self.sim.device) if dist.get_backend() == "nccl" else s
            dist.all_reduce(s, op=dist.ReduceOp.SUM)
        return self.sim.diag_from_sums(s.tolist())

    def owned(self, t):
        """Strip the ghost layers from a local field / population tensor ([..., layers, ...rest])."""
        glo, ghi = self.ghosts
        axis = -2 if self.sim.dim == 2 else -3
        n = t.shape[axis]
        return t.narrow(axis, glo, n - glo - ghi)

    def close(self):
        self.sim.close()


def connect_local(slabs):
    """Fused halo exchange among slabs that live in ONE process on ONE device: each handle gets its neighbours'
    workspaces as peers.  The slabs must be stepped ONE STEP AT A TIME in turn on the shared stream (as the tests do):
    then every neighbour flag is already set when a kernel starts and no kernel ever waits."""
    for a in range(len(slabs) - 1):
        lower, upper = slabs[a].sim, slabs[a + 1].sim
        lo_layout, up_layout = lower.halo_layout(1), upper.halo_layout(0)
        lower.set_peer(1, upper.workspace.data_ptr(), up_layout)
        upper.set_peer(0, lower.workspace.data_ptr(), lo_layout)
    for s in slabs:
        s._fused = True
        s._exchange = lambda: None


def exchange_local(slabs):
    """Halo exchange among slabs that live in ONE process on ONE device (tests, single-GPU runs): direct copies."""
    views = [s.halo_views() for s in slabs]
    for a in range(len(slabs) - 1):
        _, _, s_hi, r_hi = views[a]
        s_lo, r_lo, _, _ = views[a + 1]
        for p in range(len(s_hi)):
            r_lo[p].copy_(s_hi[p])
            r_hi[p].copy_(s_lo[p])
