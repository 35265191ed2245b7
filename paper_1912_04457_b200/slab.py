"""Slab decomposition of a periodic spatial domain over ranks: one process per GPU, the domain split
along z, ONE halo exchange per Euler step.

Why this is the whole multi-GPU story of the path: the collision term is local in x (Eq. 5 has a single x), so
every kinematic sample, |M|^2, bracket and deposit of a spatial cell stays on the rank that owns the cell; only the
drift stencil of Eq. 13 reads a neighbouring cell, and first-order upwind reads exactly one cell away.
Each rank therefore keeps nz_local own z layers plus one halo layer below and one above; before a step it sends its
lowest own layer down and its highest own layer up (two contiguous blocks of f: a z layer is contiguous in the layout
f[xcell][species][pcell]) and receives the neighbours' into its halo layers.  The totals of bz_moments are summed with
one all-reduce of 2*S doubles.  Results are those of the undecomposed domain: the Philox spatial counter of a cell is
its global index (bz_set_slab), so every cell draws the same samples on any number of ranks.

This module holds only host logic (who sends which layer to whom); every step of the path runs in libbz.so through
`paper_1912_04457_b200.bz.Boltzmann`, the "engine".  The engine is duck-typed (set_slab, get_layers, set_layers,
step, moments, layer_values) so that the exchange logic is covered on CPU by world_size-2 gloo tests that plug the
oracle in (tests/test_slab_gloo.py); there is no CPU engine in this package.
"""
import contextlib

import torch
import torch.distributed as dist


def slab_range(nz_global, rank, world):
    """Own z layers [z0, z1) of `rank`: a balanced split, the first nz_global % world ranks get one layer more."""
    if not (0 <= rank < world) or nz_global < world:
        raise ValueError("need 0 <= rank < world <= nz_global")
    base, extra = divmod(nz_global, world)
    z0 = rank * base + min(rank, extra)
    return z0, z0 + base + (1 if rank < extra else 0)


class SlabDomain:
    """The slab of `rank` of a periodic nx x ny x nz_global domain.

    make_engine(nz_with_halo) must return an engine on an nx x ny x nz_with_halo grid; layer 0 and layer
    nz_with_halo - 1 are the halo layers, layers 1 .. nz_local the slab's own."""

    def __init__(self, make_engine, nx, ny, nz_global, rank=0, world=1, group=None):
        self.nx, self.ny, self.nz_global, self.rank, self.world, self.group = nx, ny, nz_global, rank, world, group
        self.z0, self.z1 = slab_range(nz_global, rank, world)
        self.nz_local = self.z1 - self.z0
        self.engine = make_engine(self.nz_local + 2)
        layer_cells = nx * ny
        # local cell x (halo layer included) is global cell x + (z0 - 1) * layer_cells; the Philox counter is 32 bits wide
        self.engine.set_slab(((self.z0 - 1) * layer_cells) & 0xFFFFFFFF, 1, self.nz_local + 1)
        self.down = (rank - 1) % world
        self.up = (rank + 1) % world
        self._recv_lo = self._recv_hi = None
        self._stage_lo = self._stage_hi = None

    # ---- state
    def set_own(self, f_own):
        """f_own: tensor with the slab's own layers [nz_local * nx * ny, S, Np] on the engine's device."""
        self.engine.set_layers(1, self.nz_local, f_own.reshape(-1))

    def get_own(self):
        return self.engine.get_layers(1, self.nz_local)

    # ---- the exchange step
    def exchange_halos(self):
        """Refresh both halo layers from the neighbours' boundary layers (periodic in z)."""
        e = self.engine
        lo = e.get_layers(1, 1)                     # lowest own layer  -> the lower neighbour's upper halo
        hi = e.get_layers(self.nz_local, 1)         # highest own layer -> the upper neighbour's lower halo
        self._exchange(lo, hi)

    def _on_engine_stream(self):
        """Context manager: makes the engine's CUDA stream torch's current stream (a no-op for a host engine).  bz_copy_layers
        enqueues on the engine's stream, while torch's copies and the process group's send/recv order themselves against the
        CURRENT stream: with the two made one, every producer and consumer of the boundary layers is on a single stream."""
        s = getattr(self.engine, "torch_stream", None)
        return torch.cuda.stream(s) if s is not None else contextlib.nullcontext()

    def _exchange(self, lo, hi):
        """lo / hi: this rank's lowest / highest own layer as flat tensors on the engine's device, produced on the
        engine's stream.  They go to the lower / upper neighbour; what comes back fills the two halo layers."""
        e = self.engine
        if self.world == 1:
            e.set_layers(self.nz_local + 1, 1, lo)
            e.set_layers(0, 1, hi)
            return
        if self._recv_lo is None:
            self._recv_lo, self._recv_hi = torch.empty_like(lo), torch.empty_like(hi)
        with self._on_engine_stream():
            # NCCL's send/recv kernels run on the process group's own stream, which waits for the current torch stream (here
            # the engine's: lo and hi are complete before they are sent), and req.wait() makes the current stream (again the
            # engine's) wait for the transfer, so that the halo copies below, which bz_copy_layers enqueues on the engine's
            # stream, read the receive buffers after they have landed.
            # Message order between a pair of ranks is the same on both sides (down-going first, tag 0; up-going second,
            # tag 1), which is what NCCL matches by (it ignores tags) and gloo matches by tag; with two ranks both
            # neighbours are the same peer.
            ops = [dist.P2POp(dist.isend, lo, self.down, self.group, 0),
                   dist.P2POp(dist.isend, hi, self.up, self.group, 1),
                   dist.P2POp(dist.irecv, self._recv_hi, self.up, self.group, 0),
                   dist.P2POp(dist.irecv, self._recv_lo, self.down, self.group, 1)]
            for req in dist.batch_isend_irecv(ops):
                req.wait()
            if lo.is_cuda:
                # This branch has not run on two or more GPUs yet (no multi-GPU box in the build): until it has, the host
                # also waits for the transfer, so that the result does not hang on the stream reasoning above alone.
                torch.cuda.current_stream(lo.device).synchronize()
            e.set_layers(self.nz_local + 1, 1, self._recv_hi)
            e.set_layers(0, 1, self._recv_lo)

    # ---- the path
    def step(self, dt):
        """One Euler step of the whole domain's share on this rank: halo exchange, then bz_step."""
        self.exchange_halos()
        self.engine.step(dt)

    def step_host(self, dt, f_in_host, f_out_host):
        """The same step end to end from HOST memory (pinned): f_in_host / f_out_host have the size of the whole local
        context (nz_local + 2 layers), of which only the own layers 1 .. nz_local are read / written.  The two boundary
        layers go to the device first and are exchanged with the neighbours; bz_step_host then pipelines the own layers
        (host-to-device copy, collision, stream + Euler, device-to-host copy by chunks of z layers).  The exchange is NOT
        overlapped with that pipeline: its copy streams start behind the halo copies on the engine's stream (two layers
        over NVLink, a fraction of a millisecond per step)."""
        e = self.engine
        lv = e.layer_values()
        flat = f_in_host.reshape(-1)
        if self._stage_lo is None:
            self._stage_lo = torch.empty(lv, dtype=torch.float64, device=e.device)
            self._stage_hi = torch.empty(lv, dtype=torch.float64, device=e.device)
        with self._on_engine_stream():              # the staging copies are consumed on the engine's stream (set_layers, send)
            self._stage_lo.copy_(flat[lv:2 * lv], non_blocking=True)
            self._stage_hi.copy_(flat[self.nz_local * lv:(self.nz_local + 1) * lv], non_blocking=True)
        self._exchange(self._stage_lo, self._stage_hi)
        e.step_host(dt, f_in_host, f_out_host)

    def moments_totals(self):
        """[S, 2] totals (N_a, E_a) over the WHOLE domain: the local totals (own layers only) all-reduced."""
        tot = self.engine.moments()["tot"].clone()
        if self.world > 1:
            t = tot.to(self.engine.device)                  # NCCL reduces device tensors, gloo host tensors
            dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.group)
            tot = t.cpu()
        return tot


def exchange_in_process(slabs):
    """The same halo refresh for slabs that live in ONE process (rank order, periodic): used to run several slabs
    back to back on one GPU, e.g. to check the decomposition against the undecomposed domain on a 1-GPU box."""
    n = len(slabs)
    los = [s.engine.get_layers(1, 1) for s in slabs]
    his = [s.engine.get_layers(s.nz_local, 1) for s in slabs]
    for r, s in enumerate(slabs):
        s.engine.set_layers(s.nz_local + 1, 1, los[(r + 1) % n])
        s.engine.set_layers(0, 1, his[(r - 1) % n])
