"""z-slab domain decomposition with overlapped halo exchange.

Host-side orchestration only.  Every slab is one context of the CUDA library whose z faces towards its neighbours are
`BC_HALO`; all arithmetic runs in the library's kernels through the staged C-ABI calls (include/streams.h):

    step_begin | MAX of red[2] | for each stage: swap halos, stage_rhs(interior) while the swap is in flight,
    stage_rhs(boundary), SUM of red[0..1] (forcing), swap of the node-flag words (hybrid switch), stage_end
    (forcing AND hybrid switch: flag swap, stage_mid, SUM, stage_end).

The messages move by `torch.distributed` point-to-point operations between processes (NCCL on GPUs, one process per
GPU) and by device-to-device copies between slabs of the same process.

A "slab" is duck-typed (binding.Streams provides it): `halo_pack(face, out, stream)`, `halo_unpack(face, buf, stream)`,
`step_begin()`, `stage_rhs(stage, part)`, `stage_end(stage)`, `red`, `stream`, `halo_shape()`, `new_buffer()` (and
`flag_halo_pack/unpack`, `new_flag_buffer()` with the hybrid switch); the
stream handling is delegated to a small `Sync` object so that the CPU (gloo) tests can run the same logic on NumPy /
CPU-tensor slabs.
"""
from dataclasses import dataclass

import numpy as np

FACE_ZMIN, FACE_ZMAX = 4, 5
PART_ALL, PART_INTERIOR, PART_BOUNDARY = 0, 1, 2
BC_PERIODIC, BC_HALO = 0, 8


# ---- partition (pure host logic) ------------------------------------------------------------------------------------
def slab_range(nz: int, nslabs: int, index: int):
    """Planes [k0, k1) of slab `index` when nz planes are split into nslabs contiguous slabs (sizes differ by <= 1)."""
    if not (0 <= index < nslabs) or nslabs < 1 or nz < nslabs:
        raise ValueError("bad slab partition")
    base, rem = divmod(nz, nslabs)
    k0 = index * base + min(index, rem)
    return k0, k0 + base + (1 if index < rem else 0)


def neighbours(index: int, nslabs: int, periodic: bool):
    """(lower, upper) slab index across the zmin / zmax face, None at a physical (non-periodic) boundary."""
    lo = index - 1 if index > 0 else (nslabs - 1 if periodic else None)
    hi = index + 1 if index < nslabs - 1 else (0 if periodic else None)
    return lo, hi


@dataclass
class SlabSpec:
    """What streams_create needs for one slab of a global grid."""
    grid: dict
    z: np.ndarray          # node coordinates incl. the three ghost coordinates on every HALO face (include/streams.h)
    params: dict
    k0: int
    k1: int
    lower: object          # neighbour slab index or None
    upper: object


def slab_spec(grid: dict, z, params: dict, nslabs: int, index: int) -> SlabSpec:
    """Grid, coordinates and parameters of slab `index`: internal z faces become BC_HALO; the ghost coordinates are the
    neighbour's nodes (shifted by the period across the periodic seam)."""
    nz = int(grid["nz"])
    z = np.asarray(z, dtype=np.float64)
    k0, k1 = slab_range(nz, nslabs, index)
    if k1 - k0 < 4:
        raise ValueError("a z-slab needs at least 4 planes")
    periodic = params["bc"][4] == BC_PERIODIC
    if periodic != (params["bc"][5] == BC_PERIODIC):
        raise ValueError("periodic must be set on both z faces")
    lo, hi = neighbours(index, nslabs, periodic)
    Lz = grid["len"][2]

    def coord(k):
        return z[k % nz] + Lz * (k // nz) if periodic else z[k]

    p = dict(params)
    bc = list(params["bc"])
    parts = []
    if lo is not None:
        bc[4] = BC_HALO
        parts.append(np.array([coord(k) for k in range(k0 - 3, k0)]))
    parts.append(z[k0:k1])
    if hi is not None:
        bc[5] = BC_HALO
        parts.append(np.array([coord(k) for k in range(k1, k1 + 3)]))
    p["bc"] = bc
    g = dict(grid)
    g["nz"] = k1 - k0
    g["len"] = list(grid["len"])
    return SlabSpec(g, np.concatenate(parts), p, k0, k1, lo, hi)


# ---- stream handling ------------------------------------------------------------------------------------------------
class CudaSync:
    """Events between the context stream and the communication stream of one slab."""

    def __init__(self, torch, slab):
        self.torch = torch
        self.main = slab.stream
        self.comm = torch.cuda.Stream(device=slab.device)

    def main_done(self):
        return self.main.record_event()

    def comm_done(self):
        return self.comm.record_event()

    def comm_wait(self, ev):
        if ev is not None:
            self.comm.wait_event(ev)

    def main_wait(self, ev):
        if ev is not None:
            self.main.wait_event(ev)

    def on_comm(self):
        return self.torch.cuda.stream(self.comm)

    def on_main(self):
        return self.torch.cuda.stream(self.main)


class NoSync:
    """CPU slabs (tests of the host logic): everything is synchronous."""
    comm = None

    class _Null:
        def __enter__(self):
            return self

        def __exit__(self, *a):
            return False

    def main_done(self):
        return None

    comm_done = main_done

    def comm_wait(self, ev):
        pass

    main_wait = comm_wait

    def on_comm(self):
        return self._Null()

    on_main = on_comm


# ---- reductions across slabs ----------------------------------------------------------------------------------------
class DistReducer:
    """red[0..1] summed / red[2] maximised over the processes of a torch.distributed group, in place on the context
    stream (one slab per process)."""

    def __init__(self, dist, group=None):
        self.dist, self.group = dist, group

    def sum(self, slabs, syncs):
        assert len(slabs) == 1, "DistReducer: one slab per process"
        with syncs[0].on_main():
            self.dist.all_reduce(slabs[0].red[0:2], op=self.dist.ReduceOp.SUM, group=self.group)

    def max(self, slabs, syncs):
        assert len(slabs) == 1, "DistReducer: one slab per process"
        with syncs[0].on_main():
            self.dist.all_reduce(slabs[0].red[2:3], op=self.dist.ReduceOp.MAX, group=self.group)


# ---- the stepping loop ----------------------------------------------------------------------------------------------
class SlabGroup:
    """The slabs this process owns (consecutive in z) of a domain cut into `nslabs` slabs, stepped in lockstep.

    slabs[i] is global slab  rank * len(slabs) + i.  `dist` (torch.distributed, initialised) moves the messages of the
    first / last local slab to the neighbouring processes; without it the group must hold every slab (a periodic seam
    is then a local copy).  `reducer` combines the partial reductions (DistReducer, or a test's own)."""

    def __init__(self, slabs, nslabs, rank=0, periodic=True, dist=None, group=None, reducer=None, syncs=None,
                 forcing=False, cfl_dt=True, overlap=True, weno=False):
        self.slabs = list(slabs)
        K = len(self.slabs)
        if K < 1 or nslabs % K:
            raise ValueError("every process holds the same number of slabs")
        self.nslabs, self.rank, self.periodic = nslabs, rank, periodic
        self.world = nslabs // K
        self.dist, self.group = dist, group
        if dist is None and self.world != 1:
            raise ValueError("several processes need torch.distributed")
        self.reducer = reducer if reducer is not None else (DistReducer(dist, group) if dist is not None else None)
        self.forcing, self.cfl_dt, self.overlap = bool(forcing), bool(cfl_dt), bool(overlap)
        # one slab without torch.distributed has nothing to combine; with it the collectives run even for one process
        self.combine = self.reducer is not None and (nslabs > 1 or dist is not None)
        if syncs is None:
            import torch
            syncs = [CudaSync(torch, s) for s in self.slabs]
        self.syncs = syncs
        self.first = rank * K
        self.nb = [neighbours(self.first + i, nslabs, periodic) for i in range(K)]
        # send buffers [face][i] and receive buffers for messages that cross the process boundary
        self.sbuf = {f: [s.new_buffer() for s in self.slabs] for f in (FACE_ZMIN, FACE_ZMAX)}
        self.rbuf = {FACE_ZMIN: self.slabs[0].new_buffer(), FACE_ZMAX: self.slabs[-1].new_buffer()}
        self._consumed = [[] for _ in range(K)]      # events of the unpacks that read slab i's send buffers
        self.weno = bool(weno)
        if self.weno:                                # node-flag words of the hybrid switch: a second, small message per face
            self.fsbuf = {f: [s.new_flag_buffer() for s in self.slabs] for f in (FACE_ZMIN, FACE_ZMAX)}
            self.frbuf = {FACE_ZMIN: self.slabs[0].new_flag_buffer(), FACE_ZMAX: self.slabs[-1].new_flag_buffer()}
        self.messages_sent = 0                       # bench / test accounting (messages that left a slab)

    # -- helpers
    def _local(self, g):
        """Local index of global slab g, or None if another process owns it."""
        i = g - self.first
        return i if 0 <= i < len(self.slabs) else None

    def _owner(self, g):
        return g // len(self.slabs)

    def swap_halos(self):
        """Pack, move and unpack the ghost planes of the current state of every local slab; returns one event per
        slab after which its ghost planes are in place (None on CPU)."""
        return self._swap("halo_pack", "halo_unpack", self.sbuf, self.rbuf)

    def swap_flags(self):
        """The same for the node-flag words of the hybrid switch (between stage_rhs and stage_end); the context
        streams wait for it."""
        for i, ev in enumerate(self._swap("flag_halo_pack", "flag_halo_unpack", self.fsbuf, self.frbuf)):
            self.syncs[i].main_wait(ev)

    def _swap(self, pack, unpack, sbuf, rbuf):
        K = len(self.slabs)
        sy = self.syncs
        packed = []
        for i, s in enumerate(self.slabs):
            sy[i].comm_wait(sy[i].main_done())                 # the state of the previous stage is final
            for ev in self._consumed[i]:
                sy[i].comm_wait(ev)                            # last swap's readers of the send buffers are done
            self._consumed[i] = []
            lo, hi = self.nb[i]
            if lo is not None:
                getattr(s, pack)(FACE_ZMIN, sbuf[FACE_ZMIN][i], stream=sy[i].comm)
            if hi is not None:
                getattr(s, pack)(FACE_ZMAX, sbuf[FACE_ZMAX][i], stream=sy[i].comm)
            packed.append(sy[i].comm_done())
        # messages between slabs of this process (incl. the periodic seam when this process holds every slab)
        via_dist = self.dist is not None and (self.world > 1 or K == 1)
        remote = {}                                            # face -> local slab whose message crosses the process boundary
        for i, s in enumerate(self.slabs):
            lo, hi = self.nb[i]
            for face, g, src_face in ((FACE_ZMIN, lo, FACE_ZMAX), (FACE_ZMAX, hi, FACE_ZMIN)):
                if g is None:
                    continue
                j = self._local(g)
                crosses = via_dist and ((face == FACE_ZMIN and i == 0) or (face == FACE_ZMAX and i == K - 1))
                if j is not None and not crosses:
                    sy[i].comm_wait(packed[j])
                    getattr(s, unpack)(face, sbuf[src_face][j], stream=sy[i].comm)
                    self._consumed[j].append(sy[i].comm_done())
                    self.messages_sent += 1
                else:
                    remote[face] = (i, self._owner(g))
        # Messages across the process boundary (torch.distributed point-to-point; NCCL on GPUs).  Every process posts its
        # sends in the order (zmax message, zmin message) and its receives in the order (through zmin, through zmax): the
        # message a slab sends upwards is what its upper neighbour receives through its zmin face, so two messages
        # between the same pair of processes (two processes or one, periodic) match in order.
        if remote:
            dist = self.dist
            with sy[0].on_comm():
                for face, (i, peer) in remote.items():
                    if i != 0:
                        sy[0].comm_wait(packed[i])
                p2p = []
                for face in (FACE_ZMAX, FACE_ZMIN):
                    if face in remote:
                        i, peer = remote[face]
                        p2p.append(dist.P2POp(dist.isend, sbuf[face][i], peer, group=self.group))
                for face in (FACE_ZMIN, FACE_ZMAX):
                    if face in remote:
                        i, peer = remote[face]
                        p2p.append(dist.P2POp(dist.irecv, rbuf[face], peer, group=self.group))
                for w in dist.batch_isend_irecv(p2p):
                    w.wait()
                self.messages_sent += len(remote)
                done = sy[0].comm_done()
            for face, (i, peer) in remote.items():
                sy[i].comm_wait(done)
                getattr(self.slabs[i], unpack)(face, rbuf[face], stream=sy[i].comm)
        return [sy[i].comm_done() for i in range(K)]

    def step(self, nsteps=1):
        sl, sy = self.slabs, self.syncs
        for _ in range(nsteps):
            for s in sl:
                s.step_begin()
            if self.cfl_dt and self.combine:
                self.reducer.max(sl, sy)
            for stage in range(3):
                halo_ready = self.swap_halos()
                if self.overlap:
                    for s in sl:
                        s.stage_rhs(stage, PART_INTERIOR)       # runs while the halos move
                for i, s in enumerate(sl):
                    sy[i].main_wait(halo_ready[i])
                    s.stage_rhs(stage, PART_BOUNDARY if self.overlap else PART_ALL)
                if self.forcing and self.weno:
                    # the body force is the sum of the residual AFTER its WENO correction, which needs the neighbours' flags
                    self.swap_flags()
                    for s in sl:
                        s.stage_mid(stage)
                    if self.combine:
                        self.reducer.sum(sl, sy)
                else:
                    if self.forcing and self.combine:
                        self.reducer.sum(sl, sy)
                    if self.weno:
                        self.swap_flags()
                for s in sl:
                    s.stage_end(stage)

    def residual_ready(self):
        """Ghost planes of the current state in place on every local slab (for streams_rhs on slabs)."""
        for i, ev in enumerate(self.swap_halos()):
            self.syncs[i].main_wait(ev)
