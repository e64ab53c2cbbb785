"""Host logic of the z-slab decomposition (paper_2004_02276_b200/slab.py) on CPU: partition, neighbour and ghost-coordinate
rules, and the lockstep stepping loop with its halo swap and reductions -- in one process (three slabs, local copies) and
across two gloo ranks (torch.distributed point-to-point + all-reduce).  The slabs here are stand-ins with a toy update that
needs exactly what the real contexts need (three ghost planes per face before every stage, a global sum every stage, a
global maximum every step), so a wrong neighbour, message order, face or reduction changes the result."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2004_02276_b200 import slab

NY, NX = 3, 4
COEF = np.array([0.03, -0.1, 0.25, 0.0, -0.2, 0.12, -0.05])       # asymmetric: lower and upper ghosts are not interchangeable


class ToySlab:
    """q[7][nz + 6][NY][NX]; stage: r_k = sum_m COEF[m] q_{k-3+m} (field 0), state += dt (r - mean r) scaled per stage."""
    device = "cpu"
    stream = None

    def __init__(self, q_int, lower, upper):
        self.nz = q_int.shape[1]
        self.q = np.zeros((7, self.nz + 6, NY, NX))
        self.q[:, 3:-3] = q_int
        self.q[:, :3] = np.nan
        self.q[:, -3:] = np.nan
        self.has = (lower is not None, upper is not None)
        self.red = torch.zeros(4, dtype=torch.float64)
        self.log = []

    def halo_shape(self):
        return (7, 3, NY, NX)

    def new_buffer(self):
        return torch.full(self.halo_shape(), float("nan"), dtype=torch.float64)

    def halo_pack(self, face, out, stream=None):
        src = self.q[:, 3:6] if face == slab.FACE_ZMIN else self.q[:, -6:-3]
        out.copy_(torch.from_numpy(np.ascontiguousarray(src)))
        self.log.append(("pack", face))

    def halo_unpack(self, face, buf, stream=None):
        if face == slab.FACE_ZMIN:
            self.q[:, :3] = buf.numpy()
        else:
            self.q[:, -3:] = buf.numpy()
        self.log.append(("unpack", face))

    def interior(self):
        return self.q[:, 3:-3]

    def step_begin(self):
        self.red[2] = float(np.abs(self.interior()).max())
        self.log.append(("begin",))

    def stage_rhs(self, stage, part):
        self.log.append(("rhs", stage, part))
        if part == slab.PART_INTERIOR:
            return
        if stage == 0:
            self.dt = 0.1 / float(self.red[2])
        ext = self.q.copy()
        if not self.has[0]:
            ext[:, :3] = ext[:, 3:4]
        if not self.has[1]:
            ext[:, -3:] = ext[:, -4:-3]
        assert np.isfinite(ext).all(), "ghost planes were not in place"
        self.r = sum(COEF[m] * ext[:, m:m + self.nz] for m in range(7))
        self.red[0] = float(self.r[0].sum())
        self.red[1] = float(self.r[0].size)
        self.q[:, :3] = np.nan                      # ghosts are stale after the update
        self.q[:, -3:] = np.nan

    def stage_end(self, stage):
        mean = float(self.red[0]) / float(self.red[1])
        self.q[:, 3:-3] += self.dt * (stage + 1) * (self.r - mean)
        self.log.append(("end", stage))


def toy_reference(q, periodic, nsteps):
    q = q.copy()
    nz = q.shape[1]
    for _ in range(nsteps):
        dt = 0.1 / np.abs(q).max()
        for stage in range(3):
            if periodic:
                ext = np.concatenate([q[:, -3:], q, q[:, :3]], axis=1)
            else:
                ext = np.concatenate([q[:, :1]] * 3 + [q] + [q[:, -1:]] * 3, axis=1)
            r = sum(COEF[m] * ext[:, m:m + nz] for m in range(7))
            q = q + dt * (stage + 1) * (r - r[0].sum() / r[0].size)
    return q


class LocalReducer:
    def sum(self, slabs, syncs):
        tot = sum(s.red[0:2].clone() for s in slabs)
        for s in slabs:
            s.red[0:2] = tot

    def max(self, slabs, syncs):
        m = max(float(s.red[2]) for s in slabs)
        for s in slabs:
            s.red[2] = m


def field(nz, seed=3):
    return np.random.default_rng(seed).uniform(0.5, 1.5, size=(7, nz, NY, NX))


def test_partition_and_neighbours():
    assert [slab.slab_range(10, 3, i) for i in range(3)] == [(0, 4), (4, 7), (7, 10)]
    assert slab.slab_range(512, 4, 3) == (384, 512)
    with pytest.raises(ValueError):
        slab.slab_range(2, 3, 0)
    assert slab.neighbours(0, 4, True) == (3, 1) and slab.neighbours(3, 4, True) == (2, 0)
    assert slab.neighbours(0, 4, False) == (None, 1) and slab.neighbours(3, 4, False) == (2, None)
    assert slab.neighbours(0, 1, True) == (0, 0) and slab.neighbours(0, 1, False) == (None, None)


def test_slab_spec_ghost_coordinates_and_faces():
    nz, Lz = 24, 6.0
    z = Lz * np.arange(nz) / nz + 0.125
    grid = dict(nx=8, ny=8, nz=nz, len=[1.0, 1.0, Lz])
    per = dict(bc=[0, 0, 1, 1, 0, 0])
    s0, s1, s2 = (slab.slab_spec(grid, z, per, 3, i) for i in range(3))
    assert s0.params["bc"][4:] == [8, 8] and s1.params["bc"][4:] == [8, 8] and per["bc"][4:] == [0, 0]
    assert (s0.k0, s0.k1, s1.k0, s2.k1) == (0, 8, 8, 24) and s1.grid["nz"] == 8 and grid["nz"] == 24
    assert np.array_equal(s1.z, z[5:19])                                   # neighbours' nodes on both sides
    assert np.array_equal(s0.z[:3], z[-3:] - Lz) and np.array_equal(s2.z[-3:], z[:3] + Lz)   # periodic seam: shifted by the period
    assert (s0.lower, s0.upper, s2.upper) == (2, 1, 0)
    wall = dict(bc=[0, 0, 1, 1, 6, 6])
    t0, t2 = slab.slab_spec(grid, z, wall, 3, 0), slab.slab_spec(grid, z, wall, 3, 2)
    assert t0.params["bc"][4:] == [6, 8] and t2.params["bc"][4:] == [8, 6]
    assert len(t0.z) == 8 + 3 and np.array_equal(t0.z, z[:11]) and np.array_equal(t2.z, z[13:])
    with pytest.raises(ValueError):
        slab.slab_spec(grid, z, per, 8, 0)                                  # 3 planes per slab: too thin


@pytest.mark.parametrize("periodic,overlap", [(True, True), (True, False), (False, True)])
def test_three_local_slabs_follow_the_undivided_toy(periodic, overlap):
    nz, nsl = 30, 3
    q0 = field(nz)
    slabs = []
    for i in range(nsl):
        k0, k1 = slab.slab_range(nz, nsl, i)
        lo, hi = slab.neighbours(i, nsl, periodic)
        slabs.append(ToySlab(q0[:, k0:k1], lo, hi))
    grp = slab.SlabGroup(slabs, nsl, periodic=periodic, reducer=LocalReducer(), syncs=[slab.NoSync() for _ in slabs],
                         forcing=True, cfl_dt=True, overlap=overlap)
    grp.step(2)
    got = np.concatenate([s.interior() for s in slabs], axis=1)
    ref = toy_reference(q0, periodic, 2)
    assert np.abs(got - ref).max() < 1e-13
    # call order of one slab: begin, then per stage swap (packs before unpacks), rhs part(s), end
    log = slabs[1].log
    per_stage = 2 + 2 + (2 if overlap else 1) + 1
    assert log[0] == ("begin",) and len(log) == 2 * (1 + 3 * per_stage)
    st0 = log[1:1 + per_stage]
    assert [e[0] for e in st0[:4]] == ["pack", "pack", "unpack", "unpack"]
    assert st0[4:] == ([("rhs", 0, slab.PART_INTERIOR), ("rhs", 0, slab.PART_BOUNDARY)] if overlap else [("rhs", 0, slab.PART_ALL)]) + [("end", 0)]
    assert grp.messages_sent == 2 * 3 * (2 * nsl if periodic else 2 * nsl - 2)


def _worker(rank, world, port, periodic, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    nz = 16
    q0 = field(nz, seed=11)
    k0, k1 = slab.slab_range(nz, world, rank)
    lo, hi = slab.neighbours(rank, world, periodic)
    s = ToySlab(q0[:, k0:k1], lo, hi)
    grp = slab.SlabGroup([s], world, rank=rank, periodic=periodic, dist=dist, syncs=[slab.NoSync()], forcing=True, cfl_dt=True)
    grp.step(2)
    ref = toy_reference(q0, periodic, 2)[:, k0:k1]
    q.put((rank, float(np.abs(s.interior() - ref).max()), grp.messages_sent))
    dist.destroy_process_group()


@pytest.mark.parametrize("periodic", [True, False])
def test_two_gloo_ranks_exchange_and_reduce(periodic):
    """world_size 2: with a periodic z both messages of a rank go to the SAME peer, so the send / receive order matters."""
    sk = socket.socket()
    sk.bind(("127.0.0.1", 0))
    port = sk.getsockname()[1]
    sk.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, periodic, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, err, sent in res:
        assert err < 1e-13, (rank, err)
        assert sent == 2 * 3 * (2 if periodic else 1)


# ---- forcing together with the hybrid switch: flag swap | stage_mid | SUM | stage_end (include/streams.h) --------------
class ToyFlagSlab(ToySlab):
    """The toy with node flags (r > 0 of field 0) whose neighbours' values enter a correction of r (a 7-plane window
    of flags, like the interface flags of the hybrid switch) BEFORE r is summed: the sum left by stage_rhs is poison."""

    def flag_shape(self):
        return (3, NY, NX)

    def new_flag_buffer(self):
        return torch.full(self.flag_shape(), -7, dtype=torch.int32)

    def stage_rhs(self, stage, part):
        super().stage_rhs(stage, part)
        if part == slab.PART_INTERIOR:
            return
        self.flag = (self.r[0] > 0).astype(np.int32) * (1 + np.arange(self.nz)[:, None, None] % 3)
        self.fl = [None, None]
        self.red[0] = float("nan")                  # only stage_mid knows the sum
        self.mid = False

    def flag_halo_pack(self, face, out, stream=None):
        out.copy_(torch.from_numpy(np.ascontiguousarray(self.flag[:3] if face == slab.FACE_ZMIN else self.flag[-3:])))
        self.log.append(("fpack", face))

    def flag_halo_unpack(self, face, buf, stream=None):
        self.fl[0 if face == slab.FACE_ZMIN else 1] = buf.numpy().copy()
        self.log.append(("funpack", face))

    def stage_mid(self, stage):
        lo = self.fl[0] if self.has[0] else np.repeat(self.flag[:1], 3, axis=0)
        hi = self.fl[1] if self.has[1] else np.repeat(self.flag[-1:], 3, axis=0)
        assert lo is not None and hi is not None and (lo >= 0).all() and (hi >= 0).all(), "flag words were not in place"
        ext = np.concatenate([lo, self.flag, hi], axis=0)
        self.r = self.r + 0.01 * sum((m + 1) * ext[m:m + self.nz] for m in range(7))[None]
        self.red[0] = float(self.r[0].sum())
        self.red[1] = float(self.r[0].size)
        self.mid = True
        self.log.append(("mid", stage))

    def stage_end(self, stage):
        assert self.mid, "stage_end before stage_mid"
        super().stage_end(stage)


def toy_flag_reference(q, periodic, nsteps):
    q = q.copy()
    nz = q.shape[1]
    for _ in range(nsteps):
        dt = 0.1 / np.abs(q).max()
        for stage in range(3):
            pad = (lambda a: np.concatenate([a[-3:], a, a[:3]], axis=0)) if periodic else \
                  (lambda a: np.concatenate([a[:1]] * 3 + [a] + [a[-1:]] * 3, axis=0))
            ext = np.stack([pad(q[v]) for v in range(7)])
            r = sum(COEF[m] * ext[:, m:m + nz] for m in range(7))
            # the flag multiplier is the plane index inside the OWNING slab; the test cuts nz into equal slabs of `per` planes
            flag = (r[0] > 0).astype(np.int32) * (1 + (np.arange(nz) % toy_flag_reference.per)[:, None, None] % 3)
            fe = pad(flag)
            r = r + 0.01 * sum((m + 1) * fe[m:m + nz] for m in range(7))[None]
            q = q + dt * (stage + 1) * (r - r[0].sum() / r[0].size)
    return q


@pytest.mark.parametrize("periodic", [True, False])
def test_three_local_slabs_with_flags_and_forcing(periodic):
    nz, nsl = 30, 3
    toy_flag_reference.per = nz // nsl
    q0 = field(nz, seed=5) - 1.0                   # both signs: the flags are not all equal
    slabs = []
    for i in range(nsl):
        k0, k1 = slab.slab_range(nz, nsl, i)
        lo, hi = slab.neighbours(i, nsl, periodic)
        slabs.append(ToyFlagSlab(q0[:, k0:k1], lo, hi))
    grp = slab.SlabGroup(slabs, nsl, periodic=periodic, reducer=LocalReducer(), syncs=[slab.NoSync() for _ in slabs],
                         forcing=True, cfl_dt=True, overlap=True, weno=True)
    grp.step(2)
    got = np.concatenate([s.interior() for s in slabs], axis=1)
    ref = toy_flag_reference(q0, periodic, 2)
    assert np.abs(got - ref).max() < 1e-13
    names = [e[0] for e in slabs[1].log[1:13]]      # first stage of the middle slab
    assert names == ["pack", "pack", "unpack", "unpack", "rhs", "rhs", "fpack", "fpack", "funpack", "funpack", "mid", "end"]


def _flag_worker(rank, world, port, periodic, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    nz = 16
    toy_flag_reference.per = nz // world
    q0 = field(nz, seed=13) - 1.0
    k0, k1 = slab.slab_range(nz, world, rank)
    lo, hi = slab.neighbours(rank, world, periodic)
    s = ToyFlagSlab(q0[:, k0:k1], lo, hi)
    grp = slab.SlabGroup([s], world, rank=rank, periodic=periodic, dist=dist, syncs=[slab.NoSync()], forcing=True, cfl_dt=True,
                         weno=True)
    grp.step(2)
    ref = toy_flag_reference(q0, periodic, 2)[:, k0:k1]
    q.put((rank, float(np.abs(s.interior() - ref).max()), grp.messages_sent))
    dist.destroy_process_group()


def test_two_gloo_ranks_with_flags_and_forcing():
    sk = socket.socket()
    sk.bind(("127.0.0.1", 0))
    port = sk.getsockname()[1]
    sk.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_flag_worker, args=(r, 2, port, True, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, err, sent in res:
        assert err < 1e-13, (rank, err)
        assert sent == 2 * 3 * 2 * 2                # halos and flag words: two messages each per stage
