"""z-slab decomposition on ONE GPU: several contexts of the CUDA library,
one per slab, exchange their ghost planes through the C-ABI halo calls and are stepped by the staged calls.

What the decomposed run must compute is fixed by the undivided problem: it is compared (a) bit for bit with the
single-context run of the same library (every node sees the same stencil values; the maximum of S10 is exact; the body-force
sum of S9 is either fed from the undivided run -> bitwise, or combined from the slabs' partial sums -> summation-order
round-off only) and (b) with the CPU oracle on the undivided grid, to the step tolerance of DESIGN.md A18.
Kernels of different slabs never wait on one another: the exchange is ordered by stream events on one device.
"""
import os

import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu
STEP_TOL = 1e-9


@pytest.fixture(scope="module")
def env():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2004_02276_b200 import build
    build.build()
    from paper_2004_02276_b200 import binding, slab
    from oracle import binding as ob
    binding.lib()
    return torch, binding, slab, ob


class HostReducer:
    """Combines the slabs' partial reductions on the host (test only): fixed slab order."""

    def __init__(self, torch):
        self.torch = torch

    def _combine(self, slabs, lo, hi, fn):
        vals = []
        for s in slabs:
            s.stream.synchronize()
            vals.append(s.red[lo:hi].cpu().numpy().copy())
        tot = vals[0]
        for v in vals[1:]:
            tot = fn(tot, v)
        t = self.torch.from_numpy(tot)
        for s in slabs:
            with self.torch.cuda.stream(s.stream):
                s.red[lo:hi].copy_(t.to(s.device))
            s.stream.synchronize()

    def sum(self, slabs, syncs):
        self._combine(slabs, 0, 2, lambda a, b: a + b)

    def max(self, slabs, syncs):
        self._combine(slabs, 2, 3, np.maximum)


def make_slabs(env, wl, nslabs):
    torch, binding, slab, _ = env
    w0 = wl.state()
    ctxs, specs = [], []
    for r in range(nslabs):
        sp = slab.slab_spec(wl.grid, wl.z, wl.params, nslabs, r)
        c = binding.Streams(sp.grid, wl.x, wl.y, sp.z, sp.params)
        c.set_state(torch.from_numpy(np.ascontiguousarray(w0[:, sp.k0:sp.k1])).cuda())
        ctxs.append(c)
        specs.append(sp)
    return ctxs, specs, w0


def gather(ctxs):
    return np.concatenate([c.get_state().cpu().numpy() for c in ctxs], axis=1)


def l2(a, b):
    return max(np.linalg.norm(a[v] - b[v]) / np.linalg.norm(b[v]) for v in range(5))


@pytest.mark.parametrize("nslabs,overlap", [(2, False), (3, True), (4, True)])
def test_periodic_box_slabs_are_bitwise_the_undivided_run(env, nslabs, overlap):
    """No forcing, CFL time step (max-reduction across slabs): the concatenated slabs equal the single context bit for bit,
    with and without the interior / boundary split of the fused kernel."""
    torch, binding, slab, ob = env
    wl = W.random_periodic(40, 20, 48, params=W.default_params(Rgas=1 / 1.4, mu_ref=5e-3))
    w0 = wl.state()
    one = binding.Streams(wl.grid, wl.x, wl.y, wl.z, wl.params)
    one.set_state(torch.from_numpy(w0).cuda())
    one.step(3)
    ref = one.get_state().cpu().numpy()
    ctxs, specs, _ = make_slabs(env, wl, nslabs)
    grp = slab.SlabGroup(ctxs, nslabs, periodic=True, reducer=HostReducer(torch), forcing=False, cfl_dt=True, overlap=overlap)
    grp.step(3)
    got = gather(ctxs)
    assert np.array_equal(got, ref), np.abs(got - ref).max()
    assert grp.messages_sent == 3 * 3 * 2 * nslabs
    d1, ds = one.diagnostics(), [c.diagnostics() for c in ctxs]
    assert all(d.dt == d1.dt and d.time == d1.time and d.step == 3 for d in ds)
    o = ob.Oracle(wl.grid, wl.x, wl.y, wl.z, wl.params)
    o.set_state(w0)
    o.step(3)
    assert l2(got, o.get_state()) < STEP_TOL
    for c in ctxs + [one]:
        c.close()
    o.close()


def test_slab_residual_equals_the_undivided_residual(env):
    """streams_rhs on slabs after one halo swap = the rows of the undivided residual, bit for bit."""
    torch, binding, slab, ob = env
    wl = W.random_periodic(36, 18, 30, params=W.default_params(Rgas=1 / 1.4, mu_ref=5e-3), stretched_y=True)
    one = binding.Streams(wl.grid, wl.x, wl.y, wl.z, wl.params)
    one.set_state(torch.from_numpy(wl.state()).cuda())
    ref = one.rhs().cpu().numpy()
    ctxs, specs, _ = make_slabs(env, wl, 3)
    grp = slab.SlabGroup(ctxs, 3, periodic=True, reducer=HostReducer(torch))
    grp.residual_ready()
    got = np.concatenate([c.rhs().cpu().numpy() for c in ctxs], axis=1)
    assert np.array_equal(got, ref), np.abs(got - ref).max()
    for c in ctxs + [one]:
        c.close()


def test_channel_slabs_with_forcing(env):
    """Lazy forcing across slabs: the body force needs the sum of R_rhou vol over ALL slabs every stage.
    (1) fed: the staged calls on the undivided context run in lockstep and its red[] goes to every slab -> bitwise;
    (2) combined: the slabs' partial sums are added (another summation order) -> round-off; oracle parity for both."""
    torch, binding, slab, ob = env
    wl = W.config3_channel(64, 32, 40)
    w0 = wl.state()
    nsl, nsteps = 2, 3
    # (1) fed
    one = binding.Streams(wl.grid, wl.x, wl.y, wl.z, wl.params)
    one.set_state(torch.from_numpy(w0).cuda())
    ctxs, specs, _ = make_slabs(env, wl, nsl)
    grp = slab.SlabGroup(ctxs, nsl, periodic=True, reducer=HostReducer(torch), forcing=True)

    def feed(lo, hi):
        one.stream.synchronize()
        v = one.red[lo:hi].clone()
        for c in ctxs:
            with torch.cuda.stream(c.stream):
                c.red[lo:hi].copy_(v)
            c.stream.synchronize()

    for _ in range(nsteps):
        one.step_begin()
        for c in ctxs:
            c.step_begin()
        feed(2, 3)
        for stage in range(3):
            ready = grp.swap_halos()
            one.stage_rhs(stage, one.PART_ALL)
            for i, c in enumerate(ctxs):
                grp.syncs[i].main_wait(ready[i])
                c.stage_rhs(stage, c.PART_INTERIOR)
                c.stage_rhs(stage, c.PART_BOUNDARY)
            feed(0, 2)
            one.stage_end(stage)
            for c in ctxs:
                c.stage_end(stage)
    ref = one.get_state().cpu().numpy()
    got = gather(ctxs)
    assert np.array_equal(got, ref), np.abs(got - ref).max()
    # the staged calls on one context are streams_step
    two = binding.Streams(wl.grid, wl.x, wl.y, wl.z, wl.params)
    two.set_state(torch.from_numpy(w0).cuda())
    two.step(nsteps)
    assert np.array_equal(two.get_state().cpu().numpy(), ref)
    # (2) combined
    ctxs2, _, _ = make_slabs(env, wl, nsl)
    grp2 = slab.SlabGroup(ctxs2, nsl, periodic=True, reducer=HostReducer(torch), forcing=True)
    grp2.step(nsteps)
    got2 = gather(ctxs2)
    assert l2(got2, ref) < 1e-13
    f1, f2 = one.diagnostics().forcing, ctxs2[0].diagnostics().forcing
    assert abs(f1 - f2) <= 1e-12 * abs(f1)
    o = ob.Oracle(wl.grid, wl.x, wl.y, wl.z, wl.params)
    o.set_state(w0)
    o.step(nsteps)
    assert l2(got2, o.get_state()) < STEP_TOL
    for c in ctxs + ctxs2 + [one, two]:
        c.close()
    o.close()


def test_channel_slabs_with_forcing_and_the_hybrid_switch(env):
    """forcing = 1 with weno_enable = 1 on slabs: the body force is the sum of the residual after its
    WENO correction, which needs the neighbours' flag words: stage_rhs | flag swap | stage_mid | SUM | stage_end.
    (1) fed: the undivided context runs the same staged calls in lockstep and its red[0..1] go to every slab -> bitwise,
    and equal to streams_step; (2) combined: the slabs' sums are added -> summation-order round-off; oracle parity."""
    import dataclasses
    torch, binding, slab, ob = env
    wl = W.config3_channel(64, 32, 40)
    wl = dataclasses.replace(wl, params=dict(wl.params, weno_enable=1, sensor_threshold=0.2, sensor_eps=0.1))
    w0 = wl.state()
    nsl, nsteps = 2, 3
    one = binding.Streams(wl.grid, wl.x, wl.y, wl.z, wl.params)
    one.set_state(torch.from_numpy(w0).cuda())
    ctxs, specs, _ = make_slabs(env, wl, nsl)
    grp = slab.SlabGroup(ctxs, nsl, periodic=True, reducer=HostReducer(torch), forcing=True, weno=True)

    def feed(lo, hi):
        one.stream.synchronize()
        v = one.red[lo:hi].clone()
        for c in ctxs:
            with torch.cuda.stream(c.stream):
                c.red[lo:hi].copy_(v)
            c.stream.synchronize()

    for _ in range(nsteps):
        one.step_begin()
        for c in ctxs:
            c.step_begin()
        feed(2, 3)
        for stage in range(3):
            ready = grp.swap_halos()
            one.stage_rhs(stage, one.PART_ALL)
            for i, c in enumerate(ctxs):
                grp.syncs[i].main_wait(ready[i])
                c.stage_rhs(stage, c.PART_INTERIOR)
                c.stage_rhs(stage, c.PART_BOUNDARY)
            if stage == 0:
                with pytest.raises(binding.StreamsError):          # a slab cannot sum before the flags are in
                    ctxs[0].stage_end(stage)
            grp.swap_flags()
            one.stage_mid(stage)
            for c in ctxs:
                c.stage_mid(stage)
            feed(0, 2)
            one.stage_end(stage)
            for c in ctxs:
                c.stage_end(stage)
    ref = one.get_state().cpu().numpy()
    assert sum(one.diagnostics().weno_ifaces) > 0, "the case must exercise the WENO branch"
    got = gather(ctxs)
    assert np.array_equal(got, ref), np.abs(got - ref).max()
    two = binding.Streams(wl.grid, wl.x, wl.y, wl.z, wl.params)    # streams_step = the staged calls without stage_mid
    two.set_state(torch.from_numpy(w0).cuda())
    two.step(nsteps)
    assert np.array_equal(two.get_state().cpu().numpy(), ref)
    with pytest.raises(binding.StreamsError):
        two.stage_mid(0)                                           # no staged step is open
    # (2) combined
    ctxs2, _, _ = make_slabs(env, wl, nsl)
    grp2 = slab.SlabGroup(ctxs2, nsl, periodic=True, reducer=HostReducer(torch), forcing=True, weno=True)
    grp2.step(nsteps)
    got2 = gather(ctxs2)
    assert l2(got2, ref) < 1e-13
    f1, f2 = one.diagnostics().forcing, ctxs2[0].diagnostics().forcing
    assert abs(f1 - f2) <= 1e-12 * abs(f1)
    o = ob.Oracle(wl.grid, wl.x, wl.y, wl.z, wl.params)
    o.set_state(w0)
    o.step(nsteps)
    assert l2(got2, o.get_state()) < STEP_TOL
    for c in ctxs + ctxs2 + [one, two]:
        c.close()
    o.close()


def test_staged_calls_enforce_their_order(env):
    torch, binding, slab, _ = env
    wl = W.random_periodic(32, 16, 16, params=W.default_params(Rgas=1 / 1.4, mu_ref=5e-3))
    sp = slab.slab_spec(wl.grid, wl.z, wl.params, 2, 0)
    c = binding.Streams(sp.grid, wl.x, wl.y, sp.z, sp.params)
    c.set_state(torch.from_numpy(np.ascontiguousarray(wl.state()[:, sp.k0:sp.k1])).cuda())
    with pytest.raises(binding.StreamsError):
        c.step(1)                                    # a slab advances by the staged calls only
    with pytest.raises(binding.StreamsError):
        c.stage_rhs(0)                               # before step_begin
    c.step_begin()
    with pytest.raises(binding.StreamsError):
        c.stage_end(0)                               # before stage_rhs
    with pytest.raises(binding.StreamsError):
        c.stage_rhs(1)                               # wrong stage
    c.close()
    # streams_rhs is one call: it refuses the slabs whose residual needs an exchange in the middle of it
    for wl2 in (W.config3_channel(32, 16, 16), W.random_periodic(32, 16, 16, params=W.default_params(
            Rgas=1 / 1.4, mu_ref=5e-3, weno_enable=1, sensor_threshold=0.3, sensor_eps=0.1))):
        sp2 = slab.slab_spec(wl2.grid, wl2.z, wl2.params, 2, 0)
        c2 = binding.Streams(sp2.grid, wl2.x, wl2.y, sp2.z, sp2.params)
        c2.set_state(torch.from_numpy(np.ascontiguousarray(wl2.state()[:, sp2.k0:sp2.k1])).cuda())
        with pytest.raises(binding.StreamsError):
            c2.rhs()                                 # forcing: sum over all slabs; hybrid switch: neighbours' flag words
        c2.close()
    # a non-periodic direction cannot take BC_HALO outside z
    p = dict(wl.params)
    p["bc"] = [8, 8, 0, 0, 0, 0]
    with pytest.raises(binding.StreamsError):
        binding.Streams(wl.grid, wl.x, wl.y, wl.z, p)


@pytest.mark.parametrize("case", ["channel_forcing", "sbli_weno"])
def test_nccl_self_exchange_world_size_one(env, case):
    """The torch.distributed (NCCL) path of SlabGroup on one GPU: a single periodic slab whose two faces are BC_HALO
    sends its messages to itself through ncclSend/ncclRecv and all-reduces its partial reductions (world size 1: no rank
    waits on another rank's kernels).  Result: bitwise the periodic single-context run.  `sbli_weno` also moves the
    node-flag words of the hybrid switch (int32 messages) and captures the frozen inflow after the first swap."""
    torch, binding, slab, ob = env
    import torch.distributed as dist
    if not dist.is_nccl_available():
        pytest.skip("NCCL backend not available")
    wl = W.config3_channel(48, 24, 24) if case == "channel_forcing" else W.config4_sbli(64, 40, 16)
    weno = bool(wl.params["weno_enable"])
    w0 = wl.state()
    one = binding.Streams(wl.grid, wl.x, wl.y, wl.z, wl.params)
    one.set_state(torch.from_numpy(w0).cuda())
    one.step(2)
    ref = one.get_state().cpu().numpy()
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29533")
    created = not dist.is_initialized()
    if created:
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        # one slab of the whole domain, but with both z faces as internal (HALO) boundaries: its own planes come back
        sp = slab.slab_spec(wl.grid, wl.z, wl.params, 1, 0)
        assert sp.params["bc"][4] == 8 and sp.params["bc"][5] == 8 and len(sp.z) == wl.grid["nz"] + 6
        c = binding.Streams(sp.grid, wl.x, wl.y, sp.z, sp.params)
        c.set_state(torch.from_numpy(w0).cuda())
        grp = slab.SlabGroup([c], 1, rank=0, periodic=True, dist=dist, forcing=bool(wl.params["forcing"]), weno=weno)
        grp.step(2)
        got = c.get_state().cpu().numpy()
        assert np.array_equal(got, ref), np.abs(got - ref).max()
        assert grp.messages_sent == 2 * 3 * 2 * (2 if weno else 1)
        c.close()
    finally:
        if created:
            dist.destroy_process_group()
    one.close()


@pytest.mark.parametrize("case", ["weno_box", "weno3_box", "sbli"])
def test_hybrid_switch_on_slabs_is_bitwise_the_undivided_run(env, case):
    """The hybrid switch across slab faces: the node-flag words of the neighbour's three planes are
    swapped between stage_rhs and stage_end; the interfaces next to a face are then flagged, listed and corrected exactly as
    in the undivided run.  `sbli` adds the frozen inflow (captured with its ghost planes after the first halo swap), the
    node wall, the shock generator and the characteristic outflow."""
    torch, binding, slab, ob = env
    if case in ("weno_box", "weno3_box"):
        wl = W.random_periodic(32, 16, 36, params=W.default_params(Rgas=1 / 1.4, mu_ref=5e-3, weno_enable=1,
                                                                   sensor_threshold=0.3, sensor_eps=0.1,
                                                                   weno_order=3 if case == "weno3_box" else 5))
        nsl = 3
    else:
        wl = W.config4_sbli(64, 40, 16)
        nsl = 2
    w0 = wl.state()
    one = binding.Streams(wl.grid, wl.x, wl.y, wl.z, wl.params)
    one.set_state(torch.from_numpy(w0).cuda())
    one.step(3)
    ref = one.get_state().cpu().numpy()
    d1 = one.diagnostics()
    assert sum(d1.weno_ifaces) > 0, "the case must exercise the WENO branch"
    ctxs, specs, _ = make_slabs(env, wl, nsl)
    grp = slab.SlabGroup(ctxs, nsl, periodic=True, reducer=HostReducer(torch), forcing=False, cfl_dt=True, weno=True)
    grp.step(3)
    got = gather(ctxs)
    assert np.array_equal(got, ref), np.abs(got - ref).max()
    o = ob.Oracle(wl.grid, wl.x, wl.y, wl.z, wl.params)
    o.set_state(w0)
    o.step(3)
    assert l2(got, o.get_state()) < STEP_TOL
    for c in ctxs + [one]:
        c.close()
    o.close()


def test_config5_size_two_slabs_one_step_bitwise(env):
    """The 1024x512x512 channel block (config 5: 32 x 64 tiles, wall tiles, lazy forcing, four 128-plane chunks) cut into
    two 1024x512x256 slabs on the same device, in the launch configuration bench.py --decomp slab times (interior chunks
    while the halos move, boundary chunks after): one RK3 step, fed reductions, bit for bit the undivided context."""
    torch, binding, slab, _ = env
    wl = W.config5_channel_big()
    nz, planes = wl.grid["nz"], 32

    def upload(ctx, k0, k1):
        w = torch.empty((5, k1 - k0, wl.grid["ny"], wl.grid["nx"]), dtype=torch.float64, device="cuda")
        for a in range(k0, k1, planes):
            b = min(k1, a + planes)
            w[:, a - k0:b - k0].copy_(torch.from_numpy(wl.state(a, b)))
        ctx.set_state(w)
        del w

    one = binding.Streams(wl.grid, wl.x, wl.y, wl.z, wl.params)
    upload(one, 0, nz)
    ctxs, specs = [], []
    for r in range(2):
        sp = slab.slab_spec(wl.grid, wl.z, wl.params, 2, r)
        c = binding.Streams(sp.grid, wl.x, wl.y, sp.z, sp.params)
        upload(c, sp.k0, sp.k1)
        ctxs.append(c)
        specs.append(sp)
    grp = slab.SlabGroup(ctxs, 2, periodic=True, reducer=HostReducer(torch), forcing=True)

    def feed(lo, hi):
        one.stream.synchronize()
        v = one.red[lo:hi].clone()
        for c in ctxs:
            with torch.cuda.stream(c.stream):
                c.red[lo:hi].copy_(v)
            c.stream.synchronize()

    one.step_begin()
    for c in ctxs:
        c.step_begin()
    feed(2, 3)
    for stage in range(3):
        ready = grp.swap_halos()
        one.stage_rhs(stage, one.PART_ALL)
        for c in ctxs:
            c.stage_rhs(stage, c.PART_INTERIOR)
        for i, c in enumerate(ctxs):
            grp.syncs[i].main_wait(ready[i])
            c.stage_rhs(stage, c.PART_BOUNDARY)
        feed(0, 2)
        one.stage_end(stage)
        for c in ctxs:
            c.stage_end(stage)
    ref = one.get_state()
    for c, sp in zip(ctxs, specs):
        got = c.get_state()
        assert torch.equal(got, ref[:, sp.k0:sp.k1]), float((got - ref[:, sp.k0:sp.k1]).abs().max())
        del got
    d = [c.diagnostics() for c in ctxs + [one]]
    assert d[0].dt == d[2].dt and d[0].forcing == d[2].forcing and d[1].forcing == d[2].forcing
    assert abs(d[0].mass + d[1].mass - d[2].mass) <= 1e-12 * d[2].mass
    for c in ctxs + [one]:
        c.close()


def test_non_periodic_z_ends_keep_their_boundary(env):
    """z faces that are physical boundaries (zeroth-order extrapolation) stay with the first and the last slab; only the
    internal faces become BC_HALO (one-sided halos): three slabs are bitwise the undivided run."""
    torch, binding, slab, ob = env
    p = W.default_params(Rgas=1 / 1.4, mu_ref=5e-3)
    p["bc"] = [0, 0, 0, 0, W.BC_EXTRAP, W.BC_EXTRAP]
    wl = W.random_periodic(40, 20, 36, params=p)
    w0 = wl.state()
    one = binding.Streams(wl.grid, wl.x, wl.y, wl.z, wl.params)
    one.set_state(torch.from_numpy(w0).cuda())
    one.step(3)
    ref = one.get_state().cpu().numpy()
    ctxs, specs, _ = make_slabs(env, wl, 3)
    assert [sp.params["bc"][4:] for sp in specs] == [[W.BC_EXTRAP, 8], [8, 8], [8, W.BC_EXTRAP]]
    grp = slab.SlabGroup(ctxs, 3, periodic=False, reducer=HostReducer(torch), forcing=False, cfl_dt=True)
    grp.step(3)
    got = gather(ctxs)
    assert np.array_equal(got, ref), np.abs(got - ref).max()
    assert grp.messages_sent == 3 * 3 * 4
    o = ob.Oracle(wl.grid, wl.x, wl.y, wl.z, wl.params)
    o.set_state(w0)
    o.step(3)
    assert l2(got, o.get_state()) < STEP_TOL
    for c in ctxs + [one]:
        c.close()
    o.close()
