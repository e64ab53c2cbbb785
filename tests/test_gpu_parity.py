"""Parity of the CUDA path (through the C-ABI) against the CPU oracle on the same seeded inputs.

Tolerances (BASELINE.json north_star; A18): per RHS evaluation
max|R_gpu - R_oracle| / max|R_oracle| <= 1e-11 per variable; after the stated step counts
||w_gpu - w_oracle||_2 / ||w_oracle||_2 <= 1e-9 per variable.  Sensor flags are integers decided
in fp64 on both sides and must agree exactly.
"""
import math
import os

import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu
GAM = 1.4
RHS_TOL = 1e-11
STEP_TOL = 1e-9


@pytest.fixture(scope="module")
def env():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2004_02276_b200 import build
    build.build()
    from paper_2004_02276_b200 import binding
    from oracle import binding as ob
    binding.lib()
    return torch, binding, ob


def pair(env, wl):
    torch, binding, ob = env
    w0 = wl.state()
    o = ob.Oracle(wl.grid, wl.x, wl.y, wl.z, wl.params)
    o.set_state(w0)
    g = binding.Streams(wl.grid, wl.x, wl.y, wl.z, wl.params)
    g.set_state(torch.from_numpy(w0).cuda())
    return o, g


def rhs_scale(ro, w=None, lam=None):
    """Per-variable scale of the RHS parity check (A18): max|R_oracle|, but never below
    1e-3 * max|w_v| * lambda_max -- R_v is a sum of flux differences of size |w_v| lambda_max
    (lambda_max = max (|u_d|+c)/h_d), and where those cancel to truncation level (the mass equation of a
    solenoidal, uniform-density field: config 2) max|R_v| itself says nothing about round-off."""
    sc = [np.abs(ro[v]).max() for v in range(5)]
    if w is not None and lam is not None:
        sc = [max(sc[v], 1e-3 * np.abs(w[v]).max() * lam) for v in range(5)]
    return sc


def rhs_err(rg, ro, w=None, lam=None):
    sc = rhs_scale(ro, w, lam)
    out = []
    for v in range(5):
        d = np.abs(rg[v] - ro[v]).max()
        out.append(d / sc[v] if sc[v] > 0 else d)
    return out


def l2_err(wg, wo):
    out = []
    for v in range(5):
        n = np.linalg.norm(wo[v])
        d = np.linalg.norm(wg[v] - wo[v])
        out.append(d / n if n > 0 else d)
    return out


def check_rhs(env, wl, tol=RHS_TOL):
    o, g = pair(env, wl)
    ro, rg = o.rhs(), g.rhs().cpu().numpy()
    assert np.isfinite(rg).all()
    lam = max(o.diagnostics(check=False).max_speed)
    e = rhs_err(rg, ro, wl.state(), lam)
    assert max(e) <= tol, (wl.name, e)
    return o, g


def check_flags(env, o, g, sync=False):
    """theta to 1e-12 and interface flags exactly, on the SAME state (sync=True first hands the oracle's
    current state to the GPU context: after independent runs the two states differ at the 1e-10 level)."""
    if sync:
        g.set_state(env[0].from_numpy(o.get_state()).cuda())
    th_o, fl_o = o.sensor()
    th_g, fl_g = g.sensor()
    # theta = -div / sqrt(div^2 + |curl|^2 + eps): a velocity rounding error delta gives |d theta| <= delta/(h sqrt(eps));
    # with delta ~ 2e-16 |u|, 1/h ~ 2e2 and eps down to 1e-6 (Sod tube) that is ~1e-10; the flags must agree exactly
    assert np.abs(th_g.cpu().numpy() - th_o).max() < 1e-10
    assert np.array_equal(fl_g.cpu().numpy(), fl_o)
    return int(fl_o.sum())


def check_steps(env, wl, nsteps, tol=STEP_TOL):
    o, g = pair(env, wl)
    o.step(nsteps)
    g.step(nsteps)
    wo, wg = o.get_state(), g.get_state().cpu().numpy()
    e = l2_err(wg, wo)
    assert max(e) <= tol, (wl.name, e)
    do, dg = o.diagnostics(check=False), g.diagnostics(check=False)
    assert do.nonfinite == 0 and dg.nonfinite == 0
    assert dg.step == nsteps and abs(dg.time - do.time) <= 1e-12 * abs(do.time)
    assert abs(dg.dt - do.dt) <= 1e-12 * do.dt
    assert abs(dg.mass - do.mass) <= 1e-12 * abs(do.mass)
    assert abs(dg.kinetic - do.kinetic) <= 1e-9 * abs(do.kinetic)
    return o, g, do, dg


# ----------------------------------------------------------------------------- RHS, small cases
def P(**kw):
    return W.default_params(Rgas=1 / GAM, mu_ref=5e-3, **kw)


def mod(wl, **kw):
    """The same workload with some parameters replaced."""
    import dataclasses
    return dataclasses.replace(wl, params=dict(wl.params, **kw))


NODE_WALLS = [W.BC_PERIODIC, W.BC_PERIODIC, W.BC_WALL_NODE, W.BC_WALL_NODE, W.BC_PERIODIC, W.BC_PERIODIC]

SMALL = {
    "inviscid_ragged": lambda: W.random_periodic(40, 20, 12, params=P(viscous_enable=0)),
    "viscous_ragged": lambda: W.random_periodic(40, 20, 12, params=P()),
    "viscous_stretched_y": lambda: W.random_periodic(33, 17, 9, params=P(), stretched_y=True),
    "several_tiles_and_chunks": lambda: W.random_periodic(70, 27, 40, params=P()),
    "order4": lambda: W.random_periodic(24, 12, 10, params=P(order=4)),
    "order2": lambda: W.random_periodic(24, 12, 10, params=P(order=2)),
    "sutherland": lambda: W.random_periodic(24, 12, 10, params=P(visc_model=W.VISC_SUTHERLAND)),
    "weno_mixed": lambda: W.random_periodic(40, 20, 12, params=P(weno_enable=1, sensor_threshold=0.3, sensor_eps=0.1)),
    "weno_everywhere": lambda: W.random_periodic(20, 12, 10, params=P(weno_enable=1, sensor_threshold=-1.0, sensor_eps=0.1)),
    "tiny_4x4x4": lambda: W.random_periodic(4, 4, 4, params=P()),
    "line_x": lambda: W.random_periodic(50, 1, 1, params=P()),
    "line_y": lambda: W.random_periodic(1, 50, 1, params=P()),
    "line_z": lambda: W.random_periodic(1, 1, 50, params=P()),
    "channel_small": lambda: W.config3_channel(48, 24, 16),
    "channel_ragged": lambda: W.config3_channel(37, 19, 11),
    "sbli_small": lambda: W.config4_sbli(64, 40, 8, Lx=12.0),
    "sbli_ragged": lambda: W.config4_sbli(45, 30, 7, Lx=10.0),
    # every interface WENO with non-periodic x and y: the interface lists hold N + a boundary plane of entries
    "sbli_weno_everywhere": lambda: mod(W.config4_sbli(45, 30, 7, Lx=10.0), sensor_threshold=-1.0),
    # forcing and the hybrid switch together (unfused fallback: k_rhs<0>, WENO correction, k_update)
    "channel_weno_forcing": lambda: mod(W.config3_channel(37, 19, 11), weno_enable=1, sensor_threshold=0.2, sensor_eps=0.1),
    # forcing with Dirichlet wall nodes (lazy forcing must leave the overridden wall rows alone)
    "channel_node_walls": lambda: mod(W.config3_channel(48, 24, 16), bc=NODE_WALLS),
}

STEPPED = ["channel_ragged", "channel_weno_forcing", "channel_node_walls", "sbli_weno_everywhere", "weno_mixed", "several_tiles_and_chunks"]


@pytest.mark.parametrize("name", list(SMALL))
def test_rhs_small(env, name):
    wl = SMALL[name]()
    o, g = check_rhs(env, wl)
    if wl.params["weno_enable"]:
        nflag = check_flags(env, o, g)
        if name.startswith(("weno", "sbli")):
            assert nflag > 0


@pytest.mark.parametrize("name", STEPPED)
def test_steps_small(env, name):
    """Three RK3 steps of the small cases that take a different path through streams_step (lazy forcing, forcing with
    WENO, Dirichlet wall rows, full interface lists, several chunks): state, dt, time, mass against the oracle."""
    check_steps(env, SMALL[name](), 3)


def test_uniform_flow_is_bitwise_steady(env):
    """Free-stream preservation (oracle pin P3 is bitwise; the CUDA path shares z pair products between
    nodes through running sums, so it is exact to round-off of the flux terms, not bitwise)."""
    wl = W.random_periodic(40, 20, 12, amp=0.0, params=P())
    o, g = pair(env, wl)
    w0 = wl.state()
    lam = max(o.diagnostics(check=False).max_speed)
    r = g.rhs().cpu().numpy()
    for v in range(5):
        assert np.abs(r[v]).max() <= 1e-14 * np.abs(w0[v]).max() * lam
    g.step(2)
    w2 = g.get_state().cpu().numpy()
    for v in range(5):
        assert np.abs(w2[v] - w0[v]).max() <= 1e-14 * np.abs(w0[v]).max()


def test_errors_and_noop(env):
    torch, binding, ob = env
    wl = W.random_periodic(8, 8, 8, params=P())
    g = binding.Streams(wl.grid, wl.x, wl.y, wl.z, wl.params)
    with pytest.raises(binding.StreamsError) as ei:
        g.step(1)
    assert ei.value.code == binding.STREAMS_ESTATE
    w0 = torch.from_numpy(wl.state()).cuda()
    g.set_state(w0)
    g.step(0)
    # the library keeps the state as primitives: get_state(set_state(w)) is w up to the
    # rounding of one division and one multiplication per component, not bitwise
    back = g.get_state()
    for v in range(5):
        assert float((back[v] - w0[v]).abs().max()) <= 4e-16 * float(w0[v].abs().max())
    assert g.diagnostics().step == 0
    bad = w0.clone()
    bad[0, 0, 0, 0] = -1.0
    g.set_state(bad)
    d = g.diagnostics(check=False)
    assert d.nonfinite == 1
    with pytest.raises(binding.StreamsError) as ei:
        g.diagnostics()
    assert ei.value.code == binding.STREAMS_ENONFINITE
    # host-buffer path gives the same state as the device path
    g.set_state(wl.state())
    g.step(1)
    a = g.get_state_host()
    g.set_state(w0)
    g.step(1)
    assert np.array_equal(a, g.get_state().cpu().numpy())


def test_fp64_peak_probe_and_step_repeatability(env):
    """The roofline probe returns a plausible fp64 rate for a B200-class part, and the path is deterministic: the same
    state stepped twice through fresh contexts gives bit-identical results (fixed-order reductions, no float atomics)."""
    torch, binding, ob = env
    rate = binding.fp64_peak()
    assert 5.0 < rate < 25.0, rate                       # 1e12 fp64 lane-instructions/s (nominal 18.6 at 1.965 GHz)
    outs = []
    for wl in (SMALL["channel_small"](), SMALL["weno_mixed"](), SMALL["sbli_small"]()):
        res = []
        for _ in range(2):
            g = binding.Streams(wl.grid, wl.x, wl.y, wl.z, wl.params)
            g.set_state(torch.from_numpy(wl.state()).cuda())
            g.step(3)
            res.append(g.get_state().cpu().numpy())
            g.close()
        assert np.array_equal(res[0], res[1]), wl.name
        outs.append(res[0])
    assert all(np.isfinite(o).all() for o in outs)


def test_split_stepping_is_bitwise_the_same(env):
    """streams_step(5) == streams_step(2); diagnostics; streams_step(3): the CFL step carried from the last stage of a step
    (dt_next), the lazy body force and the ping-pong buffers survive call boundaries and a diagnostics pass in between."""
    torch, binding, ob = env
    for wl in (SMALL["channel_small"](), SMALL["weno_mixed"](), SMALL["channel_weno_forcing"]()):
        w0 = torch.from_numpy(wl.state()).cuda()
        a = binding.Streams(wl.grid, wl.x, wl.y, wl.z, wl.params)
        a.set_state(w0)
        a.step(5)
        b = binding.Streams(wl.grid, wl.x, wl.y, wl.z, wl.params)
        b.set_state(w0)
        b.step(2)
        d = b.diagnostics()
        assert d.step == 2
        b.rhs()                                           # a residual evaluation in between must not disturb the state
        b.step(3)
        assert np.array_equal(a.get_state().cpu().numpy(), b.get_state().cpu().numpy()), wl.name
        da, db = a.diagnostics(), b.diagnostics()
        assert da.time == db.time and da.dt == db.dt and da.step == db.step == 5
        a.close()
        b.close()


def test_sod_tube_gpu(env):
    """Hybrid recipe end to end on the GPU along x: same answer as the oracle after the full run."""
    n = 200
    xs = (np.arange(n) + 0.5) / n
    p = W.default_params(viscous_enable=0, weno_enable=1, sensor_threshold=0.5, sensor_eps=1e-6, Rgas=1.0, cfl=0.5,
                         bc=[W.BC_EXTRAP, W.BC_EXTRAP] + [W.BC_PERIODIC] * 4)
    grid = dict(nx=n, ny=1, nz=1, len=[1.0, 1.0, 1.0])
    left = (xs < 0.5).reshape(1, 1, n)
    w0 = W.prim_to_cons(np.where(left, 1.0, 0.125), np.zeros((1, 1, n)), np.zeros((1, 1, n)), np.zeros((1, 1, n)),
                        np.where(left, 1.0, 0.1), GAM)
    wl = W.Workload("sod", grid, xs, np.zeros(1), np.zeros(1), p, 60, 0, state_fn=lambda a, b: w0.copy())
    o, g, do, dg = check_steps(env, wl, 60, tol=1e-9)
    assert dg.min_rho > 0.12 and 0.05 < dg.time < 0.1
    assert check_flags(env, o, g, sync=True) > 0


# ----------------------------------------------------------------------------- the five configs
def test_config1_tgv_full(env):
    """config 1: 32^3 TGV, 20 RK3 steps at CFL 0.5; the sensor must stay inactive."""
    wl = W.config1_tgv()
    o, g = check_rhs(env, wl)
    assert check_flags(env, o, g) == 0
    o, g, do, dg = check_steps(env, wl, wl.steps)
    assert list(dg.weno_ifaces) == [0, 0, 0]


def test_config2_isotropic_full(env):
    """config 2: 128^3 decaying isotropic turbulence, Mt = 0.6, 100 RK3 steps; shocklets trigger WENO."""
    wl = W.config2_isotropic()
    o, g = check_rhs(env, wl)
    nflag = check_flags(env, o, g)
    o, g, do, dg = check_steps(env, wl, wl.steps)
    assert check_flags(env, o, g, sync=True) >= 0
    frac = sum(dg.weno_ifaces) / sum(dg.total_ifaces)
    print("config2: flagged interface fraction after 100 steps %.4f, initial flags %d" % (frac, nflag))


def test_config3_channel(env):
    """config 3: channel with staggered walls and bulk forcing: reduced grid for the stated 200 steps,
    and the full 256x128x128 grid for one RHS and 10 steps."""
    wl = W.config3_channel(128, 64, 64)
    o, g, do, dg = check_steps(env, wl, wl.steps)
    assert abs(dg.forcing - do.forcing) <= 1e-9 * abs(do.forcing)
    full = W.config3_channel()
    check_rhs(env, full)
    o, g, do, dg = check_steps(env, full, 10)
    d0 = None
    # P11/P12 on the GPU path: mass and bulk momentum constant to round-off
    torch = env[0]
    g.set_state(torch.from_numpy(full.state()).cuda())
    d0 = g.diagnostics()
    g.step(10)
    d1 = g.diagnostics()
    assert abs(d1.mass - d0.mass) <= 1e-13 * d0.mass
    assert abs(d1.mom[0] - d0.mom[0]) <= 1e-12 * abs(d0.mom[0])


def slab_check(env, wl, gpu_rhs, slabs, planes=8):
    """Compare planes [k0, k0+planes) of a full-size GPU RHS with the oracle run on the slab plus `halo`
    wrapped planes each side (forcing off on both sides).  Every stencil has z-radius 3; with the WENO
    switch on, an interface flag looks at theta of nodes up to 3 planes away, each of which needs 3 more
    planes, so the slab then carries 6."""
    torch, binding, ob = env
    worst = [0.0] * 5
    scale = [float(gpu_rhs[v].abs().max()) for v in range(5)]
    halo = 6 if wl.params["weno_enable"] else 3
    for k0 in slabs:
        sub = wl.slab(k0, k0 + planes, halo=halo)
        o = ob.Oracle(sub.grid, sub.x, sub.y, sub.z, sub.params)
        o.set_state(sub.state())
        ro = o.rhs()[:, halo:halo + planes]
        rg = gpu_rhs[:, k0:k0 + planes].cpu().numpy()
        for v in range(5):
            worst[v] = max(worst[v], np.abs(rg[v] - ro[v]).max() / scale[v])
        o.close()
    return worst


def test_config4_sbli(env):
    """config 4: reduced grid for the stated 100 steps (all boundary kinds, WENO across the shock), and the
    full 1024x256x128 grid for one RHS, checked on sampled z-slabs."""
    wl = W.config4_sbli(256, 64, 32)
    o, g = check_rhs(env, wl)
    assert check_flags(env, o, g) > 0
    o, g, do, dg = check_steps(env, wl, wl.steps)
    assert sum(dg.weno_ifaces) > 0
    torch, binding, ob = env
    full = W.config4_sbli()
    s = binding.Streams(full.grid, full.x, full.y, full.z, full.params)
    s.set_state(torch.from_numpy(full.state()).cuda())
    r = s.rhs()
    worst = slab_check(env, full, r, [0, 60, 120])
    assert max(worst) <= RHS_TOL, worst
    s.step(2)
    d = s.diagnostics()
    assert d.nonfinite == 0 and sum(d.weno_ifaces) > 0
    s.close()


def test_config5_big_channel_spot_check(env):
    """config 5: 1024x512x512 (268M points) in the launch configuration bench.py times: one RHS checked
    against the oracle on three 8-plane z-slabs; then invariants that hold at any size over 5 steps."""
    torch, binding, ob = env
    wl = W.config5_channel_big()
    if torch.cuda.get_device_properties(0).total_memory < 70e9:
        pytest.skip("needs ~55 GB of device memory")
    nofo = dict(wl.params, forcing=0)
    s = binding.Streams(wl.grid, wl.x, wl.y, wl.z, nofo)
    w = torch.empty(wl.shape, dtype=torch.float64, device="cuda")
    for k0 in range(0, wl.grid["nz"], 16):
        w[:, k0:k0 + 16].copy_(torch.from_numpy(wl.state(k0, k0 + 16)))
    s.set_state(w)
    r = s.rhs()
    worst = slab_check(env, wl, r, [0, 252, 504])
    assert max(worst) <= RHS_TOL, worst
    # full-field forcing sum against an independent float64 pairwise/fsum reduction of the GPU-produced R
    hx = np.full(wl.grid["nx"], wl.grid["len"][0] / wl.grid["nx"])
    s.close()
    del r
    s = binding.Streams(wl.grid, wl.x, wl.y, wl.z, wl.params)
    s.set_state(w)
    d0 = s.diagnostics()
    s.step(5)
    d1 = s.diagnostics()
    assert d1.nonfinite == 0 and d1.forcing > 0
    assert abs(d1.mass - d0.mass) <= 1e-13 * d0.mass
    assert abs(d1.mom[0] - d0.mom[0]) <= 1e-12 * abs(d0.mom[0])
    assert abs(d0.volume - 6 * math.pi * 2 * 2 * math.pi) < 1e-6 * d0.volume
    assert hx[0] > 0
    s.close()
