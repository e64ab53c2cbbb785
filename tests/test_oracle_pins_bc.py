"""Pins of the oracle's boundary closures (S1), viscosity law, sensor, forcing power and Roe state.

Each test fails under one plausible mistake in `oracle/streams_oracle.c` that the pins of
tests/test_oracle_pins.py do not see (a wrong ghost rule for rho, p, T at a wall, a shifted mirror
index, a missing Dirichlet override, shock-generator ghosts that never switch to the post-shock
state, a wrong Sutherland exponent, a vorticity component dropped from Eq. 8, the f u_1 power of
Eq. 1c dropped, an arithmetic instead of a Roe mean).  None of them touches the CUDA path, and none
compares the oracle with itself: the expected values are closed forms (linear profiles continued
through a wall, normal-shock relations, Roe's property U), sympy-manufactured fields, or ghost
arrays built by hand in NumPy from the rule as DESIGN.md S1 states it.
"""
import math

import numpy as np
import pytest

import workloads as W
from tests import helpers as H

GAM = 1.4
R_GAS = 1.0 / GAM
CV = R_GAS / (GAM - 1.0)
CP = GAM * CV


@pytest.fixture(scope="module")
def ob(oracle_mod):
    return oracle_mod


def column(ob, y, params, rho, u, v, w, p):
    """One column of ny nodes along y (x, z: one periodic node each)."""
    ny = len(y)
    grid = dict(nx=1, ny=ny, nz=1, len=[1.0, float(y[-1] - y[0]), 1.0])
    o = ob.Oracle(grid, np.zeros(1), y, np.zeros(1), params)
    sh = (1, ny, 1)
    o.set_state(W.prim_to_cons(rho.reshape(sh), u.reshape(sh), v.reshape(sh), w.reshape(sh), p.reshape(sh), GAM))
    return o


def prim_of(wg):
    rho = wg[0]
    u, v, w = wg[1] / rho, wg[2] / rho, wg[3] / rho
    p = (GAM - 1.0) * (wg[4] - 0.5 * rho * (u * u + v * v + w * w))
    return rho, u, v, w, p, p / (rho * R_GAS)


# ------------------------------------------------------------------ (a) staggered isothermal wall, S1 / PAPER.md:110
def stag_setup(ob, ny=24, Tw=(1.1, 1.5), c=0.4, visc_exp=1.0):
    """Linear u and T between staggered walls at y = -1, +1: u = c (y + 1) vanishes at the lower wall,
    T runs from Tw[0] to Tw[1]; p uniform.  mu ~ T (visc_exp = 1) so that mu is linear in y as well."""
    y = -1.0 + (2.0 * np.arange(ny) + 1.0) / ny
    d = 0.5 * (Tw[1] - Tw[0])
    T = Tw[0] + d * (y + 1.0)
    u = c * (y + 1.0)
    p = np.full(ny, 0.9)
    bc = [W.BC_PERIODIC] * 2 + [W.BC_WALL_STAG] * 2 + [W.BC_PERIODIC] * 2
    prm = W.default_params(Rgas=R_GAS, mu_ref=0.02, T_ref=1.0, visc_exp=visc_exp, T_wall=list(Tw), y_wall=[-1.0, 1.0], bc=bc)
    o = column(ob, y, prm, p / (R_GAS * T), u, np.zeros(ny), np.zeros(ny), p)
    return o, y, T, u, p, d, c, prm


def test_wall_staggered_ghost_rule_direct(ob):
    """Ghost node -l mirrors node l-1 about the wall plane: u -> -u, T -> 2 T_w - T, p -> p, rho = p / (R T)
    (S1; the wall sits half-way between the ghost and its mirror)."""
    o, y, T, u, p, d, c, prm = stag_setup(ob)
    ny = len(y)
    wg = o.ghosted()[:, 3, :, 3]                      # the column, ghost-extended in y
    rho_g, u_g, v_g, w_g, p_g, T_g = prim_of(wg)
    for l in (1, 2, 3):
        for side, (g, m, Tw) in enumerate([(3 - l, 3 + l - 1, prm["T_wall"][0]), (3 + ny - 1 + l, 3 + ny - l, prm["T_wall"][1])]):
            assert abs(u_g[g] + u_g[m]) < 1e-15 and abs(w_g[g] + w_g[m]) < 1e-15           # velocity odd
            assert abs(p_g[g] - p_g[m]) < 1e-15                                           # pressure even
            assert abs((T_g[g] - Tw) + (T_g[m] - Tw)) < 1e-15                             # T - T_w odd
            assert abs(rho_g[g] - p_g[m] / (R_GAS * (2 * Tw - T_g[m]))) < 1e-15            # rho from the gas law


def test_wall_staggered_linear_profiles_continue_through_the_wall(ob):
    """Closed form.  With the S1 rule a profile that is linear in y and takes the wall value on the wall plane is
    continued linearly into the ghosts, so the discrete derivatives at the wall-adjacent nodes are exact:
    u_y = c, u_yy = 0, T_y = d, T_yy = 0, mu_y = mu_ref d / T_ref, and p_y = 0 because p is even.  Then (Eq. 2-3, 9)
      V_rhou = mu_y u_y,   V_rhoE = u V_rhou + mu u_y^2 + (c_p / Pr) mu_y T_y,   convective part = 0 exactly.
    A ghost temperature T_w (instead of 2 T_w - T) kinks T; a ghost density rho (instead of p / R T_g) breaks p_y = 0."""
    o, y, T, u, p, d, c, prm = stag_setup(ob)
    conv, visc = o.rhs_parts()
    conv, visc = conv[:, 0, :, 0], visc[:, 0, :, 0]
    mu = prm["mu_ref"] * T / prm["T_ref"]
    mu_y = prm["mu_ref"] * d / prm["T_ref"]
    low = slice(0, 8)                                 # u is linear about the LOWER wall only
    Vx = mu_y * c
    assert np.abs(visc[1][low] - Vx).max() < 1e-10 * abs(Vx)
    VE = u * Vx + mu * c * c + CP / prm["Pr"] * mu_y * d
    assert np.abs(visc[4][low] - VE[low]).max() < 1e-10 * np.abs(VE).max()
    # T is linear between BOTH walls (different wall temperatures): no conduction residual anywhere if u = 0
    o2, y, T, u, p, d, c, prm = stag_setup(ob, c=0.0)
    conv2, visc2 = o2.rhs_parts()
    heat = CP / prm["Pr"] * mu_y * d
    assert np.abs(visc2[4, 0, :, 0] - heat).max() < 1e-10 * abs(heat)
    for cv in (conv, conv2[:, 0, :, 0]):
        assert np.abs(cv).max() < 1e-13 * p.max() * len(y)      # v = 0, p uniform and even: nothing convective


# ------------------------------------------------------------------ (b) isothermal wall on the boundary node, S1 / PAPER.md:126
def node_setup(ob, ny=24, Tw=(1.2, 1.8), c=0.4):
    y = np.linspace(0.0, 2.0, ny)
    d = (Tw[1] - Tw[0]) / 2.0
    T = Tw[0] + d * y
    u = c * y                                          # no slip on node 0
    p = np.full(ny, 0.8)
    bc = [W.BC_PERIODIC] * 2 + [W.BC_WALL_NODE] * 2 + [W.BC_PERIODIC] * 2
    prm = W.default_params(Rgas=R_GAS, mu_ref=0.02, T_ref=1.0, visc_exp=1.0, T_wall=list(Tw), bc=bc)
    o = column(ob, y, prm, p / (R_GAS * T), u, np.zeros(ny), np.zeros(ny), p)
    return o, y, T, u, p, d, c, prm


def test_wall_node_ghost_rule_and_linear_continuation(ob):
    """Ghost node -l mirrors node +l about the wall NODE (odd for u and T - T_w, even for p).  A shifted mirror index
    breaks both the direct comparison and the closed form u_y = c, u_yy = 0 at the first interior nodes."""
    o, y, T, u, p, d, c, prm = node_setup(ob)
    ny = len(y)
    rho_g, u_g, v_g, w_g, p_g, T_g = prim_of(o.ghosted()[:, 3, :, 3])
    for l in (1, 2, 3):
        for g, m, Tw in [(3 - l, 3 + l, prm["T_wall"][0]), (3 + ny - 1 + l, 3 + ny - 1 - l, prm["T_wall"][1])]:
            assert abs(u_g[g] + u_g[m]) < 1e-15 and abs(p_g[g] - p_g[m]) < 1e-15
            assert abs((T_g[g] - Tw) + (T_g[m] - Tw)) < 1e-15
            assert abs(rho_g[g] - p_g[m] / (R_GAS * (2 * Tw - T_g[m]))) < 1e-15
    conv, visc = o.rhs_parts()
    mu_y = prm["mu_ref"] * d / prm["T_ref"]
    low = slice(0, 8)
    assert np.abs(visc[1, 0, low, 0] - mu_y * c).max() < 1e-10 * abs(mu_y * c)
    mu = prm["mu_ref"] * T / prm["T_ref"]
    VE = u * mu_y * c + mu * c * c + CP / prm["Pr"] * mu_y * d
    assert np.abs(visc[4, 0, low, 0] - VE[low]).max() < 1e-10 * np.abs(VE).max()
    assert np.abs(conv).max() < 1e-13 * p.max() * ny


def test_wall_node_dirichlet_override_after_every_stage(ob):
    """S1: after every RK stage the wall node has rho u = rho v = rho w = 0 and rho E = rho c_v T_w (rho evolves)."""
    wl = W.config4_sbli(16, 12, 4, Lx=4.0)
    p = dict(wl.params, bc=[W.BC_PERIODIC] * 2 + [W.BC_WALL_NODE] * 2 + [W.BC_PERIODIC] * 2, weno_enable=0,
             T_wall=[1.3, 0.9], dt_fixed=1e-3)
    w0 = W.random_periodic(16, 12, 4, seed=21).state()           # slipping, non-isothermal wall rows to start with
    o = ob.Oracle(wl.grid, wl.x, wl.y, wl.z, p)
    o.set_state(w0)
    o.step(1)
    w = o.get_state()
    for j, Tw in ((0, 1.3), (-1, 0.9)):
        assert np.abs(w[1:4, :, j, :]).max() == 0.0
        assert np.abs(w[4, :, j, :] - w[0, :, j, :] * CV * Tw).max() < 1e-15 * np.abs(w[4]).max()
        assert np.abs(w[0, :, j, :] - w0[0, :, j, :]).max() > 1e-6            # the density of the wall row does evolve
    assert np.abs(w[1, :, 1, :]).max() > 0.0                                   # the first interior row is free


# ------------------------------------------------------------------ (c) shock generator ghosts, S1 / PAPER.md:146
def test_shock_generator_ghost_rows_and_residual(ob):
    """Uniform free stream below a SHOCKGEN top boundary.  The ghost rows hold the free stream for x < x_shock and the
    oblique-shock post state (values of SURVEY S1, pinned from the jump conditions by P10) for x >= x_shock.  Hence the
    inviscid central residual is 0 wherever the stencil sees free stream only, and where the ghosts hold the post state
    it is the split form (P2) of the y-derivative across a jump (g_post - g_fs) A_j / h_y(j), A_j = sum_{l >= ny - j} a_l."""
    M = 2.28
    nx, ny = 40, 16
    x = np.linspace(0.0, 4.0, nx)
    y = np.linspace(0.0, 1.5, ny)
    xs = 0.5 * (x[19] + x[20])
    bc = [W.BC_EXTRAP, W.BC_EXTRAP, W.BC_EXTRAP, W.BC_SHOCKGEN, W.BC_PERIODIC, W.BC_PERIODIC]
    prm = W.default_params(Rgas=R_GAS, viscous_enable=0, fs=[1.0, M, 0.0, 0.0, 1.0], shock_angle_deg=8.0, x_shock=xs, bc=bc)
    grid = dict(nx=nx, ny=ny, nz=1, len=[4.0, 1.5, 1.0])
    o = ob.Oracle(grid, x, y, np.zeros(1), prm)
    one = np.ones((1, ny, nx))
    o.set_state(W.prim_to_cons(one, M * one, 0 * one, 0 * one, one / GAM, GAM))
    post = dict(rho=1.395939, u=2.091408, v=-0.293928, T=1.147604)          # SURVEY S1 closed-form values (c_1 = 1)
    rho_g, u_g, v_g, w_g, p_g, T_g = prim_of(o.ghosted()[:, 3])            # [ny+6][nx+6]
    for l in (1, 2, 3):
        row = 3 + ny - 1 + l
        left = slice(3, 3 + 20)
        right = slice(3 + 20, 3 + nx)
        assert np.abs(rho_g[row, left] - 1.0).max() < 1e-15 and np.abs(u_g[row, left] - M).max() < 1e-15
        assert np.abs(v_g[row, left]).max() == 0.0 and np.abs(T_g[row, left] - 1.0).max() < 1e-15
        assert np.abs(rho_g[row, right] - post["rho"]).max() < 1e-6 and np.abs(u_g[row, right] - post["u"]).max() < 1e-6
        assert np.abs(v_g[row, right] - post["v"]).max() < 1e-6 and np.abs(T_g[row, right] - post["T"]).max() < 1e-6
    r = o.rhs()[:, 0]
    assert np.abs(r[:, : ny - 3, :]).max() == 0.0                            # rows whose stencil stays inside the grid
    assert np.abs(r[:, :, :20]).max() == 0.0                                  # columns in front of the jump
    # expected residual of the top rows behind the jump (exact post state from the oracle's P10-pinned routine)
    pp, _beta = ob.shock_state(prm)
    a = [3 / 4, -3 / 20, 1 / 60]
    hy, _ = o.metrics(1)
    fs = dict(rho=1.0, u=M, v=0.0, w=0.0, p=1.0 / GAM)
    ps = dict(rho=pp[0], u=pp[1], v=pp[2], w=pp[3], p=pp[0] * R_GAS * pp[4])
    for s_ in (fs, ps):
        s_["H"] = GAM / (GAM - 1.0) * s_["p"] / s_["rho"] + 0.5 * (s_["u"] ** 2 + s_["v"] ** 2 + s_["w"] ** 2)
    for j in range(ny - 3, ny):
        A = sum(a[l - 1] for l in range(ny - j, 4))
        exp = np.zeros(5)
        for m, key in enumerate([None, "u", "v", "w", "H"]):
            ph = (lambda s_: 1.0) if key is None else (lambda s_, key=key: s_[key])
            dl = lambda g: g(ps) - g(fs)                  # jump of a product between the post state and the free stream
            rho, vn, phi = fs["rho"], fs["v"], ph(fs)
            split = 0.25 * (dl(lambda s_: s_["rho"] * s_["v"] * ph(s_)) + rho * dl(lambda s_: s_["v"] * ph(s_))
                            + vn * dl(lambda s_: s_["rho"] * ph(s_)) + phi * dl(lambda s_: s_["rho"] * s_["v"])
                            + rho * vn * dl(ph) + rho * phi * dl(lambda s_: s_["v"]) + vn * phi * dl(lambda s_: s_["rho"]))
            exp[m] = -split * A / hy[j]
        exp[2] -= (ps["p"] - fs["p"]) * A / hy[j]
        got = r[:, j, 24:]                                # columns whose x-stencil sees post-state ghosts only
        for m in range(5):
            assert np.abs(got[m] - exp[m]).max() < 1e-12 * max(1.0, abs(exp[m])), (j, m, got[m][:3], exp[m])
    assert abs(r[2, ny - 1, 30]) > 0.05                    # and the jump is really there


def test_inflow_frozen_and_corner_fill_order(ob):
    """INFLOW_FROZEN ghosts keep plane 0 of the state given to set_state, also after stepping (A16); edge ghosts follow
    the fill order x -> y -> z: the (x < 0, y < 0) corner of a node wall is the wall reflection of the x-ghost."""
    wl = W.config4_sbli(24, 16, 4, Lx=6.0)
    o = ob.Oracle(wl.grid, wl.x, wl.y, wl.z, wl.params)
    w0 = wl.state()
    o.set_state(w0)
    o.step(2)
    wg = o.ghosted()
    ny = wl.grid["ny"]
    for l in (1, 2, 3):
        assert np.array_equal(wg[:, 3:-3, 3:-3, 3 - l], w0[:, :, :, 0])
    w1 = o.get_state()
    assert np.abs(w1[:, :, :, 0] - w0[:, :, :, 0]).max() > 0.0             # the boundary node itself evolves
    for l in (1, 2, 3):                                                     # outflow: zeroth-order copy of the last node
        assert np.array_equal(wg[:, 3:-3, 3:-3, 3 + wl.grid["nx"] - 1 + l], w1[:, :, :, -1])
    # corner (i = -1, j = -2): reflection about wall node 0 of the x-ghost (i = -1, j = +2) = frozen inflow at j = 2
    Tw = wl.params["T_wall"][0]
    src = w0[:, 1, 2, 0]
    rho, u, v, w_, p, T = prim_of(src[:, None])
    Tg = 2 * Tw - T
    rg = p / (R_GAS * Tg)
    exp = np.array([rg, -rg * u, -rg * v, -rg * w_, p / (GAM - 1) + 0.5 * rg * (u * u + v * v + w_ * w_)])[:, 0]
    assert np.abs(wg[:, 3 + 1, 3 - 2, 3 - 1] - exp).max() < 1e-14 * np.abs(exp).max()
    # z is filled last over the extended x and y ranges: periodic copy of the (ghost-filled) plane
    assert np.array_equal(wg[:, 3 - 1], wg[:, 3 + wl.grid["nz"] - 1])


# ------------------------------------------------------------------ (d) Sutherland's law
def test_sutherland_law_through_prims(ob):
    """mu / mu_ref = (T/T_ref)^(3/2) (T_ref + S) / (T + S) (Sutherland's law): exactly 1 at T_ref, the
    closed form at T_ref/2 and 2 T_ref, and -- for air, T_ref = 273.15 K, mu_ref = 1.716e-5 Pa s, S = 110.4 K -- the
    tabulated viscosity of air at 546.3 K (2.87e-5 Pa s) and 136.6 K (0.947e-5 Pa s) within the law's 2 % accuracy."""
    n = 3
    S = 110.4 / 273.15
    prm = W.default_params(Rgas=R_GAS, visc_model=W.VISC_SUTHERLAND, mu_ref=1.716e-5, T_ref=1.0, suth_S=S)
    grid = dict(nx=n, ny=1, nz=1, len=[1.0, 1.0, 1.0])
    T = np.array([0.5, 1.0, 2.0]).reshape(1, 1, n)
    rho = np.ones_like(T)
    o = ob.Oracle(grid, np.arange(n) / n, np.zeros(1), np.zeros(1), prm)
    o.set_state(W.prim_to_cons(rho, 0 * T, 0 * T, 0 * T, rho * R_GAS * T, GAM))
    mu = o.prims()[8].ravel() / 1.716e-5
    assert abs(mu[1] - 1.0) < 1e-15
    assert abs(mu[2] - 2 ** 1.5 * (1 + S) / (2 + S)) < 1e-14 and abs(mu[2] * 1.716e-5 / 2.87e-5 - 1) < 0.02
    assert abs(mu[0] - 0.5 ** 1.5 * (1 + S) / (0.5 + S)) < 1e-14 and abs(mu[0] * 1.716e-5 / 0.947e-5 - 1) < 0.02
    # power law for comparison: (T/T_ref)^0.76
    prm2 = dict(prm, visc_model=W.VISC_POWER, visc_exp=0.76)
    o2 = ob.Oracle(grid, np.arange(n) / n, np.zeros(1), np.zeros(1), prm2)
    o2.set_state(W.prim_to_cons(rho, 0 * T, 0 * T, 0 * T, rho * R_GAS * T, GAM))
    assert np.abs(o2.prims()[8].ravel() / 1.716e-5 - np.array([0.5, 1.0, 2.0]) ** 0.76).max() < 1e-14


# ------------------------------------------------------------------ (e) shock sensor on a manufactured field, Eq. 8
def test_sensor_manufactured_field_all_nine_gradients(ob):
    """theta = max(-div u / sqrt(div^2 + |curl u|^2 + eps), 0) (Eq. 8 with reading G1) on a periodic
    velocity field whose nine gradients are all non-zero, against the sympy expression, on a grid stretched in y."""
    import sympy as sp
    x, y, z = sp.symbols("x y z")
    vel = [sp.Rational(3, 10) * sp.sin(x + 2 * y) * sp.cos(z) + sp.Rational(1, 5) * sp.cos(y - z),
           sp.Rational(1, 4) * sp.cos(2 * x - z) * sp.sin(y) + sp.Rational(1, 5) * sp.sin(x + z),
           sp.Rational(1, 5) * sp.sin(x - y) * sp.sin(2 * z) + sp.Rational(3, 10) * sp.cos(x + y)]
    X = [x, y, z]
    div = sum(sp.diff(vel[i], X[i]) for i in range(3))
    curl = [sp.diff(vel[2], y) - sp.diff(vel[1], z), sp.diff(vel[0], z) - sp.diff(vel[2], x), sp.diff(vel[1], x) - sp.diff(vel[0], y)]
    eps = sp.Rational(1, 20)
    f = sp.lambdify((x, y, z), vel + [div] + curl, "numpy")
    n = 32
    L = 2 * np.pi
    xs = L * np.arange(n) / n
    ys = xs + 0.2 * np.sin(xs)
    prm = W.default_params(Rgas=R_GAS, weno_enable=1, sensor_eps=float(eps), sensor_threshold=0.4)
    grid = dict(nx=n, ny=n, nz=n, len=[L, L, L])
    Z, Y, Xg = np.meshgrid(xs, ys, xs, indexing="ij")
    u, v, w, dv, cx, cy, cz = [np.broadcast_to(np.asarray(a, dtype=float), Xg.shape) for a in f(Xg, Y, Z)]
    for g in (cx, cy, cz):
        assert np.abs(g).max() > 0.2                                        # every vorticity component matters
    exact = np.maximum(-dv / np.sqrt(dv * dv + cx * cx + cy * cy + cz * cz + float(eps)), 0.0)
    o = ob.Oracle(grid, xs, ys, xs, prm)
    one = np.ones_like(u)
    o.set_state(W.prim_to_cons(one, u, v, w, one / GAM, GAM))
    th, fl = o.sensor()
    assert np.abs(th - exact).max() < 1e-4
    assert exact.max() > 0.8 and (exact > 0.4).mean() > 0.01


# ------------------------------------------------------------------ (f) power of the body force, Eq. 1b-c
def test_forcing_power_term(ob):
    """Eq. 1b-c: f enters the x-momentum equation and f u_1 the total-energy equation."""
    wl = W.config3_channel(16, 12, 8)
    o1 = ob.Oracle(wl.grid, wl.x, wl.y, wl.z, wl.params)
    o0 = ob.Oracle(wl.grid, wl.x, wl.y, wl.z, dict(wl.params, forcing=0))
    w0 = wl.state()
    o1.set_state(w0)
    o0.set_state(w0)
    r1, r0 = o1.rhs(), o0.rhs()
    f = o1.diagnostics().forcing
    assert f > 0.0
    u = w0[1] / w0[0]
    hx, hy, hz = (o1.metrics(d)[0] for d in range(3))
    vol = hz[:, None, None] * hy[None, :, None] * hx[None, None, :]
    assert np.abs((r1[1] - r0[1]) - f).max() < 1e-13 * np.abs(r0[1]).max()
    assert np.abs((r1[4] - r0[4]) - f * u).max() < 1e-13 * np.abs(r0[4]).max()
    lhs = math.fsum(((r1[4] - r0[4]) * vol).ravel())
    rhs = f * math.fsum((u * vol).ravel())
    assert abs(lhs - rhs) < 1e-13 * abs(rhs)
    for m in (0, 2, 3):
        assert np.array_equal(r1[m], r0[m])


# ------------------------------------------------------------------ (g) Roe state, S6 step 1
def normal_shock(Ms, rho1=1.0, p1=1.0 / GAM):
    """State behind a shock of Mach number Ms running in +x into gas at rest (normal-shock relations)."""
    c1 = math.sqrt(GAM * p1 / rho1)
    s = Ms * c1
    rr = (GAM + 1) * Ms * Ms / ((GAM - 1) * Ms * Ms + 2)
    pr = 1 + 2 * GAM / (GAM + 1) * (Ms * Ms - 1)
    return rho1 * rr, s * (1 - 1 / rr), p1 * pr, s


def cons(rho, vel, p):
    return np.array([rho, rho * vel[0], rho * vel[1], rho * vel[2], p / (GAM - 1) + 0.5 * rho * float(np.dot(vel, vel))])


@pytest.mark.parametrize("d", [0, 1, 2])
def test_roe_state_property_U(ob, d):
    """Roe's property U: with the sqrt(rho)-weighted state, R Lambda L (w_b - w_a) = F(w_b) - F(w_a) for ANY two states.
    An arithmetic mean does not have it."""
    rng = np.random.default_rng(40 + d)
    for _ in range(5):
        ra, rb = rng.uniform(0.3, 3.0, 2)
        ua, ubv = rng.uniform(-1, 1, 3), rng.uniform(-1, 1, 3)
        pa, pb = rng.uniform(0.3, 3.0, 2)
        wa, wb = cons(ra, ua, pa), cons(rb, ubv, pb)
        Ha, Hb = (wa[4] + pa) / ra, (wb[4] + pb) / rb
        ubar, Hbar = ob.roe_state(ra, ua, Ha, rb, ubv, Hb)
        Lm, Rm, lam = ob.eigen(d, GAM, ubar, Hbar)
        lhs = Rm @ np.diag(lam) @ Lm @ (wb - wa)
        rhs = H.euler_flux(wb, d, GAM) - H.euler_flux(wa, d, GAM)
        assert np.abs(lhs - rhs).max() < 1e-12 * np.abs(rhs).max()
        # the arithmetic mean fails the same identity by orders of magnitude
        Lm2, Rm2, lam2 = ob.eigen(d, GAM, 0.5 * (ua + ubv), 0.5 * (Ha + Hb))
        assert np.abs(Rm2 @ np.diag(lam2) @ Lm2 @ (wb - wa) - rhs).max() > 1e-4 * np.abs(rhs).max()


@pytest.mark.parametrize("order", [5, 3])
@pytest.mark.parametrize("d", [0, 1, 2])
def test_weno_flux_at_a_moving_shock_and_a_contact(ob, d, order):
    """End to end through the oracle's WENO flux (every interface WENO).  Two uniform states that satisfy the
    Rankine-Hugoniot conditions of a shock of speed s: by property U the jump lies in ONE characteristic field of the
    Roe matrix, the other four fields are constant across the stencil, and the Lax-Friedrichs WENO flux at the jump is
      F = (F_a + F_b)/2 - alpha (w_b - w_a)/2,   alpha = max over the stencil of |u_n + c|
    (the upwind candidate stencils are smooth; the others are weighted ~ (eps/beta)^2 ~ 1e-10).  With a wrong average
    the other fields see a jump too and add their own dissipation.  A stationary contact gives exactly (0, p, 0, 0, 0)."""
    n = 24
    rho2, u2, p2, s = normal_shock(3.0)
    xs = np.arange(n) / n
    bc = [W.BC_PERIODIC] * 6
    bc[2 * d] = bc[2 * d + 1] = W.BC_EXTRAP
    prm = W.default_params(Rgas=R_GAS, viscous_enable=0, weno_enable=1, sensor_threshold=-1.0, sensor_eps=1.0, bc=bc, weno_order=order)
    nn = [1, 1, 1]
    nn[d] = n
    coords = [np.zeros(1)] * 3
    coords[d] = xs
    grid = dict(nx=nn[0], ny=nn[1], nz=nn[2], len=[1.0, 1.0, 1.0])
    shape = (nn[2], nn[1], nn[0])
    left = (np.arange(n) < n // 2).reshape(shape)
    vel = [np.zeros(shape), np.zeros(shape), np.zeros(shape)]
    vel[d] = np.where(left, u2, 0.0)
    vel[(d + 1) % 3] = np.full(shape, 0.37)                                   # a uniform transverse velocity rides along
    o = ob.Oracle(grid, *coords, prm)
    o.set_state(W.prim_to_cons(np.where(left, rho2, 1.0), vel[0], vel[1], vel[2], np.where(left, p2, 1.0 / GAM), GAM))
    r = o.rhs().reshape(5, n)
    va, vb = np.zeros(3), np.zeros(3)
    va[d], vb[d] = u2, 0.0
    va[(d + 1) % 3] = vb[(d + 1) % 3] = 0.37
    wa, wb = cons(rho2, va, p2), cons(1.0, vb, 1.0 / GAM)
    Fa, Fb = H.euler_flux(wa, d, GAM), H.euler_flux(wb, d, GAM)
    assert np.abs((Fb - Fa) - s * (wb - wa)).max() < 1e-12 * np.abs(Fa).max()          # Rankine-Hugoniot holds
    alpha = max(abs(u2 + math.sqrt(GAM * p2 / rho2)), 1.0)
    Fhat = 0.5 * (Fa + Fb) - 0.5 * alpha * (wb - wa)
    h = 1.0 / n
    ia = n // 2 - 1
    scale = np.abs(Fa).max() / h
    assert np.abs(r[:, ia] + (Fhat - Fa) / h).max() < 1e-7 * scale
    assert np.abs(r[:, ia + 1] + (Fb - Fhat) / h).max() < 1e-7 * scale
    rest = np.delete(r, [ia, ia + 1], axis=1)
    assert np.abs(rest).max() < 1e-7 * scale
    # stationary contact: rho jumps, u = 0, p equal
    zero = np.zeros(shape)
    o.set_state(W.prim_to_cons(np.where(left, 2.5, 0.4), zero, zero, zero, np.full(shape, 0.7), GAM))
    assert np.abs(o.rhs()).max() < 1e-13 * 0.7 / h


# ------------------------------------------------------------------ statistics
def stats_field(nx, ny, nz, A, seedless=True):
    """rho = rho0 (1 + D cos z), u = U(y) + A sin x cos z, v = C sin x cos z, w = 0.2, T = T0(y) + B cos 2x on
    equispaced periodic x, z: every x-z node mean below is exact (trigonometric sums below the Nyquist limit)."""
    L = 2 * np.pi
    x, z = L * np.arange(nx) / nx, L * np.arange(nz) / nz
    y = np.linspace(-0.9, 0.9, ny)
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    rho0, D, C_, B = 1.3, 0.2, 0.15, 0.1
    U, T0 = 1.0 - Y ** 2, 1.0 + 0.3 * Y
    rho = rho0 * (1 + D * np.cos(Z))
    u = U + A * np.sin(X) * np.cos(Z)
    v = C_ * np.sin(X) * np.cos(Z)
    w = 0.2 + 0 * X
    T = T0 + B * np.cos(2 * X)
    grid = dict(nx=nx, ny=ny, nz=nz, len=[L, 1.8, L])
    Uy, T0y = 1.0 - y ** 2, 1.0 + 0.3 * y
    exact = dict(rho=rho0 + 0 * y, u=Uy, v=0 * y, w=0.2 + 0 * y, p=R_GAS * rho0 * T0y, T=T0y, rho_u=rho0 * Uy, rho_v=0 * y,
                 rho_w=0.2 * rho0 + 0 * y, rho_T=rho0 * T0y, rho_uu=rho0 * (Uy ** 2 + A * A / 4), rho_vv=rho0 * C_ * C_ / 4 + 0 * y,
                 rho_ww=0.04 * rho0 + 0 * y, rho_uv=rho0 * A * C_ / 4 + 0 * y, TT=T0y ** 2 + B * B / 2, mu=0.02 * T0y)
    return grid, (x, y, z), W.prim_to_cons(rho, u, v, w, rho * R_GAS * T, GAM), exact


STAT_ORDER = ["rho", "u", "v", "w", "p", "T", "mu", "rho_u", "rho_v", "rho_w", "rho_T", "rho_uu", "rho_vv", "rho_ww", "rho_uv", "TT"]


def test_statistics_closed_form_plane_means(ob):
    """averaging over the homogeneous directions and time.  Plane means of a trigonometric field are
    known in closed form; the time average of two samples is their mean; Favre u~ = mean(rho u) / mean(rho)."""
    prm = W.default_params(Rgas=R_GAS, mu_ref=0.02, T_ref=1.0, visc_exp=1.0, bc=[W.BC_PERIODIC] * 2 + [W.BC_EXTRAP] * 2 + [W.BC_PERIODIC] * 2)
    grid, (x, y, z), w1, ex1 = stats_field(16, 7, 12, A=0.3)
    _g, _c, w2, ex2 = stats_field(16, 7, 12, A=0.5)
    o = ob.Oracle(grid, x, y, z, prm)
    o.set_state(w1)
    o.stats_accumulate()
    st, n = o.stats_read()
    assert n == 1
    for m, key in enumerate(STAT_ORDER):
        assert np.abs(st[m] - ex1[key]).max() < 1e-14 * max(1.0, np.abs(ex1[key]).max()), key
    o.set_state(w2)
    o.stats_accumulate()
    st, n = o.stats_read()
    assert n == 2
    for m, key in enumerate(STAT_ORDER):
        assert np.abs(st[m] - 0.5 * (ex1[key] + ex2[key])).max() < 1e-14 * max(1.0, np.abs(ex1[key]).max()), key
    # Favre-averaged velocity and the density-scaled normal stress rho u''u'' = mean(rho uu) - mean(rho u)^2 / mean(rho)
    assert np.abs(st[7] / st[0] - ex1["u"]).max() < 1e-14
    tau = st[11] - st[7] ** 2 / st[0]
    assert np.abs(tau - 1.3 * 0.5 * (0.3 ** 2 + 0.5 ** 2) / 4).max() < 1e-14
    o.stats_reset()
    assert o.stats_read()[1] == 0 and np.abs(o.stats_read()[0]).max() == 0.0


# ------------------------------------------------------------------ characteristic boundaries, PAPER.md:126 (8.f rank 3)
def ycolumn(ob, ny, bc_lo, bc_hi, rho, v, p, u=None, Tw=1.0, visc=0):
    y = np.arange(ny) / ny
    bc = [W.BC_PERIODIC] * 2 + [bc_lo, bc_hi] + [W.BC_PERIODIC] * 2
    prm = W.default_params(Rgas=R_GAS, viscous_enable=visc, T_wall=[Tw, Tw], bc=bc)
    return column(ob, y, prm, rho, np.zeros(ny) if u is None else u, v, np.zeros(ny), p), y


def test_characteristic_faces_reduce_to_the_LODI_relations(ob):
    """Poinsot & Lele's locally one-dimensional inviscid relations in primitive variables, gas at rest plus a small
    smooth perturbation (amplitude 1e-6: the conservative-variable form of S8 and the primitive form differ at second
    order).  With L_1 = (v - c)(p_y - rho c v_y), L_5 = (v + c)(p_y + rho c v_y):
      non-reflecting top (L_1 = 0):  rho_t = -L_5 / (2 c^2),  (rho v)_t = -L_5 / (2 c)    -> both from p_y + rho c v_y
      reflecting wall (L_5 = L_1):   rho_t = -L_1 / c^2 = (p_y - rho c v_y) / c,  (rho v)_t = 0
    with one-sided second-order differences at the boundary node."""
    ny = 32
    eps = 1e-6
    yy = np.arange(ny) / ny
    rho = 1.0 + eps * np.sin(3 * yy + 0.4)
    v = eps * np.cos(2 * yy + 0.1)
    v[0] = 0.0                                             # no slip at the wall node
    p = 1.0 / GAM + eps * np.sin(5 * yy - 0.3)
    o, y = ycolumn(ob, ny, W.BC_WALL_CHAR, W.BC_OUTFLOW, rho, v, p, Tw=float(p[0] / (R_GAS * rho[0])))
    conv, _ = o.rhs_parts()
    conv = conv[:, 0, :, 0]
    h = 1.0 / ny
    # top node: backward differences
    py = (3 * p[-1] - 4 * p[-2] + p[-3]) / (2 * h)
    vy = (3 * v[-1] - 4 * v[-2] + v[-3]) / (2 * h)
    c_ = math.sqrt(GAM * p[-1] / rho[-1])
    L5 = (v[-1] + c_) * (py + rho[-1] * c_ * vy)
    assert abs(conv[0, -1] + L5 / (2 * c_ * c_)) < 1e-4 * abs(L5)
    assert abs(conv[2, -1] + L5 / (2 * c_)) < 1e-4 * abs(L5)
    # wall node: forward differences
    py = (-3 * p[0] + 4 * p[1] - p[2]) / (2 * h)
    vy = (-3 * v[0] + 4 * v[1] - v[2]) / (2 * h)
    c_ = math.sqrt(GAM * p[0] / rho[0])
    L1 = (v[0] - c_) * (py - rho[0] * c_ * vy)
    assert abs(conv[0, 0] + L1 / (c_ * c_)) < 1e-4 * abs(L1)
    assert abs(conv[2, 0]) < 1e-6 * abs(L1)
    # a uniform state gives exactly zero at both faces
    one = np.ones(ny)
    o2, _ = ycolumn(ob, ny, W.BC_WALL_CHAR, W.BC_OUTFLOW, one, 0 * one, one / GAM)
    assert np.abs(o2.rhs()).max() < 1e-13


def run_pulse(ob, bc_lo, bc_hi, centre, direction, T_end, ny=96):
    """Acoustic pulse of amplitude 1e-3 in gas at rest (rho = c = 1) running up (+1) or down (-1) the column."""
    amp = 1e-3
    yy = np.arange(ny) / ny
    g = amp * np.exp(-((yy - centre) / 0.05) ** 2)
    o, y = ycolumn(ob, ny, bc_lo, bc_hi, 1.0 + g, direction * g, 1.0 / GAM + g)
    while o.diagnostics().time < T_end:
        o.step(1)
    w = o.get_state()[:, 0, :, 0]
    return yy, w, amp


def test_nonreflecting_top_lets_a_pulse_out(ob):
    yy, w, amp = run_pulse(ob, W.BC_EXTRAP, W.BC_OUTFLOW, 0.7, +1, 0.6)
    assert np.abs(w[0][8:] - 1.0).max() < 0.05 * amp                       # nothing comes back from the top


def test_characteristic_wall_reflects_a_pulse(ob):
    """A pulse running down to the characteristic wall comes back with the same sign and (nearly) the same amplitude,
    the wall pressure peaks near twice the incident amplitude, and the wall row stays at rest (rigid, isothermal)."""
    yy, w, amp = run_pulse(ob, W.BC_WALL_CHAR, W.BC_OUTFLOW, 0.3, -1, 0.6)
    rho, v = w[0], w[2] / w[0]
    k = int(np.argmax(np.abs(rho - 1.0)))
    assert 0.2 < yy[k] < 0.4 and 0.85 * amp < rho[k] - 1.0 < 1.1 * amp       # back where it started, same sign
    assert v[k] > 0.8 * amp                                                  # and now running upwards
    assert w[2][0] == 0.0
