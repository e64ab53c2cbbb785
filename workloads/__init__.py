"""Seeded synthetic inputs for the five BASELINE.json configs.

This module holds NO arithmetic of the method: it only builds grids, parameter dicts and
initial conservative states w[5][nz][ny][nx] with NumPy.  It is the one module that both
the CUDA binding's callers and the CPU oracle's callers use (the oracle and the CUDA path
never import each other).  Every random field uses one `np.random.default_rng([seed, k])`
stream per z-plane k, so a slab [k0, k1) of a big case can be generated on its own.

The paper's own workloads are turbulent fields from long runs that need
data not available here; these inputs take their shapes, physics and grid structure and
stand in for them.
"""
from dataclasses import dataclass, field

import numpy as np

BC_PERIODIC, BC_WALL_STAG, BC_WALL_NODE, BC_INFLOW, BC_OUTFLOW, BC_SHOCKGEN, BC_EXTRAP, BC_WALL_CHAR = range(8)
VISC_POWER, VISC_SUTHERLAND = 0, 1


def default_params(**over) -> dict:
    p = dict(gamma=1.4, Pr=0.72, Rgas=1.0 / 1.4, mu_ref=1e-3, T_ref=1.0, visc_exp=0.76, suth_S=110.4 / 273.15,
             sensor_threshold=0.5, sensor_eps=1.0, T_wall=[1.0, 1.0], y_wall=[-1.0, 1.0],
             fs=[1.0, 0.0, 0.0, 0.0, 1.0], shock_angle_deg=0.0, x_shock=0.0, cfl=0.5, dt_fixed=0.0,
             visc_model=VISC_POWER, order=6, weno_enable=0, forcing=0, viscous_enable=1,
             bc=[BC_PERIODIC] * 6, weno_order=5)
    for k, v in over.items():
        if k not in p:
            raise KeyError(k)
        p[k] = v
    return p


@dataclass
class Workload:
    name: str
    grid: dict                      # nx, ny, nz, len[3]
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    params: dict
    steps: int
    seed: int
    state_fn: object = field(repr=False, default=None)   # (k0, k1) -> w[5][k1-k0][ny][nx]

    @property
    def shape(self):
        return (5, self.grid["nz"], self.grid["ny"], self.grid["nx"])

    @property
    def npoints(self):
        return self.grid["nx"] * self.grid["ny"] * self.grid["nz"]

    def state(self, k0=0, k1=None):
        """Initial conservative state for z-planes [k0, k1)."""
        return self.state_fn(k0, self.grid["nz"] if k1 is None else k1)

    def slab(self, k0, k1, halo=3, keep_forcing=False):
        """A sub-workload holding planes [k0-halo, k1+halo) (periodic wrap in z): the oracle's
        RHS on its middle planes equals the full problem's (every stencil has z-radius 3).
        Forcing is a global reduction, so it is switched off unless keep_forcing."""
        nz = self.grid["nz"]
        ks = [(k % nz) for k in range(k0 - halo, k1 + halo)]
        g = dict(self.grid)
        g["nz"] = len(ks)
        g["len"] = list(self.grid["len"])
        dz = self.z[1] - self.z[0] if nz > 1 else self.grid["len"][2]
        zz = self.z[0] + dz * np.arange(k0 - halo, k1 + halo)
        g["len"][2] = dz * len(ks)
        parts = [self.state_fn(k, k + 1) for k in ks]
        w = np.concatenate(parts, axis=1)
        p = dict(self.params)
        if not keep_forcing:
            p["forcing"] = 0
        sub = Workload(self.name + f"_slab{k0}_{k1}", g, self.x, self.y, zz, p, 0, self.seed,
                       state_fn=lambda a, b, w=w: w[:, a:b].copy())
        return sub


def prim_to_cons(rho, u, v, w, p, gamma):
    out = np.empty((5,) + rho.shape)
    out[0] = rho
    out[1] = rho * u
    out[2] = rho * v
    out[3] = rho * w
    out[4] = p / (gamma - 1.0) + 0.5 * rho * (u * u + v * v + w * w)
    return out


def _noise(seed, k, shape, amp):
    rng = np.random.default_rng([seed, k])
    return rng.uniform(-amp, amp, size=(3,) + shape)


# ---------------------------------------------------------------------------------------------
# config 1: Taylor-Green vortex
def config1_tgv(n=32, seed=1001, steps=20, weno=1) -> Workload:
    gamma, M0 = 1.4, 0.1
    p0 = 1.0 / (gamma * M0 * M0)
    L = 2.0 * np.pi
    x = L * np.arange(n) / n
    params = default_params(Rgas=p0, mu_ref=1.0 / 1600.0, T_ref=1.0, weno_enable=weno, sensor_threshold=0.5,
                            sensor_eps=1.0, cfl=0.5)
    grid = dict(nx=n, ny=n, nz=n, len=[L, L, L])

    def state(k0, k1):
        Z, Y, X = np.meshgrid(x[k0:k1], x, x, indexing="ij")
        u = np.sin(X) * np.cos(Y) * np.cos(Z)
        v = -np.cos(X) * np.sin(Y) * np.cos(Z)
        w = np.zeros_like(u)
        p = p0 + (1.0 / 16.0) * (np.cos(2 * X) + np.cos(2 * Y)) * (np.cos(2 * Z) + 2.0)
        rho = p / (p0 * 1.0)
        for i, k in enumerate(range(k0, k1)):
            nz_ = _noise(seed, k, (n, n), 1e-3)
            u[i] += nz_[0]
            v[i] += nz_[1]
            w[i] += nz_[2]
        return prim_to_cons(rho, u, v, w, p, gamma)

    return Workload("tgv", grid, x, x.copy(), x.copy(), params, steps, seed, state)


# ---------------------------------------------------------------------------------------------
# config 2: decaying compressible isotropic turbulence
def config2_isotropic(n=128, seed=1002, steps=100, mt=0.6, k0=4.0, threshold=0.5) -> Workload:
    gamma = 1.4
    L = 2.0 * np.pi
    x = L * np.arange(n) / n
    lam = 2.0 / k0
    uprime = mt / np.sqrt(3.0)
    params = default_params(Rgas=1.0 / gamma, mu_ref=uprime * lam / 100.0, T_ref=1.0, weno_enable=1,
                            sensor_threshold=threshold, sensor_eps=(uprime / lam) ** 2, cfl=0.5)
    grid = dict(nx=n, ny=n, nz=n, len=[L, L, L])
    cache = {}

    def velocity():
        if "u" in cache:
            return cache["u"]
        rng = np.random.default_rng(seed)
        a = rng.standard_normal((3, n, n, n))
        ah = np.fft.fftn(a, axes=(1, 2, 3))
        kk = np.fft.fftfreq(n, 1.0 / n)
        KZ, KY, KX = np.meshgrid(kk, kk, kk, indexing="ij")
        K = np.stack([KX, KY, KZ])            # component order u,v,w <-> kx,ky,kz
        k2 = KX ** 2 + KY ** 2 + KZ ** 2
        nyq = (np.abs(KX) == n // 2) | (np.abs(KY) == n // 2) | (np.abs(KZ) == n // 2)
        k2s = np.where(k2 == 0, 1.0, k2)
        ah = ah - K * (K * ah).sum(axis=0) / k2s                     # solenoidal projection
        kmag = np.sqrt(k2s)
        E = kmag ** 4 * np.exp(-2.0 * (kmag / k0) ** 2)
        ah = ah * np.sqrt(E) / kmag
        ah[:, (k2 == 0) | nyq] = 0.0
        u = np.real(np.fft.ifftn(ah, axes=(1, 2, 3)))
        u *= mt / np.sqrt((u ** 2).sum(axis=0).mean())
        cache["u"] = u
        return u

    def state(ka, kb):
        u = velocity()[:, ka:kb]
        rho = np.ones_like(u[0])
        p = rho * (1.0 / gamma) * 1.0
        return prim_to_cons(rho, u[0], u[1], u[2], p, gamma)

    return Workload("isotropic", grid, x, x.copy(), x.copy(), params, steps, seed, state)


# ---------------------------------------------------------------------------------------------
# configs 3 and 5: supersonic plane channel, staggered isothermal walls, bulk forcing
def tanh_nodes(ny, b=1.7):
    eta = -1.0 + (2.0 * np.arange(1, ny + 1) - 1.0) / ny
    return np.tanh(b * eta) / np.tanh(b)


def erf_nodes(ny, a=1.4):
    """Error-function wall-normal mapping of the paper's channel, staggered nodes (the walls at y = -1, +1
    fall half-way between a ghost and the first node): y_j = erf(a eta_j) / erf(a), eta_j = -1 + (2j - 1)/ny.
    a = 1.4 gives the paper's spacing ratio: centre / wall = exp(a^2) = 7.1 (its dy+ = 0.8 ... 5.7 at ny = 256)."""
    from math import erf
    eta = -1.0 + (2.0 * np.arange(1, ny + 1) - 1.0) / ny
    return np.array([erf(a * e) for e in eta]) / erf(a)


def _smooth121(a, axis, periodic, passes=4):
    for _ in range(passes):
        if periodic:
            a = 0.25 * np.roll(a, 1, axis) + 0.5 * a + 0.25 * np.roll(a, -1, axis)
        else:
            lo = np.take(a, [0], axis)
            hi = np.take(a, [-1], axis)
            ap = np.concatenate([lo, a, hi], axis)
            n = a.shape[axis]
            a = 0.25 * np.take(ap, range(0, n), axis) + 0.5 * a + 0.25 * np.take(ap, range(2, n + 2), axis)
    return a


def config3_channel(nx=256, ny=128, nz=128, seed=1003, steps=200, name="channel", smooth=False, zcopies=1) -> Workload:
    """zcopies > 1: a box zcopies times as long in z (nz and L_z scaled together, so the spacing stays; every plane has
    its own noise stream): the weak-scaling input of the z-slab decomposition, nz planes per GPU (Fig. 11)."""
    gamma = 1.4
    nz = nz * zcopies
    Lx, Lz = 6.0 * np.pi, 2.0 * np.pi * zcopies
    x = Lx * np.arange(nx) / nx
    z = Lz * np.arange(nz) / nz
    y = tanh_nodes(ny)
    ub, Reb = 1.5, 6000.0
    params = default_params(Rgas=1.0 / gamma, mu_ref=2.0 * 1.0 * ub * 1.0 / Reb, T_ref=1.0, weno_enable=0,
                            forcing=1, T_wall=[1.0, 1.0], y_wall=[-1.0, 1.0], cfl=0.5,
                            bc=[BC_PERIODIC, BC_PERIODIC, BC_WALL_STAG, BC_WALL_STAG, BC_PERIODIC, BC_PERIODIC])
    grid = dict(nx=nx, ny=ny, nz=nz, len=[Lx, 2.0, Lz])
    env = (1.0 - y * y)[None, :, None]

    def state(k0, k1):
        nk = k1 - k0
        u = np.empty((nk, ny, nx))
        v = np.empty_like(u)
        w = np.empty_like(u)
        for i, k in enumerate(range(k0, k1)):
            nz_ = _noise(seed, k, (ny, nx), 0.1 * ub)
            if smooth:   # in-plane (1,2,1)/4 smoothing only, so that slabs stay independent
                for c in range(3):
                    nz_[c] = _smooth121(_smooth121(nz_[c], 1, True), 0, False)
                nz_ *= 0.1 * ub / np.abs(nz_).max()
            u[i] = 1.5 * ub * env[0] + nz_[0] * env[0]
            v[i] = nz_[1] * env[0]
            w[i] = nz_[2] * env[0]
        rho = np.ones_like(u)
        p = rho * (1.0 / gamma) * 1.0
        return prim_to_cons(rho, u, v, w, p, gamma)

    return Workload(name, grid, x, y, z, params, steps, seed, state)


def config6_channel_paper(nx=128, ny=64, nz=64, seed=1006, steps=20) -> Workload:
    """The paper's OWN channel numerics (section 8.f rank 2 of SURVEY.md) on the seeded channel input: fourth-order
    central flux and viscous terms, Sutherland's law, error-function wall-normal
    mapping, M_b = 1.5, Re_b = 14725."""
    wl = config3_channel(nx, ny, nz, seed, steps, name="channel_paper")
    wl.y = erf_nodes(ny)
    Reb = 14725.0
    wl.params.update(order=4, visc_model=VISC_SUTHERLAND, mu_ref=2.0 * 1.0 * 1.5 * 1.0 / Reb, T_ref=1.0,
                     suth_S=110.4 / 273.15)
    return wl


def config5_channel_big(nx=1024, ny=512, nz=512, seed=1005, steps=50, smooth=False, zcopies=1) -> Workload:
    return config3_channel(nx, ny, nz, seed, steps, name="channel_big", smooth=smooth, zcopies=zcopies)


# ---------------------------------------------------------------------------------------------
# config 4: oblique shock / laminar boundary layer interaction
def sinh_nodes(ny, Ly=8.0, b=3.5):
    eta = np.arange(ny) / (ny - 1.0)
    return Ly * np.sinh(b * eta) / np.sinh(b)


def _similarity_profile(M, gamma, Pr, Tw, expo=0.76, eta_max=12.0, n=4801):
    """Compressible laminar flat-plate similarity solution (Illingworth-Levy variables):
    (C f'')' + f f'' = 0, (C g'/Pr)' + f g' + C (gamma-1) M^2 f''^2 = 0, C = g^(expo-1),
    f(0)=f'(0)=0, g(0)=Tw, f'(inf)=g(inf)=1; RK4 shooting on (f''(0), g'(0))."""
    h = eta_max / (n - 1)

    def rhs(s):
        f, fp, a, g, bq = s          # a = C f'', bq = C g'/Pr
        C = g ** (expo - 1.0)
        fpp = a / C
        return np.array([fp, fpp, -f * fpp, bq * Pr / C, -f * bq * Pr / C - C * (gamma - 1.0) * M * M * fpp * fpp])

    def shoot(p0, p1, keep=False):
        s = np.array([0.0, 0.0, p0, Tw, p1])
        out = [s.copy()] if keep else None
        for _ in range(n - 1):
            k1 = rhs(s)
            k2 = rhs(s + 0.5 * h * k1)
            k3 = rhs(s + 0.5 * h * k2)
            k4 = rhs(s + h * k3)
            s = s + h / 6.0 * (k1 + 2 * k2 + 2 * k3 + k4)
            if keep:
                out.append(s.copy())
        return (np.array(out) if keep else s)

    pr = np.array([0.47 * Tw ** (expo - 1.0), 0.0])
    for _ in range(40):
        s = shoot(pr[0], pr[1])
        res = np.array([s[1] - 1.0, s[3] - 1.0])
        if np.abs(res).max() < 1e-12:
            break
        J = np.empty((2, 2))
        for c in range(2):
            dp = pr.copy()
            e = 1e-6 * max(1.0, abs(pr[c]))
            dp[c] += e
            s2 = shoot(dp[0], dp[1])
            J[:, c] = (np.array([s2[1] - 1.0, s2[3] - 1.0]) - res) / e
        pr = pr - np.linalg.solve(J, res)
    sol = shoot(pr[0], pr[1], keep=True)
    eta = np.linspace(0.0, eta_max, n)
    fp, g = sol[:, 1], sol[:, 3]
    yphys = np.concatenate([[0.0], np.cumsum(0.5 * (g[1:] + g[:-1]) * h)])   # y ~ int g d(eta)
    return eta, yphys, fp, g


def config7_boundary_layer(nx=256, ny=64, nz=32, seed=1007, steps=20, Lx=24.0, Ly=8.0, Lz=4.0) -> Workload:
    """Spatially developing supersonic boundary layer in the paper's set-up:
    M_inf = 2, characteristic wave treatment at the no-slip wall at the recovery temperature, non-reflecting upper and
    outflow boundaries, central flux only; the digital-filter inflow needs the database of ref. [40] (absent): frozen
    laminar similarity inflow plus seeded fluctuations stand in for it."""
    return config4_sbli(nx, ny, nz, seed, steps, Lx, Ly, Lz, M=2.0, shock=False, name="boundary_layer")


def config4_sbli(nx=1024, ny=256, nz=128, seed=1004, steps=100, Lx=48.0, Ly=8.0, Lz=4.0, M=2.28, shock=True, name="sbli", zcopies=1) -> Workload:
    """zcopies > 1: a span zcopies times as wide (nz and L_z scaled together): the weak-scaling input of the z-slab mode."""
    gamma, Pr = 1.4, 0.72
    nz, Lz = nz * zcopies, Lz * zcopies
    x = Lx * np.arange(nx) / (nx - 1.0)
    z = Lz * np.arange(nz) / nz
    y = sinh_nodes(ny, Ly)
    Tr = 1.0 + 0.5 * (gamma - 1.0) * Pr ** (1.0 / 3.0) * M * M     # recovery temperature
    x_shock = 17.4 * Lx / 48.0
    params = default_params(Rgas=1.0 / gamma, mu_ref=M / 1.0e4, T_ref=1.0, weno_enable=1, sensor_threshold=0.5,
                            sensor_eps=(M / 1.0) ** 2, T_wall=[Tr, Tr], fs=[1.0, M, 0.0, 0.0, 1.0],
                            shock_angle_deg=8.0, x_shock=x_shock, cfl=0.5,
                            bc=[BC_INFLOW, BC_OUTFLOW, BC_WALL_NODE, BC_SHOCKGEN, BC_PERIODIC, BC_PERIODIC])
    if not shock:
        params.update(weno_enable=0, shock_angle_deg=0.0, bc=[BC_INFLOW, BC_OUTFLOW, BC_WALL_CHAR, BC_OUTFLOW, BC_PERIODIC, BC_PERIODIC])
    grid = dict(nx=nx, ny=ny, nz=nz, len=[Lx, Ly, Lz])
    cache = {}

    def base():
        if "b" in cache:
            return cache["b"]
        _eta, yp, fp, g = _similarity_profile(M, gamma, Pr, Tr)
        y99 = np.interp(0.99, fp, yp)
        ys = yp / y99                                   # u(y=1) = 0.99 u_inf
        u1 = M * np.interp(y, ys, fp, right=1.0)
        T1 = np.interp(y, ys, g, right=1.0)
        u1[0] = 0.0
        T1[0] = Tr
        p_inf = 1.0 / gamma
        # oblique-shock ratios for the initial field (input recipe; closed form of gas dynamics)
        phi = np.deg2rad(8.0)
        lo, hi = np.arcsin(1.0 / M), np.deg2rad(60.0)
        fun = lambda be: 2.0 / np.tan(be) * (M * M * np.sin(be) ** 2 - 1.0) / (M * M * (gamma + np.cos(2 * be)) + 2.0)
        for _ in range(200):
            mid = 0.5 * (lo + hi)
            if fun(mid) < np.tan(phi):
                lo = mid
            else:
                hi = mid
        beta = 0.5 * (lo + hi)
        Mn = M * np.sin(beta)
        pr_ = 1.0 + 2.0 * gamma / (gamma + 1.0) * (Mn * Mn - 1.0)
        rr_ = (gamma + 1.0) * Mn * Mn / ((gamma - 1.0) * Mn * Mn + 2.0)
        X, Y = np.meshgrid(x, y, indexing="xy")          # [ny][nx]
        behind = ((X - x_shock) > (Ly - Y) / np.tan(beta)) & shock
        u = np.broadcast_to(u1[:, None], X.shape).copy()
        T = np.broadcast_to(T1[:, None], X.shape).copy()
        v = np.zeros_like(u)
        rho = (p_inf / ((1.0 / gamma) * T))
        p = np.full_like(u, p_inf)
        un = u * np.sin(beta)
        ut = u * np.cos(beta)
        un2 = un / rr_
        u_b = ut * np.cos(beta) + un2 * np.sin(beta)
        v_b = -ut * np.sin(beta) + un2 * np.cos(beta)
        u = np.where(behind, u_b, u)
        v = np.where(behind, v_b, v)
        rho = np.where(behind, rho * rr_, rho)
        p = np.where(behind, p * pr_, p)
        cache["b"] = (rho, u, v, p)
        return cache["b"]

    def state(k0, k1):
        rho2, u2, v2, p2 = base()
        nk = k1 - k0
        rho = np.broadcast_to(rho2, (nk, ny, nx)).copy()
        p = np.broadcast_to(p2, (nk, ny, nx)).copy()
        u = np.broadcast_to(u2, (nk, ny, nx)).copy()
        v = np.broadcast_to(v2, (nk, ny, nx)).copy()
        w = np.zeros_like(u)
        env = np.exp(-y * y)[:, None]
        env[0:1] = 0.0                                   # wall node untouched
        for i, k in enumerate(range(k0, k1)):
            nz_ = _noise(seed, k, (ny, nx), 0.05 * M)
            u[i] += nz_[0] * env
            v[i] += nz_[1] * env
            w[i] += nz_[2] * env
        return prim_to_cons(rho, u, v, w, p, gamma)

    return Workload(name, grid, x, y, z, params, steps, seed, state)


# ---------------------------------------------------------------------------------------------
# generic seeded smooth/rough periodic states for unit tests
def random_periodic(nx, ny, nz, seed=7, params=None, amp=0.2, stretched_y=False) -> Workload:
    gamma = 1.4
    L = 2.0 * np.pi
    x = L * np.arange(nx) / nx
    y = L * np.arange(ny) / ny
    z = L * np.arange(nz) / nz
    if stretched_y:
        y = y + 0.3 * np.sin(y) * (L / (2 * np.pi)) * 0.5
    p_ = params or default_params(Rgas=1.0 / gamma, mu_ref=5e-3)
    grid = dict(nx=nx, ny=ny, nz=nz, len=[L, L, L])

    def state(k0, k1):
        out = np.empty((5, k1 - k0, ny, nx))
        for i, k in enumerate(range(k0, k1)):
            rng = np.random.default_rng([seed, k])
            r = rng.uniform(-amp, amp, size=(5, ny, nx))
            rho = 1.0 + r[0]
            p = (1.0 + r[4]) / gamma
            out[:, i] = prim_to_cons(rho, 0.5 + r[1], r[2], -0.3 + r[3], p, gamma)
        return out

    return Workload("random_periodic", grid, x, y, z, p_, 1, seed, state)
