"""Independent NumPy helpers for the oracle pins (textbook formulas only)."""
import numpy as np

A = {2: [0.5], 4: [2 / 3, -1 / 12], 6: [3 / 4, -3 / 20, 1 / 60]}


def ddx(f, axis, h, order=6):
    """Textbook periodic central first derivative on a uniform grid."""
    out = np.zeros_like(f)
    for l, a in enumerate(A[order], start=1):
        out += a * (np.roll(f, -l, axis) - np.roll(f, l, axis))
    return out / h


def cons_to_prim(w, gamma):
    rho = w[0]
    u, v, ww = w[1] / rho, w[2] / rho, w[3] / rho
    p = (gamma - 1) * (w[4] - 0.5 * rho * (u * u + v * v + ww * ww))
    return rho, u, v, ww, p


def euler_flux(wv, d, gamma):
    """Physical Euler flux of the conservative 5-vector along direction d (works with complex input)."""
    rho = wv[0]
    vel = [wv[1] / rho, wv[2] / rho, wv[3] / rho]
    p = (gamma - 1) * (wv[4] - 0.5 * rho * (vel[0] ** 2 + vel[1] ** 2 + vel[2] ** 2))
    F = [rho * vel[d], wv[1] * vel[d], wv[2] * vel[d], wv[3] * vel[d], (wv[4] + p) * vel[d]]
    F[1 + d] = F[1 + d] + p
    return np.array(F)


def exact_riemann(rl, ul, pl, rr, ur, pr, gamma, xi):
    """Exact solution of the 1-D Riemann problem (Toro, ch. 4) sampled at xi = x/t."""
    g = gamma
    cl, cr = np.sqrt(g * pl / rl), np.sqrt(g * pr / rr)

    def fk(p, rk, pk, ck):
        if p > pk:
            Ak, Bk = 2 / ((g + 1) * rk), (g - 1) / (g + 1) * pk
            return (p - pk) * np.sqrt(Ak / (p + Bk)), np.sqrt(Ak / (p + Bk)) * (1 - 0.5 * (p - pk) / (p + Bk))
        return 2 * ck / (g - 1) * ((p / pk) ** ((g - 1) / (2 * g)) - 1), 1 / (rk * ck) * (p / pk) ** (-(g + 1) / (2 * g))

    p = 0.5 * (pl + pr)
    for _ in range(100):
        f1, d1 = fk(p, rl, pl, cl)
        f2, d2 = fk(p, rr, pr, cr)
        dp = (f1 + f2 + ur - ul) / (d1 + d2)
        p = max(p - dp, 1e-12)
        if abs(dp) < 1e-15 * p:
            break
    f1, _ = fk(p, rl, pl, cl)
    f2, _ = fk(p, rr, pr, cr)
    us = 0.5 * (ul + ur) + 0.5 * (f2 - f1)
    rho = np.empty_like(xi)
    u = np.empty_like(xi)
    pp = np.empty_like(xi)
    for i, s in enumerate(xi):
        if s <= us:   # left of contact
            if p > pl:
                sl = ul - cl * np.sqrt((g + 1) / (2 * g) * p / pl + (g - 1) / (2 * g))
                if s < sl:
                    rho[i], u[i], pp[i] = rl, ul, pl
                else:
                    rho[i] = rl * ((p / pl + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * p / pl + 1))
                    u[i], pp[i] = us, p
            else:
                shl = ul - cl
                csl = cl * (p / pl) ** ((g - 1) / (2 * g))
                stl = us - csl
                if s < shl:
                    rho[i], u[i], pp[i] = rl, ul, pl
                elif s > stl:
                    rho[i], u[i], pp[i] = rl * (p / pl) ** (1 / g), us, p
                else:
                    c = 2 / (g + 1) * (cl + (g - 1) / 2 * (ul - s))
                    u[i] = 2 / (g + 1) * (cl + (g - 1) / 2 * ul + s)
                    rho[i] = rl * (c / cl) ** (2 / (g - 1))
                    pp[i] = pl * (c / cl) ** (2 * g / (g - 1))
        else:
            if p > pr:
                sr = ur + cr * np.sqrt((g + 1) / (2 * g) * p / pr + (g - 1) / (2 * g))
                if s > sr:
                    rho[i], u[i], pp[i] = rr, ur, pr
                else:
                    rho[i] = rr * ((p / pr + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * p / pr + 1))
                    u[i], pp[i] = us, p
            else:
                shr = ur + cr
                csr = cr * (p / pr) ** ((g - 1) / (2 * g))
                strr = us + csr
                if s > shr:
                    rho[i], u[i], pp[i] = rr, ur, pr
                elif s < strr:
                    rho[i], u[i], pp[i] = rr * (p / pr) ** (1 / g), us, p
                else:
                    c = 2 / (g + 1) * (cr - (g - 1) / 2 * (ur - s))
                    u[i] = 2 / (g + 1) * (-cr + (g - 1) / 2 * ur + s)
                    rho[i] = rr * (c / cr) ** (2 / (g - 1))
                    pp[i] = pr * (c / cr) ** (2 * g / (g - 1))
    return rho, u, pp, p, us
