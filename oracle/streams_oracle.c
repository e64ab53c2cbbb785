/*
 * streams_oracle.c -- TEST INFRASTRUCTURE, not the product (see streams_oracle.h).
 *
 * A plain CPU implementation of what the hot path computes, step by step in the order
 * and notation of DESIGN.md S0..S11, each step citing the passage of PAPER.md it follows.
 * Ghost nodes (width 3) ARE stored here (arrays [.][nz+6][ny+6][nx+6]) so that every
 * stencil is a plain loop; there is no blocking, fusion or reordering.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (oracle/build.py).
 *
 * Pins (tests/test_oracle_pins.py, tests/test_oracle_pins_bc.py, -m "not gpu"): coefficient tables against
 * polynomial exactness; flux form against the telescoped pair form; bitwise free-stream
 * preservation; discrete conservation; kinetic-energy identity; RK3 amplification
 * polynomial, Butcher tableau and order (coefficients read from tests/golden/); eigenvectors
 * against a complex-step Jacobian; Roe state against Roe's property U and a moving-shock
 * closed form of the WENO flux; WENO5 linear limit and order; Sod tube against the exact
 * Riemann solution; oblique-shock jump conditions; metric and viscous operators against
 * sympy-manufactured fields; wall ghost rules (staggered and node) against hand-built ghosts
 * and the closed forms of linear profiles continued through the wall; Dirichlet wall-node
 * override; shock-generator ghost rows and the residual they produce; frozen-inflow ghosts
 * and the x -> y -> z corner fill order; Sutherland's law; the sensor of Eq. 8 on a
 * manufactured field with all nine velocity gradients; the f u_1 power of Eq. 1c.
 * PARITY UNPINNED (choices of DESIGN.md only, nothing in the paper fixes them): the VALUES of
 * the sensor threshold / regulariser, the non-reflecting outflow formula A13 beyond "uniform
 * flow gives 0, a pulse leaves" (P14), nearest-node theta at non-periodic ghosts (A17), and the
 * CFL definition S10 beyond its closed form on a uniform state (P13).
 */
#include "streams_oracle.h"

#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NG 3
#define NV 5
enum { Q_RHO = 0, Q_U, Q_V, Q_W, Q_P, Q_T, Q_H, Q_C, Q_MU, NQ };

struct oracle_ctx {
  oracle_grid g;
  oracle_params p;
  int n[3];        /* interior nodes per direction                     */
  int N[3];        /* with ghosts                                      */
  size_t sd[3];    /* strides of the ghost-filled arrays               */
  size_t NP;       /* nodes of one ghost-filled field                  */
  size_t np;       /* interior nodes                                   */
  int L;
  double a[4], b[4]; /* a[l], b[l], l = 1..L         */
  double* xc[3];   /* ghost-extended coordinates, xc[d][i+NG]          */
  double* h[3];    /* first index-derivative of the coordinate (S2)    */
  double* gm[3];   /* second index-derivative of the coordinate (S2)   */
  double* w;       /* interior state [5][nz][ny][nx]                   */
  double* wg;      /* ghost-filled conservative state                  */
  double* q;       /* ghost-filled primitives [NQ]                     */
  double* dd[3];   /* ghost-extended d u_k / d x_k for the mixed terms */
  double* theta;   /* sensor at interior nodes                         */
  double* inflow;  /* [5][nz][ny] plane captured at set_state          */
  double* Rprev;   /* R of the previous RK stage                       */
  double* Rcur;
  double post[5];  /* shock generator post-shock primitive state       */
  double* stat_sum;  /* [ORC_NSTAT][ny] running sums of the plane means (statistics) */
  long long stat_n;
  int has_state;
  long long step;
  double time, dt, force;
  long long weno_if[3], tot_if[3];
};

/* ------------------------------------------------------------------------------------ */
/* central coefficients: "standard coefficients for central finite-difference            */
/* approximations" of the first (a_l) and second (b_l) derivative       */
int oracle_coeffs(int order, double a[3], double b[3]) {
  a[0] = a[1] = a[2] = b[0] = b[1] = b[2] = 0.0;
  switch (order) {
    case 2: a[0] = 1.0 / 2.0; b[0] = 1.0; return 1;
    case 4: a[0] = 2.0 / 3.0; a[1] = -1.0 / 12.0; b[0] = 4.0 / 3.0; b[1] = -1.0 / 12.0; return 2;
    case 6:
      a[0] = 3.0 / 4.0; a[1] = -3.0 / 20.0; a[2] = 1.0 / 60.0;
      b[0] = 3.0 / 2.0; b[1] = -3.0 / 20.0; b[2] = 1.0 / 90.0;
      return 3;
    default: return 0;
  }
}

int oracle_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

static inline size_t GI(const oracle_ctx* c, int i, int j, int k) {
  return ((size_t)(k + NG) * c->N[1] + (size_t)(j + NG)) * c->N[0] + (size_t)(i + NG);
}
static inline size_t II(const oracle_ctx* c, int i, int j, int k) {
  return ((size_t)k * c->n[1] + (size_t)j) * c->n[0] + (size_t)i;
}
static inline int imod(int a, int n) { int r = a % n; return r < 0 ? r + n : r; }

/* viscosity law: power law mu ~ T^0.76 (north_star) or Sutherland */
static double visc(const oracle_params* p, double T) {
  if (p->visc_model == ORC_VISC_SUTHERLAND)
    return p->mu_ref * pow(T / p->T_ref, 1.5) * (p->T_ref + p->suth_S) / (T + p->suth_S);
  return p->mu_ref * pow(T / p->T_ref, p->visc_exp);
}

/* ------------------------------------------------------------------------------------ */
/* S1: shock generator -- inviscid oblique shock for the deflection angle */
int oracle_shock_state(const oracle_params* p, double post[5], double* beta_out) {
  const double gam = p->gamma;
  const double rho1 = p->fs[0], u1 = p->fs[1], T1 = p->fs[4];
  const double c1 = sqrt(gam * p->Rgas * T1);
  const double M = u1 / c1;
  const double phi = p->shock_angle_deg * M_PI / 180.0;
  if (!(M > 1.0) || !(phi > 0.0)) return ORC_EINVAL;
  /* theta-beta-M relation: tan(phi) = 2 cot(beta) (M^2 sin^2 beta - 1) / (M^2 (gamma + cos 2beta) + 2);
     weak solution = the root between the Mach angle and the angle of maximum deflection */
  const double blo0 = asin(1.0 / M);
  double bmax = blo0, fmax = -1.0;
  for (int s = 0; s <= 100000; ++s) {
    double be = blo0 + (0.5 * M_PI - blo0) * s / 100000.0;
    double f = 2.0 / tan(be) * (M * M * sin(be) * sin(be) - 1.0) / (M * M * (gam + cos(2.0 * be)) + 2.0);
    if (f > fmax) { fmax = f; bmax = be; }
  }
  if (tan(phi) > fmax) return ORC_EINVAL; /* detached */
  double lo = blo0, hi = bmax;
  for (int it = 0; it < 200; ++it) {
    double be = 0.5 * (lo + hi);
    double f = 2.0 / tan(be) * (M * M * sin(be) * sin(be) - 1.0) / (M * M * (gam + cos(2.0 * be)) + 2.0);
    if (f < tan(phi)) lo = be; else hi = be;
  }
  const double beta = 0.5 * (lo + hi);
  const double Mn = M * sin(beta);
  const double pr = 1.0 + 2.0 * gam / (gam + 1.0) * (Mn * Mn - 1.0);
  const double rr = (gam + 1.0) * Mn * Mn / ((gam - 1.0) * Mn * Mn + 2.0);
  /* shock line runs down-stream and downwards: tangent (cos b, -sin b), normal (sin b, cos b) */
  const double un1 = u1 * sin(beta), ut = u1 * cos(beta);
  const double un2 = un1 / rr;
  post[0] = rho1 * rr;
  post[1] = ut * cos(beta) + un2 * sin(beta);
  post[2] = -ut * sin(beta) + un2 * cos(beta);
  post[3] = p->fs[3];
  post[4] = T1 * pr / rr;
  if (beta_out) *beta_out = beta;
  return ORC_OK;
}

static void prim_to_cons(const oracle_params* p, const double pr[5] /*rho,u,v,w,T*/, double wc[5]) {
  const double cv = p->Rgas / (p->gamma - 1.0);
  wc[0] = pr[0];
  wc[1] = pr[0] * pr[1];
  wc[2] = pr[0] * pr[2];
  wc[3] = pr[0] * pr[3];
  wc[4] = pr[0] * (cv * pr[4] + 0.5 * (pr[1] * pr[1] + pr[2] * pr[2] + pr[3] * pr[3])); /* E = cv T + u.u/2 */
}

/* S1 isothermal no-slip reflection: u -> -u, T -> 2 Tw - T, p -> p, rho = p / (R T) */
static void reflect_wall(const oracle_params* p, double Tw, const double ws[5], double wgst[5]) {
  const double gam = p->gamma;
  const double rho = ws[0], u = ws[1] / rho, v = ws[2] / rho, w = ws[3] / rho;
  const double pres = (gam - 1.0) * (ws[4] - 0.5 * rho * (u * u + v * v + w * w));
  const double T = pres / (rho * p->Rgas);
  const double Tg = 2.0 * Tw - T;
  const double rg = pres / (p->Rgas * Tg);
  wgst[0] = rg;
  wgst[1] = -rg * u;
  wgst[2] = -rg * v;
  wgst[3] = -rg * w;
  wgst[4] = pres / (gam - 1.0) + 0.5 * rg * (u * u + v * v + w * w);
}

/* ------------------------------------------------------------------------------------ */
static int is_periodic(const oracle_ctx* c, int d) { return c->p.bc[2 * d] == ORC_BC_PERIODIC; }

static int check_params(const oracle_grid* g, const oracle_params* p) {
  if (g->nx < 1 || g->ny < 1 || g->nz < 1) return 0;
  if (!(p->gamma > 1.0) || !(p->Rgas > 0.0) || !(p->Pr > 0.0)) return 0;
  if (p->order != 2 && p->order != 4 && p->order != 6) return 0;
  if (p->weno_enable && !(p->sensor_eps > 0.0)) return 0;
  if (p->weno_order != 0 && p->weno_order != 3 && p->weno_order != 5) return 0;
  const int n[3] = {g->nx, g->ny, g->nz};
  for (int d = 0; d < 3; ++d) {
    int lo = p->bc[2 * d], hi = p->bc[2 * d + 1];
    if ((lo == ORC_BC_PERIODIC) != (hi == ORC_BC_PERIODIC)) return 0;
    if (lo != ORC_BC_PERIODIC && n[d] < 4) return 0;
    if (lo == ORC_BC_PERIODIC && !(g->len[d] > 0.0)) return 0;
    for (int s = 0; s < 2; ++s) {
      int b = p->bc[2 * d + s];
      if (b < 0 || b > ORC_BC_WALL_CHAR) return 0;
      if ((b == ORC_BC_WALL_STAG || b == ORC_BC_WALL_NODE) && d != 1) return 0;
      if (b == ORC_BC_WALL_CHAR && !(d == 1 && s == 0)) return 0;
      if (b == ORC_BC_INFLOW && !(d == 0 && s == 0)) return 0;
      if (b == ORC_BC_OUTFLOW && !((d == 0 || d == 1) && s == 1)) return 0;
      if (b == ORC_BC_SHOCKGEN && !(d == 1 && s == 1)) return 0;
    }
  }
  return 1;
}

int oracle_create(const oracle_grid* g, const double* x, const double* y, const double* z,
                  const oracle_params* p, oracle_ctx** out) {
  if (!g || !p || !x || !y || !z || !out) return ORC_EINVAL;
  if (!check_params(g, p)) return ORC_EINVAL;
  oracle_ctx* c = (oracle_ctx*)calloc(1, sizeof(oracle_ctx));
  c->g = *g; c->p = *p;
  c->n[0] = g->nx; c->n[1] = g->ny; c->n[2] = g->nz;
  for (int d = 0; d < 3; ++d) c->N[d] = c->n[d] + 2 * NG;
  c->sd[0] = 1; c->sd[1] = (size_t)c->N[0]; c->sd[2] = (size_t)c->N[0] * c->N[1];
  c->NP = (size_t)c->N[0] * c->N[1] * c->N[2];
  c->np = (size_t)c->n[0] * c->n[1] * c->n[2];
  double aa[3], bb[3];
  c->L = oracle_coeffs(p->order, aa, bb);
  for (int l = 1; l <= 3; ++l) { c->a[l] = aa[l - 1]; c->b[l] = bb[l - 1]; }
  if (p->bc[3] == ORC_BC_SHOCKGEN && oracle_shock_state(p, c->post, NULL) != ORC_OK) { free(c); return ORC_EINVAL; }

  /* S1 ghost coordinates, S2 metrics */
  const double* xin[3] = {x, y, z};
  for (int d = 0; d < 3; ++d) {
    const int n = c->n[d];
    for (int i = 1; i < n; ++i) if (!(xin[d][i] > xin[d][i - 1])) { free(c); return ORC_EINVAL; }
    c->xc[d] = (double*)calloc((size_t)c->N[d], sizeof(double));
    c->h[d] = (double*)calloc((size_t)n, sizeof(double));
    c->gm[d] = (double*)calloc((size_t)n, sizeof(double));
    double* xc = c->xc[d] + NG;
    for (int i = 0; i < n; ++i) xc[i] = xin[d][i];
    for (int l = 1; l <= NG; ++l) {
      for (int s = 0; s < 2; ++s) {
        const int gi = s == 0 ? -l : n - 1 + l;
        const int bc = p->bc[2 * d + s];
        if (bc == ORC_BC_PERIODIC) {
          const int r = imod(gi, n);
          const int qq = (gi - r) / n;            /* number of periods crossed */
          xc[gi] = xin[d][r] + qq * g->len[d];
        } else if (bc == ORC_BC_WALL_STAG) {      /* mirrored about the wall plane */
          const int m = s == 0 ? l - 1 : n - l;
          xc[gi] = 2.0 * p->y_wall[s] - xin[d][m];
        } else {                                   /* odd reflection about the boundary node */
          const int bn = s == 0 ? 0 : n - 1;
          const int m = s == 0 ? l : n - 1 - l;
          xc[gi] = 2.0 * xin[d][bn] - xin[d][m];
        }
      }
    }
    for (int i = 0; i < n; ++i) {
      double hh = 0.0, gg = 0.0;
      for (int l = 1; l <= c->L; ++l) {
        hh += c->a[l] * (xc[i + l] - xc[i - l]);
        gg += c->b[l] * ((xc[i + l] - xc[i]) - (xc[i] - xc[i - l]));
      }
      c->h[d][i] = hh; c->gm[d][i] = gg;
      if (!(hh > 0.0)) { free(c); return ORC_EINVAL; }
    }
  }
  c->w = (double*)calloc(NV * c->np, sizeof(double));
  c->wg = (double*)calloc(NV * c->NP, sizeof(double));
  c->q = (double*)calloc(NQ * c->NP, sizeof(double));
  for (int d = 0; d < 3; ++d) c->dd[d] = (double*)calloc(c->NP, sizeof(double));
  c->theta = (double*)calloc(c->np, sizeof(double));
  c->inflow = (double*)calloc((size_t)NV * c->n[1] * c->n[2], sizeof(double));
  c->Rprev = (double*)calloc(NV * c->np, sizeof(double));
  c->Rcur = (double*)calloc(NV * c->np, sizeof(double));
  c->stat_sum = (double*)calloc((size_t)ORC_NSTAT * c->n[1], sizeof(double));
  *out = c;
  return ORC_OK;
}

void oracle_destroy(oracle_ctx* c) {
  if (!c) return;
  for (int d = 0; d < 3; ++d) { free(c->xc[d]); free(c->h[d]); free(c->gm[d]); free(c->dd[d]); }
  free(c->w); free(c->wg); free(c->q); free(c->theta); free(c->inflow); free(c->Rprev); free(c->Rcur); free(c->stat_sum);
  free(c);
}

int oracle_set_state(oracle_ctx* c, const double* w) {
  if (!c || !w) return ORC_EINVAL;
  memcpy(c->w, w, NV * c->np * sizeof(double));
  /* S1 INFLOW_FROZEN: ghost planes keep the values of the first interior plane of the initial state */
  for (int v = 0; v < NV; ++v)
    for (int k = 0; k < c->n[2]; ++k)
      for (int j = 0; j < c->n[1]; ++j)
        c->inflow[((size_t)v * c->n[2] + k) * c->n[1] + j] = w[v * c->np + II(c, 0, j, k)];
  memset(c->Rprev, 0, NV * c->np * sizeof(double));
  c->has_state = 1; c->step = 0; c->time = 0.0; c->dt = 0.0; c->force = 0.0;
  return ORC_OK;
}

int oracle_get_state(oracle_ctx* c, double* w) {
  if (!c || !w) return ORC_EINVAL;
  if (!c->has_state) return ORC_ESTATE;
  memcpy(w, c->w, NV * c->np * sizeof(double));
  return ORC_OK;
}

int oracle_get_metrics(oracle_ctx* c, int d, double* h, double* g) {
  if (!c || d < 0 || d > 2) return ORC_EINVAL;
  for (int i = 0; i < c->n[d]; ++i) { if (h) h[i] = c->h[d][i]; if (g) g[i] = c->gm[d][i]; }
  return ORC_OK;
}

/* ------------------------------------------------------------------------------------ */
/* S1: ghost values, width 3, fill order x -> y -> z, each later direction over the full
 * extended range of the earlier ones (this defines the edge and corner ghosts).          */
static void fill_ghosts(oracle_ctx* c) {
  const oracle_params* p = &c->p;
  const size_t NP = c->NP;
  /* interior copy */
#pragma omp parallel for
  for (int k = 0; k < c->n[2]; ++k)
    for (int j = 0; j < c->n[1]; ++j)
      for (int i = 0; i < c->n[0]; ++i)
        for (int v = 0; v < NV; ++v) c->wg[v * NP + GI(c, i, j, k)] = c->w[v * c->np + II(c, i, j, k)];

  double fsc[5], postc[5];
  prim_to_cons(p, p->fs, fsc);
  prim_to_cons(p, c->post, postc);

  for (int d = 0; d < 3; ++d) {
    const int n = c->n[d];
    int lo[3], hi[3];
    for (int e = 0; e < 3; ++e) {
      if (e < d) { lo[e] = -NG; hi[e] = c->n[e] + NG; } else { lo[e] = 0; hi[e] = c->n[e]; }
    }
    const int e1 = (d + 1) % 3, e2 = (d + 2) % 3;
    for (int t2 = lo[e2]; t2 < hi[e2]; ++t2)
      for (int t1 = lo[e1]; t1 < hi[e1]; ++t1)
        for (int s = 0; s < 2; ++s)
          for (int l = 1; l <= NG; ++l) {
            int id[3]; id[e1] = t1; id[e2] = t2;
            const int gi = s == 0 ? -l : n - 1 + l;
            const int bc = p->bc[2 * d + s];
            double ws[5], wo[5];
            int src = 0;
            switch (bc) {
              case ORC_BC_PERIODIC: src = imod(gi, n); break;
              case ORC_BC_WALL_STAG: src = s == 0 ? l - 1 : n - l; break;
              case ORC_BC_WALL_NODE:
              case ORC_BC_WALL_CHAR: src = s == 0 ? l : n - 1 - l; break;
              default: src = s == 0 ? 0 : n - 1; break;
            }
            id[d] = src;
            const size_t so = GI(c, id[0], id[1], id[2]);
            for (int v = 0; v < NV; ++v) ws[v] = c->wg[v * NP + so];
            switch (bc) {
              case ORC_BC_WALL_STAG:
              case ORC_BC_WALL_NODE:
              case ORC_BC_WALL_CHAR: reflect_wall(p, p->T_wall[s], ws, wo); break;
              case ORC_BC_INFLOW:
                /* d == 0, s == 0: transverse indices are interior here because x is filled first */
                for (int v = 0; v < NV; ++v) wo[v] = c->inflow[((size_t)v * c->n[2] + id[2]) * c->n[1] + id[1]];
                break;
              case ORC_BC_SHOCKGEN: {
                /* d == 1, s == 1: piecewise-constant state, sharp jump at x_shock (A15) */
                const double xx = c->xc[0][id[0] + NG];
                for (int v = 0; v < NV; ++v) wo[v] = xx < p->x_shock ? fsc[v] : postc[v];
              } break;
              default: for (int v = 0; v < NV; ++v) wo[v] = ws[v]; break; /* periodic copy / zeroth-order extrapolation */
            }
            id[d] = gi;
            const size_t go = GI(c, id[0], id[1], id[2]);
            for (int v = 0; v < NV; ++v) c->wg[v * NP + go] = wo[v];
          }
  }
}

/* S3: primitives at every node including ghosts */
static void compute_prims(oracle_ctx* c) {
  const oracle_params* p = &c->p;
  const size_t NP = c->NP;
  const double gam = p->gamma;
#pragma omp parallel for
  for (long long o = 0; o < (long long)NP; ++o) {
    const double rho = c->wg[0 * NP + o];
    const double u = c->wg[1 * NP + o] / rho, v = c->wg[2 * NP + o] / rho, w = c->wg[3 * NP + o] / rho;
    const double rE = c->wg[4 * NP + o];
    const double pres = (gam - 1.0) * (rE - 0.5 * rho * (u * u + v * v + w * w));
    const double T = pres / (rho * p->Rgas);
    c->q[Q_RHO * NP + o] = rho;
    c->q[Q_U * NP + o] = u; c->q[Q_V * NP + o] = v; c->q[Q_W * NP + o] = w;
    c->q[Q_P * NP + o] = pres;
    c->q[Q_T * NP + o] = T;
    c->q[Q_H * NP + o] = (rE + pres) / rho;        /* H = E + p/rho */
    c->q[Q_C * NP + o] = sqrt(gam * pres / rho);
    c->q[Q_MU * NP + o] = visc(p, T);
  }
}

/* index-space first and second central differences of field f along direction d (S2 / table) */
static inline double D1(const oracle_ctx* c, const double* f, size_t o, int d) {
  const size_t s = c->sd[d];
  double r = 0.0;
  for (int l = 1; l <= c->L; ++l) r += c->a[l] * (f[o + l * s] - f[o - l * s]);
  return r;
}
static inline double D2(const oracle_ctx* c, const double* f, size_t o, int d) {
  const size_t s = c->sd[d];
  double r = 0.0;
  for (int l = 1; l <= c->L; ++l) r += c->b[l] * ((f[o + l * s] - f[o]) - (f[o] - f[o - l * s]));
  return r;
}

/* S4: shock sensor, Eq. 8 read as (div u)^2 + |curl u|^2 + (u0/L0)^2 under the root */
static void compute_theta(oracle_ctx* c) {
  const size_t NP = c->NP;
  const double* U[3] = {c->q + Q_U * NP, c->q + Q_V * NP, c->q + Q_W * NP};
#pragma omp parallel for
  for (int k = 0; k < c->n[2]; ++k)
    for (int j = 0; j < c->n[1]; ++j)
      for (int i = 0; i < c->n[0]; ++i) {
        const size_t o = GI(c, i, j, k);
        const int id[3] = {i, j, k};
        double G[3][3]; /* G[a][d] = d u_a / d x_d */
        for (int a = 0; a < 3; ++a)
          for (int d = 0; d < 3; ++d) G[a][d] = D1(c, U[a], o, d) / c->h[d][id[d]];
        const double div = G[0][0] + G[1][1] + G[2][2];
        const double ox = G[2][1] - G[1][2], oy = G[0][2] - G[2][0], oz = G[1][0] - G[0][1];
        const double den = sqrt(div * div + (ox * ox + oy * oy + oz * oz) + c->p.sensor_eps);
        const double th = -div / den;
        c->theta[II(c, i, j, k)] = th > 0.0 ? th : 0.0;
      }
}

/* theta at a (possibly ghost) index along direction d: periodic wrap, else nearest interior node (A17) */
static inline double theta_at(const oracle_ctx* c, int d, int id[3], int g) {
  int q[3] = {id[0], id[1], id[2]};
  const int n = c->n[d];
  if (is_periodic(c, d)) q[d] = imod(g, n); else q[d] = g < 0 ? 0 : (g > n - 1 ? n - 1 : g);
  return c->theta[II(c, q[0], q[1], q[2])];
}

/* interface f+1/2 (between nodes f and f+1 along d) is flagged iff any of the six WENO stencil
 * nodes f-2..f+3 has theta above the threshold (A6) */
static inline int iface_flag(const oracle_ctx* c, int d, int id[3], int f) {
  if (!c->p.weno_enable) return 0;
  double m = 0.0;
  for (int g = f - 2; g <= f + 3; ++g) { double t = theta_at(c, d, id, g); if (t > m) m = t; }
  return m > c->p.sensor_threshold;
}

/* ------------------------------------------------------------------------------------ */
/* S5: energy-preserving central flux, Eq. 6-7: o = offset of node i, interface i+1/2 */
static void central_flux(const oracle_ctx* c, int d, size_t o, int wall_plane, double F[5]) {
  const size_t NP = c->NP, s = c->sd[d];
  const double* rho = c->q + Q_RHO * NP;
  const double* un = c->q + (Q_U + d) * NP;
  const double* ph[4] = {c->q + Q_U * NP, c->q + Q_V * NP, c->q + Q_W * NP, c->q + Q_H * NP};
  const double* pr = c->q + Q_P * NP;
  double C[5] = {0, 0, 0, 0, 0}, P = 0.0;
  for (int l = 1; l <= c->L; ++l) {
    double sc[5] = {0, 0, 0, 0, 0}, sp = 0.0;
    for (int m = 0; m <= l - 1; ++m) {
      const size_t ia = o - m * s, ib = ia + l * s;
      /* (rho,u,phi)~ = 1/8 (rho_a+rho_b)(u_a+u_b)(phi_a+phi_b), Eq. 6; phi = 1 counts as (1+1) */
      const double ru = 0.25 * (rho[ia] + rho[ib]) * (un[ia] + un[ib]);
      sc[0] += ru;
      for (int v = 0; v < 4; ++v) sc[1 + v] += ru * (0.5 * (ph[v][ia] + ph[v][ib]));
      sp += 0.5 * (pr[ia] + pr[ib]);
    }
    for (int v = 0; v < 5; ++v) C[v] += 2.0 * c->a[l] * sc[v];
    P += 2.0 * c->a[l] * sp;
  }
  /* staggered wall plane: "convective fluxes are identically zero"; pressure kept */
  for (int v = 0; v < 5; ++v) F[v] = wall_plane ? 0.0 : C[v];
  F[1 + d] += P;
}

/* S6 step 6: WENO5 of Jiang & Shu (ref. [34]), epsilon = 1e-6, p = 2 */
double oracle_weno5(double a, double b, double cc, double d, double e) {
  const double q0 = (2.0 * a - 7.0 * b + 11.0 * cc) / 6.0;
  const double q1 = (-b + 5.0 * cc + 2.0 * d) / 6.0;
  const double q2 = (2.0 * cc + 5.0 * d - e) / 6.0;
  const double b0 = 13.0 / 12.0 * (a - 2.0 * b + cc) * (a - 2.0 * b + cc) + 0.25 * (a - 4.0 * b + 3.0 * cc) * (a - 4.0 * b + 3.0 * cc);
  const double b1 = 13.0 / 12.0 * (b - 2.0 * cc + d) * (b - 2.0 * cc + d) + 0.25 * (b - d) * (b - d);
  const double b2 = 13.0 / 12.0 * (cc - 2.0 * d + e) * (cc - 2.0 * d + e) + 0.25 * (3.0 * cc - 4.0 * d + e) * (3.0 * cc - 4.0 * d + e);
  const double eps = 1e-6;
  const double a0 = 0.1 / ((eps + b0) * (eps + b0));
  const double a1 = 0.6 / ((eps + b1) * (eps + b1));
  const double a2 = 0.3 / ((eps + b2) * (eps + b2));
  return (a0 * q0 + a1 * q1 + a2 * q2) / (a0 + a1 + a2);
}

/* Variant (A23): WENO3 of Jiang & Shu (ref. [34]) -- two candidate stencils {a,b}, {b,c} for the
 * interface right of b, linear weights 1/3, 2/3, smoothness (b-a)^2, (c-b)^2, same epsilon and exponent as the fifth-order one */
double oracle_weno3(double a, double b, double cc) {
  const double q0 = (-a + 3.0 * b) / 2.0;
  const double q1 = (b + cc) / 2.0;
  const double b0 = (b - a) * (b - a);
  const double b1 = (cc - b) * (cc - b);
  const double eps = 1e-6;
  const double a0 = (1.0 / 3.0) / ((eps + b0) * (eps + b0));
  const double a1 = (2.0 / 3.0) / ((eps + b1) * (eps + b1));
  return (a0 * q0 + a1 * q1) / (a0 + a1);
}

/* S6 step 2: left/right eigenvectors of dF_d/dw in conservative variables, row-major 5x5 */
void oracle_eigen(int d, double gam, const double ub[3], double Hb, double Lm[25], double Rm[25], double lam[5]) {
  const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
  const double q2 = ub[0] * ub[0] + ub[1] * ub[1] + ub[2] * ub[2];
  const double c2 = (gam - 1.0) * (Hb - 0.5 * q2);
  const double cs = sqrt(c2);
  const double b1 = (gam - 1.0) / c2, b2 = 0.5 * q2 * b1;
  const double un = ub[d];
  double nn[3] = {0, 0, 0}; nn[d] = 1.0;
  memset(Lm, 0, 25 * sizeof(double)); memset(Rm, 0, 25 * sizeof(double));
  /* rows of L */
  Lm[0 * 5 + 0] = 0.5 * (b2 + un / cs);
  for (int m = 0; m < 3; ++m) Lm[0 * 5 + 1 + m] = 0.5 * (-b1 * ub[m] - nn[m] / cs);
  Lm[0 * 5 + 4] = 0.5 * b1;
  Lm[1 * 5 + 0] = 1.0 - b2;
  for (int m = 0; m < 3; ++m) Lm[1 * 5 + 1 + m] = b1 * ub[m];
  Lm[1 * 5 + 4] = -b1;
  Lm[2 * 5 + 0] = -ub[t1]; Lm[2 * 5 + 1 + t1] = 1.0;
  Lm[3 * 5 + 0] = -ub[t2]; Lm[3 * 5 + 1 + t2] = 1.0;
  Lm[4 * 5 + 0] = 0.5 * (b2 - un / cs);
  for (int m = 0; m < 3; ++m) Lm[4 * 5 + 1 + m] = 0.5 * (-b1 * ub[m] + nn[m] / cs);
  Lm[4 * 5 + 4] = 0.5 * b1;
  /* columns of R */
  Rm[0 * 5 + 0] = 1.0; for (int m = 0; m < 3; ++m) Rm[(1 + m) * 5 + 0] = ub[m] - cs * nn[m]; Rm[4 * 5 + 0] = Hb - un * cs;
  Rm[0 * 5 + 1] = 1.0; for (int m = 0; m < 3; ++m) Rm[(1 + m) * 5 + 1] = ub[m];               Rm[4 * 5 + 1] = 0.5 * q2;
  Rm[(1 + t1) * 5 + 2] = 1.0; Rm[4 * 5 + 2] = ub[t1];
  Rm[(1 + t2) * 5 + 3] = 1.0; Rm[4 * 5 + 3] = ub[t2];
  Rm[0 * 5 + 4] = 1.0; for (int m = 0; m < 3; ++m) Rm[(1 + m) * 5 + 4] = ub[m] + cs * nn[m]; Rm[4 * 5 + 4] = Hb + un * cs;
  lam[0] = un - cs; lam[1] = un; lam[2] = un; lam[3] = un; lam[4] = un + cs;
}

/* S6 step 1: Roe state of two nodes a (lower) and b (upper): r = sqrt(rho_b / rho_a), square-root-of-density
 * weighted means of the velocity components and of the total enthalpy */
void oracle_roe_state(double rho_a, const double u_a[3], double H_a, double rho_b, const double u_b[3], double H_b,
                      double ubar[3], double* Hbar) {
  const double r = sqrt(rho_b / rho_a);
  for (int m = 0; m < 3; ++m) ubar[m] = (u_a[m] + r * u_b[m]) / (1.0 + r);
  *Hbar = (H_a + r * H_b) / (1.0 + r);
}

/* S6: characteristic-wise Lax-Friedrichs split WENO5 flux at interface i+1/2 */
static void weno_flux(const oracle_ctx* c, int d, size_t o, double F[5]) {
  const size_t NP = c->NP, s = c->sd[d];
  const double gam = c->p.gamma;
  const double* Q = c->q;
  const int w3 = c->p.weno_order == 3;
  /* 1. Roe state from nodes i, i+1 */
  const size_t oa = o, ob = o + s;
  const double ua[3] = {Q[Q_U * NP + oa], Q[Q_V * NP + oa], Q[Q_W * NP + oa]};
  const double ubn[3] = {Q[Q_U * NP + ob], Q[Q_V * NP + ob], Q[Q_W * NP + ob]};
  double ub[3], Hb;
  oracle_roe_state(Q[Q_RHO * NP + oa], ua, Q[Q_H * NP + oa], Q[Q_RHO * NP + ob], ubn, Q[Q_H * NP + ob], ub, &Hb);
  /* 2. eigenvectors */
  double Lm[25], Rm[25], lamb[5];
  oracle_eigen(d, gam, ub, Hb, Lm, Rm, lamb);
  /* 3. node states, physical Euler fluxes and their characteristic projections; 4. local LF speeds */
  double wc[6][5], fc[6][5], al[5] = {0, 0, 0, 0, 0};
  for (int qn = 0; qn < 6; ++qn) {
    const size_t oq = o + (size_t)(qn) * s - 2 * s; /* nodes i-2 .. i+3 */
    const double rho = Q[Q_RHO * NP + oq], pres = Q[Q_P * NP + oq], H = Q[Q_H * NP + oq], cs = Q[Q_C * NP + oq];
    const double uu[3] = {Q[Q_U * NP + oq], Q[Q_V * NP + oq], Q[Q_W * NP + oq]};
    const double un = uu[d];
    double wv[5], fv[5];
    wv[0] = rho; wv[1] = rho * uu[0]; wv[2] = rho * uu[1]; wv[3] = rho * uu[2]; wv[4] = rho * H - pres; /* rho E */
    fv[0] = rho * un;
    for (int m = 0; m < 3; ++m) fv[1 + m] = rho * uu[m] * un;
    fv[1 + d] += pres;
    fv[4] = rho * un * H;
    for (int sc = 0; sc < 5; ++sc) {
      double a1 = 0.0, a2 = 0.0;
      for (int v = 0; v < 5; ++v) { a1 += Lm[sc * 5 + v] * wv[v]; a2 += Lm[sc * 5 + v] * fv[v]; }
      wc[qn][sc] = a1; fc[qn][sc] = a2;
    }
    const double lq[5] = {un - cs, un, un, un, un + cs};
    /* local Lax-Friedrichs: maximum over the nodes the reconstruction reads (i-2..i+3 for WENO5, i-1..i+2 for WENO3, A23) */
    if (w3 && (qn == 0 || qn == 5)) continue;
    for (int sc = 0; sc < 5; ++sc) if (fabs(lq[sc]) > al[sc]) al[sc] = fabs(lq[sc]);
  }
  /* 5.-6. split, reconstruct; 7. project back */
  double fh[5];
  for (int sc = 0; sc < 5; ++sc) {
    double fp[6], fm[6];
    for (int qn = 0; qn < 6; ++qn) {
      fp[qn] = 0.5 * (fc[qn][sc] + al[sc] * wc[qn][sc]);
      fm[qn] = 0.5 * (fc[qn][sc] - al[sc] * wc[qn][sc]);
    }
    if (w3) fh[sc] = oracle_weno3(fp[1], fp[2], fp[3]) + oracle_weno3(fm[4], fm[3], fm[2]);
    else fh[sc] = oracle_weno5(fp[0], fp[1], fp[2], fp[3], fp[4]) + oracle_weno5(fm[5], fm[4], fm[3], fm[2], fm[1]);
  }
  for (int v = 0; v < 5; ++v) {
    double acc = 0.0;
    for (int sc = 0; sc < 5; ++sc) acc += Rm[v * 5 + sc] * fh[sc];
    F[v] = acc;
  }
}

/* ------------------------------------------------------------------------------------ */
/* S8 (part 1): convective residual  -sum_d (F_{i+1/2} - F_{i-1/2}) / h_d, Eq. 5 with the metric of S2;
 * at OUTFLOW nodes the x-difference is replaced by the characteristic form (A13).        */
static void convective(oracle_ctx* c, double* R) {
  const size_t NP = c->NP, np = c->np;
  memset(R, 0, NV * np * sizeof(double));
  for (int d = 0; d < 3; ++d) { c->weno_if[d] = 0; c->tot_if[d] = 0; }
  for (int d = 0; d < 3; ++d) {
    const int n = c->n[d];
    const int e1 = (d + 1) % 3, e2 = (d + 2) % 3;
    const int per = is_periodic(c, d);
    const int stag_lo = c->p.bc[2 * d] == ORC_BC_WALL_STAG, stag_hi = c->p.bc[2 * d + 1] == ORC_BC_WALL_STAG;
    const int outflow_hi = c->p.bc[2 * d + 1] == ORC_BC_OUTFLOW;
    const int charwall_lo = c->p.bc[2 * d] == ORC_BC_WALL_CHAR;
    long long nflag = 0;
#pragma omp parallel for reduction(+ : nflag)
    for (int t2 = 0; t2 < c->n[e2]; ++t2) {
      double* F = (double*)malloc((size_t)(n + 1) * NV * sizeof(double));
      for (int t1 = 0; t1 < c->n[e1]; ++t1) {
        int id[3]; id[e1] = t1; id[e2] = t2; id[d] = 0;
        const size_t o0 = GI(c, id[0], id[1], id[2]);
        for (int f = -1; f <= n - 1; ++f) { /* interface between nodes f and f+1 */
          const size_t o = o0 + (size_t)(f + NG) * c->sd[d] - (size_t)NG * c->sd[d];
          const int wall = (f == -1 && stag_lo) || (f == n - 1 && stag_hi);
          const int flagged = !wall && iface_flag(c, d, id, f);
          if (flagged) weno_flux(c, d, o, &F[(f + 1) * NV]);
          else central_flux(c, d, o, wall, &F[(f + 1) * NV]);
          if (flagged && !(per && f == -1)) ++nflag;
        }
        for (int i = 0; i < n; ++i) {
          id[d] = i;
          const size_t oi = II(c, id[0], id[1], id[2]);
          if (outflow_hi && i == n - 1) {
            /* S8: -sum_s r_s L_s with L_s = lambda_s (l_s . dw) for outgoing waves (lambda >= 0), 0 otherwise */
            const size_t ob = GI(c, id[0], id[1], id[2]);
            const size_t s = c->sd[d];
            double dw[5], Lm[25], Rm[25], lam[5], ub[3];
            for (int v = 0; v < NV; ++v)
              dw[v] = (3.0 * c->wg[v * NP + ob] - 4.0 * c->wg[v * NP + ob - s] + c->wg[v * NP + ob - 2 * s]) / (2.0 * c->h[d][i]);
            for (int m = 0; m < 3; ++m) ub[m] = c->q[(Q_U + m) * NP + ob];
            oracle_eigen(d, c->p.gamma, ub, c->q[Q_H * NP + ob], Lm, Rm, lam);
            double Ls[5];
            for (int sc = 0; sc < 5; ++sc) {
              double acc = 0.0;
              for (int v = 0; v < 5; ++v) acc += Lm[sc * 5 + v] * dw[v];
              Ls[sc] = lam[sc] >= 0.0 ? lam[sc] * acc : 0.0;
            }
            for (int v = 0; v < NV; ++v) {
              double acc = 0.0;
              for (int sc = 0; sc < 5; ++sc) acc += Rm[v * 5 + sc] * Ls[sc];
              R[v * np + oi] -= acc;
            }
          } else if (charwall_lo && i == 0) {
            /* Characteristic wave treatment at the no-slip wall (reading A14b): one-sided dw into the
               domain, the wave leaving through the wall (lambda_1 = u_n - c <= 0) is computed from the interior, the
               incoming acoustic wave is its reflection L_5 = L_1 (no normal momentum is created: with u_n = 0,
               -(r_1 L_1 + r_5 L_5) has no wall-normal momentum component), entropy and shear waves do not enter
               (lambda = u_n = 0 at the wall; removed if positive). */
            const size_t ob = GI(c, id[0], id[1], id[2]);
            const size_t s = c->sd[d];
            double dw[5], Lm[25], Rm[25], lam[5], ub[3];
            for (int v = 0; v < NV; ++v)
              dw[v] = (-3.0 * c->wg[v * NP + ob] + 4.0 * c->wg[v * NP + ob + s] - c->wg[v * NP + ob + 2 * s]) / (2.0 * c->h[d][i]);
            for (int m = 0; m < 3; ++m) ub[m] = c->q[(Q_U + m) * NP + ob];
            oracle_eigen(d, c->p.gamma, ub, c->q[Q_H * NP + ob], Lm, Rm, lam);
            double Ls[5];
            for (int sc = 0; sc < 5; ++sc) {
              double acc = 0.0;
              for (int v = 0; v < 5; ++v) acc += Lm[sc * 5 + v] * dw[v];
              Ls[sc] = lam[sc] <= 0.0 ? lam[sc] * acc : 0.0;
            }
            Ls[4] = Ls[0];
            for (int v = 0; v < NV; ++v) {
              double acc = 0.0;
              for (int sc = 0; sc < 5; ++sc) acc += Rm[v * 5 + sc] * Ls[sc];
              R[v * np + oi] -= acc;
            }
          } else {
            for (int v = 0; v < NV; ++v) R[v * np + oi] -= (F[(i + 1) * NV + v] - F[i * NV + v]) / c->h[d][i];
          }
        }
      }
      free(F);
    }
    c->weno_if[d] = nflag;
    c->tot_if[d] = (long long)(per ? n : n + 1) * c->n[e1] * c->n[e2];
  }
}

/* S7: viscous and heat-conduction terms in Laplacian form (Eq. 2-3, 9) */
static void viscous(oracle_ctx* c, double* V) {
  const size_t NP = c->NP, np = c->np;
  const oracle_params* p = &c->p;
  const double cp = p->gamma * p->Rgas / (p->gamma - 1.0);
  const double* U[3] = {c->q + Q_U * NP, c->q + Q_V * NP, c->q + Q_W * NP};
  const double* T = c->q + Q_T * NP;
  const double* MU = c->q + Q_MU * NP;
  memset(V, 0, NV * np * sizeof(double));
  /* inner derivatives d u_k / d x_k on the range extended in the other two directions (A8):
     they are differentiated again, along another direction, for the mixed terms */
  for (int d = 0; d < 3; ++d) {
    int lo[3], hi[3];
    for (int e = 0; e < 3; ++e) { lo[e] = e == d ? 0 : -NG; hi[e] = e == d ? c->n[e] : c->n[e] + NG; }
#pragma omp parallel for
    for (int k = lo[2]; k < hi[2]; ++k)
      for (int j = lo[1]; j < hi[1]; ++j)
        for (int i = lo[0]; i < hi[0]; ++i) {
          const int id[3] = {i, j, k};
          const size_t o = GI(c, i, j, k);
          c->dd[d][o] = D1(c, U[d], o, d) / c->h[d][id[d]];
        }
  }
#pragma omp parallel for
  for (int k = 0; k < c->n[2]; ++k)
    for (int j = 0; j < c->n[1]; ++j)
      for (int i = 0; i < c->n[0]; ++i) {
        const size_t o = GI(c, i, j, k), oi = II(c, i, j, k);
        const int id[3] = {i, j, k};
        double G[3][3], G2[3][3], Tj[3], T2[3], Mj[3];
        for (int d = 0; d < 3; ++d) {
          const double hd = c->h[d][id[d]], gd = c->gm[d][id[d]];
          for (int a = 0; a < 3; ++a) {
            const double d1 = D1(c, U[a], o, d);
            G[a][d] = d1 / hd;                                              /* d u_a / d x_d            */
            G2[a][d] = D2(c, U[a], o, d) / (hd * hd) - d1 * gd / (hd * hd * hd); /* d2 u_a / d x_d^2 (S2) */
          }
          const double t1 = D1(c, T, o, d);
          Tj[d] = t1 / hd;
          T2[d] = D2(c, T, o, d) / (hd * hd) - t1 * gd / (hd * hd * hd);
          Mj[d] = D1(c, MU, o, d) / hd;                                     /* mu differentiated numerically, as Eq. 9 */
        }
        const double Th = G[0][0] + G[1][1] + G[2][2];
        const double uu[3] = {U[0][o], U[1][o], U[2][o]};
        const double mu = MU[o];
        double Vi[3];
        for (int a = 0; a < 3; ++a) {
          /* (grad Theta)_a = d2_a u_a + sum_{k != a} d_a (d_k u_k) */
          double gth = G2[a][a];
          for (int kx = 0; kx < 3; ++kx) if (kx != a) gth += D1(c, c->dd[kx], o, a) / c->h[a][id[a]];
          double lap = G2[a][0] + G2[a][1] + G2[a][2];
          double cross = 0.0;
          for (int jx = 0; jx < 3; ++jx) cross += Mj[jx] * (G[a][jx] + G[jx][a]);
          Vi[a] = mu * (lap + gth / 3.0) + cross - 2.0 / 3.0 * Mj[a] * Th;
        }
        const double s01 = G[0][1] + G[1][0], s02 = G[0][2] + G[2][0], s12 = G[1][2] + G[2][1];
        const double Phi = mu * (2.0 * (G[0][0] * G[0][0] + G[1][1] * G[1][1] + G[2][2] * G[2][2]) + s01 * s01 + s02 * s02 + s12 * s12 - 2.0 / 3.0 * Th * Th);
        const double heat = cp / p->Pr * (mu * (T2[0] + T2[1] + T2[2]) + (Mj[0] * Tj[0] + Mj[1] * Tj[1] + Mj[2] * Tj[2]));
        V[1 * np + oi] = Vi[0];
        V[2 * np + oi] = Vi[1];
        V[3 * np + oi] = Vi[2];
        V[4 * np + oi] = uu[0] * Vi[0] + uu[1] * Vi[1] + uu[2] * Vi[2] + Phi + heat;
      }
}

/* Neumaier compensated sum accumulator */
typedef struct { double s, c; } ksum;
static inline void kadd(ksum* k, double x) {
  double t = k->s + x;
  if (fabs(k->s) >= fabs(x)) k->c += (k->s - t) + x; else k->c += (x - t) + k->s;
  k->s = t;
}

static void prepare(oracle_ctx* c) {
  fill_ghosts(c);
  compute_prims(c);
  if (c->p.weno_enable) compute_theta(c);
}

/* R(w): S8 + S9.  conv/visc (optional) receive the two parts without forcing. */
static void rhs_full(oracle_ctx* c, double* R, double* conv_out, double* visc_out) {
  const size_t np = c->np;
  prepare(c);
  convective(c, R);
  if (conv_out) memcpy(conv_out, R, NV * np * sizeof(double));
  if (c->p.viscous_enable) {
    double* V = (double*)malloc(NV * np * sizeof(double));
    viscous(c, V);
    if (visc_out) memcpy(visc_out, V, NV * np * sizeof(double));
    for (size_t o = 0; o < NV * np; ++o) R[o] += V[o];
    free(V);
  } else if (visc_out) memset(visc_out, 0, NV * np * sizeof(double));
  c->force = 0.0;
  if (c->p.forcing) {
    /* S9: f = - sum(R_rhou vol) / sum(vol); added to the x-momentum and, times u, to the energy (Eq. 1b-c) */
    ksum A = {0, 0}, Vt = {0, 0};
    for (int k = 0; k < c->n[2]; ++k)
      for (int j = 0; j < c->n[1]; ++j)
        for (int i = 0; i < c->n[0]; ++i) {
          const double vol = c->h[0][i] * c->h[1][j] * c->h[2][k];
          kadd(&A, R[1 * np + II(c, i, j, k)] * vol);
          kadd(&Vt, vol);
        }
    const double f = -(A.s + A.c) / (Vt.s + Vt.c);
    c->force = f;
    for (int k = 0; k < c->n[2]; ++k)
      for (int j = 0; j < c->n[1]; ++j)
        for (int i = 0; i < c->n[0]; ++i) {
          const size_t oi = II(c, i, j, k);
          R[1 * np + oi] += f;
          R[4 * np + oi] += f * c->q[Q_U * c->NP + GI(c, i, j, k)];
        }
  }
}

int oracle_rhs(oracle_ctx* c, double* out) {
  if (!c || !out) return ORC_EINVAL;
  if (!c->has_state) return ORC_ESTATE;
  rhs_full(c, out, NULL, NULL);
  return ORC_OK;
}

int oracle_rhs_parts(oracle_ctx* c, double* conv_out, double* visc_out) {
  if (!c) return ORC_EINVAL;
  if (!c->has_state) return ORC_ESTATE;
  double* R = (double*)malloc(NV * c->np * sizeof(double));
  rhs_full(c, R, conv_out, visc_out);
  free(R);
  return ORC_OK;
}

int oracle_get_prims(oracle_ctx* c, double* out) {
  if (!c || !out) return ORC_EINVAL;
  if (!c->has_state) return ORC_ESTATE;
  prepare(c);
  for (int v = 0; v < NQ; ++v)
    for (int k = 0; k < c->n[2]; ++k)
      for (int j = 0; j < c->n[1]; ++j)
        for (int i = 0; i < c->n[0]; ++i) out[v * c->np + II(c, i, j, k)] = c->q[v * c->NP + GI(c, i, j, k)];
  return ORC_OK;
}

/* accessor for the pins of S1: the ghost-filled conservative state [5][nz+6][ny+6][nx+6] of the current state */
int oracle_get_ghosted(oracle_ctx* c, double* wg_out) {
  if (!c || !wg_out) return ORC_EINVAL;
  if (!c->has_state) return ORC_ESTATE;
  fill_ghosts(c);
  memcpy(wg_out, c->wg, NV * c->NP * sizeof(double));
  return ORC_OK;
}

int oracle_get_sensor(oracle_ctx* c, double* theta_out, unsigned char* flags_out) {
  if (!c) return ORC_EINVAL;
  if (!c->has_state) return ORC_ESTATE;
  fill_ghosts(c);
  compute_prims(c);
  compute_theta(c);
  if (theta_out) memcpy(theta_out, c->theta, c->np * sizeof(double));
  if (flags_out)
    for (int d = 0; d < 3; ++d)
      for (int k = 0; k < c->n[2]; ++k)
        for (int j = 0; j < c->n[1]; ++j)
          for (int i = 0; i < c->n[0]; ++i) {
            int id[3] = {i, j, k};
            const int f = id[d];
            const int wall = f == c->n[d] - 1 && c->p.bc[2 * d + 1] == ORC_BC_WALL_STAG;
            flags_out[d * c->np + II(c, i, j, k)] = (unsigned char)(!wall && iface_flag(c, d, id, f));
          }
  return ORC_OK;
}

/* S10: dt = cfl / max over nodes and directions of (|u_d| + c) / h_d */
static double time_step(oracle_ctx* c, double speed[3]) {
  const size_t NP = c->NP;
  double m[3] = {0, 0, 0};
  for (int k = 0; k < c->n[2]; ++k)
    for (int j = 0; j < c->n[1]; ++j)
      for (int i = 0; i < c->n[0]; ++i) {
        const size_t o = GI(c, i, j, k);
        const int id[3] = {i, j, k};
        for (int d = 0; d < 3; ++d) {
          const double s = (fabs(c->q[(Q_U + d) * NP + o]) + c->q[Q_C * NP + o]) / c->h[d][id[d]];
          if (s > m[d]) m[d] = s;
        }
      }
  if (speed) { speed[0] = m[0]; speed[1] = m[1]; speed[2] = m[2]; }
  double mm = m[0] > m[1] ? m[0] : m[1];
  mm = mm > m[2] ? mm : m[2];
  return c->p.dt_fixed > 0.0 ? c->p.dt_fixed : c->p.cfl / mm;
}

/* S11: Eq. 11 with alpha_1 = -17/60 (reading G5: the printed +17/60 is not third order) */
int oracle_step(oracle_ctx* c, int nsteps) {
  if (!c || nsteps < 0) return ORC_EINVAL;
  if (!c->has_state) return ORC_ESTATE;
  static const double alpha[3] = {0.0, -17.0 / 60.0, -5.0 / 12.0};
  static const double beta[3] = {8.0 / 15.0, 5.0 / 12.0, 3.0 / 4.0};
  const size_t np = c->np;
  const double cv = c->p.Rgas / (c->p.gamma - 1.0);
  for (int st = 0; st < nsteps; ++st) {
    fill_ghosts(c);
    compute_prims(c);
    const double dt = time_step(c, NULL);
    c->dt = dt;
    for (int l = 0; l < 3; ++l) {
      rhs_full(c, c->Rcur, NULL, NULL);
      for (size_t o = 0; o < NV * np; ++o) c->w[o] += dt * (alpha[l] * c->Rprev[o] + beta[l] * c->Rcur[o]);
      double* t = c->Rprev; c->Rprev = c->Rcur; c->Rcur = t;
      /* S1 node wall: after every stage rho u = rho v = rho w = 0, rho E = rho cv Tw (rho evolves by the scheme) */
      for (int s = 0; s < 2; ++s)
        if (c->p.bc[2 + s] == ORC_BC_WALL_NODE || c->p.bc[2 + s] == ORC_BC_WALL_CHAR) {
          const int j = s == 0 ? 0 : c->n[1] - 1;
          for (int k = 0; k < c->n[2]; ++k)
            for (int i = 0; i < c->n[0]; ++i) {
              const size_t oi = II(c, i, j, k);
              c->w[1 * np + oi] = 0.0; c->w[2 * np + oi] = 0.0; c->w[3 * np + oi] = 0.0;
              c->w[4 * np + oi] = c->w[0 * np + oi] * cv * c->p.T_wall[s];
            }
        }
    }
    c->time += dt;
    c->step += 1;
  }
  return ORC_OK;
}

/* ------------------------------------------------------------------------------------ */
/* Statistics: "the overline symbol denotes averaging in the homogeneous space directions and in
 * time"; Reynolds means of phi and the density-weighted sums that give Favre means  phi~ = mean(rho phi) / mean(rho).
 * One call adds the x-z plane means (plain node means: the homogeneous directions are uniformly spaced) of the
 * current state to running sums, per wall-normal index j.  Order of the ORC_NSTAT quantities:
 *   rho, u, v, w, p, T, mu, rho u, rho v, rho w, rho T, rho u u, rho v v, rho w w, rho u v, T T                  */
int oracle_stats_accumulate(oracle_ctx* c) {
  if (!c) return ORC_EINVAL;
  if (!c->has_state) return ORC_ESTATE;
  fill_ghosts(c);
  compute_prims(c);
  const size_t NP = c->NP;
  const double cnt = (double)c->n[0] * (double)c->n[2];
  for (int j = 0; j < c->n[1]; ++j) {
    ksum acc[ORC_NSTAT];
    for (int m = 0; m < ORC_NSTAT; ++m) { acc[m].s = 0.0; acc[m].c = 0.0; }
    for (int k = 0; k < c->n[2]; ++k)
      for (int i = 0; i < c->n[0]; ++i) {
        const size_t o = GI(c, i, j, k);
        const double rho = c->q[Q_RHO * NP + o], u = c->q[Q_U * NP + o], v = c->q[Q_V * NP + o], w = c->q[Q_W * NP + o];
        const double pr = c->q[Q_P * NP + o], T = c->q[Q_T * NP + o], mu = c->q[Q_MU * NP + o];
        const double val[ORC_NSTAT] = {rho, u, v, w, pr, T, mu, rho * u, rho * v, rho * w, rho * T,
                                       rho * u * u, rho * v * v, rho * w * w, rho * u * v, T * T};
        for (int m = 0; m < ORC_NSTAT; ++m) kadd(&acc[m], val[m]);
      }
    for (int m = 0; m < ORC_NSTAT; ++m) c->stat_sum[(size_t)m * c->n[1] + j] += (acc[m].s + acc[m].c) / cnt;
  }
  c->stat_n += 1;
  return ORC_OK;
}

/* time-averaged profiles [ORC_NSTAT][ny] = running sums / number of accumulated samples */
int oracle_stats_read(oracle_ctx* c, double* out, long long* nsamples) {
  if (!c || !out) return ORC_EINVAL;
  const double inv = c->stat_n > 0 ? 1.0 / (double)c->stat_n : 0.0;
  for (size_t e = 0; e < (size_t)ORC_NSTAT * c->n[1]; ++e) out[e] = c->stat_sum[e] * inv;
  if (nsamples) *nsamples = c->stat_n;
  return ORC_OK;
}

int oracle_stats_reset(oracle_ctx* c) {
  if (!c) return ORC_EINVAL;
  memset(c->stat_sum, 0, (size_t)ORC_NSTAT * c->n[1] * sizeof(double));
  c->stat_n = 0;
  return ORC_OK;
}

int oracle_diagnostics(oracle_ctx* c, oracle_diag* out) {
  if (!c || !out) return ORC_EINVAL;
  if (!c->has_state) return ORC_ESTATE;
  memset(out, 0, sizeof(*out));
  prepare(c);
  const size_t NP = c->NP, np = c->np;
  ksum mass = {0, 0}, mx = {0, 0}, my = {0, 0}, mz = {0, 0}, en = {0, 0}, ke = {0, 0}, vt = {0, 0};
  double minr = INFINITY, minp = INFINITY, maxm = 0.0, maxth = 0.0;
  int bad = 0;
  for (int k = 0; k < c->n[2]; ++k)
    for (int j = 0; j < c->n[1]; ++j)
      for (int i = 0; i < c->n[0]; ++i) {
        const size_t o = GI(c, i, j, k), oi = II(c, i, j, k);
        const double vol = c->h[0][i] * c->h[1][j] * c->h[2][k];
        const double rho = c->q[Q_RHO * NP + o], u = c->q[Q_U * NP + o], v = c->q[Q_V * NP + o], w = c->q[Q_W * NP + o];
        const double pr = c->q[Q_P * NP + o], cs = c->q[Q_C * NP + o];
        kadd(&mass, rho * vol); kadd(&mx, c->w[1 * np + oi] * vol); kadd(&my, c->w[2 * np + oi] * vol);
        kadd(&mz, c->w[3 * np + oi] * vol); kadd(&en, c->w[4 * np + oi] * vol);
        kadd(&ke, 0.5 * rho * (u * u + v * v + w * w) * vol); kadd(&vt, vol);
        if (!(rho > 0.0) || !(pr > 0.0) || !isfinite(rho) || !isfinite(pr) || !isfinite(c->w[4 * np + oi])) bad = 1;
        if (rho < minr) minr = rho;
        if (pr < minp) minp = pr;
        const double ma = sqrt(u * u + v * v + w * w) / cs;
        if (ma > maxm) maxm = ma;
        if (c->p.weno_enable && c->theta[oi] > maxth) maxth = c->theta[oi];
      }
  out->step = c->step; out->time = c->time; out->dt = c->dt; out->forcing = c->force;
  out->mass = mass.s + mass.c; out->mom[0] = mx.s + mx.c; out->mom[1] = my.s + my.c; out->mom[2] = mz.s + mz.c;
  out->energy = en.s + en.c; out->kinetic = ke.s + ke.c; out->volume = vt.s + vt.c;
  out->bulk_rhou = out->mom[0] / out->volume;
  out->min_rho = minr; out->min_p = minp; out->max_mach = maxm; out->max_theta = maxth;
  time_step(c, out->max_speed);
  for (int d = 0; d < 3; ++d) { out->weno_ifaces[d] = c->weno_if[d]; out->total_ifaces[d] = c->tot_if[d]; }
  out->nonfinite = bad;
  return bad ? ORC_ENONFINITE : ORC_OK;
}
