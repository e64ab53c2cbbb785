// k_aux.cuh -- state conversion (a2), RK3 update with forcing (a7, a9), CFL reduction (a10), diagnostics.
#pragma once
#include "dev_common.cuh"

namespace streams {

constexpr int RT = 256;                 // threads of the light grid-stride kernels

// node index -> (i, j, k) in 32-bit arithmetic (validate(): N < 2^32)
__device__ __forceinline__ void node_ijk(const DevP& P, long long o, int& i, int& j, int& k) {
  const unsigned int o32 = (unsigned int)o, row = o32 / (unsigned int)P.nx;
  i = (int)(o32 - row * (unsigned int)P.nx);
  k = (int)(row / (unsigned int)P.ny);
  j = (int)(row - (unsigned int)k * (unsigned int)P.ny);
}

// device scalars kept between kernels (no host round trip inside streams_step)
struct DevScal {
  double dt;            // S10
  double force;         // S9: body force f of the last RHS evaluation
  double time;
  double vol_total;     // sum of node volumes (constant, set at creation)
  double max_theta;     // bits reinterpreted for atomicMax
  unsigned long long weno_if[3];
  unsigned int list_count;
  unsigned int pad;
  unsigned int icount[3];   // entries of the three interface lists (k_weno_list)
  unsigned int pad2;
  // Partial reductions of THIS context, combined across z-slabs by the caller between the staged calls
  // (include/streams.h, streams_reduce_ptr): red[0] = sum R_rhou vol, red[1] = sum vol  (S9: f = -red[0] / red[1]),
  // red[2] = max over nodes and directions of (|u_d| + c) / h_d  (S10: dt = cfl / red[2]).
  double red[4];
};

// ---- S3: conservative w[5][N] -> primitives Q[NQ][N]  (streams_set_state) ----
__global__ void __launch_bounds__(RT) k_cons2prim(const __grid_constant__ DevP P, const double* __restrict__ w, double* __restrict__ Q) {
  for (long long o = blockIdx.x * (long long)RT + threadIdx.x; o < P.N; o += (long long)gridDim.x * RT) {
    Prim q;
    cons2prim(P, w[o], w[o + P.N], w[o + 2 * P.N], w[o + 3 * P.N], w[o + 4 * P.N], q);
    Q[o] = q.rho; Q[o + P.QS] = q.u; Q[o + 2 * P.QS] = q.v; Q[o + 3 * P.QS] = q.w; Q[o + 4 * P.QS] = q.T; Q[o + 5 * P.QS] = q.mu; Q[o + 6 * P.QS] = q.H;
  }
}
// ---- primitives -> conservative (streams_get_state) ----
__global__ void __launch_bounds__(RT) k_prim2cons(const __grid_constant__ DevP P, const double* __restrict__ Q, double* __restrict__ w) {
  for (long long o = blockIdx.x * (long long)RT + threadIdx.x; o < P.N; o += (long long)gridDim.x * RT) {
    Prim q;
    q.rho = Q[o]; q.u = Q[o + P.QS]; q.v = Q[o + 2 * P.QS]; q.w = Q[o + 3 * P.QS]; q.T = Q[o + 4 * P.QS]; q.mu = 0.0;
    double wv[5];
    prim2cons(P, q, wv);
#pragma unroll
    for (int v = 0; v < 5; ++v) w[o + v * P.N] = wv[v];
  }
}

// ---- S11 with S9: R += f (0,1,0,0,u);  w <- w + dt (alpha R_prev + beta R), Eq. 11, state kept
// as primitives.  `keep_R` != 0 writes the two forced components of R back (the next stage reads them as R_prev).
__global__ void __launch_bounds__(RT) k_update(const __grid_constant__ DevP P, double* __restrict__ Q, const double* __restrict__ Sp,
                                               double* __restrict__ Sc, const DevScal* __restrict__ sc,
                                               double alpha, double beta, int use_force, int keep_R) {
  const double dt = sc->dt;
  const double f = use_force ? sc->force : 0.0;
  for (long long o = blockIdx.x * (long long)RT + threadIdx.x; o < P.N; o += (long long)gridDim.x * RT) {
    Prim q;
    q.rho = Q[o]; q.u = Q[o + P.QS]; q.v = Q[o + 2 * P.QS]; q.w = Q[o + 3 * P.QS]; q.T = Q[o + 4 * P.QS]; q.mu = 0.0;
    double r[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) r[v] = Sc[o + v * P.N];
    if (use_force) {
      r[1] += f; r[4] = fma(f, q.u, r[4]);           // Eq. 1b-c: f delta_i1 and f u_1
      if (keep_R) { Sc[o + 1 * P.N] = r[1]; Sc[o + 4 * P.N] = r[4]; }
    }
    double dW[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      const double sp = alpha != 0.0 ? Sp[o + v * P.N] : 0.0;
      dW[v] = dt * (alpha * sp + beta * r[v]);
    }
    advance_prim(P, q, dW);
    int i_, j, k_;
    node_ijk(P, o, i_, j, k_);
    if (j == 0 && node_wall(P.bc[2])) wall_node_override(P, P.Twall[0], P.mu_wall[0], q);
    if (j == P.ny - 1 && node_wall(P.bc[3])) wall_node_override(P, P.Twall[1], P.mu_wall[1], q);
    Q[o] = q.rho; Q[o + P.QS] = q.u; Q[o + 2 * P.QS] = q.v; Q[o + 3 * P.QS] = q.w; Q[o + 4 * P.QS] = q.T; Q[o + 5 * P.QS] = q.mu; Q[o + 6 * P.QS] = q.H;
  }
}

// ---- lazy forcing (S9 with Eq. 11): the fused k_rhs<true> advanced the state WITHOUT this stage's body force (f is
// only known once the whole R has been summed); this adds dt beta f (e_rhou + u e_rhoE), u = the velocity of the
// stage's input state `Qin`, to the new state `Q` (rho, v, w are not touched) and evaluates mu(T) of the new state.
// Same map as advance_prim.  One CTA walks grid rows (j,k); `speed` != NULL (last stage): per-CTA maxima of
// (|u_d| + c) / h_d of the finished state (S10) go to speed[3][gridDim.x], so the next step needs no extra pass.
constexpr int FIXU = 4;
__global__ void __launch_bounds__(RT) k_force_fix(const __grid_constant__ DevP P, double* __restrict__ Q, const double* __restrict__ Qin,
                                                  const DevScal* __restrict__ sc, double beta, double* __restrict__ speed) {
  __shared__ double sh[RT / 32];
  const double c = sc->dt * beta * sc->force;
  const bool wn0 = node_wall(P.bc[2]), wn1 = node_wall(P.bc[3]);
  const int nrows = P.ny * P.nz;
  double m[3] = {0.0, 0.0, 0.0};
  for (int row = blockIdx.x; row < nrows; row += gridDim.x) {
    const int j = row % P.ny, k = row / P.ny;
    const bool wallrow = (wn0 && j == 0) || (wn1 && j == P.ny - 1);      // Dirichlet wall nodes: already overridden
    const double ihy = P.ih[1][j], ihz = P.ih[2][k];
    const size_t r0 = (size_t)row * P.nx;
    for (int ib = threadIdx.x; ib < P.nx; ib += FIXU * RT) {
      // FIXU nodes per thread, all loads first (memory-level parallelism: the kernel is HBM-bound)
      double rho[FIXU], u[FIXU], T[FIXU], H[FIXU], ul[FIXU], vv[FIXU], ww[FIXU];
#pragma unroll
      for (int e = 0; e < FIXU; ++e) {
        const int i = ib + e * RT;
        if (i < P.nx) {
          const size_t o = r0 + i;
          u[e] = Q[o + P.QS]; T[e] = Q[o + 4 * P.QS];
          if (!wallrow) { rho[e] = Q[o]; H[e] = Q[o + 6 * P.QS]; ul[e] = Qin[o + P.QS]; }
          if (speed) { vv[e] = Q[o + 2 * P.QS]; ww[e] = Q[o + 3 * P.QS]; }
        }
      }
#pragma unroll
      for (int e = 0; e < FIXU; ++e) {
        const int i = ib + e * RT;
        if (i < P.nx) {
          const size_t o = r0 + i;
          double un = u[e], Tn = T[e];
          if (!wallrow) {
            const double ir = 1.0 / rho[e];
            const double du = c * ir, dE = (c * ul[e]) * ir;
            un = u[e] + du;
            const double dke = 0.5 * (du * (un + u[e]));
            const double dT = (dE - dke) * P.inv_cv;
            Tn = T[e] + dT;
            Q[o + P.QS] = un; Q[o + 4 * P.QS] = Tn; Q[o + 5 * P.QS] = visc_mu(P, Tn);
            Q[o + 6 * P.QS] = H[e] + fma(P.cp, dT, dke);
          }
          if (speed) {
            const double cs = sqrt(P.gam * P.Rgas * Tn);
            m[0] = fmax(m[0], (fabs(un) + cs) * P.ih[0][i]);
            m[1] = fmax(m[1], (fabs(vv[e]) + cs) * ihy);
            m[2] = fmax(m[2], (fabs(ww[e]) + cs) * ihz);
          }
        }
      }
    }
  }
  if (speed)
    for (int d = 0; d < 3; ++d) {
      const double t = block_max<RT>(m[d], sh, threadIdx.x);
      if (threadIdx.x == 0) speed[d * gridDim.x + blockIdx.x] = t;
    }
}

// R_rhou += f, R_rhoE += f u  (streams_rhs with forcing)
__global__ void __launch_bounds__(RT) k_apply_force(const __grid_constant__ DevP P, const double* __restrict__ Q, double* __restrict__ R,
                                                    const DevScal* __restrict__ sc) {
  const double f = sc->force;
  for (long long o = blockIdx.x * (long long)RT + threadIdx.x; o < P.N; o += (long long)gridDim.x * RT) {
    R[o + 1 * P.N] += f;
    R[o + 4 * P.N] = fma(f, Q[o + P.QS], R[o + 4 * P.N]);
  }
}

// ---- S9: per-block partial sums of R_rhou * vol ----
__global__ void __launch_bounds__(RT) k_force_partial(const __grid_constant__ DevP P, const double* __restrict__ R, double* __restrict__ partial) {
  __shared__ double sh[RT / 32];
  double acc = 0.0;
  for (long long o = blockIdx.x * (long long)RT + threadIdx.x; o < P.N; o += (long long)gridDim.x * RT) {
    int i, j, k;
    node_ijk(P, o, i, j, k);
    acc += R[o + P.N] * (P.hh[0][i] * P.hh[1][j] * P.hh[2][k]);
  }
  const double t = block_sum<RT>(acc, sh, threadIdx.x);
  if (threadIdx.x == 0) partial[blockIdx.x] = t;
}
// red[0] = sum(partials), red[1] = sum(vol), fixed summation order (one CTA); take != 0: f = - red[0] / red[1] at once
// (single context; z-slabs combine red across contexts first and then run k_force_take)
__global__ void __launch_bounds__(RT) k_force_final(const double* __restrict__ partial, int n, DevScal* sc, int take) {
  __shared__ double sh[RT / 32];
  double acc = 0.0;
  for (int e = threadIdx.x; e < n; e += RT) acc += partial[e];
  const double t = block_sum<RT>(acc, sh, threadIdx.x);
  if (threadIdx.x == 0) {
    sc->red[0] = t; sc->red[1] = sc->vol_total;
    if (take) sc->force = -t / sc->vol_total;
  }
}
__global__ void k_force_take(DevScal* sc) { sc->force = -sc->red[0] / sc->red[1]; }

// ---- S10: dt = cfl / max_d max_nodes (|u_d| + c) / h_d ----
__global__ void __launch_bounds__(RT) k_speed_partial(const __grid_constant__ DevP P, const double* __restrict__ Q, double* __restrict__ partial /*[3][grid]*/) {
  __shared__ double sh[RT / 32];
  double m[3] = {0.0, 0.0, 0.0};
  for (long long o = blockIdx.x * (long long)RT + threadIdx.x; o < P.N; o += (long long)gridDim.x * RT) {
    int i, j, k;
    node_ijk(P, o, i, j, k);
    const double cs = sqrt(P.gam * P.Rgas * Q[o + 4 * P.QS]);
    m[0] = fmax(m[0], (fabs(Q[o + P.QS]) + cs) * P.ih[0][i]);
    m[1] = fmax(m[1], (fabs(Q[o + 2 * P.QS]) + cs) * P.ih[1][j]);
    m[2] = fmax(m[2], (fabs(Q[o + 3 * P.QS]) + cs) * P.ih[2][k]);
  }
  for (int d = 0; d < 3; ++d) {
    const double t = block_max<RT>(m[d], sh, threadIdx.x);
    if (threadIdx.x == 0) partial[d * gridDim.x + blockIdx.x] = t;
  }
}
__global__ void __launch_bounds__(RT) k_dt_final(const double* __restrict__ partial, int n, DevScal* sc,
                                                 double* __restrict__ speeds_out /* 3, may be NULL */, int set_red) {
  __shared__ double sh[RT / 32];
  double mm = 0.0;
  for (int d = 0; d < 3; ++d) {
    double m = 0.0;
    for (int e = threadIdx.x; e < n; e += RT) m = fmax(m, partial[d * n + e]);
    const double t = block_max<RT>(m, sh, threadIdx.x);
    if (threadIdx.x == 0) { mm = fmax(mm, t); if (speeds_out) speeds_out[d] = t; }
  }
  if (threadIdx.x == 0 && set_red) sc->red[2] = mm;             // local maximum; k_take_dt turns it into the time step
}
__global__ void k_advance_time(DevScal* sc) { sc->time += sc->dt; }
// S10: dt = cfl / max (|u_d| + c) / h_d, the maximum taken over the whole domain (red[2], combined across z-slabs)
__global__ void k_take_dt(DevScal* sc, double cfl) { sc->dt = cfl / sc->red[2]; }

// ---- diagnostics: per-block partials, reduced on the host by streams_diagnostics ----
constexpr int NDIAG = 12;   // mass, mx, my, mz, E, ke, vol | min rho, min p, max Mach | nonfinite | spare
__global__ void __launch_bounds__(RT) k_diag_partial(const __grid_constant__ DevP P, const double* __restrict__ Q, double* __restrict__ partial /*[NDIAG][grid]*/) {
  __shared__ double sh[RT / 32];
  double s[7] = {0, 0, 0, 0, 0, 0, 0};
  double mnr = INFINITY, mnp = INFINITY, mxm = 0.0, bad = 0.0;
  for (long long o = blockIdx.x * (long long)RT + threadIdx.x; o < P.N; o += (long long)gridDim.x * RT) {
    int i, j, k;
    node_ijk(P, o, i, j, k);
    const double vol = P.hh[0][i] * P.hh[1][j] * P.hh[2][k];
    Prim q;
    q.rho = Q[o]; q.u = Q[o + P.QS]; q.v = Q[o + 2 * P.QS]; q.w = Q[o + 3 * P.QS]; q.T = Q[o + 4 * P.QS]; q.mu = 0.0;
    double wv[5];
    prim2cons(P, q, wv);
    const double q2 = q.u * q.u + q.v * q.v + q.w * q.w;
    const double ke = 0.5 * q.rho * q2;
    const double p = q.rho * (P.Rgas * q.T);
    s[0] += wv[0] * vol; s[1] += wv[1] * vol; s[2] += wv[2] * vol; s[3] += wv[3] * vol; s[4] += wv[4] * vol; s[5] += ke * vol; s[6] += vol;
    if (!(q.rho > 0.0) || !(p > 0.0) || !isfinite(q.rho) || !isfinite(p) || !isfinite(wv[4])) bad = 1.0;
    mnr = fmin(mnr, q.rho); mnp = fmin(mnp, p);
    mxm = fmax(mxm, sqrt(q2 / (P.gam * P.Rgas * q.T)));
  }
  for (int a = 0; a < 7; ++a) {
    const double t = block_sum<RT>(s[a], sh, threadIdx.x);
    if (threadIdx.x == 0) partial[a * gridDim.x + blockIdx.x] = t;
  }
  double t;
  t = -block_max<RT>(-mnr, sh, threadIdx.x); if (threadIdx.x == 0) partial[7 * gridDim.x + blockIdx.x] = t;
  t = -block_max<RT>(-mnp, sh, threadIdx.x); if (threadIdx.x == 0) partial[8 * gridDim.x + blockIdx.x] = t;
  t = block_max<RT>(mxm, sh, threadIdx.x);   if (threadIdx.x == 0) partial[9 * gridDim.x + blockIdx.x] = t;
  t = block_max<RT>(bad, sh, threadIdx.x);   if (threadIdx.x == 0) partial[10 * gridDim.x + blockIdx.x] = t;
}

// ---- fp64 pipe peak: 8 independent DFMA chains per thread, registers only (streams_fp64_peak) ----
__global__ void __launch_bounds__(1024) k_fp64_peak(double* __restrict__ out, int iters, double a, double b) {
  double x0 = threadIdx.x, x1 = x0 + 1.0, x2 = x0 + 2.0, x3 = x0 + 3.0, x4 = x0 + 4.0, x5 = x0 + 5.0, x6 = x0 + 6.0, x7 = x0 + 7.0;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
      x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
      x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
  }
  const double r = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
  if (r == 123.456) out[0] = r;              // never true: keeps the chains alive
}

// capture the frozen inflow plane (S1 INFLOW_FROZEN): inflow[v][k][j] = Q[v][k][j][0], all stored planes k (a z-slab
// keeps the ghost planes of the inflow as well: k = -zpad .. nz + zpad - 1; `Q` and `inflow` point at plane 0)
__global__ void k_capture_inflow(const __grid_constant__ DevP P, const double* __restrict__ Q, double* __restrict__ inflow) {
  const long long n = P.IS, r0 = -(long long)P.zpad * P.ny;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < NQ * n; e += (long long)gridDim.x * blockDim.x) {
    const int v = (int)(e / n);
    const long long r = r0 + e % n;
    inflow[v * n + r] = Q[v * P.QS + r * P.nx];
  }
}

}  // namespace streams
