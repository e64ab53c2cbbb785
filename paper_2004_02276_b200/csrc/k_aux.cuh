// k_aux.cuh -- RK3 update (a9), CFL reduction (a10), forcing reduction (a7), diagnostics.
#pragma once
#include "dev_common.cuh"

namespace streams {

constexpr int RT = 256;                 // threads of the reduction kernels

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
};

// ---- S11: w <- w + dt (alpha R_prev + beta R), Eq. 11, with the body force of S9 ----
__global__ void __launch_bounds__(RT) k_update(const DevP P, double* __restrict__ w, const double* __restrict__ Sp,
                                               double* __restrict__ Sc, const DevScal* __restrict__ sc,
                                               double alpha, double beta, int use_force) {
  const double dt = sc->dt;
  const double f = use_force ? sc->force : 0.0;
  for (long long o = blockIdx.x * (long long)RT + threadIdx.x; o < P.N; o += (long long)gridDim.x * RT) {
    double wv[5], r[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) { wv[v] = w[o + v * P.N]; r[v] = Sc[o + v * P.N]; }
    if (use_force) {
      const double u = wv[1] / wv[0];
      r[1] += f; r[4] += f * u;                      // Eq. 1b-c: f delta_i1 and f u_1
      Sc[o + 1 * P.N] = r[1]; Sc[o + 4 * P.N] = r[4];
    }
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      const double sp = alpha != 0.0 ? Sp[o + v * P.N] : 0.0;
      wv[v] += dt * (alpha * sp + beta * r[v]);
    }
    const int j = (int)((o / P.nx) % P.ny);
    if ((j == 0 && P.bc[2] == BC_WALL_NODE) || (j == P.ny - 1 && P.bc[3] == BC_WALL_NODE)) {
      const double Twl = j == 0 ? P.Twall[0] : P.Twall[1];
      wv[1] = 0.0; wv[2] = 0.0; wv[3] = 0.0; wv[4] = wv[0] * P.cv * Twl;
    }
#pragma unroll
    for (int v = 0; v < 5; ++v) w[o + v * P.N] = wv[v];
  }
}

// R_rhou += f, R_rhoE += f u  (streams_rhs with forcing)
__global__ void __launch_bounds__(RT) k_apply_force(const DevP P, const double* __restrict__ w, double* __restrict__ R,
                                                    const DevScal* __restrict__ sc) {
  const double f = sc->force;
  for (long long o = blockIdx.x * (long long)RT + threadIdx.x; o < P.N; o += (long long)gridDim.x * RT) {
    const double u = w[o + P.N] / w[o];
    R[o + 1 * P.N] += f;
    R[o + 4 * P.N] += f * u;
  }
}

// ---- S9: per-block partial sums of R_rhou * vol ----
__global__ void __launch_bounds__(RT) k_force_partial(const DevP P, const double* __restrict__ R, double* __restrict__ partial) {
  __shared__ double sh[RT / 32];
  double acc = 0.0;
  for (long long o = blockIdx.x * (long long)RT + threadIdx.x; o < P.N; o += (long long)gridDim.x * RT) {
    const int i = (int)(o % P.nx), j = (int)((o / P.nx) % P.ny), k = (int)(o / ((long long)P.nx * P.ny));
    acc += R[o + P.N] * (P.hh[0][i] * P.hh[1][j] * P.hh[2][k]);
  }
  const double t = block_sum<RT>(acc, sh, threadIdx.x);
  if (threadIdx.x == 0) partial[blockIdx.x] = t;
}
// f = - sum(partials) / sum(vol), fixed summation order (one CTA)
__global__ void __launch_bounds__(RT) k_force_final(const double* __restrict__ partial, int n, DevScal* sc) {
  __shared__ double sh[RT / 32];
  double acc = 0.0;
  for (int e = threadIdx.x; e < n; e += RT) acc += partial[e];
  const double t = block_sum<RT>(acc, sh, threadIdx.x);
  if (threadIdx.x == 0) sc->force = -t / sc->vol_total;
}

// ---- S10: dt = cfl / max_d max_nodes (|u_d| + c) / h_d ----
__global__ void __launch_bounds__(RT) k_speed_partial(const DevP P, const double* __restrict__ w, double* __restrict__ partial /*[3][grid]*/) {
  __shared__ double sh[RT / 32];
  double m[3] = {0.0, 0.0, 0.0};
  for (long long o = blockIdx.x * (long long)RT + threadIdx.x; o < P.N; o += (long long)gridDim.x * RT) {
    const int i = (int)(o % P.nx), j = (int)((o / P.nx) % P.ny), k = (int)(o / ((long long)P.nx * P.ny));
    Prim q;
    cons2prim_nomu(P, w[o], w[o + P.N], w[o + 2 * P.N], w[o + 3 * P.N], w[o + 4 * P.N], q);
    const double cs = sqrt(P.gam * P.Rgas * q.T);
    m[0] = fmax(m[0], (fabs(q.u) + cs) * P.ih[0][i]);
    m[1] = fmax(m[1], (fabs(q.v) + cs) * P.ih[1][j]);
    m[2] = fmax(m[2], (fabs(q.w) + cs) * P.ih[2][k]);
  }
  for (int d = 0; d < 3; ++d) {
    const double t = block_max<RT>(m[d], sh, threadIdx.x);
    if (threadIdx.x == 0) partial[d * gridDim.x + blockIdx.x] = t;
  }
}
__global__ void __launch_bounds__(RT) k_dt_final(const double* __restrict__ partial, int n, double cfl, double dt_fixed,
                                                 DevScal* sc, double* __restrict__ speeds_out /* 3, may be NULL */, int set_dt) {
  __shared__ double sh[RT / 32];
  double mm = 0.0;
  for (int d = 0; d < 3; ++d) {
    double m = 0.0;
    for (int e = threadIdx.x; e < n; e += RT) m = fmax(m, partial[d * n + e]);
    const double t = block_max<RT>(m, sh, threadIdx.x);
    if (threadIdx.x == 0) { mm = fmax(mm, t); if (speeds_out) speeds_out[d] = t; }
  }
  if (threadIdx.x == 0 && set_dt) sc->dt = dt_fixed > 0.0 ? dt_fixed : cfl / mm;
}
__global__ void k_advance_time(DevScal* sc) { sc->time += sc->dt; }

// ---- diagnostics: per-block partials, reduced on the host by streams_diagnostics ----
constexpr int NDIAG = 12;   // mass, mx, my, mz, E, ke, vol | min rho, min p, max Mach | nonfinite | spare
__global__ void __launch_bounds__(RT) k_diag_partial(const DevP P, const double* __restrict__ w, double* __restrict__ partial /*[NDIAG][grid]*/) {
  __shared__ double sh[RT / 32];
  double s[7] = {0, 0, 0, 0, 0, 0, 0};
  double mnr = INFINITY, mnp = INFINITY, mxm = 0.0, bad = 0.0;
  for (long long o = blockIdx.x * (long long)RT + threadIdx.x; o < P.N; o += (long long)gridDim.x * RT) {
    const int i = (int)(o % P.nx), j = (int)((o / P.nx) % P.ny), k = (int)(o / ((long long)P.nx * P.ny));
    const double vol = P.hh[0][i] * P.hh[1][j] * P.hh[2][k];
    const double r = w[o], ru = w[o + P.N], rv = w[o + 2 * P.N], rw = w[o + 3 * P.N], rE = w[o + 4 * P.N];
    Prim q;
    cons2prim_nomu(P, r, ru, rv, rw, rE, q);
    const double ke = 0.5 * r * (q.u * q.u + q.v * q.v + q.w * q.w);
    const double p = P.gm1 * (rE - ke);
    s[0] += r * vol; s[1] += ru * vol; s[2] += rv * vol; s[3] += rw * vol; s[4] += rE * vol; s[5] += ke * vol; s[6] += vol;
    if (!(r > 0.0) || !(p > 0.0) || !isfinite(r) || !isfinite(p) || !isfinite(rE)) bad = 1.0;
    mnr = fmin(mnr, r); mnp = fmin(mnp, p);
    mxm = fmax(mxm, sqrt((q.u * q.u + q.v * q.v + q.w * q.w) / (P.gam * P.Rgas * q.T)));
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

// capture the frozen inflow plane (S1 INFLOW_FROZEN): inflow[v][k][j] = w[v][k][j][0]
__global__ void k_capture_inflow(const DevP P, const double* __restrict__ w, double* __restrict__ inflow) {
  const long long n = (long long)P.nz * P.ny;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < 5 * n; e += (long long)gridDim.x * blockDim.x) {
    const int v = (int)(e / n);
    const long long r = e % n;
    inflow[e] = w[v * P.N + r * P.nx];
  }
}

}  // namespace streams
