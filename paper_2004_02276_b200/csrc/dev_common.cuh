// dev_common.cuh -- device-side parameters, ghost-by-index rules (S1) and primitives (S3).
//
// No ghost node is ever stored: every kernel asks `fetch_*` for node (i,j,k) with indices in
// [-3, n+3) and the boundary kind decides where the value comes from (S1; PAPER.md:110,
// 126, 146).  The composition order x -> y -> z of the ghost rules (S1) is reproduced by
// resolving z first, then y, then x (each later direction reads the earlier one's ghost).
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace streams {

constexpr int HALO = 3;

enum { BC_PERIODIC = 0, BC_WALL_STAG = 1, BC_WALL_NODE = 2, BC_INFLOW = 3, BC_OUTFLOW = 4, BC_SHOCKGEN = 5, BC_EXTRAP = 6 };
enum { VISC_POWER = 0, VISC_SUTH = 1 };

// central coefficients of order 2L, zero-padded to three entries
struct Coef { double a[3], b[3]; };

struct DevP {
  int nx, ny, nz;
  int bc[6];
  int visc_model, weno, forcing, viscous, L;
  long long N;                       // nx*ny*nz
  double gam, gm1, Rgas, inv_R, cp, cv, cp_over_Pr;
  double mu_ref, T_ref, inv_Tref, visc_exp, suth_S;
  double th_thr, th_eps;
  double Twall[2];
  double fs[6], post[6];             // shock generator states as rho,u,v,w,T,mu
  Coef c;
  // O(n) arrays on the device (owned by the context)
  const double* ih[3];               // 1 / h_d(i)                       (S2)
  const double* gh[3];               // - g_d(i) / h_d(i)^3              (S2)
  const double* hh[3];               // h_d(i)
  const unsigned char* xpost;        // [nx+6]: 1 where the ghost-extended x is behind the generator shock
  const double* inflow;              // [5][nz][ny] frozen inflow plane (conservative)
};

// the six stored primitives; p and H are derived the same way everywhere (derive_pH)
struct Prim { double rho, u, v, w, T, mu; };

__device__ __forceinline__ int wrap(int i, int n) {
  while (i < 0) i += n;
  while (i >= n) i -= n;
  return i;
}

__device__ __forceinline__ double visc_mu(const DevP& P, double T) {
  const double t = T * P.inv_Tref;
  if (P.visc_model == VISC_SUTH) return P.mu_ref * t * sqrt(t) * (P.T_ref + P.suth_S) / (T + P.suth_S);
  return P.mu_ref * exp(P.visc_exp * log(t));          // power law mu ~ T^0.76 (north_star)
}

__device__ __forceinline__ void derive_pH(const DevP& P, const Prim& q, double& p, double& H) {
  p = q.rho * (P.Rgas * q.T);
  H = P.cp * q.T + 0.5 * (q.u * q.u + q.v * q.v + q.w * q.w);
}

// S3 without the viscosity (cheap part)
__device__ __forceinline__ void cons2prim_nomu(const DevP& P, double r, double ru, double rv, double rw, double rE, Prim& q) {
  const double ir = 1.0 / r;
  q.rho = r; q.u = ru * ir; q.v = rv * ir; q.w = rw * ir;
  const double ke = 0.5 * (q.u * q.u + q.v * q.v + q.w * q.w);
  const double p0 = P.gm1 * (rE - r * ke);
  q.T = p0 * ir * P.inv_R;
}

// index maps ----------------------------------------------------------------------------------
// x: returns source index; inflow=true means "take the frozen inflow plane"
__device__ __forceinline__ int map_x(const DevP& P, int i, bool& inflow) {
  inflow = false;
  if (i < 0) {
    const int b = P.bc[0];
    if (b == BC_PERIODIC) return wrap(i, P.nx);
    if (b == BC_INFLOW) { inflow = true; return 0; }
    return 0;
  }
  if (i >= P.nx) {
    if (P.bc[1] == BC_PERIODIC) return wrap(i, P.nx);
    return P.nx - 1;
  }
  return i;
}
// y: mode 0 plain, 1 reflect about wall 0, 2 reflect about wall 1, 3 shock-generator state
__device__ __forceinline__ int map_y(const DevP& P, int j, int& mode) {
  mode = 0;
  if (j < 0) {
    const int b = P.bc[2];
    if (b == BC_PERIODIC) return wrap(j, P.ny);
    if (b == BC_WALL_STAG) { mode = 1; return -j - 1; }
    if (b == BC_WALL_NODE) { mode = 1; return -j; }
    return 0;
  }
  if (j >= P.ny) {
    const int b = P.bc[3];
    if (b == BC_PERIODIC) return wrap(j, P.ny);
    if (b == BC_WALL_STAG) { mode = 2; return 2 * P.ny - 1 - j; }
    if (b == BC_WALL_NODE) { mode = 2; return 2 * (P.ny - 1) - j; }
    if (b == BC_SHOCKGEN) { mode = 3; return P.ny - 1; }
    return P.ny - 1;
  }
  return j;
}
__device__ __forceinline__ int map_z(const DevP& P, int k) {
  if (k < 0) return P.bc[4] == BC_PERIODIC ? wrap(k, P.nz) : 0;
  if (k >= P.nz) return P.bc[5] == BC_PERIODIC ? wrap(k, P.nz) : P.nz - 1;
  return k;
}

// S1 isothermal no-slip reflection at primitive level: u -> -u, T -> 2 Tw - T, p -> p, rho = p/(R T)
__device__ __forceinline__ void reflect(const DevP& P, double Tw, Prim& q) {
  const double p = q.rho * (P.Rgas * q.T);
  const double Tg = 2.0 * Tw - q.T;
  q.rho = p / (P.Rgas * Tg);
  q.u = -q.u; q.v = -q.v; q.w = -q.w;
  q.T = Tg;
}

// Primitives of node (i,j,k), any index in [-3, n+3).  WITH_MU=false skips the viscosity.
template <bool WITH_MU>
__device__ __forceinline__ void fetch_prim(const DevP& P, const double* __restrict__ w, int i, int j, int k, Prim& q) {
  const int kk = map_z(P, k);
  int ymode;
  const int jj = map_y(P, j, ymode);
  if (ymode == 3) {
    const double* s = P.xpost[i + HALO] ? P.post : P.fs;
    q.rho = s[0]; q.u = s[1]; q.v = s[2]; q.w = s[3]; q.T = s[4]; q.mu = s[5];
    return;
  }
  bool inflow;
  const int ii = map_x(P, i, inflow);
  double r, ru, rv, rw, rE;
  if (inflow) {
    const size_t o = (size_t)kk * P.ny + jj, st = (size_t)P.nz * P.ny;
    r = P.inflow[o]; ru = P.inflow[o + st]; rv = P.inflow[o + 2 * st]; rw = P.inflow[o + 3 * st]; rE = P.inflow[o + 4 * st];
  } else {
    const size_t o = ((size_t)kk * P.ny + jj) * P.nx + ii;
    r = __ldg(w + o); ru = __ldg(w + o + P.N); rv = __ldg(w + o + 2 * P.N); rw = __ldg(w + o + 3 * P.N); rE = __ldg(w + o + 4 * P.N);
  }
  cons2prim_nomu(P, r, ru, rv, rw, rE, q);
  if (ymode == 1) reflect(P, P.Twall[0], q);
  else if (ymode == 2) reflect(P, P.Twall[1], q);
  if (WITH_MU) q.mu = visc_mu(P, q.T);
}

// velocities only (sensor, mixed-derivative look-ahead tile)
__device__ __forceinline__ void fetch_vel(const DevP& P, const double* __restrict__ w, int i, int j, int k, double& u, double& v, double& ww) {
  const int kk = map_z(P, k);
  int ymode;
  const int jj = map_y(P, j, ymode);
  if (ymode == 3) {
    const double* s = P.xpost[i + HALO] ? P.post : P.fs;
    u = s[1]; v = s[2]; ww = s[3];
    return;
  }
  bool inflow;
  const int ii = map_x(P, i, inflow);
  double r, ru, rv, rw;
  if (inflow) {
    const size_t o = (size_t)kk * P.ny + jj, st = (size_t)P.nz * P.ny;
    r = P.inflow[o]; ru = P.inflow[o + st]; rv = P.inflow[o + 2 * st]; rw = P.inflow[o + 3 * st];
  } else {
    const size_t o = ((size_t)kk * P.ny + jj) * P.nx + ii;
    r = __ldg(w + o); ru = __ldg(w + o + P.N); rv = __ldg(w + o + 2 * P.N); rw = __ldg(w + o + 3 * P.N);
  }
  const double ir = 1.0 / r;
  u = ru * ir; v = rv * ir; ww = rw * ir;
  if (ymode == 1 || ymode == 2) { u = -u; v = -v; ww = -ww; }
}

// block-wide sum / max in a fixed order (deterministic): result valid in thread 0
template <int NT_>
__device__ __forceinline__ double block_sum(double v, double* sh /* >= NT_/32 doubles */, int tid) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  const int lane = tid & 31, wid = tid >> 5;
  __syncthreads();
  if (lane == 0) sh[wid] = v;
  __syncthreads();
  double r = 0.0;
  if (tid == 0) for (int i = 0; i < NT_ / 32; ++i) r += sh[i];
  return r;
}
template <int NT_>
__device__ __forceinline__ double block_max(double v, double* sh, int tid) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
  const int lane = tid & 31, wid = tid >> 5;
  __syncthreads();
  if (lane == 0) sh[wid] = v;
  __syncthreads();
  double r = -INFINITY;
  if (tid == 0) for (int i = 0; i < NT_ / 32; ++i) r = fmax(r, sh[i]);
  return r;
}

}  // namespace streams
