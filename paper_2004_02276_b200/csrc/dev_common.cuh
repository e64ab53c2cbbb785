// dev_common.cuh -- device-side parameters, ghost-by-index rules (S1) and primitives (S3).
//
// State layout in HBM: the library keeps the flow state as PRIMITIVES
//   Q[7][nz][ny][nx] = rho, u, v, w, T, mu, H     (x fastest, no ghost nodes stored)
// so that no kernel pays a division, the power-law viscosity or the total enthalpy when it loads
// a stencil point (a tile is filled by plain asynchronous copies); the conservative vector of
// PAPER.md:95 is formed in registers where Eq. 11 needs it.
// No ghost node is ever stored: a kernel asks `resolve_xy` where the value of an in-plane
// location (i,j), indices in [-3, n+3), comes from, and `map_z` for the plane (S1;
// PAPER.md:110, 126, 146).  The composition order x -> y -> z of the ghost rules is reproduced
// by resolving z first, then y, then x (each later direction reads the earlier one's ghost).
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace streams {

constexpr int HALO = 3;
constexpr int NQ = 7;                 // stored primitives per node

enum { BC_PERIODIC = 0, BC_WALL_STAG = 1, BC_WALL_NODE = 2, BC_INFLOW = 3, BC_OUTFLOW = 4, BC_SHOCKGEN = 5, BC_EXTRAP = 6, BC_WALL_CHAR = 7, BC_HALO = 8 };
enum { VISC_POWER = 0, VISC_SUTH = 1 };

// central coefficients of order 2L, zero-padded to three entries
struct Coef {
  double a[3], b[3];
  double qa[3];      // a_l / 4        (Eq. 6: the 1/4 of the triple average times 2 a_l / 2)
  double aR[3];      // a_l * Rgas     (pressure difference formed as Rgas * (rho T) differences)
  double sb2;        // 2 (b_1 + b_2 + b_3)
};

struct DevP {
  int nx, ny, nz, nxy;
  int bc[6];
  int visc_model, weno, forcing, viscous, L;
  long long N;                       // nx*ny*nz
  long long QS;                      // doubles between two fields of a primitive-state buffer: (nz + 2 zpad) * nxy
  int zpad;                          // ghost planes stored below / above the state (3 when a z face is BC_HALO, else 0)
  int IS;                            // doubles between two fields of the frozen inflow plane: (nz + 2 zpad) * ny
  double gam, gm1, Rgas, inv_R, cp, cv, inv_cv, cp_over_Pr;
  double mu_ref, T_ref, inv_Tref, visc_exp, suth_S;
  double th_thr, th_eps;
  double Twall[2], mu_wall[2];
  double fs[NQ], post[NQ];           // shock generator states as rho,u,v,w,T,mu,H
  Coef c;
  // O(n) arrays on the device (owned by the context)
  const double* ih[3];               // 1 / h_d(i)                       (S2)
  const double* gh[3];               // - g_d(i) / h_d(i)^3              (S2)
  const double* hh[3];               // h_d(i)
  const unsigned char* xpost;        // [nx+6]: 1 where the ghost-extended x is behind the generator shock
  const double* inflow;              // [NQ][nz][ny] frozen inflow plane (primitives)
};

struct Prim { double rho, u, v, w, T, mu, H; };

__device__ __forceinline__ int wrap(int i, int n) {
  while (i < 0) i += n;
  while (i >= n) i -= n;
  return i;
}

// S3 viscosity law: power law mu ~ T^0.76 (north_star) or Sutherland
__device__ __forceinline__ double visc_mu(const DevP& P, double T) {
  const double t = T * P.inv_Tref;
  if (P.visc_model == VISC_SUTH) return P.mu_ref * t * sqrt(t) * (P.T_ref + P.suth_S) / (T + P.suth_S);
  return P.mu_ref * exp(P.visc_exp * log(t));
}

// S3: p = rho R T, H = c_p T + |u|^2/2  (E = c_v T + |u|^2/2, H = E + p/rho)
__device__ __forceinline__ void derive_pH(const DevP& P, double rho, double u, double v, double w, double T, double& p, double& H) {
  p = rho * (P.Rgas * T);
  H = fma(P.cp, T, 0.5 * fma(u, u, fma(v, v, w * w)));
}

// S3 from the conservative vector (set_state): one division, one power law
__device__ __forceinline__ void cons2prim(const DevP& P, double r, double ru, double rv, double rw, double rE, Prim& q) {
  const double ir = 1.0 / r;
  q.rho = r; q.u = ru * ir; q.v = rv * ir; q.w = rw * ir;
  const double ke = 0.5 * (q.u * q.u + q.v * q.v + q.w * q.w);
  const double p0 = P.gm1 * (rE - r * ke);
  q.T = p0 * ir * P.inv_R;
  q.mu = visc_mu(P, q.T);
  q.H = fma(P.cp, q.T, ke);
}
__device__ __forceinline__ void prim2cons(const DevP& P, const Prim& q, double wv[5]) {
  wv[0] = q.rho; wv[1] = q.rho * q.u; wv[2] = q.rho * q.v; wv[3] = q.rho * q.w;
  wv[4] = q.rho * fma(P.cv, q.T, 0.5 * (q.u * q.u + q.v * q.v + q.w * q.w));
}

// Eq. 11 applied to a node held as primitives: w' = w + dW in conservative variables, written as
// increments of the primitives (exactly the same map; dW = 0 leaves the node bit-identical):
//   rho' = rho + dW0,  u' = u + (dW_u - u dW0)/rho',  E' = E + (dW_E - E dW0)/rho',
//   c_v T' = c_v T + (E' - E) - (|u'|^2 - |u|^2)/2
template <bool WITH_MU = true>
__device__ __forceinline__ void advance_prim(const DevP& P, Prim& q, const double dW[5]) {
  const double rn = q.rho + dW[0];
  const double ir = 1.0 / rn;
  const double du = (dW[1] - q.u * dW[0]) * ir, dv = (dW[2] - q.v * dW[0]) * ir, dw = (dW[3] - q.w * dW[0]) * ir;
  const double E = fma(P.cv, q.T, 0.5 * (q.u * q.u + q.v * q.v + q.w * q.w));
  const double dE = (dW[4] - E * dW[0]) * ir;
  const double un = q.u + du, vn = q.v + dv, wn = q.w + dw;
  const double dke = 0.5 * (du * (un + q.u) + dv * (vn + q.v) + dw * (wn + q.w));
  q.T = fma(dE - dke, P.inv_cv, q.T);
  q.rho = rn; q.u = un; q.v = vn; q.w = wn;
  if (WITH_MU) q.mu = visc_mu(P, q.T);
  q.H = fma(P.cp, q.T, 0.5 * fma(un, un, fma(vn, vn, wn * wn)));
}
// S1: Dirichlet override of a WALL_ISO_NODE wall node after every stage (rho evolves by the scheme)
__device__ __forceinline__ void wall_node_override(const DevP& P, double Tw, double mu_w, Prim& q) {
  q.u = 0.0; q.v = 0.0; q.w = 0.0; q.T = Tw; q.mu = mu_w; q.H = P.cp * Tw;
}

// wall on the boundary node (Dirichlet override after every stage): plain reflected-ghost wall or its characteristic variant
__device__ __forceinline__ bool node_wall(int bc) { return bc == BC_WALL_NODE || bc == BC_WALL_CHAR; }

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
    if (b == BC_WALL_NODE || b == BC_WALL_CHAR) { mode = 1; return -j; }
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
// z: plane index relative to the first interior plane.  A BC_HALO face keeps the index (-3..-1, nz..nz+2): those planes
// are STORED around the state (DevP::zpad) and filled by streams_halo_unpack with the neighbouring slab's planes.
__device__ __forceinline__ int map_z(const DevP& P, int k) {
  if (k < 0) return P.bc[4] == BC_PERIODIC ? wrap(k, P.nz) : (P.bc[4] == BC_HALO ? k : 0);
  if (k >= P.nz) return P.bc[5] == BC_PERIODIC ? wrap(k, P.nz) : (P.bc[5] == BC_HALO ? k : P.nz - 1);
  return k;
}

// Where the value of in-plane location (i,j) comes from.  kind & 7: 0 nothing, 1 the field Q at `off`
// (= jj*nx+ii inside a plane), 2 the frozen inflow plane (off = jj), 3 / 4 the free-stream / post-shock
// constant of the shock generator; kind >> 4: 0 plain, 1 / 2 isothermal reflection about wall 0 / 1.
struct Src { int off, kind; };
enum { SRC_NONE = 0, SRC_FIELD = 1, SRC_INFLOW = 2, SRC_FS = 3, SRC_POST = 4, SRC_LOCAL = 8 /* k_rhs patch list: source inside the tile */ };

__device__ __forceinline__ Src resolve_xy(const DevP& P, int i, int j) {
  Src s;
  int ymode;
  const int jj = map_y(P, j, ymode);
  if (ymode == 3) { s.off = 0; s.kind = P.xpost[i + HALO] ? SRC_POST : SRC_FS; return s; }
  bool inflow;
  const int ii = map_x(P, i, inflow);
  s.kind = (inflow ? SRC_INFLOW : SRC_FIELD) | (ymode << 4);
  s.off = inflow ? jj : jj * P.nx + ii;
  return s;
}

// viscosity law kept out of line and fed with scalars only (register ABI: no local-memory traffic): used on
// the rare ghost-row path of wall tiles so that the hot loop does not carry three inlined exp/log bodies
__device__ __noinline__ double visc_mu_outofline(double T, double mu_ref, double T_ref, double inv_Tref, double visc_exp, double suth_S, int model) {
  const double t = T * inv_Tref;
  if (model == VISC_SUTH) return mu_ref * t * sqrt(t) * (T_ref + suth_S) / (T + suth_S);
  return mu_ref * exp(visc_exp * log(t));
}
// S1 isothermal no-slip reflection: u -> -u, T -> 2 Tw - T, p -> p, rho = p/(R T)
__device__ __forceinline__ void reflect(const DevP& P, double Tw, Prim& q) {
  const double Tg = 2.0 * Tw - q.T;
  q.rho = (q.rho * q.T) / Tg;
  q.u = -q.u; q.v = -q.v; q.w = -q.w;
  q.T = Tg;
  q.mu = visc_mu_outofline(Tg, P.mu_ref, P.T_ref, P.inv_Tref, P.visc_exp, P.suth_S, P.visc_model);
  q.H = fma(P.cp, Tg, 0.5 * fma(q.u, q.u, fma(q.v, q.v, q.w * q.w)));
}

// raw load of the stored primitives for source s in (already mapped) plane kk; reflection NOT applied
__device__ __forceinline__ void load_src_raw(const DevP& P, const double* __restrict__ Q, const Src s, int kk, Prim& q) {
  const int k = s.kind & 7;
  if (k == SRC_FIELD) {
    const long long o = (long long)kk * P.nxy + s.off;
    q.rho = __ldg(Q + o); q.u = __ldg(Q + o + P.QS); q.v = __ldg(Q + o + 2 * P.QS); q.w = __ldg(Q + o + 3 * P.QS);
    q.T = __ldg(Q + o + 4 * P.QS); q.mu = __ldg(Q + o + 5 * P.QS); q.H = __ldg(Q + o + 6 * P.QS);
  } else if (k == SRC_INFLOW) {
    const long long o = (long long)kk * P.ny + s.off, st = P.IS;
    q.rho = P.inflow[o]; q.u = P.inflow[o + st]; q.v = P.inflow[o + 2 * st]; q.w = P.inflow[o + 3 * st];
    q.T = P.inflow[o + 4 * st]; q.mu = P.inflow[o + 5 * st]; q.H = P.inflow[o + 6 * st];
  } else {
    const double* c = k == SRC_POST ? P.post : P.fs;
    q.rho = c[0]; q.u = c[1]; q.v = c[2]; q.w = c[3]; q.T = c[4]; q.mu = c[5]; q.H = c[6];
  }
}
__device__ __forceinline__ void apply_reflect(const DevP& P, const Src s, Prim& q) {
  const int r = s.kind >> 4;
  if (r) reflect(P, P.Twall[r - 1], q);
}

// Primitives of node (i,j,k), any index in [-3, n+3) (generic path of the light kernels)
__device__ __forceinline__ void fetch_prim(const DevP& P, const double* __restrict__ Q, int i, int j, int k, Prim& q) {
  const Src s = resolve_xy(P, i, j);
  load_src_raw(P, Q, s, map_z(P, k), q);
  apply_reflect(P, s, q);
}
// rho, u, v, w, T only (WENO stencils: p, H and c are derived; mu is not needed, so a reflected ghost pays no power law)
__device__ __forceinline__ void fetch_prim5(const DevP& P, const double* __restrict__ Q, int i, int j, int k, Prim& q) {
  const Src s = resolve_xy(P, i, j);
  const int kk = map_z(P, k), kd = s.kind & 7;
  if (kd == SRC_FIELD) {
    const long long o = (long long)kk * P.nxy + s.off;
    q.rho = __ldg(Q + o); q.u = __ldg(Q + o + P.QS); q.v = __ldg(Q + o + 2 * P.QS); q.w = __ldg(Q + o + 3 * P.QS); q.T = __ldg(Q + o + 4 * P.QS);
  } else if (kd == SRC_INFLOW) {
    const long long o = (long long)kk * P.ny + s.off, st = P.IS;
    q.rho = P.inflow[o]; q.u = P.inflow[o + st]; q.v = P.inflow[o + 2 * st]; q.w = P.inflow[o + 3 * st]; q.T = P.inflow[o + 4 * st];
  } else {
    const double* c = kd == SRC_POST ? P.post : P.fs;
    q.rho = c[0]; q.u = c[1]; q.v = c[2]; q.w = c[3]; q.T = c[4];
  }
  const int r = s.kind >> 4;
  if (r) {                                   // S1 isothermal no-slip reflection (see reflect())
    const double Tg = 2.0 * P.Twall[r - 1] - q.T;
    q.rho = (q.rho * q.T) / Tg;
    q.u = -q.u; q.v = -q.v; q.w = -q.w; q.T = Tg;
  }
  q.mu = 0.0; q.H = 0.0;
}
// velocities only (sensor)
__device__ __forceinline__ void fetch_vel(const DevP& P, const double* __restrict__ Q, int i, int j, int k, double& u, double& v, double& w) {
  const Src s = resolve_xy(P, i, j);
  const int kk = map_z(P, k), kd = s.kind & 7;
  if (kd == SRC_FIELD) {
    const long long o = (long long)kk * P.nxy + s.off;
    u = __ldg(Q + o + P.QS); v = __ldg(Q + o + 2 * P.QS); w = __ldg(Q + o + 3 * P.QS);
  } else if (kd == SRC_INFLOW) {
    const long long o = (long long)kk * P.ny + s.off, st = P.IS;
    u = P.inflow[o + st]; v = P.inflow[o + 2 * st]; w = P.inflow[o + 3 * st];
  } else {
    const double* c = kd == SRC_POST ? P.post : P.fs;
    u = c[1]; v = c[2]; w = c[3];
  }
  if (s.kind >> 4) { u = -u; v = -v; w = -w; }
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
