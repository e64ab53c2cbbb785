// k_rhs.cuh -- the fused right-hand-side kernel (rows a1,a4,a6,a7,a8,a9 of the scope table).
//
// One CTA owns a TX x TY tile of (x,y) nodes and marches over a chunk of z planes (2.5-D
// blocking), one node per thread.  The state arrives as primitives Q = rho,u,v,w,T,mu (see
// dev_common.cuh), so filling a tile is load + store (+ p and H); nothing transcendental runs
// per stencil point.  Per plane s a CTA holds
//   * tile[s&1] : rho,u,v,w,p,H,T,mu of plane s for the tile plus a halo of 3 (shared memory,
//                 double-buffered so that one barrier separates fill from use),
//   * z-windows of rho,u,v,w,T,mu for planes s-3..s+3 in REGISTERS,
//   * the staging rows D_y v / D_x u on the x- / y-extended tile for the xy mixed derivatives,
//   * thread-private rings (shared memory, [slot][field][tid]) of the three in-plane derivative
//     fields d_x w, d_y w, d_x u + d_y v of planes s-6..s and of the partial residual of
//     planes s-3..s: the z-mixed terms d_z(d_x w), d_z(d_y w), d_z(d_x u + d_y v) of plane s-3
//     need planes up to s, so the result of plane s-3 is completed and written at step s
//     ("delayed output") instead of loading a look-ahead tile.
// Convective terms: Eq. 6-7 in the telescoped pair form
//   F_{i+1/2} - F_{i-1/2} = 2 sum_l a_l [ (rho,u,phi)~_{i,l} - (rho,u,phi)~_{i-l,l} ],
// factored per node as phi_i * sum_l (A_l - B_l) + sum_l (A_l phi_{i+l} - B_l phi_{i-l}) with
// A_l = a_l/4 (rho_i+rho_{i+l})(un_i+un_{i+l}), B_l likewise for i-l: the same sum of the same
// pair products (equal up to rounding order).
// Viscous terms: Laplacian form, Eq. 9 and DESIGN.md S7.
// The epilogue either writes R (streams_rhs, forcing path) or applies the RK3 stage of Eq. 11
// (the paper's own update loop is PAPER.md:209-225) and writes the new primitives.
#pragma once
#include "dev_common.cuh"

namespace streams {

constexpr int TX = 32, TY = 8, NT = TX * TY;
constexpr int PX = TX + 2 * HALO, PY = TY + 2 * HALO;
constexpr int PITCH = PX;                       // doubles per tile row
constexpr int TILE = PY * PITCH;                // doubles per tile field
enum { F_RHO = 0, F_U, F_V, F_W, F_P, F_H, F_T, F_MU, NF };

constexpr int SM_TILE1 = NF * TILE;             // one plane
constexpr int SM_TILES = 2 * SM_TILE1;          // double-buffered
constexpr int SM_STGY = TY * PITCH;             // D_y v on the x-extended rows
constexpr int SM_STGX = PY * TX;                // D_x u on the y-extended columns
constexpr int SM_GRING = 7 * 3 * NT;            // private rings of d_x w, d_y w, d_x u + d_y v
constexpr int SM_RRING = 4 * 5 * NT;            // private ring of the partial residual
constexpr int SM_RED = 16;
constexpr int SM_RHS_DOUBLES = SM_TILES + SM_STGY + SM_STGX + SM_GRING + SM_RRING + SM_RED;
constexpr int NHALO = 2 * HALO * TX + 2 * HALO * TY + 4 * HALO * HALO;   // 276 halo slots per tile
constexpr int NSTAGE = 2 * HALO * TY + 2 * HALO * TX;                     // 240 staged derivatives outside the tile

struct RhsArgs {
  const double* q;        // primitives the residual is evaluated on, [6][N]
  double* out_rhs;        // !FUSED: R goes here, [5][N]
  double* q_out;          // FUSED: primitives of w + dt (alpha S_prev + beta R)
  const double* S_prev;   // FUSED: R of the previous stage (ignored when alpha == 0)
  double* S_out;          // FUSED: R of this stage (may alias S_prev)
  const double* dt_ptr;   // FUSED: time step on the device
  double alpha, beta;
  double* partial;        // per-CTA partial sums of R_rhou * vol (forcing), may be NULL
  int lz;                 // planes per CTA
};

struct Nb { double rho, u, v, w, p, H, T, mu; };
// index-space sums of one direction: convective (Dm, c*), first (d*) and second (e*) differences
struct DirAcc { double Dm, cu, cv, cw, cH, cp, du, dv, dw, dT, dmu, eu, ev, ew, eT; };

__device__ __forceinline__ void acc_zero(DirAcc& A) {
  A.Dm = A.cu = A.cv = A.cw = A.cH = A.cp = 0.0;
  A.du = A.dv = A.dw = A.dT = A.dmu = 0.0;
  A.eu = A.ev = A.ew = A.eT = 0.0;
}

// contribution of the node pair (i, i+l) and (i-l, i) along direction D  (Eq. 6-7; Eq. 9 differences)
template <int D>
__device__ __forceinline__ void dir_accum(const double a, const double b, const Nb& c, const Nb& p, const Nb& m, DirAcc& A) {
  const double unc = D == 0 ? c.u : (D == 1 ? c.v : c.w);
  const double unp = D == 0 ? p.u : (D == 1 ? p.v : p.w);
  const double unm = D == 0 ? m.u : (D == 1 ? m.v : m.w);
  const double qa = 0.25 * a;
  const double Ap = qa * ((c.rho + p.rho) * (unc + unp));
  const double Bm = qa * ((m.rho + c.rho) * (unm + unc));
  A.Dm += Ap - Bm;
  A.cu = fma(Ap, p.u, A.cu); A.cu = fma(-Bm, m.u, A.cu);
  A.cv = fma(Ap, p.v, A.cv); A.cv = fma(-Bm, m.v, A.cv);
  A.cw = fma(Ap, p.w, A.cw); A.cw = fma(-Bm, m.w, A.cw);
  A.cH = fma(Ap, p.H, A.cH); A.cH = fma(-Bm, m.H, A.cH);
  A.cp = fma(a, p.p - m.p, A.cp);
  A.du = fma(a, p.u - m.u, A.du);
  A.dv = fma(a, p.v - m.v, A.dv);
  A.dw = fma(a, p.w - m.w, A.dw);
  A.dT = fma(a, p.T - m.T, A.dT);
  A.dmu = fma(a, p.mu - m.mu, A.dmu);
  A.eu = fma(b, fma(-2.0, c.u, p.u + m.u), A.eu);
  A.ev = fma(b, fma(-2.0, c.v, p.v + m.v), A.ev);
  A.ew = fma(b, fma(-2.0, c.w, p.w + m.w), A.ew);
  A.eT = fma(b, fma(-2.0, c.T, p.T + m.T), A.eT);
}
// F_{+1/2} - F_{-1/2} (index space) of the five equations from the sums of one direction
template <int D>
__device__ __forceinline__ void conv_from_acc(const Nb& c, const DirAcc& A, double f[5]) {
  f[0] = 2.0 * A.Dm;
  f[1] = fma(c.u, A.Dm, A.cu);
  f[2] = fma(c.v, A.Dm, A.cv);
  f[3] = fma(c.w, A.Dm, A.cw);
  f[4] = fma(c.H, A.Dm, A.cH);
  f[1 + D] += A.cp;
}

__device__ __forceinline__ Nb tile_nb(const double* __restrict__ t, int o) {
  Nb q;
  q.rho = t[F_RHO * TILE + o]; q.u = t[F_U * TILE + o]; q.v = t[F_V * TILE + o]; q.w = t[F_W * TILE + o];
  q.p = t[F_P * TILE + o]; q.H = t[F_H * TILE + o]; q.T = t[F_T * TILE + o]; q.mu = t[F_MU * TILE + o];
  return q;
}

// central flux of Eq. 7 in flux form at the interface above tile offset o (rows o, o+st), y only:
// used next to a staggered wall, where the wall-plane flux keeps the pressure only
__device__ __forceinline__ void flux_y_full(const DevP& P, const double* __restrict__ t, int o, int st, double F[5]) {
#pragma unroll
  for (int v = 0; v < 5; ++v) F[v] = 0.0;
#pragma unroll
  for (int l = 1; l <= 3; ++l) {
    const double a = P.c.a[l - 1];
#pragma unroll
    for (int m = 0; m < l; ++m) {
      const int oa = o - m * st, ob = o + (l - m) * st;
      const double mm = (t[F_RHO * TILE + oa] + t[F_RHO * TILE + ob]) * (t[F_V * TILE + oa] + t[F_V * TILE + ob]);
      F[0] += (0.5 * a) * mm;
      F[1] += (0.25 * a) * (mm * (t[F_U * TILE + oa] + t[F_U * TILE + ob]));
      F[2] += (0.25 * a) * (mm * (t[F_V * TILE + oa] + t[F_V * TILE + ob]));
      F[3] += (0.25 * a) * (mm * (t[F_W * TILE + oa] + t[F_W * TILE + ob]));
      F[4] += (0.25 * a) * (mm * (t[F_H * TILE + oa] + t[F_H * TILE + ob]));
      F[2] += a * (t[F_P * TILE + oa] + t[F_P * TILE + ob]);
    }
  }
}
__device__ __forceinline__ double flux_y_pressure(const DevP& P, const double* __restrict__ t, int o, int st) {
  double F = 0.0;
#pragma unroll
  for (int l = 1; l <= 3; ++l)
#pragma unroll
    for (int m = 0; m < l; ++m) F += P.c.a[l - 1] * (t[F_P * TILE + o - m * st] + t[F_P * TILE + o + (l - m) * st]);
  return F;
}

__device__ __forceinline__ double d1_tile(const DevP& P, const double* __restrict__ f, int o, int st) {
  double d1 = 0.0;
#pragma unroll
  for (int l = 1; l <= 3; ++l) d1 = fma(P.c.a[l - 1], f[o + l * st] - f[o - l * st], d1);
  return d1;
}

__device__ __forceinline__ void tile_put(const DevP& P, double* __restrict__ t, int o, const Prim& q, bool full) {
  t[F_U * TILE + o] = q.u; t[F_V * TILE + o] = q.v; t[F_W * TILE + o] = q.w;
  if (full) {
    double pp, HH;
    derive_pH(P, q.rho, q.u, q.v, q.w, q.T, pp, HH);
    t[F_RHO * TILE + o] = q.rho; t[F_P * TILE + o] = pp; t[F_H * TILE + o] = HH; t[F_T * TILE + o] = q.T; t[F_MU * TILE + o] = q.mu;
  }
}

template <bool FUSED>
__global__ void __launch_bounds__(NT, 1) k_rhs(const DevP P, const RhsArgs A) {
  extern __shared__ double sm[];
  double* tiles = sm;
  double* sgY = tiles + SM_TILES;
  double* sgX = sgY + SM_STGY;
  double* gring = sgX + SM_STGX;
  double* rring = gring + SM_GRING;
  double* red = rring + SM_RRING;

  const int ti = threadIdx.x, tj = threadIdx.y, tid = tj * TX + ti;
  const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY;
  const int gi = i0 + ti, gj = j0 + tj;
  const int k0 = blockIdx.z * A.lz;
  const int k1 = min(k0 + A.lz, P.nz);
  const bool active = gi < P.nx && gj < P.ny;
  const int oc = (tj + HALO) * PITCH + ti + HALO;                             // own tile offset
  const int own_off = gj * P.nx + gi;

  // Tile slots this thread fills besides its own node: slot 0 = its own position when that lies outside the
  // grid but inside the ghost range (ragged tiles); slots 1,2 = halo list entries tid and tid + NT:
  // [0,192) y-halo rows, [192,240) x-halo columns, [240,276) corners.
  Src es[3];
  int eo[3];
  es[0].kind = SRC_NONE; es[0].off = 0; eo[0] = oc;
  if (!active && gi < P.nx + HALO && gj < P.ny + HALO) es[0] = resolve_xy(P, gi, gj);
#pragma unroll
  for (int r = 0; r < 2; ++r) {
    const int e = tid + r * NT;
    int io = 0, jo = 0;
    bool any = true;
    if (e < 192) { const int rr = e / TX; jo = rr < 3 ? rr - 3 : TY + rr - 3; io = e % TX; }
    else if (e < 240) { const int e2 = e - 192; jo = e2 / 6; const int c = e2 % 6; io = c < 3 ? c - 3 : TX + c - 3; }
    else if (e < NHALO) { const int e3 = e - 240; const int rr = e3 / 6, c = e3 % 6; jo = rr < 3 ? rr - 3 : TY + rr - 3; io = c < 3 ? c - 3 : TX + c - 3; }
    else any = false;
    if (any && (i0 + io >= P.nx + HALO || j0 + jo >= P.ny + HALO)) any = false;
    es[r + 1].kind = SRC_NONE; es[r + 1].off = 0;
    if (any) es[r + 1] = resolve_xy(P, i0 + io, j0 + jo);
    eo[r + 1] = (jo + HALO) * PITCH + io + HALO;
  }
  // staged derivative outside the tile: [0,48) D_y v on the x-halo columns, [48,240) D_x u on the y-halo rows
  int sj_src = 0, sj_dst = -1, sj_st = 1, sj_f = F_U;
  if (tid < 2 * HALO * TY) {
    const int r = tid / 6, c = tid % 6, io = c < 3 ? c - 3 : TX + c - 3;
    sj_src = (r + HALO) * PITCH + io + HALO; sj_dst = r * PITCH + io + HALO; sj_st = PITCH; sj_f = F_V;
  } else if (tid < NSTAGE) {
    const int e2 = tid - 2 * HALO * TY, rr = e2 / TX, col = e2 % TX, jo = rr < 3 ? rr - 3 : TY + rr - 3;
    sj_src = (jo + HALO) * PITCH + col + HALO; sj_dst = SM_STGY + (jo + HALO) * TX + col; sj_st = 1; sj_f = F_U;
  }

  const double ihx = active ? P.ih[0][gi] : 0.0, ihy = active ? P.ih[1][gj] : 0.0;
  const double ghx = active ? P.gh[0][gi] : 0.0, ghy = active ? P.gh[1][gj] : 0.0;
  const double hxy = active ? P.hh[0][gi] * P.hh[1][gj] : 0.0;
#define a1 P.c.a[0]
#define a2 P.c.a[1]
#define a3 P.c.a[2]
#define b1 P.c.b[0]
#define b2 P.c.b[1]
#define b3 P.c.b[2]

  // register windows: index a holds plane s-3+a
  double rw[7], uw[7], vw[7], ww[7], Tw[7], mw[7];
#pragma unroll
  for (int a = 0; a < 7; ++a) { rw[a] = 1.0; uw[a] = vw[a] = ww[a] = 0.0; Tw[a] = mw[a] = 1.0; }
  if (active) {
#pragma unroll
    for (int a = 4; a < 7; ++a) {          // planes k0-3 .. k0-1 (they shift down by one before first use)
      Prim q;
      Src so; so.kind = SRC_FIELD; so.off = own_off;
      load_src_raw(P, A.q, so, map_z(P, k0 - 7 + a), q);
      rw[a] = q.rho; uw[a] = q.u; vw[a] = q.v; ww[a] = q.w; Tw[a] = q.T; mw[a] = q.mu;
    }
  }
  double fsum = 0.0;
  const double dt = FUSED ? *A.dt_ptr : 0.0;
  int slot7 = 0;                                     // it % 7

  for (int s = k0 - 3, it = 0; s < k1 + 3; ++s, ++it) {
    const bool full = s >= k0 && s < k1;
    const int ks = map_z(P, s);
    // ---------------- loads: halo slots of plane s, own node of plane s+3 ----------------------
    Prim hq[3];
#pragma unroll
    for (int r = 0; r < 3; ++r)
      if (es[r].kind) load_src_raw(P, A.q, es[r], ks, hq[r]);
    Prim pq;
    pq.rho = 1.0; pq.u = pq.v = pq.w = 0.0; pq.T = 1.0; pq.mu = 1.0;
    if (active) {
      Src so; so.kind = SRC_FIELD; so.off = own_off;
      load_src_raw(P, A.q, so, map_z(P, s + 3), pq);
    }
#pragma unroll
    for (int a = 0; a < 6; ++a) { rw[a] = rw[a + 1]; uw[a] = uw[a + 1]; vw[a] = vw[a + 1]; ww[a] = ww[a + 1]; Tw[a] = Tw[a + 1]; mw[a] = mw[a + 1]; }
    rw[6] = pq.rho; uw[6] = pq.u; vw[6] = pq.v; ww[6] = pq.w; Tw[6] = pq.T; mw[6] = pq.mu;

    // ---------------- tile of plane s ----------------------------------------------------------
    double* t = tiles + (it & 1) * SM_TILE1;
    if (active) {
      Prim pc; pc.rho = rw[3]; pc.u = uw[3]; pc.v = vw[3]; pc.w = ww[3]; pc.T = Tw[3]; pc.mu = mw[3];
      tile_put(P, t, oc, pc, full);
    }
#pragma unroll
    for (int r = 0; r < 3; ++r)
      if (es[r].kind) { apply_reflect(P, es[r], hq[r]); tile_put(P, t, eo[r], hq[r], full); }
    __syncthreads();
    // ---------------- in-plane derivatives shared through the staging rows ---------------------
    const double dxu = d1_tile(P, t + F_U * TILE, oc, 1);
    const double dyv = d1_tile(P, t + F_V * TILE, oc, PITCH);
    sgX[(tj + HALO) * TX + ti] = dxu;
    sgY[tj * PITCH + ti + HALO] = dyv;
    if (sj_dst >= 0) sgY[sj_dst] = d1_tile(P, t + sj_f * TILE, sj_src, sj_st);    // sgX follows sgY in memory
    __syncthreads();
    if (!active) continue;

    const int sl7 = slot7;
    slot7 = slot7 == 6 ? 0 : slot7 + 1;
    double g1, g2, g3;
    if (!full) {
      g1 = d1_tile(P, t + F_W * TILE, oc, 1) * ihx;
      g2 = d1_tile(P, t + F_W * TILE, oc, PITCH) * ihy;
      g3 = dxu * ihx + dyv * ihy;
    } else {
      // ================= plane s: everything except the z-mixed second derivatives ==============
      const double ihz = P.ih[2][s], ghz = P.gh[2][s];
      Nb c;
      c.rho = rw[3]; c.u = uw[3]; c.v = vw[3]; c.w = ww[3]; c.T = Tw[3]; c.mu = mw[3];
      c.p = t[F_P * TILE + oc]; c.H = t[F_H * TILE + oc];
      double G[3][3], lap[3], gth[3], Tj[3], Mj[3], T2;
      double R[5];
      // ---- x ----
      {
        DirAcc X;
        acc_zero(X);
        { const Nb p = tile_nb(t, oc + 1), m = tile_nb(t, oc - 1); dir_accum<0>(a1, b1, c, p, m, X); }
        { const Nb p = tile_nb(t, oc + 2), m = tile_nb(t, oc - 2); dir_accum<0>(a2, b2, c, p, m, X); }
        { const Nb p = tile_nb(t, oc + 3), m = tile_nb(t, oc - 3); dir_accum<0>(a3, b3, c, p, m, X); }
        double f[5];
        conv_from_acc<0>(c, X, f);
        if (gi == P.nx - 1 && P.bc[1] == BC_OUTFLOW) {
          // S8: characteristic form of the x-derivative at the outflow node, incoming waves removed
          const Nb n1 = tile_nb(t, oc - 1), n2 = tile_nb(t, oc - 2);
          const double w0[5] = {c.rho, c.rho * c.u, c.rho * c.v, c.rho * c.w, c.rho * c.H - c.p};
          const double w1[5] = {n1.rho, n1.rho * n1.u, n1.rho * n1.v, n1.rho * n1.w, n1.rho * n1.H - n1.p};
          const double w2[5] = {n2.rho, n2.rho * n2.u, n2.rho * n2.v, n2.rho * n2.w, n2.rho * n2.H - n2.p};
          double dw[5];
#pragma unroll
          for (int v = 0; v < 5; ++v) dw[v] = (3.0 * w0[v] - 4.0 * w1[v] + w2[v]) * 0.5;   // * ihx below
          const double u = c.u, v_ = c.v, w_ = c.w;
          const double q2 = u * u + v_ * v_ + w_ * w_;
          const double Hc = P.cp * c.T + 0.5 * q2;
          const double c2 = P.gm1 * (Hc - 0.5 * q2), cs = sqrt(c2);
          const double bb1 = P.gm1 / c2, bb2 = 0.5 * q2 * bb1;
          const double mdw = u * dw[1] + v_ * dw[2] + w_ * dw[3];
          double Ls[5];
          Ls[0] = 0.5 * ((bb2 + u / cs) * dw[0] - bb1 * mdw - dw[1] / cs + bb1 * dw[4]);
          Ls[1] = (1.0 - bb2) * dw[0] + bb1 * mdw - bb1 * dw[4];
          Ls[2] = -v_ * dw[0] + dw[2];
          Ls[3] = -w_ * dw[0] + dw[3];
          Ls[4] = 0.5 * ((bb2 - u / cs) * dw[0] - bb1 * mdw + dw[1] / cs + bb1 * dw[4]);
          const double lam[5] = {u - cs, u, u, u, u + cs};
#pragma unroll
          for (int m = 0; m < 5; ++m) Ls[m] = lam[m] >= 0.0 ? lam[m] * Ls[m] : 0.0;
          f[0] = Ls[0] + Ls[1] + Ls[4];
          f[1] = (u - cs) * Ls[0] + u * Ls[1] + (u + cs) * Ls[4];
          f[2] = v_ * Ls[0] + v_ * Ls[1] + Ls[2] + v_ * Ls[4];
          f[3] = w_ * Ls[0] + w_ * Ls[1] + Ls[3] + w_ * Ls[4];
          f[4] = (Hc - u * cs) * Ls[0] + 0.5 * q2 * Ls[1] + v_ * Ls[2] + w_ * Ls[3] + (Hc + u * cs) * Ls[4];
        }
#pragma unroll
        for (int v = 0; v < 5; ++v) R[v] = -(ihx * f[v]);
        const double i2 = ihx * ihx;
        G[0][0] = dxu * ihx; G[1][0] = X.dv * ihx; G[2][0] = X.dw * ihx; Tj[0] = X.dT * ihx; Mj[0] = X.dmu * ihx;
        const double s0 = fma(dxu, ghx, X.eu * i2), s1 = fma(X.dv, ghx, X.ev * i2), s2 = fma(X.dw, ghx, X.ew * i2);
        lap[0] = s0; lap[1] = s1; lap[2] = s2; gth[0] = s0;
        T2 = fma(X.dT, ghx, X.eT * i2);
      }
      // ---- y ----
      {
        DirAcc Y;
        acc_zero(Y);
        { const Nb p = tile_nb(t, oc + PITCH), m = tile_nb(t, oc - PITCH); dir_accum<1>(a1, b1, c, p, m, Y); }
        { const Nb p = tile_nb(t, oc + 2 * PITCH), m = tile_nb(t, oc - 2 * PITCH); dir_accum<1>(a2, b2, c, p, m, Y); }
        { const Nb p = tile_nb(t, oc + 3 * PITCH), m = tile_nb(t, oc - 3 * PITCH); dir_accum<1>(a3, b3, c, p, m, Y); }
        double f[5];
        conv_from_acc<1>(c, Y, f);
        const bool wall_lo = gj == 0 && P.bc[2] == BC_WALL_STAG;
        const bool wall_hi = gj == P.ny - 1 && P.bc[3] == BC_WALL_STAG;
        if (wall_lo || wall_hi) {
          double Fp[5] = {0, 0, 0, 0, 0}, Fm[5] = {0, 0, 0, 0, 0};
          if (wall_hi) Fp[2] = flux_y_pressure(P, t, oc, PITCH); else flux_y_full(P, t, oc, PITCH, Fp);
          if (wall_lo) Fm[2] = flux_y_pressure(P, t, oc - PITCH, PITCH); else flux_y_full(P, t, oc - PITCH, PITCH, Fm);
#pragma unroll
          for (int v = 0; v < 5; ++v) f[v] = Fp[v] - Fm[v];
        }
#pragma unroll
        for (int v = 0; v < 5; ++v) R[v] = fma(-ihy, f[v], R[v]);
        const double i2 = ihy * ihy;
        G[0][1] = Y.du * ihy; G[1][1] = dyv * ihy; G[2][1] = Y.dw * ihy; Tj[1] = Y.dT * ihy; Mj[1] = Y.dmu * ihy;
        const double s0 = fma(Y.du, ghy, Y.eu * i2), s1 = fma(dyv, ghy, Y.ev * i2), s2 = fma(Y.dw, ghy, Y.ew * i2);
        lap[0] += s0; lap[1] += s1; lap[2] += s2; gth[1] = s1;
        T2 += fma(Y.dT, ghy, Y.eT * i2);
      }
      // ---- z (register windows) ----
      {
        DirAcc Z;
        acc_zero(Z);
#pragma unroll
        for (int l = 1; l <= 3; ++l) {
          Nb p, m;
          p.rho = rw[3 + l]; p.u = uw[3 + l]; p.v = vw[3 + l]; p.w = ww[3 + l]; p.T = Tw[3 + l]; p.mu = mw[3 + l];
          m.rho = rw[3 - l]; m.u = uw[3 - l]; m.v = vw[3 - l]; m.w = ww[3 - l]; m.T = Tw[3 - l]; m.mu = mw[3 - l];
          derive_pH(P, p.rho, p.u, p.v, p.w, p.T, p.p, p.H);
          derive_pH(P, m.rho, m.u, m.v, m.w, m.T, m.p, m.H);
          dir_accum<2>(l == 1 ? a1 : (l == 2 ? a2 : a3), l == 1 ? b1 : (l == 2 ? b2 : b3), c, p, m, Z);
        }
        double f[5];
        conv_from_acc<2>(c, Z, f);
#pragma unroll
        for (int v = 0; v < 5; ++v) R[v] = fma(-ihz, f[v], R[v]);
        const double i2 = ihz * ihz;
        G[0][2] = Z.du * ihz; G[1][2] = Z.dv * ihz; G[2][2] = Z.dw * ihz; Tj[2] = Z.dT * ihz; Mj[2] = Z.dmu * ihz;
        const double s0 = fma(Z.du, ghz, Z.eu * i2), s1 = fma(Z.dv, ghz, Z.ev * i2), s2 = fma(Z.dw, ghz, Z.ew * i2);
        lap[0] += s0; lap[1] += s1; lap[2] += s2; gth[2] = s2;
        T2 += fma(Z.dT, ghz, Z.eT * i2);
      }
      g1 = G[2][0]; g2 = G[2][1]; g3 = G[0][0] + G[1][1];
      if (P.viscous) {
        // xy mixed terms (A8): d_x(d_y v) and d_y(d_x u) from the staging rows
        const int oy = tj * PITCH + ti + HALO, ox = (tj + HALO) * TX + ti;
        double mxy = a1 * (sgY[oy + 1] - sgY[oy - 1]);
        mxy = fma(a2, sgY[oy + 2] - sgY[oy - 2], mxy);
        mxy = fma(a3, sgY[oy + 3] - sgY[oy - 3], mxy);
        double myx = a1 * (sgX[ox + TX] - sgX[ox - TX]);
        myx = fma(a2, sgX[ox + 2 * TX] - sgX[ox - 2 * TX], myx);
        myx = fma(a3, sgX[ox + 3 * TX] - sgX[ox - 3 * TX], myx);
        const double ixy = ihx * ihy;
        gth[0] = fma(mxy, ixy, gth[0]);
        gth[1] = fma(myx, ixy, gth[1]);
        const double Th = G[0][0] + G[1][1] + G[2][2];
        double Vi[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
          const double cross = Mj[0] * (G[a][0] + G[0][a]) + Mj[1] * (G[a][1] + G[1][a]) + Mj[2] * (G[a][2] + G[2][a]);
          Vi[a] = c.mu * fma(gth[a], 1.0 / 3.0, lap[a]) + cross - (2.0 / 3.0) * Mj[a] * Th;
        }
        const double s01 = G[0][1] + G[1][0], s02 = G[0][2] + G[2][0], s12 = G[1][2] + G[2][1];
        const double Phi = c.mu * (2.0 * (G[0][0] * G[0][0] + G[1][1] * G[1][1] + G[2][2] * G[2][2]) + s01 * s01 + s02 * s02 + s12 * s12 - (2.0 / 3.0) * Th * Th);
        const double heat = P.cp_over_Pr * (c.mu * T2 + (Mj[0] * Tj[0] + Mj[1] * Tj[1] + Mj[2] * Tj[2]));
        R[1] += Vi[0]; R[2] += Vi[1]; R[3] += Vi[2];
        R[4] += c.u * Vi[0] + c.v * Vi[1] + c.w * Vi[2] + Phi + heat;
      }
      double* rr = rring + (it & 3) * 5 * NT + tid;
#pragma unroll
      for (int v = 0; v < 5; ++v) rr[v * NT] = R[v];
    }
    {
      double* gr = gring + sl7 * 3 * NT + tid;
      gr[0] = g1; gr[NT] = g2; gr[2 * NT] = g3;
    }
    // ================= plane p = s-3: add the z-mixed terms, write the result ====================
    const int p = s - 3;
    if (p < k0) continue;
    double R[5];
    {
      const double* rr = rring + ((it - 3) & 3) * 5 * NT + tid;
#pragma unroll
      for (int v = 0; v < 5; ++v) R[v] = rr[v * NT];
    }
    if (P.viscous) {
      // ring slot of plane p+l is (sl7 - 3 + l) mod 7
      double dz[3] = {0.0, 0.0, 0.0};
#pragma unroll
      for (int l = 1; l <= 3; ++l) {
        int sp = sl7 - 3 + l; if (sp < 0) sp += 7;
        int sn = sl7 - 3 - l; if (sn < 0) sn += 7;
        const double* gp = gring + sp * 3 * NT + tid;
        const double* gn = gring + sn * 3 * NT + tid;
        const double a = l == 1 ? a1 : (l == 2 ? a2 : a3);
#pragma unroll
        for (int m = 0; m < 3; ++m) dz[m] = fma(a, gp[m * NT] - gn[m * NT], dz[m]);
      }
      const double f3 = mw[0] * (1.0 / 3.0) * P.ih[2][p];
      const double v0 = f3 * dz[0], v1 = f3 * dz[1], v2 = f3 * dz[2];
      R[1] += v0; R[2] += v1; R[3] += v2;
      R[4] += uw[0] * v0 + vw[0] * v1 + ww[0] * v2;
    }
    fsum += R[1] * (hxy * P.hh[2][p]);
    // ---------------- epilogue: write R, or the RK3 stage of Eq. 11 ------------------------------
    const size_t o = (size_t)p * P.nxy + own_off;
    if (!FUSED) {
#pragma unroll
      for (int v = 0; v < 5; ++v) A.out_rhs[o + v * P.N] = R[v];
    } else {
      double dW[5];
#pragma unroll
      for (int v = 0; v < 5; ++v) {
        const double sp = A.alpha != 0.0 ? A.S_prev[o + v * P.N] : 0.0;
        dW[v] = dt * (A.alpha * sp + A.beta * R[v]);
        A.S_out[o + v * P.N] = R[v];
      }
      Prim qn; qn.rho = rw[0]; qn.u = uw[0]; qn.v = vw[0]; qn.w = ww[0]; qn.T = Tw[0]; qn.mu = mw[0];
      advance_prim(P, qn, dW);
      if (gj == 0 && P.bc[2] == BC_WALL_NODE) wall_node_override(P, P.Twall[0], P.mu_wall[0], qn);
      if (gj == P.ny - 1 && P.bc[3] == BC_WALL_NODE) wall_node_override(P, P.Twall[1], P.mu_wall[1], qn);
      A.q_out[o] = qn.rho; A.q_out[o + P.N] = qn.u; A.q_out[o + 2 * P.N] = qn.v; A.q_out[o + 3 * P.N] = qn.w;
      A.q_out[o + 4 * P.N] = qn.T; A.q_out[o + 5 * P.N] = qn.mu;
    }
  }
  if (A.partial) {
    const double tot = block_sum<NT>(fsum, red, tid);
    if (tid == 0) A.partial[(blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x] = tot;
  }
}

#undef a1
#undef a2
#undef a3
#undef b1
#undef b2
#undef b3

}  // namespace streams
