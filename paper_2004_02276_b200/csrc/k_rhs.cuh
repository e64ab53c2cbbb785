// k_rhs.cuh -- the fused right-hand-side kernel (rows a1,a2,a4,a6,a7,a8,a9 of the scope table).
//
// One CTA owns a TX x TY tile of (x,y) nodes and marches over a chunk of z planes (2.5-D
// blocking).  Per plane s it holds
//   * tileS : the 8 primitives of plane s for the tile plus a halo of 3 (shared memory),
//   * tileQ : the velocities of plane s+3 (look-ahead) for the in-plane derivatives that the
//             z-mixed terms d_z(d_x w), d_z(d_y w), d_z(d_x u + d_y v) differentiate again,
//   * z-windows of u,v,w,T,mu (planes s-3..s+3) and rho (s..s+3) in REGISTERS, one node per thread,
//   * windows of the three in-plane derivative fields in thread-private shared memory.
// Convective terms: Eq. 6-7 in the telescoped pair form
//   F_{i+1/2} - F_{i-1/2} = 2 sum_l a_l [ (rho,u,phi)~_{i,l} - (rho,u,phi)~_{i-l,l} ],
// which is the same sum of the same pair products as the flux form; in z every pair is
// computed once and handed to both nodes through register accumulators.
// Viscous terms: Laplacian form, Eq. 9 and DESIGN.md S7.
// The epilogue either writes R (streams_rhs) or applies the RK3 stage of Eq. 11 in place of
// a separate update kernel (the paper's own update loop is PAPER.md:209-225).
#pragma once
#include "dev_common.cuh"

namespace streams {

constexpr int TX = 32, TY = 8, NT = TX * TY;
constexpr int PX = TX + 2 * HALO, PY = TY + 2 * HALO;
constexpr int PITCH = PX;                       // doubles per tile row
constexpr int TILE = PY * PITCH;                // doubles per tile field
enum { F_RHO = 0, F_U, F_V, F_W, F_P, F_H, F_T, F_MU, NF };

constexpr int SM_TILES = NF * TILE;             // tileS
constexpr int SM_TILEQ = 3 * TILE;              // tileQ (u,v,w of plane s+3)
constexpr int SM_STGY = TY * PITCH;             // D_y v on the x-extended rows
constexpr int SM_STGX = PY * TX;                // D_x u on the y-extended columns
constexpr int SM_MIXW = 7 * 3 * NT;             // private windows of Dxw, Dyw, divxy
constexpr int SM_RED = 16;
constexpr int SM_RHS_DOUBLES = SM_TILES + SM_TILEQ + SM_STGY + SM_STGX + SM_MIXW + SM_RED;

struct RhsArgs {
  const double* w;        // state the residual is evaluated on
  double* out_rhs;        // !FUSED: R goes here
  double* w_out;          // FUSED: w + dt (alpha S_prev + beta R)
  const double* S_prev;   // FUSED: R of the previous stage (ignored when alpha == 0)
  double* S_out;          // FUSED: R of this stage (may alias S_prev)
  const double* dt_ptr;   // FUSED: time step on the device
  double alpha, beta;
  double* partial;        // per-CTA partial sums of R_rhou * vol (forcing), may be NULL
  int lz;                 // planes per CTA
};

struct Q6 { double rho, u, v, w, H, p; };

// pair products of Eq. 6 for nodes a,b along direction D, without the constant factors
template <int D>
__device__ __forceinline__ void pair6(const Q6& a, const Q6& b, double f[6]) {
  const double una = D == 0 ? a.u : (D == 1 ? a.v : a.w);
  const double unb = D == 0 ? b.u : (D == 1 ? b.v : b.w);
  const double m = (a.rho + b.rho) * (una + unb);
  f[0] = m;
  f[1] = m * (a.u + b.u);
  f[2] = m * (a.v + b.v);
  f[3] = m * (a.w + b.w);
  f[4] = m * (a.H + b.H);
  f[5] = a.p + b.p;
}

__device__ __forceinline__ Q6 tile_q6(const double* __restrict__ t, int o) {
  Q6 q;
  q.rho = t[F_RHO * TILE + o]; q.u = t[F_U * TILE + o]; q.v = t[F_V * TILE + o]; q.w = t[F_W * TILE + o];
  q.H = t[F_H * TILE + o]; q.p = t[F_P * TILE + o];
  return q;
}

// F_{+1/2} - F_{-1/2} along D for the node at tile offset o (stride st), pair form
template <int D>
__device__ __forceinline__ void conv_inplane(const DevP& P, const double* __restrict__ t, int o, int st, double acc[5]) {
  const Q6 c = tile_q6(t, o);
#pragma unroll
  for (int l = 1; l <= 3; ++l) {
    const Q6 qp = tile_q6(t, o + l * st), qm = tile_q6(t, o - l * st);
    double fp[6], fm[6];
    pair6<D>(c, qp, fp);
    pair6<D>(qm, c, fm);
    const double a = P.c.a[l - 1];
    acc[0] += (0.5 * a) * (fp[0] - fm[0]);
#pragma unroll
    for (int v = 1; v < 5; ++v) acc[v] += (0.25 * a) * (fp[v] - fm[v]);
    acc[1 + D] += a * (fp[5] - fm[5]);
  }
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
      const Q6 qa = tile_q6(t, o - m * st), qb = tile_q6(t, o + (l - m) * st);
      double f[6];
      pair6<1>(qa, qb, f);
      F[0] += (0.5 * a) * f[0];
#pragma unroll
      for (int v = 1; v < 5; ++v) F[v] += (0.25 * a) * f[v];
      F[2] += a * f[5];
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

// first / second index-space differences from a tile (stride st)
__device__ __forceinline__ void d12_tile(const DevP& P, const double* __restrict__ f, int o, int st, double& d1, double& d2) {
  const double c0 = f[o];
  d1 = 0.0; d2 = 0.0;
#pragma unroll
  for (int l = 1; l <= 3; ++l) {
    const double fp = f[o + l * st], fm = f[o - l * st];
    d1 += P.c.a[l - 1] * (fp - fm);
    d2 += P.c.b[l - 1] * fma(-2.0, c0, fp + fm);
  }
}
__device__ __forceinline__ double d1_tile(const DevP& P, const double* __restrict__ f, int o, int st) {
  double d1 = 0.0;
#pragma unroll
  for (int l = 1; l <= 3; ++l) d1 += P.c.a[l - 1] * (f[o + l * st] - f[o - l * st]);
  return d1;
}
__device__ __forceinline__ void d12_win(const DevP& P, const double (&f)[7], double& d1, double& d2) {
  d1 = 0.0; d2 = 0.0;
#pragma unroll
  for (int l = 1; l <= 3; ++l) {
    d1 += P.c.a[l - 1] * (f[3 + l] - f[3 - l]);
    d2 += P.c.b[l - 1] * fma(-2.0, f[3], f[3 + l] + f[3 - l]);
  }
}

template <bool FUSED>
__global__ void __launch_bounds__(NT, 1) k_rhs(const DevP P, const RhsArgs A) {
  extern __shared__ double sm[];
  double* tS = sm;
  double* tQ = tS + SM_TILES;
  double* sgY = tQ + SM_TILEQ;
  double* sgX = sgY + SM_STGY;
  double* mixw = sgX + SM_STGX;
  double* red = mixw + SM_MIXW;

  const int ti = threadIdx.x, tj = threadIdx.y, tid = tj * TX + ti;
  const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY;
  const int gi = i0 + ti, gj = j0 + tj;
  const int k0 = blockIdx.z * A.lz;
  const int k1 = min(k0 + A.lz, P.nz);
  const bool active = gi < P.nx && gj < P.ny;
  const bool ghost_slot = !active && gi < P.nx + HALO && gj < P.ny + HALO;   // ragged tile: slot holds a ghost
  const int oc = (tj + HALO) * PITCH + ti + HALO;                             // own tile offset

  // halo work list: [0,192) y-halo rows, [192,240) x-halo columns, [240,276) corners
  int hio[2], hjo[2], hoff[2], hkind[2];   // kind 0 none, 1 full primitives, 2 corner (u,v only)
#pragma unroll
  for (int r = 0; r < 2; ++r) {
    const int e = tid + r * NT;
    int io = 0, jo = 0, kind = 0;
    if (e < 192) { const int rr = e / TX; jo = rr < 3 ? rr - 3 : TY + rr - 3; io = e % TX; kind = 1; }
    else if (e < 240) { const int e2 = e - 192; jo = e2 / 6; const int c = e2 % 6; io = c < 3 ? c - 3 : TX + c - 3; kind = 1; }
    else if (e < 276) { const int e3 = e - 240; const int rr = e3 / 6, c = e3 % 6; jo = rr < 3 ? rr - 3 : TY + rr - 3; io = c < 3 ? c - 3 : TX + c - 3; kind = 2; }
    if (kind && (i0 + io >= P.nx + HALO || j0 + jo >= P.ny + HALO)) kind = 0;
    hkind[r] = kind; hio[r] = i0 + io; hjo[r] = j0 + jo;
    hoff[r] = (jo + HALO) * PITCH + io + HALO;
  }

  const double ihx = active ? P.ih[0][gi] : 0.0, ihy = active ? P.ih[1][gj] : 0.0;
  const double ghx = active ? P.gh[0][gi] : 0.0, ghy = active ? P.gh[1][gj] : 0.0;
  const double hxy = active ? P.hh[0][gi] * P.hh[1][gj] : 0.0;

  // register windows (index 3 = plane s)
  double uw[7], vw[7], ww[7], Tw[7], mw[7], rw[4];
  double zc[4][5];
#pragma unroll
  for (int a = 0; a < 7; ++a) { uw[a] = vw[a] = ww[a] = 0.0; Tw[a] = mw[a] = 1.0; }
#pragma unroll
  for (int a = 0; a < 4; ++a) { rw[a] = 1.0;
#pragma unroll
    for (int v = 0; v < 5; ++v) zc[a][v] = 0.0; }
  double fsum = 0.0;
  const double dt = FUSED ? *A.dt_ptr : 0.0;

  for (int s = k0 - 6; s < k1; ++s) {
    const int q = s + 3;                     // look-ahead plane
    const bool full = s >= k0;
    // ---------------- phase A: loads, primitives, tiles --------------------------------------
    Prim pq;
    pq.rho = 1.0; pq.u = pq.v = pq.w = 0.0; pq.T = 1.0; pq.mu = 1.0;
    if (active) fetch_prim<true>(P, A.w, gi, gj, q, pq);
    // shift windows, push plane q
#pragma unroll
    for (int a = 0; a < 6; ++a) { uw[a] = uw[a + 1]; vw[a] = vw[a + 1]; ww[a] = ww[a + 1]; Tw[a] = Tw[a + 1]; mw[a] = mw[a + 1]; }
    uw[6] = pq.u; vw[6] = pq.v; ww[6] = pq.w; Tw[6] = pq.T; mw[6] = pq.mu;
#pragma unroll
    for (int a = 0; a < 3; ++a) rw[a] = rw[a + 1];
    rw[3] = pq.rho;

    __syncthreads();                         // previous plane's readers are done with the tiles
    if (active) {
      tQ[0 * TILE + oc] = pq.u; tQ[1 * TILE + oc] = pq.v; tQ[2 * TILE + oc] = pq.w;
    } else if (ghost_slot) {
      double a, b, c;
      fetch_vel(P, A.w, gi, gj, q, a, b, c);
      tQ[0 * TILE + oc] = a; tQ[1 * TILE + oc] = b; tQ[2 * TILE + oc] = c;
    }
#pragma unroll
    for (int r = 0; r < 2; ++r) {
      if (hkind[r] == 1) {
        double a, b, c;
        fetch_vel(P, A.w, hio[r], hjo[r], q, a, b, c);
        tQ[0 * TILE + hoff[r]] = a; tQ[1 * TILE + hoff[r]] = b; tQ[2 * TILE + hoff[r]] = c;
      }
    }
    if (full) {
      if (active) {
        Prim pc; pc.rho = rw[0]; pc.u = uw[3]; pc.v = vw[3]; pc.w = ww[3]; pc.T = Tw[3]; pc.mu = mw[3];
        double pp, HH;
        derive_pH(P, pc, pp, HH);
        tS[F_RHO * TILE + oc] = pc.rho; tS[F_U * TILE + oc] = pc.u; tS[F_V * TILE + oc] = pc.v; tS[F_W * TILE + oc] = pc.w;
        tS[F_P * TILE + oc] = pp; tS[F_H * TILE + oc] = HH; tS[F_T * TILE + oc] = pc.T; tS[F_MU * TILE + oc] = pc.mu;
      } else if (ghost_slot) {
        Prim pg; double pp, HH;
        fetch_prim<true>(P, A.w, gi, gj, s, pg);
        derive_pH(P, pg, pp, HH);
        tS[F_RHO * TILE + oc] = pg.rho; tS[F_U * TILE + oc] = pg.u; tS[F_V * TILE + oc] = pg.v; tS[F_W * TILE + oc] = pg.w;
        tS[F_P * TILE + oc] = pp; tS[F_H * TILE + oc] = HH; tS[F_T * TILE + oc] = pg.T; tS[F_MU * TILE + oc] = pg.mu;
      }
#pragma unroll
      for (int r = 0; r < 2; ++r) {
        const int kind = hkind[r];
        if (kind == 0) continue;
        const int o = hoff[r];
        Prim pg;
        if (kind == 1) {
          double pp, HH;
          fetch_prim<true>(P, A.w, hio[r], hjo[r], s, pg);
          derive_pH(P, pg, pp, HH);
          tS[F_RHO * TILE + o] = pg.rho; tS[F_U * TILE + o] = pg.u; tS[F_V * TILE + o] = pg.v; tS[F_W * TILE + o] = pg.w;
          tS[F_P * TILE + o] = pp; tS[F_H * TILE + o] = HH; tS[F_T * TILE + o] = pg.T; tS[F_MU * TILE + o] = pg.mu;
        } else {
          fetch_prim<false>(P, A.w, hio[r], hjo[r], s, pg);
          tS[F_U * TILE + o] = pg.u; tS[F_V * TILE + o] = pg.v;
        }
      }
    }
    __syncthreads();
    // ---------------- phase B1: in-plane derivatives of plane q; staging of plane s ----------
    {
      double dxw = 0.0, dyw = 0.0, dv = 0.0;
      if (active) {
        dxw = d1_tile(P, tQ + 2 * TILE, oc, 1);
        dyw = d1_tile(P, tQ + 2 * TILE, oc, PITCH);
        dv = d1_tile(P, tQ + 0 * TILE, oc, 1) * ihx + d1_tile(P, tQ + 1 * TILE, oc, PITCH) * ihy;
      }
      const int slot = ((q % 7) + 7) % 7;
      mixw[(slot * 3 + 0) * NT + tid] = dxw;
      mixw[(slot * 3 + 1) * NT + tid] = dyw;
      mixw[(slot * 3 + 2) * NT + tid] = dv;
    }
    if (full && P.viscous) {
      for (int e = tid; e < TY * PX; e += NT) {        // D_y v at (col, row), x-extended
        const int row = e / PX, col = e % PX;
        sgY[row * PITCH + col] = d1_tile(P, tS + F_V * TILE, (row + HALO) * PITCH + col, PITCH);
      }
      for (int e = tid; e < PY * TX; e += NT) {        // D_x u at (col, row), y-extended
        const int row = e / TX, col = e % TX;
        sgX[row * TX + col] = d1_tile(P, tS + F_U * TILE, row * PITCH + col + HALO, 1);
      }
    }
    __syncthreads();
    if (s < k0 - 3 || !active) continue;

    // ---------------- z-direction convective pairs (s, s+l): each computed once --------------
    {
      Q6 qc[4];
#pragma unroll
      for (int a = 0; a < 4; ++a) {
        Prim t; t.rho = rw[a]; t.u = uw[3 + a]; t.v = vw[3 + a]; t.w = ww[3 + a]; t.T = Tw[3 + a]; t.mu = 0.0;
        double pp, HH;
        derive_pH(P, t, pp, HH);
        qc[a].rho = t.rho; qc[a].u = t.u; qc[a].v = t.v; qc[a].w = t.w; qc[a].H = HH; qc[a].p = pp;
      }
#pragma unroll
      for (int l = 1; l <= 3; ++l) {
        double f[6];
        pair6<2>(qc[0], qc[l], f);
        const double a = P.c.a[l - 1];
        const double c0 = (0.5 * a) * f[0];
        zc[0][0] += c0; zc[l][0] -= c0;
#pragma unroll
        for (int v = 1; v < 5; ++v) { const double cv_ = (0.25 * a) * f[v]; zc[0][v] += cv_; zc[l][v] -= cv_; }
        const double cp_ = a * f[5];
        zc[0][3] += cp_; zc[l][3] -= cp_;
      }
    }
    double az[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) { az[v] = zc[0][v]; zc[0][v] = zc[1][v]; zc[1][v] = zc[2][v]; zc[2][v] = zc[3][v]; zc[3][v] = 0.0; }
    if (!full) continue;

    // ---------------- phase B2: plane s ------------------------------------------------------
    const double ihz = P.ih[2][s], ghz = P.gh[2][s];
    double R[5];
    {
      double ax[5] = {0, 0, 0, 0, 0}, ay[5] = {0, 0, 0, 0, 0};
      conv_inplane<0>(P, tS, oc, 1, ax);
      const bool wall_lo = gj == 0 && P.bc[2] == BC_WALL_STAG;
      const bool wall_hi = gj == P.ny - 1 && P.bc[3] == BC_WALL_STAG;
      if (wall_lo || wall_hi) {
        double Fp[5] = {0, 0, 0, 0, 0}, Fm[5] = {0, 0, 0, 0, 0};
        if (wall_hi) Fp[2] = flux_y_pressure(P, tS, oc, PITCH); else flux_y_full(P, tS, oc, PITCH, Fp);
        if (wall_lo) Fm[2] = flux_y_pressure(P, tS, oc - PITCH, PITCH); else flux_y_full(P, tS, oc - PITCH, PITCH, Fm);
#pragma unroll
        for (int v = 0; v < 5; ++v) ay[v] = Fp[v] - Fm[v];
      } else {
        conv_inplane<1>(P, tS, oc, PITCH, ay);
      }
      if (gi == P.nx - 1 && P.bc[1] == BC_OUTFLOW) {
        // S8: characteristic form of the x-derivative at the outflow node, incoming waves removed
        const size_t o = ((size_t)s * P.ny + gj) * P.nx + gi;
        double dw[5];
#pragma unroll
        for (int v = 0; v < 5; ++v)
          dw[v] = (3.0 * A.w[o + v * P.N] - 4.0 * A.w[o - 1 + v * P.N] + A.w[o - 2 + v * P.N]) * 0.5;   // * ihx below
        const double u = uw[3], v_ = vw[3], w_ = ww[3];
        const double q2 = u * u + v_ * v_ + w_ * w_;
        const double Hc = P.cp * Tw[3] + 0.5 * q2;
        const double c2 = P.gm1 * (Hc - 0.5 * q2), cs = sqrt(c2);
        const double b1 = P.gm1 / c2, b2 = 0.5 * q2 * b1;
        const double mdw = u * dw[1] + v_ * dw[2] + w_ * dw[3];
        double Ls[5];
        Ls[0] = 0.5 * ((b2 + u / cs) * dw[0] - b1 * mdw - dw[1] / cs + b1 * dw[4]);
        Ls[1] = (1.0 - b2) * dw[0] + b1 * mdw - b1 * dw[4];
        Ls[2] = -v_ * dw[0] + dw[2];
        Ls[3] = -w_ * dw[0] + dw[3];
        Ls[4] = 0.5 * ((b2 - u / cs) * dw[0] - b1 * mdw + dw[1] / cs + b1 * dw[4]);
        const double lam[5] = {u - cs, u, u, u, u + cs};
#pragma unroll
        for (int m = 0; m < 5; ++m) Ls[m] = lam[m] >= 0.0 ? lam[m] * Ls[m] : 0.0;
        ax[0] = Ls[0] + Ls[1] + Ls[4];
        ax[1] = (u - cs) * Ls[0] + u * Ls[1] + (u + cs) * Ls[4];
        ax[2] = v_ * Ls[0] + v_ * Ls[1] + Ls[2] + v_ * Ls[4];
        ax[3] = w_ * Ls[0] + w_ * Ls[1] + Ls[3] + w_ * Ls[4];
        ax[4] = (Hc - u * cs) * Ls[0] + 0.5 * q2 * Ls[1] + v_ * Ls[2] + w_ * Ls[3] + (Hc + u * cs) * Ls[4];
      }
#pragma unroll
      for (int v = 0; v < 5; ++v) R[v] = -(ihx * ax[v] + ihy * ay[v] + ihz * az[v]);
    }
    const double uc = uw[3], vc = vw[3], wc = ww[3], muc = mw[3];
    if (P.viscous) {
      double G[3][3], G2[3][3], Tj[3], T2[3], Mj[3];
      double d1, d2;
      // x
      d12_tile(P, tS + F_U * TILE, oc, 1, d1, d2); G[0][0] = d1 * ihx; G2[0][0] = d2 * (ihx * ihx) + d1 * ghx;
      d12_tile(P, tS + F_V * TILE, oc, 1, d1, d2); G[1][0] = d1 * ihx; G2[1][0] = d2 * (ihx * ihx) + d1 * ghx;
      d12_tile(P, tS + F_W * TILE, oc, 1, d1, d2); G[2][0] = d1 * ihx; G2[2][0] = d2 * (ihx * ihx) + d1 * ghx;
      d12_tile(P, tS + F_T * TILE, oc, 1, d1, d2); Tj[0] = d1 * ihx; T2[0] = d2 * (ihx * ihx) + d1 * ghx;
      Mj[0] = d1_tile(P, tS + F_MU * TILE, oc, 1) * ihx;
      // y
      d12_tile(P, tS + F_U * TILE, oc, PITCH, d1, d2); G[0][1] = d1 * ihy; G2[0][1] = d2 * (ihy * ihy) + d1 * ghy;
      d12_tile(P, tS + F_V * TILE, oc, PITCH, d1, d2); G[1][1] = d1 * ihy; G2[1][1] = d2 * (ihy * ihy) + d1 * ghy;
      d12_tile(P, tS + F_W * TILE, oc, PITCH, d1, d2); G[2][1] = d1 * ihy; G2[2][1] = d2 * (ihy * ihy) + d1 * ghy;
      d12_tile(P, tS + F_T * TILE, oc, PITCH, d1, d2); Tj[1] = d1 * ihy; T2[1] = d2 * (ihy * ihy) + d1 * ghy;
      Mj[1] = d1_tile(P, tS + F_MU * TILE, oc, PITCH) * ihy;
      // z
      d12_win(P, uw, d1, d2); G[0][2] = d1 * ihz; G2[0][2] = d2 * (ihz * ihz) + d1 * ghz;
      d12_win(P, vw, d1, d2); G[1][2] = d1 * ihz; G2[1][2] = d2 * (ihz * ihz) + d1 * ghz;
      d12_win(P, ww, d1, d2); G[2][2] = d1 * ihz; G2[2][2] = d2 * (ihz * ihz) + d1 * ghz;
      d12_win(P, Tw, d1, d2); Tj[2] = d1 * ihz; T2[2] = d2 * (ihz * ihz) + d1 * ghz;
      { double dm = 0.0;
#pragma unroll
        for (int l = 1; l <= 3; ++l) dm += P.c.a[l - 1] * (mw[3 + l] - mw[3 - l]);
        Mj[2] = dm * ihz; }
      // mixed terms (A8): d_a (d_k u_k), a != k
      double mxy = 0.0, myx = 0.0, mxz = 0.0, myz = 0.0, mzd = 0.0;
      {
        const int sl0 = ((s % 7) + 7) % 7;
#pragma unroll
        for (int l = 1; l <= 3; ++l) {
          const double a = P.c.a[l - 1];
          mxy += a * (sgY[tj * PITCH + ti + HALO + l] - sgY[tj * PITCH + ti + HALO - l]);
          myx += a * (sgX[(tj + HALO + l) * TX + ti] - sgX[(tj + HALO - l) * TX + ti]);
          int sp = sl0 + l; if (sp >= 7) sp -= 7;
          int sn = sl0 - l; if (sn < 0) sn += 7;
          mxz += a * (mixw[(sp * 3 + 0) * NT + tid] - mixw[(sn * 3 + 0) * NT + tid]);
          myz += a * (mixw[(sp * 3 + 1) * NT + tid] - mixw[(sn * 3 + 1) * NT + tid]);
          mzd += a * (mixw[(sp * 3 + 2) * NT + tid] - mixw[(sn * 3 + 2) * NT + tid]);
        }
        mxy *= ihx * ihy; myx *= ihx * ihy; mxz *= ihx * ihz; myz *= ihy * ihz; mzd *= ihz;
      }
      const double gth[3] = {G2[0][0] + mxy + mxz, myx + G2[1][1] + myz, mzd + G2[2][2]};
      const double Th = G[0][0] + G[1][1] + G[2][2];
      double Vi[3];
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        const double lap = G2[a][0] + G2[a][1] + G2[a][2];
        const double cross = Mj[0] * (G[a][0] + G[0][a]) + Mj[1] * (G[a][1] + G[1][a]) + Mj[2] * (G[a][2] + G[2][a]);
        Vi[a] = muc * (lap + gth[a] * (1.0 / 3.0)) + cross - (2.0 / 3.0) * Mj[a] * Th;
      }
      const double s01 = G[0][1] + G[1][0], s02 = G[0][2] + G[2][0], s12 = G[1][2] + G[2][1];
      const double Phi = muc * (2.0 * (G[0][0] * G[0][0] + G[1][1] * G[1][1] + G[2][2] * G[2][2]) + s01 * s01 + s02 * s02 + s12 * s12 - (2.0 / 3.0) * Th * Th);
      const double heat = P.cp_over_Pr * (muc * (T2[0] + T2[1] + T2[2]) + (Mj[0] * Tj[0] + Mj[1] * Tj[1] + Mj[2] * Tj[2]));
      R[1] += Vi[0]; R[2] += Vi[1]; R[3] += Vi[2];
      R[4] += uc * Vi[0] + vc * Vi[1] + wc * Vi[2] + Phi + heat;
    }
    fsum += R[1] * (hxy * P.hh[2][s]);
    // ---------------- epilogue: write R, or the RK3 stage of Eq. 11 --------------------------
    const size_t o = ((size_t)s * P.ny + gj) * P.nx + gi;
    if (!FUSED) {
#pragma unroll
      for (int v = 0; v < 5; ++v) A.out_rhs[o + v * P.N] = R[v];
    } else {
      double wn[5];
#pragma unroll
      for (int v = 0; v < 5; ++v) {
        const double sp = A.alpha != 0.0 ? A.S_prev[o + v * P.N] : 0.0;
        wn[v] = A.w[o + v * P.N] + dt * (A.alpha * sp + A.beta * R[v]);
        A.S_out[o + v * P.N] = R[v];
      }
      if ((gj == 0 && P.bc[2] == BC_WALL_NODE) || (gj == P.ny - 1 && P.bc[3] == BC_WALL_NODE)) {
        const double Twl = gj == 0 ? P.Twall[0] : P.Twall[1];
        wn[1] = 0.0; wn[2] = 0.0; wn[3] = 0.0; wn[4] = wn[0] * P.cv * Twl;
      }
#pragma unroll
      for (int v = 0; v < 5; ++v) A.w_out[o + v * P.N] = wn[v];
    }
  }
  if (A.partial) {
    const double tot = block_sum<NT>(fsum, red, tid);
    if (tid == 0) A.partial[(blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x] = tot;
  }
}

}  // namespace streams
