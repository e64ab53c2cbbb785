// k_rhs.cuh -- the fused right-hand-side kernel (rows a1,a4,a6,a7,a8,a9 of the scope table).
//
// One CTA owns a TX x TY tile of (x,y) nodes and marches over a chunk of z planes (2.5-D
// blocking).  Every node is worked on by TWO threads of different warps (warp-specialised
// roles), because the on-chip working set per node (z windows, derivative rings, halo tile)
// only allows 256 nodes in flight per SM and one thread per node cannot hide the fp64 latency:
//   role A (warps 0-7)  : x and y directions read from the shared-memory tile of plane s,
//                         the xy mixed derivatives and the assembly of the viscous terms;
//   role B (warps 8-15) : z direction from REGISTER windows (planes s-3..s+3 of its own node),
//                         the asynchronous fill of the tile two planes ahead, the z-mixed terms
//                         of plane s-3 and the epilogue (write R, or the RK3 stage of Eq. 11).
// The state arrives as primitives Q = rho,u,v,w,T,mu,H (dev_common.cuh), so filling a tile is a
// plain asynchronous copy global -> shared (cp.async completing on an mbarrier; no registers,
// nothing transcendental per stencil point); only wall-reflected / constant ghost slots go
// through registers.  Per plane s a CTA holds
//   * tile[s&1]  : the seven primitives of plane s for the tile plus a halo of 3,
//   * sgX / sgY  : D_x u on the y-extended and D_y v on the x-extended tile (xy mixed terms),
//   * xch        : the 14 z-direction sums of plane s handed from role B to role A,
//   * gring      : d_x w, d_y w, d_x u + d_y v of planes s-6..s (thread-private columns),
//   * rring      : the residual of planes s-3..s without their z-mixed terms.
// The z-mixed terms d_z(d_x w), d_z(d_y w), d_z(d_x u + d_y v) of plane s-3 need planes up to
// s, so plane s-3 is completed and written at step s ("delayed output") -- no look-ahead tile.
// Convective terms: Eq. 6-7 in the telescoped pair form
//   F_{i+1/2} - F_{i-1/2} = 2 sum_l a_l [ (rho,u,phi)~_{i,l} - (rho,u,phi)~_{i-l,l} ],
// factored per node as phi_i * sum_l (A_l - B_l) + sum_l (A_l phi_{i+l} - B_l phi_{i-l}) with
// A_l = a_l/4 (rho_i+rho_{i+l})(un_i+un_{i+l}), B_l likewise for i-l: the same sum of the same
// pair products (equal up to rounding order).  The pressure difference is formed as
// a_l R (rho_+ T_+ - rho_- T_-).
// Viscous terms: Laplacian form, Eq. 9 and DESIGN.md S7.
#pragma once
#include "dev_common.cuh"

namespace streams {

constexpr int TX = 32, TY = 8;
constexpr int NPT = TX * TY;                    // nodes per tile = threads per role
constexpr int NT = 2 * NPT;                     // threads per CTA
constexpr int XH = 4;                           // tile columns left of the tile origin (3 used)
constexpr int PITCH = TX + 2 * XH;              // doubles per tile row
constexpr int PY = TY + 2 * HALO;
constexpr int TILE = PY * PITCH;                // doubles per tile field
enum { F_RHO = 0, F_U, F_V, F_W, F_T, F_MU, F_H, NF };   // = order of the fields of Q
static_assert(NF == NQ, "tile fields are the stored primitives");

constexpr int SM_TILE1 = NF * TILE;             // one plane
constexpr int SM_TILES = 2 * SM_TILE1;          // double-buffered
constexpr int SM_STGY = TY * PITCH;             // D_y v on the x-extended rows
constexpr int SM_STGX = PY * TX;                // D_x u on the y-extended columns
constexpr int SM_GRING = 7 * 3 * NPT;
constexpr int SM_RRING = 4 * 5 * NPT;
constexpr int NXCH = 14;
constexpr int SM_XCH = NXCH * NPT;
constexpr int SM_RED = 32;
constexpr int SM_RHS_DOUBLES = SM_TILES + SM_STGY + SM_STGX + SM_GRING + SM_RRING + SM_XCH + SM_RED + 2;
constexpr int NHALO = 2 * HALO * TX + 2 * HALO * TY + 4 * HALO * HALO;   // 276 halo slots per tile
constexpr int NSTAGE = 2 * HALO * TY + 2 * HALO * TX;                     // 240 staged derivatives outside the tile

struct RhsArgs {
  const double* q;        // primitives the residual is evaluated on, [NQ][N]
  double* out_rhs;        // !FUSED: R goes here, [5][N]
  double* q_out;          // FUSED: primitives of w + dt (alpha S_prev + beta R)
  const double* S_prev;   // FUSED: R of the previous stage (ignored when alpha == 0)
  double* S_out;          // FUSED: R of this stage (may alias S_prev)
  const double* dt_ptr;   // FUSED: time step on the device
  double alpha, beta;
  double* partial;        // per-CTA partial sums of R_rhou * vol (forcing), may be NULL
  int lz;                 // planes per CTA
};

// ---- PTX helpers: mbarrier, cp.async, named barriers ----------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
  asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(bar) : "memory");
}
// arrive once all cp.async issued so far by this thread have landed; counts as one expected arrival
__device__ __forceinline__ void cp_async_arrive(unsigned bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  unsigned ok;
  do {
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  } while (!ok);
}
__device__ __forceinline__ void cp_async8(unsigned dst, const double* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void bar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }
enum { BAR_STAGE = 1, BAR_ZSUM = 2, BAR_ADONE = 3 };

struct Nb { double rho, u, v, w, T, mu, H; };
// index-space sums of one direction: convective (Dm, c*), first differences (d*), and
// s* = sum_l b_l (phi_{+l} + phi_{-l}) of the second differences
struct DirAcc { double Dm, cu, cv, cw, cH, cp, du, dv, dw, dT, dmu, su, sv, sw, sT; };

__device__ __forceinline__ void acc_zero(DirAcc& A) {
  A.Dm = A.cu = A.cv = A.cw = A.cH = A.cp = 0.0;
  A.du = A.dv = A.dw = A.dT = A.dmu = 0.0;
  A.su = A.sv = A.sw = A.sT = 0.0;
}

// contribution of the node pairs (i, i+l) and (i-l, i) along direction D  (Eq. 6-7; Eq. 9 differences)
//   qa = a_l / 4, aR = a_l R
template <int D>
__device__ __forceinline__ void dir_accum(const double a, const double b, const double qa, const double aR,
                                          const Nb& c, const Nb& p, const Nb& m, DirAcc& A) {
  const double unc = D == 0 ? c.u : (D == 1 ? c.v : c.w);
  const double unp = D == 0 ? p.u : (D == 1 ? p.v : p.w);
  const double unm = D == 0 ? m.u : (D == 1 ? m.v : m.w);
  const double Ap = qa * ((c.rho + p.rho) * (unc + unp));
  const double Bm = qa * ((m.rho + c.rho) * (unm + unc));
  A.Dm += Ap - Bm;
  A.cu = fma(Ap, p.u, A.cu); A.cu = fma(-Bm, m.u, A.cu);
  A.cv = fma(Ap, p.v, A.cv); A.cv = fma(-Bm, m.v, A.cv);
  A.cw = fma(Ap, p.w, A.cw); A.cw = fma(-Bm, m.w, A.cw);
  A.cH = fma(Ap, p.H, A.cH); A.cH = fma(-Bm, m.H, A.cH);
  A.cp = fma(aR, fma(p.rho, p.T, -(m.rho * m.T)), A.cp);
  A.du = fma(a, p.u - m.u, A.du);
  A.dv = fma(a, p.v - m.v, A.dv);
  A.dw = fma(a, p.w - m.w, A.dw);
  A.dT = fma(a, p.T - m.T, A.dT);
  A.dmu = fma(a, p.mu - m.mu, A.dmu);
  A.su = fma(b, p.u + m.u, A.su);
  A.sv = fma(b, p.v + m.v, A.sv);
  A.sw = fma(b, p.w + m.w, A.sw);
  A.sT = fma(b, p.T + m.T, A.sT);
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
  q.T = t[F_T * TILE + o]; q.mu = t[F_MU * TILE + o]; q.H = t[F_H * TILE + o];
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
      F[2] += (a * P.Rgas) * fma(t[F_RHO * TILE + oa], t[F_T * TILE + oa], t[F_RHO * TILE + ob] * t[F_T * TILE + ob]);
    }
  }
}
__device__ __forceinline__ double flux_y_pressure(const DevP& P, const double* __restrict__ t, int o, int st) {
  double F = 0.0;
#pragma unroll
  for (int l = 1; l <= 3; ++l)
#pragma unroll
    for (int m = 0; m < l; ++m) {
      const int oa = o - m * st, ob = o + (l - m) * st;
      F += (P.c.a[l - 1] * P.Rgas) * fma(t[F_RHO * TILE + oa], t[F_T * TILE + oa], t[F_RHO * TILE + ob] * t[F_T * TILE + ob]);
    }
  return F;
}

__device__ __forceinline__ double d1_tile(const DevP& P, const double* __restrict__ f, int o, int st) {
  double d1 = 0.0;
#pragma unroll
  for (int l = 1; l <= 3; ++l) d1 = fma(P.c.a[l - 1], f[o + l * st] - f[o - l * st], d1);
  return d1;
}

// ---- role B: one tile slot of plane kk, filled asynchronously when its source is a plain copy ----
struct Slot { Src s; int dst; };     // dst = tile offset, s.kind == SRC_NONE: nothing to do

__device__ __forceinline__ void fill_slot(const DevP& P, const double* __restrict__ Q, const Slot& sl, int kk,
                                          double* __restrict__ t, bool all_fields) {
  const int kind = sl.s.kind & 7;
  if (kind == SRC_NONE) return;
  const bool refl = (sl.s.kind >> 4) != 0;
  if (!refl && kind == SRC_FIELD) {
    const double* src = Q + (size_t)kk * P.nxy + sl.s.off;
    const unsigned dst = smem_u32(t + sl.dst);
    if (all_fields) {
#pragma unroll
      for (int f = 0; f < NF; ++f) cp_async8(dst + f * TILE * 8, src + (size_t)f * P.N);
    } else {
#pragma unroll
      for (int f = F_U; f <= F_W; ++f) cp_async8(dst + f * TILE * 8, src + (size_t)f * P.N);
    }
  } else if (!refl && kind == SRC_INFLOW) {
    const size_t st = (size_t)P.nz * P.ny;
    const double* src = P.inflow + (size_t)kk * P.ny + sl.s.off;
    const unsigned dst = smem_u32(t + sl.dst);
#pragma unroll
    for (int f = 0; f < NF; ++f) cp_async8(dst + f * TILE * 8, src + f * st);
  } else {
    Prim q;
    load_src_raw(P, Q, sl.s, kk, q);
    apply_reflect(P, sl.s, q);
    double* d = t + sl.dst;
    d[F_RHO * TILE] = q.rho; d[F_U * TILE] = q.u; d[F_V * TILE] = q.v; d[F_W * TILE] = q.w;
    d[F_T * TILE] = q.T; d[F_MU * TILE] = q.mu; d[F_H * TILE] = q.H;
  }
}

// sums of one direction -> what the assembly needs from it (index space -> physical space, S2):
//   o[0..4] = ih * (F_{+1/2} - F_{-1/2}),  o[5..7] = d_D (u,v,w),  o[8] = d_D T,  o[9] = d_D mu,
//   o[10..12] = d_DD (u,v,w),  o[13] = d_DD T
template <int D>
__device__ __forceinline__ void dir_finish(const DevP& P, const Nb& c, const DirAcc& S, const double f[5], double ih, double gh, double o[NXCH]) {
#pragma unroll
  for (int v = 0; v < 5; ++v) o[v] = ih * f[v];
  const double i2 = ih * ih, m2 = -P.c.sb2;
  o[5] = S.du * ih; o[6] = S.dv * ih; o[7] = S.dw * ih; o[8] = S.dT * ih; o[9] = S.dmu * ih;
  o[10] = fma(S.du, gh, fma(m2, c.u, S.su) * i2);
  o[11] = fma(S.dv, gh, fma(m2, c.v, S.sv) * i2);
  o[12] = fma(S.dw, gh, fma(m2, c.w, S.sw) * i2);
  o[13] = fma(S.dT, gh, fma(m2, c.T, S.sT) * i2);
}

template <bool FUSED>
__global__ void __launch_bounds__(NT, 1) k_rhs(const DevP P, const RhsArgs A) {
  extern __shared__ __align__(16) double sm[];
  double* tiles = sm;
  double* sgY = tiles + SM_TILES;
  double* sgX = sgY + SM_STGY;
  double* gring = sgX + SM_STGX;
  double* rring = gring + SM_GRING;
  double* xch = rring + SM_RRING;
  double* red = xch + SM_XCH;
  const unsigned bar_full = smem_u32(red + SM_RED);          // two mbarriers: tile[b] of the current plane has landed

  const int tid = threadIdx.x;
  const bool roleB = tid >= NPT;
  const int pt = tid & (NPT - 1), ti = pt & (TX - 1), tj = pt / TX;
  const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY;
  const int gi = i0 + ti, gj = j0 + tj;
  const int k0 = blockIdx.z * A.lz;
  const int k1 = min(k0 + A.lz, P.nz);
  const bool active = gi < P.nx && gj < P.ny;
  const int oc = (tj + HALO) * PITCH + ti + XH;                               // own tile offset
  const int own_off = gj * P.nx + gi;

  if (tid == 0) {
    mbar_init(bar_full, NT);            // per plane every role-B thread arrives twice: cp.async completion + plain stores
    mbar_init(bar_full + 8, NT);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  const double ihx = active ? P.ih[0][gi] : 0.0, ihy = active ? P.ih[1][gj] : 0.0;
#define a1 P.c.a[0]
#define a2 P.c.a[1]
#define a3 P.c.a[2]
  double fsum = 0.0;

  if (!roleB) {
    // ============================ role A: x, y, xy-mixed, assembly ==============================
    // staged derivative outside the tile: [0,48) D_y v on the x-halo columns, [48,240) D_x u on the y-halo rows
    int sj_src = 0, sj_dst = -1, sj_st = 1, sj_f = F_U;
    if (pt < 2 * HALO * TY) {
      const int r = pt / 6, c = pt % 6, io = c < 3 ? c - 3 : TX + c - 3;
      sj_src = (r + HALO) * PITCH + io + XH; sj_dst = r * PITCH + io + XH; sj_st = PITCH; sj_f = F_V;
    } else if (pt < NSTAGE) {
      const int e2 = pt - 2 * HALO * TY, rr = e2 / TX, col = e2 % TX, jo = rr < 3 ? rr - 3 : TY + rr - 3;
      sj_src = (jo + HALO) * PITCH + col + XH; sj_dst = SM_STGY + (jo + HALO) * TX + col; sj_st = 1; sj_f = F_U;
    }
    const double ghx = active ? P.gh[0][gi] : 0.0, ghy = active ? P.gh[1][gj] : 0.0;
    int slot7 = 0;                                     // it % 7

    for (int s = k0 - 3, it = 0; s < k1 + 3; ++s, ++it) {
      const bool full = s >= k0 && s < k1;
      const double* t = tiles + (it & 1) * SM_TILE1;
      mbar_wait(bar_full + 8 * (it & 1), (it >> 1) & 1);
      // ---------------- in-plane derivatives shared through the staging rows ---------------------
      const double dxu = d1_tile(P, t + F_U * TILE, oc, 1);
      const double dyv = d1_tile(P, t + F_V * TILE, oc, PITCH);
      sgX[(tj + HALO) * TX + ti] = dxu;
      sgY[tj * PITCH + ti + XH] = dyv;
      if (sj_dst >= 0) sgY[sj_dst] = d1_tile(P, t + sj_f * TILE, sj_src, sj_st);    // sgX follows sgY in memory
      bar_sync(BAR_STAGE, NPT);

      double g1 = 0.0, g2 = 0.0, g3 = 0.0;
      double R[5], ox[NXCH], oy[NXCH], mxy = 0.0, myx = 0.0;
      Nb c;
      if (active && !full) {
        g1 = d1_tile(P, t + F_W * TILE, oc, 1) * ihx;
        g2 = d1_tile(P, t + F_W * TILE, oc, PITCH) * ihy;
        g3 = dxu * ihx + dyv * ihy;
      }
      if (active && full) {
        c = tile_nb(t, oc);
        // ---- x ----
        {
          DirAcc X;
          acc_zero(X);
#pragma unroll
          for (int l = 1; l <= 3; ++l) {
            const Nb p = tile_nb(t, oc + l), m = tile_nb(t, oc - l);
            dir_accum<0>(P.c.a[l - 1], P.c.b[l - 1], P.c.qa[l - 1], P.c.aR[l - 1], c, p, m, X);
          }
          double f[5];
          conv_from_acc<0>(c, X, f);
          if (gi == P.nx - 1 && P.bc[1] == BC_OUTFLOW) {
            // S8: characteristic form of the x-derivative at the outflow node, incoming waves removed
            const Nb n1 = tile_nb(t, oc - 1), n2 = tile_nb(t, oc - 2);
            const double pc = c.rho * (P.Rgas * c.T), p1 = n1.rho * (P.Rgas * n1.T), p2 = n2.rho * (P.Rgas * n2.T);
            const double w0[5] = {c.rho, c.rho * c.u, c.rho * c.v, c.rho * c.w, c.rho * c.H - pc};
            const double w1[5] = {n1.rho, n1.rho * n1.u, n1.rho * n1.v, n1.rho * n1.w, n1.rho * n1.H - p1};
            const double w2[5] = {n2.rho, n2.rho * n2.u, n2.rho * n2.v, n2.rho * n2.w, n2.rho * n2.H - p2};
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
          dir_finish<0>(P, c, X, f, ihx, ghx, ox);
        }
        // ---- y ----
        {
          DirAcc Y;
          acc_zero(Y);
#pragma unroll
          for (int l = 1; l <= 3; ++l) {
            const Nb p = tile_nb(t, oc + l * PITCH), m = tile_nb(t, oc - l * PITCH);
            dir_accum<1>(P.c.a[l - 1], P.c.b[l - 1], P.c.qa[l - 1], P.c.aR[l - 1], c, p, m, Y);
          }
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
          dir_finish<1>(P, c, Y, f, ihy, ghy, oy);
        }
        if (P.viscous) {
          // xy mixed terms (A8): d_x(d_y v) and d_y(d_x u) from the staging rows
          const int sy = tj * PITCH + ti + XH, sx = (tj + HALO) * TX + ti;
          mxy = a1 * (sgY[sy + 1] - sgY[sy - 1]);
          mxy = fma(a2, sgY[sy + 2] - sgY[sy - 2], mxy);
          mxy = fma(a3, sgY[sy + 3] - sgY[sy - 3], mxy);
          myx = a1 * (sgX[sx + TX] - sgX[sx - TX]);
          myx = fma(a2, sgX[sx + 2 * TX] - sgX[sx - 2 * TX], myx);
          myx = fma(a3, sgX[sx + 3 * TX] - sgX[sx - 3 * TX], myx);
        }
      }
      bar_sync(BAR_ZSUM, NT);          // the z sums of plane s are in xch; all tile / staging reads of plane s are done
      if (active) {
        if (full) {
          double oz[NXCH];
#pragma unroll
          for (int v = 0; v < NXCH; ++v) oz[v] = xch[v * NPT + pt];
#pragma unroll
          for (int v = 0; v < 5; ++v) R[v] = -(ox[v] + oy[v] + oz[v]);
          g1 = ox[7]; g2 = oy[7]; g3 = ox[5] + oy[6];
          if (P.viscous) {
            // G[a][d] = d_d u_a: ox[5+a], oy[5+a], oz[5+a];  Tj = o[8], Mj = o[9]
            const double ixy = ihx * ihy;
            double gth[3];
            gth[0] = fma(mxy, ixy, ox[10]);
            gth[1] = fma(myx, ixy, oy[11]);
            gth[2] = oz[12];
            const double lap[3] = {ox[10] + oy[10] + oz[10], ox[11] + oy[11] + oz[11], ox[12] + oy[12] + oz[12]};
            const double T2 = ox[13] + oy[13] + oz[13];
            const double Th = ox[5] + oy[6] + oz[7];
            const double Mj[3] = {ox[9], oy[9], oz[9]};
            const double s01 = oy[5] + ox[6], s02 = oz[5] + ox[7], s12 = oz[6] + oy[7];
            double Vi[3];
            Vi[0] = c.mu * fma(gth[0], 1.0 / 3.0, lap[0]) + (Mj[0] * (2.0 * ox[5]) + Mj[1] * s01 + Mj[2] * s02) - (2.0 / 3.0) * Mj[0] * Th;
            Vi[1] = c.mu * fma(gth[1], 1.0 / 3.0, lap[1]) + (Mj[0] * s01 + Mj[1] * (2.0 * oy[6]) + Mj[2] * s12) - (2.0 / 3.0) * Mj[1] * Th;
            Vi[2] = c.mu * fma(gth[2], 1.0 / 3.0, lap[2]) + (Mj[0] * s02 + Mj[1] * s12 + Mj[2] * (2.0 * oz[7])) - (2.0 / 3.0) * Mj[2] * Th;
            const double Phi = c.mu * (2.0 * (ox[5] * ox[5] + oy[6] * oy[6] + oz[7] * oz[7]) + s01 * s01 + s02 * s02 + s12 * s12 - (2.0 / 3.0) * Th * Th);
            const double heat = P.cp_over_Pr * (c.mu * T2 + (Mj[0] * ox[8] + Mj[1] * oy[8] + Mj[2] * oz[8]));
            R[1] += Vi[0]; R[2] += Vi[1]; R[3] += Vi[2];
            R[4] += c.u * Vi[0] + c.v * Vi[1] + c.w * Vi[2] + Phi + heat;
          }
          double* rr = rring + (it & 3) * 5 * NPT + pt;
#pragma unroll
          for (int v = 0; v < 5; ++v) rr[v * NPT] = R[v];
        }
        double* gr = gring + slot7 * 3 * NPT + pt;
        gr[0] = g1; gr[NPT] = g2; gr[2 * NPT] = g3;
      }
      slot7 = slot7 == 6 ? 0 : slot7 + 1;
      __threadfence_block();
      bar_arrive(BAR_ADONE, NT);
    }
  } else {
    // ============================ role B: z, tile fill, delayed output ============================
    // Tile slots this thread fills: slot 0 = its own position (also when that lies outside the grid but
    // inside the ghost range: ragged tiles); slots 1,2 = halo list entries pt and pt + NPT:
    // [0,192) y-halo rows, [192,240) x-halo columns, [240,276) corners.
    Slot sl[3];
    sl[0].s.kind = SRC_NONE; sl[0].s.off = 0; sl[0].dst = oc;
    if (gi < P.nx + HALO && gj < P.ny + HALO) sl[0].s = resolve_xy(P, gi, gj);
#pragma unroll
    for (int r = 0; r < 2; ++r) {
      const int e = pt + r * NPT;
      int io = 0, jo = 0;
      bool any = true;
      if (e < 192) { const int rr = e / TX; jo = rr < 3 ? rr - 3 : TY + rr - 3; io = e % TX; }
      else if (e < 240) { const int e2 = e - 192; jo = e2 / 6; const int c = e2 % 6; io = c < 3 ? c - 3 : TX + c - 3; }
      else if (e < NHALO) { const int e3 = e - 240; const int rr = e3 / 6, c = e3 % 6; jo = rr < 3 ? rr - 3 : TY + rr - 3; io = c < 3 ? c - 3 : TX + c - 3; }
      else any = false;
      if (any && (i0 + io >= P.nx + HALO || j0 + jo >= P.ny + HALO)) any = false;
      sl[r + 1].s.kind = SRC_NONE; sl[r + 1].s.off = 0;
      if (any) sl[r + 1].s = resolve_xy(P, i0 + io, j0 + jo);
      sl[r + 1].dst = (jo + HALO) * PITCH + io + XH;
    }
    const int nplanes = k1 + 3 - (k0 - 3);
    // tiles of the first two planes
#pragma unroll
    for (int b = 0; b < 2; ++b) {
      if (b < nplanes) {
        const int sp = k0 - 3 + b;
        const bool fl = sp >= k0 && sp < k1;
        double* t = tiles + b * SM_TILE1;
#pragma unroll
        for (int r = 0; r < 3; ++r) fill_slot(P, A.q, sl[r], map_z(P, sp), t, fl);
        cp_async_arrive(bar_full + 8 * b);
        mbar_arrive(bar_full + 8 * b);
      }
    }
    const double hxy = active ? P.hh[0][gi] * P.hh[1][gj] : 0.0;
    const double* qown = A.q + own_off;
    // register windows: index a holds plane s-3+a
    double rw[7], uw[7], vw[7], ww[7], Tw[7], mw[7];
#pragma unroll
    for (int a = 0; a < 7; ++a) { rw[a] = 1.0; uw[a] = vw[a] = ww[a] = 0.0; Tw[a] = mw[a] = 1.0; }
    if (active) {
#pragma unroll
      for (int a = 3; a < 7; ++a) {          // planes k0-3 .. k0 sit in slots 3..6 at s = k0-3
        const double* q = qown + (size_t)map_z(P, k0 - 6 + a) * P.nxy;
        rw[a] = __ldg(q); uw[a] = __ldg(q + P.N); vw[a] = __ldg(q + 2 * P.N); ww[a] = __ldg(q + 3 * P.N);
        Tw[a] = __ldg(q + 4 * P.N); mw[a] = __ldg(q + 5 * P.N);
      }
    }
    const double dt = FUSED ? *A.dt_ptr : 0.0;
    int slot7 = 0;                                     // it % 7

    for (int s = k0 - 3, it = 0; s < k1 + 3; ++s, ++it) {
      const bool full = s >= k0 && s < k1;
      if (active && full) {
        // ---- z sums of plane s from the register windows ----
        const double ihz = P.ih[2][s], ghz = P.gh[2][s];
        Nb c;
        c.rho = rw[3]; c.u = uw[3]; c.v = vw[3]; c.w = ww[3]; c.T = Tw[3]; c.mu = mw[3];
        c.H = fma(P.cp, c.T, 0.5 * fma(c.u, c.u, fma(c.v, c.v, c.w * c.w)));
        DirAcc Z;
        acc_zero(Z);
#pragma unroll
        for (int l = 1; l <= 3; ++l) {
          Nb p, m;
          p.rho = rw[3 + l]; p.u = uw[3 + l]; p.v = vw[3 + l]; p.w = ww[3 + l]; p.T = Tw[3 + l]; p.mu = mw[3 + l];
          m.rho = rw[3 - l]; m.u = uw[3 - l]; m.v = vw[3 - l]; m.w = ww[3 - l]; m.T = Tw[3 - l]; m.mu = mw[3 - l];
          p.H = fma(P.cp, p.T, 0.5 * fma(p.u, p.u, fma(p.v, p.v, p.w * p.w)));
          m.H = fma(P.cp, m.T, 0.5 * fma(m.u, m.u, fma(m.v, m.v, m.w * m.w)));
          dir_accum<2>(P.c.a[l - 1], P.c.b[l - 1], P.c.qa[l - 1], P.c.aR[l - 1], c, p, m, Z);
        }
        double f[5], oz[NXCH];
        conv_from_acc<2>(c, Z, f);
        dir_finish<2>(P, c, Z, f, ihz, ghz, oz);
#pragma unroll
        for (int v = 0; v < NXCH; ++v) xch[v * NPT + pt] = oz[v];
      }
      __threadfence_block();
      bar_arrive(BAR_ZSUM, NT);
      bar_sync(BAR_ADONE, NT);         // role A has written R and g of plane s and is done with tile[it & 1]
      // ---------------- tile of plane s+2 into the buffer plane s just left ------------------------
      if (it + 2 < nplanes) {
        const int sp = s + 2;
        const bool fl = sp >= k0 && sp < k1;
        double* t = tiles + (it & 1) * SM_TILE1;
        const int kk = map_z(P, sp);
#pragma unroll
        for (int r = 0; r < 3; ++r) fill_slot(P, A.q, sl[r], kk, t, fl);
        cp_async_arrive(bar_full + 8 * (it & 1));
        mbar_arrive(bar_full + 8 * (it & 1));
      }
      // ================= plane p = s-3: add the z-mixed terms, write the result ====================
      const int p = s - 3;
      if (active && p >= k0) {
        double R[5];
        {
          const double* rr = rring + ((it - 3) & 3) * 5 * NPT + pt;
#pragma unroll
          for (int v = 0; v < 5; ++v) R[v] = rr[v * NPT];
        }
        if (P.viscous) {
          // ring slot of plane p+l is (slot7 - 3 + l) mod 7
          double dz[3] = {0.0, 0.0, 0.0};
#pragma unroll
          for (int l = 1; l <= 3; ++l) {
            int sp = slot7 - 3 + l; if (sp < 0) sp += 7;
            int sn = slot7 - 3 - l; if (sn < 0) sn += 7;
            const double* gp = gring + sp * 3 * NPT + pt;
            const double* gn = gring + sn * 3 * NPT + pt;
            const double a = P.c.a[l - 1];
#pragma unroll
            for (int m = 0; m < 3; ++m) dz[m] = fma(a, gp[m * NPT] - gn[m * NPT], dz[m]);
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
          Prim qn; qn.rho = rw[0]; qn.u = uw[0]; qn.v = vw[0]; qn.w = ww[0]; qn.T = Tw[0]; qn.mu = mw[0]; qn.H = 0.0;
          advance_prim(P, qn, dW);
          if (gj == 0 && P.bc[2] == BC_WALL_NODE) wall_node_override(P, P.Twall[0], P.mu_wall[0], qn);
          if (gj == P.ny - 1 && P.bc[3] == BC_WALL_NODE) wall_node_override(P, P.Twall[1], P.mu_wall[1], qn);
          A.q_out[o] = qn.rho; A.q_out[o + P.N] = qn.u; A.q_out[o + 2 * P.N] = qn.v; A.q_out[o + 3 * P.N] = qn.w;
          A.q_out[o + 4 * P.N] = qn.T; A.q_out[o + 5 * P.N] = qn.mu; A.q_out[o + 6 * P.N] = qn.H;
        }
      }
      slot7 = slot7 == 6 ? 0 : slot7 + 1;
      // ---------------- shift the windows, own node of plane s+4 ------------------------------------
#pragma unroll
      for (int a = 0; a < 6; ++a) { rw[a] = rw[a + 1]; uw[a] = uw[a + 1]; vw[a] = vw[a + 1]; ww[a] = ww[a + 1]; Tw[a] = Tw[a + 1]; mw[a] = mw[a + 1]; }
      if (active && s + 4 < k1 + 3) {
        const double* q = qown + (size_t)map_z(P, s + 4) * P.nxy;
        rw[6] = __ldg(q); uw[6] = __ldg(q + P.N); vw[6] = __ldg(q + 2 * P.N); ww[6] = __ldg(q + 3 * P.N);
        Tw[6] = __ldg(q + 4 * P.N); mw[6] = __ldg(q + 5 * P.N);
      }
    }
  }
#undef a1
#undef a2
#undef a3
  if (A.partial) {
    const double tot = block_sum<NT>(fsum, red, tid);
    if (tid == 0) A.partial[(blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x] = tot;
  }
}

}  // namespace streams
