// k_rhs.cuh -- the fused right-hand-side kernel (rows a1,a3 (flags),a4,a6,a7,a8,a9 of the scope table).
//
// One CTA owns a TX x TY tile of (x,y) nodes and marches over a chunk of z planes (2.5-D
// blocking), one thread per node, ~250 registers, one CTA per SM:
//   * the tile of plane s (seven stored primitives, halo 3, x padded to 4) is brought in by ONE
//     TMA box copy per plane (cp.async.bulk.tensor, 4-D box x,y,z,field) into one of two buffers,
//     completion on an mbarrier -- no thread issues a load for the tile; plane s+2 is requested
//     into the buffer of plane s once every thread is past its in-plane reads.  TMA zero-fills
//     outside the grid, and only tiles that touch a domain face patch their ghost slots (periodic
//     wrap, wall reflection, inflow, shock generator) by index (S1), one plane ahead, from a list
//     built once per CTA;
//   * x and y directions read the tile; the z direction reads REGISTER windows (planes s-3..s+2
//     of the thread's own node) and the own-node ring in shared memory (planes s+3..s+5, filled
//     by thread-private cp.async): z costs no tile and no exposed global load;
//   * the xy mixed derivatives go through two small staging arrays (D_x u on the y-extended,
//     D_y v on the x-extended tile); the ONE CTA-wide barrier per plane is split: arrive after the
//     staging rows are written, wait after the z direction;
//   * the z-mixed terms d_z(d_x w), d_z(d_y w), d_z(d_x u + d_y v) of plane s-3 need planes up
//     to s, so plane s-3 is completed and written at step s ("delayed output"); the pending
//     residuals and in-plane derivatives sit in thread-private shared-memory columns;
//   * the epilogue writes R (MODE 0) or applies Eq. 11 and writes the primitives of the new
//     state (MODE 1; MODE 2 = lazy forcing, see RhsArgs::f_prev), R_prev prefetched by cp.async;
//   * with the hybrid switch on, the node flags of Eq. 8 are a by-product of the velocity gradients.
// Convective terms: Eq. 6-7 in the telescoped pair form
//   F_{i+1/2} - F_{i-1/2} = 2 sum_l a_l [ (rho,u,phi)~_{i,l} - (rho,u,phi)~_{i-l,l} ],
// factored per node as phi_i * sum_l (A_l - B_l) + sum_l (A_l phi_{i+l} - B_l phi_{i-l}) with
// A_l = a_l/4 (rho_i+rho_{i+l})(un_i+un_{i+l}), B_l likewise for i-l: the same sum of the same
// pair products (equal up to rounding order).  The pressure difference is formed as
// a_l R (rho_+ T_+ - rho_- T_-).
// Viscous terms: Laplacian form, Eq. 9 and DESIGN.md S7; every direction folds its
// second differences into three running sums as soon as it is done, so that only the nine
// velocity gradients, grad mu and five residual sums stay live across directions.
#pragma once
#include <cuda.h>
#include "dev_common.cuh"

namespace streams {

constexpr int TX = 32, TY = 8;
constexpr int NPT = TX * TY;                    // nodes per tile = threads per CTA
constexpr int NT = NPT;
constexpr int XH = 4;                           // tile columns left/right of the tile (3 used; 4 keeps TMA rows 16-byte multiples)
constexpr int PITCH = TX + 2 * XH;              // doubles per tile row (40)
constexpr int PY = TY + 2 * HALO;               // tile rows (14)
constexpr int TILE = PY * PITCH;                // doubles per tile field (560)
enum { F_RHO = 0, F_U, F_V, F_W, F_T, F_MU, F_H, NF };   // = order of the fields of Q
static_assert(NF == NQ, "tile fields are the stored primitives");

constexpr int NBUF = 2;                         // tile buffers: plane s is used while s+1 lands; s+2 is requested into the
                                                // buffer of plane s once every thread is past its in-plane reads (step barrier)
constexpr int SM_TILE1 = NF * TILE;             // one plane (3920 doubles = 31360 B, a multiple of 128 B)
constexpr int SM_TILES = NBUF * SM_TILE1;
constexpr int SM_STGY = TY * PITCH;             // D_y v on the x-extended rows
constexpr int SM_STGX = PY * TX;                // D_x u on the y-extended columns
constexpr int SM_STG1 = SM_STGY + SM_STGX;      // one staging set; two sets alternate between planes
constexpr int SM_GRING = 7 * 3 * NPT;
constexpr int SM_RRING = 3 * 5 * NPT;     // R of planes s-1..s-3: read (plane s-3) before written (plane s) in a step
constexpr int NOWN = 3;                         // own-node ring: plane s+3 is read while s+4, s+5 are in flight
constexpr int SM_OWN = NOWN * NF * NPT;
constexpr int SM_SPREV = 2 * 6 * NPT;            // FUSED: R_prev (5) and u_prev of planes s-3 / s-2, prefetched by cp.async one step ahead
constexpr int SM_PCOPY = (sizeof(DevP) + 7) / 8;   // copy of the parameter block for the out-of-line helpers
constexpr int SM_RED = 32;
constexpr int LZ_MAX = 128;                     // planes per CTA (make_layout caps the chunk length)
constexpr int SM_MET = 3 * LZ_MAX + 2 * TX + 2 * TY;   // 1/h_z, -g_z/h_z^3, h_z of the chunk; 1/h, -g/h^3 of the tile's x and y
constexpr int SM_PATCH = TILE;                  // ghost-slot list of an edge tile: one int2 (8 bytes) per entry
constexpr int SM_RHS_DOUBLES = SM_TILES + 2 * SM_STG1 + SM_GRING + SM_RRING + SM_OWN + SM_SPREV + SM_MET + SM_PATCH + SM_PCOPY + SM_RED + 16;
static_assert(SM_RHS_DOUBLES * 8 <= 227 * 1024, "one CTA per SM: the shared-memory budget of sm_100a");
constexpr int NSTAGE = 2 * HALO * TY + 2 * HALO * TX;                     // 240 staged derivatives outside the tile
constexpr unsigned TILE_BYTES = SM_TILE1 * sizeof(double);
static_assert(TILE_BYTES % 128 == 0, "TMA destination buffers stay 128-byte aligned");

struct RhsArgs {
  const double* q;        // primitives the residual is evaluated on, [NQ][N]
  double* out_rhs;        // !FUSED: R goes here, [5][N]
  double* q_out;          // FUSED: primitives of w + dt (alpha S_prev + beta R)
  const double* S_prev;   // FUSED: R of the previous stage (ignored when alpha == 0)
  double* S_out;          // FUSED: R of this stage (may alias S_prev)
  const double* dt_ptr;   // FUSED: time step on the device
  const double* f_prev;   // FUSED, lazy forcing (S9): body force of the previous stage, or NULL.  S_prev then holds the
                          // previous R WITHOUT its forcing terms; they are added here as f_prev (e_rhou + u_prev e_rhoE),
                          // u_prev = the velocity still sitting in q_out (the previous stage's input state)
  double alpha, beta;
  int write_S;            // FUSED: 0 in the last stage (alpha of the next stage is 0: R is never read)
  unsigned int* fbits;    // hybrid switch on: node flags theta > theta_th of Eq. 8 (a3), a by-product of the velocity
                          // gradients, one BIT per node: word [k * ny + j][i / 32] = the ballot of a tile row (= one warp);
                          // NULL when the WENO switch is off
  double* partial;        // per-CTA partial sums of R_rhou * vol (forcing), may be NULL
  int lz;                 // planes per CTA
  int cz0, czs;           // chunk of CTA z-index c is cz0 + c * czs (whole grid: 0, 1; streams_stage_rhs launches the chunks
                          // that need no ghost plane of a BC_HALO face and the two boundary chunks separately)
  int use_tma;            // 1: tile and own-node ring by TMA box copies (tensor maps over q); 0: by index (odd nx)
};

// ---- PTX helpers: mbarrier, TMA ----------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  unsigned ok;
  do {
    // potentially blocking: the warp sleeps in hardware up to the time hint (ns) instead of spinning on issue slots
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity), "r"(4000u) : "memory");
  } while (!ok);
}
// one 4-D box (x, y, z, field) into shared memory; completes its bytes on the mbarrier
__device__ __forceinline__ void tma_box(unsigned dst, const CUtensorMap* tm, int x, int y, int z, int f, unsigned bar) {
  asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
               ::"r"(dst), "l"(tm), "r"(x), "r"(y), "r"(z), "r"(f), "r"(bar) : "memory");
}
// the tile of a plane (halo 3, all stored primitives); completes `TILE_BYTES`
__device__ __forceinline__ void tma_tile(unsigned dst, const CUtensorMap* tm, int x, int y, int z, unsigned bar) { tma_box(dst, tm, x, y, z, 0, bar); }

// Tensor maps of one launch (all 4-D: x, y, z, field):
//   tile  the state the residual is evaluated on, box (PITCH, PY, 1, NQ): a plane's tile with its halo
//   own   the same state, box (TX, TY, 1, NQ): the tile's own nodes of a later plane (z window, no halo)
struct RhsMaps { CUtensorMap tile, own; };
constexpr unsigned OWN_BYTES = NQ * NPT * sizeof(double);
// thread-private asynchronous 8-byte copies (own node of a later plane into the own-node ring)
__device__ __forceinline__ void cp_async8(unsigned dst, const double* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N_>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N_) : "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

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

// ---- S1 by index: the ghost slots of an edge tile (all = false) or every slot (all = true, no TMA) ----
// The list is built once per CTA; entry = (tile slot | kind << 16, in-plane source offset).
__device__ __noinline__ void build_patch_list(const DevP& P, int i0, int j0, bool all, int2* __restrict__ list, int* __restrict__ count, int tid) {
  for (int e = tid; e < TILE; e += NT) {
    const int r = e / PITCH, io = e - r * PITCH - XH, jo = r - HALO;
    if (io < -HALO || io >= TX + HALO) continue;
    const int gi = i0 + io, gj = j0 + jo;
    if (gi >= P.nx + HALO || gj >= P.ny + HALO) continue;
    if (!all && gi >= 0 && gi < P.nx && gj >= 0 && gj < P.ny) continue;      // TMA brings it
    Src s = resolve_xy(P, gi, gj);
    if (!all && (s.kind & 7) == SRC_FIELD) {
      // a source node that lies inside this tile's own box (the mirror rows of a wall) is read from the tile in shared
      // memory, not from global memory: kind bit 3, off = tile slot of the source
      const int jj = s.off / P.nx, ii = s.off - jj * P.nx;
      const int lo = ii - i0, ljs = jj - j0;
      if (lo >= -XH && lo < TX + XH && ljs >= -HALO && ljs < TY + HALO) { s.kind |= SRC_LOCAL; s.off = (ljs + HALO) * PITCH + lo + XH; }
    }
    const int n = atomicAdd(count, 1);
    list[n] = make_int2(e | (s.kind << 16), s.off);
  }
}
// fill the listed slots of tile `t` for (already mapped) plane kk
__device__ __noinline__ void patch_tile(const DevP& P, const double* __restrict__ Q, const int2* __restrict__ list, int n, int kk,
                                        double* __restrict__ t, int tid) {
  for (int e = tid; e < n; e += NT) {
    const int2 en = list[e];
    Src s; s.kind = en.x >> 16; s.off = en.y;
    Prim q;
    if (s.kind & SRC_LOCAL) {
      const double* r = t + s.off;
      q.rho = r[F_RHO * TILE]; q.u = r[F_U * TILE]; q.v = r[F_V * TILE]; q.w = r[F_W * TILE];
      q.T = r[F_T * TILE]; q.mu = r[F_MU * TILE]; q.H = r[F_H * TILE];
    } else {
      load_src_raw(P, Q, s, kk, q);
    }
    apply_reflect(P, s, q);
    double* d = t + (en.x & 0xffff);
    d[F_RHO * TILE] = q.rho; d[F_U * TILE] = q.u; d[F_V * TILE] = q.v; d[F_W * TILE] = q.w;
    d[F_T * TILE] = q.T; d[F_MU * TILE] = q.mu; d[F_H * TILE] = q.H;
  }
}

// what stays live across the three directions of one node (S7):
//   R[5]  residual sums, G[3*a+d] = d_d u_a, M[d] = d_d mu,
//   Va[a] = sum_j d_jj u_a + (1/3) d_aa u_a (+ (1/3) mixed terms), LT = sum_j d_jj T, heat = sum_j d_j mu d_j T
struct NodeAcc { double R[5], G[9], M[3], Va[3], LT, heat; };

// sums of direction D -> physical space (S2) and into the node accumulators
template <int D>
__device__ __forceinline__ void dir_fold(const DevP& P, const Nb& c, const DirAcc& S, const double f[5], double ih, double gh, NodeAcc& N) {
#pragma unroll
  for (int v = 0; v < 5; ++v) N.R[v] = fma(-ih, f[v], N.R[v]);
  const double i2 = ih * ih, m2 = -P.c.sb2;
  const double gT = S.dT * ih, gm = S.dmu * ih;
  N.G[0 + D] = S.du * ih; N.G[3 + D] = S.dv * ih; N.G[6 + D] = S.dw * ih;
  N.M[D] = gm;
  const double d2u = fma(S.du, gh, fma(m2, c.u, S.su) * i2);
  const double d2v = fma(S.dv, gh, fma(m2, c.v, S.sv) * i2);
  const double d2w = fma(S.dw, gh, fma(m2, c.w, S.sw) * i2);
  const double d2T = fma(S.dT, gh, fma(m2, c.T, S.sT) * i2);
  N.Va[0] = fma(D == 0 ? 4.0 / 3.0 : 1.0, d2u, N.Va[0]);
  N.Va[1] = fma(D == 1 ? 4.0 / 3.0 : 1.0, d2v, N.Va[1]);
  N.Va[2] = fma(D == 2 ? 4.0 / 3.0 : 1.0, d2w, N.Va[2]);
  N.LT += d2T;
  N.heat = fma(gm, gT, N.heat);
}

// viscous stresses, dissipation and heat conduction from the node accumulators (Eq. 2-3, 9; S7) into R
__device__ __forceinline__ void visc_assemble(const DevP& P, const Nb& c, NodeAcc& N) {
  const double* G = N.G;
  const double Th = G[0] + G[4] + G[8];
  const double s01 = G[1] + G[3], s02 = G[2] + G[6], s12 = G[5] + G[7];
  const double t23 = (2.0 / 3.0) * Th;
  const double V0 = fma(c.mu, N.Va[0], fma(N.M[0], 2.0 * G[0] - t23, fma(N.M[1], s01, N.M[2] * s02)));
  const double V1 = fma(c.mu, N.Va[1], fma(N.M[1], 2.0 * G[4] - t23, fma(N.M[0], s01, N.M[2] * s12)));
  const double V2 = fma(c.mu, N.Va[2], fma(N.M[2], 2.0 * G[8] - t23, fma(N.M[0], s02, N.M[1] * s12)));
  const double Phi = c.mu * (2.0 * fma(G[0], G[0], fma(G[4], G[4], G[8] * G[8])) + fma(s01, s01, fma(s02, s02, s12 * s12)) - t23 * Th);
  const double heat = P.cp_over_Pr * fma(c.mu, N.LT, N.heat);
  N.R[1] += V0; N.R[2] += V1; N.R[3] += V2;
  N.R[4] += fma(c.u, V0, fma(c.v, V1, c.w * V2)) + Phi + heat;
}

// S8: characteristic form of the derivative along D at a boundary node, incoming waves removed.
// Replaces the index-space flux difference f of direction D.  side = +1: max-index face (one-sided difference
// backwards, waves with lambda >= 0 leave), side = -1: min-index face (forwards, lambda <= 0 leave).  wall = true:
// characteristic wall (reading A14b): the incoming acoustic wave is the reflection of the outgoing one, L_5 = L_1.
// Rare path (one column / row): kept out of line.
struct F5 { double v[5]; };   // returned by value: stays in registers across the call (no local-memory frame)
template <int D>
__device__ __noinline__ F5 char_face(const DevP& P, const double* __restrict__ t, int oc, int st, int side, bool wall) {
  F5 r;
  double* f = r.v;
  const Nb c = tile_nb(t, oc), n1 = tile_nb(t, oc - side * st), n2 = tile_nb(t, oc - 2 * side * st);
  const double pc = c.rho * (P.Rgas * c.T), p1 = n1.rho * (P.Rgas * n1.T), p2 = n2.rho * (P.Rgas * n2.T);
  const double w0[5] = {c.rho, c.rho * c.u, c.rho * c.v, c.rho * c.w, c.rho * c.H - pc};
  const double w1[5] = {n1.rho, n1.rho * n1.u, n1.rho * n1.v, n1.rho * n1.w, n1.rho * n1.H - p1};
  const double w2[5] = {n2.rho, n2.rho * n2.u, n2.rho * n2.v, n2.rho * n2.w, n2.rho * n2.H - p2};
  double dw[5];
  const double sg = (double)side;
#pragma unroll
  for (int v = 0; v < 5; ++v) dw[v] = sg * (3.0 * w0[v] - 4.0 * w1[v] + w2[v]) * 0.5;   // * ih by the caller
  constexpr int T1 = (D + 1) % 3, T2 = (D + 2) % 3;
  const double vel[3] = {c.u, c.v, c.w};
  const double un = vel[D];
  const double q2 = c.u * c.u + c.v * c.v + c.w * c.w;
  const double Hc = P.cp * c.T + 0.5 * q2;
  const double c2 = P.gm1 * (Hc - 0.5 * q2), cs = sqrt(c2);
  const double bb1 = P.gm1 / c2, bb2 = 0.5 * q2 * bb1;
  const double mdw = c.u * dw[1] + c.v * dw[2] + c.w * dw[3];
  double Ls[5];
  Ls[0] = 0.5 * ((bb2 + un / cs) * dw[0] - bb1 * mdw - dw[1 + D] / cs + bb1 * dw[4]);
  Ls[1] = (1.0 - bb2) * dw[0] + bb1 * mdw - bb1 * dw[4];
  Ls[2] = -vel[T1] * dw[0] + dw[1 + T1];
  Ls[3] = -vel[T2] * dw[0] + dw[1 + T2];
  Ls[4] = 0.5 * ((bb2 - un / cs) * dw[0] - bb1 * mdw + dw[1 + D] / cs + bb1 * dw[4]);
  const double lam[5] = {un - cs, un, un, un, un + cs};
#pragma unroll
  for (int m = 0; m < 5; ++m) Ls[m] = (side > 0 ? lam[m] >= 0.0 : lam[m] <= 0.0) ? lam[m] * Ls[m] : 0.0;
  if (wall) Ls[4] = Ls[0];
  const double sm = Ls[0] + Ls[1] + Ls[4];
  f[0] = sm;
  f[1] = c.u * sm; f[2] = c.v * sm; f[3] = c.w * sm;
  f[1 + D] += cs * (Ls[4] - Ls[0]);
  f[1 + T1] += Ls[2];
  f[1 + T2] += Ls[3];
  f[4] = (Hc - un * cs) * Ls[0] + 0.5 * q2 * Ls[1] + vel[T1] * Ls[2] + vel[T2] * Ls[3] + (Hc + un * cs) * Ls[4];
  return r;
}

// flux difference of the y direction next to a staggered wall: the wall-plane flux keeps the pressure only
__device__ __noinline__ F5 wall_y(const DevP& P, const double* __restrict__ t, int oc, bool wall_lo, bool wall_hi) {
  F5 r;
  double Fp[5] = {0, 0, 0, 0, 0}, Fm[5] = {0, 0, 0, 0, 0};
  if (wall_hi) Fp[2] = flux_y_pressure(P, t, oc, PITCH); else flux_y_full(P, t, oc, PITCH, Fp);
  if (wall_lo) Fm[2] = flux_y_pressure(P, t, oc - PITCH, PITCH); else flux_y_full(P, t, oc - PITCH, PITCH, Fm);
#pragma unroll
  for (int v = 0; v < 5; ++v) r.v[v] = Fp[v] - Fm[v];
  return r;
}


// The whole kernel body.  PLAIN = true is the instantiation for tiles that lie fully inside the grid and hold no
// special node (no staggered-wall row, no Dirichlet wall row, no characteristic outflow column), with TMA and the
// viscous terms on: every such test folds at compile time and no out-of-line call remains in the plane loop, which
// frees ~30 registers for the scheduler.  Ghost slots (periodic wrap, reflection, ...) are handled in both.
// MODE: 0 = residual only (streams_rhs), 1 = fused RK stage, 2 = fused RK stage with lazy forcing (mu(T) left to k_force_fix)
template <int MODE, bool PLAIN, bool WENO, int STAGE>
__device__ __forceinline__ void rhs_body(const DevP& P, const RhsArgs& A, const RhsMaps& M, double* sm, const int3 cta) {
  const CUtensorMap& tmap = M.tile;
  constexpr bool FUSED = MODE != 0, LAZY = MODE == 2;
  // STAGE (fused launches): 0 = first RK stage (alpha = 0: no R_prev), 1 = middle, 2 = last (R is not stored: never read)
  constexpr bool HAS_PREV = FUSED && STAGE > 0, WRITE_S = STAGE < 2, HAS_FPREV = LAZY && STAGE > 0;
  double* tiles = sm;
  double* stg = tiles + SM_TILES;
  double* gring = stg + 2 * SM_STG1;
  double* rring = gring + SM_GRING;
  double* oring = rring + SM_RRING;
  double* spring = oring + SM_OWN;
  double* met = spring + SM_SPREV;
  int2* plist = reinterpret_cast<int2*>(met + SM_MET);
  // The out-of-line helpers (ghost list, ghost patch, wall and outflow closures) take the parameters by reference.  A
  // reference to the kernel parameter itself makes every field a generic load from the parameter bank, which misses the
  // small L1 left beside 208 KB of shared memory (measured: ~2500 cycles per plane on edge tiles); they get this copy.
  DevP* sP = reinterpret_cast<DevP*>(met + SM_MET + SM_PATCH);
  double* red = met + SM_MET + SM_PATCH + SM_PCOPY;
  const unsigned bar0 = smem_u32(red + SM_RED);          // NBUF mbarriers: tile buffer b holds its plane
  const unsigned sbar = bar0 + 8 * NBUF;                 // the per-plane CTA barrier, split into arrive / wait
  int* pcount = reinterpret_cast<int*>(red + SM_RED + NBUF + 1);
  const unsigned obar = bar0 + 8 * 8;                    // NOWN mbarriers: own-node ring slot holds its plane (TMA path)
  const double* zi = met;                                // 1/h_z, -g_z/h_z^3, h_z of planes k0 .. k1-1
  const double* zg = met + LZ_MAX;
  const double* zh = met + 2 * LZ_MAX;
  const double* xi = met + 3 * LZ_MAX;                   // 1/h_x, -g_x/h_x^3 of the tile's columns
  const double* xg = xi + TX;
  const double* yi = xg + TX;                            // 1/h_y, -g_y/h_y^3 of the tile's rows
  const double* yg = yi + TY;

  const int tid = threadIdx.x;
  const int ti = tid & (TX - 1), tj = tid / TX;
  const int i0 = cta.x * TX, j0 = cta.y * TY;
  const int gi = i0 + ti, gj = j0 + tj;
  const int k0 = cta.z * A.lz;
  const int k1 = min(k0 + A.lz, P.nz);
  const bool active = PLAIN || (gi < P.nx && gj < P.ny);
  const int own_off = gj * P.nx + gi;
  const bool use_tma = PLAIN || A.use_tma != 0;
  // with TMA the own-node ring is filled by box copies too (one request per plane by one thread instead of seven
  // thread-private copies with their address arithmetic): config 5 -1.4 %, config 4 -0.7 % per launch, the L2-resident
  // configs 2, 3 +1 ... 1.5 %; choosing between the two at run time costs more than either (both bodies in the loop)
  const bool own_tma = use_tma;
  // tiles that see a domain face fill their ghost slots by index (S1); without TMA every tile fills every slot
  const bool edge = !use_tma || i0 < HALO || i0 + TX + HALO > P.nx || j0 < HALO || j0 + TY + HALO > P.ny;
  const int nplanes = k1 + 3 - (k0 - 3);

  if (tid == 0) {
    *pcount = 0;
    mbar_init(sbar, NT / 32);
    if (use_tma) {
#pragma unroll
      for (int b = 0; b < NBUF; ++b) mbar_init(bar0 + 8 * b, 1);
#pragma unroll
      for (int b = 0; b < NOWN; ++b) mbar_init(obar + 8 * b, 1);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    fence_proxy_async();
    if (use_tma) {
#pragma unroll
      for (int b = 0; b < 2; ++b)
        if (b < nplanes) {
          mbar_expect_tx(bar0 + 8 * b, TILE_BYTES);
          tma_tile(smem_u32(tiles + b * SM_TILE1), &tmap, i0 - XH, j0 - HALO, map_z(P, k0 - 3 + b) + P.zpad, bar0 + 8 * b);
        }
      // own nodes of planes k0, k0+1, k0+2 (ring slots 0, 1, 2): plane q sits in slot (q - k0) % 3; later planes are
      // requested by the same thread at the end of the step that read the slot's previous plane
#pragma unroll
      for (int b = 0; b < NOWN; ++b)
        if (own_tma && k0 + b < k1 + 3) {
          mbar_expect_tx(obar + 8 * b, OWN_BYTES);
          tma_box(smem_u32(oring + b * NF * NPT), &M.own, i0, j0, map_z(P, k0 + b) + P.zpad, 0, obar + 8 * b);
        }
    }
  }
  for (int e = tid; e < (int)(sizeof(DevP) / sizeof(int)); e += NT) reinterpret_cast<int*>(sP)[e] = reinterpret_cast<const int*>(&P)[e];
  for (int e = tid; e < k1 - k0; e += NT) {
    met[e] = P.ih[2][k0 + e]; met[LZ_MAX + e] = P.gh[2][k0 + e]; met[2 * LZ_MAX + e] = P.hh[2][k0 + e];
  }
  if (tid < TX) {
    const bool ok = i0 + tid < P.nx;
    met[3 * LZ_MAX + tid] = ok ? P.ih[0][i0 + tid] : 0.0;
    met[3 * LZ_MAX + TX + tid] = ok ? P.gh[0][i0 + tid] : 0.0;
  } else if (tid < TX + TY) {
    const int r = tid - TX;
    const bool ok = j0 + r < P.ny;
    met[3 * LZ_MAX + 2 * TX + r] = ok ? P.ih[1][j0 + r] : 0.0;
    met[3 * LZ_MAX + 2 * TX + TY + r] = ok ? P.gh[1][j0 + r] : 0.0;
  }
  __syncthreads();
  int npatch = 0;
  if (edge) {
    build_patch_list(*sP, i0, j0, !use_tma, plist, pcount, tid);
    __syncthreads();
    npatch = *pcount;
    if (use_tma) mbar_wait(bar0, 0);
    patch_tile(*sP, A.q, plist, npatch, map_z(P, k0 - 3), tiles, tid);     // first plane; later planes one step ahead
    __syncthreads();
  }

  double fsum = 0.0;

  // register windows of the own node: index a holds plane s-3+a
  // (plane s+3 stays in the own-node ring: read for the l = 3 pair and again when it enters the window)
  double rw[6], uw[6], vw[6], ww[6], Tw[6], mw[6], Hw[6];
#pragma unroll
  for (int a = 0; a < 6; ++a) { rw[a] = 1.0; uw[a] = vw[a] = ww[a] = 0.0; Tw[a] = mw[a] = 1.0; Hw[a] = 0.0; }
  if (active) {
#pragma unroll
    for (int a = 3; a < 6; ++a) {          // planes k0-3 .. k0-1 sit in slots 3..5 at s = k0-3
      const double* q = A.q + own_off + (long long)map_z(P, k0 - 6 + a) * P.nxy;
      rw[a] = __ldg(q); uw[a] = __ldg(q + P.QS); vw[a] = __ldg(q + 2 * P.QS); ww[a] = __ldg(q + 3 * P.QS);
      Tw[a] = __ldg(q + 4 * P.QS); mw[a] = __ldg(q + 5 * P.QS); Hw[a] = __ldg(q + 6 * P.QS);
    }
  }
  // own node of the planes ahead: plane s+5 is requested at the top of step s (cp.async, thread-private
  // slot, no register and no barrier) into ring slot (it+5) % 3; plane s+3 is read from slot it % 3
  // (with TMA the ring is filled by box copies of the tile's own nodes instead: one request per plane, no per-thread
  // address arithmetic, completion on the slot's mbarrier)
  if (!own_tma) {
#pragma unroll
    for (int b = 0; b < 2; ++b) {
      if (active) {
        const double* q = A.q + own_off + (long long)map_z(P, k0 + b) * P.nxy;
#pragma unroll
        for (int f = 0; f < NF; ++f) cp_async8(smem_u32(oring + tid) + ((b * NF + f) * NPT) * 8, q + f * P.QS);
      }
      cp_async_commit();
    }
  }
  // dt and the previous stage's body force sit in shared memory (read once per plane in the epilogue)
  double* scal = red + SM_RED + NBUF + 2;
  if (FUSED && tid == 0) {
    scal[0] = *A.dt_ptr;
    scal[1] = HAS_FPREV ? *A.f_prev : 0.0;
  }
  __syncthreads();
  int slot7 = 0, b3 = 0;                                 // it % 7, it % 3
  unsigned own_par = 0;                                  // (it / 3) & 1: phase of the own-node ring slot read in this step

  for (int s = k0 - 3, it = 0; s < k1 + 3; ++s, ++it) {
    const bool full = s >= k0 && s < k1;
    const int buf = it & 1;                              // tile buffer of plane s; its mbarrier is in phase (it >> 1) & 1
    const unsigned phase = (unsigned)(it >> 1) & 1u;
    double* t = tiles + buf * SM_TILE1;
    // Addresses: a warp-uniform pointer (plane, field) plus the node's 32-bit offset inside a plane (two instructions per
    // address; a 64-bit per-thread element index costs four, and the loop forms 24 addresses per plane)
    const unsigned own32 = (unsigned)own_off;
    if (!own_tma && active && s + 5 < k1 + 3) {
      // own node of plane s+5 by thread-private copies (with TMA: a box copy per plane, requested at the end of a step)
      const double* q = (A.q + (long long)map_z(P, s + 5) * P.nxy) + own32;
      const unsigned d = smem_u32(oring + tid) + ((b3 == 0 ? 2 : b3 - 1) * NF * NPT) * 8;       // (it + 5) % 3
#pragma unroll
      for (int f = 0; f < NF; ++f) cp_async8(d + f * NPT * 8, q + f * P.QS);
    }
    if (HAS_PREV && active && s - 2 >= k0 && s - 2 < k1) {
      // R_prev (and u_prev for the lazy forcing) of plane s-2, read in the NEXT step's epilogue (one step of slack:
      // the epilogue sits before the plane barrier and must not wait for HBM).  Thread-private slots: a thread's own
      // program order keeps the copy behind its reads of the slot, which happen between barrier arrive and wait.
      const long long zo = (long long)(s - 2) * P.nxy;
      const double* sp = (A.S_prev + zo) + own32;
      const unsigned d = smem_u32(spring + tid) + (((it + 1) & 1) * 6 * NPT) * 8;
#pragma unroll
      for (int v = 0; v < 5; ++v) cp_async8(d + v * NPT * 8, sp + v * P.N);
      if (HAS_FPREV) cp_async8(d + 5 * NPT * 8, (A.q_out + zo + P.QS) + own32);
    }
    cp_async_commit();
    cp_async_wait<1>();                                  // the groups of steps <= s-1 have landed: R_prev of plane s-3 (and
                                                         // without TMA the own node of planes s+3, s+4)
    int tl = tid;                                        // opaque copy: keeps per-thread shared-memory addresses from being
    asm volatile("" : "+r"(tl));                         // hoisted out of the loop (and then spilled) instead of recomputed
    const int li = tl & (TX - 1), lj = tl / TX, loc = (lj + HALO) * PITCH + li + XH;
    const double* own3 = oring + b3 * NF * NPT + tl;     // own node of plane s+3
    // ---- z, from the register windows (no shared tile, no barrier): the upper half of the warps does it FIRST, the
    // lower half after arriving at the barrier, so that the two warps of a scheduler are in different phases
    // (fp64-dense z against the shared-memory-heavy x, y)
    NodeAcc N;
    Nb o3;                                               // own node of plane s+3: read ONCE (l = 3 pair, then the window)
    auto zdir = [&]() {
      Nb c;
      c.rho = rw[3]; c.u = uw[3]; c.v = vw[3]; c.w = ww[3]; c.T = Tw[3]; c.mu = mw[3]; c.H = Hw[3];
      DirAcc Z;
      acc_zero(Z);
#pragma unroll
      for (int l = 1; l <= 3; ++l) {
        Nb p, m;
        if (l < 3) {
          p.rho = rw[3 + l]; p.u = uw[3 + l]; p.v = vw[3 + l]; p.w = ww[3 + l]; p.T = Tw[3 + l]; p.mu = mw[3 + l]; p.H = Hw[3 + l];
        } else {
          p = o3;
        }
        m.rho = rw[3 - l]; m.u = uw[3 - l]; m.v = vw[3 - l]; m.w = ww[3 - l]; m.T = Tw[3 - l]; m.mu = mw[3 - l]; m.H = Hw[3 - l];
        dir_accum<2>(P.c.a[l - 1], P.c.b[l - 1], P.c.qa[l - 1], P.c.aR[l - 1], c, p, m, Z);
      }
      double f[5];
      conv_from_acc<2>(c, Z, f);
      dir_fold<2>(P, c, Z, f, zi[s - k0], zg[s - k0], N);
    };
    if (active && full) {
#pragma unroll
      for (int v = 0; v < 5; ++v) N.R[v] = 0.0;
      N.Va[0] = N.Va[1] = N.Va[2] = 0.0; N.LT = 0.0; N.heat = 0.0;
    }
    if (use_tma) mbar_wait(bar0 + 8 * buf, phase);
    double* sgY = stg + (it & 1) * SM_STG1;
    double* sgX = sgY + SM_STGY;
    // staged derivative outside the tile: threads [0,48) D_y v on the x-halo columns, [48,240) D_x u on the y-halo rows
    // (indices recomputed every plane: cheaper than three registers carried through the loop)
    if (tl < 2 * HALO * TY) {
      const int r = tl / 6, c = tl % 6, io = c < 3 ? c - 3 : TX + c - 3;
      sgY[r * PITCH + io + XH] = d1_tile(P, t + F_V * TILE, (r + HALO) * PITCH + io + XH, PITCH);
    } else if (tl < NSTAGE) {
      const int e2 = tl - 2 * HALO * TY, rr = e2 / TX, col = e2 % TX, jo = rr < 3 ? rr - 3 : TY + rr - 3;
      sgX[(jo + HALO) * TX + col] = d1_tile(P, t + F_U * TILE, (jo + HALO) * PITCH + col + XH, 1);
    }

    if (!active || !full) {
      // ghost planes of the chunk, and tile nodes beyond the grid (their staging entries are the
      // neighbours' ghost columns / rows): in-plane first derivatives only
      const double dxu = d1_tile(P, t + F_U * TILE, loc, 1);
      const double dyv = d1_tile(P, t + F_V * TILE, loc, PITCH);
      sgX[(lj + HALO) * TX + li] = dxu;
      sgY[lj * PITCH + li + XH] = dyv;
      if (active) {
        const double ihx = xi[li], ihy = yi[lj];
        double* gr = gring + slot7 * 3 * NPT + tl;
        gr[0] = d1_tile(P, t + F_W * TILE, loc, 1) * ihx;
        gr[NPT] = d1_tile(P, t + F_W * TILE, loc, PITCH) * ihy;
        gr[2 * NPT] = __dadd_rn(__dmul_rn(dxu, ihx), __dmul_rn(dyv, ihy));   // = G[0] + G[4] of a full plane, bit for bit
      }
    } else {
      const double ihx = xi[li], ihy = yi[lj];
      {
        Nb c;
        c.rho = rw[3]; c.u = uw[3]; c.v = vw[3]; c.w = ww[3]; c.T = Tw[3]; c.mu = mw[3]; c.H = Hw[3];
        // ---- x ----
        {
          DirAcc X;
          acc_zero(X);
#pragma unroll
          for (int l = 1; l <= 3; ++l) {
            const Nb p = tile_nb(t, loc + l), m = tile_nb(t, loc - l);
            dir_accum<0>(P.c.a[l - 1], P.c.b[l - 1], P.c.qa[l - 1], P.c.aR[l - 1], c, p, m, X);
          }
          sgX[(lj + HALO) * TX + li] = X.du;                                 // D_x u, for d_y(d_x u) of the neighbours
          double f[5];
          conv_from_acc<0>(c, X, f);
          if (!PLAIN && gi == P.nx - 1 && P.bc[1] == BC_OUTFLOW) {
            const F5 r = char_face<0>(*sP, t, loc, 1, 1, false);
#pragma unroll
            for (int v = 0; v < 5; ++v) f[v] = r.v[v];
          }
          dir_fold<0>(P, c, X, f, ihx, xg[li], N);
        }
        // ---- y ----
        {
          DirAcc Y;
          acc_zero(Y);
#pragma unroll
          for (int l = 1; l <= 3; ++l) {
            const Nb p = tile_nb(t, loc + l * PITCH), m = tile_nb(t, loc - l * PITCH);
            dir_accum<1>(P.c.a[l - 1], P.c.b[l - 1], P.c.qa[l - 1], P.c.aR[l - 1], c, p, m, Y);
          }
          sgY[lj * PITCH + li + XH] = Y.dv;                                  // D_y v, for d_x(d_y v) of the neighbours
          double f[5];
          conv_from_acc<1>(c, Y, f);
          const bool wall_lo = gj == 0 && P.bc[2] == BC_WALL_STAG;
          const bool wall_hi = gj == P.ny - 1 && P.bc[3] == BC_WALL_STAG;
          if (!PLAIN && (wall_lo || wall_hi)) {
            const F5 r = wall_y(*sP, t, loc, wall_lo, wall_hi);
#pragma unroll
            for (int v = 0; v < 5; ++v) f[v] = r.v[v];
          }
          const bool nr_top = gj == P.ny - 1 && P.bc[3] == BC_OUTFLOW, ch_wall = gj == 0 && P.bc[2] == BC_WALL_CHAR;
          if (!PLAIN && (nr_top || ch_wall)) {
            const F5 r = char_face<1>(*sP, t, loc, PITCH, nr_top ? 1 : -1, ch_wall);
#pragma unroll
            for (int v = 0; v < 5; ++v) f[v] = r.v[v];
          }
          dir_fold<1>(P, c, Y, f, ihy, yg[lj], N);
        }
      }
      double* gr = gring + slot7 * 3 * NPT + tl;
      // no FMA contraction here: a plane next to a chunk is a ghost plane of that chunk (branch above) and must give
      // the same bits, so that the result does not depend on how z is cut into chunks or slabs
      gr[0] = N.G[6]; gr[NPT] = N.G[7]; gr[2 * NPT] = __dadd_rn(N.G[0], N.G[4]);
    }
    if (edge && it + 1 < nplanes) {
      // ghost slots of the NEXT plane's tile: written before this step's barrier, read after it.  Done here, after the
      // in-plane work, because that tile was requested at the end of the previous step: waiting for it at the top of the
      // step exposed the whole TMA latency on the patching warps, and through the barrier on everybody
      const int b1 = buf ^ 1;
      if (use_tma && tl < npatch) mbar_wait(bar0 + 8 * b1, (unsigned)((it + 1) >> 1) & 1u);
      patch_tile(*sP, A.q, plist, npatch, map_z(P, s + 1), tiles + b1 * SM_TILE1, tl);
    }
    // own node of plane s+3: read BEFORE the arrive, so that every thread is done with the ring slot when the barrier
    // completes and the slot can take the box copy of plane s+6 (requested three steps before it is read)
    if (own_tma && s + 3 < k1 + 3) mbar_wait(obar + 8 * b3, own_par);
    o3.rho = own3[F_RHO * NPT]; o3.u = own3[F_U * NPT]; o3.v = own3[F_V * NPT]; o3.w = own3[F_W * NPT];
    o3.T = own3[F_T * NPT]; o3.mu = own3[F_MU * NPT]; o3.H = own3[F_H * NPT];
    // ---- the plane's barrier, first half: everything other threads read of this step is written ----
    __syncwarp();
    if ((tl & 31) == 0) mbar_arrive(sbar);

    // ================= between arrive and wait: everything that needs no other thread's data of this plane.  The z
    // direction, the viscous assembly of plane s without its xy mixed terms, and the completion + epilogue of plane
    // p = s-3 (z-mixed terms from the thread-private rings, Eq. 11, global stores) -- more than half of the step's
    // work, so that the wait below finds the barrier complete (measured: the wait was 6 % of all warp cycles when it
    // sat directly after the z direction).
    const int p = s - 3;
    const bool do_fin = active && p >= k0, do_asm = active && full;
    bool flagged = false;
    if (do_asm) {
      zdir();
      if (WENO) {
        // S4 / Eq. 8: same expression, same order as k_sensor (the flags must agree bit for bit)
        const double* G = N.G;
        const double div = G[0] + G[4] + G[8];
        const double ox = G[7] - G[5], oy = G[2] - G[6], oz = G[3] - G[1];
        const double th = fmax(-div / sqrt(div * div + (ox * ox + oy * oy + oz * oz) + P.th_eps), 0.0);
        flagged = th > P.th_thr;
      }
      if (PLAIN || P.viscous) {
        Nb c;
        c.rho = rw[3]; c.u = uw[3]; c.v = vw[3]; c.w = ww[3]; c.T = Tw[3]; c.mu = mw[3]; c.H = Hw[3];
        visc_assemble(P, c, N);                          // N.R is final up to the xy mixed terms (added after the wait)
      }
    }
    if (WENO && full) {
      // a tile row is one warp and starts at a multiple of 32: its ballot IS the flag word (0 for nodes beyond the grid)
      const unsigned bits = __ballot_sync(0xffffffffu, flagged);
      if ((tl & 31) == 0 && gj < P.ny) A.fbits[((long long)s * P.ny + gj) * ((P.nx + 31) >> 5) + (i0 >> 5)] = bits;
    }
    if (do_fin) {
      double R[5];
      {
        const double* rr = rring + b3 * 5 * NPT + tl;               // plane s-3 sits in slot it % 3
#pragma unroll
        for (int v = 0; v < 5; ++v) R[v] = rr[v * NPT];
      }
      if (PLAIN || P.viscous) {
        // ring slot of plane p+l is (slot7 - 3 + l) mod 7
        double dz[3] = {0.0, 0.0, 0.0};
#pragma unroll
        for (int l = 1; l <= 3; ++l) {
          int sp = slot7 - 3 + l; if (sp < 0) sp += 7;
          int sn = slot7 - 3 - l; if (sn < 0) sn += 7;
          const double* gp = gring + sp * 3 * NPT + tl;
          const double* gn = gring + sn * 3 * NPT + tl;
          const double a = P.c.a[l - 1];
#pragma unroll
          for (int m = 0; m < 3; ++m) dz[m] = fma(a, gp[m * NPT] - gn[m * NPT], dz[m]);
        }
        const double f3 = mw[0] * (1.0 / 3.0) * zi[p - k0];
        const double v0 = f3 * dz[0], v1 = f3 * dz[1], v2 = f3 * dz[2];
        R[1] += v0; R[2] += v1; R[3] += v2;
        R[4] += uw[0] * v0 + vw[0] * v1 + ww[0] * v2;
      }
      fsum = fma(R[1], zh[p - k0], fsum);                                      // times h_x h_y after the loop
      // ---------------- epilogue: write R, or the RK3 stage of Eq. 11 ------------------------------
      const long long zo = (long long)p * P.nxy;
      if (!FUSED) {
        double* ro = (A.out_rhs + zo) + own32;
#pragma unroll
        for (int v = 0; v < 5; ++v) ro[v * P.N] = R[v];
      } else {
        double dW[5];
        const double dt = scal[0], fprev = scal[1];
        const double* pv = spring + (it & 1) * 6 * NPT + tl;        // requested at the top of step s-1
#pragma unroll
        for (int v = 0; v < 5; ++v) {
          double sp = HAS_PREV ? pv[v * NPT] : 0.0;
          if (v == 1) sp += fprev;
          if (v == 4 && HAS_FPREV) sp = fma(fprev, pv[5 * NPT], sp);
          dW[v] = HAS_PREV ? dt * (A.alpha * sp + A.beta * R[v]) : dt * (A.beta * R[v]);
        }
        if (WRITE_S) {
          double* so = (A.S_out + zo) + own32;
#pragma unroll
          for (int v = 0; v < 5; ++v) so[v * P.N] = R[v];
        }
        Prim qn; qn.rho = rw[0]; qn.u = uw[0]; qn.v = vw[0]; qn.w = ww[0]; qn.T = Tw[0]; qn.mu = mw[0]; qn.H = 0.0;
        bool store_mu = !LAZY;
        advance_prim<!LAZY>(P, qn, dW);
        if (!PLAIN && gj == 0 && node_wall(P.bc[2])) { wall_node_override(P, P.Twall[0], P.mu_wall[0], qn); store_mu = true; }
        if (!PLAIN && gj == P.ny - 1 && node_wall(P.bc[3])) { wall_node_override(P, P.Twall[1], P.mu_wall[1], qn); store_mu = true; }
        double* qo = (A.q_out + zo) + own32;
        qo[0] = qn.rho; qo[P.QS] = qn.u; qo[2 * P.QS] = qn.v; qo[3 * P.QS] = qn.w;
        qo[4 * P.QS] = qn.T; qo[6 * P.QS] = qn.H;
        if (store_mu) qo[5 * P.QS] = qn.mu;
      }
    }
    // ---------------- shift the windows (own node of plane s+3 enters) BEFORE the wait: 70 register moves that need no
    // other thread, done while the barrier completes.  After the shift the plane's own node sits in slot 2.
#pragma unroll
    for (int a = 0; a < 5; ++a) {
      rw[a] = rw[a + 1]; uw[a] = uw[a + 1]; vw[a] = vw[a + 1]; ww[a] = ww[a + 1]; Tw[a] = Tw[a + 1]; mw[a] = mw[a + 1]; Hw[a] = Hw[a + 1];
    }
    if (active && s + 3 < k1 + 3) {
      rw[5] = o3.rho; uw[5] = o3.u; vw[5] = o3.v; ww[5] = o3.w; Tw[5] = o3.T; mw[5] = o3.mu; Hw[5] = o3.H;
    }
    // ---- second half of the barrier: the staging rows of this plane are complete ----
    mbar_wait(sbar, (unsigned)(it & 1));
    // every thread is past its reads of this plane's tile: the buffer takes plane s+2
    if (use_tma && tl == 0 && it + 2 < nplanes) {
      const int b2 = buf;                                // (it + 2) % NBUF
      fence_proxy_async();
      mbar_expect_tx(bar0 + 8 * b2, TILE_BYTES);
      tma_tile(smem_u32(tiles + b2 * SM_TILE1), &tmap, i0 - XH, j0 - HALO, map_z(P, s + 2) + P.zpad, bar0 + 8 * b2);
    }
    // ... and the ring slot read in this step (plane s+3; every thread read it before arriving) takes plane s+6
    if (own_tma && tl == 0 && s + 6 < k1 + 3) {
      fence_proxy_async();
      mbar_expect_tx(obar + 8 * b3, OWN_BYTES);
      tma_box(smem_u32(oring + b3 * NF * NPT), &M.own, i0, j0, map_z(P, s + 6) + P.zpad, 0, obar + 8 * b3);
    }
    // ================= after the barrier: the xy mixed terms of plane s (A8), d_x(d_y v) and d_y(d_x u) from the
    // staging rows; they enter V_0, V_1 times mu / 3 and the viscous work u V_0 + v V_1.  R of plane s goes to the
    // residual ring (its slot was read above: plane s-3).
    if (do_asm) {
      if (PLAIN || P.viscous) {
        const int sy = lj * PITCH + li + XH, sx = (lj + HALO) * TX + li;
        double mxy = P.c.a[0] * (sgY[sy + 1] - sgY[sy - 1]);
        mxy = fma(P.c.a[1], sgY[sy + 2] - sgY[sy - 2], mxy);
        mxy = fma(P.c.a[2], sgY[sy + 3] - sgY[sy - 3], mxy);
        double myx = P.c.a[0] * (sgX[sx + TX] - sgX[sx - TX]);
        myx = fma(P.c.a[1], sgX[sx + 2 * TX] - sgX[sx - 2 * TX], myx);
        myx = fma(P.c.a[2], sgX[sx + 3 * TX] - sgX[sx - 3 * TX], myx);
        const double m3 = mw[2] * (xi[li] * yi[lj] * (1.0 / 3.0));        // slot 2: the windows are already shifted
        const double v0 = m3 * mxy, v1 = m3 * myx;
        N.R[1] += v0; N.R[2] += v1;
        N.R[4] += fma(uw[2], v0, vw[2] * v1);
      }
      double* rr = rring + b3 * 5 * NPT + tl;
#pragma unroll
      for (int v = 0; v < 5; ++v) rr[v * NPT] = N.R[v];
    }
    slot7 = slot7 == 6 ? 0 : slot7 + 1;
    if (b3 == 2) { b3 = 0; own_par ^= 1u; } else ++b3;
  }
  if (A.partial) {
    const double hxy = active ? P.hh[0][gi] * P.hh[1][gj] : 0.0;
    const double tot = block_sum<NT>(fsum * hxy, red, tid);
    if (tid == 0) A.partial[(cta.z * gridDim.y + cta.y) * gridDim.x + cta.x] = tot;
  }
}

// WENO: the hybrid switch is on (the kernel also writes the node flag words); a template parameter, so that the flag code
// does not exist in the launches of the central-only configs (it cost them 1.7 % as a run-time branch)
// STAGE: the RK stage of a fused launch (0, 1, 2; residual-only launches use 0): whether R_prev exists and whether R is
// stored are compile-time facts of the launch
template <int MODE, bool WENO, int STAGE>
__global__ void __launch_bounds__(NT, 1) k_rhs(const __grid_constant__ DevP P, const RhsArgs A, const __grid_constant__ RhsMaps M) {
  extern __shared__ __align__(128) double sm[];
  // CTA -> (tile, chunk): the chunk index varies fastest with the launch order, so that the CTAs resident at any time
  // march through different z ranges (spreads the DRAM traffic; one wave in lockstep through z measured 24 % slower)
  const int lin = blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z);
  const int tix = lin / gridDim.z;
  const int3 cta = make_int3(tix % gridDim.x, tix / gridDim.x, A.cz0 + (lin % gridDim.z) * A.czs);
  const int i0 = cta.x * TX, j0 = cta.y * TY;
  const bool inside = i0 + TX <= P.nx && j0 + TY <= P.ny;
  const bool outflow = P.bc[1] == BC_OUTFLOW && i0 + TX >= P.nx;
  const bool wall_lo = (P.bc[2] == BC_WALL_STAG || node_wall(P.bc[2])) && j0 == 0;
  const bool wall_hi = (P.bc[3] == BC_WALL_STAG || node_wall(P.bc[3]) || P.bc[3] == BC_OUTFLOW) && j0 + TY >= P.ny;
  if (inside && A.use_tma && P.viscous && !outflow && !wall_lo && !wall_hi) rhs_body<MODE, true, WENO, STAGE>(P, A, M, sm, cta);
  else rhs_body<MODE, false, WENO, STAGE>(P, A, M, sm, cta);
}

}  // namespace streams
