// k_weno.cuh -- shock sensor (a3) and the WENO5 correction on flagged interfaces (a5).
//
// The hybrid switch is hard (A6): interface i+1/2 takes the characteristic-wise
// Lax-Friedrichs WENO5 flux when any of its six stencil nodes has theta > theta_th, the
// central flux otherwise.  The fused kernel evaluates the central flux
// everywhere; here the flagged interfaces add  dF = F_weno - F_central  to their two nodes.
// Work is compacted and done ONCE per interface: k_weno_list appends every flagged interface
// i+1/2 (by its lower node) to the list of its direction and every node with at least one
// flagged interface to the node list; k_weno_flux<D> runs one thread per listed interface (no
// divergence) and leaves dF in a node-indexed scratch array; k_weno_apply runs one thread per
// listed node and sums the corrections of its up to six interfaces in a fixed order (no
// floating-point atomics: deterministic).
#pragma once
#include "dev_common.cuh"
#include "k_aux.cuh"

namespace streams {

// ---- S4: theta of Eq. 8 per node -> byte flag theta > theta_th ----
__global__ void __launch_bounds__(RT) k_sensor(const __grid_constant__ DevP P, const double* __restrict__ w, unsigned char* __restrict__ nflag,
                                               double* __restrict__ theta_out, DevScal* sc) {
  __shared__ double sh[RT / 32];
  double tmax = 0.0;
  for (long long o = blockIdx.x * (long long)RT + threadIdx.x; o < P.N; o += (long long)gridDim.x * RT) {
    const int i = (int)(o % P.nx), j = (int)((o / P.nx) % P.ny), k = (int)(o / P.nxy);
    double G[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
#pragma unroll
    for (int d = 0; d < 3; ++d) {
#pragma unroll
      for (int l = 1; l <= 3; ++l) {
        double up, vp, wp, um, vm, wm;
        fetch_vel(P, w, i + (d == 0 ? l : 0), j + (d == 1 ? l : 0), k + (d == 2 ? l : 0), up, vp, wp);
        fetch_vel(P, w, i - (d == 0 ? l : 0), j - (d == 1 ? l : 0), k - (d == 2 ? l : 0), um, vm, wm);
        const double a = P.c.a[l - 1];
        G[0][d] += a * (up - um); G[1][d] += a * (vp - vm); G[2][d] += a * (wp - wm);
      }
    }
    const double ih[3] = {P.ih[0][i], P.ih[1][j], P.ih[2][k]};
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int d = 0; d < 3; ++d) G[a][d] *= ih[d];
    const double div = G[0][0] + G[1][1] + G[2][2];
    const double ox = G[2][1] - G[1][2], oy = G[0][2] - G[2][0], oz = G[1][0] - G[0][1];
    const double th = fmax(-div / sqrt(div * div + (ox * ox + oy * oy + oz * oz) + P.th_eps), 0.0);
    nflag[o] = th > P.th_thr ? 1 : 0;
    if (theta_out) theta_out[o] = th;
    tmax = fmax(tmax, th);
  }
  const double t = block_max<RT>(tmax, sh, threadIdx.x);
  if (threadIdx.x == 0) atomicMax(reinterpret_cast<unsigned long long*>(&sc->max_theta), (unsigned long long)__double_as_longlong(t));
}

constexpr unsigned int IFACE_BELOW = 0x80000000u;      // interface-list entry: the interface BELOW the (first) node
// offset of node (i,j,k) inside the boundary plane of direction D (scratch of the IFACE_BELOW entries)
template <int D>
__device__ __forceinline__ size_t plane_index(const DevP& P, int i, int j, int k) {
  return D == 0 ? (size_t)k * P.ny + j : (D == 1 ? (size_t)k * P.nx + i : (size_t)j * P.nx + i);
}
template <int D>
__device__ __forceinline__ size_t plane_size(const DevP& P) {
  return D == 0 ? (size_t)P.ny * P.nz : (D == 1 ? (size_t)P.nx * P.nz : (size_t)P.nx * P.ny);
}
// boundary scratch dFb: [x: 5 * ny*nz][y: 5 * nx*nz][z: 5 * nx*ny]
template <int D>
__device__ __forceinline__ size_t plane_base(const DevP& P) {
  return D == 0 ? 0 : (D == 1 ? 5 * plane_size<0>(P) : 5 * (plane_size<0>(P) + plane_size<1>(P)));
}

// ---- node flags as bits: fbits[row][wi], row = k * ny + j, bit b of word wi = node i = 32 wi + b (0 beyond nx) ----
__device__ __forceinline__ int words_per_row(const DevP& P) { return (P.nx + 31) >> 5; }

__global__ void __launch_bounds__(RT) k_flag_pack(const __grid_constant__ DevP P, const unsigned char* __restrict__ nflag,
                                                  unsigned int* __restrict__ fbits) {
  const int nw = words_per_row(P);
  const unsigned int nwords = (unsigned int)(P.ny * P.nz) * (unsigned int)nw;
  const int lane = threadIdx.x & 31;
  for (unsigned int wd = (blockIdx.x * RT + threadIdx.x) >> 5; wd < nwords; wd += (gridDim.x * RT) >> 5) {
    const unsigned int row = wd / (unsigned int)nw, wi = wd - row * (unsigned int)nw;
    const int i = (int)(wi << 5) + lane;
    const int f = i < P.nx ? nflag[(size_t)row * P.nx + i] : 0;
    const unsigned int bits = __ballot_sync(0xffffffffu, f != 0);
    if (lane == 0) fbits[wd] = bits;
  }
}

// one node flag by (possibly ghost) x index of row `rw`: periodic wrap, else nearest interior node (A17)
__device__ __forceinline__ unsigned int xbit(const DevP& P, const unsigned int* __restrict__ rw, int i) {
  const int ii = P.bc[0] == BC_PERIODIC ? wrap(i, P.nx) : min(max(i, 0), P.nx - 1);
  return (rw[ii >> 5] >> (ii & 31)) & 1u;
}
// row index of (j, k) with the ghost rule of the sensor along y / z; beyond a BC_HALO face the row is one of the
// neighbouring slab's (stored around the flag words like the ghost planes around the state: negative / >= nz*ny)
__device__ __forceinline__ int row_of(const DevP& P, int j, int k) {
  const int jj = P.bc[2] == BC_PERIODIC ? wrap(j, P.ny) : min(max(j, 0), P.ny - 1);
  int kk = k;
  if (k < 0) kk = P.bc[4] == BC_PERIODIC ? wrap(k, P.nz) : (P.bc[4] == BC_HALO ? k : 0);
  else if (k >= P.nz) kk = P.bc[5] == BC_PERIODIC ? wrap(k, P.nz) : (P.bc[5] == BC_HALO ? k : P.nz - 1);
  return kk * P.ny + jj;
}

// Warp-cooperative append: every lane holds the bit word of ITS 32 nodes (`bits`), the list position of its first entry
// (`pos`) and its first node (`o0`); the warp walks the non-empty words and lane b writes the entry of node b, so that one
// store instruction writes consecutive entries (a thread writing its own run costs one sector per entry).
template <class F>
__device__ __forceinline__ void warp_emit(unsigned int bits, unsigned int pos, unsigned int o0, int lane, F&& store) {
  for (unsigned int todo = __ballot_sync(0xffffffffu, bits != 0u); todo; todo &= todo - 1) {
    const int src = __ffs(todo) - 1;
    const unsigned int b = __shfl_sync(0xffffffffu, bits, src), p0 = __shfl_sync(0xffffffffu, pos, src);
    const unsigned int on = __shfl_sync(0xffffffffu, o0, src);
    if ((b >> lane) & 1u) store(on + (unsigned int)lane, p0 + (unsigned int)__popc(b & ((1u << lane) - 1u)));
  }
}

// Interface flags and lists from the packed node flags, ONE THREAD PER WORD (32 nodes of a row): interface i+1/2 along
// d is flagged iff any of nodes i-2..i+3 is (A6), i.e. an OR of six shifted words (x) or of six words of neighbouring
// rows / planes (y, z).  Entries: node list (node index + 6-bit mask, bit 2d = interface below, 2d+1 = above) of the
// nodes with a flagged interface, and per direction the list of flagged interfaces by their lower node (the interface
// below the first node of a non-periodic direction: node | IFACE_BELOW).  A CTA reserves its slots with one atomic
// per list and round; inside a CTA the entries follow the words, i.e. x, so that the consumers read their stencils coalesced.
__global__ void __launch_bounds__(RT) k_weno_list(const __grid_constant__ DevP P, const unsigned int* __restrict__ fbits,
                                                  unsigned int* __restrict__ list, unsigned char* __restrict__ lmask,
                                                  unsigned int* __restrict__ ilist /* [3][istride] or NULL */, size_t istride,
                                                  unsigned char* __restrict__ iflags_out /* [3][N] or NULL */, DevScal* sc) {
  const int nw = words_per_row(P);
  const unsigned int nwords = (unsigned int)(P.ny * P.nz) * (unsigned int)nw;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  __shared__ unsigned int s_wtot[2][4][RT / 32], s_base[2][4];
  unsigned long long cnt[3] = {0, 0, 0};
  const unsigned int nround = (nwords + gridDim.x * RT - 1) / (gridDim.x * RT);
  for (unsigned int it = 0; it < nround; ++it) {
    const unsigned int wd = (it * gridDim.x + blockIdx.x) * RT + threadIdx.x;
    const bool in = wd < nwords;
    unsigned int lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0};
    unsigned int row = 0, i0 = 0;
    int j = 0, k = 0;
    if (in) {
      row = wd / (unsigned int)nw;
      const unsigned int wi = wd - row * (unsigned int)nw;
      i0 = wi << 5;
      k = (int)(row / (unsigned int)P.ny); j = (int)(row - (unsigned int)k * (unsigned int)P.ny);
      const int nvalid = min(32, P.nx - (int)i0);
      const unsigned int valid = nvalid == 32 ? 0xffffffffu : ((1u << nvalid) - 1u);
      // ---- x: 38-bit window, bit b = node i0 - 3 + b
      {
        const unsigned int* rw = fbits + (size_t)row * nw;
        unsigned long long V = (unsigned long long)rw[wi] << 3;
#pragma unroll
        for (int b = 0; b < 3; ++b) V |= (unsigned long long)xbit(P, rw, (int)i0 - 3 + b) << b;
        // nodes right of the word: the next word when it is whole inside the row, else bit by bit (row end, ghosts)
        if ((int)i0 + 35 <= P.nx) V |= (unsigned long long)(rw[wi + 1] & 7u) << 35;
        else {
#pragma unroll
          for (int b = 0; b < 3; ++b) V |= (unsigned long long)xbit(P, rw, (int)i0 + 32 + b) << (35 + b);
          // the word's own bits beyond nx hold 0: ghost nodes inside the word take the rule as well
          for (int b = nvalid; b < min(32, nvalid + 3); ++b) V |= (unsigned long long)xbit(P, rw, (int)i0 + b) << (3 + b);
        }
        unsigned long long H = 0, L = 0;
#pragma unroll
        for (int sft = 1; sft <= 6; ++sft) H |= V >> sft;          // nodes i-2 .. i+3  <->  window bits n+1 .. n+6
#pragma unroll
        for (int sft = 0; sft <= 5; ++sft) L |= V >> sft;          // nodes i-3 .. i+2
        hi[0] = (unsigned int)H & valid; lo[0] = (unsigned int)L & valid;
      }
      // ---- y and z: the same word of six neighbouring rows / planes
      {
        unsigned int wy[7], wz[7];
#pragma unroll
        for (int g = 0; g < 7; ++g) {
          wy[g] = fbits[(long long)row_of(P, j - 3 + g, k) * nw + wi];
          wz[g] = fbits[(long long)row_of(P, j, k - 3 + g) * nw + wi];
        }
        lo[1] = wy[0] | wy[1] | wy[2] | wy[3] | wy[4] | wy[5]; hi[1] = wy[1] | wy[2] | wy[3] | wy[4] | wy[5] | wy[6];
        lo[2] = wz[0] | wz[1] | wz[2] | wz[3] | wz[4] | wz[5]; hi[2] = wz[1] | wz[2] | wz[3] | wz[4] | wz[5] | wz[6];
      }
      // the staggered wall plane is never flagged (A6)
      if (P.bc[0] == BC_WALL_STAG && i0 == 0) lo[0] &= ~1u;
      if (P.bc[1] == BC_WALL_STAG && (int)i0 + nvalid == P.nx) hi[0] &= ~(1u << (nvalid - 1));
      if (P.bc[2] == BC_WALL_STAG && j == 0) lo[1] = 0;
      if (P.bc[3] == BC_WALL_STAG && j == P.ny - 1) hi[1] = 0;
      if (P.bc[4] == BC_WALL_STAG && k == 0) lo[2] = 0;
      if (P.bc[5] == BC_WALL_STAG && k == P.nz - 1) hi[2] = 0;
      cnt[0] += __popc(hi[0]) + ((i0 == 0 && P.bc[0] != BC_PERIODIC) ? (lo[0] & 1u) : 0u);
      cnt[1] += __popc(hi[1]) + ((j == 0 && P.bc[2] != BC_PERIODIC) ? __popc(lo[1]) : 0);
      cnt[2] += __popc(hi[2]) + ((k == 0 && P.bc[4] != BC_PERIODIC) ? __popc(lo[2]) : 0);
      if (iflags_out) {
        for (int b = 0; b < nvalid; ++b) {
          const size_t o = (size_t)row * P.nx + i0 + b;
#pragma unroll
          for (int d = 0; d < 3; ++d) iflags_out[d * P.N + o] = (unsigned char)((hi[d] >> b) & 1u);
        }
      }
    }
    const unsigned int o0 = row * (unsigned int)P.nx + i0;           // node of bit 0 (N < 2^31 with the switch on)
    // ---- entries of this word in the four lists (0..2: interfaces along d, 3: nodes)
    unsigned int lb[3] = {0, 0, 0};                                  // below-entries: first node of a non-periodic direction
    if (in && ilist) {
      if (P.bc[0] != BC_PERIODIC && i0 == 0) lb[0] = lo[0] & 1u;
      if (P.bc[2] != BC_PERIODIC && j == 0) lb[1] = lo[1];
      if (P.bc[4] != BC_PERIODIC && k == 0) lb[2] = lo[2];
    }
    const unsigned int any = (in && list) ? (lo[0] | hi[0] | lo[1] | hi[1] | lo[2] | hi[2]) : 0u;
    unsigned int n_me[4], pre[4];
#pragma unroll
    for (int l = 0; l < 3; ++l) n_me[l] = (in && ilist) ? (unsigned int)(__popc(hi[l]) + __popc(lb[l])) : 0u;
    n_me[3] = (unsigned int)__popc(any);
    // The CTA reserves its slots with ONE atomic per list and round (a warp-wise reservation made 4 x 32 768 atomics on
    // four neighbouring counters for config 4: the kernel ran at the rate of same-address atomics).  Two sets of the
    // shared counters alternate between rounds, so that a warp that runs ahead cannot overwrite what a slower one reads.
    unsigned int* wt = s_wtot[it & 1][0];
#pragma unroll
    for (int l = 0; l < 4; ++l) {
      unsigned int v = n_me[l];                                      // inclusive warp prefix sum
#pragma unroll
      for (int sft = 1; sft < 32; sft <<= 1) { const unsigned int t = __shfl_up_sync(0xffffffffu, v, sft); if (lane >= sft) v += t; }
      pre[l] = v;
      if (lane == 31) wt[l * (RT / 32) + wid] = v;
    }
    __syncthreads();
    if (threadIdx.x < 4) {
      unsigned int tot = 0;
#pragma unroll
      for (int w = 0; w < RT / 32; ++w) tot += wt[threadIdx.x * (RT / 32) + w];
      unsigned int* counter = threadIdx.x < 3 ? &sc->icount[threadIdx.x] : &sc->list_count;
      s_base[it & 1][threadIdx.x] = tot ? atomicAdd(counter, tot) : 0u;
    }
    __syncthreads();
    unsigned int pos[4];
#pragma unroll
    for (int l = 0; l < 4; ++l) {
      unsigned int base = s_base[it & 1][l];
      for (int w = 0; w < wid; ++w) base += wt[l * (RT / 32) + w];
      pos[l] = base + pre[l] - n_me[l];
    }
    // ---- interface lists: the warp writes the entries of one word at a time (lane b = node b of the word)
    if (ilist) {
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        unsigned int* li = ilist + d * istride;
        warp_emit(hi[d], pos[d], o0, lane, [&](unsigned int node, unsigned int at) { li[at] = node; });
        warp_emit(lb[d], pos[d] + (unsigned int)__popc(hi[d]), o0, lane, [&](unsigned int node, unsigned int at) { li[at] = node | IFACE_BELOW; });
      }
    }
    // ---- node list
    if (list) {
      for (unsigned int todo = __ballot_sync(0xffffffffu, any != 0u); todo; todo &= todo - 1) {
        const int src = __ffs(todo) - 1;
        const unsigned int bw = __shfl_sync(0xffffffffu, any, src), p0 = __shfl_sync(0xffffffffu, pos[3], src);
        const unsigned int on = __shfl_sync(0xffffffffu, o0, src);
        unsigned int m = 0;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
          m |= ((__shfl_sync(0xffffffffu, lo[d], src) >> lane) & 1u) << (2 * d);
          m |= ((__shfl_sync(0xffffffffu, hi[d], src) >> lane) & 1u) << (2 * d + 1);
        }
        if ((bw >> lane) & 1u) {
          const unsigned int at = p0 + (unsigned int)__popc(bw & ((1u << lane) - 1u));
          list[at] = on + (unsigned int)lane;
          lmask[at] = (unsigned char)m;
        }
      }
    }
  }
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    for (int sft = 16; sft > 0; sft >>= 1) cnt[d] += __shfl_down_sync(0xffffffffu, cnt[d], sft);
    if ((threadIdx.x & 31) == 0 && cnt[d]) atomicAdd(&sc->weno_if[d], cnt[d]);
  }
}

// WENO5-JS reconstruction (ref. [34]) as numerator and denominator: value = num / den.
// Weights a_k = d_k / (eps + b_k)^2 written over the common denominator e0 e1 e2: w_k = d_k prod_{j != k} e_j,
// value = sum w_k q_k / sum w_k.  The caller adds the upwind and the downwind reconstruction of a characteristic field
// over ONE division: n+/d+ + n-/d- = (n+ d- + n- d+) / (d+ d-)  (one division per field instead of four in the textbook form).
__device__ __forceinline__ void weno5_nd(double a, double b, double c, double d, double e, double& num, double& den) {
  const double q0 = (2.0 * a - 7.0 * b + 11.0 * c) * (1.0 / 6.0);
  const double q1 = (-b + 5.0 * c + 2.0 * d) * (1.0 / 6.0);
  const double q2 = (2.0 * c + 5.0 * d - e) * (1.0 / 6.0);
  const double t0 = a - 2.0 * b + c, u0 = a - 4.0 * b + 3.0 * c;
  const double t1 = b - 2.0 * c + d, u1 = b - d;
  const double t2 = c - 2.0 * d + e, u2 = 3.0 * c - 4.0 * d + e;
  const double b0 = (13.0 / 12.0) * t0 * t0 + 0.25 * u0 * u0;
  const double b1 = (13.0 / 12.0) * t1 * t1 + 0.25 * u1 * u1;
  const double b2 = (13.0 / 12.0) * t2 * t2 + 0.25 * u2 * u2;
  const double eps = 1e-6;
  const double e0 = (eps + b0) * (eps + b0), e1 = (eps + b1) * (eps + b1), e2 = (eps + b2) * (eps + b2);
  const double a0 = 0.1 * (e1 * e2), a1 = 0.6 * (e0 * e2), a2 = 0.3 * (e0 * e1);
  num = a0 * q0 + a1 * q1 + a2 * q2;
  den = a0 + a1 + a2;
}
// Third-order variant (reading A23): candidates {a,b}, {b,c}, linear weights 1/3, 2/3, smoothness (b-a)^2, (c-b)^2; as
// numerator and denominator over the common denominator e0 e1 like weno5_nd.
__device__ __forceinline__ void weno3_nd(double a, double b, double c, double& num, double& den) {
  const double q0 = 0.5 * (3.0 * b - a), q1 = 0.5 * (b + c);
  const double t0 = b - a, t1 = c - b;
  const double e0 = 1e-6 + t0 * t0, e1 = 1e-6 + t1 * t1;
  const double w0 = (1.0 / 3.0) * (e1 * e1), w1 = (2.0 / 3.0) * (e0 * e0);
  num = w0 * q0 + w1 * q1;
  den = w0 + w1;
}

// rho, u, v, w, T of a (possibly ghost) node by the rules of S1, out of line and returned by value (stays in registers)
struct P5 { double rho, u, v, w, T; };
__device__ __noinline__ P5 fetch_prim5_ghost(const DevP& P, const double* __restrict__ w, int i, int j, int k) {
  Prim q;
  fetch_prim5(P, w, i, j, k, q);
  P5 r;
  r.rho = q.rho; r.u = q.u; r.v = q.v; r.w = q.w; r.T = q.T;
  return r;
}

// dF = F_weno - F_central at the interface between node (i,j,k) and its upper neighbour along D (S5, S6)
template <int D, int ORD>
__device__ void weno_delta(const DevP& P, const double* __restrict__ w, int i, int j, int k, double dF[5]) {
  double rho[6], vel[6][3], Hh[6], pp[6], cs[6];
  // The six stencil nodes i-2 .. i+3 along D.  Nearly every listed interface has all six inside the grid: plain strided
  // loads.  The ghost rules of S1 (index maps, reflection, inflow / free-stream sources) cost ~150 instructions per node
  // when inlined six times (the kernel was 3700 instructions, 60 KB: `no_instruction` was its second largest stall);
  // stencils that reach a face take them through ONE out-of-line copy.
  // A periodic direction only wraps the index and a BC_HALO face stores its ghost planes around the state: both stay
  // on the plain path (all of config 2; a warp whose lanes disagree pays both paths).
  const int id = D == 0 ? i : (D == 1 ? j : k), nd = D == 0 ? P.nx : (D == 1 ? P.ny : P.nz);
  const bool per = P.bc[2 * D] == BC_PERIODIC;
  const bool inside = (id >= 2 || per || (D == 2 && P.bc[4] == BC_HALO)) && (id + 3 < nd || per || (D == 2 && P.bc[5] == BC_HALO));
  const long long st = D == 0 ? 1 : (D == 1 ? (long long)P.nx : P.nxy);
  const double* q0 = w + (((long long)k * P.ny + j) * P.nx + i) - id * st;      // index 0 along D
#pragma unroll
  for (int n = 0; n < 6; ++n) {
    P5 q;
    if (inside) {
      int m = id + n - 2;
      if (per) m = m < 0 ? m + nd : (m >= nd ? m - nd : m);
      const double* qn = q0 + m * st;
      q.rho = __ldg(qn); q.u = __ldg(qn + P.QS); q.v = __ldg(qn + 2 * P.QS); q.w = __ldg(qn + 3 * P.QS); q.T = __ldg(qn + 4 * P.QS);
    } else {
      const int off = n - 2;
      q = fetch_prim5_ghost(P, w, i + (D == 0 ? off : 0), j + (D == 1 ? off : 0), k + (D == 2 ? off : 0));
    }
    rho[n] = q.rho; vel[n][0] = q.u; vel[n][1] = q.v; vel[n][2] = q.w;
    derive_pH(P, q.rho, q.u, q.v, q.w, q.T, pp[n], Hh[n]);
    cs[n] = sqrt(P.gam * P.Rgas * q.T);
  }
  // central flux, flux form of Eq. 7: pairs (i-m, i-m+l); local index of node i is 2
  double Fc[5] = {0, 0, 0, 0, 0};
#pragma unroll
  for (int l = 1; l <= 3; ++l) {
    const double a = P.c.a[l - 1];
#pragma unroll
    for (int m = 0; m < l; ++m) {
      const int ia = 2 - m, ib = 2 - m + l;
      const double mm = (rho[ia] + rho[ib]) * (vel[ia][D] + vel[ib][D]);
      Fc[0] += (0.5 * a) * mm;
      Fc[1] += (0.25 * a) * (mm * (vel[ia][0] + vel[ib][0]));
      Fc[2] += (0.25 * a) * (mm * (vel[ia][1] + vel[ib][1]));
      Fc[3] += (0.25 * a) * (mm * (vel[ia][2] + vel[ib][2]));
      Fc[4] += (0.25 * a) * (mm * (Hh[ia] + Hh[ib]));
      Fc[1 + D] += a * (pp[ia] + pp[ib]);
    }
  }
  // Roe state (S6 step 1) and eigenvectors (step 2)
  constexpr int T1 = (D + 1) % 3, T2 = (D + 2) % 3;
  const double r = sqrt(rho[3] / rho[2]), ir1 = 1.0 / (1.0 + r);
  double ub[3];
#pragma unroll
  for (int m = 0; m < 3; ++m) ub[m] = (vel[2][m] + r * vel[3][m]) * ir1;
  const double Hb = (Hh[2] + r * Hh[3]) * ir1;
  const double q2 = ub[0] * ub[0] + ub[1] * ub[1] + ub[2] * ub[2];
  const double c2 = P.gm1 * (Hb - 0.5 * q2), cb = sqrt(c2), icb = 1.0 / cb;
  const double b1 = P.gm1 / c2, b2 = 0.5 * q2 * b1;
  const double un = ub[D];
  // steps 3-4: characteristic variables/fluxes at the six nodes, local LF speeds.  With w = (rho, rho u, rho H - p) and
  // f = vn w + p (e_{1+D} + vn e_5) the projections l_s . w and l_s . f collapse to a few operations per node:
  //   a = rho (b2 + b1 (H - ub.u)) - b1 p,   d = rho (un - vn) / cb
  //   l_1,5 . w = (a +- d) / 2,  l_2 . w = rho - a,  l_3,4 . w = rho (u_T - ub_T)
  //   l_s . f = vn (l_s . w) + p (l_s[1+D] + vn l_s[5]):  e = b1 (vn - un) p, h = p / cb:  (e -+ h)/2, -e, 0, 0
  // (the same left eigenvectors as SURVEY S6, multiplied out; equal to the matrix-vector products up to rounding)
  double wc[6][5], fc[6][5], al[5] = {0, 0, 0, 0, 0};
#pragma unroll
  for (int n = 0; n < 6; ++n) {
    const double vn = vel[n][D];
    const double m = ub[0] * vel[n][0] + ub[1] * vel[n][1] + ub[2] * vel[n][2];
    const double g = b2 + b1 * (Hh[n] - m);
    const double a = rho[n] * g - b1 * pp[n];
    const double d = icb * (rho[n] * (un - vn));
    wc[n][0] = 0.5 * (a + d);
    wc[n][1] = rho[n] - a;
    wc[n][2] = rho[n] * (vel[n][T1] - ub[T1]);
    wc[n][3] = rho[n] * (vel[n][T2] - ub[T2]);
    wc[n][4] = 0.5 * (a - d);
    const double e = b1 * ((vn - un) * pp[n]), h = icb * pp[n];
    fc[n][0] = vn * wc[n][0] + 0.5 * (e - h);
    fc[n][1] = vn * wc[n][1] - e;
    fc[n][2] = vn * wc[n][2];
    fc[n][3] = vn * wc[n][3];
    fc[n][4] = vn * wc[n][4] + 0.5 * (e + h);
    if (ORD == 5 || (n >= 1 && n <= 4)) {                // local LF: the nodes the reconstruction reads (A23)
      al[0] = fmax(al[0], fabs(vn - cs[n]));
      al[1] = fmax(al[1], fabs(vn));
      al[4] = fmax(al[4], fabs(vn + cs[n]));
    }
  }
  al[2] = al[1]; al[3] = al[1];
  // steps 5-6: split and reconstruct
  double fh[5];
#pragma unroll
  for (int s = 0; s < 5; ++s) {
    double fp[6], fm[6];
#pragma unroll
    for (int n = 0; n < 6; ++n) { fp[n] = 0.5 * (fc[n][s] + al[s] * wc[n][s]); fm[n] = 0.5 * (fc[n][s] - al[s] * wc[n][s]); }
    double np_, dp_, nm_, dm_;
    if (ORD == 5) {
      weno5_nd(fp[0], fp[1], fp[2], fp[3], fp[4], np_, dp_);
      weno5_nd(fm[5], fm[4], fm[3], fm[2], fm[1], nm_, dm_);
    } else {
      weno3_nd(fp[1], fp[2], fp[3], np_, dp_);
      weno3_nd(fm[4], fm[3], fm[2], nm_, dm_);
    }
    // range: den ~ (eps + beta)^4 with beta ~ F^2 (F = characteristic flux), so d+ d- ~ F^16 between 1e-48 (smooth
    // data, eps^8) and fp64 overflow at F ~ 1e19: no rescaling needed in any sensible unit system
    fh[s] = (np_ * dm_ + nm_ * dp_) / (dp_ * dm_);
  }
  // step 7: back to conservative variables
  double Fw[5];
  Fw[0] = fh[0] + fh[1] + fh[4];
#pragma unroll
  for (int m = 0; m < 3; ++m) Fw[1 + m] = ub[m] * (fh[0] + fh[1] + fh[4]);
  Fw[1 + D] += cb * (fh[4] - fh[0]);
  Fw[1 + T1] += fh[2];
  Fw[1 + T2] += fh[3];
  Fw[4] = (Hb - un * cb) * fh[0] + 0.5 * q2 * fh[1] + ub[T1] * fh[2] + ub[T2] * fh[3] + (Hb + un * cb) * fh[4];
#pragma unroll
  for (int v = 0; v < 5; ++v) dF[v] = Fw[v] - Fc[v];
}

// one thread per listed interface of direction D: dF of the interface above node o -> dFbuf[D][v][o]
// (IFACE_BELOW entries: the interface below the first node -> dFb, the boundary-plane scratch)
template <int D, int MB, int ORD>
__global__ void __launch_bounds__(128, MB) k_weno_flux(const __grid_constant__ DevP P, const double* __restrict__ w, const unsigned int* __restrict__ ilist,
                                                   size_t istride, const DevScal* __restrict__ sc, double* __restrict__ dFbuf, double* __restrict__ dFb) {
  const unsigned int n = sc->icount[D];
  const unsigned int* li = ilist + D * istride;
  double* out = dFbuf + (size_t)D * 5 * P.N;
  for (unsigned int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
    const unsigned int en = li[e];
    const bool below = (en & IFACE_BELOW) != 0;
    const unsigned int o = en & ~IFACE_BELOW, row = o / (unsigned int)P.nx;
    const int i = (int)(o - row * (unsigned int)P.nx), k = (int)(row / (unsigned int)P.ny), j = (int)(row - (unsigned int)k * (unsigned int)P.ny);
    double dF[5];
    weno_delta<D, ORD>(P, w, i - (below && D == 0), j - (below && D == 1), k - (below && D == 2), dF);
    if (below) {
      double* ob = dFb + plane_base<D>(P) + plane_index<D>(P, i, j, k);
#pragma unroll
      for (int v = 0; v < 5; ++v) ob[v * plane_size<D>(P)] = dF[v];
    } else {
#pragma unroll
      for (int v = 0; v < 5; ++v) out[o + v * P.N] = dF[v];
    }
  }
}

// dF of the interface BELOW node (i,j,k) along D: the scratch entry of the lower neighbour, or of the boundary plane
template <int D>
__device__ __forceinline__ void dF_below(const DevP& P, const double* __restrict__ dFbuf, const double* __restrict__ dFb, int i, int j, int k, double dF[5]) {
  const int id = D == 0 ? i : (D == 1 ? j : k), n = D == 0 ? P.nx : (D == 1 ? P.ny : P.nz);
  if (id == 0 && P.bc[2 * D] != BC_PERIODIC) {
    const double* ib = dFb + plane_base<D>(P) + plane_index<D>(P, i, j, k);
#pragma unroll
    for (int v = 0; v < 5; ++v) dF[v] = ib[v * plane_size<D>(P)];
    return;
  }
  const int im = id == 0 ? n - 1 : id - 1;
  const size_t o = ((size_t)(D == 2 ? im : k) * P.ny + (D == 1 ? im : j)) * P.nx + (D == 0 ? im : i);
  const double* in = dFbuf + (size_t)D * 5 * P.N;
#pragma unroll
  for (int v = 0; v < 5; ++v) dF[v] = in[o + v * P.N];
}

// one thread per listed node: R += dR (if R), and (if q_new) the node of the already advanced state takes the
// conservative increment dt beta dR  (Eq. 11 is linear in R)
__global__ void __launch_bounds__(RT) k_weno_apply(const __grid_constant__ DevP P, const double* __restrict__ w, const unsigned int* __restrict__ list,
                                                   const unsigned char* __restrict__ lmask, const DevScal* __restrict__ sc,
                                                   const double* __restrict__ dFbuf, const double* __restrict__ dFb,
                                                   double* __restrict__ R, double* __restrict__ q_new, double beta) {
  const unsigned int n = sc->list_count;
  const double dtb = sc->dt * beta;
  for (unsigned int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
    const unsigned int o = list[e], row = o / (unsigned int)P.nx;
    const int mask = lmask[e];
    const int i = (int)(o - row * (unsigned int)P.nx), k = (int)(row / (unsigned int)P.ny), j = (int)(row - (unsigned int)k * (unsigned int)P.ny);
    double dR[5] = {0, 0, 0, 0, 0};
    double dF[5];
    const bool skip_x = i == P.nx - 1 && P.bc[1] == BC_OUTFLOW;   // S8 replaces the x-difference there
    if (!skip_x) {
      const double ih = P.ih[0][i];
      if (mask & 1) { dF_below<0>(P, dFbuf, dFb, i, j, k, dF);
#pragma unroll
        for (int v = 0; v < 5; ++v) dR[v] += ih * dF[v]; }
      if (mask & 2) {
#pragma unroll
        for (int v = 0; v < 5; ++v) dR[v] -= ih * dFbuf[o + v * P.N]; }
    }
    // the characteristic forms at a non-reflecting top / characteristic wall replace the y-difference of those rows
    const bool skip_y = (j == P.ny - 1 && P.bc[3] == BC_OUTFLOW) || (j == 0 && P.bc[2] == BC_WALL_CHAR);
    if (!skip_y) {
      const double ih = P.ih[1][j];
      if (mask & 4) { dF_below<1>(P, dFbuf, dFb, i, j, k, dF);
#pragma unroll
        for (int v = 0; v < 5; ++v) dR[v] += ih * dF[v]; }
      if (mask & 8) {
#pragma unroll
        for (int v = 0; v < 5; ++v) dR[v] -= ih * dFbuf[(size_t)5 * P.N + o + v * P.N]; }
    }
    {
      const double ih = P.ih[2][k];
      if (mask & 16) { dF_below<2>(P, dFbuf, dFb, i, j, k, dF);
#pragma unroll
        for (int v = 0; v < 5; ++v) dR[v] += ih * dF[v]; }
      if (mask & 32) {
#pragma unroll
        for (int v = 0; v < 5; ++v) dR[v] -= ih * dFbuf[(size_t)10 * P.N + o + v * P.N]; }
    }
    if (R) {                                             // NULL in the last RK stage: its R is never read
#pragma unroll
      for (int v = 0; v < 5; ++v) R[o + v * P.N] += dR[v];
    }
    if (q_new) {
      const bool wall = (j == 0 && node_wall(P.bc[2])) || (j == P.ny - 1 && node_wall(P.bc[3]));
      if (wall) {
        q_new[o] += dtb * dR[0];                      // u = v = w = 0 and T = T_w stay as overridden (S1)
      } else {
        Prim q;
        q.rho = q_new[o]; q.u = q_new[o + P.QS]; q.v = q_new[o + 2 * P.QS]; q.w = q_new[o + 3 * P.QS]; q.T = q_new[o + 4 * P.QS]; q.mu = 0.0;
        double dW[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) dW[v] = dtb * dR[v];
        advance_prim(P, q, dW);
        q_new[o] = q.rho; q_new[o + P.QS] = q.u; q_new[o + 2 * P.QS] = q.v; q_new[o + 3 * P.QS] = q.w; q_new[o + 4 * P.QS] = q.T; q_new[o + 5 * P.QS] = q.mu; q_new[o + 6 * P.QS] = q.H;
      }
    }
  }
}

}  // namespace streams
