// k_stats.cuh -- Reynolds / Favre statistics in the homogeneous directions: x-z plane means per
// wall-normal index j of NSTAT quantities, added to running sums on the device (time average = sums / samples).
//
// HBM-bound: one pass over six stored primitives (48 B per node).  One CTA per (row j, z-chunk): threads walk the
// x rows of the chunk's planes (coalesced), 16 register accumulators per thread, fixed-order block reduction into
// partial[zc][m][j]; k_stats_final adds the chunks in a fixed order (deterministic: no floating-point atomics).
#pragma once
#include "dev_common.cuh"
#include "k_aux.cuh"

namespace streams {

constexpr int NSTAT = 16;   // rho, u, v, w, p, T, mu, rho u, rho v, rho w, rho T, rho u u, rho v v, rho w w, rho u v, T T
constexpr int STAT_ZC = 8;  // z-chunks per row (at most)

__global__ void __launch_bounds__(RT) k_stats_partial(const __grid_constant__ DevP P, const double* __restrict__ Q, int nzc,
                                                      double* __restrict__ partial /* [nzc][NSTAT][ny] */) {
  __shared__ double sh[RT / 32];
  const int j = blockIdx.x, zc = blockIdx.y;
  const int kz0 = (int)((long long)P.nz * zc / nzc), kz1 = (int)((long long)P.nz * (zc + 1) / nzc);
  double a[NSTAT];
#pragma unroll
  for (int m = 0; m < NSTAT; ++m) a[m] = 0.0;
  for (int k = kz0; k < kz1; ++k) {
    const size_t r0 = ((size_t)k * P.ny + j) * P.nx;
    for (int i = threadIdx.x; i < P.nx; i += RT) {
      const size_t o = r0 + i;
      const double rho = Q[o], u = Q[o + P.QS], v = Q[o + 2 * P.QS], w = Q[o + 3 * P.QS], T = Q[o + 4 * P.QS], mu = Q[o + 5 * P.QS];
      const double ru = rho * u, rv = rho * v, rw = rho * w;
      a[0] += rho; a[1] += u; a[2] += v; a[3] += w; a[4] += rho * (P.Rgas * T); a[5] += T; a[6] += mu;
      a[7] += ru; a[8] += rv; a[9] += rw; a[10] += rho * T;
      a[11] = fma(ru, u, a[11]); a[12] = fma(rv, v, a[12]); a[13] = fma(rw, w, a[13]); a[14] = fma(ru, v, a[14]);
      a[15] = fma(T, T, a[15]);
    }
  }
#pragma unroll
  for (int m = 0; m < NSTAT; ++m) {
    const double t = block_sum<RT>(a[m], sh, threadIdx.x);
    if (threadIdx.x == 0) partial[((size_t)zc * NSTAT + m) * P.ny + j] = t;
  }
}

// sums[m][j] += (sum over chunks of partial) / (nx nz);  one thread per (m, j); thread 0 counts the sample
__global__ void k_stats_final(const __grid_constant__ DevP P, const double* __restrict__ partial, int nzc,
                              double* __restrict__ sums /* [NSTAT][ny] */, unsigned long long* __restrict__ count) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e == 0) *count += 1ull;
  if (e >= NSTAT * P.ny) return;
  double t = 0.0;
  for (int zc = 0; zc < nzc; ++zc) t += partial[(size_t)zc * NSTAT * P.ny + e];
  sums[e] += t / ((double)P.nx * (double)P.nz);
}

}  // namespace streams
