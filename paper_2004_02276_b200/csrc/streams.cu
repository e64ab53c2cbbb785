// streams.cu -- C-ABI entry points of include/streams.h: context, metrics, launch sequence.
//
// Host logic only: every field-sized operation is a kernel from k_rhs.cuh / k_aux.cuh /
// k_weno.cuh enqueued on the caller's stream.  There is no CPU fallback: any CUDA failure
// is reported as STREAMS_ECUDA.
#include "../../include/streams.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "dev_common.cuh"
#include "k_aux.cuh"
#include "k_rhs.cuh"
#include "k_stats.cuh"
#include "k_weno.cuh"

using namespace streams;

namespace {
thread_local char g_err[256] = "no error";
constexpr int RGRID = 148 * 8;           // CTAs of the grid-stride reduction kernels (148 SMs)
constexpr size_t ALIGN = 256;
inline size_t up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }
}  // namespace

struct streams_ctx {
  streams_grid g;
  streams_params p;
  DevP P;
  cudaStream_t st;
  // workspace carve-up (caller memory)
  double *qbuf[2], *S[2], *theta, *partial, *inflow, *speeds;   // qbuf: primitives [NQ][N]; S: R registers [5][N]
  unsigned char *nflag, *lmask;
  unsigned int* fbits;                 // node flags as bits, [nz*ny][ceil(nx/32)]
  unsigned int* list;
  unsigned int* ilist;                 // [3][N] interface lists (lower node of each flagged interface)
  double* dFbuf;                       // [3][5][N] dF of the interface above each node (flagged entries only)
  double* dFb;                         // dF of the interfaces below the first node of a non-periodic direction
  int npartial;
  // context-owned small device memory
  void* small_dev;
  DevScal* sc;
  int cur, scur;                 // current state buffer, current "previous-R" buffer
  int has_state;
  long long step;
  long long launches;
  dim3 rhs_grid;
  int lz;
  size_t istride;                      // entries per direction of ilist
  int dt_ready;                        // sc->red[2] holds the CFL maximum of the current state (last k_force_fix of a step)
  int zpad;                            // ghost planes stored around each state buffer (3 with a BC_HALO z face)
  int stage_next;                      // staged stepping: -1 = between steps, else the stage whose streams_stage_rhs /
  int stage_half;                      // streams_stage_end comes next (half: 0 = rhs pending, 1 = end pending)
  int inflow_pending;                  // z-slab with INFLOW_FROZEN: the frozen plane is captured once the ghost planes are in
  int parts_done;                      // bit 0: interior chunks launched, bit 1: boundary chunks launched (this stage)
  int mid_done;                        // forcing + hybrid switch: streams_stage_mid has corrected R and summed it (this stage)
  // TMA descriptors, 4-D (x, y, z, field): per state buffer the tile box (halo 3) and the own-node box (no halo)
  CUtensorMap tmap[2], tmap_own[2];
  int use_tma;                   // 0 when nx is odd (TMA needs 16-byte row strides): tiles are filled by index
  int prof_on, prof_n;
  std::vector<cudaEvent_t>* prof_ev;   // pairs (start, stop) around k_rhs
  int device;                          // CUDA device the context was created on; every entry point switches to it
  // one RK3 step as a CUDA graph (launch-bound small grids): one executable per host-state key, see step_key()
  int graph_ok;                        // 0: direct launches only (legacy default stream, capture failed, disabled)
  cudaGraphExec_t gexec[8];
  int g_after[8];                      // host state (key) after the step captured from key k
  int g_launches[8];                   // kernel launches inside the graph (bench accounting)
  double* stat_partial;                // [STAT_ZC][NSTAT][ny] chunk sums of the statistics pass (context-owned, O(ny))
  double* stat_sum;                    // [NSTAT][ny] running sums of the plane means
  unsigned long long* stat_n;          // accumulated samples
  DevScal* h_sc;                       // pinned host copies for streams_diagnostics (no pageable-memory async copies)
  double* h_part;
  char err[256];
};

namespace {

int fail(streams_ctx* c, int code, const char* msg) {
  snprintf(g_err, sizeof g_err, "%s", msg);
  if (c) snprintf(c->err, sizeof c->err, "%s", msg);
  return code;
}
int cuda_fail(streams_ctx* c, cudaError_t e, const char* where) {
  char b[256];
  snprintf(b, sizeof b, "CUDA error at %s: %s", where, cudaGetErrorString(e));
  return fail(c, STREAMS_ECUDA, b);
}
#define CK(call)                                                   \
  do {                                                             \
    cudaError_t e_ = (call);                                       \
    if (e_ != cudaSuccess) return cuda_fail(c, e_, #call);         \
  } while (0)
#define LAUNCH_CHECK(name)                                         \
  do {                                                             \
    c->launches++;                                                 \
    cudaError_t e_ = cudaGetLastError();                           \
    if (e_ != cudaSuccess) return cuda_fail(c, e_, name);          \
  } while (0)

// every entry point runs on the device the context was created on, whatever the caller's current device is
struct DevGuard {
  int prev = -1, dev;
  explicit DevGuard(int d) : dev(d) { if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) cudaSetDevice(dev); else prev = dev; }
  ~DevGuard() { if (prev != dev) cudaSetDevice(prev); }
};

bool coeffs(int order, Coef& k) {
  for (int i = 0; i < 3; ++i) k.a[i] = k.b[i] = k.qa[i] = k.aR[i] = 0.0;
  k.sb2 = 0.0;
  if (order == 2) { k.a[0] = 0.5; k.b[0] = 1.0; return true; }
  if (order == 4) { k.a[0] = 2.0 / 3.0; k.a[1] = -1.0 / 12.0; k.b[0] = 4.0 / 3.0; k.b[1] = -1.0 / 12.0; return true; }
  if (order == 6) { k.a[0] = 0.75; k.a[1] = -0.15; k.a[2] = 1.0 / 60.0; k.b[0] = 1.5; k.b[1] = -0.15; k.b[2] = 1.0 / 90.0; return true; }
  return false;
}

const char* validate(const streams_grid* g, const streams_params* p) {
  if (g->nx < 1 || g->ny < 1 || g->nz < 1) return "grid sizes must be >= 1";
  if ((long long)g->nx * g->ny * g->nz > 0xffffffffLL) return "more than 2^32 nodes";
  if ((long long)g->nx * g->ny > 0x3fffffffLL) return "more than 2^30 nodes per z-plane";
  if ((long long)g->ny * g->nz > 0x7fffffffLL) return "more than 2^31 grid rows (ny * nz)";
  if (!(p->gamma > 1.0) || !(p->Rgas > 0.0) || !(p->Pr > 0.0)) return "gamma > 1, Rgas > 0, Pr > 0 required";
  if (p->order != 2 && p->order != 4 && p->order != 6) return "order must be 2, 4 or 6";
  if (p->weno_enable && (long long)g->nx * g->ny * g->nz > 0x7fffffffLL) return "more than 2^31 nodes with the hybrid switch on (interface lists)";
  if (p->weno_enable && !(p->sensor_eps > 0.0)) return "sensor_eps must be > 0 (Eq. 8 is 0/0 in uniform flow otherwise)";
  if (p->weno_order != 0 && p->weno_order != 3 && p->weno_order != 5) return "weno_order must be 3 or 5 (0 = 5)";
  if (p->visc_model != STREAMS_VISC_POWER && p->visc_model != STREAMS_VISC_SUTHERLAND) return "unknown visc_model";
  if (!(p->cfl > 0.0) && !(p->dt_fixed > 0.0)) return "cfl > 0 or dt_fixed > 0 required";
  const int n[3] = {g->nx, g->ny, g->nz};
  for (int d = 0; d < 3; ++d) {
    const int lo = p->bc[2 * d], hi = p->bc[2 * d + 1];
    if ((lo == STREAMS_BC_PERIODIC) != (hi == STREAMS_BC_PERIODIC)) return "periodic must be set on both faces of a direction";
    if (lo != STREAMS_BC_PERIODIC && n[d] < 4) return "non-periodic directions need >= 4 nodes";
    if (lo == STREAMS_BC_PERIODIC && !(g->len[d] > 0.0)) return "periodic directions need len > 0";
    for (int s = 0; s < 2; ++s) {
      const int b = p->bc[2 * d + s];
      if (b < 0 || b > STREAMS_BC_HALO) return "unknown boundary kind";
      if (b == STREAMS_BC_HALO && d != 2) return "HALO (z-slab decomposition) is supported on z faces only";
      if (b == STREAMS_BC_WALL_ISO_CHAR && !(d == 1 && s == 0)) return "WALL_ISO_CHAR is supported on ymin only";
      if ((b == STREAMS_BC_WALL_ISO_STAGGERED || b == STREAMS_BC_WALL_ISO_NODE) && d != 1) return "walls are supported on y faces only";
      if (b == STREAMS_BC_INFLOW_FROZEN && !(d == 0 && s == 0)) return "INFLOW_FROZEN is supported on xmin only";
      if (b == STREAMS_BC_OUTFLOW_NR && !((d == 0 || d == 1) && s == 1)) return "OUTFLOW_NR is supported on xmax and ymax only";
      if (b == STREAMS_BC_SHOCKGEN && !(d == 1 && s == 1)) return "SHOCKGEN is supported on ymax only";
    }
  }
  if (p->forcing && p->bc[0] != STREAMS_BC_PERIODIC) return "bulk forcing needs a periodic x direction";
  return nullptr;
}

double visc_host(const streams_params& p, double T) {
  if (p.visc_model == STREAMS_VISC_SUTHERLAND) return p.mu_ref * std::pow(T / p.T_ref, 1.5) * (p.T_ref + p.suth_S) / (T + p.suth_S);
  return p.mu_ref * std::pow(T / p.T_ref, p.visc_exp);
}

// S1 shock generator: weak oblique-shock solution for the deflection angle
bool shock_post_state(const streams_params& p, double post[NQ]) {
  const double g = p.gamma, u1 = p.fs[1], T1 = p.fs[4];
  const double M = u1 / std::sqrt(g * p.Rgas * T1);
  const double tphi = std::tan(p.shock_angle_deg * 3.14159265358979323846 / 180.0);
  if (!(M > 1.0) || !(tphi > 0.0)) return false;
  auto f = [&](double b) { const double s = std::sin(b); return 2.0 / std::tan(b) * (M * M * s * s - 1.0) / (M * M * (g + std::cos(2.0 * b)) + 2.0); };
  // golden-section search of the maximum-deflection angle, then bisection on the weak branch
  const double mu = std::asin(1.0 / M);
  double a = mu, b = 0.5 * 3.14159265358979323846;
  const double gr = 0.6180339887498949;
  for (int it = 0; it < 200; ++it) {
    const double x1 = b - gr * (b - a), x2 = a + gr * (b - a);
    if (f(x1) < f(x2)) a = x1; else b = x2;
  }
  const double bmax = 0.5 * (a + b);
  if (f(bmax) < tphi) return false;
  double lo = mu, hi = bmax;
  for (int it = 0; it < 200; ++it) { const double m = 0.5 * (lo + hi); if (f(m) < tphi) lo = m; else hi = m; }
  const double be = 0.5 * (lo + hi), sb = std::sin(be), cb = std::cos(be);
  const double Mn = M * sb;
  const double pr = 1.0 + 2.0 * g / (g + 1.0) * (Mn * Mn - 1.0);
  const double rr = (g + 1.0) * Mn * Mn / ((g - 1.0) * Mn * Mn + 2.0);
  const double ut = u1 * cb, un2 = u1 * sb / rr;
  post[0] = p.fs[0] * rr;
  post[1] = ut * cb + un2 * sb;
  post[2] = -ut * sb + un2 * cb;
  post[3] = p.fs[3];
  post[4] = T1 * pr / rr;
  post[5] = visc_host(p, post[4]);
  post[6] = p.gamma * p.Rgas / (p.gamma - 1.0) * post[4] + 0.5 * (post[1] * post[1] + post[2] * post[2] + post[3] * post[3]);
  return true;
}

// TMA descriptor of one primitive-state buffer: tensor (x, y, z, field), box = one tile plane with its halo.
// cuTensorMapEncodeTiled is fetched through the runtime (no link-time dependency on libcuda).
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
bool make_box_map(CUtensorMap* tm, double* base, int nx, int ny, int nz, int nf, int bx, int by, int bf) {
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
      qres != cudaDriverEntryPointSuccess)
    return false;
  const cuuint64_t dims[4] = {(cuuint64_t)nx, (cuuint64_t)ny, (cuuint64_t)nz, (cuuint64_t)nf};
  const cuuint64_t strides[3] = {(cuuint64_t)nx * 8, (cuuint64_t)nx * ny * 8, (cuuint64_t)nx * ny * nz * 8};
  const cuuint32_t box[4] = {(cuuint32_t)bx, (cuuint32_t)by, 1u, (cuuint32_t)bf};
  const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
  const CUresult r = ((EncodeTiledFn)fn)(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, base, dims, strides, box, estr,
                                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                         CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

struct Carve { size_t off = 0; size_t take(size_t bytes) { size_t o = off; off += up(bytes); return o; } };

struct Layout { size_t w[2], S[2], theta, nflag, fbits, lmask, list, ilist, dFbuf, dFb, partial, inflow, speeds, sc, total; int npartial; dim3 grid; int lz; size_t istride; int zpad; };

Layout make_layout(const streams_grid& g, const streams_params& p) {
  Layout L;
  const size_t N = (size_t)g.nx * g.ny * g.nz;
  Carve c;
  // a BC_HALO z face stores three ghost planes below AND above each state buffer (the neighbouring slab's planes)
  L.zpad = (p.bc[4] == STREAMS_BC_HALO || p.bc[5] == STREAMS_BC_HALO) ? HALO : 0;
  const size_t NS = (size_t)g.nx * g.ny * (g.nz + 2 * L.zpad);
  for (int i = 0; i < 2; ++i) L.w[i] = c.take(NQ * NS * sizeof(double));
  for (int i = 0; i < 2; ++i) L.S[i] = c.take(5 * N * sizeof(double));
  L.theta = L.nflag = L.fbits = L.lmask = L.list = L.ilist = L.dFbuf = L.dFb = 0;
  if (p.weno_enable) {
    L.nflag = c.take(N);
    L.fbits = c.take((size_t)g.ny * (g.nz + 2 * L.zpad) * ((g.nx + 31) / 32) * sizeof(unsigned int));
    L.lmask = c.take(N);
    L.list = c.take(N * sizeof(unsigned int));
    L.istride = N + std::max({(size_t)g.ny * g.nz, (size_t)g.nx * g.nz, (size_t)g.nx * g.ny});
    L.ilist = c.take(3 * L.istride * sizeof(unsigned int));
    L.dFbuf = c.take(15 * N * sizeof(double));
    L.dFb = c.take(5 * ((size_t)g.ny * g.nz + (size_t)g.nx * g.nz + (size_t)g.nx * g.ny) * sizeof(double));
  }
  const int tiles_x = (g.nx + TX - 1) / TX, tiles_y = (g.ny + TY - 1) / TY;
  const int tiles = tiles_x * tiles_y;
  // planes per CTA.  Grids with at least half a wave of tiles (148 SMs, one CTA each): a launch takes about
  //   (tiles c / 148) (nz / c + G) + kappa (nz / c + G),   c chunks of nz / c planes, G ~ the cost of a chunk's 6 ghost planes,
  // the second term being the tail: CTAs differ (a wall tile takes twice the time of an interior one) and the last ones
  // run on a partly empty GPU.  Minimum at c = sqrt(kappa 148 nz / (G tiles)); kappa / G = 0.43 fits the measured optima
  // (sweep of c on one box: config 3 / 6 (128 tiles, nz 128) c = 8: -6 % per step against c = 3; config 4 (1024 tiles,
  // nz 128) c = 2 ... 3: -3 % against c = 1; config 5 (2048 tiles, nz 512) c = 4 as before), chunks of at most LZ_MAX and
  // at least 8 planes.  CTAs at different z also spread the DRAM traffic better than one wave marching in lockstep.
  // Smaller grids cannot fill the SMs with tiles: there the chunk count minimises  waves x (lz + 3.5)  (ghost planes
  // cost ~40 % of a full one; config 2: one wave of 128 CTAs beats every finer cut).
  int nchunk;
  if (tiles >= 74) {
    nchunk = (int)std::lround(std::sqrt(0.43 * 148.0 * g.nz / tiles));
    nchunk = std::max(nchunk, (g.nz + LZ_MAX - 1) / LZ_MAX);
    nchunk = std::min(nchunk, std::max(1, g.nz / 8));
  } else {
    nchunk = 1;
    double best = 1e300;
    for (int c = (g.nz + LZ_MAX - 1) / LZ_MAX; c <= g.nz; ++c) {
      const int lz = (g.nz + c - 1) / c;
      const int cc = (g.nz + lz - 1) / lz;
      const double cost = std::ceil((double)tiles * cc / 148.0) * (lz + 3.5);
      if (cost < best) { best = cost; nchunk = cc; }
      if (lz == 1) break;
    }
  }
  // z-slabs: at least four chunks where the slab allows it, so that the chunks between the two boundary chunks (which
  // need no ghost plane) can run while the halo exchange is in flight (Fig. 8)
  if (L.zpad) nchunk = std::max(nchunk, std::min(4, std::max(1, g.nz / 8)));
  L.lz = (g.nz + nchunk - 1) / nchunk;
  nchunk = (g.nz + L.lz - 1) / L.lz;
  L.grid = dim3(tiles_x, tiles_y, nchunk);
  L.npartial = std::max(tiles * nchunk, NDIAG * RGRID);
  L.partial = c.take((size_t)L.npartial * sizeof(double));
  L.inflow = c.take((size_t)NQ * (g.nz + 2 * L.zpad) * g.ny * sizeof(double));
  L.speeds = c.take(8 * sizeof(double));
  L.sc = c.take(sizeof(DevScal));        // device scalars in caller memory: the caller may run collectives on streams_reduce_ptr
  L.total = c.off;
  return L;
}

// the instantiations of the fused kernel: mode (0 residual only, 1 fused RK stage, 2 fused stage with lazy forcing),
// hybrid switch, RK stage.  Lazy forcing never runs with the hybrid switch; residual-only launches have no stage.
typedef void (*RhsKernel)(const DevP, const RhsArgs, const RhsMaps);
RhsKernel rhs_kernel(int mode, bool weno, int stage) {
  if (mode == 0) return stage != 0 ? nullptr : (weno ? (RhsKernel)k_rhs<0, true, 0> : (RhsKernel)k_rhs<0, false, 0>);
  if (mode == 2) {
    if (weno) return nullptr;
    return stage == 0 ? (RhsKernel)k_rhs<2, false, 0> : (stage == 1 ? (RhsKernel)k_rhs<2, false, 1> : (RhsKernel)k_rhs<2, false, 2>);
  }
  if (weno) return stage == 0 ? (RhsKernel)k_rhs<1, true, 0> : (stage == 1 ? (RhsKernel)k_rhs<1, true, 1> : (RhsKernel)k_rhs<1, true, 2>);
  return stage == 0 ? (RhsKernel)k_rhs<1, false, 0> : (stage == 1 ? (RhsKernel)k_rhs<1, false, 1> : (RhsKernel)k_rhs<1, false, 2>);
}

int rgrid_for(long long N) { return (int)std::min<long long>(RGRID, (N + RT - 1) / RT); }

}  // namespace

extern "C" {

size_t streams_workspace_bytes(const streams_grid* g, const streams_params* p) {
  if (!g || !p || validate(g, p)) return 0;
  return make_layout(*g, *p).total;
}

const char* streams_last_error(const streams_ctx* c) { return c ? c->err : g_err; }

long long streams_launch_count(const streams_ctx* c) { return c ? c->launches : 0; }

int streams_fp64_peak(void* cuda_stream, double* h_tinstr) {
  if (!h_tinstr) return fail(nullptr, STREAMS_EINVAL, "null argument");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return cuda_fail(nullptr, e, "streams_fp64_peak: no CUDA device");
  double* d_out = nullptr;
  cudaEvent_t e0, e1;
  if ((e = cudaMalloc(&d_out, sizeof(double))) != cudaSuccess) return cuda_fail(nullptr, e, "cudaMalloc");
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int grid = 2 * sms, iters = 4096;
  double best = 0.0;
  for (int rep = 0; rep < 4; ++rep) {                 // first pass warms up; best of the next three
    cudaEventRecord(e0, st);
    k_fp64_peak<<<grid, 1024, 0, st>>>(d_out, iters, 0.999999, 1e-9);
    cudaEventRecord(e1, st);
    e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) break;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double n = (double)grid * 1024.0 * iters * 64.0;
    if (rep > 0 && ms > 0.f) best = std::max(best, n / (ms * 1e-3) / 1e12);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d_out);
  if (e != cudaSuccess) return cuda_fail(nullptr, e, "k_fp64_peak");
  *h_tinstr = best;
  return STREAMS_OK;
}

void streams_destroy(streams_ctx* c) {
  if (!c) return;
  DevGuard dg(c->device);
  cudaStreamSynchronize(c->st);
  for (int k = 0; k < 8; ++k) if (c->gexec[k]) cudaGraphExecDestroy(c->gexec[k]);
  if (c->h_sc) cudaFreeHost(c->h_sc);
  if (c->h_part) cudaFreeHost(c->h_part);
  if (c->small_dev) cudaFree(c->small_dev);
  if (c->prof_ev) { for (cudaEvent_t e : *c->prof_ev) cudaEventDestroy(e); delete c->prof_ev; }
  delete c;
}

int streams_profile(streams_ctx* c, int enable) {
  if (!c) return fail(c, STREAMS_EINVAL, "null argument");
  DevGuard dg(c->device);
  if (enable && !c->prof_ev) {
    c->prof_ev = new std::vector<cudaEvent_t>(2 * 4096);
    for (cudaEvent_t& e : *c->prof_ev) CK(cudaEventCreate(&e));
  }
  if (enable) c->prof_n = 0;
  c->prof_on = enable ? 1 : 0;
  return STREAMS_OK;
}

int streams_profile_read(streams_ctx* c, double* ms_total, long long* launches) {
  if (!c || !ms_total || !launches) return fail(c, STREAMS_EINVAL, "null argument");
  DevGuard dg(c->device);
  CK(cudaStreamSynchronize(c->st));
  double tot = 0.0;
  for (int i = 0; i < c->prof_n; ++i) {
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, (*c->prof_ev)[2 * i], (*c->prof_ev)[2 * i + 1]));
    tot += ms;
  }
  *ms_total = tot; *launches = c->prof_n;
  return STREAMS_OK;
}

int streams_create(const streams_grid* g, const double* hx, const double* hy, const double* hz, const streams_params* p,
                   void* d_workspace, size_t workspace_bytes, void* cuda_stream, streams_ctx** out) {
  streams_ctx* c = nullptr;
  if (!g || !hx || !hy || !hz || !p || !out) return fail(nullptr, STREAMS_EINVAL, "null argument");
  if (const char* m = validate(g, p)) return fail(nullptr, STREAMS_EINVAL, m);
  const Layout L = make_layout(*g, *p);
  if (!d_workspace || workspace_bytes < L.total) return fail(nullptr, STREAMS_ENOMEM, "workspace too small");
  if (((size_t)d_workspace) % ALIGN) return fail(nullptr, STREAMS_ENOMEM, "workspace must be 256-byte aligned");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return fail(nullptr, STREAMS_ECUDA, "no CUDA device: this library has no CPU path");

  c = new (std::nothrow) streams_ctx();
  if (!c) return fail(nullptr, STREAMS_ENOMEM, "host allocation failed");
  std::memset(c, 0, sizeof *c);
  snprintf(c->err, sizeof c->err, "no error");
  c->g = *g; c->p = *p;
  c->st = (cudaStream_t)cuda_stream;
  if (cudaGetDevice(&c->device) != cudaSuccess) { delete c; return fail(nullptr, STREAMS_ECUDA, "cudaGetDevice failed"); }
  // stream capture is not allowed on the legacy default stream: graphs need a stream of the caller's own
  c->graph_ok = (c->st != nullptr && c->st != cudaStreamLegacy && c->st != cudaStreamPerThread) ? 1 : 0;
  char* base = (char*)d_workspace;
  c->zpad = L.zpad;
  const size_t zoff = (size_t)L.zpad * g->nx * g->ny;      // qbuf points at the first INTERIOR plane
  for (int i = 0; i < 2; ++i) { c->qbuf[i] = (double*)(base + L.w[i]) + zoff; c->S[i] = (double*)(base + L.S[i]); }
  if (p->weno_enable) {
    c->theta = nullptr; c->nflag = (unsigned char*)(base + L.nflag);
    c->fbits = (unsigned int*)(base + L.fbits) + (size_t)L.zpad * g->ny * ((g->nx + 31) / 32); c->lmask = (unsigned char*)(base + L.lmask); c->list = (unsigned int*)(base + L.list);
    c->ilist = (unsigned int*)(base + L.ilist); c->dFbuf = (double*)(base + L.dFbuf); c->dFb = (double*)(base + L.dFb);
  }
  c->partial = (double*)(base + L.partial); c->inflow = (double*)(base + L.inflow) + (size_t)L.zpad * g->ny; c->speeds = (double*)(base + L.speeds);
  c->npartial = L.npartial; c->rhs_grid = L.grid; c->lz = L.lz; c->istride = L.istride;
  c->sc = (DevScal*)(base + L.sc);
  c->stage_next = -1;

  // ---- S1 ghost coordinates and S2 metrics (host, O(n)) ----
  const int n[3] = {g->nx, g->ny, g->nz};
  // h_z of a slab: [3 ghost coordinates if bc[zmin] == HALO][nz nodes][3 ghost coordinates if bc[zmax] == HALO]
  const double* hz_lo = p->bc[4] == STREAMS_BC_HALO ? hz : nullptr;
  const double* hz_in = hz + (hz_lo ? HALO : 0);
  const double* hz_hi = p->bc[5] == STREAMS_BC_HALO ? hz_in + g->nz : nullptr;
  const double* xin[3] = {hx, hy, hz_in};
  Coef K;
  coeffs(p->order, K);
  std::vector<double> ih[3], gh[3], hh[3], xg0;
  double voltot_dir[3];
  for (int d = 0; d < 3; ++d) {
    for (int i = 1; i < n[d]; ++i)
      if (!(xin[d][i] > xin[d][i - 1])) { delete c; return fail(nullptr, STREAMS_EINVAL, "coordinates must be strictly increasing"); }
    std::vector<double> xc(n[d] + 2 * HALO);
    for (int i = 0; i < n[d]; ++i) xc[i + HALO] = xin[d][i];
    for (int l = 1; l <= HALO; ++l)
      for (int s = 0; s < 2; ++s) {
        const int gi = s == 0 ? -l : n[d] - 1 + l;
        const int bc = p->bc[2 * d + s];
        double v;
        if (bc == STREAMS_BC_HALO) {
          v = s == 0 ? hz_lo[HALO - l] : hz_hi[l - 1];       // the neighbouring slab's node coordinates
          if (s == 0 ? !(v < xin[d][0]) : !(v > xin[d][n[d] - 1])) { delete c; return fail(nullptr, STREAMS_EINVAL, "HALO ghost coordinates must continue the z nodes monotonically"); }
        } else if (bc == STREAMS_BC_PERIODIC) {
          int r = gi % n[d]; if (r < 0) r += n[d];
          v = xin[d][r] + (double)((gi - r) / n[d]) * g->len[d];
        } else if (bc == STREAMS_BC_WALL_ISO_STAGGERED) {
          v = 2.0 * p->y_wall[s] - xin[d][s == 0 ? l - 1 : n[d] - l];
        } else {
          v = 2.0 * xin[d][s == 0 ? 0 : n[d] - 1] - xin[d][s == 0 ? l : n[d] - 1 - l];
        }
        xc[gi + HALO] = v;
      }
    ih[d].resize(n[d]); gh[d].resize(n[d]); hh[d].resize(n[d]);
    double tot = 0.0;
    for (int i = 0; i < n[d]; ++i) {
      double h = 0.0, gg = 0.0;
      for (int l = 1; l <= 3; ++l) {
        h += K.a[l - 1] * (xc[i + HALO + l] - xc[i + HALO - l]);
        gg += K.b[l - 1] * ((xc[i + HALO + l] - xc[i + HALO]) - (xc[i + HALO] - xc[i + HALO - l]));
      }
      if (!(h > 0.0)) { delete c; return fail(nullptr, STREAMS_EINVAL, "non-positive metric"); }
      hh[d][i] = h; ih[d][i] = 1.0 / h; gh[d][i] = -gg / (h * h * h);
      tot += h;
    }
    voltot_dir[d] = tot;
    if (d == 0) xg0 = xc;
  }
  // total volume: sum over nodes of hx hy hz, summed the same way a serial loop would (used only as a divisor)
  double voltot = 0.0;
  for (int k = 0; k < n[2]; ++k)
    for (int j = 0; j < n[1]; ++j) voltot += voltot_dir[0] * hh[1][j] * hh[2][k];

  // ---- device parameter block ----
  DevP& P = c->P;
  P.nx = n[0]; P.ny = n[1]; P.nz = n[2]; P.nxy = n[0] * n[1]; P.N = (long long)n[0] * n[1] * n[2];
  P.zpad = L.zpad; P.QS = (long long)n[0] * n[1] * (n[2] + 2 * L.zpad); P.IS = n[1] * (n[2] + 2 * L.zpad);
  for (int i = 0; i < 6; ++i) P.bc[i] = p->bc[i];
  P.visc_model = p->visc_model; P.weno = p->weno_enable; P.forcing = p->forcing; P.viscous = p->viscous_enable; P.L = p->order / 2;
  P.gam = p->gamma; P.gm1 = p->gamma - 1.0; P.Rgas = p->Rgas; P.inv_R = 1.0 / p->Rgas;
  P.cp = p->gamma * p->Rgas / (p->gamma - 1.0); P.cv = p->Rgas / (p->gamma - 1.0); P.inv_cv = 1.0 / P.cv; P.cp_over_Pr = P.cp / p->Pr;
  P.mu_ref = p->mu_ref; P.T_ref = p->T_ref; P.inv_Tref = 1.0 / p->T_ref; P.visc_exp = p->visc_exp; P.suth_S = p->suth_S;
  P.th_thr = p->sensor_threshold; P.th_eps = p->sensor_eps;
  P.Twall[0] = p->T_wall[0]; P.Twall[1] = p->T_wall[1];
  P.mu_wall[0] = visc_host(*p, p->T_wall[0]); P.mu_wall[1] = visc_host(*p, p->T_wall[1]);
  for (int i = 0; i < 3; ++i) { K.qa[i] = 0.25 * K.a[i]; K.aR[i] = K.a[i] * p->Rgas; }
  K.sb2 = 2.0 * (K.b[0] + K.b[1] + K.b[2]);
  P.c = K;
  for (int i = 0; i < 5; ++i) P.fs[i] = p->fs[i];
  P.fs[5] = visc_host(*p, p->fs[4]);
  P.fs[6] = P.cp * p->fs[4] + 0.5 * (p->fs[1] * p->fs[1] + p->fs[2] * p->fs[2] + p->fs[3] * p->fs[3]);
  for (int i = 0; i < NQ; ++i) P.post[i] = P.fs[i];
  std::vector<unsigned char> xpost(n[0] + 2 * HALO, 0);
  if (p->bc[3] == STREAMS_BC_SHOCKGEN) {
    if (!shock_post_state(*p, P.post)) { delete c; return fail(nullptr, STREAMS_EINVAL, "shock generator: no attached weak shock for these parameters"); }
    for (int i = 0; i < n[0] + 2 * HALO; ++i) xpost[i] = xg0[i] < p->x_shock ? 0 : 1;   // sharp jump (A15)
  }

  // ---- small device arrays ----
  size_t off = 0, o_arr[9], o_xpost, o_stat;
  for (int a = 0; a < 9; ++a) { o_arr[a] = off; off += up((size_t)n[a % 3] * sizeof(double)); }
  o_xpost = off; off += up(xpost.size());
  o_stat = off; off += up(((size_t)(STAT_ZC + 1) * NSTAT * n[1] + 1) * sizeof(double));
  cudaError_t e = cudaMalloc(&c->small_dev, off);
  if (e != cudaSuccess) { delete c; return cuda_fail(nullptr, e, "cudaMalloc(metrics)"); }
  char* sb = (char*)c->small_dev;
  std::vector<double>* src[9] = {&ih[0], &ih[1], &ih[2], &gh[0], &gh[1], &gh[2], &hh[0], &hh[1], &hh[2]};
  for (int a = 0; a < 9; ++a) {
    e = cudaMemcpyAsync(sb + o_arr[a], src[a]->data(), src[a]->size() * sizeof(double), cudaMemcpyHostToDevice, c->st);
    if (e != cudaSuccess) { cudaFree(c->small_dev); delete c; return cuda_fail(nullptr, e, "cudaMemcpy(metrics)"); }
  }
  for (int d = 0; d < 3; ++d) { P.ih[d] = (const double*)(sb + o_arr[d]); P.gh[d] = (const double*)(sb + o_arr[3 + d]); P.hh[d] = (const double*)(sb + o_arr[6 + d]); }
  cudaMemcpyAsync(sb + o_xpost, xpost.data(), xpost.size(), cudaMemcpyHostToDevice, c->st);
  P.xpost = (const unsigned char*)(sb + o_xpost);
  P.inflow = c->inflow;
  c->stat_partial = (double*)(sb + o_stat);
  c->stat_sum = c->stat_partial + (size_t)STAT_ZC * NSTAT * n[1];
  c->stat_n = (unsigned long long*)(c->stat_sum + (size_t)NSTAT * n[1]);
  cudaMemsetAsync(c->stat_sum, 0, ((size_t)NSTAT * n[1] + 1) * sizeof(double), c->st);
  DevScal hs;
  std::memset(&hs, 0, sizeof hs);
  hs.vol_total = voltot;
  hs.dt = p->dt_fixed > 0.0 ? p->dt_fixed : 0.0;
  cudaMemcpyAsync(c->sc, &hs, sizeof hs, cudaMemcpyHostToDevice, c->st);
  e = cudaStreamSynchronize(c->st);     // host vectors go out of scope
  if (e != cudaSuccess) { cudaFree(c->small_dev); delete c; return cuda_fail(nullptr, e, "create sync"); }

  // TMA needs 16-byte global strides: rows of an even number of doubles.  Odd nx takes the by-index fill.
  c->use_tma = (n[0] % 2 == 0) ? 1 : 0;
  if (c->use_tma)
    for (int i = 0; i < 2; ++i)
      if (!make_box_map(&c->tmap[i], c->qbuf[i] - zoff, n[0], n[1], n[2] + 2 * L.zpad, NQ, PITCH, PY, NQ) ||
          !make_box_map(&c->tmap_own[i], c->qbuf[i] - zoff, n[0], n[1], n[2] + 2 * L.zpad, NQ, TX, TY, NQ)) {
        cudaFree(c->small_dev); delete c;
        return fail(nullptr, STREAMS_ECUDA, "cuTensorMapEncodeTiled failed");
      }
  e = cudaMallocHost((void**)&c->h_sc, sizeof(DevScal));
  if (e == cudaSuccess) e = cudaMallocHost((void**)&c->h_part, ((size_t)NDIAG * RGRID + 8) * sizeof(double));
  if (e != cudaSuccess) { cudaFree(c->small_dev); delete c; return cuda_fail(nullptr, e, "cudaMallocHost(diagnostics)"); }
  e = cudaSuccess;
  for (int m = 0; m < 3 && e == cudaSuccess; ++m)
    for (int w = 0; w < 2 && e == cudaSuccess; ++w)
      for (int st = 0; st < 3 && e == cudaSuccess; ++st)
        if (RhsKernel k = rhs_kernel(m, w != 0, st))
          e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, SM_RHS_DOUBLES * (int)sizeof(double));
  if (e != cudaSuccess) { cudaFree(c->small_dev); delete c; return cuda_fail(nullptr, e, "cudaFuncSetAttribute(k_rhs)"); }
  *out = c;
  return STREAMS_OK;
}

// conservative state in d_w (device) -> primitives in qbuf[0]; captures the frozen inflow plane
static int after_set_state(streams_ctx* c, const double* d_w) {
  c->cur = 0;
  k_cons2prim<<<rgrid_for(c->P.N), RT, 0, c->st>>>(c->P, d_w, c->qbuf[0]);
  LAUNCH_CHECK("k_cons2prim");
  c->inflow_pending = 0;
  if (c->p.bc[0] == STREAMS_BC_INFLOW_FROZEN) {
    // a z-slab freezes its ghost planes of the inflow as well: they arrive with the first halo swap (ensure_inflow)
    if (c->zpad) c->inflow_pending = 1;
    else { k_capture_inflow<<<64, 256, 0, c->st>>>(c->P, c->qbuf[0], c->inflow); LAUNCH_CHECK("k_capture_inflow"); }
  }
  // keep vol_total: reset the other scalars one by one
  CK(cudaMemsetAsync(&c->sc->force, 0, sizeof(double), c->st));
  CK(cudaMemsetAsync(&c->sc->time, 0, sizeof(double), c->st));
  if (!(c->p.dt_fixed > 0.0)) CK(cudaMemsetAsync(&c->sc->dt, 0, sizeof(double), c->st));
  c->has_state = 1; c->step = 0; c->scur = 0; c->dt_ready = 0; c->stage_next = -1; c->stage_half = 0; c->parts_done = 0; c->mid_done = 0;
  return STREAMS_OK;
}

int streams_set_state(streams_ctx* c, const double* d_w) {
  if (!c || !d_w) return fail(c, STREAMS_EINVAL, "null argument");
  DevGuard dg(c->device);
  return after_set_state(c, d_w);
}
int streams_set_state_host(streams_ctx* c, const double* h_w) {
  if (!c || !h_w) return fail(c, STREAMS_EINVAL, "null argument");
  DevGuard dg(c->device);
  // the RK register S[1] is free between steps: it stages the conservative vector
  CK(cudaMemcpyAsync(c->S[1], h_w, 5 * (size_t)c->P.N * sizeof(double), cudaMemcpyHostToDevice, c->st));
  const int rc = after_set_state(c, c->S[1]);
  if (rc) return rc;
  CK(cudaStreamSynchronize(c->st));
  return STREAMS_OK;
}
int streams_get_state(streams_ctx* c, double* d_w) {
  if (!c || !d_w) return fail(c, STREAMS_EINVAL, "null argument");
  DevGuard dg(c->device);
  if (!c->has_state) return fail(c, STREAMS_ESTATE, "no state set");
  k_prim2cons<<<rgrid_for(c->P.N), RT, 0, c->st>>>(c->P, c->qbuf[c->cur], d_w);
  LAUNCH_CHECK("k_prim2cons");
  return STREAMS_OK;
}
int streams_get_state_host(streams_ctx* c, double* h_w) {
  if (!c || !h_w) return fail(c, STREAMS_EINVAL, "null argument");
  DevGuard dg(c->device);
  if (!c->has_state) return fail(c, STREAMS_ESTATE, "no state set");
  k_prim2cons<<<rgrid_for(c->P.N), RT, 0, c->st>>>(c->P, c->qbuf[c->cur], c->S[1]);
  LAUNCH_CHECK("k_prim2cons");
  CK(cudaMemcpyAsync(h_w, c->S[1], 5 * (size_t)c->P.N * sizeof(double), cudaMemcpyDeviceToHost, c->st));
  CK(cudaStreamSynchronize(c->st));
  return STREAMS_OK;
}

// grid of the one-thread-per-flag-word list kernel
static int wgrid_for(const streams_ctx* c) {
  const long long words = (long long)c->P.ny * c->P.nz * ((c->P.nx + 31) / 32);
  return (int)std::min<long long>(RGRID, (words + RT - 1) / RT);
}

// sensor + list of nodes with flagged interfaces for the state in `w`
static int run_sensor(streams_ctx* c, const double* w, double* theta_out, unsigned char* iflags_out, bool build_list) {
  CK(cudaMemsetAsync(&c->sc->max_theta, 0, sizeof(double) + 3 * sizeof(unsigned long long) + 2 * sizeof(unsigned int), c->st));
  const int rg = rgrid_for(c->P.N);
  k_sensor<<<rg, RT, 0, c->st>>>(c->P, w, c->nflag, theta_out, c->sc);
  LAUNCH_CHECK("k_sensor");
  k_flag_pack<<<rg, RT, 0, c->st>>>(c->P, c->nflag, c->fbits);
  LAUNCH_CHECK("k_flag_pack");
  k_weno_list<<<wgrid_for(c), RT, 0, c->st>>>(c->P, c->fbits, build_list ? c->list : nullptr, c->lmask, nullptr, 0, iflags_out, c->sc);
  LAUNCH_CHECK("k_weno_list");
  return STREAMS_OK;
}

// z-slab with a frozen inflow: capture the inflow plane (ghost planes included) the first time the state is used after
// set_state -- the caller has swapped the halos of the initial state by then (include/streams.h)
static int ensure_inflow(streams_ctx* c) {
  if (!c->inflow_pending) return STREAMS_OK;
  k_capture_inflow<<<64, 256, 0, c->st>>>(c->P, c->qbuf[c->cur], c->inflow);
  LAUNCH_CHECK("k_capture_inflow");
  c->inflow_pending = 0;
  return STREAMS_OK;
}

// lists of flagged interfaces and of the nodes next to them from the flag words k_rhs has just written (a3); on a z-slab
// the caller has swapped the words of the three planes next to each BC_HALO face in between (streams_flag_halo_*)
static int run_list(streams_ctx* c) {
  CK(cudaMemsetAsync(&c->sc->max_theta, 0, sizeof(double) + 3 * sizeof(unsigned long long) + 2 * sizeof(unsigned int), c->st));
  CK(cudaMemsetAsync(&c->sc->icount[0], 0, 4 * sizeof(unsigned int), c->st));
  k_weno_list<<<wgrid_for(c), RT, 0, c->st>>>(c->P, c->fbits, c->list, c->lmask, c->ilist, c->istride, nullptr, c->sc);
  LAUNCH_CHECK("k_weno_list");
  return STREAMS_OK;
}

// a5: lists from the flags of the last k_rhs, dF once per flagged interface, then the listed nodes take
// R += dR and (q_new != NULL) the advanced state takes dt beta dR
static int run_weno(streams_ctx* c, const double* w, double* R, double* q_new, double beta) {
  int rc;
  if ((rc = run_list(c))) return rc;
  // 3 CTAs of 128 threads per SM (168 registers, no spills, 12 warps): config 4, ms per RK3 step with 2 / 3 / 4 CTAs per SM:
  // 18.33 / 16.30 / 16.56 (4 CTAs = 128 registers with 120 B of spills; before the plain-load path of weno_delta 4 was as good)
  if (c->p.weno_order == 3) {      // third-order variant (include/streams.h, weno_order): same lists, same launch shape
    k_weno_flux<0, 3, 3><<<148 * 3, 128, 0, c->st>>>(c->P, w, c->ilist, c->istride, c->sc, c->dFbuf, c->dFb);
    LAUNCH_CHECK("k_weno_flux<0,3>");
    k_weno_flux<1, 3, 3><<<148 * 3, 128, 0, c->st>>>(c->P, w, c->ilist, c->istride, c->sc, c->dFbuf, c->dFb);
    LAUNCH_CHECK("k_weno_flux<1,3>");
    k_weno_flux<2, 3, 3><<<148 * 3, 128, 0, c->st>>>(c->P, w, c->ilist, c->istride, c->sc, c->dFbuf, c->dFb);
    LAUNCH_CHECK("k_weno_flux<2,3>");
  } else {
    k_weno_flux<0, 3, 5><<<148 * 3, 128, 0, c->st>>>(c->P, w, c->ilist, c->istride, c->sc, c->dFbuf, c->dFb);
    LAUNCH_CHECK("k_weno_flux<0>");
    k_weno_flux<1, 3, 5><<<148 * 3, 128, 0, c->st>>>(c->P, w, c->ilist, c->istride, c->sc, c->dFbuf, c->dFb);
    LAUNCH_CHECK("k_weno_flux<1>");
    k_weno_flux<2, 3, 5><<<148 * 3, 128, 0, c->st>>>(c->P, w, c->ilist, c->istride, c->sc, c->dFbuf, c->dFb);
    LAUNCH_CHECK("k_weno_flux<2>");
  }
  k_weno_apply<<<rgrid_for(c->P.N), RT, 0, c->st>>>(c->P, w, c->list, c->lmask, c->sc, c->dFbuf, c->dFb, R, q_new, beta);
  LAUNCH_CHECK("k_weno_apply");
  return STREAMS_OK;
}

static int launch_rhs(streams_ctx* c, int mode, const RhsArgs& A_in, dim3 grid) {
  RhsArgs A = A_in;
  A.use_tma = c->use_tma;
  A.fbits = c->p.weno_enable ? c->fbits : nullptr;
  const int qi = A.q == c->qbuf[1] ? 1 : 0;
  RhsMaps tm;
  tm.tile = c->tmap[qi]; tm.own = c->tmap_own[qi];
  const size_t smem = SM_RHS_DOUBLES * sizeof(double);
  const bool rec = c->prof_on && c->prof_n < 4096;
  if (rec) CK(cudaEventRecord((*c->prof_ev)[2 * c->prof_n], c->st));
  // instantiation: mode, hybrid switch (the kernel writes the flag words), RK stage (0: alpha = 0, no R_prev; 2: R not stored)
  const int stage = mode == 0 ? 0 : (A.alpha == 0.0 ? 0 : (A.write_S ? 1 : 2));
  rhs_kernel(mode, A.fbits != nullptr, stage)<<<grid, NT, smem, c->st>>>(c->P, A, tm);
  LAUNCH_CHECK("k_rhs");
  if (rec) { CK(cudaEventRecord((*c->prof_ev)[2 * c->prof_n + 1], c->st)); c->prof_n++; }
  return STREAMS_OK;
}

static int force_from_partials(streams_ctx* c, const double* R, bool have_rhs_partials, bool take) {
  int n = (int)(c->rhs_grid.x * c->rhs_grid.y * c->rhs_grid.z);
  if (!have_rhs_partials) {
    n = rgrid_for(c->P.N);
    k_force_partial<<<n, RT, 0, c->st>>>(c->P, R, c->partial);
    LAUNCH_CHECK("k_force_partial");
  }
  k_force_final<<<1, RT, 0, c->st>>>(c->partial, n, c->sc, take ? 1 : 0);
  LAUNCH_CHECK("k_force_final");
  return STREAMS_OK;
}

int streams_rhs(streams_ctx* c, double* d_rhs) {
  if (!c || !d_rhs) return fail(c, STREAMS_EINVAL, "null argument");
  DevGuard dg(c->device);
  if (!c->has_state) return fail(c, STREAMS_ESTATE, "no state set");
  if (c->zpad && c->p.weno_enable) return fail(c, STREAMS_EINVAL, "streams_rhs on a z-slab with the hybrid switch: the flag words are swapped between the staged calls");
  if (c->zpad && c->p.forcing) return fail(c, STREAMS_EINVAL, "streams_rhs on a z-slab with forcing: the body force is a sum over all slabs, combined between the staged calls");
  const double* w = c->qbuf[c->cur];
  int rc;
  if ((rc = ensure_inflow(c))) return rc;
  RhsArgs A;
  std::memset(&A, 0, sizeof A);
  A.q = w; A.out_rhs = d_rhs; A.lz = c->lz; A.cz0 = 0; A.czs = 1;
  const bool partial_ok = c->p.forcing && !c->p.weno_enable;
  A.partial = partial_ok ? c->partial : nullptr;
  if ((rc = launch_rhs(c, 0, A, c->rhs_grid))) return rc;
  if (c->p.weno_enable) {
    if ((rc = run_weno(c, w, d_rhs, nullptr, 0.0))) return rc;
  }
  if (c->p.forcing) {
    if ((rc = force_from_partials(c, d_rhs, partial_ok, true))) return rc;
    k_apply_force<<<rgrid_for(c->P.N), RT, 0, c->st>>>(c->P, w, d_rhs, c->sc);
    LAUNCH_CHECK("k_apply_force");
  }
  return STREAMS_OK;
}

int streams_sensor(streams_ctx* c, double* d_theta, unsigned char* d_flags) {
  if (!c) return fail(c, STREAMS_EINVAL, "null argument");
  DevGuard dg(c->device);
  if (!c->has_state) return fail(c, STREAMS_ESTATE, "no state set");
  if (!c->p.weno_enable) return fail(c, STREAMS_EINVAL, "streams_sensor needs weno_enable = 1");
  if (int rc = ensure_inflow(c)) return rc;
  return run_sensor(c, c->qbuf[c->cur], d_theta, d_flags, false);
}

// host state that decides which kernels one RK3 step launches and on which buffers
static int step_key(const streams_ctx* c) { return c->cur | (c->scur << 1) | (c->dt_ready << 2); }

static const double RK_ALPHA[3] = {0.0, -17.0 / 60.0, -5.0 / 12.0};   // Eq. 11 with the sign of reading G5
static const double RK_BETA[3] = {8.0 / 15.0, 5.0 / 12.0, 3.0 / 4.0};
enum { PART_ALL = 0, PART_INTERIOR = 1, PART_BOUNDARY = 2 };

// S10, first half: the CFL maximum of the current state into sc->red[2] (already there after a lazy-forcing step)
static int do_step_begin(streams_ctx* c) {
  if (c->p.dt_fixed > 0.0 || c->dt_ready) return STREAMS_OK;
  const int rg = rgrid_for(c->P.N);
  k_speed_partial<<<rg, RT, 0, c->st>>>(c->P, c->qbuf[c->cur], c->partial);
  LAUNCH_CHECK("k_speed_partial");
  k_dt_final<<<1, RT, 0, c->st>>>(c->partial, rg, c->sc, nullptr, 1);
  LAUNCH_CHECK("k_dt_final");
  return STREAMS_OK;
}

// chunks of the fused kernel launched by one part: whole grid, the chunks between the first and the last one (they read
// no ghost plane of a z face), or the first and the last chunk
static bool part_chunks(const streams_ctx* c, int part, RhsArgs& A, dim3& grid) {
  const int nch = (int)c->rhs_grid.z;
  grid = c->rhs_grid;
  A.cz0 = 0; A.czs = 1;
  if (part == PART_INTERIOR) { if (nch < 3) return false; A.cz0 = 1; grid.z = nch - 2; }
  if (part == PART_BOUNDARY) { A.czs = std::max(1, nch - 1); grid.z = std::min(2, nch); }
  return true;
}

// first half of RK stage l (Eq. 11): dt (l = 0), the fused residual + stage kernel, and the partial body-force sums
// into sc->red[0..1].  part: PART_ALL, or PART_INTERIOR then PART_BOUNDARY (the reductions follow the boundary part).
static int do_stage_rhs(streams_ctx* c, int l, int part, bool single) {
  int rc;
  const bool first = part != PART_BOUNDARY, last = part != PART_INTERIOR;
  if (first && (rc = ensure_inflow(c))) return rc;
  if (l == 0 && first && !(c->p.dt_fixed > 0.0)) {
    k_take_dt<<<1, 1, 0, c->st>>>(c->sc, c->p.cfl);
    LAUNCH_CHECK("k_take_dt");
    c->dt_ready = 0;
  }
  double* w = c->qbuf[c->cur];
  RhsArgs A;
  std::memset(&A, 0, sizeof A);
  A.q = w; A.lz = c->lz; A.alpha = RK_ALPHA[l]; A.beta = RK_BETA[l]; A.dt_ptr = &c->sc->dt;
  dim3 grid;
  const bool any = part_chunks(c, part, A, grid);
  if (c->p.forcing && !c->p.weno_enable) {
    // lazy forcing: the fused kernel advances with alpha (R_prev + f_prev ...) + beta R and sums R_rhou; once f is
    // known a light kernel adds dt beta f (e_rhou + u e_rhoE).  S[0] keeps R without the forcing terms.
    A.q_out = c->qbuf[c->cur ^ 1]; A.S_prev = c->S[0]; A.S_out = c->S[0]; A.partial = c->partial;
    A.f_prev = l > 0 ? &c->sc->force : nullptr;
    A.write_S = l < 2 ? 1 : 0;
    if (any && (rc = launch_rhs(c, 2, A, grid))) return rc;
    if (last && (rc = force_from_partials(c, nullptr, true, single))) return rc;
  } else if (c->p.forcing) {
    // forcing with the hybrid switch: R -> S[scur^1]; WENO, f and the update kernel follow in do_stage_end
    const bool partial_ok = !c->p.weno_enable;
    A.out_rhs = c->S[c->scur ^ 1]; A.partial = partial_ok ? c->partial : nullptr;
    if (any && (rc = launch_rhs(c, 0, A, grid))) return rc;
  } else {
    // fused: w_new = w + dt (alpha S + beta R) written to the other state buffer, S updated in place
    // R of the last stage is never read (alpha_0 = 0): neither this kernel nor k_weno_apply stores it
    A.q_out = c->qbuf[c->cur ^ 1]; A.S_prev = c->S[0]; A.S_out = c->S[0]; A.write_S = l < 2 ? 1 : 0;
    if (any && (rc = launch_rhs(c, 1, A, grid))) return rc;
  }
  return STREAMS_OK;
}

// forcing with the hybrid switch, between the halves: the body force needs the sum of the CORRECTED R, and on z-slabs the
// correction needs the neighbours' flag words, which the caller swaps after do_stage_rhs: WENO correction of R, then the
// partial sums into red[0..1] (not taken: the caller combines them across the slabs before do_stage_end)
static int do_stage_mid(streams_ctx* c) {
  if (!(c->p.forcing && c->p.weno_enable)) return STREAMS_OK;
  int rc;
  double* Sc = c->S[c->scur ^ 1];
  if ((rc = run_weno(c, c->qbuf[c->cur], Sc, nullptr, 0.0))) return rc;
  if ((rc = force_from_partials(c, Sc, false, false))) return rc;
  c->mid_done = 1;
  return STREAMS_OK;
}

// second half of RK stage l: f = -red[0] / red[1] (combined across z-slabs by the caller), the forcing fix, the WENO
// correction; after the last stage the CFL maximum of the new state and the time
static int do_stage_end(streams_ctx* c, int l, bool single) {
  const int rg = rgrid_for(c->P.N);
  int rc;
  double* w = c->qbuf[c->cur];
  if (c->p.forcing && !c->p.weno_enable) {
    double* wn = c->qbuf[c->cur ^ 1];
    if (!single) { k_force_take<<<1, 1, 0, c->st>>>(c->sc); LAUNCH_CHECK("k_force_take"); }
    const bool want_dt = l == 2 && !(c->p.dt_fixed > 0.0);
    k_force_fix<<<rg, RT, 0, c->st>>>(c->P, wn, w, c->sc, RK_BETA[l], want_dt ? c->partial : nullptr);
    LAUNCH_CHECK("k_force_fix");
    if (want_dt) {
      k_dt_final<<<1, RT, 0, c->st>>>(c->partial, rg, c->sc, nullptr, 1);
      LAUNCH_CHECK("k_dt_final");
      c->dt_ready = 1;
    }
    c->cur ^= 1;
  } else if (c->p.forcing) {
    double* Sp = c->S[c->scur];
    double* Sc = c->S[c->scur ^ 1];
    if (c->mid_done) {
      // streams_stage_mid has corrected R and left its sums in red[0..1]; the caller has combined them across the slabs
      k_force_take<<<1, 1, 0, c->st>>>(c->sc);
      LAUNCH_CHECK("k_force_take");
    } else {
      if (c->p.weno_enable && (rc = run_weno(c, w, Sc, nullptr, 0.0))) return rc;
      if ((rc = force_from_partials(c, Sc, !c->p.weno_enable, true))) return rc;
    }
    k_update<<<rg, RT, 0, c->st>>>(c->P, w, Sp, Sc, c->sc, RK_ALPHA[l], RK_BETA[l], 1, l < 2 ? 1 : 0);
    LAUNCH_CHECK("k_update");
    c->scur ^= 1;
  } else {
    if (c->p.weno_enable && (rc = run_weno(c, w, l < 2 ? c->S[0] : nullptr, c->qbuf[c->cur ^ 1], RK_BETA[l]))) return rc;
    c->cur ^= 1;
  }
  if (l == 2) {
    k_advance_time<<<1, 1, 0, c->st>>>(c->sc);
    LAUNCH_CHECK("k_advance_time");
  }
  return STREAMS_OK;
}

// enqueue ONE RK3 step (Eq. 11) on the context stream and advance the host-side state (buffers, dt_ready)
static int step_once(streams_ctx* c) {
  int rc;
  if ((rc = do_step_begin(c))) return rc;
  for (int l = 0; l < 3; ++l) {
    if ((rc = do_stage_rhs(c, l, PART_ALL, true))) return rc;
    if ((rc = do_stage_end(c, l, true))) return rc;
  }
  return STREAMS_OK;
}

// Small grids are launch-bound (config 1: 27 launches of a few microseconds per step): one RK3 step is captured into
// a CUDA graph per host-state key and replayed.  Grids of >= GRAPH_MAX_POINTS launch directly (nothing to gain).
constexpr long long GRAPH_MAX_POINTS = 1LL << 24;

int streams_step(streams_ctx* c, int nsteps) {
  if (!c || nsteps < 0) return fail(c, STREAMS_EINVAL, "bad argument");
  DevGuard dg(c->device);
  if (!c->has_state) return fail(c, STREAMS_ESTATE, "no state set");
  if (c->zpad) return fail(c, STREAMS_EINVAL, "a z-slab (BC_HALO) advances by the staged calls: its ghost planes are exchanged between stages");
  if (c->stage_next >= 0) return fail(c, STREAMS_ESTATE, "a staged step is open (streams_step_begin without the third streams_stage_end)");
  int rc;
  for (int s = 0; s < nsteps; ++s) {
    const bool graph = c->graph_ok && !c->prof_on && c->P.N < GRAPH_MAX_POINTS;
    if (!graph) {
      if ((rc = step_once(c))) return rc;
      c->step++;
      continue;
    }
    const int key = step_key(c);
    if (!c->gexec[key]) {
      // capture: the launches of step_once are recorded, not run; the host state it leaves is what a replay leaves
      const int cur0 = c->cur, scur0 = c->scur, dtr0 = c->dt_ready;
      const long long l0 = c->launches;
      cudaGraph_t gph = nullptr;
      cudaError_t e = cudaStreamBeginCapture(c->st, cudaStreamCaptureModeThreadLocal);
      if (e != cudaSuccess) { c->graph_ok = 0; cudaGetLastError(); --s; continue; }
      rc = step_once(c);
      e = cudaStreamEndCapture(c->st, &gph);
      const int after = step_key(c);
      const int nl = (int)(c->launches - l0);
      c->cur = cur0; c->scur = scur0; c->dt_ready = dtr0; c->launches = l0;
      if (rc || e != cudaSuccess || !gph) { if (gph) cudaGraphDestroy(gph); c->graph_ok = 0; cudaGetLastError(); --s; continue; }
      e = cudaGraphInstantiate(&c->gexec[key], gph, 0);
      cudaGraphDestroy(gph);
      if (e != cudaSuccess) { c->gexec[key] = nullptr; c->graph_ok = 0; cudaGetLastError(); --s; continue; }
      c->g_after[key] = after; c->g_launches[key] = nl;
    }
    CK(cudaGraphLaunch(c->gexec[key], c->st));
    const int after = c->g_after[key];
    c->cur = after & 1; c->scur = (after >> 1) & 1; c->dt_ready = (after >> 2) & 1;
    c->launches += c->g_launches[key];
    c->step++;
  }
  return STREAMS_OK;
}

// ---- staged stepping and z-slab halos ----------------------------------------------------

int streams_step_begin(streams_ctx* c) {
  if (!c) return fail(c, STREAMS_EINVAL, "null argument");
  DevGuard dg(c->device);
  if (!c->has_state) return fail(c, STREAMS_ESTATE, "no state set");
  if (c->stage_next >= 0) return fail(c, STREAMS_ESTATE, "streams_step_begin: the previous staged step is not finished");
  const int rc = do_step_begin(c);
  if (rc) return rc;
  c->stage_next = 0; c->stage_half = 0; c->parts_done = 0; c->mid_done = 0;
  return STREAMS_OK;
}

int streams_stage_rhs(streams_ctx* c, int stage, int part) {
  if (!c || part < PART_ALL || part > PART_BOUNDARY) return fail(c, STREAMS_EINVAL, "bad argument");
  DevGuard dg(c->device);
  if (c->stage_next != stage || c->stage_half != 0) return fail(c, STREAMS_ESTATE, "streams_stage_rhs out of order (step_begin, then rhs / end of stages 0, 1, 2)");
  if (part == PART_ALL && c->parts_done) return fail(c, STREAMS_ESTATE, "streams_stage_rhs: PART_ALL after a partial launch");
  if (part == PART_INTERIOR && c->parts_done) return fail(c, STREAMS_ESTATE, "streams_stage_rhs: the interior part comes first, once");
  if (part == PART_BOUNDARY && (c->parts_done & 2)) return fail(c, STREAMS_ESTATE, "streams_stage_rhs: boundary part launched twice");
  int rc;
  if (part == PART_BOUNDARY && !(c->parts_done & 1)) {
    // no interior launch was asked for: the boundary part then stands for the whole grid
    part = PART_ALL;
  }
  if ((rc = do_stage_rhs(c, stage, part, false))) return rc;
  if (part == PART_INTERIOR) c->parts_done = 1;
  else { c->parts_done = 3; c->stage_half = 1; }
  return STREAMS_OK;
}

int streams_stage_mid(streams_ctx* c, int stage) {
  if (!c) return fail(c, STREAMS_EINVAL, "null argument");
  DevGuard dg(c->device);
  if (c->stage_next != stage || c->stage_half != 1 || c->mid_done) return fail(c, STREAMS_ESTATE, "streams_stage_mid out of order (once, between streams_stage_rhs and streams_stage_end)");
  return do_stage_mid(c);
}

int streams_stage_end(streams_ctx* c, int stage) {
  if (!c) return fail(c, STREAMS_EINVAL, "null argument");
  DevGuard dg(c->device);
  if (c->stage_next != stage || c->stage_half != 1) return fail(c, STREAMS_ESTATE, "streams_stage_end out of order");
  if (c->zpad && c->p.forcing && c->p.weno_enable && !c->mid_done)
    return fail(c, STREAMS_ESTATE, "streams_stage_end: a z-slab with forcing and the hybrid switch needs streams_stage_mid first");
  const int rc = do_stage_end(c, stage, false);
  if (rc) return rc;
  c->stage_half = 0; c->parts_done = 0; c->mid_done = 0;
  if (stage == 2) { c->stage_next = -1; c->step++; } else c->stage_next = stage + 1;
  return STREAMS_OK;
}

double* streams_reduce_ptr(streams_ctx* c) { return c ? c->sc->red : nullptr; }

size_t streams_halo_bytes(const streams_ctx* c) { return c ? (size_t)NQ * HALO * c->P.nxy * sizeof(double) : 0; }

// the three planes next to a z face <-> a contiguous message [NQ][3][ny][nx] (seven copies of 3 nx ny doubles)
static int halo_copy(streams_ctx* c, int face, double* buf, void* stream, bool pack) {
  if (!c || !buf || (face != 4 && face != 5)) return fail(c, STREAMS_EINVAL, "bad argument (face: 4 = zmin, 5 = zmax)");
  DevGuard dg(c->device);
  if (!c->has_state) return fail(c, STREAMS_ESTATE, "no state set");
  if (!pack && c->p.bc[face] != STREAMS_BC_HALO) return fail(c, STREAMS_EINVAL, "streams_halo_unpack: this face is not BC_HALO");
  cudaStream_t st = stream ? (cudaStream_t)stream : c->st;
  const long long k = pack ? (face == 4 ? 0 : c->P.nz - HALO) : (face == 4 ? -HALO : c->P.nz);
  const size_t n = (size_t)HALO * c->P.nxy;
  double* q = c->qbuf[c->cur] + k * c->P.nxy;
  for (int f = 0; f < NQ; ++f) {
    if (pack) CK(cudaMemcpyAsync(buf + f * n, q + f * c->P.QS, n * sizeof(double), cudaMemcpyDeviceToDevice, st));
    else CK(cudaMemcpyAsync(q + f * c->P.QS, buf + f * n, n * sizeof(double), cudaMemcpyDeviceToDevice, st));
  }
  return STREAMS_OK;
}
// node-flag words (one bit per node) of the three planes next to a z face <-> a contiguous message [3][ny][ceil(nx/32)]
static int flag_halo_copy(streams_ctx* c, int face, unsigned int* buf, void* stream, bool pack) {
  if (!c || !buf || (face != 4 && face != 5)) return fail(c, STREAMS_EINVAL, "bad argument (face: 4 = zmin, 5 = zmax)");
  DevGuard dg(c->device);
  if (!c->p.weno_enable) return fail(c, STREAMS_EINVAL, "flag halos need weno_enable = 1");
  if (!pack && c->p.bc[face] != STREAMS_BC_HALO) return fail(c, STREAMS_EINVAL, "streams_flag_halo_unpack: this face is not BC_HALO");
  cudaStream_t st = stream ? (cudaStream_t)stream : c->st;
  const long long k = pack ? (face == 4 ? 0 : c->P.nz - HALO) : (face == 4 ? -HALO : c->P.nz);
  const size_t rowwords = (size_t)c->P.ny * ((c->P.nx + 31) / 32), n = HALO * rowwords;
  unsigned int* f = c->fbits + k * (long long)rowwords;
  if (pack) CK(cudaMemcpyAsync(buf, f, n * sizeof(unsigned int), cudaMemcpyDeviceToDevice, st));
  else CK(cudaMemcpyAsync(f, buf, n * sizeof(unsigned int), cudaMemcpyDeviceToDevice, st));
  return STREAMS_OK;
}
size_t streams_flag_halo_bytes(const streams_ctx* c) {
  return c && c->p.weno_enable ? (size_t)HALO * c->P.ny * ((c->P.nx + 31) / 32) * sizeof(unsigned int) : 0;
}
int streams_flag_halo_pack(streams_ctx* c, int face, unsigned int* d_buf, void* cuda_stream) { return flag_halo_copy(c, face, d_buf, cuda_stream, true); }
int streams_flag_halo_unpack(streams_ctx* c, int face, const unsigned int* d_buf, void* cuda_stream) {
  return flag_halo_copy(c, face, const_cast<unsigned int*>(d_buf), cuda_stream, false);
}
int streams_halo_pack(streams_ctx* c, int face, double* d_buf, void* cuda_stream) { return halo_copy(c, face, d_buf, cuda_stream, true); }
int streams_halo_unpack(streams_ctx* c, int face, const double* d_buf, void* cuda_stream) {
  return halo_copy(c, face, const_cast<double*>(d_buf), cuda_stream, false);
}

int streams_stats_accumulate(streams_ctx* c) {
  if (!c) return fail(c, STREAMS_EINVAL, "null argument");
  DevGuard dg(c->device);
  if (!c->has_state) return fail(c, STREAMS_ESTATE, "no state set");
  const int nzc = std::min(STAT_ZC, c->P.nz);
  k_stats_partial<<<dim3(c->P.ny, nzc), RT, 0, c->st>>>(c->P, c->qbuf[c->cur], nzc, c->stat_partial);
  LAUNCH_CHECK("k_stats_partial");
  k_stats_final<<<(NSTAT * c->P.ny + 127) / 128, 128, 0, c->st>>>(c->P, c->stat_partial, nzc, c->stat_sum, c->stat_n);
  LAUNCH_CHECK("k_stats_final");
  return STREAMS_OK;
}

int streams_stats_read(streams_ctx* c, double* h_out, long long* h_nsamples) {
  if (!c || !h_out) return fail(c, STREAMS_EINVAL, "null argument");
  DevGuard dg(c->device);
  const size_t n = (size_t)NSTAT * c->P.ny;
  std::vector<double> tmp(n + 1);
  CK(cudaMemcpyAsync(tmp.data(), c->stat_sum, (n + 1) * sizeof(double), cudaMemcpyDeviceToHost, c->st));
  CK(cudaStreamSynchronize(c->st));
  unsigned long long cnt;
  std::memcpy(&cnt, &tmp[n], sizeof cnt);
  const double inv = cnt > 0 ? 1.0 / (double)cnt : 0.0;
  for (size_t e = 0; e < n; ++e) h_out[e] = tmp[e] * inv;
  if (h_nsamples) *h_nsamples = (long long)cnt;
  return STREAMS_OK;
}

int streams_stats_reset(streams_ctx* c) {
  if (!c) return fail(c, STREAMS_EINVAL, "null argument");
  DevGuard dg(c->device);
  CK(cudaMemsetAsync(c->stat_sum, 0, ((size_t)NSTAT * c->P.ny + 1) * sizeof(double), c->st));
  return STREAMS_OK;
}

int streams_diagnostics(streams_ctx* c, streams_diag* out) {
  if (!c || !out) return fail(c, STREAMS_EINVAL, "null argument");
  DevGuard dg(c->device);
  if (!c->has_state) return fail(c, STREAMS_ESTATE, "no state set");
  std::memset(out, 0, sizeof *out);
  const int rg = rgrid_for(c->P.N);
  const double* w = c->qbuf[c->cur];
  int rc;
  if ((rc = ensure_inflow(c))) return rc;
  // sensor statistics of the current state (interface counts as the next RHS would see them)
  if (c->p.weno_enable && (rc = run_sensor(c, w, nullptr, nullptr, false))) return rc;
  DevScal& hs = *c->h_sc;
  CK(cudaMemcpyAsync(c->h_sc, c->sc, sizeof hs, cudaMemcpyDeviceToHost, c->st));
  k_speed_partial<<<rg, RT, 0, c->st>>>(c->P, w, c->partial);
  LAUNCH_CHECK("k_speed_partial");
  k_dt_final<<<1, RT, 0, c->st>>>(c->partial, rg, c->sc, c->speeds, 0);
  LAUNCH_CHECK("k_dt_final");
  double* sp = c->h_part + (size_t)NDIAG * RGRID;
  CK(cudaMemcpyAsync(sp, c->speeds, 3 * sizeof(double), cudaMemcpyDeviceToHost, c->st));
  k_diag_partial<<<rg, RT, 0, c->st>>>(c->P, w, c->partial);
  LAUNCH_CHECK("k_diag_partial");
  double* part = c->h_part;
  CK(cudaMemcpyAsync(part, c->partial, (size_t)NDIAG * rg * sizeof(double), cudaMemcpyDeviceToHost, c->st));
  CK(cudaStreamSynchronize(c->st));
  double s[7] = {0, 0, 0, 0, 0, 0, 0}, mnr = INFINITY, mnp = INFINITY, mxm = 0.0, bad = 0.0;
  for (int a = 0; a < 7; ++a) {
    // pairwise-free Neumaier sum over the CTA partials (fixed order)
    double sum = 0.0, comp = 0.0;
    for (int b = 0; b < rg; ++b) {
      const double x = part[(size_t)a * rg + b], t = sum + x;
      comp += std::fabs(sum) >= std::fabs(x) ? (sum - t) + x : (x - t) + sum;
      sum = t;
    }
    s[a] = sum + comp;
  }
  for (int b = 0; b < rg; ++b) {
    mnr = std::fmin(mnr, part[(size_t)7 * rg + b]); mnp = std::fmin(mnp, part[(size_t)8 * rg + b]);
    mxm = std::fmax(mxm, part[(size_t)9 * rg + b]); bad = std::fmax(bad, part[(size_t)10 * rg + b]);
  }
  out->step = c->step; out->time = hs.time; out->dt = hs.dt; out->forcing = hs.force;
  out->mass = s[0]; out->mom[0] = s[1]; out->mom[1] = s[2]; out->mom[2] = s[3]; out->energy = s[4]; out->kinetic = s[5];
  out->volume = s[6]; out->bulk_rhou = s[1] / s[6];
  out->min_rho = mnr; out->min_p = mnp; out->max_mach = mxm; out->max_theta = c->p.weno_enable ? hs.max_theta : 0.0;
  for (int d = 0; d < 3; ++d) out->max_speed[d] = sp[d];
  const long long n[3] = {c->P.nx, c->P.ny, c->P.nz};
  for (int d = 0; d < 3; ++d) {
    const bool per = c->p.bc[2 * d] == STREAMS_BC_PERIODIC;
    out->weno_ifaces[d] = c->p.weno_enable ? (long long)hs.weno_if[d] : 0;
    out->total_ifaces[d] = (per ? n[d] : n[d] + 1) * n[(d + 1) % 3] * n[(d + 2) % 3];
  }
  const bool nonfinite = bad > 0.0 || !std::isfinite(s[0]) || !std::isfinite(s[4]);
  out->nonfinite = nonfinite ? 1 : 0;
  if (nonfinite) return fail(c, STREAMS_ENONFINITE, "state is not physical (NaN/Inf, rho <= 0 or p <= 0)");
  return STREAMS_OK;
}

}  // extern "C"

// ---- S10 maxima without any allocation (include/streams.h, streams_max_speed_static) --------------------------------
// The scratch of this ONE entry point is a file-scope device array instead of caller workspace: per-CTA partial maxima
// [3][STATIC_MAX_CTAS] followed by a 256-byte line whose first word is the "CTAs finished" ticket.  Every device that
// loads the library holds the 98 560 bytes until exit; all calls on a device share it (overlapping calls race) and it
// keeps the last call's contents: the partials are overwritten before they are read, the ticket is zeroed before each
// launch.  In HOST code the array's name is a host-side stand-in, not a device address: static_scratch() resolves the
// address once per device with cudaGetSymbolAddress and the kernel takes it as an argument.
namespace {
constexpr int STATIC_CHUNK = RT * 32;           // nodes reduced by one CTA
constexpr int STATIC_MAX_CTAS = 4096;
constexpr int STATIC_WORDS = 3 * STATIC_MAX_CTAS + 32;
static_assert((long long)STATIC_CHUNK * STATIC_MAX_CTAS == STREAMS_STATIC_MAX_NODES, "streams.h states the limit");
constexpr int STATIC_MAX_DEV = 64;
}  // namespace

static __device__ __align__(256) double g_static_scratch[STATIC_WORDS];

namespace {
// one CTA = STATIC_CHUNK consecutive nodes of the conservative state; the last CTA to finish (ticket) reduces the
// partials and writes the three maxima.  The maximum is exact, so the result does not depend on the CTA order.
__global__ void __launch_bounds__(RT) k_speed_static(const __grid_constant__ DevP P, const double* __restrict__ w,
                                                     double* scratch, double* __restrict__ out) {
  __shared__ double sh[RT / 32];
  __shared__ int is_last;
  double m[3] = {0.0, 0.0, 0.0};
  const long long o0 = blockIdx.x * (long long)STATIC_CHUNK;
  const long long o1 = o0 + STATIC_CHUNK < P.N ? o0 + STATIC_CHUNK : P.N;
  for (long long o = o0 + threadIdx.x; o < o1; o += RT) {
    int i, j, k;
    node_ijk(P, o, i, j, k);
    Prim q;
    cons2prim(P, w[o], w[o + P.N], w[o + 2 * P.N], w[o + 3 * P.N], w[o + 4 * P.N], q);      // S3 (mu is not used)
    const double cs = sqrt(P.gam * P.Rgas * q.T);
    m[0] = fmax(m[0], (fabs(q.u) + cs) * P.ih[0][i]);
    m[1] = fmax(m[1], (fabs(q.v) + cs) * P.ih[1][j]);
    m[2] = fmax(m[2], (fabs(q.w) + cs) * P.ih[2][k]);
  }
  for (int d = 0; d < 3; ++d) {
    const double t = block_max<RT>(m[d], sh, threadIdx.x);
    if (threadIdx.x == 0) scratch[d * STATIC_MAX_CTAS + blockIdx.x] = t;
  }
  unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch + 3 * STATIC_MAX_CTAS);
  if (threadIdx.x == 0) {
    __threadfence();                                              // the partials are visible before the ticket moves
    is_last = atomicAdd(ticket, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!is_last) return;
  __threadfence();
  const volatile double* part = scratch;
  for (int d = 0; d < 3; ++d) {
    double mm = 0.0;
    for (int e = threadIdx.x; e < (int)gridDim.x; e += RT) mm = fmax(mm, part[d * STATIC_MAX_CTAS + e]);
    const double t = block_max<RT>(mm, sh, threadIdx.x);
    if (threadIdx.x == 0) out[d] = t;
  }
  if (threadIdx.x == 0) *ticket = 0u;                             // left at zero for the next call
}

// device address of g_static_scratch on `device` (current), resolved once per device
int static_scratch(streams_ctx* c, int device, double** ptr) {
  static double* addr[STATIC_MAX_DEV];
  static std::mutex mu;
  if (device < 0 || device >= STATIC_MAX_DEV) return fail(c, STREAMS_EINVAL, "streams_max_speed_static: device index beyond 63");
  std::lock_guard<std::mutex> lock(mu);
  if (!addr[device]) {
    double* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
    if (e != cudaSuccess || !p) return cuda_fail(c, e, "cudaGetSymbolAddress(g_static_scratch)");
    addr[device] = p;
  }
  *ptr = addr[device];
  return STREAMS_OK;
}
}  // namespace

extern "C" int streams_max_speed_static(streams_ctx* c, const double* d_w, double* d_speeds) {
  if (!c || !d_w || !d_speeds) return fail(c, STREAMS_EINVAL, "null argument");
  if (c->P.N > STREAMS_STATIC_MAX_NODES) {
    char b[200];
    snprintf(b, sizeof b, "streams_max_speed_static: %lld nodes exceeds the static scratch limit of %lld nodes (use streams_diagnostics)",
             (long long)c->P.N, (long long)STREAMS_STATIC_MAX_NODES);
    return fail(c, STREAMS_EINVAL, b);
  }
  DevGuard dg(c->device);
  double* scratch = nullptr;
  int rc;
  if ((rc = static_scratch(c, c->device, &scratch))) return rc;
  const int grid = (int)((c->P.N + STATIC_CHUNK - 1) / STATIC_CHUNK);
  CK(cudaMemsetAsync(scratch + 3 * STATIC_MAX_CTAS, 0, sizeof(unsigned int), c->st));
  k_speed_static<<<grid, RT, 0, c->st>>>(c->P, d_w, scratch, d_speeds);
  LAUNCH_CHECK("k_speed_static");
  return STREAMS_OK;
}
