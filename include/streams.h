/*
 * streams.h -- C-ABI boundary of the B200-native STREAmS hot path.
 *
 * The library evaluates the explicit right-hand side R(w) of the 3-D compressible
 * Navier-Stokes equations (Eq. 1-3) on a Cartesian grid that may be
 * stretched, and advances the conservative state w = [rho, rho u, rho v, rho w, rho E]
 * with the three-stage low-storage Runge-Kutta scheme of PAPER.md:89-99
 * (Eq. 10-11).  Everything between `streams_set_state` and `streams_get_state` runs in
 * hand-written fp64 CUDA kernels for sm_100a on ONE GPU; there is no CPU fallback.
 *
 * Conventions
 *  - Every call returns an int: STREAMS_OK (0) or a negative STREAMS_E* code.  No
 *    exception crosses the boundary.  `streams_last_error` gives a text for the last
 *    failure of a context (or of `streams_create` when ctx == NULL).
 *  - Pointers named d_* are DEVICE pointers, h_* are HOST pointers.  The library never
 *    takes ownership of a caller pointer.  All field arrays are fp64, layout
 *    [5][nz][ny][nx] (variable slowest, x fastest), NO ghost nodes stored.
 *  - The library does not allocate field-sized device memory.  The caller (PyTorch in
 *    this repository) allocates `streams_workspace_bytes()` bytes, 256-byte aligned,
 *    hands them to `streams_create`, and keeps them alive until `streams_destroy`.
 *    The context owns only O(nx+ny+nz) metric arrays and a few scalars on the device.
 *    Workspace: two states of 7 stored primitives (112 B/node), two RK registers
 *    (80 B/node), reduction partials; with weno_enable also the node flags, node and
 *    interface lists and the interface-flux scratch (about 146 B/node more).
 *  - All kernels are enqueued on the `cuda_stream` given at creation (a cudaStream_t
 *    passed as void*, NULL = legacy default stream).  Only `streams_diagnostics`,
 *    the *_host copies and `streams_destroy` synchronise that stream.
 *  - Index/ghost convention: nodes 0..n-1 per direction; ghost values (width 3) are
 *    never stored, they are evaluated by index arithmetic from the boundary kind
 *    (DESIGN.md "S1").
 */
#ifndef STREAMS_H
#define STREAMS_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct streams_ctx streams_ctx; /* opaque; created by streams_create, freed by streams_destroy */

/* error codes */
enum {
  STREAMS_OK = 0,
  STREAMS_EINVAL = -1,     /* bad argument or unsupported combination of parameters   */
  STREAMS_ECUDA = -2,      /* a CUDA runtime call or kernel launch failed             */
  STREAMS_ENOMEM = -3,     /* caller workspace too small / misaligned                  */
  STREAMS_ENONFINITE = -4, /* diagnostics saw NaN/Inf or rho <= 0 or p <= 0            */
  STREAMS_ESTATE = -5      /* call needs a state but streams_set_state was not called  */
};

/* boundary kinds, one per face: bc[0..5] = xmin, xmax, ymin, ymax, zmin, zmax */
enum {
  STREAMS_BC_PERIODIC = 0,           /* PAPER.md:110, 126 (homogeneous directions)            */
  STREAMS_BC_WALL_ISO_STAGGERED = 1, /* isothermal no-slip wall half-way between the first two
                                        nodes, convective flux zero there       */
  STREAMS_BC_WALL_ISO_NODE = 2,      /* isothermal no-slip wall on the boundary node */
  STREAMS_BC_INFLOW_FROZEN = 3,      /* Dirichlet ghost planes frozen at set_state (stands in for the
                                        digital-filter inflow of PAPER.md:126, A16) */
  STREAMS_BC_OUTFLOW_NR = 4,         /* characteristic non-reflecting boundary: xmax (outflow) or ymax (upper boundary) */
  STREAMS_BC_SHOCKGEN = 5,           /* inviscid oblique-shock state imposed in the ghosts of ymax
                                                                                 */
  STREAMS_BC_EXTRAP = 6,             /* zeroth-order extrapolation (1-D tube tests)            */
  STREAMS_BC_WALL_ISO_CHAR = 7,      /* ymin only: isothermal no-slip wall on the boundary node with the "similar
                                        characteristic wave treatment" of PAPER.md:126: the wall-normal convective
                                        derivative at the wall node in characteristic form, incoming acoustic wave =
                                        reflection of the outgoing one (A14b)        */
  STREAMS_BC_HALO = 8                /* zmin / zmax only: the face is an internal boundary of a domain decomposed into
                                        z-slabs ("ghost nodes ... are exchanged between neighbouring
                                        processes").  The three ghost planes beyond the face are STORED with the state and
                                        filled by streams_halo_unpack; the context advances by the staged calls below */
};

enum { STREAMS_VISC_POWER = 0, STREAMS_VISC_SUTHERLAND = 1 };

/* Grid: node counts and the domain length per direction (the period for periodic
 * directions; otherwise informational).  Node coordinates are passed to streams_create. */
typedef struct {
  int nx, ny, nz;
  int pad_;
  double len[3];
} streams_grid;

/* Gas, scheme, boundary and forcing parameters.  Plain data, copied at creation. */
typedef struct {
  double gamma;            /* ratio of specific heats (1.4)                                   */
  double Pr;               /* Prandtl number (0.72)                              */
  double Rgas;             /* gas constant in the caller's units: p = rho Rgas T              */
  double mu_ref, T_ref;    /* viscosity law reference values                                  */
  double visc_exp;         /* POWER:  mu = mu_ref (T/T_ref)^visc_exp                          */
  double suth_S;           /* SUTHERLAND: mu = mu_ref (T/T_ref)^1.5 (T_ref+S)/(T+S)           */
  double sensor_threshold; /* theta_th of the hybrid switch (Eq. 8)              */
  double sensor_eps;       /* (u0/L0)^2 regulariser of Eq. 8, must be > 0                     */
  double T_wall[2];        /* wall temperature for the ymin / ymax walls                      */
  double y_wall[2];        /* wall-plane coordinate for STAGGERED walls (ymin, ymax)          */
  double fs[5];            /* free-stream primitive state rho,u,v,w,T (SHOCKGEN)              */
  double shock_angle_deg;  /* flow deflection of the shock generator                          */
  double x_shock;          /* x at which the jump enters through the ymax ghosts              */
  double cfl;              /* Courant number for the on-device time step (S10)      */
  double dt_fixed;         /* > 0: use this time step instead of the CFL reduction            */
  int visc_model;          /* STREAMS_VISC_*                                                  */
  int order;               /* 2L: 2, 4 or 6 (6 = measured path)                               */
  int weno_enable;         /* 1: Ducros-switched WENO5 flux on flagged interfaces             */
  int forcing;             /* 1: constant bulk mass-flow forcing in x      */
  int viscous_enable;      /* 0: Euler equations (conservation / KE tests)                    */
  int bc[6];               /* STREAMS_BC_* for xmin,xmax,ymin,ymax,zmin,zmax                   */
  int weno_order;          /* order of the WENO reconstruction on flagged interfaces (PAPER.md:77-79 names none): 5 =
                            * Jiang-Shu WENO5 (default, the measured path; 0 means 5) or 3 (variant, A23: nodes
                            * i-1..i+2, also for the Lax-Friedrichs maximum); the flag rule (six nodes) does not change */
} streams_params;

/* Reductions over the current state (and the last RHS evaluation). */
typedef struct {
  long long step;          /* completed RK3 steps                                             */
  double time, dt, forcing;/* physical time, last time step, last body force f                */
  double mass, mom[3], energy, kinetic; /* sum over nodes of q * vol, vol = h_x h_y h_z       */
  double volume;           /* sum of vol                                                      */
  double bulk_rhou;        /* mom[0] / volume                                                 */
  double min_rho, min_p, max_mach, max_theta;
  double max_speed[3];     /* max over nodes of (|u_d| + c) / h_d                             */
  long long weno_ifaces[3], total_ifaces[3]; /* flagged / total interfaces of the last RHS   */
  int nonfinite;           /* 1 if NaN/Inf, rho<=0 or p<=0 was seen                           */
  int pad_;
} streams_diag;

/* Bytes of device workspace `streams_create` needs for this grid/params (0 on bad input).
 * Passage: PAPER.md:183-225 (section 4.2: the state array w_gpu and the RK increment array fln_gpu live in
 * device memory for the whole time loop); here the caller owns that memory. */
size_t streams_workspace_bytes(const streams_grid* grid, const streams_params* params);

/* Create a context for one Cartesian grid, stretched or uniform per direction (PAPER.md:110 error-function /
 * PAPER.md:124 hyperbolic-sine wall-normal mappings are the caller's: the library takes node coordinates and forms
 * the metrics of Eq. 5 generalised to non-uniform spacing, S2), gas model (Eq. 2-3),
 * scheme order, boundary kinds and forcing.
 * h_x/h_y/h_z: HOST arrays of nx/ny/nz node coordinates, strictly
 * increasing.  A z face of kind BC_HALO adds the three node coordinates of the neighbouring slab on that side: h_z then
 * holds [3 ghost coordinates if bc[zmin] == HALO][nz nodes][3 ghost coordinates if bc[zmax] == HALO], increasing.  d_workspace: DEVICE memory, >= streams_workspace_bytes(), 256-B aligned,
 * owned by the caller.  cuda_stream: cudaStream_t as void*.  On success *out is set. */
int streams_create(const streams_grid* grid, const double* h_x, const double* h_y, const double* h_z,
                   const streams_params* params, void* d_workspace, size_t workspace_bytes,
                   void* cuda_stream, streams_ctx** out);

/* Copy a state w = [rho, rho u, rho v, rho w, rho E] (Eq. 10) into the context: the paper's
 * `w_gpu = w`.  Device->device, async; converts to the stored primitives.  Captures the frozen inflow
 * plane when bc[xmin] == INFLOW_FROZEN.  Resets step counter, time and RK register. */
int streams_set_state(streams_ctx* ctx, const double* d_w);
/* Same from pageable or pinned HOST memory (host->device copy on the context stream; synchronises). */
int streams_set_state_host(streams_ctx* ctx, const double* h_w);

/* Copy the current conservative state w out: the paper's `w = w_gpu`.  Device->device, async. */
int streams_get_state(streams_ctx* ctx, double* d_w_out);
/* Same into HOST memory (synchronises). */
int streams_get_state_host(streams_ctx* ctx, double* h_w_out);

/* The residual vector R(w) of Eq. 10: convective terms by the energy-preserving central flux of
 * Eq. 5-7 or, on interfaces flagged by the sensor of Eq. 8, the characteristic
 * Lax-Friedrichs WENO flux; viscous terms in the Laplacian form of Eq. 9.
 * R of the current state goes into d_rhs_out ([5][nz][ny][nx]); includes the body force
 * (forcing=1) and the characteristic replacement at OUTFLOW_NR nodes, excludes the
 * Dirichlet node overrides of NODE walls.  State, time and step counter unchanged. */
int streams_rhs(streams_ctx* ctx, double* d_rhs_out);

/* Node flags of the shock sensor for the current state: d_theta_out[nz][ny][nx] fp64
 * (may be NULL) receives theta of Eq. 8; d_flags_out[3][nz][ny][nx] bytes (may be NULL)
 * receives 1 where interface i+1/2 (resp. j+1/2, k+1/2) above node (i,j,k) is flagged. */
int streams_sensor(streams_ctx* ctx, double* d_theta_out, unsigned char* d_flags_out);

/* Advance nsteps full steps of Wray's three-stage scheme, Eq. 11 (alpha_1 = -17/60, G5);
 * dt recomputed on the device every step unless dt_fixed > 0 (S10); the body force is re-evaluated at every
 * stage.  No host synchronisation.  On a stream of the caller's own (not the legacy default
 * stream) grids below 2^24 nodes replay one captured CUDA graph per step instead of launching kernel by kernel. */
int streams_step(streams_ctx* ctx, int nsteps);

/* ---- Staged stepping and z-slab halos: the domain decomposition of PAPER.md:168 and the overlapped ghost-node swap of
 * PAPER.md:229-237 (section 4.3, Fig. 8), restricted to slabs along z (one slab per context / GPU; the caller moves the
 * messages: NCCL, MPI or a device-to-device copy).  One RK3 step of Eq. 11 is
 *     streams_step_begin                        local CFL maximum -> red[2]          [caller: MAX of red[2] over the slabs]
 *     for stage = 0, 1, 2:
 *         [caller: exchange the halos of the current state: pack / send / receive / unpack]
 *         streams_stage_rhs(stage, part)        fused residual + stage kernel; body-force sums -> red[0], red[1]
 *                                               [caller: SUM of red[0..1] over the slabs (forcing = 1 only)]
 *         streams_stage_end(stage)              f = -red[0] / red[1], forcing fix, WENO correction, (stage 2) time += dt
 * and gives bit for bit the state of streams_step when there is one slab (no BC_HALO face) and nothing is combined.
 * `part`: STREAMS_PART_ALL launches the whole grid.  For overlap, STREAMS_PART_INTERIOR launches the z-chunks that read
 * no ghost plane (possibly none on a thin slab) and may run while the halos are in flight; STREAMS_PART_BOUNDARY then
 * launches the first and the last chunk and the reductions.  Calls out of this order return STREAMS_ESTATE.
 * streams_step refuses a context with a BC_HALO face.  All calls are asynchronous on the context stream.
 * forcing = 1 TOGETHER WITH weno_enable = 1: the body force is the sum of the residual AFTER its WENO correction
 * (PAPER.md:57, 77-79), and on a slab that correction needs the neighbours' flag words.  The stage is then
 *         streams_stage_rhs | [caller: swap the flag words] | streams_stage_mid(stage): WENO correction of R, sums ->
 *         red[0], red[1] | [caller: SUM of red[0..1]] | streams_stage_end(stage): f, Eq. 11.
 * streams_stage_mid is optional on a context without a BC_HALO face (streams_stage_end then does its work) and does
 * nothing for other parameter combinations; at most once per stage, else STREAMS_ESTATE. */
enum { STREAMS_PART_ALL = 0, STREAMS_PART_INTERIOR = 1, STREAMS_PART_BOUNDARY = 2 };
int streams_step_begin(streams_ctx* ctx);
int streams_stage_rhs(streams_ctx* ctx, int stage, int part);
int streams_stage_mid(streams_ctx* ctx, int stage);
int streams_stage_end(streams_ctx* ctx, int stage);

/* DEVICE pointer (inside the caller's workspace, valid for the life of the context) to four doubles:
 *   red[0] = sum over the context's nodes of R_rhou vol, red[1] = sum of vol   (S9),
 *   red[2] = max over nodes and directions of (|u_d| + c) / h_d                (S10), red[3] unused.
 * The caller combines them across slabs in place (sum, sum, max) on the context stream between the staged calls. */
double* streams_reduce_ptr(streams_ctx* ctx);

/* Ghost-plane messages of the CURRENT state (the swap of the ghost nodes).  A message is the three planes
 * next to a z face as stored primitives, [7][3][ny][nx] fp64 = streams_halo_bytes() bytes (rho, u, v, w, T, mu, H: sending
 * mu and H as well saves the receiver a power law per ghost node and keeps slabs bit-identical to the undivided run).
 * streams_halo_pack copies the INTERIOR planes next to `face` (4 = zmin: planes 0..2, 5 = zmax: planes nz-3..nz-1) into
 * d_buf; streams_halo_unpack copies d_buf into the GHOST planes beyond `face` (which must be BC_HALO).  The message packed
 * at the zmax face of slab r is what slab r+1 unpacks at its zmin face, and vice versa.  Device-to-device, asynchronous on
 * `cuda_stream` (NULL = the context stream; another stream lets the swap overlap STREAMS_PART_INTERIOR, ordering between
 * the two streams is the caller's: events). */
size_t streams_halo_bytes(const streams_ctx* ctx);
int streams_halo_pack(streams_ctx* ctx, int face, double* d_buf, void* cuda_stream);
int streams_halo_unpack(streams_ctx* ctx, int face, const double* d_buf, void* cuda_stream);

/* The hybrid switch on z-slabs (weno_enable = 1): interface k+1/2 is flagged when any of the nodes
 * k-2 .. k+3 has theta > theta_th (S4), so the interfaces next to a slab face need the node flags of the
 * neighbour's three planes.  streams_stage_rhs leaves the node flags of the stage's state packed one bit per node; between
 * streams_stage_rhs and streams_stage_end the caller swaps the flag words of the three planes next to every BC_HALO face
 * the same way as the state halos: message [3][ny][ceil(nx/32)] 32-bit words = streams_flag_halo_bytes() bytes (0 when
 * the switch is off).  With a frozen inflow the slab captures the inflow plane (its ghost planes included) at the first
 * use of the state after streams_set_state, i.e. after the caller's first halo swap.  streams_rhs refuses a slab with the
 * hybrid switch (one call cannot contain the swap) and a slab with forcing (the body force is a sum over all slabs); streams_sensor and the interface counts of streams_diagnostics on a
 * slab use the ghost flag words of the last stage. */
size_t streams_flag_halo_bytes(const streams_ctx* ctx);
int streams_flag_halo_pack(streams_ctx* ctx, int face, unsigned int* d_buf, void* cuda_stream);
int streams_flag_halo_unpack(streams_ctx* ctx, int face, const unsigned int* d_buf, void* cuda_stream);

/* Reductions of the current state into *h_out (host struct): the volume integrals of PAPER.md:107 (bulk density
 * rho_b = 1/V int rho dV and bulk momentum, "both exactly constant in time"), total energy and kinetic energy
 * (PAPER.md:77), the last body force f, extrema and sensor statistics (Eq. 8).  Synchronises.  Returns
 * STREAMS_ENONFINITE (with *h_out filled) if the state is not physical. */
int streams_diagnostics(streams_ctx* ctx, streams_diag* h_out);

/* Reynolds / Favre statistics ("the overline symbol denotes averaging in the homogeneous space
 * directions and in time"; phi~ = mean(rho phi) / mean(rho)).  streams_stats_accumulate adds the x-z plane means
 * (plain node means: x and z are the homogeneous, uniformly spaced directions) of the current state to running sums
 * on the device, one profile over the wall-normal index j per quantity; async, no host synchronisation.
 * streams_stats_read returns the time average (sums / samples) into h_out[STREAMS_NSTAT][ny] (HOST) and the number
 * of samples; synchronises.  Order of the quantities:
 *   rho, u, v, w, p, T, mu, rho u, rho v, rho w, rho T, rho u u, rho v v, rho w w, rho u v, T T
 * e.g. Favre mean u~ = out[7]/out[0]; density-scaled stress rho u''u'' = out[11] - out[7]^2/out[0] (Fig. 3).
 * streams_stats_reset clears sums and sample count. */
enum { STREAMS_NSTAT = 16 };
int streams_stats_accumulate(streams_ctx* ctx);
int streams_stats_read(streams_ctx* ctx, double* h_out, long long* h_nsamples);
int streams_stats_reset(streams_ctx* ctx);

/* Kernel timing for roofline accounting.  streams_profile(ctx, 1) clears the record and makes
 * every following launch of the fused RHS kernel (k_rhs) be bracketed by CUDA events on the
 * context stream; streams_profile(ctx, 0) stops.  streams_profile_read synchronises and returns
 * the summed device time in ms and the number of k_rhs launches recorded (at most 4096). */
int streams_profile(streams_ctx* ctx, int enable);
int streams_profile_read(streams_ctx* ctx, double* h_ms_total, long long* h_launches);

/* Roofline denominator of an fp64-ALU-bound kernel: runs a register-only kernel of independent DFMA
 * chains (one CTA of 1024 threads x 2 per SM) on `cuda_stream` (may be NULL = default stream) and
 * returns in *h_tinstr the measured rate of fp64 lane-instructions in 1e12 per second (one DFMA of
 * one thread = one; multiply by 2 for flop/s).  Nominal: 148 SMs x 64 lanes x SM clock.  Synchronises.
 * Not part of the method (PAPER.md gives no peak); used by bench.py next to MEASURED_PEAKS.json. */
int streams_fp64_peak(void* cuda_stream, double* h_tinstr);

/* The S10 maxima (PAPER.md:89-99 is silent on the time step; north_star "CFL reduction", S10)
 * WITHOUT ANY ALLOCATION, for callers that cannot allocate (CUDA graph capture, serving loops): the maxima over the
 * nodes of (|u_d| + c) / h_d, d = x, y, z, of the conservative state d_w (device, [5][nz][ny][nx], caller-owned, read
 * only; any state of the context's grid, not necessarily the one set by streams_set_state) are written to d_speeds
 * (device, 3 doubles, caller-owned) by ONE kernel enqueued on the context stream (asynchronous); the time step of
 * S10 is cfl / max(d_speeds[0..2]).  Same numbers as streams_diagnostics().max_speed of that state.  The grid
 * metrics and gas constants are the context's; the per-CTA partial maxima and the "last CTA" ticket live in a
 * file-scope `static __device__` array of the library (98 560 bytes: 3 x 4096 doubles + a 256-byte ticket line; every
 * GPU that loads the library holds it until exit), NOT in the workspace.  Calls neither cudaMalloc / cudaFree nor any
 * allocating routine; the first call on a device resolves the array's device address (cudaGetSymbolAddress, no
 * allocation: make it once before a capture starts), later calls enqueue one 4-byte memset (the ticket must start at
 * zero) and the kernel.
 * Limit: one CTA reduces 8192 nodes and the array holds 4096 CTAs: grids of more than STREAMS_STATIC_MAX_NODES nodes
 * are rejected with STREAMS_EINVAL ("... exceeds the static scratch limit ...") before anything is enqueued.
 * Every call on a device, of every context, shares the one array: calls that OVERLAP on the GPU (different
 * streams, no ordering between them) race on it and return garbage; calls on one stream, or ordered by events, are safe.
 * STREAMS_EINVAL for null arguments; STREAMS_ECUDA for a CUDA failure. */
#define STREAMS_STATIC_MAX_NODES 33554432LL
int streams_max_speed_static(streams_ctx* ctx, const double* d_w, double* d_speeds);

/* Number of kernel launches enqueued by this context so far (for bench accounting). */
long long streams_launch_count(const streams_ctx* ctx);

/* Text of the last error (never NULL).  ctx may be NULL for streams_create failures. */
const char* streams_last_error(const streams_ctx* ctx);

void streams_destroy(streams_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* STREAMS_H */
