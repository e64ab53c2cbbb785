/*
 * streams_oracle.h -- TEST INFRASTRUCTURE, not the product.
 *
 * Plain, slow, fp64 CPU restatement of the STREAmS right-hand side and RK3 time advance,
 * written from /root/reference/PAPER.md (section 2, Eq. 1-11) and the readings listed in
 * DESIGN.md ("S0".."S11").  It shares no code, header, table or helper with the CUDA path
 * under paper_2004_02276_b200/csrc and include/streams.h; the structs below are its own.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
 * may load it.
 *
 * All pointers are HOST pointers; fields are fp64 [5][nz][ny][nx], x fastest.
 */
#ifndef STREAMS_ORACLE_H
#define STREAMS_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

enum { ORC_OK = 0, ORC_EINVAL = -1, ORC_ENONFINITE = -4, ORC_ESTATE = -5 };
enum { ORC_BC_PERIODIC = 0, ORC_BC_WALL_STAG = 1, ORC_BC_WALL_NODE = 2, ORC_BC_INFLOW = 3,
       ORC_BC_OUTFLOW = 4, ORC_BC_SHOCKGEN = 5, ORC_BC_EXTRAP = 6, ORC_BC_WALL_CHAR = 7 };
enum { ORC_VISC_POWER = 0, ORC_VISC_SUTHERLAND = 1 };
enum { ORC_NSTAT = 16 };   /* statistics per wall-normal index, see oracle_stats_accumulate */

typedef struct { int nx, ny, nz; int pad_; double len[3]; } oracle_grid;

typedef struct {
  double gamma, Pr, Rgas, mu_ref, T_ref, visc_exp, suth_S;
  double sensor_threshold, sensor_eps;
  double T_wall[2], y_wall[2], fs[5];
  double shock_angle_deg, x_shock, cfl, dt_fixed;
  int visc_model, order, weno_enable, forcing, viscous_enable;
  int bc[6];
  int weno_order; /* order of the WENO reconstruction on flagged interfaces: 5 (default; 0 means 5) or 3 (reading A23) */
} oracle_params;

typedef struct {
  long long step;
  double time, dt, forcing;
  double mass, mom[3], energy, kinetic, volume, bulk_rhou;
  double min_rho, min_p, max_mach, max_theta;
  double max_speed[3];
  long long weno_ifaces[3], total_ifaces[3];
  int nonfinite, pad_;
} oracle_diag;

typedef struct oracle_ctx oracle_ctx;

int  oracle_create(const oracle_grid*, const double* x, const double* y, const double* z,
                   const oracle_params*, oracle_ctx** out);
int  oracle_set_state(oracle_ctx*, const double* w);
int  oracle_get_state(oracle_ctx*, double* w_out);
int  oracle_rhs(oracle_ctx*, double* rhs_out);
int  oracle_step(oracle_ctx*, int nsteps);
int  oracle_diagnostics(oracle_ctx*, oracle_diag* out);
void oracle_destroy(oracle_ctx*);
int  oracle_threads(void);
/* Reynolds / Favre statistics: plane means over the homogeneous directions x, z, averaged over calls */
int  oracle_stats_accumulate(oracle_ctx*);
int  oracle_stats_read(oracle_ctx*, double* out /* [ORC_NSTAT][ny] */, long long* nsamples);
int  oracle_stats_reset(oracle_ctx*);

/* pieces exposed so that tests can pin them one by one */
int  oracle_coeffs(int order, double a_out[3], double b_out[3]);            /* a_l, b_l tables        */
double oracle_weno5(double a, double b, double c, double d, double e);      /* S6 step 6               */
double oracle_weno3(double a, double b, double c);                          /* A23: third-order variant */
void oracle_eigen(int d, double gamma, const double ubar[3], double Hbar,
                  double Lm[25], double Rm[25], double lam[5]);             /* S6 step 2 (row-major)   */
int  oracle_shock_state(const oracle_params*, double post_prim[5], double* beta_rad); /* S1 shock generator */
int  oracle_get_metrics(oracle_ctx*, int d, double* h_out, double* g_out);  /* S2                      */
int  oracle_get_sensor(oracle_ctx*, double* theta_out, unsigned char* flags_out); /* S4: theta[nz][ny][nx], flags[3][nz][ny][nx] */
int  oracle_get_prims(oracle_ctx*, double* prim_out);                       /* S3: [9][nz][ny][nx] rho,u,v,w,p,T,H,c,mu */
int  oracle_rhs_parts(oracle_ctx*, double* conv_out, double* visc_out);     /* convective / viscous split of R (no forcing) */
int  oracle_get_ghosted(oracle_ctx*, double* wg_out);                       /* S1: ghost-filled state [5][nz+6][ny+6][nx+6] */
void oracle_roe_state(double rho_a, const double u_a[3], double H_a, double rho_b, const double u_b[3], double H_b,
                      double ubar[3], double* Hbar);                        /* S6 step 1               */

#ifdef __cplusplus
}
#endif
#endif
