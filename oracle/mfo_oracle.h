/*
 * mfo_oracle.h — C ABI of the CPU ORACLE for the MUSTA-FORCE step of arXiv 1510.06340.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT. Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may load it. It shares no code with the
 * CUDA path (paper_1510_06340_b200/csrc) and neither includes the other.
 *
 * It mirrors the product boundary (include/mustaforce.h) with prefix mfo_ and host memory only,
 * so one harness can drive both.  All arrays are host pointers, nx*ny*nz doubles, x fastest:
 * idx = i + nx*(j + ny*k).  Enumerations carry the same numeric values as the product header
 * but are re-declared here on purpose (no shared header).
 *
 * Readings of the paper (A1..A17) are listed in DESIGN.md; each function cites PAPER.md lines.
 */
#ifndef MFO_ORACLE_H
#define MFO_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mfo_ctx mfo_ctx;

enum { MFO_EOS_CS2 = 0, MFO_EOS_TABLE = 1 };
enum { MFO_LIM_NONE = 0, MFO_LIM_MINMOD = 1, MFO_LIM_SUPERBEE = 2, MFO_LIM_VANALBADA = 3,
       MFO_LIM_VANLEER = 4, MFO_LIM_MC = 5, MFO_LIM_FIRST = 6 };
enum { MFO_BC_OUTFLOW = 0, MFO_BC_PERIODIC = 1 };
enum { MFO_OK = 0, MFO_EINVAL = -1, MFO_ENOMEM = -2, MFO_ESTATE = -4 };

mfo_ctx* mfo_create(int nx, int ny, int nz, double dx, int eos, int limiter, int k_stages);
void     mfo_destroy(mfo_ctx*);

int mfo_set_state(mfo_ctx*, const double* E, const double* Mx, const double* My, const double* Mz, const double* R);
int mfo_get_state(mfo_ctx*, double* E, double* Mx, double* My, double* Mz, double* R);
int mfo_set_state_prim(mfo_ctx*, const double* e, const double* vx, const double* vy, const double* vz, const double* n);
int mfo_get_state_prim(mfo_ctx*, double* e, double* vx, double* vy, double* vz, double* n);

int mfo_step(mfo_ctx*, int n, double cfl);      /* dt = cfl*dx/S_max from U^n, once per step   */
int mfo_step_dt(mfo_ctx*, int n, double dt);    /* fixed dt (paper Tables 1-3) */
int mfo_conserved_totals(mfo_ctx*, double out[5]);
int mfo_get_time(mfo_ctx*, double* t, double* last_dt, long long* steps);
int mfo_max_signal_speed(mfo_ctx*, double* smax);

int mfo_set_rk(mfo_ctx*, int order);
int mfo_set_boundary(mfo_ctx*, int bc);
int mfo_set_cs2(mfo_ctx*, double cs2);
int mfo_set_predictor(mfo_ctx*, int on);
/* 32: the stored state is single precision as in the paper's own code (reading A19) - the state handed in and the
 * result of every Runge-Kutta stage are rounded to float, arithmetic stays double.  64 (default): no rounding.  Rounds the current state. */
int mfo_set_state_precision(mfo_ctx*, int bits);
int mfo_set_alpha(mfo_ctx*, double alpha);
int mfo_set_jet_source(mfo_ctx*, double dEdx, double sigma, double x0, double y0, double z0);
/* tabulated EOS (context created with MFO_EOS_TABLE): ln p on a grid uniform in ln e (ne points) and in n (nn points, e fastest) */
int mfo_set_eos_table(mfo_ctx*, int ne, int nn, double ln_e0, double dln_e, double n0, double dn, const double* ln_p);
int mfo_eos(mfo_ctx*, double e, double n, double out[3]);   /* p, dp/de, dp/dn of the context's EOS */
int mfo_sync(mfo_ctx*);
const char* mfo_last_error(mfo_ctx*);

/* ---- pieces exposed so the pins can reach them one by one (tests only) ---- */
double mfo_slope(int limiter, double a, double b);                    /* Eq.14-21, two-argument form  */
int mfo_flux(mfo_ctx*, int d, const double U[5], double F[5]);        /* Eq.3 with Eq.23 inside       */
int mfo_con2prim(mfo_ctx*, const double U[5], double prim[5]);        /* Eq.23: (e,vx,vy,vz,n)        */
int mfo_prim2con(mfo_ctx*, const double prim[5], double U[5]);        /* Eq.4                          */
int mfo_musta_flux(mfo_ctx*, int d, double lam, const double UL[5], const double UR[5], double F[5]); /* Eq.8-11 */
int mfo_eval_L(mfo_ctx*, double dt, double* L_E, double* L_Mx, double* L_My, double* L_Mz, double* L_R); /* L(U) of the stored state */
int mfo_eval_faces(mfo_ctx*, double dt, int d, int side, double* out5); /* evolved face states of interior cells, 5*N doubles, comp-major */
int mfo_num_threads(void);                                              /* 1 unless built with -fopenmp */

#ifdef __cplusplus
}
#endif
#endif
