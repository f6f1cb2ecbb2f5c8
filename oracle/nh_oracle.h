/* nh_oracle.h -- CPU ORACLE (test infrastructure, NOT the product).
 *
 * Plain, slow, obviously-correct fp64 implementation of one time step of the hybrid
 * finite-volume / finite-difference projection scheme of Escalante, Morales de Luna & Castro
 * (arXiv 1706.04551; /root/reference/PAPER.md) for Yamazaki's depth-integrated
 * non-hydrostatic system, written from the paper step by step.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * use anything under oracle/.  It shares no code, header, table or helper with the CUDA path
 * (paper_1706_04551_b200/csrc, include/nh_b200.h); the structs below are this file's own.
 *
 * All pointers are HOST pointers.  Cell arrays: nx*ny doubles, x fastest.  Node arrays:
 * (nx+1)*(ny+1) doubles, x fastest, always (in a periodic direction the last line duplicates
 * the first: ignored on input, filled on output).  Node (I,J) is the common corner of cells
 * (I-1,J-1),(I,J-1),(I-1,J),(I,J); it is the paper's (i+1/2,j+1/2) with i=I-1, j=J-1.
 *
 * Return value: 0 on success, negative code otherwise (no exceptions, no aborts).
 */
#ifndef NH_ORACLE_H
#define NH_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

enum { NHO_BC_PERIODIC = 0, NHO_BC_WALL = 1, NHO_BC_OUTFLOW = 2 };
enum { NHO_OK = 0, NHO_EINVAL = -1, NHO_ENOMEM = -2, NHO_ENOCONV = -4, NHO_ENAN = -5 };

typedef struct {
  double g;            /* gravity                                        */
  double cfl;          /* CFL number in (0,1] (eq. (23))                      */
  double delta;        /* velocity desingularisation delta (L447-451), paper: 1e-5      */
  double eps_dry;      /* dry threshold on h (reading R1: = delta)                      */
  double B1, B2;       /* breaking onset / termination coefficients (L141-143, L635)    */
  double solver_rtol;  /* stop at ||r||_2 <= rtol*||b||_2 (reading R14), 1e-12          */
  double gen_A, gen_h0, gen_x0, gen_Lrel; /* solitary-wave generating zone at x-lo (L417-431, R18) */
  double manning_n;    /* Gauckler-Manning coefficient n (L61-65, L773-775); 0 = frictionless     */
  double srj_eps;      /* solver 1: stop when the Jacobi increment of (32) is < srj_eps (L507-514) */
  double srj_rel;      /* solver 1: if > 0 the tolerance of (32) is srj_rel * max|b/A_C| instead    */
  double abs_xlo, abs_xhi, abs_ylo, abs_yhi; /* widths L_Rel of absorbing relaxation zones on the
                          four sides (L415-440; R18, R29); 0 = none                                */
  int breaking;        /* 1: eddy-viscosity breaking sources on (section 3)             */
  int nonhydro;        /* 0: hydrostatic SWE path only (p = 0, w frozen)                */
  int time_order;      /* 1 or 2 (TVD RK2, L406, L516)                                  */
  int space_order;     /* 1 (eqs (16)-(19)) or 2 (MUSCL+minmod, eqs (20)-(22))          */
  int bc_xlo, bc_xhi, bc_ylo, bc_yhi;
  int solver_maxit;
  int gen_on;
  int precision;       /* 64 only in the oracle                                         */
  int solver;          /* 0: Jacobi-preconditioned BiCGStab (R14); 1: the paper's Jacobi method
                          with scheduled relaxation (L507-514; reading R28)                     */
  int srj_mmax;        /* solver 1: longest relaxation cycle (power of two), default 256        */
  int w_advect;        /* 1: vertical-velocity equation of [7], (hw)_t + div(hw u) = p (L109-113), instead of
                          h w_t = p: w transported by first-order upwind differences (reading R30) */
  int warm_start;      /* 1 (default): start vector of a solve = previous solution + quadratic extrapolation of
                          the same-kind increments of the last three steps (reading R32; solver 0 with solver_rtol <= 1e-8
                          only); 0: previous solution */
  int reserved;
} nho_params;

typedef struct {
  double t;            /* simulated time                                                */
  double dt_last;      /* last time step used                                           */
  double res_last;     /* last solve: true ||b-Ax||_2/||b||_2 before the polish iteration */
  long long steps;
  long long iters_total; /* BiCGStab iterations over all solves (polish not counted)    */
  long long clamps;    /* number of h<0 -> 0 clamps (reading R7)                        */
  long long solves;
  int iters_last, iters_max;
  int flags;           /* bit0: a solve failed to converge                              */
  int reserved;
  double clamp_max;    /* largest |h*| of a clamped negative depth (R7, R24)              */
  long long clamp_hist[6]; /* clamps by size of |h*| in metres: < 1e-15, < 1e-12, < 1e-9, < 1e-6,
                          < 1e-3, >= 1e-3                                                  */
} nho_info;

typedef struct nho_ctx nho_ctx;

void nho_default_params(nho_params* prm);
int  nho_create(nho_ctx** out, int nx, int ny, double dx, double dy, const double* H,
                const nho_params* prm);
void nho_destroy(nho_ctx* c);
int  nho_set_state(nho_ctx* c, const double* h, const double* qx, const double* qy,
                   const double* w, const double* p);          /* w,p NULL => zeros; a new run:
                                                                  the solution history of R32 is dropped */
int  nho_continue_state(nho_ctx* c, const double* h, const double* qx, const double* qy,
                        const double* w, const double* p);     /* the same for the running state coming
                                                                  back: the solution history is kept   */
int  nho_get_state(nho_ctx* c, double* h, double* qx, double* qy, double* w, double* p); /* NULL => skip */
int  nho_set_time(nho_ctx* c, double t);          /* simulated time of the current state (restart) */
int  nho_step(nho_ctx* c, int nsteps);            /* CFL dt each step, RK per time_order */
int  nho_hydrostatic_step(nho_ctx* c, double dt); /* S0-S5 only, in place; dt<=0 => CFL  */
int  nho_nonhydro_correct(nho_ctx* c, double dt); /* S6-S10 on the current state         */
int  nho_get_info(nho_ctx* c, nho_info* out);
const char* nho_last_error(nho_ctx* c);

/* test hooks */
int  nho_compute_dt(nho_ctx* c, double* dt);                        /* full-step dt rule (R20)      */
int  nho_apply_A(nho_ctx* c, const double* x_nodes, double* y_nodes); /* y = A(h,z) x (S8)          */
int  nho_coeffs(nho_ctx* c, double* AC, double* AE, double* AW, double* AN, double* AS);
int  nho_rhs(nho_ctx* c, double dt, double* b_nodes);   /* b = -B/dt of the current state (S7), breaking ignored */
int  nho_constraint(nho_ctx* c, double* B_nodes);       /* discrete B, eq. (37), current state */
int  nho_w_advect(nho_ctx* c, double dt, double* w_out); /* S5b alone (R30): w of the current state transported over dt */
int  nho_start_vector(nho_ctx* c, double* x0_nodes); /* R32: the vector the next solve of a step would start from */
int  nho_solve(nho_ctx* c, const double* b_nodes, double* x_nodes, int* iters, double* relres); /* S9; x in: start */
int  nho_breaking(nho_ctx* c, double dt, double* qx2, double* qy2, double* w2); /* S6 alone: the current
                   state taken as U*, w -> q** = q* + dt R_u (cells), w** = w + dt R_w (nodes); updates the
                   hysteresis flags of R11 (they persist across set_state); requires prm.breaking     */
void nho_face_fluct(double g, double hm, double etam, double um, double vm,
                    double hp, double etap, double up, double vp,
                    double Dm[3], double Dp[3]);                     /* S4 */
double nho_dsg(double h, double q, double delta);                    /* S0 */
double nho_minmod(double a, double b);                               /* S2 */
double nho_cbrt_fixed(double a);   /* R31: cube root of a > 0 by the fixed algorithm (friction, R27) */
double nho_sech2_fixed(double a);  /* R31: sech^2 by the fixed algorithm (solitary-wave target, S11)  */

#ifdef __cplusplus
}
#endif
#endif
