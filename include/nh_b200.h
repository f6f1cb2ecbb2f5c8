/* nh_b200.h -- C ABI of libnh_b200.so: the per-time-step hot path of the hybrid finite-volume /
 * finite-difference projection scheme of Escalante, Morales de Luna & Castro (arXiv 1706.04551,
 * cited below as PAPER.md L<line>) for Yamazaki's depth-integrated non-hydrostatic system,
 * hand-written CUDA for NVIDIA B200 (sm_100a), SoA, fp64 (optional fp32 variant: nh_params.precision).
 *
 * Every step of the path runs in CUDA kernels of this library; there is no CPU fallback.  No
 * torch types appear here: plain pointers and sizes.
 *
 * POINTERS.  Every array pointer may be a DEVICE pointer (valid on the device of the context's
 * stream) or a HOST pointer (pageable or pinned): copies use cudaMemcpyAsync(cudaMemcpyDefault)
 * on the context's stream, so unified virtual addressing decides.  With pageable host memory the
 * copy is synchronous with respect to the host.  The caller owns every buffer it passes; the
 * library copies on create/set and copies out on get; nothing but the context is returned by
 * pointer.  The context owns all device memory it uses (cudaMalloc at nh_create).
 *
 * LAYOUT.  Cell arrays: nx*ny doubles, x fastest (cell (i,j) at j*nx+i, centre ((i+1/2)dx,
 * (j+1/2)dy)).  Node arrays: (nx+1)*(ny+1) doubles, x fastest, always; node (I,J) is the common
 * corner of cells (I-1,J-1),(I,J-1),(I-1,J),(I,J) -- the paper's staggered point
 * (i+1/2,j+1/2) with i=I-1, j=J-1.  In a periodic direction the
 * last node line duplicates the first: ignored on input, filled on output.
 *
 * ASYNCHRONY.  nh_step / nh_hydrostatic_step / nh_nonhydro_correct only enqueue work on the
 * context's stream and return (no host synchronisation inside; dt, the solver's convergence tests
 * and all reductions stay on the device).  nh_set_state, nh_get_state, nh_sync, nh_get_info and the
 * test hooks synchronise with the stream (nh_set_state once, to report the validation of its
 * input).  Sticky run-time conditions (a solve that did not converge, a NaN time step) are
 * reported by nh_sync / nh_get_info.
 *
 * ERRORS.  0 on success, a negative nh_status otherwise; no exceptions, no aborts, no global
 * state.  One context may be used by one host thread at a time.
 */
#ifndef NH_B200_H
#define NH_B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nh_ctx nh_ctx; /* opaque */

/* boundary types (the wall type is this build's extension, R9) */
typedef enum { NH_BC_PERIODIC = 0, NH_BC_WALL = 1, NH_BC_OUTFLOW = 2 } nh_bc;

typedef enum {
  NH_OK = 0,
  NH_EINVAL = -1,  /* invalid argument (also: h < 0 or non-finite input found by nh_set_state) */
  NH_ENOMEM = -2,  /* host or device allocation failed                                     */
  NH_ECUDA = -3,   /* a CUDA call failed (nh_last_error has the text)                      */
  NH_ENOCONV = -4, /* a pressure solve hit maxit / still not converged after 8 restart cycles */
  NH_ENAN = -5     /* NaN/Inf time step or right-hand side                                 */
} nh_status;

/* Parameters, passed by pointer, copied.  Fill with nh_default_params first. */
typedef struct {
  double g;           /* gravity, default 9.81                               */
  double cfl;         /* CFL number in (0,1], default 0.5 (eq. (23))              */
  double delta;       /* velocity desingularisation delta, default 1e-5 (L447-451)          */
  double eps_dry;     /* cell is dry iff h <= eps_dry, default 1e-5 (R1)          */
  double B1, B2;      /* breaking onset / termination coefficients, 0.15 / 0.5 (L141-143, L635) */
  double solver_rtol; /* BiCGStab stops at ||r||_2 <= rtol ||b||_2, default 1e-12 (R14)     */
  double gen_A, gen_h0, gen_x0, gen_Lrel; /* solitary-wave generating zone at x-lo (L417-431, R18) */
  double manning_n;   /* Gauckler-Manning n (L61-65, L773-775), semi-implicit (R27); default 0 = off */
  double srj_eps;     /* solver 1: stop when the Jacobi increment of eq. (32) is < srj_eps; 1e-5  */
  double srj_rel;     /* solver 1: if > 0, the tolerance of (32) is srj_rel * max|b / A_C| instead */
  double abs_xlo, abs_xhi, abs_ylo, abs_yhi; /* widths L_Rel of the absorbing relaxation zones on
                         the four sides (L415-440; R18, R29); 0 = none (default).  Not on
                         a periodic side; abs_xlo not together with gen_on: NH_EINVAL           */
  int breaking;       /* 1: eddy-viscosity breaking sources on (section 3, eqs (8)-(12))    */
  int nonhydro;       /* 0: hydrostatic SWE path only (p = 0, w frozen); default 1          */
  int time_order;     /* 1, or 2 = two-stage TVD Runge-Kutta (L406, L516, L544); default 2  */
  int space_order;    /* 1 = eqs (16)-(19), 2 = MUSCL+minmod eqs (20)-(22); default 2       */
  int bc_xlo, bc_xhi, bc_ylo, bc_yhi; /* nh_bc; periodic must be set on both sides of a direction */
  int solver_maxit;   /* default 10000                                                      */
  int gen_on;         /* 1: generating relaxation zone active                               */
  int precision;      /* 64 (default): fp64 throughout, the parity contract.  32: the optional fp32
                         variant -- every field plane and its arithmetic in fp32 (eta = h - H is
                         stored beside h so that metres of signal survive on kilometres of depth),
                         dt, the clock and all dot products in fp64; arrays at this boundary stay
                         fp64 (converted at set / get); solver_rtol below 1e-4 is raised to 1e-4.
                         Tolerances against the fp64 oracle: DESIGN.md section 10                 */
  int solver;         /* 0 (default): Jacobi-preconditioned BiCGStab to solver_rtol (R14);
                         1: the paper's Jacobi method with scheduled relaxation and stopping
                         rule (32) (L507-514; R28): no dot products, results bit-identical
                         to the CPU oracle's                                                 */
  int srj_mmax;       /* solver 1: longest relaxation cycle, a power of two <= 4096; default 256 */
  int w_advect;       /* 1: the vertical-velocity equation of [7], (hw)_t + div(hw u) = p (PAPER.md
                         L109-113), instead of h w_t = p: in every stage the node values w are first
                         transported by first-order upwind differences with the 4-cell mean of the
                         desingularised velocities (R30); default 0                       */
  int warm_start;     /* 1 (default): a pressure solve starts from the previous solution plus the quadratic
                         extrapolation of the same-kind increments of the last three steps,
                         x0 = s1 + 3 (s2 - s3) - 3 (s4 - s5) + (s6 - s7) (R32), once seven
                         solutions exist since the last nh_set_state, for solver 0 with solver_rtol
                         <= 1e-8 (looser stopping rules start from the previous solution, as 0 does) */
  int reserved;
} nh_params;

typedef struct {
  double t;              /* simulated time                                                  */
  double dt_last;        /* last time step used                                             */
  double res_last;       /* last solve: solver 0: true ||b-Ax||_2/||b||_2 before the polish iteration;
                            solver 1: the last max|Jacobi increment| E of eq. (32)           */
  long long steps;
  long long iters_total; /* solver iterations over all solves (solver 0: BiCGStab iterations, polish
                            not counted; solver 1: Jacobi sweeps that updated x)             */
  long long clamps;      /* number of h<0 -> 0 clamps in the predictor (R7)                 */
  long long solves;
  int iters_last, iters_max;
  int flags;             /* bit0: a solve failed to converge; bit1: NaN/Inf dt or rhs;
                            bit2: the last set_state saw h<0 or a non-finite value (rejected);
                            bit3 (fp32 variant only, informational, sticky, no error code): a solve was
                            accepted because its true residual stopped improving ABOVE
                            solver_rtol_effective -- look at res_last                         */
  int reserved;
  double clamp_max;      /* largest |h*| of a clamped negative depth (R7, R24)             */
  long long clamp_hist[6]; /* clamps by size of |h*| in metres: < 1e-15, < 1e-12, < 1e-9, < 1e-6,
                            < 1e-3, >= 1e-3                                                 */
  double solver_rtol_effective; /* the tolerance solver 0 really stops at: nh_params.solver_rtol, except
                            that the fp32 variant raises anything below 1e-4 to 1e-4            */
} nh_info;

void nh_default_params(nh_params* prm);

/* Problem statement of the paper: a structured Cartesian mesh of nx*ny cells of size dx*dy with
 * still-water depth H per cell (may be negative = emerged land; bed elevation z_b = -H)
 * (PAPER.md L462-470, L528).  cuda_stream: a cudaStream_t (NULL = the default stream); all work
 * of this context is ordered on it.  Requires nx,ny >= 4 (two-cell MUSCL halo), dx,dy > 0,
 * finite H.  Fails with NH_ECUDA when no sm_100 device / kernel image is available. */
int nh_create(nh_ctx** out, int nx, int ny, double dx, double dy, const double* H,
              const nh_params* prm, void* cuda_stream);
void nh_destroy(nh_ctx* ctx);

/* State = conserved variables (h, qx, qy) per cell (L45-59, L528) and (w, p) per staggered node
 * (L245-247, L464-466, L535).  w, p NULL => zeros.  set stages the arrays in a free slot,
 * validates h >= 0 and finiteness there on the device, waits for that result (one stream
 * synchronisation) and returns NH_EINVAL leaving the current state untouched if it fails.
 * nh_set_state starts a NEW run: the solver forgets its history of earlier pressure solutions
 * (R32), so the next solves start from p alone.  nh_continue_state is the same call for a
 * state that IS the running one coming back -- a checkpoint restored into the context that wrote it,
 * a round trip through the host: the history is kept, and the run goes on exactly as if the state had
 * never left (same iteration counts, same bits).  The caller says which it is; the library does not
 * look at the contents to guess.  Handing nh_continue_state an unrelated state is not an error: the
 * first solves merely start from a poor vector (more iterations, same converged result).
 * get: NULL => skip that field; synchronises (the arrays are complete on return). */
int nh_set_state(nh_ctx* ctx, const double* h, const double* qx, const double* qy,
                 const double* w, const double* p);
int nh_continue_state(nh_ctx* ctx, const double* h, const double* qx, const double* qy,
                      const double* w, const double* p);
int nh_get_state(nh_ctx* ctx, double* h, double* qx, double* qy, double* w, double* p);
/* Simulated time of the current state (default 0 at nh_create).  Together with nh_get_state /
 * nh_set_state and nh_get_info().t this is the checkpoint / restart of the FIELDS: the generating
 * relaxation zone (L417-431) is the only part of the step that reads the clock.  Enqueued on the stream.
 * Two pieces of state are NOT in that checkpoint and stay inside the context:
 *  (1) the onset / termination flags of the breaking criterion (eq. (9)).  They survive
 *      nh_set_state and start cleared in a new context.  With B1 < B2 (the default 0.15 / 0.5) the
 *      criterion does not consult them, so a restart in a fresh context is equivalent; with B1 >= B2
 *      (true hysteresis) it is not, and there is no call to export them.
 *  (2) the solver's history of the last seven pressure solutions (start vector, R32).
 *      nh_set_state drops it, nh_continue_state keeps it; a fresh context always starts without one
 *      (seven solves from the previous solution alone: more iterations, same converged result).
 * Neither changes what a converged step computes beyond the solver tolerance, except (1) with
 * B1 >= B2. */
int nh_set_time(nh_ctx* ctx, double t);

/* nsteps full time steps: dt = CFL / max[(|u|+sqrt(gh))/dx + (|v|+sqrt(gh))/dy] (eq. (23),
 * DESIGN.md R20), then per Runge-Kutta stage: hydrostatic predictor (eqs (16)-(22), (30)),
 * semi-implicit Manning friction if manning_n > 0 (L61-65, L249), breaking sources (eqs (8)-(12),
 * (28)), pressure system assembly and solve (eqs (24)-(29), (36)-(43); prm.solver: BiCGStab to
 * solver_rtol, or the paper's Jacobi method with scheduled relaxation and rule (32)), Chorin-Temam
 * correction (eqs (28), (31), (41)), generating / absorbing relaxation zones (L415-440); stages
 * combined as U^{n+1} = (U^n + U^(2))/2 (L406, L516, L544). */
int nh_step(nh_ctx* ctx, int nsteps);

/* First part alone: predictor (S0-S5) on the current state, in place; w, p untouched.
 * dt <= 0 => the CFL time step of the current state. */
int nh_hydrostatic_step(nh_ctx* ctx, double dt);
/* Second + third part alone: breaking sources, right-hand side, solve, correction (S6-S10) on
 * the current state, in place; h unchanged.  dt > 0 required. */
int nh_nonhydro_correct(nh_ctx* ctx, double dt);

/* Wait for the stream; returns the sticky run-time status (NH_OK / NH_ENOCONV / NH_ENAN /
 * NH_ECUDA) and clears nothing. */
int nh_sync(nh_ctx* ctx);
int nh_get_info(nh_ctx* ctx, nh_info* out); /* synchronises */
const char* nh_last_error(nh_ctx* ctx);

/* Launch counters (host side, for bench.py's gpu_launches): number of kernels this context has
 * launched since creation. */
long long nh_launch_count(nh_ctx* ctx);

/* Per-phase device timing for the roofline report (bench.py): when enabled, every kernel group of
 * nh_step is bracketed by a pair of CUDA events recorded on the context's stream (no host
 * synchronisation is added).  nh_profile_read synchronises, returns the summed milliseconds and
 * the number of brackets per phase since the last read (arrays of NH_PROF_CATS entries, HOST
 * pointers) and resets them.  Phases: the hydrostatic predictor (a1-a3), the assembly (a4-a5 and
 * the rows of A), the pressure solve (a6: one cooperative kernel per bracket), and the correction
 * with the Runge-Kutta combine (a7-a8). */
enum { NH_PROF_PREDICTOR = 0, NH_PROF_ASSEMBLY = 1, NH_PROF_SOLVER = 2, NH_PROF_CORRECT = 3,
       NH_PROF_CATS = 4 };
int nh_profile(nh_ctx* ctx, int enable);
int nh_profile_read(nh_ctx* ctx, double* ms, long long* groups);

/* Measurement hook (bench.py's predictor roofline): the fp64 instruction rate of the current device,
 * thread-level fused multiply-adds per second, measured with CUDA events on a kernel of independent
 * DFMA chains (2 flops each; / 32 = warp instructions as ncu counts them).  Needs no context;
 * synchronises.  dfma_per_second is a HOST pointer. */
int nh_fp64_rate(void* cuda_stream, double* dfma_per_second);
/* Measurement hook (bench.py --streammix): the DRAM rate, in GB/s of algorithmic bytes, that a plain
 * streaming kernel reaches with nread planes read and nwrite planes written per element -- the mix of
 * one pass of the matrix-free solver (5 + 1 and 8 + 4), of a Jacobi sweep
 * (6 + 1), or of a copy (1 + 1) -- with ideal access.  Planes of doubles_per_plane doubles (even) are
 * allocated and freed inside (NH_ENOMEM if they do not fit); other mixes: NH_EINVAL.  Needs no
 * context; synchronises.  gbytes_per_second is a HOST pointer. */
int nh_stream_mix_rate(void* cuda_stream, int nread, int nwrite, long long doubles_per_plane,
                       double* gbytes_per_second);

/* ---- the CFL time step for callers that must not allocate ------------------------------------
 * nh_cfl_dt_static computes dt = cfl / max_ij[(|u|+sqrt(g h))/dx + (|v|+sqrt(g h))/dy] (eq. (23),
 * PAPER.md L339-341, with the desingularised velocities of L447-451; R20) of a state held
 * in the CALLER's device arrays, without a context: no cudaMalloc, cudaFree, cudaMallocHost or any
 * other allocating call happens inside, on the first call or later.  Everything else in this
 * library needs nh_create, which allocates some fifty field planes.
 *
 * Who this is for.  Code that wants to know the admissible time step of a state it already has on
 * the GPU, but runs where device allocation is off the table: a coupled model whose memory manager
 * has claimed the whole device up front, so that a cudaMalloc from a guest library fails or eats
 * into a reserve it does not own; a latency-bound loop (real-time forecasting, an in-situ monitor
 * that sub-cycles on dt) that cannot afford the device-wide synchronisation cudaMalloc / cudaFree
 * imply; a plug-in that by house rule may not own device memory at all.
 *
 * How.  The reduction's scratch memory (one partial maximum per 4096 cells) is a fixed array
 * compiled into the library: 16384 doubles = 128 KiB.  Every GPU that loads libnh_b200.so holds that
 * array from load until the process exits, used or not.  Its size is the limit: nx * ny must not
 * exceed NH_STATIC_MAX_CELLS (= nh_cfl_dt_static_max_cells() = 8192 * 8192); a larger grid is
 * refused with NH_EINVAL and a message in nh_static_last_error(), nothing is launched.
 *
 * Arguments.  h, qx, qy: nx*ny doubles each, cell layout as above, DEVICE pointers (read only);
 * dt_out: DEVICE pointer to one double (written).  Host pointers are refused with NH_EINVAL.  h is
 * expected >= 0 and finite, as nh_set_state demands; NaN rates are skipped; dt_out = 0 when no cell
 * has a positive rate.  g, delta, cfl: nh_params' g, delta, cfl.  cuda_stream: a cudaStream_t of the
 * CURRENT device (NULL = default stream).  The two kernels are only enqueued; the result is in
 * dt_out once the stream reaches that point; the caller owns all four arrays throughout.  fp64, same
 * operation order as the context path: bit-identical to nh_compute_dt on the same state.
 *
 * First call on a device.  It looks up, once per device and with that device current, the device
 * address of the built-in array (cudaGetSymbolAddress) and checks that the device is sm_100.  Make
 * this first call before starting any stream capture on that device.
 *
 * Sharing.  All calls on one device use the SAME array, and it keeps what the last call left.  Each
 * call overwrites every slot before reading it, so no clearing is needed between calls that follow
 * one another -- in one stream, or in streams ordered by events.  Two calls that can run on the GPU
 * at the same time (different streams, different host threads, no ordering) race on the array and
 * both results are then undefined: serialise them.
 *
 * Errors: NH_EINVAL (sizes, parameters, null / host pointers), NH_ECUDA (no sm_100 device, a CUDA
 * call failed); nh_static_last_error() returns the text for the calling thread's last call. */
#define NH_STATIC_MAX_CELLS 67108864LL
int nh_cfl_dt_static(int nx, int ny, double dx, double dy, double g, double cfl, double delta,
                     const double* h, const double* qx, const double* qy, double* dt_out,
                     void* cuda_stream);
long long nh_cfl_dt_static_max_cells(void);
const char* nh_static_last_error(void);

/* ---- test hooks (not on the timed path); node arrays in/out use the public node layout ---- */
int nh_compute_dt(nh_ctx* ctx, double* dt_host);          /* CFL dt of the current state; synchronises */
int nh_apply_A(nh_ctx* ctx, const double* x_nodes, double* y_nodes); /* y = A(h,z) x, matrix-free (S8) */
int nh_coeffs(nh_ctx* ctx, double* AC, double* AE, double* AW, double* AN, double* AS); /* rows of A */
int nh_rhs(nh_ctx* ctx, double dt, double* b_nodes);      /* b = -B/dt of the current state (S7)   */
int nh_constraint(nh_ctx* ctx, double* B_nodes);          /* discrete constraint B, eq. (37)       */
/* S9 on the current state's operator with the context's solver: x_nodes in = start, out = solution;
 * iters/relres are HOST pointers (may be NULL; relres = res_last of nh_info); synchronises. */
int nh_solve(nh_ctx* ctx, const double* b_nodes, double* x_nodes, int* iters, double* relres);
/* S6 alone (eqs (9)-(12), L136-165, L224; second stage of (28), L379-396): the current state taken
 * as U*, -> q** = q* + dt R_u (cell arrays qx2, qy2) and w** = w + dt R_w (node array w2); updates
 * the onset / termination flags of the breaking criterion (they persist across nh_set_state).
 * Requires prm.breaking and dt > 0 (NH_EINVAL otherwise); synchronises. */
int nh_breaking(nh_ctx* ctx, double dt, double* qx2, double* qy2, double* w2);
/* The transport step of the w-advection variant alone (L109-113, R30): w of the current
 * state carried over dt by the node velocities of the current state -> node array w_out; the state
 * is not changed.  dt > 0 required; works whatever prm.w_advect says; synchronises. */
int nh_w_advect(nh_ctx* ctx, double dt, double* w_out);
/* The vector the next pressure solve of a step would start from (R32) -> node array; the
 * state is not changed; synchronises. */
int nh_start_vector(nh_ctx* ctx, double* x0_nodes);

#ifdef __cplusplus
}
#endif
#endif
