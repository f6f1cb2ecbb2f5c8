// nh_internal.cuh -- shared declarations of the CUDA path (libnh_b200.so).  Not part of the ABI.
//
// Steps S0..S11 and readings R1..R23 are those of DESIGN.md (restating SURVEY.md 8(c));
// "L<n>" are PAPER.md line numbers (arXiv 1706.04551).
//
// Arithmetic contract: fp64, compiled with -fmad=false so that every formula is evaluated in
// source order with IEEE-754 round-to-nearest operations (CUDA's fp64 div and sqrt are correctly
// rounded).  The predictor, the breaking sources, the right-hand side, the coefficients and the
// correction therefore take every discrete decision (minmod branch, wet/dry test, emerging-bottom
// clip, breaking flag, clamp) on the same values a plain CPU evaluation of the paper's formulas
// sees; only the Krylov solver's dot products are summed in a different (tree) order.
//
// Precision.  Every kernel file and nh_core.cu are compiled twice, with NH_PREC = 64 (namespace
// nh64, real = double: the contract above) and NH_PREC = 32 (namespace nh32, real = float: the
// optional fp32 variant of north_star -- all field planes and their arithmetic in fp32, eta stored
// beside h so that metres of signal survive on kilometres of depth, the scalar reductions (dt, dot
// products, the clock) in fp64).  RC(x) types a literal as real.  nh_abi.cu
// holds the extern "C" entry points and dispatches on nh_params.precision.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <utility>
#include <vector>

#include "../../include/nh_b200.h"

#ifndef NH_PREC
#define NH_PREC 64
#endif
#if NH_PREC == 64
#define NH_NS nh64
#define NH_REAL double
#define NH_REAL2 double2
#elif NH_PREC == 32
#define NH_NS nh32
#define NH_REAL float
#define NH_REAL2 float2
#else
#error "NH_PREC must be 64 or 32"
#endif
#define RC(x) ((NH_REAL)(x))

#ifndef NH_SHARED_TYPES
#define NH_SHARED_TYPES


// Device-resident scalars: the time step, the clock and the counters never visit the host
// inside nh_step.
struct NhScal {
  double dt;        // time step of the step in flight
  double t;         // simulated time
  double dt_last;
  double res_last;
  unsigned long long lam_bits;  // max over cells of the CFL rate, as the bits of a non-negative double
  long long steps, iters_total, clamps, solves;
  int iters_last, iters_max, flags, pad;
  // solver 1 (nh_solver.cu, k_srj): bits of non-negative doubles, reduced by integer atomicMax
  unsigned long long srj_rho_bits;   // Gershgorin radius of D^-1 A about 1 (k_scale_rows)
  unsigned long long srj_bmax_bits;  // max |b / A_C| (k_scale_rows)
  unsigned long long srj_E_bits[3];  // max |Jacobi increment| of sweep k in slot k % 3
  int srj_bad, pad2;                 // a NaN appeared in a sweep
  // size statistics of the negative depths clamped by the predictor (R7, R24): exact integer atomics
  unsigned long long clamp_max_bits;  // max |h*|, as the bits of a non-negative double
  unsigned long long clamp_hist[6];   // < 1e-15, < 1e-12, < 1e-9, < 1e-6, < 1e-3, >= 1e-3 (metres)
};

enum { NH_FLAG_NOCONV = 1, NH_FLAG_NAN = 2, NH_FLAG_BADSTATE = 4, NH_FLAG_STAGNATED = 8 };
#endif  // NH_SHARED_TYPES

namespace NH_NS {

typedef NH_REAL real;
typedef NH_REAL2 real2;
// grid geometry handed to every kernel by value
struct NhGrid {
  int nx, ny;    // cells
  int nnx, nny;  // distinct node lines: n in a periodic direction, n+1 otherwise
  int np;        // internal node pitch (nh_node_pitch: multiple of 16, ghost / padding columns on both sides)
  int bxlo, bxhi, bylo, byhi;
  real dx, dy;
};

constexpr bool kEta = (NH_PREC == 32);  // eta stored beside h (fp32 variant)
__host__ __device__ __forceinline__ real2 make_real2(real a, real b) { real2 v; v.x = a; v.y = b; return v; }

// ---- S1: ghost access by index maps (R9) ------------------------------------------------
// cells: periodic wraps; wall / outflow mirror (-1->0, -2->1, n->n-1, n+1->n-2); sgn = -1 only
// in a wall ghost (applied by the caller to the normal discharge / velocity).
__device__ __forceinline__ int nh_map_cell(int i, int n, int bclo, int bchi, real& sgn) {
  sgn = RC(1.0);
  if (i < 0) {
    if (bclo == NH_BC_PERIODIC) return i + n;
    if (bclo == NH_BC_WALL) sgn = -RC(1.0);
    return -1 - i;
  }
  if (i >= n) {
    if (bchi == NH_BC_PERIODIC) return i - n;
    if (bchi == NH_BC_WALL) sgn = -RC(1.0);
    return 2 * n - 1 - i;
  }
  return i;
}
__device__ __forceinline__ int nh_map_cell_even(int i, int n, int bclo, int bchi) {
  if (i < 0) return (bclo == NH_BC_PERIODIC) ? i + n : -1 - i;
  if (i >= n) return (bchi == NH_BC_PERIODIC) ? i - n : 2 * n - 1 - i;
  return i;
}
// nodes: periodic: node n == node 0 (n distinct lines, n = number of cells); mirror: -1 -> 1,
// n+1 -> n-1 (R10).  Valid for -n <= I <= 2n.
__device__ __forceinline__ int nh_map_node(int I, int n, int bclo) {
  if (bclo == NH_BC_PERIODIC) {
    if (I < 0) return I + n;
    if (I >= n) return I - n;
    return I;
  }
  if (I < 0) return -I;
  if (I > n) return 2 * n - I;
  return I;
}

// S0: desingularised velocity u = sqrt(2) h q / sqrt(h^4 + max(h^4, delta^4))  (L447-451)
#define NH_SQRT2 RC(1.4142135623730951)
__device__ __forceinline__ real nh_dsg(real h, real q, real delta) {
  real h2 = h * h, h4 = h2 * h2;
  real d2 = delta * delta, d4 = d2 * d2;
  real den = sqrt(h4 + fmax(h4, d4));
  real num = NH_SQRT2 * h * q;
  // 0 / den = 0 (den > 0): same bits, but a zero dividend would send the fp64 division down its slow
  // path, and still water is common (2.8 M of 3.5 M warp-divisions on the config-5 basin)
  return (num == RC(0.0)) ? num : num / den;
}
// R16: dinv(h) = sqrt(2) h / sqrt(h^4 + max(h^4, delta^4))  (= 1/h for h >= delta)
__device__ __forceinline__ real nh_dinv_h(real h, real delta) {
  real h2 = h * h, h4 = h2 * h2;
  real d2 = delta * delta, d4 = d2 * d2;
  return (NH_SQRT2 * h) / sqrt(h4 + fmax(h4, d4));
}
// S2: minmod(a,b) = 0 if ab <= 0 else sign(a) min(|a|,|b|)  (L335)
__device__ __forceinline__ real nh_minmod(real a, real b) {
  if (a * b <= RC(0.0)) return RC(0.0);
  return (a > RC(0.0)) ? fmin(a, b) : fmax(a, b);
}

// R31: the two transcendentals of the path -- the cube root in h^(4/3) of the friction law (L61-65)
// and sech^2 of the solitary-wave target (33) -- are evaluated by a stated sequence of IEEE
// operations (frexp / ldexp / floor are exact) instead of library routines whose last place is
// not specified, so that the results do not depend on who evaluates them.
// cube root of a > 0: a = t 8^q, t in [0.5, 4); six Halley steps from y = 1
__device__ __forceinline__ real nh_cbrt_fixed(real a) {
  int e;
  real m = frexp(a, &e);
  int q = (e + 3072) / 3 - 1024;  // floor(e / 3)
  real t = ldexp(m, e - 3 * q);
  real y = RC(1.0);
#pragma unroll 1
  for (int k = 0; k < 6; ++k) {
    real y3 = y * y * y;
    y = y * (y3 + RC(2.0) * t) / (RC(2.0) * y3 + t);
  }
  return ldexp(y, q);
}
// sech^2(a) = 4 e / (1 + e)^2, e = exp(-2|a|) = 2^-n exp(-r), r = 2|a| - n ln 2 (two pieces),
// exp(-r) by its Taylor series to r^14 in Horner form
__device__ __forceinline__ real nh_sech2_fixed(real a) {
  real y = RC(2.0) * fabs(a);
  if (y > RC(745.0)) return RC(0.0);
  real n = floor(y * RC(1.4426950408889634) + RC(0.5));
  real r = (y - n * RC(0.693147180369123816490)) - n * RC(1.90821492927058770002e-10);
  real p = RC(1.0);
#pragma unroll 1
  for (int k = 14; k >= 1; --k) p = RC(1.0) - (r / (real)k) * p;
  real e = ldexp(p, -(int)n);
  real d = RC(1.0) + e;
  return RC(4.0) * e / (d * d);
}

// Internal node planes: NH_COL_PAD ghost / padding columns on the left, >= 2 on the right, pitch NP
// a multiple of 16 doubles (every row starts on a 128-byte line), ny + 5 rows; the pointer handed
// to kernels addresses node (0,0) = physical element (2 rows, 4 columns), so that a[J * np + I] is
// valid for -4 <= I < np - 4 and -2 <= J <= ny + 2: ghost lines need no index map, every even
// column is 16-byte aligned, and the 60-column strips of the solver's marching warps
// (nh_solver.cu) start on 32-byte sectors: 60 s + 4 columns = 480 s + 32 bytes, so no two warps
// ever write parts of the same sector (measured: +39 % store bandwidth over a 16-byte offset).
constexpr int NH_STRIP = 60, NH_ROW_PAD = 2, NH_COL_PAD = 4;
inline int nh_node_pitch(int nnx) {
  int n = NH_STRIP * ((nnx + NH_STRIP - 1) / NH_STRIP) + NH_COL_PAD + 2;
  return (n + 15) / 16 * 16;
}

// ---- context ------------------------------------------------------------------------------
struct Ctx {
  NhGrid g;
  nh_params prm;
  cudaStream_t stream;
  int device;
  int sm_count;
  long long launches;
  char err[512];
  int host_status;  // sticky host-side error (NH_ECUDA)
  bool lam_valid;   // sc->lam_bits holds the CFL rate of the current state

  size_t nc, nn;  // cells, nodes (public node layout)
  // cells
  real* H;
  real* eta[3];   // fp32 variant only (kEta): eta = h - H of the three state slots, the master copy
  double* Hd;     // fp32 variant only: the bathymetry as given (fp64), for eta = h - H at set / get
  double* stage;  // fp32 variant only: fp64 staging plane for set / get (max(cells, nodes) doubles)
  real *h[3], *qx[3], *qy[3];  // three state slots (rotating): current, stage 1, stage 2
  real *qx1, *qy1;             // predictor output q*
  real *qx2, *qy2;             // q** (breaking on)
  real* z;                     // z = 2 eta - h of U*
  real *hc, *zc;               // h, z of U* in the node layout shifted by one column, ghost cells
                                 // filled (operands of the matrix-free solver, nh_solver.cu)
  unsigned char *flag_c, *flag_n;
  // nodes
  real* w[3];
  real* w2;  // w** (breaking on)
  real* wadv;  // w after the transport step of the w-advection variant (R30)
  real* hist[7];  // R32: the last seven pressure solutions, hist[0] the most recent
  int nhist;      // how many of them are valid (reset by set_state)
  real* p;   // pressure multiplier p~ (warm start of the next solve)
  real* b;   // right-hand side
  real *dg, *dinv, *cE, *cW, *cN, *cS;  // diag(A), its inverse, off-diagonals (solver 1: row-scaled; hooks: raw)
  real *ky, *kr, *krB, *kr0, *kpA, *kpB, *kvA, *kvB, *kt;  // BiCGStab vectors (r, p, v double-buffered)
  double* pub;   // dense (nx+1) x (ny+1) staging plane for the public node layout
  std::vector<void*> raw;  // allocation bases (node planes are handed out offset to node (0,0))
  double* part;  // per-CTA partial sums of the solver
  int solver_grid, solver_occ, solver_nstrips, solver_R, solver_nbands;
  int srj_grid, srj_R, srj_nbands;  // solver 1: cooperative grid and band height of k_srj
  double* srj_cos;                  // solver 1: cos(pi (2 perm_i - 1) / 2M), tables of M = 1, 2, 4, ... at offset M - 1
  size_t nni;  // doubles per internal node plane (ghost ring included)
  NhScal* sc;       // device scalars
  NhScal* sc_host;  // pinned mirror
  int cur;          // index of the cell slot (h, qx, qy) holding the current state
  int curw;         // index of the node slot (w) holding the current state
  // per-phase CUDA-event brackets (nh_profile): predictor / assembly / solver / correction
  bool prof_on;
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> prof_ev[NH_PROF_CATS];
};

// fp32 variant: the eta plane that goes with a state slot's h plane (nullptr in the fp64 build)
inline real* nh_eta_of(const Ctx* c, const real* h) {
  if (kEta)
    for (int s = 0; s < 3; ++s)
      if (c->h[s] == h) return c->eta[s];
  return nullptr;
}

// ---- kernel launchers (each enqueues on c->stream and bumps c->launches) --------------------
// nh_predictor.cu
void nh_launch_lambda(Ctx* c, const real* h, const real* qx, const real* qy);
void nh_launch_set_dt(Ctx* c, double dt_fixed /* <=0: CFL from lam */);
void nh_launch_end_step(Ctx* c, int advance_time);
void nh_launch_predictor(Ctx* c, const real* h, const real* qx, const real* qy,
                         real* h1, real* qx1, real* qy1);
void nh_launch_combine(Ctx* c, real* h0, real* qx0, real* qy0, real* w0,
                       const real* h2, const real* qx2, const real* qy2, const real* w2);
void nh_launch_validate(Ctx* c, const real* h, const real* qx, const real* qy);
// nh_pressure.cu
void nh_launch_compute_z(Ctx* c, const real* h, real* z);
void nh_launch_cell_planes(Ctx* c, const real* h);  // z (dense) and hc, zc (solver 0)
void nh_launch_breaking(Ctx* c, const real* h, const real* qx1, const real* qy1,
                        const real* w_in, real* qx2, real* qy2, real* w2);
void nh_launch_rhs(Ctx* c, const real* h, const real* qx, const real* qy, const real* z,
                   const real* w, real* b, int constraint_only);
void nh_launch_coeffs(Ctx* c, const real* h, const real* z);  // -> dg, dinv, raw cE..cS
void nh_launch_scale_rows(Ctx* c, const real* b, real* bp);
void nh_launch_assemble_rows(Ctx* c, const real* h, const real* qx, const real* qy,
                             const real* z, const real* w, real* bp);  // solver 1: rhs + rows + scaling fused  // solver 1: cX *= dinv, bp = b dinv, rho, max|bp|
void nh_launch_apply_A(Ctx* c, const real* h, const real* z, const real* x, real* y);
void nh_launch_correct(Ctx* c, const real* h, const real* z, const real* qx2,
                       const real* qy2, const real* w2, const real* p, real* qx_out,
                       real* qy_out, real* w_out);
void nh_launch_w_advect(Ctx* c, const real* h, const real* qx, const real* qy,
                        const real* w_in, real* w_out);  // R30
void nh_launch_start_vector(Ctx* c, real* x0);  // R32: x0 <- extrapolation of c->hist (all 7 valid)
void nh_launch_relax(Ctx* c, real* h, real* qx, real* qy, real* w, real* p, int stage);
void nh_launch_absorb(Ctx* c, real* h, real* qx, real* qy, real* w, real* p);
void nh_launch_nodes_out(Ctx* c, const real* src, double* dst);
// nh_solver.cu
int nh_solver_setup(Ctx* c);  // occupancy -> cooperative grid, partial buffer
void nh_launch_solve(Ctx* c, const real* b, real* x, int count_stats);

#define NH_CUDA_OK(c, call)                                                                   \
  do {                                                                                        \
    cudaError_t e_ = (call);                                                                  \
    if (e_ != cudaSuccess) {                                                                  \
      snprintf((c)->err, sizeof((c)->err), "%s:%d: %s: %s", __FILE__, __LINE__, #call,        \
               cudaGetErrorString(e_));                                                       \
      (c)->host_status = NH_ECUDA;                                                            \
    }                                                                                         \
  } while (0)

}  // namespace NH_NS
