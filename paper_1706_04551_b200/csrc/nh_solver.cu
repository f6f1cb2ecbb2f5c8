// nh_solver.cu -- a6: Jacobi-preconditioned BiCGStab (R14, R25) for the compact
// finite-difference pressure system (eqs (29), (36)-(43)) as ONE persistent
// cooperative kernel per solve, with the operator applied matrix-free (L535).
//
// The whole solve -- true-residual (re)starts, the iteration loop with its convergence tests, the
// half-step exit, breakdown restarts and the final polish iteration -- runs on the device: no
// host round trip per iteration (the paper's loop reads the error on the host every sweep,
// L535-539).
//
// Formulation.  Right preconditioning with M = diag(A) (van der Vorst's p^ = M^-1 p, s^ = M^-1 s;
// r is the residual of the unpreconditioned system) is carried in SCALED VECTORS: the planes hold
// r^ = M^-1 r, p^ = M^-1 p, v^ = M^-1 v, t^ = M^-1 t.  Every recurrence of the method is linear, so
// it holds unchanged between the scaled vectors; the operator input (p^, s^) is then read as stored
// and the output is divided by the diagonal of its OWN row only, so no neighbour's diagonal is ever
// needed and the rows of A can be recomputed on the fly from the two cell planes h and z = 2 eta - h
// (S8; ~55 flops per node and apply) instead of being read as four stored coefficient planes.  The
// iterate is x itself (x += alpha p^ + omega s^).  Dot products are those of the UNSCALED vectors
// (t.s = sum A_C^2 t^ s^ ...), so alpha, omega, beta, the residual norm and hence the iterates are
// the ones of the textbook right-preconditioned method up to rounding.
//
// Two passes over memory per iteration (d = one double per node):
//   pass B : s^ = r^ - alpha v^;  t = A s^;  dots t.s, t.t, s.s, r0.s, r0.t
//            reads r^, v^, r0, h, z   writes t^                                        6 d
//   pass CA: s^ = r^ - alpha v^;  x += alpha p^ + omega s^;  r^' = s^ - omega t^;
//            p^' = r^' + beta (p^ - omega v^);  v' = A p^';  dots r0.v', r'.r'
//            reads r^, v^, t^, p^, x, r0, h, z   writes x, r^', p^', v^'              12 d
// with rho' = r0.s - omega r0.t (R25), so that every scalar of iteration i+1 is known after pass B
// of iteration i and the x/r update of iteration i shares its pass with the p/v update of
// iteration i+1.  s is never stored.  r^, p^, v^ are double-buffered (a pass reads the old planes
// with their halo and writes the new ones).  18 d = 144 B per node-iteration (the stored-matrix
// version of round 1 moved 22 d = 176 B).
//
// Sweep geometry ("marching warps").  Node planes are stored with a ghost ring (4 columns left,
// >= 2 right, 2 rows above and below; pitch NP a multiple of 16, so every strip starts on a 32-byte
// sector and every row on a 128-byte line, nh_internal.cuh) whose
// distance-1 ghosts hold the mirrored / wrapped images of the boundary nodes (R10); the writer of
// a boundary node stores its images, so no pass ever maps an index.  A warp owns a strip of 60
// columns and marches down a band of R rows: lane l holds columns 60 s - 2 + 2 l and the next one
// (one 16-byte load per plane per row), lanes 0 and 31 are halo lanes, the rows j-1, j, j+1 of the
// stencil operand and the cell rows the coefficients need live in registers, east/west neighbours
// come from warp shuffles.  No shared memory tiles, no block-level synchronisation inside a pass;
// all global accesses are coalesced 512-byte row segments.
//
// Dot products are two-stage and deterministic: per-CTA partials in a fixed order, one grid
// barrier, then every CTA sums all partials in the same order, so all CTAs take every branch
// alike.  Partials are double-buffered: one grid barrier per pass.
#include <cooperative_groups.h>
#include <math.h>
#include <stdio.h>

#include "nh_internal.cuh"

namespace cg = cooperative_groups;

namespace NH_NS {
namespace {

#define D(x) ((double)(x))  // dot products, norms and the scalars of the method are fp64 in both builds

#ifndef NH_NT
#define NH_NT 192
#endif
#ifndef NH_MINB
#define NH_MINB 2
#endif
constexpr int NT = NH_NT, NW = NT / 32;  // CTA size, warps per CTA
constexpr int SW = 60;                 // owned columns per warp strip
constexpr int MAXDOT = 5;
// small grids: at least this many rows per warp before CTAs are added (a warp marches its rows one
// memory latency at a time; us per iteration at 512 x 8 / 256^2 / 512^2: 4 rows 13.8 / 14.3 / 17.4,
// 2 rows 10.5 / 11.9 / 15.6, 1 row 8.5 / 11.3 / 15.6; no effect from 1024^2 up)
#ifndef NH_MINROWS
#define NH_MINROWS 1
#endif

struct SolveP {
  NhGrid G;
  int nstrips, R, nbands;  // strips of SW columns, band height, bands
  const real *hc, *zc;   // cell planes h, z = 2 eta - h of U* (node layout shifted by one column)
  const real* b;
  real* x;               // the iterate: start vector in, solution out (the pressure plane)
  real *r0, *t;          // shadow residual (unscaled); t^
  real *rA, *rB, *pA, *pB, *vA, *vB;  // r^, p^, v^ (double-buffered)
  double* part;  // [2][MAXDOT][gridDim.x]
  NhScal* sc;
  double rtol;
  real mx2, my2;  // -1 / (16 dx^2), -1 / (16 dy^2)
  int maxit;
  int count_stats;
};

__device__ __forceinline__ size_t nidx(const NhGrid& G, int I, int J) {
  return (size_t)((long long)J * G.np + I);
}

// ghost image of a real node line (distance-1 ghosts only): -2 = none.  Mirror (wall / outflow):
// line 1 -> ghost -1, line n-2 -> ghost n; periodic: line n-1 -> ghost -1, line 0 -> ghost n
// (n = number of distinct lines; R10).
__device__ __forceinline__ int ghost_image(int I, int n, int bclo) {
  if (bclo == NH_BC_PERIODIC) {
    if (I == n - 1) return -1;
    if (I == 0) return n;
    return -2;
  }
  if (I == 1) return -1;
  if (I == n - 2) return n;
  return -2;
}

// store a real node value and its ghost images (slow path: boundary nodes only)
__device__ __forceinline__ void store_images(const NhGrid& G, real* a, int I, int J, real v) {
  int gi = ghost_image(I, G.nnx, G.bxlo), gj = ghost_image(J, G.nny, G.bylo);
  a[nidx(G, I, J)] = v;
  if (gi != -2) a[nidx(G, gi, J)] = v;
  if (gj != -2) a[nidx(G, I, gj)] = v;
}

// per-CTA partials of K values into part[buf][k][cta] (fixed order: lanes by shuffle tree, warps
// in index order)
template <int K>
__device__ __forceinline__ void block_partials(const double (&v)[K], double* part, int buf,
                                               double (*red)[NW]) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < K; ++k) {
    double a = v[k];
    for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
    if (lane == 0) red[k][wid] = a;
  }
  __syncthreads();
  if (threadIdx.x < K) {
    double a = 0.0;
#pragma unroll
    for (int w = 0; w < NW; ++w) a += red[threadIdx.x][w];
    part[((size_t)buf * MAXDOT + threadIdx.x) * gridDim.x + blockIdx.x] = a;
  }
  __syncthreads();
}

// every CTA sums all partials in the same fixed order -> bit-identical scalars everywhere.
// Warp k sums the partials of value k (lane-strided loads all in flight at once, then a shuffle
// tree): one load latency and one block barrier per call (the first version summed the K values one
// after the other with three block barriers: 4 us per pass, half of an iteration on small grids).
template <int K>
__device__ __forceinline__ void grid_sums(const double* part, int buf, double (&out)[K],
                                          double (*red)[NW], double* bc) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int nb = gridDim.x;
  for (int k = wid; k < K; k += NW) {
    const double* src = part + ((size_t)buf * MAXDOT + k) * nb;
    double a = 0.0;
    for (int i = lane; i < nb; i += 32) a += __ldcg(&src[i]);
    for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
    if (lane == 0) bc[k] = a;
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < K; ++k) out[k] = bc[k];
  __syncthreads();  // bc is reused by the next call
}

// ---- marching-warp geometry ----------------------------------------------------------------
struct Unit {
  int c0;        // first of the lane's two columns (even; may be a ghost / padding column)
  int Ja, Jb;    // owned rows [Ja, Jb)
  bool own0, own1;  // the lane owns column c0 / c0+1 (real node of this strip)
  int g0, g1;       // ghost column holding the image of owned column c0 / c0+1 (-2: none)
};

__device__ __forceinline__ Unit make_unit(const SolveP& P, int u, int lane) {
  Unit U;
  int strip = u % P.nstrips, band = u / P.nstrips;
  U.c0 = strip * SW - 2 + 2 * lane;
  U.Ja = band * P.R;
  U.Jb = min(U.Ja + P.R, P.G.nny);
  bool inner = (lane >= 1) && (lane <= 30);
  U.own0 = inner && U.c0 < P.G.nnx;
  U.own1 = inner && U.c0 + 1 < P.G.nnx;
  U.g0 = U.own0 ? ghost_image(U.c0, P.G.nnx, P.G.bxlo) : -2;
  U.g1 = U.own1 ? ghost_image(U.c0 + 1, P.G.nnx, P.G.bxlo) : -2;
  return U;
}

// 16-byte load of the lane's column pair of row j
__device__ __forceinline__ real2 ld2(const real* a, const NhGrid& G, int c0, int j) {
  return *reinterpret_cast<const real2*>(a + nidx(G, c0, j));
}

// store the lane's pair of row j (owned columns only) and its ghost images: the same pair again on
// the ghost row of a boundary row, single values on the ghost column of a boundary column (the
// warps of the first and last strip used to take a scalar path for every row and finished 8 %
// (8192^2) to 34 % (2048^2) after the others, which every pass then waited for)
__device__ __forceinline__ void st2(real* a, const SolveP& P, const Unit& U, int j, real2 v) {
  const NhGrid& G = P.G;
  const int gj = ghost_image(j, G.nny, G.bylo);
  if (U.own1) {  // own1 implies own0
    *reinterpret_cast<real2*>(a + nidx(G, U.c0, j)) = v;
    if (gj != -2) *reinterpret_cast<real2*>(a + nidx(G, U.c0, gj)) = v;
  } else if (U.own0) {
    a[nidx(G, U.c0, j)] = v.x;
    if (gj != -2) a[nidx(G, U.c0, gj)] = v.x;
  }
  if (U.g0 != -2) a[nidx(G, U.g0, j)] = v.x;
  if (U.g1 != -2) a[nidx(G, U.g1, j)] = v.y;
}

// ---- matrix-free rows of A on the march ("coefficients are computed on the fly") ----
// The cell planes hc, zc (h and z = 2 eta - h of U*, written once per stage by k_cell_planes) use
// the node layout shifted by one column: plane column P holds cell P - 1, ghost cells filled through
// the cell index maps (R9).  The lane that owns nodes c0, c0+1 loads cells c0-1, c0 as its own pair
// and gets cell c0+1 from the next lane: k = 0, 1, 2 below.  Node A = c0 lies between the cell
// columns k = 0 (west) and 1 (east), node B = c0+1 between k = 1 and 2.  A warp keeps the cell rows
// J-1, J (and z of row J+1, xi^y of row J-1) in registers while it marches: per sweep step one row
// of h and one of z are loaded, 16 bytes per node instead of the 32 of four stored coefficients.
#define NH_FULL 0xffffffffu
struct Coef {  // row of A at the lane's two nodes: A_E, A_W, A_N, A_S, A_C (S8)
  real e[2], w[2], n[2], s[2], c[2];
};
__device__ __forceinline__ void lane3(real2 own, real (&q)[3]) {
  q[0] = own.x; q[1] = own.y; q[2] = __shfl_down_sync(NH_FULL, own.x, 1);
}
struct March {
  // S = cell row J-1, N = cell row J.  Carried between sweep steps: the raw rows h(J-1), z(J-1), z(J)
  // (column sums), and the row-pair sums of row J-1 at the lane's two nodes (they were the "north"
  // sums of the previous step): h, z, and dz2 = z(J) - z(J-2) = 2 xi^y of row J-1.
  real hS[3], zS[3], zN[3];
  real hSr[2], zSr[2], tS[2];
  // state for the first node row Ja of a band
  __device__ __forceinline__ void start(const SolveP& P, int c0, int Ja) {
    real zSS[3];
    lane3(ld2(P.zc, P.G, c0, Ja - 2), zSS);
    lane3(ld2(P.zc, P.G, c0, Ja - 1), zS);
    lane3(ld2(P.zc, P.G, c0, Ja), zN);
    lane3(ld2(P.hc, P.G, c0, Ja - 1), hS);
#pragma unroll
    for (int n = 0; n < 2; ++n) {
      hSr[n] = hS[n] + hS[n + 1];
      zSr[n] = zS[n] + zS[n + 1];
      tS[n] = (zN[n] - zSS[n]) + (zN[n + 1] - zSS[n + 1]);
    }
  }
  // rows of A at node row J from the cell rows h(J) and z(J+1) just loaded, then roll to J+1.
  // S8 with the sums shared between the two nodes and the factors 1/2, 1/4 folded into the
  // multipliers: 2 h_E = h_NE + h_SE is a column sum (sh), 4 xi_E the difference of the z column
  // sums two cells apart, 2 h_N a row sum, 4 xi_N the row-pair sum of z(J+1) - z(J-1);
  // mx2 = -1 / (16 dx^2), my2 = -1 / (16 dy^2).
  __device__ __forceinline__ Coef step(const SolveP& P, real2 hrow, real2 zrow) {
    real hN[3], zNN[3], sh[3], sz[3];
    lane3(hrow, hN);
    lane3(zrow, zNN);
#pragma unroll
    for (int k = 0; k < 3; ++k) { sh[k] = hS[k] + hN[k]; sz[k] = zS[k] + zN[k]; }
    const real szm = __shfl_up_sync(NH_FULL, sz[1], 1), szp = __shfl_down_sync(NH_FULL, sz[1], 1);
    const real x4[3] = {sz[1] - szm, sz[2] - sz[0], szp - sz[1]};  // 4 xi of the three cell columns
    const real q = RC(0.25);
    Coef C;
#pragma unroll
    for (int n = 0; n < 2; ++n) {
      const real a = sh[n] + sh[n + 1];   // 4 h_n, (38)
      const real bx = sz[n + 1] - sz[n];  // 2 (z_E - z_W)
      const real am = (a - bx) * P.mx2, ap = (a + bx) * P.mx2;
      C.e[n] = am * fma(q, x4[n + 1], sh[n + 1]);
      C.w[n] = ap * fma(-q, x4[n], sh[n]);
      const real cx = fma(am, fma(-q, x4[n + 1], sh[n + 1]), ap * fma(q, x4[n], sh[n]));
      const real hNr = hN[n] + hN[n + 1], zNr = zN[n] + zN[n + 1];
      const real tN = (zNN[n] - zS[n]) + (zNN[n + 1] - zS[n + 1]);  // 4 xi_N
      const real by = zNr - zSr[n];                                 // 2 (z_N - z_S)
      const real bm = (a - by) * P.my2, bp = (a + by) * P.my2;
      C.n[n] = bm * fma(q, tN, hNr);
      C.s[n] = bp * fma(-q, tS[n], hSr[n]);
      const real cy = fma(bm, fma(-q, tN, hNr), bp * fma(q, tS[n], hSr[n]));
      C.c[n] = RC(2.0) - (cx + cy);
      hSr[n] = hNr; zSr[n] = zNr; tS[n] = tN;
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) { hS[k] = hN[k]; zS[k] = zN[k]; zN[k] = zNN[k]; }
    return C;
  }
};

// 1 / a for a >= 2 (the diagonal of A): hardware seed (20+ bits) and two Newton steps.  Not correctly
// rounded; the scaling only has to be the same number wherever a node's diagonal is used.
#if NH_PREC == 64
__device__ __forceinline__ double rcp_diag(double a) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a));
  double e = fma(-a, r, 1.0);
  r = fma(r, e, r);
  e = fma(-a, r, 1.0);
  return fma(r, e, r);
}
#else
__device__ __forceinline__ float rcp_diag(float a) { return __frcp_rn(a); }
#endif

// off-diagonal part of (A x) at the lane's two nodes of row j from the operand rows m: j-1, c: j, n: j+1
__device__ __forceinline__ real2 offdiag2(const Coef& C, real2 m, real2 c, real2 n) {
  const real west0 = __shfl_up_sync(NH_FULL, c.y, 1);
  const real east1 = __shfl_down_sync(NH_FULL, c.x, 1);
  real2 o;
  o.x = fma(C.s[0], m.x, fma(C.n[0], n.x, fma(C.w[0], west0, C.e[0] * c.y)));
  o.y = fma(C.s[1], m.y, fma(C.n[1], n.y, fma(C.w[1], c.x, C.e[1] * east1)));
  return o;
}

// Every pass is software-pipelined by hand: the loads of the NEXT row are issued before the current
// row is computed and stored (the compiler cannot hoist them itself across the stores of possibly
// aliasing planes), so each warp keeps one full row of every plane in flight while it computes.

#define NH_STR_(x) #x
#define NH_STR(x) NH_STR_(x)
#ifndef NH_UNROLL
#define NH_UNROLL 2  // sweep loops unrolled by two: the rolling rows need no register moves (-2 %)
#endif

// residual pass: r = b - A x (S9: the true residual decides), r0 = r, r^ = r / A_C; partials r.r, b.b
__device__ __forceinline__ void pass_R(const SolveP& P, real* rh, int buf, double (*red)[NW]) {
  const NhGrid& G = P.G;
  const int lane = threadIdx.x & 31;
  const int gw = blockIdx.x * NW + (threadIdx.x >> 5), tw = gridDim.x * NW;
  const int nunits = P.nstrips * P.nbands;
  double acc[2] = {0.0, 0.0};
  for (int k = gw; k < nunits; k += tw) {
    Unit U = make_unit(P, k, lane);
    March M;
    M.start(P, U.c0, U.Ja);
    real2 xm = ld2(P.x, G, U.c0, U.Ja - 1), xc = ld2(P.x, G, U.c0, U.Ja);
    for (int j = U.Ja; j < U.Jb; ++j) {
      const real2 xn = ld2(P.x, G, U.c0, j + 1), bb = ld2(P.b, G, U.c0, j);
      const Coef C = M.step(P, ld2(P.hc, G, U.c0, j), ld2(P.zc, G, U.c0, j + 1));
      const real2 off = offdiag2(C, xm, xc, xn);
      const real2 rr = make_real2(bb.x - fma(C.c[0], xc.x, off.x), bb.y - fma(C.c[1], xc.y, off.y));
      st2(P.r0, P, U, j, rr);
      st2(rh, P, U, j, make_real2(rr.x * rcp_diag(C.c[0]), rr.y * rcp_diag(C.c[1])));
      if (U.own0) { acc[0] = fma(D(rr.x), D(rr.x), acc[0]); acc[1] = fma(D(bb.x), D(bb.x), acc[1]); }
      if (U.own1) { acc[0] = fma(D(rr.y), D(rr.y), acc[0]); acc[1] = fma(D(bb.y), D(bb.y), acc[1]); }
      xm = xc; xc = xn;
    }
  }
  block_partials<2>(acc, P.part, buf, red);
}

// pass B: s^ = r^ - alpha v^ (rows Ja-1..Jb), t = A s^ (rows Ja..Jb-1), stored as t^ = t / A_C;
// partials of the unscaled vectors: t.s, t.t, s.s, r0.s, r0.t
struct RowB {  // operands of sweep step j: r^, v^ of row j+1; r0, h of row j; z of row j+1
  real2 r, v, q, h, z;
};
__device__ __forceinline__ void ld_rowb(RowB& X, const SolveP& P, const real* r, const real* v,
                                        int c0, int j) {
  X.r = ld2(r, P.G, c0, j + 1); X.v = ld2(v, P.G, c0, j + 1);
  X.q = ld2(P.r0, P.G, c0, j);
  X.h = ld2(P.hc, P.G, c0, j); X.z = ld2(P.zc, P.G, c0, j + 1);
}

__device__ __forceinline__ void pass_B(const SolveP& P, real alpha, const real* r, const real* v,
                                    int buf, double (*red)[NW]) {
  const NhGrid& G = P.G;
  const int lane = threadIdx.x & 31;
  const int gw = blockIdx.x * NW + (threadIdx.x >> 5), tw = gridDim.x * NW;
  const int nunits = P.nstrips * P.nbands;
  double acc[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
  for (int k = gw; k < nunits; k += tw) {
    Unit U = make_unit(P, k, lane);
    auto srow = [&](real2 a, real2 b) {
      return make_real2(fma(-alpha, b.x, a.x), fma(-alpha, b.y, a.y));
    };
    March M;
    M.start(P, U.c0, U.Ja);
    real2 sm = srow(ld2(r, G, U.c0, U.Ja - 1), ld2(v, G, U.c0, U.Ja - 1));
    real2 sc = srow(ld2(r, G, U.c0, U.Ja), ld2(v, G, U.c0, U.Ja));
    // One operand set; the loads of step j+1 are issued as soon as step j has moved its operands
    // into the marching state, before the arithmetic of the step (row index clamped: the last
    // request is never used).
    RowB X;
    ld_rowb(X, P, r, v, U.c0, U.Ja);
    _Pragma(NH_STR(unroll NH_UNROLL))
    for (int j = U.Ja; j < U.Jb; ++j) {
      const real2 sn = srow(X.r, X.v);
      const real2 q = X.q;
      const Coef C = M.step(P, X.h, X.z);
      if (j + 1 < U.Jb) ld_rowb(X, P, r, v, U.c0, j + 1);
      const real2 off = offdiag2(C, sm, sc, sn);
      const real2 tu = make_real2(fma(C.c[0], sc.x, off.x), fma(C.c[1], sc.y, off.y));  // t
      const real2 su = make_real2(C.c[0] * sc.x, C.c[1] * sc.y);                        // s
      st2(P.t, P, U, j, make_real2(fma(rcp_diag(C.c[0]), off.x, sc.x), fma(rcp_diag(C.c[1]), off.y, sc.y)));
      if (U.own0) {
        acc[0] = fma(D(tu.x), D(su.x), acc[0]); acc[1] = fma(D(tu.x), D(tu.x), acc[1]);
        acc[2] = fma(D(su.x), D(su.x), acc[2]);
        acc[3] = fma(D(q.x), D(su.x), acc[3]); acc[4] = fma(D(q.x), D(tu.x), acc[4]);
      }
      if (U.own1) {
        acc[0] = fma(D(tu.y), D(su.y), acc[0]); acc[1] = fma(D(tu.y), D(tu.y), acc[1]);
        acc[2] = fma(D(su.y), D(su.y), acc[2]);
        acc[3] = fma(D(q.y), D(su.y), acc[3]); acc[4] = fma(D(q.y), D(tu.y), acc[4]);
      }
      sm = sc; sc = sn;
    }
  }
  block_partials<5>(acc, P.part, buf, red);
}

// pass CA: FIRST: p^' = r^' = r^ (start of a cycle).  Otherwise s^ = r^ - alpha v^;
// x += alpha p^ + omega s^; r^' = s^ - omega t^; p^' = r^' + beta (p^ - omega v^).  Then v' = A p^',
// stored as v^' = v' / A_C.  partials of the unscaled vectors: r0.v', r'.r'
struct RowV {  // vector row of pass CA
  real2 r, v, t, p, x;
};
template <bool FIRST>
__device__ __forceinline__ void ld_rowv(RowV& V, const SolveP& P, const real* r, const real* p,
                                        const real* v, int c0, int j) {
  V.r = ld2(r, P.G, c0, j);
  if (!FIRST) {
    V.v = ld2(v, P.G, c0, j); V.t = ld2(P.t, P.G, c0, j);
    V.p = ld2(p, P.G, c0, j); V.x = ld2(P.x, P.G, c0, j);
  }
}
struct RowCA {  // operands of sweep step j: vectors of row j+1; r0, h of row j; z of row j+1
  RowV V;
  real2 q, h, z;
};

template <bool FIRST>
__device__ __forceinline__ void pass_CA(const SolveP& P, real alpha, real omega, real beta,
                                     const real* r, const real* p, const real* v, real* rN,
                                     real* pN, real* vN, int buf, double (*red)[NW]) {
  const int lane = threadIdx.x & 31;
  const int gw = blockIdx.x * NW + (threadIdx.x >> 5), tw = gridDim.x * NW;
  const int nunits = P.nstrips * P.nbands;
  double acc[2] = {0.0, 0.0};
  for (int k = gw; k < nunits; k += tw) {
    Unit U = make_unit(P, k, lane);
    // new r^, p^, x of a row from its loaded operands
    auto vrow = [&](const RowV& V, real2& rn, real2& pn, real2& xx) {
      if (FIRST) {
        rn = V.r; pn = V.r; xx = V.r;
      } else {
        const real2 s = make_real2(fma(-alpha, V.v.x, V.r.x), fma(-alpha, V.v.y, V.r.y));
        rn = make_real2(fma(-omega, V.t.x, s.x), fma(-omega, V.t.y, s.y));
        pn = make_real2(fma(beta, fma(-omega, V.v.x, V.p.x), rn.x),
                          fma(beta, fma(-omega, V.v.y, V.p.y), rn.y));
        xx = make_real2(V.x.x + fma(omega, s.x, alpha * V.p.x), V.x.y + fma(omega, s.y, alpha * V.p.y));
      }
    };
    auto store_row = [&](int j, real2 rn, real2 pn, real2 xx) {
      if (!FIRST) st2(P.x, P, U, j, xx);
      st2(rN, P, U, j, rn);
      st2(pN, P, U, j, pn);
    };
    auto ld_set = [&](RowCA& X, int j) {
      ld_rowv<FIRST>(X.V, P, r, p, v, U.c0, j + 1);
      X.q = ld2(P.r0, P.G, U.c0, j);
      X.h = ld2(P.hc, P.G, U.c0, j); X.z = ld2(P.zc, P.G, U.c0, j + 1);
    };
    March M;
    M.start(P, U.c0, U.Ja);
    real2 pm, pc, rc;  // p^' of rows j-1, j; r^' of row j (its A_C is known one step later)
    {
      RowV V0, V1;
      ld_rowv<FIRST>(V0, P, r, p, v, U.c0, U.Ja - 1);
      ld_rowv<FIRST>(V1, P, r, p, v, U.c0, U.Ja);
      real2 r0_, x0_, x1_;
      vrow(V0, r0_, pm, x0_);
      vrow(V1, rc, pc, x1_);
      store_row(U.Ja, rc, pc, x1_);
    }
    // One operand set; the loads of step j+1 are issued as soon as step j has consumed its operands,
    // BEFORE its stores (ghost-image logic included) and its dot-product terms, which then run in
    // the shadow of the memory latency.
    RowCA X;
    ld_set(X, U.Ja);
    _Pragma(NH_STR(unroll NH_UNROLL))
    for (int j = U.Ja; j < U.Jb; ++j) {
      const bool own_next = j + 1 < U.Jb;
      real2 rn, pn, xx;
      vrow(X.V, rn, pn, xx);
      const Coef C = M.step(P, X.h, X.z);
      const real2 q = X.q;
      if (own_next) ld_set(X, min(j + 1, U.Jb - 1));  // operands of the next step
      const real2 off = offdiag2(C, pm, pc, pn);
      const real2 vu = make_real2(fma(C.c[0], pc.x, off.x), fma(C.c[1], pc.y, off.y));  // v'
      if (own_next) store_row(j + 1, rn, pn, xx);
      st2(vN, P, U, j, make_real2(fma(rcp_diag(C.c[0]), off.x, pc.x), fma(rcp_diag(C.c[1]), off.y, pc.y)));
      const real2 ru = make_real2(C.c[0] * rc.x, C.c[1] * rc.y);  // r' of row j
      if (U.own0) { acc[0] = fma(D(q.x), D(vu.x), acc[0]); acc[1] = fma(D(ru.x), D(ru.x), acc[1]); }
      if (U.own1) { acc[0] = fma(D(q.y), D(vu.y), acc[0]); acc[1] = fma(D(ru.y), D(ru.y), acc[1]); }
      pm = pc; pc = pn; rc = rn;
    }
  }
  block_partials<2>(acc, P.part, buf, red);
}

// ---- simple phases (a handful per solve): rows over CTAs, columns over threads --------------
// ghost images of the start vector
__device__ void phase_images(const SolveP& P) {
  const NhGrid& G = P.G;
  for (int J = blockIdx.x; J < G.nny; J += gridDim.x)
    for (int I = threadIdx.x; I < G.nnx; I += NT) store_images(G, P.x, I, J, P.x[nidx(G, I, J)]);
}

// x += alpha p^ + omega s^, s^ = r^ - alpha v^  (final update of an iteration whose pass CA never
// ran: half-step exit with omega = 0, and the polish iteration)
__device__ void phase_update_x(const SolveP& P, real alpha, real omega, const real* r,
                               const real* p, const real* v) {
  const NhGrid& G = P.G;
  for (int J = blockIdx.x; J < G.nny; J += gridDim.x)
    for (int I = threadIdx.x; I < G.nnx; I += NT) {
      size_t k = nidx(G, I, J);
      real s = r[k] - alpha * v[k];
      store_images(G, P.x, I, J, P.x[k] + (alpha * p[k] + omega * s));
    }
}

__device__ void phase_zero_x(const SolveP& P) {
  const NhGrid& G = P.G;
  for (int J = blockIdx.x; J < G.nny; J += gridDim.x)
    for (int I = threadIdx.x; I < G.nnx; I += NT) store_images(G, P.x, I, J, RC(0.0));
}

__global__ void __launch_bounds__(NT, NH_MINB) k_bicgstab(SolveP P) {
  cg::grid_group grid = cg::this_grid();
  __shared__ double red[MAXDOT][NW];
  __shared__ double bc[MAXDOT];

  real *rC = P.rA, *rN = P.rB, *pC = P.pA, *pN = P.pB, *vC = P.vA, *vN = P.vB;  // current / next
  auto flip = [&]() {
    real* t;
    t = rC; rC = rN; rN = t;
    t = pC; pC = pN; pN = t;
    t = vC; vC = vN; vN = t;
  };
  int buf = 0;  // partial buffer of the pass in flight (alternates: one grid barrier per pass)
  int iters = 0, converged = 0, status = 0, stagnated = 0;
  double rnorm = 0.0, bnorm = 0.0, tol = 0.0, rnorm_prev = 0.0;

  phase_images(P);
  grid.sync();
  for (int cycle = 0; cycle < 8 && !converged; ++cycle) {
    double d2[2], d5[5];
    pass_R(P, rC, buf, red);
    grid.sync();
    grid_sums<2>(P.part, buf, d2, red, bc);
    buf ^= 1;
    rnorm = sqrt(d2[0]);
    if (cycle == 0) {
      bnorm = sqrt(d2[1]);
      if (!(bnorm == bnorm) || isinf(bnorm)) { status = NH_ENAN; break; }
      if (bnorm == 0.0) break;
      tol = P.rtol * bnorm;
    }
    if (!(rnorm == rnorm)) { status = NH_ENAN; break; }
    if (rnorm <= tol) { converged = 1; break; }
    // fp32 variant: an fp32 iterate cannot satisfy the system better than ~ kappa u32 ||b||.  When a
    // whole cycle (recursive residual below tol) no longer halves the TRUE residual, the attainable
    // accuracy has been reached: accept the iterate; res_last reports what was reached, and because
    // that residual is ABOVE the tolerance the acceptance is flagged (NH_FLAG_STAGNATED, nh_info.flags
    // bit 3): a breakdown that stalls at 1e-2 must not look like a solve that met 1e-4.
    if (kEta && cycle > 0 && rnorm > 0.5 * rnorm_prev) { converged = 1; stagnated = 1; break; }
    rnorm_prev = rnorm;
    if (iters >= P.maxit) break;
    // first direction of the cycle: p = r, v = A M^-1 p, sigma = r0.v
    double rho = d2[0];
    pass_CA<true>(P, RC(0.0), RC(0.0), RC(0.0), rC, pC, vC, rN, pN, vN, buf, red);
    flip();
    grid.sync();
    grid_sums<2>(P.part, buf, d2, red, bc);
    buf ^= 1;
    double sigma = d2[0];
    while (iters < P.maxit) {
      if (fabs(rho) < 1e-300 || fabs(sigma) < 1e-300) break;  // breakdown -> restart
      double alpha = rho / sigma;
      iters++;
      pass_B(P, (real)alpha, rC, vC, buf, red);
      grid.sync();
      grid_sums<5>(P.part, buf, d5, red, bc);
      buf ^= 1;
      if (sqrt(d5[2]) <= tol) {  // half-step exit: x += alpha p^
        phase_update_x(P, (real)alpha, RC(0.0), rC, pC, vC);
        grid.sync();
        break;
      }
      if (d5[1] == 0.0) break;
      double omega = d5[0] / d5[1];
      if (fabs(omega) < 1e-300 || !(omega == omega)) break;
      double rho_new = d5[3] - omega * d5[4];  // r0.r' = r0.s - omega r0.t  (R25)
      double beta = (rho_new / rho) * (alpha / omega);
      rho = rho_new;
      pass_CA<false>(P, (real)alpha, (real)omega, (real)beta, rC, pC, vC, rN, pN, vN, buf, red);
      flip();
      grid.sync();
      grid_sums<2>(P.part, buf, d2, red, bc);
      buf ^= 1;
      sigma = d2[0];
      rnorm = sqrt(d2[1]);
      if (!(rnorm == rnorm)) break;
      if (rnorm <= tol) break;
    }
    // loop back: the true residual decides (the recursive residual may have drifted)
  }
  if (status == 0 && bnorm > 0.0 && !converged) status = NH_ENOCONV;

  // one extra "polish" iteration from the true residual (R14): r0 = r, p = r
  if (converged && rnorm > 0.0) {
    double d2[2], d5[5];
    double rho = rnorm * rnorm;
    pass_CA<true>(P, RC(0.0), RC(0.0), RC(0.0), rC, pC, vC, rN, pN, vN, buf, red);
    flip();
    grid.sync();
    grid_sums<2>(P.part, buf, d2, red, bc);
    buf ^= 1;
    double sigma = d2[0];
    if (fabs(rho) >= 1e-300 && fabs(sigma) >= 1e-300) {
      double alpha = rho / sigma;
      pass_B(P, (real)alpha, rC, vC, buf, red);
      grid.sync();
      grid_sums<5>(P.part, buf, d5, red, bc);
      buf ^= 1;
      double omega = (d5[1] > 0.0) ? d5[0] / d5[1] : 0.0;
      phase_update_x(P, (real)alpha, (real)omega, rC, pC, vC);
      grid.sync();
    }
  }
  if (status != NH_ENAN && bnorm == 0.0) phase_zero_x(P);  // b = 0 => p~ = 0, zero iterations

  if (blockIdx.x == 0 && threadIdx.x == 0) {
    NhScal* sc = P.sc;
    if (status == NH_ENOCONV) sc->flags |= NH_FLAG_NOCONV;
    if (status == NH_ENAN) sc->flags |= NH_FLAG_NAN;
    if (stagnated) sc->flags |= NH_FLAG_STAGNATED;
    sc->iters_last = iters;
    sc->res_last = (bnorm > 0.0) ? rnorm / bnorm : 0.0;
    if (P.count_stats) {
      sc->iters_total += iters;
      sc->solves += 1;
      if (iters > sc->iters_max) sc->iters_max = iters;
    }
  }
}

// ---- solver 1: the paper's Jacobi method with scheduled relaxation (L507-514, L535-539; R28) ----
// One persistent cooperative kernel per solve; one sweep and one grid barrier per iteration, no dot
// products.  Sweep k:  z = b' - (x + ((c_E x_E + c_W x_W) + c_N x_N) + c_S x_S)  (the increment of
// the plain Jacobi method), E_k = max |z| (eq. (32)), x' = x + omega_k z, with the row-scaled
// coefficients and b' of k_scale_rows.  Every operation is a plain IEEE multiply / add in the
// order the oracle uses (no FMA), a max is exact, and a Jacobi sweep does not depend on the sweep
// order: the iterates, the iteration count and E are bit-identical to the CPU oracle's.
// Traffic: reads x, b', 4 c; writes x': 7 doubles = 56 B per node-iteration.
constexpr int NT1 = 256, NW1 = NT1 / 32;  // CTA shape of k_srj (128 registers, 16 warps per SM)
struct SrjP {
  NhGrid G;
  int nstrips, R, nbands;
  const real *cE, *cW, *cN, *cS, *bp;
  const double* costab;
  real *xA, *xB;  // xA = the pressure plane p (start and result), xB = scratch
  NhScal* sc;
  double eps, rel;  // tolerance of (32): eps, or rel * max|b'| when rel > 0
  int maxit, mmax, count_stats;
};

__device__ __forceinline__ void srj_sweep(const SrjP& P, const SolveP& Q, real om, const real* x,
                                          real* xn, unsigned long long* Eslot) {
  const NhGrid& G = P.G;
  const int lane = threadIdx.x & 31;
  const int gw = blockIdx.x * NW1 + (threadIdx.x >> 5), tw = gridDim.x * NW1;
  const int nunits = P.nstrips * P.nbands;
  real emax = RC(0.0);
  bool bad = false;
  struct Row { real2 xn, b, e, w, n, s; };
  for (int u = gw; u < nunits; u += tw) {
    Unit U = make_unit(Q, u, lane);
    real2 xm = ld2(x, G, U.c0, U.Ja - 1), xc = ld2(x, G, U.c0, U.Ja);
    auto ld_row = [&](Row& X, int j) {  // operands of sweep step j (x of row j+1, the rest of row j)
      X.xn = ld2(x, G, U.c0, min(j + 1, U.Jb));
      const int jc = min(j, U.Jb - 1);
      X.b = ld2(P.bp, G, U.c0, jc);
      X.e = ld2(P.cE, G, U.c0, jc); X.w = ld2(P.cW, G, U.c0, jc);
      X.n = ld2(P.cN, G, U.c0, jc); X.s = ld2(P.cS, G, U.c0, jc);
    };
    auto step = [&](int j, Row& cur, Row& nxt) {
      ld_row(nxt, j + 1);  // request the next step's operands first
      real west0 = __shfl_up_sync(0xffffffffu, xc.y, 1);
      real east1 = __shfl_down_sync(0xffffffffu, xc.x, 1);
      real ax0 = xc.x + (((cur.e.x * xc.y + cur.w.x * west0) + cur.n.x * cur.xn.x) + cur.s.x * xm.x);
      real ax1 = xc.y + (((cur.e.y * east1 + cur.w.y * xc.x) + cur.n.y * cur.xn.y) + cur.s.y * xm.y);
      real z0 = cur.b.x - ax0, z1 = cur.b.y - ax1;
      if (U.own0) { emax = fmax(emax, fabs(z0)); bad |= !(z0 == z0); }
      if (U.own1) { emax = fmax(emax, fabs(z1)); bad |= !(z1 == z1); }
      st2(xn, Q, U, j, make_real2(xc.x + om * z0, xc.y + om * z1));
      xm = xc; xc = cur.xn;
    };
    Row A, B;
    ld_row(A, U.Ja);
    for (int j = U.Ja; j < U.Jb; j += 2) {
      step(j, A, B);
      if (j + 1 < U.Jb) step(j + 1, B, A);
    }
  }
  // CTA max -> one integer atomicMax (exact, order independent)
  for (int o = 16; o > 0; o >>= 1) emax = fmax(emax, __shfl_xor_sync(0xffffffffu, emax, o));
  __shared__ real wmax[NW1];
  if (lane == 0) wmax[threadIdx.x >> 5] = emax;
  int anybad = __syncthreads_or(bad);
  if (threadIdx.x == 0) {
    real m = RC(0.0);
#pragma unroll
    for (int w = 0; w < NW1; ++w) m = fmax(m, wmax[w]);
    if (m > RC(0.0)) atomicMax(Eslot, (unsigned long long)__double_as_longlong((double)m));
    if (anybad) atomicOr(&P.sc->srj_bad, 1);
  }
}

#ifndef NH_SRJ_MINB
#define NH_SRJ_MINB 2
#endif
__global__ void __launch_bounds__(NT1, NH_SRJ_MINB) k_srj(SrjP P) {
  cg::grid_group grid = cg::this_grid();
  const NhGrid& G = P.G;
  NhScal* sc = P.sc;
  SolveP Q;  // geometry view for make_unit / st2
  Q.G = P.G; Q.nstrips = P.nstrips; Q.R = P.R; Q.nbands = P.nbands;
  const double rho = __longlong_as_double((long long)sc->srj_rho_bits);
  const double bmax = __longlong_as_double((long long)sc->srj_bmax_bits);
  int iters = 0, status = 0;
  double E = 0.0;
  real *x = P.xA, *xn = P.xB;
  if (!(bmax == bmax) || isinf(bmax)) {
    status = NH_ENAN;
  } else if (bmax == 0.0) {  // b = 0 => p~ = 0, zero iterations (same convention as solver 0)
    for (int J = blockIdx.x; J < G.nny; J += gridDim.x)
      for (int I = threadIdx.x; I < G.nnx; I += NT1) P.xA[nidx(G, I, J)] = RC(0.0);
  } else {
    // cycle length: smallest power of two with M sqrt(2 (1 - rho)) >= 7.6, at most mmax.  Where a
    // row is not strictly diagonally dominant (rho >= 1, e.g. across a discontinuous free surface)
    // there is no interval to place Chebyshev nodes on: plain Jacobi (one factor, 1).
    const bool dominant = rho < 1.0;
    const double gap = dominant ? sqrt(2.0 * (1.0 - rho)) : 0.0;
    int M = 1;
    if (dominant)
      while (M < P.mmax && (double)M * gap < 7.6) M *= 2;
    const double* cosv = P.costab + (M - 1);
    const double tol = (P.rel > 0.0) ? P.rel * bmax : P.eps;
    // ghost images of the start vector
    for (int J = blockIdx.x; J < G.nny; J += gridDim.x)
      for (int I = threadIdx.x; I < G.nnx; I += NT1) store_images(G, x, I, J, x[nidx(G, I, J)]);
    grid.sync();
    for (;;) {
      const double om = dominant ? 1.0 / (1.0 - rho * cosv[iters % M]) : 1.0;
      unsigned long long* slot = &sc->srj_E_bits[iters % 3];
      srj_sweep(P, Q, (real)om, x, xn, slot);
      grid.sync();
      E = __longlong_as_double((long long)__ldcg(slot));
      const int bad = __ldcg(&sc->srj_bad);
      if (blockIdx.x == 0 && threadIdx.x == 0) sc->srj_E_bits[(iters + 2) % 3] = 0ULL;
      if (bad) { status = NH_ENAN; break; }
      if (E < tol) break;  // eq. (32): x is the accepted iterate
      if (iters >= P.maxit) { status = NH_ENOCONV; break; }
      real* t = x; x = xn; xn = t;
      iters++;
    }
    if (x != P.xA) {  // the accepted iterate lives in the scratch plane
      for (int J = blockIdx.x; J < G.nny; J += gridDim.x)
        for (int I = threadIdx.x; I < G.nnx; I += NT1) P.xA[nidx(G, I, J)] = x[nidx(G, I, J)];
    }
  }
  grid.sync();
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    if (status == NH_ENOCONV) sc->flags |= NH_FLAG_NOCONV;
    if (status == NH_ENAN) sc->flags |= NH_FLAG_NAN;
    sc->iters_last = iters;
    sc->res_last = E;
    if (P.count_stats) {
      sc->iters_total += iters;
      sc->solves += 1;
      if (iters > sc->iters_max) sc->iters_max = iters;
    }
    // reset the reductions for the next solve
    sc->srj_rho_bits = 0ULL; sc->srj_bmax_bits = 0ULL; sc->srj_bad = 0;
    sc->srj_E_bits[0] = sc->srj_E_bits[1] = sc->srj_E_bits[2] = 0ULL;
  }
}

}  // namespace

// Cooperative grid (one wave of co-resident CTAs) and the band height R: every warp takes the
// units u = gw, gw + tw, ... (strip fastest, so neighbouring warps sweep neighbouring strips of the
// same band); R minimises rounds x (R + 2 halo rows).
int nh_solver_setup(Ctx* c) {
  int occ = 0;
  cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_bicgstab, NT, 0);
  if (e != cudaSuccess || occ < 1) {
    snprintf(c->err, sizeof(c->err), "solver occupancy query failed: %s", cudaGetErrorString(e));
    return NH_ECUDA;
  }
  const int nnx = c->g.nnx, nny = c->g.nny;
  const int nstrips = (nnx + SW - 1) / SW;
  long long small_units = (long long)nstrips * ((nny + NH_MINROWS - 1) / NH_MINROWS);
  long long grid = (long long)occ * c->sm_count;
  if (grid > (small_units + NW - 1) / NW) grid = (small_units + NW - 1) / NW;
  if (grid < 1) grid = 1;
  const long long tw = grid * NW;
  int bestR = nny;
  long long best = -1;
  for (int R = NH_MINROWS; R <= nny; ++R) {
    long long nb = (nny + R - 1) / R;
    long long rounds = (nstrips * nb + tw - 1) / tw;
    long long cost = rounds * (R + 2);
    if (best < 0 || cost < best) { best = cost; bestR = R; }
  }
  if (nny < NH_MINROWS) bestR = nny;
  c->solver_occ = occ;
  c->solver_grid = (int)grid;
  c->solver_nstrips = nstrips;
  c->solver_R = bestR;
  c->solver_nbands = (nny + bestR - 1) / bestR;
  e = cudaMalloc(&c->part, sizeof(double) * 2 * MAXDOT * (size_t)grid);
  if (e != cudaSuccess) return NH_ENOMEM;
  c->srj_cos = nullptr;
  if (c->prm.solver == 1) {
    // solver 1: its own cooperative grid / band height, and the relaxation schedule:
    // cos(pi (2 perm_i - 1) / 2M) in Lebedev-Finogenov order for M = 1, 2, 4, ..., mmax (R28),
    // evaluated on the host so that the factors are the ones a CPU evaluation produces.
    int occ1 = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ1, k_srj, NT1, 0);
    if (e != cudaSuccess || occ1 < 1) {
      snprintf(c->err, sizeof(c->err), "srj occupancy query failed: %s", cudaGetErrorString(e));
      return NH_ECUDA;
    }
    long long g1 = (long long)occ1 * c->sm_count;
    if (g1 > (small_units + NW1 - 1) / NW1) g1 = (small_units + NW1 - 1) / NW1;
    if (g1 < 1) g1 = 1;
    const long long tw1 = g1 * NW1;
    int R1 = nny;
    long long best1 = -1;
    for (int R = NH_MINROWS; R <= nny; ++R) {
      long long nb = (nny + R - 1) / R;
      long long rounds = (nstrips * nb + tw1 - 1) / tw1;
      long long cost = rounds * (R + 2);
      if (best1 < 0 || cost < best1) { best1 = cost; R1 = R; }
    }
    if (nny < NH_MINROWS) R1 = nny;
    c->srj_grid = (int)g1; c->srj_R = R1; c->srj_nbands = (nny + R1 - 1) / R1;
    const int mmax = c->prm.srj_mmax;
    std::vector<double> tab((size_t)2 * mmax - 1);
    std::vector<int> perm((size_t)mmax);
    for (int M = 1; M <= mmax; M *= 2) {
      perm[0] = 1;
      for (int m = 1; m < M; m *= 2)
        for (int i = m - 1; i >= 0; --i) {
          int a = perm[i];
          perm[2 * i] = a; perm[2 * i + 1] = 2 * m + 1 - a;
        }
      for (int i = 0; i < M; ++i)
        tab[(size_t)(M - 1) + i] = cos(3.14159265358979323846 * (double)(2 * perm[i] - 1) / (double)(2 * M));
    }
    e = cudaMalloc(&c->srj_cos, sizeof(double) * tab.size());
    if (e != cudaSuccess) return NH_ENOMEM;
    e = cudaMemcpy(c->srj_cos, tab.data(), sizeof(double) * tab.size(), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return NH_ECUDA;
  }
  return NH_OK;
}

void nh_launch_solve(Ctx* c, const real* b, real* x, int count_stats) {
  if (c->prm.solver == 1) {  // b is c->kr = b / A_C here (nh_launch_scale_rows)
    SrjP S;
    S.G = c->g;
    S.nstrips = c->solver_nstrips; S.R = c->srj_R; S.nbands = c->srj_nbands;
    S.cE = c->cE; S.cW = c->cW; S.cN = c->cN; S.cS = c->cS; S.bp = c->kr; S.costab = c->srj_cos;
    S.xA = x; S.xB = c->ky; S.sc = c->sc; S.eps = c->prm.srj_eps; S.rel = c->prm.srj_rel;
    S.maxit = c->prm.solver_maxit; S.mmax = c->prm.srj_mmax; S.count_stats = count_stats;
    void* args[] = {&S};
    NH_CUDA_OK(c, cudaLaunchCooperativeKernel((void*)k_srj, dim3(c->srj_grid), dim3(NT1), args, 0,
                                              c->stream));
    c->launches++;
    return;
  }
  SolveP P;
  P.G = c->g;
  P.nstrips = c->solver_nstrips; P.R = c->solver_R; P.nbands = c->solver_nbands;
  P.hc = c->hc; P.zc = c->zc;
  P.b = b; P.x = x;
  P.r0 = c->kr0; P.t = c->kt;
  P.rA = c->kr; P.rB = c->krB; P.pA = c->kpA; P.pB = c->kpB; P.vA = c->kvA; P.vB = c->kvB;
  P.part = c->part; P.sc = c->sc; P.rtol = c->prm.solver_rtol; P.maxit = c->prm.solver_maxit;
  P.mx2 = (real)(-1.0 / (16.0 * (double)c->g.dx * (double)c->g.dx));
  P.my2 = (real)(-1.0 / (16.0 * (double)c->g.dy * (double)c->g.dy));
  P.count_stats = count_stats;
  void* args[] = {&P};
  NH_CUDA_OK(c, cudaLaunchCooperativeKernel((void*)k_bicgstab, dim3(c->solver_grid), dim3(NT), args,
                                            0, c->stream));
  c->launches++;
}

}  // namespace NH_NS
