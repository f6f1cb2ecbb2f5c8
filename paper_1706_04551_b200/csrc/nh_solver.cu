// nh_solver.cu -- a6: Jacobi-preconditioned BiCGStab (R14, R25) for the compact
// finite-difference pressure system (eqs (29), (36)-(43)) as ONE persistent
// cooperative kernel per solve.
//
// The whole solve -- true-residual (re)starts, the iteration loop with its convergence tests, the
// half-step exit, breakdown restarts and the final polish iteration -- runs on the device: no
// host round trip per iteration (the paper's loop reads the error on the host every sweep,
// L535-539).  Right preconditioning is folded into the operator: with M = diag(A) the iteration
// runs on A M^-1 (unit diagonal, column-scaled off-diagonals cE..cS prepared once per solve by
// k_scale_coeffs) with the iterate y = M x; r is the residual of the
// unpreconditioned system.
//
// Two passes over memory per iteration (d = one double per node):
//   pass B : s = r - alpha v;  t = (A M^-1) s;  dots t.s, t.t, s.s, r0.s, r0.t
//            reads r, v, r0, 4c   writes t                                            8 d
//   pass CA: s = r - alpha v;  y += alpha p + omega s;  r' = s - omega t;
//            p' = r' + beta (p - omega v);  v' = (A M^-1) p';  dots r0.v', r'.r'
//            reads r, v, t, p, y, r0, 4c   writes y, r', p', v'                      14 d
// with rho' = r0.s - omega r0.t (R25), so that every scalar of iteration i+1 is known after pass B
// of iteration i and the x/r update of iteration i shares its pass with the p/v update of
// iteration i+1.  s is never stored.  r, p, v are double-buffered (a pass reads the old planes
// with their halo and writes the new ones).
//
// Sweep geometry ("marching warps").  Node planes are stored with a ghost ring (4 columns left,
// >= 2 right, 2 rows above and below; pitch NP a multiple of 16, so every strip starts on a 32-byte
// sector and every row on a 128-byte line, nh_internal.cuh) whose
// distance-1 ghosts hold the mirrored / wrapped images of the boundary nodes (R10); the writer of
// a boundary node stores its images, so no pass ever maps an index.  A warp owns a strip of 60
// columns and marches down a band of R rows: lane l holds columns 60 s - 2 + 2 l and the next one
// (one 16-byte load per plane per row), lanes 0 and 31 are halo lanes, the rows j-1, j, j+1 of the
// stencil operand live in registers, east/west neighbours come from warp shuffles.  No shared
// memory tiles, no block-level synchronisation inside a pass; all global accesses are coalesced
// 512-byte row segments.
//
// Dot products are two-stage and deterministic: per-CTA partials in a fixed order, one grid
// barrier, then every CTA sums all partials in the same order, so all CTAs take every branch
// alike.  Partials are double-buffered: one grid barrier per pass.
#include <cooperative_groups.h>
#include <math.h>
#include <stdio.h>

#include "nh_internal.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int NT = 256, NW = NT / 32;  // CTA size, warps per CTA
constexpr int SW = 60;                 // owned columns per warp strip
constexpr int MAXDOT = 5;
// small grids: at least this many rows per warp before CTAs are added (a warp marches its rows one
// memory latency at a time; measured at 512 x 8 ... 512^2: 8 rows 18-20 us per iteration, 4 rows 13-15)
#ifndef NH_MINROWS
#define NH_MINROWS 4
#endif

struct SolveP {
  NhGrid G;
  int nstrips, R, nbands;  // strips of SW columns, band height, bands
  const double *cE, *cW, *cN, *cS, *dg, *dinv, *b;
  double* x;
  double *y, *r0, *t;
  double *rA, *rB, *pA, *pB, *vA, *vB;
  double* part;  // [2][MAXDOT][gridDim.x]
  NhScal* sc;
  double rtol;
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
__device__ __forceinline__ void store_images(const NhGrid& G, double* a, int I, int J, double v) {
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
  static_assert(K <= NW, "one warp per value");
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int nb = gridDim.x;
  if (wid < K) {
    const double* src = part + ((size_t)buf * MAXDOT + wid) * nb;
    double a = 0.0;
    for (int i = lane; i < nb; i += 32) a += __ldcg(&src[i]);
    for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
    if (lane == 0) bc[wid] = a;
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
__device__ __forceinline__ double2 ld2(const double* a, const NhGrid& G, int c0, int j) {
  return *reinterpret_cast<const double2*>(a + nidx(G, c0, j));
}

// store the lane's pair of row j (owned columns only) and its ghost images: the same pair again on
// the ghost row of a boundary row, single values on the ghost column of a boundary column (the
// warps of the first and last strip used to take a scalar path for every row and finished 8 %
// (8192^2) to 34 % (2048^2) after the others, which every pass then waited for)
__device__ __forceinline__ void st2(double* a, const SolveP& P, const Unit& U, int j, double2 v) {
  const NhGrid& G = P.G;
  const int gj = ghost_image(j, G.nny, G.bylo);
  if (U.own1) {  // own1 implies own0
    *reinterpret_cast<double2*>(a + nidx(G, U.c0, j)) = v;
    if (gj != -2) *reinterpret_cast<double2*>(a + nidx(G, U.c0, gj)) = v;
  } else if (U.own0) {
    a[nidx(G, U.c0, j)] = v.x;
    if (gj != -2) a[nidx(G, U.c0, gj)] = v.x;
  }
  if (U.g0 != -2) a[nidx(G, U.g0, j)] = v.x;
  if (U.g1 != -2) a[nidx(G, U.g1, j)] = v.y;
}

// Register-resident operands of one sweep row.  Every pass is software-pipelined by hand: the
// loads of the NEXT row are issued before the current row is computed and stored (the compiler
// cannot hoist them itself across the stores of possibly aliasing planes), so each warp keeps one
// full row of every plane (~3-5 KB) in flight while it computes.
struct RowC {  // coefficient row j of (A M^-1) and the shadow residual
  double2 q, e, w, n, s;
};
__device__ __forceinline__ RowC ld_rowc(const SolveP& P, int c0, int j) {
  RowC C;
  C.q = ld2(P.r0, P.G, c0, j);
  C.e = ld2(P.cE, P.G, c0, j); C.w = ld2(P.cW, P.G, c0, j);
  C.n = ld2(P.cN, P.G, c0, j); C.s = ld2(P.cS, P.G, c0, j);
  return C;
}

// (A M^-1) applied to the operand rows (m: j-1, c: j, n: j+1) at the lane's two columns of row j
__device__ __forceinline__ double2 stencil2(const RowC& C, double2 m, double2 c, double2 n) {
  double west0 = __shfl_up_sync(0xffffffffu, c.y, 1);
  double east1 = __shfl_down_sync(0xffffffffu, c.x, 1);
  double2 o;
  o.x = fma(C.s.x, m.x, fma(C.n.x, n.x, fma(C.w.x, west0, fma(C.e.x, c.y, c.x))));
  o.y = fma(C.s.y, m.y, fma(C.n.y, n.y, fma(C.w.y, c.x, fma(C.e.y, east1, c.y))));
  return o;
}

// Operand requests per sweep step (measured on config 5, 8192 x 8192, us per iteration: old
// load-at-use order 2297; B prefetched + CA grouped 2069; both prefetched 2447 (CA's second operand
// set spills); both passes out of line 2611 (the parameter block then lives in local memory);
// cp.async rings in shared memory, 2 or 3 rows deep, 2362 / 2443; t recomputed in pass CA instead
// of stored by pass B and read back, 20 instead of 22 doubles per node-iteration, 2165 (its extra
// live rows spill at 128 registers; 2271 with 192-thread CTAs and 168 registers)).
constexpr bool PF_B = true;    // pass B: request the next step's operands before computing this one
constexpr bool PF_CA = false;  // pass CA: all ten operand loads of a step up front, then compute
#ifndef NH_DEFER_CA
#define NH_DEFER_CA 1
#endif
constexpr bool DEFER_CA = NH_DEFER_CA;  // pass CA: next step's loads issued before this step's stores

// pass B: s = r - alpha v (rows Ja-1..Jb), t = (A M^-1) s (rows Ja..Jb-1);
// partials: t.s, t.t, s.s, r0.s, r0.t
struct RowB {  // operands of one sweep step of pass B: vectors of row j+1, coefficients of row j
  double2 r, v;
  RowC C;
};
__device__ __forceinline__ void ld_rowb(RowB& X, const SolveP& P, const double* r, const double* v,
                                        int c0, int jv, int jc) {
  X.r = ld2(r, P.G, c0, jv); X.v = ld2(v, P.G, c0, jv);
  X.C = ld_rowc(P, c0, jc);
}

__device__ __forceinline__ void pass_B(const SolveP& P, double alpha, const double* r, const double* v,
                                    int buf, double (*red)[NW]) {
  const NhGrid& G = P.G;
  const int lane = threadIdx.x & 31;
  const int gw = blockIdx.x * NW + (threadIdx.x >> 5), tw = gridDim.x * NW;
  const int nunits = P.nstrips * P.nbands;
  double acc[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
  for (int u = gw; u < nunits; u += tw) {
    Unit U = make_unit(P, u, lane);
    auto srow = [&](double2 a, double2 b) {
      return make_double2(fma(-alpha, b.x, a.x), fma(-alpha, b.y, a.y));
    };
    double2 sm = srow(ld2(r, G, U.c0, U.Ja - 1), ld2(v, G, U.c0, U.Ja - 1));
    double2 sc = srow(ld2(r, G, U.c0, U.Ja), ld2(v, G, U.c0, U.Ja));
    // one sweep step: row j from the operand set `cur`; the set of the next step is requested
    // first (`nxt`; row indices clamped, the last request is never used)
    auto step = [&](int j, RowB& cur, RowB& nxt) {
      if (PF_B) ld_rowb(nxt, P, r, v, U.c0, min(j + 2, U.Jb), min(j + 1, U.Jb - 1));
      else ld_rowb(cur, P, r, v, U.c0, j + 1, j);
      double2 sn = srow(cur.r, cur.v);
      double2 t = stencil2(cur.C, sm, sc, sn);
      st2(P.t, P, U, j, t);
      const double2 q = cur.C.q;
      if (U.own0) {
        acc[0] = fma(t.x, sc.x, acc[0]); acc[1] = fma(t.x, t.x, acc[1]); acc[2] = fma(sc.x, sc.x, acc[2]);
        acc[3] = fma(q.x, sc.x, acc[3]); acc[4] = fma(q.x, t.x, acc[4]);
      }
      if (U.own1) {
        acc[0] = fma(t.y, sc.y, acc[0]); acc[1] = fma(t.y, t.y, acc[1]); acc[2] = fma(sc.y, sc.y, acc[2]);
        acc[3] = fma(q.y, sc.y, acc[3]); acc[4] = fma(q.y, t.y, acc[4]);
      }
      sm = sc; sc = sn;
    };
    RowB A, B;
    if (PF_B) ld_rowb(A, P, r, v, U.c0, U.Ja + 1, U.Ja);
    for (int j = U.Ja; j < U.Jb; j += 2) {  // ping-pong operand sets: no register rotation
      step(j, A, B);
      if (j + 1 < U.Jb) step(j + 1, B, A);
    }
  }
  block_partials<5>(acc, P.part, buf, red);
}

// pass CA: FIRST: p' = r' = r (start of a cycle).  Otherwise s = r - alpha v; y += alpha p + omega s;
// r' = s - omega t; p' = r' + beta (p - omega v).  Then v' = (A M^-1) p'.  partials: r0.v', r'.r'
struct RowV {  // vector row of pass CA
  double2 r, v, t, p, y;
};
template <bool FIRST>
__device__ __forceinline__ void ld_rowv(RowV& V, const SolveP& P, const double* r, const double* p,
                                        const double* v, int c0, int j) {
  V.r = ld2(r, P.G, c0, j);
  if (!FIRST) {
    V.v = ld2(v, P.G, c0, j); V.t = ld2(P.t, P.G, c0, j);
    V.p = ld2(p, P.G, c0, j); V.y = ld2(P.y, P.G, c0, j);
  }
}
struct RowCA {  // operands of one sweep step of pass CA: vectors of row j+1, coefficients of row j
  RowV V;
  RowC C;
};

template <bool FIRST>
__device__ __forceinline__ void pass_CA(const SolveP& P, double alpha, double omega, double beta,
                                     const double* r, const double* p, const double* v, double* rN,
                                     double* pN, double* vN, int buf, double (*red)[NW]) {
  const int lane = threadIdx.x & 31;
  const int gw = blockIdx.x * NW + (threadIdx.x >> 5), tw = gridDim.x * NW;
  const int nunits = P.nstrips * P.nbands;
  double acc[2] = {0.0, 0.0};
  for (int u = gw; u < nunits; u += tw) {
    Unit U = make_unit(P, u, lane);
    // new p of row j from its loaded operands; on owned rows also the y / r' / p' stores and the
    // r'.r' partial
    auto prow = [&](const RowV& V, int j, bool owned_row) {
      double2 rn, pn;
      if (FIRST) {
        rn = V.r; pn = V.r;
      } else {
        double2 s = make_double2(fma(-alpha, V.v.x, V.r.x), fma(-alpha, V.v.y, V.r.y));
        rn = make_double2(fma(-omega, V.t.x, s.x), fma(-omega, V.t.y, s.y));
        pn = make_double2(fma(beta, fma(-omega, V.v.x, V.p.x), rn.x),
                          fma(beta, fma(-omega, V.v.y, V.p.y), rn.y));
        if (owned_row) {
          double2 yy;
          yy.x = V.y.x + fma(omega, s.x, alpha * V.p.x);
          yy.y = V.y.y + fma(omega, s.y, alpha * V.p.y);
          st2(P.y, P, U, j, yy);
        }
      }
      if (owned_row) {
        st2(rN, P, U, j, rn);
        st2(pN, P, U, j, pn);
        if (U.own0) acc[1] = fma(rn.x, rn.x, acc[1]);
        if (U.own1) acc[1] = fma(rn.y, rn.y, acc[1]);
      }
      return pn;
    };
    double2 pm, pc;
    {
      RowV V0, V1;
      ld_rowv<FIRST>(V0, P, r, p, v, U.c0, U.Ja - 1);
      ld_rowv<FIRST>(V1, P, r, p, v, U.c0, U.Ja);
      pm = prow(V0, U.Ja - 1, false);
      pc = prow(V1, U.Ja, true);
    }
    auto ld_set = [&](RowCA& X, int jv, int jc) {
      ld_rowv<FIRST>(X.V, P, r, p, v, U.c0, jv);
      X.C = ld_rowc(P, U.c0, jc);
    };
    auto step = [&](int j, RowCA& cur, RowCA& nxt) {
      if (PF_CA) ld_set(nxt, min(j + 2, U.Jb), min(j + 1, U.Jb - 1));
      else ld_set(cur, j + 1, j);
      double2 pn = prow(cur.V, j + 1, j + 1 < U.Jb);
      double2 vv = stencil2(cur.C, pm, pc, pn);
      st2(vN, P, U, j, vv);
      if (U.own0) acc[0] = fma(cur.C.q.x, vv.x, acc[0]);
      if (U.own1) acc[0] = fma(cur.C.q.y, vv.y, acc[0]);
      pm = pc; pc = pn;
    };
    if (!FIRST && DEFER_CA) {
      // One operand set; the loads of step j+1 are issued as soon as step j has consumed its
      // operands, BEFORE its four stores (ghost-image logic included) and its dot-product terms,
      // which then run in the shadow of the memory latency.
      RowCA X;
      ld_set(X, U.Ja + 1, U.Ja);
      for (int j = U.Ja; j < U.Jb; ++j) {
        const RowV& V = X.V;
        const bool own_next = j + 1 < U.Jb;
        double2 sv = make_double2(fma(-alpha, V.v.x, V.r.x), fma(-alpha, V.v.y, V.r.y));
        double2 rn = make_double2(fma(-omega, V.t.x, sv.x), fma(-omega, V.t.y, sv.y));
        double2 pn = make_double2(fma(beta, fma(-omega, V.v.x, V.p.x), rn.x),
                                  fma(beta, fma(-omega, V.v.y, V.p.y), rn.y));
        double2 yy = make_double2(V.y.x + fma(omega, sv.x, alpha * V.p.x),
                                  V.y.y + fma(omega, sv.y, alpha * V.p.y));
        double2 vv = stencil2(X.C, pm, pc, pn);
        const double2 q = X.C.q;
        if (own_next) ld_set(X, min(j + 2, U.Jb), j + 1);  // operands of the next step
        if (own_next) {
          st2(P.y, P, U, j + 1, yy);
          st2(rN, P, U, j + 1, rn);
          st2(pN, P, U, j + 1, pn);
          if (U.own0) acc[1] = fma(rn.x, rn.x, acc[1]);
          if (U.own1) acc[1] = fma(rn.y, rn.y, acc[1]);
        }
        st2(vN, P, U, j, vv);
        if (U.own0) acc[0] = fma(q.x, vv.x, acc[0]);
        if (U.own1) acc[0] = fma(q.y, vv.y, acc[0]);
        pm = pc; pc = pn;
      }
    } else {
      RowCA A, B;
      if (PF_CA) ld_set(A, U.Ja + 1, U.Ja);
      for (int j = U.Ja; j < U.Jb; j += 2) {  // ping-pong operand sets: no register rotation
        step(j, A, B);
        if (j + 1 < U.Jb) step(j + 1, B, A);
      }
    }
  }
  block_partials<2>(acc, P.part, buf, red);
}

// ---- simple phases (a handful per solve): rows over CTAs, columns over threads --------------
// y = dg * x at the real nodes, with ghost images
__device__ void phase_y_from_x(const SolveP& P) {
  const NhGrid& G = P.G;
  for (int J = blockIdx.x; J < G.nny; J += gridDim.x)
    for (int I = threadIdx.x; I < G.nnx; I += NT) {
      size_t k = nidx(G, I, J);
      store_images(G, P.y, I, J, P.x[k] * P.dg[k]);
    }
}

// true residual r = b - (A M^-1) y, r0 = r (S9: the true residual decides); partials r.r, b.b
__device__ void phase_init(const SolveP& P, double* r, int buf, double (*red)[NW]) {
  const NhGrid& G = P.G;
  double acc[2] = {0.0, 0.0};
  for (int J = blockIdx.x; J < G.nny; J += gridDim.x)
    for (int I = threadIdx.x; I < G.nnx; I += NT) {
      size_t k = nidx(G, I, J);
      const double* y = P.y;
      double ay = y[k] + P.cE[k] * y[k + 1] + P.cW[k] * y[k - 1] + P.cN[k] * y[k + G.np] +
                  P.cS[k] * y[k - G.np];
      double bb = P.b[k];
      double rr = bb - ay;
      store_images(G, r, I, J, rr);
      P.r0[k] = rr;
      acc[0] += rr * rr; acc[1] += bb * bb;
    }
  block_partials<2>(acc, P.part, buf, red);
}

// y += alpha p + omega s, s = r - alpha v  (final update of an iteration whose pass CA never ran:
// half-step exit with omega = 0, and the polish iteration)
__device__ void phase_update_y(const SolveP& P, double alpha, double omega, const double* r,
                               const double* p, const double* v) {
  const NhGrid& G = P.G;
  for (int J = blockIdx.x; J < G.nny; J += gridDim.x)
    for (int I = threadIdx.x; I < G.nnx; I += NT) {
      size_t k = nidx(G, I, J);
      double s = r[k] - alpha * v[k];
      store_images(G, P.y, I, J, P.y[k] + (alpha * p[k] + omega * s));
    }
}

// x = M^-1 y  (or zeros when b = 0)
__device__ void phase_out(const SolveP& P, bool zero) {
  const NhGrid& G = P.G;
  for (int J = blockIdx.x; J < G.nny; J += gridDim.x)
    for (int I = threadIdx.x; I < G.nnx; I += NT) {
      size_t k = nidx(G, I, J);
      P.x[k] = zero ? 0.0 : P.y[k] * P.dinv[k];
    }
}

__global__ void __launch_bounds__(NT, 2) k_bicgstab(SolveP P) {
  cg::grid_group grid = cg::this_grid();
  __shared__ double red[MAXDOT][NW];
  __shared__ double bc[MAXDOT];

  double *rC = P.rA, *rN = P.rB, *pC = P.pA, *pN = P.pB, *vC = P.vA, *vN = P.vB;  // current / next
  auto flip = [&]() {
    double* t;
    t = rC; rC = rN; rN = t;
    t = pC; pC = pN; pN = t;
    t = vC; vC = vN; vN = t;
  };
  int buf = 0;  // partial buffer of the pass in flight (alternates: one grid barrier per pass)
  int iters = 0, converged = 0, status = 0;
  double rnorm = 0.0, bnorm = 0.0, tol = 0.0;

  phase_y_from_x(P);
  grid.sync();
  for (int cycle = 0; cycle < 8 && !converged; ++cycle) {
    double d2[2], d5[5];
    phase_init(P, rC, buf, red);
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
    if (iters >= P.maxit) break;
    // first direction of the cycle: p = r, v = (A M^-1) p, sigma = r0.v
    double rho = d2[0];
    pass_CA<true>(P, 0.0, 0.0, 0.0, rC, pC, vC, rN, pN, vN, buf, red);
    flip();
    grid.sync();
    grid_sums<2>(P.part, buf, d2, red, bc);
    buf ^= 1;
    double sigma = d2[0];
    while (iters < P.maxit) {
      if (fabs(rho) < 1e-300 || fabs(sigma) < 1e-300) break;  // breakdown -> restart
      double alpha = rho / sigma;
      iters++;
      pass_B(P, alpha, rC, vC, buf, red);
      grid.sync();
      grid_sums<5>(P.part, buf, d5, red, bc);
      buf ^= 1;
      if (sqrt(d5[2]) <= tol) {  // half-step exit: x += alpha p^
        phase_update_y(P, alpha, 0.0, rC, pC, vC);
        grid.sync();
        break;
      }
      if (d5[1] == 0.0) break;
      double omega = d5[0] / d5[1];
      if (fabs(omega) < 1e-300 || !(omega == omega)) break;
      double rho_new = d5[3] - omega * d5[4];  // r0.r' = r0.s - omega r0.t  (R25)
      double beta = (rho_new / rho) * (alpha / omega);
      rho = rho_new;
      pass_CA<false>(P, alpha, omega, beta, rC, pC, vC, rN, pN, vN, buf, red);
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
    pass_CA<true>(P, 0.0, 0.0, 0.0, rC, pC, vC, rN, pN, vN, buf, red);
    flip();
    grid.sync();
    grid_sums<2>(P.part, buf, d2, red, bc);
    buf ^= 1;
    double sigma = d2[0];
    if (fabs(rho) >= 1e-300 && fabs(sigma) >= 1e-300) {
      double alpha = rho / sigma;
      pass_B(P, alpha, rC, vC, buf, red);
      grid.sync();
      grid_sums<5>(P.part, buf, d5, red, bc);
      buf ^= 1;
      double omega = (d5[1] > 0.0) ? d5[0] / d5[1] : 0.0;
      phase_update_y(P, alpha, omega, rC, pC, vC);
      grid.sync();
    }
  }
  if (status != NH_ENAN) phase_out(P, bnorm == 0.0);

  if (blockIdx.x == 0 && threadIdx.x == 0) {
    NhScal* sc = P.sc;
    if (status == NH_ENOCONV) sc->flags |= NH_FLAG_NOCONV;
    if (status == NH_ENAN) sc->flags |= NH_FLAG_NAN;
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
struct SrjP {
  NhGrid G;
  int nstrips, R, nbands;
  const double *cE, *cW, *cN, *cS, *bp, *costab;
  double *xA, *xB;  // xA = the pressure plane p (start and result), xB = scratch
  NhScal* sc;
  double eps, rel;  // tolerance of (32): eps, or rel * max|b'| when rel > 0
  int maxit, mmax, count_stats;
};

__device__ __forceinline__ void srj_sweep(const SrjP& P, const SolveP& Q, double om, const double* x,
                                          double* xn, unsigned long long* Eslot) {
  const NhGrid& G = P.G;
  const int lane = threadIdx.x & 31;
  const int gw = blockIdx.x * NW + (threadIdx.x >> 5), tw = gridDim.x * NW;
  const int nunits = P.nstrips * P.nbands;
  double emax = 0.0;
  bool bad = false;
  struct Row { double2 xn, b, e, w, n, s; };
  for (int u = gw; u < nunits; u += tw) {
    Unit U = make_unit(Q, u, lane);
    double2 xm = ld2(x, G, U.c0, U.Ja - 1), xc = ld2(x, G, U.c0, U.Ja);
    auto ld_row = [&](Row& X, int j) {  // operands of sweep step j (x of row j+1, the rest of row j)
      X.xn = ld2(x, G, U.c0, min(j + 1, U.Jb));
      const int jc = min(j, U.Jb - 1);
      X.b = ld2(P.bp, G, U.c0, jc);
      X.e = ld2(P.cE, G, U.c0, jc); X.w = ld2(P.cW, G, U.c0, jc);
      X.n = ld2(P.cN, G, U.c0, jc); X.s = ld2(P.cS, G, U.c0, jc);
    };
    auto step = [&](int j, Row& cur, Row& nxt) {
      ld_row(nxt, j + 1);  // request the next step's operands first
      double west0 = __shfl_up_sync(0xffffffffu, xc.y, 1);
      double east1 = __shfl_down_sync(0xffffffffu, xc.x, 1);
      double ax0 = xc.x + (((cur.e.x * xc.y + cur.w.x * west0) + cur.n.x * cur.xn.x) + cur.s.x * xm.x);
      double ax1 = xc.y + (((cur.e.y * east1 + cur.w.y * xc.x) + cur.n.y * cur.xn.y) + cur.s.y * xm.y);
      double z0 = cur.b.x - ax0, z1 = cur.b.y - ax1;
      if (U.own0) { emax = fmax(emax, fabs(z0)); bad |= !(z0 == z0); }
      if (U.own1) { emax = fmax(emax, fabs(z1)); bad |= !(z1 == z1); }
      st2(xn, Q, U, j, make_double2(xc.x + om * z0, xc.y + om * z1));
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
  __shared__ double wmax[NW];
  if (lane == 0) wmax[threadIdx.x >> 5] = emax;
  int anybad = __syncthreads_or(bad);
  if (threadIdx.x == 0) {
    double m = 0.0;
#pragma unroll
    for (int w = 0; w < NW; ++w) m = fmax(m, wmax[w]);
    if (m > 0.0) atomicMax(Eslot, (unsigned long long)__double_as_longlong(m));
    if (anybad) atomicOr(&P.sc->srj_bad, 1);
  }
}

#ifndef NH_SRJ_MINB
#define NH_SRJ_MINB 2
#endif
__global__ void __launch_bounds__(NT, NH_SRJ_MINB) k_srj(SrjP P) {
  cg::grid_group grid = cg::this_grid();
  const NhGrid& G = P.G;
  NhScal* sc = P.sc;
  SolveP Q;  // geometry view for make_unit / st2
  Q.G = P.G; Q.nstrips = P.nstrips; Q.R = P.R; Q.nbands = P.nbands;
  const double rho = __longlong_as_double((long long)sc->srj_rho_bits);
  const double bmax = __longlong_as_double((long long)sc->srj_bmax_bits);
  int iters = 0, status = 0;
  double E = 0.0;
  double *x = P.xA, *xn = P.xB;
  if (!(bmax == bmax) || isinf(bmax)) {
    status = NH_ENAN;
  } else if (bmax == 0.0) {  // b = 0 => p~ = 0, zero iterations (same convention as solver 0)
    for (int J = blockIdx.x; J < G.nny; J += gridDim.x)
      for (int I = threadIdx.x; I < G.nnx; I += NT) P.xA[nidx(G, I, J)] = 0.0;
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
      for (int I = threadIdx.x; I < G.nnx; I += NT) store_images(G, x, I, J, x[nidx(G, I, J)]);
    grid.sync();
    for (;;) {
      const double om = dominant ? 1.0 / (1.0 - rho * cosv[iters % M]) : 1.0;
      unsigned long long* slot = &sc->srj_E_bits[iters % 3];
      srj_sweep(P, Q, om, x, xn, slot);
      grid.sync();
      E = __longlong_as_double((long long)__ldcg(slot));
      const int bad = __ldcg(&sc->srj_bad);
      if (blockIdx.x == 0 && threadIdx.x == 0) sc->srj_E_bits[(iters + 2) % 3] = 0ULL;
      if (bad) { status = NH_ENAN; break; }
      if (E < tol) break;  // eq. (32): x is the accepted iterate
      if (iters >= P.maxit) { status = NH_ENOCONV; break; }
      double* t = x; x = xn; xn = t;
      iters++;
    }
    if (x != P.xA) {  // the accepted iterate lives in the scratch plane
      for (int J = blockIdx.x; J < G.nny; J += gridDim.x)
        for (int I = threadIdx.x; I < G.nnx; I += NT) P.xA[nidx(G, I, J)] = x[nidx(G, I, J)];
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
int nh_solver_setup(nh_ctx* c) {
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
  for (int R = 4; R <= nny; ++R) {
    long long nb = (nny + R - 1) / R;
    long long rounds = (nstrips * nb + tw - 1) / tw;
    long long cost = rounds * (R + 2);
    if (best < 0 || cost < best) { best = cost; bestR = R; }
  }
  if (nny < 4) bestR = nny;
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
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ1, k_srj, NT, 0);
    if (e != cudaSuccess || occ1 < 1) {
      snprintf(c->err, sizeof(c->err), "srj occupancy query failed: %s", cudaGetErrorString(e));
      return NH_ECUDA;
    }
    long long g1 = (long long)occ1 * c->sm_count;
    if (g1 > (small_units + NW - 1) / NW) g1 = (small_units + NW - 1) / NW;
    if (g1 < 1) g1 = 1;
    const long long tw1 = g1 * NW;
    int R1 = nny;
    long long best1 = -1;
    for (int R = 4; R <= nny; ++R) {
      long long nb = (nny + R - 1) / R;
      long long rounds = (nstrips * nb + tw1 - 1) / tw1;
      long long cost = rounds * (R + 2);
      if (best1 < 0 || cost < best1) { best1 = cost; R1 = R; }
    }
    if (nny < 4) R1 = nny;
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

void nh_launch_solve(nh_ctx* c, const double* b, double* x, int count_stats) {
  if (c->prm.solver == 1) {  // b is c->kr = b / A_C here (nh_launch_scale_rows)
    SrjP S;
    S.G = c->g;
    S.nstrips = c->solver_nstrips; S.R = c->srj_R; S.nbands = c->srj_nbands;
    S.cE = c->cE; S.cW = c->cW; S.cN = c->cN; S.cS = c->cS; S.bp = c->kr; S.costab = c->srj_cos;
    S.xA = x; S.xB = c->ky; S.sc = c->sc; S.eps = c->prm.srj_eps; S.rel = c->prm.srj_rel;
    S.maxit = c->prm.solver_maxit; S.mmax = c->prm.srj_mmax; S.count_stats = count_stats;
    void* args[] = {&S};
    NH_CUDA_OK(c, cudaLaunchCooperativeKernel((void*)k_srj, dim3(c->srj_grid), dim3(NT), args, 0,
                                              c->stream));
    c->launches++;
    return;
  }
  SolveP P;
  P.G = c->g;
  P.nstrips = c->solver_nstrips; P.R = c->solver_R; P.nbands = c->solver_nbands;
  P.cE = c->cE; P.cW = c->cW; P.cN = c->cN; P.cS = c->cS; P.dg = c->dg; P.dinv = c->dinv;
  P.b = b; P.x = x;
  P.y = c->ky; P.r0 = c->kr0; P.t = c->kt;
  P.rA = c->kr; P.rB = c->krB; P.pA = c->kpA; P.pB = c->kpB; P.vA = c->kvA; P.vB = c->kvB;
  P.part = c->part; P.sc = c->sc; P.rtol = c->prm.solver_rtol; P.maxit = c->prm.solver_maxit;
  P.count_stats = count_stats;
  void* args[] = {&P};
  NH_CUDA_OK(c, cudaLaunchCooperativeKernel((void*)k_bicgstab, dim3(c->solver_grid), dim3(NT), args,
                                            0, c->stream));
  c->launches++;
}
