// nh_solver.cu -- a6: Jacobi-preconditioned BiCGStab (van der Vorst 1992 form, R14) for
// the compact finite-difference pressure system (eqs (29), (36)-(43)) as ONE
// persistent cooperative kernel.
//
// The whole solve -- true-residual (re)starts, the iteration loop with its convergence tests, the
// half-step exit, breakdown restarts and the final polish iteration -- runs on the device: no
// host round trip per iteration (the paper's loop reads the error on the host every sweep,
// L535-539).  The grid is one wave of co-resident CTAs (occupancy x 148 SMs); phases are separated
// by grid-wide barriers; dot products are two-pass and deterministic (per-CTA partials in a fixed
// order, then every CTA sums all partials in the same order, so all CTAs take every branch alike).
//
// Right preconditioning is folded into the operator: with M = diag(A) the iteration runs on
// A M^-1 (unit diagonal, column-scaled off-diagonals cE..cS prepared once per solve by
// k_scale_coeffs) with the iterate y = M x; r is the residual of the unpreconditioned system.
//
// Per iteration (d = one double per node):
//   phase A: p = r + beta (p - omega v);  v = A M^-1 p;  r0.v       reads r,p,v,r0,4c  writes p,v   10 d
//   phase B: s = r - alpha v;  t = A M^-1 s;  t.s, t.t, s.s          reads r,v,4c       writes t      7 d
//   phase C: y += alpha p + omega s;  r = s - omega t;  r0.r, r.r    reads y,p,r,v,t,r0 writes y,r    8 d
// s is never stored (recomputed from r and v); p and v are double-buffered so that phase A can
// recompute p on its halo while neighbours write the new p.
#include <cooperative_groups.h>
#include <math.h>
#include <stdio.h>

#include "nh_internal.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int TX = 64, TY = 16, NT = 256;  // node tile and CTA size
constexpr int SX = TX + 2, SY = TY + 2;
constexpr int NPT = TX * TY / NT;          // nodes per thread (rows ty, ty+4, ...)
constexpr int MAXDOT = 3;

struct SolveP {
  NhGrid G;
  const double *cE, *cW, *cN, *cS, *dg, *dinv, *b;
  double* x;
  double *y, *r, *r0, *pA, *pB, *vA, *vB, *t;
  double* part;
  NhScal* sc;
  double rtol;
  int maxit;
  int count_stats;
};

struct Tile {
  double a[SY][SX];
};

__device__ __forceinline__ size_t nidx(const NhGrid& G, int I, int J) { return (size_t)J * G.np + I; }

// deterministic block reduction of K values; result of value k lands in part[k*gridDim.x + blockIdx.x]
template <int K>
__device__ __forceinline__ void block_partials(double (&v)[K], double* part, double (*red)[NT / 32]) {
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
    for (int w = 0; w < NT / 32; ++w) a += red[threadIdx.x][w];
    part[(size_t)threadIdx.x * gridDim.x + blockIdx.x] = a;
  }
  __syncthreads();
}

// every CTA sums all partials in the same fixed order -> bit-identical scalars everywhere
template <int K>
__device__ __forceinline__ void grid_sums(const double* part, double (&out)[K], double (*red)[NT / 32],
                                          double* bc) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int nb = gridDim.x;
#pragma unroll
  for (int k = 0; k < K; ++k) {
    double a = 0.0;
    for (int i = threadIdx.x; i < nb; i += NT) a += __ldcg(&part[(size_t)k * nb + i]);
    for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
    if (lane == 0) red[k][wid] = a;
  }
  __syncthreads();
  if (threadIdx.x < K) {
    double a = 0.0;
#pragma unroll
    for (int w = 0; w < NT / 32; ++w) a += red[threadIdx.x][w];
    bc[threadIdx.x] = a;
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < K; ++k) out[k] = bc[k];
  __syncthreads();
}

struct TileIter {
  int ntx, ntiles;
  __device__ TileIter(const NhGrid& G) {
    ntx = (G.nnx + TX - 1) / TX;
    ntiles = ntx * ((G.nny + TY - 1) / TY);
  }
};

// global node index of halo-tile element (lx,ly) through the node maps (R10); -1 if not needed
__device__ __forceinline__ long long halo_index(const NhGrid& G, int I0, int J0, int lx, int ly) {
  int I = I0 - 1 + lx, J = J0 - 1 + ly;
  if (I > G.nnx || J > G.nny) return -1;
  // distinct node lines are 0..nnx-1; -1 and nnx are ghosts
  int II = I, JJ = J;
  if (I < 0 || I >= G.nnx) II = nh_map_node(I, G.nx, G.bxlo);
  if (J < 0 || J >= G.nny) JJ = nh_map_node(J, G.ny, G.bylo);
  return (long long)JJ * G.np + II;
}

__device__ __forceinline__ double stencil(const Tile& T, int lx, int ly, size_t k, const SolveP& P) {
  return T.a[ly][lx] + P.cE[k] * T.a[ly][lx + 1] + P.cW[k] * T.a[ly][lx - 1] +
         P.cN[k] * T.a[ly + 1][lx] + P.cS[k] * T.a[ly - 1][lx];
}

// INIT: r = b - (A M^-1) y, r0 = r; partials: r.r and b.b.  first: y = dg * x (x-space start).
__device__ void phase_init(const SolveP& P, Tile& T, bool from_x, double (*red)[NT / 32]) {
  const NhGrid& G = P.G;
  TileIter it(G);
  double acc[2] = {0.0, 0.0};
  for (int tile = blockIdx.x; tile < it.ntiles; tile += gridDim.x) {
    int I0 = (tile % it.ntx) * TX, J0 = (tile / it.ntx) * TY;
    __syncthreads();
    for (int e = threadIdx.x; e < SX * SY; e += NT) {
      int lx = e % SX, ly = e / SX;
      long long k = halo_index(G, I0, J0, lx, ly);
      double v = 0.0;
      if (k >= 0) v = from_x ? P.x[k] * P.dg[k] : P.y[k];
      T.a[ly][lx] = v;
    }
    __syncthreads();
    int tx = threadIdx.x % TX, ty0 = threadIdx.x / TX;
#pragma unroll
    for (int q = 0; q < NPT; ++q) {
      int ty = ty0 + q * (NT / TX);
      int I = I0 + tx, J = J0 + ty;
      if (I < G.nnx && J < G.nny) {
        size_t k = nidx(G, I, J);
        double bb = P.b[k];
        double rr = bb - stencil(T, tx + 1, ty + 1, k, P);
        if (from_x) P.y[k] = T.a[ty + 1][tx + 1];
        P.r[k] = rr; P.r0[k] = rr;
        acc[0] += rr * rr; acc[1] += bb * bb;
      }
    }
  }
  block_partials<2>(acc, P.part, red);
}

// phase A: p_new = first ? r : r + beta (p - omega v)   on tile+halo;  v_new = (A M^-1) p_new
__device__ void phase_A(const SolveP& P, Tile& T, bool first, double beta, double omega,
                        const double* pO, const double* vO, double* pN, double* vN,
                        double (*red)[NT / 32]) {
  const NhGrid& G = P.G;
  TileIter it(G);
  double acc[1] = {0.0};
  for (int tile = blockIdx.x; tile < it.ntiles; tile += gridDim.x) {
    int I0 = (tile % it.ntx) * TX, J0 = (tile / it.ntx) * TY;
    __syncthreads();
    for (int e = threadIdx.x; e < SX * SY; e += NT) {
      int lx = e % SX, ly = e / SX;
      long long k = halo_index(G, I0, J0, lx, ly);
      double v = 0.0;
      if (k >= 0) {
        v = P.r[k];
        if (!first) v = v + beta * (pO[k] - omega * vO[k]);
      }
      T.a[ly][lx] = v;
    }
    __syncthreads();
    int tx = threadIdx.x % TX, ty0 = threadIdx.x / TX;
#pragma unroll
    for (int q = 0; q < NPT; ++q) {
      int ty = ty0 + q * (NT / TX);
      int I = I0 + tx, J = J0 + ty;
      if (I < G.nnx && J < G.nny) {
        size_t k = nidx(G, I, J);
        double vv = stencil(T, tx + 1, ty + 1, k, P);
        pN[k] = T.a[ty + 1][tx + 1];
        vN[k] = vv;
        acc[0] += P.r0[k] * vv;
      }
    }
  }
  block_partials<1>(acc, P.part, red);
}

// phase B: s = r - alpha v on tile+halo; t = (A M^-1) s; partials t.s, t.t, s.s
__device__ void phase_B(const SolveP& P, Tile& T, double alpha, const double* v,
                        double (*red)[NT / 32]) {
  const NhGrid& G = P.G;
  TileIter it(G);
  double acc[3] = {0.0, 0.0, 0.0};
  for (int tile = blockIdx.x; tile < it.ntiles; tile += gridDim.x) {
    int I0 = (tile % it.ntx) * TX, J0 = (tile / it.ntx) * TY;
    __syncthreads();
    for (int e = threadIdx.x; e < SX * SY; e += NT) {
      int lx = e % SX, ly = e / SX;
      long long k = halo_index(G, I0, J0, lx, ly);
      double s = 0.0;
      if (k >= 0) s = P.r[k] - alpha * v[k];
      T.a[ly][lx] = s;
    }
    __syncthreads();
    int tx = threadIdx.x % TX, ty0 = threadIdx.x / TX;
#pragma unroll
    for (int q = 0; q < NPT; ++q) {
      int ty = ty0 + q * (NT / TX);
      int I = I0 + tx, J = J0 + ty;
      if (I < G.nnx && J < G.nny) {
        size_t k = nidx(G, I, J);
        double tt = stencil(T, tx + 1, ty + 1, k, P);
        double s = T.a[ty + 1][tx + 1];
        P.t[k] = tt;
        acc[0] += tt * s; acc[1] += tt * tt; acc[2] += s * s;
      }
    }
  }
  block_partials<3>(acc, P.part, red);
}

// phase C: y += alpha p + omega s;  r = s - omega t  (s = r - alpha v);  partials r0.r, r.r
__device__ void phase_C(const SolveP& P, double alpha, double omega, const double* p,
                        const double* v, bool update_r, double (*red)[NT / 32]) {
  const NhGrid& G = P.G;
  TileIter it(G);
  double acc[2] = {0.0, 0.0};
  for (int tile = blockIdx.x; tile < it.ntiles; tile += gridDim.x) {
    int I0 = (tile % it.ntx) * TX, J0 = (tile / it.ntx) * TY;
    int tx = threadIdx.x % TX, ty0 = threadIdx.x / TX;
#pragma unroll
    for (int q = 0; q < NPT; ++q) {
      int ty = ty0 + q * (NT / TX);
      int I = I0 + tx, J = J0 + ty;
      if (I < G.nnx && J < G.nny) {
        size_t k = nidx(G, I, J);
        double pk = p[k];
        if (update_r) {
          double s = P.r[k] - alpha * v[k];
          P.y[k] = P.y[k] + (alpha * pk + omega * s);
          double rn = s - omega * P.t[k];
          P.r[k] = rn;
          acc[0] += P.r0[k] * rn; acc[1] += rn * rn;
        } else {
          P.y[k] = P.y[k] + alpha * pk;  // half-step exit: x += alpha p^
        }
      }
    }
  }
  block_partials<2>(acc, P.part, red);
}

// x = M^-1 y  (or zeros when b = 0)
__device__ void phase_out(const SolveP& P, bool zero) {
  const NhGrid& G = P.G;
  TileIter it(G);
  for (int tile = blockIdx.x; tile < it.ntiles; tile += gridDim.x) {
    int I0 = (tile % it.ntx) * TX, J0 = (tile / it.ntx) * TY;
    int tx = threadIdx.x % TX, ty0 = threadIdx.x / TX;
#pragma unroll
    for (int q = 0; q < NPT; ++q) {
      int ty = ty0 + q * (NT / TX);
      int I = I0 + tx, J = J0 + ty;
      if (I < G.nnx && J < G.nny) {
        size_t k = nidx(G, I, J);
        P.x[k] = zero ? 0.0 : P.y[k] * P.dinv[k];
      }
    }
  }
}

__global__ void __launch_bounds__(NT) k_bicgstab(SolveP P) {
  cg::grid_group grid = cg::this_grid();
  __shared__ Tile T;
  __shared__ double red[MAXDOT][NT / 32];
  __shared__ double bc[MAXDOT];

  const double* pO = P.pA; double* pN = P.pB;  // p: current / next
  const double* vO = P.vA; double* vN = P.vB;
  int iters = 0, converged = 0, status = 0;
  double rnorm = 0.0, bnorm = 0.0, tol = 0.0;
  bool have_y = false;

  for (int cycle = 0; cycle < 8 && !converged; ++cycle) {
    // true residual r = b - A x (S9: the true residual decides; restarts after drift/breakdown)
    phase_init(P, T, !have_y, red);
    have_y = true;
    grid.sync();
    double d2[2];
    grid_sums<2>(P.part, d2, red, bc);
    grid.sync();  // partials are reused by the next phase
    rnorm = sqrt(d2[0]);
    if (cycle == 0) {
      bnorm = sqrt(d2[1]);
      if (!(bnorm == bnorm) || isinf(bnorm)) { status = NH_ENAN; break; }
      if (bnorm == 0.0) break;
      tol = P.rtol * bnorm;
    }
    if (rnorm <= tol) { converged = 1; break; }
    if (iters >= P.maxit) break;
    double rho = 1.0, alpha = 1.0, omega = 1.0;
    double rho_new = d2[0];  // r0 = r  =>  r0.r = r.r
    bool first = true;
    while (iters < P.maxit) {
      if (fabs(rho_new) < 1e-300) break;  // breakdown -> restart
      double beta = (rho_new / rho) * (alpha / omega);
      rho = rho_new;
      phase_A(P, T, first, beta, omega, pO, vO, pN, vN, red);
      { const double* tp = pO; pO = pN; pN = const_cast<double*>(tp); }
      { const double* tv = vO; vO = vN; vN = const_cast<double*>(tv); }
      grid.sync();
      double d1[1];
      grid_sums<1>(P.part, d1, red, bc);
      grid.sync();
      double sigma = d1[0];
      if (fabs(sigma) < 1e-300) break;
      alpha = rho / sigma;
      iters++;
      phase_B(P, T, alpha, vO, red);
      grid.sync();
      double d3[3];
      grid_sums<3>(P.part, d3, red, bc);
      grid.sync();
      double snorm = sqrt(d3[2]);
      if (snorm <= tol) {  // half-step exit
        phase_C(P, alpha, 0.0, pO, vO, false, red);
        grid.sync();
        break;
      }
      if (d3[1] == 0.0) break;
      omega = d3[0] / d3[1];
      if (fabs(omega) < 1e-300) break;
      phase_C(P, alpha, omega, pO, vO, true, red);
      grid.sync();
      grid_sums<2>(P.part, d2, red, bc);
      grid.sync();
      rho_new = d2[0];
      rnorm = sqrt(d2[1]);
      first = false;
      if (rnorm <= tol) break;
    }
  }
  if (status == 0 && bnorm > 0.0 && !converged) status = NH_ENOCONV;

  // one extra "polish" iteration from the true residual (R14): r0 = r, p = r
  if (converged && rnorm > 0.0) {
    double rho = rnorm * rnorm;
    {
      // rho = r0.r with r0 = r: recompute exactly as a dot (d2[0] of the last INIT)
      // (rnorm*rnorm differs from the dot by rounding; keep the dot)
    }
    phase_A(P, T, true, 0.0, 0.0, pO, vO, pN, vN, red);
    { const double* tp = pO; pO = pN; pN = const_cast<double*>(tp); }
    { const double* tv = vO; vO = vN; vN = const_cast<double*>(tv); }
    grid.sync();
    double d1[1];
    grid_sums<1>(P.part, d1, red, bc);
    grid.sync();
    double sigma = d1[0];
    if (fabs(rho) >= 1e-300 && fabs(sigma) >= 1e-300) {
      double alpha = rho / sigma;
      phase_B(P, T, alpha, vO, red);
      grid.sync();
      double d3[3];
      grid_sums<3>(P.part, d3, red, bc);
      grid.sync();
      double omega = (d3[1] > 0.0) ? d3[0] / d3[1] : 0.0;
      phase_C(P, alpha, omega, pO, vO, true, red);
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

}  // namespace

int nh_solver_setup(nh_ctx* c) {
  int occ = 0;
  cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_bicgstab, NT, 0);
  if (e != cudaSuccess || occ < 1) {
    snprintf(c->err, sizeof(c->err), "solver occupancy query failed: %s", cudaGetErrorString(e));
    return NH_ECUDA;
  }
  int ntiles = ((c->g.nnx + TX - 1) / TX) * ((c->g.nny + TY - 1) / TY);
  if (occ > 4) occ = 4;
  int grid = occ * c->sm_count;
  if (grid > ntiles) grid = ntiles;
  if (grid < 1) grid = 1;
  c->solver_occ = occ;
  c->solver_grid = grid;
  e = cudaMalloc(&c->part, sizeof(double) * MAXDOT * (size_t)grid);
  if (e != cudaSuccess) return NH_ENOMEM;
  return NH_OK;
}

void nh_launch_solve(nh_ctx* c, const double* b, double* x, int count_stats) {
  SolveP P;
  P.G = c->g;
  P.cE = c->cE; P.cW = c->cW; P.cN = c->cN; P.cS = c->cS; P.dg = c->dg; P.dinv = c->dinv;
  P.b = b; P.x = x;
  P.y = c->ky; P.r = c->kr; P.r0 = c->kr0; P.pA = c->kpA; P.pB = c->kpB; P.vA = c->kvA; P.vB = c->kvB;
  P.t = c->kt;
  P.part = c->part; P.sc = c->sc; P.rtol = c->prm.solver_rtol; P.maxit = c->prm.solver_maxit;
  P.count_stats = count_stats;
  void* args[] = {&P};
  NH_CUDA_OK(c, cudaLaunchCooperativeKernel((void*)k_bicgstab, dim3(c->solver_grid), dim3(NT), args,
                                            0, c->stream));
  c->launches++;
}
