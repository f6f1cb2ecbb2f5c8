// nh_pressure.cu -- second and third parts of the time step, outside the Krylov loop:
// breaking sources (a4), right-hand side (a5), the rows of the compact finite-difference pressure
// operator (S8) and their column scaling for the Jacobi-preconditioned solver, the matrix-free
// operator apply (test hook), the Chorin-Temam correction (a7) and the relaxation zone (a9).
//
// These kernels run once per Runge-Kutta stage (the solver runs 10^2 iterations per stage), so
// they read their small stencils straight from global memory through the boundary index maps
// (L1/L2 serve the overlap) instead of staging tiles.
#include <math.h>
#include <stdio.h>

#include "nh_internal.cuh"

namespace {

constexpr int BX = 32, BY = 8;

struct Fld {  // read-only field + grid: ghost access S1 (R9)
  const NhGrid& G;
  bool fast;  // every cell / node this thread touches is inside the grid: no index maps, no signs
  __device__ __forceinline__ double even(const double* __restrict__ a, int i, int j) const {
    if (fast) return a[(size_t)j * G.nx + i];
    int ii = nh_map_cell_even(i, G.nx, G.bxlo, G.bxhi);
    int jj = nh_map_cell_even(j, G.ny, G.bylo, G.byhi);
    return a[(size_t)jj * G.nx + ii];
  }
  __device__ __forceinline__ double xn(const double* __restrict__ a, int i, int j) const {
    if (fast) return a[(size_t)j * G.nx + i];
    double sx;
    int ii = nh_map_cell(i, G.nx, G.bxlo, G.bxhi, sx);
    int jj = nh_map_cell_even(j, G.ny, G.bylo, G.byhi);
    return sx * a[(size_t)jj * G.nx + ii];
  }
  __device__ __forceinline__ double yn(const double* __restrict__ a, int i, int j) const {
    if (fast) return a[(size_t)j * G.nx + i];
    double sy;
    int ii = nh_map_cell_even(i, G.nx, G.bxlo, G.bxhi);
    int jj = nh_map_cell(j, G.ny, G.bylo, G.byhi, sy);
    return sy * a[(size_t)jj * G.nx + ii];
  }
  __device__ __forceinline__ double node(const double* __restrict__ a, int I, int J) const {
    if (fast) return a[(size_t)J * G.np + I];
    int II = nh_map_node(I, G.nx, G.bxlo);
    int JJ = nh_map_node(J, G.ny, G.bylo);
    return a[(size_t)JJ * G.np + II];
  }
  __device__ __forceinline__ double xi_x(const double* __restrict__ z, int i, int j) const {
    return 0.5 * (even(z, i + 1, j) - even(z, i - 1, j));
  }
  __device__ __forceinline__ double xi_y(const double* __restrict__ z, int i, int j) const {
    return 0.5 * (even(z, i, j + 1) - even(z, i, j - 1));
  }
  __device__ __forceinline__ double hnode(const double* __restrict__ h, int I, int J) const {
    return 0.25 * (even(h, I - 1, J - 1) + even(h, I, J - 1) + even(h, I, J) + even(h, I - 1, J));
  }
};

// node (I,J) whose stencils (cells I-2..I+1, J-2..J+1; nodes I-1..I+1, J-1..J+1) stay inside the grid
__device__ __forceinline__ bool node_interior(const NhGrid& G, int I, int J) {
  return I >= 2 && I + 1 <= G.nx - 1 && J >= 2 && J + 1 <= G.ny - 1;
}

// z = 2 eta - h, eq. (6)
__global__ void __launch_bounds__(256)
k_compute_z(size_t nc, const double* __restrict__ h, const double* __restrict__ H,
            double* __restrict__ z) {
  for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < nc;
       k += (size_t)gridDim.x * blockDim.x) {
    double eta = h[k] - H[k];
    z[k] = 2.0 * eta - h[k];
  }
}

// z = 2 eta - h (eq. (6)) as the dense cell plane, and the operands of the matrix-free solver
// (nh_solver.cu): h and z in the node layout shifted by one column (plane column P = cell P - 1),
// cells -2 .. nx+1 by -2 .. ny+1 through the even cell maps (R9: h, H, eta are even in every ghost).
__global__ void __launch_bounds__(BX* BY)
k_cell_planes(NhGrid G, const double* __restrict__ h, const double* __restrict__ H,
              double* __restrict__ z, double* __restrict__ hc, double* __restrict__ zc) {
  int i = (int)(blockIdx.x * BX + threadIdx.x) - 2, j = (int)(blockIdx.y * BY + threadIdx.y) - 2;
  if (i > G.nx + 1 || j > G.ny + 1) return;
  int ii = nh_map_cell_even(i, G.nx, G.bxlo, G.bxhi);
  int jj = nh_map_cell_even(j, G.ny, G.bylo, G.byhi);
  size_t k = (size_t)jj * G.nx + ii;
  double hv = h[k];
  double eta = hv - H[k];
  double zv = 2.0 * eta - hv;
  if (ii == i && jj == j) z[k] = zv;
  long long kp = (long long)j * G.np + (i + 1);
  hc[kp] = hv; zc[kp] = zv;
}

// S8: the five coefficients of row (I,J), derived from (36)-(41); 1D restriction = (43).
__device__ __forceinline__ void node_coeffs(const Fld& F, const double* __restrict__ h,
                                            const double* __restrict__ z, int I, int J, double& AC,
                                            double& AE, double& AW, double& AN, double& AS) {
  const NhGrid& G = F.G;
  // SW=(I-1,J-1), SE=(I,J-1), NW=(I-1,J), NE=(I,J)
  double hSW = F.even(h, I - 1, J - 1), hSE = F.even(h, I, J - 1);
  double hNW = F.even(h, I - 1, J), hNE = F.even(h, I, J);
  double zSW = F.even(z, I - 1, J - 1), zSE = F.even(z, I, J - 1);
  double zNW = F.even(z, I - 1, J), zNE = F.even(z, I, J);
  double hn = 0.25 * (hSW + hSE + hNE + hNW);  // (38)
  double hE = 0.5 * (hNE + hSE), hW = 0.5 * (hNW + hSW);
  double hN = 0.5 * (hNE + hNW), hS = 0.5 * (hSE + hSW);
  double xE = 0.5 * (F.xi_x(z, I, J) + F.xi_x(z, I, J - 1));
  double xW = 0.5 * (F.xi_x(z, I - 1, J) + F.xi_x(z, I - 1, J - 1));
  double xN = 0.5 * (F.xi_y(z, I, J) + F.xi_y(z, I - 1, J));
  double xS = 0.5 * (F.xi_y(z, I, J - 1) + F.xi_y(z, I - 1, J - 1));
  double zx = 0.5 * (zNE + zSE) - 0.5 * (zNW + zSW);  // (2eta-h)_E - (2eta-h)_W, L896-898
  double zy = 0.5 * (zNE + zNW) - 0.5 * (zSE + zSW);
  double ex = 8.0 * G.dx * G.dx, ey = 8.0 * G.dy * G.dy;
  double am = 2.0 * hn - zx, ap = 2.0 * hn + zx;
  double bm = 2.0 * hn - zy, bp = 2.0 * hn + zy;
  AE = -(am * (2.0 * hE + xE)) / ex;
  AW = -(ap * (2.0 * hW - xW)) / ex;
  AN = -(bm * (2.0 * hN + xN)) / ey;
  AS = -(bp * (2.0 * hS - xS)) / ey;
  AC = 2.0 + (am * (2.0 * hE - xE) + ap * (2.0 * hW + xW)) / ex +
       (bm * (2.0 * hN - xN) + bp * (2.0 * hS + xS)) / ey;
}

__global__ void __launch_bounds__(BX* BY)
k_coeffs(NhGrid G, const double* __restrict__ h, const double* __restrict__ z,
         double* __restrict__ dg, double* __restrict__ dinv, double* __restrict__ cE,
         double* __restrict__ cW, double* __restrict__ cN, double* __restrict__ cS) {
  int I = blockIdx.x * BX + threadIdx.x, J = blockIdx.y * BY + threadIdx.y;
  if (I >= G.nnx || J >= G.nny) return;
  Fld F{G, node_interior(G, I, J)};
  double AC, AE, AW, AN, AS;
  node_coeffs(F, h, z, I, J, AC, AE, AW, AN, AS);
  size_t k = (size_t)J * G.np + I;
  dg[k] = AC; dinv[k] = 1.0 / AC;
  cE[k] = AE; cW[k] = AW; cN[k] = AN; cS[k] = AS;
}

// Column scaling for the right-preconditioned operator A M^-1, M = diag(A_C) (R14):
// (A M^-1)_{n,nb} = A_{n,nb} / A_C(nb); its diagonal is 1.
__global__ void __launch_bounds__(BX* BY)
k_scale_coeffs(NhGrid G, const double* __restrict__ dinv, double* __restrict__ cE,
               double* __restrict__ cW, double* __restrict__ cN, double* __restrict__ cS) {
  int I = blockIdx.x * BX + threadIdx.x, J = blockIdx.y * BY + threadIdx.y;
  if (I >= G.nnx || J >= G.nny) return;
  Fld F{G, node_interior(G, I, J)};
  size_t k = (size_t)J * G.np + I;
  cE[k] = cE[k] * F.node(dinv, I + 1, J);
  cW[k] = cW[k] * F.node(dinv, I - 1, J);
  cN[k] = cN[k] * F.node(dinv, I, J + 1);
  cS[k] = cS[k] * F.node(dinv, I, J - 1);
}

// Row scaling for solver 1 (the paper's Jacobi method, R28): c_X = A_X / A_C, b' = b / A_C; the
// Gershgorin radius rho = max_n ((|c_E|+|c_W|)+|c_N|)+|c_S| and max |b'| are reduced exactly
// (max of non-negative doubles = integer max of their bit patterns).
__global__ void __launch_bounds__(BX* BY)
k_scale_rows(NhGrid G, const double* __restrict__ dinv, double* __restrict__ cE,
             double* __restrict__ cW, double* __restrict__ cN, double* __restrict__ cS,
             const double* __restrict__ b, double* __restrict__ bp, NhScal* sc) {
  int I = blockIdx.x * BX + threadIdx.x, J = blockIdx.y * BY + threadIdx.y;
  double rad = 0.0, bm = 0.0;
  if (I < G.nnx && J < G.nny) {
    size_t k = (size_t)J * G.np + I;
    double di = dinv[k];
    double e = cE[k] * di, w = cW[k] * di, n = cN[k] * di, s = cS[k] * di;
    cE[k] = e; cW[k] = w; cN[k] = n; cS[k] = s;
    double v = b[k] * di;
    bp[k] = v;
    rad = ((fabs(e) + fabs(w)) + fabs(n)) + fabs(s);
    bm = fabs(v);
  }
  // NaN sorts above every finite pattern, so a NaN in b' or in a coefficient survives the max
  unsigned long long rb = (unsigned long long)__double_as_longlong(rad);
  unsigned long long bb = (unsigned long long)__double_as_longlong(bm);
  for (int o = 16; o > 0; o >>= 1) {
    unsigned long long t = __shfl_xor_sync(0xffffffffu, rb, o);
    rb = t > rb ? t : rb;
    t = __shfl_xor_sync(0xffffffffu, bb, o);
    bb = t > bb ? t : bb;
  }
  if (((threadIdx.y * BX + threadIdx.x) & 31) == 0) {
    if (rb) atomicMax(&sc->srj_rho_bits, rb);
    if (bb) atomicMax(&sc->srj_bmax_bits, bb);
  }
}

// y = A x on the distinct nodes, coefficients recomputed from (h, z) on the fly (matrix-free,
// L535-537); neighbours through the node maps (R10).
__global__ void __launch_bounds__(BX* BY)
k_apply_A(NhGrid G, const double* __restrict__ h, const double* __restrict__ z,
          const double* __restrict__ x, double* __restrict__ y) {
  int I = blockIdx.x * BX + threadIdx.x, J = blockIdx.y * BY + threadIdx.y;
  if (I >= G.nnx || J >= G.nny) return;
  Fld F{G, node_interior(G, I, J)};
  double AC, AE, AW, AN, AS;
  node_coeffs(F, h, z, I, J, AC, AE, AW, AN, AS);
  size_t k = (size_t)J * G.np + I;
  y[k] = AC * x[k] + AE * F.node(x, I + 1, J) + AW * F.node(x, I - 1, J) +
         AN * F.node(x, I, J + 1) + AS * F.node(x, I, J - 1);
}

// S7: discrete constraint B of (37)-(40) at node (I,J); b = -B/dt (R15).
__device__ __forceinline__ double node_B(const Fld& F, const double* __restrict__ h,
                                         const double* __restrict__ qx,
                                         const double* __restrict__ qy,
                                         const double* __restrict__ z, double wn, int I, int J) {
  const NhGrid& G = F.G;
  double hn = F.hnode(h, I, J);
  double q1E = 0.5 * (F.xn(qx, I, J) + F.xn(qx, I, J - 1));
  double q1W = 0.5 * (F.xn(qx, I - 1, J) + F.xn(qx, I - 1, J - 1));
  double q2N = 0.5 * (F.yn(qy, I, J) + F.yn(qy, I - 1, J));
  double q2S = 0.5 * (F.yn(qy, I, J - 1) + F.yn(qy, I - 1, J - 1));
  double zE = 0.5 * (F.even(z, I, J) + F.even(z, I, J - 1));
  double zW = 0.5 * (F.even(z, I - 1, J) + F.even(z, I - 1, J - 1));
  double zN = 0.5 * (F.even(z, I, J) + F.even(z, I - 1, J));
  double zS = 0.5 * (F.even(z, I, J - 1) + F.even(z, I - 1, J - 1));
  double divq = (q1E - q1W) / G.dx + (q2N - q2S) / G.dy;
  return hn * divq - 0.5 * (q1E + q1W) * (zE - zW) / G.dx - 0.5 * (q2N + q2S) * (zN - zS) / G.dy +
         2.0 * hn * wn;
}

__global__ void __launch_bounds__(BX* BY)
k_rhs(NhGrid G, const NhScal* sc, int constraint_only, const double* __restrict__ h,
      const double* __restrict__ qx, const double* __restrict__ qy, const double* __restrict__ z,
      const double* __restrict__ w, double* __restrict__ b) {
  int I = blockIdx.x * BX + threadIdx.x, J = blockIdx.y * BY + threadIdx.y;
  if (I >= G.nnx || J >= G.nny) return;
  Fld F{G, node_interior(G, I, J)};
  size_t k = (size_t)J * G.np + I;
  double B = node_B(F, h, qx, qy, z, w[k], I, J);
  const double dt = sc->dt;
  b[k] = constraint_only ? B : ((dt > 0.0) ? -B / dt : 0.0);  // R26: dt = 0 (all dry) => b = 0
}

// Solver 1, whole assembly of a stage in one kernel (k_rhs + k_coeffs + k_scale_rows with the same
// arithmetic, 3 kernels and 11 plane round trips less): right-hand side, rows, row scaling,
// Gershgorin radius and max |b'|.
__global__ void __launch_bounds__(BX* BY)
k_assemble_rows(NhGrid G, NhScal* sc, const double* __restrict__ h, const double* __restrict__ qx,
                const double* __restrict__ qy, const double* __restrict__ z,
                const double* __restrict__ w, double* __restrict__ cE, double* __restrict__ cW,
                double* __restrict__ cN, double* __restrict__ cS, double* __restrict__ bp) {
  int I = blockIdx.x * BX + threadIdx.x, J = blockIdx.y * BY + threadIdx.y;
  double rad = 0.0, bm = 0.0;
  if (I < G.nnx && J < G.nny) {
    Fld F{G, node_interior(G, I, J)};
    size_t k = (size_t)J * G.np + I;
    double AC, AE, AW, AN, AS;
    node_coeffs(F, h, z, I, J, AC, AE, AW, AN, AS);
    double B = node_B(F, h, qx, qy, z, w[k], I, J);
    const double dt = sc->dt;
    double bv = (dt > 0.0) ? -B / dt : 0.0;
    double di = 1.0 / AC;
    double e = AE * di, ww = AW * di, n = AN * di, s = AS * di;
    cE[k] = e; cW[k] = ww; cN[k] = n; cS[k] = s;
    double v = bv * di;
    bp[k] = v;
    rad = ((fabs(e) + fabs(ww)) + fabs(n)) + fabs(s);
    bm = fabs(v);
  }
  unsigned long long rb = (unsigned long long)__double_as_longlong(rad);
  unsigned long long bb = (unsigned long long)__double_as_longlong(bm);
  for (int o = 16; o > 0; o >>= 1) {
    unsigned long long t = __shfl_xor_sync(0xffffffffu, rb, o);
    rb = t > rb ? t : rb;
    t = __shfl_xor_sync(0xffffffffu, bb, o);
    bb = t > bb ? t : bb;
  }
  if (((threadIdx.y * BX + threadIdx.x) & 31) == 0) {
    if (rb) atomicMax(&sc->srj_rho_bits, rb);
    if (bb) atomicMax(&sc->srj_bmax_bits, bb);
  }
}

// S6: breaking sources at cells (section 3, eqs (9)-(12); 2D reading R12): q** = q* + dt R_u
__global__ void __launch_bounds__(BX* BY)
k_break_cells(NhGrid G, const NhScal* sc, double g, double delta, double eps, double B1, double B2,
              const double* __restrict__ H, const double* __restrict__ h,
              const double* __restrict__ qx1, const double* __restrict__ qy1,
              unsigned char* __restrict__ flag_c, double* __restrict__ qx2,
              double* __restrict__ qy2) {
  int i = blockIdx.x * BX + threadIdx.x, j = blockIdx.y * BY + threadIdx.y;
  if (i >= G.nx || j >= G.ny) return;
  Fld F{G};
  const double dt = sc->dt;
  size_t k = (size_t)j * G.nx + i;
  double nu = 0.0, divu = 0.0;
  double hk = h[k];
  if (hk > eps) {
    double qxp = F.xn(qx1, i + 1, j), qxm = F.xn(qx1, i - 1, j);
    double qyp = F.yn(qy1, i, j + 1), qym = F.yn(qy1, i, j - 1);
    double divq = (qxp - qxm) / (2.0 * G.dx) + (qyp - qym) / (2.0 * G.dy);
    // velocities of U* at the four neighbours (ghost sign applied to the velocity, like the
    // discharge: dsg is odd in q)
    double sx, sy;
    int ip = nh_map_cell(i + 1, G.nx, G.bxlo, G.bxhi, sx);
    double up = sx * nh_dsg(h[(size_t)j * G.nx + ip], qx1[(size_t)j * G.nx + ip], delta);
    int im = nh_map_cell(i - 1, G.nx, G.bxlo, G.bxhi, sx);
    double um = sx * nh_dsg(h[(size_t)j * G.nx + im], qx1[(size_t)j * G.nx + im], delta);
    int jp = nh_map_cell(j + 1, G.ny, G.bylo, G.byhi, sy);
    double vp = sy * nh_dsg(h[(size_t)jp * G.nx + i], qy1[(size_t)jp * G.nx + i], delta);
    int jm = nh_map_cell(j - 1, G.ny, G.bylo, G.byhi, sy);
    double vm = sy * nh_dsg(h[(size_t)jm * G.nx + i], qy1[(size_t)jm * G.nx + i], delta);
    divu = (up - um) / (2.0 * G.dx) + (vp - vm) / (2.0 * G.dy);
    double cc = sqrt(g * hk);
    double U1 = B1 * cc, U2 = B2 * cc;
    int fl = (fabs(divq) >= U1) || (flag_c[k] && fabs(divq) >= U2);  // R11
    flag_c[k] = (unsigned char)fl;
    if (fl) {
      double B = 1.0 - divq / U1;  // (9)
      nu = fmax(B, 0.0) * hk * fabs(divq);
    }
  } else {
    flag_c[k] = 0;
  }
  double Hx = (F.even(H, i + 1, j) - F.even(H, i - 1, j)) / (2.0 * G.dx);
  double Hy = (F.even(H, i, j + 1) - F.even(H, i, j - 1)) / (2.0 * G.dy);
  qx2[k] = qx1[k] + dt * (2.0 * nu * divu * Hx);  // R_u, L224
  qy2[k] = qy1[k] + dt * (2.0 * nu * divu * Hy);
}

// S6 at nodes (R13): w** = w + dt R_w, compact edge averages of (39)
__global__ void __launch_bounds__(BX* BY)
k_break_nodes(NhGrid G, const NhScal* sc, double g, double delta, double eps, double B1, double B2,
              const double* __restrict__ h, const double* __restrict__ qx1,
              const double* __restrict__ qy1, const double* __restrict__ w_in,
              unsigned char* __restrict__ flag_n, double* __restrict__ w2) {
  int I = blockIdx.x * BX + threadIdx.x, J = blockIdx.y * BY + threadIdx.y;
  if (I >= G.nnx || J >= G.nny) return;
  Fld F{G};
  const double dt = sc->dt;
  size_t k = (size_t)J * G.np + I;
  double hn = F.hnode(h, I, J);
  double nu = 0.0, divu = 0.0;
  if (hn > eps) {
    // the four cells around the node: index maps once, then discharge and velocity of each
    double sxm, sxp, sym, syp;
    int im = nh_map_cell(I - 1, G.nx, G.bxlo, G.bxhi, sxm), ip = nh_map_cell(I, G.nx, G.bxlo, G.bxhi, sxp);
    int jm = nh_map_cell(J - 1, G.ny, G.bylo, G.byhi, sym), jp = nh_map_cell(J, G.ny, G.bylo, G.byhi, syp);
    size_t kNE = (size_t)jp * G.nx + ip, kSE = (size_t)jm * G.nx + ip;
    size_t kNW = (size_t)jp * G.nx + im, kSW = (size_t)jm * G.nx + im;
    double qxNE = sxp * qx1[kNE], qxSE = sxp * qx1[kSE], qxNW = sxm * qx1[kNW], qxSW = sxm * qx1[kSW];
    double qyNE = syp * qy1[kNE], qyNW = syp * qy1[kNW], qySE = sym * qy1[kSE], qySW = sym * qy1[kSW];
    double uNE = sxp * nh_dsg(h[kNE], qx1[kNE], delta), uSE = sxp * nh_dsg(h[kSE], qx1[kSE], delta);
    double uNW = sxm * nh_dsg(h[kNW], qx1[kNW], delta), uSW = sxm * nh_dsg(h[kSW], qx1[kSW], delta);
    double vNE = syp * nh_dsg(h[kNE], qy1[kNE], delta), vNW = syp * nh_dsg(h[kNW], qy1[kNW], delta);
    double vSE = sym * nh_dsg(h[kSE], qy1[kSE], delta), vSW = sym * nh_dsg(h[kSW], qy1[kSW], delta);
    double q1E = 0.5 * (qxNE + qxSE), q1W = 0.5 * (qxNW + qxSW);
    double q2N = 0.5 * (qyNE + qyNW), q2S = 0.5 * (qySE + qySW);
    double u1E = 0.5 * (uNE + uSE), u1W = 0.5 * (uNW + uSW);
    double u2N = 0.5 * (vNE + vNW), u2S = 0.5 * (vSE + vSW);
    double divq = (q1E - q1W) / G.dx + (q2N - q2S) / G.dy;
    divu = (u1E - u1W) / G.dx + (u2N - u2S) / G.dy;
    double cc = sqrt(g * hn);
    double U1 = B1 * cc, U2 = B2 * cc;
    int fl = (fabs(divq) >= U1) || (flag_n[k] && fabs(divq) >= U2);
    flag_n[k] = (unsigned char)fl;
    if (fl) {
      double B = 1.0 - divq / U1;
      nu = fmax(B, 0.0) * hn * fabs(divq);
    }
  } else {
    flag_n[k] = 0;
  }
  w2[k] = w_in[k] + dt * (2.0 * nu * divu);  // R_w, L224
}

// S5b (w-advection variant of [7]; reading R30): (hw)_t + div(hw u) = p with
// h_t + div q = 0 is w_t + u . grad w = p / h.  Transport part, before S6: first-order upwind
// differences between neighbouring nodes, node velocity = mean of the desingularised velocities (S0)
// of the four cells around the node in the stage input (ghost cells through the maps of R9, so the
// normal velocity of a wall node is 0).  Same operation order as the oracle: bit-exact.
__global__ void __launch_bounds__(BX* BY)
k_w_advect(NhGrid G, const NhScal* sc, double delta, const double* __restrict__ h,
           const double* __restrict__ qx, const double* __restrict__ qy,
           const double* __restrict__ w_in, double* __restrict__ w_out) {
  int I = blockIdx.x * BX + threadIdx.x, J = blockIdx.y * BY + threadIdx.y;
  if (I >= G.nnx || J >= G.nny) return;
  Fld F{G};
  double sxm, sxp, sym, syp;
  int im = nh_map_cell(I - 1, G.nx, G.bxlo, G.bxhi, sxm), ip = nh_map_cell(I, G.nx, G.bxlo, G.bxhi, sxp);
  int jm = nh_map_cell(J - 1, G.ny, G.bylo, G.byhi, sym), jp = nh_map_cell(J, G.ny, G.bylo, G.byhi, syp);
  size_t kNE = (size_t)jp * G.nx + ip, kSE = (size_t)jm * G.nx + ip;
  size_t kNW = (size_t)jp * G.nx + im, kSW = (size_t)jm * G.nx + im;
  double uSW = sxm * nh_dsg(h[kSW], qx[kSW], delta), uSE = sxp * nh_dsg(h[kSE], qx[kSE], delta);
  double uNE = sxp * nh_dsg(h[kNE], qx[kNE], delta), uNW = sxm * nh_dsg(h[kNW], qx[kNW], delta);
  double vSW = sym * nh_dsg(h[kSW], qy[kSW], delta), vSE = sym * nh_dsg(h[kSE], qy[kSE], delta);
  double vNE = syp * nh_dsg(h[kNE], qy[kNE], delta), vNW = syp * nh_dsg(h[kNW], qy[kNW], delta);
  double un = 0.25 * (uSW + uSE + uNE + uNW);
  double vn = 0.25 * (vSW + vSE + vNE + vNW);
  double wc = w_in[(size_t)J * G.np + I];
  double wx = (un > 0.0) ? (wc - F.node(w_in, I - 1, J)) / G.dx : (F.node(w_in, I + 1, J) - wc) / G.dx;
  double wy = (vn > 0.0) ? (wc - F.node(w_in, I, J - 1)) / G.dy : (F.node(w_in, I, J + 1) - wc) / G.dy;
  w_out[(size_t)J * G.np + I] = wc - sc->dt * (un * wx + vn * wy);
}

// S10: correction, eqs (36),(41): q <- q** + dt T_NH(p) at cells
__global__ void __launch_bounds__(BX* BY)
k_correct_cells(NhGrid G, const NhScal* sc, const double* __restrict__ h,
                const double* __restrict__ z, const double* __restrict__ qx2,
                const double* __restrict__ qy2, const double* __restrict__ pt,
                double* __restrict__ qx_out, double* __restrict__ qy_out) {
  int i = blockIdx.x * BX + threadIdx.x, j = blockIdx.y * BY + threadIdx.y;
  if (i >= G.nx || j >= G.ny) return;
  // cells i-1..i+1, j-1..j+1 and nodes i..i+1, j..j+1 inside the grid (periodic: node n wraps)
  Fld F{G, i >= 1 && i <= G.nx - 2 && j >= 1 && j <= G.ny - 2};
  const double dt = sc->dt;
  size_t k = (size_t)j * G.nx + i;
  // corner nodes of cell (i,j): (i,j) (i+1,j) (i,j+1) (i+1,j+1)
  double p00 = F.node(pt, i, j), p10 = F.node(pt, i + 1, j);
  double p01 = F.node(pt, i, j + 1), p11 = F.node(pt, i + 1, j + 1);
  double pE = 0.5 * (p11 + p10), pW = 0.5 * (p01 + p00);
  double pN = 0.5 * (p11 + p01), pS = 0.5 * (p10 + p00);
  double xx = F.xi_x(z, i, j), xy = F.xi_y(z, i, j);
  double hk = h[k];
  qx_out[k] = qx2[k] - dt / (4.0 * G.dx) * ((2.0 * hk + xx) * pE + (xx - 2.0 * hk) * pW);
  qy_out[k] = qy2[k] - dt / (4.0 * G.dy) * ((2.0 * hk + xy) * pN + (xy - 2.0 * hk) * pS);
}

// S10 at nodes: w <- w** + dt p dinv(h_n)  (R16)
__global__ void __launch_bounds__(BX* BY)
k_correct_nodes(NhGrid G, const NhScal* sc, double delta, const double* __restrict__ h,
                const double* __restrict__ w2, const double* __restrict__ pt,
                double* __restrict__ w_out) {
  int I = blockIdx.x * BX + threadIdx.x, J = blockIdx.y * BY + threadIdx.y;
  if (I >= G.nnx || J >= G.nny) return;
  Fld F{G, node_interior(G, I, J)};
  size_t k = (size_t)J * G.np + I;
  double hn = F.hnode(h, I, J);
  w_out[k] = w2[k] + sc->dt * pt[k] * nh_dinv_h(hn, delta);
}

// S11: generating relaxation zone at x-lo (L417-431, reading R18), target at the stage's end time
__device__ __forceinline__ double relax_m_cell(double L, double dx, int i) {
  double x = ((double)i + 0.5) * dx;
  double d = L - x;
  if (d <= 0.0) return 1.0;
  if (d >= L) return 0.0;
  return sqrt(1.0 - (d / L) * (d / L));
}
__global__ void __launch_bounds__(256)
k_relax(NhGrid G, const NhScal* sc, int stage, double g, double A, double h0, double x0, double L,
        int krel, const double* __restrict__ H, double* __restrict__ h, double* __restrict__ qx,
        double* __restrict__ qy, double* __restrict__ w, double* __restrict__ p) {
  const double kk = sqrt(3.0 * A / (4.0 * h0 * h0 * h0));
  const double cel = sqrt(g * (h0 + A));
  // stage 0 ends at t + dt, stage 1 at (t + dt) + dt (the second stage starts from t + dt)
  double tt = sc->t + sc->dt;
  if (stage == 1) tt = tt + sc->dt;
  int ncol = krel + 1;
  size_t tot = (size_t)ncol * (G.ny + 1);
  for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < tot;
       e += (size_t)gridDim.x * blockDim.x) {
    int i = (int)(e % ncol), j = (int)(e / ncol);
    if (i < krel && j < G.ny) {
      size_t k = (size_t)j * G.nx + i;
      double m = relax_m_cell(L, G.dx, i);
      double x = ((double)i + 0.5) * G.dx;
      double etas = A * nh_sech2_fixed(kk * (x - x0 - cel * tt));  // R31
      double hs = fmax(H[k] + etas, 0.0);
      h[k] = m * h[k] + (1.0 - m) * hs;
      qx[k] = m * qx[k] + (1.0 - m) * (cel * etas);
      qy[k] = m * qy[k];
    }
    if (i <= krel && i < G.nnx && j < G.nny) {
      size_t k = (size_t)j * G.np + i;
      double mL = (i - 1 >= 0) ? relax_m_cell(L, G.dx, i - 1) : 0.0;
      double mR = (i < G.nx) ? relax_m_cell(L, G.dx, i) : 1.0;
      double m = 0.5 * (mL + mR);  // m_{i+-1/2}, L429
      w[k] = m * w[k];
      p[k] = m * p[k];
    }
  }
}

// S11b: absorbing relaxation zone on one side (L415-440; R18, R29): the relaxation of S11 towards
// eta* = 0, q* = w* = p* = 0, a <- a + (1 - m)(a* - a), m = sqrt(1 - (d/L)^2), d from the inner end
// of the zone; node coefficients are the mean of the two adjacent cell coefficients (0 beyond the
// boundary).  side: 0 x-lo, 1 x-hi, 2 y-lo, 3 y-hi; s = distance from the boundary in cells / lines.
__device__ __forceinline__ double absorb_m(double L, double dxy, int s) {
  double x = ((double)s + 0.5) * dxy;
  double d = L - x;
  if (d <= 0.0) return 1.0;
  if (d >= L) return 0.0;
  return sqrt(1.0 - (d / L) * (d / L));
}
__global__ void __launch_bounds__(256)
k_absorb(NhGrid G, int side, double L, int krel, const double* __restrict__ H,
         double* __restrict__ h, double* __restrict__ qx, double* __restrict__ qy,
         double* __restrict__ w, double* __restrict__ p) {
  const bool xdir = side < 2, hi = side & 1;
  const int n = xdir ? G.nx : G.ny;
  const double dxy = xdir ? G.dx : G.dy;
  const int nother = xdir ? G.ny : G.nx;  // both zone directions are non-periodic: n + 1 node lines
  const int nnother = xdir ? G.nny : G.nnx;
  const int ns = krel + 1;
  size_t tot = (size_t)ns * (nother + 1);
  for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < tot;
       e += (size_t)gridDim.x * blockDim.x) {
    int s = (int)(e % ns), t = (int)(e / ns);
    if (s < krel && t < nother) {
      int a = hi ? n - 1 - s : s;
      size_t k = xdir ? (size_t)t * G.nx + a : (size_t)a * G.nx + t;
      double f = 1.0 - absorb_m(L, dxy, s);
      double hs = fmax(H[k], 0.0);
      h[k] = h[k] + f * (hs - h[k]);
      qx[k] = qx[k] + f * (0.0 - qx[k]);
      qy[k] = qy[k] + f * (0.0 - qy[k]);
    }
    if (t < nnother) {
      int a = hi ? n - s : s;
      double mo = (s - 1 >= 0) ? absorb_m(L, dxy, s - 1) : 0.0;
      double mi = (s < n) ? absorb_m(L, dxy, s) : 1.0;
      double f = 1.0 - 0.5 * (mo + mi);
      size_t k = xdir ? (size_t)t * G.np + a : (size_t)a * G.np + t;
      w[k] = w[k] + f * (0.0 - w[k]);
      p[k] = p[k] + f * (0.0 - p[k]);
    }
  }
}

// internal plane -> dense public node layout: fill the duplicate lines of periodic directions
__global__ void __launch_bounds__(BX* BY)
k_nodes_out(NhGrid G, const double* __restrict__ src, double* __restrict__ dst) {
  int I = blockIdx.x * BX + threadIdx.x, J = blockIdx.y * BY + threadIdx.y;
  if (I > G.nx || J > G.ny) return;
  int II = (I == G.nx && G.nnx == G.nx) ? 0 : I;
  int JJ = (J == G.ny && G.nny == G.ny) ? 0 : J;
  dst[(size_t)J * (G.nx + 1) + I] = src[(size_t)JJ * G.np + II];
}

dim3 grid2(int nx, int ny) { return dim3((nx + BX - 1) / BX, (ny + BY - 1) / BY); }
int grid_1d(const nh_ctx* c, size_t n, int block) {
  size_t need = (n + block - 1) / block;
  size_t cap = (size_t)c->sm_count * 16;
  return (int)(need < cap ? (need ? need : 1) : cap);
}

}  // namespace

void nh_launch_compute_z(nh_ctx* c, const double* h, double* z) {
  k_compute_z<<<grid_1d(c, c->nc, 256), 256, 0, c->stream>>>(c->nc, h, c->H, z);
  c->launches++;
}
void nh_launch_cell_planes(nh_ctx* c, const double* h) {
  k_cell_planes<<<grid2(c->g.nx + 4, c->g.ny + 4), dim3(BX, BY), 0, c->stream>>>(c->g, h, c->H, c->z,
                                                                                c->hc, c->zc);
  c->launches++;
}
void nh_launch_breaking(nh_ctx* c, const double* h, const double* qx1, const double* qy1,
                        const double* w_in, double* qx2, double* qy2, double* w2) {
  const nh_params& P = c->prm;
  k_break_cells<<<grid2(c->g.nx, c->g.ny), dim3(BX, BY), 0, c->stream>>>(
      c->g, c->sc, P.g, P.delta, P.eps_dry, P.B1, P.B2, c->H, h, qx1, qy1, c->flag_c, qx2, qy2);
  k_break_nodes<<<grid2(c->g.nnx, c->g.nny), dim3(BX, BY), 0, c->stream>>>(
      c->g, c->sc, P.g, P.delta, P.eps_dry, P.B1, P.B2, h, qx1, qy1, w_in, c->flag_n, w2);
  c->launches += 2;
}
void nh_launch_rhs(nh_ctx* c, const double* h, const double* qx, const double* qy, const double* z,
                   const double* w, double* b, int constraint_only) {
  k_rhs<<<grid2(c->g.nnx, c->g.nny), dim3(BX, BY), 0, c->stream>>>(c->g, c->sc, constraint_only, h,
                                                                  qx, qy, z, w, b);
  c->launches++;
}
void nh_launch_coeffs(nh_ctx* c, const double* h, const double* z) {
  k_coeffs<<<grid2(c->g.nnx, c->g.nny), dim3(BX, BY), 0, c->stream>>>(c->g, h, z, c->dg, c->dinv,
                                                                     c->cE, c->cW, c->cN, c->cS);
  c->launches++;
}
void nh_launch_scale_coeffs(nh_ctx* c) {
  k_scale_coeffs<<<grid2(c->g.nnx, c->g.nny), dim3(BX, BY), 0, c->stream>>>(c->g, c->dinv, c->cE,
                                                                           c->cW, c->cN, c->cS);
  c->launches++;
}
void nh_launch_scale_rows(nh_ctx* c, const double* b, double* bp) {
  k_scale_rows<<<grid2(c->g.nnx, c->g.nny), dim3(BX, BY), 0, c->stream>>>(
      c->g, c->dinv, c->cE, c->cW, c->cN, c->cS, b, bp, c->sc);
  c->launches++;
}
void nh_launch_assemble_rows(nh_ctx* c, const double* h, const double* qx, const double* qy,
                             const double* z, const double* w, double* bp) {
  k_assemble_rows<<<grid2(c->g.nnx, c->g.nny), dim3(BX, BY), 0, c->stream>>>(
      c->g, c->sc, h, qx, qy, z, w, c->cE, c->cW, c->cN, c->cS, bp);
  c->launches++;
}
void nh_launch_apply_A(nh_ctx* c, const double* h, const double* z, const double* x, double* y) {
  k_apply_A<<<grid2(c->g.nnx, c->g.nny), dim3(BX, BY), 0, c->stream>>>(c->g, h, z, x, y);
  c->launches++;
}
void nh_launch_correct(nh_ctx* c, const double* h, const double* z, const double* qx2,
                       const double* qy2, const double* w2, const double* p, double* qx_out,
                       double* qy_out, double* w_out) {
  k_correct_cells<<<grid2(c->g.nx, c->g.ny), dim3(BX, BY), 0, c->stream>>>(c->g, c->sc, h, z, qx2,
                                                                          qy2, p, qx_out, qy_out);
  k_correct_nodes<<<grid2(c->g.nnx, c->g.nny), dim3(BX, BY), 0, c->stream>>>(
      c->g, c->sc, c->prm.delta, h, w2, p, w_out);
  c->launches += 2;
}
void nh_launch_w_advect(nh_ctx* c, const double* h, const double* qx, const double* qy,
                        const double* w_in, double* w_out) {
  k_w_advect<<<grid2(c->g.nnx, c->g.nny), dim3(BX, BY), 0, c->stream>>>(c->g, c->sc, c->prm.delta, h,
                                                                       qx, qy, w_in, w_out);
  c->launches++;
}
void nh_launch_relax(nh_ctx* c, double* h, double* qx, double* qy, double* w, double* p, int stage) {
  const nh_params& P = c->prm;
  int krel = (int)ceil(P.gen_Lrel / c->g.dx);
  if (krel > c->g.nx) krel = c->g.nx;
  size_t tot = (size_t)(krel + 1) * (c->g.ny + 1);
  k_relax<<<grid_1d(c, tot, 256), 256, 0, c->stream>>>(c->g, c->sc, stage, P.g, P.gen_A, P.gen_h0,
                                                       P.gen_x0, P.gen_Lrel, krel, c->H, h, qx, qy,
                                                       w, p);
  c->launches++;
}
void nh_launch_absorb(nh_ctx* c, double* h, double* qx, double* qy, double* w, double* p) {
  const double L[4] = {c->prm.abs_xlo, c->prm.abs_xhi, c->prm.abs_ylo, c->prm.abs_yhi};
  for (int side = 0; side < 4; ++side) {
    if (!(L[side] > 0.0)) continue;
    const bool xdir = side < 2;
    const int n = xdir ? c->g.nx : c->g.ny, nother = xdir ? c->g.ny : c->g.nx;
    int krel = (int)ceil(L[side] / (xdir ? c->g.dx : c->g.dy));
    if (krel > n) krel = n;
    size_t tot = (size_t)(krel + 1) * (nother + 1);
    k_absorb<<<grid_1d(c, tot, 256), 256, 0, c->stream>>>(c->g, side, L[side], krel, c->H, h, qx, qy,
                                                          w, p);
    c->launches++;
  }
}
void nh_launch_nodes_out(nh_ctx* c, const double* src, double* dst) {
  k_nodes_out<<<grid2(c->g.nx + 1, c->g.ny + 1), dim3(BX, BY), 0, c->stream>>>(c->g, src, dst);
  c->launches++;
}
