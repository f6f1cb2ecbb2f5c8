// nh_pressure.cu -- second and third parts of the time step, outside the Krylov loop:
// breaking sources (a4), right-hand side (a5), the cell planes of the matrix-free solver, the rows
// of the compact finite-difference pressure operator (S8: solver 1 and the test hooks), the
// matrix-free operator apply (test hook), the w transport (R30), the start vector (R32), the
// Chorin-Temam correction (a7) and the relaxation zones (a9).
//
// These kernels run once per Runge-Kutta stage (the solver runs 10^2 iterations per stage), so
// they read their small stencils straight from global memory through the boundary index maps
// (L1/L2 serve the overlap) instead of staging tiles.
#include <math.h>
#include <stdio.h>

#include "nh_internal.cuh"

namespace NH_NS {
namespace {

constexpr int BX = 32, BY = 8;

struct Fld {  // read-only field + grid: ghost access S1 (R9)
  const NhGrid& G;
  bool fast;  // every cell / node this thread touches is inside the grid: no index maps, no signs
  __device__ __forceinline__ real even(const real* __restrict__ a, int i, int j) const {
    if (fast) return a[(size_t)j * G.nx + i];
    int ii = nh_map_cell_even(i, G.nx, G.bxlo, G.bxhi);
    int jj = nh_map_cell_even(j, G.ny, G.bylo, G.byhi);
    return a[(size_t)jj * G.nx + ii];
  }
  __device__ __forceinline__ real xn(const real* __restrict__ a, int i, int j) const {
    if (fast) return a[(size_t)j * G.nx + i];
    real sx;
    int ii = nh_map_cell(i, G.nx, G.bxlo, G.bxhi, sx);
    int jj = nh_map_cell_even(j, G.ny, G.bylo, G.byhi);
    return sx * a[(size_t)jj * G.nx + ii];
  }
  __device__ __forceinline__ real yn(const real* __restrict__ a, int i, int j) const {
    if (fast) return a[(size_t)j * G.nx + i];
    real sy;
    int ii = nh_map_cell_even(i, G.nx, G.bxlo, G.bxhi);
    int jj = nh_map_cell(j, G.ny, G.bylo, G.byhi, sy);
    return sy * a[(size_t)jj * G.nx + ii];
  }
  __device__ __forceinline__ real node(const real* __restrict__ a, int I, int J) const {
    if (fast) return a[(size_t)J * G.np + I];
    int II = nh_map_node(I, G.nx, G.bxlo);
    int JJ = nh_map_node(J, G.ny, G.bylo);
    return a[(size_t)JJ * G.np + II];
  }
  __device__ __forceinline__ real xi_x(const real* __restrict__ z, int i, int j) const {
    return RC(0.5) * (even(z, i + 1, j) - even(z, i - 1, j));
  }
  __device__ __forceinline__ real xi_y(const real* __restrict__ z, int i, int j) const {
    return RC(0.5) * (even(z, i, j + 1) - even(z, i, j - 1));
  }
  __device__ __forceinline__ real hnode(const real* __restrict__ h, int I, int J) const {
    return RC(0.25) * (even(h, I - 1, J - 1) + even(h, I, J - 1) + even(h, I, J) + even(h, I - 1, J));
  }
};

// node (I,J) whose stencils (cells I-2..I+1, J-2..J+1; nodes I-1..I+1, J-1..J+1) stay inside the grid
__device__ __forceinline__ bool node_interior(const NhGrid& G, int I, int J) {
  return I >= 2 && I + 1 <= G.nx - 1 && J >= 2 && J + 1 <= G.ny - 1;
}

// z = 2 eta - h, eq. (6)
__global__ void __launch_bounds__(256)
k_compute_z(size_t nc, const real* __restrict__ h, const real* __restrict__ H,
            real* __restrict__ z, const real* __restrict__ etap) {
  for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < nc;
       k += (size_t)gridDim.x * blockDim.x) {
    if (kEta) {  // fp32 variant: z = eta - H from the stored eta (2 eta - h would lose it in h)
      z[k] = etap[k] - H[k];
    } else {
      real eta = h[k] - H[k];
      z[k] = RC(2.0) * eta - h[k];
    }
  }
}

// z = 2 eta - h (eq. (6)) as the dense cell plane, and the operands of the matrix-free solver
// (nh_solver.cu): h and z in the node layout shifted by one column (plane column P = cell P - 1),
// cells -2 .. nx+1 by -2 .. ny+1 through the even cell maps (R9: h, H, eta are even in every ghost).
__global__ void __launch_bounds__(BX* BY)
k_cell_planes(NhGrid G, const real* __restrict__ h, const real* __restrict__ H,
              real* __restrict__ z, real* __restrict__ hc, real* __restrict__ zc,
              const real* __restrict__ etap) {
  int i = (int)(blockIdx.x * BX + threadIdx.x) - 2, j = (int)(blockIdx.y * BY + threadIdx.y) - 2;
  if (i > G.nx + 1 || j > G.ny + 1) return;
  int ii = nh_map_cell_even(i, G.nx, G.bxlo, G.bxhi);
  int jj = nh_map_cell_even(j, G.ny, G.bylo, G.byhi);
  size_t k = (size_t)jj * G.nx + ii;
  real hv = h[k];
  real zv;
  if (kEta) {
    zv = etap[k] - H[k];
  } else {
    real eta = hv - H[k];
    zv = RC(2.0) * eta - hv;
  }
  if (ii == i && jj == j) z[k] = zv;
  long long kp = (long long)j * G.np + (i + 1);
  hc[kp] = hv; zc[kp] = zv;
}

// S8: the five coefficients of row (I,J), derived from (36)-(41); 1D restriction = (43).
__device__ __forceinline__ void node_coeffs(const Fld& F, const real* __restrict__ h,
                                            const real* __restrict__ z, int I, int J, real& AC,
                                            real& AE, real& AW, real& AN, real& AS) {
  const NhGrid& G = F.G;
  // SW=(I-1,J-1), SE=(I,J-1), NW=(I-1,J), NE=(I,J)
  real hSW = F.even(h, I - 1, J - 1), hSE = F.even(h, I, J - 1);
  real hNW = F.even(h, I - 1, J), hNE = F.even(h, I, J);
  real zSW = F.even(z, I - 1, J - 1), zSE = F.even(z, I, J - 1);
  real zNW = F.even(z, I - 1, J), zNE = F.even(z, I, J);
  real hn = RC(0.25) * (hSW + hSE + hNE + hNW);  // (38)
  real hE = RC(0.5) * (hNE + hSE), hW = RC(0.5) * (hNW + hSW);
  real hN = RC(0.5) * (hNE + hNW), hS = RC(0.5) * (hSE + hSW);
  real xE = RC(0.5) * (F.xi_x(z, I, J) + F.xi_x(z, I, J - 1));
  real xW = RC(0.5) * (F.xi_x(z, I - 1, J) + F.xi_x(z, I - 1, J - 1));
  real xN = RC(0.5) * (F.xi_y(z, I, J) + F.xi_y(z, I - 1, J));
  real xS = RC(0.5) * (F.xi_y(z, I, J - 1) + F.xi_y(z, I - 1, J - 1));
  real zx = RC(0.5) * (zNE + zSE) - RC(0.5) * (zNW + zSW);  // (2eta-h)_E - (2eta-h)_W, L896-898
  real zy = RC(0.5) * (zNE + zNW) - RC(0.5) * (zSE + zSW);
  real ex = RC(8.0) * G.dx * G.dx, ey = RC(8.0) * G.dy * G.dy;
  real am = RC(2.0) * hn - zx, ap = RC(2.0) * hn + zx;
  real bm = RC(2.0) * hn - zy, bp = RC(2.0) * hn + zy;
  AE = -(am * (RC(2.0) * hE + xE)) / ex;
  AW = -(ap * (RC(2.0) * hW - xW)) / ex;
  AN = -(bm * (RC(2.0) * hN + xN)) / ey;
  AS = -(bp * (RC(2.0) * hS - xS)) / ey;
  AC = RC(2.0) + (am * (RC(2.0) * hE - xE) + ap * (RC(2.0) * hW + xW)) / ex +
       (bm * (RC(2.0) * hN - xN) + bp * (RC(2.0) * hS + xS)) / ey;
}

__global__ void __launch_bounds__(BX* BY)
k_coeffs(NhGrid G, const real* __restrict__ h, const real* __restrict__ z,
         real* __restrict__ dg, real* __restrict__ dinv, real* __restrict__ cE,
         real* __restrict__ cW, real* __restrict__ cN, real* __restrict__ cS) {
  int I = blockIdx.x * BX + threadIdx.x, J = blockIdx.y * BY + threadIdx.y;
  if (I >= G.nnx || J >= G.nny) return;
  Fld F{G, node_interior(G, I, J)};
  real AC, AE, AW, AN, AS;
  node_coeffs(F, h, z, I, J, AC, AE, AW, AN, AS);
  size_t k = (size_t)J * G.np + I;
  dg[k] = AC; dinv[k] = RC(1.0) / AC;
  cE[k] = AE; cW[k] = AW; cN[k] = AN; cS[k] = AS;
}

// Row scaling for solver 1 (the paper's Jacobi method, R28): c_X = A_X / A_C, b' = b / A_C; the
// Gershgorin radius rho = max_n ((|c_E|+|c_W|)+|c_N|)+|c_S| and max |b'| are reduced exactly
// (max of non-negative doubles = integer max of their bit patterns).
__global__ void __launch_bounds__(BX* BY)
k_scale_rows(NhGrid G, const real* __restrict__ dinv, real* __restrict__ cE,
             real* __restrict__ cW, real* __restrict__ cN, real* __restrict__ cS,
             const real* __restrict__ b, real* __restrict__ bp, NhScal* sc) {
  int I = blockIdx.x * BX + threadIdx.x, J = blockIdx.y * BY + threadIdx.y;
  real rad = RC(0.0), bm = RC(0.0);
  if (I < G.nnx && J < G.nny) {
    size_t k = (size_t)J * G.np + I;
    real di = dinv[k];
    real e = cE[k] * di, w = cW[k] * di, n = cN[k] * di, s = cS[k] * di;
    cE[k] = e; cW[k] = w; cN[k] = n; cS[k] = s;
    real v = b[k] * di;
    bp[k] = v;
    rad = ((fabs(e) + fabs(w)) + fabs(n)) + fabs(s);
    bm = fabs(v);
  }
  // NaN sorts above every finite pattern, so a NaN in b' or in a coefficient survives the max
  unsigned long long rb = (unsigned long long)__double_as_longlong((double)rad);
  unsigned long long bb = (unsigned long long)__double_as_longlong((double)bm);
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
k_apply_A(NhGrid G, const real* __restrict__ h, const real* __restrict__ z,
          const real* __restrict__ x, real* __restrict__ y) {
  int I = blockIdx.x * BX + threadIdx.x, J = blockIdx.y * BY + threadIdx.y;
  if (I >= G.nnx || J >= G.nny) return;
  Fld F{G, node_interior(G, I, J)};
  real AC, AE, AW, AN, AS;
  node_coeffs(F, h, z, I, J, AC, AE, AW, AN, AS);
  size_t k = (size_t)J * G.np + I;
  y[k] = AC * x[k] + AE * F.node(x, I + 1, J) + AW * F.node(x, I - 1, J) +
         AN * F.node(x, I, J + 1) + AS * F.node(x, I, J - 1);
}

// S7: discrete constraint B of (37)-(40) at node (I,J); b = -B/dt (R15).
__device__ __forceinline__ real node_B(const Fld& F, const real* __restrict__ h,
                                         const real* __restrict__ qx,
                                         const real* __restrict__ qy,
                                         const real* __restrict__ z, real wn, int I, int J) {
  const NhGrid& G = F.G;
  real hn = F.hnode(h, I, J);
  real q1E = RC(0.5) * (F.xn(qx, I, J) + F.xn(qx, I, J - 1));
  real q1W = RC(0.5) * (F.xn(qx, I - 1, J) + F.xn(qx, I - 1, J - 1));
  real q2N = RC(0.5) * (F.yn(qy, I, J) + F.yn(qy, I - 1, J));
  real q2S = RC(0.5) * (F.yn(qy, I, J - 1) + F.yn(qy, I - 1, J - 1));
  real zE = RC(0.5) * (F.even(z, I, J) + F.even(z, I, J - 1));
  real zW = RC(0.5) * (F.even(z, I - 1, J) + F.even(z, I - 1, J - 1));
  real zN = RC(0.5) * (F.even(z, I, J) + F.even(z, I - 1, J));
  real zS = RC(0.5) * (F.even(z, I, J - 1) + F.even(z, I - 1, J - 1));
  real divq = (q1E - q1W) / G.dx + (q2N - q2S) / G.dy;
  return hn * divq - RC(0.5) * (q1E + q1W) * (zE - zW) / G.dx - RC(0.5) * (q2N + q2S) * (zN - zS) / G.dy +
         RC(2.0) * hn * wn;
}

__global__ void __launch_bounds__(BX* BY)
k_rhs(NhGrid G, const NhScal* sc, int constraint_only, const real* __restrict__ h,
      const real* __restrict__ qx, const real* __restrict__ qy, const real* __restrict__ z,
      const real* __restrict__ w, real* __restrict__ b) {
  int I = blockIdx.x * BX + threadIdx.x, J = blockIdx.y * BY + threadIdx.y;
  if (I >= G.nnx || J >= G.nny) return;
  Fld F{G, node_interior(G, I, J)};
  size_t k = (size_t)J * G.np + I;
  real B = node_B(F, h, qx, qy, z, w[k], I, J);
  const real dt = (real)sc->dt;
  b[k] = constraint_only ? B : ((dt > RC(0.0)) ? -B / dt : RC(0.0));  // R26: dt = 0 (all dry) => b = 0
}

// Solver 1, whole assembly of a stage in one kernel (k_rhs + k_coeffs + k_scale_rows with the same
// arithmetic, 3 kernels and 11 plane round trips less): right-hand side, rows, row scaling,
// Gershgorin radius and max |b'|.
__global__ void __launch_bounds__(BX* BY)
k_assemble_rows(NhGrid G, NhScal* sc, const real* __restrict__ h, const real* __restrict__ qx,
                const real* __restrict__ qy, const real* __restrict__ z,
                const real* __restrict__ w, real* __restrict__ cE, real* __restrict__ cW,
                real* __restrict__ cN, real* __restrict__ cS, real* __restrict__ bp) {
  int I = blockIdx.x * BX + threadIdx.x, J = blockIdx.y * BY + threadIdx.y;
  real rad = RC(0.0), bm = RC(0.0);
  if (I < G.nnx && J < G.nny) {
    Fld F{G, node_interior(G, I, J)};
    size_t k = (size_t)J * G.np + I;
    real AC, AE, AW, AN, AS;
    node_coeffs(F, h, z, I, J, AC, AE, AW, AN, AS);
    real B = node_B(F, h, qx, qy, z, w[k], I, J);
    const real dt = (real)sc->dt;
    real bv = (dt > RC(0.0)) ? -B / dt : RC(0.0);
    real di = RC(1.0) / AC;
    real e = AE * di, ww = AW * di, n = AN * di, s = AS * di;
    cE[k] = e; cW[k] = ww; cN[k] = n; cS[k] = s;
    real v = bv * di;
    bp[k] = v;
    rad = ((fabs(e) + fabs(ww)) + fabs(n)) + fabs(s);
    bm = fabs(v);
  }
  unsigned long long rb = (unsigned long long)__double_as_longlong((double)rad);
  unsigned long long bb = (unsigned long long)__double_as_longlong((double)bm);
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
k_break_cells(NhGrid G, const NhScal* sc, real g, real delta, real eps, real B1, real B2,
              const real* __restrict__ H, const real* __restrict__ h,
              const real* __restrict__ qx1, const real* __restrict__ qy1,
              unsigned char* __restrict__ flag_c, real* __restrict__ qx2,
              real* __restrict__ qy2) {
  int i = blockIdx.x * BX + threadIdx.x, j = blockIdx.y * BY + threadIdx.y;
  if (i >= G.nx || j >= G.ny) return;
  Fld F{G};
  const real dt = (real)sc->dt;
  size_t k = (size_t)j * G.nx + i;
  real nu = RC(0.0), divu = RC(0.0);
  real hk = h[k];
  if (hk > eps) {
    real qxp = F.xn(qx1, i + 1, j), qxm = F.xn(qx1, i - 1, j);
    real qyp = F.yn(qy1, i, j + 1), qym = F.yn(qy1, i, j - 1);
    real divq = (qxp - qxm) / (RC(2.0) * G.dx) + (qyp - qym) / (RC(2.0) * G.dy);
    // velocities of U* at the four neighbours (ghost sign applied to the velocity, like the
    // discharge: dsg is odd in q)
    real sx, sy;
    int ip = nh_map_cell(i + 1, G.nx, G.bxlo, G.bxhi, sx);
    real up = sx * nh_dsg(h[(size_t)j * G.nx + ip], qx1[(size_t)j * G.nx + ip], delta);
    int im = nh_map_cell(i - 1, G.nx, G.bxlo, G.bxhi, sx);
    real um = sx * nh_dsg(h[(size_t)j * G.nx + im], qx1[(size_t)j * G.nx + im], delta);
    int jp = nh_map_cell(j + 1, G.ny, G.bylo, G.byhi, sy);
    real vp = sy * nh_dsg(h[(size_t)jp * G.nx + i], qy1[(size_t)jp * G.nx + i], delta);
    int jm = nh_map_cell(j - 1, G.ny, G.bylo, G.byhi, sy);
    real vm = sy * nh_dsg(h[(size_t)jm * G.nx + i], qy1[(size_t)jm * G.nx + i], delta);
    divu = (up - um) / (RC(2.0) * G.dx) + (vp - vm) / (RC(2.0) * G.dy);
    real cc = sqrt(g * hk);
    real U1 = B1 * cc, U2 = B2 * cc;
    int fl = (fabs(divq) >= U1) || (flag_c[k] && fabs(divq) >= U2);  // R11
    flag_c[k] = (unsigned char)fl;
    if (fl) {
      real B = RC(1.0) - divq / U1;  // (9)
      nu = fmax(B, RC(0.0)) * hk * fabs(divq);
    }
  } else {
    flag_c[k] = 0;
  }
  real Hx = (F.even(H, i + 1, j) - F.even(H, i - 1, j)) / (RC(2.0) * G.dx);
  real Hy = (F.even(H, i, j + 1) - F.even(H, i, j - 1)) / (RC(2.0) * G.dy);
  qx2[k] = qx1[k] + dt * (RC(2.0) * nu * divu * Hx);  // R_u, L224
  qy2[k] = qy1[k] + dt * (RC(2.0) * nu * divu * Hy);
}

// S6 at nodes (R13): w** = w + dt R_w, compact edge averages of (39)
__global__ void __launch_bounds__(BX* BY)
k_break_nodes(NhGrid G, const NhScal* sc, real g, real delta, real eps, real B1, real B2,
              const real* __restrict__ h, const real* __restrict__ qx1,
              const real* __restrict__ qy1, const real* __restrict__ w_in,
              unsigned char* __restrict__ flag_n, real* __restrict__ w2) {
  int I = blockIdx.x * BX + threadIdx.x, J = blockIdx.y * BY + threadIdx.y;
  if (I >= G.nnx || J >= G.nny) return;
  Fld F{G};
  const real dt = (real)sc->dt;
  size_t k = (size_t)J * G.np + I;
  real hn = F.hnode(h, I, J);
  real nu = RC(0.0), divu = RC(0.0);
  if (hn > eps) {
    // the four cells around the node: index maps once, then discharge and velocity of each
    real sxm, sxp, sym, syp;
    int im = nh_map_cell(I - 1, G.nx, G.bxlo, G.bxhi, sxm), ip = nh_map_cell(I, G.nx, G.bxlo, G.bxhi, sxp);
    int jm = nh_map_cell(J - 1, G.ny, G.bylo, G.byhi, sym), jp = nh_map_cell(J, G.ny, G.bylo, G.byhi, syp);
    size_t kNE = (size_t)jp * G.nx + ip, kSE = (size_t)jm * G.nx + ip;
    size_t kNW = (size_t)jp * G.nx + im, kSW = (size_t)jm * G.nx + im;
    real qxNE = sxp * qx1[kNE], qxSE = sxp * qx1[kSE], qxNW = sxm * qx1[kNW], qxSW = sxm * qx1[kSW];
    real qyNE = syp * qy1[kNE], qyNW = syp * qy1[kNW], qySE = sym * qy1[kSE], qySW = sym * qy1[kSW];
    real uNE = sxp * nh_dsg(h[kNE], qx1[kNE], delta), uSE = sxp * nh_dsg(h[kSE], qx1[kSE], delta);
    real uNW = sxm * nh_dsg(h[kNW], qx1[kNW], delta), uSW = sxm * nh_dsg(h[kSW], qx1[kSW], delta);
    real vNE = syp * nh_dsg(h[kNE], qy1[kNE], delta), vNW = syp * nh_dsg(h[kNW], qy1[kNW], delta);
    real vSE = sym * nh_dsg(h[kSE], qy1[kSE], delta), vSW = sym * nh_dsg(h[kSW], qy1[kSW], delta);
    real q1E = RC(0.5) * (qxNE + qxSE), q1W = RC(0.5) * (qxNW + qxSW);
    real q2N = RC(0.5) * (qyNE + qyNW), q2S = RC(0.5) * (qySE + qySW);
    real u1E = RC(0.5) * (uNE + uSE), u1W = RC(0.5) * (uNW + uSW);
    real u2N = RC(0.5) * (vNE + vNW), u2S = RC(0.5) * (vSE + vSW);
    real divq = (q1E - q1W) / G.dx + (q2N - q2S) / G.dy;
    divu = (u1E - u1W) / G.dx + (u2N - u2S) / G.dy;
    real cc = sqrt(g * hn);
    real U1 = B1 * cc, U2 = B2 * cc;
    int fl = (fabs(divq) >= U1) || (flag_n[k] && fabs(divq) >= U2);
    flag_n[k] = (unsigned char)fl;
    if (fl) {
      real B = RC(1.0) - divq / U1;
      nu = fmax(B, RC(0.0)) * hn * fabs(divq);
    }
  } else {
    flag_n[k] = 0;
  }
  w2[k] = w_in[k] + dt * (RC(2.0) * nu * divu);  // R_w, L224
}

// S5b (w-advection variant of [7]; reading R30): (hw)_t + div(hw u) = p with
// h_t + div q = 0 is w_t + u . grad w = p / h.  Transport part, before S6: first-order upwind
// differences between neighbouring nodes, node velocity = mean of the desingularised velocities (S0)
// of the four cells around the node in the stage input (ghost cells through the maps of R9, so the
// normal velocity of a wall node is 0).  Same operation order as the oracle: bit-exact.
__global__ void __launch_bounds__(BX* BY)
k_w_advect(NhGrid G, const NhScal* sc, real delta, const real* __restrict__ h,
           const real* __restrict__ qx, const real* __restrict__ qy,
           const real* __restrict__ w_in, real* __restrict__ w_out) {
  int I = blockIdx.x * BX + threadIdx.x, J = blockIdx.y * BY + threadIdx.y;
  if (I >= G.nnx || J >= G.nny) return;
  Fld F{G};
  real sxm, sxp, sym, syp;
  int im = nh_map_cell(I - 1, G.nx, G.bxlo, G.bxhi, sxm), ip = nh_map_cell(I, G.nx, G.bxlo, G.bxhi, sxp);
  int jm = nh_map_cell(J - 1, G.ny, G.bylo, G.byhi, sym), jp = nh_map_cell(J, G.ny, G.bylo, G.byhi, syp);
  size_t kNE = (size_t)jp * G.nx + ip, kSE = (size_t)jm * G.nx + ip;
  size_t kNW = (size_t)jp * G.nx + im, kSW = (size_t)jm * G.nx + im;
  real uSW = sxm * nh_dsg(h[kSW], qx[kSW], delta), uSE = sxp * nh_dsg(h[kSE], qx[kSE], delta);
  real uNE = sxp * nh_dsg(h[kNE], qx[kNE], delta), uNW = sxm * nh_dsg(h[kNW], qx[kNW], delta);
  real vSW = sym * nh_dsg(h[kSW], qy[kSW], delta), vSE = sym * nh_dsg(h[kSE], qy[kSE], delta);
  real vNE = syp * nh_dsg(h[kNE], qy[kNE], delta), vNW = syp * nh_dsg(h[kNW], qy[kNW], delta);
  real un = RC(0.25) * (uSW + uSE + uNE + uNW);
  real vn = RC(0.25) * (vSW + vSE + vNE + vNW);
  real wc = w_in[(size_t)J * G.np + I];
  real wx = (un > RC(0.0)) ? (wc - F.node(w_in, I - 1, J)) / G.dx : (F.node(w_in, I + 1, J) - wc) / G.dx;
  real wy = (vn > RC(0.0)) ? (wc - F.node(w_in, I, J - 1)) / G.dy : (F.node(w_in, I, J + 1) - wc) / G.dy;
  w_out[(size_t)J * G.np + I] = wc - (real)sc->dt * (un * wx + vn * wy);
}

// R32: start vector of a pressure solve from the last seven solutions (s1 the most recent):
// x0 = ((s1 + 3 (s2 - s3)) - 3 (s4 - s5)) + (s6 - s7), in this operation order (bit-exact against
// the oracle, so that solver 1 stays bit-exact end to end)
__global__ void __launch_bounds__(BX* BY)
k_start_vector(NhGrid G, const real* __restrict__ s1, const real* __restrict__ s2,
               const real* __restrict__ s3, const real* __restrict__ s4, const real* __restrict__ s5,
               const real* __restrict__ s6, const real* __restrict__ s7, real* __restrict__ x0) {
  int I = blockIdx.x * BX + threadIdx.x, J = blockIdx.y * BY + threadIdx.y;
  if (I >= G.nnx || J >= G.nny) return;
  size_t k = (size_t)J * G.np + I;
  x0[k] = ((s1[k] + RC(3.0) * (s2[k] - s3[k])) - RC(3.0) * (s4[k] - s5[k])) + (s6[k] - s7[k]);
}

// S10: correction, eqs (36),(41): q <- q** + dt T_NH(p) at cells
__global__ void __launch_bounds__(BX* BY)
k_correct_cells(NhGrid G, const NhScal* sc, const real* __restrict__ h,
                const real* __restrict__ z, const real* __restrict__ qx2,
                const real* __restrict__ qy2, const real* __restrict__ pt,
                real* __restrict__ qx_out, real* __restrict__ qy_out) {
  int i = blockIdx.x * BX + threadIdx.x, j = blockIdx.y * BY + threadIdx.y;
  if (i >= G.nx || j >= G.ny) return;
  // cells i-1..i+1, j-1..j+1 and nodes i..i+1, j..j+1 inside the grid (periodic: node n wraps)
  Fld F{G, i >= 1 && i <= G.nx - 2 && j >= 1 && j <= G.ny - 2};
  const real dt = (real)sc->dt;
  size_t k = (size_t)j * G.nx + i;
  // corner nodes of cell (i,j): (i,j) (i+1,j) (i,j+1) (i+1,j+1)
  real p00 = F.node(pt, i, j), p10 = F.node(pt, i + 1, j);
  real p01 = F.node(pt, i, j + 1), p11 = F.node(pt, i + 1, j + 1);
  real pE = RC(0.5) * (p11 + p10), pW = RC(0.5) * (p01 + p00);
  real pN = RC(0.5) * (p11 + p01), pS = RC(0.5) * (p10 + p00);
  real xx = F.xi_x(z, i, j), xy = F.xi_y(z, i, j);
  real hk = h[k];
  qx_out[k] = qx2[k] - dt / (RC(4.0) * G.dx) * ((RC(2.0) * hk + xx) * pE + (xx - RC(2.0) * hk) * pW);
  qy_out[k] = qy2[k] - dt / (RC(4.0) * G.dy) * ((RC(2.0) * hk + xy) * pN + (xy - RC(2.0) * hk) * pS);
}

// S10 at nodes: w <- w** + dt p dinv(h_n)  (R16)
__global__ void __launch_bounds__(BX* BY)
k_correct_nodes(NhGrid G, const NhScal* sc, real delta, const real* __restrict__ h,
                const real* __restrict__ w2, const real* __restrict__ pt,
                real* __restrict__ w_out) {
  int I = blockIdx.x * BX + threadIdx.x, J = blockIdx.y * BY + threadIdx.y;
  if (I >= G.nnx || J >= G.nny) return;
  Fld F{G, node_interior(G, I, J)};
  size_t k = (size_t)J * G.np + I;
  real hn = F.hnode(h, I, J);
  w_out[k] = w2[k] + (real)sc->dt * pt[k] * nh_dinv_h(hn, delta);
}

// S11: generating relaxation zone at x-lo (L417-431, reading R18), target at the stage's end time
__device__ __forceinline__ real relax_m_cell(real L, real dx, int i) {
  real x = ((real)i + RC(0.5)) * dx;
  real d = L - x;
  if (d <= RC(0.0)) return RC(1.0);
  if (d >= L) return RC(0.0);
  return sqrt(RC(1.0) - (d / L) * (d / L));
}
__global__ void __launch_bounds__(256)
k_relax(NhGrid G, const NhScal* sc, int stage, real g, real A, real h0, real x0, real L,
        int krel, const real* __restrict__ H, real* __restrict__ h, real* __restrict__ qx,
        real* __restrict__ qy, real* __restrict__ w, real* __restrict__ p, real* __restrict__ etap) {
  const real kk = sqrt(RC(3.0) * A / (RC(4.0) * h0 * h0 * h0));
  const real cel = sqrt(g * (h0 + A));
  // stage 0 ends at t + dt, stage 1 at (t + dt) + dt (the second stage starts from t + dt)
  double tt = sc->t + sc->dt;  // the clock stays fp64 in both builds
  if (stage == 1) tt = tt + sc->dt;
  int ncol = krel + 1;
  size_t tot = (size_t)ncol * (G.ny + 1);
  for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < tot;
       e += (size_t)gridDim.x * blockDim.x) {
    int i = (int)(e % ncol), j = (int)(e / ncol);
    if (i < krel && j < G.ny) {
      size_t k = (size_t)j * G.nx + i;
      real m = relax_m_cell(L, G.dx, i);
      real x = ((real)i + RC(0.5)) * G.dx;
      real etas = A * nh_sech2_fixed(kk * (x - x0 - cel * tt));  // R31
      real hs = fmax(H[k] + etas, RC(0.0));
      if (kEta) {  // relax the stored quantity: the law is linear, eta* = h* - H
        real ev = m * etap[k] + (RC(1.0) - m) * (hs - H[k]);
        etap[k] = ev;
        h[k] = fmax(H[k] + ev, RC(0.0));
      } else {
        h[k] = m * h[k] + (RC(1.0) - m) * hs;
      }
      qx[k] = m * qx[k] + (RC(1.0) - m) * (cel * etas);
      qy[k] = m * qy[k];
    }
    if (i <= krel && i < G.nnx && j < G.nny) {
      size_t k = (size_t)j * G.np + i;
      real mL = (i - 1 >= 0) ? relax_m_cell(L, G.dx, i - 1) : RC(0.0);
      real mR = (i < G.nx) ? relax_m_cell(L, G.dx, i) : RC(1.0);
      real m = RC(0.5) * (mL + mR);  // m_{i+-1/2}, L429
      w[k] = m * w[k];
      p[k] = m * p[k];
    }
  }
}

// S11b: absorbing relaxation zone on one side (L415-440; R18, R29): the relaxation of S11 towards
// eta* = 0, q* = w* = p* = 0, a <- a + (1 - m)(a* - a), m = sqrt(1 - (d/L)^2), d from the inner end
// of the zone; node coefficients are the mean of the two adjacent cell coefficients (0 beyond the
// boundary).  side: 0 x-lo, 1 x-hi, 2 y-lo, 3 y-hi; s = distance from the boundary in cells / lines.
__device__ __forceinline__ real absorb_m(real L, real dxy, int s) {
  real x = ((real)s + RC(0.5)) * dxy;
  real d = L - x;
  if (d <= RC(0.0)) return RC(1.0);
  if (d >= L) return RC(0.0);
  return sqrt(RC(1.0) - (d / L) * (d / L));
}
__global__ void __launch_bounds__(256)
k_absorb(NhGrid G, int side, real L, int krel, const real* __restrict__ H,
         real* __restrict__ h, real* __restrict__ qx, real* __restrict__ qy,
         real* __restrict__ w, real* __restrict__ p, real* __restrict__ etap) {
  const bool xdir = side < 2, hi = side & 1;
  const int n = xdir ? G.nx : G.ny;
  const real dxy = xdir ? G.dx : G.dy;
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
      real f = RC(1.0) - absorb_m(L, dxy, s);
      real hs = fmax(H[k], RC(0.0));
      if (kEta) {
        real ev = etap[k] + f * ((hs - H[k]) - etap[k]);
        etap[k] = ev;
        h[k] = fmax(H[k] + ev, RC(0.0));
      } else {
        h[k] = h[k] + f * (hs - h[k]);
      }
      qx[k] = qx[k] + f * (RC(0.0) - qx[k]);
      qy[k] = qy[k] + f * (RC(0.0) - qy[k]);
    }
    if (t < nnother) {
      int a = hi ? n - s : s;
      real mo = (s - 1 >= 0) ? absorb_m(L, dxy, s - 1) : RC(0.0);
      real mi = (s < n) ? absorb_m(L, dxy, s) : RC(1.0);
      real f = RC(1.0) - RC(0.5) * (mo + mi);
      size_t k = xdir ? (size_t)t * G.np + a : (size_t)a * G.np + t;
      w[k] = w[k] + f * (RC(0.0) - w[k]);
      p[k] = p[k] + f * (RC(0.0) - p[k]);
    }
  }
}

// internal plane -> dense public node layout: fill the duplicate lines of periodic directions
__global__ void __launch_bounds__(BX* BY)
k_nodes_out(NhGrid G, const real* __restrict__ src, double* __restrict__ dst) {
  int I = blockIdx.x * BX + threadIdx.x, J = blockIdx.y * BY + threadIdx.y;
  if (I > G.nx || J > G.ny) return;
  int II = (I == G.nx && G.nnx == G.nx) ? 0 : I;
  int JJ = (J == G.ny && G.nny == G.ny) ? 0 : J;
  dst[(size_t)J * (G.nx + 1) + I] = (double)src[(size_t)JJ * G.np + II];
}

dim3 grid2(int nx, int ny) { return dim3((nx + BX - 1) / BX, (ny + BY - 1) / BY); }
int grid_1d(const Ctx* c, size_t n, int block) {
  size_t need = (n + block - 1) / block;
  size_t cap = (size_t)c->sm_count * 16;
  return (int)(need < cap ? (need ? need : 1) : cap);
}

}  // namespace

void nh_launch_compute_z(Ctx* c, const real* h, real* z) {
  k_compute_z<<<grid_1d(c, c->nc, 256), 256, 0, c->stream>>>(c->nc, h, c->H, z, nh_eta_of(c, h));
  c->launches++;
}
void nh_launch_cell_planes(Ctx* c, const real* h) {
  k_cell_planes<<<grid2(c->g.nx + 4, c->g.ny + 4), dim3(BX, BY), 0, c->stream>>>(c->g, h, c->H, c->z,
                                                                                c->hc, c->zc, nh_eta_of(c, h));
  c->launches++;
}
void nh_launch_breaking(Ctx* c, const real* h, const real* qx1, const real* qy1,
                        const real* w_in, real* qx2, real* qy2, real* w2) {
  const nh_params& P = c->prm;
  k_break_cells<<<grid2(c->g.nx, c->g.ny), dim3(BX, BY), 0, c->stream>>>(
      c->g, c->sc, P.g, P.delta, P.eps_dry, P.B1, P.B2, c->H, h, qx1, qy1, c->flag_c, qx2, qy2);
  k_break_nodes<<<grid2(c->g.nnx, c->g.nny), dim3(BX, BY), 0, c->stream>>>(
      c->g, c->sc, P.g, P.delta, P.eps_dry, P.B1, P.B2, h, qx1, qy1, w_in, c->flag_n, w2);
  c->launches += 2;
}
void nh_launch_rhs(Ctx* c, const real* h, const real* qx, const real* qy, const real* z,
                   const real* w, real* b, int constraint_only) {
  k_rhs<<<grid2(c->g.nnx, c->g.nny), dim3(BX, BY), 0, c->stream>>>(c->g, c->sc, constraint_only, h,
                                                                  qx, qy, z, w, b);
  c->launches++;
}
void nh_launch_coeffs(Ctx* c, const real* h, const real* z) {
  k_coeffs<<<grid2(c->g.nnx, c->g.nny), dim3(BX, BY), 0, c->stream>>>(c->g, h, z, c->dg, c->dinv,
                                                                     c->cE, c->cW, c->cN, c->cS);
  c->launches++;
}
void nh_launch_scale_rows(Ctx* c, const real* b, real* bp) {
  k_scale_rows<<<grid2(c->g.nnx, c->g.nny), dim3(BX, BY), 0, c->stream>>>(
      c->g, c->dinv, c->cE, c->cW, c->cN, c->cS, b, bp, c->sc);
  c->launches++;
}
void nh_launch_assemble_rows(Ctx* c, const real* h, const real* qx, const real* qy,
                             const real* z, const real* w, real* bp) {
  k_assemble_rows<<<grid2(c->g.nnx, c->g.nny), dim3(BX, BY), 0, c->stream>>>(
      c->g, c->sc, h, qx, qy, z, w, c->cE, c->cW, c->cN, c->cS, bp);
  c->launches++;
}
void nh_launch_apply_A(Ctx* c, const real* h, const real* z, const real* x, real* y) {
  k_apply_A<<<grid2(c->g.nnx, c->g.nny), dim3(BX, BY), 0, c->stream>>>(c->g, h, z, x, y);
  c->launches++;
}
void nh_launch_correct(Ctx* c, const real* h, const real* z, const real* qx2,
                       const real* qy2, const real* w2, const real* p, real* qx_out,
                       real* qy_out, real* w_out) {
  k_correct_cells<<<grid2(c->g.nx, c->g.ny), dim3(BX, BY), 0, c->stream>>>(c->g, c->sc, h, z, qx2,
                                                                          qy2, p, qx_out, qy_out);
  k_correct_nodes<<<grid2(c->g.nnx, c->g.nny), dim3(BX, BY), 0, c->stream>>>(
      c->g, c->sc, c->prm.delta, h, w2, p, w_out);
  c->launches += 2;
}
void nh_launch_w_advect(Ctx* c, const real* h, const real* qx, const real* qy,
                        const real* w_in, real* w_out) {
  k_w_advect<<<grid2(c->g.nnx, c->g.nny), dim3(BX, BY), 0, c->stream>>>(c->g, c->sc, c->prm.delta, h,
                                                                       qx, qy, w_in, w_out);
  c->launches++;
}
void nh_launch_start_vector(Ctx* c, real* x0) {
  real* const* h = c->hist;
  k_start_vector<<<grid2(c->g.nnx, c->g.nny), dim3(BX, BY), 0, c->stream>>>(c->g, h[0], h[1], h[2], h[3],
                                                                           h[4], h[5], h[6], x0);
  c->launches++;
}
void nh_launch_relax(Ctx* c, real* h, real* qx, real* qy, real* w, real* p, int stage) {
  const nh_params& P = c->prm;
  int krel = (int)ceil(P.gen_Lrel / c->g.dx);
  if (krel > c->g.nx) krel = c->g.nx;
  size_t tot = (size_t)(krel + 1) * (c->g.ny + 1);
  k_relax<<<grid_1d(c, tot, 256), 256, 0, c->stream>>>(c->g, c->sc, stage, P.g, P.gen_A, P.gen_h0,
                                                       P.gen_x0, P.gen_Lrel, krel, c->H, h, qx, qy,
                                                       w, p, nh_eta_of(c, h));
  c->launches++;
}
void nh_launch_absorb(Ctx* c, real* h, real* qx, real* qy, real* w, real* p) {
  const double L[4] = {c->prm.abs_xlo, c->prm.abs_xhi, c->prm.abs_ylo, c->prm.abs_yhi};
  for (int side = 0; side < 4; ++side) {
    if (!(L[side] > RC(0.0))) continue;
    const bool xdir = side < 2;
    const int n = xdir ? c->g.nx : c->g.ny, nother = xdir ? c->g.ny : c->g.nx;
    int krel = (int)ceil(L[side] / (xdir ? c->g.dx : c->g.dy));
    if (krel > n) krel = n;
    size_t tot = (size_t)(krel + 1) * (nother + 1);
    k_absorb<<<grid_1d(c, tot, 256), 256, 0, c->stream>>>(c->g, side, L[side], krel, c->H, h, qx, qy,
                                                          w, p, nh_eta_of(c, h));
    c->launches++;
  }
}
void nh_launch_nodes_out(Ctx* c, const real* src, double* dst) {
  k_nodes_out<<<grid2(c->g.nx + 1, c->g.ny + 1), dim3(BX, BY), 0, c->stream>>>(c->g, src, dst);
  c->launches++;
}

}  // namespace NH_NS
