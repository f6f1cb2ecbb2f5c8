// nh_predictor.cu -- first part of the time step: CFL time step (a0), MUSCL reconstruction (a1),
// PVM/HLL path-conservative face fluctuations (a2), fused cell update (a3), RK combine (a8).
//
// One fused kernel does a1-a3: a (TX+4) x (TY+4) halo tile of the primitive fields (h, eta, u, v,
// z_b) is staged in shared memory through the boundary index maps, then every thread owns one
// cell, reconstructs, solves the two faces on its high sides (handing D^+ to its neighbours
// through shared memory) and writes U*.  No edge colouring, no accumulator
// array (the paper's K1/K2 split, was made for write conflicts that a
// cell-centric gather does not have).  Traffic: 4 planes read, 3 written = 56 B per cell.
#include <math.h>
#include <stdio.h>

#include "nh_internal.cuh"

namespace {

constexpr int PTX = 32, PTY = 8, PH = 2;  // predictor tile and halo
constexpr int PSX = PTX + 2 * PH, PSY = PTY + 2 * PH;

struct PredTile {
  double h[PSY][PSX], eta[PSY][PSX], u[PSY][PSX], v[PSY][PSX], zb[PSY][PSX];
};

struct Prim {
  double h, eta, un, ut, zb;
};

__device__ __forceinline__ Prim get_prim(const PredTile& T, int lx, int ly, int dir) {
  Prim P;
  P.h = T.h[ly][lx];
  P.eta = T.eta[ly][lx];
  P.zb = T.zb[ly][lx];
  double uu = T.u[ly][lx], vv = T.v[ly][lx];
  if (dir == 0) { P.un = uu; P.ut = vv; } else { P.un = vv; P.ut = uu; }
  return P;
}

// S2: undivided limited slopes (eta, h, un, ut) of the cell at tile position (lx,ly) (L335-337, R2)
__device__ __forceinline__ void cell_slopes(const PredTile& T, int lx, int ly, int dir, int order,
                                            double eps_dry, double s[4]) {
  s[0] = s[1] = s[2] = s[3] = 0.0;
  if (order == 1) return;
  int di = (dir == 0), dj = (dir == 1);
  Prim Pc = get_prim(T, lx, ly, dir);
  if (Pc.h <= eps_dry) return;  // R2 (i): dry cell
  Prim Pm = get_prim(T, lx - di, ly - dj, dir);
  Prim Pp = get_prim(T, lx + di, ly + dj, dir);
  s[0] = nh_minmod(Pc.eta - Pm.eta, Pp.eta - Pc.eta);
  s[1] = nh_minmod(Pc.h - Pm.h, Pp.h - Pc.h);
  s[2] = nh_minmod(Pc.un - Pm.un, Pp.un - Pc.un);
  s[3] = nh_minmod(Pc.ut - Pm.ut, Pp.ut - Pc.ut);
  // R2 (ii): emerging bottom against either neighbour -> gradient of eta set to zero (L337)
  if (fmin(Pc.eta, Pm.eta) < fmax(Pc.zb, Pm.zb) || fmin(Pc.eta, Pp.eta) < fmax(Pc.zb, Pp.zb))
    s[0] = 0.0;
  // R2 (iii): positivity of the reconstructed depth (L335-337)
  if (Pc.h - 0.5 * fabs(s[1]) < 0.0) s[1] = copysign(2.0 * Pc.h, s[1]);
}

// S4: PVM/HLL path-conservative fluctuations at one face, eqs (18)(19) with A* (L303-322), three
// components (R3), guards (R4), emerging-bottom clip (R5).  m = U^-, p = U^+.
__device__ __forceinline__ void face_fluct(double g, double hm, double etam, double um, double vm,
                                           double hp, double etap, double up, double vp,
                                           double Dm[3], double Dp[3]) {
  double hh = 0.5 * (hm + hp);  // h_{i+1/2}, L276
  double sm = sqrt(hm), sp = sqrt(hp);
  double den = sm + sp;
  double unum = um * sm + up * sp;
  double uh = (den > 0.0) ? ((unum == 0.0) ? unum : unum / den) : 0.0;  // Roe average, L276; R4
                                                    // (zero dividend: same bits, no slow path)
  double ch = sqrt(g * hh), cm = sqrt(g * hm), cp = sqrt(g * hp);
  double SL = fmin(uh - ch, um - cm);  // L290
  double SR = fmax(uh + ch, up + cp);  // L292
  if (SR - SL <= 1e-14 * (1.0 + ch)) {  // R4: dry-dry face
#pragma unroll
    for (int k = 0; k < 3; ++k) { Dm[k] = 0.0; Dp[k] = 0.0; }
    return;
  }
  double a0 = (SR * fabs(SL) - SL * fabs(SR)) / (SR - SL);  // L286
  double a1 = (fabs(SR) - fabs(SL)) / (SR - SL);
  // R5: emerging bottom; z^+- = eta^+- - h^+- are the face bed levels
  double zm = etam - hm, zp = etap - hp;
  double zs = fmax(zm, zp);
  double deta;
  if (fmin(etam, etap) >= zs) deta = etap - etam;
  else deta = fmax(0.0, etap - zs) - fmax(0.0, etam - zs);
  double qnm = hm * um, qnp = hp * up;
  double qtm = hm * vm, qtp = hp * vp;
  double R[3], DU[3];
  R[0] = qnp - qnm;  // F_c(U+) - F_c(U-) + T_p, (19)
  R[1] = (qnp * up - qnm * um) + g * hh * deta;
  R[2] = qnp * vp - qnm * vm;
  DU[0] = deta;  // U+ - U- - (H+ - H-) e1, (18)
  DU[1] = qnp - qnm;
  DU[2] = qtp - qtm;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    Dm[k] = 0.5 * ((1.0 - a1) * R[k] - a0 * DU[k]);
    Dp[k] = 0.5 * ((1.0 + a1) * R[k] + a0 * DU[k]);
  }
}

// One face solve: the face between tile cell (lx,ly) and its neighbour in direction dir.
// sL = slopes of the left / lower cell (returned: its owner needs them for the in-cell term).
__device__ __forceinline__ void hi_face(const PredTile& T, int lx, int ly, int dir, int order,
                                        double eps_dry, double g, double sL[4], double Dm[3],
                                        double Dp[3]) {
  const int di = (dir == 0), dj = (dir == 1);
  Prim Pc = get_prim(T, lx, ly, dir);
  Prim Pp = get_prim(T, lx + di, ly + dj, dir);
  double sR[4];
  cell_slopes(T, lx, ly, dir, order, eps_dry, sL);
  cell_slopes(T, lx + di, ly + dj, dir, order, eps_dry, sR);
  // S3 face states: left = c + s/2, right = p - s/2
  double hL = Pc.h + 0.5 * sL[1], eL = Pc.eta + 0.5 * sL[0];
  double uL = Pc.un + 0.5 * sL[2], vL = Pc.ut + 0.5 * sL[3];
  double hR = Pp.h - 0.5 * sR[1], eR = Pp.eta - 0.5 * sR[0];
  double uR = Pp.un - 0.5 * sR[2], vR = Pp.ut - 0.5 * sR[3];
  face_fluct(g, hL, eL, uL, vL, hR, eR, uR, vR, Dm, Dp);
}

// Every face is solved once, by the thread of the cell on its low side, which keeps D^- for its
// own update and publishes D^+ for its neighbour through shared memory; the faces on the low
// edges of the tile (32 in y, 8 in x) are solved by the first 40 threads.  (The first version had
// every cell solve its four faces and limit five cells: 2400 instructions per cell.)
#ifndef NH_PRED_MINB
#define NH_PRED_MINB 4  // 64 registers: 10.3 ms per two launches at 8192^2 (2: 15.7, 3: 11.9, 5: 10.2, 6: 12.4)
#endif
__global__ void __launch_bounds__(PTX* PTY, NH_PRED_MINB)
k_predictor(NhGrid G, double g, double delta, double eps_dry, double manning_n, int order,
            NhScal* sc, const double* __restrict__ H, const double* __restrict__ h,
            const double* __restrict__ qx, const double* __restrict__ qy,
            double* __restrict__ h1, double* __restrict__ qx1, double* __restrict__ qy1) {
  __shared__ PredTile T;
  __shared__ double DPx[3][PTY][PTX + 1];  // D^+ of the x-face on the low side of cell lx - PH
  __shared__ double DPy[3][PTY + 1][PTX];  // D^+ of the y-face on the low side of cell ly - PH
  const int i0 = blockIdx.x * PTX, j0 = blockIdx.y * PTY;
  const int tid = threadIdx.y * PTX + threadIdx.x;
  // S0 + S1: derived fields of the halo tile through the index maps
  for (int e = tid; e < PSX * PSY; e += PTX * PTY) {
    int lx = e % PSX, ly = e / PSX;
    int gi = i0 - PH + lx, gj = j0 - PH + ly;
    double hv = 0.0, ev = 0.0, uv = 0.0, vv = 0.0, zv = 0.0;
    if (gi <= G.nx + 1 && gj <= G.ny + 1) {
      double sx, sy;
      int ii = nh_map_cell(gi, G.nx, G.bxlo, G.bxhi, sx);
      int jj = nh_map_cell(gj, G.ny, G.bylo, G.byhi, sy);
      size_t k = (size_t)jj * G.nx + ii;
      double Hv = H[k];
      hv = h[k];
      ev = hv - Hv;
      uv = sx * nh_dsg(hv, qx[k], delta);
      vv = sy * nh_dsg(hv, qy[k], delta);
      zv = -Hv;
    }
    T.h[ly][lx] = hv; T.eta[ly][lx] = ev; T.u[ly][lx] = uv; T.v[ly][lx] = vv; T.zb[ly][lx] = zv;
  }
  __syncthreads();
  const int i = i0 + threadIdx.x, j = j0 + threadIdx.y;
  const bool active = (i < G.nx && j < G.ny);
  const int lx = threadIdx.x + PH, ly = threadIdx.y + PH;
  double sown[2][4], Dm_hi[2][3];
  if (active) {
#pragma unroll
    for (int dir = 0; dir < 2; ++dir) {
      double Dp[3];
      hi_face(T, lx, ly, dir, order, eps_dry, g, sown[dir], Dm_hi[dir], Dp);
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        if (dir == 0) DPx[k][threadIdx.y][threadIdx.x + 1] = Dp[k];
        else DPy[k][threadIdx.y + 1][threadIdx.x] = Dp[k];
      }
    }
  }
  // faces on the low edges of the tile: y-faces below row 0 (threads 0..31), x-faces left of
  // column 0 (threads 32..39)
  if (tid < PTX + PTY) {
    const int dir = (tid < PTX) ? 1 : 0;
    const int cx = (dir == 1) ? tid : -1, cy = (dir == 1) ? -1 : tid - PTX;  // tile cell on the low side
    if (i0 + max(cx, 0) < G.nx && j0 + max(cy, 0) < G.ny) {
      double sl[4], Dm[3], Dp[3];
      hi_face(T, cx + PH, cy + PH, dir, order, eps_dry, g, sl, Dm, Dp);
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        if (dir == 0) DPx[k][cy][0] = Dp[k];
        else DPy[k][0][cx] = Dp[k];
      }
    }
  }
  __syncthreads();
  if (!active) return;
  const double dt = sc->dt;
  double dU[2][3];  // per direction: (h, normal q, tangential q)
#pragma unroll
  for (int dir = 0; dir < 2; ++dir) {
    Prim Pc = get_prim(T, lx, ly, dir);
    const double* s_ = sown[dir];
    // own face states: "hi" face left state = c + s/2, "lo" face right state = c - s/2
    double hL = Pc.h + 0.5 * s_[1], uL = Pc.un + 0.5 * s_[2], vL = Pc.ut + 0.5 * s_[3];
    double hr = Pc.h - 0.5 * s_[1], ur = Pc.un - 0.5 * s_[2], vr = Pc.ut - 0.5 * s_[3];
    // in-cell term I_i of (22) = F_c(U^-_{i+1/2}) - F_c(U^+_{i-1/2}) + g h_i sigma_eta e2 (S5)
    double qnL = hL * uL, qnr = hr * ur;
    double Fhi[3] = {qnL, qnL * uL, qnL * vL};
    double Flo[3] = {qnr, qnr * ur, qnr * vr};
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      double Dp_lo = (dir == 0) ? DPx[k][threadIdx.y][threadIdx.x] : DPy[k][threadIdx.y][threadIdx.x];
      dU[dir][k] = Dm_hi[dir][k] + Dp_lo + (Fhi[k] - Flo[k]);
    }
    dU[dir][1] += g * Pc.h * s_[0];
  }
  size_t k = (size_t)j * G.nx + i;
  double lxr = dt / G.dx, lyr = dt / G.dy;
  double hn = h[k] - lxr * dU[0][0] - lyr * dU[1][0];
  double qxn = qx[k] - lxr * dU[0][1] - lyr * dU[1][2];
  double qyn = qy[k] - lxr * dU[0][2] - lyr * dU[1][1];
  if (hn < 0.0) {  // R7; size statistics for R24 (rare: integer atomics, exact and order independent)
    double a = -hn;
    int bk = (a < 1e-15) ? 0 : (a < 1e-12) ? 1 : (a < 1e-9) ? 2 : (a < 1e-6) ? 3 : (a < 1e-3) ? 4 : 5;
    atomicAdd(&sc->clamp_hist[bk], 1ULL);
    atomicMax(&sc->clamp_max_bits, (unsigned long long)__double_as_longlong(a));
    atomicAdd((unsigned long long*)&sc->clamps, 1ULL);
    hn = 0.0;
  }
  if (hn <= eps_dry) { qxn = 0.0; qyn = 0.0; }          // R7
  else if (manning_n > 0.0) {
    // Manning friction tau = g h u n^2 |u| / h^(4/3) (L61-65, L773-775), semi-implicit (L249, R27):
    // q <- q / (1 + dt g n^2 |u*| / h*^(4/3)), desingularised velocities of U*, wet cells only
    double uu = nh_dsg(hn, qxn, delta), vv = nh_dsg(hn, qyn, delta);
    double speed = sqrt(uu * uu + vv * vv);
    double h43 = hn * nh_cbrt_fixed(hn);  // R31
    double den = 1.0 + dt * g * manning_n * manning_n * speed / h43;
    qxn = qxn / den; qyn = qyn / den;
  }
  h1[k] = hn; qx1[k] = qxn; qy1[k] = qyn;
}

// a0 / R20: lam = max_ij[(|u|+sqrt(gh))/dx + (|v|+sqrt(gh))/dy].  A max is exact and order
// independent; non-negative doubles order like their bit patterns, so one integer atomicMax per
// CTA finishes the device-wide reduction deterministically.
__device__ __forceinline__ double cfl_rate(double g, double delta, double dx, double dy, double h,
                                           double qx, double qy) {
  double cc = sqrt(g * h);
  double uu = nh_dsg(h, qx, delta), vv = nh_dsg(h, qy, delta);
  return (fabs(uu) + cc) / dx + (fabs(vv) + cc) / dy;
}
__device__ __forceinline__ void block_max_to_global(double l, unsigned long long* lam_bits) {
  for (int o = 16; o > 0; o >>= 1) l = fmax(l, __shfl_xor_sync(0xffffffffu, l, o));
  __shared__ double wm[32];
  int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) wm[wid] = l;
  __syncthreads();
  if (wid == 0) {
    int nw = (blockDim.x + 31) >> 5;
    l = (lane < nw) ? wm[lane] : 0.0;
    for (int o = 16; o > 0; o >>= 1) l = fmax(l, __shfl_xor_sync(0xffffffffu, l, o));
    if (lane == 0 && l > 0.0) atomicMax(lam_bits, (unsigned long long)__double_as_longlong(l));
  }
}

__global__ void __launch_bounds__(256)
k_lambda(size_t nc, double g, double delta, double dx, double dy, const double* __restrict__ h,
         const double* __restrict__ qx, const double* __restrict__ qy, NhScal* sc) {
  double l = 0.0;
  for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < nc;
       k += (size_t)gridDim.x * blockDim.x) {
    double v = cfl_rate(g, delta, dx, dy, h[k], qx[k], qy[k]);
    if (v > l) l = v;
  }
  block_max_to_global(l, &sc->lam_bits);
}

__global__ void k_set_dt(NhScal* sc, double cfl, double dt_fixed) {
  if (dt_fixed > 0.0) {
    sc->dt = dt_fixed;
  } else {
    double lam = __longlong_as_double((long long)sc->lam_bits);
    double dt = (lam > 0.0) ? cfl / lam : 0.0;
    if (!(dt == dt) || isinf(dt)) atomicOr(&sc->flags, NH_FLAG_NAN);
    sc->dt = dt;
  }
  sc->lam_bits = 0ULL;
}

__global__ void k_end_step(NhScal* sc, int advance_time) {
  if (advance_time) { sc->t += sc->dt; sc->steps += 1; }
  sc->dt_last = sc->dt;
}

// a8: U^{n+1} = U^n/2 + U^(2)/2 on h, qx, qy (cells) and w (nodes) (L406, L516, L544; R19), fused
// with the CFL rate of the new state (a0 of the next step: 0 extra bytes).
__global__ void __launch_bounds__(256)
k_combine(NhGrid G, double g, double delta, double* __restrict__ h0, double* __restrict__ qx0,
          double* __restrict__ qy0, double* __restrict__ w0, const double* __restrict__ h2,
          const double* __restrict__ qx2, const double* __restrict__ qy2,
          const double* __restrict__ w2, NhScal* sc) {
  size_t nc = (size_t)G.nx * G.ny, nn = (size_t)G.np * (G.ny + 1);
  double l = 0.0;
  size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < nc; k += stride) {
    double hv = 0.5 * h0[k] + 0.5 * h2[k];
    double qxv = 0.5 * qx0[k] + 0.5 * qx2[k];
    double qyv = 0.5 * qy0[k] + 0.5 * qy2[k];
    h0[k] = hv; qx0[k] = qxv; qy0[k] = qyv;
    double v = cfl_rate(g, delta, G.dx, G.dy, hv, qxv, qyv);
    if (v > l) l = v;
  }
  if (w2 != nullptr)  // nullptr: w did not move in this step (hydrostatic path without zones)
    for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < nn; k += stride)
      w0[k] = 0.5 * w0[k] + 0.5 * w2[k];
  block_max_to_global(l, &sc->lam_bits);
}

// set_state validation: h >= 0 and finite, q finite
__global__ void __launch_bounds__(256)
k_validate(size_t nc, const double* __restrict__ h, const double* __restrict__ qx,
           const double* __restrict__ qy, NhScal* sc) {
  bool bad = false;
  for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < nc;
       k += (size_t)gridDim.x * blockDim.x) {
    double a = h[k], b = qx[k], c = qy[k];
    if (!(a >= 0.0) || isinf(a) || !(b == b) || !(c == c)) bad = true;
  }
  if (__syncthreads_or(bad) && threadIdx.x == 0) atomicOr(&sc->flags, NH_FLAG_BADSTATE);
}

int grid_1d(const nh_ctx* c, size_t n, int block) {
  size_t need = (n + block - 1) / block;
  size_t cap = (size_t)c->sm_count * 16;
  return (int)(need < cap ? (need ? need : 1) : cap);
}

}  // namespace

void nh_launch_lambda(nh_ctx* c, const double* h, const double* qx, const double* qy) {
  k_lambda<<<grid_1d(c, c->nc, 256), 256, 0, c->stream>>>(c->nc, c->prm.g, c->prm.delta, c->g.dx,
                                                          c->g.dy, h, qx, qy, c->sc);
  c->launches++;
}
void nh_launch_set_dt(nh_ctx* c, double dt_fixed) {
  k_set_dt<<<1, 1, 0, c->stream>>>(c->sc, c->prm.cfl, dt_fixed);
  c->launches++;
}
void nh_launch_end_step(nh_ctx* c, int advance_time) {
  k_end_step<<<1, 1, 0, c->stream>>>(c->sc, advance_time);
  c->launches++;
}
void nh_launch_predictor(nh_ctx* c, const double* h, const double* qx, const double* qy, double* h1,
                         double* qx1, double* qy1) {
  dim3 grid((c->g.nx + PTX - 1) / PTX, (c->g.ny + PTY - 1) / PTY), block(PTX, PTY);
  k_predictor<<<grid, block, 0, c->stream>>>(c->g, c->prm.g, c->prm.delta, c->prm.eps_dry,
                                             c->prm.manning_n, c->prm.space_order, c->sc, c->H, h, qx, qy, h1, qx1,
                                             qy1);
  c->launches++;
}
void nh_launch_combine(nh_ctx* c, double* h0, double* qx0, double* qy0, double* w0, const double* h2,
                       const double* qx2, const double* qy2, const double* w2) {
  k_combine<<<grid_1d(c, c->nn, 256), 256, 0, c->stream>>>(c->g, c->prm.g, c->prm.delta, h0, qx0,
                                                           qy0, w0, h2, qx2, qy2, w2, c->sc);
  c->launches++;
}
void nh_launch_validate(nh_ctx* c, const double* h, const double* qx, const double* qy) {
  k_validate<<<grid_1d(c, c->nc, 256), 256, 0, c->stream>>>(c->nc, h, qx, qy, c->sc);
  c->launches++;
}
