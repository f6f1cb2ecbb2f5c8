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

namespace NH_NS {
namespace {

constexpr int PTX = 32, PTY = 8, PH = 2;  // predictor tile and halo
constexpr int PSX = PTX + 2 * PH, PSY = PTY + 2 * PH;

struct PredTile {
  real h[PSY][PSX], eta[PSY][PSX], u[PSY][PSX], v[PSY][PSX], zb[PSY][PSX];
};

struct Prim {
  real h, eta, un, ut, zb;
};

__device__ __forceinline__ Prim get_prim(const PredTile& T, int lx, int ly, int dir) {
  Prim P;
  P.h = T.h[ly][lx];
  P.eta = T.eta[ly][lx];
  P.zb = T.zb[ly][lx];
  real uu = T.u[ly][lx], vv = T.v[ly][lx];
  if (dir == 0) { P.un = uu; P.ut = vv; } else { P.un = vv; P.ut = uu; }
  return P;
}

// S2: undivided limited slopes (eta, h, un, ut) of the cell at tile position (lx,ly) (L335-337, R2)
__device__ __forceinline__ void cell_slopes(const PredTile& T, int lx, int ly, int dir, int order,
                                            real eps_dry, real s[4]) {
  s[0] = s[1] = s[2] = s[3] = RC(0.0);
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
    s[0] = RC(0.0);
  // R2 (iii): positivity of the reconstructed depth (L335-337)
  if (Pc.h - RC(0.5) * fabs(s[1]) < RC(0.0)) s[1] = copysign(RC(2.0) * Pc.h, s[1]);
}

// S4: PVM/HLL path-conservative fluctuations at one face, eqs (18)(19) with A* (L303-322), three
// components (R3), guards (R4), emerging-bottom clip (R5).  m = U^-, p = U^+.
__device__ __forceinline__ void face_fluct(real g, real hm, real etam, real um, real vm,
                                           real hp, real etap, real up, real vp,
                                           real Dm[3], real Dp[3]) {
  real hh = RC(0.5) * (hm + hp);  // h_{i+1/2}, L276
  real sm = sqrt(hm), sp = sqrt(hp);
  real den = sm + sp;
  real unum = um * sm + up * sp;
  real uh = (den > RC(0.0)) ? ((unum == RC(0.0)) ? unum : unum / den) : RC(0.0);  // Roe average, L276; R4
                                                    // (zero dividend: same bits, no slow path)
  real ch = sqrt(g * hh), cm = sqrt(g * hm), cp = sqrt(g * hp);
  real SL = fmin(uh - ch, um - cm);  // L290
  real SR = fmax(uh + ch, up + cp);  // L292
  if (SR - SL <= RC(1e-14) * (RC(1.0) + ch)) {  // R4: dry-dry face
#pragma unroll
    for (int k = 0; k < 3; ++k) { Dm[k] = RC(0.0); Dp[k] = RC(0.0); }
    return;
  }
  real a0 = (SR * fabs(SL) - SL * fabs(SR)) / (SR - SL);  // L286
  real a1 = (fabs(SR) - fabs(SL)) / (SR - SL);
  // R5: emerging bottom; z^+- = eta^+- - h^+- are the face bed levels
  real zm = etam - hm, zp = etap - hp;
  real zs = fmax(zm, zp);
  real deta;
  if (fmin(etam, etap) >= zs) deta = etap - etam;
  else deta = fmax(RC(0.0), etap - zs) - fmax(RC(0.0), etam - zs);
  real qnm = hm * um, qnp = hp * up;
  real qtm = hm * vm, qtp = hp * vp;
  real R[3], DU[3];
  R[0] = qnp - qnm;  // F_c(U+) - F_c(U-) + T_p, (19)
  R[1] = (qnp * up - qnm * um) + g * hh * deta;
  R[2] = qnp * vp - qnm * vm;
  DU[0] = deta;  // U+ - U- - (H+ - H-) e1, (18)
  DU[1] = qnp - qnm;
  DU[2] = qtp - qtm;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    Dm[k] = RC(0.5) * ((RC(1.0) - a1) * R[k] - a0 * DU[k]);
    Dp[k] = RC(0.5) * ((RC(1.0) + a1) * R[k] + a0 * DU[k]);
  }
}

// One face solve: the face between tile cell (lx,ly) and its neighbour in direction dir.
// sL = slopes of the left / lower cell (returned: its owner needs them for the in-cell term).
__device__ __forceinline__ void hi_face(const PredTile& T, int lx, int ly, int dir, int order,
                                        real eps_dry, real g, real sL[4], real Dm[3],
                                        real Dp[3]) {
  const int di = (dir == 0), dj = (dir == 1);
  Prim Pc = get_prim(T, lx, ly, dir);
  Prim Pp = get_prim(T, lx + di, ly + dj, dir);
  real sR[4];
  cell_slopes(T, lx, ly, dir, order, eps_dry, sL);
  cell_slopes(T, lx + di, ly + dj, dir, order, eps_dry, sR);
  // S3 face states: left = c + s/2, right = p - s/2
  real hL = Pc.h + RC(0.5) * sL[1], eL = Pc.eta + RC(0.5) * sL[0];
  real uL = Pc.un + RC(0.5) * sL[2], vL = Pc.ut + RC(0.5) * sL[3];
  real hR = Pp.h - RC(0.5) * sR[1], eR = Pp.eta - RC(0.5) * sR[0];
  real uR = Pp.un - RC(0.5) * sR[2], vR = Pp.ut - RC(0.5) * sR[3];
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
k_predictor(NhGrid G, real g, real delta, real eps_dry, real manning_n, int order,
            NhScal* sc, const real* __restrict__ H, const real* __restrict__ h,
            const real* __restrict__ qx, const real* __restrict__ qy,
            real* __restrict__ h1, real* __restrict__ qx1, real* __restrict__ qy1,
            const real* __restrict__ eta_in, real* __restrict__ eta_out) {  // fp32 variant: eta planes
  __shared__ PredTile T;
  __shared__ real DPx[3][PTY][PTX + 1];  // D^+ of the x-face on the low side of cell lx - PH
  __shared__ real DPy[3][PTY + 1][PTX];  // D^+ of the y-face on the low side of cell ly - PH
  const int i0 = blockIdx.x * PTX, j0 = blockIdx.y * PTY;
  const int tid = threadIdx.y * PTX + threadIdx.x;
  // S0 + S1: derived fields of the halo tile through the index maps
  for (int e = tid; e < PSX * PSY; e += PTX * PTY) {
    int lx = e % PSX, ly = e / PSX;
    int gi = i0 - PH + lx, gj = j0 - PH + ly;
    real hv = RC(0.0), ev = RC(0.0), uv = RC(0.0), vv = RC(0.0), zv = RC(0.0);
    if (gi <= G.nx + 1 && gj <= G.ny + 1) {
      real sx, sy;
      int ii = nh_map_cell(gi, G.nx, G.bxlo, G.bxhi, sx);
      int jj = nh_map_cell(gj, G.ny, G.bylo, G.byhi, sy);
      size_t k = (size_t)jj * G.nx + ii;
      real Hv = H[k];
      if (kEta) { ev = eta_in[k]; hv = Hv + ev; }  // fp32 variant: eta is the stored quantity
      else { hv = h[k]; ev = hv - Hv; }
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
  real sown[2][4], Dm_hi[2][3];
  if (active) {
#pragma unroll
    for (int dir = 0; dir < 2; ++dir) {
      real Dp[3];
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
      real sl[4], Dm[3], Dp[3];
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
  const real dt = (real)sc->dt;
  real dU[2][3];  // per direction: (h, normal q, tangential q)
#pragma unroll
  for (int dir = 0; dir < 2; ++dir) {
    Prim Pc = get_prim(T, lx, ly, dir);
    const real* s_ = sown[dir];
    // own face states: "hi" face left state = c + s/2, "lo" face right state = c - s/2
    real hL = Pc.h + RC(0.5) * s_[1], uL = Pc.un + RC(0.5) * s_[2], vL = Pc.ut + RC(0.5) * s_[3];
    real hr = Pc.h - RC(0.5) * s_[1], ur = Pc.un - RC(0.5) * s_[2], vr = Pc.ut - RC(0.5) * s_[3];
    // in-cell term I_i of (22) = F_c(U^-_{i+1/2}) - F_c(U^+_{i-1/2}) + g h_i sigma_eta e2 (S5)
    real qnL = hL * uL, qnr = hr * ur;
    real Fhi[3] = {qnL, qnL * uL, qnL * vL};
    real Flo[3] = {qnr, qnr * ur, qnr * vr};
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      real Dp_lo = (dir == 0) ? DPx[k][threadIdx.y][threadIdx.x] : DPy[k][threadIdx.y][threadIdx.x];
      dU[dir][k] = Dm_hi[dir][k] + Dp_lo + (Fhi[k] - Flo[k]);
    }
    dU[dir][1] += g * Pc.h * s_[0];
  }
  size_t k = (size_t)j * G.nx + i;
  real lxr = dt / G.dx, lyr = dt / G.dy;
  real hn, en = RC(0.0);
  if (kEta) { en = eta_in[k] - lxr * dU[0][0] - lyr * dU[1][0]; hn = H[k] + en; }
  else hn = h[k] - lxr * dU[0][0] - lyr * dU[1][0];
  real qxn = qx[k] - lxr * dU[0][1] - lyr * dU[1][2];
  real qyn = qy[k] - lxr * dU[0][2] - lyr * dU[1][1];
  if (hn < RC(0.0)) {  // R7; size statistics for R24 (rare: integer atomics, exact and order independent)
    double a = (double)(-hn);
    int bk = (a < 1e-15) ? 0 : (a < 1e-12) ? 1 : (a < 1e-9) ? 2 : (a < 1e-6) ? 3 : (a < 1e-3) ? 4 : 5;
    atomicAdd(&sc->clamp_hist[bk], 1ULL);
    atomicMax(&sc->clamp_max_bits, (unsigned long long)__double_as_longlong(a));
    atomicAdd((unsigned long long*)&sc->clamps, 1ULL);
    hn = RC(0.0);
    if (kEta) en = -H[k];
  }
  if (hn <= eps_dry) { qxn = RC(0.0); qyn = RC(0.0); }          // R7
  else if (manning_n > RC(0.0)) {
    // Manning friction tau = g h u n^2 |u| / h^(4/3) (L61-65, L773-775), semi-implicit (L249, R27):
    // q <- q / (1 + dt g n^2 |u*| / h*^(4/3)), desingularised velocities of U*, wet cells only
    real uu = nh_dsg(hn, qxn, delta), vv = nh_dsg(hn, qyn, delta);
    real speed = sqrt(uu * uu + vv * vv);
    real h43 = hn * nh_cbrt_fixed(hn);  // R31
    real den = RC(1.0) + dt * g * manning_n * manning_n * speed / h43;
    qxn = qxn / den; qyn = qyn / den;
  }
  h1[k] = hn; qx1[k] = qxn; qy1[k] = qyn;
  if (kEta) eta_out[k] = en;
}

// a0 / R20: lam = max_ij[(|u|+sqrt(gh))/dx + (|v|+sqrt(gh))/dy].  A max is exact and order
// independent; non-negative doubles order like their bit patterns, so one integer atomicMax per
// CTA finishes the device-wide reduction deterministically.
__device__ __forceinline__ real cfl_rate(real g, real delta, real dx, real dy, real h,
                                           real qx, real qy) {
  real cc = sqrt(g * h);
  real uu = nh_dsg(h, qx, delta), vv = nh_dsg(h, qy, delta);
  return (fabs(uu) + cc) / dx + (fabs(vv) + cc) / dy;
}
__device__ __forceinline__ void block_max_to_global(real l, unsigned long long* lam_bits) {
  for (int o = 16; o > 0; o >>= 1) l = fmax(l, __shfl_xor_sync(0xffffffffu, l, o));
  __shared__ real wm[32];
  int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) wm[wid] = l;
  __syncthreads();
  if (wid == 0) {
    int nw = (blockDim.x + 31) >> 5;
    l = (lane < nw) ? wm[lane] : RC(0.0);
    for (int o = 16; o > 0; o >>= 1) l = fmax(l, __shfl_xor_sync(0xffffffffu, l, o));
    if (lane == 0 && l > RC(0.0)) atomicMax(lam_bits, (unsigned long long)__double_as_longlong((double)l));
  }
}

__global__ void __launch_bounds__(256)
k_lambda(size_t nc, real g, real delta, real dx, real dy, const real* __restrict__ h,
         const real* __restrict__ qx, const real* __restrict__ qy, NhScal* sc) {
  real l = RC(0.0);
  for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < nc;
       k += (size_t)gridDim.x * blockDim.x) {
    real v = cfl_rate(g, delta, dx, dy, h[k], qx[k], qy[k]);
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
k_combine(NhGrid G, real g, real delta, real* __restrict__ h0, real* __restrict__ qx0,
          real* __restrict__ qy0, real* __restrict__ w0, const real* __restrict__ h2,
          const real* __restrict__ qx2, const real* __restrict__ qy2,
          const real* __restrict__ w2, NhScal* sc, const real* __restrict__ H,
          real* __restrict__ eta0, const real* __restrict__ eta2) {  // fp32 variant: eta planes
  size_t nc = (size_t)G.nx * G.ny, nn = (size_t)G.np * (G.ny + 1);
  real l = RC(0.0);
  size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < nc; k += stride) {
    real hv;
    if (kEta) {  // combine the stored quantity, then h = H + eta
      real ev = RC(0.5) * eta0[k] + RC(0.5) * eta2[k];
      eta0[k] = ev;
      hv = fmax(H[k] + ev, RC(0.0));
    } else {
      hv = RC(0.5) * h0[k] + RC(0.5) * h2[k];
    }
    real qxv = RC(0.5) * qx0[k] + RC(0.5) * qx2[k];
    real qyv = RC(0.5) * qy0[k] + RC(0.5) * qy2[k];
    h0[k] = hv; qx0[k] = qxv; qy0[k] = qyv;
    real v = cfl_rate(g, delta, G.dx, G.dy, hv, qxv, qyv);
    if (v > l) l = v;
  }
  if (w2 != nullptr)  // nullptr: w did not move in this step (hydrostatic path without zones)
    for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < nn; k += stride)
      w0[k] = RC(0.5) * w0[k] + RC(0.5) * w2[k];
  block_max_to_global(l, &sc->lam_bits);
}

// set_state validation: h >= 0 and finite, q finite
__global__ void __launch_bounds__(256)
k_validate(size_t nc, const real* __restrict__ h, const real* __restrict__ qx,
           const real* __restrict__ qy, NhScal* sc) {
  bool bad = false;
  for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < nc;
       k += (size_t)gridDim.x * blockDim.x) {
    real a = h[k], b = qx[k], c = qy[k];
    if (!(a >= RC(0.0)) || isinf(a) || !(b == b) || !(c == c)) bad = true;
  }
  if (__syncthreads_or(bad) && threadIdx.x == 0) atomicOr(&sc->flags, NH_FLAG_BADSTATE);
}

int grid_1d(const Ctx* c, size_t n, int block) {
  size_t need = (n + block - 1) / block;
  size_t cap = (size_t)c->sm_count * 16;
  return (int)(need < cap ? (need ? need : 1) : cap);
}

}  // namespace

void nh_launch_lambda(Ctx* c, const real* h, const real* qx, const real* qy) {
  k_lambda<<<grid_1d(c, c->nc, 256), 256, 0, c->stream>>>(c->nc, c->prm.g, c->prm.delta, c->g.dx,
                                                          c->g.dy, h, qx, qy, c->sc);
  c->launches++;
}
void nh_launch_set_dt(Ctx* c, double dt_fixed) {
  k_set_dt<<<1, 1, 0, c->stream>>>(c->sc, c->prm.cfl, dt_fixed);
  c->launches++;
}
void nh_launch_end_step(Ctx* c, int advance_time) {
  k_end_step<<<1, 1, 0, c->stream>>>(c->sc, advance_time);
  c->launches++;
}
void nh_launch_predictor(Ctx* c, const real* h, const real* qx, const real* qy, real* h1,
                         real* qx1, real* qy1) {
  dim3 grid((c->g.nx + PTX - 1) / PTX, (c->g.ny + PTY - 1) / PTY), block(PTX, PTY);
  k_predictor<<<grid, block, 0, c->stream>>>(c->g, c->prm.g, c->prm.delta, c->prm.eps_dry,
                                             c->prm.manning_n, c->prm.space_order, c->sc, c->H, h, qx, qy, h1, qx1,
                                             qy1, nh_eta_of(c, h), nh_eta_of(c, h1));
  c->launches++;
}
void nh_launch_combine(Ctx* c, real* h0, real* qx0, real* qy0, real* w0, const real* h2,
                       const real* qx2, const real* qy2, const real* w2) {
  k_combine<<<grid_1d(c, c->nn, 256), 256, 0, c->stream>>>(c->g, c->prm.g, c->prm.delta, h0, qx0,
                                                           qy0, w0, h2, qx2, qy2, w2, c->sc, c->H,
                                                           nh_eta_of(c, h0), nh_eta_of(c, h2));
  c->launches++;
}
void nh_launch_validate(Ctx* c, const real* h, const real* qx, const real* qy) {
  k_validate<<<grid_1d(c, c->nc, 256), 256, 0, c->stream>>>(c->nc, h, qx, qy, c->sc);
  c->launches++;
}

}  // namespace NH_NS
