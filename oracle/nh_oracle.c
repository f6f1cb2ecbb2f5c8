/* nh_oracle.c -- CPU ORACLE (test infrastructure, NOT the product; see nh_oracle.h).
 *
 * One time step of the scheme of arXiv 1706.04551, written step by step in the
 * paper's order and notation.  Steps S0..S11 and readings R1..R23 refer to SURVEY.md 8(c)
 * (restated in DESIGN.md; R24..R31 are DESIGN.md's own); "L<n>" are PAPER.md line numbers.
 *
 * Plain C, fp64, scalar loops, no blocking / fusion / reordering beyond what the formulas
 * state.  OpenMP only splits loops over rows j (every row is independent inside a loop).
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/build.py).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): lake at rest (P1), mass (P2), textbook HLL +
 * Stoker dam break (P3), printed 1D coefficients (43) + x<->y symmetry (P4), constraint after
 * correction via an independent transcription of (36)-(41) (P5), dense LU (P6), dry-slope
 * closed form (P7), linear dispersion relation (P8), 2nd-order convergence (P9), diagonal
 * dominance (P10), flat-bottom symmetry (P11), breaking properties and the printed 1D magnitudes
 * (P12), closed forms of the generating / absorbing zones (R18, R29), of the CFL time step (23), of
 * Manning friction (R27) and of the w transport (R30), the all-dry branch (R26), the fixed-algorithm
 * cube root and sech^2 against libm (R31).
 * Parity unpinned (internal consistency only): the 3-component 2D face solver reading R3 and the
 * 2D extension R12 of the breaking terms.
 */
#include "nh_oracle.h"
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

struct nho_ctx {
  int nx, ny;        /* cells                                                     */
  int nnx, nny;      /* distinct node lines: n in a periodic direction, else n+1  */
  double dx, dy;
  nho_params prm;
  nho_info info;
  char err[256];
  /* state */
  double *H, *h, *qx, *qy;   /* cells */
  double *w, *p;             /* nodes, full (nx+1)*(ny+1) layout */
  unsigned char *flag_c, *flag_n; /* breaking hysteresis flags (R11) */
  /* stage scratch (cells) */
  double *eta, *u, *v;       /* S0 derived fields of the stage input */
  double *h1, *qx1, *qy1;    /* predictor output U* */
  double *qx2, *qy2;         /* q** (after breaking sources) */
  double *z;                 /* z = 2 eta - h of U* */
  /* stage scratch (nodes) */
  double *w2, *b;            /* w**, rhs */
  double *kr, *kr0, *kp, *kv, *ks, *kt, *kph, *ksh, *kdiag; /* BiCGStab vectors */
  /* RK copies */
  double *h0, *qx0, *qy0, *w0;
  double *wadv;              /* w after the transport step of the w-advection variant (R30) */
  double *hist[7];           /* R32: the last seven pressure solutions, hist[0] the most recent */
  int nhist;                 /* how many of them are valid (reset by nho_set_state) */
};

/* ------------------------------------------------------------------------------------ */
/* S1 ghost access by index maps (reading R9).                                           */
/* cells: periodic wraps; wall / outflow mirror (-1->0, -2->1, n->n-1, n+1->n-2);        */
/* *sgn = -1 only for a wall ghost (the caller applies it to the normal discharge).      */
static int map_cell(int i, int n, int bclo, int bchi, int* sgn) {
  *sgn = 1;
  if (i < 0) {
    if (bclo == NHO_BC_PERIODIC) return i + n;
    if (bclo == NHO_BC_WALL) *sgn = -1;
    return -1 - i;
  }
  if (i >= n) {
    if (bchi == NHO_BC_PERIODIC) return i - n;
    if (bchi == NHO_BC_WALL) *sgn = -1;
    return 2 * n - 1 - i;
  }
  return i;
}
/* nodes: periodic: node n == node 0 (n distinct lines); mirror: -1->1, n+1->n-1.         */
static int map_node(int I, int n, int bclo, int bchi) {
  if (bclo == NHO_BC_PERIODIC) { /* both sides periodic */
    (void)bchi;
    int r = I % n;
    return r < 0 ? r + n : r;
  }
  if (I < 0) return -I;
  if (I > n) return 2 * n - I;
  return I;
}

/* OpenMP splits loops over rows when the grid is worth it (scheduling only: every reduction used is
 * exact or has a fixed order, so results do not depend on the number of threads) */
#define NHO_PAR(c) ((c)->ny >= 8 && (long long)(c)->nx * (c)->ny >= 4096)

#define CIDX(c, i, j) ((size_t)(j) * (size_t)(c)->nx + (size_t)(i))
#define NIDX(c, I, J) ((size_t)(J) * (size_t)((c)->nx + 1) + (size_t)(I))

/* even cell field (h, H, eta, z, ...) at a possibly-ghost index */
static double cell_even(const nho_ctx* c, const double* a, int i, int j) {
  int sx, sy;
  int ii = map_cell(i, c->nx, c->prm.bc_xlo, c->prm.bc_xhi, &sx);
  int jj = map_cell(j, c->ny, c->prm.bc_ylo, c->prm.bc_yhi, &sy);
  return a[CIDX(c, ii, jj)];
}
/* x-normal field (qx, u): flips sign in an x-wall ghost */
static double cell_xn(const nho_ctx* c, const double* a, int i, int j) {
  int sx, sy;
  int ii = map_cell(i, c->nx, c->prm.bc_xlo, c->prm.bc_xhi, &sx);
  int jj = map_cell(j, c->ny, c->prm.bc_ylo, c->prm.bc_yhi, &sy);
  return (double)sx * a[CIDX(c, ii, jj)];
}
/* y-normal field (qy, v): flips sign in a y-wall ghost */
static double cell_yn(const nho_ctx* c, const double* a, int i, int j) {
  int sx, sy;
  int ii = map_cell(i, c->nx, c->prm.bc_xlo, c->prm.bc_xhi, &sx);
  int jj = map_cell(j, c->ny, c->prm.bc_ylo, c->prm.bc_yhi, &sy);
  return (double)sy * a[CIDX(c, ii, jj)];
}
/* node field (p, w, Krylov vectors) at a possibly-ghost node index */
static double node_val(const nho_ctx* c, const double* a, int I, int J) {
  int II = map_node(I, c->nx, c->prm.bc_xlo, c->prm.bc_xhi);
  int JJ = map_node(J, c->ny, c->prm.bc_ylo, c->prm.bc_yhi);
  return a[NIDX(c, II, JJ)];
}

/* ------------------------------------------------------------------------------------ */
/* S0: desingularised velocity, L447-451:  u = sqrt(2) h q / sqrt(h^4 + max(h^4, delta^4)) */
double nho_dsg(double h, double q, double delta) {
  double h2 = h * h, h4 = h2 * h2;
  double d2 = delta * delta, d4 = d2 * d2;
  double den = sqrt(h4 + fmax(h4, d4));
  return (sqrt(2.0) * h * q) / den;
}
/* R16: dinv(h) = sqrt(2) h / sqrt(h^4 + max(h^4, delta^4))  (= 1/h for h >= delta) */
static double dinv_h(double h, double delta) {
  double h2 = h * h, h4 = h2 * h2;
  double d2 = delta * delta, d4 = d2 * d2;
  return (sqrt(2.0) * h) / sqrt(h4 + fmax(h4, d4));
}
/* S2: minmod(a,b) = 0 if ab <= 0 else sign(a) min(|a|,|b|)   (L335, [25]) */
double nho_minmod(double a, double b) {
  if (a * b <= 0.0) return 0.0;
  return (a > 0.0) ? fmin(a, b) : fmax(a, b);
}

/* Reading R31 (two transcendentals evaluated by a FIXED algorithm).  h^(4/3) of the friction law
 * (L61-65) and sech^2 of the solitary-wave target (33) need a cube root and an exponential; libm's
 * are not correctly rounded and differ from library to library in the last place, and a wet/dry
 * front amplifies last-place differences.  Both are therefore evaluated by a stated sequence of
 * IEEE operations (frexp / ldexp / floor are exact), which any implementation reproduces bit for bit.
 * Accuracy: a few ulp (pinned against libm in tests/test_oracle_pins.py). */
/* cube root of a > 0: a = t 8^q with t in [0.5, 4); six Halley steps y <- y (y^3 + 2t) / (2y^3 + t)
 * from y = 1 (cubic convergence: 0.37 -> 3e-2 -> 3e-5 -> 1e-14 -> rounding) */
static double cbrt_fixed(double a) {
  int e;
  double m = frexp(a, &e);             /* a = m 2^e, m in [0.5, 1) */
  int q = (e + 3072) / 3 - 1024;       /* floor(e / 3), non-negative dividend */
  double t = ldexp(m, e - 3 * q);      /* t in [0.5, 4) */
  double y = 1.0;
  for (int k = 0; k < 6; ++k) {
    double y3 = y * y * y;
    y = y * (y3 + 2.0 * t) / (2.0 * y3 + t);
  }
  return ldexp(y, q);
}
/* sech^2(a) = 4 e / (1 + e)^2, e = exp(-2|a|) = 2^-n exp(-r), n = nearest integer to 2|a| / ln 2,
 * r = 2|a| - n ln 2 in two pieces (|r| <= 0.35), exp(-r) by its Taylor series to r^14 (Horner) */
static double sech2_fixed(double a) {
  double y = 2.0 * fabs(a);
  if (y > 745.0) return 0.0;
  double n = floor(y * 1.4426950408889634 + 0.5);
  double r = (y - n * 0.693147180369123816490) - n * 1.90821492927058770002e-10;
  double p = 1.0;
  for (int k = 14; k >= 1; --k) p = 1.0 - (r / (double)k) * p;
  double e = ldexp(p, -(int)n);
  double d = 1.0 + e;
  return 4.0 * e / (d * d);
}
double nho_cbrt_fixed(double a) { return cbrt_fixed(a); }   /* test hooks (pins) */
double nho_sech2_fixed(double a) { return sech2_fixed(a); }

static void derived_fields(nho_ctx* c, const double* h, const double* qx, const double* qy) {
  const double delta = c->prm.delta;
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
  for (int j = 0; j < c->ny; ++j)
    for (int i = 0; i < c->nx; ++i) {
      size_t k = CIDX(c, i, j);
      c->eta[k] = h[k] - c->H[k];
      c->u[k] = nho_dsg(h[k], qx[k], delta);
      c->v[k] = nho_dsg(h[k], qy[k], delta);
    }
}

/* ------------------------------------------------------------------------------------ */
/* S4: PVM/HLL path-conservative fluctuations at one face, eqs (18)(19) with A* (L303-322),  */
/* three components (R3), guards (R4), emerging-bottom clip (R5).                           */
/* "m" = state left of the face (U^-), "p" = right (U^+); u normal, v tangential velocity.  */
/* D[0]: h, D[1]: normal discharge, D[2]: tangential discharge.                            */
void nho_face_fluct(double g, double hm, double etam, double um, double vm,
                    double hp, double etap, double up, double vp,
                    double Dm[3], double Dp[3]) {
  double hh = 0.5 * (hm + hp);                       /* h_{i+1/2}, L276 */
  double sm = sqrt(hm), sp = sqrt(hp);
  double den = sm + sp;
  double uh = (den > 0.0) ? (um * sm + up * sp) / den : 0.0; /* Roe average, L276; R4 */
  double ch = sqrt(g * hh), cm = sqrt(g * hm), cp = sqrt(g * hp);
  double SL = fmin(uh - ch, um - cm);                /* L290 */
  double SR = fmax(uh + ch, up + cp);                /* L292 */
  if (SR - SL <= 1e-14 * (1.0 + ch)) {               /* R4: dry-dry face */
    for (int k = 0; k < 3; ++k) { Dm[k] = 0.0; Dp[k] = 0.0; }
    return;
  }
  double a0 = (SR * fabs(SL) - SL * fabs(SR)) / (SR - SL);   /* L286 */
  double a1 = (fabs(SR) - fabs(SL)) / (SR - SL);
  /* R5: emerging bottom.  z^+- = eta^+- - h^+- are the face bed levels. */
  double zm = etam - hm, zp = etap - hp;
  double zs = fmax(zm, zp);
  double deta;
  if (fmin(etam, etap) >= zs) deta = etap - etam;
  else deta = fmax(0.0, etap - zs) - fmax(0.0, etam - zs);
  double qnm = hm * um, qnp = hp * up;               /* normal discharges */
  double qtm = hm * vm, qtp = hp * vp;               /* tangential discharges */
  double R[3], DU[3];
  R[0] = qnp - qnm;                                  /* F_c(U+) - F_c(U-) + T_p, (19) */
  R[1] = (qnp * up - qnm * um) + g * hh * deta;
  R[2] = qnp * vp - qnm * vm;
  DU[0] = deta;                                      /* U+ - U- - (H+ - H-) e1, (18) */
  DU[1] = qnp - qnm;
  DU[2] = qtp - qtm;
  for (int k = 0; k < 3; ++k) {
    Dm[k] = 0.5 * ((1.0 - a1) * R[k] - a0 * DU[k]);
    Dp[k] = 0.5 * ((1.0 + a1) * R[k] + a0 * DU[k]);
  }
}

/* primitive state of a (possibly ghost) cell, as seen in direction dir (0: x, 1: y):      */
/* un = velocity normal to the faces of that direction, ut = tangential.                   */
typedef struct { double h, eta, un, ut, zb; } prim_t;

static prim_t get_prim(const nho_ctx* c, const double* h, int i, int j, int dir) {
  prim_t P;
  P.h = cell_even(c, h, i, j);
  P.eta = cell_even(c, c->eta, i, j);
  P.zb = -cell_even(c, c->H, i, j);
  double uu = cell_xn(c, c->u, i, j), vv = cell_yn(c, c->v, i, j);
  if (dir == 0) { P.un = uu; P.ut = vv; } else { P.un = vv; P.ut = uu; }
  return P;
}

/* S2: undivided limited slopes (eta, h, un, ut) of cell (i,j) in direction dir. */
static void cell_slopes(const nho_ctx* c, const double* h, int i, int j, int dir, double s[4]) {
  s[0] = s[1] = s[2] = s[3] = 0.0;
  if (c->prm.space_order == 1) return;
  int di = (dir == 0), dj = (dir == 1);
  prim_t Pc = get_prim(c, h, i, j, dir);
  if (Pc.h <= c->prm.eps_dry) return;                         /* R2 (i): dry cell */
  prim_t Pm = get_prim(c, h, i - di, j - dj, dir);
  prim_t Pp = get_prim(c, h, i + di, j + dj, dir);
  s[0] = nho_minmod(Pc.eta - Pm.eta, Pp.eta - Pc.eta);
  s[1] = nho_minmod(Pc.h - Pm.h, Pp.h - Pc.h);
  s[2] = nho_minmod(Pc.un - Pm.un, Pp.un - Pc.un);
  s[3] = nho_minmod(Pc.ut - Pm.ut, Pp.ut - Pc.ut);
  /* R2 (ii): emerging bottom against either neighbour -> gradient of eta set to zero (L337) */
  if (fmin(Pc.eta, Pm.eta) < fmax(Pc.zb, Pm.zb) || fmin(Pc.eta, Pp.eta) < fmax(Pc.zb, Pp.zb))
    s[0] = 0.0;
  /* R2 (iii): positivity of the reconstructed depth (L335-337) */
  if (Pc.h - 0.5 * fabs(s[1]) < 0.0) s[1] = copysign(2.0 * Pc.h, s[1]);
}

/* S2-S5: hydrostatic predictor, eqs (20)-(22) per direction = eq. (30) (R6).              */
/* in: (h,qx,qy) + derived fields; out: (h1,qx1,qy1).                                       */
static void predictor(nho_ctx* c, const double* h, const double* qx, const double* qy, double dt) {
  const double g = c->prm.g;
  long long clamps = 0, hist[6] = {0, 0, 0, 0, 0, 0};
  double cmax = 0.0;
  derived_fields(c, h, qx, qy);
#pragma omp parallel for if (NHO_PAR(c)) schedule(static) reduction(+ : clamps, hist[:6]) reduction(max : cmax)
  for (int j = 0; j < c->ny; ++j)
    for (int i = 0; i < c->nx; ++i) {
      double dU[2][3]; /* per direction: (h, normal q, tangential q) */
      for (int dir = 0; dir < 2; ++dir) {
        int di = (dir == 0), dj = (dir == 1);
        prim_t Pc = get_prim(c, h, i, j, dir);
        prim_t Pm = get_prim(c, h, i - di, j - dj, dir);
        prim_t Pp = get_prim(c, h, i + di, j + dj, dir);
        double sc[4], sm[4], sp[4];
        cell_slopes(c, h, i, j, dir, sc);
        cell_slopes(c, h, i - di, j - dj, dir, sm);
        cell_slopes(c, h, i + di, j + dj, dir, sp);
        /* S3 face states.  "hi" face (i+1/2): left = c + s/2, right = p - s/2 */
        double hL = Pc.h + 0.5 * sc[1], eL = Pc.eta + 0.5 * sc[0];
        double uL = Pc.un + 0.5 * sc[2], vL = Pc.ut + 0.5 * sc[3];
        double hR = Pp.h - 0.5 * sp[1], eR = Pp.eta - 0.5 * sp[0];
        double uR = Pp.un - 0.5 * sp[2], vR = Pp.ut - 0.5 * sp[3];
        double Dm_hi[3], Dp_hi[3];
        nho_face_fluct(g, hL, eL, uL, vL, hR, eR, uR, vR, Dm_hi, Dp_hi);
        /* "lo" face (i-1/2): left = m + s/2, right = c - s/2 */
        double hl = Pm.h + 0.5 * sm[1], el = Pm.eta + 0.5 * sm[0];
        double ul = Pm.un + 0.5 * sm[2], vl = Pm.ut + 0.5 * sm[3];
        double hr = Pc.h - 0.5 * sc[1], er = Pc.eta - 0.5 * sc[0];
        double ur = Pc.un - 0.5 * sc[2], vr = Pc.ut - 0.5 * sc[3];
        double Dm_lo[3], Dp_lo[3];
        nho_face_fluct(g, hl, el, ul, vl, hr, er, ur, vr, Dm_lo, Dp_lo);
        /* in-cell term I_i of (22) = F_c(U^-_{i+1/2}) - F_c(U^+_{i-1/2}) + g h_i sigma_eta e2 (S5) */
        double qnL = hL * uL, qnr = hr * ur;
        double Fhi[3] = { qnL, qnL * uL, qnL * vL };
        double Flo[3] = { qnr, qnr * ur, qnr * vr };
        for (int k = 0; k < 3; ++k) dU[dir][k] = Dm_hi[k] + Dp_lo[k] + (Fhi[k] - Flo[k]);
        dU[dir][1] += g * Pc.h * sc[0];
      }
      size_t k = CIDX(c, i, j);
      double lx = dt / c->dx, ly = dt / c->dy;
      double hn = h[k] - lx * dU[0][0] - ly * dU[1][0];
      double qxn = qx[k] - lx * dU[0][1] - ly * dU[1][2];
      double qyn = qy[k] - lx * dU[0][2] - ly * dU[1][1];
      if (hn < 0.0) {                                       /* R7; size statistics for R24 */
        double a = -hn;
        int bk = (a < 1e-15) ? 0 : (a < 1e-12) ? 1 : (a < 1e-9) ? 2 : (a < 1e-6) ? 3 : (a < 1e-3) ? 4 : 5;
        hist[bk]++;
        if (a > cmax) cmax = a;
        hn = 0.0; clamps++;
      }
      if (hn <= c->prm.eps_dry) { qxn = 0.0; qyn = 0.0; }   /* R7 */
      else if (c->prm.manning_n > 0.0) {
        /* Manning friction tau = g h u n^2 |u| / h^(4/3) (L61-65, L773-775), "discretized
         * semi-implicitly" (L249, L484; reading R27): q <- q / (1 + dt g n^2 |u*| / h*^(4/3))
         * with the desingularised velocities of U* (S0); wet cells only. */
        double uu = nho_dsg(hn, qxn, c->prm.delta), vv = nho_dsg(hn, qyn, c->prm.delta);
        double speed = sqrt(uu * uu + vv * vv);
        double h43 = hn * cbrt_fixed(hn);   /* R31 */
        double den = 1.0 + dt * g * c->prm.manning_n * c->prm.manning_n * speed / h43;
        qxn = qxn / den; qyn = qyn / den;
      }
      c->h1[k] = hn; c->qx1[k] = qxn; c->qy1[k] = qyn;
    }
  c->info.clamps += clamps;
  for (int k = 0; k < 6; ++k) c->info.clamp_hist[k] += hist[k];
  if (cmax > c->info.clamp_max) c->info.clamp_max = cmax;
}

/* A4 / R20: dt = CFL / max_ij[(|u|+sqrt(gh))/dx + (|v|+sqrt(gh))/dy] */
static double cfl_dt(nho_ctx* c, const double* h, const double* qx, const double* qy) {
  double lam = 0.0;
  const double g = c->prm.g, delta = c->prm.delta;
#pragma omp parallel for if (NHO_PAR(c)) schedule(static) reduction(max : lam)
  for (int j = 0; j < c->ny; ++j)
    for (int i = 0; i < c->nx; ++i) {
      size_t k = CIDX(c, i, j);
      double cc = sqrt(g * h[k]);
      double uu = nho_dsg(h[k], qx[k], delta), vv = nho_dsg(h[k], qy[k], delta);
      double l = (fabs(uu) + cc) / c->dx + (fabs(vv) + cc) / c->dy;
      if (l > lam) lam = l;
    }
  return (lam > 0.0) ? c->prm.cfl / lam : 0.0;
}

/* ------------------------------------------------------------------------------------ */
/* S7/S8 geometry at node (I,J): the four cells around it and the compact edge values.     */
typedef struct {
  double hn;                  /* (38) */
  double hE, hW, hN, hS;      /* edge averages of h */
  double xE, xW, xN, xS;      /* edge averages of xi^x (E,W) and xi^y (N,S) */
  double zx, zy;              /* zeta^x = z_E - z_W, zeta^y = z_N - z_S */
} node_geo;

static double xi_x(const nho_ctx* c, const double* z, int i, int j) {
  return 0.5 * (cell_even(c, z, i + 1, j) - cell_even(c, z, i - 1, j));
}
static double xi_y(const nho_ctx* c, const double* z, int i, int j) {
  return 0.5 * (cell_even(c, z, i, j + 1) - cell_even(c, z, i, j - 1));
}

static node_geo node_geometry(const nho_ctx* c, const double* h, const double* z, int I, int J) {
  node_geo G;
  /* SW=(I-1,J-1), SE=(I,J-1), NW=(I-1,J), NE=(I,J) */
  double hSW = cell_even(c, h, I - 1, J - 1), hSE = cell_even(c, h, I, J - 1);
  double hNW = cell_even(c, h, I - 1, J), hNE = cell_even(c, h, I, J);
  double zSW = cell_even(c, z, I - 1, J - 1), zSE = cell_even(c, z, I, J - 1);
  double zNW = cell_even(c, z, I - 1, J), zNE = cell_even(c, z, I, J);
  G.hn = 0.25 * (hSW + hSE + hNE + hNW);
  G.hE = 0.5 * (hNE + hSE); G.hW = 0.5 * (hNW + hSW);
  G.hN = 0.5 * (hNE + hNW); G.hS = 0.5 * (hSE + hSW);
  G.xE = 0.5 * (xi_x(c, z, I, J) + xi_x(c, z, I, J - 1));
  G.xW = 0.5 * (xi_x(c, z, I - 1, J) + xi_x(c, z, I - 1, J - 1));
  G.xN = 0.5 * (xi_y(c, z, I, J) + xi_y(c, z, I - 1, J));
  G.xS = 0.5 * (xi_y(c, z, I, J - 1) + xi_y(c, z, I - 1, J - 1));
  G.zx = 0.5 * (zNE + zSE) - 0.5 * (zNW + zSW);   /* (2eta-h)_E - (2eta-h)_W, L896-898 */
  G.zy = 0.5 * (zNE + zNW) - 0.5 * (zSE + zSW);
  return G;
}

/* S8: the five coefficients of row (I,J) (derived from (36)-(41); 1D restriction = (43)). */
static void node_coeffs(const nho_ctx* c, const double* h, const double* z, int I, int J,
                        double* AC, double* AE, double* AW, double* AN, double* AS) {
  node_geo G = node_geometry(c, h, z, I, J);
  double ex = 8.0 * c->dx * c->dx, ey = 8.0 * c->dy * c->dy;
  double am = 2.0 * G.hn - G.zx, ap = 2.0 * G.hn + G.zx;
  double bm = 2.0 * G.hn - G.zy, bp = 2.0 * G.hn + G.zy;
  *AE = -(am * (2.0 * G.hE + G.xE)) / ex;
  *AW = -(ap * (2.0 * G.hW - G.xW)) / ex;
  *AN = -(bm * (2.0 * G.hN + G.xN)) / ey;
  *AS = -(bp * (2.0 * G.hS - G.xS)) / ey;
  *AC = 2.0 + (am * (2.0 * G.hE - G.xE) + ap * (2.0 * G.hW + G.xW)) / ex
            + (bm * (2.0 * G.hN - G.xN) + bp * (2.0 * G.hS + G.xS)) / ey;
}

/* y = A x on the distinct nodes; neighbours through the node maps (R10). */
static void apply_A(const nho_ctx* c, const double* h, const double* z, const double* x, double* y) {
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
  for (int J = 0; J < c->nny; ++J)
    for (int I = 0; I < c->nnx; ++I) {
      double AC, AE, AW, AN, AS;
      node_coeffs(c, h, z, I, J, &AC, &AE, &AW, &AN, &AS);
      y[NIDX(c, I, J)] = AC * x[NIDX(c, I, J)] + AE * node_val(c, x, I + 1, J)
                       + AW * node_val(c, x, I - 1, J) + AN * node_val(c, x, I, J + 1)
                       + AS * node_val(c, x, I, J - 1);
    }
}

/* S7: discrete constraint B of (37)-(40) at node (I,J) from cell fields (h, qx, qy, z) and w. */
static double node_B(const nho_ctx* c, const double* h, const double* qx, const double* qy,
                     const double* z, const double* w, int I, int J) {
  double hn = 0.25 * (cell_even(c, h, I - 1, J - 1) + cell_even(c, h, I, J - 1)
                      + cell_even(c, h, I, J) + cell_even(c, h, I - 1, J));
  double q1E = 0.5 * (cell_xn(c, qx, I, J) + cell_xn(c, qx, I, J - 1));
  double q1W = 0.5 * (cell_xn(c, qx, I - 1, J) + cell_xn(c, qx, I - 1, J - 1));
  double q2N = 0.5 * (cell_yn(c, qy, I, J) + cell_yn(c, qy, I - 1, J));
  double q2S = 0.5 * (cell_yn(c, qy, I, J - 1) + cell_yn(c, qy, I - 1, J - 1));
  double zE = 0.5 * (cell_even(c, z, I, J) + cell_even(c, z, I, J - 1));
  double zW = 0.5 * (cell_even(c, z, I - 1, J) + cell_even(c, z, I - 1, J - 1));
  double zN = 0.5 * (cell_even(c, z, I, J) + cell_even(c, z, I - 1, J));
  double zS = 0.5 * (cell_even(c, z, I, J - 1) + cell_even(c, z, I - 1, J - 1));
  double divq = (q1E - q1W) / c->dx + (q2N - q2S) / c->dy;
  return hn * divq - 0.5 * (q1E + q1W) * (zE - zW) / c->dx
                   - 0.5 * (q2N + q2S) * (zN - zS) / c->dy + 2.0 * hn * w[NIDX(c, I, J)];
}

static void compute_z(nho_ctx* c, const double* h, double* z) {
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
  for (int j = 0; j < c->ny; ++j)
    for (int i = 0; i < c->nx; ++i) {
      size_t k = CIDX(c, i, j);
      double eta = h[k] - c->H[k];
      z[k] = 2.0 * eta - h[k];                 /* 2 eta - h, eq. (6) */
    }
}

/* dot products over the distinct nodes: row sums, then the sum of the row sums (fixed order) */
static double dot_nodes(const nho_ctx* c, const double* a, const double* b2) {
  double* rows = (double*)malloc(sizeof(double) * (size_t)c->nny);
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
  for (int J = 0; J < c->nny; ++J) {
    double s = 0.0;
    for (int I = 0; I < c->nnx; ++I) s += a[NIDX(c, I, J)] * b2[NIDX(c, I, J)];
    rows[J] = s;
  }
  double s = 0.0;
  for (int J = 0; J < c->nny; ++J) s += rows[J];
  free(rows);
  return s;
}

/* S9: Jacobi-preconditioned BiCGStab (van der Vorst 1992 form), R14.  x: start -> solution. */
static int bicgstab(nho_ctx* c, const double* h, const double* z, const double* b, double* x,
                    int* iters_out, double* relres_out) {
  const double rtol = c->prm.solver_rtol;
  const int maxit = c->prm.solver_maxit;
  double *r = c->kr, *r0 = c->kr0, *p = c->kp, *v = c->kv, *s = c->ks, *t = c->kt;
  double *ph = c->kph, *sh = c->ksh, *dg = c->kdiag;
  const int nnx = c->nnx, nny = c->nny;
  int iters = 0, status = NHO_OK;
  *iters_out = 0; *relres_out = 0.0;
  double bnorm = sqrt(dot_nodes(c, b, b));
  if (!(bnorm == bnorm) || isinf(bnorm)) return NHO_ENAN;
  if (bnorm == 0.0) {
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
    for (int J = 0; J < nny; ++J)
      for (int I = 0; I < nnx; ++I) x[NIDX(c, I, J)] = 0.0;
    return NHO_OK;
  }
  const double tol = rtol * bnorm;
  /* M = diag(A_C) */
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
  for (int J = 0; J < nny; ++J)
    for (int I = 0; I < nnx; ++I) {
      double AC, AE, AW, AN, AS;
      node_coeffs(c, h, z, I, J, &AC, &AE, &AW, &AN, &AS);
      dg[NIDX(c, I, J)] = AC;
    }
  int converged = 0;
  double rnorm = 0.0;
  for (int cycle = 0; cycle < 8 && !converged; ++cycle) {
    /* true residual r = b - A x */
    apply_A(c, h, z, x, r);
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
    for (int J = 0; J < nny; ++J)
      for (int I = 0; I < nnx; ++I) {
        size_t k = NIDX(c, I, J);
        r[k] = b[k] - r[k]; r0[k] = r[k]; p[k] = 0.0; v[k] = 0.0;
      }
    rnorm = sqrt(dot_nodes(c, r, r));
    if (rnorm <= tol) { converged = 1; break; }
    if (iters >= maxit) break;
    double rho = 1.0, alpha = 1.0, omega = 1.0;
    while (iters < maxit) {
      double rho_new = dot_nodes(c, r0, r);
      if (fabs(rho_new) < 1e-300) break;                    /* breakdown -> restart */
      double beta = (rho_new / rho) * (alpha / omega);
      rho = rho_new;
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
      for (int J = 0; J < nny; ++J)
        for (int I = 0; I < nnx; ++I) {
          size_t k = NIDX(c, I, J);
          p[k] = r[k] + beta * (p[k] - omega * v[k]);
          ph[k] = p[k] / dg[k];
        }
      apply_A(c, h, z, ph, v);
      double sigma = dot_nodes(c, r0, v);
      if (fabs(sigma) < 1e-300) break;
      alpha = rho / sigma;
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
      for (int J = 0; J < nny; ++J)
        for (int I = 0; I < nnx; ++I) {
          size_t k = NIDX(c, I, J);
          s[k] = r[k] - alpha * v[k];
        }
      iters++;
      double snorm = sqrt(dot_nodes(c, s, s));
      if (snorm <= tol) {                                   /* half-step exit */
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
        for (int J = 0; J < nny; ++J)
          for (int I = 0; I < nnx; ++I) {
            size_t k = NIDX(c, I, J);
            x[k] += alpha * ph[k];
          }
        break;
      }
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
      for (int J = 0; J < nny; ++J)
        for (int I = 0; I < nnx; ++I) {
          size_t k = NIDX(c, I, J);
          sh[k] = s[k] / dg[k];
        }
      apply_A(c, h, z, sh, t);
      double tt = dot_nodes(c, t, t);
      if (tt == 0.0) break;
      omega = dot_nodes(c, t, s) / tt;
      if (fabs(omega) < 1e-300) break;
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
      for (int J = 0; J < nny; ++J)
        for (int I = 0; I < nnx; ++I) {
          size_t k = NIDX(c, I, J);
          x[k] += alpha * ph[k] + omega * sh[k];
          r[k] = s[k] - omega * t[k];
        }
      rnorm = sqrt(dot_nodes(c, r, r));
      if (rnorm <= tol) break;
    }
    /* loop back: the true residual decides (recursive residual may have drifted) */
  }
  if (!converged) status = NHO_ENOCONV;
  *relres_out = rnorm / bnorm;
  *iters_out = iters;
  /* one extra "polish" iteration from a fresh start (R14, SURVEY hard parts) */
  if (converged && rnorm > 0.0) {
    /* r, r0 hold the true residual; p = r */
    double rho = dot_nodes(c, r0, r);
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
    for (int J = 0; J < nny; ++J)
      for (int I = 0; I < nnx; ++I) {
        size_t k = NIDX(c, I, J);
        ph[k] = r[k] / dg[k];
      }
    apply_A(c, h, z, ph, v);
    double sigma = dot_nodes(c, r0, v);
    if (fabs(rho) >= 1e-300 && fabs(sigma) >= 1e-300) {
      double alpha = rho / sigma;
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
      for (int J = 0; J < nny; ++J)
        for (int I = 0; I < nnx; ++I) {
          size_t k = NIDX(c, I, J);
          s[k] = r[k] - alpha * v[k];
          sh[k] = s[k] / dg[k];
        }
      apply_A(c, h, z, sh, t);
      double tt = dot_nodes(c, t, t);
      double omega = (tt > 0.0) ? dot_nodes(c, t, s) / tt : 0.0;
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
      for (int J = 0; J < nny; ++J)
        for (int I = 0; I < nnx; ++I) {
          size_t k = NIDX(c, I, J);
          x[k] += alpha * ph[k] + omega * sh[k];
        }
    }
  }
  return status;
}

/* ------------------------------------------------------------------------------------ */
/* S6: breaking sources (section 3, eqs (9)-(12); 2D reading R12, node reading R13).        */
/* S9' (solver = 1): the paper's solver, "an iterative Jacobi method combined with a scheduled
 * relaxation method following [2]" with the stopping rule (32).
 * The paper prints neither the relaxation factors nor the cycle; reading R28:
 *   - row-scaled system: dinv = 1/A_C, c_X = A_X dinv, b' = b dinv (Jacobi's D^-1);
 *   - rho = max_n ((|c_E|+|c_W|)+|c_N|)+|c_S| < 1 is the Gershgorin radius of D^-1 A about 1
 *     (strict diagonal dominance, L503-505), so the spectrum lies in [1-rho, 1+rho];
 *   - one relaxation cycle has M factors, the reciprocals of the Chebyshev nodes of that interval,
 *       omega_k = 1 / (1 - rho cos(pi (2k-1) / (2M))),  k = 1..M
 *     (the optimal scheduled-relaxation factors are exactly these: Adsuara et al.'s follow-up to
 *     [2]), applied in the Lebedev-Finogenov order for powers of two (perm_1 = (1); perm_2m =
 *     (p_1, 2m+1-p_1, p_2, 2m+1-p_2, ...)), which keeps round-off bounded for long cycles;
 *   - M = smallest power of two with M sqrt(2 (1-rho)) >= 7.6 (one cycle then damps every mode
 *     about 1000-fold), at most srj_mmax;
 *   - iteration k: z = b' - (x + c_E x_E + c_W x_W + c_N x_N + c_S x_S) is the increment of the
 *     plain Jacobi method; stop if E = ||z||_inf < tol, eq. (32) (x is then the answer), with
 *     tol = srj_eps (the paper's absolute epsilon) or, if srj_rel > 0, tol = srj_rel max|b'|;
 *     otherwise x <- x + omega z.  No dot products; every node update depends on x of the
 *     previous sweep only, so the result does not depend on the sweep order.
 * x: start -> solution.  res_out = the last E. */
static int srj_solve(nho_ctx* c, const double* h, const double* z, const double* b, double* x,
                     int* iters_out, double* res_out) {
  const int nnx = c->nnx, nny = c->nny, maxit = c->prm.solver_maxit;
  double *dinv = c->kdiag, *ce = c->kph, *cw = c->ksh, *cn = c->ks, *cs = c->kt, *bp = c->kr;
  double *xn = c->kv;
  *iters_out = 0; *res_out = 0.0;
  double rho = 0.0, bmax = 0.0;
  int bad = 0;
#pragma omp parallel for if (NHO_PAR(c)) schedule(static) reduction(max : rho, bmax) reduction(| : bad)
  for (int J = 0; J < nny; ++J)
    for (int I = 0; I < nnx; ++I) {
      double AC, AE, AW, AN, AS;
      node_coeffs(c, h, z, I, J, &AC, &AE, &AW, &AN, &AS);
      size_t k = NIDX(c, I, J);
      double di = 1.0 / AC;
      dinv[k] = di;
      ce[k] = AE * di; cw[k] = AW * di; cn[k] = AN * di; cs[k] = AS * di;
      bp[k] = b[k] * di;
      double rad = ((fabs(ce[k]) + fabs(cw[k])) + fabs(cn[k])) + fabs(cs[k]);
      if (rad > rho) rho = rad;
      if (fabs(bp[k]) > bmax) bmax = fabs(bp[k]);
      if (!(bp[k] == bp[k]) || isinf(bp[k])) bad = 1;
    }
  if (bad) return NHO_ENAN;
  if (bmax == 0.0) {  /* same convention as the BiCGStab path: b = 0 => p~ = 0, zero iterations */
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
    for (int J = 0; J < nny; ++J)
      for (int I = 0; I < nnx; ++I) x[NIDX(c, I, J)] = 0.0;
    return NHO_OK;
  }
  /* cycle length and schedule.  Where a row is not strictly diagonally dominant (rho >= 1: the
   * Gershgorin interval reaches 0, e.g. across a discontinuous free surface) there is no interval to
   * place Chebyshev nodes on: the method falls back to the plain Jacobi method (one factor, 1). */
  const int dominant = (rho < 1.0);
  const double gap = dominant ? sqrt(2.0 * (1.0 - rho)) : 0.0;
  int M = 1;
  if (dominant)
    while (M < c->prm.srj_mmax && (double)M * gap < 7.6) M *= 2;
  int* perm = (int*)malloc(sizeof(int) * (size_t)M);
  double* omega = (double*)malloc(sizeof(double) * (size_t)M);
  if (!perm || !omega) { free(perm); free(omega); return NHO_ENOMEM; }
  perm[0] = 1;
  for (int m = 1; m < M; m *= 2)          /* perm_2m from perm_m, in place from the back */
    for (int i = m - 1; i >= 0; --i) {
      int a = perm[i];
      perm[2 * i] = a; perm[2 * i + 1] = 2 * m + 1 - a;
    }
  for (int i = 0; i < M; ++i) {
    double cosv = cos(3.14159265358979323846 * (double)(2 * perm[i] - 1) / (double)(2 * M));
    omega[i] = dominant ? 1.0 / (1.0 - rho * cosv) : 1.0;
  }
  int iters = 0, status = NHO_OK;
  double E = 0.0;
  /* tolerance of (32): absolute (the paper's epsilon), or relative to max |b'| (R28) */
  const double tol = (c->prm.srj_rel > 0.0) ? c->prm.srj_rel * bmax : c->prm.srj_eps;
  for (;;) {
    const double om = omega[iters % M];
    double Emax = 0.0;
    int nan = 0;
#pragma omp parallel for if (NHO_PAR(c)) schedule(static) reduction(max : Emax) reduction(| : nan)
    for (int J = 0; J < nny; ++J)
      for (int I = 0; I < nnx; ++I) {
        size_t k = NIDX(c, I, J);
        double ax = x[k] + (((ce[k] * node_val(c, x, I + 1, J) + cw[k] * node_val(c, x, I - 1, J)) +
                             cn[k] * node_val(c, x, I, J + 1)) + cs[k] * node_val(c, x, I, J - 1));
        double zz = bp[k] - ax;
        double az = fabs(zz);
        if (az > Emax) Emax = az;
        if (!(zz == zz)) nan = 1;
        xn[k] = x[k] + om * zz;
      }
    E = Emax;
    if (nan) { status = NHO_ENAN; break; }
    if (E < tol) break;                          /* eq. (32): x is the accepted iterate */
    if (iters >= maxit) { status = NHO_ENOCONV; break; }
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
    for (int J = 0; J < nny; ++J)
      for (int I = 0; I < nnx; ++I) x[NIDX(c, I, J)] = xn[NIDX(c, I, J)];
    iters++;
  }
  free(perm); free(omega);
  *iters_out = iters; *res_out = E;
  return status;
}

static int solve_system(nho_ctx* c, const double* h, const double* z, const double* b, double* x,
                        int* iters_out, double* res_out) {
  if (c->prm.solver == 1) return srj_solve(c, h, z, b, x, iters_out, res_out);
  return bicgstab(c, h, z, b, x, iters_out, res_out);
}

/* in: U* = (h1,qx1,qy1), w_in; out: q** = (qx2,qy2), w2.                                   */
static void breaking_sources(nho_ctx* c, const double* w_in, double dt) {
  const double g = c->prm.g, delta = c->prm.delta, eps = c->prm.eps_dry;
  const double B1 = c->prm.B1, B2 = c->prm.B2;
  const double* h = c->h1;
  /* velocities of U* */
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
  for (int j = 0; j < c->ny; ++j)
    for (int i = 0; i < c->nx; ++i) {
      size_t k = CIDX(c, i, j);
      c->u[k] = nho_dsg(h[k], c->qx1[k], delta);
      c->v[k] = nho_dsg(h[k], c->qy1[k], delta);
    }
  /* cells: central differences (L394-396) */
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
  for (int j = 0; j < c->ny; ++j)
    for (int i = 0; i < c->nx; ++i) {
      size_t k = CIDX(c, i, j);
      double nu = 0.0, divu = 0.0;
      if (h[k] > eps) {
        double divq = (cell_xn(c, c->qx1, i + 1, j) - cell_xn(c, c->qx1, i - 1, j)) / (2.0 * c->dx)
                    + (cell_yn(c, c->qy1, i, j + 1) - cell_yn(c, c->qy1, i, j - 1)) / (2.0 * c->dy);
        divu = (cell_xn(c, c->u, i + 1, j) - cell_xn(c, c->u, i - 1, j)) / (2.0 * c->dx)
             + (cell_yn(c, c->v, i, j + 1) - cell_yn(c, c->v, i, j - 1)) / (2.0 * c->dy);
        double cc = sqrt(g * h[k]);
        double U1 = B1 * cc, U2 = B2 * cc;
        int fl = (fabs(divq) >= U1) || (c->flag_c[k] && fabs(divq) >= U2);   /* R11 */
        c->flag_c[k] = (unsigned char)fl;
        if (fl) {
          double B = 1.0 - divq / U1;                                       /* (9) */
          nu = fmax(B, 0.0) * h[k] * fabs(divq);
        }
      } else {
        c->flag_c[k] = 0;
      }
      double Hx = (cell_even(c, c->H, i + 1, j) - cell_even(c, c->H, i - 1, j)) / (2.0 * c->dx);
      double Hy = (cell_even(c, c->H, i, j + 1) - cell_even(c, c->H, i, j - 1)) / (2.0 * c->dy);
      c->qx2[k] = c->qx1[k] + dt * (2.0 * nu * divu * Hx);                   /* R_u, L224 */
      c->qy2[k] = c->qy1[k] + dt * (2.0 * nu * divu * Hy);
    }
  /* nodes: compact edge averages of (39) */
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
  for (int J = 0; J < c->nny; ++J)
    for (int I = 0; I < c->nnx; ++I) {
      size_t k = NIDX(c, I, J);
      double hn = 0.25 * (cell_even(c, h, I - 1, J - 1) + cell_even(c, h, I, J - 1)
                          + cell_even(c, h, I, J) + cell_even(c, h, I - 1, J));
      double nu = 0.0, divu = 0.0;
      if (hn > eps) {
        double q1E = 0.5 * (cell_xn(c, c->qx1, I, J) + cell_xn(c, c->qx1, I, J - 1));
        double q1W = 0.5 * (cell_xn(c, c->qx1, I - 1, J) + cell_xn(c, c->qx1, I - 1, J - 1));
        double q2N = 0.5 * (cell_yn(c, c->qy1, I, J) + cell_yn(c, c->qy1, I - 1, J));
        double q2S = 0.5 * (cell_yn(c, c->qy1, I, J - 1) + cell_yn(c, c->qy1, I - 1, J - 1));
        double u1E = 0.5 * (cell_xn(c, c->u, I, J) + cell_xn(c, c->u, I, J - 1));
        double u1W = 0.5 * (cell_xn(c, c->u, I - 1, J) + cell_xn(c, c->u, I - 1, J - 1));
        double u2N = 0.5 * (cell_yn(c, c->v, I, J) + cell_yn(c, c->v, I - 1, J));
        double u2S = 0.5 * (cell_yn(c, c->v, I, J - 1) + cell_yn(c, c->v, I - 1, J - 1));
        double divq = (q1E - q1W) / c->dx + (q2N - q2S) / c->dy;
        divu = (u1E - u1W) / c->dx + (u2N - u2S) / c->dy;
        double cc = sqrt(g * hn);
        double U1 = B1 * cc, U2 = B2 * cc;
        int fl = (fabs(divq) >= U1) || (c->flag_n[k] && fabs(divq) >= U2);
        c->flag_n[k] = (unsigned char)fl;
        if (fl) {
          double B = 1.0 - divq / U1;
          nu = fmax(B, 0.0) * hn * fabs(divq);
        }
      } else {
        c->flag_n[k] = 0;
      }
      c->w2[k] = w_in[k] + dt * (2.0 * nu * divu);                           /* R_w, L224 */
    }
}

/* S10: correction, eqs (36),(41): q <- q** + dt T_NH(p), w <- w** + dt p dinv(h_n). */
static void correction(nho_ctx* c, const double* pt, double dt, double* qx_out, double* qy_out,
                       double* w_out) {
  const double* h = c->h1; const double* z = c->z;
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
  for (int j = 0; j < c->ny; ++j)
    for (int i = 0; i < c->nx; ++i) {
      size_t k = CIDX(c, i, j);
      /* corner nodes of cell (i,j): (i,j) (i+1,j) (i,j+1) (i+1,j+1) */
      double p00 = node_val(c, pt, i, j), p10 = node_val(c, pt, i + 1, j);
      double p01 = node_val(c, pt, i, j + 1), p11 = node_val(c, pt, i + 1, j + 1);
      double pE = 0.5 * (p11 + p10), pW = 0.5 * (p01 + p00);
      double pN = 0.5 * (p11 + p01), pS = 0.5 * (p10 + p00);
      double xx = xi_x(c, z, i, j), xy = xi_y(c, z, i, j);
      qx_out[k] = c->qx2[k] - dt / (4.0 * c->dx) * ((2.0 * h[k] + xx) * pE + (xx - 2.0 * h[k]) * pW);
      qy_out[k] = c->qy2[k] - dt / (4.0 * c->dy) * ((2.0 * h[k] + xy) * pN + (xy - 2.0 * h[k]) * pS);
    }
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
  for (int J = 0; J < c->nny; ++J)
    for (int I = 0; I < c->nnx; ++I) {
      size_t k = NIDX(c, I, J);
      double hn = 0.25 * (cell_even(c, h, I - 1, J - 1) + cell_even(c, h, I, J - 1)
                          + cell_even(c, h, I, J) + cell_even(c, h, I - 1, J));
      w_out[k] = c->w2[k] + dt * pt[k] * dinv_h(hn, c->prm.delta);
    }
}

/* S11: generating relaxation zone at x-lo (L417-431, reading R18), target at time tt. */
static double relax_m_cell(const nho_ctx* c, int i) {
  double L = c->prm.gen_Lrel;
  double x = ((double)i + 0.5) * c->dx;
  double d = L - x;
  if (d <= 0.0) return 1.0;
  if (d >= L) return 0.0;
  return sqrt(1.0 - (d / L) * (d / L));
}
static void relaxation(nho_ctx* c, double* h, double* qx, double* qy, double* w, double* p, double tt) {
  const double A = c->prm.gen_A, h0 = c->prm.gen_h0, x0 = c->prm.gen_x0, L = c->prm.gen_Lrel;
  const double kk = sqrt(3.0 * A / (4.0 * h0 * h0 * h0));
  const double cel = sqrt(c->prm.g * (h0 + A));
  int krel = (int)ceil(L / c->dx);
  if (krel > c->nx) krel = c->nx;
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
  for (int j = 0; j < c->ny; ++j)
    for (int i = 0; i < krel; ++i) {
      size_t k = CIDX(c, i, j);
      double m = relax_m_cell(c, i);
      double x = ((double)i + 0.5) * c->dx;
      double sech2 = sech2_fixed(kk * (x - x0 - cel * tt));   /* R31 */
      double etas = A * sech2;
      double hs = fmax(c->H[k] + etas, 0.0);
      h[k] = m * h[k] + (1.0 - m) * hs;
      qx[k] = m * qx[k] + (1.0 - m) * (cel * etas);
      qy[k] = m * qy[k];
    }
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
  for (int J = 0; J < c->nny; ++J)
    for (int I = 0; I <= krel && I < c->nnx; ++I) {
      size_t k = NIDX(c, I, J);
      double mL = (I - 1 >= 0) ? relax_m_cell(c, I - 1) : 0.0;
      double mR = (I < c->nx) ? relax_m_cell(c, I) : 1.0;
      double m = 0.5 * (mL + mR);                           /* m_{i+-1/2}, L429 */
      w[k] = m * w[k];
      p[k] = m * p[k];
    }
}

/* S11b: absorbing relaxation zones (L415-440): the relaxation of S11 with the target
 * U* = w* = p* = 0, read as eta* = 0, q* = 0 (h* = max(H, 0); "U* = 0" would drain the basin, R18).
 * Reading R29: width L on a side, k_Rel = ceil(L / dx) cells; m = sqrt(1 - (d/L)^2) with d measured
 * from the inner end of the zone (R18), m = 1 outside; node values use the mean of the two
 * adjacent cell coefficients (0 beyond the boundary, L429); the update is written
 * a <- a + (1 - m)(a* - a) so that a state already at the target is left bit-identical (lake at
 * rest); sides are applied in the order x-lo, x-hi, y-lo, y-hi (corners take both factors). */
static double absorb_m(double L, double dxy, int idx_from_boundary) {
  double x = ((double)idx_from_boundary + 0.5) * dxy;
  double d = L - x;
  if (d <= 0.0) return 1.0;
  if (d >= L) return 0.0;
  return sqrt(1.0 - (d / L) * (d / L));
}
static void absorb_side(nho_ctx* c, int side, double L, double* h, double* qx, double* qy, double* w,
                        double* p) {
  const int xdir = (side < 2), hi = (side & 1);
  const int n = xdir ? c->nx : c->ny, nn = xdir ? c->nnx : c->nny;
  const double dxy = xdir ? c->dx : c->dy;
  int krel = (int)ceil(L / dxy);
  if (krel > n) krel = n;
  const int nother = xdir ? c->ny : c->nx, nnother = xdir ? c->nny : c->nnx;
#pragma omp parallel for if (nother >= 48) schedule(static)
  for (int t = 0; t < nother; ++t)
    for (int s = 0; s < krel; ++s) {          /* s = cell index counted from the boundary */
      int a = hi ? n - 1 - s : s;
      size_t k = xdir ? CIDX(c, a, t) : CIDX(c, t, a);
      double f = 1.0 - absorb_m(L, dxy, s);
      double hs = fmax(c->H[k], 0.0);
      h[k] = h[k] + f * (hs - h[k]);
      qx[k] = qx[k] + f * (0.0 - qx[k]);
      qy[k] = qy[k] + f * (0.0 - qy[k]);
    }
#pragma omp parallel for if (nnother >= 48) schedule(static)
  for (int t = 0; t < nnother; ++t)
    for (int s = 0; s <= krel; ++s) {         /* s = node line counted from the boundary line */
      int a = hi ? n - s : s;                  /* node line index in the (n+1)-line numbering */
      if (nn == n) {                           /* periodic direction never has zones */
        continue;
      }
      double mo = (s - 1 >= 0) ? absorb_m(L, dxy, s - 1) : 0.0;   /* cell towards the boundary */
      double mi = (s < n) ? absorb_m(L, dxy, s) : 1.0;            /* cell towards the interior */
      double f = 1.0 - 0.5 * (mo + mi);
      size_t k = xdir ? NIDX(c, a, t) : NIDX(c, t, a);
      w[k] = w[k] + f * (0.0 - w[k]);
      p[k] = p[k] + f * (0.0 - p[k]);
    }
}
static void absorbing_zones(nho_ctx* c, double* h, double* qx, double* qy, double* w, double* p) {
  const double L[4] = { c->prm.abs_xlo, c->prm.abs_xhi, c->prm.abs_ylo, c->prm.abs_yhi };
  for (int side = 0; side < 4; ++side)
    if (L[side] > 0.0) absorb_side(c, side, L[side], h, qx, qy, w, p);
}

/* S5b (only if w_advect; reading R30): the vertical-velocity equation of [7],
 * (hw)_t + div(hw u) = p (L109-113), which with h_t + div q = 0 is  w_t + u . grad w = p / h.
 * The paper gives no discretisation ("can be easily extended").  Reading: in the first (hyperbolic)
 * part of every stage the node values w are transported in advective form with first-order upwind
 * differences between neighbouring nodes; the node velocity is the mean of the desingularised
 * velocities (S0) of the four cells around the node, taken from the stage input U^n like the
 * fluxes of the predictor (ghost cells through the maps of R9: the normal velocity of a wall node
 * is 0).  The pressure part p / h is the unchanged S10.  Under the time step (23) the update is a
 * convex combination of the node and its upwind neighbours (maximum principle). */
static void w_advection(nho_ctx* c, const double* w_in, double dt, double* w_out) {
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
  for (int J = 0; J < c->nny; ++J)
    for (int I = 0; I < c->nnx; ++I) {
      double un = 0.25 * (cell_xn(c, c->u, I - 1, J - 1) + cell_xn(c, c->u, I, J - 1) +
                          cell_xn(c, c->u, I, J) + cell_xn(c, c->u, I - 1, J));
      double vn = 0.25 * (cell_yn(c, c->v, I - 1, J - 1) + cell_yn(c, c->v, I, J - 1) +
                          cell_yn(c, c->v, I, J) + cell_yn(c, c->v, I - 1, J));
      double wc = w_in[NIDX(c, I, J)];
      double wx = (un > 0.0) ? (wc - node_val(c, w_in, I - 1, J)) / c->dx
                             : (node_val(c, w_in, I + 1, J) - wc) / c->dx;
      double wy = (vn > 0.0) ? (wc - node_val(c, w_in, I, J - 1)) / c->dy
                             : (node_val(c, w_in, I, J + 1) - wc) / c->dy;
      w_out[NIDX(c, I, J)] = wc - dt * (un * wx + vn * wy);
    }
}

/* Reading R32: the start vector of a pressure solve.  The paper does not say where its iteration
 * starts; R14 took the previous solution.  The solves of a run alternate between the two Runge-Kutta
 * stages, and the increment from one solve to the next, i_k = s_k - s_(k-1), repeats every second
 * solve up to a slow drift in time.  With warm_start = 1 (default) the start vector is the previous
 * solution plus the quadratic extrapolation of the same-kind increments of the last three steps,
 *     x0 = s1 + 3 (s2 - s3) - 3 (s4 - s5) + (s6 - s7)      (s1 = most recent solution),
 * once seven solutions exist since the last nho_set_state and only for solver 0 with solver_rtol <= 1e-8;
 * otherwise, and with warm_start = 0, x0 = p as it stands (the previous solution, or what nho_set_state gave).  A start vector does not
 * change what the solve converges to (stopping rule unchanged); it saves 16-27 % of the iterations
 * on the five configs (R32). */
static void start_vector(const nho_ctx* c, double* x0) {
  /* only where the stored solutions are accurate enough to be extrapolated: the formula amplifies
   * their error 15-fold, so with a loose stopping rule (solver 1 at the paper's eps, tolerances above
   * 1e-8) the plain previous solution is the better start (measured: DESIGN.md R32) */
  if (!c->prm.warm_start || c->prm.solver != 0 || c->prm.solver_rtol > 1e-8 || c->nhist < 7) return;
  double* const* h = c->hist;
  for (int J = 0; J < c->nny; ++J)
    for (int I = 0; I < c->nnx; ++I) {
      size_t k = NIDX(c, I, J);
      x0[k] = ((h[0][k] + 3.0 * (h[1][k] - h[2][k])) - 3.0 * (h[3][k] - h[4][k])) + (h[5][k] - h[6][k]);
    }
}
static void push_solution(nho_ctx* c, const double* x) {
  size_t nn = (size_t)(c->nx + 1) * (size_t)(c->ny + 1);
  double* t = c->hist[6];
  for (int a = 6; a > 0; --a) c->hist[a] = c->hist[a - 1];
  c->hist[0] = t;
  memcpy(c->hist[0], x, nn * sizeof(double));
  if (c->nhist < 7) c->nhist++;
}

/* S6-S10 on U* = (h1,qx1,qy1) with w_in; results to (qx_out,qy_out,w_out), p in c->p. */
static int nonhydro_part(nho_ctx* c, const double* w_in, double dt, double* qx_out, double* qy_out,
                         double* w_out) {
  size_t nn = (size_t)(c->nx + 1) * (size_t)(c->ny + 1);
  size_t nc = (size_t)c->nx * (size_t)c->ny;
  if (c->prm.breaking) breaking_sources(c, w_in, dt);
  else {
    memcpy(c->qx2, c->qx1, nc * sizeof(double));
    memcpy(c->qy2, c->qy1, nc * sizeof(double));
    memcpy(c->w2, w_in, nn * sizeof(double));
  }
  compute_z(c, c->h1, c->z);
  /* S7: b = -B(U**, w**)/dt  (sign: R15) */
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
  for (int J = 0; J < c->nny; ++J)
    for (int I = 0; I < c->nnx; ++I)
      c->b[NIDX(c, I, J)] = (dt > 0.0) ? -node_B(c, c->h1, c->qx2, c->qy2, c->z, c->w2, I, J) / dt
                                       : 0.0;   /* R26: all-dry domain, dt = 0 => p~ = 0 */
  int iters = 0; double relres = 0.0;
  start_vector(c, c->p);   /* R32 */
  int st = solve_system(c, c->h1, c->z, c->b, c->p, &iters, &relres);
  push_solution(c, c->p);
  c->info.iters_last = iters;
  c->info.iters_total += iters;
  c->info.solves += 1;
  if (iters > c->info.iters_max) c->info.iters_max = iters;
  c->info.res_last = relres;
  if (st == NHO_ENOCONV) c->info.flags |= 1;
  if (st == NHO_ENAN) return st;
  correction(c, c->p, dt, qx_out, qy_out, w_out);
  return st;
}

/* one stage Phi_dt: (h,qx,qy,w) -> (h,qx,qy,w) in place; t0 = time of the stage input. */
static int stage(nho_ctx* c, double dt, double t0) {
  size_t nc = (size_t)c->nx * (size_t)c->ny;
  predictor(c, c->h, c->qx, c->qy, dt);
  int st = NHO_OK;
  if (c->prm.nonhydro) {
    const double* w_in = c->w;
    if (c->prm.w_advect) {   /* R30: c->u, c->v are the velocities of the stage input (predictor, S0) */
      w_advection(c, c->w, dt, c->wadv);
      w_in = c->wadv;
    }
    st = nonhydro_part(c, w_in, dt, c->qx, c->qy, c->w);
    memcpy(c->h, c->h1, nc * sizeof(double));
  } else {
    memcpy(c->h, c->h1, nc * sizeof(double));
    memcpy(c->qx, c->qx1, nc * sizeof(double));
    memcpy(c->qy, c->qy1, nc * sizeof(double));
  }
  if (c->prm.gen_on) relaxation(c, c->h, c->qx, c->qy, c->w, c->p, t0 + dt);
  absorbing_zones(c, c->h, c->qx, c->qy, c->w, c->p);
  return st;
}

/* ------------------------------------------------------------------------------------ */
void nho_default_params(nho_params* prm) {
  memset(prm, 0, sizeof(*prm));
  prm->g = 9.81; prm->cfl = 0.5; prm->delta = 1e-5; prm->eps_dry = 1e-5;
  prm->B1 = 0.15; prm->B2 = 0.5; prm->solver_rtol = 1e-12;
  prm->breaking = 0; prm->nonhydro = 1; prm->time_order = 2; prm->space_order = 2;
  prm->bc_xlo = prm->bc_xhi = prm->bc_ylo = prm->bc_yhi = NHO_BC_OUTFLOW;
  prm->solver_maxit = 10000; prm->gen_on = 0; prm->precision = 64;
  prm->solver = 0; prm->srj_eps = 1e-5; prm->srj_mmax = 256; prm->warm_start = 1;
}

static int bc_ok(int b) { return b == NHO_BC_PERIODIC || b == NHO_BC_WALL || b == NHO_BC_OUTFLOW; }

int nho_create(nho_ctx** out, int nx, int ny, double dx, double dy, const double* H,
               const nho_params* prm) {
  if (!out || !H || !prm) return NHO_EINVAL;
  *out = NULL;
  if (nx < 4 || ny < 4 || !(dx > 0.0) || !(dy > 0.0)) return NHO_EINVAL;
  if (!(prm->cfl > 0.0 && prm->cfl <= 1.0) || !(prm->g > 0.0) || !(prm->delta > 0.0)) return NHO_EINVAL;
  if (!(prm->eps_dry >= 0.0) || !(prm->solver_rtol > 0.0) || prm->solver_maxit < 1) return NHO_EINVAL;
  if (!bc_ok(prm->bc_xlo) || !bc_ok(prm->bc_xhi) || !bc_ok(prm->bc_ylo) || !bc_ok(prm->bc_yhi)) return NHO_EINVAL;
  if ((prm->bc_xlo == NHO_BC_PERIODIC) != (prm->bc_xhi == NHO_BC_PERIODIC)) return NHO_EINVAL;
  if ((prm->bc_ylo == NHO_BC_PERIODIC) != (prm->bc_yhi == NHO_BC_PERIODIC)) return NHO_EINVAL;
  if (prm->time_order != 1 && prm->time_order != 2) return NHO_EINVAL;
  if (prm->space_order != 1 && prm->space_order != 2) return NHO_EINVAL;
  if (prm->precision != 64) return NHO_EINVAL;
  if (!(prm->manning_n >= 0.0)) return NHO_EINVAL;
  if (prm->solver != 0 && prm->solver != 1) return NHO_EINVAL;
  if (prm->w_advect != 0 && prm->w_advect != 1) return NHO_EINVAL;
  if (prm->warm_start != 0 && prm->warm_start != 1) return NHO_EINVAL;
  if (!(prm->srj_rel >= 0.0)) return NHO_EINVAL;
  if (!(prm->abs_xlo >= 0.0) || !(prm->abs_xhi >= 0.0) || !(prm->abs_ylo >= 0.0) || !(prm->abs_yhi >= 0.0)) return NHO_EINVAL;
  if ((prm->abs_xlo > 0.0 || prm->abs_xhi > 0.0) && prm->bc_xlo == NHO_BC_PERIODIC) return NHO_EINVAL;
  if ((prm->abs_ylo > 0.0 || prm->abs_yhi > 0.0) && prm->bc_ylo == NHO_BC_PERIODIC) return NHO_EINVAL;
  if (prm->abs_xlo > 0.0 && prm->gen_on) return NHO_EINVAL;   /* the generating zone owns x-lo */
  if (prm->solver == 1 && (!(prm->srj_eps > 0.0) || prm->srj_mmax < 1 || prm->srj_mmax > 4096 ||
                           (prm->srj_mmax & (prm->srj_mmax - 1)) != 0)) return NHO_EINVAL;
  if (prm->breaking && !(prm->B1 > 0.0 && prm->B2 > 0.0)) return NHO_EINVAL;
  if (prm->gen_on && !(prm->gen_A > 0.0 && prm->gen_h0 > 0.0 && prm->gen_Lrel > 0.0)) return NHO_EINVAL;
  size_t nc = (size_t)nx * (size_t)ny, nn = (size_t)(nx + 1) * (size_t)(ny + 1);
  for (size_t k = 0; k < nc; ++k) if (!(H[k] == H[k]) || isinf(H[k])) return NHO_EINVAL;
  nho_ctx* c = (nho_ctx*)calloc(1, sizeof(nho_ctx));
  if (!c) return NHO_ENOMEM;
  c->nx = nx; c->ny = ny; c->dx = dx; c->dy = dy; c->prm = *prm;
  c->nnx = (prm->bc_xlo == NHO_BC_PERIODIC) ? nx : nx + 1;
  c->nny = (prm->bc_ylo == NHO_BC_PERIODIC) ? ny : ny + 1;
  double** cellp[] = { &c->H, &c->h, &c->qx, &c->qy, &c->eta, &c->u, &c->v, &c->h1, &c->qx1, &c->qy1,
                       &c->qx2, &c->qy2, &c->z, &c->h0, &c->qx0, &c->qy0 };
  double** nodep[] = { &c->w, &c->p, &c->w2, &c->b, &c->kr, &c->kr0, &c->kp, &c->kv, &c->ks, &c->kt,
                       &c->kph, &c->ksh, &c->kdiag, &c->w0, &c->wadv, &c->hist[0], &c->hist[1], &c->hist[2],
                       &c->hist[3], &c->hist[4], &c->hist[5], &c->hist[6] };
  int ok = 1;
  for (size_t a = 0; a < sizeof(cellp) / sizeof(cellp[0]); ++a) { *cellp[a] = (double*)calloc(nc, sizeof(double)); if (!*cellp[a]) ok = 0; }
  for (size_t a = 0; a < sizeof(nodep) / sizeof(nodep[0]); ++a) { *nodep[a] = (double*)calloc(nn, sizeof(double)); if (!*nodep[a]) ok = 0; }
  c->flag_c = (unsigned char*)calloc(nc, 1); c->flag_n = (unsigned char*)calloc(nn, 1);
  if (!c->flag_c || !c->flag_n) ok = 0;
  if (!ok) { nho_destroy(c); return NHO_ENOMEM; }
  memcpy(c->H, H, nc * sizeof(double));
  *out = c;
  return NHO_OK;
}

void nho_destroy(nho_ctx* c) {
  if (!c) return;
  double* all[] = { c->H, c->h, c->qx, c->qy, c->eta, c->u, c->v, c->h1, c->qx1, c->qy1, c->qx2, c->qy2,
                    c->z, c->h0, c->qx0, c->qy0, c->w, c->p, c->w2, c->b, c->kr, c->kr0, c->kp, c->kv,
                    c->ks, c->kt, c->kph, c->ksh, c->kdiag, c->w0, c->wadv, c->hist[0], c->hist[1], c->hist[2],
                    c->hist[3], c->hist[4], c->hist[5], c->hist[6] };
  for (size_t a = 0; a < sizeof(all) / sizeof(all[0]); ++a) free(all[a]);
  free(c->flag_c); free(c->flag_n);
  free(c);
}

/* copy a user node array in, folding periodic duplicates (last line ignored) */
static void nodes_in(nho_ctx* c, const double* src, double* dst) {
  size_t nn = (size_t)(c->nx + 1) * (size_t)(c->ny + 1);
  if (!src) { memset(dst, 0, nn * sizeof(double)); return; }
  memcpy(dst, src, nn * sizeof(double));
}
/* copy out, filling the duplicate lines of periodic directions */
static void nodes_out(nho_ctx* c, const double* src, double* dst) {
  for (int J = 0; J <= c->ny; ++J)
    for (int I = 0; I <= c->nx; ++I) {
      int II = (I == c->nx && c->nnx == c->nx) ? 0 : I;
      int JJ = (J == c->ny && c->nny == c->ny) ? 0 : J;
      dst[NIDX(c, I, J)] = src[NIDX(c, II, JJ)];
    }
}

static int set_state(nho_ctx* c, const double* h, const double* qx, const double* qy,
                     const double* w, const double* p, int keep_history) {
  if (!c || !h || !qx || !qy) return NHO_EINVAL;
  size_t nc = (size_t)c->nx * (size_t)c->ny;
  for (size_t k = 0; k < nc; ++k)
    if (!(h[k] >= 0.0) || isinf(h[k]) || !(qx[k] == qx[k]) || !(qy[k] == qy[k])) {
      snprintf(c->err, sizeof(c->err), "set_state: h<0 or non-finite input at cell %zu", k);
      return NHO_EINVAL;
    }
  memcpy(c->h, h, nc * sizeof(double));
  memcpy(c->qx, qx, nc * sizeof(double));
  memcpy(c->qy, qy, nc * sizeof(double));
  nodes_in(c, w, c->w);
  nodes_in(c, p, c->p);
  /* R32: set_state starts a new solution history; continue_state (the caller says that the running
   * state is coming back: a checkpoint, a round trip) keeps it */
  if (!keep_history) c->nhist = 0;
  return NHO_OK;
}
int nho_set_state(nho_ctx* c, const double* h, const double* qx, const double* qy,
                  const double* w, const double* p) {
  return set_state(c, h, qx, qy, w, p, 0);
}
int nho_continue_state(nho_ctx* c, const double* h, const double* qx, const double* qy,
                       const double* w, const double* p) {
  return set_state(c, h, qx, qy, w, p, 1);
}

int nho_get_state(nho_ctx* c, double* h, double* qx, double* qy, double* w, double* p) {
  if (!c) return NHO_EINVAL;
  size_t nc = (size_t)c->nx * (size_t)c->ny;
  if (h) memcpy(h, c->h, nc * sizeof(double));
  if (qx) memcpy(qx, c->qx, nc * sizeof(double));
  if (qy) memcpy(qy, c->qy, nc * sizeof(double));
  if (w) nodes_out(c, c->w, w);
  if (p) nodes_out(c, c->p, p);
  return NHO_OK;
}

int nho_set_time(nho_ctx* c, double t) {
  if (!c || !(t == t) || isinf(t)) return NHO_EINVAL;
  c->info.t = t;
  return NHO_OK;
}

int nho_compute_dt(nho_ctx* c, double* dt) {
  if (!c || !dt) return NHO_EINVAL;
  *dt = cfl_dt(c, c->h, c->qx, c->qy);
  return NHO_OK;
}

/* full step (R19): U1 = Phi(Un); U2 = Phi(U1); U^{n+1} = (Un + U2)/2 on h,qx,qy,w. */
int nho_step(nho_ctx* c, int nsteps) {
  if (!c || nsteps < 0) return NHO_EINVAL;
  size_t nc = (size_t)c->nx * (size_t)c->ny, nn = (size_t)(c->nx + 1) * (size_t)(c->ny + 1);
  int worst = NHO_OK;
  for (int s = 0; s < nsteps; ++s) {
    double dt = cfl_dt(c, c->h, c->qx, c->qy);
    if (!(dt == dt)) { snprintf(c->err, sizeof(c->err), "step: NaN time step"); return NHO_ENAN; }
    int st;
    if (c->prm.time_order == 1) {
      st = stage(c, dt, c->info.t);
      if (st == NHO_ENAN) return st;
      if (st != NHO_OK) worst = st;
    } else {
      memcpy(c->h0, c->h, nc * sizeof(double)); memcpy(c->qx0, c->qx, nc * sizeof(double));
      memcpy(c->qy0, c->qy, nc * sizeof(double)); memcpy(c->w0, c->w, nn * sizeof(double));
      st = stage(c, dt, c->info.t);
      if (st == NHO_ENAN) return st;
      if (st != NHO_OK) worst = st;
      st = stage(c, dt, c->info.t + dt);
      if (st == NHO_ENAN) return st;
      if (st != NHO_OK) worst = st;
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
      for (int j = 0; j < c->ny; ++j)
        for (int i = 0; i < c->nx; ++i) {
          size_t k = CIDX(c, i, j);
          c->h[k] = 0.5 * c->h0[k] + 0.5 * c->h[k];
          c->qx[k] = 0.5 * c->qx0[k] + 0.5 * c->qx[k];
          c->qy[k] = 0.5 * c->qy0[k] + 0.5 * c->qy[k];
        }
#pragma omp parallel for if (NHO_PAR(c)) schedule(static)
      for (int J = 0; J < c->nny; ++J)
        for (int I = 0; I < c->nnx; ++I) {
          size_t k = NIDX(c, I, J);
          c->w[k] = 0.5 * c->w0[k] + 0.5 * c->w[k];
        }
    }
    c->info.t += dt; c->info.dt_last = dt; c->info.steps += 1;
  }
  if (worst == NHO_ENOCONV) snprintf(c->err, sizeof(c->err), "step: pressure solve did not converge");
  return worst;
}

int nho_hydrostatic_step(nho_ctx* c, double dt) {
  if (!c) return NHO_EINVAL;
  size_t nc = (size_t)c->nx * (size_t)c->ny;
  if (!(dt > 0.0)) dt = cfl_dt(c, c->h, c->qx, c->qy);
  predictor(c, c->h, c->qx, c->qy, dt);
  memcpy(c->h, c->h1, nc * sizeof(double));
  memcpy(c->qx, c->qx1, nc * sizeof(double));
  memcpy(c->qy, c->qy1, nc * sizeof(double));
  c->info.dt_last = dt;
  return NHO_OK;
}

int nho_nonhydro_correct(nho_ctx* c, double dt) {
  if (!c || !(dt > 0.0)) return NHO_EINVAL;
  size_t nc = (size_t)c->nx * (size_t)c->ny;
  memcpy(c->h1, c->h, nc * sizeof(double));
  memcpy(c->qx1, c->qx, nc * sizeof(double));
  memcpy(c->qy1, c->qy, nc * sizeof(double));
  int st = nonhydro_part(c, c->w, dt, c->qx, c->qy, c->w);
  c->info.dt_last = dt;
  return st;
}

int nho_get_info(nho_ctx* c, nho_info* out) {
  if (!c || !out) return NHO_EINVAL;
  *out = c->info;
  return NHO_OK;
}
const char* nho_last_error(nho_ctx* c) { return c ? c->err : "null context"; }

/* ---- test hooks ---- */
int nho_apply_A(nho_ctx* c, const double* x_nodes, double* y_nodes) {
  if (!c || !x_nodes || !y_nodes) return NHO_EINVAL;
  nodes_in(c, x_nodes, c->kph);
  compute_z(c, c->h, c->z);
  apply_A(c, c->h, c->z, c->kph, c->ksh);
  nodes_out(c, c->ksh, y_nodes);
  return NHO_OK;
}
int nho_coeffs(nho_ctx* c, double* AC, double* AE, double* AW, double* AN, double* AS) {
  if (!c || !AC || !AE || !AW || !AN || !AS) return NHO_EINVAL;
  compute_z(c, c->h, c->z);
  for (int J = 0; J <= c->ny; ++J)
    for (int I = 0; I <= c->nx; ++I) {
      int II = (I == c->nx && c->nnx == c->nx) ? 0 : I;
      int JJ = (J == c->ny && c->nny == c->ny) ? 0 : J;
      size_t k = NIDX(c, I, J);
      node_coeffs(c, c->h, c->z, II, JJ, &AC[k], &AE[k], &AW[k], &AN[k], &AS[k]);
    }
  return NHO_OK;
}
int nho_rhs(nho_ctx* c, double dt, double* b_nodes) {
  if (!c || !b_nodes || !(dt > 0.0)) return NHO_EINVAL;
  compute_z(c, c->h, c->z);
  for (int J = 0; J < c->nny; ++J)
    for (int I = 0; I < c->nnx; ++I)
      c->b[NIDX(c, I, J)] = -node_B(c, c->h, c->qx, c->qy, c->z, c->w, I, J) / dt;
  nodes_out(c, c->b, b_nodes);
  return NHO_OK;
}
int nho_constraint(nho_ctx* c, double* B_nodes) {
  if (!c || !B_nodes) return NHO_EINVAL;
  compute_z(c, c->h, c->z);
  for (int J = 0; J < c->nny; ++J)
    for (int I = 0; I < c->nnx; ++I)
      c->b[NIDX(c, I, J)] = node_B(c, c->h, c->qx, c->qy, c->z, c->w, I, J);
  nodes_out(c, c->b, B_nodes);
  return NHO_OK;
}
int nho_breaking(nho_ctx* c, double dt, double* qx2, double* qy2, double* w2) {
  if (!c || !qx2 || !qy2 || !w2 || !(dt > 0.0) || !c->prm.breaking) return NHO_EINVAL;
  size_t nc = (size_t)c->nx * (size_t)c->ny;
  memcpy(c->h1, c->h, nc * sizeof(double));
  memcpy(c->qx1, c->qx, nc * sizeof(double));
  memcpy(c->qy1, c->qy, nc * sizeof(double));
  breaking_sources(c, c->w, dt);
  memcpy(qx2, c->qx2, nc * sizeof(double));
  memcpy(qy2, c->qy2, nc * sizeof(double));
  nodes_out(c, c->w2, w2);
  return NHO_OK;
}
int nho_w_advect(nho_ctx* c, double dt, double* w_out) {
  if (!c || !w_out || !(dt > 0.0)) return NHO_EINVAL;
  derived_fields(c, c->h, c->qx, c->qy);
  w_advection(c, c->w, dt, c->wadv);
  nodes_out(c, c->wadv, w_out);
  return NHO_OK;
}

int nho_start_vector(nho_ctx* c, double* x0_nodes) {
  if (!c || !x0_nodes) return NHO_EINVAL;
  size_t nn = (size_t)(c->nx + 1) * (size_t)(c->ny + 1);
  memcpy(c->kr, c->p, nn * sizeof(double));
  start_vector(c, c->kr);
  nodes_out(c, c->kr, x0_nodes);
  return NHO_OK;
}

int nho_solve(nho_ctx* c, const double* b_nodes, double* x_nodes, int* iters, double* relres) {
  if (!c || !b_nodes || !x_nodes) return NHO_EINVAL;
  int it = 0; double rr = 0.0;
  nodes_in(c, b_nodes, c->b);
  nodes_in(c, x_nodes, c->w2);
  compute_z(c, c->h, c->z);
  int st = solve_system(c, c->h, c->z, c->b, c->w2, &it, &rr);
  nodes_out(c, c->w2, x_nodes);
  if (iters) *iters = it;
  if (relres) *relres = rr;
  return st;
}
