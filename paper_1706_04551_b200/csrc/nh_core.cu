// nh_core.cu -- context, state, and the step driver behind the C ABI (nh_abi.cu dispatches here;
// compiled once per precision, nh_internal.cuh): sequences the kernels of nh_predictor.cu / nh_pressure.cu / nh_solver.cu on the
// context's stream.  Nothing here computes on the host: dt, the solver's convergence tests, the
// clock and all counters stay in device memory (NhScal) until nh_get_info / nh_sync read them.
//
// Step order (PAPER.md L524-544 and Fig. 4, repackaged):
//   dt = CFL / lam_max(U^n)                       (lam_max produced by the previous step's combine)
//   for each Runge-Kutta stage:  predictor -> [breaking] -> z, rhs, rows of A -> BiCGStab
//                                -> correction -> [relaxation zone]
//   U^{n+1} = (U^n + U^(2)) / 2  fused with lam_max(U^{n+1})
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "nh_internal.cuh"
#include "nh_core.h"

namespace NH_NS {
namespace {

__global__ void __launch_bounds__(256)
k_all_finite(size_t n, const double* __restrict__ a, int* bad) {
  bool b = false;
  for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n;
       k += (size_t)gridDim.x * blockDim.x) {
    double v = a[k];
    if (!(v == v) || isinf(v)) b = true;
  }
  if (__syncthreads_or(b) && threadIdx.x == 0) atomicOr(bad, 1);
}

__global__ void k_clear_flag(NhScal* sc, int mask) { sc->flags &= ~mask; }
// ---- fp32 variant: the user's arrays are fp64, the planes fp32 (conversion at set / get only) ----
__global__ void __launch_bounds__(256) k_to_real(size_t n, const double* __restrict__ a, real* __restrict__ b) {
  for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (size_t)gridDim.x * blockDim.x)
    b[k] = (real)a[k];
}
__global__ void __launch_bounds__(256) k_to_double(size_t n, const real* __restrict__ a, double* __restrict__ b) {
  for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (size_t)gridDim.x * blockDim.x)
    b[k] = (double)a[k];
}
// eta = h - H formed in fp64 from the user's h and the bathymetry as given, stored in fp32 beside
// h = H + eta (fp32 H); h < 0 or non-finite input raises the bad-state flag
__global__ void __launch_bounds__(256)
k_eta_in(size_t n, const double* __restrict__ hd, const double* __restrict__ Hd, const real* __restrict__ H,
         real* __restrict__ eta, real* __restrict__ h, NhScal* sc) {
  bool bad = false;
  for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (size_t)gridDim.x * blockDim.x) {
    double hv = hd[k];
    if (!(hv >= 0.0) || isinf(hv)) bad = true;
    real e = (hv == 0.0) ? -H[k] : (real)(hv - Hd[k]);   // a dry cell is exactly dry in fp32 too
    eta[k] = e;
    h[k] = fmax(H[k] + e, RC(0.0));
  }
  if (__syncthreads_or(bad) && threadIdx.x == 0) atomicOr(&sc->flags, NH_FLAG_BADSTATE);
}
__global__ void __launch_bounds__(256)
k_h_out(size_t n, const real* __restrict__ eta, const real* __restrict__ h, const double* __restrict__ Hd,
        double* __restrict__ out) {
  for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (size_t)gridDim.x * blockDim.x)
    out[k] = (h[k] == RC(0.0)) ? 0.0 : fmax(Hd[k] + (double)eta[k], 0.0);
}
__global__ void __launch_bounds__(256)
k_nodes_in(NhGrid G, const double* __restrict__ dense, real* __restrict__ plane) {
  int I = blockIdx.x * 32 + threadIdx.x, J = blockIdx.y * 8 + threadIdx.y;
  if (I >= G.nnx || J >= G.nny) return;
  plane[(size_t)J * G.np + I] = (real)dense[(size_t)J * (G.nx + 1) + I];
}
inline int grid1(const Ctx* c, size_t n) {
  size_t need = (n + 255) / 256, cap = (size_t)c->sm_count * 16;
  return (int)(need < cap ? (need ? need : 1) : cap);
}
__global__ void k_set_time(NhScal* sc, double t) { sc->t = t; }

bool bc_ok(int b) { return b == NH_BC_PERIODIC || b == NH_BC_WALL || b == NH_BC_OUTFLOW; }

int fail(Ctx* c, int code, const char* msg) {
  if (c) snprintf(c->err, sizeof(c->err), "%s", msg);
  return code;
}

template <typename T>
bool dalloc(Ctx* c, T** p, size_t count) {
  cudaError_t e = cudaMalloc((void**)p, count * sizeof(T));
  if (e != cudaSuccess) {
    *p = nullptr;
    snprintf(c->err, sizeof(c->err), "cudaMalloc(%zu bytes): %s", count * sizeof(T),
             cudaGetErrorString(e));
    (void)cudaGetLastError();
    return false;
  }
  c->raw.push_back((void*)*p);
  e = cudaMemsetAsync(*p, 0, count * sizeof(T), c->stream);
  return e == cudaSuccess;
}

// internal node plane (ghost ring, nh_internal.cuh): the handed-out pointer addresses node (0,0)
inline size_t node_origin(const Ctx* c) { return (size_t)NH_ROW_PAD * c->g.np + NH_COL_PAD; }
bool nalloc(Ctx* c, real** p) {
  real* base = nullptr;
  if (!dalloc(c, &base, c->nni)) { *p = nullptr; return false; }
  *p = base + node_origin(c);
  return true;
}

void free_all(Ctx* c) {
  for (void* p : c->raw) if (p) cudaFree(p);
  c->raw.clear();
  if (c->part) cudaFree(c->part);
  if (c->srj_cos) cudaFree(c->srj_cos);
  if (c->sc_host) cudaFreeHost(c->sc_host);
  for (int k = 0; k < NH_PROF_CATS; ++k)
    for (auto& ev : c->prof_ev[k]) { cudaEventDestroy(ev.first); cudaEventDestroy(ev.second); }
}

// copy in/out with cudaMemcpyDefault: the pointer may be host or device (UVA decides)
int copy_async(Ctx* c, void* dst, const void* src, size_t bytes) {
  cudaError_t e = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDefault, c->stream);
  if (e != cudaSuccess) {
    snprintf(c->err, sizeof(c->err), "cudaMemcpyAsync: %s", cudaGetErrorString(e));
    (void)cudaGetLastError();
    c->host_status = NH_ECUDA;
    return NH_ECUDA;
  }
  return NH_OK;
}

// cell array in / out: fp64 build: a plain copy; fp32 build: through the fp64 staging plane
int cell_in(Ctx* c, real* dst, const double* src_user) {
  if (!kEta) return copy_async(c, dst, src_user, c->nc * sizeof(double));
  if (copy_async(c, c->stage, src_user, c->nc * sizeof(double))) return NH_ECUDA;
  k_to_real<<<grid1(c, c->nc), 256, 0, c->stream>>>(c->nc, c->stage, dst);
  c->launches++;
  return NH_OK;
}
int cell_out(Ctx* c, double* dst_user, const real* src) {
  if (!kEta) return copy_async(c, dst_user, src, c->nc * sizeof(double));
  k_to_double<<<grid1(c, c->nc), 256, 0, c->stream>>>(c->nc, src, c->stage);
  c->launches++;
  return copy_async(c, dst_user, c->stage, c->nc * sizeof(double));
}

// public node array (dense (nx+1) x (ny+1), host or device) -> internal plane: the distinct lines
// only (a periodic duplicate line is ignored on input); NULL -> zeros
int node_in(Ctx* c, real* dst, const double* src_user) {
  cudaError_t e;
  if (!src_user) {
    e = cudaMemsetAsync(dst - node_origin(c), 0, c->nni * sizeof(real), c->stream);
  } else if (!kEta) {
    e = cudaMemcpy2DAsync(dst, (size_t)c->g.np * sizeof(real), src_user,
                          (size_t)(c->g.nx + 1) * sizeof(double), (size_t)c->g.nnx * sizeof(double),
                          (size_t)c->g.nny, cudaMemcpyDefault, c->stream);
  } else {  // fp32 variant: through the dense fp64 staging plane, converted by a kernel
    e = cudaMemcpyAsync(c->pub, src_user, c->nn * sizeof(double), cudaMemcpyDefault, c->stream);
    if (e == cudaSuccess) {
      dim3 blk(32, 8), grd((c->g.nnx + 31) / 32, (c->g.nny + 7) / 8);
      k_nodes_in<<<grd, blk, 0, c->stream>>>(c->g, c->pub, dst);
      c->launches++;
    }
  }
  if (e != cudaSuccess) {
    snprintf(c->err, sizeof(c->err), "node copy in: %s", cudaGetErrorString(e));
    (void)cudaGetLastError();
    c->host_status = NH_ECUDA;
    return NH_ECUDA;
  }
  return NH_OK;
}

int check_launch(Ctx* c) {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    snprintf(c->err, sizeof(c->err), "kernel launch: %s", cudaGetErrorString(e));
    c->host_status = NH_ECUDA;
    return NH_ECUDA;
  }
  return c->host_status;
}

int sticky_status(Ctx* c, int flags) {
  if (c->host_status != NH_OK) return c->host_status;
  if (flags & NH_FLAG_NAN) return fail(c, NH_ENAN, "NaN/Inf time step or right-hand side");
  if (flags & NH_FLAG_NOCONV) return fail(c, NH_ENOCONV, "step: pressure solve did not converge");
  return NH_OK;
}

int read_scalars(Ctx* c) {
  cudaError_t e = cudaMemcpyAsync(c->sc_host, c->sc, sizeof(NhScal), cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) {
    snprintf(c->err, sizeof(c->err), "synchronise: %s", cudaGetErrorString(e));
    c->host_status = NH_ECUDA;
    return NH_ECUDA;
  }
  return NH_OK;
}

// other two slots, given the current one
inline void other_slots(int cur, int& s1, int& s2) { s1 = (cur + 1) % 3; s2 = (cur + 2) % 3; }

struct ProfScope {  // CUDA-event bracket of one kernel group on the context's stream
  Ctx* c; int cat; cudaEvent_t e0, e1; bool on;
  ProfScope(Ctx* c_, int cat_) : c(c_), cat(cat_), on(c_->prof_on) {
    if (!on) return;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    cudaEventRecord(e0, c->stream);
  }
  ~ProfScope() {
    if (!on) return;
    cudaEventRecord(e1, c->stream);
    c->prof_ev[cat].push_back({e0, e1});
  }
};

// R32: the extrapolated start vector is used once seven solutions exist, and only where the stored
// solutions are accurate enough to be extrapolated (the formula amplifies their error 15-fold):
// solver 0 with solver_rtol <= 1e-8
inline bool extrapolate_start(const Ctx* c) {
  return c->prm.warm_start && c->prm.solver == 0 && c->prm.solver_rtol <= 1e-8 && c->nhist == 7;
}

// S6-S10 on U* = (h1, qx1, qy1) with w_in -> (qx_out, qy_out, w_out); p~ in c->p (warm start).
void nonhydro_part(Ctx* c, const real* h1, const real* qx1, const real* qy1,
                   const real* w_in, real* qx_out, real* qy_out, real* w_out) {
  const real *qxs = qx1, *qys = qy1, *ws = w_in;
  {
    ProfScope ps(c, NH_PROF_ASSEMBLY);
    if (c->prm.breaking) {
      nh_launch_breaking(c, h1, qx1, qy1, w_in, c->qx2, c->qy2, c->w2);
      qxs = c->qx2; qys = c->qy2; ws = c->w2;
    }
    if (c->prm.solver == 1) {
      nh_launch_compute_z(c, h1, c->z);
      nh_launch_assemble_rows(c, h1, qxs, qys, c->z, ws, c->kr);
    } else {  // matrix-free solver: no rows of A are stored, only h and z with their ghost cells
      nh_launch_cell_planes(c, h1);
      nh_launch_rhs(c, h1, qxs, qys, c->z, ws, c->b, 0);
    }
  }
  {
    ProfScope ps(c, NH_PROF_SOLVER);
    if (extrapolate_start(c)) nh_launch_start_vector(c, c->p);  // R32
    nh_launch_solve(c, c->b, c->p, 1);
    // the solution joins the history (rotate the seven planes, copy into the oldest)
    real* t = c->hist[6];
    for (int a = 6; a > 0; --a) c->hist[a] = c->hist[a - 1];
    c->hist[0] = t;
    copy_async(c, c->hist[0] - node_origin(c), c->p - node_origin(c), c->nni * sizeof(real));
    if (c->nhist < 7) c->nhist++;
  }
  {
    ProfScope ps(c, NH_PROF_CORRECT);
    nh_launch_correct(c, h1, c->z, qxs, qys, ws, c->p, qx_out, qy_out, w_out);
  }
}

// w changes within a stage only through the correction (nonhydro) or the relaxation zone
inline bool absorbing(const Ctx* c) {
  return c->prm.abs_xlo > 0.0 || c->prm.abs_xhi > 0.0 || c->prm.abs_ylo > 0.0 || c->prm.abs_yhi > 0.0;
}
inline bool w_moves(const Ctx* c) { return c->prm.nonhydro || c->prm.gen_on || absorbing(c); }

// one stage Phi_dt: cell slot `in` -> `out`, node slot `inw` -> `outw` (== inw when w does not
// move); stage_idx selects the relaxation clock (end time of the stage).
void stage(Ctx* c, int in, int inw, int out, int outw, int stage_idx) {
  if (c->prm.nonhydro) {
    {
      ProfScope ps(c, NH_PROF_PREDICTOR);
      nh_launch_predictor(c, c->h[in], c->qx[in], c->qy[in], c->h[out], c->qx1, c->qy1);
    }
    const real* w_in = c->w[inw];
    if (c->prm.w_advect) {  // R30: w is first carried by the velocities of the stage input
      ProfScope ps(c, NH_PROF_PREDICTOR);
      nh_launch_w_advect(c, c->h[in], c->qx[in], c->qy[in], c->w[inw], c->wadv);
      w_in = c->wadv;
    }
    nonhydro_part(c, c->h[out], c->qx1, c->qy1, w_in, c->qx[out], c->qy[out], c->w[outw]);
  } else {
    ProfScope ps(c, NH_PROF_PREDICTOR);
    nh_launch_predictor(c, c->h[in], c->qx[in], c->qy[in], c->h[out], c->qx[out], c->qy[out]);
    if (outw != inw)
      copy_async(c, c->w[outw] - node_origin(c), c->w[inw] - node_origin(c), c->nni * sizeof(real));
  }
  if (c->prm.gen_on)
    nh_launch_relax(c, c->h[out], c->qx[out], c->qy[out], c->w[outw], c->p, stage_idx);
  if (absorbing(c)) nh_launch_absorb(c, c->h[out], c->qx[out], c->qy[out], c->w[outw], c->p);
}

void ensure_lambda(Ctx* c) {
  if (!c->lam_valid) nh_launch_lambda(c, c->h[c->cur], c->qx[c->cur], c->qy[c->cur]);
}

}  // namespace


int core_create(Ctx** out, int nx, int ny, double dx, double dy, const double* H,
              const nh_params* prm, void* cuda_stream) {
  if (!out || !H || !prm) return NH_EINVAL;
  *out = nullptr;
  if (nx < 4 || ny < 4 || !(dx > 0.0) || !(dy > 0.0)) return NH_EINVAL;
  if (!(prm->cfl > 0.0 && prm->cfl <= 1.0) || !(prm->g > 0.0) || !(prm->delta > 0.0)) return NH_EINVAL;
  if (!(prm->eps_dry >= 0.0) || !(prm->solver_rtol > 0.0) || prm->solver_maxit < 1) return NH_EINVAL;
  if (!bc_ok(prm->bc_xlo) || !bc_ok(prm->bc_xhi) || !bc_ok(prm->bc_ylo) || !bc_ok(prm->bc_yhi)) return NH_EINVAL;
  if ((prm->bc_xlo == NH_BC_PERIODIC) != (prm->bc_xhi == NH_BC_PERIODIC)) return NH_EINVAL;
  if ((prm->bc_ylo == NH_BC_PERIODIC) != (prm->bc_yhi == NH_BC_PERIODIC)) return NH_EINVAL;
  if (prm->time_order != 1 && prm->time_order != 2) return NH_EINVAL;
  if (prm->space_order != 1 && prm->space_order != 2) return NH_EINVAL;
  if (prm->precision != NH_PREC) return NH_EINVAL;
  if (!(prm->manning_n >= 0.0)) return NH_EINVAL;
  if (prm->solver != 0 && prm->solver != 1) return NH_EINVAL;
  if (prm->w_advect != 0 && prm->w_advect != 1) return NH_EINVAL;
  if (prm->warm_start != 0 && prm->warm_start != 1) return NH_EINVAL;
  if (!(prm->srj_rel >= 0.0)) return NH_EINVAL;
  if (!(prm->abs_xlo >= 0.0) || !(prm->abs_xhi >= 0.0) || !(prm->abs_ylo >= 0.0) || !(prm->abs_yhi >= 0.0)) return NH_EINVAL;
  if ((prm->abs_xlo > 0.0 || prm->abs_xhi > 0.0) && prm->bc_xlo == NH_BC_PERIODIC) return NH_EINVAL;
  if ((prm->abs_ylo > 0.0 || prm->abs_yhi > 0.0) && prm->bc_ylo == NH_BC_PERIODIC) return NH_EINVAL;
  if (prm->abs_xlo > 0.0 && prm->gen_on) return NH_EINVAL;  // the generating zone owns x-lo
  if (prm->solver == 1 && (!(prm->srj_eps > 0.0) || prm->srj_mmax < 1 || prm->srj_mmax > 4096 ||
                           (prm->srj_mmax & (prm->srj_mmax - 1)) != 0)) return NH_EINVAL;
  if (prm->breaking && !(prm->B1 > 0.0 && prm->B2 > 0.0)) return NH_EINVAL;
  if (prm->gen_on && !(prm->gen_A > 0.0 && prm->gen_h0 > 0.0 && prm->gen_Lrel > 0.0)) return NH_EINVAL;

  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); return NH_ECUDA; }
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) { (void)cudaGetLastError(); return NH_ECUDA; }
  if (prop.major != 10) return NH_ECUDA;  // the library carries sm_100a code only

  Ctx* c = new (std::nothrow) Ctx();
  if (!c) return NH_ENOMEM;
  c->g.nx = nx; c->g.ny = ny; c->g.dx = (real)dx; c->g.dy = (real)dy;
  c->g.bxlo = prm->bc_xlo; c->g.bxhi = prm->bc_xhi; c->g.bylo = prm->bc_ylo; c->g.byhi = prm->bc_yhi;
  c->g.nnx = (prm->bc_xlo == NH_BC_PERIODIC) ? nx : nx + 1;
  c->g.nny = (prm->bc_ylo == NH_BC_PERIODIC) ? ny : ny + 1;
  c->g.np = nh_node_pitch(c->g.nnx);
  c->prm = *prm;
  // fp32 variant: the true residual of this operator bottoms out near 1e-5 of ||b|| in fp32
  // (profiles/r02d_fp32.md), so smaller tolerances are raised to 1e-4
  if (kEta && c->prm.solver_rtol < 1e-4) c->prm.solver_rtol = 1e-4;
  c->stream = (cudaStream_t)cuda_stream;
  c->device = dev;
  c->sm_count = prop.multiProcessorCount;
  c->nc = (size_t)nx * ny;
  c->nn = (size_t)(nx + 1) * (ny + 1);
  c->nni = (size_t)c->g.np * (ny + 1 + 2 * NH_ROW_PAD);
  c->cur = 0; c->curw = 0; c->nhist = 0;
  c->lam_valid = false;
  c->host_status = NH_OK;

  bool ok = true;
  real** cells[] = {&c->H, &c->h[0], &c->h[1], &c->h[2], &c->qx[0], &c->qx[1], &c->qx[2],
                      &c->qy[0], &c->qy[1], &c->qy[2], &c->qx1, &c->qy1, &c->z};
  real** nodes[] = {&c->w[0], &c->w[1], &c->w[2], &c->p, &c->b, &c->dg, &c->dinv, &c->cE, &c->cW,
                      &c->cN, &c->cS, &c->ky, &c->kr, &c->krB, &c->kr0, &c->kpA, &c->kpB, &c->kvA,
                      &c->kvB, &c->kt, &c->w2, &c->hc, &c->zc, &c->wadv, &c->hist[0], &c->hist[1], &c->hist[2],
                    &c->hist[3], &c->hist[4], &c->hist[5], &c->hist[6]};
  for (real** p : cells) ok = ok && dalloc(c, p, c->nc);
  for (real** p : nodes) ok = ok && nalloc(c, p);
  if (kEta) {  // fp32 variant: eta planes, the bathymetry as given, an fp64 staging plane
    for (int k = 0; k < 3; ++k) ok = ok && dalloc(c, &c->eta[k], c->nc);
    ok = ok && dalloc(c, &c->Hd, c->nc) && dalloc(c, &c->stage, c->nc > c->nn ? c->nc : c->nn);
  }
  ok = ok && dalloc(c, &c->pub, c->nn);
  if (prm->breaking) {
    ok = ok && dalloc(c, &c->qx2, c->nc) && dalloc(c, &c->qy2, c->nc);
    ok = ok && dalloc(c, &c->flag_c, c->nc) && dalloc(c, &c->flag_n, c->nni);
  }
  ok = ok && dalloc(c, &c->sc, 1);
  if (ok && cudaMallocHost((void**)&c->sc_host, sizeof(NhScal)) != cudaSuccess) ok = false;
  if (ok && nh_solver_setup(c) != NH_OK) ok = false;
  if (!ok) { (void)cudaGetLastError(); free_all(c); delete c; return NH_ENOMEM; }

  // bathymetry: copy, then validate finiteness on the device (create may synchronise)
  double* Hd = kEta ? c->Hd : (double*)c->H;
  int st = copy_async(c, Hd, H, c->nc * sizeof(double));
  int* bad = (int*)&c->sc->pad;
  if (st == NH_OK) {
    k_all_finite<<<grid1(c, c->nc), 256, 0, c->stream>>>(c->nc, Hd, bad);
    c->launches++;
    if (kEta) {
      k_to_real<<<grid1(c, c->nc), 256, 0, c->stream>>>(c->nc, Hd, c->H);
      c->launches++;
    }
    st = check_launch(c);
  }
  if (st == NH_OK) st = read_scalars(c);
  if (st == NH_OK && c->sc_host->pad != 0) st = NH_EINVAL;
  if (st != NH_OK) { free_all(c); delete c; return st; }
  cudaMemsetAsync(c->sc, 0, sizeof(NhScal), c->stream);
  *out = c;
  return NH_OK;
}

void core_destroy(Ctx* c) {
  if (!c) return;
  cudaStreamSynchronize(c->stream);
  free_all(c);
  delete c;
}

int core_set_state(Ctx* c, const double* h, const double* qx, const double* qy, const double* w,
                 const double* p, int keep_history) {
  if (!c || !h || !qx || !qy) return NH_EINVAL;
  int s1, s2; other_slots(c->cur, s1, s2);
  // stage into a free slot, validate there, then make it current (an invalid state changes nothing)
  k_clear_flag<<<1, 1, 0, c->stream>>>(c->sc, NH_FLAG_BADSTATE);
  c->launches++;
  if (kEta) {  // fp32 variant: eta = h - H in fp64, then both planes in fp32
    if (copy_async(c, c->stage, h, c->nc * sizeof(double))) return NH_ECUDA;
    k_eta_in<<<grid1(c, c->nc), 256, 0, c->stream>>>(c->nc, c->stage, c->Hd, c->H, c->eta[s1], c->h[s1], c->sc);
    c->launches++;
  } else if (cell_in(c, c->h[s1], h)) {
    return NH_ECUDA;
  }
  if (cell_in(c, c->qx[s1], qx) || cell_in(c, c->qy[s1], qy)) return NH_ECUDA;
  nh_launch_validate(c, c->h[s1], c->qx[s1], c->qy[s1]);
  // p goes through a scratch plane (an invalid state must leave the current one untouched)
  if (node_in(c, c->wadv, p)) return NH_ECUDA;
  if (check_launch(c) != NH_OK) return NH_ECUDA;
  if (read_scalars(c) != NH_OK) return NH_ECUDA;
  if (c->sc_host->flags & NH_FLAG_BADSTATE)
    return fail(c, NH_EINVAL, "set_state: h<0 or non-finite input");
  c->cur = s1;
  // R32: nh_set_state starts a new solution history; nh_continue_state (the caller says that this is
  // the running state coming back: a checkpoint, a round trip through the host) keeps it
  if (!keep_history) c->nhist = 0;
  if (node_in(c, c->w[c->curw], w)) return NH_ECUDA;
  if (copy_async(c, c->p - node_origin(c), c->wadv - node_origin(c), c->nni * sizeof(real))) return NH_ECUDA;
  // the CFL rate left by the last RK combine belongs to the replaced state: k_lambda takes a max
  // onto lam_bits, so it has to start from zero (eq. (23) of the NEW state only)
  c->lam_valid = false;
  if (cudaMemsetAsync(&c->sc->lam_bits, 0, sizeof(c->sc->lam_bits), c->stream) != cudaSuccess) {
    (void)cudaGetLastError();
    c->host_status = NH_ECUDA;
    return fail(c, NH_ECUDA, "set_state: cudaMemsetAsync");
  }
  return NH_OK;
}

// node plane out in the public layout (periodic duplicate lines filled), via the dense staging plane
static int node_out(Ctx* c, const real* src, double* dst_user) {
  nh_launch_nodes_out(c, src, c->pub);
  if (check_launch(c) != NH_OK) return NH_ECUDA;
  return copy_async(c, dst_user, c->pub, c->nn * sizeof(double));
}

int core_get_state(Ctx* c, double* h, double* qx, double* qy, double* w, double* p) {
  if (!c) return NH_EINVAL;
  if (h) {
    if (kEta) {  // fp32 variant: h = H + eta with the bathymetry as given, so that h - H is the stored eta
      k_h_out<<<grid1(c, c->nc), 256, 0, c->stream>>>(c->nc, c->eta[c->cur], c->h[c->cur], c->Hd, c->stage);
      c->launches++;
      if (copy_async(c, h, c->stage, c->nc * sizeof(double))) return NH_ECUDA;
    } else if (cell_out(c, h, c->h[c->cur])) {
      return NH_ECUDA;
    }
  }
  if (qx && cell_out(c, qx, c->qx[c->cur])) return NH_ECUDA;
  if (qy && cell_out(c, qy, c->qy[c->cur])) return NH_ECUDA;
  if (w && node_out(c, c->w[c->curw], w)) return NH_ECUDA;
  if (p && node_out(c, c->p, p)) return NH_ECUDA;
  cudaError_t e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) { c->host_status = NH_ECUDA; return fail(c, NH_ECUDA, cudaGetErrorString(e)); }
  return NH_OK;
}

int core_set_time(Ctx* c, double t) {
  if (!c || !(t == t) || isinf(t)) return NH_EINVAL;
  k_set_time<<<1, 1, 0, c->stream>>>(c->sc, t);
  c->launches++;
  return check_launch(c);
}

int core_step(Ctx* c, int nsteps) {
  if (!c || nsteps < 0) return NH_EINVAL;
  if (c->host_status != NH_OK) return c->host_status;
  for (int s = 0; s < nsteps; ++s) {
    ensure_lambda(c);
    nh_launch_set_dt(c, 0.0);
    c->lam_valid = false;
    int s1, s2, w1, w2;
    other_slots(c->cur, s1, s2);
    other_slots(c->curw, w1, w2);
    if (!w_moves(c)) w1 = w2 = c->curw;
    if (c->prm.time_order == 1) {
      stage(c, c->cur, c->curw, s1, w1, 0);
      c->cur = s1; c->curw = w1;
    } else {
      stage(c, c->cur, c->curw, s1, w1, 0);
      stage(c, s1, w1, s2, w2, 1);
      ProfScope ps(c, NH_PROF_CORRECT);
      nh_launch_combine(c, c->h[c->cur], c->qx[c->cur], c->qy[c->cur], c->w[c->curw], c->h[s2],
                        c->qx[s2], c->qy[s2], w2 == c->curw ? nullptr : c->w[w2]);
      c->lam_valid = true;
    }
    nh_launch_end_step(c, 1);
  }
  return check_launch(c);
}

int core_hydrostatic_step(Ctx* c, double dt) {
  if (!c) return NH_EINVAL;
  if (c->host_status != NH_OK) return c->host_status;
  if (!(dt > 0.0)) { ensure_lambda(c); nh_launch_set_dt(c, 0.0); }
  else nh_launch_set_dt(c, dt);
  c->lam_valid = false;
  int s1, s2; other_slots(c->cur, s1, s2);
  nh_launch_predictor(c, c->h[c->cur], c->qx[c->cur], c->qy[c->cur], c->h[s1], c->qx[s1], c->qy[s1]);
  c->cur = s1;
  nh_launch_end_step(c, 0);
  return check_launch(c);
}

int core_nonhydro_correct(Ctx* c, double dt) {
  if (!c || !(dt > 0.0)) return NH_EINVAL;
  if (c->host_status != NH_OK) return c->host_status;
  nh_launch_set_dt(c, dt);
  c->lam_valid = false;
  int s1, s2, w1, w2;
  other_slots(c->cur, s1, s2);
  other_slots(c->curw, w1, w2);
  // U* := current state; h is not changed by S6-S10
  nonhydro_part(c, c->h[c->cur], c->qx[c->cur], c->qy[c->cur], c->w[c->curw], c->qx[s1], c->qy[s1],
                c->w[w1]);
  if (copy_async(c, c->h[s1], c->h[c->cur], c->nc * sizeof(real))) return NH_ECUDA;
  if (kEta && copy_async(c, c->eta[s1], c->eta[c->cur], c->nc * sizeof(real))) return NH_ECUDA;
  c->cur = s1; c->curw = w1;
  nh_launch_end_step(c, 0);
  return check_launch(c);
}

int core_sync(Ctx* c) {
  if (!c) return NH_EINVAL;
  if (read_scalars(c) != NH_OK) return NH_ECUDA;
  return sticky_status(c, c->sc_host->flags);
}

int core_get_info(Ctx* c, nh_info* out) {
  if (!c || !out) return NH_EINVAL;
  if (read_scalars(c) != NH_OK) return NH_ECUDA;
  const NhScal& s = *c->sc_host;
  memset(out, 0, sizeof(*out));
  out->t = s.t; out->dt_last = s.dt_last; out->res_last = s.res_last;
  out->steps = s.steps; out->iters_total = s.iters_total; out->clamps = s.clamps;
  out->solves = s.solves; out->iters_last = s.iters_last; out->iters_max = s.iters_max;
  out->flags = s.flags;
  memcpy(&out->clamp_max, &s.clamp_max_bits, sizeof(double));
  for (int k = 0; k < 6; ++k) out->clamp_hist[k] = (long long)s.clamp_hist[k];
  out->solver_rtol_effective = c->prm.solver_rtol;  // fp32 variant: raised to 1e-4 at create
  return NH_OK;
}

const char* core_last_error(Ctx* c) { return c ? c->err : "null context"; }

long long core_launch_count(Ctx* c) { return c ? c->launches : 0; }

// ---- per-phase device timing (bench.py's roofline: CUDA events on the context's stream) ----
int core_profile(Ctx* c, int enable) {
  if (!c) return NH_EINVAL;
  cudaStreamSynchronize(c->stream);
  for (int k = 0; k < NH_PROF_CATS; ++k) {
    for (auto& ev : c->prof_ev[k]) { cudaEventDestroy(ev.first); cudaEventDestroy(ev.second); }
    c->prof_ev[k].clear();
  }
  c->prof_on = enable != 0;
  return NH_OK;
}

int core_profile_read(Ctx* c, double* ms, long long* groups) {
  if (!c || !ms || !groups) return NH_EINVAL;
  cudaError_t e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) { c->host_status = NH_ECUDA; return fail(c, NH_ECUDA, cudaGetErrorString(e)); }
  for (int k = 0; k < NH_PROF_CATS; ++k) {
    double tot = 0.0;
    for (auto& ev : c->prof_ev[k]) {
      float t = 0.f;
      if (cudaEventElapsedTime(&t, ev.first, ev.second) == cudaSuccess) tot += t;
      cudaEventDestroy(ev.first); cudaEventDestroy(ev.second);
    }
    ms[k] = tot;
    groups[k] = (long long)c->prof_ev[k].size();
    c->prof_ev[k].clear();
  }
  return NH_OK;
}

// ---- test hooks (not on the timed path) ----------------------------------------------------
int core_compute_dt(Ctx* c, double* dt_host) {
  if (!c || !dt_host) return NH_EINVAL;
  ensure_lambda(c);
  nh_launch_set_dt(c, 0.0);
  c->lam_valid = false;
  if (check_launch(c) != NH_OK) return NH_ECUDA;
  if (read_scalars(c) != NH_OK) return NH_ECUDA;
  *dt_host = c->sc_host->dt;
  return NH_OK;
}

int core_apply_A(Ctx* c, const double* x_nodes, double* y_nodes) {
  if (!c || !x_nodes || !y_nodes) return NH_EINVAL;
  if (node_in(c, c->kpA, x_nodes)) return NH_ECUDA;
  nh_launch_compute_z(c, c->h[c->cur], c->z);
  nh_launch_apply_A(c, c->h[c->cur], c->z, c->kpA, c->kpB);
  if (node_out(c, c->kpB, y_nodes)) return NH_ECUDA;
  cudaStreamSynchronize(c->stream);
  return check_launch(c);
}

int core_coeffs(Ctx* c, double* AC, double* AE, double* AW, double* AN, double* AS) {
  if (!c || !AC || !AE || !AW || !AN || !AS) return NH_EINVAL;
  nh_launch_compute_z(c, c->h[c->cur], c->z);
  nh_launch_coeffs(c, c->h[c->cur], c->z);  // raw (unscaled) rows
  const real* src[5] = {c->dg, c->cE, c->cW, c->cN, c->cS};
  double* dst[5] = {AC, AE, AW, AN, AS};
  for (int k = 0; k < 5; ++k)
    if (node_out(c, src[k], dst[k])) return NH_ECUDA;
  cudaStreamSynchronize(c->stream);
  return check_launch(c);
}

static int rhs_hook(Ctx* c, double dt, double* out, int constraint_only) {
  if (!constraint_only) { nh_launch_set_dt(c, dt); c->lam_valid = false; }
  nh_launch_compute_z(c, c->h[c->cur], c->z);
  nh_launch_rhs(c, c->h[c->cur], c->qx[c->cur], c->qy[c->cur], c->z, c->w[c->curw], c->b,
                constraint_only);
  if (node_out(c, c->b, out)) return NH_ECUDA;
  cudaStreamSynchronize(c->stream);
  return check_launch(c);
}
int core_rhs(Ctx* c, double dt, double* b_nodes) {
  if (!c || !b_nodes || !(dt > 0.0)) return NH_EINVAL;
  return rhs_hook(c, dt, b_nodes, 0);
}
int core_constraint(Ctx* c, double* B_nodes) {
  if (!c || !B_nodes) return NH_EINVAL;
  return rhs_hook(c, 1.0, B_nodes, 1);
}

int core_breaking(Ctx* c, double dt, double* qx2, double* qy2, double* w2) {
  if (!c || !qx2 || !qy2 || !w2 || !(dt > 0.0) || !c->prm.breaking) return NH_EINVAL;
  nh_launch_set_dt(c, dt);
  c->lam_valid = false;
  nh_launch_breaking(c, c->h[c->cur], c->qx[c->cur], c->qy[c->cur], c->w[c->curw], c->qx2, c->qy2,
                     c->w2);
  if (cell_out(c, qx2, c->qx2) || cell_out(c, qy2, c->qy2)) return NH_ECUDA;
  if (node_out(c, c->w2, w2)) return NH_ECUDA;
  cudaStreamSynchronize(c->stream);
  return check_launch(c);
}

int core_w_advect(Ctx* c, double dt, double* w_out) {
  if (!c || !w_out || !(dt > 0.0)) return NH_EINVAL;
  nh_launch_set_dt(c, dt);
  c->lam_valid = false;
  nh_launch_w_advect(c, c->h[c->cur], c->qx[c->cur], c->qy[c->cur], c->w[c->curw], c->wadv);
  if (node_out(c, c->wadv, w_out)) return NH_ECUDA;
  cudaStreamSynchronize(c->stream);
  return check_launch(c);
}

int core_start_vector(Ctx* c, double* x0_nodes) {
  if (!c || !x0_nodes) return NH_EINVAL;
  if (copy_async(c, c->w2 - node_origin(c), c->p - node_origin(c), c->nni * sizeof(real))) return NH_ECUDA;
  if (extrapolate_start(c)) nh_launch_start_vector(c, c->w2);
  if (node_out(c, c->w2, x0_nodes)) return NH_ECUDA;
  cudaStreamSynchronize(c->stream);
  return check_launch(c);
}

int core_solve(Ctx* c, const double* b_nodes, double* x_nodes, int* iters, double* relres) {
  if (!c || !b_nodes || !x_nodes) return NH_EINVAL;
  if (node_in(c, c->b, b_nodes) || node_in(c, c->w2, x_nodes)) return NH_ECUDA;
  if (c->prm.solver == 1) {
    nh_launch_compute_z(c, c->h[c->cur], c->z);
    nh_launch_coeffs(c, c->h[c->cur], c->z);
    nh_launch_scale_rows(c, c->b, c->kr);
  } else {
    nh_launch_cell_planes(c, c->h[c->cur]);
  }
  nh_launch_solve(c, c->b, c->w2, 0);
  if (node_out(c, c->w2, x_nodes)) return NH_ECUDA;
  if (check_launch(c) != NH_OK) return NH_ECUDA;
  if (read_scalars(c) != NH_OK) return NH_ECUDA;
  if (iters) *iters = c->sc_host->iters_last;
  if (relres) *relres = c->sc_host->res_last;
  int fl = c->sc_host->flags;
  // the hook reports its own solve; clear the sticky bits it may have set
  k_clear_flag<<<1, 1, 0, c->stream>>>(c->sc, NH_FLAG_NOCONV | NH_FLAG_NAN | NH_FLAG_STAGNATED);
  c->launches++;
  if (fl & NH_FLAG_NAN) return NH_ENAN;
  if (fl & NH_FLAG_NOCONV) return NH_ENOCONV;
  return NH_OK;
}

}  // namespace NH_NS
