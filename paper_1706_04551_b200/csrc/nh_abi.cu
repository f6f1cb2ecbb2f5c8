// nh_abi.cu -- the C ABI of libnh_b200.so (include/nh_b200.h).  Nothing here computes: every entry
// point forwards to the implementation of the context's precision, nh64 (fp64, the default and the
// parity contract) or nh32 (the optional fp32 variant), both defined by nh_core.cu (nh_core.h).
#include <string.h>

#include <new>

#include "nh_core.h"

struct nh_ctx {
  int prec;  // 64 or 32
  nh64::Ctx* c64;
  nh32::Ctx* c32;
};

#define NH_FWD(c, call64, call32) ((c)->prec == 32 ? (call32) : (call64))

extern "C" {

void nh_default_params(nh_params* prm) {
  if (!prm) return;
  memset(prm, 0, sizeof(*prm));
  prm->g = 9.81; prm->cfl = 0.5; prm->delta = 1e-5; prm->eps_dry = 1e-5;
  prm->B1 = 0.15; prm->B2 = 0.5; prm->solver_rtol = 1e-12;
  prm->breaking = 0; prm->nonhydro = 1; prm->time_order = 2; prm->space_order = 2;
  prm->bc_xlo = prm->bc_xhi = prm->bc_ylo = prm->bc_yhi = NH_BC_OUTFLOW;
  prm->solver_maxit = 10000; prm->gen_on = 0; prm->precision = 64;
  prm->solver = 0; prm->srj_eps = 1e-5; prm->srj_mmax = 256; prm->w_advect = 0; prm->warm_start = 1;
}

int nh_create(nh_ctx** out, int nx, int ny, double dx, double dy, const double* H,
              const nh_params* prm, void* cuda_stream) {
  if (!out || !H || !prm) return NH_EINVAL;
  *out = nullptr;
  if (prm->precision != 64 && prm->precision != 32) return NH_EINVAL;
  nh_ctx* c = new (std::nothrow) nh_ctx();
  if (!c) return NH_ENOMEM;
  c->prec = prm->precision; c->c64 = nullptr; c->c32 = nullptr;
  int st = (c->prec == 32) ? nh32::core_create(&c->c32, nx, ny, dx, dy, H, prm, cuda_stream)
                           : nh64::core_create(&c->c64, nx, ny, dx, dy, H, prm, cuda_stream);
  if (st != NH_OK) { delete c; return st; }
  *out = c;
  return NH_OK;
}

void nh_destroy(nh_ctx* c) {
  if (!c) return;
  if (c->prec == 32) nh32::core_destroy(c->c32); else nh64::core_destroy(c->c64);
  delete c;
}

int nh_set_state(nh_ctx* c, const double* h, const double* qx, const double* qy, const double* w,
                 const double* p) {
  if (!c) return NH_EINVAL;
  return NH_FWD(c, nh64::core_set_state(c->c64, h, qx, qy, w, p, 0), nh32::core_set_state(c->c32, h, qx, qy, w, p, 0));
}
int nh_continue_state(nh_ctx* c, const double* h, const double* qx, const double* qy, const double* w,
                      const double* p) {
  if (!c) return NH_EINVAL;
  return NH_FWD(c, nh64::core_set_state(c->c64, h, qx, qy, w, p, 1), nh32::core_set_state(c->c32, h, qx, qy, w, p, 1));
}
int nh_get_state(nh_ctx* c, double* h, double* qx, double* qy, double* w, double* p) {
  if (!c) return NH_EINVAL;
  return NH_FWD(c, nh64::core_get_state(c->c64, h, qx, qy, w, p), nh32::core_get_state(c->c32, h, qx, qy, w, p));
}
int nh_set_time(nh_ctx* c, double t) {
  if (!c) return NH_EINVAL;
  return NH_FWD(c, nh64::core_set_time(c->c64, t), nh32::core_set_time(c->c32, t));
}
int nh_step(nh_ctx* c, int nsteps) {
  if (!c) return NH_EINVAL;
  return NH_FWD(c, nh64::core_step(c->c64, nsteps), nh32::core_step(c->c32, nsteps));
}
int nh_hydrostatic_step(nh_ctx* c, double dt) {
  if (!c) return NH_EINVAL;
  return NH_FWD(c, nh64::core_hydrostatic_step(c->c64, dt), nh32::core_hydrostatic_step(c->c32, dt));
}
int nh_nonhydro_correct(nh_ctx* c, double dt) {
  if (!c) return NH_EINVAL;
  return NH_FWD(c, nh64::core_nonhydro_correct(c->c64, dt), nh32::core_nonhydro_correct(c->c32, dt));
}
int nh_sync(nh_ctx* c) {
  if (!c) return NH_EINVAL;
  return NH_FWD(c, nh64::core_sync(c->c64), nh32::core_sync(c->c32));
}
int nh_get_info(nh_ctx* c, nh_info* out) {
  if (!c) return NH_EINVAL;
  return NH_FWD(c, nh64::core_get_info(c->c64, out), nh32::core_get_info(c->c32, out));
}
const char* nh_last_error(nh_ctx* c) {
  if (!c) return "null context";
  return NH_FWD(c, nh64::core_last_error(c->c64), nh32::core_last_error(c->c32));
}
long long nh_launch_count(nh_ctx* c) {
  if (!c) return 0;
  return NH_FWD(c, nh64::core_launch_count(c->c64), nh32::core_launch_count(c->c32));
}
int nh_profile(nh_ctx* c, int enable) {
  if (!c) return NH_EINVAL;
  return NH_FWD(c, nh64::core_profile(c->c64, enable), nh32::core_profile(c->c32, enable));
}
int nh_profile_read(nh_ctx* c, double* ms, long long* groups) {
  if (!c) return NH_EINVAL;
  return NH_FWD(c, nh64::core_profile_read(c->c64, ms, groups), nh32::core_profile_read(c->c32, ms, groups));
}
int nh_compute_dt(nh_ctx* c, double* dt_host) {
  if (!c) return NH_EINVAL;
  return NH_FWD(c, nh64::core_compute_dt(c->c64, dt_host), nh32::core_compute_dt(c->c32, dt_host));
}
int nh_apply_A(nh_ctx* c, const double* x_nodes, double* y_nodes) {
  if (!c) return NH_EINVAL;
  return NH_FWD(c, nh64::core_apply_A(c->c64, x_nodes, y_nodes), nh32::core_apply_A(c->c32, x_nodes, y_nodes));
}
int nh_coeffs(nh_ctx* c, double* AC, double* AE, double* AW, double* AN, double* AS) {
  if (!c) return NH_EINVAL;
  return NH_FWD(c, nh64::core_coeffs(c->c64, AC, AE, AW, AN, AS), nh32::core_coeffs(c->c32, AC, AE, AW, AN, AS));
}
int nh_rhs(nh_ctx* c, double dt, double* b_nodes) {
  if (!c) return NH_EINVAL;
  return NH_FWD(c, nh64::core_rhs(c->c64, dt, b_nodes), nh32::core_rhs(c->c32, dt, b_nodes));
}
int nh_constraint(nh_ctx* c, double* B_nodes) {
  if (!c) return NH_EINVAL;
  return NH_FWD(c, nh64::core_constraint(c->c64, B_nodes), nh32::core_constraint(c->c32, B_nodes));
}
int nh_breaking(nh_ctx* c, double dt, double* qx2, double* qy2, double* w2) {
  if (!c) return NH_EINVAL;
  return NH_FWD(c, nh64::core_breaking(c->c64, dt, qx2, qy2, w2), nh32::core_breaking(c->c32, dt, qx2, qy2, w2));
}
int nh_w_advect(nh_ctx* c, double dt, double* w_out) {
  if (!c) return NH_EINVAL;
  return NH_FWD(c, nh64::core_w_advect(c->c64, dt, w_out), nh32::core_w_advect(c->c32, dt, w_out));
}
int nh_start_vector(nh_ctx* c, double* x0_nodes) {
  if (!c) return NH_EINVAL;
  return NH_FWD(c, nh64::core_start_vector(c->c64, x0_nodes), nh32::core_start_vector(c->c32, x0_nodes));
}
int nh_solve(nh_ctx* c, const double* b_nodes, double* x_nodes, int* iters, double* relres) {
  if (!c) return NH_EINVAL;
  return NH_FWD(c, nh64::core_solve(c->c64, b_nodes, x_nodes, iters, relres),
                nh32::core_solve(c->c32, b_nodes, x_nodes, iters, relres));
}

}  // extern "C"
