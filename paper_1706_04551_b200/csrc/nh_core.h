// nh_core.h -- the precision-specific implementation behind the C ABI.  nh_core.cu defines these
// functions once per build of the kernels (namespace nh64: fp64, namespace nh32: the fp32 variant);
// nh_abi.cu holds the extern "C" entry points of include/nh_b200.h and dispatches on
// nh_params.precision.  User-facing arrays are fp64 in both builds (the fp32 build converts at
// nh_set_state / nh_get_state).
#pragma once
#include "../../include/nh_b200.h"

#define NH_DECLARE_CORE(NS)                                                                        \
  namespace NS {                                                                                   \
  struct Ctx;                                                                                      \
  int core_create(Ctx** out, int nx, int ny, double dx, double dy, const double* H,               \
                  const nh_params* prm, void* cuda_stream);                                        \
  void core_destroy(Ctx* c);                                                                       \
  int core_set_state(Ctx* c, const double* h, const double* qx, const double* qy, const double* w, \
                     const double* p, int keep_history);                                           \
  int core_get_state(Ctx* c, double* h, double* qx, double* qy, double* w, double* p);            \
  int core_set_time(Ctx* c, double t);                                                             \
  int core_step(Ctx* c, int nsteps);                                                               \
  int core_hydrostatic_step(Ctx* c, double dt);                                                    \
  int core_nonhydro_correct(Ctx* c, double dt);                                                    \
  int core_sync(Ctx* c);                                                                           \
  int core_get_info(Ctx* c, nh_info* out);                                                         \
  const char* core_last_error(Ctx* c);                                                             \
  long long core_launch_count(Ctx* c);                                                             \
  int core_profile(Ctx* c, int enable);                                                            \
  int core_profile_read(Ctx* c, double* ms, long long* groups);                                    \
  int core_compute_dt(Ctx* c, double* dt_host);                                                    \
  int core_apply_A(Ctx* c, const double* x_nodes, double* y_nodes);                                \
  int core_coeffs(Ctx* c, double* AC, double* AE, double* AW, double* AN, double* AS);            \
  int core_rhs(Ctx* c, double dt, double* b_nodes);                                                \
  int core_constraint(Ctx* c, double* B_nodes);                                                    \
  int core_breaking(Ctx* c, double dt, double* qx2, double* qy2, double* w2);                     \
  int core_w_advect(Ctx* c, double dt, double* w_out);                                             \
  int core_start_vector(Ctx* c, double* x0_nodes);                                                 \
  int core_solve(Ctx* c, const double* b_nodes, double* x_nodes, int* iters, double* relres);     \
  }

NH_DECLARE_CORE(nh64)
NH_DECLARE_CORE(nh32)
