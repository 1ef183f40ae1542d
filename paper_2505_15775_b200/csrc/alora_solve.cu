// placeholder until the solver lands
#include "alora_internal.h"
namespace alora { void free_solve_workspace(alora_ctx*) {} }
extern "C" void alora_default_params(alora_params* p) {
  if (!p) return;
  p->eps = 1e-5; p->stop_mode = 0; p->T_max = 100; p->tol0 = 1e-2; p->c_in = 0.1; p->tol_min = 1e-7;
  p->it_max = 500; p->lbfgs_mem = 5; p->p_max = 1; p->k_max = 300; p->tau_neg = -1.0; p->tol_eig = -1.0;
  p->gamma = 2.0; p->kappa = 0.25; p->sigma_max = 1e8; p->tau_shrink = 1e-8; p->s_max = 1e6; p->seed = 12345;
}
extern "C" alora_status alora_lanczos(alora_ctx* c, const double*, int32_t, double, uint64_t, double*, void*, int32_t*, double*) {
  return alora::fail(c, ALORA_ESTATE, "not built yet");
}
extern "C" alora_status alora_solve(alora_ctx* c, const alora_params*, void*, int32_t*, int32_t, double*, double*, alora_iter_record*, int32_t, alora_result*) {
  return alora::fail(c, ALORA_ESTATE, "not built yet");
}
