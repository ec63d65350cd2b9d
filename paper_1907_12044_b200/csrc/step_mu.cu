// step_mu.cu -- TDVP-MU step driver.  Placeholder until the SVD path lands.
#include "handle.cuh"
extern "C" {
int tdvp_step_mu(tdvp_handle *h, double dt, double *err_est) {
  (void)dt; (void)err_est;
  return set_err(h, TDVP_ESTATE, "tdvp_step_mu: not built yet in this revision");
}
int tdvp_mu_derivative(tdvp_handle *h, tdvp_c128 *const *out_host) {
  (void)out_host;
  return set_err(h, TDVP_ESTATE, "tdvp_mu_derivative: not built yet in this revision");
}
int tdvp_svd_bond(tdvp_handle *h, int Ml, int d, int Mr, const tdvp_c128 *C, tdvp_c128 *U, double *lam, tdvp_c128 *Vh) {
  (void)Ml; (void)d; (void)Mr; (void)C; (void)U; (void)lam; (void)Vh;
  return set_err(h, TDVP_ESTATE, "tdvp_svd_bond: not built yet in this revision");
}
}
