// step_mu.cu -- TDVP-MU step driver.  Placeholder until the SVD path lands.
#include "handle.cuh"
extern "C" int tdvp_step_mu(tdvp_handle *h, double dt, double *err_est) {
  (void)dt; (void)err_est;
  return set_err(h, TDVP_ESTATE, "tdvp_step_mu: not built yet in this revision");
}
