// tridiag.cuh -- eigen-decomposition of the small real symmetric tridiagonal Lanczos matrix and
// the Krylov coefficients c = beta0 * V exp(z Lambda) V^T e_1 ("diagonalize the
// tridiagonal matrix in the subspace").  Implicit symmetric QR iteration with Wilkinson shift and
// deflation (Golub & Van Loan, "Matrix Computations", sec. 8.3), written so that the same source
// runs as one warp on the device (every lane repeats the scalar recurrence and rotates only the
// eigenvector rows it owns: no intra-sweep synchronisation) and as plain host code for the CPU
// unit test (nl = 1).
#pragma once
#include <math.h>

#ifdef __CUDACC__
#define TD_HD __host__ __device__
#else
#define TD_HD
#endif

// a[0..m) diagonal, b[0..m-1) off-diagonal (both overwritten; a ends as the eigenvalues).
// V: m x m row-major with leading dimension ldv, must hold the identity in rows lane, lane+nl, ...
// on entry; on exit rows owned by this lane hold the eigenvectors' components (T = V diag(a) V^T).
TD_HD inline void tridiag_qr_eig(int m, double *a, double *b, double *V, int ldv, int lane, int nl) {
  const double eps = 2.220446049250313e-16;
  int hi = m - 1;
  int guard = 0;
  while (hi > 0 && guard < 64 * m) {
    guard++;
    for (int i = 0; i < hi; i++)
      if (fabs(b[i]) <= eps * (fabs(a[i]) + fabs(a[i + 1]))) b[i] = 0.0;
    if (b[hi - 1] == 0.0) { hi--; continue; }
    int lo = hi - 1;
    while (lo > 0 && b[lo - 1] != 0.0) lo--;
    // Wilkinson shift from the trailing 2x2 of the unreduced block [lo, hi]
    double dd = 0.5 * (a[hi - 1] - a[hi]), bb = b[hi - 1];
    double den = dd + (dd >= 0.0 ? 1.0 : -1.0) * sqrt(dd * dd + bb * bb);
    double mu = a[hi] - bb * bb / den;
    double x = a[lo] - mu, z = b[lo];
    for (int k = lo; k < hi; k++) {
      double r = sqrt(x * x + z * z);
      double c = 1.0, s = 0.0;
      if (r > 0.0) { c = x / r; s = z / r; }
      if (k > lo) b[k - 1] = r;
      double ak = a[k], ak1 = a[k + 1], bk = b[k];
      a[k] = c * c * ak + 2.0 * c * s * bk + s * s * ak1;
      a[k + 1] = s * s * ak - 2.0 * c * s * bk + c * c * ak1;
      b[k] = c * s * (ak1 - ak) + (c * c - s * s) * bk;
      x = b[k];
      if (k < hi - 1) { z = s * b[k + 1]; b[k + 1] = c * b[k + 1]; }
      for (int row = lane; row < m; row += nl) {
        double vk = V[row * ldv + k], vk1 = V[row * ldv + k + 1];
        V[row * ldv + k] = c * vk + s * vk1;
        V[row * ldv + k + 1] = -s * vk + c * vk1;
      }
    }
  }
}
