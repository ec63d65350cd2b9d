// step_mu.cu -- TDVP-MU: the right-hand side of the
// equations of motion in the left-canonical gauge and one Dormand-Prince 5(4) step of it.
//   Eq. 27:        i dC_N/dt = H[N] C_N
//   Eq. 37:    i dL_i/dt = (1 - p[i]) H[i](L_i U Lambda) Lambda~^{-1} U^dagger
//   Eq. 33:        p[i] = L_i L_i^dagger, applied as G - L (L^dagger G)
//   Eq. 36:    the centre of site i+1 unfolded by SVD, U Lambda R
//   Eq. 38:    Lambda~ = Lambda + eps^{1/2} exp(-Lambda / eps^{1/2})
// Reading c13: G = H_eff(C_i) Lambda~^{-1} U^dagger with C_i = L_i U Lambda; only the
// inverse factor is regularised.  Reading c12: one call = one fixed Dormand-Prince step (the
// paper's VMF integrator); step-size control is the caller's loop.
// Everything is enqueued on the handle's stream; the SVDs run on the device (svd.cu).
#include <algorithm>
#include <cmath>

#include <cstdlib>
#include <utility>

#include <functional>

#include "handle.cuh"

int move_gauge(tdvp_handle *h, int centre);

namespace {

constexpr int VT = 256;
inline int grid_for(long long n) { long long g = (n + VT - 1) / VT; return (int)(g > 1184 ? 1184 : (g < 1 ? 1 : g)); }
inline size_t up256(size_t x) { return (x + 255) & ~size_t(255); }
long long site_elems(const tdvp_handle *h, int i) { return (long long)h->M[i] * h->d[i] * h->M[i + 1]; }

// X[row][c] *= f(lam[c]);  mode 0: f = lam (U Lambda); mode 1: f = 1 / (lam + sq exp(-lam / sq))  (Eq. 38)
__global__ void scale_cols_kernel(c128 *X, long long rows, int n, const double *lam, int mode, double sq) {
  const long long total = rows * n;
  for (long long e = blockIdx.x * (long long)VT + threadIdx.x; e < total; e += (long long)gridDim.x * VT) {
    const double l = lam[e % n];
    const double f = mode == 0 ? l : 1.0 / (l + sq * exp(-l / sq));
    c128 v = X[e];
    X[e] = make_double2(v.x * f, v.y * f);
  }
}
// out = -i (G - T)   (T may be NULL: out = -i G)
__global__ void minus_i_diff_kernel(c128 *out, const c128 *G, const c128 *T, long long n) {
  for (long long e = blockIdx.x * (long long)VT + threadIdx.x; e < n; e += (long long)gridDim.x * VT) {
    c128 g = G[e];
    if (T) { c128 t = T[e]; g.x -= t.x; g.y -= t.y; }
    out[e] = make_double2(g.y, -g.x);
  }
}
struct Comb { const c128 *k[7]; double c[7]; int n; };
// out = base + sum_j c_j k_j   (base may be NULL)
__global__ void lincomb_kernel(c128 *out, const c128 *base, Comb cb, long long n) {
  for (long long e = blockIdx.x * (long long)VT + threadIdx.x; e < n; e += (long long)gridDim.x * VT) {
    c128 v = base ? base[e] : make_double2(0.0, 0.0);
    for (int j = 0; j < cb.n; j++) { c128 k = cb.k[j][e]; v.x += cb.c[j] * k.x; v.y += cb.c[j] * k.y; }
    out[e] = v;
  }
}
// out[0] = sqrt(sum_i parts[i])
__global__ void err_final_kernel(const double *parts, int n, double *out) {
  double s = 0.0;
  for (int i = 0; i < n; i++) s += parts[i];
  out[0] = sqrt(s);
}

struct MuScratch {
  c128 *U, *UL, *P, *Vh, *C0, *C1, *HC, *G, *T;
  double *lam;
};

size_t mu_scratch_bytes(const tdvp_handle *h, size_t *sb_out, size_t *bb_out) {
  long long ms = 0; int mm = 1;
  for (int i = 0; i < h->n; i++) { ms = std::max(ms, site_elems(h, i)); mm = std::max(mm, h->M[i + 1]); }
  const size_t sb = up256(ms * 16), bb = up256((size_t)mm * mm * 16);
  if (sb_out) *sb_out = sb;
  if (bb_out) *bb_out = bb;
  return 6 * sb + 3 * bb + up256(mm * 8) + 1024;
}

MuScratch mu_carve(const tdvp_handle *h, void *mem) {
  size_t sb = 0, bb = 0;
  mu_scratch_bytes(h, &sb, &bb);
  MuScratch s{};
  char *p = reinterpret_cast<char *>(mem);
  if (!p) return s;
  s.Vh = reinterpret_cast<c128 *>(p); p += sb;
  s.C0 = reinterpret_cast<c128 *>(p); p += sb;
  s.C1 = reinterpret_cast<c128 *>(p); p += sb;
  s.HC = reinterpret_cast<c128 *>(p); p += sb;
  s.G = reinterpret_cast<c128 *>(p); p += sb;
  s.T = reinterpret_cast<c128 *>(p); p += sb;
  s.U = reinterpret_cast<c128 *>(p); p += bb;
  s.UL = reinterpret_cast<c128 *>(p); p += bb;
  s.P = reinterpret_cast<c128 *>(p); p += bb;
  s.lam = reinterpret_cast<double *>(p);
  return s;
}

MuScratch mu_scratch(tdvp_handle *h) {
  if (!h->mu_scratch) {
    if (cudaMalloc(&h->mu_scratch, mu_scratch_bytes(h, nullptr, nullptr)) != cudaSuccess) { h->mu_scratch = nullptr; }
  }
  return mu_carve(h, h->mu_scratch);
}

void gemm1(cudaStream_t st, const ZGemm &g) { zgemm(st, g); }

int mu_rhs_pipelined(tdvp_handle *h, const std::vector<c128 *> &Y, const std::vector<c128 *> &K);

// K = F(Y): the TDVP-MU right-hand side.  Uses the handle's Lenv / Renv storage as scratch caches.
// (One queue, everything in sequence: kept as the reference order, TDVP_MU_PIPELINE=0; mu_rhs below is what runs.)
int mu_rhs_serial(tdvp_handle *h, const std::vector<c128 *> &Y, const std::vector<c128 *> &K) {
  cudaStream_t st = h->stream;
  const int n = h->n;
  MuScratch s = mu_scratch(h);
  if (!s.U) return set_err(h, TDVP_ENOMEM, "TDVP-MU scratch allocation failed");
  void *ws = h->step_ws;
  const double sq = std::sqrt(h->opt.mu_eps);
  for (int i = 0; i < n - 1; i++)                                                        // "Get Env"
    env_update(st, 0, h->M[i], h->M[i + 1], h->d[i], h->Dw[i], h->Dw[i + 1], h->Lenv[i], h->Wsp[i], Y[i],
               h->Lenv[i + 1], ws);
  {                                                                                      // Eq. 27
    const int i = n - 1;
    heff_apply(st, h->M[i], h->M[i + 1], h->d[i], h->Dw[i], h->Dw[i + 1], h->Lenv[i], h->Wsp[i], Y[i], h->Renv[i],
               s.HC, ws);
    TDVP_LAUNCH(minus_i_diff_kernel, grid_for(site_elems(h, i)), VT, 0, st, K[i], s.HC, (const c128 *)nullptr,
                site_elems(h, i));
  }
  const c128 *C = Y[n - 1];
  c128 *Cnext = s.C0;
  for (int i = n - 1; i >= 1; i--) {
    const int Ml = h->M[i], Mr = h->M[i + 1], d = h->d[i];
    svd_bond(st, Ml, d, Mr, C, s.U, s.lam, s.Vh, ws, h->status_dev);                                    // Eq. 36
    env_update(st, 1, Ml, Mr, d, h->Dw[i], h->Dw[i + 1], h->Renv[i], h->Wsp[i], s.Vh, h->Renv[i - 1], ws);
    // site i-1: centre form C' = L (U Lambda)
    const int j = i - 1, Jl = h->M[j], Jr = h->M[j + 1], dj = h->d[j];                    // Jr == Ml
    const long long ne = site_elems(h, j), rows = (long long)Jl * dj;
    vec_copy(st, s.UL, s.U, (long long)Jr * Jr);
    TDVP_LAUNCH(scale_cols_kernel, grid_for((long long)Jr * Jr), VT, 0, st, s.UL, (long long)Jr, Jr, s.lam, 0, sq);
    ZGemm g{};
    g.A = Y[j]; g.B = s.UL; g.C = Cnext;                    // C'[(a,s)][r] = sum_l L[(a,s)][l] UL[l][r]
    g.M = (int)rows; g.K = Jr; g.N = Jr; g.a_ms = Jr; g.a_ks = 1; g.b_ks = Jr; g.b_ns = 1; g.ldc = Jr;
    gemm1(st, g);
    heff_apply(st, Jl, Jr, dj, h->Dw[j], h->Dw[j + 1], h->Lenv[j], h->Wsp[j], Cnext, h->Renv[j], s.HC, ws);
    TDVP_LAUNCH(scale_cols_kernel, grid_for(ne), VT, 0, st, s.HC, rows, Jr, s.lam, 1, sq);  // Lambda~^{-1}, Eq. 38
    ZGemm g2{};
    g2.A = s.HC; g2.B = s.U; g2.C = s.G;                    // G[(a,s)][l] = sum_r HC[(a,s)][r] conj(U[l][r])
    g2.M = (int)rows; g2.K = Jr; g2.N = Jr; g2.a_ms = Jr; g2.a_ks = 1; g2.b_ns = Jr; g2.b_ks = 1; g2.conjB = 1; g2.ldc = Jr;
    gemm1(st, g2);
    ZGemm g3{};
    g3.A = Y[j]; g3.B = s.G; g3.C = s.P;                    // P[b][l] = sum_{(a,s)} conj(L[(a,s)][b]) G[(a,s)][l]
    g3.M = Jr; g3.N = Jr; g3.K = (int)rows; g3.a_ms = 1; g3.a_ks = Jr; g3.conjA = 1; g3.b_ks = Jr; g3.b_ns = 1; g3.ldc = Jr;
    gemm1(st, g3);
    ZGemm g4{};
    g4.A = Y[j]; g4.B = s.P; g4.C = s.T;                    // T = L P
    g4.M = (int)rows; g4.K = Jr; g4.N = Jr; g4.a_ms = Jr; g4.a_ks = 1; g4.b_ks = Jr; g4.b_ns = 1; g4.ldc = Jr;
    gemm1(st, g4);
    TDVP_LAUNCH(minus_i_diff_kernel, grid_for(ne), VT, 0, st, K[j], s.G, s.T, ne);         // -i (1 - p) G, Eq. 33/37
    C = Cnext;
    Cnext = (Cnext == s.C0) ? s.C1 : s.C0;
  }
  return check_cuda(h, cudaGetLastError(), "TDVP-MU derivative");
}

int mu_rhs(tdvp_handle *h, const std::vector<c128 *> &Y, const std::vector<c128 *> &K) {
  static const bool pipeline = [] { const char *e = getenv("TDVP_MU_PIPELINE"); return !(e && e[0] == '0'); }();
  if (pipeline && !h->cmf_streams.empty() && !h->cmf_mem.empty()) return mu_rhs_pipelined(h, Y, K);
  return mu_rhs_serial(h, Y, K);
}

int mu_alloc(tdvp_handle *h) {
  if (!h->mu_y.empty()) return TDVP_OK;
  std::vector<c128 *> tmp;
  for (int sidx = 0; sidx < 8; sidx++) {
    std::vector<c128 *> v(h->n, nullptr);
    for (int i = 0; i < h->n; i++)
      if (int rc = check_cuda(h, cudaMalloc(&v[i], site_elems(h, i) * 16), "cudaMalloc TDVP-MU stage")) return rc;
    if (sidx < 7) h->mu_k[sidx] = v; else h->mu_y = v;
  }
  if (int rc = check_cuda(h, cudaMalloc(&h->mu_err_dev, (h->n + 1) * sizeof(double)), "cudaMalloc")) return rc;
  return TDVP_OK;
}

// Dormand-Prince 5(4) Butcher tableau (the RK45 of PAPER.md:224)
const double DP_A[7][6] = {
    {0, 0, 0, 0, 0, 0},
    {1.0 / 5, 0, 0, 0, 0, 0},
    {3.0 / 40, 9.0 / 40, 0, 0, 0, 0},
    {44.0 / 45, -56.0 / 15, 32.0 / 9, 0, 0, 0},
    {19372.0 / 6561, -25360.0 / 2187, 64448.0 / 6561, -212.0 / 729, 0, 0},
    {9017.0 / 3168, -355.0 / 33, 46732.0 / 5247, 49.0 / 176, -5103.0 / 18656, 0},
    {35.0 / 384, 0.0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84}};
const double DP_B5[7] = {35.0 / 384, 0.0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84, 0.0};
const double DP_B4[7] = {5179.0 / 57600, 0.0, 7571.0 / 16695, 393.0 / 640, -92097.0 / 339200, 187.0 / 2100, 1.0 / 40};

int enqueue_mu_step(tdvp_handle *h, double dt) {
  cudaStream_t st = h->stream;
  const int n = h->n;
  // first-same-as-last: stage 7 of the previous step was evaluated at what is now the state, so its
  // right-hand side is stage 1 of this step (any call that changes the tensors clears the flag;
  // TDVP_NO_FSAL=1, read at every step, recomputes it -- the exactness test toggles it)
  const bool fsal = h->mu_fsal && !getenv("TDVP_NO_FSAL");
  if (fsal) std::swap(h->mu_k[0], h->mu_k[6]);
  h->mu_fsal = false;
  for (int sidx = fsal ? 1 : 0; sidx < 7; sidx++) {
    const std::vector<c128 *> *Y = &h->A;
    if (sidx > 0) {
      for (int i = 0; i < n; i++) {
        Comb cb{}; cb.n = 0;
        for (int j = 0; j < sidx; j++)
          if (DP_A[sidx][j] != 0.0) { cb.k[cb.n] = h->mu_k[j][i]; cb.c[cb.n] = dt * DP_A[sidx][j]; cb.n++; }
        TDVP_LAUNCH(lincomb_kernel, grid_for(site_elems(h, i)), VT, 0, st, h->mu_y[i], (const c128 *)h->A[i], cb,
                    site_elems(h, i));
      }
      Y = &h->mu_y;
    }
    if (int rc = mu_rhs(h, *Y, h->mu_k[sidx])) return rc;
  }
  void *scratch = h->step_ws;
  for (int i = 0; i < n; i++) {
    Comb ce{}; ce.n = 0;
    for (int j = 0; j < 7; j++)
      if (DP_B5[j] - DP_B4[j] != 0.0) { ce.k[ce.n] = h->mu_k[j][i]; ce.c[ce.n] = dt * (DP_B5[j] - DP_B4[j]); ce.n++; }
    TDVP_LAUNCH(lincomb_kernel, grid_for(site_elems(h, i)), VT, 0, st, h->mu_y[i], (const c128 *)nullptr, ce, site_elems(h, i));
    vec_norm_sq(st, h->mu_y[i], site_elems(h, i), h->mu_err_dev + 1 + i, scratch);
    Comb cb{}; cb.n = 0;
    for (int j = 0; j < 7; j++)
      if (DP_B5[j] != 0.0) { cb.k[cb.n] = h->mu_k[j][i]; cb.c[cb.n] = dt * DP_B5[j]; cb.n++; }
    TDVP_LAUNCH(lincomb_kernel, grid_for(site_elems(h, i)), VT, 0, st, h->A[i], (const c128 *)h->A[i], cb, site_elems(h, i));
  }
  TDVP_LAUNCH(err_final_kernel, 1, 1, 0, st, h->mu_err_dev + 1, n, h->mu_err_dev);
  if (int rc = check_cuda(h, cudaGetLastError(), "tdvp_step_mu")) return rc;
  h->mu_fsal = true;
  return TDVP_OK;
}


// ---------------------------------------------------------------------------------------------
// TDVP-MU with constant-mean-field (CMF) integration, second-order midpoint scheme
// (cost PAPER.md:253 and Table I; readings: DESIGN.md c19).
// The mean field of site j < N-1 is (h[1:j-1], h[j+1:N] rebuilt from the R of Eq. 36, U, Lambda of
// the bond to its right); it is held constant while L_j is integrated by classical RK4 sub-steps of
//     i dL_j/dt = (1 - L_j L_j^dagger) H[j](L_j U Lambda) Lambda~^{-1} U^dagger       (Eq. 37, 33, 38)
// and C_N by the Lanczos exponential of Eq. 27.  One step: mean field at t = 0 -> every local
// matrix to tau/2 -> mean field there -> every local matrix from 0 to tau with that mean field.
// SVDs and environment updates run twice per step, whatever the number of local sub-steps.
struct CmfFields {                 // per bond b = 1..n-1 (between sites b-1 and b): U, U*Lambda, Lambda
  std::vector<c128 *> U, UL;
  std::vector<double *> lam;
};

int cmf_alloc(tdvp_handle *h) {
  if (!h->cmf_mem.empty()) return TDVP_OK;
  const int n = h->n;
  h->cmf_mem.assign(3 * n, nullptr);
  for (int b = 1; b < n; b++) {
    const size_t m = (size_t)h->M[b];
    if (int rc = check_cuda(h, cudaMalloc(&h->cmf_mem[3 * b], m * m * 16), "cudaMalloc CMF U")) return rc;
    if (int rc = check_cuda(h, cudaMalloc(&h->cmf_mem[3 * b + 1], m * m * 16), "cudaMalloc CMF U Lambda")) return rc;
    if (int rc = check_cuda(h, cudaMalloc(&h->cmf_mem[3 * b + 2], m * 8), "cudaMalloc CMF Lambda")) return rc;
  }
  return TDVP_OK;
}

// Mean fields of the left-canonical state Y: Lenv[i] for every site, Renv[j] / U / Lambda for j < n-1.
// `released(j)` (optional) is called as soon as everything the local problem of site j reads has been enqueued on
// h->stream -- L[j] from the forward pass, R[j] and U, Lambda of the bond to its right from the backward pass at bond
// j + 1 -- i.e. while the unfoldings of the bonds further left are still to come: the caller starts site j there.
int cmf_mean_fields(tdvp_handle *h, const std::vector<c128 *> &Y, const std::function<void(int)> &released = nullptr) {
  cudaStream_t st = h->stream;
  const int n = h->n;
  MuScratch s = mu_scratch(h);
  if (!s.U) return set_err(h, TDVP_ENOMEM, "TDVP-MU scratch allocation failed");
  void *ws = h->step_ws;
  for (int i = 0; i < n - 1; i++)                                                        // "Get Env"
    env_update(st, 0, h->M[i], h->M[i + 1], h->d[i], h->Dw[i], h->Dw[i + 1], h->Lenv[i], h->Wsp[i], Y[i],
               h->Lenv[i + 1], ws);
  // The backward pass.  On the chain (queue st): R factor of the centre, Jacobi iteration, U Lambda, the next centre.
  // Off the chain, one bond behind it on the queue cmf_env when the handle has one: Q and Vh of the bond, the R block
  // built from Vh, and with that the release of site i - 1 (event cmf_rel[i - 1]).  The unfolding workspaces alternate
  // with the bond's parity: bond i's first half waits until bond i + 2's second half has let go of the workspace.
  cudaStream_t eq = (h->cmf_env && released) ? h->cmf_env : st;
  const bool split = eq != st;
  const c128 *C = Y[n - 1];
  c128 *Cnext = s.C0;
  for (int i = n - 1; i >= 1; i--) {
    const int Ml = h->M[i], Mr = h->M[i + 1], d = h->d[i];
    c128 *U = reinterpret_cast<c128 *>(h->cmf_mem[3 * i]), *UL = reinterpret_cast<c128 *>(h->cmf_mem[3 * i + 1]);
    double *lam = reinterpret_cast<double *>(h->cmf_mem[3 * i + 2]);
    void *sws = split ? h->cmf_svd_ws[i & 1] : ws;
    if (split && i + 2 <= n - 1) cudaStreamWaitEvent(st, h->cmf_rel[i + 1], 0);
    svd_bond_factor(st, Ml, d, Mr, C, U, lam, sws, h->status_dev);                                     // Eq. 36
    vec_copy(st, UL, U, (long long)Ml * Ml);
    TDVP_LAUNCH(scale_cols_kernel, grid_for((long long)Ml * Ml), VT, 0, st, UL, (long long)Ml, Ml, lam, 0, 0.0);
    if (split) { cudaEventRecord(h->cmf_fac[i], st); cudaStreamWaitEvent(eq, h->cmf_fac[i], 0); }
    svd_bond_vh(eq, Ml, d, Mr, s.Vh, sws);
    env_update(eq, 1, Ml, Mr, d, h->Dw[i], h->Dw[i + 1], h->Renv[i], h->Wsp[i], s.Vh, h->Renv[i - 1], split ? h->cmf_env_ws : ws);
    if (released) {
      cudaEventRecord(h->cmf_rel[i - 1], eq);              // the mean fields of site i - 1 are ready
      released(i - 1);
    }
    if (i > 1) {                                           // centre form of site i-1, unfolded next
      const int j = i - 1;
      ZGemm g{};
      g.A = Y[j]; g.B = UL; g.C = Cnext;
      g.M = h->M[j] * h->d[j]; g.K = Ml; g.N = Ml; g.a_ms = Ml; g.a_ks = 1; g.b_ks = Ml; g.b_ns = 1; g.ldc = Ml;
      gemm1(st, g);
      C = Cnext;
      Cnext = (Cnext == s.C0) ? s.C1 : s.C0;
    }
  }
  if (split && n >= 2) cudaStreamWaitEvent(st, h->cmf_rel[0], 0);   // the environment queue joins the chain again
  return check_cuda(h, cudaGetLastError(), "CMF mean fields");
}

// K = dL_j/dt of Eq. 37 at the local matrix Yj, mean fields of site j held in the handle.
void cmf_local_rhs(tdvp_handle *h, int j, const c128 *Yj, c128 *K, const MuScratch &s, cudaStream_t st, void *ws) {
  const double sq = std::sqrt(h->opt.mu_eps);
  const int Jl = h->M[j], Jr = h->M[j + 1], dj = h->d[j];
  const long long ne = site_elems(h, j), rows = (long long)Jl * dj;
  const c128 *U = reinterpret_cast<const c128 *>(h->cmf_mem[3 * (j + 1)]);
  const c128 *UL = reinterpret_cast<const c128 *>(h->cmf_mem[3 * (j + 1) + 1]);
  const double *lam = reinterpret_cast<const double *>(h->cmf_mem[3 * (j + 1) + 2]);
  ZGemm g{};
  g.A = Yj; g.B = UL; g.C = s.C0;                          // C[(a,s)][r] = sum_l L[(a,s)][l] (U Lambda)[l][r]
  g.M = (int)rows; g.K = Jr; g.N = Jr; g.a_ms = Jr; g.a_ks = 1; g.b_ks = Jr; g.b_ns = 1; g.ldc = Jr;
  gemm1(st, g);
  heff_apply(st, Jl, Jr, dj, h->Dw[j], h->Dw[j + 1], h->Lenv[j], h->Wsp[j], s.C0, h->Renv[j], s.HC, ws);
  TDVP_LAUNCH(scale_cols_kernel, grid_for(ne), VT, 0, st, s.HC, rows, Jr, lam, 1, sq);   // Lambda~^{-1}, Eq. 38
  ZGemm g2{};
  g2.A = s.HC; g2.B = U; g2.C = s.G;                       // G = HC U^dagger
  g2.M = (int)rows; g2.K = Jr; g2.N = Jr; g2.a_ms = Jr; g2.a_ks = 1; g2.b_ns = Jr; g2.b_ks = 1; g2.conjB = 1; g2.ldc = Jr;
  gemm1(st, g2);
  ZGemm g3{};
  g3.A = Yj; g3.B = s.G; g3.C = s.P;                       // P = L^dagger G
  g3.M = Jr; g3.N = Jr; g3.K = (int)rows; g3.a_ms = 1; g3.a_ks = Jr; g3.conjA = 1; g3.b_ks = Jr; g3.b_ns = 1; g3.ldc = Jr;
  gemm1(st, g3);
  ZGemm g4{};
  g4.A = Yj; g4.B = s.P; g4.C = s.T;                       // T = L P
  g4.M = (int)rows; g4.K = Jr; g4.N = Jr; g4.a_ms = Jr; g4.a_ks = 1; g4.b_ks = Jr; g4.b_ns = 1; g4.ldc = Jr;
  gemm1(st, g4);
  TDVP_LAUNCH(minus_i_diff_kernel, grid_for(ne), VT, 0, st, K, s.G, s.T, ne);             // -i (1 - p) G
}

// Side queues for the local propagation: once the mean fields are fixed the local problems of
// different sites are independent, and each is a chain of small GEMMs that leaves
// most of the GPU idle, so sites are dealt round-robin to a few queues, each with its own scratch.
int cmf_queues(tdvp_handle *h) {
  if (!h->cmf_streams.empty()) return TDVP_OK;
  int nq = 6;
  if (const char *e = getenv("TDVP_CMF_QUEUES")) nq = atoi(e);
  if (nq < 1) nq = 1;
  if (nq > 16) nq = 16;
  if (int rc = check_cuda(h, cudaEventCreateWithFlags(&h->cmf_fork, cudaEventDisableTiming), "event")) return rc;
  {
    static const bool hi = [] { const char *e = getenv("TDVP_CMF_PRIORITY"); return !(e && e[0] == '0'); }();
    int least = 0, greatest = 0;
    if (hi && cudaDeviceGetStreamPriorityRange(&least, &greatest) == cudaSuccess && greatest != least) {
      if (int rc = check_cuda(h, cudaStreamCreateWithPriority(&h->cmf_hi, cudaStreamNonBlocking, greatest), "CMF mean-field queue")) return rc;
      if (int rc = check_cuda(h, cudaEventCreateWithFlags(&h->cmf_hi_done, cudaEventDisableTiming), "event")) return rc;
      zgemm_prepare_stream(h->cmf_hi);
    }
  }
  {
    // Vh of a bond and the R block built from it hang off the chain of unfoldings without being on it (the next
    // unfolding needs U Lambda only): they run on a queue of their own, one bond behind the chain
    static const bool split = [] { const char *e = getenv("TDVP_CMF_SPLIT_SVD"); return !(e && e[0] == '0'); }();
    if (split) {
      if (int rc = check_cuda(h, cudaStreamCreateWithFlags(&h->cmf_env, cudaStreamNonBlocking), "CMF environment queue")) return rc;
      zgemm_prepare_stream(h->cmf_env);
      if (int rc = check_cuda(h, cudaMalloc(&h->cmf_env_ws, h->step_ws_bytes), "cudaMalloc CMF workspace")) return rc;
      for (int k = 0; k < 2; k++)
        if (int rc = check_cuda(h, cudaMalloc(&h->cmf_svd_ws[k], h->step_ws_bytes), "cudaMalloc CMF workspace")) return rc;
      for (int j = 0; j < h->n; j++) {
        cudaEvent_t ev = nullptr;
        if (int rc = check_cuda(h, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming), "event")) return rc;
        h->cmf_fac.push_back(ev);
      }
    }
  }
  for (int j = 0; j < h->n; j++) {                           // "mean fields of site j are ready"
    cudaEvent_t ev = nullptr;
    if (int rc = check_cuda(h, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming), "event")) return rc;
    h->cmf_rel.push_back(ev);
  }
  for (int q = 0; q < nq; q++) {
    cudaStream_t st = nullptr; cudaEvent_t ev = nullptr; void *ws = nullptr, *sc = nullptr;
    if (int rc = check_cuda(h, cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking), "CMF queue")) return rc;
    if (int rc = check_cuda(h, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming), "event")) return rc;
    if (int rc = check_cuda(h, cudaMalloc(&ws, h->step_ws_bytes), "cudaMalloc CMF workspace")) return rc;
    if (int rc = check_cuda(h, cudaMalloc(&sc, mu_scratch_bytes(h, nullptr, nullptr)), "cudaMalloc CMF scratch")) return rc;
    zgemm_prepare_stream(st);
    // the side queues run beside the unfolding chain's cluster kernels (16 SMs for a QR, 8 for the Jacobi sweeps, up
    // to 2 ms each): their GEMMs leave those SMs out of their grids, or every cut (cooperative) launch would wait
    {
      static const int spare = [] { const char *e = getenv("TDVP_CMF_SPARE_SMS"); return e ? atoi(e) : 24; }();
      const int sms = zgemm_device_sms();
      if (spare > 0 && sms > 2 * spare) zgemm_set_stream_cap(st, 2 * (sms - spare));
      // ... and beyond that a quarter of the device's CTA slots each (TDVP_CMF_QUEUE_CTAS, default SMs / 2): with every
      // queue's GEMMs spread over all slots the queues took turns and each launch's ramp and drain stayed exposed; on a
      // share of its own a queue's kernels overlap the others' (measured, six queues: 498 -> 467 ms per CMF step for
      // 48..90 CTAs per queue, 6..12 queues alike)
      {
        static const int qc = [] { const char *ec = getenv("TDVP_CMF_QUEUE_CTAS"); return ec ? atoi(ec) : -1; }();
        const int c = qc >= 0 ? qc : sms / 2;
        if (c > 0) zgemm_set_stream_cap(st, c);
      }
    }
    h->cmf_streams.push_back(st); h->cmf_join.push_back(ev); h->cmf_ws.push_back(ws); h->cmf_scratch.push_back(sc);
  }
  if (h->cmf_env) {                                          // (the same grid cap as the side queues, for the same reason)
    const char *e = getenv("TDVP_CMF_SPARE_SMS");
    const int spare = e ? atoi(e) : 24, sms = zgemm_device_sms();
    if (spare > 0 && sms > 2 * spare) zgemm_set_stream_cap(h->cmf_env, 2 * (sms - spare));
  }
  return TDVP_OK;
}

// RK4 sub-steps of site j on queue st
void cmf_site(tdvp_handle *h, int j, const c128 *Xj, c128 *y, double t, int n_sub, const MuScratch &s, cudaStream_t st, void *ws) {
  const double hs = t / n_sub;
  const long long ne = site_elems(h, j);
  c128 *ys = h->mu_y[j];
  c128 *k1 = h->mu_k[0][j], *k2 = h->mu_k[1][j], *k3 = h->mu_k[2][j], *k4 = h->mu_k[3][j];
  vec_copy(st, y, Xj, ne);
  for (int q = 0; q < n_sub; q++) {                        // classical RK4
    cmf_local_rhs(h, j, y, k1, s, st, ws);
    { Comb c{}; c.n = 1; c.k[0] = k1; c.c[0] = 0.5 * hs;
      TDVP_LAUNCH(lincomb_kernel, grid_for(ne), VT, 0, st, ys, (const c128 *)y, c, ne); }
    cmf_local_rhs(h, j, ys, k2, s, st, ws);
    { Comb c{}; c.n = 1; c.k[0] = k2; c.c[0] = 0.5 * hs;
      TDVP_LAUNCH(lincomb_kernel, grid_for(ne), VT, 0, st, ys, (const c128 *)y, c, ne); }
    cmf_local_rhs(h, j, ys, k3, s, st, ws);
    { Comb c{}; c.n = 1; c.k[0] = k3; c.c[0] = hs;
      TDVP_LAUNCH(lincomb_kernel, grid_for(ne), VT, 0, st, ys, (const c128 *)y, c, ne); }
    cmf_local_rhs(h, j, ys, k4, s, st, ws);
    { Comb c{}; c.n = 4; c.k[0] = k1; c.k[1] = k2; c.k[2] = k3; c.k[3] = k4;
      c.c[0] = hs / 6.0; c.c[1] = hs / 3.0; c.c[2] = hs / 3.0; c.c[3] = hs / 6.0;
      TDVP_LAUNCH(lincomb_kernel, grid_for(ne), VT, 0, st, y, (const c128 *)y, c, ne); }
  }
}

// The right-hand side with the same pipeline as the CMF step below: the bond unfoldings (Eq. 36) are a sequential
// chain, site j's share of Eq. 37 (the H_eff apply and four GEMMs) needs only the bond to its right -- it runs on a
// side queue as soon as that bond is done, with the per-bond U, Lambda kept in the handle (cmf_mem) instead of one
// scratch copy the next unfolding overwrites.  Same kernels on the same data as mu_rhs_serial.
int mu_rhs_pipelined(tdvp_handle *h, const std::vector<c128 *> &Y, const std::vector<c128 *> &K) {
  cudaStream_t st = h->stream;
  const int n = h->n;
  const int nq = (int)h->cmf_streams.size();
  cudaStream_t mf = h->cmf_hi ? h->cmf_hi : st;
  if (mf != st) { cudaEventRecord(h->cmf_fork, st); cudaStreamWaitEvent(mf, h->cmf_fork, 0); }
  h->stream = mf;
  const int rc = cmf_mean_fields(h, Y, [&](int j) {
    const int q = j % nq;
    cudaStreamWaitEvent(h->cmf_streams[q], h->cmf_rel[j], 0);
    cmf_local_rhs(h, j, Y[j], K[j], mu_carve(h, h->cmf_scratch[q]), h->cmf_streams[q], h->cmf_ws[q]);
  });
  h->stream = st;
  if (mf != st) { cudaEventRecord(h->cmf_hi_done, mf); cudaStreamWaitEvent(st, h->cmf_hi_done, 0); }
  if (rc) return rc;
  {                                                                                      // Eq. 27
    const int i = n - 1;
    MuScratch s = mu_scratch(h);
    heff_apply(st, h->M[i], h->M[i + 1], h->d[i], h->Dw[i], h->Dw[i + 1], h->Lenv[i], h->Wsp[i], Y[i], h->Renv[i],
               s.HC, h->step_ws);
    TDVP_LAUNCH(minus_i_diff_kernel, grid_for(site_elems(h, i)), VT, 0, st, K[i], s.HC, (const c128 *)nullptr,
                site_elems(h, i));
  }
  for (int q = 0; q < nq && q < n - 1; q++) {
    cudaEventRecord(h->cmf_join[q], h->cmf_streams[q]);
    cudaStreamWaitEvent(st, h->cmf_join[q], 0);
  }
  return check_cuda(h, cudaGetLastError(), "TDVP-MU derivative");
}

// Mean fields of the state Y, then Z[i] = every local matrix of X propagated over time t with them.  The two are
// pipelined: the backward pass of the mean-field build is a chain of bond unfoldings (one 8-SM cluster kernel at a
// time, ~2.5 ms per bond at M = 128), and site j's local problem needs nothing left of bond j + 1 -- so site j starts
// on its side queue the moment that bond is done (an event per site), and the local propagation, which is where the
// step's GEMM work is, fills the SMs the unfolding chain leaves idle.  Same kernels in the same order on every
// queue: bit-identical to running the two phases one after the other (TDVP_CMF_PIPELINE=0).
int cmf_fields_and_propagate(tdvp_handle *h, const std::vector<c128 *> &Y, const std::vector<c128 *> &X, const std::vector<c128 *> &Z,
                             double t, int n_sub) {
  cudaStream_t st = h->stream;
  const int n = h->n;
  const int nq = (int)h->cmf_streams.size();
  static const bool pipeline = [] { const char *e = getenv("TDVP_CMF_PIPELINE"); return !(e && e[0] == '0'); }();
  auto start_site = [&](int j) {
    const int q = j % nq;
    cmf_site(h, j, X[j], Z[j], t, n_sub, mu_carve(h, h->cmf_scratch[q]), h->cmf_streams[q], h->cmf_ws[q]);
  };
  if (pipeline) {
    // the unfolding chain is the critical path: it runs on a queue of its own with the highest priority, so that its
    // short cluster kernels are scheduled ahead of the side queues' GEMM CTAs whenever SMs come free
    cudaStream_t mf = h->cmf_hi ? h->cmf_hi : st;
    if (mf != st) { cudaEventRecord(h->cmf_fork, st); cudaStreamWaitEvent(mf, h->cmf_fork, 0); }
    h->stream = mf;
    const int rc = cmf_mean_fields(h, Y, [&](int j) {          // (cmf_rel[j] has been recorded: mean fields of site j are ready)
      cudaStreamWaitEvent(h->cmf_streams[j % nq], h->cmf_rel[j], 0);
      start_site(j);
    });
    h->stream = st;
    if (mf != st) { cudaEventRecord(h->cmf_hi_done, mf); cudaStreamWaitEvent(st, h->cmf_hi_done, 0); }
    if (rc) return rc;
  } else {
    if (int rc = cmf_mean_fields(h, Y)) return rc;
    cudaEventRecord(h->cmf_fork, st);
    for (int q = 0; q < nq && q < n - 1; q++) cudaStreamWaitEvent(h->cmf_streams[q], h->cmf_fork, 0);
    for (int j = 0; j < n - 1; j++) start_site(j);
  }
  {                                                        // Eq. 27 by the Krylov exponential
    const int i = n - 1;
    LanczosOp op{};
    op.kind = 0; op.Ml = h->M[i]; op.Mr = h->M[i + 1]; op.d = h->d[i]; op.Dl = h->Dw[i]; op.Dr = h->Dw[i + 1];
    op.L = h->Lenv[i]; op.R = h->Renv[i]; op.W = &h->Wsp[i];
    lanczos_expm(st, op, h->opt.krylov_dim, h->opt.krylov_tol, 0.0, -t, X[i], Z[i], h->step_ws, nullptr, h->status_dev);
  }
  for (int q = 0; q < nq && q < n - 1; q++) {
    cudaEventRecord(h->cmf_join[q], h->cmf_streams[q]);
    cudaStreamWaitEvent(st, h->cmf_join[q], 0);
  }
  return check_cuda(h, cudaGetLastError(), "CMF local propagation");
}

int enqueue_cmf_step(tdvp_handle *h, double dt, int n_sub) {
  h->mu_fsal = false;
  if (int rc = cmf_fields_and_propagate(h, h->A, h->A, h->mu_k[4], 0.5 * dt, (n_sub + 1) / 2)) return rc;
  if (int rc = cmf_fields_and_propagate(h, h->mu_k[4], h->A, h->mu_k[5], dt, n_sub)) return rc;
  for (int i = 0; i < h->n; i++) vec_copy(h->stream, h->A[i], h->mu_k[5][i], site_elems(h, i));
  return check_cuda(h, cudaGetLastError(), "tdvp_step_mu_cmf");
}

int prepare_mu(tdvp_handle *h) {
  if (!h || h->n < 1) return set_err(h, TDVP_EINVAL, "handle has no chain");
  if (h->n < 2) return set_err(h, TDVP_EINVAL, "TDVP-MU needs at least two sites");
  if (int rc = mu_alloc(h)) return rc;
  if (!getenv("TDVP_MU_PIPELINE") || getenv("TDVP_MU_PIPELINE")[0] != '0') {   // per-bond U, Lambda and the side queues of mu_rhs
    if (int rc = cmf_alloc(h)) return rc;
    if (int rc = cmf_queues(h)) return rc;
  }
  return TDVP_OK;
}

}  // namespace

extern "C" {

int tdvp_step_mu(tdvp_handle *h, double dt, double *err_est) {
  if (int rc = prepare_mu(h)) return rc;
  if (h->centre != h->n - 1) {
    if (int rc = move_gauge(h, h->n - 1)) return rc;
  }
  if (int rc = enqueue_mu_step(h, dt)) return rc;
  if (err_est) {
    if (int rc = check_cuda(h, cudaMemcpyAsync(err_est, h->mu_err_dev, sizeof(double), cudaMemcpyDeviceToHost, h->stream), "memcpy")) return rc;
    return finish_blocking(h, "tdvp_step_mu");
  }
  return TDVP_OK;
}

int tdvp_step_mu_cmf(tdvp_handle *h, double dt, int n_sub) {
  if (int rc = prepare_mu(h)) return rc;
  if (n_sub < 1) return set_err(h, TDVP_EINVAL, "n_sub must be >= 1");
  if (int rc = cmf_alloc(h)) return rc;
  if (int rc = cmf_queues(h)) return rc;
  if (h->centre != h->n - 1) {
    if (int rc = move_gauge(h, h->n - 1)) return rc;
  }
  // one CUDA graph per (dt, n_sub): the ~46 000 launches of a step of the 71-site chain, the four side queues of the
  // local propagation as parallel branches, cost one graph launch on the host
  if (!mu_scratch(h).U) return set_err(h, TDVP_ENOMEM, "TDVP-MU scratch allocation failed");   // (allocates on first use: not inside a capture)
  int rc_enq = TDVP_OK;
  h->mu_fsal = false;
  const int rc = run_step(h, h->cmf_graph, dt, [&] { rc_enq = enqueue_cmf_step(h, dt, n_sub); }, "tdvp_step_mu_cmf", n_sub);
  return rc_enq != TDVP_OK ? rc_enq : rc;
}

int tdvp_mu_derivative(tdvp_handle *h, tdvp_c128 *const *out_host) {
  if (int rc = prepare_mu(h)) return rc;
  if (!out_host) return set_err(h, TDVP_EINVAL, "null pointer");
  if (h->centre != h->n - 1) return set_err(h, TDVP_ESTATE, "tdvp_mu_derivative needs the MU gauge (centre N-1): call tdvp_set_gauge");
  if (int rc = mu_rhs(h, h->A, h->mu_k[0])) return rc;
  for (int i = 0; i < h->n; i++) {
    if (!out_host[i]) return set_err(h, TDVP_EINVAL, "null output tensor");
    if (int rc = check_cuda(h, cudaMemcpyAsync(out_host[i], h->mu_k[0][i], site_elems(h, i) * 16, cudaMemcpyDeviceToHost, h->stream), "memcpy")) return rc;
  }
  return finish_blocking(h, "tdvp_mu_derivative");
}

int tdvp_svd_bond(tdvp_handle *h, int Ml, int d, int Mr, const tdvp_c128 *C, tdvp_c128 *U, double *lam, tdvp_c128 *Vh) {
  tdvp_handle *hh = h ? h : default_handle();
  if (!C || !U || !lam || !Vh) return set_err(h, TDVP_EINVAL, "null pointer");
  if (Ml < 1 || d < 1 || Mr < 1) return set_err(h, TDVP_EINVAL, "dimensions must be >= 1");
  if ((long long)d * Mr < Ml) return set_err(h, TDVP_EINVAL, "matrix unfolding needs Ml <= d*Mr");
  if ((long long)d * Mr > QR_MAX_TALL) return set_err(h, TDVP_EINVAL, "matrix unfolding: d*Mr above 12800 is not supported");
  size_t sb = svd_ws_bytes(Ml, d, Mr);
  if (int rc = check_cuda(h, hh->arena.reserve(sb + 1024, hh->stream), "workspace")) return rc;
  hh->arena.reset();
  void *ws = hh->arena.take(sb);
  svd_bond(hh->stream, Ml, d, Mr, reinterpret_cast<const c128 *>(C), reinterpret_cast<c128 *>(U), lam,
           reinterpret_cast<c128 *>(Vh), ws, hh->status_dev);
  return check_cuda(h, cudaGetLastError(), "tdvp_svd_bond");
}

}  // extern "C"
