// observe.cu -- observables on the resident MPS: one-site reduced density
// matrix / site populations P^(n)(t), norm, energy; tdvp_get_mps / tdvp_set_mps.
// Identity transfer matrices are contracted from both ends over ALL sites (no canonical-form
// shortcut), so the result is gauge-agnostic: it also serves the slowly drifting gauge of TDVP-MU
// (PAPER.md:220).
#include <algorithm>
#include <vector>

#include "handle.cuh"

int chain_rebuild_right_envs(tdvp_handle *h);
int chain_rebuild_left_envs(tdvp_handle *h);
int chain_canonical_defect(tdvp_handle *h, int side, int lo, int hi, double *defect);

namespace {

__global__ void set_one_k(c128 *p) { p[0] = make_double2(1.0, 0.0); }

// rho[s][t] = sum_{a,b} T2[a,s,b] conj(A[a,t,b]);  one CTA per (s,t)
__global__ void rdm_kernel(const c128 *T2, const c128 *A, int Ml, int d, int Mr, c128 *rho) {
  const int s = blockIdx.x / d, t = blockIdx.x % d;
  double sx = 0.0, sy = 0.0;
  const long long n = (long long)Ml * Mr;
  for (long long e = threadIdx.x; e < n; e += blockDim.x) {
    long long a = e / Mr, b = e % Mr;
    c128 x = T2[(a * d + s) * Mr + b], y = A[(a * d + t) * Mr + b];
    sx += x.x * y.x + x.y * y.y;
    sy += x.y * y.x - x.x * y.y;
  }
  __shared__ double rx[256], ry[256];
  rx[threadIdx.x] = sx; ry[threadIdx.x] = sy;
  __syncthreads();
  for (int k = blockDim.x / 2; k > 0; k >>= 1) {
    if (threadIdx.x < k) { rx[threadIdx.x] += rx[threadIdx.x + k]; ry[threadIdx.x] += ry[threadIdx.x + k]; }
    __syncthreads();
  }
  if (threadIdx.x == 0) rho[blockIdx.x] = make_double2(rx[0], ry[0]);
}

void gemm1(tdvp_handle *h, const ZGemm &g) { zgemm(h->stream, g); }

// E'[b][y] = sum_{a,x,s} conj(A[a,s,b]) E[a][x] A[x,s,y]
void transfer_left(tdvp_handle *h, int i, const c128 *E, c128 *Eout, c128 *T) {
  const int Ml = h->M[i], Mr = h->M[i + 1], d = h->d[i];
  ZGemm g{};
  g.A = E; g.B = h->A[i]; g.C = T;                       // T[a][(s,y)] = sum_x E[a][x] A[x][(s,y)]
  g.M = Ml; g.K = Ml; g.N = d * Mr; g.a_ms = Ml; g.a_ks = 1; g.b_ks = g.N; g.b_ns = 1; g.ldc = g.N;
  gemm1(h, g);
  ZGemm q{};
  q.A = h->A[i]; q.B = T; q.C = Eout;                    // E'[b][y] = sum_{(a,s)} conj(A[(a,s)][b]) T[(a,s)][y]
  q.M = Mr; q.N = Mr; q.K = Ml * d; q.a_ms = 1; q.a_ks = Mr; q.conjA = 1; q.b_ks = Mr; q.b_ns = 1; q.ldc = Mr;
  gemm1(h, q);
}
// E'[a][x] = sum_{s,b,y} conj(A[a,s,b]) E[b][y] A[x,s,y]
void transfer_right(tdvp_handle *h, int i, const c128 *E, c128 *Eout, c128 *T) {
  const int Ml = h->M[i], Mr = h->M[i + 1], d = h->d[i];
  ZGemm g{};
  g.A = h->A[i]; g.B = E; g.C = T;                       // T[(x,s)][b] = sum_y A[(x,s)][y] E[b][y]
  g.M = Ml * d; g.K = Mr; g.N = Mr; g.a_ms = Mr; g.a_ks = 1; g.b_ns = Mr; g.b_ks = 1; g.ldc = Mr;
  gemm1(h, g);
  ZGemm q{};
  q.A = h->A[i]; q.B = T; q.C = Eout;                    // E'[a][x] = sum_{(s,b)} conj(A[a][(s,b)]) T[x][(s,b)]
  q.M = Ml; q.N = Ml; q.K = d * Mr; q.a_ms = q.K; q.a_ks = 1; q.conjA = 1; q.b_ns = q.K; q.b_ks = 1; q.ldc = Ml;
  gemm1(h, q);
}

// one-site RDM at `site` -> host rho[d*d] (rho[s][t] = sum psi_s conj(psi_t)).  Blocks.
int site_rdm(tdvp_handle *h, int site, std::vector<c128> &rho) {
  int maxM = *std::max_element(h->M.begin(), h->M.end());
  char *p = reinterpret_cast<char *>(h->step_ws);
  auto up = [](size_t x) { return (x + 255) & ~size_t(255); };
  c128 *E0 = reinterpret_cast<c128 *>(p); p += up((size_t)maxM * maxM * 16);
  c128 *E1 = reinterpret_cast<c128 *>(p); p += up((size_t)maxM * maxM * 16);
  c128 *Er = reinterpret_cast<c128 *>(p); p += up((size_t)maxM * maxM * 16);
  c128 *Er1 = reinterpret_cast<c128 *>(p); p += up((size_t)maxM * maxM * 16);
  c128 *rho_dev = reinterpret_cast<c128 *>(p); p += up((size_t)h->d[site] * h->d[site] * 16);
  c128 *T = h->tmpA, *T2 = h->tmpB;
  cudaStream_t st = h->stream;
  TDVP_LAUNCH(set_one_k, 1, 1, 0, st, E0);
  c128 *El = E0, *Eln = E1;
  for (int i = 0; i < site; i++) { transfer_left(h, i, El, Eln, T); std::swap(El, Eln); }
  TDVP_LAUNCH(set_one_k, 1, 1, 0, st, Er);
  c128 *Ec = Er, *Ecn = Er1;
  for (int i = h->n - 1; i > site; i--) { transfer_right(h, i, Ec, Ecn, T); std::swap(Ec, Ecn); }
  const int Ml = h->M[site], Mr = h->M[site + 1], d = h->d[site];
  ZGemm g{};
  g.A = El; g.B = h->A[site]; g.C = T;                    // T[a][(s,y)] = sum_x El[a][x] A[x][(s,y)]
  g.M = Ml; g.K = Ml; g.N = d * Mr; g.a_ms = Ml; g.a_ks = 1; g.b_ks = g.N; g.b_ns = 1; g.ldc = g.N;
  gemm1(h, g);
  ZGemm q{};
  q.A = T; q.B = Ec; q.C = T2;                            // T2[(a,s)][b] = sum_y T[(a,s)][y] Er[b][y]
  q.M = Ml * d; q.K = Mr; q.N = Mr; q.a_ms = Mr; q.a_ks = 1; q.b_ns = Mr; q.b_ks = 1; q.ldc = Mr;
  gemm1(h, q);
  TDVP_LAUNCH(rdm_kernel, d * d, 256, 0, st, T2, h->A[site], Ml, d, Mr, rho_dev);
  rho.resize((size_t)d * d);
  if (int rc = check_cuda(h, cudaMemcpyAsync(rho.data(), rho_dev, (size_t)d * d * 16, cudaMemcpyDeviceToHost, st), "memcpy")) return rc;
  return finish_blocking(h, "site observable");
}

}  // namespace

extern "C" {

int tdvp_observe(tdvp_handle *h, int site, const tdvp_c128 *op, tdvp_c128 *out) {
  if (!h || h->n < 1) return set_err(h, TDVP_EINVAL, "handle has no chain");
  if (site < 0 || site >= h->n || !op || !out) return set_err(h, TDVP_EINVAL, "bad site or null pointer");
  std::vector<c128> rho;
  if (int rc = site_rdm(h, site, rho)) return rc;
  const int d = h->d[site];
  double sx = 0.0, sy = 0.0;
  for (int s = 0; s < d; s++)
    for (int t = 0; t < d; t++) {                           // <O> = sum O[s][t] rho[t][s]
      c128 r = rho[(size_t)t * d + s];
      sx += op[s * d + t].re * r.x - op[s * d + t].im * r.y;
      sy += op[s * d + t].re * r.y + op[s * d + t].im * r.x;
    }
  out->re = sx; out->im = sy;
  return TDVP_OK;
}

int tdvp_populations(tdvp_handle *h, int site, double *out) {
  if (!h || h->n < 1) return set_err(h, TDVP_EINVAL, "handle has no chain");
  if (site < 0 || site >= h->n || !out) return set_err(h, TDVP_EINVAL, "bad site or null pointer");
  std::vector<c128> rho;
  if (int rc = site_rdm(h, site, rho)) return rc;
  const int d = h->d[site];
  for (int s = 0; s < d; s++) out[s] = rho[(size_t)s * d + s].x;
  return TDVP_OK;
}

int tdvp_norm_energy(tdvp_handle *h, double *norm_sq, double *energy) {
  if (!h || h->n < 1) return set_err(h, TDVP_EINVAL, "handle has no chain");
  if (norm_sq) {
    std::vector<c128> rho;
    if (int rc = site_rdm(h, 0, rho)) return rc;
    double t = 0.0;
    for (int s = 0; s < h->d[0]; s++) t += rho[(size_t)s * h->d[0] + s].x;
    *norm_sq = t;
  }
  if (energy) {
    // <psi|H|psi>: the full network contracted left to right (Eq. 30); scratch environments live
    // in the arena so that the cached blocks stay untouched.
    int maxM = *std::max_element(h->M.begin(), h->M.end());
    int maxD = *std::max_element(h->Dw.begin(), h->Dw.end());
    size_t eb = ((size_t)maxM * maxD * maxM * 16 + 255) & ~size_t(255);
    if (int rc = check_cuda(h, h->arena.reserve(2 * eb + 1024, h->stream), "workspace")) return rc;
    h->arena.reset();
    c128 *E0 = reinterpret_cast<c128 *>(h->arena.take(eb)), *E1 = reinterpret_cast<c128 *>(h->arena.take(eb));
    TDVP_LAUNCH(set_one_k, 1, 1, 0, h->stream, E0);
    for (int i = 0; i < h->n; i++) {
      env_update(h->stream, 0, h->M[i], h->M[i + 1], h->d[i], h->Dw[i], h->Dw[i + 1], E0, h->Wsp[i], h->A[i], E1, h->step_ws);
      std::swap(E0, E1);
    }
    c128 e;
    if (int rc = check_cuda(h, cudaMemcpyAsync(&e, E0, 16, cudaMemcpyDeviceToHost, h->stream), "memcpy")) return rc;
    if (int rc = finish_blocking(h, "tdvp_norm_energy")) return rc;
    *energy = e.x;
  }
  return TDVP_OK;
}

int tdvp_get_mps(tdvp_handle *h, int site, tdvp_c128 *out_host, int *Ml, int *Mr) {
  if (!h || h->n < 1) return set_err(h, TDVP_EINVAL, "handle has no chain");
  if (site < 0 || site >= h->n) return set_err(h, TDVP_EINVAL, "bad site");
  if (Ml) *Ml = h->M[site];
  if (Mr) *Mr = h->M[site + 1];
  if (!out_host) return TDVP_OK;
  size_t n = (size_t)h->M[site] * h->d[site] * h->M[site + 1];
  if (int rc = check_cuda(h, cudaMemcpyAsync(out_host, h->A[site], n * 16, cudaMemcpyDeviceToHost, h->stream), "memcpy")) return rc;
  return finish_blocking(h, "tdvp_get_mps");
}

int tdvp_set_mps(tdvp_handle *h, const tdvp_c128 *const *mps_host, int centre) {
  if (h) h->mu_fsal = false;
  if (!h || h->n < 1) return set_err(h, TDVP_EINVAL, "handle has no chain");
  if (!mps_host) return set_err(h, TDVP_EINVAL, "null pointer");
  if (centre != 0 && centre != h->n - 1) return set_err(h, TDVP_EINVAL, "centre must be 0 or N-1");
  for (int i = 0; i < h->n; i++) {
    if (!mps_host[i]) return set_err(h, TDVP_EINVAL, "null tensor");
    size_t n = (size_t)h->M[i] * h->d[i] * h->M[i + 1];
    if (int rc = check_cuda(h, cudaMemcpyAsync(h->A[i], mps_host[i], n * 16, cudaMemcpyHostToDevice, h->stream), "memcpy")) return rc;
  }
  if (int rc = check_cuda(h, cudaStreamSynchronize(h->stream), "tdvp_set_mps")) return rc;   // host buffers are free again
  h->centre = centre;
  if (!(h->opt.flags & TDVP_FLAG_SKIP_CANONICAL_CHECK) && h->n > 1) {
    double defect = 0.0;
    int rc = centre == 0 ? chain_canonical_defect(h, 1, 1, h->n, &defect) : chain_canonical_defect(h, 0, 0, h->n - 1, &defect);
    if (rc) return rc;
    if (!(defect <= 1e-10)) return set_err(h, TDVP_EINVAL, "MPS is not canonical around the stated centre");
  }
  return centre == 0 ? chain_rebuild_right_envs(h) : chain_rebuild_left_envs(h);
}

}  // extern "C"
