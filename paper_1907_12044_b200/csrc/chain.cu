// chain.cu -- the resident chain: tdvp_create / tdvp_destroy, the environment-block cache in HBM,
// the TDVP-PS step driver (Eq. 42-44) and the observables.
#include <algorithm>
#include <cmath>
#include <cstring>

#include "handle.cuh"

namespace {

inline size_t up256(size_t x) { return (x + 255) & ~size_t(255); }

long long site_elems(const tdvp_handle *h, int i) { return (long long)h->M[i] * h->d[i] * h->M[i + 1]; }
long long lenv_elems(const tdvp_handle *h, int i) { return (long long)h->M[i] * h->Dw[i] * h->M[i]; }
long long renv_elems(const tdvp_handle *h, int i) { return (long long)h->M[i + 1] * h->Dw[i + 1] * h->M[i + 1]; }

LanczosOp heff_op(const tdvp_handle *h, int i) {
  return LanczosOp{0, h->M[i], h->M[i + 1], h->d[i], h->Dw[i], h->Dw[i + 1], h->Lenv[i], h->Renv[i], &h->Wsp[i]};
}
// bond between sites b-1 and b (b = 1..n-1): L = Lenv[b], R = Renv[b-1]
LanczosOp bond_op(const tdvp_handle *h, int b) {
  return LanczosOp{1, h->M[b], h->M[b], 1, h->Dw[b], h->Dw[b], h->Lenv[b], h->Renv[b - 1], nullptr};
}

__global__ void set_one_kernel(c128 *p) { p[0] = make_double2(1.0, 0.0); }

// fmax drops a NaN operand; the canonical check must not (a tensor with NaN / Inf entries has no
// defect of zero): NaN if either is NaN, else the larger.
__device__ __forceinline__ double nan_max(double a, double b) { return (a != a || b != b) ? a + b : fmax(a, b); }

// max |G - I| over an n x n matrix -> out[0] (single block); NaN if G holds a non-finite entry
__global__ void max_dev_identity_kernel(const c128 *G, int n, double *out) {
  __shared__ double red[256];
  double m = 0.0;
  for (int e = threadIdx.x; e < n * n; e += blockDim.x) {
    int i = e / n, j = e % n;
    double dx = G[e].x - (i == j ? 1.0 : 0.0), dy = G[e].y;
    m = nan_max(m, nan_max(fabs(dx), fabs(dy)));           // Inf - Inf and 0 * Inf in the Gram matrix give NaN
  }
  red[threadIdx.x] = m;
  __syncthreads();
  for (int s = blockDim.x / 2; s > 0; s >>= 1) {
    if (threadIdx.x < s) red[threadIdx.x] = nan_max(red[threadIdx.x], red[threadIdx.x + s]);
    __syncthreads();
  }
  if (threadIdx.x == 0) out[0] = nan_max(out[0], red[0]);
}

}  // namespace

// Workspace needed by any single sub-step of a PS / MU step on this chain.
size_t chain_step_ws_bytes(const tdvp_handle *h) {
  size_t need = 0;
  const int k = h->opt.krylov_dim;
  for (int i = 0; i < h->n; i++) {
    need = std::max(need, lanczos_ws_bytes(heff_op(h, i), k));
    need = std::max(need, env_ws_bytes(h->M[i], h->M[i + 1], h->d[i], h->Dw[i], h->Dw[i + 1]));
    if (i < h->n - 1) need = std::max(need, qr_ws_bytes(h->M[i] * h->d[i], h->M[i + 1]));
    if (i > 0) {
      need = std::max(need, qr_ws_bytes(h->d[i] * h->M[i + 1], h->M[i]));
      need = std::max(need, lanczos_ws_bytes(bond_op(h, i), k));
      need = std::max(need, svd_ws_bytes(h->M[i], h->d[i], h->M[i + 1]));
    }
  }
  return need + 4096;
}

int chain_rebuild_right_envs(tdvp_handle *h) {
  for (int i = h->n - 1; i >= 1; i--)
    env_update(h->stream, 1, h->M[i], h->M[i + 1], h->d[i], h->Dw[i], h->Dw[i + 1], h->Renv[i], h->Wsp[i],
               h->A[i], h->Renv[i - 1], h->step_ws);
  return check_cuda(h, cudaGetLastError(), "right environments");
}
int chain_rebuild_left_envs(tdvp_handle *h) {
  for (int i = 0; i < h->n - 1; i++)
    env_update(h->stream, 0, h->M[i], h->M[i + 1], h->d[i], h->Dw[i], h->Dw[i + 1], h->Lenv[i], h->Wsp[i],
               h->A[i], h->Lenv[i + 1], h->step_ws);
  return check_cuda(h, cudaGetLastError(), "left environments");
}

// max over sites in [lo, hi) of || isometry condition - I ||_max.  side 1: right-canonical (Eq. 8),
// side 0: left-canonical (Eq. 7).  Blocks.
int chain_canonical_defect(tdvp_handle *h, int side, int lo, int hi, double *defect) {
  double *dev = reinterpret_cast<double *>(h->step_ws);
  c128 *G = reinterpret_cast<c128 *>(reinterpret_cast<char *>(h->step_ws) + 256);
  cudaMemsetAsync(dev, 0, sizeof(double), h->stream);
  for (int i = lo; i < hi; i++) {
    ZGemm g{};
    const int Ml = h->M[i], Mr = h->M[i + 1], d = h->d[i];
    g.A = h->A[i]; g.B = h->A[i]; g.C = G;
    if (side == 1) {        // G[a][a'] = sum_k A[a][k] conj(A[a'][k]),  k = (s, b)
      g.M = Ml; g.N = Ml; g.K = d * Mr;
      g.a_ms = (long long)d * Mr; g.a_ks = 1; g.b_ns = (long long)d * Mr; g.b_ks = 1; g.conjB = 1; g.ldc = Ml;
    } else {                // G[b][b'] = sum_k conj(A[k][b]) A[k][b'],  k = (a, s)
      g.M = Mr; g.N = Mr; g.K = Ml * d;
      g.a_ms = 1; g.a_ks = Mr; g.conjA = 1; g.b_ks = Mr; g.b_ns = 1; g.ldc = Mr;
    }
    zgemm(h->stream, g);
    TDVP_LAUNCH(max_dev_identity_kernel, 1, 256, 0, h->stream, G, g.M, dev);
  }
  if (int rc = check_cuda(h, cudaMemcpyAsync(defect, dev, sizeof(double), cudaMemcpyDeviceToHost, h->stream), "memcpy")) return rc;
  return check_cuda(h, cudaStreamSynchronize(h->stream), "canonical check");
}

static void free_chain(tdvp_handle *h) {
  auto fr = [](void *p) { if (p) cudaFree(p); };
  for (auto p : h->W) fr(p);
  for (auto p : h->Wsp_mem) fr(p);
  for (auto p : h->A) fr(p);
  for (auto p : h->Lenv) fr(p);
  for (auto p : h->Renv) fr(p);
  for (int s = 0; s < 7; s++) for (auto p : h->mu_k[s]) fr(p);
  for (auto p : h->mu_y) fr(p);
  for (auto p : h->cmf_mem) fr(p);
  for (auto p : h->cmf_ws) fr(p);
  for (auto p : h->cmf_scratch) fr(p);
  for (auto q : h->cmf_streams) { cudaStreamSynchronize(q); zgemm_release_stream(q); cudaStreamDestroy(q); }
  for (auto e : h->cmf_join) cudaEventDestroy(e);
  for (auto e : h->cmf_rel) cudaEventDestroy(e);
  for (auto e : h->cmf_fac) cudaEventDestroy(e);
  if (h->cmf_env) { cudaStreamSynchronize(h->cmf_env); zgemm_release_stream(h->cmf_env); cudaStreamDestroy(h->cmf_env); }
  fr(h->cmf_env_ws); fr(h->cmf_svd_ws[0]); fr(h->cmf_svd_ws[1]);
  if (h->cmf_fork) cudaEventDestroy(h->cmf_fork);
  if (h->cmf_hi) { cudaStreamSynchronize(h->cmf_hi); zgemm_release_stream(h->cmf_hi); cudaStreamDestroy(h->cmf_hi); }
  if (h->cmf_hi_done) cudaEventDestroy(h->cmf_hi_done);
  fr(h->tmpA); fr(h->tmpB); fr(h->bondD); fr(h->bondD2); fr(h->step_ws); fr(h->mu_err_dev); fr(h->mu_scratch);
  if (h->ps2_graph.exec) cudaGraphExecDestroy(h->ps2_graph.exec);
  fr(h->ps2_ws);
  if (h->ps_graph.exec) cudaGraphExecDestroy(h->ps_graph.exec);
  if (h->mu_graph.exec) cudaGraphExecDestroy(h->mu_graph.exec);
  if (h->cmf_graph.exec) cudaGraphExecDestroy(h->cmf_graph.exec);
  h->arena.release();
}

extern "C" {

int tdvp_destroy(tdvp_handle *h) {
  if (!h) return TDVP_OK;
  cudaStreamSynchronize(h->stream);
  free_chain(h);
  if (h->status_dev) cudaFree(h->status_dev);
  if (h->owns_zgemm_ctx) zgemm_release_stream(h->stream);   // the last handle on the stream frees the context
  if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
  if (h->ev_first) cudaEventDestroy(h->ev_first);
  if (h->ev_w) cudaEventDestroy(h->ev_w);
  if (h->ev_r) cudaEventDestroy(h->ev_r);
  for (int i = 0; i < 4; i++) if (h->ev_l[i]) cudaEventDestroy(h->ev_l[i]);
  delete h;
  return TDVP_OK;
}

int tdvp_create(tdvp_handle **out, int n_sites, const int *phys_dim, const int *mpo_bond,
                const tdvp_c128 *const *mpo, const int *mps_bond, const tdvp_c128 *const *mps,
                int on_device, const tdvp_options *opt, void *cuda_stream) {
  if (!out || !phys_dim || !mpo_bond || !mpo || !mps_bond || !mps) return set_err(nullptr, TDVP_EINVAL, "null pointer");
  if (n_sites < 1) return set_err(nullptr, TDVP_EINVAL, "n_sites must be >= 1");
  if (mpo_bond[0] != 1 || mpo_bond[n_sites] != 1 || mps_bond[0] != 1 || mps_bond[n_sites] != 1)
    return set_err(nullptr, TDVP_EINVAL, "boundary bond dimensions must be 1");
  for (int i = 0; i < n_sites; i++) {
    if (phys_dim[i] < 1 || mpo_bond[i + 1] < 1 || mps_bond[i + 1] < 1 || !mpo[i] || !mps[i])
      return set_err(nullptr, TDVP_EINVAL, "bad dimension or null tensor");
    if ((long long)mps_bond[i] * phys_dim[i] < mps_bond[i + 1] || (long long)mps_bond[i + 1] * phys_dim[i] < mps_bond[i])
      return set_err(nullptr, TDVP_EINVAL, "MPS bonds must satisfy M_i*d_i >= M_{i+1} and M_{i+1}*d_i >= M_i");
    if ((long long)mps_bond[i] * phys_dim[i] > QR_MAX_TALL || (long long)mps_bond[i + 1] * phys_dim[i] > QR_MAX_TALL)
      return set_err(nullptr, TDVP_EINVAL, "M_i * d_i above 12800 is not supported (QR gauge move, SURVEY.md 8(a) a7)");
  }
  tdvp_handle *h = nullptr;
  if (int rc = tdvp_create_context(&h, opt, cuda_stream)) return rc;
  h->n = n_sites;
  h->d.assign(phys_dim, phys_dim + n_sites);
  h->Dw.assign(mpo_bond, mpo_bond + n_sites + 1);
  h->M.assign(mps_bond, mps_bond + n_sites + 1);
  const int n = n_sites;
  h->W.assign(n, nullptr); h->Wsp.resize(n); h->Wsp_mem.assign(n, nullptr);
  h->A.assign(n, nullptr); h->Lenv.assign(n, nullptr); h->Renv.assign(n, nullptr);
  const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  auto fail = [&](int rc) { std::string e = h->err; tdvp_destroy(h); return set_err(nullptr, rc, e); };
  long long max_site = 0, max_bond = 0;
  for (int i = 0; i < n; i++) {
    size_t wn = (size_t)h->Dw[i] * h->d[i] * h->d[i] * h->Dw[i + 1];
    if (int rc = check_cuda(h, cudaMalloc(&h->W[i], wn * 16), "cudaMalloc W")) return fail(rc);
    if (int rc = check_cuda(h, cudaMalloc(&h->Wsp_mem[i], wsparse_bytes(h->Dw[i], h->d[i], h->Dw[i + 1])), "cudaMalloc W csr")) return fail(rc);
    if (int rc = check_cuda(h, cudaMalloc(&h->A[i], site_elems(h, i) * 16), "cudaMalloc A")) return fail(rc);
    if (int rc = check_cuda(h, cudaMalloc(&h->Lenv[i], lenv_elems(h, i) * 16), "cudaMalloc L")) return fail(rc);
    if (int rc = check_cuda(h, cudaMalloc(&h->Renv[i], renv_elems(h, i) * 16), "cudaMalloc R")) return fail(rc);
    if (int rc = check_cuda(h, cudaMemcpyAsync(h->W[i], mpo[i], wn * 16, kind, h->stream), "copy W")) return fail(rc);
    if (int rc = check_cuda(h, cudaMemcpyAsync(h->A[i], mps[i], site_elems(h, i) * 16, kind, h->stream), "copy A")) return fail(rc);
    wsparse_build(h->stream, h->Wsp[i], h->Wsp_mem[i], h->Dw[i], h->d[i], h->Dw[i + 1], h->W[i], h->opt.w_zero_tol);
    wsparse_classify(h->Wsp[i], h->stream);             // long or short rows: known on the host from here on
    max_site = std::max(max_site, site_elems(h, i));
    max_bond = std::max(max_bond, (long long)h->M[i + 1] * h->M[i + 1]);
  }
  if (int rc = check_cuda(h, cudaMalloc(&h->tmpA, max_site * 16), "cudaMalloc")) return fail(rc);
  if (int rc = check_cuda(h, cudaMalloc(&h->tmpB, max_site * 16), "cudaMalloc")) return fail(rc);
  if (int rc = check_cuda(h, cudaMalloc(&h->bondD, max_bond * 16), "cudaMalloc")) return fail(rc);
  if (int rc = check_cuda(h, cudaMalloc(&h->bondD2, max_bond * 16), "cudaMalloc")) return fail(rc);
  h->step_ws_bytes = chain_step_ws_bytes(h);
  if (int rc = check_cuda(h, cudaMalloc(&h->step_ws, h->step_ws_bytes), "cudaMalloc step workspace")) return fail(rc);
  TDVP_LAUNCH(set_one_kernel, 1, 1, 0, h->stream, h->Lenv[0]);
  TDVP_LAUNCH(set_one_kernel, 1, 1, 0, h->stream, h->Renv[n - 1]);
  h->centre = 0;
  if (!(h->opt.flags & TDVP_FLAG_SKIP_CANONICAL_CHECK) && n > 1) {
    double defect = 0.0;
    if (int rc = chain_canonical_defect(h, 1, 1, n, &defect)) return fail(rc);
    if (!(defect <= 1e-10)) {
      h->err = "MPS is not right-canonical on sites 1..N-1 (Eq. 8 violated by " + std::to_string(defect) + ")";
      return fail(TDVP_EINVAL);
    }
  }
  if (int rc = chain_rebuild_right_envs(h)) return fail(rc);
  if (int rc = check_cuda(h, cudaStreamSynchronize(h->stream), "tdvp_create")) return fail(rc);
  *out = h;
  return TDVP_OK;
}

}  // extern "C"
