// pc_rk4.cu -- propagation and compression with the classical Runge-Kutta method (P&C-RK4), used as the
// paper's warm-up of the TDVP runs, from its building blocks:
//   MPO x MPS       Eq. 12-13   A'[(w,a), s', (v,b)] = sum_s W[w,s',s,v] A[a,s,b]
//   MPS + MPS       Eq. 14-15  block-diagonal merge of the site tensors
//   canonicalise    Eq. 9        QR sweep from site 1 to N-1 (qr.cu)
//   compress        Eq. 10       SVD sweep from site N to 2 keeping min(M, k) singular values (svd.cu)
//   RK4             Eq. 16
// Readings (DESIGN.md c20, the same as oracle/pc_rk4.py): every MPO x MPS product and every linear
// combination is compressed to M_max; scalars multiply the first site tensor; a compression keeps
// min(M, k) singular values, zeros included, so the bond dimensions depend on the shapes only.
// Unlike the TDVP steps, the bond dimensions change from operation to operation, so the working states
// live in buffers of their own (allocated per operation: the warm-up runs once per trajectory).
#include <algorithm>
#include <vector>

#include "handle.cuh"

namespace {

constexpr int PT = 256;
inline int grid_for(long long n) { long long g = (n + PT - 1) / PT; return (int)(g > 2368 ? 2368 : (g < 1 ? 1 : g)); }
inline size_t up256(size_t x) { return (x + 255) & ~size_t(255); }

struct DMps {                      // an MPS in device memory with its own bond dimensions
  std::vector<c128 *> t;
  std::vector<int> bond;           // [n + 1]
  void release() { for (auto p : t) if (p) cudaFree(p); t.clear(); bond.clear(); }
};

// out[(w,a), p, (v,b)] = sum_s W[w,p,s,v] A[a,s,b]  (Eq. 13), zeros of W skipped; coef multiplies the result
__global__ void mpo_site_kernel(const c128 *__restrict__ W, const c128 *__restrict__ A, c128 *out, int Dl, int d, int Dr, int Ml, int Mr,
                                c128 coef) {
  const long long total = (long long)Dl * Ml * d * Dr * Mr;
  for (long long e = blockIdx.x * (long long)PT + threadIdx.x; e < total; e += (long long)gridDim.x * PT) {
    const int b = (int)(e % Mr);
    long long r = e / Mr;
    const int v = (int)(r % Dr); r /= Dr;
    const int p = (int)(r % d); r /= d;
    const int a = (int)(r % Ml);
    const int w = (int)(r / Ml);
    double sx = 0.0, sy = 0.0;
    for (int s = 0; s < d; s++) {
      const c128 wv = __ldg(W + (((long long)w * d + p) * d + s) * Dr + v);
      if (wv.x == 0.0 && wv.y == 0.0) continue;
      const c128 x = A[((long long)a * d + s) * Mr + b];
      sx += wv.x * x.x - wv.y * x.y;
      sy += wv.x * x.y + wv.y * x.x;
    }
    out[e] = make_double2(coef.x * sx - coef.y * sy, coef.x * sy + coef.y * sx);
  }
}
// dst[(r0 + a), s, (c0 + b)] = coef * src[a, s, b]   (one block of Eq. 15)
__global__ void place_block_kernel(c128 *dst, int Mr_dst, int r0, int c0, const c128 *src, int Ml, int d, int Mr, c128 coef) {
  const long long total = (long long)Ml * d * Mr;
  for (long long e = blockIdx.x * (long long)PT + threadIdx.x; e < total; e += (long long)gridDim.x * PT) {
    const int b = (int)(e % Mr);
    const long long as = e / Mr;                           // a * d + s
    const long long a = as / d, s = as % d;
    const c128 x = src[e];
    dst[((r0 + a) * d + s) * Mr_dst + c0 + b] = make_double2(coef.x * x.x - coef.y * x.y, coef.x * x.y + coef.y * x.x);
  }
}
// out[r][c] = U[r][c] * lam[c], c < keep (the kept columns of U Lambda, compact)
__global__ void ulam_kernel(const c128 *U, int ldu, const double *lam, c128 *out, int rows, int keep) {
  const long long total = (long long)rows * keep;
  for (long long e = blockIdx.x * (long long)PT + threadIdx.x; e < total; e += (long long)gridDim.x * PT) {
    const int c = (int)(e % keep);
    const long long r = e / keep;
    const c128 u = U[r * ldu + c];
    const double l = lam[c];
    out[e] = make_double2(u.x * l, u.y * l);
  }
}
// T[a, s, (a', s')] = delta: the identity as a left-isometric site tensor [Ml, d, Ml * d]
__global__ void identity_site_kernel(c128 *T, int n) {
  const long long total = (long long)n * n;
  for (long long e = blockIdx.x * (long long)PT + threadIdx.x; e < total; e += (long long)gridDim.x * PT)
    T[e] = make_double2((e / n) == (e % n) ? 1.0 : 0.0, 0.0);
}

struct Ctx {
  tdvp_handle *h;
  cudaStream_t st;
  void *ws = nullptr; size_t ws_cap = 0;
  int rc = TDVP_OK;
  bool ok() const { return rc == TDVP_OK; }
  void fail(int code, const char *msg) { if (rc == TDVP_OK) rc = set_err(h, code, msg); }
  c128 *alloc(long long elems) {
    void *p = nullptr;
    if (cudaMalloc(&p, (size_t)(elems > 0 ? elems : 1) * 16) != cudaSuccess) { cudaGetLastError(); fail(TDVP_ENOMEM, "P&C-RK4: device allocation failed"); return nullptr; }
    return reinterpret_cast<c128 *>(p);
  }
  void *scratch(size_t bytes) {
    if (bytes > ws_cap) {
      cudaStreamSynchronize(st);
      if (ws) cudaFree(ws);
      ws = nullptr; ws_cap = 0;
      if (cudaMalloc(&ws, bytes + bytes / 4) != cudaSuccess) { cudaGetLastError(); fail(TDVP_ENOMEM, "P&C-RK4: scratch allocation failed"); return nullptr; }
      ws_cap = bytes + bytes / 4;
    }
    return ws;
  }
};

void gemm_nn(Ctx &cx, const c128 *A, const c128 *B, c128 *C, long long M, long long K, long long N) {   // C[M,N] = A[M,K] B[K,N], row-major
  ZGemm g{};
  g.A = A; g.B = B; g.C = C;
  g.M = (int)M; g.K = (int)K; g.N = (int)N;
  g.a_ms = K; g.a_ks = 1; g.b_ks = N; g.b_ns = 1; g.ldc = N;
  zgemm(cx.st, g);
}

// |out> = coef * H |in>   (Eq. 12-13)
DMps mpo_times_mps(Ctx &cx, const tdvp_handle *mo /*holds W, d, Dw*/, const std::vector<c128 *> &W, const std::vector<int> &d,
                   const std::vector<int> &Dw, const DMps &in, c128 coef) {
  (void)mo;
  DMps out;
  const int n = (int)in.t.size();
  out.bond.resize(n + 1);
  out.t.assign(n, nullptr);
  for (int i = 0; i <= n; i++) out.bond[i] = Dw[i] * in.bond[i];
  for (int i = 0; i < n && cx.ok(); i++) {
    const long long total = (long long)out.bond[i] * d[i] * out.bond[i + 1];
    if (total > 2000000000LL) { cx.fail(TDVP_EINVAL, "P&C-RK4: an MPO x MPS site tensor exceeds 2e9 elements"); break; }
    out.t[i] = cx.alloc(total);
    if (!out.t[i]) break;
    TDVP_LAUNCH(mpo_site_kernel, grid_for(total), PT, 0, cx.st, W[i], in.t[i], out.t[i], Dw[i], d[i], Dw[i + 1], in.bond[i], in.bond[i + 1],
                i == 0 ? coef : make_double2(1.0, 0.0));
  }
  return out;
}

// sum_k coef_k |term_k>   (Eq. 14-15)
DMps mps_add(Ctx &cx, const std::vector<int> &d, const std::vector<const DMps *> &terms, const std::vector<c128> &coef) {
  DMps out;
  const int n = (int)terms[0]->t.size();
  out.bond.assign(n + 1, 1);
  out.t.assign(n, nullptr);
  for (int i = 1; i < n; i++) { int s = 0; for (auto t : terms) s += t->bond[i]; out.bond[i] = s; }
  for (int i = 0; i < n && cx.ok(); i++) {
    const long long total = (long long)out.bond[i] * d[i] * out.bond[i + 1];
    out.t[i] = cx.alloc(total);
    if (!out.t[i]) break;
    cudaMemsetAsync(out.t[i], 0, (size_t)total * 16, cx.st);
    int r0 = 0, c0 = 0;
    for (size_t k = 0; k < terms.size(); k++) {
      const DMps &m = *terms[k];
      const long long be = (long long)m.bond[i] * d[i] * m.bond[i + 1];
      TDVP_LAUNCH(place_block_kernel, grid_for(be), PT, 0, cx.st, out.t[i], out.bond[i + 1], i == 0 ? 0 : r0, i == n - 1 ? 0 : c0, m.t[i],
                  m.bond[i], d[i], m.bond[i + 1], i == 0 ? coef[k] : make_double2(1.0, 0.0));
      r0 += m.bond[i]; c0 += m.bond[i + 1];
    }
  }
  return out;
}

// Canonicalise (Eq. 9: QR from site 1 to N-1), then SVD from site N to 2 keeping min(M, k) singular values
// (Eq. 10).  In place: m becomes right-canonical with the gauge centre at site 0.
void compress(Ctx &cx, const std::vector<int> &d, DMps &m, int M) {
  const int n = (int)m.t.size();
  cudaStream_t st = cx.st;
  int *status = cx.h ? cx.h->status_dev : nullptr;
  for (int i = 0; i < n - 1 && cx.ok(); i++) {
    const int Ml = m.bond[i], Mr = m.bond[i + 1], di = d[i], Mrr = m.bond[i + 2], dn = d[i + 1];
    const long long rows = (long long)Ml * di;
    if (rows > QR_MAX_TALL) { cx.fail(TDVP_EINVAL, "P&C-RK4: a canonicalisation QR has more than 12800 rows (M_O * M_max * d too large)"); break; }
    if (rows >= Mr) {
      c128 *Q = cx.alloc(rows * Mr), *D = cx.alloc((long long)Mr * Mr), *nx = cx.alloc((long long)Mr * dn * Mrr);
      void *ws = cx.scratch(qr_ws_bytes((int)rows, Mr) + 1024);
      if (!Q || !D || !nx || !ws) { if (Q) cudaFree(Q); if (D) cudaFree(D); if (nx) cudaFree(nx); break; }
      qr_gauge(st, 0, Ml, di, Mr, m.t[i], Q, D, ws);
      gemm_nn(cx, D, m.t[i + 1], nx, Mr, Mr, (long long)dn * Mrr);          // C_{i+1} = D R_{i+1}
      cudaStreamSynchronize(st);
      cudaFree(m.t[i]); cudaFree(m.t[i + 1]); cudaFree(D);
      m.t[i] = Q; m.t[i + 1] = nx;
    } else {
      // wide: (Ml d) x Mr with Ml d < Mr.  Q = identity (a unitary of dimension Ml d), D = the matrix itself: a
      // valid gauge move (any unitary-equivalent choice is) with the same new bond min(rows, cols)
      const int nb = (int)rows;
      c128 *Q = cx.alloc((long long)nb * nb), *nx = cx.alloc((long long)nb * dn * Mrr);
      if (!Q || !nx) { if (Q) cudaFree(Q); if (nx) cudaFree(nx); break; }
      TDVP_LAUNCH(identity_site_kernel, grid_for((long long)nb * nb), PT, 0, st, Q, nb);
      gemm_nn(cx, m.t[i], m.t[i + 1], nx, nb, Mr, (long long)dn * Mrr);
      cudaStreamSynchronize(st);
      cudaFree(m.t[i]); cudaFree(m.t[i + 1]);
      m.t[i] = Q; m.t[i + 1] = nx;
      m.bond[i + 1] = nb;
    }
  }
  for (int i = n - 1; i >= 1 && cx.ok(); i--) {
    const int Ml = m.bond[i], Mr = m.bond[i + 1], di = d[i], Mll = m.bond[i - 1], dp = d[i - 1];
    const long long cols = (long long)di * Mr;
    const int k = (int)std::min<long long>(Ml, cols), keep = std::min(M, k);
    c128 *B = cx.alloc((long long)keep * cols), *carry = cx.alloc((long long)Ml * keep), *pv = cx.alloc((long long)Mll * dp * keep);
    if (!B || !carry || !pv) { if (B) cudaFree(B); if (carry) cudaFree(carry); if (pv) cudaFree(pv); break; }
    if (Ml <= cols) {
      if (cols > QR_MAX_TALL) { cx.fail(TDVP_EINVAL, "P&C-RK4: a compression SVD has d * M above 12800"); break; }
      c128 *U = cx.alloc((long long)Ml * Ml), *Vh = cx.alloc((long long)Ml * cols);
      double *lam = reinterpret_cast<double *>(cx.alloc((Ml + 1) / 2 + 1));
      void *ws = cx.scratch(svd_ws_bytes(Ml, di, Mr) + 1024);
      if (U && Vh && lam && ws) {
        svd_bond(st, Ml, di, Mr, m.t[i], U, lam, Vh, ws, status);                  // Eq. 10
        cudaMemcpyAsync(B, Vh, (size_t)keep * cols * 16, cudaMemcpyDeviceToDevice, st);   // the first `keep` rows of V^dagger
        TDVP_LAUNCH(ulam_kernel, grid_for((long long)Ml * keep), PT, 0, st, U, Ml, lam, carry, Ml, keep);
      }
      cudaStreamSynchronize(st);
      if (U) cudaFree(U); if (Vh) cudaFree(Vh); if (lam) cudaFree(lam);
    } else {
      // tall unfolding (Ml > d Mr): QR first, C = Q R with R (d Mr) x (d Mr), then the SVD of R
      const int kk = (int)cols;
      if (Ml > QR_MAX_TALL) { cx.fail(TDVP_EINVAL, "P&C-RK4: a compression QR has more than 12800 rows"); break; }
      c128 *Q = cx.alloc((long long)Ml * kk), *R = cx.alloc((long long)kk * kk), *U = cx.alloc((long long)kk * kk), *Vh = cx.alloc((long long)kk * kk),
           *UL = cx.alloc((long long)kk * keep);
      double *lam = reinterpret_cast<double *>(cx.alloc((kk + 1) / 2 + 1));
      size_t wb = std::max(qr_ws_bytes(Ml, kk), svd_ws_bytes(kk, 1, kk)) + 1024;
      void *ws = cx.scratch(wb);
      if (Q && R && U && Vh && UL && lam && ws) {
        qr_gauge(st, 0, Ml, 1, kk, m.t[i], Q, R, ws);
        svd_bond(st, kk, 1, kk, R, U, lam, Vh, ws, status);
        cudaMemcpyAsync(B, Vh, (size_t)keep * cols * 16, cudaMemcpyDeviceToDevice, st);
        TDVP_LAUNCH(ulam_kernel, grid_for((long long)kk * keep), PT, 0, st, U, kk, lam, UL, kk, keep);
        gemm_nn(cx, Q, UL, carry, Ml, kk, keep);
      }
      cudaStreamSynchronize(st);
      for (c128 *p : {Q, R, U, Vh, UL}) if (p) cudaFree(p);
      if (lam) cudaFree(lam);
    }
    gemm_nn(cx, m.t[i - 1], carry, pv, (long long)Mll * dp, Ml, keep);            // C_{i-1} = L_{i-1} (U Lambda)
    cudaStreamSynchronize(st);
    cudaFree(m.t[i]); cudaFree(m.t[i - 1]); cudaFree(carry);
    m.t[i] = B; m.t[i - 1] = pv;
    m.bond[i] = keep;
  }
  if (cx.ok()) cx.rc = check_cuda(cx.h, cudaGetLastError(), "P&C-RK4 compression");
}

// One Runge-Kutta step, Eq. 16 (time-independent H)
void rk4_step(Ctx &cx, const std::vector<c128 *> &W, const std::vector<int> &d, const std::vector<int> &Dw, DMps &psi, double tau, int M) {
  const c128 minus_i = make_double2(0.0, -1.0), one = make_double2(1.0, 0.0);
  auto h_times = [&](const DMps &x) { DMps k = mpo_times_mps(cx, nullptr, W, d, Dw, x, minus_i); if (cx.ok()) compress(cx, d, k, M); return k; };
  auto combo = [&](double c, const DMps &k) {
    DMps y = mps_add(cx, d, {&psi, &k}, {one, make_double2(c, 0.0)});
    if (cx.ok()) compress(cx, d, y, M);
    return y;
  };
  DMps k1, k2, k3, k4, y;
  k1 = h_times(psi);
  if (cx.ok()) { y = combo(0.5 * tau, k1); if (cx.ok()) k2 = h_times(y); y.release(); }
  if (cx.ok()) { y = combo(0.5 * tau, k2); if (cx.ok()) k3 = h_times(y); y.release(); }
  if (cx.ok()) { y = combo(tau, k3); if (cx.ok()) k4 = h_times(y); y.release(); }
  if (cx.ok()) {
    const double s = tau / 6.0;
    DMps nw = mps_add(cx, d, {&psi, &k1, &k2, &k3, &k4}, {one, make_double2(s, 0.0), make_double2(2.0 * s, 0.0), make_double2(2.0 * s, 0.0), make_double2(s, 0.0)});
    if (cx.ok()) compress(cx, d, nw, M);
    cudaStreamSynchronize(cx.st);
    psi.release();
    psi = nw;
  }
  cudaStreamSynchronize(cx.st);
  k1.release(); k2.release(); k3.release(); k4.release();
}

}  // namespace

extern "C" {

int tdvp_pc_rk4_warmup(tdvp_handle *h, int n_sites, const int *phys_dim, const int *mpo_bond, const tdvp_c128 *const *mpo,
                       const int *mps_bond, const tdvp_c128 *const *mps, double tau, int n_steps, int M_max, int M_out,
                       int *mps_bond_out, tdvp_c128 *const *mps_out) {
  tdvp_handle *hh = h ? h : default_handle();
  if (!phys_dim || !mpo_bond || !mpo || !mps_bond || !mps || !mps_bond_out || !mps_out) return set_err(h, TDVP_EINVAL, "null pointer");
  if (n_sites < 2) return set_err(h, TDVP_EINVAL, "P&C-RK4 needs at least two sites");
  if (n_steps < 0 || M_max < 1 || M_out < 1) return set_err(h, TDVP_EINVAL, "n_steps >= 0, M_max >= 1 and M_out >= 1 are required");
  if (mpo_bond[0] != 1 || mpo_bond[n_sites] != 1 || mps_bond[0] != 1 || mps_bond[n_sites] != 1)
    return set_err(h, TDVP_EINVAL, "boundary bond dimensions must be 1");
  const int n = n_sites;
  for (int i = 0; i < n; i++)
    if (phys_dim[i] < 1 || mpo_bond[i + 1] < 1 || mps_bond[i + 1] < 1 || !mpo[i] || !mps[i] || !mps_out[i])
      return set_err(h, TDVP_EINVAL, "bad dimension or null tensor");
  Ctx cx; cx.h = hh; cx.st = hh->stream;
  std::vector<int> d(phys_dim, phys_dim + n), Dw(mpo_bond, mpo_bond + n + 1);
  std::vector<c128 *> W(n, nullptr);
  DMps psi;
  psi.bond.assign(mps_bond, mps_bond + n + 1);
  psi.t.assign(n, nullptr);
  for (int i = 0; i < n && cx.ok(); i++) {
    const long long wn = (long long)Dw[i] * d[i] * d[i] * Dw[i + 1], an = (long long)psi.bond[i] * d[i] * psi.bond[i + 1];
    W[i] = cx.alloc(wn); psi.t[i] = cx.alloc(an);
    if (!W[i] || !psi.t[i]) break;
    cudaMemcpyAsync(W[i], mpo[i], (size_t)wn * 16, cudaMemcpyHostToDevice, cx.st);
    cudaMemcpyAsync(psi.t[i], mps[i], (size_t)an * 16, cudaMemcpyHostToDevice, cx.st);
  }
  for (int s = 0; s < n_steps && cx.ok(); s++) rk4_step(cx, W, d, Dw, psi, tau, M_max);     // Eq. 16
  if (cx.ok()) compress(cx, d, psi, M_out);                                                // "compressed to the pre-defined M_S"
  if (cx.ok()) {
    for (int i = 0; i <= n; i++) mps_bond_out[i] = psi.bond[i];
    for (int i = 0; i < n; i++)
      cudaMemcpyAsync(mps_out[i], psi.t[i], (size_t)psi.bond[i] * d[i] * psi.bond[i + 1] * 16, cudaMemcpyDeviceToHost, cx.st);
    cx.rc = finish_blocking(hh, "tdvp_pc_rk4_warmup");
    if (cx.rc && !h) set_err(nullptr, cx.rc, hh->err);
  } else {
    cudaStreamSynchronize(cx.st);
    if (!h) set_err(nullptr, cx.rc, hh->err);
  }
  psi.release();
  for (auto p : W) if (p) cudaFree(p);
  if (cx.ws) cudaFree(cx.ws);
  return cx.rc;
}

}  // extern "C"
