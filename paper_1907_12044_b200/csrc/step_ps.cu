// step_ps.cu -- TDVP-PS step driver (Eq. 42-44) and gauge
// sweeps.  Everything is enqueue-only on the handle's stream; a whole step is captured once into a
// CUDA graph (keyed by dt) and replayed, so that the ~10^4 small launches of a step cost one
// graph launch on the host.
#include <algorithm>

#include "handle.cuh"

size_t chain_step_ws_bytes(const tdvp_handle *h);
int chain_rebuild_right_envs(tdvp_handle *h);
int chain_rebuild_left_envs(tdvp_handle *h);

namespace {

LanczosOp heff_op(const tdvp_handle *h, int i) {
  return LanczosOp{0, h->M[i], h->M[i + 1], h->d[i], h->Dw[i], h->Dw[i + 1], h->Lenv[i], h->Renv[i], &h->Wsp[i]};
}
LanczosOp bond_op(const tdvp_handle *h, int b) {
  return LanczosOp{1, h->M[b], h->M[b], 1, h->Dw[b], h->Dw[b], h->Lenv[b], h->Renv[b - 1], nullptr};
}
long long site_elems(const tdvp_handle *h, int i) { return (long long)h->M[i] * h->d[i] * h->M[i + 1]; }

// out[a][(s,c)] = sum_b D[a][b] A[b][(s,c)]     (C_{i+1} = D R_{i+1}, "MatMul-QR")
void absorb_right(tdvp_handle *h, int i, const c128 *D, const c128 *A, c128 *out) {
  ZGemm g{};
  g.A = D; g.B = A; g.C = out;
  g.M = h->M[i]; g.K = h->M[i]; g.N = h->d[i] * h->M[i + 1];
  g.a_ms = h->M[i]; g.a_ks = 1; g.b_ks = g.N; g.b_ns = 1; g.ldc = g.N;
  zgemm(h->stream, g);
}
// out[(a,s)][c] = sum_b A[(a,s)][b] D[b][c]     (C_{i-1} = A_{i-1} D)
void absorb_left(tdvp_handle *h, int i, const c128 *A, const c128 *D, c128 *out) {
  ZGemm g{};
  g.A = A; g.B = D; g.C = out;
  g.M = h->M[i] * h->d[i]; g.K = h->M[i + 1]; g.N = h->M[i + 1];
  g.a_ms = h->M[i + 1]; g.a_ks = 1; g.b_ks = g.N; g.b_ns = 1; g.ldc = g.N;
  zgemm(h->stream, g);
}

// Eq. 42: one symmetric sweep pair.  The centre tensor travels through tmpA / tmpB.
void enqueue_ps_step(tdvp_handle *h, double dt) {
  cudaStream_t st = h->stream;
  const int n = h->n, k = h->opt.krylov_dim;
  const double ktol = h->opt.krylov_tol;
  void *ws = h->step_ws;
  const c128 *cur = h->A[0];
  for (int i = 0; i < n - 1; i++) {
    lanczos_expm(st, heff_op(h, i), k, ktol, 0.0, -0.5 * dt, cur, h->tmpA, ws, nullptr, h->status_dev);            // Eq. 43
    qr_gauge(st, 0, h->M[i], h->d[i], h->M[i + 1], h->tmpA, h->A[i], h->bondD, ws);            // Eq. 9
    env_update(st, 0, h->M[i], h->M[i + 1], h->d[i], h->Dw[i], h->Dw[i + 1], h->Lenv[i], h->Wsp[i], h->A[i],
               h->Lenv[i + 1], ws);                                                             // Eq. 30-32
    lanczos_expm(st, bond_op(h, i + 1), k, ktol, 0.0, +0.5 * dt, h->bondD, h->bondD2, ws, nullptr, h->status_dev);  // Eq. 44
    absorb_right(h, i + 1, h->bondD2, h->A[i + 1], h->tmpB);
    cur = h->tmpB;
  }
  lanczos_expm(st, heff_op(h, n - 1), k, ktol, 0.0, -dt, cur, h->tmpA, ws, nullptr, h->status_dev);                 // last site, full step
  for (int i = n - 1; i >= 1; i--) {
    qr_gauge(st, 1, h->M[i], h->d[i], h->M[i + 1], h->tmpA, h->A[i], h->bondD, ws);
    env_update(st, 1, h->M[i], h->M[i + 1], h->d[i], h->Dw[i], h->Dw[i + 1], h->Renv[i], h->Wsp[i], h->A[i],
               h->Renv[i - 1], ws);
    lanczos_expm(st, bond_op(h, i), k, ktol, 0.0, +0.5 * dt, h->bondD, h->bondD2, ws, nullptr, h->status_dev);
    absorb_left(h, i - 1, h->A[i - 1], h->bondD2, h->tmpB);
    lanczos_expm(st, heff_op(h, i - 1), k, ktol, 0.0, -0.5 * dt, h->tmpB, h->tmpA, ws, nullptr, h->status_dev);
  }
  vec_copy(st, h->A[0], h->tmpA, site_elems(h, 0));
}

// ---- two-site TDVP-PS (PAPER.md:290 and its ref. 32) --------------------------------
// out[r][c] = src[r * sr + c * sc] * (mode 1: lam[c]; mode 2: lam[r]; mode 0: 1)
__global__ void gather_scale_kernel(c128 *out, long long R, long long Cn, const c128 *src, long long sr, long long sc,
                                    const double *lam, int mode) {
  const long long total = R * Cn;
  for (long long e = blockIdx.x * 256LL + threadIdx.x; e < total; e += (long long)gridDim.x * 256) {
    const long long r = e / Cn, c = e % Cn;
    const c128 x = src[r * sr + c * sc];
    const double f = mode == 1 ? lam[c] : (mode == 2 ? lam[r] : 1.0);
    out[e] = make_double2(x.x * f, x.y * f);
  }
}
inline int gs_grid(long long n) { long long g = (n + 255) / 256; return (int)(g > 1184 ? 1184 : (g < 1 ? 1 : g)); }

struct Ps2Ws { c128 *th, *th2, *U, *Vh; double *lam; void *lz; void *svd; };
inline size_t up256s(size_t x) { return (x + 255) & ~size_t(255); }

LanczosOp heff2_op(const tdvp_handle *h, int i) {
  LanczosOp op{2, h->M[i], h->M[i + 2], h->d[i], h->Dw[i], h->Dw[i + 2], h->Lenv[i], h->Renv[i + 1], &h->Wsp[i]};
  op.d2 = h->d[i + 1]; op.Dm = h->Dw[i + 1]; op.W2 = &h->Wsp[i + 1];
  return op;
}

// sizes of the two-site workspace; carve() hands out its pieces
size_t ps2_layout(const tdvp_handle *h, Ps2Ws *w, char *base) {
  size_t th = 0, umax = 0, lz = 0, sv = 0, lam = 0;
  for (int i = 0; i + 1 < h->n; i++) {
    const size_t rows = (size_t)h->M[i] * h->d[i], cols = (size_t)h->d[i + 1] * h->M[i + 2];
    const size_t mn = rows < cols ? rows : cols;
    th = std::max(th, rows * cols);
    umax = std::max(umax, mn * mn);
    lam = std::max(lam, mn);
    lz = std::max(lz, lanczos_ws_bytes(heff2_op(h, i), h->opt.krylov_dim));
    sv = std::max(sv, rows <= cols ? svd_ws_bytes((int)rows, h->d[i + 1], h->M[i + 2]) : svd_ws_bytes((int)cols, 1, (int)rows));
  }
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off += up256s(bytes); return base ? base + o : nullptr; };
  char *a = take(th * 16), *b = take(th * 16), *u = take(umax * 16), *v = take(th * 16), *l = take(lam * 8), *z = take(lz), *q = take(sv);
  if (w) { w->th = (c128 *)a; w->th2 = (c128 *)b; w->U = (c128 *)u; w->Vh = (c128 *)v; w->lam = (double *)l; w->lz = z; w->svd = q; }
  return off + 256;
}

// Theta of the pair (i, i + 1), rows = M_i d_i, cols = d_{i+1} M_{i+2}, split by SVD (Eq. 10) keeping chi = M_{i+1} values:
//   to_right = true : A_i <- U (left-canonical), centre <- S V^dagger  (a site tensor of site i + 1)
//   to_right = false: B_{i+1} <- V^dagger (right-canonical), centre <- U S (a site tensor of site i)
void split_pair(tdvp_handle *h, const Ps2Ws &w, int i, const c128 *theta, bool to_right, c128 *iso_out, c128 *centre_out) {
  cudaStream_t st = h->stream;
  const long long rows = (long long)h->M[i] * h->d[i], cols = (long long)h->d[i + 1] * h->M[i + 2];
  const long long chi = h->M[i + 1];
  if (rows <= cols) {
    svd_bond(st, (int)rows, h->d[i + 1], h->M[i + 2], theta, w.U, w.lam, w.Vh, w.svd, h->status_dev);    // Theta = U S Vh
    if (to_right) {
      TDVP_LAUNCH(gather_scale_kernel, gs_grid(rows * chi), 256, 0, st, iso_out, rows, chi, w.U, rows, 1LL, w.lam, 0);     // U[:, :chi]
      TDVP_LAUNCH(gather_scale_kernel, gs_grid(chi * cols), 256, 0, st, centre_out, chi, cols, w.Vh, cols, 1LL, w.lam, 2);  // S Vh[:chi]
    } else {
      TDVP_LAUNCH(gather_scale_kernel, gs_grid(chi * cols), 256, 0, st, iso_out, chi, cols, w.Vh, cols, 1LL, w.lam, 0);     // Vh[:chi]
      TDVP_LAUNCH(gather_scale_kernel, gs_grid(rows * chi), 256, 0, st, centre_out, rows, chi, w.U, rows, 1LL, w.lam, 1);   // U[:, :chi] S
    }
  } else {
    // tall: SVD of the transpose, Theta^T = U2 S Vh2  =>  Theta = Vh2^T S U2^T
    TDVP_LAUNCH(gather_scale_kernel, gs_grid(rows * cols), 256, 0, st, w.th2, cols, rows, theta, 1LL, cols, w.lam, 0);      // Theta^T
    svd_bond(st, (int)cols, 1, (int)rows, w.th2, w.U, w.lam, w.Vh, w.svd, h->status_dev);                // U2 [cols,cols], Vh2 [cols,rows]
    if (to_right) {
      TDVP_LAUNCH(gather_scale_kernel, gs_grid(rows * chi), 256, 0, st, iso_out, rows, chi, w.Vh, 1LL, rows, w.lam, 0);     // Vh2^T[:, :chi]
      TDVP_LAUNCH(gather_scale_kernel, gs_grid(chi * cols), 256, 0, st, centre_out, chi, cols, w.U, 1LL, cols, w.lam, 2);   // S U2^T[:chi]
    } else {
      TDVP_LAUNCH(gather_scale_kernel, gs_grid(chi * cols), 256, 0, st, iso_out, chi, cols, w.U, 1LL, cols, w.lam, 0);      // U2^T[:chi]
      TDVP_LAUNCH(gather_scale_kernel, gs_grid(rows * chi), 256, 0, st, centre_out, rows, chi, w.Vh, 1LL, rows, w.lam, 1);  // Vh2^T[:, :chi] S
    }
  }
}

// Theta[(a,s),(t,b)] = sum_c X[(a,s),c] Y[c,(t,b)]
void form_pair(tdvp_handle *h, int i, const c128 *X, const c128 *Y, c128 *theta) {
  ZGemm g{};
  g.A = X; g.B = Y; g.C = theta;
  g.M = h->M[i] * h->d[i]; g.K = h->M[i + 1]; g.N = h->d[i + 1] * h->M[i + 2];
  g.a_ms = g.K; g.a_ks = 1; g.b_ks = g.N; g.b_ns = 1; g.ldc = g.N;
  zgemm(h->stream, g);
}

// One two-site step (oracle/tdvp_ps2.py is the statement of the algorithm)
void enqueue_ps2_step(tdvp_handle *h, double dt) {
  cudaStream_t st = h->stream;
  const int n = h->n, k = h->opt.krylov_dim;
  const double ktol = h->opt.krylov_tol;
  Ps2Ws w;
  ps2_layout(h, &w, reinterpret_cast<char *>(h->ps2_ws));
  void *ws = h->step_ws;
  const c128 *centre = h->A[0];
  c128 *theta = w.th;
  for (int i = 0; i < n - 1; i++) {
    const bool last = i == n - 2;
    form_pair(h, i, centre, h->A[i + 1], w.th2);
    lanczos_expm(st, heff2_op(h, i), k, ktol, 0.0, last ? -dt : -0.5 * dt, w.th2, theta, w.lz, nullptr, h->status_dev);
    if (last) break;
    split_pair(h, w, i, theta, true, h->A[i], h->tmpA);
    env_update(st, 0, h->M[i], h->M[i + 1], h->d[i], h->Dw[i], h->Dw[i + 1], h->Lenv[i], h->Wsp[i], h->A[i], h->Lenv[i + 1], ws);
    lanczos_expm(st, heff_op(h, i + 1), k, ktol, 0.0, +0.5 * dt, h->tmpA, h->tmpB, ws, nullptr, h->status_dev);   // backward, one site
    centre = h->tmpB;
  }
  for (int i = n - 1; i >= 1; i--) {
    split_pair(h, w, i - 1, theta, false, h->A[i], h->tmpA);          // B_i, centre of site i - 1 in tmpA
    env_update(st, 1, h->M[i], h->M[i + 1], h->d[i], h->Dw[i], h->Dw[i + 1], h->Renv[i], h->Wsp[i], h->A[i], h->Renv[i - 1], ws);
    if (i - 1 > 0) {
      lanczos_expm(st, heff_op(h, i - 1), k, ktol, 0.0, +0.5 * dt, h->tmpA, h->tmpB, ws, nullptr, h->status_dev);
      form_pair(h, i - 2, h->A[i - 2], h->tmpB, w.th2);
      lanczos_expm(st, heff2_op(h, i - 2), k, ktol, 0.0, -0.5 * dt, w.th2, theta, w.lz, nullptr, h->status_dev);
    } else {
      vec_copy(st, h->A[0], h->tmpA, site_elems(h, 0));
    }
  }
}

}  // namespace

int move_gauge(tdvp_handle *h, int centre);

extern "C" {

int tdvp_step_ps(tdvp_handle *h, double dt) {
  if (!h || h->n < 1) return set_err(h, TDVP_EINVAL, "handle has no chain");
  h->mu_fsal = false;
  if (h->centre != 0) {
    if (int rc = move_gauge(h, 0)) return rc;
  }
  return run_step(h, h->ps_graph, dt, [&] { enqueue_ps_step(h, dt); }, "tdvp_step_ps");
}

int tdvp_step_ps2(tdvp_handle *h, double dt) {
  if (!h || h->n < 1) return set_err(h, TDVP_EINVAL, "handle has no chain");
  if (h->n < 2) return set_err(h, TDVP_EINVAL, "two-site TDVP needs at least two sites");
  for (int i = 0; i + 1 < h->n; i++) {
    const long long rows = (long long)h->M[i] * h->d[i], cols = (long long)h->d[i + 1] * h->M[i + 2];
    if (std::max(rows, cols) > QR_MAX_TALL) return set_err(h, TDVP_EINVAL, "two-site TDVP: M * d above 12800 is not supported (pair SVD)");
    if (h->M[i + 1] > std::min(rows, cols)) return set_err(h, TDVP_EINVAL, "two-site TDVP: a bond is larger than its pair matrix allows");
  }
  h->mu_fsal = false;
  if (h->centre != 0) {
    if (int rc = move_gauge(h, 0)) return rc;
  }
  if (!h->ps2_ws) {
    const size_t bytes = ps2_layout(h, nullptr, nullptr);
    if (int rc = check_cuda(h, cudaMalloc(&h->ps2_ws, bytes), "cudaMalloc two-site workspace")) return rc;
    h->ps2_ws_bytes = bytes;
  }
  return run_step(h, h->ps2_graph, dt, [&] { enqueue_ps2_step(h, dt); }, "tdvp_step_ps2");
}

int tdvp_apply_heff_site(tdvp_handle *h, int site, const tdvp_c128 *A_dev, tdvp_c128 *out_dev) {
  if (!h || h->n < 1) return set_err(h, TDVP_EINVAL, "handle has no chain");
  if (site < 0 || site >= h->n || !A_dev || !out_dev) return set_err(h, TDVP_EINVAL, "bad site or null pointer");
  heff_apply(h->stream, h->M[site], h->M[site + 1], h->d[site], h->Dw[site], h->Dw[site + 1], h->Lenv[site],
             h->Wsp[site], reinterpret_cast<const c128 *>(A_dev), h->Renv[site], reinterpret_cast<c128 *>(out_dev),
             h->step_ws);
  return check_cuda(h, cudaGetLastError(), "tdvp_apply_heff_site");
}

int tdvp_update_env_site(tdvp_handle *h, int site, int side) {
  if (!h || h->n < 1) return set_err(h, TDVP_EINVAL, "handle has no chain");
  if (side != 0 && side != 1) return set_err(h, TDVP_EINVAL, "side must be 0 or 1");
  if (site < 0 || site >= h->n || (side == 0 && site == h->n - 1) || (side == 1 && site == 0))
    return set_err(h, TDVP_EINVAL, "no neighbouring block on that side");
  const int i = site;
  if (side == 0)
    env_update(h->stream, 0, h->M[i], h->M[i + 1], h->d[i], h->Dw[i], h->Dw[i + 1], h->Lenv[i], h->Wsp[i], h->A[i],
               h->Lenv[i + 1], h->step_ws);
  else
    env_update(h->stream, 1, h->M[i], h->M[i + 1], h->d[i], h->Dw[i], h->Dw[i + 1], h->Renv[i], h->Wsp[i], h->A[i],
               h->Renv[i - 1], h->step_ws);
  return check_cuda(h, cudaGetLastError(), "tdvp_update_env_site");
}

int tdvp_set_gauge(tdvp_handle *h, int centre) {
  if (!h || h->n < 1) return set_err(h, TDVP_EINVAL, "handle has no chain");
  if (centre != 0 && centre != h->n - 1) return set_err(h, TDVP_EINVAL, "centre must be 0 or N-1");
  return move_gauge(h, centre);
}

int tdvp_get_centre(tdvp_handle *h) {
  if (!h || h->n < 1) return set_err(h, TDVP_EINVAL, "handle has no chain");
  return h->centre;
}

}  // extern "C"

// QR / RQ sweep without time evolution (Eq. 9); rebuilds the environments the sweep passes.
int move_gauge(tdvp_handle *h, int centre) {
  h->mu_fsal = false;
  cudaStream_t st = h->stream;
  while (h->centre < centre) {
    const int i = h->centre;
    qr_gauge(st, 0, h->M[i], h->d[i], h->M[i + 1], h->A[i], h->tmpA, h->bondD, h->step_ws);
    vec_copy(st, h->A[i], h->tmpA, site_elems(h, i));
    env_update(st, 0, h->M[i], h->M[i + 1], h->d[i], h->Dw[i], h->Dw[i + 1], h->Lenv[i], h->Wsp[i], h->A[i],
               h->Lenv[i + 1], h->step_ws);
    absorb_right(h, i + 1, h->bondD, h->A[i + 1], h->tmpB);
    vec_copy(st, h->A[i + 1], h->tmpB, site_elems(h, i + 1));
    h->centre = i + 1;
  }
  while (h->centre > centre) {
    const int i = h->centre;
    qr_gauge(st, 1, h->M[i], h->d[i], h->M[i + 1], h->A[i], h->tmpA, h->bondD, h->step_ws);
    vec_copy(st, h->A[i], h->tmpA, site_elems(h, i));
    env_update(st, 1, h->M[i], h->M[i + 1], h->d[i], h->Dw[i], h->Dw[i + 1], h->Renv[i], h->Wsp[i], h->A[i],
               h->Renv[i - 1], h->step_ws);
    absorb_left(h, i - 1, h->A[i - 1], h->bondD, h->tmpB);
    vec_copy(st, h->A[i - 1], h->tmpB, site_elems(h, i - 1));
    h->centre = i - 1;
  }
  return check_cuda(h, cudaGetLastError(), "gauge sweep");
}
