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

}  // namespace

// Capture `enqueue` into a graph (once per dt) and launch it; falls back to direct enqueue when
// graphs are disabled.
template <class F>
static int run_step(tdvp_handle *h, StepGraph &sg, double dt, F enqueue, const char *what) {
  if (h->opt.flags & TDVP_FLAG_NO_GRAPH) {
    enqueue();
    return check_cuda(h, cudaGetLastError(), what);
  }
  if (!sg.exec || sg.dt != dt) {
    if (sg.exec) { cudaGraphExecDestroy(sg.exec); sg.exec = nullptr; }
    cudaStream_t cap = h->stream;
    cudaStream_t own = nullptr;
    if (cap == nullptr || cap == cudaStreamLegacy || cap == cudaStreamPerThread) {
      // the legacy default stream cannot be captured: record on a private stream, replay on h->stream
      if (int rc = check_cuda(h, cudaStreamCreateWithFlags(&own, cudaStreamNonBlocking), "stream")) return rc;
      cap = own;
      zgemm_alias_stream(own, h->stream);
    }
    cudaStream_t saved = h->stream;
    h->stream = cap;
    long long tally = 0;
    cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
    cudaGraph_t graph = nullptr;
    if (e == cudaSuccess) {
      g_capture_tally = &tally;
      enqueue();
      g_capture_tally = nullptr;
      e = cudaStreamEndCapture(cap, &graph);
    }
    h->stream = saved;
    if (e == cudaSuccess) e = cudaGraphInstantiate(&sg.exec, graph, 0);
    if (graph) cudaGraphDestroy(graph);
    if (own) { zgemm_forget_stream(own); cudaStreamDestroy(own); }
    if (e != cudaSuccess) { sg.exec = nullptr; cudaGetLastError(); return check_cuda(h, e, what); }
    sg.dt = dt; sg.launches = tally;
  }
  if (int rc = check_cuda(h, cudaGraphLaunch(sg.exec, h->stream), what)) return rc;
  g_launch_count.fetch_add(sg.launches);
  return TDVP_OK;
}

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
