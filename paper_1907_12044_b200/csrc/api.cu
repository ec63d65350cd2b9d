// api.cu -- C ABI entry points that work on caller-provided device buffers (include/tdvp.h),
// handle bookkeeping, error reporting and the FP64 tensor-pipe probe.
#include <mutex>
#include <vector>

#include "handle.cuh"

std::atomic<long long> g_launch_count{0};
thread_local long long *g_capture_tally = nullptr;
static thread_local std::string g_null_err;

// ---- phase profiler ---------------------------------------------------------------------------
// Process-wide measurement state (include/tdvp.h says so): the record list is guarded by a mutex,
// the on/off switch is atomic, the nesting depth belongs to the enqueueing host thread.
std::atomic<bool> g_prof_on{false};
thread_local int g_prof_depth = 0;
namespace {
struct ProfRec { cudaEvent_t e0, e1; int phase; bool closed; };
std::mutex g_prof_mu;
std::vector<ProfRec> g_prof_recs;
size_t g_prof_used = 0;
constexpr size_t PROF_MAX = 1 << 16;
}
int prof_begin(cudaStream_t st, int phase) {
  std::lock_guard<std::mutex> lk(g_prof_mu);
  if (g_prof_used >= PROF_MAX) return -1;
  if (g_prof_used == g_prof_recs.size()) {
    ProfRec r; r.phase = phase; r.closed = false;
    if (cudaEventCreate(&r.e0) != cudaSuccess || cudaEventCreate(&r.e1) != cudaSuccess) { cudaGetLastError(); return -1; }
    g_prof_recs.push_back(r);
  }
  const int rec = (int)g_prof_used++;
  g_prof_recs[rec].phase = phase; g_prof_recs[rec].closed = false;
  cudaEventRecord(g_prof_recs[rec].e0, st);
  return rec;
}
void prof_end(cudaStream_t st, int rec) {
  std::lock_guard<std::mutex> lk(g_prof_mu);
  if (rec < 0 || (size_t)rec >= g_prof_used) return;       // the list was read and reset in between
  cudaEventRecord(g_prof_recs[rec].e1, st);
  g_prof_recs[rec].closed = true;
}

// ---- errors -----------------------------------------------------------------------------------
namespace {
thread_local int g_sticky_code = 0;
thread_local std::string g_sticky_msg;
}
void sticky_error(int code, const std::string &msg) {
  if (g_sticky_code == 0 && code != 0) { g_sticky_code = code; g_sticky_msg = msg; }
}
int sticky_take(std::string *msg) {
  const int c = g_sticky_code;
  if (c && msg) *msg = g_sticky_msg;
  g_sticky_code = 0; g_sticky_msg.clear();
  return c;
}

int set_err(tdvp_handle *h, int code, const std::string &msg) {
  if (h) h->err = msg; else g_null_err = msg;
  return code;
}
// End of (a stage of) a public call: a pending internal error (see sticky_error) wins over the CUDA
// status, because whatever was enqueued after it ran on missing data.
int check_cuda(tdvp_handle *h, cudaError_t e, const char *what) {
  std::string smsg;
  if (const int sc = sticky_take(&smsg)) {
    if (e != cudaSuccess) cudaGetLastError();
    return set_err(h, sc, std::string(what) + ": " + smsg);
  }
  if (e == cudaSuccess) return TDVP_OK;
  return set_err(h, e == cudaErrorMemoryAllocation ? TDVP_ENOMEM : TDVP_ECUDA,
                 std::string(what) + ": " + cudaGetErrorString(e));
}

int finish_blocking(tdvp_handle *h, const char *what) {
  if (int rc = check_cuda(h, cudaStreamSynchronize(h->stream), what)) return rc;
  if (!h->status_dev) return TDVP_OK;
  int bits = 0;
  if (int rc = check_cuda(h, cudaMemcpy(&bits, h->status_dev, sizeof(int), cudaMemcpyDeviceToHost), what)) return rc;
  if (!bits) return TDVP_OK;
  cudaMemset(h->status_dev, 0, sizeof(int));
  if (bits & TDVP_STATUS_KRYLOV_RANGE)
    return set_err(h, TDVP_ESTATE, std::string(what) + ": a Krylov exponential had |z| * (spectral width of the tridiagonal matrix) above "
                                                       "the ~1850 the coefficient series covers; use a smaller step");
  if (bits & TDVP_STATUS_SVD_UNCONVERGED)
    return set_err(h, TDVP_ESTATE, std::string(what) + ": a bond SVD (Eq. 36) used up its Jacobi sweeps without converging; "
                                                       "results since the last blocking call are not to tolerance");
  return set_err(h, TDVP_ESTATE, std::string(what) + ": unknown device status");
}

cudaError_t Arena::reserve(size_t bytes, cudaStream_t st) {
  if (bytes <= cap) return cudaSuccess;
  if (base) {                                   // kernels in flight may still use the old arena
    cudaError_t e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return e;
    cudaFree(base); base = nullptr; cap = 0;
  }
  size_t want = bytes + bytes / 4 + (1 << 20);
  cudaError_t e = cudaMalloc(&base, want);
  if (e != cudaSuccess) { base = nullptr; cap = 0; return e; }
  cap = want; off = 0;
  return cudaSuccess;
}
void Arena::release() { if (base) cudaFree(base); base = nullptr; cap = 0; off = 0; }

void configure_kernels_once() {
  static std::once_flag once;
  std::call_once(once, [] { zgemm_configure(); wstage_configure(); qr_configure(); lanczos_configure(); svd_configure(); });
}

tdvp_handle *default_handle() {
  configure_kernels_once();
  static tdvp_handle *h = nullptr;
  static std::mutex mu;
  std::lock_guard<std::mutex> g(mu);
  if (!h) {
    h = new tdvp_handle(); tdvp_default_options(&h->opt); h->stream = nullptr; zgemm_prepare_stream(nullptr);
    if (cudaMalloc(&h->status_dev, sizeof(int)) == cudaSuccess) cudaMemset(h->status_dev, 0, sizeof(int));
    else { h->status_dev = nullptr; cudaGetLastError(); }
  }
  return h;   // if the context could not be made, the sticky error surfaces at the caller's first GEMM
}

static int check_opts(tdvp_handle *h, const tdvp_options &o) {
  if (o.krylov_dim < 1 || o.krylov_dim > TDVP_MAX_KRYLOV)
    return set_err(h, TDVP_EINVAL, "krylov_dim must be in [1, 64]");
  if (!(o.krylov_tol >= 0.0)) return set_err(h, TDVP_EINVAL, "krylov_tol must be >= 0 (0 = fixed Krylov dimension)");
  if (!(o.mu_eps > 0.0)) return set_err(h, TDVP_EINVAL, "mu_eps must be > 0");
  if (o.w_zero_tol < 0.0) return set_err(h, TDVP_EINVAL, "w_zero_tol must be >= 0");
  return TDVP_OK;
}

extern "C" {

void tdvp_default_options(tdvp_options *opt) {
  if (!opt) return;
  opt->krylov_dim = 10;
  opt->krylov_tol = 0.0;
  opt->mu_eps = 1e-10;
  opt->w_zero_tol = 0.0;
  opt->flags = 0;
}

int tdvp_create_context(tdvp_handle **out, const tdvp_options *opt, void *cuda_stream) {
  if (!out) return set_err(nullptr, TDVP_EINVAL, "out is NULL");
  tdvp_handle *h = new (std::nothrow) tdvp_handle();
  if (!h) return set_err(nullptr, TDVP_ENOMEM, "host allocation failed");
  if (opt) h->opt = *opt; else tdvp_default_options(&h->opt);
  int rc = check_opts(nullptr, h->opt);
  if (rc) { delete h; return rc; }
  h->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
  configure_kernels_once();
  if (zgemm_prepare_stream(h->stream) != TDVP_OK) {
    const int rc2 = check_cuda(nullptr, cudaSuccess, "tdvp_create_context");
    delete h;
    return rc2 ? rc2 : TDVP_ECUDA;
  }
  h->owns_zgemm_ctx = true;
  cudaError_t e = cudaMalloc(&h->status_dev, sizeof(int));
  if (e == cudaSuccess) e = cudaMemset(h->status_dev, 0, sizeof(int));
  if (e != cudaSuccess) {
    const int rc2 = check_cuda(nullptr, e, "tdvp_create_context");
    tdvp_destroy(h);
    return rc2;
  }
  *out = h;
  return TDVP_OK;
}

const char *tdvp_last_error(const tdvp_handle *h) { return h ? h->err.c_str() : g_null_err.c_str(); }

long long tdvp_launch_count(void) { return g_launch_count.load(); }

int tdvp_profile_enable(int on) { g_prof_on.store(on != 0); return TDVP_OK; }

int tdvp_profile_read(double *ms, long long *count) {
  if (!ms || !count) return set_err(nullptr, TDVP_EINVAL, "null pointer");
  for (int i = 0; i < TDVP_PROFILE_PHASES; i++) { ms[i] = 0.0; count[i] = 0; }
  if (int rc = check_cuda(nullptr, cudaDeviceSynchronize(), "tdvp_profile_read")) return rc;
  std::lock_guard<std::mutex> lk(g_prof_mu);
  for (size_t i = 0; i < g_prof_used; i++) {
    float t = 0.f;
    if (g_prof_recs[i].closed && cudaEventElapsedTime(&t, g_prof_recs[i].e0, g_prof_recs[i].e1) == cudaSuccess) {
      ms[g_prof_recs[i].phase] += t; count[g_prof_recs[i].phase]++;
    }
  }
  g_prof_used = 0;
  cudaGetLastError();
  return TDVP_OK;
}

int tdvp_sync(tdvp_handle *h) {
  tdvp_handle *hh = h ? h : default_handle();
  const int rc = finish_blocking(hh, "tdvp_sync");
  if (rc && !h) set_err(nullptr, rc, hh->err);
  return rc;
}

static int bad_dims(tdvp_handle *h, int Ml, int Mr, int d, int Dl, int Dr) {
  if (Ml < 1 || Mr < 1 || d < 1 || Dl < 1 || Dr < 1) return set_err(h, TDVP_EINVAL, "dimensions must be >= 1");
  const double lim = 2.0e9;
  if ((double)Ml * Dl * d * Mr > lim || (double)Ml * Dr * d * Mr > lim || (double)Ml * Ml * Dl > lim ||
      (double)Mr * Mr * Dr > lim)
    return set_err(h, TDVP_EINVAL, "problem too large (an intermediate exceeds 2e9 elements)");
  return 0;
}

namespace {
// second queue + events of a handle (host-entry copies; sparse build of W beside stage 1)
int ensure_side_queue(tdvp_handle *h, tdvp_handle *hh) {
  if (hh->copy_stream) return 0;
  if (int rc = check_cuda(h, cudaStreamCreateWithFlags(&hh->copy_stream, cudaStreamNonBlocking), "copy stream")) return rc;
  cudaEventCreateWithFlags(&hh->ev_first, cudaEventDisableTiming);
  cudaEventCreateWithFlags(&hh->ev_w, cudaEventDisableTiming);
  cudaEventCreateWithFlags(&hh->ev_r, cudaEventDisableTiming);
  for (int i = 0; i < 4; i++) cudaEventCreateWithFlags(&hh->ev_l[i], cudaEventDisableTiming);
  return 0;
}
// The stateless calls get a dense W and must build its sparse form first; that build does not depend
// on stage 1, so it runs on the side queue (fork after the arena's previous users, join before the
// W stage) and its ~8 us latency disappears behind the first GEMM.
int build_w_beside(tdvp_handle *h, tdvp_handle *hh, WSparse &wsp, void *wmem, int Dl, int d, int Dr, const c128 *W,
                   int Ml, int Mr) {
  if (int rc = ensure_side_queue(h, hh)) return rc;
  cudaEventRecord(hh->ev_first, hh->stream);
  cudaStreamWaitEvent(hh->copy_stream, hh->ev_first, 0);
  const bool many_panels = (long long)Ml * ((Mr + 63) / 64) >= W_QUAD_MIN_PANELS;
  wsparse_build(hh->copy_stream, wsp, wmem, Dl, d, Dr, W, hh->opt.w_zero_tol, many_panels);
  cudaEventRecord(hh->ev_w, hh->copy_stream);
  return 0;
}
}  // namespace

int tdvp_apply_heff(tdvp_handle *h, int Ml, int Mr, int d, int Dl, int Dr, const tdvp_c128 *L,
                    const tdvp_c128 *W, const tdvp_c128 *A, const tdvp_c128 *R, tdvp_c128 *out) {
  tdvp_handle *hh = h ? h : default_handle();
  if (!L || !W || !A || !R || !out) return set_err(h, TDVP_EINVAL, "null pointer");
  if (int rc = bad_dims(h, Ml, Mr, d, Dl, Dr)) return rc;
  size_t wb = wsparse_bytes(Dl, d, Dr), hb = heff_ws_bytes(Ml, Mr, d, Dl, Dr);
  if (int rc = check_cuda(h, hh->arena.reserve(wb + hb + 1024, hh->stream), "workspace")) return rc;
  hh->arena.reset();
  void *wmem = hh->arena.take(wb);
  void *ws = hh->arena.take(hb);
  WSparse wsp;
  if (int rc = build_w_beside(h, hh, wsp, wmem, Dl, d, Dr, reinterpret_cast<const c128 *>(W), Ml, Mr)) return rc;
  heff_apply(hh->stream, Ml, Mr, d, Dl, Dr, reinterpret_cast<const c128 *>(L), wsp,
             reinterpret_cast<const c128 *>(A), reinterpret_cast<const c128 *>(R),
             reinterpret_cast<c128 *>(out), ws, hh->ev_w);
  return check_cuda(h, cudaGetLastError(), "tdvp_apply_heff");
}

int tdvp_apply_heff_host(tdvp_handle *h, int Ml, int Mr, int d, int Dl, int Dr, const tdvp_c128 *L,
                         const tdvp_c128 *W, const tdvp_c128 *A, const tdvp_c128 *R, tdvp_c128 *out) {
  tdvp_handle *hh = h ? h : default_handle();
  if (!L || !W || !A || !R || !out) return set_err(h, TDVP_EINVAL, "null pointer");
  if (int rc = bad_dims(h, Ml, Mr, d, Dl, Dr)) return rc;
  const size_t nL = (size_t)Ml * Dl * Ml * 16, nW = (size_t)Dl * d * d * Dr * 16, nA = (size_t)Ml * d * Mr * 16,
               nR = (size_t)Mr * Dr * Mr * 16;
  auto up = [](size_t x) { return (x + 255) & ~size_t(255); };
  size_t wb = wsparse_bytes(Dl, d, Dr), hb = heff_ws_bytes(Ml, Mr, d, Dl, Dr);
  size_t io = up(nL) + up(nW) + 2 * up(nA) + up(nR);
  if (int rc = check_cuda(h, hh->arena.reserve(io + wb + hb + 4096, hh->stream), "workspace")) return rc;
  hh->arena.reset();
  c128 *dL = reinterpret_cast<c128 *>(hh->arena.take(nL)), *dW = reinterpret_cast<c128 *>(hh->arena.take(nW));
  c128 *dA = reinterpret_cast<c128 *>(hh->arena.take(nA)), *dR = reinterpret_cast<c128 *>(hh->arena.take(nR));
  c128 *dO = reinterpret_cast<c128 *>(hh->arena.take(nA));
  void *wmem = hh->arena.take(wb);
  void *ws = hh->arena.take(hb);
  cudaStream_t st = hh->stream;
  if (int rc = ensure_side_queue(h, hh)) return rc;
  // all H2D copies go to the copy queue in the order the stages need them -- A, L in slices of the
  // bond index, W, R -- and the compute stream waits for each piece by event, so stage 1 starts
  // after A and the first slice of L and the W stage / stage 3 never wait if the link keeps up
  cudaStream_t cq = hh->copy_stream;
  const int nsl = Ml >= 64 ? 4 : 1;
  cudaEventRecord(hh->ev_first, st);                     // the arena's previous users are done
  cudaStreamWaitEvent(cq, hh->ev_first, 0);
  if (int rc = check_cuda(h, cudaMemcpyAsync(dA, A, nA, cudaMemcpyHostToDevice, cq), "h2d A")) return rc;
  for (int s = 0; s < nsl; s++) {
    const size_t a0 = (size_t)Ml * s / nsl, a1 = (size_t)Ml * (s + 1) / nsl, row = (size_t)Dl * Ml;
    if (a1 > a0)
      if (int rc = check_cuda(h, cudaMemcpyAsync(dL + a0 * row, reinterpret_cast<const c128 *>(L) + a0 * row, (a1 - a0) * row * 16,
                                                 cudaMemcpyHostToDevice, cq), "h2d L")) return rc;
    cudaEventRecord(hh->ev_l[s], cq);
  }
  if (int rc = check_cuda(h, cudaMemcpyAsync(dW, W, nW, cudaMemcpyHostToDevice, cq), "h2d W")) return rc;
  cudaEventRecord(hh->ev_w, cq);
  if (int rc = check_cuda(h, cudaMemcpyAsync(dR, R, nR, cudaMemcpyHostToDevice, cq), "h2d R")) return rc;
  cudaEventRecord(hh->ev_r, cq);
  heff_apply_staged(st, Ml, Mr, d, Dl, Dr, dL, dW, wmem, hh->opt.w_zero_tol, dA, dR, dO, ws, nsl, hh->ev_l, hh->ev_w, hh->ev_r);
  if (int rc = check_cuda(h, cudaGetLastError(), "tdvp_apply_heff_host")) return rc;
  if (int rc = check_cuda(h, cudaMemcpyAsync(out, dO, nA, cudaMemcpyDeviceToHost, st), "d2h out")) return rc;
  return check_cuda(h, cudaStreamSynchronize(st), "tdvp_apply_heff_host sync");
}

int tdvp_update_env(tdvp_handle *h, int side, int Ml, int Mr, int d, int Dl, int Dr,
                    const tdvp_c128 *env_in, const tdvp_c128 *W, const tdvp_c128 *A,
                    tdvp_c128 *env_out) {
  tdvp_handle *hh = h ? h : default_handle();
  if (!env_in || !W || !A || !env_out) return set_err(h, TDVP_EINVAL, "null pointer");
  if (side != 0 && side != 1) return set_err(h, TDVP_EINVAL, "side must be 0 or 1");
  if (int rc = bad_dims(h, Ml, Mr, d, Dl, Dr)) return rc;
  size_t wb = wsparse_bytes(Dl, d, Dr), eb = env_ws_bytes(Ml, Mr, d, Dl, Dr);
  if (int rc = check_cuda(h, hh->arena.reserve(wb + eb + 1024, hh->stream), "workspace")) return rc;
  hh->arena.reset();
  void *wmem = hh->arena.take(wb);
  void *ws = hh->arena.take(eb);
  WSparse wsp;
  if (int rc = build_w_beside(h, hh, wsp, wmem, Dl, d, Dr, reinterpret_cast<const c128 *>(W), Ml, Mr)) return rc;
  env_update(hh->stream, side, Ml, Mr, d, Dl, Dr, reinterpret_cast<const c128 *>(env_in), wsp,
             reinterpret_cast<const c128 *>(A), reinterpret_cast<c128 *>(env_out), ws, hh->ev_w);
  return check_cuda(h, cudaGetLastError(), "tdvp_update_env");
}

int tdvp_apply_bond(tdvp_handle *h, int Ml, int Mr, int Dw, const tdvp_c128 *L,
                    const tdvp_c128 *D, const tdvp_c128 *R, tdvp_c128 *out) {
  tdvp_handle *hh = h ? h : default_handle();
  if (!L || !D || !R || !out) return set_err(h, TDVP_EINVAL, "null pointer");
  if (int rc = bad_dims(h, Ml, Mr, 1, Dw, Dw)) return rc;
  size_t bb = bond_ws_bytes(Ml, Mr, Dw);
  if (int rc = check_cuda(h, hh->arena.reserve(bb + 1024, hh->stream), "workspace")) return rc;
  hh->arena.reset();
  void *ws = hh->arena.take(bb);
  bond_apply(hh->stream, Ml, Mr, Dw, reinterpret_cast<const c128 *>(L),
             reinterpret_cast<const c128 *>(D), reinterpret_cast<const c128 *>(R),
             reinterpret_cast<c128 *>(out), ws);
  return check_cuda(h, cudaGetLastError(), "tdvp_apply_bond");
}

int tdvp_expm_heff(tdvp_handle *h, int Ml, int Mr, int d, int Dl, int Dr, const tdvp_c128 *L,
                   const tdvp_c128 *W, const tdvp_c128 *R, double z_re, double z_im,
                   const tdvp_c128 *v, tdvp_c128 *y, int *krylov_used) {
  tdvp_handle *hh = h ? h : default_handle();
  if (!L || !W || !R || !v || !y) return set_err(h, TDVP_EINVAL, "null pointer");
  if (int rc = bad_dims(h, Ml, Mr, d, Dl, Dr)) return rc;
  LanczosOp op{0, Ml, Mr, d, Dl, Dr, reinterpret_cast<const c128 *>(L), reinterpret_cast<const c128 *>(R), nullptr};
  const int k = hh->opt.krylov_dim;
  size_t wb = wsparse_bytes(Dl, d, Dr), lb = lanczos_ws_bytes(op, k);
  if (int rc = check_cuda(h, hh->arena.reserve(wb + lb + 2048, hh->stream), "workspace")) return rc;
  hh->arena.reset();
  void *wmem = hh->arena.take(wb);
  void *ws = hh->arena.take(lb);
  int *m_dev = reinterpret_cast<int *>(hh->arena.take(256));
  WSparse wsp;
  wsparse_build(hh->stream, wsp, wmem, Dl, d, Dr, reinterpret_cast<const c128 *>(W), hh->opt.w_zero_tol);
  op.W = &wsp;
  lanczos_expm(hh->stream, op, k, hh->opt.krylov_tol, z_re, z_im, reinterpret_cast<const c128 *>(v),
               reinterpret_cast<c128 *>(y), ws, m_dev, hh->status_dev);
  if (int rc = check_cuda(h, cudaGetLastError(), "tdvp_expm_heff")) return rc;
  if (krylov_used) {
    if (int rc = check_cuda(h, cudaMemcpyAsync(krylov_used, m_dev, sizeof(int), cudaMemcpyDeviceToHost, hh->stream), "memcpy")) return rc;
    return check_cuda(h, cudaStreamSynchronize(hh->stream), "tdvp_expm_heff sync");
  }
  return TDVP_OK;
}

int tdvp_expm_bond(tdvp_handle *h, int Ml, int Mr, int Dw, const tdvp_c128 *L, const tdvp_c128 *R,
                   double z_re, double z_im, const tdvp_c128 *v, tdvp_c128 *y, int *krylov_used) {
  tdvp_handle *hh = h ? h : default_handle();
  if (!L || !R || !v || !y) return set_err(h, TDVP_EINVAL, "null pointer");
  if (int rc = bad_dims(h, Ml, Mr, 1, Dw, Dw)) return rc;
  LanczosOp op{1, Ml, Mr, 1, Dw, Dw, reinterpret_cast<const c128 *>(L), reinterpret_cast<const c128 *>(R), nullptr};
  const int k = hh->opt.krylov_dim;
  size_t lb = lanczos_ws_bytes(op, k);
  if (int rc = check_cuda(h, hh->arena.reserve(lb + 2048, hh->stream), "workspace")) return rc;
  hh->arena.reset();
  void *ws = hh->arena.take(lb);
  int *m_dev = reinterpret_cast<int *>(hh->arena.take(256));
  lanczos_expm(hh->stream, op, k, hh->opt.krylov_tol, z_re, z_im, reinterpret_cast<const c128 *>(v),
               reinterpret_cast<c128 *>(y), ws, m_dev, hh->status_dev);
  if (int rc = check_cuda(h, cudaGetLastError(), "tdvp_expm_bond")) return rc;
  if (krylov_used) {
    if (int rc = check_cuda(h, cudaMemcpyAsync(krylov_used, m_dev, sizeof(int), cudaMemcpyDeviceToHost, hh->stream), "memcpy")) return rc;
    return check_cuda(h, cudaStreamSynchronize(hh->stream), "tdvp_expm_bond sync");
  }
  return TDVP_OK;
}

int tdvp_qr_gauge(tdvp_handle *h, int side, int Ml, int d, int Mr, const tdvp_c128 *C,
                  tdvp_c128 *Q, tdvp_c128 *D) {
  tdvp_handle *hh = h ? h : default_handle();
  if (!C || !Q || !D) return set_err(h, TDVP_EINVAL, "null pointer");
  if (side != 0 && side != 1) return set_err(h, TDVP_EINVAL, "side must be 0 or 1");
  if (Ml < 1 || d < 1 || Mr < 1) return set_err(h, TDVP_EINVAL, "dimensions must be >= 1");
  long long tall = side == 0 ? (long long)Ml * d : (long long)d * Mr;
  int thin = side == 0 ? Mr : Ml;
  if (tall < thin) return set_err(h, TDVP_EINVAL, "gauge move needs a tall or square matrix");
  if (tall > QR_MAX_TALL) return set_err(h, TDVP_EINVAL, "gauge move: tall side above 12800 rows is not supported");
  size_t qb = qr_ws_bytes((int)tall, thin);
  if (int rc = check_cuda(h, hh->arena.reserve(qb + 1024, hh->stream), "workspace")) return rc;
  hh->arena.reset();
  void *ws = hh->arena.take(qb);
  qr_gauge(hh->stream, side, Ml, d, Mr, reinterpret_cast<const c128 *>(C),
           reinterpret_cast<c128 *>(Q), reinterpret_cast<c128 *>(D), ws);
  return check_cuda(h, cudaGetLastError(), "tdvp_qr_gauge");
}

}  // extern "C"

// ---- FP64 tensor-pipe issue-rate probe ------------------------------------------------------
// F independent integer instructions (LOP3) follow every DMMA: F = 0 measures the pipe's peak, F > 0
// how much of it other instructions of the same warps cost (they do not issue under a DMMA).
template <int F>
__global__ void dmma_probe_kernel(double *out, int iters, double a, double b, int z) {
  double c0[8], c1[8];
  int x[4] = {(int)threadIdx.x, 1, 2, 3};
#pragma unroll
  for (int i = 0; i < 8; i++) { c0[i] = threadIdx.x; c1[i] = i; }
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < 8; i++) {
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                   : "+d"(c0[i]), "+d"(c1[i]) : "d"(a), "d"(b));
#pragma unroll
      for (int f = 0; f < F; f++) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x[f & 3]) : "r"(z), "r"(it));
    }
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 8; i++) s += c0[i] + c1[i];
  if (s == 1.2345 || x[0] + x[1] + x[2] + x[3] == 12345) out[0] = s;
}

static void launch_probe(int fillers, int blocks, int threads, double *out, int iters) {
  switch (fillers) {
    case 0: dmma_probe_kernel<0><<<blocks, threads>>>(out, iters, 1.0000001, 1e-9, iters); break;
    case 1: dmma_probe_kernel<1><<<blocks, threads>>>(out, iters, 1.0000001, 1e-9, iters); break;
    case 2: dmma_probe_kernel<2><<<blocks, threads>>>(out, iters, 1.0000001, 1e-9, iters); break;
    case 4: dmma_probe_kernel<4><<<blocks, threads>>>(out, iters, 1.0000001, 1e-9, iters); break;
    case 8: dmma_probe_kernel<8><<<blocks, threads>>>(out, iters, 1.0000001, 1e-9, iters); break;
    default: dmma_probe_kernel<16><<<blocks, threads>>>(out, iters, 1.0000001, 1e-9, iters); break;
  }
}

extern "C" {

int tdvp_probe_dmma_issue(int fillers, int iters, double *tflops) {
  if (!tflops || iters < 1 || !(fillers == 0 || fillers == 1 || fillers == 2 || fillers == 4 || fillers == 8 || fillers == 16))
    return set_err(nullptr, TDVP_EINVAL, "bad arguments (fillers must be 0, 1, 2, 4, 8 or 16)");
  int dev = 0, nsm = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
  double *out = nullptr;
  if (int rc = check_cuda(nullptr, cudaMalloc(&out, 8), "cudaMalloc")) return rc;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  // F = 0: eight warps per CTA (the peak); F > 0: two CTAs of four warps per SM, the residency of
  // zgemm_kernel (two warps per SMSP)
  const int blocks = 2 * nsm, threads = fillers == 0 ? 256 : 128;
  launch_probe(fillers, blocks, threads, out, iters / 10 + 1);
  float best = 1e30f;
  for (int r = 0; r < 3; r++) {
    cudaEventRecord(e0);
    launch_probe(fillers, blocks, threads, out, iters);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) best = ms;
  }
  cudaError_t e = cudaGetLastError();
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(out);
  if (e != cudaSuccess) return check_cuda(nullptr, e, "probe");
  double fma = 256.0 * 8 * (double)iters * (threads / 32) * blocks;
  *tflops = 2.0 * fma / (best * 1e-3) / 1e12;
  return TDVP_OK;
}

int tdvp_set_gemm_products(int products) {
  if (products != 3 && products != 4) return TDVP_EINVAL;
  zgemm_set_mode(products);
  return 0;
}
int tdvp_get_gemm_products(void) { return zgemm_get_mode(); }

int tdvp_probe_fp64_tensor_peak(int iters, double *tflops) { return tdvp_probe_dmma_issue(0, iters, tflops); }

}  // extern "C"
