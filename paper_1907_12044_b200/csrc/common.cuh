// common.cuh -- shared declarations of libtdvp.so (CUDA path; shares nothing with oracle/).
#pragma once
#include <cuda_runtime.h>
#include <atomic>
#include <cstdint>
#include <cstdio>
#include <string>

#include "../../include/tdvp.h"

typedef double2 c128;  // (x = re, y = im), same memory layout as tdvp_c128

extern std::atomic<long long> g_launch_count;   // kernels enqueued (tdvp_launch_count)
// While a stream capture is recording, launches are counted into the graph's own tally instead.
extern thread_local long long *g_capture_tally;

// Phase profiler (tdvp_profile_enable / tdvp_profile_read): CUDA-event pairs around the launches
// of a kernel class, recorded on the launching stream; off by default, skipped during capture.
enum { PH_ZGEMM = 0, PH_WSTAGE = 1, PH_VEC = 2, PH_QR = 3, PH_SVD = 4, PH_COUNT = 5 };
static_assert(PH_COUNT == TDVP_PROFILE_PHASES, "phase list of include/tdvp.h");
// Process-wide, guarded by a mutex (several handles / host threads may enqueue at once); the nesting
// depth is per host thread.  prof_begin returns the record it opened, or -1.
int prof_begin(cudaStream_t st, int phase);
void prof_end(cudaStream_t st, int rec);
extern std::atomic<bool> g_prof_on;
extern thread_local int g_prof_depth;   // nested scopes: only the outermost one records
struct ProfScope {
  cudaStream_t st; bool counted; int rec;
  ProfScope(cudaStream_t s, int phase) : st(s), counted(g_prof_on.load(std::memory_order_relaxed) && !g_capture_tally), rec(-1) {
    if (counted && g_prof_depth++ == 0) rec = prof_begin(st, phase);
  }
  ~ProfScope() { if (counted) { g_prof_depth--; if (rec >= 0) prof_end(st, rec); } }
};

// Errors of internal stages whose call chain returns void (a GEMM that cannot get its scheduling
// context or tensor maps): recorded per host thread, FIRST error wins, reported -- and cleared -- by
// the next check_cuda() of the API layer, so that every public call still returns a TDVP_E* code
// (include/tdvp.h: no signal or exception crosses the boundary).
void sticky_error(int code, const std::string &msg);
int sticky_take(std::string *msg);   // returns the pending code (0 = none) and clears it

static inline void count_launch() {
  if (g_capture_tally) ++*g_capture_tally; else g_launch_count.fetch_add(1, std::memory_order_relaxed);
}

// Launch wrapper: counts the launch; errors are picked up by the API layer via cudaGetLastError.
#define TDVP_LAUNCH(kernel, grid, block, smem, stream, ...)              \
  do {                                                                   \
    kernel<<<(grid), (block), (smem), (stream)>>>(__VA_ARGS__);          \
    count_launch();                                                      \
  } while (0)

__host__ __device__ static inline c128 cmul(c128 a, c128 b) {
  return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__host__ __device__ static inline c128 cconj(c128 a) { return make_double2(a.x, -a.y); }

// One-time kernel attribute setup (dynamic shared memory limits); called when a handle is made.
void zgemm_configure();
void wstage_configure();
void qr_configure();
void svd_configure();
void lanczos_configure();
void configure_kernels_once();

static inline long long ceil_div_ll(long long a, long long b) { return (a + b - 1) / b; }

// ---------------------------------------------------------------------------------------------
// zgemm.cu : complex128 GEMM on the FP64 tensor pipe (DMMA m8n8k4), batched, split-K.
// C[bi](m,n) = sum_k opA[bi](m,k) * opB[bi](k,n),  m < M, n < N, k < K
//   opA(m,k) = conjA ? conj(A[m*a_ms + k*a_ks]) : A[m*a_ms + k*a_ks]   (one of a_ms, a_ks is 1)
//   opB(k,n) = conjB ? conj(B[k*b_ks + n*b_ns]) : B[k*b_ks + n*b_ns]   (one of b_ks, b_ns is 1)
//   C(m,n)   = C[m*ldc + n]
// batch index bi = bo*batch_inner + bin; each operand has an (outer, inner) pair of strides.
struct ZGemm {
  const c128 *A; const c128 *B; c128 *C;
  int M, N, K;
  long long a_ms, a_ks, b_ks, b_ns, ldc;
  int batch_inner = 1, batch_outer = 1;
  long long a_bsi = 0, b_bsi = 0, c_bsi = 0;   // inner batch strides
  long long a_bso = 0, b_bso = 0, c_bso = 0;   // outer batch strides
  int conjA = 0, conjB = 0;
  const int *skip = nullptr;     // DEVICE, nullable: if *skip != 0 when the kernel starts, every CTA returns at once
};
// The kernel is a persistent stream-K schedule; its partial-tile slots and flags belong to the
// stream (one reference-counted context per stream, made by zgemm_prepare_stream outside any capture
// and dropped by zgemm_release_stream; a private capture stream is aliased to the stream the graph
// will be replayed on).  Returns TDVP_OK or a TDVP_E* code, which is also left as the thread's sticky
// error (callers with a void chain need not look at it).
int zgemm(cudaStream_t st, const ZGemm &p);
int zgemm_prepare_stream(cudaStream_t st);
void zgemm_set_stream_cap(cudaStream_t st, int max_ctas);   // GEMMs on st use at most this many CTAs (0: no limit)
int zgemm_device_sms();
void zgemm_set_mode(int products);   // 3 or 4 real DMMA products per complex product
int zgemm_get_mode();
void zgemm_alias_stream(cudaStream_t alias, cudaStream_t of);
void zgemm_forget_stream(cudaStream_t alias);
void zgemm_release_stream(cudaStream_t st);

// ---------------------------------------------------------------------------------------------
// wstage.cu : sparse MPO stage.
// Device CSR of a dense W[Dl,d,d,Dr], rows r = s*Dr + v (heff order) and columns c = w*d + t.
struct WSparse {
  int Dl, d, Dr;
  // row-padded sparse form: row r holds cnt[r] entries, sorted by column, at [r*ncols, r*ncols + cnt[r])
  int *cnt;         // DEVICE [d*Dr]
  int *col;         // DEVICE [capacity]
  c128 *val;        // DEVICE [capacity]
  // transposed-role form used by the right-to-left order: rows r = w*d + s, columns c = t*Dr + v
  int *cnt_r; int *col_r; c128 *val_r;
  int capacity;     // Dl*d*d*Dr
  // rows sorted by entry count, longest first (both forms): the long-row kernel works on groups of
  // four consecutive rows of this order, so that the rows of a group are about equally long
  int *order, *order_r;
  // are the rows long (entries >= 8 per row on average)?  -1 = only known on the device (stateless
  // calls: both W-stage kernels are launched and the one whose turn it is not returns at once),
  // 0 / 1 = known on the host (resident chains: read back once at create)
  int long_rows = -1, long_rows_r = -1;
};
void wsparse_classify(WSparse &ws, cudaStream_t st);   // fills long_rows / long_rows_r (blocks on st)
size_t wsparse_bytes(int Dl, int d, int Dr);
// carve a WSparse out of `mem` (DEVICE, wsparse_bytes) and build both CSRs from dense W (DEVICE)
void wsparse_build(cudaStream_t st, WSparse &ws, void *mem, int Dl, int d, int Dr,
                   const c128 *W, double zero_tol, bool want_order = true);
constexpr int W_QUAD_MIN_PANELS = 48;   // fewer (a, 64-y) panels than this: the long-row kernel is not considered
// T2[a,s,v,y] = sum_{w,t} W[w,s,t,v] T1[a,w,t,y];  T1 [Ml,Dl,d,Mr] -> T2 [Ml,d,Dr,Mr]
void wstage_left(cudaStream_t st, const WSparse &ws, int Ml, int Mr, const c128 *T1, c128 *T2, const int *skip = nullptr);
// T2[w,x,s,b] = sum_{t,v} W[w,s,t,v] T1[x,t,v,b];  T1 [Ml,d,Dr,Mr] -> T2 [Dl,Ml,d,Mr]
void wstage_right(cudaStream_t st, const WSparse &ws, int Ml, int Mr, const c128 *T1, c128 *T2, const int *skip = nullptr);

// ---------------------------------------------------------------------------------------------
// Workspace: one growable device arena per handle (cudaMalloc only when it has to grow).
struct Arena {
  char *base = nullptr; size_t cap = 0; size_t off = 0;
  cudaError_t reserve(size_t bytes, cudaStream_t st);
  void reset() { off = 0; }
  void *take(size_t bytes) {
    size_t a = (off + 255) & ~size_t(255);
    if (a + bytes > cap) return nullptr;
    off = a + bytes; return base + a;
  }
  void release();
};

// ---------------------------------------------------------------------------------------------
// contract.cu : the local contractions on explicit device pointers.
size_t heff_ws_bytes(int Ml, int Mr, int d, int Dl, int Dr);
void heff_apply(cudaStream_t st, int Ml, int Mr, int d, int Dl, int Dr, const c128 *L,
                const WSparse &W, const c128 *A, const c128 *R, c128 *out, void *ws,
                cudaEvent_t w_ready = nullptr,    // if set: the W stage waits for it (W built on a side queue)
                const int *skip = nullptr);       // DEVICE flag: non-zero turns the three kernels into no-ops
// The same for the host-entry path, whose inputs are still arriving on a copy queue: stage 1 runs in
// nsl slices of the bond index a, slice s after ev_l[s] (A and rows [s*Ml/nsl, (s+1)*Ml/nsl) of L
// have landed); the sparse form of W is built after ev_w, stage 3 waits for ev_r (R).
void heff_apply_staged(cudaStream_t st, int Ml, int Mr, int d, int Dl, int Dr, const c128 *L, const c128 *W_dense,
                       void *wmem, double zero_tol, const c128 *A, const c128 *R, c128 *out, void *ws,
                       int nsl, const cudaEvent_t *ev_l, cudaEvent_t ev_w, cudaEvent_t ev_r);
// Two-site H_eff (Eq. 29 with two sites between the blocks): out[a,s1,s2,b] = sum L[a,w,x] W1[w,s1,t1,u]
// W2[u,s2,t2,v] Theta[x,t1,t2,y] R[b,v,y] -- stage 1, the W stage once per site, stage 3, on the same kernels.
size_t heff2_ws_bytes(int Ml, int Mr, int d1, int d2, int Dl, int Dm, int Dr);
void heff2_apply(cudaStream_t st, int Ml, int Mr, int d1, int d2, int Dl, int Dm, int Dr, const c128 *L, const WSparse &W1,
                 const WSparse &W2, const c128 *Theta, const c128 *R, c128 *out, void *ws, const int *skip = nullptr);
size_t env_ws_bytes(int Ml, int Mr, int d, int Dl, int Dr);
void env_update(cudaStream_t st, int side, int Ml, int Mr, int d, int Dl, int Dr,
                const c128 *env_in, const WSparse &W, const c128 *A, c128 *env_out, void *ws, cudaEvent_t w_ready = nullptr);
size_t bond_ws_bytes(int Ml, int Mr, int Dw);
void bond_apply(cudaStream_t st, int Ml, int Mr, int Dw, const c128 *L, const c128 *D,
                const c128 *R, c128 *out, void *ws, const int *skip = nullptr);

// ---------------------------------------------------------------------------------------------
// lanczos.cu : Krylov exponential with all scalars on the device.
struct LanczosOp {           // which operator: heff (site), bond, or two-site heff
  int kind;                  // 0 = heff, 1 = bond, 2 = two-site heff (sites i, i + 1 between L and R)
  int Ml, Mr, d, Dl, Dr;     // bond: d = 1, Dl = Dr = Dw
  const c128 *L; const c128 *R; const WSparse *W;
  int d2 = 1, Dm = 1;        // two-site: physical dimension of the second site, MPO bond between the two sites
  const WSparse *W2 = nullptr;   // (W: Dl x d x d x Dm, W2: Dm x d2 x d2 x Dr)
  long long elems() const { return kind == 1 ? (long long)Ml * Mr : (long long)Ml * d * (kind == 2 ? d2 : 1) * Mr; }
};
size_t lanczos_ws_bytes(const LanczosOp &op, int k);
// y = exp(z H) v with at most k Krylov vectors; tol > 0 (and z purely imaginary): stop at the first j with
// beta_j |[exp(z T_j) e_1]_j| < tol.  m_used_dev: DEVICE int (nullable) receiving the Krylov dimension used;
// status_dev: the handle's sticky device status (nullable).
constexpr int TDVP_STATUS_KRYLOV_RANGE = 2;   // |z| * spectral width of T beyond the Chebyshev series kept
void lanczos_expm(cudaStream_t st, const LanczosOp &op, int k, double tol, double z_re, double z_im,
                  const c128 *v, c128 *y, void *ws, int *m_used_dev, int *status_dev);

// ---------------------------------------------------------------------------------------------
// qr.cu : Householder QR gauge move on the device.
// Tallest matrix the panel kernels take: beyond 20 * 256 rows a one-column panel must still fit in
// 200 KB of shared memory.  The API layer rejects taller gauge moves / unfoldings with TDVP_EINVAL.
constexpr int QR_MAX_TALL = 12800;
size_t qr_ws_bytes(int rows, int cols);
// side 0: C (rows x cols, row-major, rows = Ml*d, cols = Mr) = Q D, Q rows x cols, D cols x cols
// side 1: C (Ml x (d*Mr)) = D Q, i.e. QR of C^T: tall = d*Mr, thin = Ml; Q [Ml, d*Mr], D [Ml, Ml]
// gate (DEVICE, nullable): if it points at zero when the kernels start, the two expensive ones (cluster factorisation
// and Q formation, matrices of up to 1280 rows) return at once and Q, D are left undefined -- for callers that decide
// on the device whether the factorisation is needed at all (svd.cu)
void qr_gauge(cudaStream_t st, int side, int Ml, int d, int Mr, const c128 *C, c128 *Q, c128 *D,
              void *ws, const int *gate = nullptr);
// its two halves on the same workspace: factor (writes D, leaves the reflectors in ws), then form Q from them
void qr_factor(cudaStream_t st, int side, int Ml, int d, int Mr, const c128 *C, c128 *D, void *ws, const int *gate = nullptr);
void qr_form_q(cudaStream_t st, int side, int Ml, int d, int Mr, c128 *Q, void *ws, const int *gate = nullptr);

// ---------------------------------------------------------------------------------------------
// svd.cu : matrix unfolding C[Ml, d*Mr] = U diag(lam) Vh (Eq. 36) on the device, Ml <= d*Mr.
size_t svd_ws_bytes(int Ml, int d, int Mr);
// status: DEVICE int of the handle (nullable); bit TDVP_STATUS_SVD_UNCONVERGED is set when the Jacobi
// iteration used up its sweeps with columns still rotating (reported by the next blocking call).
constexpr int TDVP_STATUS_SVD_UNCONVERGED = 1;
void svd_bond(cudaStream_t st, int Ml, int d, int Mr, const c128 *C, c128 *U, double *lam, c128 *Vh, void *ws,
              int *status);
// its two halves on the same workspace (svd.cu): U and lam first, Vh later -- possibly on another queue
void svd_bond_factor(cudaStream_t st, int Ml, int d, int Mr, const c128 *C, c128 *U, double *lam, void *ws, int *status);
void svd_bond_vh(cudaStream_t st, int Ml, int d, int Mr, c128 *Vh, void *ws);

// ---------------------------------------------------------------------------------------------
// small vector kernels shared by the drivers (vecops.cu)
void vec_copy(cudaStream_t st, c128 *dst, const c128 *src, long long n);
void vec_zero(cudaStream_t st, c128 *dst, long long n);
// partial-free deterministic reductions: out_dev[0] = sum |x|^2 ; uses scratch of vec_red_scratch()
size_t vec_red_scratch_bytes();
void vec_norm_sq(cudaStream_t st, const c128 *x, long long n, double *out_dev, void *scratch);
void vec_dotc(cudaStream_t st, const c128 *x, const c128 *y, long long n, c128 *out_dev, void *scratch);
