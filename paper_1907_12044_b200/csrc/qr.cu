// qr.cu -- QR gauge move C = Q D (Eq. 9) by blocked Householder reflections, on
// the device.  The paper runs this on one CPU core with a PCIe copy each way
// and names the transfer overhead; here the matrix never leaves HBM.
//
// Householder (not Cholesky-QR): centre tensors of a padded / delta-seeded MPS are numerically
// rank deficient (relative singular values down to 1e-8 and below), and Q must still be an exact
// isometry (Eq. 7/8).
//
// Layout: the tall matrix (rows x cols, rows >= cols) is held column-major in a workspace X (every
// column contiguous), so all passes are coalesced.  side 1 (RQ = QR of the plain transpose,
// SURVEY.md 8(c) c9) is natively that layout; side 0 is transposed on the way in and out.
//   panel kernel : one CTA keeps an nb-column panel in shared memory, factors it column by column
//                  (zlarfg-style reflectors), builds the compact-WY factor T, emits R entries
//   trail kernel : X[:, c] <- (I - V T^H V^H) X[:, c] for the trailing columns (a few columns/CTA)
//   the same kernel with T instead of T^H applied to identity columns, panels in reverse, forms Q.
#include <cstdlib>

#include "common.cuh"

namespace {

constexpr int NB_MAX = 8;
constexpr int PANEL_THREADS = 1024;
constexpr int TRAIL_THREADS = 256;
constexpr int CB = 4;   // columns per CTA in the trailing update
// A column whose squared norm is below this (entries below ~1e-145: products of round-off residues along a
// chain of rank-deficient bonds get there) is treated as zero: H = I, the entries below the diagonal are dropped.
// Its squared norm would underflow and the reflector scalars 1 / beta, 1 / |alpha - beta|^2 would be Inf / NaN.
constexpr double TINY_NORM2 = 1e-290;

inline size_t up256(size_t x) { return (x + 255) & ~size_t(255); }

__device__ __forceinline__ double warp_sum_d(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// X[j][i] (column-major, ld = rows) <- C[i*cols + j]     (tiled transpose)
__global__ void transpose_in_kernel(const c128 *C, c128 *X, int rows, int cols) {
  __shared__ c128 t[32][33];
  int i0 = blockIdx.y * 32, j0 = blockIdx.x * 32;
  for (int r = threadIdx.y; r < 32; r += blockDim.y) {
    int i = i0 + r, j = j0 + threadIdx.x;
    if (i < rows && j < cols) t[r][threadIdx.x] = C[(long long)i * cols + j];
  }
  __syncthreads();
  for (int r = threadIdx.y; r < 32; r += blockDim.y) {
    int j = j0 + r, i = i0 + threadIdx.x;
    if (i < rows && j < cols) X[(long long)j * rows + i] = t[threadIdx.x][r];
  }
}
// Q[i*cols + j] <- Y[j][i]
__global__ void transpose_out_kernel(const c128 *Y, c128 *Q, int rows, int cols) {
  __shared__ c128 t[32][33];
  int i0 = blockIdx.y * 32, j0 = blockIdx.x * 32;
  for (int r = threadIdx.y; r < 32; r += blockDim.y) {
    int j = j0 + r, i = i0 + threadIdx.x;
    if (i < rows && j < cols) t[r][threadIdx.x] = Y[(long long)j * rows + i];
  }
  __syncthreads();
  for (int r = threadIdx.y; r < 32; r += blockDim.y) {
    int i = i0 + r, j = j0 + threadIdx.x;
    if (i < rows && j < cols) Q[(long long)i * cols + j] = t[threadIdx.x][r];
  }
}

__global__ void copy_kernel(c128 *dst, const c128 *src, long long n) {
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x)
    dst[e] = src[e];
}
// Y[c][i] = delta(i, c)
__global__ void identity_kernel(c128 *Y, int rows, int cols) {
  long long n = (long long)rows * cols;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
    int i = e % rows, c = e / rows;
    Y[e] = make_double2(i == c ? 1.0 : 0.0, 0.0);
  }
}
// D out: transpose_d = 0: D[i][j] = R[i][j]; 1: D[i][j] = R[j][i]
__global__ void store_d_kernel(const c128 *Rm, c128 *D, int cols, int transpose_d) {
  int n = cols * cols;
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
    int i = e / cols, j = e % cols;
    D[e] = transpose_d ? Rm[j * cols + i] : Rm[e];
  }
}

// ---- register-resident panel factorisation ---------------------------------------------------
// Same contract as qr_panel_kernel below, for rows - j0 <= RP_THREADS * RPT (256 x 5, 512 x 5, 512 x 10).  Every thread keeps
// its RPT rows of the NB panel columns in registers; each column costs ONE block-wide reduction:
// the sums s = sum_{i>=jj} |x_i|^2 and d_c = sum_{i>=jj} conj(x_i) y_c[i] give the reflector AND
// its products with the remaining panel columns, because v differs from x only in the pivot row:
//   v^H y_c = y_c[jj] + conj(scal) (d_c - conj(alpha) y_c[jj]),   v = [1; x_{i>jj} scal].

// Sum N doubles over the CTA: warp shuffles, then one shared-memory round over the warps in a fixed
// order (deterministic).  sm: [RP_WARPS][N] + [N].
template <int N, int RP_THREADS>
__device__ __forceinline__ void block_sum(double (&v)[N], double *sm) {
  constexpr int RP_WARPS = RP_THREADS / 32;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int i = 0; i < N; i++) {
    const double t = warp_sum_d(v[i]);
    if (lane == 0) sm[warp * N + i] = t;
  }
  __syncthreads();
  if (threadIdx.x < N) {
    double t = 0.0;
#pragma unroll
    for (int k = 0; k < RP_WARPS; k++) t += sm[k * N + threadIdx.x];
    sm[RP_WARPS * N + threadIdx.x] = t;
  }
  __syncthreads();
#pragma unroll
  for (int i = 0; i < N; i++) v[i] = sm[RP_WARPS * N + i];
  __syncthreads();
}

// Compact-WY factor T (w x w upper triangular, H_1...H_w = I - V T V^H) from the strictly upper Gram
// entries G[a][b] = v_a^H v_b and the tau's; one warp, lane a owns row a of the new column.
__device__ __noinline__ void build_T(const c128 *Gs, const c128 *tau_s, c128 *Ts, c128 *Tm, int w) {
  const int lane = threadIdx.x & 31;
  for (int a = lane; a < NB_MAX * NB_MAX; a += 32) Ts[a] = make_double2(0.0, 0.0);
  __syncwarp();
  // column c: T[a][c] = -tau_c sum_{qq<c} T[a][qq] G[qq][c]; lane = 4 a' + part handles two rows a (a', a' + 4... )
  // spread as: lane = a * 4 + s, s = quarter of the qq range; partial sums are combined by two shuffles
  for (int c = 0; c < w; c++) {
    if (lane == 0) Ts[c * NB_MAX + c] = tau_s[c];
    const int a = lane >> 2, sgm = lane & 3;             // 8 rows x 4 segments of two qq each
    c128 acc = make_double2(0.0, 0.0);
    if (a < c) {
#pragma unroll
      for (int u = 0; u < 2; u++) {
        const int qq = 2 * sgm + u;
        if (qq >= a && qq < c) { const c128 t = cmul(Ts[a * NB_MAX + qq], Gs[qq * NB_MAX + c]); acc.x += t.x; acc.y += t.y; }
      }
    }
    acc.x += __shfl_xor_sync(0xffffffffu, acc.x, 1); acc.y += __shfl_xor_sync(0xffffffffu, acc.y, 1);
    acc.x += __shfl_xor_sync(0xffffffffu, acc.x, 2); acc.y += __shfl_xor_sync(0xffffffffu, acc.y, 2);
    if (a < c && sgm == 0) {
      const c128 t = cmul(tau_s[c], acc);
      Ts[a * NB_MAX + c] = make_double2(-t.x, -t.y);
    }
    __syncwarp();
  }
  for (int a = lane; a < NB_MAX * NB_MAX; a += 32) Tm[a] = Ts[a];
}

// One column step with a RUN-TIME column index jj: the column being eliminated is always x[.][0]
// and the panel is shifted left by one column afterwards, so the same (small) code runs for every
// column (unrolling the step per column made the kernel 9000 instructions long and instruction-
// fetch bound).  The finished reflector goes straight to X; R entries to Rm.
template <int RP_THREADS, int RPT, int NB>
__device__ __forceinline__ void qr_panel_col(c128 (&x)[RPT][NB], c128 (*pivot)[NB], double *sm, c128 *tau_s, c128 *Rm,
                                             c128 *X, int rows, int cols, int j0, int len, int tid, int jj) {
  constexpr int NRED = 1 + 2 * (NB - 1);
  double red[NRED];
#pragma unroll
  for (int q = 0; q < NRED; q++) red[q] = 0.0;
#pragma unroll
  for (int r = 0; r < RPT; r++) {
    const int i = tid + r * RP_THREADS;
    if (i >= jj && i < len) {
      const c128 u = x[r][0];
      red[0] = fma(u.x, u.x, fma(u.y, u.y, red[0]));     // explicit FMA chains: the step is FP64-issue bound
      if (i == jj) pivot[jj & 1][0] = u;
#pragma unroll
      for (int c = 1; c < NB; c++) {
        const c128 yv = x[r][c];
        red[1 + 2 * (c - 1)] = fma(u.x, yv.x, fma(u.y, yv.y, red[1 + 2 * (c - 1)]));
        red[2 + 2 * (c - 1)] = fma(u.x, yv.y, fma(-u.y, yv.x, red[2 + 2 * (c - 1)]));
        if (i == jj) pivot[jj & 1][c] = yv;
      }
    }
  }
  block_sum<NRED, RP_THREADS>(red, sm);
  const c128 alpha = pivot[jj & 1][0];
  double xn2 = red[0] - (alpha.x * alpha.x + alpha.y * alpha.y);
  if (xn2 < 0.0) xn2 = 0.0;
  c128 tau, scal;
  double beta;
  if ((xn2 == 0.0 && alpha.y == 0.0) || alpha.x * alpha.x + alpha.y * alpha.y + xn2 < TINY_NORM2) {
    tau = make_double2(0.0, 0.0); scal = make_double2(0.0, 0.0); beta = alpha.x;
  } else {
    const double nrm = sqrt(alpha.x * alpha.x + alpha.y * alpha.y + xn2);
    beta = alpha.x >= 0.0 ? -nrm : nrm;
    const double ib = 1.0 / beta;
    tau = make_double2((beta - alpha.x) * ib, -alpha.y * ib);
    const double dr = alpha.x - beta, di = alpha.y, idn = 1.0 / (dr * dr + di * di);
    scal = make_double2(dr * idn, -di * idn);
  }
  if (tid == 0) { tau_s[jj] = tau; Rm[(long long)(j0 + jj) * cols + j0 + jj] = make_double2(beta, 0.0); }
  c128 g[NB];                                            // conj(tau) * (v^H y_c)
#pragma unroll
  for (int c = 1; c < NB; c++) {
    const c128 dc = make_double2(red[1 + 2 * (c - 1)], red[2 + 2 * (c - 1)]);
    const c128 yj = pivot[jj & 1][c];
    const c128 t1 = cmul(cconj(alpha), yj);
    const c128 t2 = cmul(cconj(scal), make_double2(dc.x - t1.x, dc.y - t1.y));
    g[c] = cmul(cconj(tau), make_double2(yj.x + t2.x, yj.y + t2.y));
  }
  c128 *Xc = X + (long long)(j0 + jj) * rows + j0;
#pragma unroll
  for (int r = 0; r < RPT; r++) {
    const int i = tid + r * RP_THREADS;
    if (i < len) {
      if (i < jj) {                                      // above the diagonal: an R entry, zero in V
        Rm[(long long)(j0 + i) * cols + j0 + jj] = x[r][0];
        Xc[i] = make_double2(0.0, 0.0);
      } else {
        const c128 v = (i == jj) ? make_double2(1.0, 0.0) : cmul(x[r][0], scal);
        Xc[i] = v;
#pragma unroll
        for (int c = 1; c < NB; c++) {
          x[r][c].x = fma(g[c].y, v.y, fma(-g[c].x, v.x, x[r][c].x));
          x[r][c].y = fma(-g[c].y, v.x, fma(-g[c].x, v.y, x[r][c].y));
        }
      }
    }
#pragma unroll
    for (int c = 0; c < NB - 1; c++) x[r][c] = x[r][c + 1];
    x[r][NB - 1] = make_double2(0.0, 0.0);
  }
}

template <int RP_THREADS, int RPT, int NB>
__global__ void __maxnreg__(RP_THREADS <= 256 ? 255 : 128) qr_panel_reg_kernel(c128 *X, int rows, int cols, int j0, int w,
                                                                   c128 *Rm, c128 *Tm /*[NB_MAX][NB_MAX]*/) {
  constexpr int NRED = 1 + 2 * (NB - 1);                 // s and d_c for the other columns
  constexpr int NGRAM = NB * (NB - 1);                   // re/im of the strictly upper Gram entries
  constexpr int NSM = NRED > NGRAM ? NRED : NGRAM;
  constexpr int RP_WARPS = RP_THREADS / 32;
  __shared__ c128 pivot[2][NB];                          // pivot row (alpha, y_c[jj]), double-buffered over jj
  __shared__ double sm[(RP_WARPS + 1) * (NSM > 0 ? NSM : 1)];
  __shared__ c128 tau_s[NB];
  __shared__ c128 Ts[NB_MAX * NB_MAX];
  __shared__ c128 Gs[NB_MAX * NB_MAX];
  const int len = rows - j0, tid = threadIdx.x;
  c128 x[RPT][NB];
#pragma unroll
  for (int r = 0; r < RPT; r++) {
    const int i = tid + r * RP_THREADS;
#pragma unroll
    for (int c = 0; c < NB; c++)
      x[r][c] = (i < len && c < w) ? X[(long long)(j0 + c) * rows + j0 + i] : make_double2(0.0, 0.0);
  }
  for (int i = tid; i < j0; i += RP_THREADS)              // R entries above the panel rows are final
    for (int c = 0; c < w; c++) Rm[(long long)i * cols + j0 + c] = X[(long long)(j0 + c) * rows + i];
  for (int i = j0 + 1 + tid; i < cols; i += RP_THREADS)   // zeros below the diagonal of R
    for (int c = 0; c < w; c++)
      if (i > j0 + c) Rm[(long long)i * cols + j0 + c] = make_double2(0.0, 0.0);
  // columns one by one; every finished reflector is written to X by the step itself
  for (int jj = 0; jj < w; jj++) qr_panel_col<RP_THREADS, RPT, NB>(x, pivot, sm, tau_s, Rm, X, rows, cols, j0, len, tid, jj);
  // read the reflector block back (own writes: same thread, same addresses) for the Gram matrix
#pragma unroll
  for (int r = 0; r < RPT; r++) {
    const int i = tid + r * RP_THREADS;
#pragma unroll
    for (int c = 0; c < NB; c++)
      x[r][c] = (i < len && c < w) ? X[(long long)(j0 + c) * rows + j0 + i] : make_double2(0.0, 0.0);
  }
  // compact WY factor from the strictly upper Gram entries v_a^H v_b
  if (NB > 1) {
    // all strictly upper Gram entries v_a^H v_b in ONE block reduction
    double gr[NGRAM > 0 ? NGRAM : 1];
#pragma unroll
    for (int q = 0; q < NGRAM; q++) gr[q] = 0.0;
#pragma unroll
    for (int r = 0; r < RPT; r++) {
      int q = 0;
#pragma unroll
      for (int a = 0; a < NB - 1; a++) {
        const c128 u = x[r][a];
#pragma unroll
        for (int b = a + 1; b < NB; b++) {
          const c128 v = x[r][b];
          gr[q] = fma(u.x, v.x, fma(u.y, v.y, gr[q]));
          gr[q + 1] = fma(u.x, v.y, fma(-u.y, v.x, gr[q + 1]));
          q += 2;
        }
      }
    }
    block_sum<NGRAM, RP_THREADS>(gr, sm);
    if (tid == 0) {
      int q = 0;
#pragma unroll
      for (int a = 0; a < NB - 1; a++)
#pragma unroll
        for (int b = a + 1; b < NB; b++) { Gs[a * NB_MAX + b] = make_double2(gr[q], gr[q + 1]); q += 2; }
    }
  }
  __syncthreads();
  if (tid < 32) build_T(Gs, tau_s, Ts, Tm, w);
}

// ---- cluster panel factorisation ---------------------------------------------------------------
// The same column-by-column Householder elimination (one combined reduction per column, see above), with
// the panel's rows spread over a thread-block CLUSTER of QC CTAs (QC SMs): a column step is bound by the
// FP64 and shuffle throughput of the SM(s) that hold the panel -- 2.9 us per column for 1280 rows on one
// SM -- and by the reduction's latency.  Here every CTA reduces its rows (warp level: a transposed
// butterfly, 16 values in 16 shuffle steps instead of 75), pushes its 16 partial sums into the shared
// memory of ALL CTAs of the cluster (st.shared::cluster), and after ONE cluster barrier every CTA adds
// the QC partials in the same order, so all hold bit-identical scalars.  The pivot row (alpha and the
// pivot entries of the other columns) travels in the same message from the CTA that owns it.  Exchange
// slots are double-buffered by column parity, which makes one barrier per column enough.
// Rows are dealt round-robin: local row i = r * (QC * QT) + cta * QT + tid.
constexpr int QC = 16;                // CTAs per cluster (non-portable size: allowed explicitly in qr_configure)
constexpr int QT = 256;               // threads per CTA
constexpr int QW = QT / 32;

__device__ __forceinline__ unsigned cluster_ctarank() { unsigned r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ void cluster_barrier() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n" ::: "memory");
  asm volatile("barrier.cluster.wait.acquire.aligned;\n" ::: "memory");
}
__device__ __forceinline__ void st_cluster_f64(const double *local_addr, unsigned cta, double v) {
  const unsigned la = (unsigned)__cvta_generic_to_shared(local_addr);
  unsigned ra;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(la), "r"(cta));
  asm volatile("st.shared::cluster.f64 [%0], %1;" ::"r"(ra), "d"(v) : "memory");
}
// Sum 16 values per lane over the warp: afterwards lane l holds the total of value index
// 8 b4 + 4 b3 + 2 b2 + b1 (b_k = bit k of l), in a fixed order.  16 shuffle steps.
__device__ __forceinline__ double warp_reduce16(double (&v)[16], int lane, int &index) {
#pragma unroll
  for (int o = 16, half = 8; o >= 2; o >>= 1, half >>= 1) {
    const bool bit = (lane & o) != 0;
#pragma unroll
    for (int i = 0; i < half; i++) {
      const double send = bit ? v[i] : v[i + half];
      const double keep = bit ? v[i + half] : v[i];
      v[i] = keep + __shfl_xor_sync(0xffffffffu, send, o);
    }
  }
  index = ((lane >> 4) & 1) * 8 + ((lane >> 3) & 1) * 4 + ((lane >> 2) & 1) * 2 + ((lane >> 1) & 1);
  return v[0] + __shfl_xor_sync(0xffffffffu, v[0], 1);
}

// Exchange: every CTA contributes `n` doubles (n <= 64; loc[] in its own shared memory; entries >= n_sum are
// taken from CTA `owner` only); afterwards tot[t] = sum over CTAs (t < n_sum) or owner's value, in all CTAs.
__device__ __forceinline__ void cluster_exchange(const double *loc, int n, int n_sum, unsigned owner, double *exch /*[QC][64]*/,
                                                 double *tot /*[64]*/, unsigned me) {
  const int t = threadIdx.x;
  if (t < n && (t < n_sum || me == owner)) {
    const double v = loc[t];
#pragma unroll
    for (unsigned c = 0; c < QC; c++) st_cluster_f64(exch + me * 64 + t, c, v);
  }
  cluster_barrier();
  if (t < n) {
    double a;
    if (t < n_sum) {
      a = 0.0;
#pragma unroll
      for (int c = 0; c < QC; c++) a += exch[c * 64 + t];
    } else {
      a = exch[owner * 64 + t];
    }
    tot[t] = a;
  }
  __syncthreads();
}


// ---- fast panel: the column steps' reductions predicted from ONE Gram matrix -------------------------
// The column-by-column elimination pays one cluster-wide reduction per COLUMN (2.2 us each: 17 us per panel of
// eight).  What a column step jj reduces -- s = sum_{i>=jj} |x_i,jj|^2 and d_c = sum_{i>=jj} conj(x_i,jj) x_i,c over
// the CURRENT (partly eliminated) panel -- follows from the panel's Gram matrix G = P^H P and its top 8 x 8 block
// alone: a reflector is unitary on the rows it acts on, so the sums over rows >= jj of the updated columns equal
// those of the columns before the update, and leaving out row jj afterwards subtracts conj(R[jj][a]) R[jj][b] -- the
// Cholesky downdate with the new row of R.  One warp runs that 8-step recurrence on 8 x 8 data (lane = column, in
// registers, neighbours by shuffles) and writes, for every step, the reflector's scalars and its products with the
// columns to its right (what every thread otherwise derives, redundantly, from the exchanged sums: a square root,
// two divisions and seven complex products per thread and column, about half of a column step's 2.2 us on its
// own); all threads then run the eight column updates back to back, without a barrier.  One cluster reduction per
// panel instead of eight.
// The predicted sums are differences: s loses log10(G_jj / s) digits.  A panel in which some column keeps less than
// FAST_TAIL_MIN of its squared norm after the columns before it have been eliminated (nearly dependent or zero
// columns: the padded / delta-seeded centres this file's header is about; typically also the first panel of a
// centre dominated by one singular vector) is left to the exact column-by-column path, untouched.  With the
// threshold at 1e-2 the reflectors' scalars carry at most ~100 eps: isometry and reconstruction stay at 1e-15
// (tests/test_gpu_parity.py::test_qr_gauge).  The decision is taken from the exchanged sums, which are
// bit-identical in every CTA.  TDVP_QR_FAST=0 switches the path off.
constexpr double FAST_TAIL_MIN = 1e-2;

// 64 Gram sums of one row's eight entries, added to acc: acc[c] += |x_c|^2, acc[8 + 2 q], acc[9 + 2 q] += conj(x_a) x_b
// (q = index of the pair a < b in row-major order)
__device__ __forceinline__ void gram8_accumulate(double (&acc)[64], const c128 (&x)[NB_MAX]) {
  int q = 0;
#pragma unroll
  for (int a = 0; a < NB_MAX; a++) {
    acc[a] = fma(x[a].x, x[a].x, fma(x[a].y, x[a].y, acc[a]));
#pragma unroll
    for (int b = a + 1; b < NB_MAX; b++) {
      acc[8 + 2 * q] = fma(x[a].x, x[b].x, fma(x[a].y, x[b].y, acc[8 + 2 * q]));
      acc[9 + 2 * q] = fma(x[a].x, x[b].y, fma(-x[a].y, x[b].x, acc[9 + 2 * q]));
      q++;
    }
  }
}
__device__ __forceinline__ c128 shfl_c(c128 v, int src) {
  return make_double2(__shfl_sync(0xffffffffu, v.x, src), __shfl_sync(0xffffffffu, v.y, src));
}
// The reflector of a column with pivot alpha and squared norm xn2 below it (the scalars of the column step)
__device__ __forceinline__ void house_scalars(c128 alpha, double xn2, c128 &tau, c128 &scal, double &beta) {
  if ((xn2 == 0.0 && alpha.y == 0.0) || alpha.x * alpha.x + alpha.y * alpha.y + xn2 < TINY_NORM2) {
    tau = make_double2(0.0, 0.0); scal = make_double2(0.0, 0.0); beta = alpha.x;
  } else {
    const double nrm = sqrt(alpha.x * alpha.x + alpha.y * alpha.y + xn2);
    beta = alpha.x >= 0.0 ? -nrm : nrm;
    const double ib = 1.0 / beta;
    tau = make_double2((beta - alpha.x) * ib, -alpha.y * ib);
    const double dr = alpha.x - beta, di = alpha.y, idn = 1.0 / (dr * dr + di * di);
    scal = make_double2(dr * idn, -di * idn);
  }
}
// One warp, lane c < 8 = column c of the panel: g = the 64 Gram sums (layout of gram8_accumulate), B[i] = entry
// (row i, column c) of the panel's top block.  Writes tab[jj][.] = what column step jj applies: [0], [1] scal, [2], [3]
// tau, [4] beta, [8 + 2 c'], [9 + 2 c'] g = conj(tau) v^H y for the column c' = c - jj places to the right (the kernel
// keeps the current column in slot 0), and returns whether every column kept FAST_TAIL_MIN of its norm (all lanes).
__device__ __forceinline__ bool predict_panel(const double *g, c128 (&B)[NB_MAX], double (*tab)[32], int lane) {
  constexpr int N = NB_MAX;
  c128 G[N];                                              // G[a] = Gram entry (a, lane)
  {
    int q = 0;
#pragma unroll
    for (int a = 0; a < N; a++) {
      G[a] = make_double2(0.0, 0.0);
#pragma unroll
      for (int b = a + 1; b < N; b++) {
        if (lane < N) {
          if (b == lane) G[a] = make_double2(g[8 + 2 * q], g[9 + 2 * q]);
        }
        q++;
      }
    }
    q = 0;
#pragma unroll
    for (int a = 0; a < N; a++)
#pragma unroll
      for (int b = a + 1; b < N; b++) { if (a == lane) G[b] = make_double2(g[8 + 2 * q], -g[9 + 2 * q]); q++; }
#pragma unroll
    for (int a = 0; a < N; a++) if (a == lane) G[a] = make_double2(g[a], 0.0);
  }
  const double g0 = lane < N ? g[lane] : 0.0;
  if (lane >= N) {
#pragma unroll
    for (int i = 0; i < N; i++) B[i] = make_double2(0.0, 0.0);
  }
  bool ok = true;
#pragma unroll
  for (int jj = 0; jj < N; jj++) {
    const c128 alpha = shfl_c(B[jj], jj);
    const double s = __shfl_sync(0xffffffffu, G[jj].x, jj);
    const double g0j = __shfl_sync(0xffffffffu, g0, jj);
    if (!(s >= FAST_TAIL_MIN * g0j) || !(g0j > 0.0) || !(g0j < 1e300)) ok = false;
    double xn2 = s - (alpha.x * alpha.x + alpha.y * alpha.y);
    if (xn2 < 0.0) xn2 = 0.0;
    c128 tau, scal;
    double beta;
    house_scalars(alpha, xn2, tau, scal, beta);
    const c128 dc = G[jj], yj = B[jj];
    c128 gg = make_double2(0.0, 0.0);
    if (lane > jj && lane < N) {
      const c128 t1 = cmul(cconj(alpha), yj);
      const c128 t2 = cmul(cconj(scal), make_double2(dc.x - t1.x, dc.y - t1.y));
      gg = cmul(cconj(tau), make_double2(yj.x + t2.x, yj.y + t2.y));
      const int cp = lane - jj;
      tab[jj][8 + 2 * cp] = gg.x; tab[jj][9 + 2 * cp] = gg.y;
    } else if (lane == jj) {
      tab[jj][0] = scal.x; tab[jj][1] = scal.y; tab[jj][2] = tau.x; tab[jj][3] = tau.y; tab[jj][4] = beta;
    } else if (lane < jj) {                                // slots of finished reflectors at the back: no column there
      const int cp = N - jj + lane;
      tab[jj][8 + 2 * cp] = 0.0; tab[jj][9 + 2 * cp] = 0.0;
    }
    // row jj of R as this step leaves it (this lane's entry), the top block's rows below it, the Gram downdate
    const c128 rrow = lane == jj ? make_double2(beta, 0.0) : make_double2(yj.x - gg.x, yj.y - gg.y);
#pragma unroll
    for (int i = jj + 1; i < N; i++) {
      const c128 v = cmul(shfl_c(B[i], jj), scal);
      if (lane > jj) { const c128 u = cmul(gg, v); B[i].x -= u.x; B[i].y -= u.y; }
    }
#pragma unroll
    for (int a = jj + 1; a < N; a++) {
      const c128 ra = shfl_c(rrow, a);
      if (lane > jj) { const c128 u = cmul(cconj(ra), rrow); G[a].x -= u.x; G[a].y -= u.y; }
    }
  }
  return ok;
}

// The WHOLE factorisation in one kernel, by one cluster: for every panel (1) the column-by-column
// elimination above with the panel's rows spread over the cluster, (2) the compact-WY factor T, built by
// every CTA for itself from the exchanged Gram sums, (3) the trailing update X[:, c] <- (I - V T^H V^H) X[:, c]
// with the COLUMNS dealt round-robin to the CTAs (all rows of a column in one CTA: its reductions stay
// inside the CTA, V is read back from global memory / L2 into registers once per panel and CTA).  Cluster
// barriers separate the phases (their release / acquire covers global memory).  Against one launch per
// panel and per update (2 x 16 launches for 128 columns) this removes the launch gaps and the cold
// instruction fetch of every launch -- the panel kernel's stall profile was dominated by both -- and the
// per-column reduction no longer waits on one SM's FP64 and shuffle throughput.
// RA = rows per thread in the update (rows <= RA * QT), NB = panel width; rows per thread in the panel
// phase RPT = ceil(RA / QC).  Forming Q stays a kernel of its own (one CTA per column, all SMs).
template <int RA, int NB>
__global__ void __cluster_dims__(QC, 1, 1) __launch_bounds__(QT, 1)
qr_factor_cluster_kernel(c128 *X, int rows, int cols, c128 *Rm, c128 *Tm /*[npanels][NB_MAX][NB_MAX]*/,
                         const int *gate /*DEVICE, nullable: run only if non-zero (written by an earlier kernel of the stream)*/,
                         int fast /*try the one-reduction panel (predict_panel) first*/) {
  if (gate && __ldcg(gate) == 0) return;                   // every CTA of the cluster reads the same value
  constexpr int RPT = (RA + QC - 1) / QC;
  constexpr int NGRAM = NB * (NB - 1);                   // re / im of the strictly upper Gram entries (<= 56)
  constexpr int NGB = (NGRAM + 15) / 16;                 // 16-value reduction rounds for them
  extern __shared__ __align__(16) unsigned char qr_dyn_smem[];
  c128 *vsm = reinterpret_cast<c128 *>(qr_dyn_smem);     // [NB][RA * QT]: the reflector block during the update
  __shared__ double exch[2][QC * 64];
  __shared__ double loc[64], tot[64];
  __shared__ double wpart[QW][64];
  __shared__ c128 tau_s[NB_MAX];
  __shared__ c128 Ts[NB_MAX * NB_MAX];
  __shared__ c128 Tl[NB_MAX * NB_MAX];
  __shared__ c128 Gs[NB_MAX * NB_MAX];
  __shared__ double ftab[NB_MAX][32];                     // fast panel: the predicted sums of every column step
  __shared__ int fOk;
  const unsigned me = cluster_ctarank();
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int gthread = (int)me * QT + tid;
  unsigned par = 0;                                         // parity of the exchange slots
  cluster_barrier();                                        // every CTA of the cluster is running: its shared memory may be written
  const int npanels = (cols + NB - 1) / NB;
  for (int pz = 0; pz < npanels; pz++) {
    const int j0 = pz * NB, w = cols - j0 < NB ? cols - j0 : NB;
    const int len = rows - j0;
    c128 *Tp = Tm + (size_t)pz * NB_MAX * NB_MAX;
    auto row_of = [&](int r) { return r * (QC * QT) + gthread; };
    // ---- (1) panel: rows round-robin over the cluster, in registers ----
    c128 x[RPT][NB];
#pragma unroll
    for (int r = 0; r < RPT; r++) {
      const int i = row_of(r);
#pragma unroll
      for (int c = 0; c < NB; c++)
        x[r][c] = (i < len && c < w) ? __ldcg(X + (long long)(j0 + c) * rows + j0 + i) : make_double2(0.0, 0.0);
    }
    for (int i = gthread; i < j0; i += QC * QT)               // R entries above the panel rows are final
      for (int c = 0; c < w; c++) Rm[(long long)i * cols + j0 + c] = __ldcg(X + (long long)(j0 + c) * rows + i);
    for (int i = j0 + 1 + gthread; i < cols; i += QC * QT)    // zeros below the diagonal of R
      for (int c = 0; c < w; c++)
        if (i > j0 + c) Rm[(long long)i * cols + j0 + c] = make_double2(0.0, 0.0);
    // ---- fast panel: one Gram reduction, then the column steps' sums by recurrence (predict_panel) ----
    bool predicted = false;
    if (fast && RPT == 1 && NB == NB_MAX && w == NB) {
      c128 ptop[NB_MAX];                                    // top block, lane = column (warp 0 of every CTA)
      if (tid < NB_MAX) {
#pragma unroll
        for (int i = 0; i < NB_MAX; i++) ptop[i] = __ldcg(X + (long long)(j0 + tid) * rows + j0 + i);
      }
      double acc[64];
#pragma unroll
      for (int t = 0; t < 64; t++) acc[t] = 0.0;
      if (row_of(0) < len) {
        c128 xr[NB_MAX];
#pragma unroll
        for (int c = 0; c < NB_MAX; c++) xr[c] = x[0][c < NB ? c : 0];
        gram8_accumulate(acc, xr);
      }
#pragma unroll
      for (int blk = 0; blk < 4; blk++) {
        double v16[16];
#pragma unroll
        for (int q = 0; q < 16; q++) v16[q] = acc[blk * 16 + q];
        int idx;
        const double part = warp_reduce16(v16, lane, idx);
        if ((lane & 1) == 0) wpart[warp][blk * 16 + idx] = part;
      }
      __syncthreads();
      if (tid < 64) { double a = 0.0; for (int k = 0; k < QW; k++) a += wpart[k][tid]; loc[tid] = a; }
      __syncthreads();
      cluster_exchange(loc, 64, 64, 0u, exch[par], tot, me);
      par ^= 1u;
      if (warp == 0) { const bool ok = predict_panel(tot, ptop, ftab, lane); if (lane == 0) fOk = ok ? 1 : 0; }
      __syncthreads();
      predicted = fOk != 0;                                 // (same sums, hence the same decision, in every CTA)
    }
    for (int jj = 0; jj < w; jj++) {
      const double *tt = tot;                               // where the step's sums come from
      if (predicted) {
        tt = ftab[jj];
      } else {
      double red[16];
#pragma unroll
      for (int q = 0; q < 16; q++) red[q] = 0.0;
#pragma unroll
      for (int r = 0; r < RPT; r++) {
        const int i = row_of(r);
        if (i >= jj && i < len) {
          const c128 u = x[r][0];
          red[0] = fma(u.x, u.x, fma(u.y, u.y, red[0]));
#pragma unroll
          for (int c = 1; c < NB; c++) {
            const c128 yv = x[r][c];
            red[1 + 2 * (c - 1)] = fma(u.x, yv.x, fma(u.y, yv.y, red[1 + 2 * (c - 1)]));
            red[2 + 2 * (c - 1)] = fma(u.x, yv.y, fma(-u.y, yv.x, red[2 + 2 * (c - 1)]));
          }
          if (i == jj) {                                      // pivot row: owner is CTA 0, thread jj (jj < NB <= QT)
#pragma unroll
            for (int c = 0; c < NB; c++) { loc[16 + 2 * c] = x[r][c].x; loc[17 + 2 * c] = x[r][c].y; }
          }
        }
      }
      int idx;
      const double part = warp_reduce16(red, lane, idx);
      if ((lane & 1) == 0) wpart[warp][idx] = part;
      __syncthreads();
      if (tid < 16) { double a = 0.0; for (int k = 0; k < QW; k++) a += wpart[k][tid]; loc[tid] = a; }
      __syncthreads();
      cluster_exchange(loc, 16 + 2 * NB, 16, 0u, exch[par], tot, me);
      par ^= 1u;
      }
      c128 tau, scal, alpha = make_double2(0.0, 0.0);
      double beta;
      if (predicted) {
        scal = make_double2(tt[0], tt[1]); tau = make_double2(tt[2], tt[3]); beta = tt[4];
      } else {
        alpha = make_double2(tt[16], tt[17]);
        double xn2 = tt[0] - (alpha.x * alpha.x + alpha.y * alpha.y);
        if (xn2 < 0.0) xn2 = 0.0;
        house_scalars(alpha, xn2, tau, scal, beta);
      }
      if (tid == 0) {
        tau_s[jj] = tau;                                    // every CTA keeps the taus: it builds T itself
        if (me == 0) Rm[(long long)(j0 + jj) * cols + j0 + jj] = make_double2(beta, 0.0);
      }
      c128 g[NB];                                            // conj(tau) * (v^H y_c)
#pragma unroll
      for (int c = 1; c < NB; c++) {
        if (predicted) {
          g[c] = make_double2(tt[8 + 2 * c], tt[9 + 2 * c]);
        } else {
          const c128 dc = make_double2(tt[1 + 2 * (c - 1)], tt[2 + 2 * (c - 1)]);
          const c128 yj = make_double2(tt[16 + 2 * c], tt[17 + 2 * c]);
          const c128 t1 = cmul(cconj(alpha), yj);
          const c128 t2 = cmul(cconj(scal), make_double2(dc.x - t1.x, dc.y - t1.y));
          g[c] = cmul(cconj(tau), make_double2(yj.x + t2.x, yj.y + t2.y));
        }
        if (c >= NB - jj) g[c] = make_double2(0.0, 0.0);     // slots at the back hold finished reflectors: not columns
      }
      c128 *Xc = X + (long long)(j0 + jj) * rows + j0;
#pragma unroll
      for (int r = 0; r < RPT; r++) {
        const int i = row_of(r);
        if (i < len) {
          if (i < jj) {                                      // above the diagonal: an R entry, zero in V
            Rm[(long long)(j0 + i) * cols + j0 + jj] = x[r][0];
            Xc[i] = make_double2(0.0, 0.0);
          } else {
            const c128 v = (i == jj) ? make_double2(1.0, 0.0) : cmul(x[r][0], scal);
            Xc[i] = v;
            x[r][0] = v;                                     // kept (rotated to the back below) for the Gram matrix
#pragma unroll
            for (int c = 1; c < NB; c++) {
              x[r][c].x = fma(g[c].y, v.y, fma(-g[c].x, v.x, x[r][c].x));
              x[r][c].y = fma(-g[c].y, v.x, fma(-g[c].x, v.y, x[r][c].y));
            }
          }
        }
        if (i >= len || i < jj) x[r][0] = make_double2(0.0, 0.0);
        // rotate: the finished reflector goes to the back, so after w steps x[r][NB - w + a] = v_a[row]
        const c128 fin = x[r][0];
#pragma unroll
        for (int c = 0; c < NB - 1; c++) x[r][c] = x[r][c + 1];
        x[r][NB - 1] = fin;
      }
    }
    // ---- (2) compact WY factor from the strictly upper Gram entries v_a^H v_b (reflector a sits in x[.][NB - w + a]) ----
    if (NB > 1 && w > 1) {
      double gr[NGB * 16];
#pragma unroll
      for (int q = 0; q < NGB * 16; q++) gr[q] = 0.0;
      if (w == NB) {                                        // full panel: reflector a sits in slot a (static indexing)
#pragma unroll
        for (int r = 0; r < RPT; r++) {
          int q = 0;
#pragma unroll
          for (int a = 0; a < NB - 1; a++) {
            const c128 u = x[r][a];
#pragma unroll
            for (int b = a + 1; b < NB; b++) {
              const c128 v = x[r][b];
              gr[q] = fma(u.x, v.x, fma(u.y, v.y, gr[q]));
              gr[q + 1] = fma(u.x, v.y, fma(-u.y, v.x, gr[q + 1]));
              q += 2;
            }
          }
        }
      } else {                                              // the ragged last panel: slots NB - w + a, selected at run time
#pragma unroll 1
        for (int r = 0; r < RPT; r++) {
          int q = 0;
#pragma unroll
          for (int a = 0; a < NB - 1; a++) {
#pragma unroll
            for (int b = a + 1; b < NB; b++) {
              const int sa = NB - w + a, sb = NB - w + b;
              if (b < w) {
                c128 u = make_double2(0.0, 0.0), v = make_double2(0.0, 0.0);
#pragma unroll
                for (int c = 0; c < NB; c++) { if (c == sa) u = x[r][c]; if (c == sb) v = x[r][c]; }
                gr[q] = fma(u.x, v.x, fma(u.y, v.y, gr[q]));
                gr[q + 1] = fma(u.x, v.y, fma(-u.y, v.x, gr[q + 1]));
              }
              q += 2;
            }
          }
        }
      }
#pragma unroll
      for (int blk = 0; blk < NGB; blk++) {
        double v16[16];
#pragma unroll
        for (int q = 0; q < 16; q++) v16[q] = gr[blk * 16 + q];
        int idx;
        const double part = warp_reduce16(v16, lane, idx);
        if ((lane & 1) == 0) wpart[warp][blk * 16 + idx] = part;
      }
      __syncthreads();
      if (tid < NGB * 16) { double a = 0.0; for (int k = 0; k < QW; k++) a += wpart[k][tid]; loc[tid] = a; }
      __syncthreads();
      cluster_exchange(loc, NGB * 16, NGB * 16, 0u, exch[par], tot, me);
      par ^= 1u;
      if (tid == 0) {
        int q = 0;
        for (int a = 0; a < NB - 1; a++)
          for (int b = a + 1; b < NB; b++) { Gs[a * NB_MAX + b] = make_double2(tot[q], tot[q + 1]); q += 2; }
      }
    }
    __syncthreads();
    if (tid < 32) build_T(Gs, tau_s, Ts, me == 0 ? Tp : Tl, w);
    cluster_barrier();                                      // V (global) complete and visible; Ts ready in every CTA
    // ---- (3) trailing update: column c to CTA (c - c_begin) % QC, all its rows >= j0 in this CTA ----
    const int c_begin = j0 + w;
    if (c_begin + (int)me < cols) {
      // the reflector block V of this panel: global memory / L2 -> shared memory, [q][row - j0] (its registers
      // are needed for two columns in flight and the prefetch of the next two)
#pragma unroll
      for (int r = 0; r < RA; r++) {
        const int i = j0 + tid + r * QT;
#pragma unroll
        for (int q = 0; q < NB; q++)
          vsm[q * (RA * QT) + tid + r * QT] = (i < rows && q < w) ? __ldcg(X + (long long)(j0 + q) * rows + i) : make_double2(0.0, 0.0);
      }
      // (each thread reads back only what it wrote: no barrier needed)
      auto v = [&](int r, int q) -> c128 { return vsm[q * (RA * QT) + tid + r * QT]; };
      // two columns per pass (one pair of block barriers for both), the next pair's loads issued before the
      // reductions of this one: a pass is a chain of latencies (L2 load, shuffles, barriers), not of flops
      auto load_col = [&](int c, c128 (&y)[RA]) {
#pragma unroll
        for (int r = 0; r < RA; r++) {
          const int i = j0 + tid + r * QT;
          y[r] = (c < cols && i < rows) ? __ldcg(X + (long long)c * rows + i) : make_double2(0.0, 0.0);
        }
      };
      c128 ya[RA], yb[RA];
      int c = c_begin + (int)me;
      load_col(c, ya); load_col(c + QC, yb);
      for (; c < cols; c += 2 * QC) {
        double acc[16], acc2[16];
#pragma unroll
        for (int q = 0; q < 16; q++) acc[q] = acc2[q] = 0.0;
#pragma unroll
        for (int r = 0; r < RA; r++)
#pragma unroll
          for (int q = 0; q < NB; q++) {
            const c128 vv = v(r, q);
            acc[2 * q] = fma(vv.x, ya[r].x, fma(vv.y, ya[r].y, acc[2 * q]));
            acc[2 * q + 1] = fma(vv.x, ya[r].y, fma(-vv.y, ya[r].x, acc[2 * q + 1]));
            acc2[2 * q] = fma(vv.x, yb[r].x, fma(vv.y, yb[r].y, acc2[2 * q]));
            acc2[2 * q + 1] = fma(vv.x, yb[r].y, fma(-vv.y, yb[r].x, acc2[2 * q + 1]));
          }
        int idx;
        const double part = warp_reduce16(acc, lane, idx);
        const double part2 = warp_reduce16(acc2, lane, idx);
        if ((lane & 1) == 0) { wpart[warp][idx] = part; wpart[warp][16 + idx] = part2; }
        __syncthreads();
        if (tid < 32) { double a = 0.0; for (int k = 0; k < QW; k++) a += wpart[k][tid]; loc[tid] = a; }
        __syncthreads();
        if (tid < 2 * NB) {                                 // T^H (V^H y): one component of one column per thread, then shared
          const int col = tid / NB, q = tid % NB;
          c128 a = make_double2(0.0, 0.0);
#pragma unroll
          for (int r = 0; r < NB; r++) {
            const c128 pr = cmul(cconj(Ts[r * NB_MAX + q]), make_double2(loc[16 * col + 2 * r], loc[16 * col + 2 * r + 1]));
            a.x += pr.x; a.y += pr.y;
          }
          tot[16 * col + 2 * q] = a.x; tot[16 * col + 2 * q + 1] = a.y;
        }
        __syncthreads();
        c128 na[RA], nb2[RA];
        load_col(c + 2 * QC, na); load_col(c + 3 * QC, nb2);    // next pair: in flight during the update below
#pragma unroll
        for (int r = 0; r < RA; r++) {
#pragma unroll
          for (int q = 0; q < NB; q++) {
            const c128 s1 = make_double2(tot[2 * q], tot[2 * q + 1]), s2 = make_double2(tot[16 + 2 * q], tot[17 + 2 * q]);
            const c128 vv = v(r, q);
            ya[r].x = fma(vv.y, s1.y, fma(-vv.x, s1.x, ya[r].x));
            ya[r].y = fma(-vv.y, s1.x, fma(-vv.x, s1.y, ya[r].y));
            yb[r].x = fma(vv.y, s2.y, fma(-vv.x, s2.x, yb[r].x));
            yb[r].y = fma(-vv.y, s2.x, fma(-vv.x, s2.y, yb[r].y));
          }
          const int i = j0 + tid + r * QT;
          if (i < rows) {
            X[(long long)c * rows + i] = ya[r];
            if (c + QC < cols) X[(long long)(c + QC) * rows + i] = yb[r];
          }
          ya[r] = na[r]; yb[r] = nb2[r];
        }
        // wpart / loc / tot are rewritten only after the next pass's first barrier ... tot after its second
      }
    }
    cluster_barrier();                                      // the updated columns are visible before the next panel is read
  }
}

// Factor the panel of columns [j0, j0+w) on rows [j0, rows).  Writes reflectors back into X (unit
// diagonal explicit, zeros above it inside the panel rows), R entries of these columns into Rm
// (row-major cols x cols, zeros below the diagonal), tau and the w x w upper-triangular T.
__global__ void __launch_bounds__(PANEL_THREADS) qr_panel_kernel(c128 *X, int rows, int cols, int j0, int w,
                                                                  c128 *Rm, c128 *Tm /*[NB_MAX][NB_MAX]*/) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int len = rows - j0;
  c128 *P = reinterpret_cast<c128 *>(smem_raw);                // [w][len]
  __shared__ double red[PANEL_THREADS / 32];
  __shared__ c128 wdot[NB_MAX];
  __shared__ c128 tau_s[NB_MAX];
  __shared__ c128 gram[NB_MAX][NB_MAX];
  __shared__ c128 scal_s;
  __shared__ double beta_s;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  constexpr int NW = PANEL_THREADS / 32;

  for (int e = tid; e < w * len; e += PANEL_THREADS) {
    int c = e / len, i = e % len;
    P[e] = X[(long long)(j0 + c) * rows + j0 + i];
  }
  // R entries above the panel rows are final already
  for (int e = tid; e < w * j0; e += PANEL_THREADS) {
    int c = e / j0, i = e % j0;
    Rm[(long long)i * cols + j0 + c] = X[(long long)(j0 + c) * rows + i];
  }
  // zeros below the diagonal of R in these columns
  for (int e = tid; e < w * cols; e += PANEL_THREADS) {
    int c = e / cols, i = e % cols;
    if (i > j0 + c) Rm[(long long)i * cols + j0 + c] = make_double2(0.0, 0.0);
  }
  __syncthreads();

  for (int jj = 0; jj < w; jj++) {
    c128 *x = P + (long long)jj * len;
    // ---- reflector for x[jj..len) ----
    double s = 0.0;
    for (int i = jj + 1 + tid; i < len; i += PANEL_THREADS) { c128 v = x[i]; s += v.x * v.x + v.y * v.y; }
    s = warp_sum_d(s);
    if (lane == 0) red[warp] = s;
    __syncthreads();
    if (tid == 0) {
      double xn2 = 0.0;
      for (int i = 0; i < NW; i++) xn2 += red[i];
      c128 alpha = x[jj];
      c128 tau, scal;
      double beta;
      if ((xn2 == 0.0 && alpha.y == 0.0) || alpha.x * alpha.x + alpha.y * alpha.y + xn2 < TINY_NORM2) {
        tau = make_double2(0.0, 0.0); scal = make_double2(0.0, 0.0); beta = alpha.x;
      } else {
        double nrm = sqrt(alpha.x * alpha.x + alpha.y * alpha.y + xn2);
        beta = alpha.x >= 0.0 ? -nrm : nrm;
        tau = make_double2((beta - alpha.x) / beta, -alpha.y / beta);
        // scal = 1 / (alpha - beta)
        double dr = alpha.x - beta, di = alpha.y, dn = dr * dr + di * di;
        scal = make_double2(dr / dn, -di / dn);
      }
      tau_s[jj] = tau; scal_s = scal; beta_s = beta;
    }
    __syncthreads();
    {
      const c128 scal = scal_s;
      for (int i = jj + 1 + tid; i < len; i += PANEL_THREADS) x[i] = cmul(x[i], scal);
      if (tid == 0) {
        Rm[(long long)(j0 + jj) * cols + j0 + jj] = make_double2(beta_s, 0.0);
        x[jj] = make_double2(1.0, 0.0);
      }
      for (int i = tid; i < jj; i += PANEL_THREADS) {       // entries above the diagonal -> R, then 0
        Rm[(long long)(j0 + i) * cols + j0 + jj] = x[i];
        x[i] = make_double2(0.0, 0.0);
      }
    }
    __syncthreads();
    // ---- apply H^H = I - conj(tau) v v^H to the remaining panel columns ----
    const int nrem = w - jj - 1;
    if (nrem > 0) {
      // each remaining column gets NW / nrem warps (at least one)
      const int wpc = NW / nrem > 0 ? NW / nrem : 1;
      const int cc = warp / wpc, part = warp % wpc;
      if (warp < wpc * nrem) {
        const c128 *y = P + (long long)(jj + 1 + cc) * len;
        double sx = 0.0, sy = 0.0;
        for (int i = jj + part * 32 + lane; i < len; i += wpc * 32) {
          c128 v = x[i], u = y[i];
          sx += v.x * u.x + v.y * u.y;
          sy += v.x * u.y - v.y * u.x;
        }
        sx = warp_sum_d(sx); sy = warp_sum_d(sy);
        if (lane == 0) { red[warp] = sx; }
        // second array for imaginary parts: reuse gram storage rows as scratch
        if (lane == 0) reinterpret_cast<double *>(&gram[0][0])[warp] = sy;
      }
      __syncthreads();
      if (tid < nrem) {
        double sx = 0.0, sy = 0.0;
        for (int pz = 0; pz < wpc; pz++) {
          sx += red[tid * wpc + pz];
          sy += reinterpret_cast<double *>(&gram[0][0])[tid * wpc + pz];
        }
        // coefficient conj(tau) * (v^H y)
        c128 ct = cconj(tau_s[jj]);
        wdot[tid] = cmul(ct, make_double2(sx, sy));
      }
      __syncthreads();
      for (int e = tid; e < nrem * (len - jj); e += PANEL_THREADS) {
        int c2 = e / (len - jj), i = jj + e % (len - jj);
        c128 *y = P + (long long)(jj + 1 + c2) * len;
        c128 t = cmul(wdot[c2], x[i]);
        y[i].x -= t.x; y[i].y -= t.y;
      }
      __syncthreads();
    }
  }
  // ---- compact WY factor: T upper triangular with H_1...H_w = I - V T V^H ----
  for (int pr = warp; pr < w * w; pr += NW) {
    int a = pr / w, bq = pr % w;
    double sx = 0.0, sy = 0.0;
    if (a < bq) {
      const c128 *va = P + (long long)a * len, *vb = P + (long long)bq * len;
      for (int i = lane; i < len; i += 32) {
        c128 v = va[i], u = vb[i];
        sx += v.x * u.x + v.y * u.y;
        sy += v.x * u.y - v.y * u.x;
      }
      sx = warp_sum_d(sx); sy = warp_sum_d(sy);
    }
    if (lane == 0) gram[a][bq] = make_double2(sx, sy);      // v_a^H v_b
  }
  __syncthreads();
  if (tid == 0) {
    c128 T[NB_MAX][NB_MAX];
    for (int a = 0; a < NB_MAX; a++) for (int c = 0; c < NB_MAX; c++) T[a][c] = make_double2(0.0, 0.0);
    for (int c = 0; c < w; c++) {
      T[c][c] = tau_s[c];
      // T[0:c, c] = -tau_c * T[0:c, 0:c] * (V[:, 0:c]^H v_c)
      for (int a = 0; a < c; a++) {
        c128 acc = make_double2(0.0, 0.0);
        for (int q = a; q < c; q++) { c128 t = cmul(T[a][q], gram[q][c]); acc.x += t.x; acc.y += t.y; }
        c128 t = cmul(tau_s[c], acc);
        T[a][c] = make_double2(-t.x, -t.y);
      }
    }
    for (int a = 0; a < NB_MAX; a++) for (int c = 0; c < NB_MAX; c++) Tm[a * NB_MAX + c] = T[a][c];
  }
  for (int e = tid; e < w * len; e += PANEL_THREADS) {
    int c = e / len, i = e % len;
    X[(long long)(j0 + c) * rows + j0 + i] = P[e];
  }
}

// For columns c in [c_begin, c_end): Y[c][j0:rows) <- (I - V Top V^H) Y[c][j0:rows) with
// Top = T (adjoint = 0) or T^H (adjoint = 1); V = X[j0 .. j0+w)[j0:rows).
__global__ void __launch_bounds__(TRAIL_THREADS) qr_apply_kernel(const c128 *X, c128 *Y, int rows, int j0, int w,
                                                                  const c128 *Tm, int adjoint, int c_begin, int c_end) {
  const int len = rows - j0;
  const int c0 = c_begin + blockIdx.x * CB;
  const int nc = (c_end - c0) < CB ? (c_end - c0) : CB;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  constexpr int NW = TRAIL_THREADS / 32;
  __shared__ c128 part[NW][CB][NB_MAX];
  __shared__ c128 Wc[CB][NB_MAX];
  c128 acc[CB][NB_MAX];
#pragma unroll
  for (int c = 0; c < CB; c++)
#pragma unroll
    for (int q = 0; q < NB_MAX; q++) acc[c][q] = make_double2(0.0, 0.0);
  for (int i = tid; i < len; i += TRAIL_THREADS) {
    c128 yv[CB];
#pragma unroll
    for (int c = 0; c < CB; c++) yv[c] = c < nc ? Y[(long long)(c0 + c) * rows + j0 + i] : make_double2(0.0, 0.0);
#pragma unroll
    for (int q = 0; q < NB_MAX; q++) {
      if (q < w) {
        c128 v = X[(long long)(j0 + q) * rows + j0 + i];
#pragma unroll
        for (int c = 0; c < CB; c++) {
          acc[c][q].x += v.x * yv[c].x + v.y * yv[c].y;
          acc[c][q].y += v.x * yv[c].y - v.y * yv[c].x;
        }
      }
    }
  }
#pragma unroll
  for (int c = 0; c < CB; c++)
#pragma unroll
    for (int q = 0; q < NB_MAX; q++) {
      double sx = warp_sum_d(acc[c][q].x), sy = warp_sum_d(acc[c][q].y);
      if (lane == 0) part[warp][c][q] = make_double2(sx, sy);
    }
  __syncthreads();
  if (tid < CB * NB_MAX) {
    int c = tid / NB_MAX, q = tid % NB_MAX;
    double sx = 0.0, sy = 0.0;
    for (int ww = 0; ww < NW; ww++) { sx += part[ww][c][q].x; sy += part[ww][c][q].y; }
    part[0][c][q] = make_double2(sx, sy);               // V^H y
  }
  __syncthreads();
  if (tid < CB * NB_MAX) {
    int c = tid / NB_MAX, q = tid % NB_MAX;
    c128 s = make_double2(0.0, 0.0);
    if (q < w) {
      for (int r = 0; r < w; r++) {
        c128 t = adjoint ? cconj(Tm[r * NB_MAX + q]) : Tm[q * NB_MAX + r];
        c128 pr = cmul(t, part[0][c][r]);
        s.x += pr.x; s.y += pr.y;
      }
    }
    Wc[c][q] = s;
  }
  __syncthreads();
  for (int i = tid; i < len; i += TRAIL_THREADS) {
    c128 d[CB];
#pragma unroll
    for (int c = 0; c < CB; c++) d[c] = make_double2(0.0, 0.0);
#pragma unroll
    for (int q = 0; q < NB_MAX; q++) {
      if (q < w) {
        c128 v = X[(long long)(j0 + q) * rows + j0 + i];
#pragma unroll
        for (int c = 0; c < CB; c++) { c128 t = cmul(v, Wc[c][q]); d[c].x += t.x; d[c].y += t.y; }
      }
    }
#pragma unroll
    for (int c = 0; c < CB; c++)
      if (c < nc) {
        c128 *dst = Y + (long long)(c0 + c) * rows + j0 + i;
        c128 o = *dst;
        *dst = make_double2(o.x - d[c].x, o.y - d[c].y);
      }
  }
}

// One column per CTA, rows distributed over the threads, the reflector block V and the column kept
// in registers between the product V^H y and the update y -= V (Top V^H y): V is read once.
// NBW = widest panel of this mode (RA * NBW <= 40 keeps V in registers without spills).
//   FORMQ = false: trailing update of column c_begin + blockIdx.x by panel (j0, w), Top = T^H.
//   FORMQ = true : column c = blockIdx.x of Q = H_1 ... H_n [I; 0]: starts from e_c and applies the
//                  panels p = c / nb .. 0 with Top = T (panels above leave e_c untouched), ONE launch
//                  for the whole Q instead of one per panel.
template <int AT, int RA, int NBW, bool FORMQ>
__global__ void __launch_bounds__(AT) qr_apply1_kernel(const c128 *__restrict__ X, c128 *Y, int rows, int j0_in, int w_in,
                                                        const c128 *__restrict__ Tm, int nb, int cols, int c_begin,
                                                        const int *gate = nullptr /*DEVICE, nullable: run only if non-zero*/) {
  if (gate && __ldcg(gate) == 0) return;
  __shared__ double sm[(AT / 32 + 1) * 2 * NBW];
  __shared__ c128 Tsm[NB_MAX * NB_MAX];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int c = c_begin + blockIdx.x;
  c128 y[RA];
  int p_hi = 0, p_lo = 0;
  if (FORMQ) {
    p_hi = c / nb;
#pragma unroll
    for (int r = 0; r < RA; r++) y[r] = make_double2((tid + r * AT) == c ? 1.0 : 0.0, 0.0);
  } else {
#pragma unroll
    for (int r = 0; r < RA; r++) {
      const int i = j0_in + tid + r * AT;
      y[r] = i < rows ? Y[(long long)c * rows + i] : make_double2(0.0, 0.0);
    }
  }
  for (int pz = p_hi; pz >= p_lo; pz--) {
    const int j0 = FORMQ ? pz * nb : j0_in;
    const int w = FORMQ ? (cols - j0 < nb ? cols - j0 : nb) : w_in;
    const c128 *Tp = FORMQ ? Tm + (size_t)pz * NB_MAX * NB_MAX : Tm;
    // rows of this thread: FORMQ indexes rows from 0 (i >= j0 take part), else from j0
    c128 v[RA][NBW];
#pragma unroll
    for (int r = 0; r < RA; r++) {
      const int i = FORMQ ? tid + r * AT : j0 + tid + r * AT;
      const bool in = i < rows && i >= j0;
#pragma unroll
      for (int q = 0; q < NBW; q++)
        v[r][q] = (in && q < w) ? X[(long long)(j0 + q) * rows + i] : make_double2(0.0, 0.0);
    }
    if (tid < NB_MAX * NB_MAX) Tsm[tid] = Tp[tid];
    double acc[2 * NBW];
#pragma unroll
    for (int q = 0; q < 2 * NBW; q++) acc[q] = 0.0;
#pragma unroll
    for (int r = 0; r < RA; r++)
#pragma unroll
      for (int q = 0; q < NBW; q++) {
        acc[2 * q] = fma(v[r][q].x, y[r].x, fma(v[r][q].y, y[r].y, acc[2 * q]));
        acc[2 * q + 1] = fma(v[r][q].x, y[r].y, fma(-v[r][q].y, y[r].x, acc[2 * q + 1]));
      }
#pragma unroll
    for (int q = 0; q < 2 * NBW; q++) {
      const double t = warp_sum_d(acc[q]);
      if (lane == 0) sm[warp * 2 * NBW + q] = t;
    }
    __syncthreads();
    if (tid < 2 * NBW) {
      double t = 0.0;
#pragma unroll
      for (int k = 0; k < AT / 32; k++) t += sm[k * 2 * NBW + tid];   // fixed order: deterministic
      sm[(AT / 32) * 2 * NBW + tid] = t;
    }
    __syncthreads();
    c128 sv[NBW];
#pragma unroll
    for (int q = 0; q < NBW; q++) {
      c128 a = make_double2(0.0, 0.0);
#pragma unroll
      for (int r = 0; r < NBW; r++) {
        const c128 dv = make_double2(sm[(AT / 32) * 2 * NBW + 2 * r], sm[(AT / 32) * 2 * NBW + 2 * r + 1]);
        const c128 t = FORMQ ? Tsm[q * NB_MAX + r] : cconj(Tsm[r * NB_MAX + q]);
        const c128 pr = cmul(t, dv);
        a.x += pr.x; a.y += pr.y;
      }
      sv[q] = a;
    }
#pragma unroll
    for (int r = 0; r < RA; r++)
#pragma unroll
      for (int q = 0; q < NBW; q++) {
        y[r].x = fma(v[r][q].y, sv[q].y, fma(-v[r][q].x, sv[q].x, y[r].x));
        y[r].y = fma(-v[r][q].y, sv[q].x, fma(-v[r][q].x, sv[q].y, y[r].y));
      }
    __syncthreads();                                     // sm / Tsm are reused by the next panel
  }
#pragma unroll
  for (int r = 0; r < RA; r++) {
    const int i = FORMQ ? tid + r * AT : j0_in + tid + r * AT;
    if (i < rows) Y[(long long)c * rows + i] = y[r];
  }
}

void launch_apply(cudaStream_t st, int mode, const c128 *X, c128 *Y, int rows, int j0, int w, const c128 *Tp, int adjoint,
                  int c_begin, int c_end) {
  if (c_begin >= c_end) return;
  const int n = c_end - c_begin;
  if (mode == 1 && adjoint) TDVP_LAUNCH((qr_apply1_kernel<256, 5, 8, false>), n, 256, 0, st, X, Y, rows, j0, w, Tp, 0, 0, c_begin);
  else if (mode == 2 && adjoint) TDVP_LAUNCH((qr_apply1_kernel<256, 10, 4, false>), n, 256, 0, st, X, Y, rows, j0, w, Tp, 0, 0, c_begin);
  else if (mode == 3 && adjoint) TDVP_LAUNCH((qr_apply1_kernel<256, 20, 2, false>), n, 256, 0, st, X, Y, rows, j0, w, Tp, 0, 0, c_begin);
  else TDVP_LAUNCH(qr_apply_kernel, (n + CB - 1) / CB, TRAIL_THREADS, 0, st, X, Y, rows, j0, w, Tp, adjoint, c_begin, c_end);
}

int panel_width(int rows) {
  long long budget = 200 * 1024;
  int nb = (int)(budget / ((long long)rows * 16));
  if (nb > NB_MAX) nb = NB_MAX;
  if (nb < 1) nb = 1;                                     // rows > QR_MAX_TALL are rejected by the API layer
  return nb;
}

}  // namespace

constexpr int QF_SMEM = 40 * QT * 16;   // RA * NB = 40 reflector entries per thread in every mode
int g_qr_cluster = 1;            // TDVP_QR_CLUSTER=0: one launch per panel and per trailing update (diagnostic switch)
int g_qr_cluster_min = 0;        // matrices with more rows than this use the cluster kernel (TDVP_QR_CLUSTER_MIN)
int g_qr_fast = 1;               // TDVP_QR_FAST=0: every panel column by column with one cluster reduction per column (diagnostic switch)

void qr_configure() {
  cudaFuncSetAttribute(qr_factor_cluster_kernel<5, 8>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
  cudaFuncSetAttribute(qr_factor_cluster_kernel<5, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, QF_SMEM);
  {                                                       // can a 16-CTA cluster of this kernel be resident at all?
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(QC); cfg.blockDim = dim3(QT); cfg.dynamicSmemBytes = QF_SMEM;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = QC; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    int nclusters = 0;
    if (cudaOccupancyMaxActiveClusters(&nclusters, qr_factor_cluster_kernel<5, 8>, &cfg) != cudaSuccess || nclusters < 1) {
      cudaGetLastError();
      g_qr_cluster = 0;
    }
  }
  if (const char *e = getenv("TDVP_QR_CLUSTER")) g_qr_cluster = g_qr_cluster && e[0] != '0';
  if (const char *e = getenv("TDVP_QR_CLUSTER_MIN")) g_qr_cluster_min = atoi(e);
  if (const char *e = getenv("TDVP_QR_FAST")) g_qr_fast = e[0] != '0';
  cudaFuncSetAttribute(qr_panel_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024 + 1024);
}

// Panel variant by height: register-resident panels up to 5120 rows (512 threads, 3/5/10 rows per
// thread, 8/4/2 columns per panel: at most 48 doubles of panel per thread), the shared-memory panel beyond.
int panel_mode(int rows, int *nb) {
  if (rows <= 5 * 256) { *nb = 8; return 1; }
  if (rows <= 10 * 256) { *nb = 4; return 2; }
  if (rows <= 20 * 256) { *nb = 2; return 3; }
  *nb = panel_width(rows);
  return 0;
}

size_t qr_ws_bytes(int rows, int cols) {
  size_t mat = up256((size_t)rows * cols * 16);
  int nb = 1;
  panel_mode(rows, &nb);
  if (nb < 1) nb = 1;
  size_t npanels = (cols + nb - 1) / nb;
  return 2 * mat + up256((size_t)cols * cols * 16) + up256(npanels * NB_MAX * NB_MAX * 16) + 512;
}

// The two halves of a gauge move on one workspace: qr_factor leaves the reflectors (X), their T factors and R in `ws`
// and writes D; qr_form_q forms Q from them.  A caller that needs D first (the chain of bond unfoldings: svd.cu) can
// run the second half later, on another queue, as long as nothing else uses `ws` in between.
void qr_factor(cudaStream_t st, int side, int Ml, int d, int Mr, const c128 *C, c128 *D, void *ws, const int *gate) {
  const int rows = side == 0 ? Ml * d : d * Mr;
  const int cols = side == 0 ? Mr : Ml;
  int nb = 1;
  const int mode = panel_mode(rows, &nb);
  ProfScope ps(st, PH_QR);
  char *p = reinterpret_cast<char *>(up256(reinterpret_cast<size_t>(ws)));
  size_t mat = up256((size_t)rows * cols * 16);
  c128 *X = reinterpret_cast<c128 *>(p); p += mat;
  c128 *Y = reinterpret_cast<c128 *>(p); p += mat;
  c128 *Rm = reinterpret_cast<c128 *>(p); p += up256((size_t)cols * cols * 16);
  c128 *Tm = reinterpret_cast<c128 *>(p);
  const long long n = (long long)rows * cols;
  const int gcopy = (int)((n + 255) / 256 > 592 ? 592 : (n + 255) / 256);
  dim3 tb(32, 8), tg((cols + 31) / 32, (rows + 31) / 32);
  (void)Y;
  if (side == 0) TDVP_LAUNCH(transpose_in_kernel, tg, tb, 0, st, C, X, rows, cols);
  else TDVP_LAUNCH(copy_kernel, gcopy, 256, 0, st, X, C, n);
  const int npanels = (cols + nb - 1) / nb;
  if (g_qr_cluster && mode == 1 && rows > g_qr_cluster_min) {
    // up to 1280 rows: the whole factorisation (panels + trailing updates) in ONE cluster kernel.  Measured
    // (B200, 1280 x 128): 580 us against 698 us with one launch per panel and per update; at 2560 x 256 the
    // 16 SMs of the cluster are too few for the trailing updates (2170 against 1924 us), so taller matrices
    // keep the launch-per-panel path below.
    TDVP_LAUNCH((qr_factor_cluster_kernel<5, 8>), QC, QT, QF_SMEM, st, X, rows, cols, Rm, Tm, gate, g_qr_fast);
  } else
  for (int pz = 0; pz < npanels; pz++) {
    int j0 = pz * nb, w = cols - j0 < nb ? cols - j0 : nb;
    size_t smem = (size_t)w * (rows - j0) * 16;
    c128 *Tp = Tm + (size_t)pz * NB_MAX * NB_MAX;
    const int plen = rows - j0;                            // the panel only lives on rows >= j0
    if (mode == 1 && plen <= 128) TDVP_LAUNCH((qr_panel_reg_kernel<128, 1, 8>), 1, 128, 0, st, X, rows, cols, j0, w, Rm, Tp);
    else if (mode == 1 && plen <= 256) TDVP_LAUNCH((qr_panel_reg_kernel<256, 1, 8>), 1, 256, 0, st, X, rows, cols, j0, w, Rm, Tp);
    else if (mode == 1 && plen <= 512) TDVP_LAUNCH((qr_panel_reg_kernel<256, 2, 8>), 1, 256, 0, st, X, rows, cols, j0, w, Rm, Tp);
    else if (mode == 1) TDVP_LAUNCH((qr_panel_reg_kernel<256, 5, 8>), 1, 256, 0, st, X, rows, cols, j0, w, Rm, Tp);
    else if (mode == 2) TDVP_LAUNCH((qr_panel_reg_kernel<512, 5, 4>), 1, 512, 0, st, X, rows, cols, j0, w, Rm, Tp);
    else if (mode == 3) TDVP_LAUNCH((qr_panel_reg_kernel<512, 10, 2>), 1, 512, 0, st, X, rows, cols, j0, w, Rm, Tp);
    else TDVP_LAUNCH(qr_panel_kernel, 1, PANEL_THREADS, smem, st, X, rows, cols, j0, w, Rm, Tp);
    int c_begin = j0 + w;
    launch_apply(st, mode, X, X, rows, j0, w, Tp, 1, c_begin, cols);
  }
  TDVP_LAUNCH(store_d_kernel, (cols * cols + 255) / 256 > 296 ? 296 : (cols * cols + 255) / 256, 256, 0, st, Rm, D, cols, side);
}

void qr_form_q(cudaStream_t st, int side, int Ml, int d, int Mr, c128 *Q, void *ws, const int *gate) {
  const int rows = side == 0 ? Ml * d : d * Mr;
  const int cols = side == 0 ? Mr : Ml;
  int nb = 1;
  const int mode = panel_mode(rows, &nb);
  ProfScope ps(st, PH_QR);
  char *p = reinterpret_cast<char *>(up256(reinterpret_cast<size_t>(ws)));
  size_t mat = up256((size_t)rows * cols * 16);
  c128 *X = reinterpret_cast<c128 *>(p); p += mat;
  c128 *Y = reinterpret_cast<c128 *>(p); p += mat;
  c128 *Rm = reinterpret_cast<c128 *>(p); p += up256((size_t)cols * cols * 16);
  c128 *Tm = reinterpret_cast<c128 *>(p);
  const long long n = (long long)rows * cols;
  const int gcopy = (int)((n + 255) / 256 > 592 ? 592 : (n + 255) / 256);
  dim3 tb(32, 8), tg((cols + 31) / 32, (rows + 31) / 32);
  (void)Rm;
  const int npanels = (cols + nb - 1) / nb;
  if (mode == 1) TDVP_LAUNCH((qr_apply1_kernel<256, 5, 8, true>), cols, 256, 0, st, X, Y, rows, 0, 0, Tm, nb, cols, 0, gate);
  else if (mode == 2) TDVP_LAUNCH((qr_apply1_kernel<256, 10, 4, true>), cols, 256, 0, st, X, Y, rows, 0, 0, Tm, nb, cols, 0);
  else if (mode == 3) TDVP_LAUNCH((qr_apply1_kernel<256, 20, 2, true>), cols, 256, 0, st, X, Y, rows, 0, 0, Tm, nb, cols, 0);
  else {
    TDVP_LAUNCH(identity_kernel, gcopy, 256, 0, st, Y, rows, cols);
    for (int pz = npanels - 1; pz >= 0; pz--) {
      int j0 = pz * nb, w = cols - j0 < nb ? cols - j0 : nb;
      launch_apply(st, mode, X, Y, rows, j0, w, Tm + (size_t)pz * NB_MAX * NB_MAX, 0, j0, cols);
    }
  }
  if (side == 0) TDVP_LAUNCH(transpose_out_kernel, tg, tb, 0, st, Y, Q, rows, cols);
  else TDVP_LAUNCH(copy_kernel, gcopy, 256, 0, st, Q, Y, n);
}

void qr_gauge(cudaStream_t st, int side, int Ml, int d, int Mr, const c128 *C, c128 *Q, c128 *D, void *ws, const int *gate) {
  qr_factor(st, side, Ml, d, Mr, C, D, ws, gate);
  qr_form_q(st, side, Ml, d, Mr, Q, ws, gate);
}

// ---------------------------------------------------------------------------------------------
// tdvp_qr_gauge_noalloc: the QR gauge move (Eq. 9) for callers that cannot allocate --
// code under CUDA-graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The same kernels
// and the same host driver (qr_gauge above) as tdvp_qr_gauge; only the scratch block (column-major copy X,
// the Q workspace Y, R, the compact-WY factors T) differs: instead of the handle's growable arena it is the
// file-scope device array below, which every GPU that loads libtdvp.so holds until the process exits.
//
// In host code `g_qr_static_scratch` is a host-side stand-in for the symbol, NOT a device address: its
// device address is taken once per device, with that device current, by cudaGetSymbolAddress, and only that
// pointer is handed to the kernels.
//
// Nothing in the block has to start at zero: every kernel of the move writes each scratch element before
// any kernel reads it (X by the transpose / copy, R and T by the panel phase, Y by the Q formation), which is
// also why the arena path may reuse its memory from call to call; the block keeps the previous call's
// contents and the test calls twice in a row with different shapes to show that stale contents are harmless.
// All calls share the one block: calls that overlap on the GPU (two streams, or two host threads) RACE --
// serialise them on one stream.
#include <mutex>

#include "handle.cuh"

constexpr size_t QR_STATIC_SCRATCH_BYTES = 6u << 20;     // 6 MiB: up to the 1280 x 128 move of configs[3] (5.3 MiB)
static __device__ __align__(256) unsigned char g_qr_static_scratch[QR_STATIC_SCRATCH_BYTES];

namespace {
constexpr int QR_STATIC_MAX_DEVICES = 64;
std::mutex g_qr_static_mu;
void *g_qr_static_ptr[QR_STATIC_MAX_DEVICES] = {nullptr};
}  // namespace

extern "C" int tdvp_qr_gauge_noalloc(void *cuda_stream, int side, int Ml, int d, int Mr, const tdvp_c128 *C,
                                     tdvp_c128 *Q, tdvp_c128 *D) {
  if (!C || !Q || !D) return set_err(nullptr, TDVP_EINVAL, "tdvp_qr_gauge_noalloc: null pointer");
  if (side != 0 && side != 1) return set_err(nullptr, TDVP_EINVAL, "tdvp_qr_gauge_noalloc: side must be 0 or 1");
  if (Ml < 1 || d < 1 || Mr < 1) return set_err(nullptr, TDVP_EINVAL, "tdvp_qr_gauge_noalloc: dimensions must be >= 1");
  const long long tall = side == 0 ? (long long)Ml * d : (long long)d * Mr;
  const int thin = side == 0 ? Mr : Ml;
  if (tall < thin) return set_err(nullptr, TDVP_EINVAL, "tdvp_qr_gauge_noalloc: gauge move needs a tall or square matrix");
  if (tall > QR_MAX_TALL) return set_err(nullptr, TDVP_EINVAL, "tdvp_qr_gauge_noalloc: tall side above 12800 rows is not supported");
  const size_t need = qr_ws_bytes((int)tall, thin) + 256;
  if (need > QR_STATIC_SCRATCH_BYTES)
    return set_err(nullptr, TDVP_EINVAL, "tdvp_qr_gauge_noalloc: needs " + std::to_string(need) + " bytes of scratch, the static block holds " +
                                             std::to_string(QR_STATIC_SCRATCH_BYTES) + " (6 MiB: e.g. up to 1280 x 128); use tdvp_qr_gauge");
  configure_kernels_once();                              // kernel attributes only: no allocation
  int dev = 0;
  if (int rc = check_cuda(nullptr, cudaGetDevice(&dev), "tdvp_qr_gauge_noalloc")) return rc;
  if (dev < 0 || dev >= QR_STATIC_MAX_DEVICES) return set_err(nullptr, TDVP_EINVAL, "tdvp_qr_gauge_noalloc: device ordinal above 63");
  void *scratch = nullptr;
  {
    std::lock_guard<std::mutex> lk(g_qr_static_mu);
    if (!g_qr_static_ptr[dev]) {                         // once per device, with that device current
      void *p = nullptr;
      if (int rc = check_cuda(nullptr, cudaGetSymbolAddress(&p, g_qr_static_scratch), "tdvp_qr_gauge_noalloc: cudaGetSymbolAddress")) return rc;
      g_qr_static_ptr[dev] = p;
    }
    scratch = g_qr_static_ptr[dev];
  }
  qr_gauge(reinterpret_cast<cudaStream_t>(cuda_stream), side, Ml, d, Mr, reinterpret_cast<const c128 *>(C), reinterpret_cast<c128 *>(Q),
           reinterpret_cast<c128 *>(D), scratch);
  return check_cuda(nullptr, cudaGetLastError(), "tdvp_qr_gauge_noalloc");
}
