// wstage.cu -- the MPO ("W") stage of H_eff / environment updates as a sparse-aware contraction
// (the M_S^2 M_O^2 d^2 term of Table I, with the zeros of W
// skipped: vibronic MPO tensors are ~3 % dense, Eq. 45 / SURVEY.md 8(c) c3).
//
// For every bond-index pair the stage is a sparse (rows x cols) matrix applied to a dense
// cols x Mr panel whose rows are contiguous in y.  HBM/L2 traffic is exactly one read of T1 and one
// write of T2; see wstage_persistent_kernel for the work split and what bounds it.
#include <vector>

#include "common.cuh"

namespace {

constexpr int YT = 64;          // y per work item: lane l owns y0 + l and y0 + 32 + l
constexpr int CSR_WARPS = 8;

// Sparse form of the (nrows x ncols) matrix view of W, built in ONE pass by one warp per row:
// row r keeps its non-zeros, sorted by column, at [r * ncols, r * ncols + cnt[r]) of col[] / val[]
// (row-padded: no prefix sum over rows is needed, so there is no second kernel and no atomics).
// which = 0: rows (s,v), cols (w,t) ["left"]; which = 1: rows (w,s), cols (t,v) ["right"].
__device__ __forceinline__ long long csr_widx(int which, int r, int c, int Dl, int d, int Dr, int ncols) {
  if (which == 0) { int s = r / Dr, v = r % Dr, w = c / d, t = c % d;
                    return (((long long)w * d + s) * d + t) * Dr + v; }
  return (long long)r * ncols + c;
}

__global__ void __launch_bounds__(CSR_WARPS * 32) csr_build_kernel(const c128 *__restrict__ W, int Dl, int d, int Dr, double tol,
                                                                    int *cnt0, int *col0, c128 *val0,
                                                                    int *cnt1, int *col1, c128 *val1) {
  const int which = blockIdx.y;
  const int nrows = which == 0 ? d * Dr : Dl * d, ncols = which == 0 ? Dl * d : d * Dr;
  int *cnt = which == 0 ? cnt0 : cnt1;
  int *col = which == 0 ? col0 : col1;
  c128 *val = which == 0 ? val0 : val1;
  const int lane = threadIdx.x & 31, r = blockIdx.x * CSR_WARPS + (threadIdx.x >> 5);
  if (r >= nrows) return;
  int o = r * ncols;
  for (int c0 = 0; c0 < ncols; c0 += 32) {
    const int c = c0 + lane;
    bool nz = false;
    c128 x = make_double2(0.0, 0.0);
    if (c < ncols) { x = __ldg(W + csr_widx(which, r, c, Dl, d, Dr, ncols)); nz = fabs(x.x) > tol || fabs(x.y) > tol; }
    const unsigned m = __ballot_sync(0xffffffffu, nz);
    if (nz) { const int q = o + __popc(m & ((1u << lane) - 1u)); col[q] = c; val[q] = x; }
    o += __popc(m);
  }
  if (lane == 0) cnt[r] = o - r * ncols;
}

struct WStageParams {
  const c128 *in; c128 *out;
  int nrows, ncols, Mr;
  long long in_bs;                 // input batch stride (per a); input row stride is Mr
  int rdiv; long long o_s1, o_s2;  // output offset of row r: (r / rdiv) * o_s1 + (r % rdiv) * o_s2
  long long o_bs;                  // output batch stride
  const int *cnt; const int *col; const c128 *val;   // row-padded sparse W (see csr_build_kernel)
  const int *order;                // rows by entry count, longest first
  int long_rows;                   // -1 unknown on the host, 0, 1
  const int *skip;                 // nullable: non-zero at kernel start = nothing to do (see ZGemm::skip)
};

__device__ __forceinline__ void cfma(double &sx, double &sy, c128 w, c128 t) {
  sx = fma(w.x, t.x, sx); sx = fma(-w.y, t.y, sx);
  sy = fma(w.x, t.y, sy); sy = fma(w.y, t.x, sy);
}

// Persistent kernel: one CTA of 32 warps per SM walks over its contiguous range of (panel, row) units.
// The panel T1[a, :, y0:y0+64] is staged in shared memory by 16 B cp.async copies; each warp then
// produces output rows, every lane owning TWO y (l and l + 32), so that the warp-uniform loads of an
// entry's value and column are amortised over two panel loads (the kernel is bound by shared-memory
// wavefronts, not by the FP64 pipe or HBM: 4 per LDS.128 of panel, 1 per broadcast).  The sparse W
// is compacted into shared memory when it fits beside the panel (every MPO of the paper's
// workloads); otherwise (configs[1]: 6000 entries + a 200 KB panel) its entries are read through
// L1/L2 with the next four prefetched into registers.  Entry batches are padded with zero weights,
// so the inner loop has no tail.
constexpr int WP_THREADS = 1024;
constexpr int WP_SMEM = 227 * 1024 - 64;   // dynamic part; the row counter is static

template <bool CSR_SMEM>
__device__ __forceinline__ void wp_rows(const WStageParams &p, const c128 *tile, const c128 *__restrict__ vals,
                                        const int *__restrict__ cols, const int *rbeg, const int *rend, c128 *out,
                                        int y0, int lane, int r0, int r1, int *next_row) {
  const c128 zero = make_double2(0.0, 0.0);
  int rs = r0 + (threadIdx.x >> 5) - WP_THREADS / 32;
  for (;;) {
    // long rows (they differ in length) are handed out one at a time, so that the warps of the CTA
    // stay busy until the segment is used up; short rows (real MPOs: ~2 entries) go round-robin
    int r = 0;
    if (next_row) {
      if (lane == 0) r = atomicAdd(next_row, 1);
      r = __shfl_sync(0xffffffffu, r, 0);
    } else {
      r = (rs += WP_THREADS / 32);
    }
    if (r >= r1) break;
    const int e0 = rbeg[r], e1 = rend[r];
    double ax = 0.0, ay = 0.0, bx = 0.0, by = 0.0;     // y0 + lane ; y0 + 32 + lane
    int c[4]; c128 w[4];
#pragma unroll
    for (int i = 0; i < 4; i++) {
      const bool ok = e0 + i < e1;
      c[i] = ok ? (CSR_SMEM ? cols[e0 + i] : __ldg(cols + e0 + i)) : 0;
      w[i] = ok ? (CSR_SMEM ? vals[e0 + i] : __ldg(vals + e0 + i)) : zero;
    }
    for (int e = e0; e < e1; e += 4) {
      int cn[4]; c128 wn[4];
#pragma unroll
      for (int i = 0; i < 4; i++) {
        const bool ok = e + 4 + i < e1;
        cn[i] = ok ? (CSR_SMEM ? cols[e + 4 + i] : __ldg(cols + e + 4 + i)) : 0;
        wn[i] = ok ? (CSR_SMEM ? vals[e + 4 + i] : __ldg(vals + e + 4 + i)) : zero;
      }
      c128 ta[4], tb[4];
#pragma unroll
      for (int i = 0; i < 4; i++) { ta[i] = tile[c[i] * YT + lane]; tb[i] = tile[c[i] * YT + 32 + lane]; }
#pragma unroll
      for (int i = 0; i < 4; i++) { cfma(ax, ay, w[i], ta[i]); cfma(bx, by, w[i], tb[i]); }
#pragma unroll
      for (int i = 0; i < 4; i++) { c[i] = cn[i]; w[i] = wn[i]; }
    }
    c128 *o = out + (r / p.rdiv) * p.o_s1 + (r % p.rdiv) * p.o_s2;
    if (y0 + lane < p.Mr) o[y0 + lane] = make_double2(ax, ay);
    if (y0 + 32 + lane < p.Mr) o[y0 + 32 + lane] = make_double2(bx, by);
  }
}

__global__ void __launch_bounds__(WP_THREADS, 1) wstage_persistent_kernel(WStageParams p, int ntile, int npanels, int quad_follows) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ int s_next_row;
  if (p.skip && *reinterpret_cast<const volatile int *>(p.skip)) return;
  c128 *tile = reinterpret_cast<c128 *>(smem_raw);                        // [ncols][YT]
  const int tile_elems = p.ncols * YT;
  int *rbeg = reinterpret_cast<int *>(smem_raw + (size_t)tile_elems * 16);   // [nrows]
  int *rend = rbeg + p.nrows;                                             // [nrows]
  const size_t csr_off = (((size_t)tile_elems * 16 + (size_t)p.nrows * 8) + 15) & ~size_t(15);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  c128 *sval = reinterpret_cast<c128 *>(smem_raw + csr_off);
  // exclusive prefix of the row counts (one warp); the sparse W is then compacted into shared memory
  // if its 20 B per entry fit beside the panel, else rows keep pointing into the padded global arrays
  if (warp == 0) {
    int run = 0;
    for (int r0 = 0; r0 < p.nrows; r0 += 32) {
      const int r = r0 + lane;
      const int n = r < p.nrows ? __ldg(p.cnt + r) : 0;
      int incl = n;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { int t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
      if (r < p.nrows) { rbeg[r] = run + incl - n; rend[r] = run + incl; }
      run += __shfl_sync(0xffffffffu, incl, 31);
    }
  }
  __syncthreads();
  const int nnz = rend[p.nrows - 1];
  const bool csr_smem = csr_off + (size_t)nnz * 20 + 16 <= (size_t)WP_SMEM;
  int *scol = reinterpret_cast<int *>(sval + nnz);
  const bool dyn = nnz >= 8 * p.nrows;
  if (dyn && quad_follows) return;                     // long rows: wstage_quad_kernel does the stage
  __syncthreads();
  if (csr_smem) {
    for (int r = warp; r < p.nrows; r += WP_THREADS / 32) {
      const int b = rbeg[r], n = rend[r] - b;
      for (int e = lane; e < n; e += 32) {
        sval[b + e] = __ldg(p.val + (size_t)r * p.ncols + e);
        scol[b + e] = __ldg(p.col + (size_t)r * p.ncols + e);
      }
    }
  } else {
    for (int r = threadIdx.x; r < p.nrows; r += WP_THREADS) {
      const int n = rend[r] - rbeg[r];
      rbeg[r] = r * p.ncols; rend[r] = r * p.ncols + n;
    }
  }
  // Work = (panel, row) units in panel-major order, cut into gridDim.x equal contiguous ranges: a CTA
  // stages at most (its share of panels + 2) panels, each once, whatever the row count.
  const long long units = (long long)npanels * p.nrows;
  long long u = units * blockIdx.x / gridDim.x;
  long long u_end = units * (blockIdx.x + 1) / gridDim.x;
  if (!dyn) {   // short rows: staging a panel costs as much as its rows, so ranges are whole panels
    u = ((long long)npanels * blockIdx.x / gridDim.x) * p.nrows;
    u_end = ((long long)npanels * (blockIdx.x + 1) / gridDim.x) * p.nrows;
  }
  while (u < u_end) {
    const int panel = (int)(u / p.nrows), r0 = (int)(u - (long long)panel * p.nrows);
    const int r1 = (u_end - u) < (long long)(p.nrows - r0) ? r0 + (int)(u_end - u) : p.nrows;
    u += r1 - r0;
    const int a = panel / ntile, y0 = (panel % ntile) * YT;
    const c128 *in = p.in + a * p.in_bs;
    __syncthreads();                                   // previous segment's readers are done with the panel
    if (threadIdx.x == 0) s_next_row = r0;
    for (int e = threadIdx.x; e < tile_elems; e += WP_THREADS) {
      const int c = e / YT, yy = e % YT;
      const bool ok = (y0 + yy) < p.Mr;
      const c128 *src = ok ? in + (long long)c * p.Mr + y0 + yy : in;
      unsigned sa = (unsigned)__cvta_generic_to_shared(tile + e);
      int sz = ok ? 16 : 0;
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(sa), "l"(src), "r"(sz));
    }
    asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;\n" ::);
    __syncthreads();
    c128 *out = p.out + a * p.o_bs;
    if (csr_smem) {
      wp_rows<true>(p, tile, sval, scol, rbeg, rend, out, y0, lane, r0, r1, dyn ? &s_next_row : nullptr);
    } else {
      wp_rows<false>(p, tile, p.val, p.col, rbeg, rend, out, y0, lane, r0, r1, dyn ? &s_next_row : nullptr);
    }
  }
}


// rank of every row by entry count (longest first, ties by row index): order[rank] = row
__global__ void row_order_kernel(const int *cnt0, int n0, int *ord0, const int *cnt1, int n1, int *ord1) {
  const int *cnt = blockIdx.x ? cnt1 : cnt0;
  const int n = blockIdx.x ? n1 : n0;
  int *ord = blockIdx.x ? ord1 : ord0;
  for (int r = threadIdx.x; r < n; r += blockDim.x) {
    const int c = cnt[r];
    int rank = 0;
    for (int q = 0; q < n; q++) { const int cq = cnt[q]; rank += (cq > c) || (cq == c && q < r); }
    ord[rank] = r;
  }
}

// ---- long rows (configs[1]: ~30 entries per row, the sparse W does not fit beside the panel) ----
// In the row-at-a-time kernel a warp-uniform load of an entry (value + column) costs the LSU pipe
// about 5.4 wavefronts, 40 % of the kernel's total, because it serves one row only.  Here a warp
// works on FOUR rows at once: lane = (row slot g = lane / 8, j = lane % 8) owns y = j + 8 m,
// m = 0..7, of its row, so one load instruction fetches the next entry of four rows, while the
// panel loads stay what they were (a quarter-warp reads 128 contiguous bytes of its row's column:
// 4 conflict-free wavefronts per LDS.128, 16 B per entry and y).  Rows are taken in groups of four
// from the order sorted by length, so the four rows of a group finish together.
constexpr int WQ_THREADS = 512;
constexpr int WQ_MIN_PANELS = W_QUAD_MIN_PANELS;       // below this the stage is launch-bound: one kernel, no row order
constexpr int WQ_SMEM = 227 * 1024 - 64;

__global__ void __launch_bounds__(WQ_THREADS, 1) wstage_quad_kernel(WStageParams p, int ntile, int npanels, int forced) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ int s_next, s_nnz;
  __shared__ __align__(8) unsigned long long s_bar;       // completion barrier of the bulk panel copies
  if (p.skip && *reinterpret_cast<const volatile int *>(p.skip)) return;
  c128 *tile = reinterpret_cast<c128 *>(smem_raw);                        // [ncols][YT]
  const int tile_elems = p.ncols * YT;
  int *scnt = reinterpret_cast<int *>(smem_raw + (size_t)tile_elems * 16);    // [nrows], in sorted order
  int *srow = scnt + p.nrows;                                              // [nrows] the row itself
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int g = lane >> 3, j = lane & 7;
  if (warp == 0) {
    int t = 0;
    for (int r = lane; r < p.nrows; r += 32) t += __ldg(p.cnt + r);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if (lane == 0) s_nnz = t;
  }
  for (int i = threadIdx.x; i < p.nrows; i += WQ_THREADS) { const int r = __ldg(p.order + i); srow[i] = r; scnt[i] = __ldg(p.cnt + r); }
  const unsigned bar_sa = (unsigned)__cvta_generic_to_shared(&s_bar);
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" ::"r"(bar_sa));
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  unsigned bar_phase = 0;
  __syncthreads();
  if (!forced && s_nnz < 8 * p.nrows) return;          // short rows: the row-at-a-time kernel does the stage
  const int ngroups = (p.nrows + 3) / 4;
  const long long units = (long long)npanels * ngroups;
  long long u = units * blockIdx.x / gridDim.x;
  const long long u_end = units * (blockIdx.x + 1) / gridDim.x;
  const c128 zero = make_double2(0.0, 0.0);
  while (u < u_end) {
    const int panel = (int)(u / ngroups), g0 = (int)(u - (long long)panel * ngroups);
    const int g1 = (u_end - u) < (long long)(ngroups - g0) ? g0 + (int)(u_end - u) : ngroups;
    u += g1 - g0;
    const int a = panel / ntile, y0 = (panel % ntile) * YT;
    const c128 *in = p.in + a * p.in_bs;
    __syncthreads();
    if (threadIdx.x == 0) s_next = g0;
    if (y0 + YT <= p.Mr) {
      // whole tile in range: one 1 KB bulk copy per panel row (TMA engine), completion on the mbarrier
      asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");   // earlier reads of the panel before async writes
      if (threadIdx.x == 0)
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar_sa), "r"((unsigned)(p.ncols * YT * 16)) : "memory");
      for (int c = threadIdx.x; c < p.ncols; c += WQ_THREADS) {
        const unsigned sa = (unsigned)__cvta_generic_to_shared(tile + (size_t)c * YT);
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
                     ::"r"(sa), "l"(in + (long long)c * p.Mr + y0), "r"((unsigned)(YT * 16)), "r"(bar_sa) : "memory");
      }
      unsigned ok;
      do {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}\n"
                     : "=r"(ok) : "r"(bar_sa), "r"(bar_phase) : "memory");
      } while (!ok);
      bar_phase ^= 1u;
    } else {
      for (int e = threadIdx.x; e < tile_elems; e += WQ_THREADS) {
        const int c = e / YT, yy = e % YT;
        const bool ok = (y0 + yy) < p.Mr;
        const c128 *src = ok ? in + (long long)c * p.Mr + y0 + yy : in;
        unsigned sa = (unsigned)__cvta_generic_to_shared(tile + e);
        int sz = ok ? 16 : 0;
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(sa), "l"(src), "r"(sz));
      }
      asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;\n" ::);
    }
    __syncthreads();
    c128 *out = p.out + a * p.o_bs;
    for (;;) {
      int grp = 0;
      if (lane == 0) grp = atomicAdd(&s_next, 1);
      grp = __shfl_sync(0xffffffffu, grp, 0);
      if (grp >= g1) break;
      const int slot = 4 * grp + g;
      const bool have = slot < p.nrows;
      const int r = have ? srow[slot] : 0;
      const int len = have ? scnt[slot] : 0;
      int steps = len;                                  // the longest of the four rows
      steps = max(steps, __shfl_xor_sync(0xffffffffu, steps, 8));
      steps = max(steps, __shfl_xor_sync(0xffffffffu, steps, 16));
      const c128 *__restrict__ vp = p.val + (size_t)r * p.ncols;
      const int *__restrict__ cp = p.col + (size_t)r * p.ncols;
      double ax[8], ay[8];
#pragma unroll
      for (int m = 0; m < 8; m++) ax[m] = ay[m] = 0.0;
      c128 w0 = 0 < len ? __ldg(vp) : zero, w1 = 1 < len ? __ldg(vp + 1) : zero;
      int c0 = 0 < len ? __ldg(cp) : 0, c1 = 1 < len ? __ldg(cp + 1) : 0;
      const c128 *tl = tile + j;
      for (int sI = 0; sI < steps; sI += 2) {
        const c128 wn0 = sI + 2 < len ? __ldg(vp + sI + 2) : zero, wn1 = sI + 3 < len ? __ldg(vp + sI + 3) : zero;
        const int cn0 = sI + 2 < len ? __ldg(cp + sI + 2) : 0, cn1 = sI + 3 < len ? __ldg(cp + sI + 3) : 0;
        {
          c128 t[8];
#pragma unroll
          for (int m = 0; m < 8; m++) t[m] = tl[c0 * YT + 8 * m];
#pragma unroll
          for (int m = 0; m < 8; m++) cfma(ax[m], ay[m], w0, t[m]);
        }
        {
          c128 t[8];
#pragma unroll
          for (int m = 0; m < 8; m++) t[m] = tl[c1 * YT + 8 * m];
#pragma unroll
          for (int m = 0; m < 8; m++) cfma(ax[m], ay[m], w1, t[m]);
        }
        w0 = wn0; w1 = wn1; c0 = cn0; c1 = cn1;
      }
      if (have) {
        c128 *o = out + (r / p.rdiv) * p.o_s1 + (r % p.rdiv) * p.o_s2 + y0 + j;
#pragma unroll
        for (int m = 0; m < 8; m++)
          if (y0 + j + 8 * m < p.Mr) o[8 * m] = make_double2(ax[m], ay[m]);
      }
    }
  }
}

// Fallback for panels that do not fit in shared memory (ncols * 1 KB > ~220 KB): one warp per
// (a, 32 y, row), panel and entries read through L1/L2.
__global__ void __launch_bounds__(256) wstage_direct_kernel(WStageParams p) {
  if (p.skip && *reinterpret_cast<const volatile int *>(p.skip)) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int a = blockIdx.y, y = blockIdx.x * 32 + lane;
  const bool yok = y < p.Mr;
  const c128 *__restrict__ in = p.in + a * p.in_bs + (yok ? y : 0);
  c128 *out = p.out + a * p.o_bs;
  for (int r = blockIdx.z * 8 + warp; r < p.nrows; r += gridDim.z * 8) {
    const int e0 = r * p.ncols, e1 = e0 + __ldg(p.cnt + r);
    double sx = 0.0, sy = 0.0;
    for (int e = e0; e < e1; e++) cfma(sx, sy, __ldg(p.val + e), __ldg(in + (long long)__ldg(p.col + e) * p.Mr));
    if (yok) out[(r / p.rdiv) * p.o_s1 + (r % p.rdiv) * p.o_s2 + y] = make_double2(sx, sy);
  }
}

int g_num_sms = 0;

void launch_wstage(cudaStream_t st, const WStageParams &p, int nbatch) {
  const int ntile = (p.Mr + YT - 1) / YT;
  const size_t panel = (size_t)p.ncols * YT * 16 + (size_t)p.nrows * 8 + 64;
  ProfScope ps(st, PH_WSTAGE);
  if (panel <= (size_t)WP_SMEM) {
    if (!g_num_sms) { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&g_num_sms, cudaDevAttrMultiProcessorCount, dev); }
    // one CTA per SM when there is enough work; never more CTAs than 32-row chunks or panels
    const long long npanels = (long long)nbatch * ntile, units = npanels * p.nrows;
    long long want = (units + 31) / 32;
    if (want < npanels) want = npanels;
    if (want > units) want = units;
    const int grid = want < g_num_sms ? (int)(want < 1 ? 1 : want) : g_num_sms;
    // long rows that do not fit beside the panel go to the four-rows-per-warp kernel.  Whether the rows
    // are long is known on the host for resident chains; for the stateless calls both kernels are
    // launched and the one whose turn it is not returns at once.
    const bool quad_fits = (size_t)p.ncols * YT * 16 + (size_t)p.nrows * 8 + 64 <= (size_t)WQ_SMEM &&
                           (long long)p.nrows * p.ncols >= 4096 && npanels >= WQ_MIN_PANELS;
    const int lr = quad_fits ? p.long_rows : 0;
    if (lr != 1) TDVP_LAUNCH(wstage_persistent_kernel, grid, WP_THREADS, WP_SMEM, st, p, ntile, (int)npanels, lr == -1 ? 1 : 0);
    if (lr != 0) {
      const long long qunits = npanels * ((p.nrows + 3) / 4);
      long long qw = (qunits + (WQ_THREADS / 32) - 1) / (WQ_THREADS / 32);
      if (qw < npanels) qw = npanels;
      if (qw > qunits) qw = qunits;
      const int qgrid = qw < g_num_sms ? (int)(qw < 1 ? 1 : qw) : g_num_sms;
      TDVP_LAUNCH(wstage_quad_kernel, qgrid, WQ_THREADS, WQ_SMEM, st, p, ntile, (int)npanels, lr == 1 ? 1 : 0);
    }
    return;
  }
  dim3 grid((p.Mr + 31) / 32, nbatch, (p.nrows + 7) / 8 < 8 ? (p.nrows + 7) / 8 : 8);
  TDVP_LAUNCH(wstage_direct_kernel, grid, 256, 0, st, p);
}

}  // namespace

void wstage_configure() {
  cudaFuncSetAttribute(wstage_persistent_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, WP_SMEM);
  cudaFuncSetAttribute(wstage_quad_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, WQ_SMEM);
}

size_t wsparse_bytes(int Dl, int d, int Dr) {
  size_t cap = (size_t)Dl * d * d * Dr;
  size_t rows0 = (size_t)d * Dr + 1, rows1 = (size_t)Dl * d + 1;
  auto up = [](size_t x) { return (x + 255) & ~size_t(255); };
  return 2 * up(rows0 * 4) + 2 * up(rows1 * 4) + 2 * up(cap * 4) + 2 * up(cap * 16) + 256;
}

void wsparse_build(cudaStream_t st, WSparse &ws, void *mem, int Dl, int d, int Dr, const c128 *W,
                   double zero_tol, bool want_order) {
  size_t cap = (size_t)Dl * d * d * Dr;
  auto up = [](size_t x) { return (x + 255) & ~size_t(255); };
  char *p = reinterpret_cast<char *>(mem);
  p = reinterpret_cast<char *>(up(reinterpret_cast<size_t>(p)));
  ws.Dl = Dl; ws.d = d; ws.Dr = Dr; ws.capacity = (int)cap;
  ws.val = reinterpret_cast<c128 *>(p); p += up(cap * 16);
  ws.val_r = reinterpret_cast<c128 *>(p); p += up(cap * 16);
  ws.col = reinterpret_cast<int *>(p); p += up(cap * 4);
  ws.col_r = reinterpret_cast<int *>(p); p += up(cap * 4);
  ws.cnt = reinterpret_cast<int *>(p); p += up(((size_t)d * Dr + 1) * 4);
  ws.cnt_r = reinterpret_cast<int *>(p); p += up(((size_t)Dl * d + 1) * 4);
  ws.order = reinterpret_cast<int *>(p); p += up(((size_t)d * Dr + 1) * 4);
  ws.order_r = reinterpret_cast<int *>(p);
  ws.long_rows = ws.long_rows_r = -1;
  int maxrows = (d * Dr > Dl * d ? d * Dr : Dl * d);
  dim3 grid((maxrows + CSR_WARPS - 1) / CSR_WARPS, 2);
  TDVP_LAUNCH(csr_build_kernel, grid, CSR_WARPS * 32, 0, st, W, Dl, d, Dr, zero_tol,
              ws.cnt, ws.col, ws.val, ws.cnt_r, ws.col_r, ws.val_r);
  // the sorted row order serves the long-row kernel only; callers that know it will not run (few
  // panels: the stage is launch-bound there) skip it and pin the choice
  if (want_order) TDVP_LAUNCH(row_order_kernel, 2, 256, 0, st, ws.cnt, d * Dr, ws.order, ws.cnt_r, Dl * d, ws.order_r);
  else ws.long_rows = ws.long_rows_r = 0;
}

void wsparse_classify(WSparse &ws, cudaStream_t st) {
  const int n0 = ws.d * ws.Dr, n1 = ws.Dl * ws.d;
  std::vector<int> c0(n0), c1(n1);
  cudaMemcpyAsync(c0.data(), ws.cnt, n0 * sizeof(int), cudaMemcpyDeviceToHost, st);
  cudaMemcpyAsync(c1.data(), ws.cnt_r, n1 * sizeof(int), cudaMemcpyDeviceToHost, st);
  if (cudaStreamSynchronize(st) != cudaSuccess) return;
  long long t0 = 0, t1 = 0;
  for (int x : c0) t0 += x;
  for (int x : c1) t1 += x;
  ws.long_rows = t0 >= 8LL * n0 ? 1 : 0;
  ws.long_rows_r = t1 >= 8LL * n1 ? 1 : 0;
}

void wstage_left(cudaStream_t st, const WSparse &ws, int Ml, int Mr, const c128 *T1, c128 *T2, const int *skip) {
  WStageParams p;
  p.in = T1; p.out = T2; p.skip = skip;
  p.nrows = ws.d * ws.Dr; p.ncols = ws.Dl * ws.d; p.Mr = Mr;
  p.in_bs = (long long)ws.Dl * ws.d * Mr;
  p.rdiv = p.nrows > 0 ? p.nrows : 1; p.o_s1 = 0; p.o_s2 = Mr;
  p.o_bs = (long long)ws.d * ws.Dr * Mr;
  p.cnt = ws.cnt; p.col = ws.col; p.val = ws.val; p.order = ws.order; p.long_rows = ws.long_rows;
  launch_wstage(st, p, Ml);
}

void wstage_right(cudaStream_t st, const WSparse &ws, int Ml, int Mr, const c128 *T1, c128 *T2, const int *skip) {
  WStageParams p;
  p.in = T1; p.out = T2; p.skip = skip;
  p.nrows = ws.Dl * ws.d; p.ncols = ws.d * ws.Dr; p.Mr = Mr;
  p.in_bs = (long long)ws.d * ws.Dr * Mr;
  p.rdiv = ws.d; p.o_s1 = (long long)Ml * ws.d * Mr; p.o_s2 = Mr;
  p.o_bs = (long long)ws.d * Mr;
  p.cnt = ws.cnt_r; p.col = ws.col_r; p.val = ws.val_r; p.order = ws.order_r; p.long_rows = ws.long_rows_r;
  launch_wstage(st, p, Ml);
}
