// wstage.cu -- the MPO ("W") stage of H_eff / environment updates as a sparse-aware contraction
// (the M_S^2 M_O^2 d^2 term of Table I, with the zeros of W
// skipped: vibronic MPO tensors are ~3 % dense, Eq. 45 / SURVEY.md 8(c) c3).
//
// For every bond-index pair the stage is a sparse (rows x cols) matrix applied to a dense
// cols x Mr panel whose rows are contiguous in y.  One CTA owns (batch index a, 32 consecutive y):
// it stages the panel T1[a, :, y0:y0+32] in shared memory with 16 B cp.async copies, then each
// warp produces output rows r = warp, warp + 16, ... with lane = y (coalesced 512 B row writes,
// conflict-free LDS.128), walking the row's CSR entries (warp-uniform loads).  HBM/L2 traffic is
// exactly one read of T1 and one write of T2.
#include "common.cuh"

namespace {

constexpr int YT = 32;          // y per CTA (one lane each)
constexpr int WS_THREADS = 512;

// CSR of the (nrows x ncols) matrix view of W.  which = 0: rows (s,v), cols (w,t) ["left"];
// which = 1: rows (w,s), cols (t,v) ["right"].  One warp per row; blockIdx.y = which.
// Pass 1 counts the non-zeros of every row, pass 2 sums the counts of the rows before its own
// (a few hundred integers) and writes the row's entries in column order (ballot prefix).
constexpr int CSR_WARPS = 8;

__device__ __forceinline__ long long csr_widx(int which, int r, int c, int Dl, int d, int Dr, int ncols) {
  if (which == 0) { int s = r / Dr, v = r % Dr, w = c / d, t = c % d;
                    return (((long long)w * d + s) * d + t) * Dr + v; }
  return (long long)r * ncols + c;
}

__global__ void __launch_bounds__(CSR_WARPS * 32) csr_count_kernel(const c128 *W, int Dl, int d, int Dr, double tol,
                                                                    int *cnt0, int *cnt1) {
  const int which = blockIdx.y;
  const int nrows = which == 0 ? d * Dr : Dl * d, ncols = which == 0 ? Dl * d : d * Dr;
  const int lane = threadIdx.x & 31, r = blockIdx.x * CSR_WARPS + (threadIdx.x >> 5);
  if (r >= nrows) return;
  int n = 0;
  for (int c0 = 0; c0 < ncols; c0 += 32) {
    int c = c0 + lane;
    bool nz = false;
    if (c < ncols) { c128 x = W[csr_widx(which, r, c, Dl, d, Dr, ncols)]; nz = fabs(x.x) > tol || fabs(x.y) > tol; }
    n += __popc(__ballot_sync(0xffffffffu, nz));
  }
  if (lane == 0) (which == 0 ? cnt0 : cnt1)[r] = n;
}

__global__ void __launch_bounds__(CSR_WARPS * 32) csr_fill_kernel(const c128 *W, int Dl, int d, int Dr, double tol,
                                                                   const int *cnt0, const int *cnt1,
                                                                   int *rowptr0, int *col0, c128 *val0,
                                                                   int *rowptr1, int *col1, c128 *val1) {
  const int which = blockIdx.y;
  const int nrows = which == 0 ? d * Dr : Dl * d, ncols = which == 0 ? Dl * d : d * Dr;
  const int *cnt = which == 0 ? cnt0 : cnt1;
  int *rowptr = which == 0 ? rowptr0 : rowptr1;
  int *col = which == 0 ? col0 : col1;
  c128 *val = which == 0 ? val0 : val1;
  const int lane = threadIdx.x & 31, r = blockIdx.x * CSR_WARPS + (threadIdx.x >> 5);
  if (r >= nrows) return;
  int o = 0;
  for (int i = lane; i < r; i += 32) o += cnt[i];
#pragma unroll
  for (int k = 16; k > 0; k >>= 1) o += __shfl_xor_sync(0xffffffffu, o, k);
  if (lane == 0) { rowptr[r] = o; if (r == nrows - 1) rowptr[nrows] = o + cnt[r]; }
  for (int c0 = 0; c0 < ncols; c0 += 32) {
    int c = c0 + lane;
    bool nz = false;
    c128 x = make_double2(0.0, 0.0);
    if (c < ncols) { x = W[csr_widx(which, r, c, Dl, d, Dr, ncols)]; nz = fabs(x.x) > tol || fabs(x.y) > tol; }
    unsigned m = __ballot_sync(0xffffffffu, nz);
    if (nz) { int q = o + __popc(m & ((1u << lane) - 1u)); col[q] = c; val[q] = x; }
    o += __popc(m);
  }
}

struct WStageParams {
  const c128 *in; c128 *out;
  int nrows, ncols, Mr;
  long long in_bs;                 // input batch stride (per a); input row stride is Mr
  int rdiv; long long o_s1, o_s2;  // output offset of row r: (r / rdiv) * o_s1 + (r % rdiv) * o_s2
  long long o_bs;                  // output batch stride
  const int *rowptr; const int *col; const c128 *val;
};

__device__ __forceinline__ void cfma(double &sx, double &sy, c128 w, c128 t) {
  sx = fma(w.x, t.x, sx); sx = fma(-w.y, t.y, sx);
  sy = fma(w.x, t.y, sy); sy = fma(w.y, t.x, sy);
}

// 16 warps per CTA and two CTAs per SM keep 8 warps per scheduler in flight; the entry loop is
// unrolled by four with all index / value / panel loads issued before the FMAs, so that the DFMA
// pipe (4 per entry and lane), not load latency, sets the pace at 15 % density, and HBM at ~3 %.
template <bool STAGE_SMEM>
__global__ void __launch_bounds__(WS_THREADS, 2) wstage_kernel(WStageParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  c128 *tile = reinterpret_cast<c128 *>(smem_raw);      // [ncols][YT]
  const int a = blockIdx.y;
  const int y0 = blockIdx.x * YT;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const c128 *__restrict__ in = p.in + a * p.in_bs;
  const int y = y0 + lane;
  const bool yok = y < p.Mr;
  if (STAGE_SMEM) {
    for (int e = threadIdx.x; e < p.ncols * YT; e += WS_THREADS) {
      int c = e / YT, yy = e % YT;
      bool ok = (y0 + yy) < p.Mr;
      const c128 *src = ok ? in + (long long)c * p.Mr + y0 + yy : in;
      unsigned s = (unsigned)__cvta_generic_to_shared(tile + e);
      int sz = ok ? 16 : 0;
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(src), "r"(sz));
    }
    asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;\n" ::);
    __syncthreads();
  }
  const int *__restrict__ colp = p.col;
  const c128 *__restrict__ valp = p.val;
  const long long yc = yok ? y : 0;
  auto panel = [&](int c) -> c128 {
    if (STAGE_SMEM) return tile[c * YT + lane];
    return __ldg(in + (long long)c * p.Mr + yc);
  };
  c128 *out = p.out + a * p.o_bs;
  for (int r = warp; r < p.nrows; r += WS_THREADS / 32) {
    const int e0 = __ldg(p.rowptr + r), e1 = __ldg(p.rowptr + r + 1);
    double sx0 = 0.0, sy0 = 0.0, sx1 = 0.0, sy1 = 0.0;
    int e = e0;
    for (; e + 4 <= e1; e += 4) {
      const int c0 = __ldg(colp + e), c1 = __ldg(colp + e + 1), c2 = __ldg(colp + e + 2), c3 = __ldg(colp + e + 3);
      const c128 w0 = __ldg(valp + e), w1 = __ldg(valp + e + 1), w2 = __ldg(valp + e + 2), w3 = __ldg(valp + e + 3);
      const c128 t0 = panel(c0), t1 = panel(c1), t2 = panel(c2), t3 = panel(c3);
      cfma(sx0, sy0, w0, t0); cfma(sx1, sy1, w1, t1); cfma(sx0, sy0, w2, t2); cfma(sx1, sy1, w3, t3);
    }
    for (; e < e1; e++) cfma(sx0, sy0, __ldg(valp + e), panel(__ldg(colp + e)));
    if (yok) out[(r / p.rdiv) * p.o_s1 + (r % p.rdiv) * p.o_s2 + y] = make_double2(sx0 + sx1, sy0 + sy1);
  }
}

// Persistent variant: one CTA of 32 warps per SM walks over (a, y-tile) work items.  The CSR of W
// (values, columns, row pointers) is staged ONCE per CTA in shared memory when it fits beside the
// panel (it does for every MPO of the paper's workloads and for the 15 % microbench), so the entry
// loop issues shared-memory loads only.  At 15 % density the loop is bound by the shared-memory
// crossbar (16 B of panel per 4 DFMA and lane); at the ~3 % density of real MPOs by HBM.
constexpr int WP_THREADS = 1024;
constexpr int WP_SMEM = 227 * 1024;

template <bool CSR_SMEM>
__device__ __forceinline__ void wp_rows(const WStageParams &p, const c128 *tile, const c128 *__restrict__ gval,
                                        const int *__restrict__ gcol, const int *__restrict__ grow, c128 *out,
                                        int y, int lane, int warp, int split, int nsplit) {
  for (int r = split + nsplit * warp; r < p.nrows; r += nsplit * (WP_THREADS / 32)) {
    const int e0 = grow[r], e1 = grow[r + 1];
    double sx0 = 0.0, sy0 = 0.0, sx1 = 0.0, sy1 = 0.0;
    int e = e0;
    for (; e + 4 <= e1; e += 4) {
      const int c0 = gcol[e], c1 = gcol[e + 1], c2 = gcol[e + 2], c3 = gcol[e + 3];
      const c128 w0 = gval[e], w1 = gval[e + 1], w2 = gval[e + 2], w3 = gval[e + 3];
      const c128 t0 = tile[c0 * YT + lane], t1 = tile[c1 * YT + lane], t2 = tile[c2 * YT + lane], t3 = tile[c3 * YT + lane];
      cfma(sx0, sy0, w0, t0); cfma(sx1, sy1, w1, t1); cfma(sx0, sy0, w2, t2); cfma(sx1, sy1, w3, t3);
    }
    for (; e < e1; e++) cfma(sx0, sy0, gval[e], tile[gcol[e] * YT + lane]);
    if (y < p.Mr) out[(r / p.rdiv) * p.o_s1 + (r % p.rdiv) * p.o_s2 + y] = make_double2(sx0 + sx1, sy0 + sy1);
  }
}

__global__ void __launch_bounds__(WP_THREADS, 1) wstage_persistent_kernel(WStageParams p, int ntile, int nitems, int nsplit) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  c128 *tile = reinterpret_cast<c128 *>(smem_raw);                        // [ncols][YT]
  const int tile_elems = p.ncols * YT;
  const int nnz = __ldg(p.rowptr + p.nrows);
  const size_t csr_off = (size_t)tile_elems * 16;
  const bool csr_smem = csr_off + (size_t)nnz * 20 + (size_t)(p.nrows + 1) * 4 + 64 <= (size_t)WP_SMEM;
  c128 *sval = reinterpret_cast<c128 *>(smem_raw + csr_off);
  int *scol = reinterpret_cast<int *>(smem_raw + csr_off + (size_t)nnz * 16);
  int *srow = scol + nnz;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (csr_smem) {
    for (int e = threadIdx.x; e < nnz; e += WP_THREADS) { sval[e] = __ldg(p.val + e); scol[e] = __ldg(p.col + e); }
    for (int e = threadIdx.x; e <= p.nrows; e += WP_THREADS) srow[e] = __ldg(p.rowptr + e);
  }
  for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
    const int split = item % nsplit, panel = item / nsplit;
    const int a = panel / ntile, y0 = (panel % ntile) * YT;
    const c128 *in = p.in + a * p.in_bs;
    __syncthreads();                                   // previous item's readers are done with the panel
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
    if (csr_smem) wp_rows<true>(p, tile, sval, scol, srow, out, y0 + lane, lane, warp, split, nsplit);
    else wp_rows<false>(p, tile, p.val, p.col, p.rowptr, out, y0 + lane, lane, warp, split, nsplit);
  }
}

int g_num_sms = 0;

void launch_wstage(cudaStream_t st, const WStageParams &p, int nbatch) {
  const int ntile = (p.Mr + YT - 1) / YT;
  size_t smem = (size_t)p.ncols * YT * 16;
  ProfScope ps(st, PH_WSTAGE);
  if (smem + 4096 <= (size_t)WP_SMEM) {
    if (!g_num_sms) { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&g_num_sms, cudaDevAttrMultiProcessorCount, dev); }
    // split the rows of a panel over several work items when the panels alone balance badly
    int nsplit = 1;
    while (nsplit < 4 && p.nrows >= 64 * nsplit) {
      const long long it = (long long)nbatch * ntile * nsplit;
      const long long rounds = (it + g_num_sms - 1) / g_num_sms;
      if (it >= g_num_sms && (double)it / (double)(rounds * g_num_sms) > 0.93) break;
      nsplit *= 2;
    }
    const int nitems = nbatch * ntile * nsplit;
    const int grid = nitems < g_num_sms ? nitems : g_num_sms;
    TDVP_LAUNCH(wstage_persistent_kernel, grid, WP_THREADS, WP_SMEM, st, p, ntile, nitems, nsplit);
    return;
  }
  dim3 grid(ntile, nbatch);
  if (smem <= 200 * 1024) {
    TDVP_LAUNCH(wstage_kernel<true>, grid, WS_THREADS, smem, st, p);
  } else {
    TDVP_LAUNCH(wstage_kernel<false>, grid, WS_THREADS, 0, st, p);
  }
}

}  // namespace

void wstage_configure() {
  cudaFuncSetAttribute(wstage_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
  cudaFuncSetAttribute(wstage_persistent_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, WP_SMEM);
}

size_t wsparse_bytes(int Dl, int d, int Dr) {
  size_t cap = (size_t)Dl * d * d * Dr;
  size_t rows0 = (size_t)d * Dr + 1, rows1 = (size_t)Dl * d + 1;
  auto up = [](size_t x) { return (x + 255) & ~size_t(255); };
  return 2 * up(rows0 * 4) + 2 * up(rows1 * 4) + 2 * up(cap * 4) + 2 * up(cap * 16) + 256;
}

void wsparse_build(cudaStream_t st, WSparse &ws, void *mem, int Dl, int d, int Dr, const c128 *W,
                   double zero_tol) {
  size_t cap = (size_t)Dl * d * d * Dr;
  auto up = [](size_t x) { return (x + 255) & ~size_t(255); };
  char *p = reinterpret_cast<char *>(mem);
  p = reinterpret_cast<char *>(up(reinterpret_cast<size_t>(p)));
  ws.Dl = Dl; ws.d = d; ws.Dr = Dr; ws.capacity = (int)cap;
  ws.val = reinterpret_cast<c128 *>(p); p += up(cap * 16);
  ws.val_r = reinterpret_cast<c128 *>(p); p += up(cap * 16);
  ws.col = reinterpret_cast<int *>(p); p += up(cap * 4);
  ws.col_r = reinterpret_cast<int *>(p); p += up(cap * 4);
  ws.rowptr = reinterpret_cast<int *>(p); p += up(((size_t)d * Dr + 1) * 4);
  ws.rowptr_r = reinterpret_cast<int *>(p);
  p += up(((size_t)Dl * d + 1) * 4);
  int *cnt0 = reinterpret_cast<int *>(p); p += up(((size_t)d * Dr + 1) * 4);
  int *cnt1 = reinterpret_cast<int *>(p);
  int maxrows = (d * Dr > Dl * d ? d * Dr : Dl * d);
  dim3 grid((maxrows + CSR_WARPS - 1) / CSR_WARPS, 2);
  TDVP_LAUNCH(csr_count_kernel, grid, CSR_WARPS * 32, 0, st, W, Dl, d, Dr, zero_tol, cnt0, cnt1);
  TDVP_LAUNCH(csr_fill_kernel, grid, CSR_WARPS * 32, 0, st, W, Dl, d, Dr, zero_tol, cnt0, cnt1,
              ws.rowptr, ws.col, ws.val, ws.rowptr_r, ws.col_r, ws.val_r);
}

void wstage_left(cudaStream_t st, const WSparse &ws, int Ml, int Mr, const c128 *T1, c128 *T2) {
  WStageParams p;
  p.in = T1; p.out = T2;
  p.nrows = ws.d * ws.Dr; p.ncols = ws.Dl * ws.d; p.Mr = Mr;
  p.in_bs = (long long)ws.Dl * ws.d * Mr;
  p.rdiv = p.nrows > 0 ? p.nrows : 1; p.o_s1 = 0; p.o_s2 = Mr;
  p.o_bs = (long long)ws.d * ws.Dr * Mr;
  p.rowptr = ws.rowptr; p.col = ws.col; p.val = ws.val;
  launch_wstage(st, p, Ml);
}

void wstage_right(cudaStream_t st, const WSparse &ws, int Ml, int Mr, const c128 *T1, c128 *T2) {
  WStageParams p;
  p.in = T1; p.out = T2;
  p.nrows = ws.Dl * ws.d; p.ncols = ws.d * ws.Dr; p.Mr = Mr;
  p.in_bs = (long long)ws.d * ws.Dr * Mr;
  p.rdiv = ws.d; p.o_s1 = (long long)Ml * ws.d * Mr; p.o_s2 = Mr;
  p.o_bs = (long long)ws.d * Mr;
  p.rowptr = ws.rowptr_r; p.col = ws.col_r; p.val = ws.val_r;
  launch_wstage(st, p, Ml);
}
