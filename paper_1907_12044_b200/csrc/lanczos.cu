// lanczos.cu -- y = exp(z H) v by the Lanczos / Krylov method (SURVEY.md 8(a) a6,
// 8(c) O3/c11): fixed Krylov dimension k, alpha_j = Re<q_j, H q_j>, full re-orthogonalisation (two
// classical Gram-Schmidt passes against all previous vectors), breakdown rule
// beta_j < 1e-14 * max(1, |alpha_j|).
//
// The paper attributes a large share of its GPU step time to this sub-step because every alpha and
// beta crossed PCIe.  Here every scalar of the recurrence lives in device
// memory: reductions finish in the last CTA to arrive (fixed summation order: deterministic), the
// breakdown decision is a device flag that turns the remaining iterations into no-ops (q = 0), and
// the k x k tridiagonal eigenproblem runs in one warp.  Nothing is read back by the host.
#include <cooperative_groups.h>
#include <cstdlib>

#include "common.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int VT = 256;                 // threads per CTA of the vector kernels
constexpr int MAXG = 296;               // max CTAs of a vector kernel (2 per SM)
constexpr double BREAKDOWN_TOL = 1e-14;

struct LzState {
  int m;            // Krylov dimension used (valid once done)
  int done;
  double beta0;
  double inv_beta;  // 1/beta_j of the current iteration, 0 after breakdown
};

struct LzBuffers {
  c128 *Q;          // [(k+1)][n]
  c128 *dots;       // [k+1]
  c128 *coef;       // [k]
  double *alpha;    // [k]
  double *beta;     // [k]
  LzState *state;
  unsigned *counter;
  c128 *partial;    // [MAXG][k+1]
  double *npartial; // [MAXG]
  void *apply_ws;
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// True in exactly one CTA: the last one to arrive.  Resets the counter for the next kernel.
__device__ __forceinline__ bool last_block(unsigned *counter) {
  __shared__ bool is_last;
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned t = atomicAdd(counter, 1u);
    is_last = (t == gridDim.x - 1);
    if (is_last) *counter = 0u;
  }
  __syncthreads();
  if (is_last) __threadfence();
  return is_last;
}

__device__ __forceinline__ void chunk_of(long long n, long long &e0, long long &e1) {
  long long per = (n + gridDim.x - 1) / gridDim.x;
  e0 = (long long)blockIdx.x * per;
  e1 = e0 + per; if (e1 > n) e1 = n;
}

// beta0 = ||v||, state reset.
__global__ void __launch_bounds__(VT) lz_init_kernel(const c128 *v, long long n, LzBuffers b) {
  long long e0, e1; chunk_of(n, e0, e1);
  double s = 0.0;
  for (long long e = e0 + threadIdx.x; e < e1; e += VT) { c128 x = v[e]; s += x.x * x.x + x.y * x.y; }
  __shared__ double red[VT / 32];
  s = warp_sum(s);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) { double t = 0; for (int i = 0; i < VT / 32; i++) t += red[i]; b.npartial[blockIdx.x] = t; }
  if (last_block(b.counter) && threadIdx.x < 32) {
    double t = 0.0;
    for (int g = threadIdx.x; g < gridDim.x; g += 32) t += b.npartial[g];
    t = warp_sum(t);
    if (threadIdx.x == 0) {
      double beta0 = sqrt(t);
      b.state->beta0 = beta0;
      b.state->inv_beta = beta0 > 0.0 ? 1.0 / beta0 : 0.0;
      b.state->done = 0;
      b.state->m = 0;
    }
  }
}

// dst = src * state.inv_beta
__global__ void __launch_bounds__(VT) lz_scale_kernel(c128 *dst, const c128 *src, long long n, const LzState *st) {
  const double f = st->inv_beta;
  for (long long e = blockIdx.x * (long long)VT + threadIdx.x; e < n; e += (long long)gridDim.x * VT) {
    c128 x = src[e];
    dst[e] = make_double2(x.x * f, x.y * f);
  }
}

// dots[i] = <q_i, w> for i < nd (conjugate on q).  first_pass: alpha[j] = Re dots[j].
__global__ void __launch_bounds__(VT) lz_dots_kernel(long long n, int nd, int j, int first_pass, LzBuffers b) {
  const c128 *w = b.Q + (long long)(j + 1) * n;
  long long e0, e1; chunk_of(n, e0, e1);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int i = warp; i < nd; i += VT / 32) {
    const c128 *q = b.Q + (long long)i * n;
    double sx = 0.0, sy = 0.0;
    for (long long e = e0 + lane; e < e1; e += 32) {
      c128 a = q[e], x = w[e];
      sx += a.x * x.x + a.y * x.y;
      sy += a.x * x.y - a.y * x.x;
    }
    sx = warp_sum(sx); sy = warp_sum(sy);
    if (lane == 0) b.partial[(long long)blockIdx.x * nd + i] = make_double2(sx, sy);
  }
  if (last_block(b.counter)) {
    for (int i = warp; i < nd; i += VT / 32) {
      double sx = 0.0, sy = 0.0;
      for (int g = lane; g < gridDim.x; g += 32) { c128 p = b.partial[(long long)g * nd + i]; sx += p.x; sy += p.y; }
      sx = warp_sum(sx); sy = warp_sum(sy);
      if (lane == 0) {
        b.dots[i] = make_double2(sx, sy);
        if (first_pass && i == j && !b.state->done) b.alpha[j] = sx;
      }
    }
  }
}

// w -= sum_{i<nd} dots[i] q_i.  If with_norm: beta_j = ||w|| and the breakdown decision.
__global__ void __launch_bounds__(VT) lz_update_kernel(long long n, int nd, int j, int k, int with_norm, LzBuffers b) {
  c128 *w = b.Q + (long long)(j + 1) * n;
  long long e0, e1; chunk_of(n, e0, e1);
  __shared__ c128 cs[TDVP_MAX_KRYLOV + 1];
  for (int i = threadIdx.x; i < nd; i += VT) cs[i] = b.dots[i];
  __syncthreads();
  double s = 0.0;
  for (long long e = e0 + threadIdx.x; e < e1; e += VT) {
    c128 x = w[e];
    for (int i = 0; i < nd; i++) {
      c128 q = b.Q[(long long)i * n + e], c = cs[i];
      x.x -= c.x * q.x - c.y * q.y;
      x.y -= c.x * q.y + c.y * q.x;
    }
    w[e] = x;
    s += x.x * x.x + x.y * x.y;
  }
  if (!with_norm) return;
  __shared__ double red[VT / 32];
  s = warp_sum(s);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) { double t = 0; for (int i = 0; i < VT / 32; i++) t += red[i]; b.npartial[blockIdx.x] = t; }
  if (last_block(b.counter) && threadIdx.x < 32) {
    double t = 0.0;
    for (int g = threadIdx.x; g < gridDim.x; g += 32) t += b.npartial[g];
    t = warp_sum(t);
    if (threadIdx.x == 0) {
      LzState *st = b.state;
      double beta = sqrt(t);
      if (!st->done) {
        double aj = fabs(b.alpha[j]);
        if (j == k - 1 || beta < BREAKDOWN_TOL * (aj > 1.0 ? aj : 1.0)) {
          st->done = 1; st->m = j + 1; st->inv_beta = 0.0;
        } else {
          b.beta[j] = beta; st->inv_beta = 1.0 / beta;
        }
      } else {
        st->inv_beta = 0.0;
      }
    }
  }
}

// ---- fused orthogonalisation step (cooperative launch) ---------------------------------------
// One kernel per Lanczos iteration instead of five: every CTA keeps its chunk of w = H q_j and of
// q_0..q_j in shared memory (one pass over HBM/L2), and the three global reductions (the two
// Gram-Schmidt passes and the norm) are grid-wide barriers of a cooperative launch.  Partial sums are
// added in a fixed order by every CTA, so all CTAs hold bit-identical scalars: deterministic.
constexpr int FT = 256;
constexpr size_t FUSED_SMEM_MAX = 200 * 1024;

__device__ __forceinline__ void fused_dots(const c128 *sw, const c128 *sq, int chunk, int len, int nd, c128 *partial,
                                           int lane, int warp) {
  for (int i = warp; i < nd; i += FT / 32) {
    const c128 *q = sq + (size_t)i * chunk;
    double sx = 0.0, sy = 0.0;
    for (int e = lane; e < len; e += 32) {
      c128 a = q[e], x = sw[e];
      sx += a.x * x.x + a.y * x.y;
      sy += a.x * x.y - a.y * x.x;
    }
    sx = warp_sum(sx); sy = warp_sum(sy);
    if (lane == 0) partial[(size_t)blockIdx.x * nd + i] = make_double2(sx, sy);
  }
}
// every CTA: cs[i] = sum_g partial[g][i] in a fixed order
__device__ __forceinline__ void fused_gather(const c128 *partial, int nd, c128 *cs, int lane, int warp) {
  for (int i = warp; i < nd; i += FT / 32) {
    double sx = 0.0, sy = 0.0;
    for (int g = lane; g < (int)gridDim.x; g += 32) { c128 pz = __ldcg(partial + (size_t)g * nd + i); sx += pz.x; sy += pz.y; }
    sx = warp_sum(sx); sy = warp_sum(sy);
    if (lane == 0) cs[i] = make_double2(sx, sy);
  }
  __syncthreads();
}

// Grid barrier on a counter that only grows during one exponential (zeroed by the host before the
// first iteration): arrival = one atomic add per CTA, release when the count reaches `target`.  The
// launch is cooperative, so all CTAs are resident.  (cg::grid_group::sync does the same with more
// bookkeeping; three barriers per call are most of this kernel's time.)
__device__ __forceinline__ void lz_grid_bar(unsigned *ctr, unsigned target) {
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    atomicAdd(ctr, 1u);
    unsigned v;
    do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(ctr) : "memory"); } while (v < target);
  }
  __syncthreads();
}

__global__ void __launch_bounds__(FT) lz_fused_orth_kernel(long long n, int chunk, int j, int k, LzBuffers b) {
  unsigned *bar = b.counter + 1;
  const unsigned bar0 = 3u * (unsigned)j * gridDim.x;     // every earlier iteration passed three barriers
  extern __shared__ __align__(16) unsigned char fsm[];
  c128 *sw = reinterpret_cast<c128 *>(fsm);                       // [chunk]
  c128 *sq = sw + chunk;                                          // [j + 1][chunk]
  __shared__ c128 cs[TDVP_MAX_KRYLOV + 1];
  __shared__ double red[FT / 32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nd = j + 1;
  const long long e0 = (long long)blockIdx.x * chunk;
  const int len = (int)((e0 + chunk <= n) ? chunk : (n > e0 ? n - e0 : 0));
  const int was_done = b.state->done;                             // read before anybody can change it
  c128 *wg = b.Q + (long long)(j + 1) * n + e0;
  if (j == k - 1) {
    // last iteration: only alpha_j = Re<q_j, w> is needed (the recurrence stops before q_{k+1} is
    // formed, PAPER.md:292-296 / oracle O3) -- one reduction, one grid barrier, no orthogonalisation
    const c128 *qg = b.Q + (long long)j * n + e0;
    double s = 0.0;
    for (int e = tid; e < len; e += FT) {
      const c128 q = __ldcg(qg + e), x = __ldcg(wg + e);
      s = fma(q.x, x.x, fma(q.y, x.y, s));
    }
    s = warp_sum(s);
    if (lane == 0) red[warp] = s;
    __syncthreads();
    if (tid == 0) { double t = 0; for (int i = 0; i < FT / 32; i++) t += red[i]; b.npartial[blockIdx.x] = t; }
    lz_grid_bar(bar, bar0 + gridDim.x);
    if (blockIdx.x == 0 && warp == 0) {
      double t = 0.0;
      for (int g = lane; g < (int)gridDim.x; g += 32) t += __ldcg(b.npartial + g);
      t = warp_sum(t);
      if (lane == 0) {
        LzState *st = b.state;
        if (!was_done) { b.alpha[j] = t; st->done = 1; st->m = j + 1; }
        st->inv_beta = 0.0;
      }
    }
    return;
  }
  // all loads of the chunk in flight at once (16 B asynchronous copies), one wait
  for (int e = tid; e < len; e += FT) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(sw + e);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sa), "l"(wg + e));
  }
  for (int i = 0; i < nd; i++) {
    const c128 *qg = b.Q + (long long)i * n + e0;
    for (int e = tid; e < len; e += FT) {
      const unsigned sa = (unsigned)__cvta_generic_to_shared(sq + (size_t)i * chunk + e);
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sa), "l"(qg + e));
    }
  }
  asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;\n" ::: "memory");
  __syncthreads();
  for (int pass = 0; pass < 2; pass++) {
    c128 *partial = b.partial + (size_t)pass * MAXG * (TDVP_MAX_KRYLOV + 1);
    fused_dots(sw, sq, chunk, len, nd, partial, lane, warp);
    lz_grid_bar(bar, bar0 + (unsigned)(pass + 1) * gridDim.x);
    fused_gather(partial, nd, cs, lane, warp);
    if (pass == 0 && blockIdx.x == 0 && tid == 0 && !was_done) b.alpha[j] = cs[j].x;
    for (int e = tid; e < len; e += FT) {
      c128 x = sw[e];
      for (int i = 0; i < nd; i++) {
        c128 q = sq[(size_t)i * chunk + e], c = cs[i];
        x.x -= c.x * q.x - c.y * q.y;
        x.y -= c.x * q.y + c.y * q.x;
      }
      sw[e] = x;
    }
    __syncthreads();
  }
  double s = 0.0;
  for (int e = tid; e < len; e += FT) { c128 x = sw[e]; s += x.x * x.x + x.y * x.y; }
  s = warp_sum(s);
  if (lane == 0) red[warp] = s;
  __syncthreads();
  if (tid == 0) { double t = 0; for (int i = 0; i < FT / 32; i++) t += red[i]; b.npartial[blockIdx.x] = t; }
  lz_grid_bar(bar, bar0 + 3u * gridDim.x);
  double t = 0.0;
  for (int g = lane; g < (int)gridDim.x; g += 32) t += __ldcg(b.npartial + g);
  t = warp_sum(t);
  const double beta = sqrt(t);
  double inv_beta = 0.0;
  bool now_done = was_done;
  if (!was_done) {
    const double aj = fabs(__ldcg(b.alpha + j));
    if (j == k - 1 || beta < BREAKDOWN_TOL * (aj > 1.0 ? aj : 1.0)) now_done = true;
    else inv_beta = 1.0 / beta;
  }
  if (blockIdx.x == 0 && tid == 0) {
    LzState *st = b.state;
    if (!was_done) {
      if (now_done) { st->done = 1; st->m = j + 1; st->inv_beta = 0.0; }
      else { b.beta[j] = beta; st->inv_beta = inv_beta; }
    } else {
      st->inv_beta = 0.0;
    }
  }
  if (j < k - 1)
    for (int e = tid; e < len; e += FT) { c128 x = sw[e]; wg[e] = make_double2(x.x * inv_beta, x.y * inv_beta); }
}

// One warp: coef = beta0 * V exp(z Lambda) V^T e_1 for the m x m tridiagonal (alpha, beta)
// ("diagonalize the tridiagonal matrix in the subspace").  Implicit symmetric QR
// iteration with Wilkinson shift and deflation (Golub & Van Loan, "Matrix Computations", sec. 8.3).
// The scalar recurrence of a sweep is a dependent FP64 chain: lane 0 alone runs it on shared-memory
// copies of the diagonals and records the sweep's rotations; then every lane applies them to the
// eigenvector rows it owns.  (All 32 lanes used to repeat the chain on local-memory arrays: 66 us.)
__global__ void __launch_bounds__(32) lz_coef_kernel(int k, double zr, double zi, LzBuffers b, int *m_out) {
  __shared__ double V[TDVP_MAX_KRYLOV * TDVP_MAX_KRYLOV];
  __shared__ double a[TDVP_MAX_KRYLOV], off[TDVP_MAX_KRYLOV], rc[TDVP_MAX_KRYLOV], rs[TDVP_MAX_KRYLOV];
  __shared__ int s_lo, s_hi;
  const int lane = threadIdx.x;
  const int m = b.state->m;
  if (lane == 0 && m_out) *m_out = m;
  for (int i = lane; i < m; i += 32) { a[i] = b.alpha[i]; off[i] = (i < m - 1) ? b.beta[i] : 0.0; }
  for (int r = lane; r < m; r += 32)
    for (int c = 0; c < m; c++) V[r * m + c] = (r == c) ? 1.0 : 0.0;
  __syncwarp();
  const double eps = 2.220446049250313e-16;
  int hi = m - 1, guard = 0;
  while (true) {
    if (lane == 0) {
      int lo = -1;
      while (hi > 0 && guard < 64 * m) {
        guard++;
        for (int i = 0; i < hi; i++)
          if (fabs(off[i]) <= eps * (fabs(a[i]) + fabs(a[i + 1]))) off[i] = 0.0;
        if (off[hi - 1] == 0.0) { hi--; continue; }
        lo = hi - 1;
        while (lo > 0 && off[lo - 1] != 0.0) lo--;
        break;
      }
      if (hi > 0 && guard < 64 * m && lo >= 0) {
        // Wilkinson shift from the trailing 2x2 of the unreduced block [lo, hi]
        const double dd = 0.5 * (a[hi - 1] - a[hi]), bb = off[hi - 1];
        const double den = dd + (dd >= 0.0 ? 1.0 : -1.0) * sqrt(dd * dd + bb * bb);
        const double mu = a[hi] - bb * bb / den;
        double x = a[lo] - mu, z = off[lo];
        for (int q = lo; q < hi; q++) {
          // the chain sqrt -> two divisions is the latency of the sweep: one reciprocal square root instead
          const double r2 = x * x + z * z;
          double c = 1.0, sn = 0.0, r = 0.0;
          if (r2 > 0.0) { const double ri = rsqrt(r2); c = x * ri; sn = z * ri; r = r2 * ri; }
          if (q > lo) off[q - 1] = r;
          const double ak = a[q], ak1 = a[q + 1], bk = off[q];
          a[q] = c * c * ak + 2.0 * c * sn * bk + sn * sn * ak1;
          a[q + 1] = sn * sn * ak - 2.0 * c * sn * bk + c * c * ak1;
          off[q] = c * sn * (ak1 - ak) + (c * c - sn * sn) * bk;
          x = off[q];
          if (q < hi - 1) { z = sn * off[q + 1]; off[q + 1] = c * off[q + 1]; }
          rc[q] = c; rs[q] = sn;
        }
        s_lo = lo; s_hi = hi;
      } else {
        s_lo = 0; s_hi = 0;                              // converged (or the guard tripped)
      }
    }
    __syncwarp();
    const int lo = s_lo, h2 = s_hi;
    if (h2 == 0) break;
    for (int row = lane; row < m; row += 32)
      for (int q = lo; q < h2; q++) {
        const double c = rc[q], sn = rs[q];
        const double vk = V[row * m + q], vk1 = V[row * m + q + 1];
        V[row * m + q] = c * vk + sn * vk1;
        V[row * m + q + 1] = -sn * vk + c * vk1;
      }
    __syncwarp();
  }
  const double beta0 = b.state->beta0;
  for (int r = lane; r < k; r += 32) {
    double cx = 0.0, cy = 0.0;
    if (r < m) {
      for (int i = 0; i < m; i++) {
        double mag = exp(zr * a[i]), sn, cn;
        sincos(zi * a[i], &sn, &cn);
        double wgt = V[r * m + i] * V[i] * mag;      // V[0][i] = V[i]
        cx += wgt * cn; cy += wgt * sn;
      }
    }
    b.coef[r] = make_double2(beta0 * cx, beta0 * cy);
  }
}

// y = sum_{j<k} coef[j] q_j
__global__ void __launch_bounds__(VT) lz_combine_kernel(long long n, int k, LzBuffers b, c128 *y) {
  __shared__ c128 cs[TDVP_MAX_KRYLOV];
  for (int i = threadIdx.x; i < k; i += VT) cs[i] = b.coef[i];
  __syncthreads();
  for (long long e = blockIdx.x * (long long)VT + threadIdx.x; e < n; e += (long long)gridDim.x * VT) {
    double sx = 0.0, sy = 0.0;
    for (int i = 0; i < k; i++) {
      c128 q = b.Q[(long long)i * n + e], c = cs[i];
      sx += c.x * q.x - c.y * q.y;
      sy += c.x * q.y + c.y * q.x;
    }
    y[e] = make_double2(sx, sy);
  }
}

inline size_t up256(size_t x) { return (x + 255) & ~size_t(255); }

size_t apply_ws_bytes(const LanczosOp &op) {
  return op.kind == 0 ? heff_ws_bytes(op.Ml, op.Mr, op.d, op.Dl, op.Dr) : bond_ws_bytes(op.Ml, op.Mr, op.Dl);
}

}  // namespace

bool g_lanczos_unfused = false;   // test hook (TDVP_LANCZOS_UNFUSED=1): force the five-kernel path

void lanczos_configure() {
  cudaFuncSetAttribute(lz_fused_orth_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FUSED_SMEM_MAX);
  const char *e = getenv("TDVP_LANCZOS_UNFUSED");
  g_lanczos_unfused = e && e[0] == '1';
}

size_t lanczos_ws_bytes(const LanczosOp &op, int k) {
  size_t n = (size_t)op.Ml * (op.kind == 0 ? op.d : 1) * op.Mr;
  return up256((k + 1) * n * 16) + up256((k + 1) * 16) + up256(k * 16) + 2 * up256(k * 8) +
         up256(sizeof(LzState)) + 256 + up256((size_t)2 * MAXG * (TDVP_MAX_KRYLOV + 1) * 16) + up256(MAXG * 8) +
         apply_ws_bytes(op) + 512;
}

void lanczos_expm(cudaStream_t st, const LanczosOp &op, int k, double z_re, double z_im,
                  const c128 *v, c128 *y, void *ws, int *m_used_dev) {
  const long long n = (long long)op.Ml * (op.kind == 0 ? op.d : 1) * op.Mr;
  char *p = reinterpret_cast<char *>(up256(reinterpret_cast<size_t>(ws)));
  LzBuffers b;
  b.Q = reinterpret_cast<c128 *>(p); p += up256((k + 1) * n * 16);
  b.dots = reinterpret_cast<c128 *>(p); p += up256((k + 1) * 16);
  b.coef = reinterpret_cast<c128 *>(p); p += up256(k * 16);
  b.alpha = reinterpret_cast<double *>(p); p += up256(k * 8);
  b.beta = reinterpret_cast<double *>(p); p += up256(k * 8);
  b.state = reinterpret_cast<LzState *>(p); p += up256(sizeof(LzState));
  b.counter = reinterpret_cast<unsigned *>(p); p += 256;
  b.partial = reinterpret_cast<c128 *>(p); p += up256((size_t)2 * MAXG * (TDVP_MAX_KRYLOV + 1) * 16);
  b.npartial = reinterpret_cast<double *>(p); p += up256(MAXG * 8);
  b.apply_ws = p;

  int G = (int)((n + VT - 1) / VT);
  if (G > MAXG) G = MAXG;
  if (G < 1) G = 1;
  // fused cooperative path: one CTA per SM at most, the chunk of all k + 1 vectors in shared memory
  static int num_sms = 0;
  if (!num_sms) { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev); }
  int FG = (int)((n + FT - 1) / FT);
  if (FG > num_sms) FG = num_sms;
  if (FG < 1) FG = 1;
  const int chunk = (int)((n + FG - 1) / FG);
  const bool fused = !g_lanczos_unfused && (size_t)(k + 1) * chunk * 16 <= FUSED_SMEM_MAX;
  {
    ProfScope ps(st, PH_VEC);
    cudaMemsetAsync(b.counter, 0, 2 * sizeof(unsigned), st);   // [0] last-block counter, [1] grid-barrier counter
    TDVP_LAUNCH(lz_init_kernel, G, VT, 0, st, v, n, b);
    TDVP_LAUNCH(lz_scale_kernel, G, VT, 0, st, b.Q, v, n, b.state);
  }
  for (int j = 0; j < k; j++) {
    c128 *qj = b.Q + (long long)j * n, *w = b.Q + (long long)(j + 1) * n;
    if (op.kind == 0)
      heff_apply(st, op.Ml, op.Mr, op.d, op.Dl, op.Dr, op.L, *op.W, qj, op.R, w, b.apply_ws);
    else
      bond_apply(st, op.Ml, op.Mr, op.Dl, op.L, qj, op.R, w, b.apply_ws);
    ProfScope ps(st, PH_VEC);
    if (fused) {
      long long nn = n; int ch = chunk, jj = j, kk = k;
      void *args[] = {&nn, &ch, &jj, &kk, &b};
      cudaLaunchCooperativeKernel((void *)lz_fused_orth_kernel, dim3(FG), dim3(FT), args, (size_t)(j + 2) * chunk * 16, st);
      count_launch();
    } else {
      TDVP_LAUNCH(lz_dots_kernel, G, VT, 0, st, n, j + 1, j, 1, b);
      TDVP_LAUNCH(lz_update_kernel, G, VT, 0, st, n, j + 1, j, k, 0, b);
      TDVP_LAUNCH(lz_dots_kernel, G, VT, 0, st, n, j + 1, j, 0, b);
      TDVP_LAUNCH(lz_update_kernel, G, VT, 0, st, n, j + 1, j, k, 1, b);
      if (j < k - 1) TDVP_LAUNCH(lz_scale_kernel, G, VT, 0, st, w, w, n, b.state);
    }
  }
  ProfScope ps(st, PH_VEC);
  TDVP_LAUNCH(lz_coef_kernel, 1, 32, 0, st, k, z_re, z_im, b, m_used_dev);
  TDVP_LAUNCH(lz_combine_kernel, G, VT, 0, st, n, k, b, y);
}
