// lanczos.cu -- y = exp(z H) v by the Lanczos / Krylov method (SURVEY.md 8(a) a6,
// 8(c) O3/c11): Krylov dimension k, alpha_j = Re<q_j, H q_j>, full re-orthogonalisation (two
// classical Gram-Schmidt passes against all previous vectors), breakdown rule
// beta_j < 1e-14 * max(1, |alpha_j|), and -- when krylov_tol > 0 -- the adaptive stop at the first j
// with beta_j |[exp(z T_j) e_1]_j| < krylov_tol (the paper: "continues until |Psi(t + tau)> converges",
// PAPER.md:292, no formula given; reading c11).
//
// The paper attributes a large share of its GPU step time to this sub-step because every alpha and
// beta crossed PCIe.  Here every scalar of the recurrence lives in device
// memory and the whole exponential is enqueue-only.  Per iteration there are two kernels: the
// operator apply (GEMM / W stage / GEMM) and ONE cooperative orthogonalisation kernel with two grid
// barriers (one per Gram-Schmidt pass).  What used to be a third barrier (the norm beta_j) and two
// extra kernels (norm of v, scaling) are gone, because normalisation is DEFERRED: H is linear, so the
// next apply runs on the unnormalised vector u_{j+1} and the next orthogonalisation kernel scales
// both u_{j+1} and H u_{j+1} by 1 / beta_j, which every CTA sums for itself, in a fixed order, from the
// per-CTA partial norms the previous kernel left behind.  The stop decisions (breakdown, adaptive
// tolerance) are taken the same way -- redundantly and identically by every CTA -- and recorded per
// iteration in hist[], which the following apply kernels read as a "skip" flag.  The coefficients
// c = exp(z T) e_1 of the k x k tridiagonal T ("diagonalize the tridiagonal matrix in the subspace",
// PAPER.md:294) are evaluated for z = i zeta by a Chebyshev (Jacobi-Anger) expansion of exp(i zeta T) e_1
// inside the kernel that combines the basis vectors (one warp, ~3 us, no eigen-decomposition: the
// implicit-QR iteration it replaces was a 50 us dependent chain); for z with a real part the
// eigen-decomposition kernel is kept.  Nothing is read back by the host.
#include <cooperative_groups.h>
#include <cstdlib>

#include "common.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int VT = 256;                 // threads per CTA of the vector kernels
constexpr int MAXG = 296;               // max CTAs of a vector kernel
constexpr double BREAKDOWN_TOL = 1e-14;
constexpr int CHEB_MAX = 2048;          // Bessel coefficients kept: |zeta| * (half width of T's Gershgorin interval) <= ~1850

struct LzState {
  int m;            // Krylov dimension used (valid once the last orthogonalisation kernel has run)
  int pad;
  double beta0;
};

struct LzBuffers {
  c128 *Q;          // [(k+1)][n]: slot j holds u_j, normalised in place to q_j by iteration j
  c128 *coef;       // [k] (only written by the eigen-decomposition path)
  double *alpha;    // [k]
  double *beta;     // [k]
  LzState *state;
  int *hist;        // [k + 1]: hist[j] = 1 if the recurrence had stopped when iteration j decided
  unsigned *bar;    // [2 k + 2] grid-barrier counters, two per iteration, zeroed per exponential
  c128 *partial;    // [2][MAXG][k + 1]
  double *npartial; // [MAXG]
  int *status;      // handle's sticky device status (nullable)
  void *apply_ws;
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// ---- c = exp(i zeta T) e_1 for the real symmetric tridiagonal T = (alpha[0..m), beta[0..m-1)) -------
// One warp, m <= 64: lane l owns components l and l + 32.  Jacobi-Anger: with T~ = (T - c0) / r in
// [-1, 1] (Gershgorin), exp(i zeta T) = e^{i zeta c0} (J_0(x) + 2 sum_n i^n J_n(x) T_n(T~)), x = zeta r.
// J_n by Miller's backward recurrence (lane 0, into jn[]), T_n(T~) e_1 by the three-term recurrence
// with neighbour components fetched by shuffles.  Returns the two components of the lane; sets
// *range_error if the series would need more than CHEB_MAX terms.
__device__ void cheb_expm_e1(int m, const double *alpha, const double *beta, double zeta, double *jn /*[CHEB_MAX + 64] shared*/,
                             c128 &c_lo, c128 &c_hi, int *range_error) {
  const int lane = threadIdx.x & 31;
  const int i0 = lane, i1 = lane + 32;
  double a0 = i0 < m ? __ldcg(alpha + i0) : 0.0, a1 = i1 < m ? __ldcg(alpha + i1) : 0.0;
  double bu0 = i0 < m - 1 ? __ldcg(beta + i0) : 0.0, bu1 = i1 < m - 1 ? __ldcg(beta + i1) : 0.0;     // coupling to i + 1
  double bl0 = (i0 >= 1 && i0 < m) ? __ldcg(beta + i0 - 1) : 0.0, bl1 = i1 < m ? __ldcg(beta + i1 - 1) : 0.0;   // to i - 1
  double lo = 1e300, hi = -1e300;
  if (i0 < m) { lo = fmin(lo, a0 - fabs(bu0) - fabs(bl0)); hi = fmax(hi, a0 + fabs(bu0) + fabs(bl0)); }
  if (i1 < m) { lo = fmin(lo, a1 - fabs(bu1) - fabs(bl1)); hi = fmax(hi, a1 + fabs(bu1) + fabs(bl1)); }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o)); hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o)); }
  const double c0 = 0.5 * (lo + hi), r = 0.5 * (hi - lo);
  double ps, pc;
  sincos(zeta * c0, &ps, &pc);
  const double x = zeta * r, ax = fabs(x);
  if (!(r > 0.0) || ax == 0.0) {             // T = c0 I (m = 1, or nothing to evolve)
    c_lo = i0 == 0 ? make_double2(pc, ps) : make_double2(0.0, 0.0);
    c_hi = make_double2(0.0, 0.0);
    return;
  }
  int N = (int)(ax + 12.0 * cbrt(ax) + 30.0);
  if (N > CHEB_MAX) { N = CHEB_MAX; if (range_error) *range_error = 1; }
  if (lane == 0) {                            // Miller: J_{n-1} = (2 n / x) J_n - J_{n+1} downwards from n = nstart
    int nstart = N + 20 + (int)sqrt(40.0 * N);
    nstart += nstart & 1;
    double jp1 = 0.0, jc = 1e-280, sum = 0.0;
    const double two_over_x = 2.0 / ax;
    for (int n = nstart; n >= 1; n--) {
      if (n <= N) jn[n] = jc;
      if ((n & 1) == 0) sum += jc;
      const double jm = (double)n * two_over_x * jc - jp1;
      jp1 = jc; jc = jm;
    }
    jn[0] = jc;
    const double inv = 1.0 / (jc + 2.0 * sum);       // 1 = J_0 + 2 sum_{k >= 1} J_{2k}
    jn[N + 1] = inv;
  }
  __syncwarp();
  const double norm = jn[N + 1];
  const double ir = 1.0 / r;
  a0 = (a0 - c0) * ir; a1 = (a1 - c0) * ir; bu0 *= ir; bu1 *= ir; bl0 *= ir; bl1 *= ir;
  const bool two = m > 32;
  auto matvec = [&](double t0, double t1, double &o0, double &o1) {
    // neighbours: below component l is lane l - 1's first; above is lane l + 1's first, or lane 0's second for l = 31
    const double dn0 = __shfl_up_sync(0xffffffffu, t0, 1);
    double up0 = __shfl_down_sync(0xffffffffu, t0, 1);
    o0 = a0 * t0 + bl0 * dn0;
    if (two) {
      const double first_hi = __shfl_sync(0xffffffffu, t1, 0);
      const double last_lo = __shfl_sync(0xffffffffu, t0, 31);
      const double dn1s = __shfl_up_sync(0xffffffffu, t1, 1);
      const double up1 = __shfl_down_sync(0xffffffffu, t1, 1);
      if (lane == 31) up0 = first_hi;
      const double dn1 = lane == 0 ? last_lo : dn1s;
      o1 = a1 * t1 + bl1 * dn1 + bu1 * (lane == 31 ? 0.0 : up1);
    } else {
      o1 = 0.0;
      if (lane == 31) up0 = 0.0;
    }
    o0 += bu0 * up0;
  };
  // (i s)^n cycles through 1, i s, -1, -i s
  const double s = x > 0.0 ? 1.0 : -1.0;
  double tp0 = i0 == 0 ? 1.0 : 0.0, tp1 = 0.0, tc0, tc1;
  matvec(tp0, tp1, tc0, tc1);
  double re0 = jn[0] * tp0, re1 = 0.0, im0 = 2.0 * s * jn[1] * tc0, im1 = 2.0 * s * jn[1] * tc1;
  for (int n = 2; n <= N; n++) {
    double m0, m1;
    matvec(tc0, tc1, m0, m1);
    const double tn0 = 2.0 * m0 - tp0, tn1 = 2.0 * m1 - tp1;
    tp0 = tc0; tp1 = tc1; tc0 = tn0; tc1 = tn1;
    const double w = 2.0 * jn[n];
    switch (n & 3) {
      case 0: re0 += w * tn0; re1 += w * tn1; break;
      case 1: im0 += s * w * tn0; im1 += s * w * tn1; break;
      case 2: re0 -= w * tn0; re1 -= w * tn1; break;
      default: im0 -= s * w * tn0; im1 -= s * w * tn1; break;
    }
  }
  re0 *= norm; re1 *= norm; im0 *= norm; im1 *= norm;
  c_lo = make_double2(pc * re0 - ps * im0, pc * im0 + ps * re0);
  c_hi = make_double2(pc * re1 - ps * im1, pc * im1 + ps * re1);
}

// Per-CTA partial of ||v||^2 with the chunking of the orthogonalisation kernels.
__global__ void __launch_bounds__(VT) lz_norm_kernel(const c128 *v, long long n, int chunk, double *npartial) {
  const long long e0 = (long long)blockIdx.x * chunk;
  const int len = (int)((e0 + chunk <= n) ? chunk : (n > e0 ? n - e0 : 0));
  double s = 0.0;
  for (int e = threadIdx.x; e < len; e += VT) { const c128 x = __ldcg(v + e0 + e); s += x.x * x.x + x.y * x.y; }
  __shared__ double red[VT / 32];
  s = warp_sum(s);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) { double t = 0; for (int i = 0; i < VT / 32; i++) t += red[i]; npartial[blockIdx.x] = t; }
}

// Grid barrier on a counter of its own (zeroed by the host before the exponential starts): one atomic
// add per CTA, released when the count reaches the grid size.  The launch is cooperative, so all CTAs
// are resident.
__device__ __forceinline__ void lz_grid_bar(unsigned *ctr) {
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    atomicAdd(ctr, 1u);
    unsigned v;
    do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(ctr) : "memory"); } while (v < gridDim.x);
  }
  __syncthreads();
}

// dots of the nd vectors q_i (chunk pointers via qptr) with w over `len` elements -> partial[blockIdx][i].
// All eight warps work whatever nd is: vector i is cut into nseg segments, the segment sums are added
// in a fixed order (deterministic).
template <class QP>
__device__ __forceinline__ void chunk_dots(const c128 *w, QP qptr, int len, int nd, c128 *partial, c128 *seg /*[8] shared*/) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  constexpr int NW = VT / 32;
  const int nseg = nd >= NW ? 1 : NW / nd;
  for (int i0 = 0; i0 < nd; i0 += NW / nseg) {
    const int i = i0 + warp / nseg, sg = warp % nseg;
    double sx = 0.0, sy = 0.0;
    if (i < nd) {
      const c128 *q = qptr(i);
      const int per = (len + nseg - 1) / nseg;
      const int b0 = sg * per, b1 = (b0 + per) < len ? (b0 + per) : len;
      for (int e = b0 + lane; e < b1; e += 32) {
        const c128 a = q[e], x = w[e];
        sx = fma(a.x, x.x, fma(a.y, x.y, sx));
        sy = fma(a.x, x.y, fma(-a.y, x.x, sy));
      }
      sx = warp_sum(sx); sy = warp_sum(sy);
    }
    if (nseg > 1) {
      if (lane == 0) seg[warp] = make_double2(sx, sy);
      __syncthreads();
      if (i < nd && sg == 0 && lane == 0) {
        double tx = 0.0, ty = 0.0;
        for (int q2 = 0; q2 < nseg; q2++) { tx += seg[warp + q2].x; ty += seg[warp + q2].y; }
        partial[(size_t)blockIdx.x * nd + i] = make_double2(tx, ty);
      }
      __syncthreads();
    } else if (i < nd && lane == 0) {
      partial[(size_t)blockIdx.x * nd + i] = make_double2(sx, sy);
    }
  }
}
// every CTA: cs[i] = sum_g partial[g][i], fixed order
__device__ __forceinline__ void gather_dots(const c128 *partial, int nd, c128 *cs) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int i = warp; i < nd; i += VT / 32) {
    double sx = 0.0, sy = 0.0;
    for (int g = lane; g < (int)gridDim.x; g += 32) { const c128 pz = __ldcg(partial + (size_t)g * nd + i); sx += pz.x; sy += pz.y; }
    sx = warp_sum(sx); sy = warp_sum(sy);
    if (lane == 0) cs[i] = make_double2(sx, sy);
  }
  __syncthreads();
}

// One Lanczos iteration after the apply w_raw = H u_j (slot j + 1 of Q; u_j in slot j):
//   beta_{j-1} = ||u_j|| from the partial norms of the previous kernel; stop decisions; q_j = u_j / beta;
//   w = w_raw / beta; two Gram-Schmidt passes against q_0..q_j (alpha_j = Re<q_j, w> from the first);
//   u_{j+1} = w to slot j + 1, partial norms of it for the next kernel.
// qs / wsm: keep the chunk of q_0..q_j / of w in shared memory (else they stay in global memory / L2).
__global__ void __launch_bounds__(VT) lz_orth_kernel(long long n, int chunk, int j, int k, double zeta, double tol, int qs, int wsm,
                                                     const c128 *u_src /*u_j: v itself for j = 0, else slot j*/, LzBuffers b) {
  extern __shared__ __align__(16) unsigned char fsm[];
  __shared__ c128 cs[TDVP_MAX_KRYLOV + 1];
  __shared__ c128 seg[VT / 32];
  __shared__ double red[VT / 32];
  __shared__ double s_inv;
  __shared__ int s_done;
  __shared__ double jn[CHEB_MAX + 64];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nd = j + 1;
  const long long e0 = (long long)blockIdx.x * chunk;
  const int len = (int)((e0 + chunk <= n) ? chunk : (n > e0 ? n - e0 : 0));
  c128 *ug = b.Q + (long long)j * n + e0;                 // q_j goes here
  const c128 *us = u_src + e0;                            // u_j comes from here
  c128 *wg = b.Q + (long long)(j + 1) * n + e0;           // w_raw -> u_{j+1}
  c128 *sw = wsm ? reinterpret_cast<c128 *>(fsm) : wg;
  c128 *sq = reinterpret_cast<c128 *>(fsm) + (wsm ? chunk : 0);          // [j + 1][chunk] if qs
  // loads that do not depend on the decision go first (16 B asynchronous copies)
  if (wsm)
    for (int e = tid; e < len; e += VT) {
      const unsigned sa = (unsigned)__cvta_generic_to_shared(sw + e);
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sa), "l"(wg + e));
    }
  if (qs)
    for (int i = 0; i < nd; i++) {
      const c128 *qg = i == j ? us : b.Q + (long long)i * n + e0;
      for (int e = tid; e < len; e += VT) {
        const unsigned sa = (unsigned)__cvta_generic_to_shared(sq + (size_t)i * chunk + e);
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sa), "l"(qg + e));
      }
    }
  asm volatile("cp.async.commit_group;\n" ::: "memory");
  // ---- beta_{j-1} and the stop decision: every CTA, same data, same order ----
  if (warp == 0) {
    double t = 0.0;
    for (int g = lane; g < (int)gridDim.x; g += 32) t += __ldcg(b.npartial + g);
    t = warp_sum(t);
    const double beta = sqrt(t);
    const int prior = j > 0 ? __ldcg(b.hist + j - 1) : 0;
    int done = prior;
    if (!prior) {
      if (j == 0) {
        done = !(beta > 0.0);
      } else {
        const double aj = fabs(__ldcg(b.alpha + j - 1));
        if (beta < BREAKDOWN_TOL * (aj > 1.0 ? aj : 1.0)) done = 1;
        else if (tol > 0.0) {
          // adaptive rule: T_j = tridiag(alpha_0..alpha_{j-1}; beta_0..beta_{j-2}), c = exp(i zeta T_j) e_1
          c128 clo, chi;
          int range = 0;
          cheb_expm_e1(j, b.alpha, b.beta, zeta, jn, clo, chi, &range);
          const int il = j - 1;
          const c128 mine = il < 32 ? clo : chi;
          const double cx = __shfl_sync(0xffffffffu, mine.x, il & 31), cy = __shfl_sync(0xffffffffu, mine.y, il & 31);
          if (beta * sqrt(cx * cx + cy * cy) < tol) done = 1;
          if (range && blockIdx.x == 0 && lane == 0 && b.status) atomicOr(b.status, TDVP_STATUS_KRYLOV_RANGE);
        }
      }
    }
    if (lane == 0) {
      s_done = done;
      s_inv = done ? 0.0 : 1.0 / beta;
      if (blockIdx.x == 0) {
        b.hist[j] = done;
        if (j == 0) b.state->beta0 = beta;
        if (!prior && done) b.state->m = j;
        if (!prior && !done && j > 0) b.beta[j - 1] = beta;
      }
    }
  }
  __syncthreads();
  if (s_done) { asm volatile("cp.async.wait_group 0;\n" ::: "memory"); return; }   // all CTAs take this branch together
  const double inv = s_inv;
  asm volatile("cp.async.wait_group 0;\n" ::: "memory");
  __syncthreads();
  // ---- normalise: q_j = u_j / beta (in place, global and shared copy), w = w_raw / beta ----
  c128 *sqj = qs ? sq + (size_t)j * chunk : ug;
  for (int e = tid; e < len; e += VT) {
    const c128 u = qs ? sqj[e] : __ldcg(us + e);
    const c128 qn = make_double2(u.x * inv, u.y * inv);
    ug[e] = qn;
    if (qs) sqj[e] = qn;
    const c128 x = wsm ? sw[e] : __ldcg(wg + e);
    sw[e] = make_double2(x.x * inv, x.y * inv);
  }
  __syncthreads();
  auto qptr = [&](int i) -> const c128 * { return qs ? sq + (size_t)i * chunk : b.Q + (long long)i * n + e0; };
  if (j == k - 1) {
    // last iteration: only alpha_j = Re<q_j, w> is needed (the recurrence stops before q_{k+1} is formed,
    // PAPER.md:292-296 / oracle O3): one reduction, one grid barrier, no orthogonalisation
    const c128 *q = qptr(j);
    double s = 0.0;
    for (int e = tid; e < len; e += VT) { const c128 a = q[e], x = sw[e]; s = fma(a.x, x.x, fma(a.y, x.y, s)); }
    s = warp_sum(s);
    if (lane == 0) red[warp] = s;
    __syncthreads();
    // (not into npartial: slower CTAs may still be summing the norms there)
    if (tid == 0) { double t = 0; for (int i = 0; i < VT / 32; i++) t += red[i]; b.partial[blockIdx.x] = make_double2(t, 0.0); }
    lz_grid_bar(b.bar + 2 * j);
    if (blockIdx.x == 0 && warp == 0) {
      double t = 0.0;
      for (int g = lane; g < (int)gridDim.x; g += 32) t += __ldcg(b.partial + g).x;
      t = warp_sum(t);
      if (lane == 0) { b.alpha[j] = t; b.state->m = k; }
    }
    return;
  }
  for (int pass = 0; pass < 2; pass++) {
    c128 *partial = b.partial + (size_t)pass * MAXG * (TDVP_MAX_KRYLOV + 1);
    chunk_dots(sw, qptr, len, nd, partial, seg);
    lz_grid_bar(b.bar + 2 * j + pass);
    gather_dots(partial, nd, cs);
    if (pass == 0 && blockIdx.x == 0 && tid == 0) b.alpha[j] = cs[j].x;
    for (int e = tid; e < len; e += VT) {
      c128 x = sw[e];
      for (int i = 0; i < nd; i++) {
        const c128 q = qptr(i)[e], c = cs[i];
        x.x -= c.x * q.x - c.y * q.y;
        x.y -= c.x * q.y + c.y * q.x;
      }
      sw[e] = x;
    }
    __syncthreads();
  }
  double s = 0.0;
  for (int e = tid; e < len; e += VT) {
    const c128 x = sw[e];
    s += x.x * x.x + x.y * x.y;
    if (wsm) wg[e] = x;                                   // u_{j+1}, normalised by the next kernel
  }
  s = warp_sum(s);
  if (lane == 0) red[warp] = s;
  __syncthreads();
  if (tid == 0) { double t = 0; for (int i = 0; i < VT / 32; i++) t += red[i]; b.npartial[blockIdx.x] = t; }
}

// One warp: coef = beta0 * V exp(z Lambda) V^T e_1 for the m x m tridiagonal (alpha, beta), for z with a
// real part ("diagonalize the tridiagonal matrix in the subspace").  Implicit symmetric QR
// iteration with Wilkinson shift and deflation (Golub & Van Loan, "Matrix Computations", sec. 8.3).
// The scalar recurrence of a sweep is a dependent FP64 chain: lane 0 alone runs it on shared-memory
// copies of the diagonals and records the sweep's rotations; then every lane applies them to the
// eigenvector rows it owns.
__global__ void __launch_bounds__(32) lz_coef_kernel(int k, double zr, double zi, LzBuffers b) {
  __shared__ double V[TDVP_MAX_KRYLOV * TDVP_MAX_KRYLOV];
  __shared__ double a[TDVP_MAX_KRYLOV], off[TDVP_MAX_KRYLOV], rc[TDVP_MAX_KRYLOV], rs[TDVP_MAX_KRYLOV];
  __shared__ int s_lo, s_hi;
  const int lane = threadIdx.x;
  const int m = b.state->m;
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

// y = sum_{j<m} coef[j] q_j with coef = beta0 exp(i zeta T) e_1 evaluated here by warp 0 of every CTA
// (have_coef = 0), or read from b.coef (have_coef = 1: the eigen-decomposition kernel ran).
__global__ void __launch_bounds__(VT) lz_combine_kernel(long long n, int k, double zeta, int have_coef, LzBuffers b, c128 *y, int *m_out) {
  __shared__ c128 cs[TDVP_MAX_KRYLOV];
  __shared__ double jn[CHEB_MAX + 64];
  const int m = b.state->m;
  if (blockIdx.x == 0 && threadIdx.x == 0 && m_out) *m_out = m;
  if (have_coef) {
    for (int i = threadIdx.x; i < m; i += VT) cs[i] = b.coef[i];
  } else if (threadIdx.x < 32 && m > 0) {
    c128 clo, chi;
    int range = 0;
    cheb_expm_e1(m, b.alpha, b.beta, zeta, jn, clo, chi, &range);
    const double beta0 = b.state->beta0;
    const int lane = threadIdx.x;
    if (lane < m) cs[lane] = make_double2(beta0 * clo.x, beta0 * clo.y);
    if (lane + 32 < m) cs[lane + 32] = make_double2(beta0 * chi.x, beta0 * chi.y);
    if (range && blockIdx.x == 0 && lane == 0 && b.status) atomicOr(b.status, TDVP_STATUS_KRYLOV_RANGE);
  }
  __syncthreads();
  for (long long e = blockIdx.x * (long long)VT + threadIdx.x; e < n; e += (long long)gridDim.x * VT) {
    double sx = 0.0, sy = 0.0;
    for (int i = 0; i < m; i++) {
      const c128 q = b.Q[(long long)i * n + e], c = cs[i];
      sx += c.x * q.x - c.y * q.y;
      sy += c.x * q.y + c.y * q.x;
    }
    y[e] = make_double2(sx, sy);
  }
}

inline size_t up256(size_t x) { return (x + 255) & ~size_t(255); }

size_t apply_ws_bytes(const LanczosOp &op) {
  if (op.kind == 2) return heff2_ws_bytes(op.Ml, op.Mr, op.d, op.d2, op.Dl, op.Dm, op.Dr);
  return op.kind == 0 ? heff_ws_bytes(op.Ml, op.Mr, op.d, op.Dl, op.Dr) : bond_ws_bytes(op.Ml, op.Mr, op.Dl);
}

constexpr size_t ORTH_SMEM_MAX = 196 * 1024;   // dynamic part; ~20 KB of static arrays beside it
int g_num_sms = 0;
int g_orth_per_sm = 1;

}  // namespace

void lanczos_configure() {
  cudaFuncSetAttribute(lz_orth_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ORTH_SMEM_MAX);
  int dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&g_num_sms, cudaDevAttrMultiProcessorCount, dev);
  if (g_num_sms < 1) g_num_sms = 1;
}

size_t lanczos_ws_bytes(const LanczosOp &op, int k) {
  size_t n = (size_t)op.elems();
  return up256((k + 1) * n * 16) + up256(k * 16) + 2 * up256(k * 8) + 1024 +
         up256((size_t)2 * MAXG * (TDVP_MAX_KRYLOV + 1) * 16) + up256(MAXG * 8) + apply_ws_bytes(op) + 512;
}

void lanczos_expm(cudaStream_t st, const LanczosOp &op, int k, double tol, double z_re, double z_im,
                  const c128 *v, c128 *y, void *ws, int *m_used_dev, int *status_dev) {
  const long long n = op.elems();
  char *p = reinterpret_cast<char *>(up256(reinterpret_cast<size_t>(ws)));
  LzBuffers b;
  b.Q = reinterpret_cast<c128 *>(p); p += up256((k + 1) * n * 16);
  b.coef = reinterpret_cast<c128 *>(p); p += up256(k * 16);
  b.alpha = reinterpret_cast<double *>(p); p += up256(k * 8);
  b.beta = reinterpret_cast<double *>(p); p += up256(k * 8);
  // one block zeroed per exponential: state, hist[k + 1], barrier counters [2 k + 2]   (<= 16 + 260 + 520 bytes)
  char *zero0 = p;
  b.state = reinterpret_cast<LzState *>(p); p += 16;
  b.hist = reinterpret_cast<int *>(p); p += 4 * (TDVP_MAX_KRYLOV + 2);
  b.bar = reinterpret_cast<unsigned *>(p); p += 4 * (2 * TDVP_MAX_KRYLOV + 2);
  p = zero0 + 1024;
  b.partial = reinterpret_cast<c128 *>(p); p += up256((size_t)2 * MAXG * (TDVP_MAX_KRYLOV + 1) * 16);
  b.npartial = reinterpret_cast<double *>(p); p += up256(MAXG * 8);
  b.status = status_dev;
  b.apply_ws = p;

  // one CTA per SM at most; the chunk of w -- and of all k + 1 vectors if they fit -- in shared memory
  int FG = (int)((n + VT - 1) / VT);
  if (FG > g_num_sms) FG = g_num_sms;
  if (FG < 1) FG = 1;
  const int chunk = (int)((n + FG - 1) / FG);
  const int wsm = (size_t)chunk * 16 <= ORTH_SMEM_MAX ? 1 : 0;
  const int qs = (size_t)(k + 1) * chunk * 16 <= ORTH_SMEM_MAX ? 1 : 0;
  const bool imaginary = (z_re == 0.0);
  {
    ProfScope ps(st, PH_VEC);
    cudaMemsetAsync(zero0, 0, 1024, st);
    TDVP_LAUNCH(lz_norm_kernel, FG, VT, 0, st, v, n, chunk, b.npartial);
  }
  for (int j = 0; j < k; j++) {
    const c128 *uj = j == 0 ? v : b.Q + (long long)j * n;    // u_0 = v is read in place
    c128 *w = b.Q + (long long)(j + 1) * n;
    // adaptive mode: once the recurrence has stopped the remaining applies return at once.  (Fixed k: no flag --
    // a stop before k is the rare breakdown at a chain end, and the flag-free GEMM instance is 5 % faster; the
    // applies then run on stale vectors nobody reads.)
    const int *skip = (j > 0 && tol > 0.0 && imaginary) ? b.hist + (j - 1) : nullptr;
    if (op.kind == 0)
      heff_apply(st, op.Ml, op.Mr, op.d, op.Dl, op.Dr, op.L, *op.W, uj, op.R, w, b.apply_ws, nullptr, skip);
    else if (op.kind == 2)
      heff2_apply(st, op.Ml, op.Mr, op.d, op.d2, op.Dl, op.Dm, op.Dr, op.L, *op.W, *op.W2, uj, op.R, w, b.apply_ws, skip);
    else
      bond_apply(st, op.Ml, op.Mr, op.Dl, op.L, uj, op.R, w, b.apply_ws, skip);
    ProfScope ps(st, PH_VEC);
    long long nn = n; int ch = chunk, jj = j, kk = k, qq = qs, ww = wsm;
    double zz = z_im, tt = imaginary ? tol : 0.0;
    void *args[] = {&nn, &ch, &jj, &kk, &zz, &tt, &qq, &ww, &uj, &b};
    const size_t smem = ((size_t)(wsm ? chunk : 0) + (qs ? (size_t)(j + 1) * chunk : 0)) * 16;
    cudaLaunchCooperativeKernel((void *)lz_orth_kernel, dim3(FG), dim3(VT), args, smem, st);
    count_launch();
  }
  ProfScope ps(st, PH_VEC);
  if (!imaginary) TDVP_LAUNCH(lz_coef_kernel, 1, 32, 0, st, k, z_re, z_im, b);
  int G = (int)((n + VT - 1) / VT);
  if (G > MAXG) G = MAXG;
  if (G < 1) G = 1;
  TDVP_LAUNCH(lz_combine_kernel, G, VT, 0, st, n, k, z_im, imaginary ? 0 : 1, b, y, m_used_dev);
}
