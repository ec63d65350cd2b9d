// svd.cu -- matrix unfolding of a bond (Eq. 36): C[Ml, d, Mr] viewed as
// Ml x (d*Mr) = U diag(lam) Vh, on the device (the paper runs its SVDs on one CPU
// core and names them "prominent" in the GPU run).
//
//   1. RQ of C (qr.cu, side 1):            C = D Q,      D n x n (n = Ml), Q row-orthonormal
//   2. one-sided (Hestenes) Jacobi on D:   D J = X,      columns of X mutually orthogonal, J unitary
//      -- high relative accuracy for the small singular values that Eq. 38 regularises
//   3. Householder QR of X (qr.cu):        X = U' R',    R' diagonal up to round-off, U' EXACTLY unitary
//      even when C is rank deficient (columns of X with norm ~ 0)
//   4. lam = |diag R'| sorted descending, U = U' sgn(R') permuted, Vh = (J permuted)^H Q  (DMMA GEMM)
//
// The Jacobi sweeps run in one thread-block cluster (8 CTAs, a column pair per warp and round,
// round-robin ordering, cluster barrier between rounds; X and J live in L2): no host round trip,
// deterministic, capturable in the step graph.
#include <cooperative_groups.h>

#include <cstdlib>

#include "common.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int MAX_SWEEPS = 40;
// A sweep that still rotates only pairs whose cosine is below this is "hovering at round-off" (the threshold
// sqrt(n) eps sits at the error level of the dot product itself), not a failure to converge.
constexpr double COARSE_TOL2 = 1e-20;
// A column whose squared norm is below this (norm below 1e-75: products of round-off residues along a chain of
// rank-deficient bonds get there) is zero for every purpose of the path.  The product a * b of the convergence
// test underflows for two such columns, the test then always fires and the pair would be rotated for ever.
constexpr double TINY_COL2 = 1e-150;
// ... and RELATIVE to the matrix: a column more than three orders of magnitude below the round-off floor of the
// largest column (norm < 1e-3 eps max_c |x_c|) is noise of noise.  Orthogonalising two such columns against
// each other leaves one of them smaller still, with a direction that is round-off again: a cascade down to the
// underflow threshold that used up all 40 sweeps on the graded bonds of a P&C-RK4 stage (singular values 6.6,
// 1e-3 ..., a degenerate cluster at 6.6e-16, columns at 5e-34).  Pairs with such a column are left alone: the
// reconstruction U Lambda V^dagger changes by less than those norms, J stays unitary by construction, and the
// Householder step that follows makes U exactly unitary whatever the tiny columns look like.
constexpr double REL_TINY2 = 4.9e-38;     // (1e-3 * 2.2e-16)^2

inline size_t up256(size_t x) { return (x + 255) & ~size_t(255); }

__device__ __forceinline__ double wsum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// max_c |x_c|^2 over the columns of the n x n column-major Xt, identically in every CTA (fixed order)
template <int NWARPS>
__device__ double max_col_norm2(const c128 *Xt, int n, double *sm /*[NWARPS]*/) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double m = 0.0;
  for (int c = warp; c < n; c += NWARPS) {
    double a = 0.0;
    for (int i = lane; i < n; i += 32) { const c128 u = __ldcg(Xt + (size_t)c * n + i); a += u.x * u.x + u.y * u.y; }
    a = wsum(a);
    m = fmax(m, a);
  }
  if (lane == 0) sm[warp] = m;
  __syncthreads();
  double r = 0.0;
  for (int k = 0; k < NWARPS; k++) r = fmax(r, sm[k]);
  __syncthreads();
  return r;
}

// Xt[c][r] = D[r][c];  Jt[c][r] = delta(c, r)          (column-major copies: contiguous columns)
__global__ void svd_init_kernel(const c128 *D, c128 *Xt, c128 *Jt, int n) {
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n * n; e += gridDim.x * blockDim.x) {
    int c = e / n, r = e % n;
    Xt[e] = D[(long long)r * n + c];
    Jt[e] = make_double2(r == c ? 1.0 : 0.0, 0.0);
  }
}

// One-sided Jacobi: rotate column pairs of X (and J) until all columns are mutually orthogonal.
// The n/2 pairs of a round are independent; the scalar FP64 work per pair (three square roots, three
// divisions) is what a single SM cannot issue fast enough, so the round is spread over a thread-block
// CLUSTER of 8 CTAs (8 SMs, one pair per warp and round at n = 128) with a hardware cluster barrier
// between rounds.  X and J live in L2: loads bypass L1 (ld.global.cg), the barrier's release /
// acquire orders the stores of one round before the loads of the next.
// NPL = rows per lane held in registers (n <= 32 * NPL); NPL = 0 is the generic looped variant.
constexpr int JC = 8;               // CTAs per cluster
constexpr int JW = 8;               // warps per CTA
// flags[] of one unfolding (ints, zeroed): [0, 40) a sweep rotated, [64, 104) ... a pair far from orthogonal, and
constexpr int FLAG_FORCE_QR = 120;  // the Jacobi kernel ran out of sweeps
constexpr int FLAG_NEED_QR = 121;   // decided by svd_sortcols_kernel: the Householder step has to make U unitary

template <int NPL>
__global__ void __cluster_dims__(JC, 1, 1) __launch_bounds__(JW * 32)
svd_jacobi_kernel(c128 *Xt, c128 *Jt, int n, int *flags /*[MAX_SWEEPS] zeroed*/, int max_sweeps, int *status) {
  cg::cluster_group cluster = cg::this_cluster();
  const int lane = threadIdx.x & 31;
  const int gwarp = blockIdx.x * JW + (threadIdx.x >> 5), nwarps = JC * JW;
  const int np = (n + 1) & ~1;             // players of the round-robin tournament (a bye if n is odd)
  const int npairs = np / 2;
  const double tol = 2.220446049250313e-16 * sqrt((double)n);   // LAPACK zgesvj: sqrt(m) * eps
  const double tol2 = tol * tol;
  __shared__ double s_cmax[JW];
  const double thr = fmax(TINY_COL2, REL_TINY2 * max_col_norm2<JW>(Xt, n, s_cmax));
  cluster.sync();                                       // everybody has read the initial columns
  int sweep = 0;
  for (; sweep < max_sweeps; sweep++) {
    bool any = false, coarse = false;
    for (int round = 0; round < np - 1; round++) {
      for (int k = gwarp; k < npairs; k += nwarps) {
        int p, q;
        if (k == 0) { p = round; q = np - 1; }
        else { p = (round + k) % (np - 1); q = (round - k + (np - 1)) % (np - 1); }
        if (p > q) { int t = p; p = q; q = t; }
        if (q >= n) continue;                                    // the bye
        c128 *xp = Xt + (long long)p * n, *xq = Xt + (long long)q * n;
        c128 *jp = Jt + (long long)p * n, *jq = Jt + (long long)q * n;
        constexpr int NR = NPL > 0 ? NPL : 1;
        c128 xu[NR], xv[NR], ju[NR], jv[NR];
        double a = 0.0, b = 0.0, cr = 0.0, ci = 0.0;
        if (NPL > 0) {
#pragma unroll
          for (int r = 0; r < NR; r++) {
            const int i = lane + 32 * r;
            const bool ok = i < n;
            xu[r] = ok ? __ldcg(xp + i) : make_double2(0.0, 0.0);
            xv[r] = ok ? __ldcg(xq + i) : make_double2(0.0, 0.0);
            ju[r] = ok ? __ldcg(jp + i) : make_double2(0.0, 0.0);
            jv[r] = ok ? __ldcg(jq + i) : make_double2(0.0, 0.0);
          }
#pragma unroll
          for (int r = 0; r < NR; r++) {
            const c128 u = xu[r], v = xv[r];
            a += u.x * u.x + u.y * u.y;
            b += v.x * v.x + v.y * v.y;
            cr += u.x * v.x + u.y * v.y;                         // conj(u) * v
            ci += u.x * v.y - u.y * v.x;
          }
        } else {
          for (int i = lane; i < n; i += 32) {
            c128 u = __ldcg(xp + i), v = __ldcg(xq + i);
            a += u.x * u.x + u.y * u.y;
            b += v.x * v.x + v.y * v.y;
            cr += u.x * v.x + u.y * v.y;
            ci += u.x * v.y - u.y * v.x;
          }
        }
        a = wsum(a); b = wsum(b); cr = wsum(cr); ci = wsum(ci);
        const double c2 = cr * cr + ci * ci;
        if (!(c2 > tol2 * a * b) || c2 == 0.0 || a < thr || b < thr) continue;
        any = true;
        if (c2 > COARSE_TOL2 * a * b) coarse = true;
        // y_q = e^{-i phi} x_q makes <x_p, y_q> = |c| real; then a real rotation (cs, sn)
        const double cabs = sqrt(c2), icabs = 1.0 / cabs;
        const double er = cr * icabs, ei = -ci * icabs;          // e^{-i phi}
        const double zeta = 0.5 * (b - a) * icabs;
        const double t = (zeta >= 0.0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
        const double cs = 1.0 / sqrt(1.0 + t * t), sn = cs * t;
        auto rot = [&](c128 u, c128 v, c128 &o1, c128 &o2) {
          const c128 y = make_double2(er * v.x - ei * v.y, er * v.y + ei * v.x);
          o1 = make_double2(cs * u.x - sn * y.x, cs * u.y - sn * y.y);
          o2 = make_double2(sn * u.x + cs * y.x, sn * u.y + cs * y.y);
        };
        if (NPL > 0) {
#pragma unroll
          for (int r = 0; r < NR; r++) {
            const int i = lane + 32 * r;
            if (i < n) {
              c128 o1, o2;
              rot(xu[r], xv[r], o1, o2); xp[i] = o1; xq[i] = o2;
              rot(ju[r], jv[r], o1, o2); jp[i] = o1; jq[i] = o2;
            }
          }
        } else {
          for (int i = lane; i < n; i += 32) {
            c128 o1, o2;
            rot(__ldcg(xp + i), __ldcg(xq + i), o1, o2); xp[i] = o1; xq[i] = o2;
            rot(__ldcg(jp + i), __ldcg(jq + i), o1, o2); jp[i] = o1; jq[i] = o2;
          }
        }
      }
      if (round == np - 2 && any && lane == 0) flags[sweep] = 1;   // benign race: every writer stores 1
      if (round == np - 2 && coarse && lane == 0) flags[64 + sweep] = 1;
      cluster.sync();
    }
    if (np < 2) break;
    if (__ldcg(flags + sweep) == 0) break;                          // nobody rotated in this sweep
    // ... or every pair it met was orthogonal to 1e-10 already (no "coarse" pair): a rotation by an angle <= 1e-10
    // disturbs the other products of its two columns by <= 1e-10 * 1e-10 each, so after this sweep every cosine is
    // below ~2 n 1e-20 << sqrt(n) eps and the next sweep would only confirm it (a sweep is ~0.2 ms at n = 128)
    if (__ldcg(flags + 64 + sweep) == 0) break;
  }
  // every sweep allowed still rotated, and the last one still saw a pair far from orthogonal (rotations that
  // hover at the round-off threshold of sqrt(n) eps are convergence): tell the host
  if (sweep == max_sweeps && np >= 2 && gwarp == 0 && lane == 0) {
    flags[FLAG_FORCE_QR] = 1;                           // columns may still be far from orthogonal: U comes from the Householder step
    if (status && __ldcg(flags + 64 + max_sweeps - 1)) atomicOr(status, TDVP_STATUS_SVD_UNCONVERGED);
  }
}

// Block variant for n <= 128: the same rotations, but the cluster barrier is paid once per BLOCK pair
// instead of once per column pair.  Columns are grouped into 16 blocks of bw = ceil(n / 16); a sweep
// is (i) all pairs inside a block (CTA c takes blocks 2c, 2c + 1) and (ii) a round-robin tournament
// of the 16 blocks, 15 outer rounds of 8 block pairs, one per CTA: the CTA copies its two blocks of X
// and J into shared memory, orthogonalises every column of one against every column of the other in
// bw inner rounds (one pair per warp, __syncthreads between), and writes them back.  127 cluster
// barriers per sweep become 16.  Same pair set per sweep, fixed order: deterministic.
constexpr int JB = 16;              // column blocks

template <int NPL>
__device__ __forceinline__ int jacobi_pair_smem(c128 *xp, c128 *xq, c128 *jp, c128 *jq, int n, int lane, double tol2, double thr) {
  c128 xu[NPL], xv[NPL], ju[NPL], jv[NPL];
  double a = 0.0, b = 0.0, cr = 0.0, ci = 0.0;
#pragma unroll
  for (int r = 0; r < NPL; r++) {
    const int i = lane + 32 * r;
    const bool ok = i < n;
    xu[r] = ok ? xp[i] : make_double2(0.0, 0.0);
    xv[r] = ok ? xq[i] : make_double2(0.0, 0.0);
    ju[r] = ok ? jp[i] : make_double2(0.0, 0.0);
    jv[r] = ok ? jq[i] : make_double2(0.0, 0.0);
    const c128 u = xu[r], v = xv[r];
    a += u.x * u.x + u.y * u.y;
    b += v.x * v.x + v.y * v.y;
    cr += u.x * v.x + u.y * v.y;                                 // conj(u) * v
    ci += u.x * v.y - u.y * v.x;
  }
  a = wsum(a); b = wsum(b); cr = wsum(cr); ci = wsum(ci);
  const double c2 = cr * cr + ci * ci;
  if (!(c2 > tol2 * a * b) || c2 == 0.0 || a < thr || b < thr) return 0;
  const int result = c2 > COARSE_TOL2 * a * b ? 3 : 1;
  // the scalar chain is the critical path of a round: reciprocal square roots instead of sqrt + divide
  const double icabs = rsqrt(c2);
  const double er = cr * icabs, ei = -ci * icabs;                // e^{-i phi}
  const double zeta = 0.5 * (b - a) * icabs;
  const double t = (zeta >= 0.0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
  const double cs = rsqrt(1.0 + t * t), sn = cs * t;
  auto rot = [&](c128 u, c128 v, c128 &o1, c128 &o2) {
    const c128 y = make_double2(er * v.x - ei * v.y, er * v.y + ei * v.x);
    o1 = make_double2(cs * u.x - sn * y.x, cs * u.y - sn * y.y);
    o2 = make_double2(sn * u.x + cs * y.x, sn * u.y + cs * y.y);
  };
#pragma unroll
  for (int r = 0; r < NPL; r++) {
    const int i = lane + 32 * r;
    if (i < n) {
      c128 o1, o2;
      rot(xu[r], xv[r], o1, o2); xp[i] = o1; xq[i] = o2;
      rot(ju[r], jv[r], o1, o2); jp[i] = o1; jq[i] = o2;
    }
  }
  return result;
}

// The same rotation with the first column of the pair (X and J) held in REGISTERS by the warp across the inner
// rounds of a block pair -- a warp keeps its column of the first block and meets a different column of the second
// block every round -- so that a round moves one column through shared memory, not two: the inner rounds of a
// block pair are bound by shared-memory traffic (8 warps x 8 KB each way per round).
template <int NPL>
__device__ __forceinline__ int jacobi_pair_preg(c128 (&xu)[NPL], c128 (&ju)[NPL], c128 *xq, c128 *jq, int n, int lane, double tol2, double thr) {
  c128 xv[NPL], jv[NPL];
  double a = 0.0, b = 0.0, cr = 0.0, ci = 0.0;
#pragma unroll
  for (int r = 0; r < NPL; r++) {
    const int i = lane + 32 * r;
    const bool ok = i < n;
    xv[r] = ok ? xq[i] : make_double2(0.0, 0.0);
    const c128 u = xu[r], v = xv[r];
    a += u.x * u.x + u.y * u.y;
    b += v.x * v.x + v.y * v.y;
    cr += u.x * v.x + u.y * v.y;                                 // conj(u) * v
    ci += u.x * v.y - u.y * v.x;
  }
  a = wsum(a); b = wsum(b); cr = wsum(cr); ci = wsum(ci);
  const double c2 = cr * cr + ci * ci;
  if (!(c2 > tol2 * a * b) || c2 == 0.0 || a < thr || b < thr) return 0;
  const int result = c2 > COARSE_TOL2 * a * b ? 3 : 1;
#pragma unroll
  for (int r = 0; r < NPL; r++) { const int i = lane + 32 * r; jv[r] = i < n ? jq[i] : make_double2(0.0, 0.0); }
  const double icabs = rsqrt(c2);
  const double er = cr * icabs, ei = -ci * icabs;                // e^{-i phi}
  const double zeta = 0.5 * (b - a) * icabs;
  const double t = (zeta >= 0.0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
  const double cs = rsqrt(1.0 + t * t), sn = cs * t;
  auto rot = [&](c128 u, c128 v, c128 &o1, c128 &o2) {
    const c128 y = make_double2(er * v.x - ei * v.y, er * v.y + ei * v.x);
    o1 = make_double2(cs * u.x - sn * y.x, cs * u.y - sn * y.y);
    o2 = make_double2(sn * u.x + cs * y.x, sn * u.y + cs * y.y);
  };
#pragma unroll
  for (int r = 0; r < NPL; r++) {
    const int i = lane + 32 * r;
    c128 o1, o2;
    rot(xu[r], xv[r], o1, o2); xu[r] = o1; if (i < n) xq[i] = o2;
    rot(ju[r], jv[r], o1, o2); ju[r] = o1; if (i < n) jq[i] = o2;
  }
  return result;
}

// Geometry: JB_ column blocks, JC_ = JB_ / 2 CTAs (one block pair each), JW_ warps per CTA (>= columns per block).
// (16, 8, 8) is what runs.  (8, 4, 16) -- 8 phases of 16 inner rounds per sweep instead of 16 of 8, half the block
// exchanges and cluster barriers -- measured SLOWER (3.04 against 2.42 ms per 128 x 128 bond): a sweep's time is in its
// 127 inner rounds, which are bound by shared-memory traffic, and 16 warps per CTA double that traffic per round.
template <int NPL, int JB_, int JC_, int JW_>
__global__ void __cluster_dims__(JC_, 1, 1) __launch_bounds__(JW_ * 32)
svd_jacobi_block_kernel(c128 *Xt, c128 *Jt, int n, int *flags /*[MAX_SWEEPS] zeroed*/, int max_sweeps, int *status) {
  cg::cluster_group cluster = cg::this_cluster();
  extern __shared__ __align__(16) unsigned char jsm[];
  const int bw = (n + JB_ - 1) / JB_;                     // columns per block (<= JW_)
  c128 *Xs = reinterpret_cast<c128 *>(jsm);               // [2 bw][n]
  c128 *Js = Xs + (size_t)2 * bw * n;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int cta = blockIdx.x;                             // one cluster: rank == blockIdx.x
  const double tol = 2.220446049250313e-16 * sqrt((double)n);
  const double tol2 = tol * tol;
  __shared__ double s_cmax[JW_];
  const double thr = fmax(TINY_COL2, REL_TINY2 * max_col_norm2<JW_>(Xt, n, s_cmax));
  cluster.sync();                                       // everybody has read the initial columns
  auto load_blocks = [&](int bp, int bq) {
    for (int e = tid; e < 2 * bw * n; e += JW_ * 32) {
      const int lc = e / n, i = e - lc * n;
      const int g = (lc < bw ? bp * bw + lc : bq * bw + (lc - bw));
      if (g < n) { Xs[e] = __ldcg(Xt + (size_t)g * n + i); Js[e] = __ldcg(Jt + (size_t)g * n + i); }
    }
    __syncthreads();
  };
  auto store_blocks = [&](int bp, int bq) {
    __syncthreads();
    for (int e = tid; e < 2 * bw * n; e += JW_ * 32) {
      const int lc = e / n, i = e - lc * n;
      const int g = (lc < bw ? bp * bw + lc : bq * bw + (lc - bw));
      if (g < n) { Xt[(size_t)g * n + i] = Xs[e]; Jt[(size_t)g * n + i] = Js[e]; }
    }
  };
  const int bwp = (bw + 1) & ~1;                          // players of the in-block tournament
  int sweep = 0;
  for (; sweep < max_sweeps; sweep++) {
    int any = 0;
    // (i) pairs inside blocks 2 cta and 2 cta + 1: the first half of the warps takes the first block, the second half the other
    {
      const int b0 = 2 * cta, b1 = 2 * cta + 1;
      load_blocks(b0, b1);
      for (int round = 0; round < bwp - 1; round++) {
        const int half = warp / (JW_ / 2), k = warp % (JW_ / 2);
        if (k < bwp / 2) {
          int p, q;
          if (k == 0) { p = round; q = bwp - 1; }
          else { p = (round + k) % (bwp - 1); q = (round - k + (bwp - 1)) % (bwp - 1); }
          if (p > q) { const int t = p; p = q; q = t; }
          const int base = half ? b1 * bw : b0 * bw;
          if (q < bw && base + q < n) {
            const int lp = half * bw + p, lq = half * bw + q;
            any |= jacobi_pair_smem<NPL>(Xs + (size_t)lp * n, Xs + (size_t)lq * n, Js + (size_t)lp * n, Js + (size_t)lq * n, n, lane, tol2, thr);
          }
        }
        __syncthreads();
      }
      store_blocks(b0, b1);
      cluster.sync();
    }
    // (ii) tournament of the blocks: CTA k plays block pair k of the round
    for (int round = 0; round < JB_ - 1; round++) {
      int bp, bq;
      if (cta == 0) { bp = round; bq = JB_ - 1; }
      else { bp = (round + cta) % (JB_ - 1); bq = (round - cta + (JB_ - 1)) % (JB_ - 1); }
      if (bp > bq) { const int t = bp; bp = bq; bq = t; }
      if (bq * bw < n) {                                   // both blocks hold real columns
        load_blocks(bp, bq);
        const bool have_p = warp < bw && bp * bw + warp < n;
        c128 xu[NPL], ju[NPL];                              // this warp's column of block bp, in registers for all bw rounds
        if (have_p) {
#pragma unroll
          for (int q = 0; q < NPL; q++) {
            const int i = lane + 32 * q;
            xu[q] = i < n ? Xs[(size_t)warp * n + i] : make_double2(0.0, 0.0);
            ju[q] = i < n ? Js[(size_t)warp * n + i] : make_double2(0.0, 0.0);
          }
        }
        for (int r = 0; r < bw; r++) {
          if (have_p) {
            const int lq = bw + (warp + r) % bw;
            if (bq * bw + (lq - bw) < n)
              any |= jacobi_pair_preg<NPL>(xu, ju, Xs + (size_t)lq * n, Js + (size_t)lq * n, n, lane, tol2, thr);
          }
          __syncthreads();
        }
        if (have_p) {
#pragma unroll
          for (int q = 0; q < NPL; q++) {
            const int i = lane + 32 * q;
            if (i < n) { Xs[(size_t)warp * n + i] = xu[q]; Js[(size_t)warp * n + i] = ju[q]; }
          }
        }
        store_blocks(bp, bq);
      }
      if (round == JB_ - 2 && any && lane == 0) flags[sweep] = 1;   // benign race: every writer stores 1
      if (round == JB_ - 2 && (any & 2) && lane == 0) flags[64 + sweep] = 1;
      cluster.sync();
    }
    if (__ldcg(flags + sweep) == 0) break;                          // nobody rotated in this sweep
    // ... or every pair it met was orthogonal to 1e-10 already (no "coarse" pair): a rotation by an angle <= 1e-10
    // disturbs the other products of its two columns by <= 1e-10 * 1e-10 each, so after this sweep every cosine is
    // below ~2 n 1e-20 << sqrt(n) eps and the next sweep would only confirm it (a sweep is ~0.2 ms at n = 128)
    if (__ldcg(flags + 64 + sweep) == 0) break;
  }
  if (sweep == max_sweeps && cta == 0 && tid == 0) {
    flags[FLAG_FORCE_QR] = 1;
    if (status && __ldcg(flags + 64 + max_sweeps - 1)) atomicOr(status, TDVP_STATUS_SVD_UNCONVERGED);
  }
}

// Columns of the rotated X (and of J with them) in the order of decreasing norm, before the Householder step:
// that step reads the singular values off the diagonal of R', which needs every column orthogonal -- in
// DIRECTION -- to the columns before it.  The columns the Jacobi iteration leaves alone (below the REL_TINY2
// floor) have arbitrary directions; placed last they can only couple among themselves, at their own magnitude.
__global__ void svd_colnorm_kernel(const c128 *Xt, int n, double *nrm) {
  const int lane = threadIdx.x & 31, c = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (c >= n) return;
  double a = 0.0;
  for (int i = lane; i < n; i += 32) { const c128 u = Xt[(size_t)c * n + i]; a += u.x * u.x + u.y * u.y; }
  a = wsum(a);
  if (lane == 0) nrm[c] = a;
}
// It also decides (CTA 0) whether the Householder step is needed: the rotated columns are mutually orthogonal to
// sqrt(n) eps RELATIVE to their norms -- U = X diag(1 / |x_c|) is then unitary to round-off as it stands -- unless the
// iteration left columns alone (below the REL_TINY2 / TINY_COL2 floors: their directions are arbitrary) or ran out of
// sweeps.  Only then does the factorisation X = U' R' run (flags[FLAG_NEED_QR] gates its kernels).
__global__ void svd_sortcols_kernel(const c128 *Xt, const c128 *Jt, const double *nrm, int n, c128 *Xs, c128 *Js, int *flags, int always_qr) {
  __shared__ int s_rank;
  const int c = blockIdx.x;
  if (threadIdx.x == 0) s_rank = 0;
  __syncthreads();
  if (c == 0 && threadIdx.x < 32) {
    double mx = 0.0, mn = 1e308;
    for (int q = threadIdx.x; q < n; q += 32) { const double o = nrm[q]; mx = fmax(mx, o); mn = (o < mn || o != o) ? o : mn; }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
      const double t = __shfl_xor_sync(0xffffffffu, mn, o);
      mn = (t < mn || t != t) ? t : mn;
    }
    if (threadIdx.x == 0)
      flags[FLAG_NEED_QR] = (always_qr || flags[FLAG_FORCE_QR] || !(mn >= fmax(TINY_COL2, REL_TINY2 * mx)) || !(mx < 1e300)) ? 1 : 0;
  }
  const double mine = nrm[c];
  int cnt = 0;
  for (int q = threadIdx.x; q < n; q += blockDim.x) { const double o = nrm[q]; cnt += (o > mine || (o == mine && q < c)) ? 1 : 0; }
  if (cnt) atomicAdd(&s_rank, cnt);
  __syncthreads();
  const int k = s_rank;
  for (int i = threadIdx.x; i < n; i += blockDim.x) {
    Xs[(size_t)k * n + i] = Xt[(size_t)c * n + i];
    Js[(size_t)k * n + i] = Jt[(size_t)c * n + i];
  }
}

// lam (descending), U and the permuted J from X = U' R' (Qp = U'^T, Dp = R'^T as qr_gauge side 1 returns them).
// U[i][k] = Qp[r][i] * sgn(Dp[r][r]),  JtP[k][j] = Jt[r][j]   with k = rank of r.
// Without the Householder step (flags[FLAG_NEED_QR] == 0): column k of the sorted X is sigma_k u_k as it stands.
__global__ void svd_finish_kernel(const c128 *Qp, const c128 *Dp, const c128 *Jt, int n, c128 *U, double *lam,
                                  c128 *JtP, const c128 *Xs, const double *nrm_unused, const int *flags) {
  extern __shared__ double sl[];                                  // [n] |R'_rr|
  if (__ldcg(flags + FLAG_NEED_QR) == 0) {
    __shared__ double s_part[4];
    for (int k = blockIdx.x; k < n; k += gridDim.x) {
      double a = 0.0;
      for (int i = threadIdx.x; i < n; i += blockDim.x) { const c128 u = Xs[(long long)k * n + i]; a += u.x * u.x + u.y * u.y; }
      a = wsum(a);
      if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = a;
      __syncthreads();
      const double nrm2 = s_part[0] + s_part[1] + s_part[2] + s_part[3];      // (128 threads: four warps, fixed order)
      const double nr = sqrt(nrm2), inv = 1.0 / nr;
      if (threadIdx.x == 0) lam[k] = nr;
      for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const c128 u = Xs[(long long)k * n + i];
        U[(long long)i * n + k] = make_double2(u.x * inv, u.y * inv);
        JtP[(long long)k * n + i] = Jt[(long long)k * n + i];
      }
      __syncthreads();
    }
    return;
  }
  for (int r = threadIdx.x; r < n; r += blockDim.x) {
    c128 v = Dp[(long long)r * n + r];
    sl[r] = sqrt(v.x * v.x + v.y * v.y);
  }
  __syncthreads();
  for (int r = blockIdx.x; r < n; r += gridDim.x) {
    __shared__ int rank_s;
    if (threadIdx.x == 0) rank_s = 0;
    __syncthreads();
    int cnt = 0;
    const double lr = sl[r];
    for (int s = threadIdx.x; s < n; s += blockDim.x) cnt += (sl[s] > lr || (sl[s] == lr && s < r)) ? 1 : 0;
    if (cnt) atomicAdd(&rank_s, cnt);
    __syncthreads();
    const int k = rank_s;
    c128 v = Dp[(long long)r * n + r];
    c128 ph = lr > 0.0 ? make_double2(v.x / lr, v.y / lr) : make_double2(1.0, 0.0);
    if (threadIdx.x == 0) lam[k] = lr;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
      U[(long long)i * n + k] = cmul(Qp[(long long)r * n + i], ph);
      JtP[(long long)k * n + i] = Jt[(long long)r * n + i];
    }
    __syncthreads();
  }
}

}  // namespace

void svd_configure() {
  const int bytes = 4 * 8 * 128 * (int)sizeof(c128);     // X and J of two blocks at n = 128
  cudaFuncSetAttribute(svd_jacobi_block_kernel<1, JB, JC, JW>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  cudaFuncSetAttribute(svd_jacobi_block_kernel<2, JB, JC, JW>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  cudaFuncSetAttribute(svd_jacobi_block_kernel<4, JB, JC, JW>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);

}

namespace {
struct SvdWs { c128 *Q, *D, *Xt, *Jt, *Qp, *Dp, *JtP, *Js; double *cnorm; int *flags; void *qws1, *qws2; };
SvdWs svd_carve(int Ml, int d, int Mr, void *ws) {
  const size_t n = Ml, nn = up256(n * n * 16);
  char *p = reinterpret_cast<char *>(up256(reinterpret_cast<size_t>(ws)));
  SvdWs w;
  w.Q = reinterpret_cast<c128 *>(p); p += up256((size_t)Ml * d * Mr * 16);
  w.D = reinterpret_cast<c128 *>(p); p += nn;
  w.Xt = reinterpret_cast<c128 *>(p); p += nn;
  w.Jt = reinterpret_cast<c128 *>(p); p += nn;
  w.Qp = reinterpret_cast<c128 *>(p); p += nn;
  w.Dp = reinterpret_cast<c128 *>(p); p += nn;
  w.JtP = reinterpret_cast<c128 *>(p); p += nn;
  w.Js = reinterpret_cast<c128 *>(p); p += nn;              // J with its columns in the sorted order (X sorted goes into D's buffer)
  w.cnorm = reinterpret_cast<double *>(p); p += up256(n * 8);
  w.flags = reinterpret_cast<int *>(p); p += 512;           // see FLAG_*
  w.qws1 = p; p += up256(qr_ws_bytes(d * Mr, Ml));          // the RQ of C: its reflectors must survive until svd_bond_vh forms Q
  w.qws2 = p;                                               // the (gated) Householder step on the rotated matrix
  return w;
}
}  // namespace

size_t svd_ws_bytes(int Ml, int d, int Mr) {
  const size_t n = Ml, nn = up256(n * n * 16);
  size_t q1 = qr_ws_bytes(d * Mr, Ml), q2 = qr_ws_bytes(Ml, Ml);
  return up256((size_t)Ml * d * Mr * 16) + 7 * nn + 512 + up256(n * 8) + up256(q1) + up256(q2) + 1024;
}

// The unfolding in two halves on one workspace.  svd_bond_factor: everything the NEXT bond of a chain of unfoldings
// needs (U, lam) -- the R factor of C = D Q without forming Q, the Jacobi iteration, U.  svd_bond_vh: Q and
// Vh = (J permuted)^H Q, which only the bond's own consumers need; it may run later and on another queue, as long as the
// workspace is left alone in between (step_mu.cu runs it beside the next bond's factor phase).
void svd_bond_factor(cudaStream_t st, int Ml, int d, int Mr, const c128 *C, c128 *U, double *lam, void *ws, int *status) {
  ProfScope ps(st, PH_SVD);
  // sweeps allowed (diagnostic switch TDVP_SVD_MAX_SWEEPS, read at every call: the error-path test lowers it)
  int max_sweeps = MAX_SWEEPS;
  if (const char *e = getenv("TDVP_SVD_MAX_SWEEPS")) { const int v = atoi(e); if (v >= 1 && v <= MAX_SWEEPS) max_sweeps = v; }
  const int n = Ml;
  const SvdWs w = svd_carve(Ml, d, Mr, ws);
  c128 *D = w.D, *Xt = w.Xt, *Jt = w.Jt, *Qp = w.Qp, *Dp = w.Dp, *JtP = w.JtP, *Js = w.Js;
  double *cnorm = w.cnorm;
  int *flags = w.flags;
  qr_factor(st, 1, Ml, d, Mr, C, D, w.qws1);                              // C = D Q (Q formed later)
  const int g = (n * n + 255) / 256 > 296 ? 296 : (n * n + 255) / 256;
  TDVP_LAUNCH(svd_init_kernel, g, 256, 0, st, D, Xt, Jt, n);
  cudaMemsetAsync(flags, 0, 128 * sizeof(int), st);
  const size_t bsm = (size_t)4 * ((n + JB - 1) / JB) * n * sizeof(c128);      // X and J of two blocks
  if (n <= 16) TDVP_LAUNCH(svd_jacobi_kernel<1>, JC, JW * 32, 0, st, Xt, Jt, n, flags, max_sweeps, status);
  else if (n <= 32) TDVP_LAUNCH((svd_jacobi_block_kernel<1, JB, JC, JW>), JC, JW * 32, bsm, st, Xt, Jt, n, flags, max_sweeps, status);
  else if (n <= 64) TDVP_LAUNCH((svd_jacobi_block_kernel<2, JB, JC, JW>), JC, JW * 32, bsm, st, Xt, Jt, n, flags, max_sweeps, status);
  else if (n <= 128) TDVP_LAUNCH((svd_jacobi_block_kernel<4, JB, JC, JW>), JC, JW * 32, bsm, st, Xt, Jt, n, flags, max_sweeps, status);
  else TDVP_LAUNCH(svd_jacobi_kernel<0>, JC, JW * 32, 0, st, Xt, Jt, n, flags, max_sweeps, status);
  // X = U' R'  <=>  Xt = R'^T U'^T: "side 1" factorisation of the n x n matrix Xt (d = 1)
  c128 *Xs = D;                                                   // D is no longer needed
  TDVP_LAUNCH(svd_colnorm_kernel, (n + 7) / 8, 256, 0, st, Xt, n, cnorm);
  // TDVP_SVD_ALWAYS_QR=1: the Householder step runs whatever the columns look like (diagnostic switch)
  static const int always_qr = [] { const char *e = getenv("TDVP_SVD_ALWAYS_QR"); return (e && e[0] == '1') ? 1 : 0; }();
  TDVP_LAUNCH(svd_sortcols_kernel, n, 128, 0, st, Xt, Jt, cnorm, n, Xs, Js, flags, always_qr);
  qr_gauge(st, 1, n, 1, n, Xs, Qp, Dp, w.qws2, flags + FLAG_NEED_QR);
  TDVP_LAUNCH(svd_finish_kernel, n < 148 ? n : 148, 128, n * sizeof(double), st, Qp, Dp, Js, n, U, lam, JtP, Xs, cnorm, flags);
}

void svd_bond_vh(cudaStream_t st, int Ml, int d, int Mr, c128 *Vh, void *ws) {
  ProfScope ps(st, PH_SVD);
  const int n = Ml;
  const SvdWs w = svd_carve(Ml, d, Mr, ws);
  qr_form_q(st, 1, Ml, d, Mr, w.Q, w.qws1);
  ZGemm gm{};                                   // Vh[k][:] = sum_j conj(JtP[k][j]) Q[j][:]
  gm.A = w.JtP; gm.B = w.Q; gm.C = Vh;
  gm.M = n; gm.K = n; gm.N = d * Mr;
  gm.a_ms = n; gm.a_ks = 1; gm.conjA = 1; gm.b_ks = gm.N; gm.b_ns = 1; gm.ldc = gm.N;
  zgemm(st, gm);
}

// C [Ml, d, Mr] -> U [Ml, Ml], lam [Ml], Vh [Ml, d, Mr]
void svd_bond(cudaStream_t st, int Ml, int d, int Mr, const c128 *C, c128 *U, double *lam, c128 *Vh, void *ws, int *status) {
  svd_bond_factor(st, Ml, d, Mr, C, U, lam, ws, status);
  svd_bond_vh(st, Ml, d, Mr, Vh, ws);
}
