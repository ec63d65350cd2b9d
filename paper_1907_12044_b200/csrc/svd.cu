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
// The Jacobi sweeps run in ONE CTA (32 warps, a column pair per warp and round, round-robin
// ordering, __syncthreads between rounds; X and J live in L2): no host round trip, deterministic,
// capturable in the step graph.
#include "common.cuh"

namespace {

constexpr int JT = 1024;            // threads of the Jacobi CTA
constexpr int MAX_SWEEPS = 40;
inline size_t up256(size_t x) { return (x + 255) & ~size_t(255); }

__device__ __forceinline__ double wsum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
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
__global__ void __launch_bounds__(JT) svd_jacobi_kernel(c128 *Xt, c128 *Jt, int n, int *sweeps_out) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = JT / 32;
  const int np = (n + 1) & ~1;             // players of the round-robin tournament (a bye if n is odd)
  const int npairs = np / 2;
  __shared__ int rotated;
  const double tol = 1e-15;
  int sweep = 0;
  for (; sweep < MAX_SWEEPS; sweep++) {
    if (threadIdx.x == 0) rotated = 0;
    __syncthreads();
    for (int round = 0; round < np - 1; round++) {
      for (int k = warp; k < npairs; k += nwarps) {
        int p, q;
        if (k == 0) { p = round; q = np - 1; }
        else { p = (round + k) % (np - 1); q = (round - k + (np - 1)) % (np - 1); }
        if (p > q) { int t = p; p = q; q = t; }
        if (q >= n) continue;                                    // the bye
        c128 *xp = Xt + (long long)p * n, *xq = Xt + (long long)q * n;
        double a = 0.0, b = 0.0, cr = 0.0, ci = 0.0;
        for (int i = lane; i < n; i += 32) {
          c128 u = xp[i], v = xq[i];
          a += u.x * u.x + u.y * u.y;
          b += v.x * v.x + v.y * v.y;
          cr += u.x * v.x + u.y * v.y;                           // conj(u) * v
          ci += u.x * v.y - u.y * v.x;
        }
        a = wsum(a); b = wsum(b); cr = wsum(cr); ci = wsum(ci);
        const double cabs = sqrt(cr * cr + ci * ci);
        if (!(cabs > tol * sqrt(a) * sqrt(b)) || cabs == 0.0) continue;
        if (lane == 0) rotated = 1;
        // y_q = e^{-i phi} x_q makes <x_p, y_q> = |c| real; then a real rotation (cs, sn)
        const double er = cr / cabs, ei = -ci / cabs;            // e^{-i phi}
        const double zeta = (b - a) / (2.0 * cabs);
        const double t = (zeta >= 0.0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
        const double cs = 1.0 / sqrt(1.0 + t * t), sn = cs * t;
        c128 *jp = Jt + (long long)p * n, *jq = Jt + (long long)q * n;
        for (int i = lane; i < n; i += 32) {
          c128 u = xp[i], v = xq[i];
          c128 y = make_double2(er * v.x - ei * v.y, er * v.y + ei * v.x);
          xp[i] = make_double2(cs * u.x - sn * y.x, cs * u.y - sn * y.y);
          xq[i] = make_double2(sn * u.x + cs * y.x, sn * u.y + cs * y.y);
          u = jp[i]; v = jq[i];
          y = make_double2(er * v.x - ei * v.y, er * v.y + ei * v.x);
          jp[i] = make_double2(cs * u.x - sn * y.x, cs * u.y - sn * y.y);
          jq[i] = make_double2(sn * u.x + cs * y.x, sn * u.y + cs * y.y);
        }
      }
      __syncthreads();
    }
    if (!rotated) break;
    __syncthreads();
  }
  if (threadIdx.x == 0 && sweeps_out) *sweeps_out = sweep;
}

// lam (descending), U and the permuted J from X = U' R' (Qp = U'^T, Dp = R'^T as qr_gauge side 1 returns them).
// U[i][k] = Qp[r][i] * sgn(Dp[r][r]),  JtP[k][j] = Jt[r][j]   with k = rank of r.
__global__ void svd_finish_kernel(const c128 *Qp, const c128 *Dp, const c128 *Jt, int n, c128 *U, double *lam,
                                  c128 *JtP) {
  extern __shared__ double sl[];                                  // [n] |R'_rr|
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

size_t svd_ws_bytes(int Ml, int d, int Mr) {
  const size_t n = Ml, nn = up256(n * n * 16);
  size_t q1 = qr_ws_bytes(d * Mr, Ml), q2 = qr_ws_bytes(Ml, Ml);
  return up256((size_t)Ml * d * Mr * 16) + 6 * nn + up256(q1 > q2 ? q1 : q2) + 1024;
}

// C [Ml, d, Mr] -> U [Ml, Ml], lam [Ml], Vh [Ml, d, Mr]
void svd_bond(cudaStream_t st, int Ml, int d, int Mr, const c128 *C, c128 *U, double *lam, c128 *Vh, void *ws) {
  ProfScope ps(st, PH_SVD);
  const int n = Ml;
  const size_t nn = up256((size_t)n * n * 16);
  char *p = reinterpret_cast<char *>(up256(reinterpret_cast<size_t>(ws)));
  c128 *Q = reinterpret_cast<c128 *>(p); p += up256((size_t)Ml * d * Mr * 16);
  c128 *D = reinterpret_cast<c128 *>(p); p += nn;
  c128 *Xt = reinterpret_cast<c128 *>(p); p += nn;
  c128 *Jt = reinterpret_cast<c128 *>(p); p += nn;
  c128 *Qp = reinterpret_cast<c128 *>(p); p += nn;
  c128 *Dp = reinterpret_cast<c128 *>(p); p += nn;
  c128 *JtP = reinterpret_cast<c128 *>(p); p += nn;
  void *qws = p;
  qr_gauge(st, 1, Ml, d, Mr, C, Q, D, qws);                               // C = D Q
  const int g = (n * n + 255) / 256 > 296 ? 296 : (n * n + 255) / 256;
  TDVP_LAUNCH(svd_init_kernel, g, 256, 0, st, D, Xt, Jt, n);
  TDVP_LAUNCH(svd_jacobi_kernel, 1, JT, 0, st, Xt, Jt, n, (int *)nullptr);
  // X = U' R'  <=>  Xt = R'^T U'^T: "side 1" factorisation of the n x n matrix Xt (d = 1)
  qr_gauge(st, 1, n, 1, n, Xt, Qp, Dp, qws);
  TDVP_LAUNCH(svd_finish_kernel, n < 148 ? n : 148, 128, n * sizeof(double), st, Qp, Dp, Jt, n, U, lam, JtP);
  ZGemm gm{};                                   // Vh[k][:] = sum_j conj(JtP[k][j]) Q[j][:]
  gm.A = JtP; gm.B = Q; gm.C = Vh;
  gm.M = n; gm.K = n; gm.N = d * Mr;
  gm.a_ms = n; gm.a_ks = 1; gm.conjA = 1; gm.b_ks = gm.N; gm.b_ns = 1; gm.ldc = gm.N;
  gm.splitk = 1;
  zgemm(st, gm, nullptr);
}
