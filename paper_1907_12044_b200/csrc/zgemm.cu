// zgemm.cu -- complex128 GEMM on the B200 FP64 tensor pipe (DMMA m8n8k4 via mma.sync f64).
//
// Used by every dense stage of the hot path: the
// "M_S^3 M_O d" terms of Table I.  tcgen05/UMMA has no FP64 operand type, so on
// sm_100a the FP64 tensor path is the warp-level DMMA; it issues at 64 FMA/clk/SM (measured:
// 37.15 TFLOP/s), slow enough that shared-memory and L2 bandwidth are never the limit -- the
// kernel is designed around keeping all four SMSPs issuing DMMA back to back:
//   * CTA tile 64x64 complex, 4 warps, each warp a 32x32 complex tile = 4x4 m8n8 blocks, real and
//     imaginary accumulators (64 f64 per thread); the complex product is 4 real MMAs per block
//     pair, with -Im(A) made by a sign-bit XOR on the ALU pipe (no FP64 pipe work);
//   * operands stay in their global layout (complex interleaved) in shared memory, staged by a
//     4-stage cp.async (LDGSTS, 16 B = one complex number per copy, zero-fill at ragged edges);
//     row paddings make every fragment LDS.128 bank-conflict free;
//   * two CTAs per SM; split-K (deterministic: partials to a workspace, then one reduce kernel)
//     when the output has too few tiles to fill 148 SMs (stage 3 of H_eff, the bond operator).
#include "common.cuh"

namespace {

constexpr int BM = 64, BN = 64, BK = 8, STAGES = 4;
constexpr int WM = 32, WN = 32;
constexpr int NTHREADS = (BM / WM) * (BN / WN) * 32;   // 128
constexpr int LDK = BK + 4;    // K-major tile row stride (complex): 12 == 4 (mod 8)
constexpr int LDM = BM + 2;    // MN-major tile row stride: 66 == 2 (mod 8)
constexpr int A_TILE = (BM * LDK > BK * LDM) ? BM * LDK : BK * LDM;   // complex elements
constexpr int B_TILE = A_TILE;
constexpr int SMEM_BYTES = STAGES * (A_TILE + B_TILE) * 16;

struct KParams {
  const c128 *A; const c128 *B; c128 *C;
  int M, N, K;
  long long a_ms, a_ks, b_ks, b_ns, ldc;
  int batch_inner;
  long long a_bsi, b_bsi, c_bsi, a_bso, b_bso, c_bso;
  unsigned a_sign;      // 0x80000000 if conjA
  unsigned b_sign;      // 0x80000000 if conjB
  int splitk, ktiles_per_split;
  int tiles_m, tiles_n;
  c128 *partial;        // split-K workspace [split][batch][M][N]
  long long partial_split_stride;
};

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem, bool pred) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  int sz = pred ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}
__device__ __forceinline__ double flip(double x, unsigned mask) {
  return __hiloint2double(__double2hiint(x) ^ (int)mask, __double2loint(x));
}
__device__ __forceinline__ void dmma(double &c0, double &c1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
      : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

template <bool A_KMAJOR, bool B_KMAJOR>
__global__ void __launch_bounds__(NTHREADS, 2) zgemm_kernel(KParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  c128 *sA = reinterpret_cast<c128 *>(smem_raw);
  c128 *sB = sA + STAGES * A_TILE;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm0 = (warp / (BN / WN)) * WM, wn0 = (warp % (BN / WN)) * WN;
  const int tile = blockIdx.x;
  const int tn = tile % p.tiles_n, tm = tile / p.tiles_n;
  const int m0 = tm * BM, n0 = tn * BN;
  const int split = blockIdx.y;
  const int bz = blockIdx.z, bin = bz % p.batch_inner, bo = bz / p.batch_inner;

  const c128 *Ab = p.A + bin * p.a_bsi + bo * p.a_bso;
  const c128 *Bb = p.B + bin * p.b_bsi + bo * p.b_bso;

  const int ktiles_total = (p.K + BK - 1) / BK;
  const int kt_begin = split * p.ktiles_per_split;
  int kt_end = kt_begin + p.ktiles_per_split;
  if (kt_end > ktiles_total) kt_end = ktiles_total;
  const int nkt = kt_end - kt_begin;   // may be <= 0 for a trailing split: writes zeros

  auto load_tile = [&](int stage, int kt) {
    const int k0 = kt * BK;
    c128 *a = sA + stage * A_TILE;
    c128 *b = sB + stage * B_TILE;
#pragma unroll
    for (int i = 0; i < (BM * BK) / NTHREADS; i++) {
      int e = tid + i * NTHREADS;
      int r, k, so;
      if (A_KMAJOR) { r = e / BK; k = e % BK; so = r * LDK + k; }
      else          { k = e / BM; r = e % BM; so = k * LDM + r; }
      bool ok = (m0 + r < p.M) && (k0 + k < p.K);
      const c128 *src = ok ? Ab + (long long)(m0 + r) * p.a_ms + (long long)(k0 + k) * p.a_ks : Ab;
      cp_async16(a + so, src, ok);
    }
#pragma unroll
    for (int i = 0; i < (BN * BK) / NTHREADS; i++) {
      int e = tid + i * NTHREADS;
      int r, k, so;
      if (B_KMAJOR) { r = e / BK; k = e % BK; so = r * LDK + k; }
      else          { k = e / BN; r = e % BN; so = k * LDM + r; }
      bool ok = (n0 + r < p.N) && (k0 + k < p.K);
      const c128 *src = ok ? Bb + (long long)(n0 + r) * p.b_ns + (long long)(k0 + k) * p.b_ks : Bb;
      cp_async16(b + so, src, ok);
    }
  };

  double cr[4][4][2], ci[4][4][2];
#pragma unroll
  for (int i = 0; i < 4; i++)
#pragma unroll
    for (int j = 0; j < 4; j++) { cr[i][j][0] = cr[i][j][1] = ci[i][j][0] = ci[i][j][1] = 0.0; }

#pragma unroll
  for (int s = 0; s < STAGES - 1; s++) {
    if (s < nkt) load_tile(s, kt_begin + s);
    cp_async_commit();
  }

  const int lr = lane >> 2, lk = lane & 3;
  for (int it = 0; it < nkt; it++) {
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    {
      int nx = it + STAGES - 1;
      if (nx < nkt) load_tile(nx % STAGES, kt_begin + nx);
      cp_async_commit();
    }
    const c128 *a = sA + (it % STAGES) * A_TILE;
    const c128 *b = sB + (it % STAGES) * B_TILE;
#pragma unroll
    for (int ks = 0; ks < BK / 4; ks++) {
      double ar[4], ai[4], nai[4], br[4], bi[4];
#pragma unroll
      for (int i = 0; i < 4; i++) {
        c128 v = A_KMAJOR ? a[(wm0 + i * 8 + lr) * LDK + ks * 4 + lk]
                          : a[(ks * 4 + lk) * LDM + wm0 + i * 8 + lr];
        ar[i] = v.x;
        ai[i] = flip(v.y, p.a_sign);
        nai[i] = flip(ai[i], 0x80000000u);
      }
#pragma unroll
      for (int j = 0; j < 4; j++) {
        c128 v = B_KMAJOR ? b[(wn0 + j * 8 + lr) * LDK + ks * 4 + lk]
                          : b[(ks * 4 + lk) * LDM + wn0 + j * 8 + lr];
        br[j] = v.x;
        bi[j] = flip(v.y, p.b_sign);
      }
#pragma unroll
      for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < 4; j++) {
          dmma(cr[i][j][0], cr[i][j][1], ar[i], br[j]);
          dmma(ci[i][j][0], ci[i][j][1], ar[i], bi[j]);
        }
#pragma unroll
      for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < 4; j++) {
          dmma(cr[i][j][0], cr[i][j][1], nai[i], bi[j]);
          dmma(ci[i][j][0], ci[i][j][1], ai[i], br[j]);
        }
    }
  }
  cp_async_wait<0>();

  // epilogue: thread holds C(row = lane/4, cols = 2*(lane%4) + {0,1}) of every 8x8 block
  c128 *Cb;
  long long ldc;
  if (p.splitk > 1) {
    Cb = p.partial + (long long)split * p.partial_split_stride + (long long)bz * p.M * p.N;
    ldc = p.N;
  } else {
    Cb = p.C + bin * p.c_bsi + bo * p.c_bso;
    ldc = p.ldc;
  }
#pragma unroll
  for (int i = 0; i < 4; i++) {
    int m = m0 + wm0 + i * 8 + lr;
    if (m >= p.M) continue;
#pragma unroll
    for (int j = 0; j < 4; j++) {
      int n = n0 + wn0 + j * 8 + 2 * lk;
      c128 *dst = Cb + (long long)m * ldc + n;
      if (n < p.N) dst[0] = make_double2(cr[i][j][0], ci[i][j][0]);
      if (n + 1 < p.N) dst[1] = make_double2(cr[i][j][1], ci[i][j][1]);
    }
  }
}

// C[b](m,n) = sum_s partial[s][b][m][n]   (fixed order: deterministic)
__global__ void splitk_reduce_kernel(const c128 *partial, long long split_stride, int splitk,
                                     c128 *C, int M, int N, long long ldc, int batch_inner,
                                     long long c_bsi, long long c_bso, long long total) {
  long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (idx >= total) return;
  int n = idx % N;
  long long t = idx / N;
  int m = t % M;
  int bz = t / M;
  double sx = 0.0, sy = 0.0;
  for (int s = 0; s < splitk; s++) {
    c128 v = partial[s * split_stride + idx];
    sx += v.x; sy += v.y;
  }
  int bin = bz % batch_inner, bo = bz / batch_inner;
  C[bin * c_bsi + bo * c_bso + (long long)m * ldc + n] = make_double2(sx, sy);
}

constexpr int SLOTS = 148 * 2;   // resident CTAs: 2 per SM on 148 SMs

int choose_splitk(long long tiles, int ktiles) {
  // cost model in k-tile units: waves * ktiles-per-split, plus the reduce pass for s > 1
  int best_s = 1;
  double best = 1e300;
  int smax = ktiles < 32 ? ktiles : 32;
  for (int s = 1; s <= smax; s++) {
    int kps = (ktiles + s - 1) / s;
    if (s > 1 && (ktiles + kps - 1) / kps != s) continue;     // skip splits that leave empty slices
    long long waves = (tiles * s + SLOTS - 1) / SLOTS;
    double cost = (double)waves * (kps + 2.0) + (s > 1 ? 3.0 + 0.5 * s : 0.0);
    if (cost < best - 1e-9) { best = cost; best_s = s; }
  }
  return best_s;
}

template <bool AK, bool BK_>
void launch(cudaStream_t st, const KParams &kp, dim3 grid) {
  TDVP_LAUNCH((zgemm_kernel<AK, BK_>), grid, NTHREADS, SMEM_BYTES, st, kp);
}

}  // namespace

void zgemm_configure() {
  cudaFuncSetAttribute(zgemm_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
  cudaFuncSetAttribute(zgemm_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
  cudaFuncSetAttribute(zgemm_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
  cudaFuncSetAttribute(zgemm_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
}

size_t zgemm_ws_elems(const ZGemm &p) {
  long long batch = (long long)p.batch_inner * p.batch_outer;
  long long tiles = ceil_div_ll(p.M, BM) * ceil_div_ll(p.N, BN) * batch;
  int ktiles = (p.K + BK - 1) / BK;
  int s = p.splitk > 0 ? p.splitk : choose_splitk(tiles, ktiles);
  if (s <= 1) return 0;
  return (size_t)s * batch * p.M * p.N;
}

void zgemm(cudaStream_t st, const ZGemm &p, c128 *ws) {
  if (p.M <= 0 || p.N <= 0) return;
  KParams kp;
  kp.A = p.A; kp.B = p.B; kp.C = p.C;
  kp.M = p.M; kp.N = p.N; kp.K = p.K;
  kp.a_ms = p.a_ms; kp.a_ks = p.a_ks; kp.b_ks = p.b_ks; kp.b_ns = p.b_ns; kp.ldc = p.ldc;
  kp.batch_inner = p.batch_inner;
  kp.a_bsi = p.a_bsi; kp.b_bsi = p.b_bsi; kp.c_bsi = p.c_bsi;
  kp.a_bso = p.a_bso; kp.b_bso = p.b_bso; kp.c_bso = p.c_bso;
  kp.a_sign = p.conjA ? 0x80000000u : 0u;
  kp.b_sign = p.conjB ? 0x80000000u : 0u;
  kp.tiles_m = (p.M + BM - 1) / BM;
  kp.tiles_n = (p.N + BN - 1) / BN;
  long long batch = (long long)p.batch_inner * p.batch_outer;
  long long tiles = (long long)kp.tiles_m * kp.tiles_n * batch;
  int ktiles = (p.K + BK - 1) / BK;
  if (ktiles < 1) ktiles = 1;
  int s = p.splitk > 0 ? p.splitk : choose_splitk(tiles, ktiles);
  if (s > ktiles) s = ktiles;
  if (ws == nullptr) s = 1;
  kp.splitk = s;
  kp.ktiles_per_split = (ktiles + s - 1) / s;
  kp.partial = ws;
  kp.partial_split_stride = batch * p.M * p.N;
  dim3 grid((unsigned)(kp.tiles_m * kp.tiles_n), (unsigned)s, (unsigned)batch);
  const bool ak = (p.a_ks == 1), bk = (p.b_ks == 1);
  {
    ProfScope ps(st, PH_ZGEMM);
    if (ak && bk) launch<true, true>(st, kp, grid);
    else if (ak && !bk) launch<true, false>(st, kp, grid);
    else if (!ak && bk) launch<false, true>(st, kp, grid);
    else launch<false, false>(st, kp, grid);
  }
  if (s > 1) {
    ProfScope ps(st, PH_SPLITK);
    long long total = batch * p.M * p.N;
    TDVP_LAUNCH(splitk_reduce_kernel, (unsigned)ceil_div_ll(total, 256), 256, 0, st, ws,
                kp.partial_split_stride, s, p.C, p.M, p.N, p.ldc, p.batch_inner, p.c_bsi, p.c_bso, total);
  }
}
