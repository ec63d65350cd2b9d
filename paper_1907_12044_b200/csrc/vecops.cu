// vecops.cu -- small vector kernels shared by the step drivers (copies, deterministic reductions).
#include "common.cuh"

namespace {
constexpr int VT = 256;
constexpr int RED_BLOCKS = 296;

__device__ __forceinline__ double wsum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

__global__ void copy_k(c128 *dst, const c128 *src, long long n) {
  for (long long e = blockIdx.x * (long long)VT + threadIdx.x; e < n; e += (long long)gridDim.x * VT) dst[e] = src[e];
}
__global__ void zero_k(c128 *dst, long long n) {
  for (long long e = blockIdx.x * (long long)VT + threadIdx.x; e < n; e += (long long)gridDim.x * VT)
    dst[e] = make_double2(0.0, 0.0);
}

// partial[b] = sum over block b's chunk of conj(x) * y  (y == nullptr: |x|^2 in .x)
__global__ void __launch_bounds__(VT) dot_partial_k(const c128 *x, const c128 *y, long long n, c128 *partial) {
  long long per = (n + gridDim.x - 1) / gridDim.x;
  long long e0 = blockIdx.x * per, e1 = e0 + per;
  if (e1 > n) e1 = n;
  double sx = 0.0, sy = 0.0;
  for (long long e = e0 + threadIdx.x; e < e1; e += VT) {
    c128 a = x[e];
    if (y) { c128 b = y[e]; sx += a.x * b.x + a.y * b.y; sy += a.x * b.y - a.y * b.x; }
    else sx += a.x * a.x + a.y * a.y;
  }
  __shared__ double rx[VT / 32], ry[VT / 32];
  sx = wsum(sx); sy = wsum(sy);
  if ((threadIdx.x & 31) == 0) { rx[threadIdx.x >> 5] = sx; ry[threadIdx.x >> 5] = sy; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double tx = 0, ty = 0;
    for (int i = 0; i < VT / 32; i++) { tx += rx[i]; ty += ry[i]; }
    partial[blockIdx.x] = make_double2(tx, ty);
  }
}
// one warp: out = sum_b partial[b]
__global__ void dot_final_k(const c128 *partial, int nb, double *out_re, c128 *out_c) {
  double sx = 0.0, sy = 0.0;
  for (int g = threadIdx.x; g < nb; g += 32) { sx += partial[g].x; sy += partial[g].y; }
  sx = wsum(sx); sy = wsum(sy);
  if (threadIdx.x == 0) {
    if (out_re) *out_re = sx;
    if (out_c) *out_c = make_double2(sx, sy);
  }
}
int grid_for(long long n) {
  long long g = (n + VT - 1) / VT;
  if (g > RED_BLOCKS) g = RED_BLOCKS;
  if (g < 1) g = 1;
  return (int)g;
}
}  // namespace

void vec_copy(cudaStream_t st, c128 *dst, const c128 *src, long long n) {
  if (n <= 0 || dst == src) return;
  TDVP_LAUNCH(copy_k, grid_for(n), VT, 0, st, dst, src, n);
}
void vec_zero(cudaStream_t st, c128 *dst, long long n) {
  if (n <= 0) return;
  TDVP_LAUNCH(zero_k, grid_for(n), VT, 0, st, dst, n);
}
size_t vec_red_scratch_bytes() { return RED_BLOCKS * sizeof(c128) + 256; }
void vec_norm_sq(cudaStream_t st, const c128 *x, long long n, double *out_dev, void *scratch) {
  int g = grid_for(n);
  TDVP_LAUNCH(dot_partial_k, g, VT, 0, st, x, (const c128 *)nullptr, n, reinterpret_cast<c128 *>(scratch));
  TDVP_LAUNCH(dot_final_k, 1, 32, 0, st, reinterpret_cast<const c128 *>(scratch), g, out_dev, (c128 *)nullptr);
}
void vec_dotc(cudaStream_t st, const c128 *x, const c128 *y, long long n, c128 *out_dev, void *scratch) {
  int g = grid_for(n);
  TDVP_LAUNCH(dot_partial_k, g, VT, 0, st, x, y, n, reinterpret_cast<c128 *>(scratch));
  TDVP_LAUNCH(dot_final_k, 1, 32, 0, st, reinterpret_cast<const c128 *>(scratch), g, (double *)nullptr, out_dev);
}
