// zgemm.cu -- complex128 GEMM on the B200 FP64 tensor pipe (DMMA m8n8k4 via mma.sync f64).
//
// Used by every dense stage of the hot path: the
// "M_S^3 M_O d" terms of Table I.  tcgen05/UMMA has no FP64 operand type, so on
// sm_100a the FP64 tensor path is the warp-level DMMA; it issues at 64 FMA/clk/SM (measured:
// 37.15 TFLOP/s), slow enough that shared-memory and L2 bandwidth are never the limit -- the
// kernel is designed around keeping all four SMSPs issuing DMMA back to back:
//   * CTA tile 64x64 complex, 4 warps, each warp a 32x32 complex tile = 4x4 m8n8 blocks; the complex
//     product is formed from THREE real MMAs per block pair by default (X1 = Ar Br, X2 = Ai Bi,
//     X3 = (Ar + Ai)(Br + Bi): 96 f64 accumulators per thread, combined once per tile segment;
//     DESIGN.md reading c15) or from four (64 accumulators, -Im(A) by a sign-bit XOR on the ALU pipe);
//   * operands stay in their global layout (complex interleaved) in shared memory, staged by TMA
//     (cp.async.bulk.tensor, dense boxes, zero fill at ragged edges) into a 3-slot ring guarded by
//     full/empty mbarriers; one thread issues the loads.  Measured: every non-DMMA instruction a
//     warp issues costs the FP64 tensor pipe ~1.6 cycles (no overlap with a DMMA in flight), so
//     the loop carries no address arithmetic, predicates or per-element copies at all;
//     box shapes are chosen so that every fragment LDS.128 is bank-conflict free;
//   * two CTAs per SM, persistent, with a stream-K schedule: every CTA gets the same number of
//     (tile, k-tile) units, tiles cut across CTAs are summed inside the kernel in a fixed order
//     (deterministic), so neither wave quantisation (stage 1: 800 tiles on 296 CTA slots) nor a
//     separate split-K reduce pass (stage 3 of H_eff, the bond operator: 40 tiles) is paid.
#include <cuda.h>

#include <mutex>
#include <unordered_map>

#include "common.cuh"

namespace {

constexpr int BM = 64, BN = 64, BK = 16, STAGES = 3;
constexpr int LOOKAHEAD = STAGES - 2;                  // k-tiles in flight ahead of the consumer
constexpr int WM = 32, WN = 32;
constexpr int NTHREADS = (BM / WM) * (BN / WN) * 32;   // 128
constexpr int KG = BK / 4;     // k-groups of 4 complex numbers (one DMMA k-step) per k-tile
// Shared-memory operand tiles, written by TMA (dense boxes, no swizzle), read by LDS.128:
//   K-major operand  : [KG][64 rows][4 complex]  -- a quarter-warp (2 rows x 4 k) reads 128
//                      contiguous bytes: bank-conflict free;
//   MN-major operand : [BK][LDM = 66 complex]    -- the box is 66 wide (2 columns over-fetched) so
//                      that the 4 k-rows of a quarter-warp start 8 banks apart: conflict free.
constexpr int LDM = BM + 2;
constexpr int TILE_K_BYTES = KG * BM * 4 * 16;         // 16384
constexpr int TILE_MN_BYTES = BK * LDM * 16;           // 16896
constexpr int TILE_BYTES = TILE_MN_BYTES;              // slot size of either layout (128 B multiple)
constexpr int SMEM_BYTES = STAGES * 2 * TILE_BYTES + 128;
constexpr int SMEM_BYTES_32 = STAGES * 2 * (BK * (32 + 2) * 16) + 128;   // the 32 x 32 tile instance

struct KParams {
  c128 *C;
  int M, N, K;
  long long ldc;
  int batch_inner;
  long long c_bsi, c_bso;
  int a_batched_i, a_batched_o, b_batched_i, b_batched_o;   // 0: operand shared by the batch (coordinate 0)
  int a5, b5;           // K-major operand has a 5-D map (k-group as its own dimension): one TMA per k-tile
  unsigned a_sign;      // 0x80000000 if conjA
  unsigned b_sign;      // 0x80000000 if conjB
  int tiles_m, tiles_n, ktiles;
  int G;                // CTAs of this launch (cooperative: all resident)
  int upc_base, upc_rem;// units (tile, k-tile) per CTA: base, +1 for the first upc_rem CTAs
  int tile;             // 64 or 32: edge of the CTA tile of this launch
  const int *skip;      // nullable: non-zero at kernel start = the caller no longer needs this product
  c128 *slots;          // [2 G][BM*BN] partial tiles of segments that do not cover their tile's whole K
  int *cnt;             // [G] partial segments published for the cut tile whose LAST unit CTA j holds
  int *done;            // [G] contributors that have finished reducing it (the last one zeroes both)
};

__device__ __forceinline__ double flip(double x, unsigned mask) {
  return __hiloint2double(__double2hiint(x) ^ (int)mask, __double2loint(x));
}
__device__ __forceinline__ void dmma(double &c0, double &c1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
      : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__device__ __forceinline__ int ld_acquire(const int *p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void red_release_add(int *p, int v) {
  asm volatile("red.release.gpu.global.add.s32 [%0], %1;\n" ::"l"(p), "r"(v) : "memory");
}
// ---- mbarrier / TMA (cp.async.bulk.tensor) ----
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  unsigned ok;
  do {
    asm volatile(
        "{\n.reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  } while (!ok);
}
__device__ __forceinline__ void tma_load_4d(unsigned dst, const CUtensorMap *tm, unsigned bar, int c0, int c1, int c2, int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];\n"
      ::"r"(dst), "l"(reinterpret_cast<unsigned long long>(tm)), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}

__device__ __forceinline__ void tma_load_5d(unsigned dst, const CUtensorMap *tm, unsigned bar, int c0, int c1, int c2, int c3, int c4) {
  asm volatile(
      "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];\n"
      ::"r"(dst), "l"(reinterpret_cast<unsigned long long>(tm)), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
      : "memory");
}

// Work decomposition ("stream-K"): the (tile, k-tile) units of the whole batched GEMM, tile-major,
// are cut into G equal contiguous ranges, one per CTA, G <= resident CTAs (cooperative launch), so
// every SM carries the same number of DMMAs whatever the tile count.  A range is at most: the tail
// of a tile begun by lower CTAs, whole tiles, and the head of a tile continued by higher CTAs.
// Whole tiles go straight to C.  A partial segment is written to a slot (2 per CTA: [0] the CTA's
// first segment, [1] its last) and counted on the tile's counter; when a CTA has finished its
// units it waits for the counters of its (at most two) cut tiles and reduces ITS SLICE of each:
// the C contributors of a tile each sum 1/C of its elements over all C slots in CTA order (fixed
// order: deterministic, whoever does it) and write them to C.  The fix-up is therefore one
// round trip deep whatever the split, and there is no separate reduce kernel.
__device__ __forceinline__ int cta_of_unit(int u, int base, int rem) {
  const int cut = rem * (base + 1);
  return u < cut ? u / (base + 1) : rem + (u - cut) / base;
}

template <bool A_KMAJOR, bool B_KMAJOR, bool CONJ, bool M3, int TB>
__device__ __forceinline__ void zgemm_body(const CUtensorMap &tmA, const CUtensorMap &tmB, const KParams &p) {
  // tile geometry of this instance (TB = 64: the default; TB = 32: small problems, see choose_tile)
  constexpr int BM = TB, BN = TB, WM = TB / 2, WN = TB / 2, NB8 = WM / 8;      // NB8 x NB8 m8n8 blocks per warp
  constexpr int LDM = TB + 2;
  constexpr int TILE_K_BYTES = KG * TB * 4 * 16, TILE_MN_BYTES = BK * LDM * 16, TILE_BYTES = TILE_MN_BYTES;
  extern __shared__ __align__(128) unsigned char smem_dyn[];
  __shared__ int s_fix_tile[2];
  __shared__ __align__(8) unsigned long long s_full[STAGES], s_empty[STAGES];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm0 = (warp / (BN / WN)) * WM, wn0 = (warp % (BN / WN)) * WN;
  // the dynamic segment is only guaranteed 16 B alignment: round up to 128 B for TMA destinations
  const unsigned smem_base = ((unsigned)__cvta_generic_to_shared(smem_dyn) + 127u) & ~127u;
  unsigned char *smem_gen = smem_dyn + (smem_base - (unsigned)__cvta_generic_to_shared(smem_dyn));
  const unsigned full0 = (unsigned)__cvta_generic_to_shared(s_full);
  const unsigned empty0 = (unsigned)__cvta_generic_to_shared(s_empty);
  if (tid == 0) {
    asm volatile("prefetch.tensormap [%0];\n" ::"l"(reinterpret_cast<unsigned long long>(&tmA)) : "memory");
    asm volatile("prefetch.tensormap [%0];\n" ::"l"(reinterpret_cast<unsigned long long>(&tmB)) : "memory");
    s_fix_tile[0] = s_fix_tile[1] = -1;
    for (int s = 0; s < STAGES; s++) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, NTHREADS / 32); }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();
  const int cta = blockIdx.x;
  const int ktiles = p.ktiles;
  const int u0 = cta * p.upc_base + (cta < p.upc_rem ? cta : p.upc_rem);
  const int nkt = p.upc_base + (cta < p.upc_rem ? 1 : 0);
  const int t0 = u0 / ktiles, k_first = u0 - t0 * ktiles;
  const int tiles_mn = p.tiles_m * p.tiles_n;
  // order of work: the partial first segment (tail of tile t0), the partial last segment (head of
  // tile tL), then the whole tiles -- so the partials are published long before anybody needs them
  const int first_len = (ktiles - k_first) < nkt ? (ktiles - k_first) : nkt;
  const int lenF = (k_first > 0 || first_len < ktiles) ? first_len : 0;
  const int tL = (u0 + nkt - 1) / ktiles;
  const int last_len = u0 + nkt - tL * ktiles;
  const int lenL = (last_len < ktiles && tL != t0) ? last_len : 0;
  const int lenFL = lenF + lenL;
  const int tM0 = (u0 + lenF) / ktiles;                  // first whole tile

  // ---- producer: thread 0 issues the TMA loads of position `pos` into slot pos % STAGES ----
  // (its tile coordinates are decoded only when the tile changes; slot and parity are counters)
  int l_tile = lenF ? t0 : (lenL ? tL : tM0), l_kt = lenF ? k_first : 0;
  int l_m0 = 0, l_n0 = 0, l_abi = 0, l_abo = 0, l_bbi = 0, l_bbo = 0, p_slot = 0;
  unsigned p_par = 0;                                    // parity of the "empty" phase to wait for
  auto decode = [&]() {
    const int bz = l_tile / tiles_mn, tr = l_tile - bz * tiles_mn;
    l_m0 = (tr / p.tiles_n) * BM; l_n0 = (tr % p.tiles_n) * BN;
    const int bin = bz % p.batch_inner, bo = bz / p.batch_inner;
    l_abi = p.a_batched_i ? bin : 0; l_abo = p.a_batched_o ? bo : 0;
    l_bbi = p.b_batched_i ? bin : 0; l_bbo = p.b_batched_o ? bo : 0;
  };
  auto issue = [&](int pos) {
    if (pos >= STAGES) mbar_wait(empty0 + 8 * p_slot, p_par);   // consumers of pos - STAGES are done
    const int k0 = l_kt * BK;
    const unsigned bar = full0 + 8 * p_slot;
    const unsigned dA = smem_base + p_slot * (2 * TILE_BYTES), dB = dA + TILE_BYTES;
    mbar_expect_tx(bar, (A_KMAJOR ? TILE_K_BYTES : TILE_MN_BYTES) + (B_KMAJOR ? TILE_K_BYTES : TILE_MN_BYTES));
    if (A_KMAJOR) {
      if (p.a5) tma_load_5d(dA, &tmA, bar, 0, l_m0, k0 >> 2, l_abi, l_abo);
      else {
#pragma unroll
        for (int g = 0; g < KG; g++) tma_load_4d(dA + g * (BM * 64), &tmA, bar, 2 * (k0 + 4 * g), l_m0, l_abi, l_abo);
      }
    } else {
      tma_load_4d(dA, &tmA, bar, 2 * l_m0, k0, l_abi, l_abo);
    }
    if (B_KMAJOR) {
      if (p.b5) tma_load_5d(dB, &tmB, bar, 0, l_n0, k0 >> 2, l_bbi, l_bbo);
      else {
#pragma unroll
        for (int g = 0; g < KG; g++) tma_load_4d(dB + g * (BN * 64), &tmB, bar, 2 * (k0 + 4 * g), l_n0, l_bbi, l_bbo);
      }
    } else {
      tma_load_4d(dB, &tmB, bar, 2 * l_n0, k0, l_bbi, l_bbo);
    }
    if (++p_slot == STAGES) { p_slot = 0; if (pos >= STAGES) p_par ^= 1u; }
    const int np = pos + 1;
    if (np == lenF && lenL) { l_tile = tL; l_kt = 0; decode(); }
    else if (np == lenFL) { l_tile = tM0; l_kt = 0; decode(); }
    else if (++l_kt == ktiles) { l_kt = 0; ++l_tile; decode(); }
  };
  if (tid == 0) {
    decode();
    for (int s = 0; s < LOOKAHEAD && s < nkt; s++) issue(s);
  }

  // 4M: cr = sum ar br - ai bi, ci = sum ar bi + ai br.
  // 3M: cr = sum ar br, ci = sum ai bi, cs = sum (ar + ai)(br + bi); the tile is cr - ci and
  //     cs - cr - ci, formed once per segment (fin()).
  double cr[NB8][NB8][2], ci[NB8][NB8][2], cs[M3 ? NB8 : 1][M3 ? NB8 : 1][2];
#pragma unroll
  for (int i = 0; i < NB8; i++)
#pragma unroll
    for (int j = 0; j < NB8; j++) {
      cr[i][j][0] = cr[i][j][1] = ci[i][j][0] = ci[i][j][1] = 0.0;
      if (M3) cs[M3 ? i : 0][M3 ? j : 0][0] = cs[M3 ? i : 0][M3 ? j : 0][1] = 0.0;
    }
  auto fin = [&](int i, int j, int h) -> c128 {
    if (M3) {
      const double x1 = cr[i][j][h], x2 = ci[i][j][h];
      return make_double2(x1 - x2, cs[M3 ? i : 0][M3 ? j : 0][h] - x1 - x2);
    }
    return make_double2(cr[i][j][h], ci[i][j][h]);
  };

  const int lr = lane >> 2, lk = lane & 3;
  const unsigned na_sign = p.a_sign ^ 0x80000000u;
  int c_tile = lenF ? t0 : (lenL ? tL : tM0), c_kt = lenF ? k_first : 0;
  int slot = -1;
  unsigned c_par = 1;
  for (int it = 0; it < nkt; it++) {
    if (tid == 0 && it + LOOKAHEAD < nkt) issue(it + LOOKAHEAD);
    __syncwarp();
    if (++slot == STAGES) slot = 0;
    if (slot == 0) c_par ^= 1u;
    mbar_wait(full0 + 8 * slot, c_par);
    const c128 *a = reinterpret_cast<const c128 *>(smem_gen + slot * (2 * TILE_BYTES));
    const c128 *b = reinterpret_cast<const c128 *>(smem_gen + slot * (2 * TILE_BYTES) + TILE_BYTES);
#pragma unroll
    for (int ks = 0; ks < KG; ks++) {
      if (M3) {
        double ar[NB8], ai[NB8], as[NB8], br[NB8], bi[NB8], bs[NB8];
#pragma unroll
        for (int j = 0; j < NB8; j++) {
          c128 v = B_KMAJOR ? b[(ks * BN + wn0 + j * 8 + lr) * 4 + lk]
                            : b[(ks * 4 + lk) * LDM + wn0 + j * 8 + lr];
          br[j] = v.x;
          bi[j] = CONJ ? flip(v.y, p.b_sign) : v.y;
          bs[j] = br[j] + bi[j];
        }
#pragma unroll
        for (int i = 0; i < NB8; i++) {
          c128 v = A_KMAJOR ? a[(ks * BM + wm0 + i * 8 + lr) * 4 + lk]
                            : a[(ks * 4 + lk) * LDM + wm0 + i * 8 + lr];
          ar[i] = v.x;
          ai[i] = CONJ ? flip(v.y, p.a_sign) : v.y;
          as[i] = ar[i] + ai[i];
        }
        if (ks == KG - 1) {            // all operands of this slot are in registers: hand it back
          __syncwarp();
          if (lane == 0) mbar_arrive(empty0 + 8 * slot);
        }
#pragma unroll
        for (int i = 0; i < NB8; i++)
#pragma unroll
          for (int j = 0; j < NB8; j++) {
            dmma(cr[i][j][0], cr[i][j][1], ar[i], br[j]);
            dmma(ci[i][j][0], ci[i][j][1], ai[i], bi[j]);
            dmma(cs[M3 ? i : 0][M3 ? j : 0][0], cs[M3 ? i : 0][M3 ? j : 0][1], as[i], bs[j]);
          }
      } else {
      double ar[NB8], ai[NB8], nai[NB8], br[NB8], bi[NB8];
#pragma unroll
      for (int i = 0; i < NB8; i++) {
        c128 v = A_KMAJOR ? a[(ks * BM + wm0 + i * 8 + lr) * 4 + lk]
                          : a[(ks * 4 + lk) * LDM + wm0 + i * 8 + lr];
        ar[i] = v.x;
        ai[i] = CONJ ? flip(v.y, p.a_sign) : v.y;
        nai[i] = flip(v.y, CONJ ? na_sign : 0x80000000u);
      }
#pragma unroll
      for (int j = 0; j < NB8; j++) {
        c128 v = B_KMAJOR ? b[(ks * BN + wn0 + j * 8 + lr) * 4 + lk]
                          : b[(ks * 4 + lk) * LDM + wn0 + j * 8 + lr];
        br[j] = v.x;
        bi[j] = CONJ ? flip(v.y, p.b_sign) : v.y;
      }
      if (ks == KG - 1) {            // all operands of this slot are in registers: hand it back
        __syncwarp();
        if (lane == 0) mbar_arrive(empty0 + 8 * slot);
      }
#pragma unroll
      for (int i = 0; i < NB8; i++)
#pragma unroll
        for (int j = 0; j < NB8; j++) {
          dmma(cr[i][j][0], cr[i][j][1], ar[i], br[j]);
          dmma(ci[i][j][0], ci[i][j][1], ar[i], bi[j]);
        }
#pragma unroll
      for (int i = 0; i < NB8; i++)
#pragma unroll
        for (int j = 0; j < NB8; j++) {
          dmma(cr[i][j][0], cr[i][j][1], nai[i], bi[j]);
          dmma(ci[i][j][0], ci[i][j][1], ai[i], br[j]);
        }
      }
    }
    // ---- end of a segment? ----
    const bool whole = it >= lenFL;
    if (!(c_kt == ktiles - 1 || it == lenF - 1 || it == lenFL - 1)) { ++c_kt; continue; }
    if (whole) {
      const int bz = c_tile / tiles_mn, tr = c_tile - bz * tiles_mn;
      const int m0 = (tr / p.tiles_n) * BM, n0 = (tr % p.tiles_n) * BN;
      const int bin = bz % p.batch_inner, bo = bz / p.batch_inner;
      c128 *Cb = p.C + bin * p.c_bsi + bo * p.c_bso;
      // thread holds C(row = lane/4, cols = 2*(lane%4) + {0,1}) of every 8x8 block
#pragma unroll
      for (int i = 0; i < NB8; i++) {
        int m = m0 + wm0 + i * 8 + lr;
        if (m >= p.M) continue;
#pragma unroll
        for (int j = 0; j < NB8; j++) {
          int n = n0 + wn0 + j * 8 + 2 * lk;
          c128 *dst = Cb + (long long)m * p.ldc + n;
          if (n < p.N) dst[0] = fin(i, j, 0);
          if (n + 1 < p.N) dst[1] = fin(i, j, 1);
        }
      }
    } else {
      // partial tile: thread-native layout (element e = q * 128 + tid, q = (i*4 + j)*2 + h), coalesced
      const int which = it < lenF ? 0 : 1;
      c128 *sl = p.slots + (size_t)(2 * cta + which) * (BM * BN);
#pragma unroll
      for (int i = 0; i < NB8; i++)
#pragma unroll
        for (int j = 0; j < NB8; j++) {
          __stcg(sl + ((i * NB8 + j) * 2 + 0) * NTHREADS + tid, fin(i, j, 0));
          __stcg(sl + ((i * NB8 + j) * 2 + 1) * NTHREADS + tid, fin(i, j, 1));
        }
      __syncthreads();               // all stores of the CTA are ordered before thread 0's release
      if (tid == 0) {
        s_fix_tile[which] = c_tile;
        const int j1 = cta_of_unit(c_tile * ktiles + ktiles - 1, p.upc_base, p.upc_rem);
        red_release_add(p.cnt + j1, 1);
      }
    }
#pragma unroll
    for (int i = 0; i < NB8; i++)
#pragma unroll
      for (int j = 0; j < NB8; j++) {
        cr[i][j][0] = cr[i][j][1] = ci[i][j][0] = ci[i][j][1] = 0.0;
        if (M3) cs[M3 ? i : 0][M3 ? j : 0][0] = cs[M3 ? i : 0][M3 ? j : 0][1] = 0.0;
      }
    c_kt = 0;
    if (it + 1 == lenF && lenL) c_tile = tL;
    else if (it + 1 == lenFL) c_tile = tM0;
    else ++c_tile;
  }

  // ---- fix-up: reduce this CTA's slice of each tile it holds a partial segment of ----
  __syncthreads();
  for (int which = 0; which < 2; which++) {
    const int t = s_fix_tile[which];
    if (t < 0) continue;
    const int tu0 = t * ktiles;
    const int j0 = cta_of_unit(tu0, p.upc_base, p.upc_rem), j1 = cta_of_unit(tu0 + ktiles - 1, p.upc_base, p.upc_rem);
    const int nc = j1 - j0 + 1, me = cta - j0;
    if (tid == 0) while (ld_acquire(p.cnt + j1) < nc) {}
    __syncthreads();
    // slices are whole groups of 128 elements, so that element e of a slice belongs to thread e % 128
    // of the tile's thread-native layout whoever reduces it: the row / column decode is per thread
    const int chunk = ((BM * BN / NTHREADS + nc - 1) / nc) * NTHREADS;
    const int e_end = (me + 1) * chunk < BM * BN ? (me + 1) * chunk : BM * BN;
    const int bz = t / tiles_mn, tr = t - bz * tiles_mn;
    const int m0 = (tr / p.tiles_n) * BM, n0 = (tr % p.tiles_n) * BN;
    c128 *Cb = p.C + (bz % p.batch_inner) * p.c_bsi + (bz / p.batch_inner) * p.c_bso;
    // slot of contributor j: [0] if the tile holds j's first unit, else [1] (j began in an earlier
    // tile): only j0 can have begun earlier
    const int j0u0 = j0 * p.upc_base + (j0 < p.upc_rem ? j0 : p.upc_rem);
    const c128 *s0 = p.slots + (size_t)(2 * j0 + (j0u0 == tu0 ? 0 : 1)) * (BM * BN);
    const c128 *s1 = p.slots + (size_t)(2 * (j0 + 1)) * (BM * BN);
    const int fm0 = m0 + (warp / (BN / WN)) * WM + (lane >> 2), fn0 = n0 + (warp % (BN / WN)) * WN + 2 * (lane & 3);
    // four elements per thread and pass, all their loads in flight together (the fix-up is a chain
    // of L2 round trips: one element at a time it cost ~0.4 us per element and thread)
    constexpr int FU = 4;
    for (int eb = me * chunk + tid; eb < e_end; eb += FU * NTHREADS) {
      double sx[FU], sy[FU];
#pragma unroll
      for (int u = 0; u < FU; u++) {
        const int e = eb + u * NTHREADS;
        const c128 v0 = e < e_end ? __ldcg(s0 + e) : make_double2(0.0, 0.0);
        sx[u] = v0.x; sy[u] = v0.y;
      }
      for (int j = 0; j < nc - 1; j++) {
        const c128 *sj = s1 + (size_t)j * (2 * BM * BN);
#pragma unroll
        for (int u = 0; u < FU; u++) {
          const int e = eb + u * NTHREADS;
          const c128 v = e < e_end ? __ldcg(sj + e) : make_double2(0.0, 0.0);
          sx[u] += v.x; sy[u] += v.y;
        }
      }
#pragma unroll
      for (int u = 0; u < FU; u++) {
        const int e = eb + u * NTHREADS;
        if (e >= e_end) continue;
        const int q = e >> 7;                               // e & 127 == tid
        const int i = q / (2 * NB8), jb = (q >> 1) % NB8, h = q & 1;
        const int m = fm0 + i * 8, n = fn0 + jb * 8 + h;
        if (m < p.M && n < p.N) Cb[(long long)m * p.ldc + n] = make_double2(sx[u], sy[u]);
      }
    }
    __syncthreads();
    if (tid == 0) {
      if (atomicAdd(p.done + j1, 1) == nc - 1) { atomicExch(p.cnt + j1, 0); atomicExch(p.done + j1, 0); }
    }
  }
}

// The kernel proper.  SKIP = false: the body inlined, no test (every fixed-k launch: the headline path).
// SKIP = true (launches that carry a skip flag: the applies of an adaptive Krylov recurrence): the flag is
// tested first and the body is a function of its own -- with the test inlined in front of it ptxas spilled
// ~270 bytes in the 3-product instances, which sit at 244 of 255 registers; outlined it costs ~5 % instead.
template <bool A_KMAJOR, bool B_KMAJOR, bool CONJ, bool M3, int TB>
__device__ __noinline__ void zgemm_body_outlined(const CUtensorMap &tmA, const CUtensorMap &tmB, const KParams &p) {
  zgemm_body<A_KMAJOR, B_KMAJOR, CONJ, M3, TB>(tmA, tmB, p);
}
template <bool A_KMAJOR, bool B_KMAJOR, bool CONJ, bool M3, bool SKIP, int TB = 64>
__global__ void __launch_bounds__(NTHREADS, 2) zgemm_kernel(const __grid_constant__ CUtensorMap tmA,
                                                            const __grid_constant__ CUtensorMap tmB,
                                                            const __grid_constant__ KParams p) {
  if (SKIP) {
    // written by an earlier kernel of the stream, so every CTA reads the same value: all return or none does
    if (p.skip != nullptr && __ldcg(p.skip) != 0) return;
    zgemm_body_outlined<A_KMAJOR, B_KMAJOR, CONJ, M3, TB>(tmA, tmB, p);
  } else {
    zgemm_body<A_KMAJOR, B_KMAJOR, CONJ, M3, TB>(tmA, tmB, p);
  }
}

// Complex product as three real DMMA products per k-step (default) or four (TDVP_ZGEMM_4M=1 in the
// environment, or zgemm_set_mode(4)): see DESIGN.md 5, reading c15.  Process-wide by contract
// (include/tdvp.h, tdvp_set_gemm_products); atomic because handles on other host threads read it.
std::atomic<int> g_mode3m{1};

template <bool AK, bool BK_, bool CJ, bool M3>
void launch2(cudaStream_t st, const CUtensorMap &ta, const CUtensorMap &tb, const KParams &kp) {
  // cooperative: the CTAs of a cut tile wait for one another in the fix-up, so all must be resident
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(kp.G); cfg.blockDim = dim3(NTHREADS); cfg.dynamicSmemBytes = kp.tile == 32 ? SMEM_BYTES_32 : SMEM_BYTES; cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeCooperative; attr[0].val.cooperative = 1;
  // no tile is cut when the ranges are whole tiles: nobody waits for anybody, a plain launch will do
  const bool cut = kp.upc_rem != 0 || (kp.upc_base % kp.ktiles) != 0;
  cfg.attrs = attr; cfg.numAttrs = cut ? 1 : 0;
  if (kp.tile == 32) cudaLaunchKernelEx(&cfg, zgemm_kernel<AK, BK_, CJ, M3, true, 32>, ta, tb, kp);   // (tests its skip flag, if any)
  else if (kp.skip) cudaLaunchKernelEx(&cfg, zgemm_kernel<AK, BK_, CJ, M3, true>, ta, tb, kp);
  else cudaLaunchKernelEx(&cfg, zgemm_kernel<AK, BK_, CJ, M3, false>, ta, tb, kp);
  count_launch();
}
template <bool AK, bool BK_, bool CJ>
void launch1(cudaStream_t st, const CUtensorMap &ta, const CUtensorMap &tb, const KParams &kp) {
  if (g_mode3m.load(std::memory_order_relaxed)) launch2<AK, BK_, CJ, true>(st, ta, tb, kp);
  else launch2<AK, BK_, CJ, false>(st, ta, tb, kp);
}
template <bool AK, bool BK_>
void launch(cudaStream_t st, const CUtensorMap &ta, const CUtensorMap &tb, const KParams &kp) {
  if (kp.a_sign || kp.b_sign) launch1<AK, BK_, true>(st, ta, tb, kp);
  else launch1<AK, BK_, false>(st, ta, tb, kp);
}
template <bool AK, bool BK_>
void set_smem_attr() {
  cudaFuncSetAttribute(zgemm_kernel<AK, BK_, true, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
  cudaFuncSetAttribute(zgemm_kernel<AK, BK_, false, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
  cudaFuncSetAttribute(zgemm_kernel<AK, BK_, true, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
  cudaFuncSetAttribute(zgemm_kernel<AK, BK_, false, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
  cudaFuncSetAttribute(zgemm_kernel<AK, BK_, true, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
  cudaFuncSetAttribute(zgemm_kernel<AK, BK_, false, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
  cudaFuncSetAttribute(zgemm_kernel<AK, BK_, true, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
  cudaFuncSetAttribute(zgemm_kernel<AK, BK_, false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
  cudaFuncSetAttribute(zgemm_kernel<AK, BK_, true, true, true, 32>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES_32);
  cudaFuncSetAttribute(zgemm_kernel<AK, BK_, false, true, true, 32>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES_32);
  cudaFuncSetAttribute(zgemm_kernel<AK, BK_, true, false, true, 32>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES_32);
  cudaFuncSetAttribute(zgemm_kernel<AK, BK_, false, false, true, 32>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES_32);
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link-time libcuda).
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn g_encode = nullptr;
int g_no_5d = 0;       // set when the driver rejects a 5-D map once (or by TDVP_ZGEMM_NO_5D=1)

// Tensor map of one operand seen as doubles.  K-major (unit stride along k): dims (2K, rows, bi, bo),
// box (8 doubles = 4 complex, 64 rows); MN-major (unit stride along m/n): dims (2*rows, K, bi, bo),
// box (2*LDM doubles, BK).  Out-of-range box elements read as zero: ragged edges need no predicates.
bool encode_operand(CUtensorMap *tm, int tile, const c128 *base, bool kmajor, long long rows, long long K, long long ld /*complex*/,
                    int nbi, long long bsi, int nbo, long long bso) {
  cuuint64_t dims[4], strides[3];
  cuuint32_t box[4], estr[4] = {1, 1, 1, 1};
  dims[0] = (cuuint64_t)(kmajor ? 2 * K : 2 * rows);
  dims[1] = (cuuint64_t)(kmajor ? rows : K);
  if (dims[1] == 1) ld = (long long)(dims[0] / 2);   // a single row: any valid stride
  strides[0] = (cuuint64_t)ld * 16;
  const bool bi = nbi > 1 && bsi != 0, bo = nbo > 1 && bso != 0;
  dims[2] = bi ? nbi : 1; dims[3] = bo ? nbo : 1;
  const cuuint64_t dummy = strides[0] * dims[1];
  strides[1] = bi ? (cuuint64_t)bsi * 16 : dummy;
  strides[2] = bo ? (cuuint64_t)bso * 16 : dummy;
  box[0] = kmajor ? 8 : 2 * (tile + 2); box[1] = kmajor ? tile : BK; box[2] = 1; box[3] = 1;
  CUresult r = g_encode(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<c128 *>(base), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    char buf[320];
    snprintf(buf, sizeof buf, "cuTensorMapEncodeTiled failed (%d) for an operand at %p (must be 16-byte aligned): dims %llu %llu "
             "%llu %llu strides %llu %llu %llu box %u %u", (int)r, (const void *)base, (unsigned long long)dims[0],
             (unsigned long long)dims[1], (unsigned long long)dims[2], (unsigned long long)dims[3],
             (unsigned long long)strides[0], (unsigned long long)strides[1], (unsigned long long)strides[2], box[0], box[1]);
    sticky_error(TDVP_EINVAL, buf);
    return false;
  }
  return true;
}

// K-major operand with K a multiple of 4: dims (8 doubles of a k-group, rows, k-groups, bi, bo), box
// (8, 64, KG, 1, 1) -- written to shared memory as [k-group][row][4 complex], the layout the four
// separate boxes of the 4-D map produce, with one TMA instruction.  Returns false if the driver
// rejects the map (the caller then keeps the 4-D one).
bool encode_operand_5d(CUtensorMap *tm, int tile, const c128 *base, long long rows, long long K, long long ld /*complex*/,
                       int nbi, long long bsi, int nbo, long long bso) {
  if (K % 4 != 0 || g_no_5d) return false;
  cuuint64_t dims[5], strides[4];
  cuuint32_t box[5] = {8, (cuuint32_t)tile, (cuuint32_t)KG, 1, 1}, estr[5] = {1, 1, 1, 1, 1};
  dims[0] = 8; dims[1] = (cuuint64_t)rows; dims[2] = (cuuint64_t)(K / 4);
  if (rows == 1) ld = K;
  strides[0] = (cuuint64_t)ld * 16;      // rows
  strides[1] = 64;                       // k-groups
  const bool bi = nbi > 1 && bsi != 0, bo = nbo > 1 && bso != 0;
  dims[3] = bi ? nbi : 1; dims[4] = bo ? nbo : 1;
  const cuuint64_t dummy = strides[0] * dims[1];
  strides[2] = bi ? (cuuint64_t)bsi * 16 : dummy;
  strides[3] = bo ? (cuuint64_t)bso * 16 : dummy;
  CUtensorMap tmp;
  CUresult r = g_encode(&tmp, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, const_cast<c128 *>(base), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { g_no_5d = 1; return false; }
  *tm = tmp;
  return true;
}

// Per-stream scheduling state: partial-tile slots and the two counter arrays.  Kernels of one
// stream run one after the other, so one context per stream is enough; it is created outside any
// stream capture (zgemm_prepare_stream) because cudaMalloc is not allowed while capturing.
struct StreamCtx { c128 *slots = nullptr; int *cnt = nullptr; int *done = nullptr; int refs = 0; bool alias = false; int cap = 0; };
std::mutex g_ctx_mu;
std::unordered_map<cudaStream_t, StreamCtx> g_ctx;
int g_slots = 0;      // resident CTAs of zgemm_kernel on this device (2 per SM)
int g_sms = 0;

// Looks the context of a stream up; `create` makes it if missing (cudaMalloc: not inside a capture),
// `add_ref` counts one more owner (a handle).  Failures leave the thread's sticky error.
StreamCtx *get_ctx(cudaStream_t st, bool create, bool add_ref = false) {
  std::lock_guard<std::mutex> lk(g_ctx_mu);
  auto it = g_ctx.find(st);
  if (it != g_ctx.end()) { if (add_ref) it->second.refs++; return &it->second; }
  if (!create) return nullptr;
  StreamCtx c;
  cudaError_t e = cudaMalloc(&c.slots, (size_t)2 * g_slots * BM * BN * sizeof(c128));
  if (e == cudaSuccess) {
    e = cudaMalloc(&c.cnt, (size_t)2 * g_slots * sizeof(int));
    if (e != cudaSuccess) cudaFree(c.slots);
  }
  if (e == cudaSuccess) {
    e = cudaMemset(c.cnt, 0, (size_t)2 * g_slots * sizeof(int));
    if (e != cudaSuccess) { cudaFree(c.slots); cudaFree(c.cnt); }
  }
  if (e != cudaSuccess) {
    cudaGetLastError();
    sticky_error(e == cudaErrorMemoryAllocation ? TDVP_ENOMEM : TDVP_ECUDA,
                 std::string("GEMM scheduling context of the stream (first use must be outside a stream capture): ") +
                     cudaGetErrorString(e));
    return nullptr;
  }
  c.done = c.cnt + g_slots;
  c.refs = add_ref ? 1 : 0;
  return &(g_ctx[st] = c);
}

// CTAs for `units` (tile, k-tile) units: the count that minimises the modelled time, in units of
// one k-tile on an SM of its own.  Two CTAs sharing an SM take twice as long per unit (one CTA
// alone reaches ~90 % of the pipe); cutting tiles costs the publish + slice reduction, measured at
// about 8 us = four units whatever the depth of the cut.
double g_split_cost = 5.0;
// unit_cost: time of one (tile, k-tile) unit relative to a 64 x 64 unit; split: cost of cutting tiles
int choose_grid(long long units, int ktiles, double unit_cost = 1.0, double split = -1.0, double *best_out = nullptr, int cap = 0) {
  int best_g = 1;
  double best = 1e300;
  if (split < 0.0) split = g_split_cost;
  const int slots = cap > 0 && cap < g_slots ? cap : g_slots;
  const int gmax = units < slots ? (int)units : slots;
  for (int g = 1; g <= gmax; g++) {
    const long long upc = (units + g - 1) / g;
    const bool cut = (units % g != 0) || (upc % ktiles != 0);
    const double cost = unit_cost * (double)upc * (g > g_sms ? 2.0 : 1.1) + (cut ? split : 0.0) - 1e-6 * g;
    if (cost < best) { best = cost; best_g = g; }
  }
  if (best_out) *best_out = best;
  return best_g;
}
// Tile edge of a launch.  A 64 x 64 tile keeps the DMMA pipe busiest (48 DMMAs per 8 fragment loads), but a
// small product has too few of them to fill 148 SMs without cutting every tile many times (the bond operator of
// Eq. 44 at M = 128: 4 output tiles, K = 768 -- a 48-way cut whose fix-up costs more than the product).  With
// 32 x 32 tiles there are four times as many, each unit a quarter of the DMMAs at ~0.4 of the time (12 DMMAs per
// 4 fragment loads), and a cut tile's fix-up moves a quarter of the data.  The same cost model as choose_grid
// picks whichever is cheaper; TDVP_ZGEMM_TILE=64 / 32 forces one (diagnostic).
int g_force_tile = 0;
double g_unit32 = 0.4, g_split32 = 2.0;
int choose_tile(long long M, long long N, long long batch, int ktiles, int *G, int cap) {
  double c64 = 0.0, c32 = 0.0;
  const long long u64 = ((M + 63) / 64) * ((N + 63) / 64) * batch * ktiles, u32 = ((M + 31) / 32) * ((N + 31) / 32) * batch * ktiles;
  const int g64 = choose_grid(u64, ktiles, 1.0, -1.0, &c64, cap), g32 = choose_grid(u32, ktiles, g_unit32, g_split32, &c32, cap);
  const bool use32 = g_force_tile == 32 || (g_force_tile == 0 && c32 < c64);
  *G = use32 ? g32 : g64;
  return use32 ? 32 : 64;
}

}  // namespace

void zgemm_configure() {
  set_smem_attr<true, true>(); set_smem_attr<true, false>(); set_smem_attr<false, true>(); set_smem_attr<false, false>();
  int dev = 0, per_sm = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&g_sms, cudaDevAttrMultiProcessorCount, dev);
  int per_sm4 = 0;
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, zgemm_kernel<true, true, true, true, false>, NTHREADS, SMEM_BYTES);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm4, zgemm_kernel<true, true, true, false, false>, NTHREADS, SMEM_BYTES);
  if (per_sm4 < per_sm) per_sm = per_sm4;
  if (const char *es = getenv("TDVP_ZGEMM_SPLIT_COST")) g_split_cost = atof(es);
  if (const char *e5 = getenv("TDVP_ZGEMM_NO_5D")) g_no_5d = e5[0] == '1';
  if (const char *et = getenv("TDVP_ZGEMM_TILE")) g_force_tile = atoi(et);
  if (const char *eu = getenv("TDVP_ZGEMM_UNIT32")) g_unit32 = atof(eu);
  if (const char *eu = getenv("TDVP_ZGEMM_SPLIT32")) g_split32 = atof(eu);
  const char *e4 = getenv("TDVP_ZGEMM_4M");
  if (e4 && e4[0] == '1') g_mode3m.store(0);
  if (per_sm < 1) per_sm = 1;
  if (per_sm > 2) per_sm = 2;
  if (g_sms < 1) g_sms = 1;
  g_slots = g_sms * per_sm;
  void *fn = nullptr;
  cudaDriverEntryPointQueryResult q;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) == cudaSuccess &&
      q == cudaDriverEntryPointSuccess)
    g_encode = reinterpret_cast<EncodeTiledFn>(fn);
}

void zgemm_set_mode(int products) { configure_kernels_once(); g_mode3m.store(products == 4 ? 0 : 1); }
int zgemm_get_mode() { configure_kernels_once(); return g_mode3m.load() ? 3 : 4; }

// Launches on `st` use at most `max_ctas` CTAs (0 = all the device holds).  For queues that run beside long cluster
// kernels: a cut GEMM is a cooperative launch, which starts only when ALL its CTAs fit at once -- with every slot of
// the device in its grid it would wait for a 2 ms bond-unfolding kernel on 8 SMs to end.
void zgemm_set_stream_cap(cudaStream_t st, int max_ctas) {
  std::lock_guard<std::mutex> lk(g_ctx_mu);
  auto it = g_ctx.find(st);
  if (it != g_ctx.end()) it->second.cap = max_ctas;
}
int zgemm_device_sms() { configure_kernels_once(); return g_sms; }

// One more owner (a handle) of the stream's context; created if missing.
int zgemm_prepare_stream(cudaStream_t st) {
  configure_kernels_once();
  return get_ctx(st, true, true) ? TDVP_OK : TDVP_ECUDA;  // on failure the sticky error says why
}

void zgemm_alias_stream(cudaStream_t alias, cudaStream_t of) {
  configure_kernels_once();
  StreamCtx *c = get_ctx(of, true);
  if (!c) return;
  std::lock_guard<std::mutex> lk(g_ctx_mu);
  StreamCtx a = *c;
  a.alias = true; a.refs = 0;
  g_ctx[alias] = a;
}

void zgemm_forget_stream(cudaStream_t alias) {
  std::lock_guard<std::mutex> lk(g_ctx_mu);
  g_ctx.erase(alias);
}

// An owner of the stream's context is gone; the last one frees it (the caller has synchronised the
// stream).  Contexts made implicitly by a handle-less call keep refs == 0 and live until exit.
void zgemm_release_stream(cudaStream_t st) {
  std::lock_guard<std::mutex> lk(g_ctx_mu);
  auto it = g_ctx.find(st);
  if (it == g_ctx.end() || it->second.alias) return;
  if (--it->second.refs > 0) return;
  cudaFree(it->second.slots);
  cudaFree(it->second.cnt);
  g_ctx.erase(it);
}

int zgemm(cudaStream_t st, const ZGemm &p) {
  if (p.M <= 0 || p.N <= 0) return TDVP_OK;
  if (!g_encode) {
    sticky_error(TDVP_ECUDA, "no cuTensorMapEncodeTiled driver entry point (CUDA driver too old for TMA)");
    return TDVP_ECUDA;
  }
  StreamCtx *ctx = get_ctx(st, true);
  if (!ctx) return TDVP_ECUDA;                            // the sticky error says why
  const bool ak = (p.a_ks == 1), bk = (p.b_ks == 1);
  const long long batch = (long long)p.batch_inner * p.batch_outer;
  int ktiles = (p.K + BK - 1) / BK;
  if (ktiles < 1) ktiles = 1;
  int G = 1;
  const int tile = choose_tile(p.M, p.N, batch, ktiles, &G, ctx->cap);
  CUtensorMap ta, tb;
  if (!encode_operand(&ta, tile, p.A, ak, p.M, p.K, ak ? p.a_ms : p.a_ks, p.batch_inner, p.a_bsi, p.batch_outer, p.a_bso) ||
      !encode_operand(&tb, tile, p.B, bk, p.N, p.K, bk ? p.b_ns : p.b_ks, p.batch_inner, p.b_bsi, p.batch_outer, p.b_bso))
    return TDVP_EINVAL;
  if ((reinterpret_cast<size_t>(p.C) & 15) != 0) {
    sticky_error(TDVP_EINVAL, "GEMM output is not 16-byte aligned");
    return TDVP_EINVAL;
  }
  KParams kp;
  kp.a5 = ak && encode_operand_5d(&ta, tile, p.A, p.M, p.K, p.a_ms, p.batch_inner, p.a_bsi, p.batch_outer, p.a_bso) ? 1 : 0;
  kp.b5 = bk && encode_operand_5d(&tb, tile, p.B, p.N, p.K, p.b_ns, p.batch_inner, p.b_bsi, p.batch_outer, p.b_bso) ? 1 : 0;
  kp.tile = tile;
  kp.C = p.C;
  kp.M = p.M; kp.N = p.N; kp.K = p.K;
  kp.ldc = p.ldc;
  kp.batch_inner = p.batch_inner;
  kp.c_bsi = p.c_bsi; kp.c_bso = p.c_bso;
  kp.a_batched_i = p.batch_inner > 1 && p.a_bsi != 0; kp.a_batched_o = p.batch_outer > 1 && p.a_bso != 0;
  kp.b_batched_i = p.batch_inner > 1 && p.b_bsi != 0; kp.b_batched_o = p.batch_outer > 1 && p.b_bso != 0;
  kp.a_sign = p.conjA ? 0x80000000u : 0u;
  kp.b_sign = p.conjB ? 0x80000000u : 0u;
  kp.tiles_m = (p.M + tile - 1) / tile;
  kp.tiles_n = (p.N + tile - 1) / tile;
  const long long tiles = (long long)kp.tiles_m * kp.tiles_n * batch;
  kp.ktiles = ktiles;
  const long long units = tiles * ktiles;
  kp.G = G;
  kp.upc_base = (int)(units / kp.G);
  kp.upc_rem = (int)(units % kp.G);
  kp.slots = ctx->slots; kp.cnt = ctx->cnt; kp.done = ctx->done;
  kp.skip = p.skip;
  ProfScope ps(st, PH_ZGEMM);
  if (ak && bk) launch<true, true>(st, ta, tb, kp);
  else if (ak && !bk) launch<true, false>(st, ta, tb, kp);
  else if (!ak && bk) launch<false, true>(st, ta, tb, kp);
  else launch<false, false>(st, ta, tb, kp);
  return TDVP_OK;
}
