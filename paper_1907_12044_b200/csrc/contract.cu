// contract.cu -- local contractions of the TDVP hot path as GEMM / W-stage / GEMM pipelines.
//   heff_apply : Eq. 29 applied as in Eq. 43
//   env_update : Eq. 30-32
//   bond_apply : Eq. 44
// "contract small matrices one by one instead of explicitly constructing the large tensors"
// (PAPER.md:253).  All row-major views below need no materialised transposes (zgemm takes
// strides); the W stage skips the zeros of the MPO (wstage.cu).
//
// Order by cost: for one site both GEMM orders (L first or R first) cost the same
// 8 (Ml^2 Dl d Mr + Ml d Dr Mr^2) flops; the intermediates are Ml*Dl*d*Mr then Ml*d*Dr*Mr for
// "L first" and the reverse for "R first".  heff and envL run L first, envR runs R first, so that
// each environment update ends in the GEMM that produces its own layout directly.
#include "common.cuh"

namespace {
inline size_t up256(size_t x) { return (x + 255) & ~size_t(255); }

ZGemm g_stage1_left(int Ml, int Mr, int d, int Dl, const c128 *L, const c128 *A, c128 *T1) {
  // T1[(a,w)][(t,y)] = sum_x L[(a,w)][x] A[x][(t,y)]
  ZGemm g{};
  g.A = L; g.B = A; g.C = T1;
  g.M = Ml * Dl; g.N = d * Mr; g.K = Ml;
  g.a_ms = Ml; g.a_ks = 1; g.b_ks = (long long)d * Mr; g.b_ns = 1; g.ldc = (long long)d * Mr;
  return g;
}
ZGemm g_stage3_heff(int Ml, int Mr, int d, int Dr, const c128 *T2, const c128 *R, c128 *out) {
  // out[(a,s)][b] = sum_{(v,y)} T2[(a,s)][(v,y)] R[b][(v,y)]
  ZGemm g{};
  g.A = T2; g.B = R; g.C = out;
  g.M = Ml * d; g.N = Mr; g.K = Dr * Mr;
  g.a_ms = (long long)Dr * Mr; g.a_ks = 1; g.b_ns = (long long)Dr * Mr; g.b_ks = 1; g.ldc = Mr;
  return g;
}
ZGemm g_stage3_envL(int Ml, int Mr, int d, int Dr, const c128 *A, const c128 *T2, c128 *Lout) {
  // L'[b][(v,y)] = sum_{(a,s)} conj(A[(a,s)][b]) T2[(a,s)][(v,y)]
  ZGemm g{};
  g.A = A; g.B = T2; g.C = Lout;
  g.M = Mr; g.N = Dr * Mr; g.K = Ml * d;
  g.a_ms = 1; g.a_ks = Mr; g.conjA = 1;
  g.b_ks = (long long)Dr * Mr; g.b_ns = 1; g.ldc = (long long)Dr * Mr;
  return g;
}
ZGemm g_stage1_right(int Ml, int Mr, int d, int Dr, const c128 *A, const c128 *R, c128 *T1) {
  // T1[(x,t)][v][b] = sum_y A[(x,t)][y] R[b][v][y], batched over v
  ZGemm g{};
  g.A = A; g.B = R; g.C = T1;
  g.M = Ml * d; g.N = Mr; g.K = Mr;
  g.a_ms = Mr; g.a_ks = 1; g.b_ns = (long long)Dr * Mr; g.b_ks = 1; g.ldc = (long long)Dr * Mr;
  g.batch_inner = Dr; g.a_bsi = 0; g.b_bsi = Mr; g.c_bsi = Mr;
  return g;
}
ZGemm g_stage3_envR(int Ml, int Mr, int d, int Dl, const c128 *A, const c128 *T2, c128 *Rout) {
  // R'[a][(w,x)] = sum_{(s,b)} conj(A[a][(s,b)]) T2[(w,x)][(s,b)]
  ZGemm g{};
  g.A = A; g.B = T2; g.C = Rout;
  g.M = Ml; g.N = Dl * Ml; g.K = d * Mr;
  g.a_ms = (long long)d * Mr; g.a_ks = 1; g.conjA = 1;
  g.b_ns = (long long)d * Mr; g.b_ks = 1; g.ldc = (long long)Dl * Ml;
  return g;
}
ZGemm g_bond1(int Ml, int Mr, int Dw, const c128 *L, const c128 *D, c128 *T) {
  // T[(a,w)][y] = sum_x L[(a,w)][x] D[x][y]
  ZGemm g{};
  g.A = L; g.B = D; g.C = T;
  g.M = Ml * Dw; g.N = Mr; g.K = Ml;
  g.a_ms = Ml; g.a_ks = 1; g.b_ks = Mr; g.b_ns = 1; g.ldc = Mr;
  return g;
}
ZGemm g_bond2(int Ml, int Mr, int Dw, const c128 *T, const c128 *R, c128 *out) {
  // out[a][b] = sum_{(w,y)} T[a][(w,y)] R[b][(w,y)]
  ZGemm g{};
  g.A = T; g.B = R; g.C = out;
  g.M = Ml; g.N = Mr; g.K = Dw * Mr;
  g.a_ms = (long long)Dw * Mr; g.a_ks = 1; g.b_ns = (long long)Dw * Mr; g.b_ks = 1; g.ldc = Mr;
  return g;
}
}  // namespace

size_t heff_ws_bytes(int Ml, int Mr, int d, int Dl, int Dr) {
  size_t t1 = (size_t)Ml * Dl * d * Mr, t2 = (size_t)Ml * d * Dr * Mr;
  return up256(t1 * 16) + up256(t2 * 16) + 256;
}

void heff_apply(cudaStream_t st, int Ml, int Mr, int d, int Dl, int Dr, const c128 *L,
                const WSparse &W, const c128 *A, const c128 *R, c128 *out, void *ws, cudaEvent_t w_ready, const int *skip) {
  size_t t1 = (size_t)Ml * Dl * d * Mr, t2 = (size_t)Ml * d * Dr * Mr;
  char *p = reinterpret_cast<char *>(up256(reinterpret_cast<size_t>(ws)));
  c128 *T1 = reinterpret_cast<c128 *>(p); p += up256(t1 * 16);
  c128 *T2 = reinterpret_cast<c128 *>(p);
  ZGemm g1 = g_stage1_left(Ml, Mr, d, Dl, L, A, T1), g3 = g_stage3_heff(Ml, Mr, d, Dr, T2, R, out);
  g1.skip = g3.skip = skip;
  zgemm(st, g1);
  if (w_ready) cudaStreamWaitEvent(st, w_ready, 0);
  wstage_left(st, W, Ml, Mr, T1, T2, skip);
  zgemm(st, g3);
}

void heff_apply_staged(cudaStream_t st, int Ml, int Mr, int d, int Dl, int Dr, const c128 *L, const c128 *W_dense,
                       void *wmem, double zero_tol, const c128 *A, const c128 *R, c128 *out, void *ws,
                       int nsl, const cudaEvent_t *ev_l, cudaEvent_t ev_w, cudaEvent_t ev_r) {
  size_t t1 = (size_t)Ml * Dl * d * Mr, t2 = (size_t)Ml * d * Dr * Mr;
  char *p = reinterpret_cast<char *>(up256(reinterpret_cast<size_t>(ws)));
  c128 *T1 = reinterpret_cast<c128 *>(p); p += up256(t1 * 16);
  c128 *T2 = reinterpret_cast<c128 *>(p);
  for (int s = 0; s < nsl; s++) {
    const int a0 = (int)((long long)Ml * s / nsl), a1 = (int)((long long)Ml * (s + 1) / nsl);
    cudaStreamWaitEvent(st, ev_l[s], 0);
    if (a1 == a0) continue;
    ZGemm g = g_stage1_left(Ml, Mr, d, Dl, L + (size_t)a0 * Dl * Ml, A, T1 + (size_t)a0 * Dl * d * Mr);
    g.M = (a1 - a0) * Dl;
    zgemm(st, g);
  }
  cudaStreamWaitEvent(st, ev_w, 0);
  WSparse W;
  wsparse_build(st, W, wmem, Dl, d, Dr, W_dense, zero_tol);
  wstage_left(st, W, Ml, Mr, T1, T2);
  cudaStreamWaitEvent(st, ev_r, 0);
  zgemm(st, g_stage3_heff(Ml, Mr, d, Dr, T2, R, out));
}

size_t heff2_ws_bytes(int Ml, int Mr, int d1, int d2, int Dl, int Dm, int Dr) {
  const size_t per = (size_t)Ml * d1 * d2 * Mr;
  const size_t big = per * (size_t)(Dl > Dm ? (Dl > Dr ? Dl : Dr) : (Dm > Dr ? Dm : Dr));
  return 2 * up256(big * 16) + 256;
}

void heff2_apply(cudaStream_t st, int Ml, int Mr, int d1, int d2, int Dl, int Dm, int Dr, const c128 *L, const WSparse &W1,
                 const WSparse &W2, const c128 *Theta, const c128 *R, c128 *out, void *ws, const int *skip) {
  const size_t per = (size_t)Ml * d1 * d2 * Mr;
  const size_t big = per * (size_t)(Dl > Dm ? (Dl > Dr ? Dl : Dr) : (Dm > Dr ? Dm : Dr));
  char *p = reinterpret_cast<char *>(up256(reinterpret_cast<size_t>(ws)));
  c128 *Ta = reinterpret_cast<c128 *>(p); p += up256(big * 16);
  c128 *Tb = reinterpret_cast<c128 *>(p);
  // T1[(a,w),(t1,t2,y)] = L Theta: stage 1 with the pair (t1,t2) as one physical index
  ZGemm g1 = g_stage1_left(Ml, Mr, d1 * d2, Dl, L, Theta, Ta);
  g1.skip = skip;
  zgemm(st, g1);
  // site i:     T2[a, s1, u, (t2,y)] = sum_{w,t1} W1[w,s1,t1,u] T1[a, w, t1, (t2,y)]   (panel rows of length d2 Mr)
  wstage_left(st, W1, Ml, d2 * Mr, Ta, Tb, skip);
  // site i + 1: T3[(a,s1), s2, v, y] = sum_{u,t2} W2[u,s2,t2,v] T2[(a,s1), u, t2, y]    (batch index (a,s1))
  wstage_left(st, W2, Ml * d1, Mr, Tb, Ta, skip);
  // out[((a,s1),s2), b] = sum_{(v,y)} T3[((a,s1),s2), (v,y)] R[b, (v,y)]
  ZGemm g3 = g_stage3_heff(Ml * d1, Mr, d2, Dr, Ta, R, out);
  g3.skip = skip;
  zgemm(st, g3);
}

size_t env_ws_bytes(int Ml, int Mr, int d, int Dl, int Dr) {
  size_t t1 = (size_t)Ml * Dl * d * Mr, t2 = (size_t)Ml * d * Dr * Mr;
  size_t big = t1 > t2 ? t1 : t2;
  return 2 * up256(big * 16) + 256;
}

void env_update(cudaStream_t st, int side, int Ml, int Mr, int d, int Dl, int Dr,
                const c128 *env_in, const WSparse &W, const c128 *A, c128 *env_out, void *ws, cudaEvent_t w_ready) {
  size_t t1 = (size_t)Ml * Dl * d * Mr, t2 = (size_t)Ml * d * Dr * Mr;
  size_t big = t1 > t2 ? t1 : t2;
  char *p = reinterpret_cast<char *>(up256(reinterpret_cast<size_t>(ws)));
  c128 *T1 = reinterpret_cast<c128 *>(p); p += up256(big * 16);
  c128 *T2 = reinterpret_cast<c128 *>(p);
  if (side == 0) {
    zgemm(st, g_stage1_left(Ml, Mr, d, Dl, env_in, A, T1));
    if (w_ready) cudaStreamWaitEvent(st, w_ready, 0);
    wstage_left(st, W, Ml, Mr, T1, T2);
    zgemm(st, g_stage3_envL(Ml, Mr, d, Dr, A, T2, env_out));
  } else {
    zgemm(st, g_stage1_right(Ml, Mr, d, Dr, A, env_in, T1));
    if (w_ready) cudaStreamWaitEvent(st, w_ready, 0);
    wstage_right(st, W, Ml, Mr, T1, T2);
    zgemm(st, g_stage3_envR(Ml, Mr, d, Dl, A, T2, env_out));
  }
}

size_t bond_ws_bytes(int Ml, int Mr, int Dw) {
  size_t t = (size_t)Ml * Dw * Mr;
  return up256(t * 16) + 256;
}

void bond_apply(cudaStream_t st, int Ml, int Mr, int Dw, const c128 *L, const c128 *D,
                const c128 *R, c128 *out, void *ws, const int *skip) {
  size_t t = (size_t)Ml * Dw * Mr;
  char *p = reinterpret_cast<char *>(up256(reinterpret_cast<size_t>(ws)));
  c128 *T = reinterpret_cast<c128 *>(p);
  ZGemm g1 = g_bond1(Ml, Mr, Dw, L, D, T), g2 = g_bond2(Ml, Mr, Dw, T, R, out);
  g1.skip = g2.skip = skip;
  zgemm(st, g1);
  zgemm(st, g2);
}
