/*
 * tdvp.h -- C ABI of libtdvp.so: the data-parallel hot path of TDVP time evolution of a matrix
 * product state (MPS) under a matrix product operator (MPO), arXiv:1907.12044, written for one
 * NVIDIA B200 (sm_100a).  Every operation below runs in hand-written CUDA kernels; there is no CPU
 * fallback.  Citations are PAPER.md:<line> plus the equation / section the line falls in.
 *
 * Conventions (BASELINE.json north_star)
 *   complex128 everywhere, interleaved (re, im), C-contiguous arrays (last index fastest):
 *     L[a, w, x]   left  environment block h[1:i-1]  (Eq. 30-32), [Ml, Dl, Ml]
 *     R[b, v, y]   right environment block h[i+1:N]                                , [Mr, Dr, Mr]
 *                  first bond index = bra (conjugated) side, last = ket side
 *     W[w, s, t, v] MPO site tensor (Eq. 11), [Dl, d, d, Dr], s = bra/output
 *                  physical index, t = ket/input physical index
 *     A[x, t, y]   MPS site tensor (Eq. 1), [Ml, d, Mr]
 *   hbar = 1; dt is in the inverse of the MPO's energy unit (the caller converts units).
 *
 * Pointers: every argument says HOST or DEVICE.  The library copies what it keeps; the caller
 * keeps ownership of everything it passes in.  One handle = one CUDA stream = not thread safe;
 * several handles may coexist.  No call blocks on the stream unless it says so.
 *
 * Errors: every int-returning call returns TDVP_OK (0) or a negative TDVP_E* code and stores a
 * message retrievable with tdvp_last_error(h) (h may be NULL: the last error of the calling
 * thread's handle-less calls).  No exceptions or signals cross the boundary.  DEVICE pointers to
 * complex data must be 16-byte aligned (TDVP_EINVAL from the call that enqueues the first GEMM on
 * them).  Conditions only a kernel can detect (a bond SVD that ran out of Jacobi sweeps) are
 * recorded on the device and returned as TDVP_ESTATE by the NEXT blocking call on that handle
 * (tdvp_sync, tdvp_populations, tdvp_observe, tdvp_norm_energy, tdvp_get_mps, tdvp_mu_derivative,
 * tdvp_step_mu with err_est), which also clears them.
 */
#ifndef TDVP_H
#define TDVP_H

#ifdef __cplusplus
extern "C" {
#endif

#define TDVP_OK        0
#define TDVP_EINVAL   -1   /* bad shape, null pointer, non-canonical MPS, unsupported size        */
#define TDVP_ENOMEM   -2   /* device or host allocation failed                                   */
#define TDVP_ECUDA    -3   /* a CUDA call failed; tdvp_last_error has the CUDA error string      */
#define TDVP_ESTATE   -4   /* call not valid in the handle's current gauge / state               */

#define TDVP_MAX_KRYLOV 64

typedef struct tdvp_handle tdvp_handle;            /* opaque; owns all device state             */
typedef struct { double re, im; } tdvp_c128;       /* interleaved complex128                    */

typedef struct {
  int    krylov_dim;   /* k of the Lanczos exponential: the dimension used when
                          krylov_tol = 0, the largest allowed when > 0; default 10; <= 64        */
  double krylov_tol;   /* 0 (default): fixed dimension.  > 0: adaptive dimension (PAPER.md:292,
                          "continues until |Psi(t+tau)> converges"; the paper gives no criterion,
                          reading c11): stop at the first j with beta_j |[exp(z T_j) e_1]_j| < tol,
                          decided on the device; applies to purely imaginary z only             */
  double mu_eps;       /* epsilon of Eq. 38; default 1e-10                    */
  double w_zero_tol;   /* |W| <= tol is a structural zero of the MPO; default 0 (exact zeros)    */
  int    flags;        /* TDVP_FLAG_* below                                                      */
} tdvp_options;

#define TDVP_FLAG_SKIP_CANONICAL_CHECK 1  /* tdvp_create / tdvp_set_mps do not verify Eq. 8      */
#define TDVP_FLAG_NO_GRAPH             2  /* step drivers enqueue kernels directly (no CUDA graph)*/

void tdvp_default_options(tdvp_options *opt);

/* ---- handles ---------------------------------------------------------------------------- */

/* A handle without a chain: stream + workspace for the stateless calls below.
   cuda_stream: a cudaStream_t (NULL = the legacy default stream). */
int tdvp_create_context(tdvp_handle **out, const tdvp_options *opt /*HOST, nullable*/,
                        void *cuda_stream);

/* tdvp_create(mpo, mps): the paper's problem statement -- an MPO H (Eq. 11 / Eq. 45) and an MPS
   (Eq. 1) to be evolved.
     n_sites            number of sites N
     phys_dim[N]        HOST, d_i
     mpo_bond[N+1]      HOST, MPO bond dimensions, mpo_bond[0] = mpo_bond[N] = 1
     mpo[N]             HOST array of pointers; mpo[i] -> W_i[mpo_bond[i], d_i, d_i, mpo_bond[i+1]]
     mps_bond[N+1]      HOST, MPS bond dimensions, mps_bond[0] = mps_bond[N] = 1, and every
                        bond must satisfy M_i <= d_i * M_{i+1} and M_{i+1} <= M_i * d_i (so that
                        each gauge move is a tall-or-square QR)
     mps[N]             HOST array of pointers; mps[i] -> A_i[mps_bond[i], d_i, mps_bond[i+1]]
     on_device          0: the tensors pointed to are in HOST memory; 1: in DEVICE memory
   The MPS must be right-canonical (Eq. 8) on sites 1..N-1 with the gauge centre
   at site 0; this is checked to 1e-10 (TDVP_EINVAL) unless TDVP_FLAG_SKIP_CANONICAL_CHECK.
   All tensors are copied into device memory owned by the handle; all right environment blocks
   h[i+1:N] (Eq. 31-32) are built and kept resident.  Blocks on the stream before returning. */
int tdvp_create(tdvp_handle **out, int n_sites, const int *phys_dim,
                const int *mpo_bond, const tdvp_c128 *const *mpo,
                const int *mps_bond, const tdvp_c128 *const *mps,
                int on_device, const tdvp_options *opt /*HOST, nullable*/, void *cuda_stream);
int tdvp_destroy(tdvp_handle *h);

/* ---- stateless contractions on caller-provided DEVICE buffers ---------------------------- */
/* h may be NULL (legacy default stream, a library-owned workspace) or any handle (its stream
   and workspace).  Buffers must not overlap.  Enqueue only.                                   */

/* out[a,s,b] = sum_{w,x,t,v,y} L[a,w,x] W[w,s,t,v] A[x,t,y] R[b,v,y]
   (H[i] applied to a site tensor: Eq. 29, used as in Eq. 43). */
int tdvp_apply_heff(tdvp_handle *h, int Ml, int Mr, int d, int Dl, int Dr,
                    const tdvp_c128 *L /*DEVICE [Ml,Dl,Ml]*/, const tdvp_c128 *W /*DEVICE [Dl,d,d,Dr]*/,
                    const tdvp_c128 *A /*DEVICE [Ml,d,Mr]*/,  const tdvp_c128 *R /*DEVICE [Mr,Dr,Mr]*/,
                    tdvp_c128 *out /*DEVICE [Ml,d,Mr]*/);

/* Same operation with HOST buffers (all five pointers HOST, pageable or pinned): copies L, W, A, R
   to the device on the handle's stream, applies H[i], copies `out` back and BLOCKS until it has
   arrived.  This is the end-to-end entry bench.py times (h2d + kernels + d2h). */
int tdvp_apply_heff_host(tdvp_handle *h, int Ml, int Mr, int d, int Dl, int Dr,
                         const tdvp_c128 *L, const tdvp_c128 *W, const tdvp_c128 *A,
                         const tdvp_c128 *R, tdvp_c128 *out);

/* Environment update (Eq. 30-32).
   side = 0: env_in = L[Ml,Dl,Ml], env_out = L'[b,v,y] = sum conj(A[a,s,b]) L[a,w,x] W[w,s,t,v] A[x,t,y]   ([Mr,Dr,Mr])
   side = 1: env_in = R[Mr,Dr,Mr], env_out = R'[a,w,x] = sum conj(A[a,s,b]) W[w,s,t,v] A[x,t,y] R[b,v,y]   ([Ml,Dl,Ml]) */
int tdvp_update_env(tdvp_handle *h, int side, int Ml, int Mr, int d, int Dl, int Dr,
                    const tdvp_c128 *env_in /*DEVICE*/, const tdvp_c128 *W /*DEVICE [Dl,d,d,Dr]*/,
                    const tdvp_c128 *A /*DEVICE [Ml,d,Mr]*/, tdvp_c128 *env_out /*DEVICE*/);

/* Bond (zero-site) operator of the backward step (Eq. 44):
   out[a,b] = sum_{w,x,y} L[a,w,x] D[x,y] R[b,w,y];  L[Ml,Dw,Ml], R[Mr,Dw,Mr], D and out [Ml,Mr]. */
int tdvp_apply_bond(tdvp_handle *h, int Ml, int Mr, int Dw,
                    const tdvp_c128 *L /*DEVICE*/, const tdvp_c128 *D /*DEVICE*/,
                    const tdvp_c128 *R /*DEVICE*/, tdvp_c128 *out /*DEVICE*/);

/* y = exp(z * H[i]) v by the Lanczos / Krylov method with dimension k = opt.krylov_dim (fixed, or
   the cap of the adaptive rule if opt.krylov_tol > 0 and z_re = 0), full re-orthogonalisation, real
   alpha_j, breakdown rule beta_j < 1e-14 * max(1, |alpha_j|).
   For z_re = 0 the coefficients exp(z T) e_1 of the tridiagonal matrix come from a Chebyshev expansion,
   which covers |z| * (spectral width of T) up to ~1850 (beyond: TDVP_ESTATE at the next blocking call).  H[i] is the (Hermitian) operator of
   tdvp_apply_heff with the given L, W, R.  All scalars of the recurrence stay on the device.
   krylov_used: HOST, nullable; if non-NULL the call blocks on the stream and returns the Krylov
   dimension actually used. */
int tdvp_expm_heff(tdvp_handle *h, int Ml, int Mr, int d, int Dl, int Dr,
                   const tdvp_c128 *L, const tdvp_c128 *W, const tdvp_c128 *R /*DEVICE, as above*/,
                   double z_re, double z_im, const tdvp_c128 *v /*DEVICE [Ml,d,Mr]*/,
                   tdvp_c128 *y /*DEVICE [Ml,d,Mr]*/, int *krylov_used);
/* Same for the bond operator of tdvp_apply_bond. */
int tdvp_expm_bond(tdvp_handle *h, int Ml, int Mr, int Dw,
                   const tdvp_c128 *L, const tdvp_c128 *R, double z_re, double z_im,
                   const tdvp_c128 *v /*DEVICE [Ml,Mr]*/, tdvp_c128 *y /*DEVICE [Ml,Mr]*/,
                   int *krylov_used);

/* QR gauge move (Eq. 9), Householder, on the device.
   side = 0: C[Ml,d,Mr] viewed as (Ml*d) x Mr = Q D,  Q[Ml,d,Mr] left-canonical (Eq. 7), D[Mr,Mr]
   side = 1: C viewed as Ml x (d*Mr) = D Q,  Q[Ml,d,Mr] right-canonical (Eq. 8), D[Ml,Ml]
   Requires Ml*d >= Mr (side 0) or d*Mr >= Ml (side 1), and that tall side <= 12800 (TDVP_EINVAL
   otherwise; the same limit M_i * d_i <= 12800 holds in tdvp_create).  Q and D are unique only up to a unitary
   on the bond (the paper does not distinguish QR from RQ); the product is exact. */
int tdvp_qr_gauge(tdvp_handle *h, int side, int Ml, int d, int Mr,
                  const tdvp_c128 *C /*DEVICE*/, tdvp_c128 *Q /*DEVICE*/, tdvp_c128 *D /*DEVICE*/);

/* The same gauge move for callers that cannot allocate (code under CUDA-graph capture, tight serving loops,
   harnesses that forbid cudaMalloc): no handle, and NO cudaMalloc / cudaFree / allocating library call --
   the scratch lives in a 6 MiB static device array inside the library (held by every GPU that loads it,
   until exit).  Limit: the move's scratch must fit, i.e. about 2 * 16 * tall * thin + 16 * thin^2 bytes
   <= 6 MiB -- up to 1280 x 128, the M = 128, d = 10 move; larger shapes return TDVP_EINVAL (use tdvp_qr_gauge).
   Same arguments, kernels and results as tdvp_qr_gauge; cuda_stream: a cudaStream_t (NULL = legacy default).
   All calls share the one scratch block: calls that overlap on the GPU (different streams or host threads)
   race -- keep them on one stream.  Enqueue only.  Errors are those of handle-less calls (tdvp_last_error(NULL)). */
int tdvp_qr_gauge_noalloc(void *cuda_stream, int side, int Ml, int d, int Mr,
                          const tdvp_c128 *C /*DEVICE*/, tdvp_c128 *Q /*DEVICE*/, tdvp_c128 *D /*DEVICE*/);

/* Matrix unfolding of a bond (Eq. 36): C[Ml,d,Mr] viewed as Ml x (d*Mr) with
   Ml <= d*Mr is factored as U diag(lam) Vh on the device (Householder QR of C^T, then one-sided
   Jacobi on the Ml x Ml triangular factor).  U: DEVICE [Ml,Ml] unitary; lam: DEVICE double[Ml],
   non-negative, descending; Vh: DEVICE [Ml,d,Mr] with orthonormal rows (a right-canonical site,
   Eq. 8).  Singular vectors are unique only up to phases / rotations inside degenerate
   subspaces; the product is exact. */
int tdvp_svd_bond(tdvp_handle *h, int Ml, int d, int Mr, const tdvp_c128 *C /*DEVICE*/,
                  tdvp_c128 *U /*DEVICE*/, double *lam /*DEVICE*/, tdvp_c128 *Vh /*DEVICE*/);

/* Propagation and compression with the classical Runge-Kutta method (P&C-RK4), the paper's warm-up of its
   TDVP runs ("P&C-RK4 ... with M_max = 256 and time step size tau = 80 a.u. in the first 10
   steps ... Thereafter, the state is compressed to the pre-defined bond dimension M_S"), built from MPO x MPS
   (Eq. 12-13), MPS + MPS (Eq. 14-15), canonicalisation (Eq. 9) and SVD
   compression (Eq. 10), all on the device.  n_steps RK4 steps of size tau (Eq. 16,
   PAPER.md:119-131; every MPO x MPS product and every linear combination is compressed to M_max, reading
   c20), then one compression to M_out.  n_steps = 0 is a plain canonicalise-and-compress of the input.
     mpo / mps          as in tdvp_create (HOST pointers, HOST tensors); the MPS need not be canonical
     mps_bond_out[N+1]  HOST out: bond dimensions of the result, min(M_out, k_i) with k_i what the shapes allow
     mps_out[N]         HOST pointers to caller buffers; mps_out[i] must hold cap_i * d_i * cap_{i+1} elements,
                        cap_i = min(M_out, d_0...d_{i-1}, d_i...d_{N-1}); filled as [bond_i, d_i, bond_{i+1}]
   The result is right-canonical (Eq. 8) with the gauge centre at site 0: the input tdvp_create expects.
   h: stream + error slot (NULL: default).  Blocks.  Limits: M_O * M * d <= 12800 rows in every QR / SVD
   (TDVP_EINVAL beyond); bonds above 128 use the slow generic Jacobi SVD. */
int tdvp_pc_rk4_warmup(tdvp_handle *h, int n_sites, const int *phys_dim, const int *mpo_bond,
                       const tdvp_c128 *const *mpo, const int *mps_bond, const tdvp_c128 *const *mps,
                       double tau, int n_steps, int M_max, int M_out, int *mps_bond_out, tdvp_c128 *const *mps_out);

/* ---- stateful calls on the handle's resident MPS / environment cache ---------------------- */

/* H[site] applied to A_dev using the cached L[site], R[site] (valid when the gauge centre is at
   `site`).  A_dev, out_dev: DEVICE [Ml_site, d_site, Mr_site]. */
int tdvp_apply_heff_site(tdvp_handle *h, int site, const tdvp_c128 *A_dev, tdvp_c128 *out_dev);
/* Rebuild one cached block from its neighbour and the resident site tensor:
   side = 0: L[site+1] from L[site], W_site, A_site;  side = 1: R[site-1] from R[site], W_site, A_site. */
int tdvp_update_env_site(tdvp_handle *h, int site, int side);

/* One TDVP-PS step of length dt (Eq. 42-44): left-to-right sweep with dt/2
   (forward Eq. 43, QR Eq. 9, environment Eq. 30-32, backward Eq. 44), the last site evolved once
   by dt, and the mirror sweep.  Needs the PS gauge (centre at site 0); leaves it there.
   Enqueue only: no host round trip inside the step. */
int tdvp_step_ps(tdvp_handle *h, double dt);

/* One step of length dt of the TWO-SITE projector-splitting integrator ("it is also possible to
   formulate TDVP-PS into a two-site algorithm"; the paper gives no equations and declines it for its cost --
   this is the integrator of its ref. 32 built from the paper's Eq. 29-32, 10 and 43):
   left to right, every pair (i, i+1) is evolved by dt/2 with the two-site effective Hamiltonian, split by SVD
   (Eq. 10) keeping the bond dimension the chain already has, and the new centre is evolved backward by dt/2
   with the one-site H[i+1]; the last pair is evolved once by dt; then the mirror sweep.  Same gauge contract as
   tdvp_step_ps (centre at site 0 before and after); enqueue only.  The bond dimensions stay fixed, the norm is
   conserved up to the truncation.  Limit: M_i d_i <= 12800, and the pair SVDs are Jacobi iterations on
   min(M_i d_i, d_{i+1} M_{i+2}) columns -- fast up to 128, slow beyond (the paper's reason to decline it holds here). */
int tdvp_step_ps2(tdvp_handle *h, double dt);

/* One Dormand-Prince 5(4) step of length dt of the TDVP-MU equations of motion
   (Eq. 27, 33, 36-38) in the left-canonical gauge (centre at site N-1).  If the
   handle is in the PS gauge it is first moved by a QR sweep (no time evolution).
   err_est: HOST, nullable; if non-NULL the call blocks and returns the Euclidean norm of the
   embedded (5th - 4th order) difference. */
int tdvp_step_mu(tdvp_handle *h, double dt, double *err_est);

/* One step of length dt of TDVP-MU with constant-mean-field (CMF) integration, second-order
   midpoint scheme (cost PAPER.md:253, Table I): the mean
   fields -- environments h[1:i-1], h[i+1:N] and the unfolded bond U, Lambda of Eq. 36 -- are built
   at t, every local matrix is propagated to t + dt/2 with them held constant, the mean fields
   are rebuilt there, and every local matrix is propagated from t to t + dt with those.  Local
   propagation (readings, DESIGN.md c19): L_i by n_sub classical Runge-Kutta (RK4) sub-steps of
   Eq. 37/33/38 (ceil(n_sub/2) over the half step), C_N by the Lanczos exponential of Eq. 27 with
   the handle's krylov_dim.  SVDs and environment updates therefore run twice per step whatever
   n_sub is.  Same gauge handling as tdvp_step_mu; enqueue only; like tdvp_step_ps the step is captured into a
   CUDA graph once per (dt, n_sub) and replayed (not with TDVP_FLAG_NO_GRAPH, and not while the phase profiler is
   enabled: a replayed graph carries no brackets).  TDVP_EINVAL if n_sub < 1. */
int tdvp_step_mu_cmf(tdvp_handle *h, double dt, int n_sub);

/* One evaluation of the TDVP-MU right-hand side (Eq. 27 and Eq. 37-38) on the resident MPS, which
   must be in the MU gauge (centre N-1; else TDVP_ESTATE).  out_host[N]: HOST pointers to HOST
   buffers [Ml_i, d_i, Mr_i] receiving dL_i/dt (i < N-1) and dC_N/dt.  Blocks on the stream. */
int tdvp_mu_derivative(tdvp_handle *h, tdvp_c128 *const *out_host);

/* Move the gauge centre by QR / RQ sweeps without time evolution and rebuild the environment
   cache: centre = 0 (PS gauge) or centre = N-1 (MU gauge). */
int tdvp_set_gauge(tdvp_handle *h, int centre);

/* <psi| op_site |psi> / <psi|psi> is NOT normalised here: out = <psi| op |psi>.
   op: HOST [d,d] (row = bra).  Blocks on the stream.  Gauge-agnostic (identity transfer matrices
   from both ends). */
int tdvp_observe(tdvp_handle *h, int site, const tdvp_c128 *op, tdvp_c128 *out /*HOST*/);
/* Diagonal of the one-site reduced density matrix at `site` (site populations P^(n)(t),
   PAPER.md:335).  out: HOST [d_site].  Blocks on the stream. */
int tdvp_populations(tdvp_handle *h, int site, double *out);
/* <psi|psi> and <psi|H|psi>.  HOST outputs, either may be NULL.  Blocks on the stream. */
int tdvp_norm_energy(tdvp_handle *h, double *norm_sq, double *energy);

/* Copy site tensor out (HOST [Ml,d,Mr]); Ml/Mr nullable.  Blocks on the stream. */
int tdvp_get_mps(tdvp_handle *h, int site, tdvp_c128 *out_host, int *Ml, int *Mr);
/* Replace the MPS (same bond dimensions as at creation).  mps_host[N]: HOST pointers to HOST
   tensors.  centre must be 0 (right-canonical) or N-1 (left-canonical); environments are rebuilt. */
int tdvp_set_mps(tdvp_handle *h, const tdvp_c128 *const *mps_host, int centre);
int tdvp_get_centre(tdvp_handle *h);               /* current gauge centre, or a negative error  */
int tdvp_sync(tdvp_handle *h);                     /* block until the handle's stream is idle    */
const char *tdvp_last_error(const tdvp_handle *h);

/* ---- workload construction (host only, no GPU work) ------------------------------------------- */
/* The Frenkel-Holstein Hamiltonian of the paper (Eq. 45), single-exciton sector,
       H = sum_m E_m a+_m a_m + sum_{m != n} J_mn a+_m a_n + sum_{m,l} w_ml (b+ b + 1/2) + sum_{m,l} g_ml w_ml (b+ + b) a+_m a_m,
   as an MPO (Eq. 11), W_i[w, s, t, v] with s = bra, t = ket as everywhere in this header.
     layout       0: one electronic site of dimension n_el, then all modes, state-major (BASELINE configs 1, 3, 4)
                  1: the paper's own order: a two-level site per electronic state followed by its modes
     E[n_el], J[n_el * n_el] (symmetric, zero diagonal), omega[n_el * n_modes], huang_rhys[n_el * n_modes]
                  HOST; g_ml = sqrt(huang_rhys_ml) (reading c4); phonon modes truncated to n_ph number states
     energy_unit  factor applied to E, J, omega (2 pi c = 1.8836515673e-4 turns cm^-1 into rad/fs, reading c5)
     n_sites      HOST out; phys_dim[n_sites], mpo_bond[n_sites + 1]: HOST out, nullable
     mpo[n_sites] HOST pointers to caller buffers [mpo_bond[i], d_i, d_i, mpo_bond[i+1]], or NULL for a size query
                  (call once with mpo = NULL to learn n_sites, phys_dim and mpo_bond, allocate, call again).
   Bond dimensions: at most n_el + 2 (layout 0) / 2 n_el + 1 (layout 1); the tensors are real and a few per cent
   dense.  Returns TDVP_EINVAL on bad arguments; the error text is that of handle-less calls. */
int tdvp_build_vibronic_mpo(int layout, int n_el, int n_modes, int n_ph, const double *E, const double *J,
                            const double *omega, const double *huang_rhys, double energy_unit,
                            int *n_sites, int *phys_dim, int *mpo_bond, tdvp_c128 *const *mpo);

/* ---- measurement helpers ------------------------------------------------------------------- */
/* Issue-rate probe of the FP64 tensor pipe (DMMA m8n8k4 in registers, no memory traffic): runs on
   the legacy default stream, blocks, returns TFLOP/s.  This is the denominator bench.py uses for
   "fraction of FP64 tensor peak". */
int tdvp_probe_fp64_tensor_peak(int iters, double *tflops /*HOST*/);
/* The same probe with `fillers` (0, 1, 2, 4, 8 or 16) independent integer instructions issued after
   every DMMA, at the GEMM kernel's residency (two CTAs of four warps per SM): measures what the
   non-tensor instructions of a DMMA loop cost.  Blocks; TDVP_EINVAL on other
   filler counts. */
int tdvp_probe_dmma_issue(int fillers, int iters, double *tflops /*HOST*/);
/* How the complex128 GEMM stages (the M_S^3 M_O d terms of Table I,
   PAPER.md:375-388) split the complex product into real FP64 tensor-core products (north_star:
   "complex product split into real MMAs"; reading c15):
     products = 3 (default): X1 = Ar Br, X2 = Ai Bi, X3 = (Ar + Ai)(Br + Bi); C = (X1 - X2) + i (X3 - X1 - X2)
                 -- 25 % fewer DMMAs; error bounded normwise (relative to |A||B|), not per component;
     products = 4: Cr = Ar Br - Ai Bi, Ci = Ar Bi + Ai Br.
   Process-wide (every handle and stream; an atomic switch, safe to flip from any host thread), takes
   effect at the next launch; a captured step graph keeps the kernels it was captured with.  The
   environment variable TDVP_ZGEMM_4M=1 selects 4 at load time.  Returns 0, or TDVP_EINVAL. */
int tdvp_set_gemm_products(int products);
int tdvp_get_gemm_products(void);
/* Phase profiler: when enabled, launches of the dominant kernel classes are bracketed by CUDA events
   on the launching stream (not inside a captured step).  tdvp_profile_read blocks on the device,
   returns the summed elapsed milliseconds and bracket counts per phase since the last read and
   resets them.  Phases: 0 complex GEMM (DMMA), 1 MPO (W) stage, 2 Lanczos / vector kernels, 3 QR,
   4 SVD.  ms, count: HOST arrays of TDVP_PROFILE_PHASES entries.  The profiler state is process-wide
   (one record list for all handles, guarded by a mutex; safe to use from several host threads). */
#define TDVP_PROFILE_PHASES 5
int tdvp_profile_enable(int on);
int tdvp_profile_read(double *ms, long long *count);
/* Number of kernel launches this library has enqueued since load (for bench.py's gpu_launches;
   launches replayed from a captured CUDA graph are counted when the graph is launched). */
long long tdvp_launch_count(void);

/* Environment variables (diagnostic switches; none of them changes what is computed beyond rounding):
     TDVP_ZGEMM_4M=1          complex GEMM from four real products instead of three (tdvp_set_gemm_products),
                              read once when the library configures its kernels;
     TDVP_ZGEMM_SPLIT_COST=x  cost, in k-tile units, that the stream-K grid model charges for cutting
                              tiles (default 5), read once;
     TDVP_LANCZOS_UNFUSED=1   separate dot / update kernels instead of the fused cooperative kernel of a
                              Lanczos iteration, read once;
     TDVP_NO_FSAL=1           tdvp_step_mu recomputes stage 1 instead of reusing stage 7 of the step
                              before (bit-identical by construction; read at every step);
     TDVP_CMF_QUEUES=n        side queues of the local problems of TDVP-MU (1..16, default 6), read when a handle
                              first runs tdvp_step_mu / tdvp_step_mu_cmf / tdvp_mu_derivative;
     TDVP_CMF_PIPELINE=0      CMF step: build all mean fields first, then propagate all sites (default: site j starts
                              on its side queue as soon as the bond to its right is unfolded), read once;
     TDVP_MU_PIPELINE=0       the same switch for the right-hand side of tdvp_step_mu / tdvp_mu_derivative, read once;
     TDVP_CMF_PRIORITY=0      no separate highest-priority queue for the chain of bond unfoldings, read once;
     TDVP_CMF_SPLIT_SVD=0     Vh of a bond and the right block built from it stay on the queue of the unfolding chain
                              (default: on a queue of their own, one bond behind the chain), read once;
     TDVP_CMF_SPARE_SMS=n     SMs the GEMMs of the side queues leave out of their grids, for the cluster kernels of
                              the unfolding chain that run beside them (default 24; 0 = none), read once;
     TDVP_CMF_QUEUE_CTAS=n    CTAs a GEMM of one of those side queues may use (default: half the SM count, a quarter of
                              the device's CTA slots; 0 = only the TDVP_CMF_SPARE_SMS limit), read once;
     TDVP_SVD_ALWAYS_QR=1     a bond SVD always runs its final Householder step (default: only when the Jacobi
                              iteration left columns alone or ran out of sweeps; decided on the device), read once;
     TDVP_QR_CLUSTER=0        QR gauge moves of up to 1280 rows with one launch per panel and per trailing update
                              instead of the single 16-CTA cluster kernel, read once;
     TDVP_QR_FAST=0           that kernel eliminates every panel column by column, one cluster reduction per column
                              (default: one reduction per panel where its columns are well enough conditioned), read once;
     TDVP_SVD_MAX_SWEEPS=n    Jacobi sweeps a bond SVD may use (1..40, default 40; lowering it forces the
                              TDVP_ESTATE "did not converge" report: used by the error-path test), read at
                              every SVD. */

#ifdef __cplusplus
}
#endif
#endif /* TDVP_H */
