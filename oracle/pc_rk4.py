"""O8. Propagation-and-compression with classical Runge-Kutta (P&C-RK4) and its building blocks
(oracle, test infra).  PAPER.md:78-138 and :322-324.

  mpo_times_mps  Eq. 12-13:  A'[(w,a), s', (w',a')] = sum_s W[w,s',s,w'] A[a,s,a'],
                 bond dimension M_O * M_S
  mps_add        Eq. 14-15: block-diagonal merge, bond dimension M_A + M_B
  canonicalise   Eq. 9: QR sweep from site 1 to N-1 -> left-canonical, centre at N
  compress       Eq. 10: "a left-canonical MPS could be compressed by successive approximate
                 SVD decomposition from site N to 1", truncation criterion (i): a fixed M_S; "as the new MPS
                 is not canonical, canonicalisation should be carried out before the actual compression"
                  -- compress() canonicalises first
  rk4_step       Eq. 16, time-independent H
  warmup         PAPER.md:322-324: "we use P&C-RK4 to propagate the state with M_max = 256 and time step
                 size tau = 80 a.u. in the first 10 steps ... Thereafter, the state is compressed to the
                 pre-defined bond dimension M_S"

Readings (DESIGN.md c20; the paper says "after each operation ... compressed" without listing them):
  * every MPO x MPS product is compressed, and every linear combination |Psi> + c |k> (two terms) or
    |Psi> + tau/6 (|k1> + 2|k2> + 2|k3> + |k4>) (five terms, merged at once) is compressed, all to M_max;
  * a compression always keeps min(M_max, k) singular values, k = min(rows, cols) of the unfolded centre
    (zero singular values included), so the bond dimensions depend on the shapes only;
  * scalars (-i, tau/2, ...) multiply the first site tensor.
The compressed state is right-canonical with the gauge centre at site 0: what TDVP-PS starts from.
"""
import numpy as np


def mpo_times_mps(mpo, mps):
    """Eq. 13.  W[w,s',s,w'] (s' = bra/output), A[a,s,a'] -> A'[(w,a), s', (w',a')]."""
    out = []
    for W, A in zip(mpo, mps):
        Dl, d, _, Dr = W.shape
        Ml, _, Mr = A.shape
        T = np.einsum("wpsv,asb->wapvb", W, A)
        out.append(np.ascontiguousarray(T.reshape(Dl * Ml, d, Dr * Mr)))
    return out


def mps_add(terms):
    """Eq. 15 for any number of terms: sum_k coeff_k |psi_k>, terms = [(coeff, mps), ...]; the coefficient
    multiplies the first site tensor of its term."""
    n = len(terms[0][1])
    out = []
    for i in range(n):
        blocks = [(c * m[i] if i == 0 else m[i]) for c, m in terms]
        d = blocks[0].shape[1]
        if n == 1:
            out.append(sum(blocks))
        elif i == 0:                                         # [A B ...]: row vector of blocks
            out.append(np.ascontiguousarray(np.concatenate(blocks, axis=2)))
        elif i == n - 1:                                     # column vector of blocks
            out.append(np.ascontiguousarray(np.concatenate(blocks, axis=0)))
        else:                                                # block diagonal
            Ml = sum(b.shape[0] for b in blocks)
            Mr = sum(b.shape[2] for b in blocks)
            T = np.zeros((Ml, d, Mr), dtype=np.complex128)
            r0 = c0 = 0
            for b in blocks:
                T[r0:r0 + b.shape[0], :, c0:c0 + b.shape[2]] = b
                r0 += b.shape[0]
                c0 += b.shape[2]
            out.append(T)
    return out


def canonicalise(mps):
    """Eq. 9: QR from site 1 to N-1; returns a left-canonical MPS with the centre at the last site."""
    out = [np.array(A, dtype=np.complex128) for A in mps]
    for i in range(len(out) - 1):
        Ml, d, Mr = out[i].shape
        Q, D = np.linalg.qr(out[i].reshape(Ml * d, Mr))
        out[i] = Q.reshape(Ml, d, Q.shape[1])
        out[i + 1] = np.einsum("ab,bsc->asc", D, out[i + 1])
    return out


def compress(mps, M_max):
    """Canonicalise (Eq. 9), then SVD from site N to 2 keeping min(M_max, k) singular values (Eq. 10).
    Returns (right-canonical MPS with the centre at site 0, list of discarded weights sum Lambda_s^2 per bond)."""
    out = canonicalise(mps)
    discarded = []
    for i in range(len(out) - 1, 0, -1):
        Ml, d, Mr = out[i].shape
        U, lam, Vh = np.linalg.svd(out[i].reshape(Ml, d * Mr), full_matrices=False)
        keep = min(M_max, lam.shape[0])
        discarded.append(float(np.sum(lam[keep:] ** 2)))
        out[i] = np.ascontiguousarray(Vh[:keep].reshape(keep, d, Mr))
        out[i - 1] = np.einsum("asb,bc->asc", out[i - 1], U[:, :keep] * lam[None, :keep])
    return out, discarded[::-1]


def rk4_step(mpo, mps, tau, M_max):
    """One P&C-RK4 step of size tau (Eq. 16) for a time-independent H given as an MPO."""
    def h_times(psi):                                        # -i H |psi>, compressed
        k = mpo_times_mps(mpo, psi)
        k[0] = -1j * k[0]
        return compress(k, M_max)[0]

    def combo(c, k):                                         # |Psi> + c |k>, compressed
        return compress(mps_add([(1.0, mps), (c, k)]), M_max)[0]

    k1 = h_times(mps)
    k2 = h_times(combo(0.5 * tau, k1))
    k3 = h_times(combo(0.5 * tau, k2))
    k4 = h_times(combo(tau, k3))
    s = tau / 6.0
    return compress(mps_add([(1.0, mps), (s, k1), (2.0 * s, k2), (2.0 * s, k3), (s, k4)]), M_max)[0]


def warmup(mpo, mps, tau, n_steps, M_max, M_S):
    """n_steps of P&C-RK4 at bond dimension M_max, then one compression to M_S.
    Returns a right-canonical MPS (centre at site 0) with bond dimensions min(M_S, k_i)."""
    psi = [np.array(A, dtype=np.complex128) for A in mps]
    for _ in range(n_steps):
        psi = rk4_step(mpo, psi, tau, M_max)
    return compress(psi, M_S)[0]
