"""O9. Two-site TDVP-PS step (oracle, test infra).

PAPER.md:290: "Inspired by the original two-site DMRG algorithm, it is also possible to formulate TDVP-PS
into a two-site algorithm so that the bond dimension could grow up adaptively [ref 32]. However, considering
the two-site algorithm is much more expensive ... we use the one-site algorithm".  The paper gives no
equations for it; what follows is the projector-splitting integrator of its ref. 32 (Haegeman, Lubich,
Oseledets, Vandereycken, Verstraete, Phys. Rev. B 94, 165116 (2016), Sec. V) written with the paper's own
ingredients: Eq. 29-32 for the effective Hamiltonians, Eq. 10 for the SVD split, Eq. 43 for the backward
step.  PARITY UNPINNED against the paper (it prints nothing to compare with); pinned against the mathematics
in tests/test_oracle_pins.py (exact propagation with complete bonds; norm; agreement with one-site TDVP-PS).

One step of size dt, state right-canonical with the centre at site 0 and all right environments cached:
  for i = 0 .. N-3:   Theta = C_i B_{i+1};  Theta <- exp(-i H2[i,i+1] dt/2) Theta;
                      SVD (Eq. 10) keeping chi = the bond dimension the state already has: A_i = U, C_{i+1} = S V^dagger;
                      L[i+1] = envL(L[i], W_i, A_i);  C_{i+1} <- exp(+i H[i+1] dt/2) C_{i+1}     (one-site H_eff, backward)
  last pair (N-2, N-1): Theta <- exp(-i H2 dt) Theta   (ONE exponential of the full step, as reading c10 for the one-site
                      scheme: the forward sweep ends and the backward sweep starts on this pair)
  for i = N-1 .. 1:   split Theta of the pair (i-1, i): B_i = V^dagger, C_{i-1} = U S;  R[i-1] = envR(R[i], W_i, B_i);
                      if i-1 > 0: C_{i-1} <- exp(+i H[i-1] dt/2) C_{i-1};  Theta = B'_{i-2}... i.e. the pair (i-2, i-1) is
                      formed with the left-canonical A_{i-2} and evolved forward by dt/2.
Readings: the bond dimensions stay what they are (truncation criterion (i) of PAPER.md:86 with M_S = the current
bond), so that the tensors keep their shapes; no renormalisation after a truncation; fixed Krylov dimension k.
"""
import numpy as np

from .contractions import heff, envL, envR
from .lanczos import lanczos_expm
from .tdvp_ps import PSState


def heff2(L, W1, W2, Theta, R):
    """H2 applied to a two-site tensor Theta[x, t1, t2, y]: out[a,s1,s2,b] = sum L[a,w,x] W1[w,s1,t1,u] W2[u,s2,t2,v]
    Theta[x,t1,t2,y] R[b,v,y]   (Eq. 29 with two sites between the environment blocks)."""
    T = np.tensordot(L, Theta, axes=([2], [0]))                 # [a,w,t1,t2,y]
    T = np.tensordot(T, W1, axes=([1, 2], [0, 2]))              # [a,t2,y,s1,u]
    T = np.tensordot(T, W2, axes=([4, 1], [0, 2]))              # [a,y,s1,s2,v]
    return np.tensordot(T, R, axes=([4, 1], [1, 2]))            # [a,s1,s2,b]


def _split(Theta, chi):
    Ml, d1, d2, Mr = Theta.shape
    U, lam, Vh = np.linalg.svd(Theta.reshape(Ml * d1, d2 * Mr), full_matrices=False)      # Eq. 10
    keep = min(chi, lam.shape[0])
    return U[:, :keep].reshape(Ml, d1, keep), lam[:keep], Vh[:keep].reshape(keep, d2, Mr)


def step_ps2(st, dt, k):
    """Advance the PSState st by one two-site TDVP-PS step of size dt."""
    n = st.n
    assert n >= 2
    for i in range(n - 1):
        Theta = np.einsum("asc,ctb->astb", st.mps[i], st.mps[i + 1])
        last = i == n - 2
        Theta, _ = lanczos_expm(lambda x: heff2(st.Lenv[i], st.mpo[i], st.mpo[i + 1], x, st.Renv[i + 1]),
                                Theta, -1j * (dt if last else dt / 2), k)
        if last:
            break
        U, lam, Vh = _split(Theta, st.mps[i].shape[2])
        st.mps[i] = U
        st.Lenv[i + 1] = envL(st.Lenv[i], st.mpo[i], U)
        C = lam[:, None, None] * Vh
        C, _ = lanczos_expm(lambda x: heff(st.Lenv[i + 1], st.mpo[i + 1], x, st.Renv[i + 1]), C, +1j * dt / 2, k)
        st.mps[i + 1] = C
    for i in range(n - 1, 0, -1):
        U, lam, Vh = _split(Theta, st.mps[i].shape[0])
        st.mps[i] = Vh
        st.Renv[i - 1] = envR(st.Renv[i], st.mpo[i], Vh)
        C = U * lam[None, None, :]
        if i - 1 > 0:
            C, _ = lanczos_expm(lambda x: heff(st.Lenv[i - 1], st.mpo[i - 1], x, st.Renv[i - 1]), C, +1j * dt / 2, k)
            Theta = np.einsum("asc,ctb->astb", st.mps[i - 2], C)
            Theta, _ = lanczos_expm(lambda x: heff2(st.Lenv[i - 2], st.mpo[i - 2], st.mpo[i - 1], x, st.Renv[i - 1]),
                                    Theta, -1j * dt / 2, k)
        else:
            st.mps[0] = C
    return st


__all__ = ["PSState", "heff2", "step_ps2"]
