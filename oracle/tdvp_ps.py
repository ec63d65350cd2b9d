"""O4. One-site TDVP-PS step (oracle, test infra).  PAPER.md:271-290, Eq. 42-44.

State: right-canonical MPS with the gauge centre at site 0 (paper's site 1) plus all right
environments.  One step = left-to-right sweep with tau/2, the last site evolved once by the full
tau (Eq. 42 prints a single factor for site N; reading c10), then the mirror right-to-left sweep.
QR gauge move: Eq. 9; RQ = QR of the transposed matrix (reading c9).
"""
import numpy as np

from .contractions import heff, envL, envR, bond, boundary_env
from .lanczos import lanczos_expm


class PSState:
    def __init__(self, mpo, mps):
        """mps: right-canonical, centre at site 0.  Tensors are copied."""
        self.mpo = [np.array(W, dtype=np.complex128) for W in mpo]
        self.mps = [np.array(A, dtype=np.complex128) for A in mps]
        n = len(mps)
        self.n = n
        self.Lenv = [None] * n      # Lenv[i]: sites < i contracted (h[1:i-1] in the paper)
        self.Renv = [None] * n      # Renv[i]: sites > i contracted (h[i+1:N])
        self.Lenv[0] = boundary_env()
        self.Renv[n - 1] = boundary_env()
        for i in range(n - 1, 0, -1):
            self.Renv[i - 1] = envR(self.Renv[i], self.mpo[i], self.mps[i])
        self.krylov_dims = []


def step_ps(st, dt, k, tol=0.0):
    """Advance st by one TDVP-PS step of size dt (Eq. 42) with Krylov dimension k (fixed if tol = 0,
    else the cap of the adaptive rule of lanczos.py)."""
    n = st.n
    st.krylov_dims = []
    for i in range(n - 1):
        # forward evolution of the centre, Eq. 43
        C, m = lanczos_expm(lambda x: heff(st.Lenv[i], st.mpo[i], x, st.Renv[i]),
                            st.mps[i], -1j * dt / 2, k, tol)
        st.krylov_dims.append(m)
        Ml, d, Mr = C.shape
        Q, D = np.linalg.qr(C.reshape(Ml * d, Mr))                 # Eq. 9
        st.mps[i] = Q.reshape(Ml, d, Q.shape[1])
        st.Lenv[i + 1] = envL(st.Lenv[i], st.mpo[i], st.mps[i])    # Eq. 30-32
        # backward evolution of the bond matrix, Eq. 44
        D, m = lanczos_expm(lambda x: bond(st.Lenv[i + 1], x, st.Renv[i]), D, +1j * dt / 2, k, tol)
        st.krylov_dims.append(m)
        st.mps[i + 1] = np.einsum("ab,bsc->asc", D, st.mps[i + 1])
    C, m = lanczos_expm(lambda x: heff(st.Lenv[n - 1], st.mpo[n - 1], x, st.Renv[n - 1]),
                        st.mps[n - 1], -1j * dt, k, tol)
    st.krylov_dims.append(m)
    st.mps[n - 1] = C
    for i in range(n - 1, 0, -1):
        C = st.mps[i]
        Ml, d, Mr = C.shape
        Q, Rt = np.linalg.qr(C.reshape(Ml, d * Mr).T)              # RQ via QR of the transpose
        D = Rt.T                                                   # C = D . B
        st.mps[i] = Q.T.reshape(Q.shape[1], d, Mr)
        st.Renv[i - 1] = envR(st.Renv[i], st.mpo[i], st.mps[i])
        D, m = lanczos_expm(lambda x: bond(st.Lenv[i], x, st.Renv[i - 1]), D, +1j * dt / 2, k, tol)
        st.krylov_dims.append(m)
        C = np.einsum("asb,bc->asc", st.mps[i - 1], D)
        C, m = lanczos_expm(lambda x: heff(st.Lenv[i - 1], st.mpo[i - 1], x, st.Renv[i - 1]),
                            C, -1j * dt / 2, k, tol)
        st.krylov_dims.append(m)
        st.mps[i - 1] = C
    return st
