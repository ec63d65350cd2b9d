"""O5. TDVP-MU derivative and one Dormand-Prince 5(4) step (oracle, test infra).

PAPER.md:188-251.  State: left-canonical MPS L_1..L_{N-1}, C_N (gauge centre at the last site).
  Eq. 27:  i dC_N/dt = H[N] C_N
  Eq. 28/37: i dL_i/dt = (1 - p[i]) H[i](L_i U Lambda) Lambda~^{-1} U^dagger
  Eq. 33:  p[i] = L_i L_i^dagger
  Eq. 36: the centre at site i+1 is unfolded by SVD, U Lambda R
  Eq. 38:  Lambda~ = Lambda + eps^{1/2} exp(-Lambda / eps^{1/2}), eps = 1e-10
Readings: c13 the index placement of Eq. 37 is garbled in the source; the form
used is G = H_eff(C_i) Lambda~^{-1} U^dagger with C_i = L_i U Lambda, the only one for which
eps -> 0 recovers Eq. 28 and Eq. 34 holds; only the inverse factor is regularised.  c12: one call
= one fixed Dormand-Prince 5(4) step (the paper's VMF integrator); the adaptive
step-size controller has no formula in the paper -> parity unpinned, left to the caller.
"""
import numpy as np

from .contractions import heff, envL, envR, boundary_env

MU_EPS = 1e-10


def mu_derivative(mpo, mps, eps=MU_EPS):
    """Time derivatives [dL_1/dt, ..., dL_{N-1}/dt, dC_N/dt] of a left-canonical MPS."""
    n = len(mps)
    Lenv = [boundary_env()]
    for i in range(n - 1):
        Lenv.append(envL(Lenv[i], mpo[i], mps[i]))                 # "Get Env"
    deriv = [None] * n
    deriv[n - 1] = -1j * heff(Lenv[n - 1], mpo[n - 1], mps[n - 1], boundary_env())   # Eq. 27
    C = mps[n - 1]
    Renv = boundary_env()
    sq = np.sqrt(eps)
    for i in range(n - 1, 0, -1):
        Ml, d, Mr = C.shape
        U, lam, Vh = np.linalg.svd(C.reshape(Ml, d * Mr), full_matrices=False)   # Eq. 36
        Rsite = Vh.reshape(Vh.shape[0], d, Mr)
        Renv = envR(Renv, mpo[i], Rsite)                           # h[i+1:N] rebuilt from R
        Lsite = mps[i - 1]
        C = np.einsum("asl,lr->asr", Lsite, U * lam[None, :])       # centre form of site i-1
        lam_reg = lam + sq * np.exp(-lam / sq)                      # Eq. 38
        HC = heff(Lenv[i - 1], mpo[i - 1], C, Renv)
        G = np.einsum("asr,rl->asl", HC / lam_reg[None, None, :], U.conj().T)
        a, s, l = G.shape
        Lm = Lsite.reshape(a * s, l)
        Gm = G.reshape(a * s, l)
        deriv[i - 1] = (-1j * (Gm - Lm @ (Lm.conj().T @ Gm))).reshape(a, s, l)   # (1 - p[i]) G
    return deriv


# Dormand-Prince 5(4) Butcher tableau (the RK45 of PAPER.md:224).
_C = [0.0, 1 / 5, 3 / 10, 4 / 5, 8 / 9, 1.0, 1.0]
_A = [
    [],
    [1 / 5],
    [3 / 40, 9 / 40],
    [44 / 45, -56 / 15, 32 / 9],
    [19372 / 6561, -25360 / 2187, 64448 / 6561, -212 / 729],
    [9017 / 3168, -355 / 33, 46732 / 5247, 49 / 176, -5103 / 18656],
    [35 / 384, 0.0, 500 / 1113, 125 / 192, -2187 / 6784, 11 / 84],
]
_B5 = [35 / 384, 0.0, 500 / 1113, 125 / 192, -2187 / 6784, 11 / 84, 0.0]
_B4 = [5179 / 57600, 0.0, 7571 / 16695, 393 / 640, -92097 / 339200, 187 / 2100, 1 / 40]


def step_mu(mpo, mps, dt, eps=MU_EPS):
    """One Dormand-Prince step of size dt on the concatenated unknowns.  Returns (new_mps,
    err_est) with err_est the Euclidean norm of (5th-order - 4th-order) solution."""
    n = len(mps)
    ks = []
    for s in range(7):
        y = [mps[i] + dt * sum(_A[s][j] * ks[j][i] for j in range(s)) if s > 0 else mps[i]
             for i in range(n)]
        ks.append(mu_derivative(mpo, y, eps))
    new = [mps[i] + dt * sum(_B5[j] * ks[j][i] for j in range(7)) for i in range(n)]
    err2 = 0.0
    for i in range(n):
        e = dt * sum((_B5[j] - _B4[j]) * ks[j][i] for j in range(7))
        err2 += float(np.sum(np.abs(e) ** 2))
    return new, np.sqrt(err2)


def to_left_canonical(mps):
    """QR sweep (Eq. 9) moving the gauge centre from site 0 to the last site, no time evolution."""
    out = [np.array(A, dtype=np.complex128) for A in mps]
    for i in range(len(out) - 1):
        Ml, d, Mr = out[i].shape
        Q, D = np.linalg.qr(out[i].reshape(Ml * d, Mr))
        out[i] = Q.reshape(Ml, d, Q.shape[1])
        out[i + 1] = np.einsum("ab,bsc->asc", D, out[i + 1])
    return out


def to_right_canonical(mps):
    """RQ sweep moving the gauge centre from the last site to site 0."""
    out = [np.array(A, dtype=np.complex128) for A in mps]
    for i in range(len(out) - 1, 0, -1):
        Ml, d, Mr = out[i].shape
        Q, Rt = np.linalg.qr(out[i].reshape(Ml, d * Mr).T)
        out[i] = Q.T.reshape(Q.shape[1], d, Mr)
        out[i - 1] = np.einsum("asb,bc->asc", out[i - 1], Rt.T)
    return out
