"""O5b. TDVP-MU with constant-mean-field (CMF) integration, second-order midpoint scheme
(oracle, test infra).

PAPER.md:222-224: "in CMF, it is assumed that H[i] and S[i+1:N] generally change much slower in
time than the local matrices C_N and L_i.  As a result, during the integration of Eq. 27 and
Eq. 28 one may hold the 'mean field' H[i] and S[i+1:N] constant for tau and evolve only the local
matrix with time step smaller than tau ... we use a second order CMF with a midpoint scheme in
which L_i(0) and C_N(0) are integrated to L_i(tau) and C_N(tau) with 'mean field' constructed by
L_i(tau/2) and C_N(tau/2) ... in CMF, since Eq. 27 is linear, it is integrated by Krylov subspace
method instead."  Cost: PAPER.md:253 (f local steps per site within tau), Table I.

With the matrix unfolding of Eq. 36-38 the mean field of site i < N is the
quadruple (h[1:i-1], h[i+1:N] rebuilt from the R of Eq. 36, U, Lambda) of the bond to its right;
the mean field of site N is h[1:N-1].  The local equation of motion with these held constant is
    i dL_i/dt = (1 - L_i L_i^dagger) H[i](L_i U Lambda) Lambda~^{-1} U^dagger          (Eq. 37, 33, 38)
which is still non-linear in L_i through the projector.

Readings (DESIGN.md c19; the paper gives no formulas for these):
  * the state at tau/2 that defines the midpoint mean field is itself propagated from t = 0 with
    the mean field of t = 0 (a first-order predictor; the scheme stays second order);
  * the local integrator of L_i is the classical fourth-order Runge-Kutta method with `n_sub`
    equal sub-steps over tau (ceil(n_sub / 2) over the half step) -- "operations in the
    Runge-Kutta integrator" names the family only;
  * C_N is propagated by the Lanczos exponential of lanczos.py (fixed Krylov dimension k).
"""
import numpy as np

from .contractions import heff, envL, envR, boundary_env
from .lanczos import lanczos_expm
from .tdvp_mu import MU_EPS


def mean_fields(mpo, mps, eps=MU_EPS):
    """Mean fields of a left-canonical MPS (L_1..L_{N-1}, C_N): Lenv[i] = h[1:i-1] for every site,
    and for every site i < N-1 (0-based) the right block Renv[i] rebuilt from the R tensors of
    Eq. 36 together with U, Lambda of the bond to its right."""
    n = len(mps)
    Lenv = [boundary_env()]
    for i in range(n - 1):
        Lenv.append(envL(Lenv[i], mpo[i], mps[i]))
    Renv = [None] * n
    U = [None] * n
    lam = [None] * n
    Renv[n - 1] = boundary_env()
    C = mps[n - 1]
    for i in range(n - 1, 0, -1):
        Ml, d, Mr = C.shape
        u, s, Vh = np.linalg.svd(C.reshape(Ml, d * Mr), full_matrices=False)    # Eq. 36
        Renv[i - 1] = envR(Renv[i], mpo[i], Vh.reshape(Vh.shape[0], d, Mr))
        U[i - 1], lam[i - 1] = u, s
        C = np.einsum("asl,lr->asr", mps[i - 1], u * s[None, :])
    return Lenv, Renv, U, lam


def local_rhs(L, Lenv_i, W_i, Renv_i, U, lam, eps=MU_EPS):
    """dL_i/dt of Eq. 37 for given (constant) mean fields."""
    sq = np.sqrt(eps)
    C = np.einsum("asl,lr->asr", L, U * lam[None, :])
    lam_reg = lam + sq * np.exp(-lam / sq)                                       # Eq. 38
    HC = heff(Lenv_i, W_i, C, Renv_i)
    G = np.einsum("asr,rl->asl", HC / lam_reg[None, None, :], U.conj().T)
    a, s, l = G.shape
    Lm, Gm = L.reshape(a * s, l), G.reshape(a * s, l)
    return (-1j * (Gm - Lm @ (Lm.conj().T @ Gm))).reshape(a, s, l)               # (1 - p[i]) G, Eq. 33


def propagate_local(mpo, mps, fields, t, n_sub, k, eps=MU_EPS):
    """Every local matrix of `mps` propagated over time t with the mean fields held constant."""
    Lenv, Renv, U, lam = fields
    n = len(mps)
    out = [None] * n
    h = t / n_sub
    for i in range(n - 1):
        y = mps[i]
        f = lambda x: local_rhs(x, Lenv[i], mpo[i], Renv[i], U[i], lam[i], eps)
        for _ in range(n_sub):                                                   # classical RK4
            k1 = f(y)
            k2 = f(y + 0.5 * h * k1)
            k3 = f(y + 0.5 * h * k2)
            k4 = f(y + h * k3)
            y = y + (h / 6.0) * (k1 + 2.0 * k2 + 2.0 * k3 + k4)
        out[i] = y
    apply_h = lambda x: heff(Lenv[n - 1], mpo[n - 1], x, boundary_env())
    out[n - 1], _ = lanczos_expm(apply_h, mps[n - 1], -1j * t, k)                # Eq. 27 by Krylov
    return out


def step_cmf(mpo, mps, dt, n_sub, k, eps=MU_EPS):
    """One second-order CMF step of size dt (midpoint scheme)."""
    half = propagate_local(mpo, mps, mean_fields(mpo, mps, eps), 0.5 * dt, (n_sub + 1) // 2, k, eps)
    return propagate_local(mpo, mps, mean_fields(mpo, half, eps), dt, n_sub, k, eps)
