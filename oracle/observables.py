"""O6. Observables (oracle, test infra): one-site reduced density matrix / populations
(P^(n)(t) of PAPER.md:330-335), norm, energy.  Gauge-agnostic: identity transfer matrices are
contracted from both ends, so any MPS (canonical or not) is accepted.
"""
import numpy as np

from .contractions import heff, envL, envR, boundary_env


def one_site_rdm(mps, site):
    """rho[s, t] = sum_{rest} psi[.., s, ..] conj(psi[.., t, ..])."""
    El = np.ones((1, 1), dtype=np.complex128)            # El[a_bra, a_ket]
    for A in mps[:site]:
        El = np.einsum("ax,asb,xsy->by", El, A.conj(), A)
    Er = np.ones((1, 1), dtype=np.complex128)
    for A in reversed(mps[site + 1:]):
        Er = np.einsum("by,asb,xsy->ax", Er, A.conj(), A)
    A = mps[site]
    return np.einsum("ax,atb,xsy,by->st", El, A.conj(), A, Er)


def populations(mps, site=0):
    """Diagonal of the one-site RDM (layout A: exciton populations at the electronic site)."""
    return np.real(np.diag(one_site_rdm(mps, site)))


def norm_sq(mps):
    E = np.ones((1, 1), dtype=np.complex128)
    for A in mps:
        E = np.einsum("ax,asb,xsy->by", E, A.conj(), A)
    return float(np.real(E[0, 0]))


def energy(mpo, mps):
    """<psi|H|psi> by contracting the full <psi| MPO |psi> network left to right (Eq. 30)."""
    L = boundary_env()
    for W, A in zip(mpo, mps):
        L = envL(L, W, A)
    return float(np.real(L[0, 0, 0]))


def mps_to_vector(mps):
    """Full state vector, first site slowest (tiny systems)."""
    T = mps[0]
    for A in mps[1:]:
        T = np.einsum("asb,btc->astc", T, A).reshape(T.shape[0], -1, A.shape[2])
    return T.reshape(-1)
