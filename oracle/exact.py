"""O7. Full-Hilbert-space propagation e^{-iHt} psi_0 (oracle, test infra; tiny chains only)."""
import numpy as np
import scipy.sparse.linalg as spla


def propagate(H_sparse, psi0, dt, n_steps):
    """Yields psi after each step of length dt."""
    psi = psi0.astype(np.complex128)
    A = (-1j * dt) * H_sparse.astype(np.complex128)
    for _ in range(n_steps):
        psi = spla.expm_multiply(A, psi)
        yield psi


def site_populations(psi, dims, site=0):
    """Diagonal of the one-site RDM of a full vector with first site slowest."""
    T = np.abs(psi.reshape(dims)) ** 2
    axes = tuple(i for i in range(len(dims)) if i != site)
    return T.sum(axis=axes)
