"""O3. Lanczos / Krylov exponential y = exp(z * H) v for Hermitian H (oracle, test infra).

PAPER.md:292-296: "the Krylov subspace method (Lanczos algorithm for Hermitian operator here)",
the {alpha}, {beta} of the three-term recurrence, and diagonalisation of the tridiagonal matrix
in the subspace.  Readings: fixed Krylov dimension k; alpha_j = Re<q_j, w>;
two passes of full re-orthogonalisation; breakdown rule beta_j < 1e-14 * max(1, |alpha_j|).
Adaptive mode (tol > 0): the paper says the Krylov dimension "is adaptive ... continues until
|Psi(t+tau)> converges" and gives no criterion -> the rule is a reading (c11), PARITY
UNPINNED against the paper: stop at the first j with beta_j * |[exp(z T_j) e_1]_j| < tol, the usual
a-posteriori estimate of the error of the Krylov exponential of a unit vector (Saad 1992; Hochbruck
& Lubich 1997).  The rule itself IS pinned against the mathematics: tests/test_oracle_pins.py checks
that the result then agrees with scipy's dense expm to ~tol * |v|.
"""
import numpy as np

BREAKDOWN_TOL = 1e-14


def lanczos_expm(apply_h, v, z, k, tol=0.0):
    """apply_h: callable x -> H x on arrays shaped like v.  z: complex scalar.  k: max dimension.
    tol: 0 = fixed k; > 0 = adaptive stop (see the module docstring).
    Returns (y, m) with m the Krylov dimension actually used."""
    shape = v.shape
    beta0 = np.linalg.norm(v)
    if beta0 == 0.0:
        return v.copy(), 0
    q = [v.reshape(-1) / beta0]
    alpha = []
    beta = []
    for j in range(k):
        w = apply_h(q[j].reshape(shape)).reshape(-1)
        a_j = np.vdot(q[j], w).real
        alpha.append(a_j)
        w = w - a_j * q[j]
        if j > 0:
            w = w - beta[j - 1] * q[j - 1]
        for _ in range(2):                       # full re-orthogonalisation, two passes
            for qi in q:
                w = w - np.vdot(qi, w) * qi
        b_j = np.linalg.norm(w)
        if j == k - 1 or b_j < BREAKDOWN_TOL * max(1.0, abs(a_j)):
            break
        if tol > 0.0:
            Tj = np.diag(np.array(alpha))
            for i in range(j):
                Tj[i, i + 1] = Tj[i + 1, i] = beta[i]
            lam_j, V_j = np.linalg.eigh(Tj)
            c_last = V_j[j, :] @ (np.exp(z * lam_j) * V_j[0, :])      # [exp(z T_j) e_1]_j
            if b_j * abs(c_last) < tol:
                break
        beta.append(b_j)
        q.append(w / b_j)
    m = len(alpha)
    T = np.diag(np.array(alpha))
    for j in range(m - 1):
        T[j, j + 1] = beta[j]
        T[j + 1, j] = beta[j]
    lam, V = np.linalg.eigh(T)
    c = V @ (np.exp(z * lam) * V[0, :])          # V e^{z Lambda} V^T e_1
    y = np.zeros_like(q[0])
    for j in range(m):
        y = y + c[j] * q[j]
    return (beta0 * y).reshape(shape), m
