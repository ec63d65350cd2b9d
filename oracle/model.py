"""O1. Frenkel-Holstein Hamiltonian -> MPO, and its Kronecker-sum matrix (oracle, test infra).

PAPER.md:312-318, Eq. 45:
    H = sum_m E_m a+_m a_m + sum_{m!=n} J_mn a+_m a_n
      + sum_{m,l} w_ml (b+_ml b_ml + 1/2) + sum_{m,l} g_ml w_ml (b+_ml + b_ml) a+_m a_m
in the single-exciton sector, phonon modes truncated to n_ph number states.  The MPO form is
Eq. 11: W[w_{i-1}, s', s, w_i] with s' the bra (output) and s the ket (input)
index; array axes here are W[w_left, s_out, s_in, w_right].

Readings: c1 two site layouts ("A": one electronic site of dim N_el followed by
all modes site-major; "B": the paper's own, a 2-level electronic DOF followed by its modes, repeated,
PAPER.md:320); c4 g = sqrt(Huang-Rhys S), zero-point term kept; c5 energies converted from cm^-1
to rad/fs by 2*pi*c, time in fs, hbar = 1.
"""
import numpy as np
import scipy.sparse as sp

TWO_PI_C = 1.8836515673e-4  # rad fs^-1 / cm^-1


def boson_operators(n_ph):
    """Truncated harmonic-oscillator matrices: number n = b+ b and displacement x = b+ + b."""
    b = np.zeros((n_ph, n_ph))
    for v in range(1, n_ph):
        b[v - 1, v] = np.sqrt(v)          # b |v> = sqrt(v) |v-1>
    n = b.T @ b
    x = b.T + b
    return n, x


def mode_list(n_el, n_modes):
    """Site-major order of the modes: (m, l) for m = 0..N_el-1, l = 0..n_modes-1."""
    return [(m, l) for m in range(n_el) for l in range(n_modes)]


def build_mpo_layout_a(E, J, omega, S, n_ph):
    """Finite-state-machine MPO, layout A.  Bond channels: 0 = 'done' (a full term of H sits to
    the left, identities follow), 1 = 'I' (only identities so far), 2.. = 'P_m' (the projector
    |m><m| was applied at the electronic site and still waits for one of m's modes)."""
    E = np.asarray(E) * TWO_PI_C
    J = np.asarray(J) * TWO_PI_C
    w = np.asarray(omega) * TWO_PI_C
    g = np.sqrt(np.asarray(S))
    n_el, n_modes = w.shape
    num, x = boson_operators(n_ph)
    eye_ph = np.eye(n_ph)
    modes = mode_list(n_el, n_modes)

    pending = list(range(n_el))                      # channels alive on the bond right of site 0
    W0 = np.zeros((1, n_el, n_el, 2 + n_el), dtype=np.complex128)
    W0[0, :, :, 0] = np.diag(E) + J                  # electronic Hamiltonian -> done
    W0[0, :, :, 1] = np.eye(n_el)                    # identity -> I
    for c, m in enumerate(pending):
        W0[0, m, m, 2 + c] = 1.0                     # |m><m| -> P_m
    mpo = [W0]
    for idx, (m, l) in enumerate(modes):
        last = idx == len(modes) - 1
        pend_in = pending
        pend_out = [q for q in pend_in if q > m or (q == m and l < n_modes - 1)]
        Dl = 2 + len(pend_in)
        Dr = 1 if last else 2 + len(pend_out)
        Wi = np.zeros((Dl, n_ph, n_ph, Dr), dtype=np.complex128)
        Wi[0, :, :, 0] = eye_ph                                   # done -> done
        Wi[1, :, :, 0] = w[m, l] * (num + 0.5 * eye_ph)           # I -> done : w (b+b + 1/2)
        Wi[2 + pend_in.index(m), :, :, 0] = g[m, l] * w[m, l] * x  # P_m -> done : g w (b+ + b)
        if not last:
            Wi[1, :, :, 1] = eye_ph                               # I -> I
            for q in pend_out:
                Wi[2 + pend_in.index(q), :, :, 2 + pend_out.index(q)] = eye_ph   # P_q -> P_q
        mpo.append(Wi)
        pending = pend_out
    return mpo


def build_mpo_layout_b(E, J, omega, S, n_ph):
    """Layout B: for every electronic state m a 2-level site (|0>, |1>, a+_m a_m =
    |1><1|) followed by its own modes.  Channels: 0 'done', 1 'I', then for every electronic site
    q already passed that still has coupling partners to the right a pair ('a+_q', 'a_q'), and,
    inside block m only, 'n_m' (number operator applied, waiting for one of m's modes)."""
    E = np.asarray(E) * TWO_PI_C
    J = np.asarray(J) * TWO_PI_C
    w = np.asarray(omega) * TWO_PI_C
    g = np.sqrt(np.asarray(S))
    n_el, n_modes = w.shape
    num, x = boson_operators(n_ph)
    eye_ph = np.eye(n_ph)
    up = np.array([[0.0, 0.0], [1.0, 0.0]])      # a+ : |0> -> |1>   (axes [out, in])
    dn = up.T                                     # a
    nn = np.diag([0.0, 1.0])
    eye2 = np.eye(2)

    def channels(hop, with_n):
        ch = ["done", "I"]
        for q in hop:
            ch += [("a+", q), ("a", q)]
        if with_n is not None:
            ch.append(("n", with_n))
        return ch

    mpo = []
    hop_in = []                                   # electronic sites with open hopping channels
    ch_in = ["I"]                                 # left boundary: a single 'I' channel
    n_sites = n_el * (1 + n_modes)
    site = 0
    for m in range(n_el):
        # --- electronic site m ---
        hop_out = [q for q in hop_in + [m] if any(J[q, r] != 0.0 for r in range(m + 1, n_el))]
        last = site == n_sites - 1
        ch_out = ["done"] if last else channels(hop_out, m if n_modes > 0 else None)
        Wi = np.zeros((len(ch_in), 2, 2, len(ch_out)), dtype=np.complex128)
        if "done" in ch_in:
            Wi[ch_in.index("done"), :, :, 0] = eye2
        Wi[ch_in.index("I"), :, :, 0] = E[m] * nn
        for q in hop_in:                          # close a hopping term J_qm (a+_q a_m + a_q a+_m)
            if J[q, m] != 0.0:
                Wi[ch_in.index(("a+", q)), :, :, 0] = J[q, m] * dn
                Wi[ch_in.index(("a", q)), :, :, 0] = J[q, m] * up
        if not last:
            Wi[ch_in.index("I"), :, :, ch_out.index("I")] = eye2
            for q in hop_out:
                if q == m:
                    Wi[ch_in.index("I"), :, :, ch_out.index(("a+", m))] = up
                    Wi[ch_in.index("I"), :, :, ch_out.index(("a", m))] = dn
                else:
                    for kind in ("a+", "a"):
                        Wi[ch_in.index((kind, q)), :, :, ch_out.index((kind, q))] = eye2
            if n_modes > 0:
                Wi[ch_in.index("I"), :, :, ch_out.index(("n", m))] = nn
        mpo.append(Wi)
        ch_in, hop_in = ch_out, hop_out
        site += 1
        # --- modes of m ---
        for l in range(n_modes):
            last = site == n_sites - 1
            keep_n = m if l < n_modes - 1 else None
            ch_out = ["done"] if last else channels(hop_in, keep_n)
            Wi = np.zeros((len(ch_in), n_ph, n_ph, len(ch_out)), dtype=np.complex128)
            Wi[ch_in.index("done"), :, :, 0] = eye_ph
            Wi[ch_in.index("I"), :, :, 0] = w[m, l] * (num + 0.5 * eye_ph)
            Wi[ch_in.index(("n", m)), :, :, 0] = g[m, l] * w[m, l] * x
            if not last:
                Wi[ch_in.index("I"), :, :, ch_out.index("I")] = eye_ph
                for c in ch_out[2:]:
                    Wi[ch_in.index(c), :, :, ch_out.index(c)] = eye_ph
            mpo.append(Wi)
            ch_in = ch_out
            site += 1
    return mpo


def build_mpo(params):
    """params: any object with fields E, J, omega, S, n_ph, layout (synthetic_inputs.VibronicParams)."""
    if params.layout == "A":
        return build_mpo_layout_a(params.E, params.J, params.omega, params.S, params.n_ph)
    if params.layout == "B":
        return build_mpo_layout_b(params.E, params.J, params.omega, params.S, params.n_ph)
    raise ValueError(params.layout)


def mpo_to_dense(mpo):
    """Contract an MPO (Eq. 11) into its full matrix <s'_1..s'_N| O |s_1..s_N> (tiny systems)."""
    T = mpo[0][0]                                     # [s_out, s_in, w]
    for Wi in mpo[1:]:
        T = np.einsum("pqw,wstv->psqtv", T, Wi)
        p, s, q, t, v = T.shape
        T = T.reshape(p * s, q * t, v)
    return T[:, :, 0]


def _kron_site_operator(dims, site, op):
    """1 (x) ... (x) op_site (x) ... (x) 1 as a sparse matrix, first site slowest."""
    out = sp.identity(1, format="csr", dtype=np.float64)
    for i, d in enumerate(dims):
        out = sp.kron(out, sp.csr_matrix(op) if i == site else sp.identity(d, format="csr"),
                      format="csr")
    return out


def _kron_two_site_operator(dims, site_a, op_a, site_b, op_b):
    out = sp.identity(1, format="csr", dtype=np.float64)
    for i, d in enumerate(dims):
        if i == site_a:
            f = sp.csr_matrix(op_a)
        elif i == site_b:
            f = sp.csr_matrix(op_b)
        else:
            f = sp.identity(d, format="csr")
        out = sp.kron(out, f, format="csr")
    return out


def kronecker_sum_hamiltonian(params):
    """Eq. 45 written out term by term as a sparse matrix in the product basis of the layout
    (first site slowest).  Independent of the MPO construction above (pin p1)."""
    E = np.asarray(params.E) * TWO_PI_C
    J = np.asarray(params.J) * TWO_PI_C
    w = np.asarray(params.omega) * TWO_PI_C
    g = np.sqrt(np.asarray(params.S))
    n_el, n_modes = w.shape
    n_ph = params.n_ph
    num, x = boson_operators(n_ph)
    if params.layout == "A":
        dims = [n_el] + [n_ph] * (n_el * n_modes)
        H = _kron_site_operator(dims, 0, np.diag(E) + J)
        for idx, (m, l) in enumerate(mode_list(n_el, n_modes)):
            proj = np.zeros((n_el, n_el))
            proj[m, m] = 1.0
            H = H + _kron_site_operator(dims, 1 + idx, w[m, l] * (num + 0.5 * np.eye(n_ph)))
            H = H + _kron_two_site_operator(dims, 0, proj, 1 + idx, g[m, l] * w[m, l] * x)
        return H.tocsr(), dims
    dims = []
    el_site = []
    for m in range(n_el):
        el_site.append(len(dims))
        dims += [2] + [n_ph] * n_modes
    up = np.array([[0.0, 0.0], [1.0, 0.0]])
    nn = np.diag([0.0, 1.0])
    H = sp.csr_matrix((int(np.prod(dims)), int(np.prod(dims))))
    for m in range(n_el):
        H = H + _kron_site_operator(dims, el_site[m], E[m] * nn)
        for q in range(n_el):
            if q != m and J[m, q] != 0.0:
                H = H + _kron_two_site_operator(dims, el_site[m], J[m, q] * up, el_site[q], up.T)
        for l in range(n_modes):
            s = el_site[m] + 1 + l
            H = H + _kron_site_operator(dims, s, w[m, l] * (num + 0.5 * np.eye(n_ph)))
            H = H + _kron_two_site_operator(dims, el_site[m], nn, s, g[m, l] * w[m, l] * x)
    return H.tocsr(), dims
