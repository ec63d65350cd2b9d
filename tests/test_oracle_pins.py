"""Pins for the oracle: each checks oracle/ against something other than
itself -- the Kronecker-sum Hamiltonian, brute-force projection in the full Hilbert space, exact
propagation e^{-iHt}, scipy's dense expm, conservation laws, and the paper's statements that
TDVP-MU preserves the gauge (Eq. 34) and agrees with TDVP-PS."""
import dataclasses

import numpy as np
import pytest
import scipy.linalg

import synthetic_inputs as si
from oracle import contractions as oc
from oracle import exact, lanczos, model, observables as obs, tdvp_mu, tdvp_ps


def _small_params(layout="A", n_el=3, n_modes=1, n_ph=3, seed=11):
    cfg = dataclasses.replace(si.CONFIGS["tiny"], model_seed=seed, n_el=n_el, n_modes=n_modes,
                              n_ph=n_ph, nearest_neighbour=False, layout=layout)
    return si.draw_vibronic_params(cfg)


# ---------------------------------------------------------------- p1: MPO (Eq. 11, Eq. 45)
@pytest.mark.parametrize("layout", ["A", "B"])
def test_p1_mpo_equals_kronecker_sum(layout):
    p = _small_params(layout, n_el=3, n_modes=2, n_ph=2)
    H, dims = model.kronecker_sum_hamiltonian(p)
    Hd = model.mpo_to_dense(model.build_mpo(p))
    assert Hd.shape == H.shape
    assert np.abs(Hd - H.toarray()).max() < 1e-15
    assert np.abs(Hd - Hd.conj().T).max() == 0.0


def test_p1_mpo_bond_dimensions(tiny_model):
    cfg, params, mpo, dims, occ = tiny_model
    assert [W.shape[3] for W in mpo] == [5, 5, 4, 4, 3, 3, 1]
    assert [W.shape[1] for W in mpo] == dims == [3, 4, 4, 4, 4, 4, 4]


def test_p1_layout_a_and_b_same_physics():
    pa = _small_params("A")
    pb = dataclasses.replace(pa, layout="B")
    pops = []
    for p in (pa, pb):
        H, dims = model.kronecker_sum_hamiltonian(p)
        occ = si.initial_occupations(p)
        psi0 = np.zeros(int(np.prod(dims)), dtype=np.complex128)
        psi0[np.ravel_multi_index(occ, dims)] = 1.0
        psi = list(exact.propagate(H, psi0, 10.0, 5))[-1]
        if p.layout == "A":
            pops.append(exact.site_populations(psi, dims, 0))
        else:
            el = [m * (1 + p.n_modes) for m in range(p.n_el)]
            pops.append(np.array([exact.site_populations(psi, dims, s)[1] for s in el]))
    assert np.abs(pops[0] - pops[1]).max() < 1e-13
    assert abs(pops[0].sum() - 1.0) < 1e-13


# ---------------------------------------------------------------- p2: contractions (Eq. 29-32, 44)
def _mixed_canonical(mps_right_canonical, centre):
    out = [A.copy() for A in mps_right_canonical]
    for i in range(centre):
        Ml, d, Mr = out[i].shape
        Q, D = np.linalg.qr(out[i].reshape(Ml * d, Mr))
        out[i] = Q.reshape(Ml, d, -1)
        out[i + 1] = np.einsum("ab,bsc->asc", D, out[i + 1])
    return out


def _left_basis(mps, centre):
    P = np.ones((1, 1), dtype=np.complex128)                 # [sigma_left, a]
    for A in mps[:centre]:
        P = np.einsum("pa,asb->psb", P, A).reshape(-1, A.shape[2])
    return P


def _right_basis(mps, centre):
    P = np.ones((1, 1), dtype=np.complex128)                 # [b, sigma_right]
    for A in reversed(mps[centre + 1:]):
        P = np.einsum("asb,bq->asq", A, P).reshape(A.shape[0], -1)
    return P


def test_p2_staged_equals_definition():
    L, W, A, R = si.random_site_problem(5, 7, 3, 4, 6, 0.4, seed=3)
    assert np.abs(oc.heff(L, W, A, R) - oc.heff_definition(L, W, A, R)).max() < 1e-12
    assert np.abs(oc.envL(L, W, A) - oc.envL_definition(L, W, A)).max() < 1e-12
    assert np.abs(oc.envR(R, W, A) - oc.envR_definition(R, W, A)).max() < 1e-12
    D = si.complex_normal(np.random.default_rng(4), (5, 7))
    L2, _, _, R2 = si.random_site_problem(5, 7, 3, 4, 4, 0.4, seed=5)
    assert np.abs(oc.bond(L2, D, R2) - oc.bond_definition(L2, D, R2)).max() < 1e-12


@pytest.mark.parametrize("centre", [0, 1, 2, 3])
def test_p2_heff_is_projected_hamiltonian(centre):
    """H_eff[i] = P^dagger H P with P = P[1:i-1] (x) I_i (x) P[i+1:N] (Eq. 29, 43), brute force."""
    p = _small_params("A")
    H, dims = model.kronecker_sum_hamiltonian(p)
    H = H.toarray()
    mpo = model.build_mpo(p)
    mps = _mixed_canonical(si.random_right_canonical_mps(dims, 4, seed=2), centre)
    Lenv = oc.boundary_env()
    for i in range(centre):
        Lenv = oc.envL(Lenv, mpo[i], mps[i])
    Renv = oc.boundary_env()
    for i in range(len(mps) - 1, centre, -1):
        Renv = oc.envR(Renv, mpo[i], mps[i])
    PL, PR = _left_basis(mps, centre), _right_basis(mps, centre)
    d = dims[centre]
    P = np.einsum("pa,su,bq->psqaub", PL, np.eye(d), PR).reshape(H.shape[0], -1)
    assert np.abs(P.conj().T @ P - np.eye(P.shape[1])).max() < 1e-13      # Eq. 7, 8
    C = mps[centre]
    brute = (P.conj().T @ H @ P @ C.reshape(-1)).reshape(C.shape)
    got = oc.heff(Lenv, mpo[centre], C, Renv)
    assert np.abs(got - brute).max() < 1e-13
    psi = obs.mps_to_vector(mps)
    assert abs(np.vdot(C, got) - np.vdot(psi, H @ psi)) < 1e-13
    assert abs(obs.energy(mpo, mps) - np.vdot(psi, H @ psi).real) < 1e-13
    if centre < len(mps) - 1:
        # bond operator K = P[1:i] (x) P[i+1:N] projected H (Eq. 44)
        Ml, dd, Mr = C.shape
        Q, D = np.linalg.qr(C.reshape(Ml * dd, Mr))
        Lnext = oc.envL(Lenv, mpo[centre], Q.reshape(Ml, dd, -1))
        PL2 = np.einsum("pa,asb->psb", PL, Q.reshape(Ml, dd, -1)).reshape(-1, Q.shape[1])
        P2 = np.einsum("pa,bq->pqab", PL2, PR).reshape(H.shape[0], -1)
        brute = (P2.conj().T @ H @ P2 @ D.reshape(-1)).reshape(D.shape)
        assert np.abs(oc.bond(Lnext, D, Renv) - brute).max() < 1e-13


# ---------------------------------------------------------------- p8: Lanczos vs dense expm
@pytest.mark.parametrize("z", [-0.7j, +0.35j])
def test_p8_lanczos_full_dimension_is_exact(z):
    rng = np.random.default_rng(8)
    n = 12
    G = si.complex_normal(rng, (n, n))
    Hm = (G + G.conj().T) / 2
    v = si.complex_normal(rng, (3, 4))
    y, m = lanczos.lanczos_expm(lambda x: (Hm @ x.reshape(-1)).reshape(x.shape), v, z, 40)
    assert m == n                                            # Krylov space exhausted -> breakdown rule
    ref = scipy.linalg.expm(z * Hm) @ v.reshape(-1)
    assert np.abs(y.reshape(-1) - ref).max() < 1e-12


def test_p8_lanczos_truncated_is_unitary_and_accurate():
    rng = np.random.default_rng(9)
    n = 60
    G = si.complex_normal(rng, (n, n))
    Hm = (G + G.conj().T) / 2 / np.sqrt(n)
    v = si.complex_normal(rng, (n,))
    y, m = lanczos.lanczos_expm(lambda x: Hm @ x, v, -0.5j, 10)
    assert m == 10
    assert abs(np.linalg.norm(y) - np.linalg.norm(v)) < 1e-13 * np.linalg.norm(v)   # T7
    ref = scipy.linalg.expm(-0.5j * Hm) @ v
    assert np.abs(y - ref).max() < 1e-9


@pytest.mark.parametrize("tol", [1e-6, 1e-10])
def test_lanczos_adaptive_rule_meets_its_tolerance(tol):
    """Reading c11 (the paper gives no criterion): stopping at the first j with
    beta_j |[exp(z T_j) e_1]_j| < tol leaves an error of the order of tol * |v| against the dense
    exponential, with far fewer than the allowed vectors, and a tighter tol uses more of them."""
    rng = np.random.default_rng(10)
    n = 200
    G = si.complex_normal(rng, (n, n))
    Hm = (G + G.conj().T) / 2 / np.sqrt(n)                    # spectrum in about [-2, 2]
    v = si.complex_normal(rng, (n,))
    z = -3.0j
    y, m = lanczos.lanczos_expm(lambda x: Hm @ x, v, z, 64, tol=tol)
    ref = scipy.linalg.expm(z * Hm) @ v
    err = np.linalg.norm(y - ref) / np.linalg.norm(v)
    assert err < 20 * tol, (err, m)
    assert 8 < m < 40
    y1, m1 = lanczos.lanczos_expm(lambda x: Hm @ x, v, z, m - 2, tol=0.0)     # two vectors fewer: not yet converged
    assert np.linalg.norm(y1 - ref) / np.linalg.norm(v) > tol / 20
    if tol == 1e-10:
        _, m6 = lanczos.lanczos_expm(lambda x: Hm @ x, v, z, 64, tol=1e-6)
        assert m6 < m
    # tol = 0 is the fixed-k contract mode, unchanged
    y0, m0 = lanczos.lanczos_expm(lambda x: Hm @ x, v, z, 12)
    assert m0 == 12


# ---------------------------------------------------------------- p3: TDVP-PS closed form
def test_p3_ps_untruncated_equals_exact_propagation(tiny_model):
    """With complete bonds every backward step cancels a forward step and Eq. 42 reduces to
    e^{-iH tau} exactly, for ANY tau (derivation: SURVEY.md 8(c) 'Why p3 holds')."""
    cfg, params, mpo, dims, occ = tiny_model
    H, _ = model.kronecker_sum_hamiltonian(params)
    mps = si.padded_product_mps(dims, occ, 64, cfg.pad_seed)
    assert [A.shape[2] for A in mps] == [3, 12, 48, 64, 16, 4, 1]
    st = tdvp_ps.PSState(mpo, mps)
    ex = exact.propagate(H, obs.mps_to_vector(mps), 25.0, 3)
    for _ in range(3):
        tdvp_ps.step_ps(st, 25.0, 40)
        psi = next(ex)
    assert np.linalg.norm(obs.mps_to_vector(st.mps) - psi) < 2e-12
    assert np.abs(obs.populations(st.mps) - exact.site_populations(psi, dims)).max() < 1e-12


# ---------------------------------------------------------------- p4, p5, p9: config 1 as stated
def test_p4_p5_p9_config1_vs_exact(tiny_model):
    cfg, params, mpo, dims, occ = tiny_model
    H, _ = model.kronecker_sum_hamiltonian(params)
    mps = si.padded_product_mps(dims, occ, cfg.M, cfg.pad_seed)
    for A in mps[1:]:                                         # Eq. 8
        m = A.reshape(A.shape[0], -1)
        assert np.abs(m @ m.conj().T - np.eye(A.shape[0])).max() < 1e-14
    st = tdvp_ps.PSState(mpo, mps)
    e0 = obs.energy(mpo, mps)
    ex = exact.propagate(H, obs.mps_to_vector(mps), cfg.dt_fs, cfg.n_steps)
    worst = 0.0
    traj = []
    for _ in range(cfg.n_steps):
        tdvp_ps.step_ps(st, cfg.dt_fs, cfg.krylov_dim)
        pops = obs.populations(st.mps)
        traj.append(pops)
        worst = max(worst, np.abs(pops - exact.site_populations(next(ex), dims)).max())
        assert abs(pops.sum() - 1.0) < 1e-13                   # p9
    assert worst < 1e-5                                        # p5 (truncation + k = 10)
    assert abs(obs.norm_sq(st.mps) - 1.0) < 1e-13              # p4 / T7
    assert abs(obs.energy(mpo, st.mps) - e0) < 1e-13 * max(1.0, abs(e0)) * 10
    golden = np.loadtxt("tests/golden/tiny_ps_populations.txt")
    assert np.abs(np.array(traj) - golden).max() < 1e-10       # regression of the stored values


# ---------------------------------------------------------------- p6, p7, T4: TDVP-MU
@pytest.fixture(scope="module")
def warmed_up(tiny_model):
    cfg, params, mpo, dims, occ = tiny_model
    st = tdvp_ps.PSState(mpo, si.padded_product_mps(dims, occ, cfg.M, cfg.pad_seed))
    for _ in range(3):
        tdvp_ps.step_ps(st, 10.0, 30)
    return mpo, [A.copy() for A in st.mps]


def test_p7_mu_gauge_condition(warmed_up):
    """Eq. 34: L^dagger dL/dt = 0."""
    mpo, warm = warmed_up
    lc = tdvp_mu.to_left_canonical(warm)
    assert abs(abs(np.vdot(obs.mps_to_vector(lc), obs.mps_to_vector(warm))) - 1.0) < 1e-13   # T2
    deriv = tdvp_mu.mu_derivative(mpo, lc)
    for L, dL in zip(lc[:-1], deriv[:-1]):
        assert np.abs(np.einsum("asb,asc->bc", L.conj(), dL)).max() < 1e-12


def test_t4_unfolded_form_equals_overlap_inverse_form(tiny_model):
    """Eq. 37 with eps -> 0 equals Eq. 28 written with S[i+1:N]^{-1}; checked on
    a random full-rank state so that S is well conditioned."""
    cfg, params, mpo, dims, occ = tiny_model
    lc = tdvp_mu.to_left_canonical(si.random_right_canonical_mps(dims, 6, seed=13))
    n = len(lc)
    deriv = tdvp_mu.mu_derivative(mpo, lc, eps=1e-30)
    Lenv = [oc.boundary_env()]
    for i in range(n - 1):
        Lenv.append(oc.envL(Lenv[i], mpo[i], lc[i]))
    Renv = oc.boundary_env()                                  # built from the RAW (non-orthonormal) basis
    S = np.ones((1, 1), dtype=np.complex128)                  # S[l', l] = <l'|l>, Eq. 5
    checked = 0
    for i in range(n - 1, 0, -1):
        Renv = oc.envR(Renv, mpo[i], lc[i])
        S = np.einsum("asb,xsy,by->ax", lc[i].conj(), lc[i], S)
        assert np.linalg.cond(S) < 1e6
        HL = oc.heff(Lenv[i - 1], mpo[i - 1], lc[i - 1], Renv)
        G = np.einsum("asl,ml->asm", HL, np.linalg.inv(S))
        a, s, l = G.shape
        Lm, Gm = lc[i - 1].reshape(a * s, l), G.reshape(a * s, l)
        direct = (-1j * (Gm - Lm @ (Lm.conj().T @ Gm))).reshape(a, s, l)
        assert np.abs(direct - deriv[i - 1]).max() < 1e-9 * np.abs(G).max()
        checked += np.abs(direct).max() > 1e-3 * np.abs(G).max()
    assert checked >= 3                                       # not only trivially-zero derivatives


def test_p6_mu_agrees_with_ps(warmed_up):
    """both schemes give the same |Psi(t)> up to numerical error."""
    mpo, warm = warmed_up
    st = tdvp_ps.PSState(mpo, warm)
    for _ in range(4):
        tdvp_ps.step_ps(st, 1.25, 30)
    y = tdvp_mu.to_left_canonical(warm)
    for _ in range(20):
        y, err = tdvp_mu.step_mu(mpo, y, 0.25)
    assert np.abs(obs.populations(y) - obs.populations(st.mps)).max() < 1e-8
    assert err < 1e-3


# ---------------------------------------------------------------- p12, p13: TDVP-MU with CMF integration
def test_p12_cmf_local_rhs_is_the_mu_derivative(warmed_up):
    """With the mean fields taken at the state itself, the constant-mean-field right-hand side of
    every site is the (pinned: p6, p7, T4) TDVP-MU derivative of Eq. 37 -- and it obeys Eq. 34."""
    from oracle import tdvp_cmf
    mpo, warm = warmed_up
    lc = tdvp_mu.to_left_canonical(warm)
    deriv = tdvp_mu.mu_derivative(mpo, lc)
    Lenv, Renv, U, lam = tdvp_cmf.mean_fields(mpo, lc)
    big = 0
    for i in range(len(lc) - 1):
        r = tdvp_cmf.local_rhs(lc[i], Lenv[i], mpo[i], Renv[i], U[i], lam[i])
        assert np.abs(r - deriv[i]).max() <= 1e-13 * max(1.0, np.abs(deriv[i]).max())
        assert np.abs(np.einsum("asb,asc->bc", lc[i].conj(), r)).max() < 1e-12
        big += np.abs(r).max() > 1e-3
    assert big >= 3


def test_p13_cmf_is_second_order_and_agrees_with_ps(warmed_up):
    """PAPER.md:224 "second order CMF with a midpoint scheme"; Fig. 7 / PAPER.md:359: fitted slope
    2.03 of the CMF error against the step size; the TDVP schemes agree once
    the step is converged.  Reference: TDVP-PS with a converged step and Krylov dimension."""
    from oracle import tdvp_cmf
    mpo, warm = warmed_up
    T = 2.0
    ref = tdvp_ps.PSState(mpo, warm)
    for _ in range(16):
        tdvp_ps.step_ps(ref, T / 16, 30)
    p_ref = obs.populations(ref.mps)
    lc = tdvp_mu.to_left_canonical(warm)
    errs = []
    for tau in (0.5, 0.25, 0.125):
        y = [a.copy() for a in lc]
        for _ in range(int(round(T / tau))):
            y = tdvp_cmf.step_cmf(mpo, y, tau, max(2, int(tau / 0.0625)), 20)
        assert abs(obs.norm_sq(y) - 1.0) < 1e-10
        errs.append(np.abs(obs.populations(y) - p_ref).max())
    slopes = [np.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert all(1.7 < s < 2.5 for s in slopes), (errs, slopes)
    assert errs[-1] < 1e-5


# ---------------------------------------------------------------- Dormand-Prince tableau and error estimate
def _dp_tableau():
    n = 7
    A = np.zeros((n, n))
    for i, row in enumerate(tdvp_mu._A):
        A[i, :len(row)] = row
    return A, np.array(tdvp_mu._C), np.array(tdvp_mu._B5), np.array(tdvp_mu._B4)


def _order_conditions(A, c, b, order):
    """Residuals of the Runge-Kutta order conditions (one per rooted tree, Butcher / Hairer-Norsett-
    Wanner vol. I table II.2.1) up to `order`."""
    Ac, Ac2, Ac3 = A @ c, A @ c ** 2, A @ c ** 3
    AAc = A @ Ac
    res = [b.sum() - 1.0]
    if order >= 2:
        res += [b @ c - 1 / 2]
    if order >= 3:
        res += [b @ c ** 2 - 1 / 3, b @ Ac - 1 / 6]
    if order >= 4:
        res += [b @ c ** 3 - 1 / 4, b @ (c * Ac) - 1 / 8, b @ Ac2 - 1 / 12, b @ AAc - 1 / 24]
    if order >= 5:
        res += [b @ c ** 4 - 1 / 5, b @ (c ** 2 * Ac) - 1 / 10, b @ (c * Ac2) - 1 / 15, b @ (c * AAc) - 1 / 30,
                b @ (Ac * Ac) - 1 / 20, b @ Ac3 - 1 / 20, b @ (A @ (c * Ac)) - 1 / 40, b @ (A @ Ac2) - 1 / 60,
                b @ (A @ AAc) - 1 / 120]
    return np.array(res)


def test_dormand_prince_tableau_order_conditions():
    """oracle/tdvp_mu.py's tableau (the RK45 of PAPER.md:224): the propagated weights _B5 satisfy all 17
    order conditions through order 5, the embedded weights _B4 all 8 through order 4 and NOT those of
    order 5 (else the difference would not estimate the error); row sums give the nodes; stage 7 is
    evaluated at the new state (first-same-as-last)."""
    A, c, b5, b4 = _dp_tableau()
    assert np.abs(A.sum(axis=1) - c).max() < 1e-15
    assert np.abs(_order_conditions(A, c, b5, 5)).max() < 1e-15
    assert np.abs(_order_conditions(A, c, b4, 4)).max() < 1e-15
    assert np.abs(_order_conditions(A, c, b4, 5)[8:]).max() > 1e-4
    assert np.array_equal(A[6, :6], b5[:6]) and b5[6] == 0.0 and c[6] == 1.0


def test_mu_err_est_scales_as_h5(warmed_up):
    """err_est of oracle step_mu is the norm of the (5th - 4th order) difference: it falls as h^5
    (slope 4.5-5.5 per halving) on the warmed tiny chain, inside the smooth regime h <= 0.1 fs
    (SURVEY.md 8(c) c12), and the 5th-order solution's own one-step error falls faster still."""
    mpo, warm = warmed_up
    lc = tdvp_mu.to_left_canonical(warm)
    errs = []
    for h in (0.1, 0.05, 0.025):
        _, e = tdvp_mu.step_mu(mpo, lc, h)
        errs.append(e)
    slopes = [np.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert all(4.5 < s < 5.5 for s in slopes), (errs, slopes)
    # one step of h against two steps of h/2 (Richardson): the propagated solution is 5th order, local
    # error O(h^6) -> the ratio between h = 0.2 and h = 0.1 is >= 2^6 = 64 (measured 112: Dormand-Prince
    # minimises the h^6 coefficient, so the h^7 term still shows); a 4th-order weight row would give 32
    def one_vs_two(h):
        y1, _ = tdvp_mu.step_mu(mpo, lc, h)
        y2, _ = tdvp_mu.step_mu(mpo, lc, h / 2)
        y2, _ = tdvp_mu.step_mu(mpo, y2, h / 2)
        return np.linalg.norm(obs.mps_to_vector(y1) - obs.mps_to_vector(y2))
    r = one_vs_two(0.2) / one_vs_two(0.1)
    assert 45 < r < 260, r


# ---------------------------------------------------------------- observables: the full one-site RDM
@pytest.mark.parametrize("site", [0, 2, 3])
def test_one_site_rdm_all_entries_vs_full_vector(site):
    """rho[s,t] = sum_rest psi[..s..] conj(psi[..t..]) INCLUDING the off-diagonals (a transposed or
    conjugated rho passes every population check), on a random complex MPS that is NOT canonical
    (the contraction is gauge-agnostic); <psi|op|psi> = trace(op^T rho) = sum_st op[s,t]... is fixed
    by the full vector too, for a non-Hermitian op with `row = bra` (include/tdvp.h:190)."""
    dims = [3, 2, 4, 3, 2]
    rng = np.random.default_rng(31)
    bonds = [1, 3, 4, 5, 2, 1]
    mps = [si.complex_normal(rng, (bonds[i], dims[i], bonds[i + 1])) for i in range(5)]
    psi = obs.mps_to_vector(mps).reshape(dims)
    T = np.moveaxis(psi, site, 0).reshape(dims[site], -1)
    brute = T @ T.conj().T                                      # rho[s,t] = sum_rest psi_s conj(psi_t)
    rho = obs.one_site_rdm(mps, site)
    assert np.abs(rho - brute).max() < 1e-12 * np.abs(brute).max()
    assert np.abs(rho - rho.conj().T).max() < 1e-12 * np.abs(brute).max()
    assert np.abs(brute - brute.T).max() > 1e-2 * np.abs(brute).max()       # the case is not symmetric
    # <psi| O_site |psi> with O[s,t] = <s|O|t> (row = bra): sum_{s,t} conj(psi_s) O[s,t] psi_t = sum O[s,t] rho[t,s]
    op = si.complex_normal(rng, (dims[site], dims[site]))
    full = np.einsum("sr,st,tr->", T.conj(), op, T)
    assert abs(np.trace(op @ rho) - full) < 1e-12 * abs(full)
    assert abs(np.trace(op.T @ rho) - full) > 1e-3 * abs(full)


# ---------------------------------------------------------------- gauge sweeps without evolution
def test_to_right_canonical_keeps_the_state(warmed_up):
    """RQ sweep (Eq. 9): every site but the first satisfies Eq. 8
    to 1e-13 and the state is unchanged (overlap 1, same vector up to nothing at all: the sweep is
    a pure gauge change, so the VECTORS agree, not only their overlap)."""
    mpo, warm = warmed_up
    lc = tdvp_mu.to_left_canonical(warm)
    for A in lc[:-1]:                                          # Eq. 7
        m = A.reshape(-1, A.shape[2])
        assert np.abs(m.conj().T @ m - np.eye(A.shape[2])).max() < 1e-13
    rc = tdvp_mu.to_right_canonical(lc)
    for A in rc[1:]:                                           # Eq. 8
        m = A.reshape(A.shape[0], -1)
        assert np.abs(m @ m.conj().T - np.eye(A.shape[0])).max() < 1e-13
    v0, v1, v2 = (obs.mps_to_vector(x) for x in (warm, lc, rc))
    assert np.linalg.norm(v1 - v0) < 1e-12 and np.linalg.norm(v2 - v0) < 1e-12
    assert abs(np.vdot(v2, v0) - 1.0) < 1e-12
    assert [a.shape for a in rc] == [a.shape for a in warm]


# ---------------------------------------------------------------- P&C-RK4 building blocks (Eq. 10, 13, 15, 16)
def _random_mps(dims, bonds, seed):
    rng = np.random.default_rng(seed)
    return [si.complex_normal(rng, (bonds[i], dims[i], bonds[i + 1])) for i in range(len(dims))]


def test_pc_mpo_times_mps_and_add_against_dense_vectors():
    """Eq. 13: the MPS of H|Psi> contracts to H_dense @ psi and has bond dimension M_O * M_S;
    Eq. 15: the merged MPS contracts to the linear combination and has bond M_A + M_B."""
    from oracle import pc_rk4
    p = _small_params("A", n_el=3, n_modes=1, n_ph=3)
    H, dims = model.kronecker_sum_hamiltonian(p)
    mpo = model.build_mpo(p)
    a = _random_mps(dims, [1, 3, 4, 2, 1], 41)
    b = _random_mps(dims, [1, 2, 5, 3, 1], 42)
    c = _random_mps(dims, [1, 1, 1, 1, 1], 43)
    va, vb, vc = (obs.mps_to_vector(x) for x in (a, b, c))
    ha = pc_rk4.mpo_times_mps(mpo, a)
    assert np.abs(obs.mps_to_vector(ha) - H @ va).max() < 1e-12 * np.abs(H @ va).max()
    assert [t.shape[2] for t in ha] == [mpo[i].shape[3] * a[i].shape[2] for i in range(len(a))]
    s = pc_rk4.mps_add([(1.0, a), (0.5 - 2.0j, b), (-3.0, c)])
    want = va + (0.5 - 2.0j) * vb - 3.0 * vc
    assert np.abs(obs.mps_to_vector(s) - want).max() < 1e-13 * np.abs(want).max()
    assert [t.shape[2] for t in s] == [3 + 2 + 1, 4 + 5 + 1, 2 + 3 + 1, 1]
    assert s[0].shape[0] == 1


def test_pc_compress_is_the_truncated_svd():
    """Eq. 10.  Two sites: the compressed state is the best rank-M approximation of the coefficient matrix
    (Eckart-Young: same singular values kept, error^2 = discarded weight).  Four sites: no truncation leaves
    the vector unchanged and returns a right-canonical MPS (Eq. 8) with the bond dimensions capped by the
    shapes; with truncation, max(discarded) <= |Psi - Psi~|^2 <= sum(discarded)."""
    from oracle import pc_rk4
    two = _random_mps([5, 6], [1, 9, 1], 51)                 # bond 9 > min(5, 6): canonicalisation caps it at 5
    v = obs.mps_to_vector(two).reshape(5, 6)
    sv = np.linalg.svd(v, compute_uv=False)
    for M in (5, 3, 1):
        comp, disc = pc_rk4.compress(two, M)
        vc = obs.mps_to_vector(comp).reshape(5, 6)
        assert comp[0].shape == (1, 5, M) and comp[1].shape == (M, 6, 1)
        assert abs(np.linalg.norm(v - vc) ** 2 - np.sum(sv[M:] ** 2)) < 1e-12
        assert abs(disc[0] - np.sum(sv[M:] ** 2)) < 1e-12
        assert np.abs(np.linalg.svd(vc, compute_uv=False)[:M] - sv[:M]).max() < 1e-12
    dims = [3, 4, 2, 5]
    four = _random_mps(dims, [1, 7, 9, 6, 1], 52)
    v = obs.mps_to_vector(four)
    comp, disc = pc_rk4.compress(four, 64)
    assert [t.shape[2] for t in comp] == [3, 9, 5, 1] and sum(disc) < 1e-24     # min(raw bond, left cap, right cap)
    assert np.linalg.norm(obs.mps_to_vector(comp) - v) < 1e-12 * np.linalg.norm(v)
    for A in comp[1:]:
        m = A.reshape(A.shape[0], -1)
        assert np.abs(m @ m.conj().T - np.eye(A.shape[0])).max() < 1e-13
    comp, disc = pc_rk4.compress(four, 3)
    err2 = np.linalg.norm(obs.mps_to_vector(comp) - v) ** 2
    assert max(disc) * (1 - 1e-12) <= err2 <= sum(disc) * (1 + 1e-12)
    assert [t.shape[2] for t in comp] == [3, 3, 3, 1]


def test_pc_rk4_is_dense_rk4_and_fourth_order(tiny_model):
    """Eq. 16.  Without truncation (M_max = 64 holds every state of config 1's chain) P&C-RK4 is the classical
    RK4 of i d/dt psi = H psi on the full vector, to round-off; against exact propagation its global error
    falls as tau^4 (slope 3.5-4.5)."""
    from oracle import pc_rk4
    cfg, params, mpo, dims, occ = tiny_model
    H, _ = model.kronecker_sum_hamiltonian(params)
    prod = [np.zeros((1, d, 1), dtype=np.complex128) for d in dims]
    for t, o in zip(prod, occ):
        t[0, o, 0] = 1.0
    psi0 = obs.mps_to_vector(prod)
    tau = 0.5
    f = lambda y: -1j * (H @ y)
    k1 = f(psi0); k2 = f(psi0 + 0.5 * tau * k1); k3 = f(psi0 + 0.5 * tau * k2); k4 = f(psi0 + tau * k3)
    dense = psi0 + tau / 6.0 * (k1 + 2 * k2 + 2 * k3 + k4)
    got = pc_rk4.rk4_step(mpo, prod, tau, 64)
    assert np.linalg.norm(obs.mps_to_vector(got) - dense) < 1e-13
    T = 4.0
    exact_T = list(exact.propagate(H, psi0, T, 1))[-1]
    errs = []
    for n in (4, 8, 16):
        psi = prod
        for _ in range(n):
            psi = pc_rk4.rk4_step(mpo, psi, T / n, 64)
        errs.append(np.linalg.norm(obs.mps_to_vector(psi) - exact_T))
    slopes = [np.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert all(3.5 < s < 4.5 for s in slopes), (errs, slopes)


def test_pc_warmup_fills_the_bonds(tiny_model):
    """after the P&C-RK4 warm-up and the compression to M_S the state is right-canonical
    with the bond dimensions the shapes allow, close to the exactly propagated state, and its bonds are
    numerically full rank (what one-site TDVP needs) -- unlike the padded product state."""
    from oracle import pc_rk4
    cfg, params, mpo, dims, occ = tiny_model
    H, _ = model.kronecker_sum_hamiltonian(params)
    prod = [np.zeros((1, d, 1), dtype=np.complex128) for d in dims]
    for t, o in zip(prod, occ):
        t[0, o, 0] = 1.0
    tau, n = 80 * 0.0241888, 10                               # the paper's 80 a.u., in fs
    warm = pc_rk4.warmup(mpo, prod, tau, n, 32, cfg.M)
    assert [t.shape[2] for t in warm] == si.capped_bonds(dims, cfg.M)[1:]
    for A in warm[1:]:
        m = A.reshape(A.shape[0], -1)
        assert np.abs(m @ m.conj().T - np.eye(A.shape[0])).max() < 1e-13
    psi = list(exact.propagate(H, obs.mps_to_vector(prod), tau * n, 1))[-1]
    assert np.linalg.norm(obs.mps_to_vector(warm) - psi) < 1e-3
    lc = tdvp_mu.to_left_canonical(warm)
    sv = np.linalg.svd(lc[-1].reshape(lc[-1].shape[0], -1), compute_uv=False)
    assert sv[-1] > 1e-9 * sv[0]                              # the last bond carries weight in every state


# ---------------------------------------------------------------- two-site TDVP-PS (ref. 32)
def test_ps2_heff2_is_the_projected_hamiltonian():
    """H2 = P^dagger H P with P = P[1:i-1] (x) I_i (x) I_{i+1} (x) P[i+2:N], brute force in the full space."""
    from oracle import tdvp_ps2
    p = _small_params("A")
    H, dims = model.kronecker_sum_hamiltonian(p)
    H = H.toarray()
    mpo = model.build_mpo(p)
    for centre in (0, 1, 2):
        mps = _mixed_canonical(si.random_right_canonical_mps(dims, 4, seed=3), centre)
        Lenv = oc.boundary_env()
        for i in range(centre):
            Lenv = oc.envL(Lenv, mpo[i], mps[i])
        Renv = oc.boundary_env()
        for i in range(len(mps) - 1, centre + 1, -1):
            Renv = oc.envR(Renv, mpo[i], mps[i])
        PL, PR = _left_basis(mps, centre), _right_basis(mps, centre + 1)
        d1, d2 = dims[centre], dims[centre + 1]
        P = np.einsum("pa,su,tv,bq->pstqauvb", PL, np.eye(d1), np.eye(d2), PR).reshape(H.shape[0], -1)
        assert np.abs(P.conj().T @ P - np.eye(P.shape[1])).max() < 1e-13
        Theta = np.einsum("asc,ctb->astb", mps[centre], mps[centre + 1])
        brute = (P.conj().T @ H @ P @ Theta.reshape(-1)).reshape(Theta.shape)
        got = tdvp_ps2.heff2(Lenv, mpo[centre], mpo[centre + 1], Theta, Renv)
        assert np.abs(got - brute).max() < 1e-13
        rng = np.random.default_rng(centre)
        X = si.complex_normal(rng, Theta.shape)                    # not of product form
        assert np.abs(tdvp_ps2.heff2(Lenv, mpo[centre], mpo[centre + 1], X, Renv)
                      - (P.conj().T @ H @ P @ X.reshape(-1)).reshape(X.shape)).max() < 1e-12


def test_ps2_untruncated_is_exact_and_truncated_beats_nothing_worse_than_one_site(tiny_model):
    """With complete bonds (M = 64 on config 1's chain) the two-site integrator is e^{-iH tau} for any tau, like
    the one-site one (pin p3); at M = 16 it conserves the norm up to the truncation, stays within 1e-5 of exact
    propagation over 20 steps of 10 fs, and agrees with one-site TDVP-PS at the truncation level."""
    from oracle import tdvp_ps2
    cfg, params, mpo, dims, occ = tiny_model
    H, _ = model.kronecker_sum_hamiltonian(params)
    mps = si.padded_product_mps(dims, occ, 64, cfg.pad_seed)
    st = tdvp_ps.PSState(mpo, mps)
    ex = exact.propagate(H, obs.mps_to_vector(mps), 25.0, 2)
    for _ in range(2):
        tdvp_ps2.step_ps2(st, 25.0, 40)
        psi = next(ex)
    assert np.linalg.norm(obs.mps_to_vector(st.mps) - psi) < 2e-12
    for A in st.mps[1:]:                                           # back in the PS gauge
        m = A.reshape(A.shape[0], -1)
        assert np.abs(m @ m.conj().T - np.eye(A.shape[0])).max() < 1e-12
    mps = si.padded_product_mps(dims, occ, cfg.M, cfg.pad_seed)
    st2, st1 = tdvp_ps.PSState(mpo, mps), tdvp_ps.PSState(mpo, mps)
    ex = exact.propagate(H, obs.mps_to_vector(mps), cfg.dt_fs, cfg.n_steps)
    worst2 = worst12 = 0.0
    for _ in range(cfg.n_steps):
        tdvp_ps2.step_ps2(st2, cfg.dt_fs, 20)
        tdvp_ps.step_ps(st1, cfg.dt_fs, 20)
        pe = exact.site_populations(next(ex), dims)
        worst2 = max(worst2, np.abs(obs.populations(st2.mps) - pe).max())
        worst12 = max(worst12, np.abs(obs.populations(st2.mps) - obs.populations(st1.mps)).max())
    assert worst2 < 1e-5 and worst12 < 1e-5
    assert abs(obs.norm_sq(st2.mps) - 1.0) < 1e-6
    assert [a.shape for a in st2.mps] == [a.shape for a in mps]
