"""Parity of the CUDA path (through the C ABI of include/tdvp.h) against oracle/ on the same seeded
inputs.  Tolerances (BASELINE.json north_star): relative Frobenius error <= 1e-11 for one complex128
contraction; site populations within 1e-8 absolute after 20 steps."""
import dataclasses
import os

import numpy as np
import pytest

import synthetic_inputs as si
from oracle import contractions as oc
from oracle import lanczos, model, observables as obs, tdvp_ps

pytestmark = pytest.mark.gpu

REL_TOL = 1e-11


@pytest.fixture(scope="module")
def T():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1907_12044_b200 as t
    t.library_path()
    return t


def dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def host(x):
    return x.cpu().numpy()


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


# ---- single contractions --------------------------------------------------------------------
SITE_CASES = [
    # Ml, Mr, d, Dl, Dr, density
    (1, 3, 3, 1, 5, 0.5),        # left chain end
    (3, 1, 4, 4, 1, 0.5),        # right chain end
    (1, 1, 2, 1, 1, 1.0),        # degenerate 1-site chain
    (12, 16, 4, 5, 4, 0.3),
    (37, 29, 5, 7, 3, 0.2),      # ragged, several tiles with tails
    (64, 64, 10, 9, 9, 0.04),    # real-MPO-like density
    (70, 130, 3, 6, 11, 0.15),   # more than one 64-tile in both bonds, ragged
    (37, 70, 7, 9, 13, 0.3),     # long rows (row-block W kernel): 91 x 63 / 63 x 91, neither a multiple of 8 / 4
    (20, 33, 10, 20, 20, 0.5),   # long rows, half dense, 200 x 200
    (9, 64, 6, 12, 5, 1.0),      # dense W, rows 30 x cols 72 and the mirror
]


@pytest.mark.parametrize("case", SITE_CASES)
def test_apply_heff_ragged(T, case):
    Ml, Mr, d, Dl, Dr, dens = case
    L, W, A, R = si.random_site_problem(Ml, Mr, d, Dl, Dr, dens, seed=100 + Ml + Mr)
    want = oc.heff_definition(L, W, A, R) if Ml * Mr <= 600 else oc.heff(L, W, A, R)
    got = host(T.tdvp_apply_heff(dev(L), dev(W), dev(A), dev(R)))
    assert rel(got, want) <= REL_TOL


def test_gemm_products_three_and_four(T):
    """The GEMM stages with the complex product from 3 (default) or 4 real DMMA products
    (include/tdvp.h, DESIGN.md c15): both inside the 1e-11 gate, each reproducible bit for bit."""
    L, W, A, R = si.microbench_tensors(64)
    want = oc.heff(L, W, A, R)
    args = [dev(x) for x in (L, W, A, R)]
    assert T.tdvp_get_gemm_products() == 3
    try:
        res = {}
        for products in (3, 4, 3):
            T.tdvp_set_gemm_products(products)
            assert T.tdvp_get_gemm_products() == products
            got = host(T.tdvp_apply_heff(*args))
            assert rel(got, want) <= REL_TOL
            if products in res:
                assert np.array_equal(res[products], got)
            res[products] = got
        assert not np.array_equal(res[3], res[4])           # they are different arithmetic
        with pytest.raises(T.TdvpError):
            T.tdvp_set_gemm_products(5)
    finally:
        T.tdvp_set_gemm_products(3)


@pytest.mark.parametrize("M", [32, 64, 128])
def test_apply_heff_microbench_config(T, M):
    """BASELINE.json configs[1]: d = 10, D_W = 20, 6000 non-zeros of W."""
    L, W, A, R = si.microbench_tensors(M)
    want = oc.heff(L, W, A, R)
    got = host(T.tdvp_apply_heff(dev(L), dev(W), dev(A), dev(R)))
    assert rel(got, want) <= REL_TOL


def test_apply_heff_host_entry(T):
    L, W, A, R = si.microbench_tensors(32)
    out = np.empty_like(A)
    T.tdvp_apply_heff_host(L, W, A, R, out)
    assert rel(out, oc.heff(L, W, A, R)) <= REL_TOL


@pytest.mark.parametrize("case", SITE_CASES)
@pytest.mark.parametrize("side", [0, 1])
def test_update_env_ragged(T, case, side):
    Ml, Mr, d, Dl, Dr, dens = case
    L, W, A, R = si.random_site_problem(Ml, Mr, d, Dl, Dr, dens, seed=200 + Ml + Mr)
    if side == 0:
        want = oc.envL(L, W, A)
        got = host(T.tdvp_update_env(0, dev(L), dev(W), dev(A)))
    else:
        want = oc.envR(R, W, A)
        got = host(T.tdvp_update_env(1, dev(R), dev(W), dev(A)))
    assert got.shape == want.shape
    assert rel(got, want) <= REL_TOL


@pytest.mark.parametrize("M", [32, 128])
def test_update_env_microbench_config(T, M):
    L, W, A, R = si.microbench_tensors(M)
    assert rel(host(T.tdvp_update_env(0, dev(L), dev(W), dev(A))), oc.envL(L, W, A)) <= REL_TOL
    assert rel(host(T.tdvp_update_env(1, dev(R), dev(W), dev(A))), oc.envR(R, W, A)) <= REL_TOL


@pytest.mark.parametrize("M", [256, 512])
def test_apply_heff_microbench_config_sampled(T, M):
    """The sweep's largest sizes in the launch configuration bench.py times (stream-K cuts in both GEMM
    stages, several W-stage items per SM): sampled output slabs out[a, :, :], each computed by the
    oracle from the definition restricted to that a (Eq. 29: L[a] is the only place a enters)."""
    L, W, A, R = si.microbench_tensors(M)
    got = host(T.tdvp_apply_heff(dev(L), dev(W), dev(A), dev(R)))
    rng = np.random.default_rng(M)
    for a in sorted(set([0, M - 1] + list(rng.integers(0, M, 4)))):
        want = oc.heff(L[a:a + 1], W, A, R)[0]
        assert rel(got[a], want) <= REL_TOL
    # env update at the same size: sampled slabs L'[b, :, :] need conj(A[:, :, b]) only
    gotE = host(T.tdvp_update_env(0, dev(L), dev(W), dev(A)))
    t2 = np.tensordot(np.tensordot(L, A, axes=([2], [0])), W, axes=([1, 2], [0, 2]))   # [a, y, s, v]
    for b in (0, M // 2 + 1, M - 1):
        want = np.tensordot(np.conj(A[:, :, b]), t2, axes=([0, 1], [0, 2]))             # [y, v]
        assert rel(gotE[b], want.T) <= REL_TOL


@pytest.mark.parametrize("dims", [(1, 1, 1), (5, 3, 4), (40, 72, 9), (128, 128, 20), (64, 64, 1), (100, 36, 3),
                                  (257, 129, 2), (8, 300, 1)])
def test_apply_bond(T, dims):
    Ml, Mr, Dw = dims
    rng = np.random.default_rng(300 + Ml)
    L = si.complex_normal(rng, (Ml, Dw, Ml))
    R = si.complex_normal(rng, (Mr, Dw, Mr))
    D = si.complex_normal(rng, (Ml, Mr))
    got = host(T.tdvp_apply_bond(dev(L), dev(D), dev(R)))
    assert rel(got, oc.bond(L, D, R)) <= REL_TOL


def test_contractions_random_shapes(T):
    """Seeded random shapes: many different stream-K schedules of the GEMM kernel (uncut, cut once,
    cut many times, batched right-environment stage, ragged k-tiles) and W-stage panel shapes."""
    rng = np.random.default_rng(20240611)
    for _ in range(24):
        Ml, Mr, Dw = int(rng.integers(1, 200)), int(rng.integers(1, 200)), int(rng.integers(1, 7))
        L = si.complex_normal(rng, (Ml, Dw, Ml))
        R = si.complex_normal(rng, (Mr, Dw, Mr))
        D = si.complex_normal(rng, (Ml, Mr))
        assert rel(host(T.tdvp_apply_bond(dev(L), dev(D), dev(R))), oc.bond(L, D, R)) <= REL_TOL, (Ml, Mr, Dw)
    for k in range(10):
        Ml, Mr = int(rng.integers(1, 90)), int(rng.integers(1, 90))
        d, Dl, Dr = int(rng.integers(1, 6)), int(rng.integers(1, 8)), int(rng.integers(1, 8))
        L, W, A, R = si.random_site_problem(Ml, Mr, d, Dl, Dr, 0.3, seed=900 + k)
        assert rel(host(T.tdvp_apply_heff(dev(L), dev(W), dev(A), dev(R))), oc.heff(L, W, A, R)) <= REL_TOL, (Ml, Mr, d, Dl, Dr)
        assert rel(host(T.tdvp_update_env(0, dev(L), dev(W), dev(A))), oc.envL(L, W, A)) <= REL_TOL, (Ml, Mr, d, Dl, Dr)
        assert rel(host(T.tdvp_update_env(1, dev(R), dev(W), dev(A))), oc.envR(R, W, A)) <= REL_TOL, (Ml, Mr, d, Dl, Dr)


# ---- QR gauge move (Eq. 9) ------------------------------------------------------------------
# the last four shapes reach the panel variants for tall sides of 1280 / 2560 / 5120 rows and beyond
@pytest.mark.parametrize("shape", [(1, 3, 3), (3, 4, 12), (16, 4, 16), (37, 5, 29), (64, 10, 64), (130, 3, 70),
                                   (128, 10, 128), (200, 10, 200), (260, 16, 64), (90, 64, 40)])
@pytest.mark.parametrize("side", [0, 1])
def test_qr_gauge(T, shape, side):
    Ml, d, Mr = shape
    if side == 0 and Ml * d < Mr:
        pytest.skip("not tall")
    if side == 1 and d * Mr < Ml:
        pytest.skip("not tall")
    rng = np.random.default_rng(400 + Ml + Mr)
    C = si.complex_normal(rng, shape)
    # make it numerically rank deficient like a padded centre: scale trailing columns / rows down
    if side == 0:
        C = C * np.logspace(0, -9, Mr)[None, None, :]
    else:
        C = C * np.logspace(0, -9, Ml)[:, None, None]
    Q, D = T.tdvp_qr_gauge(side, dev(C))
    Q, D = host(Q), host(D)
    if side == 0:
        Qm = Q.reshape(Ml * d, Mr)
        assert np.abs(Qm.conj().T @ Qm - np.eye(Mr)).max() < 1e-13 * max(Mr, 8)      # Eq. 7
        assert rel((Qm @ D).reshape(shape), C) < 1e-13
    else:
        Qm = Q.reshape(Ml, d * Mr)
        assert np.abs(Qm @ Qm.conj().T - np.eye(Ml)).max() < 1e-13 * max(Ml, 8)      # Eq. 8
        assert rel((D @ Qm).reshape(shape), C) < 1e-13


# ---- Lanczos exponential on a Hermitian H_eff of a real chain ---------------------------------
def _tiny_state(n_warm=1):
    cfg = si.CONFIGS["tiny"]
    params = si.draw_vibronic_params(cfg)
    mpo = model.build_mpo(params)
    mps = si.padded_product_mps(si.site_dims(params), si.initial_occupations(params), cfg.M, cfg.pad_seed)
    st = tdvp_ps.PSState(mpo, mps)
    for _ in range(n_warm):
        tdvp_ps.step_ps(st, cfg.dt_fs, cfg.krylov_dim)
    return cfg, mpo, st


def test_expm_heff_and_bond(T):
    cfg, mpo, st = _tiny_state()
    # move the centre two sites to the right by hand so that L and R are both non-trivial
    for i in range(2):
        C = st.mps[i]
        Ml, d, Mr = C.shape
        Q, D = np.linalg.qr(C.reshape(Ml * d, Mr))
        st.mps[i] = Q.reshape(Ml, d, Mr)
        st.Lenv[i + 1] = oc.envL(st.Lenv[i], mpo[i], st.mps[i])
        st.mps[i + 1] = np.einsum("ab,bsc->asc", D, st.mps[i + 1])
    i = 2
    L, W, R, v = st.Lenv[i], mpo[i], st.Renv[i], st.mps[i]
    for k in (10, 4):
        ctx = T.tdvp_create_context(T.make_options(krylov_dim=k))
        z = -0.5j * cfg.dt_fs
        want, m = lanczos.lanczos_expm(lambda x: oc.heff(L, W, x, R), v, z, k)
        got, mg = T.tdvp_expm_heff(dev(L), dev(W), dev(R), z, dev(v), handle=ctx, want_dim=True)
        assert mg == m
        assert rel(host(got), want) <= REL_TOL
        # bond operator between sites 1 and 2
        Lb, Rb = st.Lenv[2], st.Renv[1]
        rng = np.random.default_rng(5)
        Dm = si.complex_normal(rng, (Lb.shape[0], Rb.shape[0]))
        want, m = lanczos.lanczos_expm(lambda x: oc.bond(Lb, x, Rb), Dm, -z, k)
        got, mg = T.tdvp_expm_bond(dev(Lb), dev(Rb), -z, dev(Dm), handle=ctx, want_dim=True)
        assert mg == m
        assert rel(host(got), want) <= REL_TOL
        ctx.close()


def test_expm_breakdown_small_space(T):
    """Krylov space exhausted (1-dimensional bond at a chain end): m < k on both sides."""
    cfg, mpo, st = _tiny_state(0)
    L, W, R, v = st.Lenv[0], mpo[0], st.Renv[0], st.mps[0]       # dimension 1*3*3 = 9 < k = 10
    z = -0.5j * cfg.dt_fs
    want, m = lanczos.lanczos_expm(lambda x: oc.heff(L, W, x, R), v, z, 10)
    got, mg = T.tdvp_expm_heff(dev(L), dev(W), dev(R), z, dev(v), want_dim=True)
    assert mg == m and m < 10
    assert rel(host(got), want) <= 1e-10


def _hermitian_product_operator(Ml, d, Mr, seed):
    """L, W, R with D_W = 1 and Hermitian factors: H = L (x) h (x) R^T is Hermitian, cheap at any size."""
    rng = np.random.default_rng(seed)
    def herm(n):
        g = si.complex_normal(rng, (n, n))
        return (g + g.conj().T) / (2.0 * np.sqrt(2.0 * n))
    L = herm(Ml).reshape(Ml, 1, Ml)
    R = herm(Mr).reshape(Mr, 1, Mr)
    W = herm(d).reshape(1, d, d, 1) * 3.0
    v = si.complex_normal(rng, (Ml, d, Mr))
    return np.ascontiguousarray(L), np.ascontiguousarray(W), np.ascontiguousarray(R), v


@pytest.mark.parametrize("case", [(100, 6, 100, 40, -0.9j),     # 41 vectors of 60 000: the basis does not fit in shared memory
                                  (450, 10, 450, 4, 1.3j),       # 2 M elements: not even the chunk of w fits
                                  (33, 3, 29, 64, -2.0j),        # k = 64: both halves of the coefficient warp
                                  (16, 2, 16, 7, -0.4 + 0.3j)])  # z with a real part: eigen-decomposition path
def test_expm_large_and_general(T, case):
    Ml, d, Mr, k, z = case
    L, W, R, v = _hermitian_product_operator(Ml, d, Mr, seed=70 + Ml)
    want, m = lanczos.lanczos_expm(lambda x: oc.heff(L, W, x, R), v, z, k)
    ctx = T.tdvp_create_context(T.make_options(krylov_dim=k))
    got, mg = T.tdvp_expm_heff(dev(L), dev(W), dev(R), z, dev(v), handle=ctx, want_dim=True)
    assert mg == m
    assert rel(host(got), want) <= REL_TOL
    ctx.close()


@pytest.mark.parametrize("tol", [1e-6, 1e-10])
def test_expm_adaptive_krylov_dimension(T, tol):
    """opt.krylov_tol > 0 (reading c11): the device stops at the same Krylov
    dimension as the oracle's rule, the result agrees to 1e-11, and the error against the dense
    exponential is of the order of tol."""
    import scipy.linalg
    Ml, d, Mr = 12, 3, 10
    L, W, R, v = _hermitian_product_operator(Ml, d, Mr, seed=5)
    z = -4.0j
    want, m = lanczos.lanczos_expm(lambda x: oc.heff(L, W, x, R), v, z, 48, tol=tol)
    assert 4 < m < 48
    ctx = T.tdvp_create_context(T.make_options(krylov_dim=48, krylov_tol=tol))
    got, mg = T.tdvp_expm_heff(dev(L), dev(W), dev(R), z, dev(v), handle=ctx, want_dim=True)
    assert mg == m
    assert rel(host(got), want) <= REL_TOL
    Hd = np.einsum("ax,st,by->asbxty", L[:, 0, :], W[0, :, :, 0], R[:, 0, :]).reshape(Ml * d * Mr, -1)
    ref = scipy.linalg.expm(z * Hd) @ v.reshape(-1)
    assert np.linalg.norm(host(got).reshape(-1) - ref) <= 20 * tol * np.linalg.norm(v)
    # the bond operator through the same rule
    rng = np.random.default_rng(6)
    Dm = si.complex_normal(rng, (Ml, Mr))
    want, m = lanczos.lanczos_expm(lambda x: oc.bond(L, x, R), Dm, -z, 48, tol=tol)
    got, mg = T.tdvp_expm_bond(dev(L), dev(R), -z, dev(Dm), handle=ctx, want_dim=True)
    assert mg == m and rel(host(got), want) <= REL_TOL
    ctx.close()


def test_tiny_chain_adaptive_krylov(T):
    """TDVP-PS with the adaptive Krylov dimension (cap 30, tol 1e-9) against the oracle running the same
    rule: 10 steps of configs[0], populations 1e-8; the converged dimension beats the fixed k = 10 run
    against exact propagation (k = 10 costs 4e-6 there)."""
    cfg = si.CONFIGS["tiny"]
    params = si.draw_vibronic_params(cfg)
    mpo = model.build_mpo(params)
    mps = si.padded_product_mps(si.site_dims(params), si.initial_occupations(params), cfg.M, cfg.pad_seed)
    st = tdvp_ps.PSState(mpo, mps)
    ch = T.tdvp_create(mpo, mps, T.make_options(krylov_dim=30, krylov_tol=1e-9))
    for s in range(10):
        tdvp_ps.step_ps(st, cfg.dt_fs, 30, tol=1e-9)
        ch.tdvp_step_ps(cfg.dt_fs)
        assert np.abs(ch.tdvp_populations(0) - obs.populations(st.mps)).max() <= 1e-8
    assert 4 < max(st.krylov_dims) < 30 and len(set(st.krylov_dims)) > 1      # the rule, not the cap, stopped every exponential
    nrm, _ = ch.tdvp_norm_energy()
    assert abs(nrm - 1.0) < 1e-8                               # unitary up to the tolerance of the rule
    ch.close()


# ---- whole trajectories ---------------------------------------------------------------------
@pytest.mark.parametrize("graph", [True, False])
def test_tiny_chain_20_steps(T, graph):
    """BASELINE.json configs[0]: populations within 1e-8 of the oracle after each of 20 steps."""
    cfg = si.CONFIGS["tiny"]
    params = si.draw_vibronic_params(cfg)
    mpo = model.build_mpo(params)
    mps = si.padded_product_mps(si.site_dims(params), si.initial_occupations(params), cfg.M, cfg.pad_seed)
    golden = np.loadtxt(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "tiny_ps_populations.txt"))
    ch = T.tdvp_create(mpo, mps, T.make_options(krylov_dim=cfg.krylov_dim, flags=0 if graph else T.TDVP_FLAG_NO_GRAPH))
    n0, e0 = ch.tdvp_norm_energy()
    assert abs(n0 - 1.0) < 1e-12
    assert abs(e0 - obs.energy(mpo, mps)) < 1e-12 * max(1.0, abs(e0))
    worst = 0.0
    for s in range(cfg.n_steps):
        ch.tdvp_step_ps(cfg.dt_fs)
        p = ch.tdvp_populations(0)
        worst = max(worst, np.abs(p - golden[s]).max())
    assert worst <= 1e-8
    n1, e1 = ch.tdvp_norm_energy()
    assert abs(n1 - 1.0) < 1e-11 and abs(e1 - e0) < 1e-11 * max(1.0, abs(e0))
    assert ch.tdvp_get_centre() == 0
    ch.close()


def test_fmo_like_chain_delta_seeded(T):
    """A short FMO-like chain (layout A, d = 10 phonon sites) at M = 12, delta-seeded start
    (SURVEY.md 8(c) c8): free-running parity over 4 steps, plus observables."""
    cfg = dataclasses.replace(si.CONFIGS["fmo64"], n_el=4, n_modes=2, n_ph=6, M=12, dt_fs=5.0)
    params = si.draw_vibronic_params(cfg)
    mpo = model.build_mpo(params)
    dims = si.site_dims(params)
    mps = si.padded_product_mps(dims, si.initial_occupations(params), cfg.M, cfg.pad_seed, cfg.delta, cfg.delta_seed)
    st = tdvp_ps.PSState(mpo, mps)
    ch = T.tdvp_create(mpo, mps, T.make_options(krylov_dim=cfg.krylov_dim))
    for s in range(4):
        tdvp_ps.step_ps(st, cfg.dt_fs, cfg.krylov_dim)
        ch.tdvp_step_ps(cfg.dt_fs)
        assert np.abs(ch.tdvp_populations(0) - obs.populations(st.mps, 0)).max() <= 1e-8
    # a phonon-site observable: <n> at site 3 through tdvp_observe
    num = np.diag(np.arange(dims[3], dtype=np.float64)).astype(np.complex128)
    want = np.trace(num @ obs.one_site_rdm(st.mps, 3))
    assert abs(ch.tdvp_observe(3, num) - want) <= 1e-8
    # state overlap |<psi_oracle|psi_gpu>| = 1 (gauge invariant)
    got = ch.tdvp_get_mps()
    E = np.ones((1, 1), dtype=np.complex128)
    for A, B in zip(st.mps, got):
        E = np.einsum("ax,asb,xsy->by", E, A.conj(), B)
    assert abs(abs(E[0, 0]) - 1.0) <= 1e-9
    ch.close()


def test_large_chain_invariants(T):
    """BASELINE.json configs[4] at full size (147 sites, layout B, M = 256): the oracle needs minutes per
    step there, so the full-size run is gated on what holds at any size -- norm, energy and the
    population sum are conserved by TDVP-PS (pin p4 for the oracle)."""
    cfg = si.CONFIGS["fmo256"]
    params = si.draw_vibronic_params(cfg)
    mpo = model.build_mpo(params)
    mps = si.padded_product_mps(si.site_dims(params), si.initial_occupations(params), cfg.M, cfg.pad_seed, cfg.delta, cfg.delta_seed)
    assert len(mps) == 147 and max(a.shape[2] for a in mps) == 256
    ch = T.tdvp_create(mpo, mps, T.make_options(krylov_dim=cfg.krylov_dim))
    n0, e0 = ch.tdvp_norm_energy()
    ch.tdvp_step_ps(cfg.dt_fs)
    n1, e1 = ch.tdvp_norm_energy()
    pops = ch.tdvp_populations(0)
    ch.close()
    assert abs(n1 - 1.0) < 1e-11 and abs(n0 - 1.0) < 1e-12
    assert abs(e1 - e0) < 1e-9 * abs(e0)
    assert abs(float(np.sum(pops)) - 1.0) < 1e-11 and np.all(pops > -1e-12)


def test_teacher_forced_step(T):
    """tdvp_set_mps with the oracle's tensors, one step, compare."""
    cfg, mpo, st = _tiny_state(3)
    ch = T.tdvp_create(mpo, st.mps, T.make_options(krylov_dim=cfg.krylov_dim))
    for _ in range(2):
        ch.tdvp_set_mps(st.mps, 0)
        tdvp_ps.step_ps(st, cfg.dt_fs, cfg.krylov_dim)
        ch.tdvp_step_ps(cfg.dt_fs)
        assert np.abs(ch.tdvp_populations(0) - obs.populations(st.mps, 0)).max() <= 1e-10
    ch.close()


def test_gauge_sweep_and_site_calls(T):
    cfg, mpo, st = _tiny_state(2)
    ch = T.tdvp_create(mpo, st.mps)
    p0 = ch.tdvp_populations(0)
    n0, e0 = ch.tdvp_norm_energy()
    ch.tdvp_set_gauge(ch.n - 1)
    assert ch.tdvp_get_centre() == ch.n - 1
    assert np.abs(ch.tdvp_populations(0) - p0).max() < 1e-12
    n1, e1 = ch.tdvp_norm_energy()
    assert abs(n1 - n0) < 1e-12 and abs(e1 - e0) < 1e-12 * max(1, abs(e0))
    # energy = <C, H_eff C> at the centre
    C = ch.tdvp_get_mps(ch.n - 1)
    HC = host(ch.tdvp_apply_heff_site(ch.n - 1, dev(C)))
    assert abs(np.vdot(C, HC).real - e0) < 1e-11 * max(1, abs(e0))
    ch.tdvp_set_gauge(0)
    assert np.abs(ch.tdvp_populations(0) - p0).max() < 1e-12
    ch.close()


def test_errors_are_reported(T):
    with pytest.raises(T.TdvpError):
        T.make_options(krylov_dim=0) and T.tdvp_create_context(T.make_options(krylov_dim=0))
    cfg, mpo, st = _tiny_state(0)
    bad = [A.copy() for A in st.mps]
    bad[3] = bad[3] * 1.5                               # not right-canonical
    with pytest.raises(T.TdvpError):
        T.tdvp_create(mpo, bad)


# ---- TDVP-MU: matrix unfolding (Eq. 36), derivative (Eq. 27, 37, 38), Dormand-Prince step ------
# the last three shapes (Ml > 128) reach the generic looped Jacobi kernel, the path of TDVP-MU at M = 256
@pytest.mark.parametrize("shape", [(1, 3, 4), (4, 3, 4), (12, 4, 16), (37, 5, 29), (64, 10, 64), (70, 3, 130),
                                   (128, 10, 128), (160, 4, 160), (256, 2, 256)])
@pytest.mark.parametrize("deficient", [False, True])
def test_svd_bond(T, shape, deficient):
    Ml, d, Mr = shape
    rng = np.random.default_rng(500 + Ml + Mr)
    C = si.complex_normal(rng, shape)
    if deficient and Ml > 2:                       # graded singular values and an exact null space
        Um, _ = np.linalg.qr(si.complex_normal(rng, (Ml, Ml)))
        Vm, _ = np.linalg.qr(si.complex_normal(rng, (d * Mr, Ml)))
        sv = np.logspace(0, -10, Ml)
        sv[-2:] = 0.0
        C = ((Um * sv[None, :]) @ Vm.conj().T).reshape(shape)
    U, lam, Vh = [host(x) for x in T.tdvp_svd_bond(dev(C))]
    Vm = Vh.reshape(Ml, d * Mr)
    tol = 1e-13 * max(Ml, 8)
    assert np.abs(U.conj().T @ U - np.eye(Ml)).max() < tol
    assert np.abs(Vm @ Vm.conj().T - np.eye(Ml)).max() < tol              # Eq. 8
    assert np.all(np.diff(lam) <= 0) and np.all(lam >= 0)
    want = np.linalg.svd(C.reshape(Ml, d * Mr), compute_uv=False)
    assert np.abs(lam - want).max() <= 1e-13 * want[0]
    assert rel(((U * lam[None, :]) @ Vm).reshape(shape), C) < 1e-13


def _warm_left_canonical(n_warm=3):
    from oracle import tdvp_mu
    cfg, mpo, st = _tiny_state(n_warm)
    return cfg, mpo, tdvp_mu.to_left_canonical(st.mps)


def test_mu_derivative(T):
    from oracle import tdvp_mu
    cfg, mpo, mpsL = _warm_left_canonical()
    want = tdvp_mu.mu_derivative(mpo, mpsL)
    ch = T.tdvp_create(mpo, tdvp_mu.to_right_canonical(mpsL))
    ch.tdvp_set_mps(mpsL, centre=ch.n - 1)
    got = ch.tdvp_mu_derivative()
    scale = max(np.linalg.norm(w) for w in want)         # complete bonds have (1 - p) = 0: dL/dt = round-off there
    for g, w in zip(got, want):
        assert np.linalg.norm(g - w) <= 1e-8 * scale
    for g, Lsite in zip(got[:-1], mpsL[:-1]):                              # Eq. 34: L^dagger dL/dt = 0
        a, s, b = Lsite.shape
        assert np.abs(Lsite.reshape(a * s, b).conj().T @ g.reshape(a * s, b)).max() < 1e-9
    ch.close()


def test_mu_step_matches_oracle_and_ps(T):
    """Dormand-Prince steps of h = 0.1 fs after a shared PS warm-up."""
    from oracle import tdvp_mu
    cfg, mpo, mpsL = _warm_left_canonical()
    ch = T.tdvp_create(mpo, tdvp_mu.to_right_canonical(mpsL))
    ch.tdvp_set_mps(mpsL, centre=ch.n - 1)
    cur = mpsL
    for s in range(4):
        cur, err_want = tdvp_mu.step_mu(mpo, cur, 0.1)
        err_got = ch.tdvp_step_mu(0.1, want_err=True)
        assert abs(err_got - err_want) <= 1e-6 * max(err_want, 1e-12) + 1e-14
        assert np.abs(ch.tdvp_populations(0) - obs.populations(cur, 0)).max() <= 1e-8
    nrm, en = ch.tdvp_norm_energy()
    assert abs(nrm - obs.norm_sq(cur)) < 1e-10 and abs(en - obs.energy(mpo, cur)) < 1e-9
    # switching back to the PS gauge leaves the state unchanged
    p = ch.tdvp_populations(0)
    ch.tdvp_set_gauge(0)
    assert np.abs(ch.tdvp_populations(0) - p).max() < 1e-12
    ch.close()


def test_mu_first_same_as_last_is_exact(T):
    """Dormand-Prince's stage 7 is evaluated at the new state, so the library reuses it as stage 1 of
    the next step; TDVP_NO_FSAL=1 (read at every step) recomputes it: both must give the same bits."""
    cfg, mpo, mpsL = _warm_left_canonical()
    from oracle import tdvp_mu
    res = []
    for no_fsal in (False, True):
        ch = T.tdvp_create(mpo, tdvp_mu.to_right_canonical(mpsL))
        ch.tdvp_set_mps(mpsL, centre=ch.n - 1)
        if no_fsal:
            os.environ["TDVP_NO_FSAL"] = "1"
        try:
            errs = [ch.tdvp_step_mu(0.1, want_err=True) for _ in range(3)]
        finally:
            os.environ.pop("TDVP_NO_FSAL", None)
        res.append((errs, ch.tdvp_populations(0)))
        ch.close()
    assert res[0][0] == res[1][0]
    assert np.array_equal(res[0][1], res[1][1])


def test_mu_cmf_step_matches_oracle(T):
    """TDVP-MU with constant-mean-field integration: CMF
    steps of 0.5 fs (8 RK4 sub-steps per site, Krylov dimension 10 at the last site) after a shared
    PS warm-up, against oracle/tdvp_cmf.py on the same tensors: populations 1e-8, norm, energy, and
    the state overlap (gauge-free) after every step."""
    from oracle import tdvp_mu, tdvp_cmf
    cfg, mpo, mpsL = _warm_left_canonical()
    ch = T.tdvp_create(mpo, tdvp_mu.to_right_canonical(mpsL), T.make_options(krylov_dim=10))
    ch.tdvp_set_mps(mpsL, centre=ch.n - 1)
    cur = mpsL
    for s in range(3):
        cur = tdvp_cmf.step_cmf(mpo, cur, 0.5, 8, 10)
        ch.tdvp_step_mu_cmf(0.5, 8)
        assert ch.tdvp_get_centre() == ch.n - 1
        assert np.abs(ch.tdvp_populations(0) - obs.populations(cur, 0)).max() <= 1e-8
        got = [ch.tdvp_get_mps(i) for i in range(ch.n)]
        ov = np.vdot(obs.mps_to_vector(cur), obs.mps_to_vector(got))
        assert abs(abs(ov) - 1.0) < 1e-9
    nrm, en = ch.tdvp_norm_energy()
    assert abs(nrm - obs.norm_sq(cur)) < 1e-10 and abs(en - obs.energy(mpo, cur)) < 1e-9
    ch.close()


def test_mu_cmf_odd_substeps_and_ps_gauge(T):
    """n_sub odd (half step uses ceil(n_sub / 2) sub-steps) and a handle that starts in the PS gauge."""
    from oracle import tdvp_mu, tdvp_cmf
    cfg, mpo, st = _tiny_state(3)
    ch = T.tdvp_create(mpo, st.mps, T.make_options(krylov_dim=10))
    cur = tdvp_cmf.step_cmf(mpo, tdvp_mu.to_left_canonical(st.mps), 0.25, 5, 10)
    ch.tdvp_step_mu_cmf(0.25, 5)
    assert ch.tdvp_get_centre() == ch.n - 1
    assert np.abs(ch.tdvp_populations(0) - obs.populations(cur, 0)).max() <= 1e-8
    with pytest.raises(T.TdvpError):
        ch.tdvp_step_mu_cmf(0.25, 0)
    ch.close()


def test_mu_cmf_fmo_like_chain(T):
    """CMF steps on a short FMO-like chain (layout A, d = 6 phonon sites, D_W up to 6, M = 12) after a
    shared PS warm-up from the delta-seeded start: populations, a phonon-site observable, overlap."""
    from oracle import tdvp_mu, tdvp_cmf
    cfg = dataclasses.replace(si.CONFIGS["fmo64"], n_el=4, n_modes=2, n_ph=6, M=12, dt_fs=5.0)
    params = si.draw_vibronic_params(cfg)
    mpo = model.build_mpo(params)
    dims = si.site_dims(params)
    mps = si.padded_product_mps(dims, si.initial_occupations(params), cfg.M, cfg.pad_seed, cfg.delta, cfg.delta_seed)
    st = tdvp_ps.PSState(mpo, mps)
    for _ in range(4):
        tdvp_ps.step_ps(st, cfg.dt_fs, cfg.krylov_dim)
    cur = tdvp_mu.to_left_canonical(st.mps)
    ch = T.tdvp_create(mpo, st.mps, T.make_options(krylov_dim=cfg.krylov_dim))
    ch.tdvp_set_mps(cur, centre=ch.n - 1)
    for s in range(2):
        cur = tdvp_cmf.step_cmf(mpo, cur, 0.05, 10, cfg.krylov_dim)
        ch.tdvp_step_mu_cmf(0.05, 10)
        assert np.abs(ch.tdvp_populations(0) - obs.populations(cur, 0)).max() <= 1e-8
    num = np.diag(np.arange(dims[3], dtype=np.float64)).astype(np.complex128)
    assert abs(ch.tdvp_observe(3, num) - np.trace(num @ obs.one_site_rdm(cur, 3))) <= 1e-8
    ov = np.vdot(obs.mps_to_vector(cur), obs.mps_to_vector(ch.tdvp_get_mps()))
    assert abs(abs(ov) - 1.0) <= 1e-8
    ch.close()


def test_mu_step_from_ps_gauge(T):
    """tdvp_step_mu on a handle in the PS gauge first moves the centre (no time evolution)."""
    cfg, mpo, st = _tiny_state(3)
    ch = T.tdvp_create(mpo, st.mps)
    p0 = ch.tdvp_populations(0)
    ch.tdvp_step_mu(1e-6)
    assert ch.tdvp_get_centre() == ch.n - 1
    assert np.abs(ch.tdvp_populations(0) - p0).max() < 1e-6
    ch.close()
