"""tdvp_qr_gauge_noalloc (include/tdvp.h): the QR gauge move with its scratch in a static device array inside
the library -- for callers that cannot call cudaMalloc.  Checked against the existing path (tdvp_qr_gauge, whose
scratch is the handle's arena) on two calls in a row with different shapes, so that the second call runs on a
scratch block full of the first call's data.  Collected last on purpose (file name): the suite runs with
pytest -x, and a failure here must not hide other tests."""
import numpy as np
import pytest

import synthetic_inputs as si

pytestmark = pytest.mark.gpu

# (shape [Ml, d, Mr], side): the 1280 x 128 move of configs[3] (the largest the 6 MiB block takes, cluster
# kernel), then a ragged RQ of another size on the same -- now stale -- scratch
CALLS = [((128, 10, 128), 0), ((37, 5, 29), 1)]


@pytest.fixture(scope="module")
def T():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1907_12044_b200 as t
    t.library_path()
    return t


def _inputs(shape, side):
    rng = np.random.default_rng(900 + shape[0] + side)
    C = si.complex_normal(rng, shape)
    n = shape[2] if side == 0 else shape[0]
    grade = np.logspace(0, -9, n)                       # numerically rank deficient, like a padded centre
    return C * (grade[None, None, :] if side == 0 else grade[:, None, None])


def test_qr_gauge_noalloc_matches_the_arena_path_twice_in_a_row(T):
    import torch
    Cs, want, outs = [], [], []
    for shape, side in CALLS:
        C = torch.from_numpy(_inputs(shape, side)).cuda()
        Q0, D0 = T.tdvp_qr_gauge(side, C)               # existing path
        n = shape[2] if side == 0 else shape[0]
        Cs.append(C)
        want.append((Q0.cpu().numpy(), D0.cpu().numpy()))
        outs.append((torch.empty_like(C), torch.empty((n, n), dtype=torch.complex128, device="cuda")))

    def run_all():
        for (shape, side), C, (Q, D) in zip(CALLS, Cs, outs):
            Q.zero_(); D.zero_()
            T.tdvp_qr_gauge_noalloc(side, C, Q, D)      # two calls in a row, one shared scratch block
        torch.cuda.synchronize()

    def check():
        for (shape, side), C, (Q, D), (Qw, Dw) in zip(CALLS, Cs, outs, want):
            Qg, Dg, Cn = Q.cpu().numpy(), D.cpu().numpy(), C.cpu().numpy()
            Ml, d, Mr = shape
            # same kernels, same order of operations: the two paths agree to the tolerance of the QR tests
            assert np.linalg.norm(Qg - Qw) <= 1e-13 * np.linalg.norm(Qw)
            assert np.linalg.norm(Dg - Dw) <= 1e-13 * np.linalg.norm(Dw)
            if side == 0:
                Qm = Qg.reshape(Ml * d, Mr)
                assert np.abs(Qm.conj().T @ Qm - np.eye(Mr)).max() < 1e-13 * max(Mr, 8)      # Eq. 7
                assert np.linalg.norm((Qm @ Dg).reshape(shape) - Cn) < 1e-13 * np.linalg.norm(Cn)
            else:
                Qm = Qg.reshape(Ml, d * Mr)
                assert np.abs(Qm @ Qm.conj().T - np.eye(Ml)).max() < 1e-13 * max(Ml, 8)      # Eq. 8
                assert np.linalg.norm((Dg @ Qm).reshape(shape) - Cn) < 1e-13 * np.linalg.norm(Cn)

    run_all()                                           # first use: symbol address taken, kernels loaded
    check()
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        run_all()
    free1 = torch.cuda.mem_get_info()[0]
    check()
    assert free1 == free0, "device memory changed by %d bytes across no-alloc calls" % (free0 - free1)


def test_qr_gauge_noalloc_rejects_what_does_not_fit(T):
    import torch
    C = torch.zeros((200, 10, 200), dtype=torch.complex128, device="cuda")     # 2000 x 200: 13 MB of scratch
    Q, D = torch.empty_like(C), torch.empty((200, 200), dtype=torch.complex128, device="cuda")
    with pytest.raises(T.TdvpError) as ei:
        T.tdvp_qr_gauge_noalloc(0, C, Q, D)
    assert ei.value.code == T.TDVP_EINVAL and "6 MiB" in str(ei.value)
    C2 = torch.zeros((64, 1, 8), dtype=torch.complex128, device="cuda")        # wide for side 1: not a gauge move
    with pytest.raises(T.TdvpError):
        T.tdvp_qr_gauge_noalloc(1, C2, torch.empty_like(C2), torch.empty((64, 64), dtype=torch.complex128, device="cuda"))
