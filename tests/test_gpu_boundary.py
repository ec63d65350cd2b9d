"""Error behaviour of the C ABI on the GPU (include/tdvp.h "Errors"): every failure is a negative
TDVP_E* return code with a message, never a signal; device memory is given back."""
import ctypes
import os

import numpy as np
import pytest

import synthetic_inputs as si

pytestmark = pytest.mark.gpu


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


def test_misaligned_operand_is_einval_not_abort(T):
    """A DEVICE pointer that is 8- but not 16-byte aligned cannot be described by a TMA tensor map: the
    GEMM stage used to abort() the process; now the call returns TDVP_EINVAL and the library keeps working."""
    import torch
    from paper_1907_12044_b200 import binding as b
    L, W, A, R = (dev(x) for x in si.random_site_problem(12, 16, 4, 5, 4, 0.3, seed=1))
    out = torch.empty_like(A)
    raw = torch.empty(A.numel() * 2 + 2, dtype=torch.float64, device="cuda")
    raw[1:1 + 2 * A.numel()] = torch.view_as_real(A).reshape(-1)
    bad_ptr = raw.data_ptr() + 8
    assert bad_ptr % 16 == 8
    ctx = T.tdvp_create_context()
    rc = b._lib.tdvp_apply_heff(ctx._h, 12, 16, 4, 5, 4, L.data_ptr(), W.data_ptr(), ctypes.c_void_p(bad_ptr), R.data_ptr(),
                                out.data_ptr())
    assert rc == T.TDVP_EINVAL
    assert b"aligned" in b._lib.tdvp_last_error(ctx._h)
    ctx.tdvp_sync()
    from oracle import contractions as oc
    got = T.tdvp_apply_heff(L, W, A, R, handle=ctx).cpu().numpy()           # the handle still works
    want = oc.heff(*(x.cpu().numpy() for x in (L, W, A, R)))
    assert np.linalg.norm(got - want) <= 1e-11 * np.linalg.norm(want)
    ctx.close()


def test_svd_out_of_sweeps_is_estate_at_next_blocking_call(T):
    rng = np.random.default_rng(3)
    C = dev(si.complex_normal(rng, (48, 3, 40)))
    ctx = T.tdvp_create_context()
    os.environ["TDVP_SVD_MAX_SWEEPS"] = "1"
    try:
        T.tdvp_svd_bond(C, handle=ctx)                     # enqueue only: cannot know yet
    finally:
        os.environ.pop("TDVP_SVD_MAX_SWEEPS", None)
    with pytest.raises(T.TdvpError) as ei:
        ctx.tdvp_sync()
    assert ei.value.code == T.TDVP_ESTATE and "SVD" in str(ei.value)
    ctx.tdvp_sync()                                        # the report clears the condition
    U, lam, Vh = T.tdvp_svd_bond(C, handle=ctx)            # default sweeps: converges
    ctx.tdvp_sync()
    want = np.linalg.svd(C.cpu().numpy().reshape(48, 120), compute_uv=False)
    assert np.abs(lam.cpu().numpy() - want).max() <= 1e-13 * want[0]
    ctx.close()


def test_too_tall_gauge_move_is_einval(T):
    """rows > 12800 used to divide by zero (SIGFPE) in the panel-width computation."""
    import torch
    C = torch.zeros((1300, 10, 2), dtype=torch.complex128, device="cuda")
    with pytest.raises(T.TdvpError) as ei:
        T.tdvp_qr_gauge(0, C)
    assert ei.value.code == T.TDVP_EINVAL
    C2 = torch.zeros((2, 10, 1300), dtype=torch.complex128, device="cuda")
    with pytest.raises(T.TdvpError):
        T.tdvp_qr_gauge(1, C2)
    with pytest.raises(T.TdvpError):
        T.tdvp_svd_bond(C2)


def _tiny():
    from oracle import model
    cfg = si.CONFIGS["tiny"]
    params = si.draw_vibronic_params(cfg)
    mpo = model.build_mpo(params)
    mps = si.padded_product_mps(si.site_dims(params), si.initial_occupations(params), cfg.M, cfg.pad_seed)
    return mpo, mps


def test_non_finite_mps_is_rejected(T):
    """fmax() drops NaN: a tensor with NaN / Inf entries used to pass the canonical check with defect 0."""
    mpo, mps = _tiny()
    for bad_value in (np.nan, np.inf):
        bad = [a.copy() for a in mps]
        bad[2][1, 2, 3] = bad_value
        with pytest.raises(T.TdvpError) as ei:
            T.tdvp_create(mpo, bad)
        assert ei.value.code == T.TDVP_EINVAL
    ch = T.tdvp_create(mpo, mps)
    bad = [a.copy() for a in mps]
    bad[4][0, 0, 0] = np.nan
    with pytest.raises(T.TdvpError):
        ch.tdvp_set_mps(bad, 0)
    ch.close()


def test_handles_on_fresh_streams_give_their_memory_back(T):
    """Every handle holds a reference on its stream's GEMM scheduling context (~39 MB); the last handle
    on a stream frees it (it used to leak until process exit)."""
    import torch
    mpo, mps = _tiny()
    L, W, A, R = (dev(x) for x in si.random_site_problem(12, 16, 4, 5, 4, 0.3, seed=1))

    def cycle():
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            ctx = T.tdvp_create_context(stream=s)
            ctx2 = T.tdvp_create_context(stream=s)        # two handles share the stream's context
            T.tdvp_apply_heff(L, W, A, R, handle=ctx)
            ch = T.tdvp_create(mpo, mps, stream=s)
            ch.tdvp_step_ps(1.0)
            ch.tdvp_sync()
            ctx.close()
            T.tdvp_apply_heff(L, W, A, R, handle=ctx2)     # still valid after the first owner left
            ctx2.tdvp_sync()
            ch.close()
            ctx2.close()
        s.synchronize()

    for _ in range(2):
        cycle()
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(6):
        cycle()
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    assert free0 - free1 < 16 * 2 ** 20, (free0 - free1) / 2 ** 20
