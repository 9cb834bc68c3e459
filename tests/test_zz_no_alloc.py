"""qw_moments_static: the moments without any allocation (block partials in a static device array of libqw, include/qw.h)
against the existing path qw_moments (partials in a cudaMalloc'ed buffer of the handle), on calls in a row that share the
static array.  Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the
other tests.  Tolerance: the moment gates of tests/test_parity_gpu.py (R24: complex128 relative 1e-10, complex64
1e-4; means relative to the extent where the mean is ~0, second moments relative to E[x^2]).
"""
import numpy as np
import pytest

from paper_1003_3779_b200 import inputs as qi

pytestmark = pytest.mark.gpu

MOM_RTOL = {np.dtype(np.complex128): 1e-10, np.dtype(np.complex64): 1e-4}


@pytest.fixture(scope="module")
def dev(qw):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    torch.cuda.init()
    return torch.device("cuda:0")


def close_moments(w, got, want):
    rt = MOM_RTOL[np.dtype(w.dtype)]
    ext = max(w.extents)
    nm = 1 if w.dim == 1 else 2
    assert got.shape == want.shape
    for b in range(w.batch):
        assert abs(got[b, 0] - want[b, 0]) <= rt * abs(want[b, 0]), ("norm", got[b], want[b])
        for j in range(1, 1 + nm):
            assert abs(got[b, j] - want[b, j]) <= rt * (abs(want[b, j]) + ext), ("mean", got[b], want[b])
        second = 1.0 + max(abs(want[b, j]) for j in range(1 + nm, want.shape[1])) + max(want[b, j] ** 2 for j in range(1, 1 + nm))
        for j in range(1 + nm, want.shape[1]):
            assert abs(got[b, j] - want[b, j]) <= rt * second, ("second moment", j, got[b], want[b])


def workloads():
    # big first, small afterwards: the second call finds the first one's partial sums in the shared array
    yield qi.k1(sites=(1 << 20) + 3, steps=40)                                          # 1D ring, complex128, batch 1
    yield qi.k3(extents=(200, 333), steps=12, coin="dft")                               # 2D torus, complex64, odd rows
    yield qi.k4(batch=40, half=100, steps=60)                                           # batch of open 1D walks, delta starts
    yield qi.k2(half=40, steps=30)                                                      # 2D open, delta start (light-cone window)


def test_moments_static_matches_moments_on_calls_in_a_row(qw, dev):
    import torch
    for w in workloads():
        h = qw.create_for(w)
        try:
            qw.load_state(h, w)
            cols = 3 if w.dim == 1 else 6
            for steps in (w.steps, 7):                                                  # two calls in a row on every handle
                qw.qw_step(h, steps)
                want = np.empty((w.batch, cols), dtype=np.float64)
                qw.qw_moments(h, want)                                                  # existing path (host buffer)
                want_dev = torch.empty((w.batch, cols), dtype=torch.float64, device=dev)
                qw.qw_moments(h, want_dev)                                              # existing path (device buffer)
                got = torch.full((w.batch, cols), float("nan"), dtype=torch.float64, device=dev)
                qw.qw_moments_static(h, got)
                again = torch.full((w.batch, cols), float("nan"), dtype=torch.float64, device=dev)
                qw.qw_moments_static(h, again)                                          # immediately again: same stream, shared scratch
                qw.qw_synchronize(h)
                g, a = got.cpu().numpy(), again.cpu().numpy()
                assert np.all(np.isfinite(g))
                assert np.array_equal(g, a)                                             # deterministic
                close_moments(w, g, want)
                close_moments(w, g, want_dev.cpu().numpy())
        finally:
            qw.qw_destroy(h)


def test_moments_static_limits_and_errors(qw, dev):
    import torch
    # the stated maximum: 8192 walks fit, 8193 do not
    for batch, ok in ((8192, True), (8193, False)):
        w = qi.k4(batch=batch, half=20, steps=10)
        h = qw.create_for(w)
        try:
            qw.load_state(h, w)
            qw.qw_step(h, w.steps)
            out = torch.empty((batch, 3), dtype=torch.float64, device=dev)
            if ok:
                qw.qw_moments_static(h, out)
                want = np.empty((batch, 3), dtype=np.float64)
                qw.qw_moments(h, want)
                close_moments(w, out.cpu().numpy(), want)
            else:
                with pytest.raises(qw.QwError) as ei:
                    qw.qw_moments_static(h, out)
                assert ei.value.code == qw.QW_EUNSUPPORTED
                assert "8192" in str(ei.value)
        finally:
            qw.qw_destroy(h)
    # a host output buffer would need a staging allocation: rejected; no state: QW_ESTATE
    w = qi.k1(sites=4096, steps=4)
    h = qw.create_for(w)
    try:
        out = torch.empty((1, 3), dtype=torch.float64, device=dev)
        with pytest.raises(qw.QwError) as ei:
            qw.qw_moments_static(h, out)
        assert ei.value.code == qw.QW_ESTATE
        qw.load_state(h, w)
        with pytest.raises(qw.QwError) as ei:
            qw.qw_moments_static(h, np.empty((1, 3), dtype=np.float64))
        assert ei.value.code == qw.QW_EINVAL
    finally:
        qw.qw_destroy(h)
