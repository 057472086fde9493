"""td_loglike_batch_static: the allocation-free entry point (include/tdlike.h) against the existing path.

Collected last on purpose (the suite runs with `pytest -x`: a failure here must not hide the other tests).  The static
device array is shared by every call of the process and keeps the last call's contents, so every case below makes two
calls in a row - the second on a different handle / different templates - and each must match td_loglike_batch on its own
inputs within the parity tolerance of tests/test_gpu_parity.py (1e-9 relative, floor 1e-9 * max(|ref|, 1))."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import td_oracle as O
from paper_2603_06010_b200 import binding as tdb
from paper_2603_06010_b200 import workloads as W

TOL = 1e-9


def _dev(x):
    return torch.as_tensor(np.ascontiguousarray(x), dtype=torch.float64).cuda()


def _close(got, ref, what):
    got, ref = np.asarray(got), np.asarray(ref)
    assert np.all(np.isfinite(got)), what
    err = np.abs(got - ref) / np.maximum(np.abs(ref), 1.0)
    assert err.max() <= TOL, f"{what}: max rel err {err.max():.3e} at {err.argmax()}"


@pytest.fixture(scope="module", autouse=True)
def _require_cuda():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    tdb.load(build_if_missing=False)   # the in-tree library must be present: no fallback


def test_static_entry_matches_existing_path_two_calls_in_a_row():
    """c1 (one 1024-sample segment) then c3 / 4 (three ragged segments of 1250 / 1500 / 1282 samples): the second
    call finds the first call's spectra in the array and must not be disturbed by them; a third call repeats the first and
    must reproduce it bit for bit."""
    tdb.static_setup(0)
    assert tdb.static_scratch_bytes() == 16 << 20
    w1 = W.make("c1", B=37)
    w2 = W.make("c3", B=21, n_scale=4)
    d1, H1, d2, H2 = _dev(w1.d), _dev(w1.H), _dev(w2.d), _dev(w2.H)
    o1 = torch.full((37,), np.nan, dtype=torch.float64, device="cuda")
    o2 = torch.full((21,), np.nan, dtype=torch.float64, device="cuda")
    o3 = torch.full((37,), np.nan, dtype=torch.float64, device="cuda")
    with tdb.TDLikelihood(w1.acf, w1.seg_lengths) as h1, tdb.TDLikelihood(w2.acf, w2.seg_lengths) as h2:
        ref1 = h1.loglike_batch(d1, H1).cpu().numpy()
        ref2 = h2.loglike_batch(d2, H2).cpu().numpy()
        h1.loglike_batch_static(d1, H1, o1)
        h2.loglike_batch_static(d2, H2, o2)            # second call in a row: same array, other handle, other sizes
        h1.loglike_batch_static(d1, H1, o3)
        n_launch = h1.last_launches()
        torch.cuda.synchronize()
    _close(o1.cpu().numpy(), ref1, "static vs td_loglike_batch, first call (c1)")
    _close(o2.cpu().numpy(), ref2, "static vs td_loglike_batch, second call (c3/4)")
    assert np.array_equal(o1.cpu().numpy(), o3.cpu().numpy())
    assert n_launch >= 4                               # the staged pipeline, not a fused kernel
    # and against the oracle itself
    _close(o1.cpu().numpy(), O.loglike_batch(w1.acf, w1.seg_lengths, w1.d, w1.H), "static vs oracle (c1)")
    _close(o2.cpu().numpy(), O.loglike_batch(w2.acf, w2.seg_lengths, w2.d, w2.H), "static vs oracle (c3/4)")


def test_static_entry_chunks_a_batch_larger_than_the_array_and_exact_zero():
    """N = 16384 needs 768.5 KiB of scratch per template: 21 templates per chunk, so B = 50 runs as three chunks that reuse
    the array; h = d gives exactly 0; two calls in a row with different templates."""
    w = W.make("c4", B=50, n_scale=4)
    H = w.H.copy()
    H[33] = w.d
    d, Ha, Hb = _dev(w.d), _dev(H), _dev(H[::-1].copy())
    oa = torch.empty(50, dtype=torch.float64, device="cuda")
    ob = torch.empty(50, dtype=torch.float64, device="cuda")
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        ref = h.loglike_batch(d, Ha).cpu().numpy()
        h.loglike_batch_static(d, Ha, oa)
        h.loglike_batch_static(d, Hb, ob)
        torch.cuda.synchronize()
    assert oa[33].item() == 0.0 and ob[49 - 33].item() == 0.0
    _close(oa.cpu().numpy(), ref, "static, chunked batch")
    _close(ob.cpu().numpy()[::-1], ref, "static, chunked batch, second call (rows reversed)")


def test_static_entry_refuses_a_segment_beyond_the_array():
    """A 2^19-sample size class needs 24 MiB per template: refused with TD_EUNSUPPORTED and a message, nothing launched.
    (White-noise autocorrelation: Levinson-Durbin is trivial, td_create stays quick.)"""
    n = (1 << 18) + 1
    acf = np.zeros(n)
    acf[0] = 2.0
    x = torch.zeros((1, n), dtype=torch.float64, device="cuda")
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    with tdb.TDLikelihood(acf, [n]) as h:
        with pytest.raises(tdb.TDError) as e:
            h.loglike_batch_static(x[0], x, out)
        assert e.value.status == tdb.TD_EUNSUPPORTED and "static array holds" in str(e.value)
