"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  Tolerance (BASELINE.json north_star): 1e-9 relative on each logL_b,
with the A12 floor |gpu - oracle| <= 1e-9 * max(|oracle|, 1)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import td_oracle as O
from oracle import templates as OT
from paper_2603_06010_b200 import binding as tdb
from paper_2603_06010_b200 import workloads as W

TOL = 1e-9


def _dev(x):
    return torch.as_tensor(np.ascontiguousarray(x), dtype=torch.float64).cuda()


def _assert_close(gpu, ref, tol=TOL, what=""):
    gpu = np.asarray(gpu)
    ref = np.asarray(ref)
    err = np.abs(gpu - ref) / np.maximum(np.abs(ref), 1.0)
    assert np.all(np.isfinite(gpu)), what
    assert err.max() <= tol, f"{what}: max rel err {err.max():.3e} at {err.argmax()}"
    return err.max()


def _gpu_loglike(w, variant=0, path=None):
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        if variant:
            h.set_fft_variant(variant)
        if path is not None:
            h.set_path(path)
        out = h.loglike_batch(_dev(w.d), _dev(w.H))
        torch.cuda.synchronize()
        return out.cpu().numpy(), h.info(), h.last_launches()


@pytest.fixture(scope="module", autouse=True)
def _require_cuda():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    tdb.load(build_if_missing=False)   # the in-tree library must be present: no fallback


# ------------------------------------------------------------------ configs of BASELINE.json
def test_c1_fused_full():
    w = W.make("c1")
    ref = O.loglike_batch(w.acf, w.seg_lengths, w.d, w.H)
    out, info, nl = _gpu_loglike(w)
    _assert_close(out, ref, what="c1")
    assert info["last_path"] == tdb.TD_PATH_FFT and nl == 1


def test_c1_staged_variant():
    w = W.make("c1")
    ref = O.loglike_batch(w.acf, w.seg_lengths, w.d, w.H)
    out, _, nl = _gpu_loglike(w, variant=2)
    _assert_close(out, ref, what="c1 staged")
    assert nl > 1


def test_c2_headline_size_subset():
    w = W.make("c2", B=96)
    ref = O.loglike_batch(w.acf, w.seg_lengths, w.d, w.H)
    out, _, _ = _gpu_loglike(w)
    _assert_close(out, ref, what="c2")
    out2, _, _ = _gpu_loglike(w, variant=2)
    _assert_close(out2, ref, what="c2 staged")


def test_c3_gapped_segments():
    w = W.make("c3", B=24)
    ref = O.loglike_batch(w.acf, w.seg_lengths, w.d, w.H)
    out, _, _ = _gpu_loglike(w)
    _assert_close(out, ref, what="c3")


def test_c5_three_detectors():
    w = W.make("c5", B=12)
    ref = O.loglike_batch(w.acf, w.seg_lengths, w.d, w.H)
    out, _, _ = _gpu_loglike(w)
    _assert_close(out, ref, what="c5")


def test_c4_long_segment_vs_library_levinson():
    """N = 65536: dense C would be 32 GiB, so the oracle route is solve_toeplitz (pin P13)."""
    w = W.make("c4", B=3)
    ref = O.loglike_batch_solve_toeplitz(w.acf, w.seg_lengths, w.d, w.H)
    out, _, nl = _gpu_loglike(w)
    _assert_close(out, ref, what="c4")
    assert nl == 2                                   # the group kernel (td_group16.cuh) + the rank-ordered sum of its partials
    out_st, _, nl_st = _gpu_loglike(w, variant=2)    # the staged kernels (what a device that cannot co-host a group runs)
    _assert_close(out_st, ref, what="c4 on the staged kernels")
    assert nl_st > 2
    # the same segment on the 16-CTA cluster kernel (td_cluster16.cuh, variant 3): all three kernel modes
    dh_ref = None
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        d, H = _dev(w.d), _dev(w.H)
        dh_s, hh_s = h.inner_batch(d, H, want_hh=True)
        dh_s, hh_s = dh_s.clone(), hh_s.clone()
        h.set_fft_variant(3)
        out16 = h.loglike_batch(d, H).cpu().numpy()
        n16 = h.last_launches()
        dh16, hh16 = h.inner_batch(d, H)
        torch.cuda.synchronize()
    _assert_close(out16, ref, what="c4 on the 16-CTA cluster kernel")
    assert n16 == 2                                  # the cluster kernel + the rank-ordered sum of the 16 partials
    scale = float(hh_s.abs().max())
    assert float((hh16 - hh_s).abs().max()) <= 1e-9 * scale and float((dh16 - dh_s).abs().max()) <= 1e-9 * scale


def test_cluster16_ragged_length_many_items_and_refusal():
    """N = 40001 (odd, unaligned rows: scalar loads) and more templates than co-resident clusters, against the staged
    kernels (themselves held to the oracle above); handles without a 65536-class segment refuse variant 3."""
    rng = np.random.default_rng(16)
    n = 40001
    rho = W.acf_from_psd(4096.0, 2 * 65536, n)
    d = rng.standard_normal(n) * 1e-21
    H = rng.standard_normal((23, n)) * 1e-21
    H[5] = d
    with tdb.TDLikelihood(rho, [n]) as h:
        ref = h.loglike_batch(_dev(d), _dev(H)).cpu().numpy()
        h.set_fft_variant(3)
        out = h.loglike_batch(_dev(d), _dev(H)).cpu().numpy()
        out2 = h.loglike_batch(_dev(d), _dev(H)).cpu().numpy()
    assert out[5] == 0.0 and np.array_equal(out, out2)
    _assert_close(out, ref, what="cluster16, N = 40001")
    w = W.make("c2", B=4)
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        with pytest.raises(tdb.TDError) as e:
            h.set_fft_variant(3)
        assert e.value.status == tdb.TD_EUNSUPPORTED


def test_group16_ragged_length_many_items_modes_graph_and_two_handles():
    """The default kernel of the 65536 class (16-CTA groups exchanging through L2, td_group16.cuh) against the staged
    kernels (variant 2, themselves held to the oracle above): N = 40001 (odd, unaligned rows: scalar loads), more templates
    than groups with an uneven remainder, all three kernel modes, bit-identical repeats, capture into a CUDA graph, and two
    handles working at the same time on two streams (cooperative launches queue behind one another; nothing may hang)."""
    rng = np.random.default_rng(161)
    n = 40001
    rho = W.acf_from_psd(4096.0, 2 * 65536, n)
    d = rng.standard_normal(n) * 1e-21
    H = rng.standard_normal((23, n)) * 1e-21
    H[5] = d
    H[7, 100] = np.nan
    dd, HH = _dev(d), _dev(H)
    with tdb.TDLikelihood(rho, [n]) as h, tdb.TDLikelihood(rho * 1.5, [n]) as h2:
        h.set_fft_variant(2)
        ref = h.loglike_batch(dd, HH).cpu().numpy()
        dh_s, hh_s = h.inner_batch(dd, HH, want_hh=True)
        dh_s, hh_s = dh_s.cpu().numpy(), hh_s.cpu().numpy()
        assert h.last_launches() > 4
        h.set_fft_variant(0)
        out = h.loglike_batch(dd, HH).cpu().numpy()
        assert h.last_launches() == 2
        out2 = h.loglike_batch(dd, HH).cpu().numpy()
        dh, hh = h.inner_batch(dd, HH, want_hh=True)
        dh, hh = dh.cpu().numpy(), hh.cpu().numpy()
        h.set_fft_variant(4)                                        # the explicit name of the same kernel
        out4 = h.loglike_batch(dd, HH).cpu().numpy()
        # graph capture: memset of the arrival counters + cooperative launch + reduction
        s = torch.cuda.Stream()
        og = torch.empty(23, dtype=torch.float64, device="cuda")
        g = torch.cuda.CUDAGraph()
        with torch.cuda.stream(s):
            h.loglike_batch(dd, HH, out=og, stream=s)               # warm
            s.synchronize()
            with torch.cuda.graph(g, stream=s):
                h.loglike_batch(dd, HH, out=og, stream=s)
            og.zero_()
            g.replay(); g.replay()
            s.synchronize()
        # two handles, two streams, interleaved calls
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        o1 = torch.empty(23, dtype=torch.float64, device="cuda")
        o2 = torch.empty(23, dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        for _ in range(4):
            h.loglike_batch(dd, HH, out=o1, stream=s1)
            h2.loglike_batch(dd, HH, out=o2, stream=s2)
        torch.cuda.synchronize()
    ok = np.isfinite(ref)
    assert not ok[7] and ok.sum() == 22 and np.isnan(out[7])
    assert out[5] == 0.0 and np.array_equal(out, out2, equal_nan=True) and np.array_equal(out, out4, equal_nan=True)
    _assert_close(out[ok], ref[ok], what="group16, N = 40001")
    assert np.array_equal(og.cpu().numpy(), out, equal_nan=True) and np.array_equal(o1.cpu().numpy(), out, equal_nan=True)
    _assert_close(o2.cpu().numpy()[ok] * 1.5, ref[ok], what="group16, second handle (C scaled by 1.5)")
    scale = np.max(np.abs(hh_s[ok]))
    assert np.max(np.abs(hh[ok] - hh_s[ok])) <= 1e-9 * scale and np.max(np.abs(dh[ok] - dh_s[ok])) <= 1e-9 * scale


@pytest.mark.parametrize("lens", [[9001], [16384], [20001], [32768], [9000, 40001, 17000, 3000]])
def test_group_kernel_sizes_4_8_16_against_staged_and_oracle(lens):
    """Size classes M = 16384 / 32768 / 65536 run on td_group_kernel<4 / 8 / 16> (td_group16.cuh) by default: against the
    staged kernels (variant 2) in all three kernel modes, and against the oracle (library Levinson solve, pin P13) on two
    templates; odd lengths take the scalar-load path; the mixed handle also has a fused-kernel class (3000)."""
    rng = np.random.default_rng(sum(lens))
    acf = np.concatenate([W.acf_from_psd(4096.0, 2 * 65536, n) * (1.0 + 0.2 * i) for i, n in enumerate(lens)])
    nt, B = sum(lens), 43                            # more templates than groups of 16, an uneven remainder for every size
    d = rng.standard_normal(nt) * 1e-21
    H = rng.standard_normal((B, nt)) * 1e-21
    H[11] = d
    dd, HH = _dev(d), _dev(H)
    with tdb.TDLikelihood(acf, lens) as h:
        out = h.loglike_batch(dd, HH).cpu().numpy()
        nl = h.last_launches()
        out_again = h.loglike_batch(dd, HH).cpu().numpy()
        dh, hh = h.inner_batch(dd, HH, want_hh=True)
        dh, hh = dh.cpu().numpy(), hh.cpu().numpy()
        h.set_fft_variant(2)
        ref_st = h.loglike_batch(dd, HH).cpu().numpy()
        nl_st = h.last_launches()
        dh_s, hh_s = h.inner_batch(dd, HH, want_hh=True)
        dh_s, hh_s = dh_s.cpu().numpy(), hh_s.cpu().numpy()
    assert out[11] == 0.0 and np.array_equal(out, out_again)
    assert nl == 2 * sum(n > 8192 for n in lens) + (1 if any(n <= 8192 for n in lens) else 0) and nl_st > nl
    _assert_close(out, ref_st, what=f"group kernel vs staged {lens}")
    scale = np.max(np.abs(hh_s))
    assert np.max(np.abs(hh - hh_s)) <= 1e-9 * scale and np.max(np.abs(dh - dh_s)) <= 1e-9 * scale
    ref = O.loglike_batch_solve_toeplitz(acf, lens, d, H[:2])
    _assert_close(out[:2], ref, what=f"group kernel vs oracle {lens}")


# ------------------------------------------------------------------ shapes: ragged, tiny, mixed classes
@pytest.mark.parametrize("n", [4097, 6001, 8192])
def test_cluster_kernel_lengths(n):
    """M = 8192: the 2-CTA cluster kernel (even, odd and unaligned rows; B not a multiple of the grid)."""
    rng = np.random.default_rng(n)
    rho = W.acf_from_psd(4096.0, 2 * 8192, n)
    d = rng.standard_normal(n) * 1e-21
    H = rng.standard_normal((5, n)) * 1e-21
    ref = O.loglike_batch(rho, [n], d, H)
    dh_ref, hh_ref = O.inner_batch(rho, [n], d, H)
    with tdb.TDLikelihood(rho, [n]) as h:
        dd, HH = _dev(d), _dev(H)
        out = h.loglike_batch(dd, HH).cpu().numpy()
        assert h.last_launches() == 1
        dh, hh = h.inner_batch(dd, HH)
        h.set_fft_variant(2)
        out2 = h.loglike_batch(dd, HH).cpu().numpy()
    _assert_close(out, ref, what=f"cluster n={n}")
    _assert_close(out2, ref, what=f"staged n={n}")
    scale = hh_ref + float(O.inner_batch(rho, [n], d, d[None, :])[1][0])
    assert np.max(np.abs(dh.cpu().numpy() - dh_ref) / scale) <= TOL
    assert np.max(np.abs(hh.cpu().numpy() - hh_ref) / np.abs(hh_ref)) <= TOL


def test_cluster_many_templates_repeatable():
    """More templates than clusters (74): every cluster loops; bitwise repeatable."""
    w = W.make("c5", B=200, n_scale=1)
    sub = slice(0, 8)
    ref = O.loglike_batch(w.acf, w.seg_lengths, w.d, w.H[sub])
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        d, H = _dev(w.d), _dev(w.H)
        o1 = h.loglike_batch(d, H)
        o2 = h.loglike_batch(d, H)
        torch.cuda.synchronize()
        assert h.last_launches() == 1
    assert torch.equal(o1, o2)
    _assert_close(o1.cpu().numpy()[sub], ref, what="c5 B=200")
    # every other template: against the staged (global-memory) variant of the same library
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        h.set_fft_variant(2)
        o3 = h.loglike_batch(_dev(w.d), _dev(w.H)).cpu().numpy()
    _assert_close(o1.cpu().numpy(), o3, tol=1e-11, what="cluster vs staged")


@pytest.mark.parametrize("n", [1, 2, 3, 5, 31, 255, 256, 257, 777, 1000, 2049, 4095])
def test_ragged_lengths(n):
    rng = np.random.default_rng(n)
    rho = W.acf_from_psd(4096.0, 2 * max(n, 64), n)
    d = rng.standard_normal(n) * 1e-21
    H = rng.standard_normal((7, n)) * 1e-21
    ref = O.loglike_batch(rho, [n], d, H)
    for variant in (0, 2):
        with tdb.TDLikelihood(rho, [n]) as h:
            h.set_fft_variant(variant)
            h.set_path(tdb.TD_PATH_FFT)        # AUTO would send n <= 512 to the dense kernel
            out = h.loglike_batch(_dev(d), _dev(H)).cpu().numpy()
        _assert_close(out, ref, what=f"n={n} variant={variant}")


def test_mixed_size_classes_and_odd_offsets():
    rng = np.random.default_rng(5)
    lens = [301, 1000, 4097, 77]
    rho = W.acf_from_psd(4096.0, 2 * 8192, max(lens))
    scales = [1.0, 0.7, 1.9, 3.0]
    acf = np.concatenate([s * rho[:n] for s, n in zip(scales, lens)])
    nt = sum(lens)
    d = rng.standard_normal(nt) * 1e-21
    H = rng.standard_normal((9, nt)) * 1e-21
    ref = O.loglike_batch(acf, lens, d, H)
    with tdb.TDLikelihood(acf, lens) as h:
        out = h.loglike_batch(_dev(d), _dev(H)).cpu().numpy()
    _assert_close(out, ref, what="mixed classes")


def test_strided_rows_and_exact_zero_and_nan_row():
    w = W.make("c1", B=8)
    n = w.n_tot
    Hpad = torch.zeros(8, n + 37, dtype=torch.float64, device="cuda")
    Hpad[:, :n] = _dev(w.H)
    Hpad[3, :n] = _dev(w.d)                       # h = d  ->  logL = 0 exactly (P8 iv)
    Hpad[5, 100] = float("nan")
    ref = O.loglike_batch(w.acf, w.seg_lengths, w.d, w.H)
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        out = h.loglike_batch(_dev(w.d), Hpad[:, :n]).cpu().numpy()
    assert out[3] == 0.0
    assert np.isnan(out[5])
    keep = [0, 1, 2, 4, 6, 7]
    _assert_close(out[keep], ref[keep], what="strided")


# ------------------------------------------------------------------ setup kernel (S0)
@pytest.mark.parametrize("n", [64, 1024, 5000])
def test_generator_matches_oracle_levinson(n):
    rho = W.acf_from_psd(4096.0, 2 * 8192, n)
    a_ref, v_ref, ld_ref = O.levinson_durbin_fast(rho)
    with tdb.TDLikelihood(rho, [n]) as h:
        a = h.generator(0)
        info = h.info()
    assert np.max(np.abs(a - a_ref)) <= 1e-10 * np.max(np.abs(a_ref))
    assert abs(info["v"][0] - v_ref) <= 1e-11 * v_ref
    assert abs(info["logdet"][0] - ld_ref) <= 1e-10 * abs(ld_ref)
    L = O.cholesky_lower(rho)
    assert abs(info["logdet"][0] - 2 * np.sum(np.log(np.diag(L)))) <= 1e-9 * abs(ld_ref)


# ------------------------------------------------------------------ td_inner_batch (Eq. 13 terms)
@pytest.mark.parametrize("name,B,variant", [("c1", 16, 0), ("c1", 16, 2), ("c3", 6, 0)])
def test_inner_batch(name, B, variant):
    w = W.make(name, B=B)
    dh_ref, hh_ref = O.inner_batch(w.acf, w.seg_lengths, w.d, w.H)
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        h.set_fft_variant(variant)
        d, H = _dev(w.d), _dev(w.H)
        dh, hh = h.inner_batch(d, H)
        ll = h.loglike_batch(d, H)
        dd, _ = h.inner_batch(d, d[None, :])
        only_hh = h.inner_batch(d, H, want_dh=False)[1]
    dh, hh, ll, dd = dh.cpu().numpy(), hh.cpu().numpy(), ll.cpu().numpy(), dd.cpu().numpy()[0]
    scale = dd + hh
    assert np.max(np.abs(dh - dh_ref) / scale) <= TOL
    assert np.max(np.abs(hh - hh_ref) / np.abs(hh_ref)) <= TOL
    assert np.max(np.abs(-2 * ll - (dd - 2 * dh + hh)) / scale) <= TOL      # bilinear identity (P11)
    assert np.array_equal(only_hh.cpu().numpy(), hh)


# ------------------------------------------------------------------ host-buffer entry point
def test_host_entry_matches_device_entry():
    w = W.make("c1", B=50)
    Hp = torch.as_tensor(w.H).pin_memory()
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        a = h.loglike_batch(_dev(w.d), _dev(w.H)).cpu().numpy()
        b = h.loglike_batch_host(w.d, Hp)
        c = h.loglike_batch_host(w.d, w.H)        # pageable numpy
    assert np.array_equal(a, b) and np.array_equal(a, c)


# ------------------------------------------------------------------ errors and edges
def test_error_paths():
    rho = W.acf_from_psd(4096.0, 2048, 512)
    bad = np.array([1.0, 0.99, 0.2, -0.9])
    with pytest.raises(tdb.TDError) as e:
        tdb.TDLikelihood(bad, [4])
    assert e.value.status == tdb.TD_ENOTSPD
    with pytest.raises(tdb.TDError) as e:
        tdb.TDLikelihood(np.array([0.0, 0.0]), [2])
    assert e.value.status == tdb.TD_ENOTSPD
    nanrho = rho.copy()
    nanrho[7] = np.nan
    with pytest.raises(tdb.TDError) as e:
        tdb.TDLikelihood(nanrho, [512])
    assert e.value.status == tdb.TD_ENOTSPD
    with pytest.raises(tdb.TDError) as e:
        tdb.TDLikelihood(rho, [0, 512][:1] + [512])   # zero-length segment
    with tdb.TDLikelihood(rho, [512]) as h:
        d = torch.zeros(512, dtype=torch.float64, device="cuda")
        H0 = torch.zeros(0, 512, dtype=torch.float64, device="cuda")
        assert h.loglike_batch(d, H0).numel() == 0          # B = 0 is a no-op
        lib = tdb.load()
        st = lib.td_loglike_batch(h._h, d.data_ptr(), d.data_ptr(), 100, 1, d.data_ptr(), None)
        assert st == tdb.TD_EINVAL                           # ldh < N_tot
        st = lib.td_loglike_batch(h._h, None, d.data_ptr(), 512, 1, d.data_ptr(), None)
        assert st == tdb.TD_EINVAL


def test_async_on_caller_stream_and_repeatable():
    w = W.make("c1", B=32)
    s = torch.cuda.Stream()
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        d, H = _dev(w.d), _dev(w.H)
        torch.cuda.synchronize()
        with torch.cuda.stream(s):
            o1 = h.loglike_batch(d, H)
            o2 = h.loglike_batch(d, H)
        s.synchronize()
    assert torch.equal(o1, o2)                               # deterministic reduction order


# ------------------------------------------------------------------ dense path (S2'-S4')
@pytest.mark.parametrize("n", [1, 5, 31, 32, 33, 64, 100, 128, 200, 256, 300, 512, 777, 1024])
def test_dense_path_lengths(n):
    """Forced dense path: every row-group / warp arrangement (NWR = 1, 2, 4, 8), ragged N and B."""
    rng = np.random.default_rng(1000 + n)
    rho = W.acf_from_psd(4096.0, 2 * 8192, n)
    d = rng.standard_normal(n) * 1e-21
    H = rng.standard_normal((37, n)) * 1e-21
    ref = O.loglike_batch(rho, [n], d, H)
    out, info, nl = _gpu_loglike(W.Workload("t", 0, 4096.0, np.array([n]), rho, d, H, np.ones(1)), path=tdb.TD_PATH_DENSE)
    _assert_close(out, ref, what=f"dense n={n}")
    assert info["last_path"] == tdb.TD_PATH_DENSE and nl == 1


@pytest.mark.parametrize("name", ["d1", "d2", "d3"])
def test_dense_configs_both_paths(name):
    """d1-d3 (ringdown-only segments): dense and FFT paths against the oracle and each other."""
    w = W.make(name, B=300)
    ref = O.loglike_batch(w.acf, w.seg_lengths, w.d, w.H)
    od, info_d, _ = _gpu_loglike(w, path=tdb.TD_PATH_DENSE)
    of, info_f, _ = _gpu_loglike(w, path=tdb.TD_PATH_FFT)
    _assert_close(od, ref, what=name + " dense")
    _assert_close(of, ref, what=name + " fft")
    assert info_d["last_path"] == tdb.TD_PATH_DENSE and info_f["last_path"] == tdb.TD_PATH_FFT


def test_dense_multi_segment_and_inner():
    rng = np.random.default_rng(77)
    lens = [64, 200, 33, 512]
    rho = W.acf_from_psd(4096.0, 2 * 8192, max(lens))
    scales = [1.0, 0.6, 2.5, 1.7]
    acf = np.concatenate([s * rho[:n] for s, n in zip(scales, lens)])
    nt = sum(lens)
    d = rng.standard_normal(nt) * 1e-21
    H = rng.standard_normal((45, nt)) * 1e-21
    ref = O.loglike_batch(acf, lens, d, H)
    dh_ref, hh_ref = O.inner_batch(acf, lens, d, H)
    with tdb.TDLikelihood(acf, lens) as h:
        h.set_path(tdb.TD_PATH_DENSE)
        dd_, HH = _dev(d), _dev(H)
        out = h.loglike_batch(dd_, HH).cpu().numpy()
        assert h.info()["last_path"] == tdb.TD_PATH_DENSE
        dh, hh = h.inner_batch(dd_, HH)
        dd, _ = h.inner_batch(dd_, dd_[None, :])
    _assert_close(out, ref, what="dense multi-segment")
    dh, hh, dd = dh.cpu().numpy(), hh.cpu().numpy(), dd.cpu().numpy()[0]
    scale = dd + hh
    assert np.max(np.abs(dh - dh_ref) / scale) <= TOL
    assert np.max(np.abs(hh - hh_ref) / np.abs(hh_ref)) <= TOL
    assert np.max(np.abs(-2 * out - (dd - 2 * dh + hh)) / scale) <= TOL


def test_auto_chooser_mixes_paths():
    """AUTO: the short segment goes to the dense kernel, the long one to the FFT kernel, one sum."""
    rng = np.random.default_rng(78)
    lens = [64, 3000]
    rho = W.acf_from_psd(4096.0, 2 * 8192, max(lens))
    acf = np.concatenate([rho[:64], 1.4 * rho[:3000]])
    nt = sum(lens)
    d = rng.standard_normal(nt) * 1e-21
    H = rng.standard_normal((19, nt)) * 1e-21
    ref = O.loglike_batch(acf, lens, d, H)
    with tdb.TDLikelihood(acf, lens) as h:
        out = h.loglike_batch(_dev(d), _dev(H)).cpu().numpy()
        assert h.last_launches() == 2 and h.info()["last_path"] == tdb.TD_PATH_FFT
        dh, hh = h.inner_batch(_dev(d), _dev(H))
        with pytest.raises(tdb.TDError) as e:
            h.set_path(tdb.TD_PATH_DENSE)          # 3000 > dense limit
        assert e.value.status == tdb.TD_EUNSUPPORTED
    _assert_close(out, ref, what="auto mixed")
    dh_ref, hh_ref = O.inner_batch(acf, lens, d, H)
    assert np.max(np.abs(hh.cpu().numpy() - hh_ref) / np.abs(hh_ref)) <= TOL


def test_probe_library_reports_plausible_peaks():
    """bench.py's roofline denominators come from the bench-only probe library (include/tdprobe.h)."""
    dfma = tdb.probe_throughput(0)
    dmma = tdb.probe_throughput(1)
    ffma = tdb.probe_throughput(4)
    assert 10.0 < dfma < 60.0 and 10.0 < dmma < 90.0 and 30.0 < ffma < 120.0


# ------------------------------------------------------------------ full sizes, in the launch configuration bench.py times
def _full_size_check(name, sample, oracle=None, path=None):
    """The whole batch of config `name` goes through the library exactly as bench.py launches it; the oracle
    recomputes the sampled rows one by one; every row is checked through properties that hold at any size:
    finite, logL <= 0, and the bilinear identity -2 logL = <d,d> - 2 <d,h> + <h,h> (pin P11) with the cross
    terms coming from td_inner_batch (a different kernel mode)."""
    w = W.make(name)
    idx = np.unique(np.concatenate([np.arange(0, w.B, max(1, w.B // sample)), [w.B - 1]]))
    fn = oracle or O.loglike_batch
    ref = fn(w.acf, w.seg_lengths, w.d, w.H[idx])
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        if path is not None:
            h.set_path(path)
        d, H = _dev(w.d), _dev(w.H)
        out = h.loglike_batch(d, H)
        dh, hh = h.inner_batch(d, H)
        dd = h.inner_batch(d, d[None, :])[1]
        torch.cuda.synchronize()
        out, dh, hh, dd = out.cpu().numpy(), dh.cpu().numpy(), hh.cpu().numpy(), float(dd.cpu().numpy()[0])
    err = _assert_close(out[idx], ref, what=f"{name} full size, sampled rows")
    print(f"[full size {name}] B = {w.B}, oracle-checked rows = {len(idx)}, max rel err = {err:.2e}")
    assert np.all(np.isfinite(out)) and np.all(out <= 0.0)
    scale = dd + hh
    assert np.max(np.abs(-2.0 * out - (dd - 2.0 * dh + hh)) / scale) <= TOL, f"{name}: bilinear identity"
    # template 0 is the injection: logL_0 = -1/2 n^T C^-1 n is chi-square distributed around -N/2 (pin P14)
    n_tot = int(np.sum(w.seg_lengths))
    assert abs(out[0] + 0.5 * n_tot) <= 5.0 * np.sqrt(0.5 * n_tot)


def test_full_size_c2_headline():
    _full_size_check("c2", sample=48)


def test_full_size_c3_gapped():
    _full_size_check("c3", sample=12)


def test_full_size_c5_network():
    _full_size_check("c5", sample=32)


def test_full_size_c4_long():
    _full_size_check("c4", sample=8, oracle=O.loglike_batch_solve_toeplitz)


@pytest.mark.parametrize("name", ["d1", "d3", "d4"])
def test_full_size_dense_regime(name):
    _full_size_check(name, sample=64, path=tdb.TD_PATH_DENSE)


@pytest.mark.parametrize("name,path", [("d1", tdb.TD_PATH_AUTO), ("d3", tdb.TD_PATH_AUTO), ("d4", tdb.TD_PATH_AUTO),
                                       ("d5", tdb.TD_PATH_CDO)])
def test_full_size_cdo_regime(name, path):
    """AUTO sends the log-likelihood of size classes up to 512 samples through the cached-L^-1 contraction (td_cdo.cuh); the
    bilinear identity inside _full_size_check ties it to the Gohberg-Semencul dense kernel (td_inner_batch)."""
    _full_size_check(name, sample=64, path=path)
    w = W.make(name, B=40)
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        h.set_path(path)
        h.loglike_batch(_dev(w.d), _dev(w.H))
        # N = 64 stays on the Gohberg-Semencul dense kernel under AUTO (measured crossover, profiles/r02_cdo.md)
        assert h.info()["last_path"] == (tdb.TD_PATH_DENSE if name == "d1" else tdb.TD_PATH_CDO)


# ------------------------------------------------------------------ cross term as a batched dot product (td_dot.cuh)
@pytest.mark.parametrize("name,B,n_scale", [("c1", 64, 1), ("c2", 40, 1), ("c3", 9, 1), ("c5", 5, 1), ("d2", 100, 1)])
def test_cross_term_dot_path(name, B, n_scale):
    """out_hh = NULL under AUTO: <d,h_b> = u . h_b with u = C^-1 d.  Against the oracle, and against the FFT kernels."""
    w = W.make(name, B=B, n_scale=n_scale)
    dh_ref, hh_ref = O.inner_batch(w.acf, w.seg_lengths, w.d, w.H)
    dd = float(O.inner_batch(w.acf, w.seg_lengths, w.d, w.d[None, :])[1][0])
    scale = dd + hh_ref
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        d, H = _dev(w.d), _dev(w.H)
        dh, none = h.inner_batch(d, H, want_hh=False)
        assert none is None and h.info()["last_path"] == tdb.TD_PATH_DOT
        dh2, _ = h.inner_batch(d, H, want_hh=False)
        assert torch.equal(dh, dh2)                       # fixed summation order
        h.set_path(tdb.TD_PATH_FFT)
        dh_fft, _ = h.inner_batch(d, H, want_hh=False)
        assert h.info()["last_path"] == tdb.TD_PATH_FFT
    assert np.max(np.abs(dh.cpu().numpy() - dh_ref) / scale) <= TOL
    assert np.max(np.abs(dh.cpu().numpy() - dh_fft.cpu().numpy()) / scale) <= TOL


def test_cross_term_dot_path_unaligned_rows_and_odd_length():
    rng = np.random.default_rng(11)
    lens = [301, 1000, 77]
    rho = W.acf_from_psd(4096.0, 2 * 8192, max(lens))
    acf = np.concatenate([s * rho[:n] for s, n in zip([1.0, 0.7, 3.0], lens)])
    nt = sum(lens)
    d = rng.standard_normal(nt) * 1e-21
    Hbig = rng.standard_normal((13, nt + 3)) * 1e-21     # odd leading dimension: scalar loads
    H = Hbig[:, :nt]
    dh_ref, hh_ref = O.inner_batch(acf, lens, d, H)
    dd = float(O.inner_batch(acf, lens, d, d[None, :])[1][0])
    with tdb.TDLikelihood(acf, lens) as h:
        dh, _ = h.inner_batch(_dev(d), _dev(Hbig)[:, :nt], want_hh=False)
        assert h.info()["last_path"] == tdb.TD_PATH_DOT
    assert np.max(np.abs(dh.cpu().numpy() - dh_ref) / (dd + hh_ref)) <= TOL


# ------------------------------------------------------------------ templates synthesised on the device (td_synth.cuh)
@pytest.mark.parametrize("name,B,n_scale", [("c1", 64, 1), ("c2", 200, 1), ("d2", 333, 1), ("c5", 10, 1), ("c3", 12, 1),
                                            ("c4", 3, 8)])
def test_family_params_entry_matches_oracle(name, B, n_scale):
    """td_loglike_family_batch: rows of 5 parameters instead of H (ringdown c1/c2/c5/d*, sine-Gaussian c3, chirp c4).
    The oracle builds H from the same parameters with its own plain family formulas (oracle/templates.py, pinned by
    P15-P18) and evaluates it; the device and host entries must agree with it and with each other."""
    w = W.make(name, B=B, n_scale=n_scale)
    H_ref = OT.family_rows(w.family, w.params, w.seg_lengths, w.fs)
    fn = O.loglike_batch_solve_toeplitz if w.n_tot > 20000 and len(w.seg_lengths) == 1 else O.loglike_batch
    ref = fn(w.acf, w.seg_lengths, w.d, H_ref)
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        out = h.loglike_family_batch(_dev(w.d), w.family, _dev(w.params), w.fs)
        torch.cuda.synchronize()
        # c1 / c2 at these batch sizes: ringdown rows synthesised inside the fused kernel's first pass (td_ring.cuh), ONE
        # launch; everything else: synthesis kernel + panel + likelihood kernels
        fused_route = name in ("c1", "c2")
        assert (h.last_launches() == 1) if fused_route else (h.last_launches() >= 2)
        out_host = h.loglike_family_batch_host(w.d, w.family, w.params, w.fs)
        h.set_fft_variant(1)                                   # the panel route for every family
        out_panel = h.loglike_family_batch(_dev(w.d), w.family, _dev(w.params), w.fs)
        torch.cuda.synchronize()
        assert h.last_launches() >= 2
    _assert_close(out.cpu().numpy(), ref, what=f"{name} params")
    _assert_close(out_panel.cpu().numpy(), ref, what=f"{name} params, panel route")
    assert np.array_equal(out.cpu().numpy(), out_host)


def test_ringdown_fused_synthesis_chooser_and_fp32():
    """Above 2 x (SM count) templates the chooser takes the panel route (measured faster, profiles/r02_ring_fused.md); the
    fused route also exists in the fp32 build (two item pipelines per CTA)."""
    w = W.make("c2", B=700, n_scale=2)
    H_ref = OT.family_rows(w.family, w.params, w.seg_lengths, w.fs)
    ref = O.loglike_batch(w.acf, w.seg_lengths, w.d, H_ref)
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        d, p = _dev(w.d), _dev(w.params)
        out_big = h.loglike_family_batch(d, w.family, p, w.fs).cpu().numpy()
        n_big = h.last_launches()
        out_small = h.loglike_family_batch(d, w.family, p[:100].contiguous(), w.fs).cpu().numpy()
        n_small = h.last_launches()
        h.set_precision(tdb.TD_PREC_F32)
        out32 = h.loglike_family_batch(d, w.family, p[:100].contiguous(), w.fs).cpu().numpy()
        n32 = h.last_launches()
    assert n_big >= 2 and n_small == 1 and n32 == 1
    _assert_close(out_big, ref, what="c2 params, large batch (panel)")
    _assert_close(out_small, ref[:100], what="c2 params, small batch (fused)")
    _assert_close(out32, ref[:100], tol=2e-5, what="c2 params, fused, fp32")


def test_ringdown_params_entry_errors_and_edges():
    w = W.make("c3", B=4)
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        with pytest.raises(ValueError):
            h.loglike_family_batch(_dev(w.d), tdb.TD_FAMILY_RINGDOWN, _dev(np.ones((4, 5))), w.fs)   # three segments need [B, 3, 5]
    w = W.make("c1", B=5)
    p = w.params.copy()
    p[1, 4] = 2.0        # t0 beyond the segment: the template is identically zero -> logL = -1/2 <d,d>
    p[2, 4] = -0.25      # t0 before the segment: live from the first sample
    H = OT.family_rows(OT.RINGDOWN, p, w.seg_lengths, w.fs)
    assert np.all(H[1] == 0.0) and H[2, 0] != 0.0
    ref = O.loglike_batch(w.acf, w.seg_lengths, w.d, H)
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        out = h.loglike_family_batch(_dev(w.d), tdb.TD_FAMILY_RINGDOWN, _dev(p), w.fs).cpu().numpy()
        with pytest.raises(tdb.TDError):
            h.loglike_family_batch(_dev(w.d), tdb.TD_FAMILY_RINGDOWN, _dev(p), 0.0)
        with pytest.raises(tdb.TDError) as e:
            h.loglike_family_batch(_dev(w.d), 7, _dev(p), w.fs)
        assert e.value.status == tdb.TD_EINVAL
    _assert_close(out, ref, what="ringdown edges")


@pytest.mark.parametrize("name,B", [("c1", 700), ("c2", 650)])
def test_fused_many_items_per_cta_repeatable(name, B):
    """More templates than SMs: every CTA loops over several items, with the counter-based hand-over between items
    (no CTA barrier at the end of an item).  Bitwise repeatable, equal to the staged global-memory variant, and a
    sample against the oracle.  (compute-sanitizer is not available on the GPU pool: races would show up here.)"""
    w = W.make(name, B=B)
    sub = np.arange(0, B, 37)
    ref = O.loglike_batch(w.acf, w.seg_lengths, w.d, w.H[sub])
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        d, H = _dev(w.d), _dev(w.H)
        outs = [h.loglike_batch(d, H) for _ in range(4)]
        inn = [h.inner_batch(d, H) for _ in range(2)]
        torch.cuda.synchronize()
        h.set_fft_variant(2)
        o_staged = h.loglike_batch(d, H).cpu().numpy()
    for o in outs[1:]:
        assert torch.equal(outs[0], o)
    assert torch.equal(inn[0][0], inn[1][0]) and torch.equal(inn[0][1], inn[1][1])
    o0 = outs[0].cpu().numpy()
    _assert_close(o0[sub], ref, what=f"{name} B={B}")
    _assert_close(o0, o_staged, tol=1e-11, what="fused vs staged")


# ------------------------------------------------------------------ degenerate rows on the dense, dot and cluster paths
@pytest.mark.parametrize("name,n_scale,path", [("d2", 1, tdb.TD_PATH_DENSE), ("d4", 1, tdb.TD_PATH_DENSE),
                                               ("d2", 1, tdb.TD_PATH_AUTO), ("d5", 1, tdb.TD_PATH_CDO),
                                               ("c5", 1, tdb.TD_PATH_AUTO), ("c4", 4, tdb.TD_PATH_AUTO)])
def test_exact_zero_nan_row_and_single_template(name, n_scale, path):
    """h = d gives exactly 0 (pin P8 iv), a NaN poisons only its own row, B = 1 and a strided H work, on the dense
    (cp.async panels), cluster and staged kernels; the dot path keeps a NaN row to itself as well."""
    w = W.make(name, B=9, n_scale=n_scale)
    n = w.n_tot
    fn = O.loglike_batch_solve_toeplitz if name == "c4" else O.loglike_batch
    ref = fn(w.acf, w.seg_lengths, w.d, w.H)
    Hpad = torch.zeros(9, n + 6, dtype=torch.float64, device="cuda")
    Hpad[:, :n] = _dev(w.H)
    Hpad[3, :n] = _dev(w.d)
    Hpad[5, n // 2] = float("nan")
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        h.set_path(path)
        out = h.loglike_batch(_dev(w.d), Hpad[:, :n]).cpu().numpy()
        one = h.loglike_batch(_dev(w.d), Hpad[7:8, :n]).cpu().numpy()
        h.set_path(tdb.TD_PATH_AUTO)
        dh, _ = h.inner_batch(_dev(w.d), Hpad[:, :n], want_hh=False)
        dh = dh.cpu().numpy()
    assert out[3] == 0.0
    assert np.isnan(out[5]) and np.isnan(dh[5])
    keep = [0, 1, 2, 4, 6, 7, 8]
    _assert_close(out[keep], ref[keep], what=f"{name} degenerate rows")
    assert one[0] == out[7]
    assert np.all(np.isfinite(dh[keep]))


def test_empty_batch_is_a_no_op_everywhere():
    w = W.make("c1", B=2)
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        d = _dev(w.d)
        H0 = torch.zeros(0, w.n_tot, dtype=torch.float64, device="cuda")
        assert h.loglike_batch(d, H0).numel() == 0
        dh, hh = h.inner_batch(d, H0)
        assert dh.numel() == 0 and hh.numel() == 0
        p0 = torch.zeros(0, 5, dtype=torch.float64, device="cuda")
        assert h.loglike_family_batch(d, tdb.TD_FAMILY_RINGDOWN, p0, w.fs).numel() == 0


def test_long_segment_five_pass_plan():
    """N = 131072 (M = 2^17 = [2,16,16,16,16]): the staged path with a generic global pass around the shared-memory
    block kernels, the longest plan exercised; oracle route = library Levinson solve (pin P13; dense C would be 128 GiB)."""
    N = 131072
    rng = np.random.default_rng(N)
    rho = W.acf_from_psd(4096.0, 2 * N, N)
    d = rng.standard_normal(N) * 1e-21
    H = rng.standard_normal((3, N)) * 1e-21
    ref = O.loglike_batch_solve_toeplitz(rho, [N], d, H[:1])
    with tdb.TDLikelihood(rho, [N]) as h:
        out = h.loglike_batch(_dev(d), _dev(H)).cpu().numpy()
        out2 = h.loglike_batch(_dev(d), _dev(H[::-1].copy())).cpu().numpy()
    _assert_close(out[:1], ref, what="N = 131072")
    assert np.array_equal(out, out2[::-1])          # a row's result does not depend on its slot in the batch
    assert np.all(out < 0.0)


def test_staged_two_lane_pipeline_on_a_side_stream():
    """The staged path alternates chunks between the caller's stream and an internal one (fork / join events).
    On a non-default stream, back to back, with the inputs produced on that same stream just before: results must be
    bitwise repeatable, complete when the caller's stream is, and equal to the oracle on a sample."""
    w = W.make("c4", B=150, n_scale=4)              # N = 16384: 61 templates per chunk and lane -> 3 chunks, both lanes
    ref = O.loglike_batch_solve_toeplitz(w.acf, w.seg_lengths, w.d, w.H[:2])
    s = torch.cuda.Stream()
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        h.set_fft_variant(2)                        # (variant 0 runs this size class on the group kernel, td_group16.cuh)
        Hc = torch.as_tensor(w.H).pin_memory()
        torch.cuda.synchronize()
        with torch.cuda.stream(s):
            d = torch.as_tensor(w.d).pin_memory().to("cuda", non_blocking=True)
            H = Hc.to("cuda", non_blocking=True)   # the kernels of both lanes must wait for this copy
            o1 = h.loglike_batch(d, H)
            o2 = h.loglike_batch(d, H)
            o1c = o1.clone()                        # ordered after the join on the caller's stream
        s.synchronize()
        assert h.last_launches() > 12               # more than two chunks' worth of kernels
    assert torch.equal(o1c, o2)
    _assert_close(o1c.cpu().numpy()[:2], ref, what="staged two-lane")


def test_many_segments_in_one_size_class():
    """Ten segments of one size class: more than the fused kernel caches in shared memory (F4_SEGCACHE = 8), so the
    segment records come from global memory; plus nine segments of the cluster class."""
    rng = np.random.default_rng(21)
    for lens in ([1024] * 10, [5000] * 9):
        rho = W.acf_from_psd(4096.0, 2 * 8192, max(lens))
        acf = np.concatenate([(1.0 + 0.1 * k) * rho[:n] for k, n in enumerate(lens)])
        nt = sum(lens)
        d = rng.standard_normal(nt) * 1e-21
        H = rng.standard_normal((5, nt)) * 1e-21
        ref = O.loglike_batch(acf, lens, d, H)
        with tdb.TDLikelihood(acf, lens) as h:
            out = h.loglike_batch(_dev(d), _dev(H)).cpu().numpy()
            assert h.last_launches() == 1
        _assert_close(out, ref, what=f"{len(lens)} segments of {lens[0]}")


@pytest.mark.parametrize("n", [16384, 20001])
def test_cooperative_setup_matches_oracle_levinson(n):
    """Segments of >= 16384 samples run the recursion on a cooperative multi-CTA grid (levinson_coop_kernel)."""
    rho = W.acf_from_psd(4096.0, 2 * 65536, n)
    a_ref, v_ref, ld_ref = O.levinson_durbin_fast(rho)
    with tdb.TDLikelihood(rho, [n]) as h:
        a = h.generator(0)
        info = h.info()
    assert np.max(np.abs(a - a_ref)) <= 1e-10 * np.max(np.abs(a_ref))
    assert abs(info["v"][0] - v_ref) <= 1e-11 * v_ref
    assert abs(info["logdet"][0] - ld_ref) <= 1e-10 * abs(ld_ref)


def test_long_non_spd_acf_is_rejected_by_the_cooperative_setup():
    bad = W.acf_from_psd(4096.0, 2 * 65536, 20000).copy()
    bad[1] = 1.5 * bad[0]                              # |rho_1| > rho_0: not positive definite
    with pytest.raises(tdb.TDError) as e:
        tdb.TDLikelihood(bad, [20000])
    assert e.value.status == tdb.TD_ENOTSPD
    bad[1] = float("nan")
    with pytest.raises(tdb.TDError) as e:
        tdb.TDLikelihood(bad, [20000])
    assert e.value.status == tdb.TD_ENOTSPD


# ------------------------------------------------------------------ allocation-free, capturable, stream-safe calls
@pytest.mark.parametrize("name,B,n_scale", [("c1", 64, 1), ("c3", 48, 1), ("c4", 40, 4), ("d2", 256, 1)])
def test_calls_capture_into_a_cuda_graph_and_replay(name, B, n_scale):
    """td_loglike_batch + td_inner_batch enqueue kernels only (no allocation, no synchronisation, every attribute set by
    td_create): both are captured into ONE CUDA graph on a side stream and replayed on new data in the same buffers."""
    w = W.make(name, B=B, n_scale=n_scale)
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        d, H = _dev(w.d), _dev(w.H)
        out = torch.empty(B, dtype=torch.float64, device="cuda")
        dh = torch.empty(B, dtype=torch.float64, device="cuda")
        eager = h.loglike_batch(d, H).clone()
        dh_e, hh_e = h.inner_batch(d, H)
        torch.cuda.synchronize()
        side = torch.cuda.Stream()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.stream(side):
            with torch.cuda.graph(g, stream=side):
                h.loglike_batch(d, H, out=out, stream=side)
                h.inner_batch(d, H, want_hh=False, stream=side, out_dh=dh)
        for rep in range(2):
            if rep == 1:                         # new templates in the captured buffers
                H.copy_(torch.flip(H, dims=[0]))
            out.zero_(); dh.zero_()
            g.replay()
            torch.cuda.synchronize()
            ref = eager if rep == 0 else torch.flip(eager, dims=[0])
            ref_dh = dh_e if rep == 0 else torch.flip(dh_e, dims=[0])
            assert torch.equal(out, ref), f"{name}: graph replay {rep} differs from the eager call"
            scale = float((hh_e.abs() + 1.0).max())
            assert float((dh - ref_dh).abs().max()) <= 1e-9 * scale * 10
    ref = O.loglike_batch(w.acf, w.seg_lengths, w.d, w.H) if w.n_tot <= 20000 else None
    if ref is not None:
        _assert_close(eager.cpu().numpy(), ref, what=f"{name} eager")


@pytest.mark.parametrize("name,B,n_scale", [("c4", 48, 4), ("c5", 32, 2)])
def test_one_handle_alternating_between_two_streams(name, B, n_scale):
    """the handle owns scratch (staged workspace, z / u of the data vector).  One host thread issuing calls on
    two different streams must get the results of serial execution: a call on another stream than the previous
    scratch-using call waits for it (include/tdlike.h, "Threads and streams")."""
    w = W.make(name, B=B, n_scale=n_scale)
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        d, H = _dev(w.d), _dev(w.H)
        H2 = torch.flip(H, dims=[0]).contiguous()
        ref1 = h.loglike_batch(d, H).clone()
        dh1, _ = h.inner_batch(d, H, want_hh=False)
        dh1 = dh1.clone()
        torch.cuda.synchronize()
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        for _ in range(3):
            o1 = h.loglike_batch(d, H, stream=s1)
            o2 = h.loglike_batch(d, H2, stream=s2)
            a1, _ = h.inner_batch(d, H, want_hh=False, stream=s1)
            a2, _ = h.inner_batch(d, H2, want_hh=False, stream=s2)
            torch.cuda.synchronize()
            assert torch.equal(o1, ref1) and torch.equal(o2, torch.flip(ref1, dims=[0]))
            assert torch.equal(a1, dh1) and torch.equal(a2, torch.flip(dh1, dims=[0]))


def test_family_host_entry_with_odd_batch_keeps_rows_aligned():
    """5 n_seg B odd used to leave d 8-byte aligned inside the packed device buffer (TMA staging silently off).
    The sections are now rounded to 16 bytes; results are bit-identical to the device-pointer call."""
    for name, B in (("c1", 7), ("c5", 5)):
        w = W.make(name, B=B, n_scale=1 if name == "c1" else 4)
        with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
            h.reserve(B)
            out_host = h.loglike_family_batch_host(w.d, w.family, w.params, w.fs)
            out_dev = h.loglike_family_batch(_dev(w.d), w.family, _dev(w.params), w.fs).cpu().numpy()
        assert np.array_equal(out_host, out_dev)
        H = OT.family_rows(w.family, w.params, w.seg_lengths, w.fs)
        _assert_close(out_host, O.loglike_batch(w.acf, w.seg_lengths, w.d, H), what=f"{name} odd B")


# ------------------------------------------------------------------ FP32 evaluation with FP64 setup
# Tolerance against the SAME fp64 oracle: |dQ|/Q <= 4 (log2(2M) + 1) eps32 kappa, eps32 = 2^-24,
# kappa = (|y1|^2 + |y2|^2) / (|y1|^2 - |y2|^2) >= 1 the cancellation factor of the Gohberg-Semencul difference
# (1.003 .. 1.05 on c1-c5, measured with the oracle's time-domain GS route).  At 2M = 16384 and kappa <= 5: 1.8e-5.
TOL32 = 2e-5


@pytest.mark.parametrize("name,B,n_scale", [("c1", 64, 1), ("c2", 96, 1), ("c3", 24, 1), ("c5", 16, 1)])
def test_f32_evaluation_matches_the_fp64_oracle(name, B, n_scale):
    w = W.make(name, B=B, n_scale=n_scale)
    ref = O.loglike_batch(w.acf, w.seg_lengths, w.d, w.H)
    dh_ref, hh_ref = O.inner_batch(w.acf, w.seg_lengths, w.d, w.H)
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        d, H = _dev(w.d), _dev(w.H)
        o64 = h.loglike_batch(d, H).clone()
        h.set_precision(tdb.TD_PREC_F32)
        o32 = h.loglike_batch(d, H).clone()
        o32b = h.loglike_batch(d, H).clone()
        dh, hh = h.inner_batch(d, H)                      # fp32 STOREZ + INNER kernels
        dh_only, _ = h.inner_batch(d, H, want_hh=False)   # the dot path stays fp64
        path_dot = h.info()["last_path"]
        h.set_precision(tdb.TD_PREC_F64)
        o64b = h.loglike_batch(d, H)
        torch.cuda.synchronize()
    e32 = _assert_close(o32.cpu().numpy(), ref, tol=TOL32, what=f"{name} f32")
    assert e32 > 1e-12, "the fp32 build was not used"            # an fp64 result would sit at 1e-14
    assert torch.equal(o32, o32b)                                 # deterministic
    assert torch.equal(o64, o64b)                                 # switching back restores the fp64 kernels bit for bit
    _assert_close(o64.cpu().numpy(), ref, what=f"{name} f64 beside it")
    scale = np.abs(hh_ref) + np.abs(dh_ref) + 1.0
    assert np.max(np.abs(hh.cpu().numpy() - hh_ref) / scale) <= TOL32
    assert np.max(np.abs(dh.cpu().numpy() - dh_ref) / scale) <= TOL32
    assert path_dot == tdb.TD_PATH_DOT
    assert np.max(np.abs(dh_only.cpu().numpy() - dh_ref) / scale) <= TOL


def test_f32_edges_exact_zero_nan_unsupported_and_mixed_classes():
    # h = d gives exactly 0 (the residual is formed in fp64 before rounding); a NaN row stays confined to its output
    w = W.make("c2", B=6, n_scale=2)
    H = w.H.copy()
    H[1] = w.d
    H[3, 17] = np.nan
    ref = O.loglike_batch(w.acf, w.seg_lengths, w.d, np.nan_to_num(H))
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        h.set_precision(tdb.TD_PREC_F32)
        out = h.loglike_batch(_dev(w.d), _dev(H)).cpu().numpy()
    assert out[1] == 0.0 and np.isnan(out[3])
    keep = [0, 2, 4, 5]
    _assert_close(out[keep], ref[keep], tol=TOL32, what="f32 edges")
    # a handle whose only segment is short (dense / small fused kernels): no fp32 kernel -> EUNSUPPORTED, setting unchanged
    w = W.make("d3", B=32)
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        with pytest.raises(tdb.TDError) as e:
            h.set_precision(tdb.TD_PREC_F32)
        assert e.value.status == tdb.TD_EUNSUPPORTED
        with pytest.raises(tdb.TDError):
            h.set_precision(7)
        out = h.loglike_batch(_dev(w.d), _dev(w.H)).cpu().numpy()
    _assert_close(out, O.loglike_batch(w.acf, w.seg_lengths, w.d, w.H), what="d3 after a refused precision switch")
    # mixed size classes: 3000 (fp32 fused kernel), 300 (dense, fp64), 5000 (fp32 cluster kernel), odd offsets
    rng = np.random.default_rng(5)
    lens = [3001, 300, 5000]
    acf = np.concatenate([W.acf_from_psd(4096.0, 2 * n, n) * s for n, s in zip(lens, (1.0, 0.7, 1.9))])
    d = rng.standard_normal(sum(lens)) * 1e-21
    Hm = rng.standard_normal((9, sum(lens))) * 1e-21
    ref = O.loglike_batch(acf, lens, d, Hm)
    with tdb.TDLikelihood(acf, lens) as h:
        h.set_precision(tdb.TD_PREC_F32)
        out = h.loglike_batch(_dev(d), _dev(Hm)).cpu().numpy()
    _assert_close(out, ref, tol=TOL32, what="f32 mixed classes")


@pytest.mark.parametrize("name", ["c2", "c5"])
def test_f32_full_size_against_the_fp64_path(name):
    """Full batch in the launch configuration bench.py --dtype f32 times: every row against the fp64 GPU result (itself
    held to 1e-9 against the oracle by test_full_size_*), a sample of rows against the oracle directly."""
    w = W.make(name)
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        d, H = _dev(w.d), _dev(w.H)
        o64 = h.loglike_batch(d, H).cpu().numpy()
        h.set_precision(tdb.TD_PREC_F32)
        o32 = h.loglike_batch(d, H).cpu().numpy()
    err = np.abs(o32 - o64) / np.maximum(np.abs(o64), 1.0)
    assert err.max() <= TOL32, f"{name}: {err.max():.2e}"
    idx = np.linspace(0, w.B - 1, 12).astype(int)
    ref = O.loglike_batch(w.acf, w.seg_lengths, w.d, w.H[idx])
    _assert_close(o32[idx], ref, tol=TOL32, what=f"{name} f32 full size")
    print(f"{name}: fp32 vs fp64 over {w.B} rows: max {err.max():.2e}, median {np.median(err):.2e}")


# ------------------------------------------------------------------ very long segments
def test_very_long_segment_2pow20():
    """N = 2^20 (transform length 2^21, five-pass plans, cooperative Levinson-Durbin over 2^20 orders).
    (a) AR(2) covariance: every row against the closed-form exact AR likelihood of the oracle (pin P19), 1e-9;
    (b) the PSD-recipe ACF of the configs: the chi-square invariant E[x^T C^-1 x] = N for x ~ N(0, C) (one draw:
        N +- 4 sqrt(2N)) and the bilinear identity of Eq. 13 between td_loglike_batch and td_inner_batch.
    Prints the td_create times (S0 is one-time and cached; reported, not part of the metric)."""
    import time
    N = 1 << 20
    rng = np.random.default_rng(20)
    phi, s2 = [1.6, -0.8], 3.0e-43
    rho = O.ar_acf(phi, s2, N)
    x = np.sqrt(s2) * rng.standard_normal(N)
    for t in range(2, N):                      # one AR(2) path (any vector would do: the identity is exact)
        x[t] += phi[0] * x[t - 1] + phi[1] * x[t - 2]
    H = np.zeros((3, N))
    H[1] = 0.25 * np.roll(x, 1000)
    H[2] = np.sqrt(s2) * rng.standard_normal(N)
    ref = np.array([-0.5 * O.ar_quadform_closed(phi, s2, x - H[b]) for b in range(3)])
    t0 = time.perf_counter()
    with tdb.TDLikelihood(rho, [N]) as h:
        t_ar = time.perf_counter() - t0
        out = h.loglike_batch(_dev(x), _dev(H)).cpu().numpy()
        v = h.info()["v"][0]
    _assert_close(out, ref, what="N = 2^20, AR(2) closed form")
    assert abs(v / s2 - 1.0) < 1e-9
    fs = 4096.0
    rho = W.acf_from_psd(fs, 2 * N, N)
    x = W._noise(rng, fs, 2 * N, N)
    Hh = 0.5 * np.roll(x, 12345)[None, :]
    t0 = time.perf_counter()
    with tdb.TDLikelihood(rho, [N]) as h:
        t_psd = time.perf_counter() - t0
        d = _dev(x)
        q = -2.0 * float(h.loglike_batch(d, _dev(np.zeros((1, N)))).item())
        ll = float(h.loglike_batch(d, _dev(Hh)).item())
        dh, hh = h.inner_batch(d, _dev(Hh))
        launches = h.last_launches()
    assert abs(q - N) <= 4.0 * np.sqrt(2.0 * N), f"chi-square invariant: Q = {q}, N = {N}"
    assert abs(-2.0 * ll - (q - 2.0 * float(dh.item()) + float(hh.item()))) <= 1e-9 * (q + float(hh.item()))
    print(f"N = 2^20: td_create {t_ar:.1f} s (AR(2) ACF), {t_psd:.1f} s (PSD-recipe ACF); Q/N = {q / N:.6f}; "
          f"{launches} launches per td_inner_batch")


# ------------------------------------------------------------------ CDO path: Y = L^-1 X with the cached whitening operator
@pytest.mark.parametrize("n", [1, 31, 64, 100, 257, 512, 777, 1024])
def test_cdo_path_lengths(n):
    """SURVEY 8(f) NEXT-3, second half: the triangular contraction against the oracle, which is the
    same quantity computed the same way (dense Cholesky, forward substitution) on the CPU."""
    rng = np.random.default_rng(400 + n)
    rho = W.acf_from_psd(4096.0, max(2 * n, 64), n)
    B = 70 if n < 600 else 37          # several 32-template tiles and a ragged tail
    d = rng.standard_normal(n) * 1e-21
    H = rng.standard_normal((B, n)) * 1e-21
    H[3] = d
    ref = O.loglike_batch(rho, [n], d, H)
    with tdb.TDLikelihood(rho, [n]) as h:
        h.set_path(tdb.TD_PATH_CDO)
        out = h.loglike_batch(_dev(d), _dev(H)).cpu().numpy()
        assert h.info()["last_path"] == tdb.TD_PATH_CDO
        dh, hh = h.inner_batch(_dev(d), _dev(H))           # cross terms keep the Gohberg-Semencul dense kernel
    assert out[3] == 0.0
    _assert_close(out, ref, what=f"cdo n={n}")
    _, hh_ref = O.inner_batch(rho, [n], d, H)
    assert np.max(np.abs(hh.cpu().numpy() - hh_ref) / np.abs(hh_ref)) <= TOL


@pytest.mark.parametrize("lens,paths", [([500], "cdo"), ([512], "cdo"), ([513], "fft"), ([700], "fft"), ([1024], "fft"),
                                        ([300, 900], "cdo+fft2"), ([40, 500, 3000], "cdo+fft")])
def test_auto_chooser_crossover_at_512(lens, paths):
    """AUTO, log-likelihood: a size class whose segments are all at most 512 samples long takes the dense kernels (CDO from 65
    samples), everything longer the FFT kernels - the M = 1024 kernel with four item pipelines per CTA beats the CDO kernel
    from 513 samples up (crossover scan in profiles/r02_cdo.md; the limit was 768 while that kernel ran one pipeline)."""
    rng = np.random.default_rng(sum(lens))
    acf = np.concatenate([W.acf_from_psd(4096.0, 2 * max(n, 32), n) * (1.0 + 0.3 * i) for i, n in enumerate(lens)])
    nt, B = sum(lens), 41
    d = rng.standard_normal(nt) * 1e-21
    H = rng.standard_normal((B, nt)) * 1e-21
    H[5] = d
    with tdb.TDLikelihood(acf, lens) as h:
        out = h.loglike_batch(_dev(d), _dev(H)).cpu().numpy()
        lp, nl = h.info()["last_path"], h.last_launches()
    _assert_close(out, O.loglike_batch(acf, lens, d, H), what=f"auto {lens}")
    assert out[5] == 0.0 or "+" in paths and abs(out[5]) <= 1e-9
    if paths == "cdo":
        assert lp == tdb.TD_PATH_CDO and nl == 1
    elif paths == "fft":
        assert lp == tdb.TD_PATH_FFT and nl == 1
    elif paths == "cdo+fft2":
        assert nl == 2                                         # CDO (300), fused FFT (900)
    else:
        assert nl == 3                                         # GS dense (40), CDO (500), fused FFT (3000)


@pytest.mark.parametrize("n,Bs", [(1000, (1, 3, 149, 300, 593)), (2000, (1, 2, 149, 297))])
def test_item_pipelines_every_batch_shape(n, Bs):
    """The one-CTA kernel runs 4 (M = 1024) / 2 (M = 2048) item pipelines per CTA, items dealt pipeline-major over min(B, SMs)
    CTAs: batches smaller than a pipeline set, one more than the SM count, between one and NGRP items per SM, and one more
    than a full wave - every row against the oracle, in fp64 and in the fp32 build (8 / 4 pipelines), rows independent of B."""
    rng = np.random.default_rng(n)
    rho = W.acf_from_psd(4096.0, 4096, n)
    d = rng.standard_normal(n) * 1e-21
    Hall = rng.standard_normal((max(Bs), n)) * 1e-21
    Hall[0] = d
    ref = O.loglike_batch(rho, [n], d, Hall)
    with tdb.TDLikelihood(rho, [n]) as h:
        for prec, tol in ((tdb.TD_PREC_F64, TOL), (tdb.TD_PREC_F32, TOL32)):
            h.set_precision(prec)
            for B in Bs:
                out = h.loglike_batch(_dev(d), _dev(Hall[:B])).cpu().numpy()
                assert h.last_launches() == 1 and out[0] == 0.0
                _assert_close(out, ref[:B], tol=tol, what=f"pipelines n={n} B={B} prec={prec}")


def test_cdo_multi_segment_odd_offsets_and_limits():
    rng = np.random.default_rng(77)
    lens = [333, 64, 1000]
    acf = np.concatenate([W.acf_from_psd(4096.0, 2 * n, n) * s for n, s in zip(lens, (1.0, 2.5, 0.6))])
    d = rng.standard_normal(sum(lens)) * 1e-21
    H = rng.standard_normal((45, sum(lens) + 3))[:, :sum(lens)] * 1e-21     # odd leading dimension: 8-byte copies
    ref = O.loglike_batch(acf, lens, d, H)
    with tdb.TDLikelihood(acf, lens) as h:
        h.set_path(tdb.TD_PATH_CDO)
        out = h.loglike_batch(_dev(d), _dev(H)).cpu().numpy()
        h.set_path(tdb.TD_PATH_DENSE)
        out_gs = h.loglike_batch(_dev(d), _dev(H)).cpu().numpy()
    _assert_close(out, ref, what="cdo multi-segment")
    _assert_close(out_gs, ref, what="gs dense beside it")
    w = W.make("c1", B=4, n_scale=1)
    acf2 = W.acf_from_psd(4096.0, 4096, 2048)
    with tdb.TDLikelihood(acf2, [2048]) as h:
        with pytest.raises(tdb.TDError) as e:
            h.set_path(tdb.TD_PATH_CDO)                      # 2048 > 1024
        assert e.value.status == tdb.TD_EUNSUPPORTED


def test_fp32_and_parameter_calls_capture_into_a_cuda_graph():
    """After td_set_precision / td_reserve the fp32 kernels and the parameter entry point (fused synthesis for a small
    batch, panel route for a large one) are launches only as well: captured and replayed."""
    w = W.make("c2", B=400, n_scale=2)
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        h.set_precision(tdb.TD_PREC_F32)
        h.reserve(400)
        d, H, p = _dev(w.d), _dev(w.H), _dev(w.params)
        p_small = p[:64].contiguous()
        e_rows = h.loglike_batch(d, H).clone()
        e_small = h.loglike_family_batch(d, w.family, p_small, w.fs).clone()
        e_big = h.loglike_family_batch(d, w.family, p, w.fs).clone()
        torch.cuda.synchronize()
        o_rows = torch.empty_like(e_rows); o_small = torch.empty_like(e_small); o_big = torch.empty_like(e_big)
        side = torch.cuda.Stream()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.stream(side):
            with torch.cuda.graph(g, stream=side):
                h.loglike_batch(d, H, out=o_rows, stream=side)
                h.loglike_family_batch(d, w.family, p_small, w.fs, out=o_small, stream=side)
                h.loglike_family_batch(d, w.family, p, w.fs, out=o_big, stream=side)
        for _ in range(2):
            o_rows.zero_(); o_small.zero_(); o_big.zero_()
            g.replay()
            torch.cuda.synchronize()
            assert torch.equal(o_rows, e_rows) and torch.equal(o_small, e_small) and torch.equal(o_big, e_big)
    ref = O.loglike_batch(w.acf, w.seg_lengths, w.d, w.H[:50])
    _assert_close(e_rows.cpu().numpy()[:50], ref, tol=TOL32, what="fp32 rows")
    _assert_close(e_big.cpu().numpy()[:50], ref, tol=TOL32, what="fp32 params")


@pytest.mark.parametrize("variant", [0, 2])
def test_f32_long_segments_on_the_group_and_staged_kernels(variant):
    """Segments of 8193+ samples run the fp32 build of the group kernel (variant 0; classes up to 65536) or of the staged
    kernels (variant 2, and every longer class) - the paper's own FP32 example is N = 16384: a sample of rows
    against the fp64 oracle (library Levinson solve), every row against the fp64 GPU result, cross terms, and the full c4
    size against the fp64 path."""
    w = W.make("c4", B=40, n_scale=4)
    ref = O.loglike_batch_solve_toeplitz(w.acf, w.seg_lengths, w.d, w.H[:4])
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        d, H = _dev(w.d), _dev(w.H)
        o64 = h.loglike_batch(d, H).cpu().numpy()
        dh64, hh64 = h.inner_batch(d, H)
        h.set_precision(tdb.TD_PREC_F32)
        h.set_fft_variant(variant)
        o32 = h.loglike_batch(d, H).cpu().numpy()
        assert (h.last_launches() == 2) == (variant == 0)
        dh32, hh32 = h.inner_batch(d, H)
        torch.cuda.synchronize()
    _assert_close(o32[:4], ref, tol=TOL32, what="c4/4 fp32 vs oracle")
    err = np.abs(o32 - o64) / np.maximum(np.abs(o64), 1.0)
    assert 1e-12 < err.max() <= TOL32
    scale = hh64.abs() + dh64.abs() + 1.0
    assert float(((hh32 - hh64).abs() / scale).max()) <= TOL32 and float(((dh32 - dh64).abs() / scale).max()) <= TOL32
    w = W.make("c4")
    with tdb.TDLikelihood(w.acf, w.seg_lengths) as h:
        d, H = _dev(w.d), _dev(w.H)
        o64 = h.loglike_batch(d, H).cpu().numpy()
        h.set_precision(tdb.TD_PREC_F32)
        h.set_fft_variant(variant)
        o32 = h.loglike_batch(d, H).cpu().numpy()
    err = np.abs(o32 - o64) / np.maximum(np.abs(o64), 1.0)
    assert 1e-12 < err.max() <= TOL32, f"c4 full size: {err.max():.2e}"


def test_f32_group_kernel_ragged_mixed_sizes_and_exact_zero():
    """fp32 group kernel: odd lengths (scalar loads), group sizes 4 / 8 / 16 and a fused-kernel class in one handle, more
    templates than groups; h = d gives exactly 0; against the fp64 oracle on two rows and the fp64 GPU path on all."""
    lens = [9001, 40001, 20000, 3000]
    rng = np.random.default_rng(3232)
    acf = np.concatenate([W.acf_from_psd(4096.0, 2 * 65536, n) * (1.0 + 0.2 * i) for i, n in enumerate(lens)])
    nt, B = sum(lens), 43
    d = rng.standard_normal(nt) * 1e-21
    H = rng.standard_normal((B, nt)) * 1e-21
    H[11] = d
    dd, HH = _dev(d), _dev(H)
    with tdb.TDLikelihood(acf, lens) as h:
        o64 = h.loglike_batch(dd, HH).cpu().numpy()
        h.set_precision(tdb.TD_PREC_F32)
        o32 = h.loglike_batch(dd, HH).cpu().numpy()
        assert h.last_launches() == 7                       # 3 x (group kernel + partial sums) + one fused kernel
        o32b = h.loglike_batch(dd, HH).cpu().numpy()
    assert o32[11] == 0.0 and np.array_equal(o32, o32b)
    _assert_close(o32, o64, tol=TOL32, what="fp32 group kernel vs fp64 path")
    _assert_close(o32[:2], O.loglike_batch_solve_toeplitz(acf, lens, d, H[:2]), tol=TOL32, what="fp32 group kernel vs oracle")


def test_f32_mixed_staged_fused_and_dense_classes():
    """One handle with a staged-class segment (20000 samples), a cluster-class one (5000), a fused-class one (3000) and a
    dense-class one (200): fp32 evaluation accumulates over all of them (the dense segment stays fp64) and agrees with the
    fp64 evaluation of the same handle, itself checked against the oracle on a few rows."""
    rng = np.random.default_rng(321)
    lens = [20000, 200, 5000, 3000]
    acf = np.concatenate([W.acf_from_psd(4096.0, 2 * 32768, n) * s for n, s in zip(lens, (1.0, 0.5, 1.7, 0.9))])
    nt = sum(lens)
    d = rng.standard_normal(nt) * 1e-21
    H = rng.standard_normal((21, nt)) * 1e-21
    ref = O.loglike_batch_solve_toeplitz(acf, lens, d, H[:3])
    with tdb.TDLikelihood(acf, lens) as h:
        o64 = h.loglike_batch(_dev(d), _dev(H)).cpu().numpy()
        dh64, hh64 = h.inner_batch(_dev(d), _dev(H))
        h.set_precision(tdb.TD_PREC_F32)
        o32 = h.loglike_batch(_dev(d), _dev(H)).cpu().numpy()
        dh32, hh32 = h.inner_batch(_dev(d), _dev(H))
        torch.cuda.synchronize()
    _assert_close(o64[:3], ref, what="mixed classes fp64")
    _assert_close(o32, o64, tol=TOL32, what="mixed classes fp32 vs fp64")
    scale = hh64.abs() + dh64.abs() + 1.0
    assert float(((hh32 - hh64).abs() / scale).max()) <= TOL32 and float(((dh32 - dh64).abs() / scale).max()) <= TOL32
