"""Pins for the CPU oracle (oracle/td_oracle.py): it is checked against what the paper and the
mathematics fix, never against itself or the CUDA path.  SURVEY.md 8(c) P1-P14.

The paper prints no numerical value of any inner product or log-likelihood (its benchmark,
Fig. 5, is an image), so there is no "paper prints X" fixture; the golden
file tests/golden/ar1_closed_form.txt holds closed-form values written out by hand from the
AR(1) tridiagonal inverse (textbook result), with its derivation.
"""
import os

import numpy as np
import pytest
import scipy.linalg as sla

from oracle import td_oracle as O
from oracle import templates as OT
from paper_2603_06010_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rel(a, b):
    return abs(a - b) / max(abs(b), 1e-300)


def _psd_rho(n, fs=4096.0):
    return W.acf_from_psd(fs, 2 * max(n, 8), n)


# ---------------------------------------------------------------- P1 brute force
@pytest.mark.parametrize("n", [1, 2, 3, 8, 64, 256])
def test_p1_bruteforce_inverse(n):
    rng = np.random.default_rng(100 + n)
    for kind in ("ar", "psd"):
        if kind == "ar":
            rho = W.ar_acf([0.6, -0.3, 0.1], 2.5, n)
        else:
            rho = _psd_rho(n) * 1e44
        x = rng.standard_normal(n)
        q_bf = O.quadform_bruteforce(rho, x)
        q_ch = O.quadform(rho, x)
        assert _rel(q_ch, q_bf) < 1e-11
        # the batched entry point on the same numbers (d = x, h = 0)
        ll = O.loglike_batch(rho, [n], x, np.zeros((1, n)))[0]
        assert _rel(-2 * ll, q_bf) < 1e-11


# ---------------------------------------------------------------- P2 white noise
def test_p2_white_noise():
    rng = np.random.default_rng(2)
    n, s2 = 300, 3.7e-44
    rho = np.zeros(n)
    rho[0] = s2
    x = rng.standard_normal(n) * 1e-21
    assert _rel(O.quadform(rho, x), x @ x / s2) < 1e-14
    a, v, logdet, kap, E = O.levinson_durbin(rho)
    assert np.array_equal(a, np.eye(n)[0]) and v == s2 and np.all(kap == 0)
    assert np.all(O.gs_generators(a) == 0)
    assert _rel(logdet, n * np.log(s2)) < 1e-14


# ---------------------------------------------------------------- P3 AR(1) closed form
def _ar1_closed(phi, s2, x):
    # C^{-1} is tridiagonal: sigma^2 Q = (1-phi^2) x_0^2 + sum_{t>=1} (x_t - phi x_{t-1})^2
    return ((1 - phi * phi) * x[0] ** 2 + np.sum((x[1:] - phi * x[:-1]) ** 2)) / s2


@pytest.mark.parametrize("phi", [0.5, 0.9, 0.99, -0.7])
def test_p3_ar1_closed_form(phi):
    rng = np.random.default_rng(3)
    n, s2 = 200, 1.7
    rho = s2 * phi ** np.arange(n) / (1 - phi * phi)
    x = rng.standard_normal(n)
    q = _ar1_closed(phi, s2, x)
    assert _rel(O.quadform(rho, x), q) < 1e-12
    a, v, logdet, kap, E = O.levinson_durbin(rho)
    expect_a = np.zeros(n)
    expect_a[0], expect_a[1] = 1.0, -phi
    assert np.max(np.abs(a - expect_a)) < 1e-12
    assert _rel(v, s2) < 1e-12
    b = O.gs_generators(a)
    assert abs(b[-1] + phi) < 1e-12 and np.max(np.abs(b[:-1])) < 1e-12
    assert _rel(O.gs_quadform_timedomain(a, v, x), q) < 1e-12
    # log det of AR(1) covariance: sigma^2n / (1-phi^2)
    assert abs(logdet - (n * np.log(s2) - np.log(1 - phi * phi))) < 1e-10


def test_p3_golden_file():
    """Hand-evaluated AR(1) values (tests/golden/ar1_closed_form.txt)."""
    rows = [l.split() for l in open(os.path.join(GOLD, "ar1_closed_form.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) >= 3
    for r in rows:
        phi, s2 = float(r[0]), float(r[1])
        x = np.array([float(v) for v in r[2].split(",")])
        q = float(r[3])
        rho = s2 * phi ** np.arange(len(x)) / (1 - phi * phi)
        assert _rel(O.quadform(rho, x), q) < 1e-13
        assert _rel(-2 * O.loglike_batch(rho, [len(x)], x, np.zeros((1, len(x))))[0], q) < 1e-13
        assert _rel(O.quadform_bruteforce(rho, x), q) < 1e-12


# ---------------------------------------------------------------- P4 two exact routes
@pytest.mark.parametrize("n", [17, 256, 1024, 4096])
def test_p4_levinson_gs_vs_cholesky(n):
    rng = np.random.default_rng(4)
    rho = _psd_rho(n)
    a, v, logdet = O.levinson_durbin_fast(rho)
    for _ in range(3):
        x = rng.standard_normal(n) * 1e-21
        assert _rel(O.gs_quadform_timedomain(a, v, x), O.quadform(rho, x)) < 1e-12


def test_p4_levinson_loop_equals_vector_form():
    rho = _psd_rho(300)
    a, v, ld, kap, E = O.levinson_durbin(rho)
    a2, v2, ld2 = O.levinson_durbin_fast(rho)
    assert np.max(np.abs(a - a2)) < 1e-13 and _rel(v2, v) < 1e-13 and abs(ld - ld2) < 1e-9


# ---------------------------------------------------------------- P5 generator residual
@pytest.mark.parametrize("n", [64, 1024, 4096])
def test_p5_generator_residual(n):
    rho = _psd_rho(n)
    a, v, _ = O.levinson_durbin_fast(rho)
    # C (a/v) = e_1 with the Toeplitz product done by an independent library routine
    r = sla.matmul_toeplitz(rho, a / v)
    e1 = np.zeros(n)
    e1[0] = 1.0
    assert np.max(np.abs(r - e1)) < 1e-11


# ---------------------------------------------------------------- P6 inverse-Cholesky row
def test_p6_inverse_cholesky_row():
    n = 512
    rho = _psd_rho(n)
    a, v, logdet = O.levinson_durbin_fast(rho)
    L = O.cholesky_lower(rho)
    Linv = sla.solve_triangular(L, np.eye(n), lower=True)
    assert np.max(np.abs(Linv[-1] - a[::-1] / np.sqrt(v))) / np.max(np.abs(Linv[-1])) < 1e-11
    Cinv = np.linalg.inv(O.toeplitz_cov(rho))
    assert _rel(v, 1.0 / Cinv[0, 0]) < 1e-11
    assert abs(logdet - 2 * np.sum(np.log(np.diag(L)))) < 1e-8 * abs(logdet)


# ---------------------------------------------------------------- P7 chi-square invariant
def test_p7_chi_square():
    """x ~ N(0, C)  =>  E[Q] = N, Var[Q] = 2N  (whitened residuals are N(0,1): PAPER.md:140, :420)."""
    fs, n, K = 4096.0, 2048, 64
    M = 2 * n
    rho = W.acf_from_psd(fs, M, n)
    rng = np.random.default_rng(7)
    X = np.stack([W._noise(rng, fs, M, n) for _ in range(K)])
    Q = -2 * O.loglike_batch(rho, [n], np.zeros(n), X)
    assert abs(Q.mean() / n - 1) < 4 * np.sqrt(2.0 / (n * K))
    assert 0.5 < Q.var() / (2 * n) < 1.8


# ---------------------------------------------------------------- P8 invariances
def test_p8_invariances():
    rng = np.random.default_rng(8)
    n = 400
    rho = _psd_rho(n)
    x = rng.standard_normal(n) * 1e-21
    q = O.quadform(rho, x)
    assert q > 0
    assert _rel(O.quadform(3.5 * rho, x), q / 3.5) < 1e-12                  # rho -> c rho
    assert _rel(O.quadform(4.0 * rho, 2.0 * x), q) < 1e-12                  # joint scaling
    assert _rel(O.quadform(rho, x[::-1]), q) < 1e-11                        # time reversal (persymmetry)
    d = rng.standard_normal(n) * 1e-21
    H = np.stack([d, d + x])
    ll = O.loglike_batch(rho, [n], d, H)
    assert ll[0] == 0.0 and ll[1] < 0                                       # h = d  =>  logL = 0 exactly
    a, v, _ = O.levinson_durbin_fast(rho)
    # both GS orderings agree: ||L^T x|| form (upper) and ||L x|| form (lower)
    La, Lb = O.lower_toeplitz(a), O.lower_toeplitz(O.gs_generators(a))
    up = (np.sum((La.T @ x) ** 2) - np.sum((Lb.T @ x) ** 2)) / v
    lo = (np.sum((La @ x) ** 2) - np.sum((Lb @ x) ** 2)) / v
    assert _rel(up, q) < 1e-11 and _rel(lo, q) < 1e-11
    mixed = (np.sum((La.T @ x) ** 2) - np.sum((Lb @ x) ** 2)) / v
    assert _rel(mixed, q) > 1e-6                                            # mixing the two is NOT valid


# ---------------------------------------------------------------- P9 block additivity
def test_p9_block_additivity():
    rng = np.random.default_rng(9)
    lens = [130, 77, 201]
    rho = _psd_rho(max(lens))
    scales = [1.0, 0.8, 2.5]
    acf = np.concatenate([s * rho[:n] for s, n in zip(scales, lens)])
    ntot = sum(lens)
    d = rng.standard_normal(ntot) * 1e-21
    H = rng.standard_normal((5, ntot)) * 1e-21
    total = O.loglike_batch(acf, lens, d, H)
    parts = np.zeros(5)
    off = 0
    for s, n in zip(scales, lens):
        parts += O.loglike_batch(rho[:n], [n], d[off:off + n], H[:, off:off + n]) / s
        off += n
    assert np.max(np.abs(total - parts) / np.abs(parts)) < 1e-12


# ---------------------------------------------------------------- P10 circulant / Whittle limit
def test_p10_circulant_limit_is_eq1():
    """If rho is taken on an M = N grid, C is circulant and Q equals the frequency-domain inner
    product of Eq. 1: Q = (1/N) sum_k |x^_k|^2 / lam_k."""
    fs, n = 1024.0, 256
    f = np.fft.fftfreq(n, 1 / fs)
    lam = 0.5 * fs * W.psd(np.abs(f))
    rho = np.fft.ifft(lam).real                                             # rho_k = rho_{N-k}
    rng = np.random.default_rng(10)
    x = rng.standard_normal(n) * 1e-21
    q_fd = np.sum(np.abs(np.fft.fft(x)) ** 2 / lam) / n
    assert _rel(O.quadform(rho, x), q_fd) < 1e-12


# ---------------------------------------------------------------- P11 bilinear identity / Eq. 13
def test_p11_bilinear_and_snr():
    w = W.make("c1", B=6, n_scale=4)
    ll = O.loglike_batch(w.acf, w.seg_lengths, w.d, w.H)
    dh, hh = O.inner_batch(w.acf, w.seg_lengths, w.d, w.H)
    dd = O.quadform(w.acf, w.d)
    assert np.max(np.abs(-2 * ll - (dd - 2 * dh + hh)) / (dd + hh)) < 1e-12
    # symmetry <x,y> = <y,x>: swap roles of d and h_1
    dh2, _ = O.inner_batch(w.acf, w.seg_lengths, w.H[1], w.d[None, :])
    assert _rel(dh2[0], dh[1]) < 1e-12


def test_p11_inner_batch_sums_over_segments():
    """<x,y> over several segments = sum of the single-segment values, with different
    scales per segment so that `=` instead of `+=` (or a dropped segment) cannot pass; <d,d> against quadform."""
    rng = np.random.default_rng(11)
    lens = [90, 41, 130]
    rho = _psd_rho(max(lens))
    scales = [1.0, 0.6, 2.2]
    acf = np.concatenate([s * rho[:n] for s, n in zip(scales, lens)])
    nt = sum(lens)
    d = rng.standard_normal(nt) * 1e-21
    H = rng.standard_normal((7, nt)) * 1e-21
    dh, hh = O.inner_batch(acf, lens, d, H)
    dh_parts, hh_parts, dd_parts = np.zeros(7), np.zeros(7), 0.0
    off = 0
    for s, n in zip(scales, lens):
        a, b = O.inner_batch(s * rho[:n], [n], d[off:off + n], H[:, off:off + n])
        dh_parts += a
        hh_parts += b
        dd_parts += O.quadform(s * rho[:n], d[off:off + n])
        off += n
    assert np.max(np.abs(dh - dh_parts)) <= 1e-12 * np.max(np.abs(hh_parts))
    assert np.max(np.abs(hh - hh_parts) / hh_parts) < 1e-12
    # every segment contributes: no single partial sum equals the total
    a0, b0 = O.inner_batch(scales[0] * rho[:lens[0]], [lens[0]], d[:lens[0]], H[:, :lens[0]])
    assert np.min(np.abs(hh - b0) / hh) > 0.1
    dd = O.inner_batch(acf, lens, d, d[None, :])[1][0]
    assert _rel(dd, dd_parts) < 1e-12
    # and per row against the brute-force bilinear form x^T C^-1 y = (Q(x+y) - Q(x-y)) / 4 at a small size
    lens2 = [12, 9]
    acf2 = np.concatenate([W.ar_acf([0.5, -0.2], 1.3, 12), 2.0 * W.ar_acf([0.5, -0.2], 1.3, 9)])
    x = rng.standard_normal(21)
    Y = rng.standard_normal((3, 21))
    dh2, hh2 = O.inner_batch(acf2, lens2, x, Y)
    for b in range(3):
        want_dh = want_hh = 0.0
        for lo, hi in ((0, 12), (12, 21)):
            r = acf2[lo:hi]
            want_dh += 0.25 * (O.quadform_bruteforce(r, x[lo:hi] + Y[b, lo:hi]) - O.quadform_bruteforce(r, x[lo:hi] - Y[b, lo:hi]))
            want_hh += O.quadform_bruteforce(r, Y[b, lo:hi])
        assert abs(dh2[b] - want_dh) < 1e-11 * want_hh and _rel(hh2[b], want_hh) < 1e-11


def test_p11_snrs_white_noise_hand_case():
    """Eq. 13 quantities where they have a closed form: white noise of variance s2 gives <x,y> = x.y / s2, so
    rho_mf = d.h / (sigma sqrt(h.h)) and rho_eff^2 = (d.d - (d-h).(d-h)) / s2."""
    rng = np.random.default_rng(13)
    lens, s2 = [50, 30], [2.5e-42, 0.4e-42]
    acf = np.zeros(80)
    acf[0], acf[50] = s2
    d = rng.standard_normal(80) * 1e-21
    H = rng.standard_normal((4, 80)) * 1e-21
    wgt = np.concatenate([np.full(50, 1 / s2[0]), np.full(30, 1 / s2[1])])
    mf, eff2 = O.snrs(acf, lens, d, H)
    want_mf = (H * wgt) @ d / np.sqrt(np.sum(H * H * wgt, axis=1))
    r = d[None, :] - H
    want_eff2 = np.sum(d * d * wgt) - np.sum(r * r * wgt, axis=1)
    assert np.max(np.abs(mf - want_mf) / np.abs(want_mf)) < 1e-12
    assert np.max(np.abs(eff2 - want_eff2)) < 1e-12 * np.sum(d * d * wgt)
    # a template equal to the data: rho_mf = sqrt(<d,d>), rho_eff^2 = <d,d>
    mf1, eff1 = O.snrs(acf, lens, d, d[None, :])
    assert _rel(mf1[0] ** 2, np.sum(d * d * wgt)) < 1e-12 and _rel(eff1[0], np.sum(d * d * wgt)) < 1e-12


def test_p1_p9_large_batch_chunk_loop_and_cached_factors():
    """B = 1500 > the 1024-row chunk of loglike_batch / inner_batch, through the `factors=` branch bench.py times:
    every row against the AR(1) closed form (P3), two segments of different variance (P9)."""
    rng = np.random.default_rng(15)
    phi, lens, s2 = 0.8, [24, 17], [1.7, 0.3]
    acf = np.concatenate([s * phi ** np.arange(n) / (1 - phi * phi) for s, n in zip(s2, lens)])
    nt, B = sum(lens), 1500
    d = rng.standard_normal(nt)
    H = rng.standard_normal((B, nt))
    R = d[None, :] - H
    want = np.zeros(B)
    off = 0
    for s, n in zip(s2, lens):
        x = R[:, off:off + n]
        want += ((1 - phi * phi) * x[:, 0] ** 2 + np.sum((x[:, 1:] - phi * x[:, :-1]) ** 2, axis=1)) / s
        off += n
    fac = O.factorize(acf, lens)
    for kw in ({}, {"factors": fac}, {"chunk": 7}):
        got = O.loglike_batch(acf, lens, d, H, **kw)
        assert np.max(np.abs(-2 * got - want) / want) < 1e-12
    # rows beyond the first chunk are really computed (not left at zero) and differ from one another
    assert np.all(want[1024:] > 0) and len(np.unique(np.round(want[1024:], 9))) == B - 1024
    dh, hh = O.inner_batch(acf, lens, d, H)
    dd = -2 * O.loglike_batch(acf, lens, d, np.zeros((1, nt)))[0]
    assert np.max(np.abs(want - (dd - 2 * dh + hh)) / (dd + hh)) < 1e-12


# ---------------------------------------------------------------- P12 Eq. 14 as printed
@pytest.mark.parametrize("n", [5, 64, 256])
def test_p12_eq14_literal(n):
    rho = _psd_rho(n) * 1e44
    Cinv = np.linalg.inv(O.toeplitz_cov(rho))
    G = O.eq14_inverse_literal(rho)
    assert np.max(np.abs(G - Cinv)) / np.max(np.abs(Cinv)) < 1e-11


# ---------------------------------------------------------------- P13 independent library
def test_p13_solve_toeplitz_route():
    w = W.make("c3", B=4, n_scale=8)
    a = O.loglike_batch(w.acf, w.seg_lengths, w.d, w.H)
    b = O.loglike_batch_solve_toeplitz(w.acf, w.seg_lengths, w.d, w.H)
    assert np.max(np.abs(a - b) / np.maximum(np.abs(a), 1)) < 1e-11


# ---------------------------------------------------------------- P14 injection sanity
@pytest.mark.parametrize("name,scale", [("c1", 1), ("c2", 4), ("c3", 8), ("c5", 8)])
def test_p14_injection(name, scale):
    w = W.make(name, B=3, n_scale=scale)
    ll = O.loglike_batch(w.acf, w.seg_lengths, w.d, w.H)
    n = w.n_tot
    assert abs(ll[0] + n / 2) < 4.5 * np.sqrt(n / 2)      # logL_0 = -1/2 n^T C^-1 n ~ -N/2 +- sqrt(N/2)
    assert ll[0] > ll[1] and ll[0] > ll[2]                # the injected template fits best


# ---------------------------------------------------------------- P15-P18 template families (oracle/templates.py)
def _golden_template_rows():
    fam = {"ringdown": OT.RINGDOWN, "sine_gaussian": OT.SINE_GAUSSIAN, "chirp": OT.CHIRP}
    for line in open(os.path.join(GOLD, "templates.txt")):
        if not line.strip() or line[0] == "#":
            continue
        head, tail = line.split("|")
        f = head.split()
        fs, n = float(f[1]), int(f[2])
        A, p1, p2, phi, p4 = float(f[3]), float(f[4]), float(f[5]), float(f[6]) * np.pi, float(f[7])
        want = {int(kv.split("=")[0]): float(kv.split("=")[1]) for kv in tail.split()}
        yield fam[f[0]], fs, n, (A, p1, p2, phi, p4), want


def test_p15_templates_golden_file():
    """Hand-evaluated samples (tests/golden/templates.txt): onset on and between samples, Gaussian envelope centred
    at t0 with the carrier counted from t = 0, chirp phase and Tukey taper."""
    rows = list(_golden_template_rows())
    assert len(rows) == 4
    for fam, fs, n, p, want in rows:
        H = OT.family_rows(fam, np.array([p]), [n], fs)[0]
        t = np.arange(n) / fs
        direct = {OT.RINGDOWN: OT.ringdown, OT.SINE_GAUSSIAN: OT.sine_gaussian, OT.CHIRP: OT.chirp}[fam](t, *p)
        assert np.array_equal(H, direct)
        for i, v in want.items():
            assert abs(H[i] - v) <= 2e-15 * max(abs(p[0]), 1.0), (fam, i, H[i], v)


@pytest.mark.parametrize("n,alpha", [(9, 0.5), (64, 0.1), (1000, 0.1), (8192, 0.1), (50, 1.0), (31, 0.25)])
def test_p16_tukey_against_scipy(n, alpha):
    import scipy.signal.windows as sw
    assert np.max(np.abs(OT.tukey(n, alpha) - sw.tukey(n, alpha, sym=True))) < 1e-14


def test_p17_projection_fold_identity():
    """F+ h_c + Fx h_s with a time shift is ONE damped sinusoid: A hypot(F+,Fx) cos(theta + phi - atan2(Fx,F+))
    = F+ cos(theta + phi) + Fx sin(theta + phi)  (the row packing of td_loglike_family_batch)."""
    rng = np.random.default_rng(17)
    fs, n = 4096.0, 700
    t = np.arange(n) / fs
    for _ in range(20):
        A, f, tau, phi = rng.uniform(0.5, 2), rng.uniform(100, 400), rng.uniform(2e-3, 2e-2), rng.uniform(0, 2 * np.pi)
        t0, Fp, Fx, dt = rng.uniform(0.02, 0.1), rng.uniform(-1, 1), rng.uniform(-1, 1), rng.uniform(-0.01, 0.01)
        literal = OT.projected_ringdown(t, A, f, tau, phi, t0, Fp, Fx, dt)
        A2, phi2, t02 = OT.fold_projection(A, phi, t0, Fp, Fx, dt)
        folded = OT.ringdown(t, A2, f, tau, phi2, t02)
        assert np.max(np.abs(literal - folded)) <= 1e-14 * A * np.hypot(Fp, Fx) + 1e-300
        assert np.all(literal[t < t0 + dt] == 0.0) and literal[t >= t0 + dt][0] != 0.0
    # the scalar identity itself, at hand-picked angles: F+ = 3, Fx = 4 -> amplitude 5, phase atan2(4, 3)
    for x in (0.0, 0.3, 2.0):
        assert abs(3 * np.cos(x) + 4 * np.sin(x) - 5 * np.cos(x - np.arctan2(4.0, 3.0))) < 1e-14


def test_p17_segment_time_fold():
    """A row written in the time of a segment that starts at ts equals the record-time waveform on that segment's
    samples (gaps: only kept samples exist on the device)."""
    fs, ts, n = 4096.0, 5128 / 4096.0, 300
    t_seg = np.arange(n) / fs
    t_rec = ts + t_seg
    row = (1.3, 180.0, 0.02, 0.7, 1.27)
    A, f, w, phi, t0 = OT.fold_segment_time(OT.SINE_GAUSSIAN, row, ts)
    assert np.max(np.abs(OT.sine_gaussian(t_seg, A, f, w, phi, t0) - OT.sine_gaussian(t_rec, *row))) < 1e-11
    A, f, tau, phi, t0 = OT.fold_segment_time(OT.RINGDOWN, row, ts)
    assert np.max(np.abs(OT.ringdown(t_seg, A, f, tau, phi, t0) - OT.ringdown(t_rec, *row))) < 1e-11


def test_p18_chirp_instantaneous_phase():
    """cos(2 pi (f0 t + fdot t^2/2) + phi): where f0 t + fdot t^2/2 is an integer the sample is +A w, at a half-integer
    -A w, at a quarter 0; f0 = 16, fdot = 32, fs = 64 -> t = 1/4: 4 + 1 = 5; t = 1/8: 2 + 1/4; t = 3/8: 6 + 9/4 = 8.25;
    t = 1/2: 8 + 4 = 12; and with phi = pi the sign flips."""
    fs, n = 64.0, 65
    t = np.arange(n) / fs
    h = OT.chirp(t, 2.0, 16.0, 32.0, 0.0, 1e-9)          # alpha -> 0: the taper touches only the end samples
    assert abs(h[16] - 2.0) < 1e-13 and abs(h[32] - 2.0) < 1e-12
    assert abs(h[8]) < 1e-13 and abs(h[24]) < 1e-12
    hp = OT.chirp(t, 2.0, 16.0, 32.0, np.pi, 1e-9)
    assert abs(hp[16] + 2.0) < 1e-13
    # instantaneous frequency f0 + fdot t: between consecutive samples the phase advances by 2 pi (f0 + fdot (t + dt/2)) dt
    ph = 2 * np.pi * (16.0 * t + 16.0 * t * t)
    assert np.allclose(np.diff(ph), 2 * np.pi * (16.0 + 32.0 * (t[:-1] + 0.5 / fs)) / fs, rtol=1e-13)


@pytest.mark.parametrize("name,B,scale", [("c1", 5, 1), ("c2", 4, 4), ("c3", 4, 4), ("c4", 3, 16), ("c5", 4, 8), ("d2", 6, 1)])
def test_input_generator_rows_equal_oracle_templates(name, B, scale):
    """The rows of H that the shared input generator draws are the oracle's family formulas at the parameters it
    reports (w.params): ties the inputs of every family test to oracle/templates.py, in both directions."""
    w = W.make(name, B=B, n_scale=scale)
    H = OT.family_rows(w.family, w.params, w.seg_lengths, w.fs)
    assert np.max(np.abs(H - w.H)) <= 1e-9 * np.max(np.abs(w.H))


def test_not_spd_is_rejected():
    rho = np.array([1.0, 0.99, 0.2, -0.9])
    with pytest.raises(np.linalg.LinAlgError):
        O.cholesky_lower(rho)
    with pytest.raises(np.linalg.LinAlgError):
        O.levinson_durbin(rho)


# ---------------------------------------------------------------- P19 AR(p) closed form (the long-N oracle route)
@pytest.mark.parametrize("phi", [[0.9], [1.6, -0.8], [0.5, -0.3, 0.1], [1.9, -0.95]])
def test_p19_ar_closed_form_against_cholesky_route(phi):
    """ar_acf / ar_quadform_closed (used at N = 2^20, where nothing else finishes) against the dense Cholesky route,
    the Levinson recursion (a = (1, -phi_1, .., -phi_p, 0, ..), v = s2) and, for p = 1, the hand-derived tridiagonal
    form of P3.  A dropped lag, a wrong sign in the Yule-Walker system or a shifted innovation window fails here."""
    rng = np.random.default_rng(19)
    n, s2 = 300, 0.37
    rho = O.ar_acf(phi, s2, n)
    p = len(phi)
    # Yule-Walker beyond the solved block, and positive definiteness
    for k in (p + 1, p + 5, n - 1):
        assert abs(rho[k] - sum(phi[j] * rho[k - 1 - j] for j in range(p))) < 1e-12 * rho[0]
    x = rng.standard_normal(n)
    q = O.ar_quadform_closed(phi, s2, x)
    assert _rel(O.quadform(rho, x), q) < 1e-9
    a, v, logdet, kap, E = O.levinson_durbin(rho)
    expect = np.zeros(n)
    expect[0] = 1.0
    expect[1 : p + 1] = -np.asarray(phi)
    assert np.max(np.abs(a - expect)) < 1e-8 and _rel(v, s2) < 1e-9
    if p == 1:
        assert _rel(_ar1_closed(phi[0], s2, x), q) < 1e-12
        assert np.max(np.abs(rho - s2 * phi[0] ** np.arange(n) / (1 - phi[0] ** 2))) < 1e-12


# ---------------------------------------------------------------- P20 the paper's GSCE route (Eqs. 14-16) against Cholesky
@pytest.mark.parametrize("name,B,scale", [("c1", 12, 4), ("c3", 6, 8), ("c5", 5, 16)])
def test_p20_gsce_route_equals_cholesky_route(name, B, scale):
    """`loglike_batch_gsce` (Levinson + circulant embedding + numpy FFT: the CPU method the paper advocates, timed by bench.py
    as a context line) against the primary oracle, on single-segment, gapped and multi-detector inputs.  A wrong conjugate,
    a b-generator off by one or an embedding shorter than 2N - 1 fails here."""
    w = W.make(name, B=B, n_scale=scale)
    ref = O.loglike_batch(w.acf, w.seg_lengths, w.d, w.H)
    got = O.loglike_batch_gsce(w.acf, w.seg_lengths, w.d, w.H)
    assert np.max(np.abs(got - ref) / np.maximum(np.abs(ref), 1.0)) < 1e-9
    fac = O.gsce_factors(w.acf, w.seg_lengths)
    assert np.array_equal(O.loglike_batch_gsce(w.acf, w.seg_lengths, w.d, w.H, factors=fac), got)
