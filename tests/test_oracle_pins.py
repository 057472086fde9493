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
@pytest.mark.parametrize("n", [17, 256, 1024])
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
    mf, eff2 = O.snrs(w.acf, w.seg_lengths, w.d, w.H)
    assert np.allclose(mf, dh / np.sqrt(hh)) and np.allclose(eff2, 2 * dh - hh, rtol=1e-9)


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


def test_not_spd_is_rejected():
    rho = np.array([1.0, 0.99, 0.2, -0.9])
    with pytest.raises(np.linalg.LinAlgError):
        O.cholesky_lower(rho)
    with pytest.raises(np.linalg.LinAlgError):
        O.levinson_durbin(rho)
