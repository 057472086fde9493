"""CPU oracle for the time-domain Gaussian log-likelihood hot path (arxiv 2603.06010).

THIS FILE IS TEST INFRASTRUCTURE, NOT PRODUCT.  Only `tests/`, `__graft_entry__.smoke()` and
`bench.py`'s cpu_baseline / `--impl reference` legs may import it.  It shares no code with the
CUDA path (paper_2603_06010_b200/csrc) and imports nothing from the package; the CUDA path
never imports it.  Plain numpy/scipy fp64, no blocking / fusion / reordering beyond what the
cited passage states.

What the hot path computes (PAPER.md:107 Eq. 5, :113 Eq. 6, :125 Eq. 7, :134-142 Eqs. 8-10,
:162 item 3):
    C_s[i][j] = rho_s(|i-j|)                      symmetric Toeplitz covariance of segment s
    <x, y>_s  = x^T C_s^{-1} y                    time-domain inner product
    logL_b    = -1/2 * sum_s <d_s - h_bs, d_s - h_bs>_s     ("const" of Eq. 7 / "+C" of Eq. 10 omitted)
The paper's GSCE method (Eqs. 14-16) reaches exactly this value ("while
maintaining exactness", :254), so the primary oracle is the plain definition evaluated the
way the paper's own whitened representation states it (Cholesky C = L L^T, Eq. 8; whitened
residual r = L^{-1}(d-h) by forward substitution, the "CDL" route :221; lnL = -1/2 r^T r,
Eq. 10).

Readings of garbled/ambiguous passages (full list: DESIGN.md "Readings of the paper"):
  A2  PAPER.md:140 "v-bar = L L^{-1} v" is read as v-bar = L^{-1} v (W = L^{-1}, same sentence).
  A3  PAPER.md:215 "C = L^T L" vs Eq. 8 "C = L L^T": Eq. 8, L lower-triangular.
  A5  PAPER.md:156-160 (Eq. 12) gaps: independent per-segment Toeplitz blocks, logL summed.
  A6  PAPER.md:148-154 (Eq. 11): a segment of N_s samples uses lags 0..N_s-1.

Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): brute-force inverse by Gauss-Jordan
loops at N <= 256 (P1), white noise closed form (P2), AR(1) tridiagonal closed form (P3),
Levinson/Gohberg-Semencul route vs Cholesky route (P4), generator residual (P5), inverse
Cholesky row (P6), chi-square invariant (P7), invariances (P8), block additivity (P9),
circulant/Whittle limit = Eq. 1 (P10), bilinear identity / Eq. 13 (P11: also the sum over
segments of inner_batch against single-segment calls and the brute-force bilinear form, and
snrs against the white-noise closed form), Eq. 14 as printed (P12), independent library
Levinson solve (P13), injection sanity (P14); the chunk loop (B > 1024) and the `factors=`
branch against the AR(1) closed form row by row (test_p1_p9_large_batch_...).
Very long segments (N = 2^20: neither the dense Cholesky nor a library Levinson solve finishes in test time): the exact
Gaussian likelihood of an AR(p) process in closed form (`ar_acf`, `ar_quadform_closed`, O(N p); pin P19 holds it to the
Cholesky route at small N and to the hand-evaluated AR(1) values of P3).
The paper's own fast CPU method (GSCE: Gohberg-Semencul + circulant embedding + FFT) is written out as
`gsce_factors` / `loglike_batch_gsce` and held to the Cholesky route by pin P20; bench.py times it as a second CPU context
line (the O(N log N) route the paper advocates) - it is not what grades the GPU.
Every function below is covered by at least one of them; nothing here is "parity unpinned".
The template families / projection of the step before the hot path live in oracle/templates.py
(pins P15-P18).
"""
from __future__ import annotations

from typing import Optional, Sequence, Tuple

import numpy as np
import scipy.linalg as sla

# ----------------------------------------------------------------------------------------
# Primary route: the definition, via the paper's whitened representation
# ----------------------------------------------------------------------------------------


def toeplitz_cov(rho: np.ndarray) -> np.ndarray:
    """Dense C with C[i][j] = rho(|i-j|)  (Eq. 5)."""
    rho = np.asarray(rho, dtype=np.float64)
    n = len(rho)
    idx = np.abs(np.arange(n)[:, None] - np.arange(n)[None, :])
    return rho[idx]


def cholesky_lower(rho: np.ndarray) -> np.ndarray:
    """L lower-triangular with C = L L^T  (Eq. 8).  Raises LinAlgError if not SPD."""
    return sla.cholesky(toeplitz_cov(rho), lower=True, check_finite=True)


def whiten(L: np.ndarray, X: np.ndarray) -> np.ndarray:
    """x-bar = L^{-1} x by forward substitution, column-wise (PAPER.md:140 reading A2; :221 CDL)."""
    return sla.solve_triangular(L, X, lower=True, check_finite=False)


def _segments(seg_lengths: Sequence[int]):
    off = 0
    for n in seg_lengths:
        n = int(n)
        yield off, off + n
        off += n


def loglike_batch(acf: np.ndarray, seg_lengths: Sequence[int], d: np.ndarray, H: np.ndarray,
                  chunk: int = 1024, factors: Optional[list] = None) -> np.ndarray:
    """out[b] = -1/2 sum_s || L_s^{-1} (d_s - h_bs) ||^2   (Eq. 10; sum over segments :162).

    acf: per-segment ACFs concatenated; d: [N_tot]; H: [B, N_tot] (same packing).
    `factors` may carry precomputed Cholesky factors (one per segment) so that timing can
    separate the one-time factorisation from the per-evaluation cost.
    """
    acf = np.asarray(acf, np.float64)
    d = np.asarray(d, np.float64)
    H = np.asarray(H, np.float64)
    B = H.shape[0]
    out = np.zeros(B)
    for s, (lo, hi) in enumerate(_segments(seg_lengths)):
        L = factors[s] if factors is not None else cholesky_lower(acf[lo:hi])
        for b0 in range(0, B, chunk):
            R = (d[None, lo:hi] - H[b0:b0 + chunk, lo:hi]).T        # residual r = d - h  (:140)
            W = whiten(L, R)                                          # r-bar = L^{-1} r
            out[b0:b0 + chunk] += np.sum(W * W, axis=0)              # r-bar^T r-bar        (Eq. 10)
    return -0.5 * out


def factorize(acf: np.ndarray, seg_lengths: Sequence[int]) -> list:
    """One Cholesky factor per segment (the one-time cost of PAPER.md:215)."""
    acf = np.asarray(acf, np.float64)
    return [cholesky_lower(acf[lo:hi]) for lo, hi in _segments(seg_lengths)]


def inner_batch(acf: np.ndarray, seg_lengths: Sequence[int], d: np.ndarray, H: np.ndarray,
                chunk: int = 1024) -> Tuple[np.ndarray, np.ndarray]:
    """(<d,h_b>, <h_b,h_b>) summed over segments: <x,y> = x-bar^T y-bar (Eq. 9; Eq. 13 terms)."""
    acf = np.asarray(acf, np.float64)
    d = np.asarray(d, np.float64)
    H = np.asarray(H, np.float64)
    B = H.shape[0]
    dh = np.zeros(B)
    hh = np.zeros(B)
    for lo, hi in _segments(seg_lengths):
        L = cholesky_lower(acf[lo:hi])
        dbar = whiten(L, d[lo:hi])
        for b0 in range(0, B, chunk):
            Hbar = whiten(L, H[b0:b0 + chunk, lo:hi].T)
            dh[b0:b0 + chunk] += dbar @ Hbar
            hh[b0:b0 + chunk] += np.sum(Hbar * Hbar, axis=0)
    return dh, hh


def quadform(rho: np.ndarray, x: np.ndarray) -> float:
    """x^T C^{-1} x for one segment via Eqs. 8-10."""
    w = whiten(cholesky_lower(rho), np.asarray(x, np.float64))
    return float(w @ w)


def snrs(acf, seg_lengths, d, H):
    """Matched-filter SNR rho_mf = <d,h>/sqrt(<h,h>) and effective SNR^2 = <d,d> - <r,r>, r = d - h
    (item 7, Eq. 13)."""
    dh, hh = inner_batch(acf, seg_lengths, d, H)
    dd = -2.0 * loglike_batch(acf, seg_lengths, d, np.zeros((1, len(d))))[0]
    rr = -2.0 * loglike_batch(acf, seg_lengths, d, H)
    return dh / np.sqrt(hh), dd - rr


# ----------------------------------------------------------------------------------------
# Brute force (pure loops, N <= 256): explicit inverse by Gauss-Jordan with partial pivoting
# ----------------------------------------------------------------------------------------


def quadform_bruteforce(rho: Sequence[float], x: Sequence[float]) -> float:
    """x^T C^{-1} x with C^{-1} formed explicitly by Gauss-Jordan elimination in Python loops
    (Eq. 6 read literally).  O(N^3) interpreted loops: keep N <= 256."""
    n = len(rho)
    A = [[float(rho[abs(i - j)]) for j in range(n)] + [1.0 if j == i else 0.0 for j in range(n)]
         for i in range(n)]
    for c in range(n):
        p = max(range(c, n), key=lambda r: abs(A[r][c]))
        if A[p][c] == 0.0:
            raise ZeroDivisionError("singular")
        A[c], A[p] = A[p], A[c]
        piv = A[c][c]
        rowc = [v / piv for v in A[c]]
        A[c] = rowc
        for r in range(n):
            if r != c:
                f = A[r][c]
                if f != 0.0:
                    rr = A[r]
                    A[r] = [rr[k] - f * rowc[k] for k in range(2 * n)]
    q = 0.0
    for i in range(n):
        row = A[i]
        acc = 0.0
        for j in range(n):
            acc += row[n + j] * float(x[j])
        q += float(x[i]) * acc
    return q


# ----------------------------------------------------------------------------------------
# Second, independent exact route: Levinson-Durbin + Gohberg-Semencul in the TIME domain
# (used to cross-check the Cholesky route; it is not what grades the GPU)
# ----------------------------------------------------------------------------------------


def levinson_durbin(rho: np.ndarray):
    """Durbin's recursion for the order-(N-1) prediction-error filter (PAPER.md:176 refs [104,105],
    :215 "O(N^2)", :239 ref [123]; the paper cites but does not print it - DESIGN.md reading R-LD).

        E_0 = rho_0; a^(0) = [1]
        kappa_k = -( sum_{j<k} a^(k-1)_j rho_{k-j} ) / E_{k-1}
        a^(k)_j = a^(k-1)_j + kappa_k a^(k-1)_{k-j}  (0<j<k);  a^(k)_0 = 1;  a^(k)_k = kappa_k
        E_k = E_{k-1} (1 - kappa_k^2)
    Returns a = a^(N-1), v = E_{N-1}, logdet = sum_k log E_k, kappa[1..N-1], E[0..N-1].
    C a = v e_1, i.e. x = C^{-1} e_1 = a / v and x_1 = 1/v in the notation of Eq. 14.
    """
    rho = np.asarray(rho, np.float64)
    n = len(rho)
    if not (rho[0] > 0.0) or not np.all(np.isfinite(rho)):
        raise np.linalg.LinAlgError("rho_0 must be positive and finite")
    a = np.zeros(n)
    a[0] = 1.0
    E = np.empty(n)
    E[0] = rho[0]
    kap = np.zeros(n)
    for k in range(1, n):
        acc = 0.0
        for j in range(k):
            acc += a[j] * rho[k - j]
        kk = -acc / E[k - 1]
        new = a.copy()
        for j in range(1, k):
            new[j] = a[j] + kk * a[k - j]
        new[k] = kk
        a = new
        E[k] = E[k - 1] * (1.0 - kk * kk)
        kap[k] = kk
        if not (E[k] > 0.0):
            raise np.linalg.LinAlgError("not positive definite at order %d" % k)
    return a, float(E[n - 1]), float(np.sum(np.log(E))), kap, E


def levinson_durbin_fast(rho: np.ndarray):
    """Same recursion as `levinson_durbin` with the two inner loops written as numpy vector
    operations (for N up to 65536).  Checked against the loop version in the pins."""
    rho = np.asarray(rho, np.float64)
    n = len(rho)
    if not (rho[0] > 0.0) or not np.all(np.isfinite(rho)):
        raise np.linalg.LinAlgError("rho_0 must be positive and finite")
    a = np.zeros(n)
    a[0] = 1.0
    E = rho[0]
    logdet = np.log(E)
    for k in range(1, n):
        kk = -np.dot(a[:k], rho[k:0:-1]) / E
        a[1:k] = a[1:k] + kk * a[k - 1:0:-1]
        a[k] = kk
        E = E * (1.0 - kk * kk)
        if not (E > 0.0):
            raise np.linalg.LinAlgError("not positive definite at order %d" % k)
        logdet += np.log(E)
    return a, float(E), float(logdet)


def gs_generators(a: np.ndarray):
    """b = (0, a_{N-1}, ..., a_1): first column of L(b), so that L(b)^T = v R_x of Eq. 14
    (R_x strictly upper-triangular Toeplitz with first row (0, x_n, ..., x_2))."""
    b = np.zeros_like(a)
    b[1:] = a[:0:-1]
    return b


def lower_toeplitz(c: np.ndarray) -> np.ndarray:
    """L(c): lower-triangular Toeplitz with first column c."""
    n = len(c)
    i = np.arange(n)[:, None] - np.arange(n)[None, :]
    return np.where(i >= 0, np.asarray(c)[np.clip(i, 0, n - 1)], 0.0)


def gs_quadform_timedomain(a: np.ndarray, v: float, x: np.ndarray) -> float:
    """x^T C^{-1} x = ( ||L(a)^T x||^2 - ||L(b)^T x||^2 ) / v  (Eq. 14 with x = a/v, x_1 = 1/v),
    with the two triangular Toeplitz products written as explicit O(N^2) sums (no FFT)."""
    x = np.asarray(x, np.float64)
    n = len(x)
    b = gs_generators(a)
    y1 = np.empty(n)
    y2 = np.empty(n)
    for i in range(n):
        y1[i] = np.dot(a[: n - i], x[i:])      # (L(a)^T x)_i = sum_{j>=i} a_{j-i} x_j
        y2[i] = np.dot(b[: n - i], x[i:])      # (L(b)^T x)_i = sum_{j>=i} b_{j-i} x_j, b_0 = 0
    return float((y1 @ y1 - y2 @ y2) / v)


def eq14_inverse_literal(rho: np.ndarray) -> np.ndarray:
    """C^{-1} built literally from Eq. 14 as printed:
    solve C x = e_1 (dense library solve), L_x lower-triangular Toeplitz with first column x,
    R_x strictly upper-triangular Toeplitz with first row (0, x_n, ..., x_2);
    C^{-1} = (L_x L_x^T - R_x^T R_x) / x_1."""
    rho = np.asarray(rho, np.float64)
    n = len(rho)
    e1 = np.zeros(n)
    e1[0] = 1.0
    x = np.linalg.solve(toeplitz_cov(rho), e1)
    Lx = lower_toeplitz(x)
    first_row = np.zeros(n)
    first_row[1:] = x[:0:-1]
    Rx = lower_toeplitz(first_row).T
    return (Lx @ Lx.T - Rx.T @ Rx) / x[0]


# ----------------------------------------------------------------------------------------
# Large-N route (N = 65536: dense C would be 32 GiB): independent library Levinson solve
# ----------------------------------------------------------------------------------------


def loglike_batch_solve_toeplitz(acf, seg_lengths, d, H) -> np.ndarray:
    """Same quantity as `loglike_batch`, with z = C^{-1} r from scipy.linalg.solve_toeplitz (a
    separate Levinson implementation in compiled code) and Q = r . z  (Eq. 6 read literally).
    Used where the dense Cholesky does not fit (config c4); pinned to `loglike_batch` in P13."""
    acf = np.asarray(acf, np.float64)
    d = np.asarray(d, np.float64)
    H = np.asarray(H, np.float64)
    out = np.zeros(H.shape[0])
    for lo, hi in _segments(seg_lengths):
        R = (d[None, lo:hi] - H[:, lo:hi]).T
        Z = sla.solve_toeplitz(acf[lo:hi], R, check_finite=False)
        out += np.sum(R * Z, axis=0)
    return -0.5 * out


# ----------------------------------------------------------------------------------------
# Closed form for very long segments: exact likelihood of a stationary AR(p) process
# ----------------------------------------------------------------------------------------
# For x_t = sum_{j=1..p} phi_j x_{t-j} + e_t, e_t ~ N(0, s2) iid, stationary, the joint density factorises as
# p(x_0..x_{p-1}) * prod_{t>=p} p(x_t | x_{t-1}..x_{t-p}), hence (the textbook exact AR likelihood; it is Eq. 10 of the
# paper, for a covariance whose Cholesky factor is known in closed form: the rows t >= p of L^{-1} are
# (.., -phi_p, .., -phi_1, 1)/sqrt(s2))
#     x^T C^{-1} x = x_{0:p}^T C_p^{-1} x_{0:p} + (1/s2) sum_{t>=p} (x_t - sum_j phi_j x_{t-j})^2 ,
# with C_p the p x p Toeplitz matrix of the first p autocovariances.  O(N p) work: the one oracle route that reaches
# N = 2^20 ("N >~ 1e7" is the paper's long-N regime).


def ar_acf(phi: Sequence[float], s2: float, n: int) -> np.ndarray:
    """Autocovariances rho_0..rho_{n-1} of the stationary AR(p) process above: rho_0..rho_p from the Yule-Walker
    equations rho_k = sum_j phi_j rho_|k-j| + s2 [k = 0] (a (p+1) x (p+1) linear solve), the rest by the recursion."""
    phi = np.asarray(phi, np.float64)
    p = phi.size
    A = np.zeros((p + 1, p + 1))
    for k in range(p + 1):
        A[k, k] += 1.0
        for j in range(1, p + 1):
            A[k, abs(k - j)] -= phi[j - 1]
    rhs = np.zeros(p + 1)
    rhs[0] = s2
    rho = np.zeros(max(n, p + 1))
    rho[: p + 1] = np.linalg.solve(A, rhs)
    for k in range(p + 1, n):
        rho[k] = np.dot(phi, rho[k - 1 : k - p - 1 : -1])
    return rho[:n].copy()


def ar_quadform_closed(phi: Sequence[float], s2: float, x: np.ndarray) -> float:
    """x^T C^{-1} x for the AR(p) covariance, by the factorisation above (no N x N object, no recursion over lags)."""
    phi = np.asarray(phi, np.float64)
    x = np.asarray(x, np.float64)
    p = phi.size
    head = quadform(ar_acf(phi, s2, p), x[:p]) if p > 0 else 0.0
    e = x[p:].copy()
    for j in range(1, p + 1):
        e -= phi[j - 1] * x[p - j : x.size - j]
    return float(head + np.dot(e, e) / s2)


# ----------------------------------------------------------------------------------------
# The paper's fast CPU route: GSCE = Gohberg-Semencul + circulant embedding + FFT
# ----------------------------------------------------------------------------------------
# Eq. 14: C^{-1} = (1/x_1)(L_x L_x^T - R_x^T R_x), C x = e_1.  With x = a / v (Levinson), x_1 = 1/v:
#     r^T C^{-1} r = ( ||L(a)^T r||^2 - ||L(b)^T r||^2 ) / v ,   b = (0, a_{N-1}, .., a_1).
# Eqs. 15-16: a triangular Toeplitz product is a slice of a circulant product of size m >= 2N - 1, and a
# circulant product is diagonal in the Fourier basis: (L(c)^T r)_i = sum_{j>=i} c_{j-i} r_j is the correlation of r with c,
# irfft( conj(rfft(c, m)) * rfft(r, m) )[:N].  numpy's FFT, written exactly in that order; the generator transforms are the
# once-per-segment "cached" part, the per-template work is one forward and two inverse real FFTs.


def gsce_factors(acf: np.ndarray, seg_lengths: Sequence[int]) -> list:
    """Per segment: (N, m, conj(rfft(a, m)), conj(rfft(b, m)), v) from the Levinson recursion (`levinson_durbin_fast`)."""
    acf = np.asarray(acf, np.float64)
    out = []
    for lo, hi in _segments(seg_lengths):
        n = hi - lo
        a, v, _ = levinson_durbin_fast(acf[lo:hi])
        b = gs_generators(a)
        m = 2 * n   # any m >= 2n - 1 is exact
        out.append((n, m, np.conj(np.fft.rfft(a, m)), np.conj(np.fft.rfft(b, m)), v))
    return out


def loglike_batch_gsce(acf: np.ndarray, seg_lengths: Sequence[int], d: np.ndarray, H: np.ndarray,
                       factors: Optional[list] = None) -> np.ndarray:
    """Same quantity as `loglike_batch` by the paper's GSCE route (Eqs. 14-16), batched over the rows of H."""
    d = np.asarray(d, np.float64)
    H = np.asarray(H, np.float64)
    if factors is None:
        factors = gsce_factors(acf, seg_lengths)
    out = np.zeros(H.shape[0])
    for (lo, hi), (n, m, Ac, Bc, v) in zip(_segments(seg_lengths), factors):
        R = np.fft.rfft(d[None, lo:hi] - H[:, lo:hi], m, axis=1)
        y1 = np.fft.irfft(Ac[None, :] * R, m, axis=1)[:, :n]
        y2 = np.fft.irfft(Bc[None, :] * R, m, axis=1)[:, :n]
        out += (np.einsum("ij,ij->i", y1, y1) - np.einsum("ij,ij->i", y2, y2)) / v
    return -0.5 * out
