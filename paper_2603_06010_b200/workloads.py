"""Seeded synthetic workloads (inputs only) for the time-domain likelihood hot path.

This module is the ONE piece shared by the CUDA path's tests/bench and the CPU oracle's
tests: it produces inputs (ACF, data, templates) and holds none of the method's arithmetic
(no Toeplitz solve, no Levinson, no Gohberg-Semencul, no quadratic form).  It depends on
numpy only.

The paper's workloads are LIGO strain around GW250114 / GW230814 with Welch PSDs and
NRSur7dq4 templates (PAPER.md:172 Fig. 3, :345, :376-382).  None of that is available, so
BASELINE.json's configs replace it with an analytic PSD and analytic templates of the same
shapes; the recipe is restated in DESIGN.md ("Input recipe") and follows SURVEY.md 8(d)-1.

Recipe (all draws from numpy default_rng(seed), PCG64, in the order written in `make`):
  PSD   S(f) = 1e-46*[x^-4.14 - 5 x^-2 + 111 (1 - x^2 + x^4/2)/(1 + x^2/2)], x = max(f,20)/215
  ACF   grid M = 2*fs*T_total, lam_j = (fs/2) S(j fs/M), rho = irfft(lam, M); segment s uses
        scale_s * rho[0:N_s]  (a principal block of an SPD circulant => SPD Toeplitz)
  noise w ~ N(0, I_M); n = irfft(sqrt(lam) * rfft(w), M)[0:N_s] * sqrt(scale_s)
        (an exact draw from N(0, C), equivalent to the paper's n = L n~)
  amplitude: frequency-domain SNR estimate on the template's own grid,
        SNR_FD^2 = 4 (fs/N) sum_k |rfft(h)_k / fs|^2 / S(f_k); h *= SNR_target / SNR_FD
  data  d = n + h_0   (template 0 is the injection)
"""
from __future__ import annotations

import dataclasses
from typing import List, Optional, Sequence, Tuple

import numpy as np

__all__ = ["Workload", "psd", "acf_from_psd", "make", "CONFIG_NAMES", "ar_acf"]


def psd(f: np.ndarray) -> np.ndarray:
    """One-sided analytic PSD of BASELINE.json's configs, held at its 20 Hz value below 20 Hz."""
    x = np.maximum(np.asarray(f, dtype=np.float64), 20.0) / 215.0
    x2 = x * x
    return 1e-46 * (x ** -4.14 - 5.0 / x2 + 111.0 * (1.0 - x2 + 0.5 * x2 * x2) / (1.0 + 0.5 * x2))


def _eigs(fs: float, M: int) -> np.ndarray:
    f = np.arange(M // 2 + 1, dtype=np.float64) * (fs / M)
    return 0.5 * fs * psd(f)


def acf_from_psd(fs: float, M: int, n: int) -> np.ndarray:
    """rho[0:n] on the M-point circular grid (M even, n <= M/2 + 1 keeps it a principal block)."""
    return np.fft.irfft(_eigs(fs, M), M)[:n].copy()


def _noise(rng: np.random.Generator, fs: float, M: int, n: int) -> np.ndarray:
    w = rng.standard_normal(M)
    return np.fft.irfft(np.sqrt(_eigs(fs, M)) * np.fft.rfft(w), M)[:n].copy()


def _snr_fd(h: np.ndarray, fs: float) -> np.ndarray:
    """FD SNR estimate of each row of h (rows are full un-gapped grids)."""
    n = h.shape[-1]
    hf = np.fft.rfft(h, axis=-1) / fs
    f = np.arange(n // 2 + 1) * (fs / n)
    return np.sqrt(4.0 * (fs / n) * np.sum((hf.real ** 2 + hf.imag ** 2) / psd(f), axis=-1))


def ar_acf(phi: Sequence[float], sigma2: float, n: int) -> np.ndarray:
    """ACF of a stationary AR(p) process x_t = sum_i phi_i x_{t-i} + e_t, Var e = sigma2.

    Input generator for small SPD Toeplitz test cases (Yule-Walker solved by a dense library
    call; no method arithmetic).  Raises if the process is not stationary.
    """
    phi = np.asarray(phi, dtype=np.float64)
    p = len(phi)
    if p == 0:
        r = np.zeros(n)
        r[0] = sigma2
        return r
    comp = np.zeros((p, p))
    comp[0, :] = phi
    comp[1:, :-1] = np.eye(p - 1)
    if np.max(np.abs(np.linalg.eigvals(comp))) >= 1.0:
        raise ValueError("AR process not stationary")
    # unknowns rho_0..rho_p:  rho_k - sum_i phi_i rho_|k-i| = sigma2 * [k == 0]
    A = np.zeros((p + 1, p + 1))
    for k in range(p + 1):
        A[k, k] += 1.0
        for i in range(1, p + 1):
            A[k, abs(k - i)] -= phi[i - 1]
    rhs = np.zeros(p + 1)
    rhs[0] = sigma2
    r0 = np.linalg.solve(A, rhs)
    r = np.zeros(max(n, p + 1))
    r[: p + 1] = r0
    for k in range(p + 1, len(r)):
        r[k] = np.dot(phi, r[k - 1 : k - p - 1 : -1])
    return r[:n].copy()


@dataclasses.dataclass
class Workload:
    name: str
    seed: int
    fs: float
    seg_lengths: np.ndarray      # int64 [n_seg]
    acf: np.ndarray              # float64 [N_tot], per-segment ACFs concatenated
    d: np.ndarray                # float64 [N_tot], kept samples only, segments concatenated
    H: np.ndarray                # float64 [B, N_tot], row b = template b, same packing
    scales: np.ndarray           # float64 [n_seg] PSD scale of each segment
    description: str = ""
    params: Optional[np.ndarray] = None   # float64 [B, 5] or [B, n_seg, 5] = (A, f, tau, phi, t0) per (template, segment)
                                          # where the rows of H come from an analytic family (time counted from each
                                          # segment's start), see FAMILIES
    family: int = 0                       # index into FAMILIES

    @property
    def n_tot(self) -> int:
        return int(self.seg_lengths.sum())

    @property
    def B(self) -> int:
        return int(self.H.shape[0])

    def offsets(self) -> np.ndarray:
        return np.concatenate(([0], np.cumsum(self.seg_lengths)))[:-1]


# analytic template families (rows of 5 parameters), the codes of include/tdlike.h:
#   0 ringdown        (A, f, tau, phi, t0):   A exp(-(t-t0)/tau) cos(2 pi f (t-t0) + phi), t >= t0
#   1 sine-Gaussian   (A, f, w, phi, t0):     A exp(-((t-t0)/w)^2) cos(2 pi f t + phi)
#   2 chirp           (A, f0, fdot, phi, alpha): A tukey_alpha(i/(n-1)) cos(2 pi (f0 t + fdot t^2 / 2) + phi)
FAMILIES = ("ringdown", "sine_gaussian", "chirp")

# name -> (seed, default B)
_SPECS = {
    "c1": (260306011, 64),
    "c2": (260306012, 4096),
    "c3": (260306013, 1024),
    "c4": (260306014, 256),
    "c5": (260306015, 8192),
    "d1": (260306021, (1 << 24) // 64),
    "d2": (260306022, (1 << 24) // 128),
    "d3": (260306023, (1 << 24) // 256),
    "d4": (260306024, (1 << 24) // 512),
    "d5": (260306025, (1 << 24) // 1024),
}
CONFIG_NAMES = tuple(_SPECS)


def _damped(t, f, tau, phi, t0, quadrature=False):
    """exp(-(t-t0)/tau) * cos(2 pi f (t-t0) + phi) for t >= t0 else 0; rows = templates."""
    dt = t[None, :] - t0[:, None]
    on = dt >= 0.0
    dtp = np.where(on, dt, 0.0)
    ph = 2.0 * np.pi * f[:, None] * dtp + phi[:, None]
    osc = np.sin(ph) if quadrature else np.cos(ph)
    return np.where(on, np.exp(-dtp / tau[:, None]) * osc, 0.0)


def _tukey(n: int, alpha: float) -> np.ndarray:
    x = np.arange(n, dtype=np.float64) / (n - 1)
    w = np.ones(n)
    lo = x < alpha / 2
    hi = x > 1 - alpha / 2
    w[lo] = 0.5 * (1 + np.cos(2 * np.pi / alpha * (x[lo] - alpha / 2)))
    w[hi] = 0.5 * (1 + np.cos(2 * np.pi / alpha * (x[hi] - 1 + alpha / 2)))
    return w


def _chunks(B: int, n: int, budget_elems: int = 1 << 25):
    step = max(1, budget_elems // max(n, 1))
    for lo in range(0, B, step):
        yield lo, min(B, lo + step)


def make(name: str, B: Optional[int] = None, n_scale: int = 1) -> Workload:
    """Build config `name` (c1..c5 of BASELINE.json, d1..d5 the dense-regime / crossover extensions).

    B overrides the number of templates (draw vectors then have that length).  n_scale > 1
    divides every length (fs kept, durations shortened) to give reduced-size versions with the
    same structure for tests the oracle must finish in seconds.
    """
    name = name.lower()
    dn = 0
    if name.startswith("d:"):   # "d:<N>": the d-type workload (one ringdown-only segment) at any length N, B = 2^24 / N
        dn = int(name[2:])
        if not 1 <= dn <= 4096:
            raise KeyError(name)
        seed, B0 = 260306100 + dn, max(1, (1 << 24) // dn)
    else:
        seed, B0 = _SPECS[name]
    B = int(B0 if B is None else B)
    rng = np.random.default_rng(seed)
    U = rng.uniform

    if name in ("c1", "c2"):
        fs = 1024.0 if name == "c1" else 4096.0
        N = int(fs) // n_scale
        M = 2 * N
        rho = acf_from_psd(fs, M, N)
        n = _noise(rng, fs, M, N)
        T = N / fs
        f, tau, phi = U(100, 400, B), U(2e-3, 20e-3, B), U(0, 2 * np.pi, B)
        t0, snr = U(0.3, 0.7, B) * T, U(8, 30, B)
        t = np.arange(N) / fs
        H = np.empty((B, N))
        amp = np.empty(B)
        for lo, hi in _chunks(B, N):
            h = _damped(t, f[lo:hi], tau[lo:hi], phi[lo:hi], t0[lo:hi])
            amp[lo:hi] = snr[lo:hi] / _snr_fd(h, fs)
            H[lo:hi] = h * amp[lo:hi, None]
        return Workload(name, seed, fs, np.array([N], np.int64), rho, n + H[0], H, np.ones(1),
                        "single segment, damped sinusoids", np.stack([amp, f, tau, phi, t0], axis=1))

    if name == "c3":
        fs = 4096.0
        Ng = 16384 // n_scale
        gap = 128 // n_scale
        l0, l1 = 5000 // n_scale, 6000 // n_scale
        ranges = [(0, l0), (l0 + gap, l0 + gap + l1), (l0 + 2 * gap + l1, Ng)]
        lens = np.array([b - a for a, b in ranges], np.int64)
        M = 2 * Ng
        scales = U(0.8, 1.2, 3)
        rho = acf_from_psd(fs, M, int(lens.max()))
        acf = np.concatenate([scales[s] * rho[: lens[s]] for s in range(3)])
        noise = np.concatenate([np.sqrt(scales[s]) * _noise(rng, fs, M, int(lens[s])) for s in range(3)])
        T = Ng / fs
        w, f, phi = U(5e-3, 50e-3, B), U(50, 500, B), U(0, 2 * np.pi, B)
        t0, snr = U(0.3, 0.7, B) * T, U(8, 30, B)
        t = np.arange(Ng) / fs
        keep = np.concatenate([np.arange(a, b) for a, b in ranges])
        H = np.empty((B, len(keep)))
        amp = np.empty(B)
        for lo, hi in _chunks(B, Ng):
            h = np.exp(-(((t[None, :] - t0[lo:hi, None]) / w[lo:hi, None]) ** 2)) * np.cos(
                2 * np.pi * f[lo:hi, None] * t[None, :] + phi[lo:hi, None])
            amp[lo:hi] = snr[lo:hi] / _snr_fd(h, fs)
            h *= amp[lo:hi, None]
            H[lo:hi] = h[:, keep]
        # per segment, in the segment's own time (start ts = a / fs): onset t0 - ts, phase phi + 2 pi f ts
        ts = np.array([a for a, _ in ranges]) / fs
        params = np.stack([np.repeat(amp[:, None], 3, 1), np.repeat(f[:, None], 3, 1), np.repeat(w[:, None], 3, 1),
                           phi[:, None] + 2 * np.pi * f[:, None] * ts[None, :], t0[:, None] - ts[None, :]], axis=2)
        return Workload(name, seed, fs, lens, acf, noise + H[0], H, scales,
                        "3 disjoint segments with 128-sample gaps, sine-Gaussians", params, 1)

    if name == "c4":
        fs = 4096.0
        N = 65536 // n_scale
        M = 2 * N
        rho = acf_from_psd(fs, M, N)
        n = _noise(rng, fs, M, N)
        f0, fdot, phi, snr = U(20, 60, B), U(5, 40, B), U(0, 2 * np.pi, B), U(8, 30, B)
        t = np.arange(N) / fs
        win = _tukey(N, 0.1)
        H = np.empty((B, N))
        amp = np.empty(B)
        for lo, hi in _chunks(B, N):
            h = win[None, :] * np.cos(2 * np.pi * (f0[lo:hi, None] * t[None, :]
                                                   + 0.5 * fdot[lo:hi, None] * t[None, :] ** 2) + phi[lo:hi, None])
            amp[lo:hi] = snr[lo:hi] / _snr_fd(h, fs)
            H[lo:hi] = h * amp[lo:hi, None]
        return Workload(name, seed, fs, np.array([N], np.int64), rho, n + H[0], H, np.ones(1),
                        "long single segment, linear chirps with Tukey(0.1) envelope",
                        np.stack([amp, f0, fdot, phi, np.full(B, 0.1)], axis=1), 2)

    if name == "c5":
        fs = 4096.0
        N = 8192 // n_scale
        M = 2 * N
        scales = np.array([1.0, 1.3, 2.0])
        rho = acf_from_psd(fs, M, N)
        acf = np.concatenate([s * rho for s in scales])
        noise = np.concatenate([np.sqrt(s) * _noise(rng, fs, M, N) for s in scales])
        T = N / fs
        f, tau, phi = U(100, 400, B), U(2e-3, 20e-3, B), U(0, 2 * np.pi, B)
        t0, snr = U(0.3, 0.7, B) * T, U(8, 30, B)
        Fp, Fx, dts = U(-1, 1, (B, 3)), U(-1, 1, (B, 3)), U(-10e-3, 10e-3, (B, 3))
        t = np.arange(N) / fs
        H = np.empty((B, 3 * N))
        amp = np.empty(B)
        for lo, hi in _chunks(B, 3 * N):
            net2 = np.zeros(hi - lo)
            for det in range(3):
                ts = t0[lo:hi] + dts[lo:hi, det]
                h = (Fp[lo:hi, det, None] * _damped(t, f[lo:hi], tau[lo:hi], phi[lo:hi], ts)
                     + Fx[lo:hi, det, None] * _damped(t, f[lo:hi], tau[lo:hi], phi[lo:hi], ts, quadrature=True))
                H[lo:hi, det * N:(det + 1) * N] = h
                net2 += _snr_fd(h, fs) ** 2 / scales[det]
            amp[lo:hi] = snr[lo:hi] / np.sqrt(net2)
            H[lo:hi] *= amp[lo:hi, None]
        # per detector the projected template F+ h_c + Fx h_s is again a damped sinusoid:
        # amplitude A hypot(F+, Fx), phase phi - atan2(Fx, F+), onset t0 + dt   ->  params [B, 3, 5]
        params = np.stack([amp[:, None] * np.hypot(Fp, Fx), np.repeat(f[:, None], 3, 1), np.repeat(tau[:, None], 3, 1),
                           phi[:, None] - np.arctan2(Fx, Fp), t0[:, None] + dts], axis=2)
        return Workload(name, seed, fs, np.array([N] * 3, np.int64), acf, noise + H[0], H, scales,
                        "3 detectors x N, projected damped sinusoids, network SNR", params)

    if name in ("d1", "d2", "d3", "d4", "d5") or dn:
        fs = 4096.0
        N = dn if dn else {"d1": 64, "d2": 128, "d3": 256, "d4": 512, "d5": 1024}[name]
        M = 2 * max(4096, 1 << int(np.ceil(np.log2(N))))   # ACF taken from the 1 s grid (longer for N > 4096), truncated (Eq. 11)
        rho = acf_from_psd(fs, M, N)
        n = _noise(rng, fs, M, N)
        f, tau, phi, snr = U(150, 400, B), U(2e-3, 10e-3, B), U(0, 2 * np.pi, B), U(8, 30, B)
        t = np.arange(N) / fs
        H = np.empty((B, N))
        amp = np.empty(B)
        # SNR estimate on a zero-padded 4096 grid so the FD estimate resolves the PSD
        for lo, hi in _chunks(B, 4096):
            h = _damped(t, f[lo:hi], tau[lo:hi], phi[lo:hi], np.zeros(hi - lo))
            hp = np.zeros((hi - lo, 4096))
            hp[:, :N] = h
            amp[lo:hi] = snr[lo:hi] / _snr_fd(hp, fs)
            H[lo:hi] = h * amp[lo:hi, None]
        return Workload(name, seed, fs, np.array([N], np.int64), rho, n + H[0], H, np.ones(1),
                        "ringdown-only short segment (dense-path regime)", np.stack([amp, f, tau, phi, np.zeros(B)], axis=1))

    raise KeyError(name)
