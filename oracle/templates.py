"""CPU oracle for the step immediately before the hot path: template generation, detector
projection and placement in the data vector (PAPER.md:164 item 5 "waveform conditioning";
:209-211 section III.A.1 "data projection and conditioning": h_+ f_+ + h_x f_x, then "placing
the projected waveform at the appropriate position in the data vector").

THIS FILE IS TEST INFRASTRUCTURE, NOT PRODUCT (same rules as td_oracle.py): only `tests/`,
`__graft_entry__.smoke()` and bench.py's cpu_baseline / `--impl reference` legs may import it;
it imports nothing from the package and shares no code with csrc/td_synth.cuh.

The paper takes its polarisations from waveform libraries (PyCBC / lalsimulation, :163) that are
not available; BASELINE.json's configs replace them by three analytic families, which are what
the CUDA library synthesises on the device (include/tdlike.h `td_family`).  Each function below is
the family's defining formula evaluated sample by sample in plain numpy fp64, with no recurrence,
no folding of parameters and no reuse of intermediate phases:

  ringdown       h_i = A exp(-(t_i - t0)/tau) cos(2 pi f (t_i - t0) + phi)   for t_i >= t0, else 0
  sine-Gaussian  h_i = A exp(-((t_i - t0)/w)^2) cos(2 pi f t_i + phi)
  chirp          h_i = A tukey_alpha(i/(n-1)) cos(2 pi (f0 t_i + fdot t_i^2/2) + phi)
  projection     h_det = F+ h_c(t - dt) + Fx h_s(t - dt)

Pins (tests/test_oracle_pins.py, `-m "not gpu"`): Tukey window against scipy.signal.windows.tukey;
hand-evaluated rows in tests/golden/templates.txt (arithmetic written beside them); the
projection fold identity; the chirp's instantaneous phase at hand-picked samples.
"""
from __future__ import annotations

from typing import Sequence

import numpy as np

RINGDOWN, SINE_GAUSSIAN, CHIRP = 0, 1, 2   # the codes of include/tdlike.h td_family


def ringdown(t: np.ndarray, A: float, f: float, tau: float, phi: float, t0: float,
             quadrature: bool = False) -> np.ndarray:
    """A exp(-(t-t0)/tau) cos(2 pi f (t-t0) + phi) for t >= t0, zero before the onset
    (the "adding zeroes to the ends of the template").  quadrature=True gives the
    sine quadrature h_s (phase advanced by -pi/2: cos(x - pi/2) = sin x)."""
    t = np.asarray(t, np.float64)
    out = np.zeros_like(t)
    on = (t - t0) >= 0.0                       # samples at or after the onset
    dt = t[on] - t0
    arg = 2.0 * np.pi * f * dt + phi
    out[on] = A * np.exp(-dt / tau) * (np.sin(arg) if quadrature else np.cos(arg))
    return out


def sine_gaussian(t: np.ndarray, A: float, f: float, w: float, phi: float, t0: float) -> np.ndarray:
    """A exp(-((t-t0)/w)^2) cos(2 pi f t + phi)   (BASELINE.json config 3)."""
    t = np.asarray(t, np.float64)
    u = (t - t0) / w
    return A * np.exp(-(u * u)) * np.cos(2.0 * np.pi * f * t + phi)


def tukey(n: int, alpha: float) -> np.ndarray:
    """Tukey (tapered-cosine) window on n samples, x_i = i/(n-1):
    w = 1/2 (1 + cos(2 pi/alpha (x - alpha/2)))        for x < alpha/2,
    w = 1                                               for alpha/2 <= x <= 1 - alpha/2,
    w = 1/2 (1 + cos(2 pi/alpha (x - 1 + alpha/2)))    for x > 1 - alpha/2."""
    out = np.ones(n)
    den = float(n - 1) if n > 1 else 1.0
    for i in range(n):
        x = i / den
        if x < 0.5 * alpha:
            out[i] = 0.5 * (1.0 + np.cos(2.0 * np.pi / alpha * (x - 0.5 * alpha)))
        elif x > 1.0 - 0.5 * alpha:
            out[i] = 0.5 * (1.0 + np.cos(2.0 * np.pi / alpha * (x - 1.0 + 0.5 * alpha)))
    return out


def chirp(t: np.ndarray, A: float, f0: float, fdot: float, phi: float, alpha: float) -> np.ndarray:
    """A tukey_alpha(i/(n-1)) cos(2 pi (f0 t + fdot t^2/2) + phi)   (BASELINE.json config 4):
    instantaneous frequency f0 + fdot t."""
    t = np.asarray(t, np.float64)
    return A * tukey(len(t), alpha) * np.cos(2.0 * np.pi * (f0 * t + 0.5 * fdot * t * t) + phi)


def project(Fp: float, Fx: float, h_c: np.ndarray, h_s: np.ndarray) -> np.ndarray:
    """Detector response h_+ f_+ + h_x f_x."""
    return Fp * np.asarray(h_c, np.float64) + Fx * np.asarray(h_s, np.float64)


def projected_ringdown(t: np.ndarray, A: float, f: float, tau: float, phi: float, t0: float,
                       Fp: float, Fx: float, dt: float) -> np.ndarray:
    """F+ h_c(t - dt) + Fx h_s(t - dt) for the damped sinusoid with quadratures h_c (cos) and h_s (sin)
    (BASELINE.json config 5; projection PAPER.md:209, placement at the shifted arrival time :211).
    Written as the literal two-term sum: no amplitude/phase fold."""
    return project(Fp, Fx, ringdown(t, A, f, tau, phi, t0 + dt), ringdown(t, A, f, tau, phi, t0 + dt, quadrature=True))


def fold_projection(A: float, phi: float, t0: float, Fp: float, Fx: float, dt: float):
    """Parameters (A', phi', t0') of the single ringdown row that equals `projected_ringdown`:
    F+ cos x + Fx sin x = hypot(F+, Fx) cos(x - atan2(Fx, F+)), so
    A' = A hypot(F+, Fx), phi' = phi - atan2(Fx, F+), t0' = t0 + dt.
    (This is how a caller packs one row per (template, detector) for td_loglike_family_batch;
    pinned against the literal sum in test_templates_projection_fold.)"""
    return A * np.hypot(Fp, Fx), phi - np.arctan2(Fx, Fp), t0 + dt


def fold_segment_time(family: int, row: Sequence[float], ts: float):
    """Parameters of a row in the time of a segment that starts at ts of a longer record (gaps: the
    kept samples of segment s have t = ts + i/fs): onset t0 - ts for the ringdown
    and the sine-Gaussian, and the sine-Gaussian's carrier phase advances by 2 pi f ts."""
    A, p1, p2, phi, p4 = [float(v) for v in row]
    if family == RINGDOWN:
        return A, p1, p2, phi, p4 - ts
    if family == SINE_GAUSSIAN:
        return A, p1, p2, phi + 2.0 * np.pi * p1 * ts, p4 - ts
    raise ValueError("the chirp's Tukey window is defined over the segment itself")


def family_rows(family: int, params: np.ndarray, seg_lengths: Sequence[int], fs: float) -> np.ndarray:
    """H [B, N_tot] from rows of 5 parameters [B, n_seg, 5] (or [B, 5] for one segment), each row in its
    segment's own time t_i = i/fs: what td_loglike_family_batch must synthesise (include/tdlike.h)."""
    params = np.asarray(params, np.float64)
    n_seg = len(seg_lengths)
    if params.ndim == 2:
        params = params[:, None, :]
    assert params.shape[1] == n_seg and params.shape[2] == 5
    B = params.shape[0]
    H = np.zeros((B, int(np.sum(seg_lengths))))
    off = 0
    for s, n in enumerate(seg_lengths):
        n = int(n)
        t = np.arange(n, dtype=np.float64) / fs
        for b in range(B):
            A, p1, p2, phi, p4 = params[b, s]
            if family == RINGDOWN:
                H[b, off:off + n] = ringdown(t, A, p1, p2, phi, p4)
            elif family == SINE_GAUSSIAN:
                H[b, off:off + n] = sine_gaussian(t, A, p1, p2, phi, p4)
            elif family == CHIRP:
                H[b, off:off + n] = chirp(t, A, p1, p2, phi, p4)
            else:
                raise ValueError("unknown family")
        off += n
    return H
