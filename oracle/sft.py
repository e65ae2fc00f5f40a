"""Oracle data SFTs by direct DFT and the plain inner products, fp64.  Test infrastructure.

* ``sft_direct``        – Eq.(26): ``x~_a[k] = dt sum_j x_a[j] exp(-i 2 pi tau_j f_k)``,
  ``tau_j = j dt``, ``f_k = k / T_SFT``, by explicit summation (a dense matrix product
  with the exponent table, no FFT).
* ``split_segments``    – P:157: disjoint segments of ``n_SFT = T_SFT/dt`` samples; a trailing
  partial segment is dropped (reading A13).
* ``time_domain_product`` – Eq.(1)/(14) P:20, P:149 for a flat PSD: ``(2 dt/S) sum_j x_j h_j``.
* ``full_band_product`` – Eq.(1) discretised per SFT: ``4 df Re sum_k x~*_k h~_k / S_k`` over
  ``1 <= k <= n/2-1`` (reading A6), optionally with DC and Nyquist at half weight,
  which makes it equal to the time-domain product exactly (Parseval, pin P2).
Pins: tests/test_oracle_sft.py (P1, P2, P4).
"""
import numpy as np


def split_segments(x, n_sft):
    """[N] -> [N_SFT][n_sft]; drops the trailing ``N mod n_sft`` samples (reading A13)."""
    x = np.asarray(x, dtype=np.float64)
    n_seg = x.shape[-1] // n_sft
    return x[..., : n_seg * n_sft].reshape(x.shape[:-1] + (n_seg, n_sft))


def dft_table(n, ks):
    """exp(-2 pi i j k / n), j<n, k in ks; the exponent is reduced with exact integers."""
    j = np.arange(n, dtype=np.int64)[:, None]
    k = np.asarray(ks, dtype=np.int64)[None, :]
    jk = (j * k) % n
    return np.exp(-2j * np.pi * jk.astype(np.float64) / n)


def sft_direct(segments, ks, dt):
    """Eq.(26): [..., n] real segments -> [..., len(ks)] complex SFT bins (units: x * s)."""
    segments = np.asarray(segments, dtype=np.float64)
    n = segments.shape[-1]
    return dt * (segments.astype(np.complex128) @ dft_table(n, ks))


def time_domain_product(x, h, dt, S_flat):
    """(2 dt / S) sum_j x_j h_j: Eq.(1) for a flat one-sided PSD, written in the time domain."""
    return 2.0 * dt / S_flat * float(np.dot(np.asarray(x, np.float64), np.asarray(h, np.float64)))


def full_band_product(xs, hs, S, df, ks, n, half_weight_edges=False):
    """4 df Re sum_k conj(xs_k) hs_k / S_k over bins ``ks`` of an n-sample segment.

    ``half_weight_edges=False`` keeps ``1 <= k <= n/2-1`` (reading A6);
    ``True`` also takes k=0 and k=n/2 at half weight (the exact Parseval partner).
    """
    ks = np.asarray(ks)
    w = np.where((ks >= 1) & (ks <= n // 2 - 1), 1.0, 0.0)
    if half_weight_edges:
        w = np.where((ks == 0) | (ks == n // 2), 0.5, w)
    return 4.0 * df * float(np.sum(w * np.real(np.conj(xs) * hs) / S))


def psd_scale_estimate(bins, psd_shape, t_sft, k_lo, n_samp, half_window=0):
    """Per-SFT noise level from the data ("whitening data on a per-SFT basis"): with ``S_a(f_k) = s_a S(f_k)`` and
    Gaussian noise ``|x~_{a,k}|^2 / (S(f_k) T/2)`` is ``s_a`` times a unit exponential variate, whose median is ln 2, so
    ``s^_a = median{...} / ln 2`` over the valid bins ``1 <= k <= n/2 - 1`` of the SFTs ``|a' - a| <= half_window`` that are not
    gaps (a gap = all bins exactly zero; its own estimate is 0).  Plain numpy.  Pin: tests/test_oracle_sft.py (recovers the
    lognormal scales of the config-2 recipe without bias; scaling law; gaps)."""
    bins = np.asarray(bins)
    n_sft, nb = bins.shape
    S = np.ones(nb) if psd_shape is None else np.asarray(psd_shape, np.float64)
    k = k_lo + np.arange(nb)
    valid = (k >= 1) & (k <= n_samp // 2 - 1)
    v = (bins.real.astype(np.float64) ** 2 + bins.imag.astype(np.float64) ** 2) / (S * 0.5 * t_sft)
    present = np.any(bins != 0, axis=1)
    out = np.zeros(n_sft)
    for a in range(n_sft):
        if not present[a]:
            continue
        rows = [b for b in range(max(0, a - half_window), min(n_sft - 1, a + half_window) + 1) if present[b]]
        pool = v[rows][:, valid].ravel()
        out[a] = np.median(pool) / np.log(2.0) if pool.size else 0.0
    return out
