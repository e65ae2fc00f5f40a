"""Pins P1, P2, P4 for oracle/sft.py (CPU only)."""
import numpy as np
from oracle import sft as osft
from oracle import kernel as kern


def _exact_sinusoid_sft(f0, phi, n, dt, ks):
    """dt * DFT of cos(2 pi f0 j dt + phi): geometric sums, exact.
    D(f) = e^{i pi (n-1) dt f} sin(pi n dt f)/sin(pi dt f)."""
    T = n * dt
    fk = np.asarray(ks) / T

    def D(f):
        return np.exp(1j * np.pi * (n - 1) * dt * f) * np.sin(np.pi * n * dt * f) / np.sin(np.pi * dt * f)
    return 0.5 * dt * (np.exp(1j * phi) * D(f0 - fk) + np.exp(-1j * phi) * D(-f0 - fk))


def test_P1_sinusoid_direct_dft_equals_closed_form_and_dirichlet_limit():
    n, fs = 4096, 512.0
    dt, T = 1 / fs, 4096 / 512.0
    f0, phi = 17.3371, 0.77
    ks = np.arange(100, 180)
    x = np.cos(2 * np.pi * f0 * np.arange(n) * dt + phi)
    got = osft.sft_direct(x, ks, dt)
    exact = _exact_sinusoid_sft(f0, phi, n, dt, ks)
    assert np.abs(got - exact).max() < 1e-12 * T
    # against the library FFT as well
    assert np.abs(got - dt * np.fft.rfft(x)[ks]).max() < 1e-12 * T
    # positive-frequency part -> (T/2) e^{i phi} e^{i pi a} sinc(a), a = (f0 - f_k) T, within O(1/n) (Eq.(B2))
    a = (f0 - ks / T) * T
    cont = 0.5 * T * np.exp(1j * phi) * kern.dirichlet(a)
    assert np.abs(got - cont).max() < 3.0 * T / n
    assert np.abs(got - cont).max() > 1e-3 * T / n      # and is not accidentally exact


def test_P1_sign_convention_of_eq26():
    """Eq.(26) has e^{-i 2 pi tau f}: a complex exponential e^{+i 2 pi f_k tau} lands in bin +k."""
    n, dt = 64, 0.25
    j = np.arange(n)
    z = np.cos(2 * np.pi * 5 * j / n)            # real: bins +5 and -5
    out = osft.sft_direct(z, np.arange(0, 33), dt)
    assert abs(out[5] - 0.5 * n * dt) < 1e-12 and np.abs(np.delete(out, 5)).max() < 1e-12
    s = np.sin(2 * np.pi * 5 * j / n)            # sin = (e^{i..} - e^{-i..})/2i -> bin +5 gets -i/2 n dt
    out = osft.sft_direct(s, np.arange(0, 33), dt)
    assert abs(out[5] - (-0.5j) * n * dt) < 1e-12


def test_P2_parseval_time_vs_sft():
    """(2 dt/S) sum_j x_j h_j = 4 df Re sum_k x~* h~ / S with DC and Nyquist at half weight: fixes
    the normalisation (4 df, and a SINGLE df: reading A1)."""
    rng = np.random.default_rng(21)
    n, dt, S = 256, 0.125, 0.37
    x = rng.standard_normal(n)
    h = rng.standard_normal(n)
    ks = np.arange(0, n // 2 + 1)
    xs, hs = osft.sft_direct(x, ks, dt), osft.sft_direct(h, ks, dt)
    lhs = osft.time_domain_product(x, h, dt, S)
    rhs = osft.full_band_product(xs, hs, np.full(ks.shape, S), 1 / (n * dt), ks, n, half_weight_edges=True)
    assert abs(lhs - rhs) < 1e-12 * abs(lhs) + 1e-12
    # a second df (Eq.(35) as printed) would be off by the factor 1/T
    assert abs(rhs / (n * dt) - lhs) > 0.1 * abs(lhs)


def test_P4_sft_folded_equals_full_resolution():
    """8 SFTs x 64 samples, flat PSD: N-point DFT product = time sum = sum over SFTs of per-SFT products (Eq.(20))."""
    rng = np.random.default_rng(22)
    n, nseg, dt, S = 64, 8, 0.5, 1.3
    N = n * nseg
    x = rng.standard_normal(N + 5)                  # trailing partial segment dropped (reading A13)
    h = rng.standard_normal(N + 5)
    xs, hs = osft.split_segments(x, n), osft.split_segments(h, n)
    assert xs.shape == (nseg, n)
    ks = np.arange(0, n // 2 + 1)
    folded = sum(osft.full_band_product(osft.sft_direct(xs[a], ks, dt), osft.sft_direct(hs[a], ks, dt),
                                        np.full(ks.shape, S), 1 / (n * dt), ks, n, True) for a in range(nseg))
    kN = np.arange(0, N // 2 + 1)
    full = osft.full_band_product(osft.sft_direct(x[:N], kN, dt), osft.sft_direct(h[:N], kN, dt),
                                  np.full(kN.shape, S), 1 / (N * dt), kN, N, True)
    tdp = osft.time_domain_product(x[:N], h[:N], dt, S)
    assert abs(folded - tdp) < 1e-11 * abs(tdp) and abs(full - tdp) < 1e-11 * abs(tdp)


def test_psd_scale_estimate_recovers_the_per_sft_noise_level():
    """oracle.sft.psd_scale_estimate ("whitening data on a per-SFT basis") on the config-2 noise recipe (coloured PSD
    shape x lognormal per-SFT scale, 10 % gaps, no signal): unbiased (the median of a unit exponential variate is ln 2) with the
    scatter of a sample median over the band, ~1/sqrt(n_bins); pooling neighbours tightens it; gaps stay gaps; scaling the
    data by c scales the estimate by c^2; a strong narrow line does not move it."""
    from paper_2502_11823_b200 import workloads as wl
    w = wl.et_bns(n_templates=1, n_sft=600, K=8, inject=False, name="noise-only")
    bins, s_true, S = w.bins[0].astype(np.complex128), w.psd_scale[0], w.psd_shape[0]
    n = int(w.desc["t_sft"] * w.desc["fs"])
    est = osft.psd_scale_estimate(bins, S, w.desc["t_sft"], w.desc["k_lo"], n, 0)
    pres = s_true > 0
    assert np.all(est[~pres] == 0.0) and np.all(est[pres] > 0.0)
    ratio = est[pres] / s_true[pres]
    nb = bins.shape[1]
    assert abs(ratio.mean() - 1.0) < 4.0 / np.sqrt(nb * pres.sum())          # unbiased
    assert 0.7 / np.sqrt(nb) < ratio.std() < 1.6 / np.sqrt(nb)                # sample median of Exp(1): sd = 1/(ln 2 sqrt(n)) x ln2... ~1/sqrt(n)
    est2 = osft.psd_scale_estimate(bins, S, w.desc["t_sft"], w.desc["k_lo"], n, 2)
    assert np.all(est2[~pres] == 0.0)
    assert np.allclose(osft.psd_scale_estimate(3.0 * bins, S, w.desc["t_sft"], w.desc["k_lo"], n, 0), 9.0 * est)
    line = bins.copy()
    line[:, 40:43] *= 100.0
    est_line = osft.psd_scale_estimate(line, S, w.desc["t_sft"], w.desc["k_lo"], n, 0)
    assert np.abs(est_line[pres] / est[pres] - 1.0).mean() < 0.06          # 3 of 153 bins boosted x 1e4 in power: a mean would move x 200
    # textbook check of the statistic itself: |CN(0, v)|^2 / v has median ln 2
    z = np.random.default_rng(0).standard_normal((200000, 2)).view(np.complex128)[:, 0] / np.sqrt(2.0)
    assert abs(np.median(np.abs(z) ** 2) - np.log(2.0)) < 0.01
