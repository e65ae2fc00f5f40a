"""GPU data-SFT generation (sft_compute_sfts / sft_ingest_timeseries) against the
oracle's direct DFT (Eq.(26), explicit summation in fp64).

Tolerance: the kernels work in fp32 (the store is complex64): an n-point fp32 FFT has a relative rms error of
about eps * log2(n) ~ 1e-6, so every bin must agree within 8e-6 of the rms bin magnitude of its SFT
(measured: ~5e-7); the direct-summation fallback accumulates in fp64 and is limited by the fp32 store (6e-8)."""
import numpy as np
import pytest

from oracle import inner as oin
from oracle import sft as osft
from paper_2502_11823_b200 import workloads as wl
from _util import to_oracle

pytestmark = pytest.mark.gpu


def _api():
    from paper_2502_11823_b200 import api
    return api


def _check_bins(g, o, tol):
    rms = np.sqrt(np.mean(np.abs(o) ** 2, axis=1, keepdims=True))
    err = np.abs(g - o) / rms
    assert err.max() <= tol, err.max()
    return float(err.max())


# The last six: the output-pruned narrow-band kernel (<= 256 bins inside [1, n/2]; block length B = 8, 16, 32) with bands that
# start at bin 1, straddle a multiple of 256 (two values of k''), sit high in the spectrum, end at n/2, hold exactly 256
# bins; 257 bins (back to the full transform); more segments than resident blocks (persistent loop).
@pytest.mark.parametrize("n,n_sft,k_lo,k_hi", [(4096, 19, 48, 168), (16384, 5, 7, 219), (64, 33, 0, 33), (1024, 3, 500, 513),
                                               (8192, 7, 1, 257), (16384, 4, 3000, 3200), (16384, 3, 7936, 8192),
                                               (4096, 5, 1900, 2048), (16384, 2, 200, 457), (16384, 450, 5, 187),
                                               (16384, 1, 100, 101), (16384, 889, 255, 258)])
def test_fft_path_matches_direct_dft(n, n_sft, k_lo, k_hi):
    api = _api()
    rng = np.random.default_rng(n + n_sft)
    dt = 1.0 / 512.0
    x = rng.standard_normal(n_sft * n + 17) * 1e-21                 # trailing partial segment: ignored (A13)
    x[: n] += 3e-21 * np.cos(2 * np.pi * (k_lo + 2.3) * np.arange(n) / n)
    bins = np.full((n_sft, k_hi - k_lo), np.nan + 0j, np.complex64)
    api.compute_sfts(np.ascontiguousarray(x[: n_sft * n]), n_sft, n, dt, k_lo, k_hi, bins)
    o = osft.sft_direct(osft.split_segments(x, n), np.arange(k_lo, k_hi), dt)
    _check_bins(bins, o, 8e-6)


def test_direct_path_any_n_and_device_pointers():
    import torch
    api = _api()
    rng = np.random.default_rng(5)
    n, n_sft, k_lo, k_hi, dt = 720, 11, 0, 41, 5.0                  # config 4's segment length
    x = rng.standard_normal(n_sft * n)
    xd = torch.from_numpy(x).cuda()
    bins = torch.zeros((n_sft, k_hi - k_lo), dtype=torch.complex64, device="cuda")
    api.compute_sfts(xd, n_sft, n, dt, k_lo, k_hi, bins)
    o = osft.sft_direct(osft.split_segments(x, n), np.arange(k_lo, k_hi), dt)
    _check_bins(bins.cpu().numpy(), o, 3e-7)
    # a non-power-of-two length above the FFT limit goes the same way
    n2 = 3000
    x2 = rng.standard_normal(2 * n2)
    b2 = np.zeros((2, 9), np.complex64)
    api.compute_sfts(x2, 2, n2, 0.01, 100, 109, b2)
    _check_bins(b2, osft.sft_direct(osft.split_segments(x2, n2), np.arange(100, 109), 0.01), 3e-7)


def test_ingest_timeseries_config1():
    """configs[0] from its 2^20-sample time series: the plan fed by sft_ingest_timeseries gives the oracle's
    inner products (the oracle uses the harness SFTs, which its own direct DFT validates)."""
    api = _api()
    w = wl.config1()
    plan_o, store = to_oracle(w)
    o = oin.inner_products(plan_o, store, w.params)
    xx = oin.xx_band(plan_o, store)
    nT = w.n_templates
    with api.Plan(w.desc) as plan:
        plan.ingest_timeseries(0, np.ascontiguousarray(w.series[0]), np.ascontiguousarray(w.psd_scale[0]),
                               np.ascontiguousarray(w.psd_shape[0]))
        xh, hh, xi = np.empty(nT), np.empty(nT), np.empty(nT)
        kc = np.empty((nT, 1, plan.n_sft), np.int32)
        plan.inner_products(np.ascontiguousarray(w.params), xh, hh, xi, kc)
    norm = np.sqrt(xx * o["hh"])
    assert (np.abs(xh - o["xh"]) / norm).max() <= 1e-4 and (np.abs(hh - o["hh"]) / o["hh"]).max() <= 1e-4
    assert not ((kc != o["kc"]) & ~(o["flags"] != 0)[:, None, :]).any()


def test_psd_scale_estimate_matches_oracle():
    """sft_estimate_psd_scale against the oracle's plain numpy medians: host and device buffers, window 0 and 2, gaps."""
    import torch
    from paper_2502_11823_b200 import api, workloads as wl
    from oracle import sft as osft
    w = wl.et_bns(n_templates=1, n_sft=300, K=8, name="psd")
    bins = np.ascontiguousarray(w.bins[0], np.complex64)
    S = np.ascontiguousarray(w.psd_shape[0])
    n = int(w.desc["t_sft"] * w.desc["fs"])
    for hw in (0, 2):
        o = osft.psd_scale_estimate(bins, S, w.desc["t_sft"], w.desc["k_lo"], n, hw)
        g = api.estimate_psd_scale(bins, w.desc["k_lo"], n, w.desc["t_sft"], S, hw)
        assert np.array_equal(g == 0.0, o == 0.0) and (o == 0.0).sum() == 30
        assert np.allclose(g, o, rtol=2e-6, atol=0.0)
        gd = api.estimate_psd_scale(torch.from_numpy(bins).cuda(), w.desc["k_lo"], n, w.desc["t_sft"], torch.from_numpy(S).cuda(), hw)
        assert np.array_equal(gd.cpu().numpy(), g)
    assert np.allclose(api.estimate_psd_scale(bins, w.desc["k_lo"], n, w.desc["t_sft"], None, 0),
                       osft.psd_scale_estimate(bins, None, w.desc["t_sft"], w.desc["k_lo"], n, 0), rtol=2e-6)
    with pytest.raises(api.SftError):
        api.estimate_psd_scale(bins, w.desc["k_lo"], n, w.desc["t_sft"], S, 40)       # pool too large
    # the estimate is close to the scales the data were made with
    pres = w.psd_scale[0] > 0
    g0 = api.estimate_psd_scale(bins, w.desc["k_lo"], n, w.desc["t_sft"], S, 0)
    assert np.abs(g0[pres] / w.psd_scale[0][pres] - 1.0).mean() < 0.1


def test_append_sfts_streaming_equals_one_shot_load():
    """sft_append_sfts (section V.A): a channel loaded with the first 700 of 1200 SFTs (the rest gaps) and completed in two
    appends gives bit-identical results to the one-shot load, for both calls; before the appends it equals the oracle on the
    truncated data."""
    import copy
    from paper_2502_11823_b200 import api, workloads as wl
    from oracle import inner as oin
    from _util import to_oracle
    w = wl.et_bns(n_templates=96, n_sft=1200, K=8, name="stream")
    N, P = 1200, np.ascontiguousarray(w.params)
    bins = np.ascontiguousarray(w.bins[0], np.complex64)
    scale, shape = np.ascontiguousarray(w.psd_scale[0]), np.ascontiguousarray(w.psd_shape[0])
    def run(plan):
        xh, hh, xi = np.empty(96), np.empty(96), np.empty(96)
        plan.inner_products(P, xh, hh, xi)
        snr = np.empty((96, N), np.float32)
        plan.cumulative_snr(P, snr)
        return xh, hh, xi, snr
    with api.plan_from_workload(w) as plan:
        full = run(plan)
    part_scale = scale.copy()
    part_scale[700:] = 0.0
    part_bins = bins.copy()
    part_bins[700:] = 0.0
    with api.Plan(w.desc) as plan:
        with pytest.raises(api.SftError):
            plan.append_sfts(0, 0, bins[:10], scale[:10])                            # SFT_ENODATA before sft_load_data
        plan.load_data(0, part_bins, part_scale, shape)
        early = run(plan)
        w2 = copy.copy(w)
        w2.bins, w2.psd_scale = part_bins[None], part_scale[None]
        po, so = to_oracle(w2)
        o = oin.inner_products(po, so, P)
        norm = np.sqrt(oin.xx_band(po, so) * o["hh"])
        assert (np.abs(early[0] - o["xh"]) / norm).max() <= 5e-6 and (np.abs(early[1] - o["hh"]) / norm).max() <= 5e-6
        plan.append_sfts(0, 700, np.ascontiguousarray(bins[700:850]), np.ascontiguousarray(scale[700:850]))
        import torch
        plan.append_sfts(0, 850, torch.from_numpy(bins[850:]).cuda(), torch.from_numpy(scale[850:]).cuda())
        plan.sync()
        done = run(plan)
        with pytest.raises(api.SftError):
            plan.append_sfts(0, 1190, np.ascontiguousarray(bins[:20]), np.ascontiguousarray(scale[:20]))   # does not fit
    for a, b in zip(full, done):
        assert np.array_equal(a, b)


def test_ingest_with_estimated_noise_level():
    """sft_ingest_timeseries with psd_scale = NULL: SFTs on the device, per-SFT noise level by the band median, whitening from it.
    Config-1 recipe (white noise of unit variance, S = 2/fs): the estimates scatter around 1 and the matched template's products
    agree with the ones computed with the true noise level to the accuracy of the estimate."""
    from paper_2502_11823_b200 import api, workloads as wl
    w = wl.config1()
    nT = w.n_templates
    P = np.ascontiguousarray(w.params)
    with api.Plan(w.desc) as plan:
        plan.ingest_timeseries(0, np.ascontiguousarray(w.series[0]), None, np.ascontiguousarray(w.psd_shape[0]))
        xh, hh = np.empty(nT), np.empty(nT)
        plan.inner_products(P, xh, hh)
    with api.plan_from_workload(w) as plan:
        xh0, hh0 = np.empty(nT), np.empty(nT)
        plan.inner_products(P, xh0, hh0)
    # (the injected chirp of config 1 is loud - SNR 230 in 120 bins - and lifts the band median by ~6 %)
    assert np.abs(hh / hh0 - 1.0).max() < 0.1 and np.abs(xh[0] / xh0[0] - 1.0) < 0.1
    assert np.abs(hh / hh0 - (hh / hh0).mean()).max() < 1e-3                  # one noise level per SFT: the same factor for every template
