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


@pytest.mark.parametrize("n,n_sft,k_lo,k_hi", [(4096, 19, 48, 168), (16384, 5, 7, 219), (64, 33, 0, 33), (1024, 3, 500, 513)])
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
