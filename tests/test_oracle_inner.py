"""Pins for oracle/inner.py: P3 (linearity, Cauchy-Schwarz), the sinusoid and matched-chirp
end-to-end pins against the exact time-domain product, and structural invariants (CPU only)."""
import copy
import numpy as np
import pytest
from oracle import inner as oin, sft as osft, waveform as owf, kernel as kern
from paper_2502_11823_b200 import workloads as wl
from _util import to_oracle


def _flat_plan(n_sft, n, fs, K, kernel, k_lo, k_hi, **kw):
    return oin.Plan(n_channels=1, n_sft=n_sft, t_sft=n / fs, fs=fs, t0=0.0, k_lo=k_lo, k_hi=k_hi, K=K,
                    kernel=kernel, **kw)


def test_sinusoid_dirichlet_against_time_domain():
    """Noiseless sinusoid, flat PSD, Dirichlet kernel: per SFT ([x,h]) = ([h,h]) =
    (T A^2/S) sum_{|m|<=K} sinc^2(x-m), i.e. the exact <h,h> = (2 dt/S) sum h^2 times the captured
    kernel power (P:238 truncation, Eq.(B1)-(B2) P:447-451)."""
    n, fs, nseg, K = 2048, 256.0, 12, 6
    T, dt, S = n / fs, 1 / fs, 2.0 / fs
    f0, A, phi0 = 40.0 + 0.3 / T, 0.7, 1.1           # offset x = 0.3 bins in every SFT
    t = np.arange(n * nseg) * dt
    h = A * np.cos(phi0 + 2 * np.pi * f0 * t)
    ks = np.arange(300, 345)
    bins = osft.sft_direct(osft.split_segments(h, n), ks, dt)[None]
    plan = _flat_plan(nseg, n, fs, K, "dirichlet", 300, 345)
    store = oin.Store(bins=bins, psd_scale=np.ones((1, nseg)), psd_shape=np.full((1, len(ks)), S))
    ta = oin.sft_times(plan)
    Z, H, k_c, act, _ = oin.band_terms_from_track(plan, store, ta, np.full(nseg, A), phi0 + 2 * np.pi * f0 * ta,
                                                  np.full(nseg, f0), np.zeros(nseg), 1e9, np.ones((1, nseg)))
    assert np.all(k_c == 320) and act.all()
    hh_time = osft.time_domain_product(h, h, dt, S)
    m = np.arange(-K, K + 1)
    captured = np.sum(np.abs(kern.dirichlet(0.3 - m)) ** 2)
    assert abs(np.sum(H) / (hh_time * captured) - 1) < 2e-3
    assert abs(np.sum(Z.real) / (hh_time * captured) - 1) < 2e-3
    assert abs(np.sum(Z.imag)) < 2e-3 * hh_time
    # a phase error of pi/2 in the template kills Re and moves everything to Im (sign pin)
    Z2, _, _, _, _ = oin.band_terms_from_track(plan, store, ta, np.full(nseg, A), phi0 + np.pi / 2 + 2 * np.pi * f0 * ta,
                                               np.full(nseg, f0), np.zeros(nseg), 1e9, np.ones((1, nseg)))
    assert abs(np.sum(Z2.real)) < 2e-3 * hh_time and abs(np.sum(Z2.imag) / (hh_time * captured) - 1) < 2e-3


@pytest.fixture(scope="module")
def chirp_case():
    """Config-1-like noiseless chirp sampled at every t_j (exact h(t)), SFTs by direct DFT."""
    fs, T, nseg = 512.0, 8.0, 24
    n = int(T * fs)
    p = np.array([1.2, 0.25, nseg * T + 216.0, 0.9, 0.5, 0, 0, 0])
    t = np.arange(n * nseg) / fs
    phi, f, _ = owf.taylor_t3(p[0], p[1], p[2], p[3], t, 0)
    h = owf.amplitude(p[4], f, 20.0) * np.cos(phi)
    ks = np.arange(60, 220)
    bins = osft.sft_direct(osft.split_segments(h, n), ks, 1 / fs)[None]
    store = oin.Store(bins=bins, psd_scale=np.ones((1, nseg)), psd_shape=np.full((1, len(ks)), 2 / fs))
    hh_time = osft.time_domain_product(h, h, 1 / fs, 2 / fs)
    return dict(fs=fs, n=n, nseg=nseg, p=p, store=store, hh_time=hh_time, h=h)


def test_matched_chirp_loss_is_small_and_fresnel_beats_dirichlet(chirp_case):
    """Eq.(36): r = 1 - sqrt(([d,h])/<d,h>) with d = h.  b = fdot T^2 reaches ~2 here, so the
    Dirichlet kernel loses tens of percent while the Fresnel kernel with a wide band loses < 1 %
    (the paper's acceptance level)."""
    c = chirp_case
    out = {}
    for kernel, K in (("fresnel", 32), ("fresnel", 4), ("dirichlet", 4)):
        plan = _flat_plan(c["nseg"], c["n"], c["fs"], K, kernel, 60, 220, f_ref=20.0)
        r = oin.inner_products(plan, c["store"], c["p"][None])
        out[(kernel, K)] = (1 - np.sqrt(r["xh"][0] / c["hh_time"]), r["hh"][0] / c["hh_time"])
    assert abs(out[("fresnel", 32)][0]) < 5e-3 and abs(out[("fresnel", 32)][1] - 1) < 1e-2
    assert 0 < out[("fresnel", 4)][0] < 3e-2
    assert out[("dirichlet", 4)][0] > 3 * out[("fresnel", 4)][0]


def test_closed_form_mode_equals_definition_mode(chirp_case):
    c = chirp_case
    res = {}
    for kernel in ("fresnel", "fresnel_quadrature"):
        plan = _flat_plan(c["nseg"], c["n"], c["fs"], 5, kernel, 60, 220, f_ref=20.0)
        res[kernel] = oin.inner_products(plan, c["store"], c["p"][None])
    for key in ("xh", "hh", "xh_im"):
        assert abs(res["fresnel"][key][0] - res["fresnel_quadrature"][key][0]) < 1e-9 * c["hh_time"]
    assert np.array_equal(res["fresnel"]["kc"], res["fresnel_quadrature"]["kc"])


@pytest.fixture(scope="module")
def c1():
    w = wl.config1(n_templates=6)
    plan, store = to_oracle(w)
    return w, plan, store


def test_P3_linearity_and_cauchy_schwarz(c1):
    w, plan, store = c1
    r0 = oin.inner_products(plan, store, w.params)
    # linear in the data
    s2 = copy.copy(store)
    rng = np.random.default_rng(5)
    other = (rng.standard_normal(store.bins.shape) + 1j * rng.standard_normal(store.bins.shape)) * 0.05
    s2.bins = other
    r1 = oin.inner_products(plan, s2, w.params)
    s3 = copy.copy(store)
    s3.bins = 2.0 * store.bins - 3.0 * other
    r2 = oin.inner_products(plan, s3, w.params)
    assert np.allclose(r2["xh"], 2 * r0["xh"] - 3 * r1["xh"], rtol=0, atol=1e-9 * np.abs(r0["xh"]).max())
    assert np.allclose(r2["hh"], r0["hh"], rtol=1e-14)
    # linear / quadratic in the template amplitude
    P = w.params.copy()
    P[:, 4] *= 1.7
    r3 = oin.inner_products(plan, store, P)
    assert np.allclose(r3["xh"], 1.7 * r0["xh"], rtol=1e-12) and np.allclose(r3["hh"], 1.7 ** 2 * r0["hh"], rtol=1e-12)
    # Cauchy-Schwarz on the band
    xx = oin.xx_band(plan, store)
    assert np.all(r0["xh"] ** 2 + r0["xh_im"] ** 2 <= xx * r0["hh"])
    # the injected template (row 0) is recovered: <x,h> ~ <h,h> within noise ~ sqrt(hh)
    assert abs(r0["xh"][0] - r0["hh"][0]) < 5 * np.sqrt(r0["hh"][0])


def test_phase_and_response_plumbing(c1):
    w, plan, store = c1
    r0 = oin.inner_products(plan, store, w.params)
    # phi_c -> phi_c + theta rotates the complex sum: (xh + i xh_im) e^{i theta}
    th = 0.83
    P = w.params.copy()
    P[:, 3] += th
    r1 = oin.inner_products(plan, store, P)
    z0 = (r0["xh"] + 1j * r0["xh_im"]) * np.exp(1j * th)
    assert np.allclose(r1["xh"] + 1j * r1["xh_im"], z0, atol=1e-8 * np.abs(z0).max())
    # a constant table response R = rho e^{i theta} does the same with |R| scalings
    p2 = copy.copy(plan)
    p2.response = "table"
    s2 = copy.copy(store)
    s2.response = np.full((1, plan.n_sft), 1.3 * np.exp(1j * th))
    r2 = oin.inner_products(p2, s2, w.params)
    assert np.allclose(r2["xh"] + 1j * r2["xh_im"], 1.3 * z0, atol=1e-8 * np.abs(z0).max())
    assert np.allclose(r2["hh"], 1.69 * r0["hh"], rtol=1e-12)


def test_psd_weights_and_gaps(c1):
    w, plan, store = c1
    r0 = oin.inner_products(plan, store, w.params)
    s2 = copy.copy(store)
    s2.psd_shape = 2.0 * store.psd_shape
    r1 = oin.inner_products(plan, s2, w.params)
    assert np.allclose(r1["xh"], 0.5 * r0["xh"], rtol=1e-12) and np.allclose(r1["hh"], 0.5 * r0["hh"], rtol=1e-12)
    # removing SFT j (gap) removes exactly that SFT's term
    Z, H, k_c, act, _ = oin.band_terms(plan, store, w.params[1])
    s3 = copy.copy(store)
    s3.psd_scale = store.psd_scale.copy()
    s3.psd_scale[0, [3, 77]] = [0.0, np.nan]
    r3 = oin.inner_products(plan, s3, w.params[1][None])
    assert abs(r3["xh"][0] - (Z.real.sum() - Z.real[0, 3] - Z.real[0, 77])) < 1e-9 * abs(Z.real).sum()
    assert abs(r3["hh"][0] - (H.sum() - H[0, 3] - H[0, 77])) < 1e-12 * H.sum()
    assert r3["kc"][0, 0, 3] == -1 and r3["kc"][0, 0, 77] == -1 and r3["kc"][0, 0, 4] == k_c[4]


def test_bin_selection_and_mask(c1):
    w, plan, store = c1
    t, A, phi, f, fdot = oin.track(plan, w.params[2])
    k_c, x, b, active, flags = oin.select_bins(plan, t, f, fdot, w.params[2][2])
    y = f * plan.t_sft + 0.5 * b                      # Fresnel centre
    assert np.all(np.abs(y[active] - k_c[active]) <= 0.5 + 1e-12)
    assert np.allclose(x[active], f[active] * plan.t_sft - k_c[active])
    assert active.all()                                # variant F: every SFT active
    pm = copy.copy(plan)
    pm.f_lo = 12.0
    k2, _, _, act2, _ = oin.select_bins(pm, t, f, fdot, w.params[2][2])
    assert np.array_equal(act2, f >= 12.0) and 0 < act2.sum() < plan.n_sft and np.all(k2[~act2] == -1)
    pd = copy.copy(plan)
    pd.kernel = "dirichlet"
    k3, _, _, _, _ = oin.select_bins(pd, t, f, fdot, w.params[2][2])
    assert np.all(np.abs(f * plan.t_sft - k3) <= 0.5 + 1e-12)
    # template that coalesces inside the data: SFTs with t_a + T >= t_c are inactive
    P = w.params[2].copy()
    P[2] = 1000.0
    pe = copy.copy(plan)
    pe.f_hi = 1e9
    t, A, phi, f, fdot = oin.track(pe, P)
    _, _, _, act4, _ = oin.select_bins(pe, t, f, fdot, P[2])
    assert np.array_equal(act4, t + plan.t_sft < 1000.0)


def test_time_origin_invariance(c1):
    w, plan, store = c1
    r0 = oin.inner_products(plan, store, w.params[:3])
    p2 = copy.copy(plan)
    p2.t0 = 12345.0
    P = w.params[:3].copy()
    P[:, 2] += 12345.0
    r1 = oin.inner_products(p2, store, P)
    assert np.allclose(r1["xh"], r0["xh"], atol=1e-6 * np.abs(r0["hh"]).max()) and np.array_equal(r1["kc"], r0["kc"])


def test_cumulative(c1):
    w, plan, store = c1
    s2 = copy.copy(store)
    s2.psd_scale = store.psd_scale.copy()
    s2.psd_scale[0, 10:20] = 0.0
    r = oin.inner_products(plan, s2, w.params)
    c = oin.cumulative_snr(plan, s2, w.params)
    assert np.allclose(c["cum_xh"][:, -1], r["xh"], rtol=1e-12, atol=1e-9)
    assert np.allclose(c["cum_hh"][:, -1], r["hh"], rtol=1e-12)
    assert np.all(np.diff(c["cum_hh"], axis=1) >= 0)
    assert np.all(c["cum_hh"][:, 19] == c["cum_hh"][:, 9])          # gaps add nothing
    Z, H, _, _, _ = oin.band_terms(plan, s2, w.params[1])
    assert np.allclose(np.diff(c["cum_xh"][1]), Z.real[0, 1:], atol=1e-9 * np.abs(Z).max())
    assert np.allclose(c["snr"][1], c["cum_xh"][1] / np.sqrt(c["cum_hh"][1]))


def test_harness_fft_matches_oracle_direct_dft(c1):
    """The store's SFTs (numpy rfft in workloads.py, complex64) equal the oracle's direct DFT of the
    same time series (Eq.(26)) to complex64 rounding."""
    w, plan, store = c1
    n = plan.n_samp
    seg = osft.split_segments(w.series[0], n)[[0, 100, 255]]
    ks = np.arange(plan.k_lo, plan.k_hi)
    ref = osft.sft_direct(seg, ks, 1 / plan.fs)
    got = w.bins[0][[0, 100, 255]].astype(np.complex128)
    assert np.abs(got - ref).max() < 2e-7 * np.abs(ref).max()
