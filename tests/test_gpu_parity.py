"""GPU parity: the CUDA path (through the C ABI) against the fp64 CPU oracle, element by element,
on the same seeded inputs.  Tolerances (BASELINE.json north_star):

* ``|d<x,h>|`` and ``|d<h,h>|`` <= 1e-4 * sqrt(<x,x> <h,h>), with ``<x,x>`` restricted to the stored
  band (stricter than the full-band normaliser the north star names, reading A14);
* stricter, also enforced here: ``|d<h,h>| <= 1e-4 <h,h>`` and ``|d<x,h>| <= 1e-4 sqrt(<x,x>_band <h,h>)``
  per template with the *band of that template* implied by the kernel - see ``_check``;
* selected central bins ``k_c`` bit-exact except pairs the oracle flags as ties (reading A5/A12),
  where either neighbour / either mask decision is accepted.
"""
import numpy as np
import pytest

from oracle import inner as oin
from paper_2502_11823_b200 import workloads as wl
from _util import to_oracle

pytestmark = pytest.mark.gpu

TOL = 1e-4
# Regression bar beside the binding one: the fp32 evaluators are built for ~2e-6 per bin and the
# measured normalised error is 5e-8 ... 5e-7, so a 10x loss of accuracy must not pass unseen.
REG = 5e-6


def _api():
    from paper_2502_11823_b200 import api
    return api


def _run_gpu(w, params=None, want_kc=True, **override):
    """Runs the library twice: with the k_c output (run-time-flag kernel variant, which also fills the
    evaluator-path counters) and without it (the compile-time-flag variant the benchmarks time, where
    the plan has one).  Returns the k_c run; the other one is returned under "hot"."""
    api = _api()
    P = np.ascontiguousarray(w.params if params is None else params, dtype=np.float64)
    nT = P.shape[0]
    with api.plan_from_workload(w, **override) as plan:
        xh, hh, xi = np.full(nT, np.nan), np.full(nT, np.nan), np.full(nT, np.nan)
        kc = np.full((nT, plan.n_channels, plan.n_sft), -7, dtype=np.int32) if want_kc else None
        plan.inner_products(P, xh, hh, xi, kc)
        paths = plan.path_counts() if want_kc else None
        xh2, hh2, xi2 = np.full(nT, np.nan), np.full(nT, np.nan), np.full(nT, np.nan)
        plan.inner_products(P, xh2, hh2, xi2, None)
    if want_kc:
        assert sum(paths.values()) == int((kc >= 0).sum()), (paths, int((kc >= 0).sum()))
    out = dict(xh=xh, hh=hh, xh_im=xi, kc=kc, paths=paths, hot=dict(xh=xh2, hh=hh2, xh_im=xi2, kc=None))
    if "evaluator" not in override:
        # the default evaluator is the moment tables (|b| <= 0.12); run the direct evaluator as well
        with api.plan_from_workload(w, evaluator="direct", **override) as plan:
            xh3, hh3, xi3 = np.full(nT, np.nan), np.full(nT, np.nan), np.full(nT, np.nan)
            plan.inner_products(P, xh3, hh3, xi3, None)
        out["hot_direct"] = dict(xh=xh3, hh=hh3, xh_im=xi3, kc=None)
    return out


def _check(w, g, o, xx, tol=TOL, reg=REG):
    norm = np.sqrt(xx * np.maximum(o["hh"], 1e-300))
    assert np.all(np.isfinite(g["xh"])) and np.all(np.isfinite(g["hh"]))
    e_xh = np.abs(g["xh"] - o["xh"]) / norm
    e_xi = np.abs(g["xh_im"] - o["xh_im"]) / norm
    e_hh = np.abs(g["hh"] - o["hh"]) / norm
    e_hh_rel = np.abs(g["hh"] - o["hh"]) / np.maximum(o["hh"], 1e-300)
    assert e_xh.max() <= tol, ("xh", e_xh.max(), int(e_xh.argmax()))
    assert e_xi.max() <= tol, ("xh_im", e_xi.max(), int(e_xi.argmax()))
    assert e_hh.max() <= tol, ("hh", e_hh.max(), int(e_hh.argmax()))
    assert e_hh_rel[o["hh"] > 0].max(initial=0.0) <= tol, ("hh rel", e_hh_rel.max())
    if reg is not None:
        assert max(e_xh.max(), e_xi.max(), e_hh.max()) <= reg, ("regression bar", e_xh.max(), e_xi.max(), e_hh.max())
    for alt in ("hot", "hot_direct"):
        if g.get(alt) is not None:
            _check(w, g[alt], o, xx, tol, reg)
    if g.get("kc") is not None:
        tie = (o["flags"] != 0)[:, None, :]
        bad = (g["kc"] != o["kc"]) & ~tie
        assert not bad.any(), ("k_c mismatch", np.argwhere(bad)[:5], g["kc"][bad][:5], o["kc"][bad][:5])
        d = np.abs(g["kc"].astype(np.int64) - o["kc"])
        assert np.all((d <= 1) | (g["kc"] == -1) | (o["kc"] == -1))
    return float(e_xh.max()), float(e_hh_rel.max())


def _oracle(w, params=None, **override):
    ww = w
    if override:
        import copy
        ww = copy.copy(w)
        ww.desc = dict(w.desc, **override)
    plan, store = to_oracle(ww)
    o = oin.inner_products(plan, store, w.params if params is None else params)
    return o, oin.xx_band(plan, store), plan, store


# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", ["F", "M"])
@pytest.mark.parametrize("kernel", ["fresnel", "dirichlet"])
def test_config1(variant, kernel):
    """BASELINE.json configs[0] whole: 64 templates x 256 SFTs, K = 4."""
    w = wl.config1(variant=variant)
    o, xx, _, _ = _oracle(w, kernel=kernel)
    g = _run_gpu(w, kernel=kernel)
    _check(w, g, o, xx)
    assert (o["kc"] >= 0).sum() > 0
    # the injected signal is template 0: its <x,h> is the largest of the bank up to noise
    if kernel == "fresnel" and variant == "F":
        assert g["xh"][0] > 0.5 * g["hh"][0]


@pytest.fixture(scope="module")
def et_small():
    """Config-2 recipe at a size the oracle finishes in seconds: 1200 SFT slots (10 % gaps,
    lognormal per-SFT PSD scale, coloured PSD shape), b up to ~4 in the last SFTs, 333 templates
    (2 full tiles of 128 + a ragged tail)."""
    return wl.et_bns(n_templates=333, n_sft=1200, K=8, name="et-small")


def test_et_small_fresnel(et_small):
    w = et_small
    o, xx, _, _ = _oracle(w)
    g = _run_gpu(w)
    _check(w, g, o, xx)
    gaps = w.psd_scale[0] <= 0
    assert gaps.sum() == 120 and np.all(g["kc"][:, 0, gaps] == -1)


def test_et_small_masked_and_dirichlet(et_small):
    """Variant "M" (f_lo = 5 Hz: only the tail is active) and the Dirichlet kernel."""
    w = et_small
    for ov in (dict(f_lo=5.0), dict(kernel="dirichlet"), dict(f_lo=5.0, f_hi=9.0, kernel="dirichlet")):
        o, xx, _, _ = _oracle(w, **ov)
        g = _run_gpu(w, **ov)
        _check(w, g, o, xx)
        assert 0 < (o["kc"] >= 0).sum() <= o["kc"].size


@pytest.mark.parametrize("K", [0, 1, 2, 5, 16, 32, 64, 128])
def test_band_half_widths(et_small, K):
    """Config 5's K axis: specialised (4, 8, 16) and generic code paths, including K = 0."""
    w = et_small
    P = w.params[:40]
    o, xx, _, _ = _oracle(w, params=P, K=K)
    g = _run_gpu(w, params=P, K=K)
    _check(w, g, o, xx)


@pytest.mark.parametrize("n_sft", [1, 2, 3, 9, 33])
def test_tiny_sft_counts(n_sft):
    """Degenerate time axes: 1, 2, 3, 9 and 33 SFT slots (the kernels take two SFTs per step and keep tracks two SFTs
    ahead; work units of at most 32 SFTs), inner products and the cumulative call, with and without gaps."""
    api = _api()
    for gap_fraction in (0.0, 0.34):
        w = wl.et_bns(n_templates=37, n_sft=n_sft, K=8, gap_fraction=gap_fraction, name="et-tiny", tau_end=129.0 + 8.0 * (1200 - n_sft))
        o, xx, plan_o, store = _oracle(w)
        g = _run_gpu(w)
        if (o["kc"] >= 0).any():
            _check(w, g, o, xx)
        else:
            assert np.all(g["xh"] == 0.0) and np.all(g["hh"] == 0.0)
        oc = oin.cumulative_snr(plan_o, store, w.params)
        with api.plan_from_workload(w) as plan:
            cx = np.full((37, n_sft), np.nan, np.float32)
            ch = np.full((37, n_sft), np.nan, np.float32)
            snr = np.full((37, n_sft), np.nan, np.float32)
            plan.cumulative_snr(np.ascontiguousarray(w.params), snr, cx, ch)
        norm = np.sqrt(max(xx, 1e-300) * np.maximum(o["hh"], 1e-300))[:, None]
        assert np.all(np.isfinite(snr))
        assert (np.abs(cx - oc["cum_xh"]) / norm).max() <= TOL * 1.0001 or np.abs(cx - oc["cum_xh"]).max() == 0.0
        assert (np.abs(ch - oc["cum_hh"]) / norm).max() <= TOL * 1.0001 or np.abs(ch - oc["cum_hh"]).max() == 0.0


@pytest.mark.parametrize("chunk", [1, 7, 32, 64, 5000])
def test_chunking_is_invisible(et_small, chunk):
    """SFT-axis tiling (grid.y) must not change results beyond fp64 summation order."""
    api = _api()
    w = et_small
    P = np.ascontiguousarray(w.params[:130])
    o, xx, _, _ = _oracle(w, params=P)
    with api.plan_from_workload(w) as plan:
        plan.set_chunk(chunk)
        xh, hh, xi = np.empty(130), np.empty(130), np.empty(130)
        plan.inner_products(P, xh, hh, xi, None)
    _check(w, dict(xh=xh, hh=hh, xh_im=xi, kc=None), o, xx)


def test_split_fp32_phase_path(et_small):
    """SFT_PHASE_SPLIT32 (config 5's phase-path axis): the track in double-float arithmetic gives the same
    results and the same bins as the fp64 track, for both kernel variants (run-time flags / CfgBNS32)."""
    w = et_small
    o, xx, _, _ = _oracle(w)
    g = _run_gpu(w, phase_path="split32")
    _check(w, g, o, xx)
    w1 = wl.config1()
    o1, xx1, _, _ = _oracle(w1)
    _check(w1, _run_gpu(w1, phase_path="split32"), o1, xx1)
    w4 = wl.config4(n_templates=64)
    o4, xx4, _, _ = _oracle(w4)
    _check(w4, _run_gpu(w4, phase_path="split32"), o4, xx4)


def test_config4_small():
    """BASELINE.json configs[3] recipe with 300 templates: 2 channels, annual response, K = 16
    clipping at k < 1, 0PN+1PN."""
    w = wl.config4(n_templates=300)
    o, xx, _, _ = _oracle(w)
    g = _run_gpu(w)
    _check(w, g, o, xx)
    assert g["xh"][0] > 0.5 * g["hh"][0]


@pytest.mark.parametrize("C", [3, 4])
def test_three_and_four_channels(C):
    """SFT_MAX_CHANNELS = 4: the run-time-flag kernel variants with 3 and 4 channels (extra channels = scaled,
    gap-punched copies of the LISA pair with their own response phases), annual response and cumulative call."""
    import copy
    w0 = wl.config4(n_templates=70)
    w = copy.copy(w0)
    rng = np.random.default_rng(90 + C)
    n_sft = w0.desc["n_sft"]
    extra = C - 2
    bins = [w0.bins[0], w0.bins[1]] + [(0.5 + 0.25 * i) * w0.bins[i % 2] for i in range(extra)]
    scale = [w0.psd_scale[0], w0.psd_scale[1]]
    for i in range(extra):
        s = w0.psd_scale[i % 2] * (1.0 + 0.5 * i)
        s = s.copy()
        s[rng.choice(n_sft, size=n_sft // 7, replace=False)] = 0.0         # gaps of their own
        scale.append(s)
    shape = [w0.psd_shape[0], w0.psd_shape[1]] + [w0.psd_shape[i % 2] * (2.0 + i) for i in range(extra)]
    w.bins = np.ascontiguousarray(np.stack(bins)).astype(np.complex64)
    w.bins[2:][np.stack(scale[2:]) <= 0.0] = 0.0
    w.psd_scale = np.stack(scale)
    w.psd_shape = np.stack(shape)
    w.desc = dict(w0.desc, n_channels=C, resp_psi=tuple(0.4 * c for c in range(C)), resp_chi=tuple(0.7 * c - 0.3 for c in range(C)))
    o, xx, plan_o, store = _oracle(w)
    g = _run_gpu(w)
    _check(w, g, o, xx)
    assert np.any(g["kc"][:, 2, :] != g["kc"][:, 0, :])                    # the extra channel's own gaps show up
    api = _api()
    oc = oin.cumulative_snr(plan_o, store, w.params[:33])
    with api.plan_from_workload(w) as plan:
        cx = np.empty((33, n_sft), np.float32)
        ch = np.empty((33, n_sft), np.float32)
        plan.cumulative_snr(np.ascontiguousarray(w.params[:33]), None, cx, ch)
    norm = np.sqrt(xx * o["hh"][:33])[:, None]
    assert (np.abs(cx - oc["cum_xh"]) / norm).max() <= TOL and (np.abs(ch - oc["cum_hh"]) / norm).max() <= TOL


def test_statistics_phase_maximised(et_small):
    """sft_statistics (NEXT-3): L = <x,h> - <h,h>/2 (Eq.(2)) and the phase-maximised statistic of Eq.(7) P:97,
    checked against the oracle's inner products of the two quadratures h_c (phi_c) and h_s (phi_c + pi/2)."""
    api = _api()
    w = et_small
    P = np.ascontiguousarray(w.params[:48])
    Ps = P.copy()
    Ps[:, 3] += 0.5 * np.pi
    oc, xx, _, _ = _oracle(w, params=P)
    os_, _, _, _ = _oracle(w, params=Ps)
    stat_o = (oc["xh"] ** 2 + os_["xh"] ** 2) / oc["hh"]
    with api.plan_from_workload(w) as plan:
        xh, hh, xi = np.empty(48), np.empty(48), np.empty(48)
        plan.inner_products(P, xh, hh, xi, None)
        L, stat = np.empty(48), np.empty(48)
        plan.statistics(xh, xi, hh, L, stat)
    assert np.allclose(L, xh - 0.5 * hh, rtol=0, atol=1e-12 * np.abs(xh).max())
    tol = 2.0 * 1e-4 * np.sqrt(xx * oc["hh"]) * np.sqrt(oc["xh"] ** 2 + os_["xh"] ** 2) / oc["hh"] + 1e-4 * stat_o
    assert np.all(np.abs(stat - stat_o) <= tol), np.abs(stat - stat_o).max()
    assert np.abs(stat - stat_o).max() <= 1e-3 * stat_o.max()


@pytest.mark.parametrize("n_channels,noise", [(1, 0.0), (1, 0.7), (2, 0.7)])
def test_fstat_matches_oracle(n_channels, noise):
    """sft_fstat (NEXT-3; Eq.(10)-(13) P:107-122): the 4 products ([x,h_nu]), the 3 distinct ([h_nu,h_mu]) and 2F against the
    oracle, which sums all 4 + 10 products bin by bin and solves the 4 x 4 system; noiseless data return the injected c_nu."""
    from oracle import stats as ost
    api = _api()
    w = wl.fstat_case(n_templates=70, n_channels=n_channels, noise=noise)
    plan_o, store = to_oracle(w)
    a, b = w.response.real.astype(np.float64), w.response.imag.astype(np.float64)
    o = ost.fstat(plan_o, store, w.params, a, b)
    xx = oin.xx_band(plan_o, store)
    nT = w.n_templates
    for ev in ("auto", "direct"):
        with api.plan_from_workload(w, evaluator=ev) as plan:
            F, x, m = np.full(nT, np.nan), np.full((4, nT), np.nan), np.full((3, nT), np.nan)
            plan.fstat(np.ascontiguousarray(w.params), F, x, m)
            F2 = np.full(nT, np.nan)
            plan.fstat(np.ascontiguousarray(w.params), F2)
        assert np.array_equal(F, F2)
        Mo = o["M"]
        for nu in range(4):
            assert (np.abs(x[nu] - o["x"][:, nu]) / np.sqrt(xx * Mo[:, nu, nu])).max() <= REG
        for i, (nu, mu) in enumerate(((0, 0), (1, 1), (0, 1))):
            assert (np.abs(m[i] - Mo[:, nu, mu]) / np.sqrt(Mo[:, nu, nu] * Mo[:, mu, mu])).max() <= REG
            assert (np.abs(m[i] - Mo[:, nu + 2, mu + 2]) / np.sqrt(Mo[:, nu, nu] * Mo[:, mu, mu])).max() <= REG
        assert np.abs(Mo[:, :2, 2:]).max() <= 1e-10 * np.abs(Mo).max()                 # what the kernel does not compute is zero
        # 2F: |d 2F| <= 2 sqrt(2F) |d x|_M  ->  bar REG sqrt(<x,x>) 2 sqrt(2F) (+ relative REG for the M part)
        assert np.all(np.abs(F - o["twoF"]) <= 4.0 * REG * np.sqrt(xx * np.maximum(o["twoF"], 1e-300)) + 10 * REG * o["twoF"])
    if noise == 0.0:
        M = np.array([[m[0][0], m[2][0], 0, 0], [m[2][0], m[1][0], 0, 0], [0, 0, m[0][0], m[2][0]], [0, 0, m[2][0], m[1][0]]])
        c = np.linalg.solve(M, x[:, 0])
        assert np.abs(c - w.notes["c_nu"]).max() < 0.02


def test_validity_flags(et_small):
    """sft_validity (NEXT-2; Eq.(33)-(34) P:244-248) against its oracle twin on a wide bank (ended, never-active and full-span
    templates), for all three PN orders; device and host buffers."""
    import torch
    api = _api()
    w = wl.et_bns_wide_bank(et_small, 300)
    for pn in (0, 1, 2):
        o, xx, plan_o, store = _oracle(w, pn1=pn)
        d_o = oin.validity(plan_o, w.params)
        with api.Plan(dict(w.desc, pn1=pn)) as plan:                       # no data loaded: not needed
            d, fl = np.full(300, np.nan), np.full(300, 9, np.uint8)
            plan.validity(np.ascontiguousarray(w.params), 0.25, d, fl)
            Pd = torch.from_numpy(np.ascontiguousarray(w.params)).cuda()
            dd = torch.full((300,), float("nan"), dtype=torch.float64, device="cuda")
            plan.validity(Pd, 0.25, dd, None)
            plan.sync()
        assert np.allclose(d, d_o, rtol=1e-9, atol=0.0) and np.array_equal(dd.cpu().numpy(), d)
        assert np.array_equal(fl, (d_o > 0.25).astype(np.uint8)) and 0 < fl.sum() < 300


def test_pn15_waveform(et_small):
    """SFT_WF_PN15 (NEXT-2): the 1.5PN tail terms in the closed-form track, the polynomial track of the clean blocks and the
    double-float track, against the oracle; k_c bit-exact.  The data hold a 1PN signal: the templates need not match it."""
    w = et_small
    P = w.params[:96]
    o, xx, _, _ = _oracle(w, params=P, pn1=2)
    assert np.abs(o["xh"] - _oracle(w, params=P)[0]["xh"]).max() > 1.0          # the tail terms matter
    _check(w, _run_gpu(w, params=P, pn1=2), o, xx)
    _check(w, _run_gpu(w, params=P, pn1=2, phase_path="split32"), o, xx)
    ww = wl.et_bns_wide_bank(w, 64)
    o2, xx2, _, _ = _oracle(ww, pn1=2)
    _check(ww, _run_gpu(ww, pn1=2), o2, xx2)


def test_response_table():
    """SFT_RESP_TABLE: an arbitrary complex per-(channel, SFT) response."""
    w = wl.config4(n_templates=40)
    rng = np.random.default_rng(77)
    R = (rng.standard_normal((2, w.desc["n_sft"])) + 1j * rng.standard_normal((2, w.desc["n_sft"]))).astype(np.complex64)
    w.response = R
    w.desc = dict(w.desc, response="table")
    o, xx, _, _ = _oracle(w)
    g = _run_gpu(w)
    _check(w, g, o, xx)


def test_cumulative_small(et_small):
    """sft_cumulative_snr: inclusive prefix sums over SFTs, every element, fp32 outputs."""
    api = _api()
    w = et_small
    P = np.ascontiguousarray(w.params[:150])
    plan_o, store = to_oracle(w)
    o = oin.cumulative_snr(plan_o, store, P)
    ref = oin.inner_products(plan_o, store, P)
    xx = oin.xx_band(plan_o, store)
    n = w.desc["n_sft"]
    for chunk in (0, 32, 96):
        with api.plan_from_workload(w) as plan:
            plan.set_chunk(chunk)
            snr = np.full((150, n), np.nan, np.float32)
            cx = np.full((150, n), np.nan, np.float32)
            ch = np.full((150, n), np.nan, np.float32)
            plan.cumulative_snr(P, snr, cx, ch)
            snr_only = np.full((150, n), np.nan, np.float32)
            plan.cumulative_snr(P, snr_only, None, None)
        norm = np.sqrt(xx * ref["hh"])[:, None]
        assert np.abs(cx - o["cum_xh"]).max() <= 1e-4 * norm.max()
        assert (np.abs(cx - o["cum_xh"]) / norm).max() <= TOL
        assert (np.abs(ch - o["cum_hh"]) / norm).max() <= TOL
        big = o["cum_hh"] > 1e-3 * ref["hh"][:, None]
        assert np.abs(snr - o["snr"])[big].max() <= 1e-3 * max(1.0, np.abs(o["snr"]).max())
        assert np.array_equal(snr, snr_only)
        assert np.all(snr[o["cum_hh"] == 0.0] == 0.0)
        # last column equals the totals
        assert np.allclose(cx[:, -1], ref["xh"], rtol=0, atol=1e-4 * norm.max())


def test_cumulative_host_slabs(et_small):
    """sft_cumulative_snr with host outputs runs the bank in slabs of templates (copy of slab i under the compute of slab
    i + 1, sft_plan_set_host_slab): the matrices must not depend on the slab size - pageable and pinned host memory, a ragged
    last slab, one and three outputs."""
    import torch
    api = _api()
    w = et_small
    nT, n = 150, w.desc["n_sft"]
    P = np.ascontiguousarray(w.params[:nT])
    with api.plan_from_workload(w) as plan:
        Pd = torch.from_numpy(P).cuda()
        ref = [torch.full((nT, n), float("nan"), dtype=torch.float32, device="cuda") for _ in range(3)]
        plan.cumulative_snr(Pd, *ref)
        plan.sync()
        ref = [r.cpu().numpy() for r in ref]
        for slab in (0, 32, 64, 100, 4096):                            # 100 -> 96: slabs of 96 + 54 templates
            plan.set_host_slab(slab)
            out = [np.full((nT, n), np.nan, np.float32) for _ in range(3)]
            plan.cumulative_snr(P, *out)
            for a, b in zip(out, ref):
                assert np.array_equal(a, b), slab
            pin = torch.full((nT, n), float("nan"), dtype=torch.float32).pin_memory()
            plan.cumulative_snr(P, pin.numpy(), None, None)
            assert np.array_equal(pin.numpy(), ref[0]), slab
        with pytest.raises(api.SftError):
            plan.set_host_slab(-1)


def test_device_pointers_and_edge_sizes(et_small):
    """Device-resident params/outputs (torch tensors), n_templates in {0, 1, 129}."""
    import torch
    api = _api()
    w = et_small
    o, xx, _, _ = _oracle(w, params=w.params[:129])
    with api.plan_from_workload(w) as plan:
        plan.inner_products(np.zeros((0, 8)), np.zeros(0), np.zeros(0))      # n = 0: SFT_OK, no work
        for nT in (1, 129):
            P = torch.from_numpy(np.ascontiguousarray(w.params[:nT])).cuda()
            xh = torch.full((nT,), float("nan"), dtype=torch.float64, device="cuda")
            hh = torch.full_like(xh, float("nan"))
            xi = torch.full_like(xh, float("nan"))
            plan.inner_products(P, xh, hh, xi, None)
            plan.sync()
            g = dict(xh=xh.cpu().numpy(), hh=hh.cpu().numpy(), xh_im=xi.cpu().numpy(), kc=None)
            oo = {k: (v[:nT] if isinstance(v, np.ndarray) else v) for k, v in o.items()}
            _check(w, g, oo, xx)
        assert plan.launch_count() > 0 and plan.last_kernel_ms() > 0.0


def test_errors_on_device(et_small):
    api = _api()
    w = et_small
    plan = api.Plan(w.desc)
    with pytest.raises(api.SftError) as ei:
        plan.inner_products(np.zeros((1, 8)), np.zeros(1), np.zeros(1))
    assert "SFT_ENODATA" in str(ei.value)
    plan.close()


def test_error_paths_leave_outputs_untouched(et_small):
    """include/sft.h: "on error the outputs are untouched".  Every error return of the three compute calls, with NaN / -7
    sentinels in the outputs (host and device buffers)."""
    import ctypes as C
    import torch
    api = _api()
    w = et_small
    n = w.desc["n_sft"]
    P = np.ascontiguousarray(w.params[:5])

    def fresh():
        return [np.full(5, np.nan) for _ in range(3)], np.full((5, 1, n), -7, np.int32), [np.full((5, n), np.nan, np.float32) for _ in range(3)]

    def untouched(v, kc, m):
        return all(np.isnan(a).all() for a in v) and (kc == -7).all() and all(np.isnan(a).all() for a in m)

    # 1. no data loaded: SFT_ENODATA from both calls
    plan = api.Plan(w.desc)
    v, kc, m = fresh()
    for call in (lambda: plan.inner_products(P, v[0], v[1], v[2], kc), lambda: plan.cumulative_snr(P, m[0], m[1], m[2])):
        with pytest.raises(api.SftError) as ei:
            call()
        assert "SFT_ENODATA" in str(ei.value)
    assert untouched(v, kc, m)
    plan.close()
    with api.plan_from_workload(w) as plan:
        lib, h = plan.lib, plan._h
        vp = lambda a: C.c_void_p(a.ctypes.data)
        # 2. argument errors straight through the C ABI (the binding would refuse some of them itself)
        assert lib.sft_inner_products(h, -1, vp(P), vp(v[0]), vp(v[1]), vp(v[2]), vp(kc), 0) == 1          # n_templates < 0
        assert lib.sft_inner_products(h, 5, vp(P), vp(v[0]), vp(v[1]), vp(v[2]), vp(kc), 7) == 1           # bad mem
        assert lib.sft_inner_products(h, 5, None, vp(v[0]), vp(v[1]), vp(v[2]), vp(kc), 0) == 1            # params NULL
        assert lib.sft_inner_products(h, 5, vp(P), None, vp(v[1]), vp(v[2]), vp(kc), 0) == 1               # xh NULL
        assert lib.sft_cumulative_snr(h, 5, vp(P), None, None, None, 0) == 1                               # no output at all
        assert lib.sft_cumulative_snr(h, -2, vp(P), vp(m[0]), vp(m[1]), vp(m[2]), 0) == 1
        assert lib.sft_cumulative_snr(h, 5, None, vp(m[0]), vp(m[1]), vp(m[2]), 0) == 1
        assert lib.sft_cumulative_snr(h, 5, vp(P), vp(m[0]), vp(m[1]), vp(m[2]), 3) == 1
        assert lib.sft_statistics(h, 5, vp(v[0]), vp(v[1]), vp(v[2]), None, None, 0) == 1                  # nothing asked for
        assert lib.sft_statistics(h, 5, None, vp(v[1]), vp(v[2]), vp(v[0]), None, 0) == 1
        assert b"" != lib.sft_last_error(h)
        assert untouched(v, kc, m)
        # n_templates == 0 is SFT_OK and touches nothing
        assert lib.sft_inner_products(h, 0, vp(P), vp(v[0]), vp(v[1]), vp(v[2]), vp(kc), 0) == 0
        assert lib.sft_cumulative_snr(h, 0, vp(P), vp(m[0]), vp(m[1]), vp(m[2]), 0) == 0
        assert untouched(v, kc, m)
        # 3. sft_load_data errors leave the channel as it was: the plan still computes the same numbers afterwards
        plan.inner_products(P, v[0], v[1], v[2], None)
        ref = [a.copy() for a in v]
        bins = np.ascontiguousarray(w.bins[0], np.complex64)
        scale = np.ascontiguousarray(w.psd_scale[0])
        bad_shape = np.ascontiguousarray(w.psd_shape[0]).copy()
        bad_shape[3] = -1.0
        assert lib.sft_load_data(h, 0, vp(bins), vp(scale), vp(bad_shape), None, 0) == 1                   # non-positive PSD
        assert lib.sft_load_data(h, 1, vp(bins), vp(scale), None, None, 0) == 1                            # channel out of range
        assert lib.sft_load_data(h, 0, None, vp(scale), None, None, 0) == 1
        assert lib.sft_load_data(h, 0, vp(bins), vp(scale), None, None, 9) == 1
        v2 = [np.full(5, np.nan) for _ in range(3)]
        plan.inner_products(P, v2[0], v2[1], v2[2], None)
        assert all(np.array_equal(a, b) for a, b in zip(ref, v2))
        # 4. device buffers: a failing call leaves them untouched as well
        Pd = torch.from_numpy(P).cuda()
        xd = torch.full((5,), float("nan"), dtype=torch.float64, device="cuda")
        dp = lambda t: C.c_void_p(t.data_ptr())
        assert lib.sft_inner_products(h, 5, dp(Pd), dp(xd), None, None, None, 1) == 1                      # hh NULL
        assert lib.sft_cumulative_snr(h, 5, dp(Pd), None, None, None, 1) == 1
        plan.sync()
        assert bool(torch.isnan(xd).all())


def test_table_track_banded_tables(et_small):
    """sft_plan_set_table_track: moment tables only along the track of a fiducial template (the SFTs serve "any template
    within a given parameter-space region").  (i) For the +-1e-3 bank the banded tables give bit-identical results to the full
    ones, for both calls, at a fraction of the memory, and the same evaluator paths; (ii) a wide bank, most of whose lanes
    leave the band of the track, falls back to the direct evaluator for those SFTs and still matches the oracle; (iii) a plan
    whose full tables could never fit (4000-bin band x 200,000 SFTs: 411 GB) gets tables with a track."""
    api = _api()
    w = et_small
    n = w.desc["n_sft"]
    P = np.ascontiguousarray(w.params)
    nT = len(P)
    def run(plan):
        xh, hh, xi = np.empty(nT), np.empty(nT), np.empty(nT)
        kc = np.empty((nT, 1, n), np.int32)
        plan.inner_products(P, xh, hh, xi, kc)
        paths = plan.path_counts()
        snr = np.empty((nT, n), np.float32)
        plan.cumulative_snr(P, snr)
        xh2, hh2 = np.empty(nT), np.empty(nT)
        plan.inner_products(P, xh2, hh2)
        return xh, hh, xi, kc, snr, xh2, hh2, paths
    with api.plan_from_workload(w) as plan:
        full = run(plan)
        full_bytes = plan.table_bytes()
        plan.set_table_track(w.injection, 3)                      # replaces the tables: data must be loaded again
        with pytest.raises(api.SftError) as ei:
            plan.inner_products(P, np.empty(nT), np.empty(nT))
        assert "SFT_ENODATA" in str(ei.value)
    with api.plan_from_workload(w, table_track=(w.injection, 3)) as plan:
        band = run(plan)
        assert 0 < plan.table_bytes() < 0.2 * full_bytes
    for i, (a, b) in enumerate(zip(full[:-1], band[:-1])):
        if i == 4:          # the SNR matrix: the two layouts run two instantiations of the cumulative kernel (fp32 rounding of the running sums)
            assert np.abs(a - b).max() <= 2e-6 * np.abs(a).max()
        else:
            assert np.array_equal(a, b)
    assert full[-1] == band[-1] and band[-1]["table"] > 0
    ww = wl.et_bns_wide_bank(w, 96)
    ww.params = np.concatenate([w.params[:64], ww.params])          # two warps inside the band of the track, three wide ones
    o, xx, _, _ = _oracle(ww)
    g = _run_gpu(ww, table_track=(w.injection, 3))
    _check(ww, g, o, xx)
    assert g["paths"]["table"] > 0 and g["paths"]["series1"] + g["paths"]["series2"] + g["paths"]["series3"] > 0
    # two channels with the annual response (config-4 recipe), tables along the injection's track
    w4 = wl.config4(n_templates=100)
    o4, xx4, _, _ = _oracle(w4)
    g4 = _run_gpu(w4, table_track=(w4.injection, 2))
    _check(w4, g4, o4, xx4)
    assert g4["paths"]["table"] > 0
    # streaming append into banded tables = one-shot load
    bins, scale, shape = np.ascontiguousarray(w.bins[0], np.complex64), np.ascontiguousarray(w.psd_scale[0]), np.ascontiguousarray(w.psd_shape[0])
    with api.Plan(w.desc) as plan:
        plan.set_table_track(w.injection, 3)
        ps, pb = scale.copy(), bins.copy()
        ps[500:] = 0.0
        pb[500:] = 0.0
        plan.load_data(0, pb, ps, shape)
        plan.append_sfts(0, 500, np.ascontiguousarray(bins[500:]), np.ascontiguousarray(scale[500:]))
        xh, hh = np.empty(nT), np.empty(nT)
        plan.inner_products(P, xh, hh)
    assert np.array_equal(xh, band[5]) and np.array_equal(hh, band[6])
    desc = dict(n_channels=1, n_sft=200000, t_sft=8.0, fs=2048.0, t0=0.0, k_lo=10, k_hi=4010, K=8, kernel="fresnel",
                pn1=1, response="none", f_lo=0.0, f_hi=1e9, f_ref=10.0)
    fid = w.injection.copy()
    fid[2] = 200000 * 8.0 + 300.0
    with api.Plan(dict(desc, evaluator="auto")) as plan:
        assert plan.table_bytes() == 0
        plan.set_table_track(fid, 8)
        assert 0 < plan.table_bytes() < 8e9


def test_evaluator_selection_by_memory():
    """SFT_EVAL_AUTO falls back to the direct evaluator when the moment tables would not fit in a quarter of the
    free device memory; SFT_EVAL_TABLE reports SFT_ENOMEM instead."""
    api = _api()
    desc = dict(n_channels=1, n_sft=200000, t_sft=8.0, fs=2048.0, t0=0.0, k_lo=10, k_hi=4010, K=8, kernel="fresnel",
                pn1=1, response="none", f_lo=0.0, f_hi=1e9, f_ref=10.0)           # tables: 411 GB
    with pytest.raises(api.SftError) as ei:
        api.Plan(dict(desc, evaluator="table"))
    assert "SFT_ENOMEM" in str(ei.value)
    api.Plan(dict(desc, evaluator="auto")).close()                                 # 12.9 GB store only: fine
    with pytest.raises(api.SftError):
        api.Plan(dict(desc, evaluator=7))


def test_ended_and_degenerate_templates(et_small):
    """Templates whose t_c lies inside / before the data (inactive from some SFT on; all inactive)."""
    w = et_small
    P = w.params[:6].copy()
    T_obs = w.desc["n_sft"] * w.desc["t_sft"]
    P[1, 2] = 0.5 * T_obs          # coalesces mid-way: later SFTs inactive, earlier ones out of band
    P[2, 2] = -10.0                # already over
    P[3, 2] = T_obs + 5000.0       # far in the future: frequencies below the stored band
    P[4, 4] = 0.0                  # zero amplitude
    o, xx, _, _ = _oracle(w, params=P)
    g = _run_gpu(w, params=P)
    norm = np.sqrt(xx * np.maximum(o["hh"].max(), 1.0))
    assert np.all(np.abs(g["xh"] - o["xh"]) <= TOL * norm) and np.all(np.abs(g["hh"] - o["hh"]) <= TOL * norm)
    tie = (o["flags"] != 0)[:, None, :]
    assert not ((g["kc"] != o["kc"]) & ~tie).any()
    assert g["hh"][2] == 0.0 and g["hh"][4] == 0.0


# ------------------------------------------------------------------------------------------
# Heterogeneous warps: every bank above is a +-1e-3 box, so the 32 lanes of a warp share k_c, the table node and the
# evaluator path.  Here neighbouring rows differ by tens of bins and by orders of magnitude in b = fdot T^2, and some
# are ended / out of band / not yet in band at the same SFT: the per-warp decisions (clean-block vote, bmax, the clamped
# windows of inactive lanes) are taken with mixed lanes.
@pytest.mark.parametrize("kernel", ["fresnel", "dirichlet"])
def test_heterogeneous_bank(et_small, kernel):
    api = _api()
    w = wl.et_bns_wide_bank(et_small, 200)
    o, xx, plan_o, store = _oracle(w, kernel=kernel)
    kc = o["kc"][:, 0, :]
    act = kc >= 0
    # the bank really is heterogeneous inside warps: at one SFT, lanes of one warp are spread over many bins, some inactive
    spread = [np.ptp(kc[32 * g:32 * g + 32][:, a][act[32 * g:32 * g + 32][:, a]]) for g in range(6) for a in range(0, 1200, 50)
              if act[32 * g:32 * g + 32][:, a].sum() > 1]
    assert max(spread) >= 30 and 0.2 < act.mean() < 0.95
    g = _run_gpu(w, kernel=kernel)
    _check(w, g, o, xx)
    if kernel == "fresnel":
        p = g["paths"]
        assert p["table"] > 0 and p["table2"] > 0 and p["fresnel"] > 0
    # the cumulative call on the same bank, every element
    oc = oin.cumulative_snr(plan_o, store, w.params)
    n = w.desc["n_sft"]
    with api.plan_from_workload(w, kernel=kernel) as plan:
        cx = np.full((200, n), np.nan, np.float32)
        ch = np.full((200, n), np.nan, np.float32)
        snr = np.full((200, n), np.nan, np.float32)
        plan.cumulative_snr(np.ascontiguousarray(w.params), snr, cx, ch)
    norm = np.sqrt(xx * np.maximum(o["hh"], 1e-300))[:, None]
    assert (np.abs(cx - oc["cum_xh"]) / norm).max() <= REG and (np.abs(ch - oc["cum_hh"]) / norm).max() <= REG
    assert np.all(np.isfinite(snr)) and np.all(snr[oc["cum_hh"] == 0.0] == 0.0)


# ------------------------------------------------------------------------------------------
# BASELINE.json's full sizes, in the launch configuration bench.py times (default work-unit size,
# hot kernel variants), against the oracle run on all host cores (tests/_util.py).
def _sample_rows(n, k, seed):
    rng = np.random.default_rng(seed)
    return np.unique(np.concatenate([[0, 1, n - 1], rng.choice(n, size=k, replace=False)]))


def _snr_bar(xx, o_snr):
    """|d SNR| allowed: the REG bar on <x,h> in SNR units (<x,h> error REG sqrt(<x,x><h,h>) / sqrt(cum_hh), taken where
    cum_hh is at least a tenth of <h,h>... the caller masks) plus fp32 rounding of the stored value."""
    return REG * np.sqrt(xx) * 4.0 + 2e-7 * np.abs(o_snr)


def test_config2_full_size_all_templates():
    """configs[1]: 4096 templates x 10,800 SFT slots, K = 8: EVERY template against the oracle; k_c on 20 of them."""
    api = _api()
    w = wl.config2()
    nT, N = w.n_templates, w.desc["n_sft"]
    P = np.ascontiguousarray(w.params)
    rows = _sample_rows(nT, 17, 21)
    with api.plan_from_workload(w) as plan:
        xh, hh, xi = np.empty(nT), np.empty(nT), np.empty(nT)
        plan.inner_products(P, xh, hh, xi, None)
        kc = np.empty((len(rows), 1, N), np.int32)
        xs, hs, is_ = np.empty(len(rows)), np.empty(len(rows)), np.empty(len(rows))
        plan.inner_products(np.ascontiguousarray(P[rows]), xs, hs, is_, kc)
        paths = plan.path_counts()
    from _util import oracle_totals_parallel
    o_xh, o_hh, o_xi = oracle_totals_parallel(w, P)
    plan_o, store = to_oracle(w)
    xx = oin.xx_band(plan_o, store)
    _check(w, dict(xh=xh, hh=hh, xh_im=xi, kc=None), dict(xh=o_xh, hh=o_hh, xh_im=o_xi), xx)
    o = oin.inner_products(plan_o, store, P[rows])
    _check(w, dict(xh=xs, hh=hs, xh_im=is_, kc=kc), o, xx)
    assert np.all(np.isfinite(xh)) and np.all(hh > 0)
    assert xh[0] > 0.8 * hh[0] and abs(hh[0] - 900.0) < 0.1 * 900.0            # the injection: SNR 30
    assert xh[0] > 0.9 * xh.max()                                               # and (nearly) the best match of the bank
    assert abs(xh[0] - o_xh[0]) <= 1e-4 * o_hh[0]
    assert sum(paths.values()) == int((kc >= 0).sum()) and paths["table"] > paths["table2"] > paths["fresnel"] > 0 and paths["series3"] == 0


def test_config3_full_size_all_templates():
    """configs[2] as BASELINE.json words it: cumulative SNR(t) for 16,384 templates x 10,800 SFTs (fp32 matrix), compared
    with oracle prefix sums at 32 seeded SFT indices for EVERY template, plus properties of every row."""
    api = _api()
    w = wl.config3()
    nT, N = w.n_templates, w.desc["n_sft"]
    P = np.ascontiguousarray(w.params)
    idx = wl.config3_check_indices(nT, N)                                             # [nT][32] seeded indices
    import torch
    with api.plan_from_workload(w) as plan:
        Pd = torch.from_numpy(P).cuda()
        snr = torch.empty((nT, N), dtype=torch.float32, device="cuda")
        cx = torch.empty_like(snr)
        ch = torch.empty_like(snr)
        plan.cumulative_snr(Pd, snr, cx, ch)
        snr_only = torch.empty_like(snr)
        plan.cumulative_snr(Pd, snr_only, None, None)                                 # the call bench.py times
        xh = torch.empty(nT, dtype=torch.float64, device="cuda")
        hh = torch.empty_like(xh)
        plan.inner_products(Pd, xh, hh, None, None)
        plan.sync()
        # properties on the device, all rows
        assert bool(torch.isfinite(snr).all())
        assert bool(torch.equal(snr, snr_only))
        assert bool((ch[:, 1:] >= ch[:, :-1] * (1.0 - 1e-6)).all())                   # <h,h> accumulates (fp32 store)
        tot_err = (cx[:, -1].double() - xh).abs() / (xh.abs() + hh.sqrt())
        assert float(tot_err.max()) < 1e-5                                            # last column = totals
        assert float(((ch[:, -1].double() - hh).abs() / hh).max()) < 1e-5
        i = torch.from_numpy(idx).cuda()
        g_snr = torch.gather(snr, 1, i).cpu().numpy()
        g_cx = torch.gather(cx, 1, i).cpu().numpy()
        g_ch = torch.gather(ch, 1, i).cpu().numpy()
        # the same call with a host matrix (slabs of templates, copies under the next slab's compute): same bits
        snr_host = np.empty((nT, N), dtype=np.float32)
        plan.cumulative_snr(P, snr_host, None, None)
        assert bool(torch.equal(torch.from_numpy(snr_host), snr.cpu()))
        del snr, cx, ch, snr_only, snr_host
    from _util import oracle_cumulative_at_parallel
    o_cx, o_ch, o_snr, o_xh, o_hh = oracle_cumulative_at_parallel(w, P, idx)
    plan_o, store = to_oracle(w)
    xx = oin.xx_band(plan_o, store)
    norm = np.sqrt(xx * o_hh)[:, None]
    assert (np.abs(g_cx - o_cx) / norm).max() <= REG, (np.abs(g_cx - o_cx) / norm).max()
    assert (np.abs(g_ch - o_ch) / norm).max() <= REG, (np.abs(g_ch - o_ch) / norm).max()
    assert (np.abs(g_ch - o_ch) / np.maximum(o_ch, 1e-300))[o_ch > 1e-3 * o_hh[:, None]].max() <= 1e-5
    big = o_ch > 0.1 * o_hh[:, None]
    assert np.all((np.abs(g_snr - o_snr) <= _snr_bar(xx, o_snr))[big]), np.abs(g_snr - o_snr)[big].max()
    assert np.abs(g_snr - o_snr)[o_ch > 1e-3 * o_hh[:, None]].max() <= 1e-3


# BASELINE.json configs[4]: the two largest axes of the sweep (bench.py --sweep), so that the GPU test record covers them.
def test_config5_43200_sfts():
    api = _api()
    w = wl.et_bns(n_templates=4096, n_sft=43200, K=8, name="config5")
    nT = w.n_templates
    P = np.ascontiguousarray(w.params)
    rows = _sample_rows(nT, 7, 24)
    with api.plan_from_workload(w) as plan:
        xh, hh, xi = np.empty(nT), np.empty(nT), np.empty(nT)
        plan.inner_products(P, xh, hh, xi, None)
    o, xx, _, _ = _oracle(w, params=P[rows])
    _check(w, dict(xh=xh[rows], hh=hh[rows], xh_im=xi[rows], kc=None), o, xx)
    assert np.all(np.isfinite(xh)) and np.all(hh > 0) and xh[0] > 0.8 * hh[0]


def test_config5_262144_templates():
    api = _api()
    w = wl.et_bns_bank(wl.config2(), 262144)
    nT = w.n_templates
    P = np.ascontiguousarray(w.params)
    rows = _sample_rows(nT, 9, 25)
    with api.plan_from_workload(w) as plan:
        xh, hh, xi = np.empty(nT), np.empty(nT), np.empty(nT)
        plan.inner_products(P, xh, hh, xi, None)
    o, xx, _, _ = _oracle(w, params=P[rows])
    _check(w, dict(xh=xh[rows], hh=hh[rows], xh_im=xi[rows], kc=None), o, xx)
    assert np.all(np.isfinite(xh)) and np.all(hh > 0) and xh[0] > 0.8 * hh[0]


def test_config4_full_size_sampled():
    """configs[3]: 65,536 templates, 2 channels x 672 SFTs, annual response, K = 16."""
    api = _api()
    w = wl.config4()
    nT = w.n_templates
    P = np.ascontiguousarray(w.params)
    rows = _sample_rows(nT, 29, 23)
    with api.plan_from_workload(w) as plan:
        xh, hh, xi = np.empty(nT), np.empty(nT), np.empty(nT)
        plan.inner_products(P, xh, hh, xi, None)
    o, xx, _, _ = _oracle(w, params=P[rows])
    _check(w, dict(xh=xh[rows], hh=hh[rows], xh_im=xi[rows], kc=None), o, xx)
    assert np.all(np.isfinite(xh)) and np.all(hh > 0)
