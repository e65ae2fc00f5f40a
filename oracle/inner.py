"""Oracle SFT inner product ``([x,h])``, ``([h,h])`` and the cumulative variant, fp64.

TEST INFRASTRUCTURE.  The method is an approximation (piecewise linear-chirp signal model +
band truncation + continuum kernel), so this follows the paper's algorithm step by step,
in the paper's order, by brute force:

1. per template, the four numbers ``{A_a, phi_a, f_a, fdot_a}`` at each SFT start ``t_a``
   (Eq.(16)-(17); P:374 step (i)) - ``oracle.waveform``;
2. per SFT, the bins ``k in [k_c-K, k_c+K]`` around ``f_k ~ f_a`` - ``select_bins``;
3. the positive-frequency SFT coefficients of the real piecewise model Eq.(18) P:166,
   ``h~_{c,a,k} = 1/2 T A_a R_{c,a} e^{i phi_a} F(a_k, b_a)`` with the kernel ``F`` of
   Eq.(27)-(29) P:208-219 - ``oracle.kernel`` - and ``Lambda z = Re[R z]`` (Eq.(5)-(6) P:80-85);
4. the sums of Eq.(20)/(24)/(35) P:178-259 with ONE ``df`` (reading A1), written as
   the discretised Eq.(1) P:20 over the selected bins with per-SFT noise ``S_{c,a}(f_k)``:

       ([x,h]) = 4 df Re sum_{c,a,k} conj(x~_{c,a,k}) h~_{c,a,k} / S_{c,a}(f_k)
               = 2 Re sum_{c,a} A_a R_{c,a} e^{i phi_a} sum_k conj(x~) F / S
       ([h,h]) = 4 df sum |h~|^2 / S = T sum_{c,a} A_a^2 |R_{c,a}|^2 sum_k |F|^2 / S

   gaps = missing SFTs add nothing; ``S_{c,a}(f_k) = s_{c,a} S_c(f_k)`` is the per-SFT
   whitening of P:139 (reading A9);
5. the cumulative variant: inclusive prefix sums over the SFT index ("accumulating the result
   over time"; early warning P:293) and ``SNR_a = cum_xh / sqrt(cum_hh)``.

Pins: tests/test_oracle_inner.py (P3, P8, P9 and the matched-signal end-to-end pin).
"""
from dataclasses import dataclass, field
import numpy as np

from . import waveform as wf
from . import kernel as kern

TIE_EPS = 1e-9          #: DESIGN.md reading A5/A12: decisions closer than this to a boundary are flagged
YEAR_S = 31557600.0     #: Julian year, for the synthetic annual response (D4)

FLAG_KC_TIE = 1
FLAG_MASK_TIE = 2


@dataclass
class Plan:
    """The analysis set-up (mirrors the fields of ``sft_plan_desc`` in include/sft.h)."""
    n_channels: int
    n_sft: int
    t_sft: float
    fs: float
    t0: float
    k_lo: int
    k_hi: int
    K: int
    kernel: str = "dirichlet"      # "dirichlet" (Eq.B2) | "fresnel" (Eq.28/29)
    pn1: int = 0                   # 0: 0PN, 1: 0PN+1PN
    response: str = "none"         # "none" | "table" | "annual"
    f_lo: float = 0.0
    f_hi: float = np.inf
    f_ref: float = 1.0
    resp_period: float = YEAR_S
    resp_depth: float = 0.3
    resp_psi: tuple = (0.0, 0.0)
    resp_chi: tuple = (0.0, 0.0)
    include_dc: int = 0            # 0: bins k < 1 never contribute (reading A6); 1: k = 0 counts ("d~[k] = 0 for k < 0")

    @property
    def n_samp(self):
        n = self.t_sft * self.fs
        assert abs(n - round(n)) < 1e-9, "t_sft*fs must be an integer (P:157)"
        return int(round(n))


@dataclass
class Store:
    """Data SFTs as handed to ``sft_load_data``: un-whitened bins + the noise description."""
    bins: np.ndarray                 # [C][N_SFT][k_hi-k_lo] complex, x~ of Eq.(26)
    psd_scale: np.ndarray            # [C][N_SFT] s_{c,a}; <=0 or non-finite => gap
    psd_shape: np.ndarray            # [C][k_hi-k_lo] S_c(f_k)
    response: np.ndarray = None      # [C][N_SFT] complex R_{c,a} for response == "table"

    def present(self):
        s = np.asarray(self.psd_scale, dtype=np.float64)
        return np.isfinite(s) & (s > 0.0)


# ---------------------------------------------------------------------------------------------
def sft_times(plan):
    """t_a = t0 + a T_SFT."""
    return plan.t0 + np.arange(plan.n_sft, dtype=np.float64) * plan.t_sft


def track(plan, p):
    """Step 1: ``{A, phi, f, fdot}`` at every SFT start for one parameter row ``p``
    = (m_chirp, eta, t_c, phi_c, amp, lambda, beta, -)."""
    t = sft_times(plan)
    phi, f, fdot = wf.taylor_t3(p[0], p[1], p[2], p[3], t, plan.pn1)
    A = wf.amplitude(p[4], f, plan.f_ref)
    return t, A, phi, f, fdot


def select_bins(plan, t, f, fdot, t_c):
    """Steps 2 + activity mask (readings A5, A12).

    ``y = f_a T`` (Dirichlet) or ``(f_a + fdot_a T/2) T`` (Fresnel: centre of the swept band);
    ``k_c = floor(y + 1/2)``; ``x = f_a T - k_c``; ``b = fdot_a T^2``.
    Active iff ``f_lo <= f_a``, ``f_a + fdot_a T <= f_hi`` and ``t_a + T < t_c``.
    """
    T = plan.t_sft
    with np.errstate(invalid="ignore"):
        fT = f * T
        b = fdot * T * T
        y = fT + (0.5 * b if plan.kernel.startswith("fresnel") else 0.0)
        yh = y + 0.5
        k_c = np.floor(yh)
        x = fT - k_c
        tau = t_c - t
        active = (tau > T) & (fT >= plan.f_lo * T) & (fT + b <= plan.f_hi * T)
        active &= np.isfinite(fT)
        flags = np.zeros(t.shape, dtype=np.uint8)
        flags[np.abs(yh - np.round(yh)) < TIE_EPS] |= FLAG_KC_TIE
        near = (np.abs(tau - T) < TIE_EPS * T) | (np.abs(fT - plan.f_lo * T) < TIE_EPS) \
            | (np.abs(fT + b - plan.f_hi * T) < TIE_EPS)
        flags[near] |= FLAG_MASK_TIE
    k_c = np.where(active, k_c, -1).astype(np.int64)
    return k_c, x, b, active, flags


def response_factor(plan, store, p, t):
    """Step 3's ``R_{c,a}`` with ``Lambda z = Re[R z]``, constant over an SFT.

    "none": 1.  "table": ``store.response``.  "annual" (D4, synthetic stand-in in the
    spirit of Eq.(40)-(41) P:332-334): ``[1 + depth cos(2 pi t_a/period + psi_c + lambda)] e^{i(chi_c + beta)}``.
    """
    C, N = plan.n_channels, plan.n_sft
    if plan.response == "none":
        return np.ones((C, N), dtype=np.complex128)
    if plan.response == "table":
        return np.asarray(store.response, dtype=np.complex128)
    if plan.response == "annual":
        lam, beta = p[5], p[6]
        R = np.empty((C, N), dtype=np.complex128)
        for c in range(C):
            amp = 1.0 + plan.resp_depth * np.cos(2.0 * np.pi * t / plan.resp_period + plan.resp_psi[c] + lam)
            R[c] = amp * np.exp(1j * (plan.resp_chi[c] + beta))
        return R
    raise ValueError(plan.response)


def kernel_coefficients(plan, x, b):
    """F(a_m, b) for m = -K..K, a_m = x - m.  [N] -> [N][2K+1]."""
    m = np.arange(-plan.K, plan.K + 1, dtype=np.float64)
    a = x[:, None] - m[None, :]
    if plan.kernel == "dirichlet":
        return kern.dirichlet(a)
    if plan.kernel == "fresnel":
        return kern.fre_closed(a, b[:, None])
    if plan.kernel == "fresnel_quadrature":      # slow path: the definition Eq.(28)
        return kern.fre_quadrature(a, b[:, None])
    raise ValueError(plan.kernel)


def band_terms(plan, store, p):
    """Per-(channel, SFT) terms of steps 1-4 for one template (parameter row ``p``).

    Returns ``Z[C][N]`` (complex, ``xh = sum Re Z``), ``H[C][N]`` (``hh = sum H``),
    ``k_c[N]`` (-1 inactive), ``act[C][N]`` and ``flags[N]``.
    """
    t, A, phi, f, fdot = track(plan, p)
    R = response_factor(plan, store, p, t)
    return band_terms_from_track(plan, store, t, A, phi, f, fdot, p[2], R)


def band_terms_from_track(plan, store, t, A, phi, f, fdot, t_c, R):
    """Steps 2-4 for ANY per-SFT track ``{A_a, phi_a, f_a, fdot_a}`` (the paper's interface,
    P:164: "described by 4 numbers") and response ``R[C][N]``."""
    C, N, K, T = plan.n_channels, plan.n_sft, plan.K, plan.t_sft
    n = plan.n_samp
    k_c, x, b, active, flags = select_bins(plan, t, f, fdot, t_c)
    present = store.present()
    Z = np.zeros((C, N), dtype=np.complex128)
    H = np.zeros((C, N), dtype=np.float64)
    act = present & active[None, :]
    idx = np.nonzero(active)[0]
    if idx.size == 0:
        return Z, H, k_c, act, flags
    Fk = kernel_coefficients(plan, x[idx], b[idx])                    # [n_act][2K+1]
    m = np.arange(-K, K + 1, dtype=np.int64)
    k = k_c[idx][:, None] + m[None, :]                                # absolute bin index
    valid = (k >= (0 if plan.include_dc else 1)) & (k <= n // 2 - 1) & (k >= plan.k_lo) & (k < plan.k_hi)   # reading A6
    col = np.clip(k - plan.k_lo, 0, plan.k_hi - plan.k_lo - 1)
    pref = A[idx] * np.exp(1j * phi[idx])                             # A_a e^{i phi_a}
    for c in range(C):
        pc = present[c][idx]
        xt = np.asarray(store.bins[c], dtype=np.complex128)[idx[:, None], col]
        with np.errstate(divide="ignore", invalid="ignore"):
            S = np.asarray(store.psd_scale[c], np.float64)[idx][:, None] * \
                np.asarray(store.psd_shape[c], np.float64)[col]
            invS = np.where(valid & pc[:, None], 1.0 / S, 0.0)
        xt = np.where(invS > 0.0, xt, 0.0)
        Rc = R[c][idx]
        Z[c, idx] = 2.0 * pref * Rc * np.sum(np.conj(xt) * invS * Fk, axis=1)
        H[c, idx] = T * (A[idx] * np.abs(Rc)) ** 2 * np.sum(np.abs(Fk) ** 2 * invS, axis=1)
    return Z, H, k_c, act, flags


def inner_products(plan, store, params):
    """``([x,h])``, ``([h,h])`` for every parameter row.  Returns a dict with
    ``xh``, ``hh``, ``xh_im`` [T]; ``kc`` [T][C][N] (int32, -1 inactive/gap); ``flags`` [T][N]."""
    params = np.atleast_2d(np.asarray(params, dtype=np.float64))
    nt = params.shape[0]
    xh = np.zeros(nt)
    hh = np.zeros(nt)
    xi = np.zeros(nt)
    kc = np.full((nt, plan.n_channels, plan.n_sft), -1, dtype=np.int32)
    flags = np.zeros((nt, plan.n_sft), dtype=np.uint8)
    for i in range(nt):
        Z, H, k_c, act, fl = band_terms(plan, store, params[i])
        xh[i] = np.sum(Z.real)
        xi[i] = np.sum(Z.imag)
        hh[i] = np.sum(H)
        kc[i] = np.where(act, k_c[None, :], -1)
        flags[i] = fl
    return dict(xh=xh, hh=hh, xh_im=xi, kc=kc, flags=flags)


def cumulative_snr(plan, store, params):
    """Step 5: inclusive prefix sums over the SFT index of the per-SFT terms (summed over
    channels); ``snr = cum_xh / sqrt(cum_hh)`` (0 where ``cum_hh == 0``).  [T][N] each."""
    params = np.atleast_2d(np.asarray(params, dtype=np.float64))
    nt = params.shape[0]
    cx = np.zeros((nt, plan.n_sft))
    ch = np.zeros((nt, plan.n_sft))
    for i in range(nt):
        Z, H, _, _, _ = band_terms(plan, store, params[i])
        cx[i] = np.cumsum(np.sum(Z.real, axis=0))
        ch[i] = np.cumsum(np.sum(H, axis=0))
    with np.errstate(divide="ignore", invalid="ignore"):
        snr = np.where(ch > 0.0, cx / np.sqrt(ch), 0.0)
    return dict(snr=snr, cum_xh=cx, cum_hh=ch)


def xx_band(plan, store):
    """<x,x> restricted to the stored band: 4 df sum |x~|^2/S over present SFTs and valid bins."""
    n = plan.n_samp
    k = np.arange(plan.k_lo, plan.k_hi)
    valid = (k >= (0 if plan.include_dc else 1)) & (k <= n // 2 - 1)
    present = store.present()
    tot = 0.0
    for c in range(plan.n_channels):
        with np.errstate(divide="ignore", invalid="ignore"):
            S = np.asarray(store.psd_scale[c], np.float64)[:, None] * np.asarray(store.psd_shape[c], np.float64)[None, :]
            w = np.where(valid[None, :] & present[c][:, None], 1.0 / S, 0.0)
        tot += 4.0 / plan.t_sft * float(np.sum(np.abs(np.asarray(store.bins[c], np.complex128)) ** 2 * w))
    return tot


def validity(plan, params):
    """Eq.(33)-(34) P:244-248 per template: ``delta_eff = 1/2 T_SFT^3 max_a fddot_a`` over the template's active SFTs (the
    delta at which Eq.(33) ``1/2 T^2 max fddot <= delta df`` holds with equality on the plan's SFT length); 0 where no SFT is
    active.  [T]"""
    params = np.atleast_2d(np.asarray(params, dtype=np.float64))
    t = sft_times(plan)
    out = np.zeros(params.shape[0])
    for i, p in enumerate(params):
        phi, f, fdot = wf.taylor_t3(p[0], p[1], p[2], p[3], t, plan.pn1)
        _, _, _, active, _ = select_bins(plan, t, f, fdot, p[2])
        if active.any():
            with np.errstate(invalid="ignore"):
                fdd = wf.taylor_t3_fddot(p[0], p[1], p[2], t, plan.pn1)
            out[i] = 0.5 * plan.t_sft ** 3 * np.max(fdd[active])
    return out
