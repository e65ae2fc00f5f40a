"""Seeded synthetic inputs shaped like the paper's workloads (ET-BNS §IV.B, LISA-MBHB
§IV.C) for BASELINE.json's five configs.  Recipe: DESIGN.md §5.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic: no SFT kernel, no bin selection, no per-SFT signal model, no inner
product.  What it does hold is the *data recipe*: Gaussian noise with a given PSD, a
continuously sampled inspiral strain added to it (the signal that is "in the data", evaluated
at every sample, not the per-SFT approximation of Eq.(16)-(19)), numpy FFTs of the segments
(SFT generation is harness work), gaps, per-SFT PSD scales, and the template
bank's parameter rows.  numpy only; no torch, no CUDA, no oracle import.

Parameter row layout (8 doubles): m_chirp[Msun], eta, t_c[s], phi_c[rad], amp, lambda, beta, 0.
"""
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field
import os
import numpy as np

GMSUN_S = 4.925491025543576e-6   # G Msun / c^3 [s]
YEAR_S = 31557600.0
NPARAM = 8


# --------------------------------------------------------------------------------------------
# the signal that is put into the data: a continuously sampled PN inspiral strain
# --------------------------------------------------------------------------------------------
def _pn_coeffs(eta, pn1):
    """1PN coefficients (pn1 >= 1) of phase and frequency, and the 1.5PN tail coefficients (pn1 >= 2)."""
    p1, p15 = float(pn1 >= 1), float(pn1 >= 2)
    return (p1 * (3715.0 / 8064.0 + 55.0 / 96.0 * eta), p1 * (743.0 / 2688.0 + 11.0 / 32.0 * eta),
            -0.75 * np.pi * p15, -0.3 * np.pi * p15)


def inspiral_phase_freq(t, m_chirp, eta, t_c, phi_c, pn1):
    """phi(t) [rad] and f(t) [Hz] of the injected inspiral at sample times t < t_c."""
    M = m_chirp * eta ** (-0.6) * GMSUN_S
    cphi, cf, tphi, tf = _pn_coeffs(eta, pn1)
    L = np.log(eta * (t_c - t) / (5.0 * M))
    q = np.exp(-0.25 * L)
    q15 = np.exp(-0.375 * L)
    phi = phi_c - (2.0 / eta) * np.exp(0.625 * L) * (1.0 + cphi * q + tphi * q15)
    f = q15 / (8.0 * np.pi * M) * (1.0 + cf * q + tf * q15)
    return phi, f


def inspiral_strain(t, p, f_ref, pn1, resp=None):
    """h(t) = Re[R(t) A(t) e^{i phi(t)}], A = amp (f/f_ref)^{2/3}; R = 1 if ``resp`` is None,
    else ``resp(t)`` (complex).  Zero at and after t_c."""
    t = np.asarray(t, dtype=np.float64)
    ok = t < p[2]
    tt = np.where(ok, t, p[2] - 1.0)
    phi, f = inspiral_phase_freq(tt, p[0], p[1], p[2], p[3], pn1)
    A = p[4] * (f / f_ref) ** (2.0 / 3.0)
    if resp is None:
        h = A * np.cos(phi)
    else:
        h = np.real(resp(tt) * A * np.exp(1j * phi))
    return np.where(ok, h, 0.0)


def tau_for_frequency(f_target, m_chirp, eta, pn1):
    """Time before coalescence at which the injected inspiral has GW frequency f_target (bisection)."""
    lo, hi = 1e-6, 1e12
    for _ in range(200):
        mid = np.sqrt(lo * hi)
        _, f = inspiral_phase_freq(np.float64(0.0), m_chirp, eta, mid, 0.0, pn1)
        if f > f_target:
            lo = mid
        else:
            hi = mid
    return float(np.sqrt(lo * hi))


# --------------------------------------------------------------------------------------------
@dataclass
class Workload:
    """One synthetic problem: what ``sft_plan_create`` / ``sft_load_data`` / ``sft_inner_products``
    receive (and, identically, what the oracle receives)."""
    name: str
    desc: dict                      # plan fields (see include/sft.h :: sft_plan_desc)
    bins: np.ndarray                # [C][N_SFT][k_hi-k_lo] complex64, x~ of Eq.(26) (strain*s)
    psd_scale: np.ndarray           # [C][N_SFT] float64, s_{c,a}; 0 => gap
    psd_shape: np.ndarray           # [C][k_hi-k_lo] float64, S_c(f_k)
    params: np.ndarray              # [n_templates][8] float64
    response: np.ndarray = None     # [C][N_SFT] complex64 or None
    injection: np.ndarray = None    # the parameter row of the injected signal
    series: np.ndarray = None       # [C][N0] float64 time series when the config is small enough
    notes: dict = field(default_factory=dict)

    @property
    def n_templates(self):
        return self.params.shape[0]


def _rows(n):
    return np.zeros((n, NPARAM), dtype=np.float64)


def _segment_rfft_bins(x_seg, dt, k_lo, k_hi):
    """numpy FFT of [.., n] segments -> dt * rfft, bins [k_lo, k_hi)."""
    return dt * np.fft.rfft(x_seg, axis=-1)[..., k_lo:k_hi]


# --------------------------------------------------------------------------------------------
# config 1: tiny single-detector chirp
# --------------------------------------------------------------------------------------------
def config1(n_templates=64, variant="F"):
    """BASELINE.json configs[0].  2048 s of unit white noise at 512 Hz (seed 0) + one 0PN chirp
    (Mc 1.2, amp 0.5 at f_ref = 20 Hz, phase from seed 1); 256 rectangular SFTs of 8 s; flat
    PSD S = 2/fs; 64 templates (seed 2); K = 4.  Variant "F" (full span, D0): t_c =
    2048 s + 216 s so the signal sweeps 7.4 -> 18 Hz across the whole data set and every SFT is
    active; variant "M" keeps the same data but sets f_lo = 12 Hz so only the tail is active."""
    fs, T, N0 = 512.0, 8.0, 1 << 20
    n = int(T * fs)
    n_sft = N0 // n
    k_lo, k_hi, K = 48, 168, 4
    f_ref = 20.0
    x = np.random.default_rng(0).standard_normal(N0)
    inj = np.zeros(NPARAM)
    inj[:5] = [1.2, 0.25, N0 / fs + 216.0, np.random.default_rng(1).uniform(0.0, 2.0 * np.pi), 0.5]
    t = np.arange(N0, dtype=np.float64) / fs
    x = x + inspiral_strain(t, inj, f_ref, 0)
    bins = _segment_rfft_bins(x.reshape(n_sft, n), 1.0 / fs, k_lo, k_hi)[None].astype(np.complex64)
    rng = np.random.default_rng(2)
    P = _rows(n_templates)
    P[:] = inj
    P[:, 0] *= 1.0 + 1e-4 * rng.standard_normal(n_templates)
    P[:, 2] += 1e-3 * rng.standard_normal(n_templates)
    P[:, 3] = rng.uniform(0.0, 2.0 * np.pi, n_templates)
    P[0] = inj                                            # template 0 is the injected signal
    desc = dict(n_channels=1, n_sft=n_sft, t_sft=T, fs=fs, t0=0.0, k_lo=k_lo, k_hi=k_hi, K=K,
                kernel="fresnel", pn1=0, response="none",
                f_lo=5.0 if variant == "F" else 12.0, f_hi=30.0, f_ref=f_ref)
    return Workload(name=f"config1-{variant}", desc=desc, bins=bins,
                    psd_scale=np.ones((1, n_sft)), psd_shape=np.full((1, k_hi - k_lo), 2.0 / fs),
                    params=P, injection=inj, series=x[None])


# --------------------------------------------------------------------------------------------
# configs 2, 3, 5: ET-like BNS bank
# --------------------------------------------------------------------------------------------
def et_psd(f):
    """S(f) = S0[(f/10)^-4 + 2 + (f/100)^2], S0 = 1e-49 (BASELINE.json configs[1])."""
    f = np.asarray(f, dtype=np.float64)
    return 1e-49 * ((f / 10.0) ** -4 + 2.0 + (f / 100.0) ** 2)


def et_bns(n_templates=4096, n_sft=10800, K=8, fs=2048.0, T=8.0, tau_end=129.0, bank_seed=5,
           inject=True, snr=30.0, kernel="fresnel", gap_fraction=0.1, variant="F", name=None,
           threads=None):
    """BASELINE.json configs[1] (and [2], [4] through the arguments).  Noise: per SFT, band bins
    drawn directly in the frequency domain, X_k ~ CN(0, s_a S(f_k) T/2) (stationary inside an
    SFT; lognormal s_a, sigma 0.2, seed 3; noise seed 30).  Gaps: ``gap_fraction`` of the SFTs
    removed (seed 4; psd_scale = 0, bins = 0).  Signal: 1.4+1.4 Msun 0PN+1PN strain sampled at
    ``fs`` over every SFT, numpy rfft, scaled to band SNR ``snr`` against s_a S(f_k).  Variant "F":
    t_c = T_obs + tau_end so that the signal spans the whole data set (f(0) = 1.88 Hz, b = fdot
    T^2 ~ 4 in the last SFT for the defaults) and plan f_lo = 0; variant "M": f_lo = 5 Hz.
    Bank: uniform box +-1e-3 (fractional in Mc and eta, eta clipped to 1/4; absolute s / rad in
    t_c, phi_c); row 0 is the injected signal."""
    n = int(round(T * fs))
    dt = 1.0 / fs
    T_obs = n_sft * T
    f_ref, pn1 = 10.0, 1
    m1 = m2 = 1.4
    eta = m1 * m2 / (m1 + m2) ** 2
    mc = (m1 + m2) * eta ** 0.6
    inj = np.zeros(NPARAM)
    inj[:5] = [mc, eta, T_obs + tau_end, 1.0, 1.0]
    # stored band from the injected track (+ margin)
    _, f0 = inspiral_phase_freq(np.float64(0.0), mc, eta, inj[2], 0.0, pn1)
    _, f1 = inspiral_phase_freq(np.float64(T_obs), mc, eta, inj[2], 0.0, pn1)
    k_lo = max(0, int(np.floor(f0 * T)) - K - 2)
    k_hi = int(np.ceil(f1 * T)) + K + 4
    nb = k_hi - k_lo
    fk = np.arange(k_lo, k_hi) / T
    S = et_psd(np.maximum(fk, 0.5 / T))
    s = np.exp(0.2 * np.random.default_rng(3).standard_normal(n_sft))
    gaps = np.random.default_rng(4).permutation(n_sft)[: int(round(gap_fraction * n_sft))]
    s[gaps] = 0.0
    rng = np.random.default_rng(30)
    noise = rng.standard_normal((n_sft, nb, 2)).view(np.complex128)[..., 0]
    noise *= np.sqrt(s[:, None] * S[None, :] * T / 4.0)
    sig = np.zeros((n_sft, nb), dtype=np.complex128)
    if inject:
        blk = 64
        starts = list(range(0, n_sft, blk))
        tau_j = np.arange(n, dtype=np.float64) * dt

        def work(a0):
            a1 = min(a0 + blk, n_sft)
            t = (np.arange(a0, a1, dtype=np.float64) * T)[:, None] + tau_j[None, :]
            return a0, a1, _segment_rfft_bins(inspiral_strain(t, inj, f_ref, pn1), dt, k_lo, k_hi)

        nthr = threads or min(16, len(os.sched_getaffinity(0)))
        with ThreadPoolExecutor(nthr) as ex:
            for a0, a1, hb in ex.map(work, starts):
                sig[a0:a1] = hb
        pres = s > 0.0
        rho2 = 4.0 / T * np.sum(np.abs(sig[pres]) ** 2 / (s[pres][:, None] * S[None, :]))
        inj[4] = snr / np.sqrt(rho2)
        sig *= inj[4]
    bins = noise + sig
    bins[s <= 0.0] = 0.0
    rng = np.random.default_rng(bank_seed)
    P = _rows(n_templates)
    P[:] = inj
    u = rng.uniform(-1e-3, 1e-3, (n_templates, 4))
    P[:, 0] *= 1.0 + u[:, 0]
    P[:, 1] = np.minimum(P[:, 1] * (1.0 + u[:, 1]), 0.25)
    P[:, 2] += u[:, 2]
    P[:, 3] += u[:, 3]
    P[0] = inj
    desc = dict(n_channels=1, n_sft=n_sft, t_sft=T, fs=fs, t0=0.0, k_lo=k_lo, k_hi=k_hi, K=K,
                kernel=kernel, pn1=pn1, response="none",
                f_lo=0.0 if variant == "F" else 5.0, f_hi=f1 + 2.0, f_ref=f_ref)
    return Workload(name=name or f"config2-{variant}", desc=desc,
                    bins=bins[None].astype(np.complex64), psd_scale=s[None], psd_shape=S[None],
                    params=P, injection=inj, notes=dict(n_gaps=int(len(gaps)), f_start=float(f0), f_end=float(f1)))


def et_bns_bank(w, n_templates, bank_seed=55):
    """The data of ``w`` (an ``et_bns`` workload) with a different bank size (config 5's template axis)."""
    import copy
    rng = np.random.default_rng(bank_seed)
    P = _rows(n_templates)
    P[:] = w.injection
    u = rng.uniform(-1e-3, 1e-3, (n_templates, 4))
    P[:, 0] *= 1.0 + u[:, 0]
    P[:, 1] = np.minimum(P[:, 1] * (1.0 + u[:, 1]), 0.25)
    P[:, 2] += u[:, 2]
    P[:, 3] += u[:, 3]
    P[0] = w.injection
    w2 = copy.copy(w)
    w2.params = P
    return w2


def et_bns_wide_bank(w, n_templates, bank_seed=56):
    """The data of ``w`` (an ``et_bns`` workload) with a WIDE, shuffled bank: chirp mass +-10 %, eta in [0.2, 0.25],
    coalescence times from a third of the way through the data to 3000 s after its end, phases uniform.  Neighbouring
    rows (the 32 templates a warp holds) then sit at different bins (tens of bins apart), at different drifts b = fdot T^2
    (0.01 ... > 4), and some are ended, out of band or not yet in band at the same SFT.  Row 0 stays the injected signal."""
    import copy
    rng = np.random.default_rng(bank_seed)
    T_obs = w.desc["n_sft"] * w.desc["t_sft"]
    P = _rows(n_templates)
    P[:] = w.injection
    P[:, 0] *= 1.0 + rng.uniform(-0.1, 0.1, n_templates)
    P[:, 1] = rng.uniform(0.2, 0.25, n_templates)
    P[:, 2] = rng.uniform(T_obs / 3.0, T_obs + 3000.0, n_templates)
    P[:, 3] = rng.uniform(0.0, 2.0 * np.pi, n_templates)
    P[0] = w.injection
    w2 = copy.copy(w)
    w2.params = P
    return w2


def config2(**kw):
    return et_bns(**kw)


def config3(n_templates=16384, **kw):
    """BASELINE.json configs[2]: config-2 data, 16,384 templates (seed 6), cumulative output."""
    kw.setdefault("bank_seed", 6)
    kw.setdefault("name", "config3-F")
    return et_bns(n_templates=n_templates, **kw)


def config3_check_indices(n_templates, n_sft, per_template=32):
    """The 32 seeded SFT indices per template at which config 3 is compared (seed 7)."""
    return np.random.default_rng(7).integers(0, n_sft, size=(n_templates, per_template))


# --------------------------------------------------------------------------------------------
# config 4: LISA-like massive BBH, two channels, annual modulation
# --------------------------------------------------------------------------------------------
def lisa_psd(f):
    """S(f) = S0 [1 + (2e-3/f)^4] (1 + (f/0.03)^2), S0 = 1e-40 (BASELINE.json configs[3])."""
    f = np.asarray(f, dtype=np.float64)
    return 1e-40 * (1.0 + (2e-3 / f) ** 4) * (1.0 + (f / 0.03) ** 2)


def config4(n_templates=65536, snr=50.0):
    """BASELINE.json configs[3].  Two channels (A, E), 28 d at 0.2 Hz, 672 SFTs of 3600 s per
    channel (n = 720); noise per SFT in the frequency domain from lisa_psd (seeds 8, 9); signal:
    M = 1e6 Msun, q = 0.5, 0PN+1PN, reaching 1.9 mHz at the end of the data, with the response
    R_c(t) = [1 + 0.3 cos(2 pi t/yr + psi_c + lambda)] e^{i(chi_c + beta)}, psi = (0, pi/2),
    chi = (0, pi/2), evaluated at every sample (D4).  Bank (seed 10): Mc, eta in a
    +-1e-3 fractional box, t_c +- 10 s, phi_c uniform, lambda uniform in [0, 2 pi), sin(beta)
    uniform; row 0 is the injected signal.  K = 16: the band clips at k < 1."""
    fs, T, n_sft, C = 0.2, 3600.0, 672, 2
    n = int(round(T * fs))
    dt = 1.0 / fs
    T_obs = n_sft * T
    K, k_lo, k_hi = 16, 0, 40
    f_ref, pn1 = 1e-3, 1
    q = 0.5
    eta = q / (1.0 + q) ** 2
    mc = 1e6 * eta ** 0.6
    psi = (0.0, np.pi / 2)
    chi = (0.0, np.pi / 2)
    tau_end = tau_for_frequency(1.9e-3, mc, eta, pn1)
    inj = np.zeros(NPARAM)
    inj[:7] = [mc, eta, T_obs + tau_end, 2.0, 1.0, 0.7, -0.3]
    fk = np.arange(k_lo, k_hi) / T
    S = lisa_psd(np.maximum(fk, 0.5 / T))
    t = np.arange(n_sft * n, dtype=np.float64) * dt
    bins = np.zeros((C, n_sft, k_hi - k_lo), dtype=np.complex128)
    sig = np.zeros_like(bins)
    for c in range(C):
        rng = np.random.default_rng(8 + c)
        nz = rng.standard_normal((n_sft, k_hi - k_lo, 2)).view(np.complex128)[..., 0]
        bins[c] = nz * np.sqrt(S[None, :] * T / 4.0)

        def resp(tt, c=c):
            return (1.0 + 0.3 * np.cos(2.0 * np.pi * tt / YEAR_S + psi[c] + inj[5])) * np.exp(1j * (chi[c] + inj[6]))

        h = inspiral_strain(t, inj, f_ref, pn1, resp)
        sig[c] = _segment_rfft_bins(h.reshape(n_sft, n), dt, k_lo, k_hi)
    valid = (np.arange(k_lo, k_hi) >= 1)
    rho2 = 4.0 / T * np.sum(np.abs(sig[:, :, valid]) ** 2 / S[None, None, valid])
    inj[4] = snr / np.sqrt(rho2)
    bins += inj[4] * sig
    rng = np.random.default_rng(10)
    P = _rows(n_templates)
    P[:] = inj
    u = rng.uniform(-1.0, 1.0, (n_templates, 6))
    P[:, 0] *= 1.0 + 1e-3 * u[:, 0]
    P[:, 1] = np.minimum(P[:, 1] * (1.0 + 1e-3 * u[:, 1]), 0.25)
    P[:, 2] += 10.0 * u[:, 2]
    P[:, 3] = np.pi * (1.0 + u[:, 3])
    P[:, 5] = np.pi * (1.0 + u[:, 4])
    P[:, 6] = np.arcsin(u[:, 5])
    P[0] = inj
    desc = dict(n_channels=C, n_sft=n_sft, t_sft=T, fs=fs, t0=0.0, k_lo=k_lo, k_hi=k_hi, K=K,
                kernel="fresnel", pn1=pn1, response="annual", f_lo=0.0, f_hi=3e-3, f_ref=f_ref,
                resp_period=YEAR_S, resp_depth=0.3, resp_psi=psi, resp_chi=chi)
    return Workload(name="config4", desc=desc, bins=bins.astype(np.complex64),
                    psd_scale=np.ones((C, n_sft)), psd_shape=np.stack([S, S]), params=P, injection=inj,
                    notes=dict(tau_end=tau_end))


# --------------------------------------------------------------------------------------------
# accuracy experiment of section IV: a noiseless fiducial signal, r(delta, Delta k) of Eq.(36)
# --------------------------------------------------------------------------------------------
ACCURACY_EXAMPLES = {
    # name: (m1, m2 [Msun], f_start, f_end [Hz], fs [Hz], modulation period [s])
    "bns": (1.4, 1.4, 1.0, 10.0, 40.0, 86400.0),
    "mbhb": (1e6, 1e6, 1e-4, 1.9e-3, 2.0, YEAR_S),
}


def accuracy_case(example, t_sft, K, f_start=None, pn1=1, kernel="fresnel"):
    """One point of the paper's accuracy maps (Fig. 3 / Fig. 4) with this library's PN waveform in place of
    IMRPhenomT (W1): the fiducial signal of section IV.B (``"bns"``: 1.4+1.4 Msun, 1 -> 10 Hz, fs = 40 Hz, daily
    modulation) or IV.C (``"mbhb"``: 1e6+1e6 Msun, 1e-4 -> 1.9e-3 Hz, fs = 2 Hz, yearly modulation),
    observed with the projector Lambda_t = [a(t) + b(t)](Re + Im), a = cos(2 pi t/P), b = sin(2 pi t/P), c_nu = 1
    (Eq.(37)-(41)), i.e. h(t) = Re[R(t) A(t) e^{i phi(t)}] with R = (a + b)(1 - i) applied at every sample.  No noise, flat
    PSD S = 1 (the experiment measures the loss of ([d,h]) against <d,h> for d = h).  ``t_sft`` is rounded to an even
    number of samples; ``f_start`` above the example's own start shortens the signal (tests).  The template (row 0 of
    ``params``) is the fiducial signal; its response table holds R at the SFT starts.
    Returns a Workload whose ``series`` is the sampled signal over the whole SFTs and ``notes["xx_time"]`` the exact
    time-domain product (2 dt / S) sum_j h_j^2 over the same samples (Eq.(1)/(14) for a flat PSD)."""
    m1, m2, f0, f1, fs, period = ACCURACY_EXAMPLES[example]
    if f_start is not None:
        f0 = float(f_start)
    eta = m1 * m2 / (m1 + m2) ** 2
    mc = (m1 + m2) * eta ** 0.6
    dt = 1.0 / fs
    n = 2 * int(round(0.5 * t_sft * fs))
    T = n * dt
    tau0, tau1 = tau_for_frequency(f0, mc, eta, pn1), tau_for_frequency(f1, mc, eta, pn1)
    n_sft = int((tau0 - tau1) // T)
    T_obs = n_sft * T
    inj = np.zeros(NPARAM)
    inj[:5] = [mc, eta, tau0, 0.7, 1.0]                      # t = 0 at f_start; the data end where f_end is reached
    f_ref = f1

    def resp(tt):
        ph = 2.0 * np.pi * tt / period
        return (np.cos(ph) + np.sin(ph)) * (1.0 - 1.0j)

    t = np.arange(n_sft * n, dtype=np.float64) * dt
    h = inspiral_strain(t, inj, f_ref, pn1, resp)
    _, fe = inspiral_phase_freq(np.float64(T_obs), mc, eta, inj[2], 0.0, pn1)
    k_lo = max(0, int(np.floor(f0 * T)) - K - 2)
    k_hi = min(n // 2, int(np.ceil(fe * T)) + K + 4)
    bins = _segment_rfft_bins(h.reshape(n_sft, n), dt, k_lo, k_hi)[None].astype(np.complex64)
    R = resp(np.arange(n_sft, dtype=np.float64) * T)[None].astype(np.complex64)
    desc = dict(n_channels=1, n_sft=n_sft, t_sft=T, fs=fs, t0=0.0, k_lo=k_lo, k_hi=k_hi, K=K, kernel=kernel, pn1=pn1,
                response="table", f_lo=0.0, f_hi=1e9, f_ref=f_ref)
    return Workload(name=f"accuracy-{example}", desc=desc, bins=bins, psd_scale=np.ones((1, n_sft)),
                    psd_shape=np.ones((1, k_hi - k_lo)), params=inj[None].copy(), response=R, injection=inj, series=h[None],
                    notes=dict(xx_time=2.0 * dt * float(np.dot(h, h)), n=n, t_obs=T_obs, f_end=float(fe)))


# --------------------------------------------------------------------------------------------
# F-statistic test case: a long signal with resolvable amplitude modulation, Eq.(10)-(12) P:107-118
# --------------------------------------------------------------------------------------------
def fstat_case(c_nu=(0.7, -0.4, 0.5, 0.9), n_templates=8, n_channels=1, noise=0.0, seed=12, K=6):
    """A 0PN+1PN chirp (Mc 1.2, 7.4 -> 18 Hz over 2048 s, fs = 512 Hz: config 1's track) observed through the antenna-pattern
    functions a_c(t) = cos(2 pi t/P + 0.4 c), b_c(t) = sin(2 pi t/P + 0.3 + 0.9 c), P = 3000 s (both vary by O(1) over the
    data, so that the two polarisations are resolvable), with amplitudes ``c_nu`` of Eq.(10): h = sum_nu c_nu h_nu,
    h_nu as in Eq.(11), evaluated at EVERY sample.  Optional white noise of standard deviation ``noise`` (seed); flat PSD
    S = 2 noise^2 / fs (1 if noise = 0).  Bank: row 0 = the signal's intrinsic parameters, the rest perturbed as in config 1.
    The Workload's ``response`` holds (a + i b) at the SFT starts: the pair (a, b) that ``sft_fstat`` reads."""
    fs, T, N0 = 512.0, 8.0, 1 << 20
    n = int(T * fs)
    n_sft = N0 // n
    k_lo, k_hi = 40, 176
    f_ref, P_mod = 20.0, 3000.0
    inj = np.zeros(NPARAM)
    inj[:5] = [1.2, 0.25, N0 / fs + 216.0, 1.3, 1.0]
    t = np.arange(N0, dtype=np.float64) / fs
    c = np.asarray(c_nu, dtype=np.float64)
    rng = np.random.default_rng(seed)
    bins, resp_tab, series = [], [], []
    for ch in range(n_channels):
        a = lambda tt, ch=ch: np.cos(2.0 * np.pi * tt / P_mod + 0.4 * ch)
        b = lambda tt, ch=ch: np.sin(2.0 * np.pi * tt / P_mod + 0.3 + 0.9 * ch)
        x = inspiral_strain(t, inj, f_ref, 1, lambda tt: (c[0] * a(tt) + c[1] * b(tt)) - 1j * (c[2] * a(tt) + c[3] * b(tt)))
        if noise > 0.0:
            x = x + noise * rng.standard_normal(N0)
        series.append(x)
        bins.append(_segment_rfft_bins(x.reshape(n_sft, n), 1.0 / fs, k_lo, k_hi))
        ta = np.arange(n_sft, dtype=np.float64) * T
        resp_tab.append(a(ta) + 1j * b(ta))
    rng = np.random.default_rng(seed + 1)
    Pm = _rows(n_templates)
    Pm[:] = inj
    Pm[:, 0] *= 1.0 + 1e-4 * rng.standard_normal(n_templates)
    Pm[:, 2] += 1e-3 * rng.standard_normal(n_templates)
    Pm[:, 3] = rng.uniform(0.0, 2.0 * np.pi, n_templates)
    Pm[0] = inj
    S = 2.0 * noise * noise / fs if noise > 0.0 else 1.0
    desc = dict(n_channels=n_channels, n_sft=n_sft, t_sft=T, fs=fs, t0=0.0, k_lo=k_lo, k_hi=k_hi, K=K, kernel="fresnel", pn1=1,
                response="table", f_lo=5.0, f_hi=30.0, f_ref=f_ref)
    return Workload(name="fstat", desc=desc, bins=np.stack(bins).astype(np.complex64), psd_scale=np.ones((n_channels, n_sft)),
                    psd_shape=np.full((n_channels, k_hi - k_lo), S), params=Pm, response=np.stack(resp_tab).astype(np.complex64),
                    injection=inj, series=np.stack(series), notes=dict(c_nu=c, S=S))
