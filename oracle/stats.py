"""Oracle detection statistics on top of the SFT inner products, fp64.  Test infrastructure.

* ``loglike`` - Eq.(2): ``L = <x,h> - <h,h>/2``.
* ``phase_maximised`` - Eq.(7)-(9) P:97-101: ``(<x,h_c>^2 + <x,h_s>^2) / <h_c,h_c>`` with ``h_c = A cos(phi)``,
  ``h_s = -A sin(phi)``: two runs of ``oracle.inner.inner_products`` (phi_c and phi_c + pi/2, which turns cos(phi) into
  -sin(phi)).
* ``fstat`` - Eq.(10)-(13) P:107-122: the four basis waveforms ``h_nu = A [a cos(phi), b cos(phi), a sin(phi), b sin(phi)]``
  (Eq.(11)) are four signals ``Re[R_nu A e^{i phi}]`` with ``R_nu = (a, b, -i a, -i b)`` (``Re[-i a z] = a Im z``), each with
  the per-SFT constant response of P:174; their SFT coefficients ``h~_nu`` follow step 3 of ``oracle.inner`` and the 4
  products ``x_nu = ([x,h_nu])`` and ALL 10 products ``M_numu = ([h_nu,h_mu])`` are summed bin by bin as in Eq.(1)/(35);
  ``2F = x^T M^-1 x`` and the maximising amplitudes ``c = M^-1 x`` (Eq.(13)), by a plain linear solve.

Pins: tests/test_oracle_stats.py - M symmetric positive definite; the cross-quadrature products vanish; 2F invariant under
an invertible re-mix of the basis; amplitudes c_nu injected sample by sample with a(t), b(t) are recovered (sign and order
of the four basis functions of Eq.(11)), and 2F of noiseless data equals <h,h> by direct integration up to the method's loss.
"""
import numpy as np

from . import inner as oin
from . import waveform as wf


def loglike(xh, hh):
    """Eq.(2) P:63."""
    return np.asarray(xh, np.float64) - 0.5 * np.asarray(hh, np.float64)


def phase_maximised(plan, store, params):
    """Eq.(7) P:97 from the two quadratures."""
    P = np.atleast_2d(np.asarray(params, np.float64))
    Ps = P.copy()
    Ps[:, 3] += 0.5 * np.pi
    c = oin.inner_products(plan, store, P)
    s = oin.inner_products(plan, store, Ps)
    return (c["xh"] ** 2 + s["xh"] ** 2) / c["hh"]


def basis_coefficients(plan, store, p, a_tab, b_tab):
    """SFT coefficients of the four basis waveforms of Eq.(11) for one parameter row ``p``.

    ``a_tab``, ``b_tab``: [C][N] antenna-pattern functions a(t_a), b(t_a) per channel (constant over an SFT).
    Returns ``hb`` [4][C][n_act][2K+1] complex (``h~_nu,c,a,k = 1/2 T A_a R_nu e^{i phi_a} F``), ``xt`` [C][n_act][2K+1]
    the data bins, ``invS`` same shape (0 for invalid bins / gaps), following steps 1-3 of ``oracle.inner``."""
    C, K, T = plan.n_channels, plan.K, plan.t_sft
    n = plan.n_samp
    t = oin.sft_times(plan)
    phi, f, fdot = wf.taylor_t3(p[0], p[1], p[2], p[3], t, plan.pn1)
    A = wf.amplitude(p[4], f, plan.f_ref)
    k_c, x, b, active, _ = oin.select_bins(plan, t, f, fdot, p[2])
    idx = np.nonzero(active)[0]
    present = store.present()
    Fk = oin.kernel_coefficients(plan, x[idx], b[idx])
    m = np.arange(-K, K + 1, dtype=np.int64)
    k = k_c[idx][:, None] + m[None, :]
    valid = (k >= (0 if plan.include_dc else 1)) & (k <= n // 2 - 1) & (k >= plan.k_lo) & (k < plan.k_hi)
    col = np.clip(k - plan.k_lo, 0, plan.k_hi - plan.k_lo - 1)
    core = 0.5 * T * (A[idx] * np.exp(1j * phi[idx]))[:, None] * Fk              # 1/2 T A e^{i phi} F
    hb = np.zeros((4, C) + core.shape, dtype=np.complex128)
    xt = np.zeros((C,) + core.shape, dtype=np.complex128)
    invS = np.zeros((C,) + core.shape)
    for c in range(C):
        pc = present[c][idx]
        with np.errstate(divide="ignore", invalid="ignore"):
            S = np.asarray(store.psd_scale[c], np.float64)[idx][:, None] * np.asarray(store.psd_shape[c], np.float64)[col]
            invS[c] = np.where(valid & pc[:, None], 1.0 / S, 0.0)
        xt[c] = np.where(invS[c] > 0.0, np.asarray(store.bins[c], np.complex128)[idx[:, None], col], 0.0)
        a, bb = np.asarray(a_tab[c], np.float64)[idx][:, None], np.asarray(b_tab[c], np.float64)[idx][:, None]
        for nu, R in enumerate((a, bb, -1j * a, -1j * bb)):
            hb[nu, c] = R * core
    return hb, xt, invS


def fstat(plan, store, params, a_tab, b_tab):
    """Eq.(13) P:122 for every parameter row: dict with ``x`` [T][4], ``M`` [T][4][4], ``c`` [T][4] (= M^-1 x) and ``twoF`` [T]."""
    P = np.atleast_2d(np.asarray(params, np.float64))
    df = 1.0 / plan.t_sft
    xs, Ms, cs, Fs = [], [], [], []
    for p in P:
        hb, xt, invS = basis_coefficients(plan, store, p, a_tab, b_tab)
        x = np.array([4.0 * df * np.sum(np.real(np.conj(xt) * hb[nu]) * invS) for nu in range(4)])
        M = np.array([[4.0 * df * np.sum(np.real(hb[nu] * np.conj(hb[mu])) * invS) for mu in range(4)] for nu in range(4)])
        if np.all(M == 0.0):
            c = np.zeros(4)
        else:
            c = np.linalg.solve(M, x)
        xs.append(x); Ms.append(M); cs.append(c); Fs.append(float(x @ c))
    return dict(x=np.array(xs), M=np.array(Ms), c=np.array(cs), twoF=np.array(Fs))
