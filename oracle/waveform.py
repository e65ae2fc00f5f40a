"""Oracle waveform: restricted TaylorT3 inspiral, 0PN or 0PN+1PN, fp64.  Test infrastructure.

The paper evaluates ``{A_a, phi_a, f_a, fdot_a}`` at every SFT start (P:157-164,
Eq.(16)-(17)) from IMRPhenomT, whose fitted coefficients are not available here;
BASELINE.json's configs prescribe "Newtonian (0PN)" and "0PN+1PN" inspirals, so this is
the textbook closed-form time-domain inspiral (reading W1):

    Theta   = eta (t_c - t) / (5 M)                       M = total mass in seconds
    phi(t)  = phi_c - (2/eta) Theta^{5/8} [1 + p1 (3715/8064 + 55 eta/96) Theta^{-1/4}]
    f(t)    = Theta^{-3/8}/(8 pi M) [1 + p1 (743/2688 + 11 eta/32) Theta^{-1/4}]
    fdot(t) = (eta/5M)/(8 pi M) [3/8 Theta^{-11/8} + 5/8 p1 (743/2688 + 11 eta/32) Theta^{-13/8}]
    A(t)    = amp (f(t)/f_ref)^{2/3}

with ``dphi/dt = 2 pi f`` and ``df/dt = fdot`` exactly (pinned numerically, P6) and the
0PN limit equal to the chirp-time closed form ``tau = (5/256) Mc^{-5/3} (pi f)^{-8/3}``
(pinned, P6/P7 with the paper's 130 h / 45 d / 5e-6 Hz/s^2 values).
"""
import numpy as np

#: G Msun / c^3 in seconds (IAU nominal solar mass parameter / c^3).
GMSUN_S = 4.925491025543576e-6

C_PHI_0 = 3715.0 / 8064.0
C_PHI_1 = 55.0 / 96.0
C_F_0 = 743.0 / 2688.0
C_F_1 = 11.0 / 32.0
#: 1.5PN (tail) terms of TaylorT3 relative to the leading one, in Theta^(-3/8): phase -3 pi/4, frequency -3 pi/10
C15_PHI = -0.75 * np.pi
C15_F = -0.3 * np.pi


def total_mass_seconds(m_chirp, eta):
    """Total mass in seconds from chirp mass [Msun] and symmetric mass ratio: M = Mc eta^{-3/5}."""
    return np.asarray(m_chirp, dtype=np.float64) * np.asarray(eta, dtype=np.float64) ** (-0.6) * GMSUN_S


def taylor_t3(m_chirp, eta, t_c, phi_c, t, pn1):
    """Phase [rad], frequency [Hz], frequency derivative [Hz/s] at times ``t``.

    ``pn1`` is the PN order code: 0 = 0PN, 1 = + 1PN terms, 2 = + 1.5PN (tail) terms
    ``phi += (2/eta)(3 pi/4) Theta^{1/4}``, ``f -= (3 pi/10) Theta^{-3/4}/(8 pi M)`` (the textbook TaylorT3 coefficients;
    ``dphi/dt = 2 pi f`` holds order by order, pinned numerically).  Where ``t >= t_c`` the outputs are NaN
    (the template has ended; such SFTs are inactive, reading A12).
    """
    t = np.asarray(t, dtype=np.float64)
    M = total_mass_seconds(m_chirp, eta)
    tau = np.float64(t_c) - t
    with np.errstate(invalid="ignore", divide="ignore"):
        theta = np.where(tau > 0.0, eta * tau / (5.0 * M), np.nan)
        cphi = C_PHI_0 + C_PHI_1 * eta
        cf = C_F_0 + C_F_1 * eta
        th_m14 = theta ** (-0.25)
        th_m38 = theta ** (-0.375)
        p1, p15 = float(pn1 >= 1), float(pn1 >= 2)
        phi = phi_c - (2.0 / eta) * theta ** 0.625 * (1.0 + p1 * cphi * th_m14 + p15 * C15_PHI * th_m38)
        f = theta ** (-0.375) / (8.0 * np.pi * M) * (1.0 + p1 * cf * th_m14 + p15 * C15_F * th_m38)
        fdot = (eta / (5.0 * M)) / (8.0 * np.pi * M) * (
            0.375 * theta ** (-1.375) + 0.625 * p1 * cf * theta ** (-1.625) + 0.75 * p15 * C15_F * theta ** (-1.75))
    return phi, f, fdot


def taylor_t3_fddot(m_chirp, eta, t_c, t, pn1):
    """Second frequency derivative [Hz/s^2], needed only by the SFT-length rule Eq.(33)-(34)."""
    t = np.asarray(t, dtype=np.float64)
    M = total_mass_seconds(m_chirp, eta)
    theta = eta * (np.float64(t_c) - t) / (5.0 * M)
    cf = C_F_0 + C_F_1 * eta
    k = eta / (5.0 * M)
    return k * k / (8.0 * np.pi * M) * (
        0.375 * 1.375 * theta ** (-2.375) + 0.625 * 1.625 * float(pn1 >= 1) * cf * theta ** (-2.625)
        + 0.75 * 1.75 * float(pn1 >= 2) * C15_F * theta ** (-2.75))


def amplitude(amp, f, f_ref):
    """A = amp (f/f_ref)^{2/3}: leading-order inspiral amplitude, constant per SFT."""
    return np.asarray(amp, dtype=np.float64) * (np.asarray(f, dtype=np.float64) / f_ref) ** (2.0 / 3.0)


def tau_newtonian(f, m_chirp):
    """Time to coalescence from GW frequency f at 0PN: (5/256) Mc^{-5/3} (pi f)^{-8/3}."""
    mc = np.asarray(m_chirp, dtype=np.float64) * GMSUN_S
    return 5.0 / 256.0 * mc ** (-5.0 / 3.0) * (np.pi * np.asarray(f, dtype=np.float64)) ** (-8.0 / 3.0)


def t_sft_rule(delta, max_fddot):
    """SFT length of Eq.(34): T_SFT(delta) = (2 delta / max fddot)^{1/3}."""
    return (2.0 * np.asarray(delta, dtype=np.float64) / max_fddot) ** (1.0 / 3.0)
