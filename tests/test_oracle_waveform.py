"""Pins P6, P7 for oracle/waveform.py (CPU only)."""
import json
import os
import numpy as np
import pytest
from oracle import waveform as wf

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.json")))


@pytest.mark.parametrize("pn1", [0, 1, 2])
@pytest.mark.parametrize("mc,eta,tau", [(1.2188, 0.25, 5000.0), (1.2188, 0.25, 200.0), (4.06e5, 0.2222, 1e6), (30.0, 0.2, 50.0)])
def test_P6_derivative_consistency(pn1, mc, eta, tau):
    """dphi/dt = 2 pi f, df/dt = fdot, d2f/dt2 = fddot by central differences (f = phi-dot)."""
    t_c = 1.0e5
    t = t_c - tau
    h = tau * 1e-5
    ts = np.array([t - h, t, t + h])
    phi, f, fd = wf.taylor_t3(mc, eta, t_c, 0.3, ts, pn1)
    assert abs((phi[2] - phi[0]) / (2 * h) / (2 * np.pi * f[1]) - 1) < 1e-7
    assert abs((f[2] - f[0]) / (2 * h) / fd[1] - 1) < 1e-7
    fdd = wf.taylor_t3_fddot(mc, eta, t_c, ts, pn1)
    assert abs((fd[2] - fd[0]) / (2 * h) / fdd[1] - 1) < 1e-6


def test_P6_newtonian_chirp_time():
    """0PN frequency equals the inverse of tau = (5/256) Mc^-5/3 (pi f)^-8/3, for any eta."""
    for eta in (0.25, 0.1):
        for tau in (1.0, 1e3, 4.6e5):
            _, f, fd = wf.taylor_t3(1.2188, eta, tau, 0.0, 0.0, 0)
            assert abs(wf.tau_newtonian(f, 1.2188) / tau - 1) < 1e-13
            # fdot = (96/5) pi^(8/3) Mc^(5/3) f^(11/3)
            mc = 1.2188 * wf.GMSUN_S
            assert abs(96 / 5 * np.pi ** (8 / 3) * mc ** (5 / 3) * f ** (11 / 3) / fd - 1) < 1e-13


def test_P6_1pn_chirp_time_textbook():
    """1PN: t_c - t(f) = tau0 [1 + (4/3)(743/336 + 11 eta/4)(pi M f)^(2/3)] + O((pi M f)^(4/3))
    (textbook 1PN chirp time); the residual must scale as (pi M f)^(4/3)."""
    mc, eta = 1.2188, 0.25
    M = wf.total_mass_seconds(mc, eta)
    res = []
    for tau in (1e5, 1e3):
        _, f, _ = wf.taylor_t3(mc, eta, tau, 0.0, 0.0, 1)
        x = (np.pi * M * f) ** (2.0 / 3.0)
        pred = wf.tau_newtonian(f, mc) * (1 + 4.0 / 3.0 * (743.0 / 336.0 + 11.0 * eta / 4.0) * x)
        res.append((pred / tau - 1, x))
    (r1, x1), (r2, x2) = res
    assert abs(r1) < 20 * x1 ** 2 and abs(r2) < 20 * x2 ** 2
    assert abs(np.log(abs(r2 / r1)) / np.log(x2 / x1) - 2.0) < 0.15   # residual ~ x^2 = (pi M f)^(4/3)


def test_P6_15pn_chirp_time_textbook():
    """1.5PN (order code 2): t_c - t(f) = tau0 [1 + (4/3)(743/336 + 11 eta/4) x - (32 pi/5) x^(3/2)] + O(x^2), x = (pi M f)^(2/3)
    (the textbook chirp times tau0 + tau1 - tau1.5): pins the sign and size of the tail terms; the residual scales as x^2."""
    mc, eta = 1.2188, 0.25
    M = wf.total_mass_seconds(mc, eta)
    res = []
    for tau in (1e5, 1e3):
        _, f, _ = wf.taylor_t3(mc, eta, tau, 0.0, 0.0, 2)
        x = (np.pi * M * f) ** (2.0 / 3.0)
        pred = wf.tau_newtonian(f, mc) * (1 + 4.0 / 3.0 * (743.0 / 336.0 + 11.0 * eta / 4.0) * x - 32.0 * np.pi / 5.0 * x ** 1.5)
        res.append((pred / tau - 1, x))
        # without the tail term the mismatch is of order x^(3/2), far above the residual
        _, f1, _ = wf.taylor_t3(mc, eta, tau, 0.0, 0.0, 1)
        assert abs(f / f1 - 1) > 0.05 * x ** 1.5
    (r1, x1), (r2, x2) = res
    assert abs(r1) < 40 * x1 ** 2 and abs(r2) < 40 * x2 ** 2
    assert abs(np.log(abs(r2 / r1)) / np.log(x2 / x1) - 2.0) < 0.25


def test_P7_bns_printed_values():
    g = GOLD["bns"]
    eta = g["m1"] * g["m2"] / (g["m1"] + g["m2"]) ** 2
    mc = (g["m1"] + g["m2"]) * eta ** 0.6
    assert abs(mc - g["chirp_mass_printed"]) < 0.01                        # "1.21 Msun" P:295
    dur = wf.tau_newtonian(g["f_start"], mc) - wf.tau_newtonian(g["f_end"], mc)
    assert abs(dur / 3600.0 / g["duration_hours_printed"] - 1) < 0.02      # "130 hours"
    assert abs(dur * g["fs"] / g["n0_printed"] - 1) < 0.1                  # "N0 ~ 2e7"
    tau10 = wf.tau_newtonian(g["f_end"], mc)
    fdd = wf.taylor_t3_fddot(mc, eta, tau10, 0.0, 0)
    assert abs(fdd / g["max_fddot_printed"] - 1) < 0.05                    # "~5e-6 Hz/s^2" P:320
    # Table I: T_SFT(delta) from Eq.(34) with the printed max fddot, and N_SFT = duration / T_SFT
    tab = GOLD["table1"]
    T = wf.t_sft_rule(np.array(tab["delta"]), g["max_fddot_printed"])
    assert np.all(np.abs(T - np.array(tab["t_sft"])) <= 1.0)
    span = np.array(tab["t_sft"]) * np.array(tab["n_sft"])
    assert np.all(np.abs(span / dur - 1) < 0.01)


def test_P7_mbhb_printed_values():
    g = GOLD["mbhb"]
    eta = 0.25
    mc = (g["m1"] + g["m2"]) * eta ** 0.6
    for pn1, tol in ((0, 0.05), (1, 0.08)):
        # duration from f_start to f_end with the oracle's own f(t): find tau(f) by bisection on taylor_t3
        def tau_of(ftarget):
            lo, hi = 1.0, 1e9
            for _ in range(200):
                mid = np.sqrt(lo * hi)
                _, f, _ = wf.taylor_t3(mc, eta, mid, 0.0, 0.0, pn1)
                lo, hi = (mid, hi) if f > ftarget else (lo, mid)
            return mid
        dur = tau_of(g["f_start"]) - tau_of(g["f_end"])
        assert abs(dur / 86400.0 / g["duration_days_printed"] - 1) < tol     # "about 45 days" P:326
    tab = GOLD["table2"]
    T = np.array(tab["t_sft"], dtype=float)
    d = np.array(tab["delta"])
    # Eq.(34): T_SFT scales as delta^(1/3)
    assert np.all(np.abs(T[0] * (d / d[0]) ** (1 / 3) - T) <= 1.0)
    # implied max fddot = 2 delta / T^3 agrees with the Newtonian fddot at 1.9 mHz to PN accuracy
    tau_end = wf.tau_newtonian(g["f_end"], mc)
    fdd = wf.taylor_t3_fddot(mc, eta, tau_end, 0.0, 0)
    assert abs(wf.t_sft_rule(1.0, fdd) / T[0] - 1) < 0.08
    span = T * np.array(tab["n_sft"])
    assert np.all(np.abs(span / span[0] - 1) < 0.01)
