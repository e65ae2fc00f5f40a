"""Pins of oracle/stats.py (Eq.(2), (7)-(13) P:63-122)."""
import numpy as np
import pytest

from oracle import stats as ost, inner as oin, sft as osft
from paper_2502_11823_b200 import workloads as wl
from _util import to_oracle


@pytest.fixture(scope="module")
def case():
    w = wl.fstat_case(n_templates=3)
    plan, store = to_oracle(w)
    a, b = w.response.real.astype(np.float64), w.response.imag.astype(np.float64)
    return w, plan, store, a, b, ost.fstat(plan, store, w.params, a, b)


def test_M_is_symmetric_positive_definite_and_block_diagonal(case):
    """([h_nu,h_mu]) is a Gram matrix; in the framework (positive-frequency coefficients, response constant per SFT) the
    cos and sin quadratures are orthogonal, and the two diagonal blocks coincide: A = sum a^2 H, B = sum b^2 H, C = sum a b H."""
    M = case[5]["M"][0]
    assert np.allclose(M, M.T, rtol=0, atol=1e-12 * np.abs(M).max())
    assert np.all(np.linalg.eigvalsh(M) > 0)
    assert np.abs(M[:2, 2:]).max() <= 1e-12 * np.abs(M).max()
    assert np.allclose(M[:2, :2], M[2:, 2:], rtol=1e-12)


def test_injected_amplitudes_are_recovered(case):
    """Noiseless data h = sum c_nu h_nu built sample by sample from Eq.(11): M^-1 x returns c (sign and order of the four basis
    functions), and 2F = c^T M c equals <h,h> by direct integration up to the method's loss."""
    w, plan, store, a, b, o = case
    c = w.notes["c_nu"]
    assert np.abs(o["c"][0] - c).max() < 0.02, o["c"][0]
    exact = osft.time_domain_product(w.series[0], w.series[0], 1.0 / w.desc["fs"], w.notes["S"])
    assert 0.95 * exact < o["twoF"][0] < 1.001 * exact
    # a sign slip in one quadrature (h_2 = +a sin phi, Eq.(11)) would move c_2, c_3 to the other side
    assert np.sign(o["c"][0][2]) == np.sign(c[2]) and np.sign(o["c"][0][3]) == np.sign(c[3])


@pytest.mark.parametrize("nu", [0, 1, 2, 3])
def test_single_basis_function(nu):
    """Data = one basis function of Eq.(11) alone: the solve returns the unit vector e_nu."""
    c = np.zeros(4)
    c[nu] = 1.0
    w = wl.fstat_case(c_nu=c, n_templates=1)
    plan, store = to_oracle(w)
    o = ost.fstat(plan, store, w.params, w.response.real.astype(np.float64), w.response.imag.astype(np.float64))
    assert np.abs(o["c"][0] - c).max() < 0.02, o["c"][0]


def test_invariance_under_remixing_and_relation_to_inner_products(case):
    w, plan, store, a, b, o = case
    G = np.random.default_rng(5).standard_normal((4, 4)) + 2.0 * np.eye(4)
    x, M = o["x"][1], o["M"][1]
    assert (G @ x) @ np.linalg.solve(G @ M @ G.T, G @ x) == pytest.approx(o["twoF"][1], rel=1e-10)
    # x_0 and M_00 are the plain inner products for the response table R = a (oracle.inner with response="table")
    import copy
    st = copy.copy(store)
    st.response = a.astype(np.complex128)
    ref = oin.inner_products(plan, st, w.params)
    assert np.allclose(o["x"][:, 0], ref["xh"], rtol=1e-10, atol=1e-10 * np.abs(ref["xh"]).max())
    assert np.allclose(o["x"][:, 2], ref["xh_im"], rtol=1e-10, atol=1e-10 * np.abs(ref["xh"]).max())
    assert np.allclose(o["M"][:, 0, 0], ref["hh"], rtol=1e-10)


def test_phase_maximised_and_loglike(case):
    w, plan, store, a, b, o = case
    st = __import__("copy").copy(store)
    st.response = (a + 0j)
    r = oin.inner_products(plan, st, w.params)
    stat = ost.phase_maximised(plan, st, w.params)
    assert np.allclose(stat, (r["xh"] ** 2 + r["xh_im"] ** 2) / r["hh"], rtol=1e-9)      # <x,h_s> = -Im Z  (shift by pi/2)
    assert np.allclose(ost.loglike(r["xh"], r["hh"]), r["xh"] - 0.5 * r["hh"])
