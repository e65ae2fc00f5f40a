"""Pin P5 (and P8) for oracle/kernel.py (CPU only)."""
import numpy as np
import mpmath
import pytest
from scipy.special import polygamma
from oracle import kernel as kern


def _mp_def(a, b):
    """Eq.(28) P:215 in dimensionless form by mpmath's adaptive quadrature (30 digits)."""
    mpmath.mp.dps = 30
    f = lambda s: mpmath.e ** (1j * mpmath.pi * (2 * a * s + b * s * s))
    pts = [mpmath.mpf(i) / 64 for i in range(65)]
    return complex(mpmath.quad(f, pts))


@pytest.mark.parametrize("a,b", [(0.0, 0.0), (0.3, 0.0), (0.3, 1e-3), (-4.7, 0.02), (8.2, 0.5), (-0.45, 2.0),
                                 (3.5, 4.0), (-10.5, 4.0), (16.4, 7.5), (0.2, -1.5), (-3.3, -0.4)])
def test_definition_vs_mpmath(a, b):
    ref = _mp_def(a, b)
    assert abs(kern.fre_quadrature(a, b) - ref) < 1e-13
    assert abs(kern.fre_closed(a, b) - ref) < 1e-11


def test_closed_form_vs_definition_random():
    rng = np.random.default_rng(11)
    a = rng.uniform(-20, 20, 4000)
    b = 10.0 ** rng.uniform(-4, 0.9, 4000) * rng.choice([1.0, 1.0, 1.0, -1.0], 4000)
    d = np.abs(kern.fre_closed(a, b) - kern.fre_quadrature(a, b))
    # fp64 rounding of the phase pi a^2/b (up to 1.3e7 rad here) limits the closed form to ~1e-10
    assert d.max() < 2e-10 and np.median(d) < 1e-13


def test_phase_guard_fallback():
    """Tiny b with large a: the closed form's phase pi a^2/b is huge; the guard must keep 1e-9."""
    a = np.array([60.3, -63.9, 17.2])
    b = np.array([1e-7, 3e-6, 1e-9])
    assert np.abs(kern.fre_closed(a, b) - kern.fre_quadrature(a, b)).max() < 1e-9
    assert np.abs(kern.fre_closed(a, b) - kern.dirichlet(a)).max() < 1e-5


def test_dirichlet_limit_and_closed_form():
    """Fre -> Dir as f1 -> 0; Dir(a) = e^{i pi a} sinc(a) equals int_0^1 e^{2 pi i a s} ds."""
    a = np.linspace(-9.3, 9.3, 77)
    assert np.abs(kern.fre_closed(a, 0.0) - kern.dirichlet(a)).max() == 0.0
    with np.errstate(all="ignore"):
        exact = np.where(a == 0, 1.0, (np.exp(2j * np.pi * a) - 1) / (2j * np.pi * a))
    assert np.abs(kern.dirichlet(a) - exact).max() < 1e-14
    for b in (1e-3, 1e-5):
        # first-order term: F(a,b) - F(a,0) = i pi b int s^2 e^{2 pi i a s} ds + O(b^2)
        d = kern.fre_closed(a, b) - kern.dirichlet(a)
        assert np.abs(d).max() < np.pi * b / 3 * 1.01
    assert abs(kern.dirichlet(0.0) - 1.0) == 0 and abs(kern.dirichlet(3.0)) < 1e-15


def test_discrete_minus_continuum_is_euler_maclaurin_end_term():
    """Eq.(27) - Eq.(28) = (g(0) - g(1))/(2n) + (g'(1) - g'(0))/(12 n^2) + O(n^-4), g the integrand
    (reading A4: the continuum kernel is the method)."""
    rng = np.random.default_rng(12)
    a = rng.uniform(-8, 8, 50)
    b = rng.uniform(0, 4, 50)
    for n in (720, 4096):
        g1 = np.exp(1j * np.pi * (2 * a + b))
        em = (1 - g1) / (2 * n) + (1j * np.pi * (2 * a + 2 * b) * g1 - 1j * np.pi * 2 * a) / (12 * n * n)
        d = kern.fre_discrete(a, b, n) - kern.fre_quadrature(a, b)
        assert np.abs(d - em).max() < 5e-3 * (40.0 / n) ** 4 * 1e3 + 1e-13
        assert np.abs(d).max() > 0.1 / n        # the difference is real: O(1/n), not rounding


def test_unit_total_power():
    """sum over ALL bins of |F(x-m, b)|^2 = int_0^1 |e^{..}|^2 ds = 1 (Parseval for one SFT)."""
    m = np.arange(-5000, 5001)     # (|a| <= 5000 keeps pi a^2/b below fre_closed's phase guard: closed form throughout)
    for x, b in ((0.37, 0.0), (-0.2, 0.8), (0.1, 3.0)):
        tot = np.sum(np.abs(kern.fre_closed(x - m, b)) ** 2)
        assert 0.0 < 1.0 - tot < 6e-5           # tail beyond +-5000 bins ~ 2/(pi^2 5000) = 4.05e-5


def test_P8_dirichlet_truncation_loss():
    """Power outside +-K at half-bin offset = [psi1(K+1/2) + psi1(K+3/2)]/pi^2 (trigamma closed
    form): 8.3/4.5/2.4/1.2/0.62/0.31 % for K = 2..64, cf. 'drops off ... at Delta k <~ 5' P:456."""
    expect = {2: 8.3e-2, 4: 4.5e-2, 8: 2.4e-2, 16: 1.2e-2, 32: 6.2e-3, 64: 3.1e-3}
    for K, e in expect.items():
        m = np.arange(-K, K + 1)
        loss = 1.0 - np.sum(np.abs(kern.dirichlet(0.5 - m)) ** 2)
        closed = float(polygamma(1, K + 0.5) + polygamma(1, K + 1.5)) / np.pi ** 2
        assert abs(loss - closed) < 1e-12
        assert abs(loss / e - 1) < 0.03
