"""Oracle kernels ``Fre`` / ``Dir`` in dimensionless form, fp64.  Test infrastructure.

Dimensionless variables (DESIGN.md notation): ``a = (f_a - f_k) T_SFT`` (offset in bins),
``b = fdot_a T_SFT^2`` (bins swept during one SFT) and

    F(a, b) = Fre(a/T, b/T^2) / T = int_0^1 exp(i pi (2 a s + b s^2)) ds        Eq.(28)

``fre_quadrature`` IS that definition (Gauss-Legendre quadrature of the integral);
``fre_closed`` is the paper's closed form Eq.(29)-(32) P:219-236 with library Fresnel
integrals; ``fre_discrete`` is the finite sum Eq.(27); ``dirichlet`` is Eq.(B2)
in the reading ``Fre(f, 0) = dt Dir(f) = T e^{i pi T f} sinc(T f)`` (reading A3).
Pins: tests/test_oracle_kernel.py (P5).
"""
import numpy as np
from scipy.special import fresnel as _fresnel_SC  # returns (S, C)

_GL_CACHE = {}


def _gauss_legendre_01(n):
    if n not in _GL_CACHE:
        x, w = np.polynomial.legendre.leggauss(n)
        _GL_CACHE[n] = (0.5 * (x + 1.0), 0.5 * w)
    return _GL_CACHE[n]


def fre_quadrature(a, b, nodes=None):
    """F(a,b) by n-point Gauss-Legendre quadrature of Eq.(28) on [0,1] (the definition).

    The integrand's phase sweeps ``2 pi (|a| + |b|/2)`` rad at most; n-point Gauss-Legendre
    is exact to rounding for ``exp(i w s)`` once ``n > w/2 + O(10)``; the default takes
    ``n = 64 + 4 ceil(max|a| + max|b|)``.
    """
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    a, b = np.broadcast_arrays(a, b)
    if nodes is None:
        span = float(np.max(np.abs(a)) + np.max(np.abs(b))) if a.size else 0.0
        nodes = 64 + 4 * int(np.ceil(span))
    s, w = _gauss_legendre_01(int(nodes))
    af, bf = a.reshape(-1), b.reshape(-1)
    out = np.empty(af.shape, dtype=np.complex128)
    step = max(1, (1 << 22) // int(nodes))          # same sums, evaluated in blocks of elements (memory only)
    for i in range(0, af.size, step):
        ph = np.pi * (2.0 * af[i:i + step, None] * s + bf[i:i + step, None] * s * s)
        out[i:i + step] = np.sum(w * np.exp(1j * ph), axis=-1)
    return out.reshape(a.shape)


def dirichlet(a):
    """F(a, 0) = e^{i pi a} sinc(a), sinc(x) = sin(pi x)/(pi x)  (Eq.(B2))."""
    a = np.asarray(a, dtype=np.float64)
    return np.exp(1j * np.pi * a) * np.sinc(a)


def fre_closed(a, b, phase_guard=1e8):
    """F(a,b) from Eq.(29)-(30) P:219-226 with ``C``, ``S`` of Eq.(31)-(32) from scipy.

    In dimensionless form ``l = a sqrt(2/b)``, ``u = l + sqrt(2 b)`` and
    ``F = exp(-i pi a^2/b)/sqrt(2 b) {C(u)-C(l) + i[S(u)-S(l)]}``.

    Readings (A10): ``b == 0`` is the Dirichlet limit; ``b < 0`` uses
    ``F(a,-b) = conj F(-a,b)`` (from the definition); where the phase ``pi a^2/b`` exceeds
    ``phase_guard`` rad the closed form loses more than ~1e-8 to fp64 rounding of that
    phase, so those elements are evaluated from the definition (``fre_quadrature``).
    """
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    a, b = np.broadcast_arrays(a, b)
    out = np.empty(a.shape, dtype=np.complex128)
    neg = b < 0.0
    aa = np.where(neg, -a, a)
    bb = np.abs(b)
    zero = bb == 0.0
    with np.errstate(divide="ignore", invalid="ignore"):
        big = (~zero) & (np.pi * aa * aa / bb > phase_guard)
    ok = ~(zero | big)
    if np.any(ok):
        a1 = aa[ok]
        b1 = bb[ok]
        l = a1 * np.sqrt(2.0 / b1)
        u = l + np.sqrt(2.0 * b1)
        Su, Cu = _fresnel_SC(u)
        Sl, Cl = _fresnel_SC(l)
        pref = np.exp(-1j * np.pi * a1 * a1 / b1) / np.sqrt(2.0 * b1)
        out[ok] = pref * ((Cu - Cl) + 1j * (Su - Sl))
    if np.any(zero):
        out[zero] = dirichlet(aa[zero])
    if np.any(big):
        out[big] = fre_quadrature(aa[big], bb[big])
    return np.where(neg, np.conj(out), out)


def fre_discrete(a, b, n):
    """Eq.(27) P:208 divided by T: (1/n) sum_{j<n} exp(i pi (2 a j/n + b (j/n)^2))."""
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    a, b = np.broadcast_arrays(a, b)
    s = np.arange(n, dtype=np.float64) / n
    ph = np.pi * (2.0 * a[..., None] * s + b[..., None] * s * s)
    return np.sum(np.exp(1j * ph), axis=-1) / n
