"""Pins for the oracle's basis functions and coupling tensors (SURVEY.md §8c 'What pins each part').

None of these retypes the oracle's own formula: they use closed-form properties, scipy's spherical
harmonics, sympy's exact Wigner-3j symbols and the worked values stored in tests/golden/.
"""
import json
import math
import os

import numpy as np
import pytest

from oracle import allegro_oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _unit(n, seed):
    v = np.random.default_rng(seed).standard_normal((n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


# ---------------------------------------------------------------- envelope (F1)
@pytest.mark.parametrize("p", [4, 6, 8])
def test_envelope_boundary_conditions(p):
    assert O.envelope(0.0, p) == 1.0
    h = 1e-4
    u = lambda x: float(O.envelope(x, p))
    # u(1)=u'(1)=u''(1)=0: one-sided differences from the inside vanish to O(h^3)
    assert abs(u(1 - h)) < 1e3 * h ** 3
    assert abs((u(1 - h) - u(1 - 2 * h)) / h) < 1e3 * h ** 2
    assert abs((u(1 - h) - 2 * u(1 - 2 * h) + u(1 - 3 * h)) / h ** 2) < 3e3 * h
    assert O.envelope(1.0, p) == 0.0 and O.envelope(1.3, p) == 0.0


def test_envelope_p6_printed_polynomial():
    # SURVEY.md §8c F1 prints the p=6 case: 1 - 28 x^6 + 48 x^7 - 21 x^8
    x = np.linspace(0, 0.999, 50)
    np.testing.assert_allclose(O.envelope(x, 6), 1 - 28 * x ** 6 + 48 * x ** 7 - 21 * x ** 8, rtol=0, atol=1e-14)


def test_envelope_derivative_matches_fd():
    x = np.linspace(0.05, 0.98, 40)
    h = 1e-6
    fd = (O.envelope(x + h, 6) - O.envelope(x - h, 6)) / (2 * h)
    np.testing.assert_allclose(O.envelope_deriv(x, 6), fd, rtol=1e-7, atol=1e-8)


# ---------------------------------------------------------------- Bessel basis (F2)
def test_bessel_orthogonality():
    # int_0^rc B_n B_m r^2 dr = (2/rc) delta_nm
    rc, nb = 5.2, 8
    r = np.linspace(1e-9, rc, 200001)
    B = O.bessel_raw(r, rc, nb)
    G = np.trapezoid(B[:, :, None] * B[:, None, :] * (r * r)[:, None, None], r, axis=0)
    np.testing.assert_allclose(G, (2 / rc) * np.eye(nb), atol=1e-8)


def test_bessel_limits_and_derivative():
    rc, nb = 4.0, 8
    n = np.arange(1, nb + 1)
    # r -> 0: sin(k r)/r -> k
    np.testing.assert_allclose(O.bessel_raw(1e-8, rc, nb), (2 / rc) * n * math.pi / rc, rtol=1e-10)
    np.testing.assert_allclose(O.bessel_raw(rc, rc, nb), 0, atol=1e-15)
    r = np.linspace(0.5, 3.9, 30)
    h = 1e-6
    fd = (O.bessel_raw(r + h, rc, nb) - O.bessel_raw(r - h, rc, nb)) / (2 * h)
    np.testing.assert_allclose(O.bessel_raw_deriv(r, rc, nb), fd, rtol=1e-6, atol=1e-8)


# ---------------------------------------------------------------- spherical harmonics (F3)
def test_sh_against_scipy():
    """Component-normalised real SH = sqrt(4 pi) x the orthonormal real SH built from scipy's complex
    Y_l^mu with the standard real combination (m<0: sqrt2 (-1)^m Im Y_l^|m|, m>0: sqrt2 (-1)^m Re Y_l^m)."""
    from scipy.special import sph_harm_y
    n = _unit(200, 0)
    theta = np.arccos(n[:, 2]); phi = np.arctan2(n[:, 1], n[:, 0])
    Y = O.spherical_harmonics(n, 3)
    for l in range(4):
        for m in range(-l, l + 1):
            yc = sph_harm_y(l, abs(m), theta, phi)
            if m < 0:
                ref = math.sqrt(2) * (-1) ** m * yc.imag
            elif m == 0:
                ref = yc.real
            else:
                ref = math.sqrt(2) * (-1) ** m * yc.real
            np.testing.assert_allclose(Y[l][:, m + l], math.sqrt(4 * math.pi) * ref, atol=1e-12)


def test_sh_norm_pole_and_addition_theorem():
    from scipy.special import eval_legendre
    a, b = _unit(100, 1), _unit(100, 2)
    Ya, Yb = O.spherical_harmonics(a, 3), O.spherical_harmonics(b, 3)
    zhat = O.spherical_harmonics(np.array([[0.0, 0.0, 1.0]]), 3)
    for l in range(4):
        np.testing.assert_allclose((Ya[l] ** 2).sum(1), 2 * l + 1, rtol=1e-13)
        expect = np.zeros(2 * l + 1); expect[l] = math.sqrt(2 * l + 1)
        np.testing.assert_allclose(zhat[l][0], expect, atol=1e-14)
        np.testing.assert_allclose((Ya[l] * Yb[l]).sum(1), (2 * l + 1) * eval_legendre(l, (a * b).sum(1)), atol=1e-12)


def test_sh_gradient_tangential_matches_fd():
    n = _unit(20, 3)
    h = 1e-6
    dY = O.spherical_harmonics_grad(n, 3)
    for k in range(3):
        t = np.zeros(3); t[k] = 1.0
        tp = t - n * n[:, k:k + 1]                      # tangential part of e_k at each n
        npl = n + h * tp; npl /= np.linalg.norm(npl, axis=1, keepdims=True)
        nmi = n - h * tp; nmi /= np.linalg.norm(nmi, axis=1, keepdims=True)
        Yp, Ym = O.spherical_harmonics(npl, 3), O.spherical_harmonics(nmi, 3)
        for l in range(4):
            fd = (Yp[l] - Ym[l]) / (2 * h)
            an = np.einsum("emk,ek->em", dY[l], tp)
            np.testing.assert_allclose(an, fd, atol=2e-8)


# ---------------------------------------------------------------- coupling tensors (A9)
TRIPLES = [(a, b, c) for a in range(4) for b in range(4) for c in range(4) if abs(a - b) <= c <= a + b]


def test_cg_trivial_cases():
    for l in range(4):
        C = O.coupling_tensor(0, l, l)
        np.testing.assert_allclose(C[0], np.eye(2 * l + 1), atol=1e-13)
        C = O.coupling_tensor(l, l, 0)
        np.testing.assert_allclose(C[:, :, 0], np.eye(2 * l + 1) / math.sqrt(2 * l + 1), atol=1e-13)


def test_cg_111_is_cross_product():
    # l=1 components are ordered (y,z,x): out = (a x b)/sqrt2 expressed in that order
    C = O.coupling_tensor(1, 1, 1)
    rng = np.random.default_rng(4)
    a, b = rng.standard_normal(3), rng.standard_normal(3)
    perm = [1, 2, 0]                                        # (y,z,x) from (x,y,z)
    out = np.einsum("abc,a,b->c", C, a[perm], b[perm])
    np.testing.assert_allclose(out, np.cross(a, b)[perm] / math.sqrt(2), atol=1e-13)


@pytest.mark.parametrize("t", TRIPLES)
def test_cg_orthogonality_and_norm(t):
    C = O.coupling_tensor(*t)
    np.testing.assert_allclose(np.einsum("abc,abd->cd", C, C), np.eye(2 * t[2] + 1), atol=1e-12)
    flat = C.ravel()
    assert flat[np.flatnonzero(np.abs(flat) > 1e-12)[0]] > 0


def _wigner_D_from_samples(l, R):
    """D^l(R) with Y_l(R n) = D Y_l(n), fitted by least squares from samples (uses only F3 via the
    oracle's SH, which test_sh_against_scipy pins independently)."""
    n = _unit(60, 10 + l)
    A = O.spherical_harmonics(n, l)[l]
    B = O.spherical_harmonics(n @ R.T, l)[l]
    X, *_ = np.linalg.lstsq(A, B, rcond=None)
    return X.T


@pytest.mark.parametrize("t", TRIPLES)
def test_cg_equivariance(t):
    from scipy.spatial.transform import Rotation
    R = Rotation.random(random_state=5).as_matrix()
    l1, l2, l3 = t
    D1, D2, D3 = (_wigner_D_from_samples(l, R) for l in t)
    C = O.coupling_tensor(*t)
    lhs = np.einsum("abc,ai,bj->ijc", C, D1, D2)            # couple rotated inputs
    rhs = np.einsum("ijk,ck->ijc", C, D3)                   # rotate the coupled output
    np.testing.assert_allclose(lhs, rhs, atol=1e-11)


@pytest.mark.parametrize("t", [(1, 1, 2), (1, 2, 3), (2, 2, 2), (2, 3, 3), (3, 3, 2), (1, 2, 1), (2, 2, 1)])
def test_cg_against_sympy_wigner3j(t):
    """Basis-independent magnitude check against sympy's exact Wigner-3j.  Product rule for
    component-normalised SH at one direction: Y_l1m1 Y_l2m2 = sum_l3 sqrt((2l1+1)(2l2+1)/(2l3+1))
    <l1 0 l2 0|l3 0> <l1m1 l2m2|l3m3> Y_l3m3 and <l1 0 l2 0|l3 0> = +-sqrt(2l3+1) (l1 l2 l3; 0 0 0);
    a coupling tensor with sum_{m1m2} C C = identity therefore gives
    sum C[m1,m2,m3] Y_l1m1(n) Y_l2m2(n) = c Y_l3m3(n), |c| = sqrt((2l1+1)(2l2+1)) |(l1 l2 l3;000)|."""
    from sympy.physics.wigner import wigner_3j
    l1, l2, l3 = t
    n = _unit(7, 6)
    Y = O.spherical_harmonics(n, 3)
    C = O.coupling_tensor(*t)
    out = np.einsum("abc,ea,eb->ec", C, Y[l1], Y[l2])
    w = float(wigner_3j(l1, l2, l3, 0, 0, 0))
    cmag = math.sqrt((2 * l1 + 1) * (2 * l2 + 1)) * abs(w)
    if (l1 + l2 + l3) % 2 == 1:
        np.testing.assert_allclose(out, 0, atol=1e-12)      # odd triples vanish on equal directions
    else:
        ratio = out / Y[l3]
        np.testing.assert_allclose(np.abs(ratio), cmag, rtol=1e-11)
        assert np.ptp(np.sign(ratio)) == 0


def test_cg_golden_worked_values():
    """Worked values printed in SURVEY.md §8c (pins row 'Coupling tensors')."""
    g = json.load(open(os.path.join(GOLD, "coupling_worked_values.json")))
    C = O.coupling_tensor(1, 1, 2)
    for (m1, m2, m3, val) in g["C112_entries"]:
        assert abs(C[m1 + 1, m2 + 1, m3 + 2] - val) < 1e-9
    assert np.count_nonzero(C) == g["C112_nnz"]
    for key, nnz in g["nnz"].items():
        t = tuple(int(c) for c in key)
        assert np.count_nonzero(O.coupling_tensor(*t)) == nnz
    n = _unit(5, 7)
    Y = O.spherical_harmonics(n, 3)
    for key, c in g["same_direction_coeff"].items():
        l1, l2, l3 = (int(ch) for ch in key)
        out = np.einsum("abc,ea,eb->ec", O.coupling_tensor(l1, l2, l3), Y[l1], Y[l2])
        np.testing.assert_allclose(out, c * Y[l3], atol=2e-9)
