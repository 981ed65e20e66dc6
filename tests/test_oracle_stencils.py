"""Pins of the oracle's linear operators -- CPU only.

Each test checks the oracle against something other than itself: coefficients the paper prints
(tests/golden/*.txt), polynomial exactness / moments (closed forms), or analytic derivatives.
"""
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import meg6_oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def impulse_response(op, half=8):
    """coefficient of f[c+m] in op(f)[c], for m = -half..half"""
    n = 4 * half + 1
    c = 2 * half
    out = {}
    for m in range(-half, half + 1):
        f = np.zeros(n)
        f[c + m] = 1.0
        out[m] = O.line_op(op, f)[c]
    return out


def read_eq41():
    rows = [l.split() for l in open(os.path.join(GOLD, "eq41_consistent_derivative.txt")) if l.strip() and l[0] != "#"]
    return {int(m): int(c) for m, c in rows}


def test_delta_matches_eq41_printed_coefficients():
    """Eq. 41: (2282,-546,89,-3,-1)/2880 on antisymmetric offsets 1..5."""
    gold = read_eq41()
    r = impulse_response("delta")
    for m in range(1, 9):
        want = gold.get(m, 0) / 2880.0
        assert r[m] == pytest.approx(want, abs=2e-16)
        assert r[-m] == pytest.approx(-want, abs=2e-16)
    assert abs(r[0]) < 1e-16


def test_H_stencil_consistent_with_eq41():
    """H must be the interface value whose difference is Eq. 41: telescoping sums of the delta
    coefficients give (-1,-4,85,-461,1821 | 1821,...)/2880 on cells i-4..i+5 (Eq. 36-37)."""
    gold = read_eq41()
    c = {m: Fraction(gold.get(abs(m), 0) * (1 if m > 0 else -1), 2880) for m in range(-6, 7)}
    c[0] = Fraction(0)
    # delta_i = H_{i+1/2} - H_{i-1/2};  H_{i+1/2} = sum_q h_q f_{i+q}  =>  c_m = h_m - h_{m+1}... solve by telescoping
    h = {}
    acc = Fraction(0)
    for q in range(-6, 7):          # h_q = sum_{m <= q} c'_m with c'_m = coefficient of f_{i+m} in delta_i, shifted
        acc += c[q]
        h[q] = -acc                 # H_{i-1/2} has weights -cumsum; H_{i+1/2}: shift by one
    r = impulse_response("H")
    for q in range(-5, 7):
        assert r[q] == pytest.approx(float(h[q - 1]), abs=3e-16), q
    want = [-1, -4, 85, -461, 1821, 1821, -461, 85, -4, -1]
    got = [r[q] * 2880 for q in range(-4, 6)]
    assert np.allclose(got, want, atol=1e-12)


def test_Lft_Rgt_stencils_and_mirror():
    """Eq. 16 with Eq. 17/19 substituted: Lft*1440 = (-1,-3,64,-309,1050,771,-152,21,-1) on i-4..i+4;
    Rgt is its mirror image."""
    L = impulse_response("Lft")
    R = impulse_response("Rgt")
    want = [-1, -3, 64, -309, 1050, 771, -152, 21, -1]
    assert np.allclose([L[m] * 1440 for m in range(-4, 5)], want, atol=1e-11)
    for m in range(-8, 9):
        assert L[m] == pytest.approx(R[-m], abs=1e-16)


def poly_at_zero(op, deg, half=8):
    x = np.arange(-2 * half, 2 * half + 1, dtype=float)
    return O.line_op(op, x ** deg)[2 * half]


def test_D1_is_sixth_order_Eq17():
    """E6 gradient exact up to degree 6; first error moment D1[x^7]_0 = 36 (= 7!/140)."""
    assert poly_at_zero("D1", 1) == pytest.approx(1.0, abs=1e-14)
    for d in (0, 2, 3, 4, 5, 6):
        assert abs(poly_at_zero("D1", d)) < 1e-9
    assert poly_at_zero("D1", 7) == pytest.approx(36.0, rel=1e-12)


def test_D2_moments_Eq19():
    """Eq. 19 with E6 gradients: exact to degree 5 (D2[x^2]=2), sixth moment -2; stencil
    {0:-13/4, 1:77/40, 2:-11/30, 3:3/40, 4:-1/120}."""
    assert poly_at_zero("D2", 2) == pytest.approx(2.0, abs=1e-13)
    for d in (0, 1, 3, 4, 5):
        assert abs(poly_at_zero("D2", d)) < 1e-9
    assert poly_at_zero("D2", 6) == pytest.approx(6 * 5 * 0 - 2.0, rel=1e-10)
    r = impulse_response("D2")
    want = {0: -13 / 4, 1: 77 / 40, 2: -11 / 30, 3: 3 / 40, 4: -1 / 120, 5: 0.0}
    for m, v in want.items():
        assert r[m] == pytest.approx(v, abs=1e-15) and r[-m] == pytest.approx(v, abs=1e-15)


def test_delta_is_fourth_order():
    """delta exact to degree 4, delta[x^5]_0 = 1/6, i.e. delta f = f' + f^(5)/720 + ...."""
    assert poly_at_zero("delta", 1) == pytest.approx(1.0, abs=1e-14)
    for d in (0, 2, 3, 4):
        assert abs(poly_at_zero("delta", d)) < 1e-10
    assert poly_at_zero("delta", 5) == pytest.approx(1.0 / 6.0, rel=1e-11)


def test_H_is_the_conservative_flux_function_to_fourth_order():
    """Eq. 15-16: the interface value is the one whose difference is the point derivative
    (flux function h = f - f2/24 + 7 f4/5760, f2/f4 = 2nd/4th derivatives): H[x^d](1/2) in
    closed form for d <= 3, and H(i+1/2) - H(i-1/2) = delta (Eq. 37)."""
    rng = np.random.default_rng(0)
    f = rng.standard_normal(40)
    H = O.line_op("H", f)
    d = O.line_op("delta", f)
    for i in range(8, 30):
        assert d[i] == pytest.approx(H[i] - H[i - 1], abs=1e-14)
    x = np.arange(-16, 17, dtype=float)
    want = {0: 1.0, 1: 0.5, 2: 0.25 - 2 / 24, 3: 0.125 - 3 / 24}
    for deg, v in want.items():
        assert O.line_op("H", x ** deg)[16] == pytest.approx(v, abs=1e-11)
    # degree 4: exact away from the origin too (delta[x^4]_i = 4 i^3)
    d4 = O.line_op("delta", x ** 4)
    for i in (-3, -1, 2, 4):
        assert d4[16 + i] == pytest.approx(4.0 * i ** 3, abs=1e-9)


def test_alpha_damping_interface_gradient_P4():
    """Eq. 29-31 with alpha^D=4, beta^D=0: stencil (1/120,-1/15,3/10,-13/8,13/8,...) on
    i-3..i+4, and the difference of consecutive interface gradients equals Eq. 19's D2 exactly
    (=> fourth order)."""
    r = impulse_response("alpha_damp")
    want = [1 / 120, -1 / 15, 3 / 10, -13 / 8, 13 / 8, -3 / 10, 1 / 15, -1 / 120]
    assert np.allclose([r[m] for m in range(-3, 5)], want, atol=1e-15)
    rng = np.random.default_rng(1)
    f = rng.standard_normal(40)
    g = O.line_op("alpha_damp", f)
    d2 = O.line_op("D2", f)
    for i in range(6, 32):
        assert g[i] - g[i - 1] == pytest.approx(d2[i], abs=2e-14)


@pytest.mark.parametrize("op,order,deriv", [("D1", 6, 1), ("delta", 4, 1), ("D2", 4, 2)])
def test_convergence_on_analytic_function(op, order, deriv):
    """brute force against analytic derivatives of sin (P9)."""
    errs = []
    for n in (32, 64):
        h = 2 * np.pi / n
        x = np.arange(-12, n + 12) * h
        f = np.sin(x + 0.3)
        num = O.line_op(op, f) / h ** deriv
        exact = np.cos(x + 0.3) if deriv == 1 else -np.sin(x + 0.3)
        sl = slice(12, n + 12)
        errs.append(np.abs(num[sl] - exact[sl]).max())
    rate = np.log2(errs[0] / errs[1])
    assert rate > order - 0.4, (errs, rate)


def test_eq43_printed_terms_of_metric_identity():
    """Eq. 43: d/dxi(xi_x-hat) over the denominator 2880^3 = 23887872000 starts with
    -1 y[i-5,j-5,k-5] z[i-5,j-5,k], -3 y[i-5,j-5,k-4] z[i-5,j-5,k] and ends with +3, +1 terms.
    Probed through the oracle's metric routine with impulse coordinates (bilinear in y and z)."""
    rows = [l.split() for l in open(os.path.join(GOLD, "eq43_metric_identity.txt")) if l.strip() and l[0] != "#"]
    den = int(rows[0][1])
    assert den == 2880 ** 3
    n, g = 12, 10
    cfg = dict(ni=n, nj=n, nk=n, periodic=[0, 0, 0], period=[[0.0] * 3] * 3)
    wl = dict(params=cfg, x=np.zeros((n + 1,) * 3), y=np.zeros((n + 1,) * 3), z=np.zeros((n + 1,) * 3))
    c = 6   # probe cell (i,j,k) = (6,6,6)
    for row in rows[1:]:
        yo, zo, num = tuple(map(int, row[0:3])), tuple(map(int, row[3:6])), int(row[6])
        G = O.Grid(wl)
        xc = np.zeros((n + 2 * g,) * 3)
        yc = np.zeros_like(xc)
        zc = np.zeros_like(xc)
        yc[c + g + yo[2], c + g + yo[1], c + g + yo[0]] = 1.0
        zc[c + g + zo[2], c + g + zo[1], c + g + zo[0]] = 1.0
        G.set_centres(xc, yc, zc)
        G.metrics_compute(0.0)
        # d/dxi of the interface-interpolated xi_x-hat = difference of the xi-family interface metric 0
        fx = G.face(0, 0)               # (nk, nj, ni+1): entry s = interface between cells s-1 and s
        val = fx[c, c, c + 1] - fx[c, c, c]
        assert val * den == pytest.approx(num, abs=1e-6), (row, val * den)
