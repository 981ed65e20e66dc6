"""Pins of the oracle's per-interface pieces (SURVEY 8(c) P3, P5, P6 and viscous special cases) -- CPU only."""
import numpy as np
import pytest

from oracle import meg6_oracle as O

G = 1.4


# ------------------------------------------------------------------ eigenvectors, App. A (P3)
def B_matrix(n, gnorm, rho, u, p, gamma=G):
    """coefficient matrix B_xi of Eq. A.2 for metric vector gnorm*n (1/J dropped, static)."""
    kx, ky, kz = gnorm * np.asarray(n)
    U = kx * u[0] + ky * u[1] + kz * u[2]
    return np.array([[U, rho * kx, rho * ky, rho * kz, 0.0],
                     [0.0, U, 0.0, 0.0, kx / rho],
                     [0.0, 0.0, U, 0.0, ky / rho],
                     [0.0, 0.0, 0.0, U, kz / rho],
                     [0.0, gamma * p * kx, gamma * p * ky, gamma * p * kz, U]]), U


@pytest.mark.parametrize("seed", range(5))
def test_eigenvectors_diagonalise_B(seed):
    """L R = I and L B R = diag(U - a|grad xi|, U, U, U, U + a|grad xi|)  (A.3-A.6)."""
    rng = np.random.default_rng(seed)
    n = rng.standard_normal(3)
    n /= np.linalg.norm(n)
    rho, p = rng.uniform(0.5, 2.0, 2)
    u = rng.standard_normal(3)
    gnorm = rng.uniform(0.3, 3.0)
    a = np.sqrt(G * p / rho)
    L, R = O.eigen(n, rho, a)
    assert np.allclose(L @ R, np.eye(5), atol=1e-14)
    B, U = B_matrix(n, gnorm, rho, u, p)
    lam = L @ B @ R
    want = np.diag([U - a * gnorm, U, U, U, U + a * gnorm])
    assert np.allclose(lam, want, atol=1e-12)


def test_eigenvector_entries_match_A6a_first_and_last_rows():
    """rows 1 and 5 of A.6a are the acoustic characteristics dp -/+ rho a n.du."""
    L, R = O.eigen([1.0, 0.0, 0.0], 2.0, 3.0)
    assert np.allclose(L[0], [0, -6.0, 0, 0, 1.0])
    assert np.allclose(L[4], [0, 6.0, 0, 0, 1.0])
    assert np.allclose(R[4], [0.5, 0, 0, 0, 0.5])          # A.4b last row
    assert np.allclose(R[0], [1 / 18.0, 1 / 9.0, 0, 0, 1 / 18.0])


# ------------------------------------------------------------------ HLLC (P5)
def flux_of_state(P, m, gamma=G):
    """Eq. 2 typed independently."""
    r, u, v, w, p = P
    mx, my, mz, mt = m
    Uh = mt + mx * u + my * v + mz * w
    E = p / (gamma - 1) + 0.5 * r * (u * u + v * v + w * w)
    return np.array([r * Uh, r * u * Uh + mx * p, r * v * Uh + my * p, r * w * Uh + mz * p, (E + p) * Uh - mt * p])


def toro_hllc_1d(PL, PR, gamma=G):
    """Textbook HLLC (Toro, Riemann Solvers, 3rd ed., Eq. 10.37-10.39) with the min/max wave speeds."""
    def cons(P):
        r, u, v, w, p = P
        return np.array([r, r * u, r * v, r * w, p / (gamma - 1) + 0.5 * r * (u * u + v * v + w * w)])

    def flx(P):
        r, u, v, w, p = P
        E = cons(P)[4]
        return np.array([r * u, r * u * u + p, r * u * v, r * u * w, u * (E + p)])
    rl, ul, vl, wl, pl = PL
    rr, ur, vr, wr, pr = PR
    cl, cr = np.sqrt(gamma * pl / rl), np.sqrt(gamma * pr / rr)
    SL, SR = min(ul - cl, ur - cr), max(ul + cl, ur + cr)
    SS = (pr - pl + rl * ul * (SL - ul) - rr * ur * (SR - ur)) / (rl * (SL - ul) - rr * (SR - ur))
    if SL >= 0:
        return flx(PL)
    if SR < 0:
        return flx(PR)

    def star(P, S):
        r, u, v, w, p = P
        E = cons(P)[4]
        f = r * (S - u) / (S - SS)
        return f * np.array([1.0, SS, v, w, E / r + (SS - u) * (SS + p / (r * (S - u)))])
    if SS >= 0:
        return flx(PL) + SL * (star(PL, SL) - cons(PL))
    return flx(PR) + SR * (star(PR, SR) - cons(PR))


@pytest.mark.parametrize("seed", range(8))
def test_hllc_reduces_to_textbook_1d(seed):
    """m = (1,0,0,0): Eq. 26-27 must equal the 1-D textbook HLLC, transverse velocities included."""
    rng = np.random.default_rng(100 + seed)
    PL = np.array([rng.uniform(0.5, 2), rng.normal(0, 0.8), rng.normal(), rng.normal(), rng.uniform(0.5, 2)])
    PR = np.array([rng.uniform(0.5, 2), rng.normal(0, 0.8), rng.normal(), rng.normal(), rng.uniform(0.5, 2)])
    if seed == 6:
        PL[1], PR[1] = 3.0, 2.5     # supersonic to the right
    if seed == 7:
        PL[1], PR[1] = -3.0, -2.5   # supersonic to the left
    F, br = O.hllc(PL, PR, [1.0, 0.0, 0.0, 0.0])
    assert np.allclose(F, toro_hllc_1d(PL, PR), rtol=1e-13, atol=1e-13)
    if seed == 6:
        assert br == 0 and np.allclose(F, flux_of_state(PL, [1, 0, 0, 0]))
    if seed == 7:
        assert br == 3 and np.allclose(F, flux_of_state(PR, [1, 0, 0, 0]))


@pytest.mark.parametrize("seed", range(6))
def test_hllc_rotated_and_scaled_normal_equals_1d_in_normal_frame(seed):
    """For m = g*n the contravariant HLLC equals g times the textbook flux in the frame aligned with n,
    rotated back (rotational invariance of the Euler equations)."""
    rng = np.random.default_rng(200 + seed)
    n = rng.standard_normal(3)
    n /= np.linalg.norm(n)
    t1 = np.cross(n, [0.3, -0.7, 0.64])
    t1 /= np.linalg.norm(t1)
    t2 = np.cross(n, t1)
    Q = np.array([n, t1, t2])      # rows: new axes
    g = rng.uniform(0.2, 4.0)

    def rnd():
        return np.array([rng.uniform(0.5, 2), *rng.normal(0, 0.7, 3), rng.uniform(0.5, 2)])
    PL, PR = rnd(), rnd()
    F, _ = O.hllc(PL, PR, [g * n[0], g * n[1], g * n[2], 0.0])
    rot = lambda P: np.array([P[0], *(Q @ P[1:4]), P[4]])
    F1 = toro_hllc_1d(rot(PL), rot(PR))
    back = np.array([F1[0], *(Q.T @ F1[1:4]), F1[4]]) * g
    assert np.allclose(F, back, rtol=1e-12, atol=1e-12)


def test_hllc_consistency_and_grid_velocity_term():
    """F(P,P,m) = F(P) of Eq. 2 including xi_t: Q*Uhat + p*(0,mx,my,mz,Uhat - mt)  (Eq. 4)."""
    rng = np.random.default_rng(5)
    for _ in range(10):
        P = np.array([rng.uniform(0.5, 2), *rng.normal(0, 0.7, 3), rng.uniform(0.5, 2)])
        m = np.array([*rng.normal(0, 1, 3), rng.normal(0, 0.5)])
        F, _ = O.hllc(P, P, m)
        assert np.allclose(F, flux_of_state(P, m), rtol=1e-12, atol=1e-12)


def test_hllc_stationary_contact_has_zero_mass_flux():
    m = np.array([0.6, -0.3, 0.5])
    uL, uR = 0.3 * np.cross(m, [1.0, 0, 0]), 0.2 * np.cross(m, [0, 1.0, 0])   # tangential only
    PL = np.array([1.0, *uL, 1.0])
    PR = np.array([0.25, *uR, 1.0])
    F, _ = O.hllc(PL, PR, [*m, 0.0])
    assert abs(F[0]) < 1e-15 and abs(F[4]) < 1e-15
    assert np.allclose(F[1:4], [0.6, -0.3, 0.5])


def test_hllc_moving_interface_galilean_invariance():
    """An interface moving with normal speed s (mt = -s*g) sees the flux F(static, u - s n) + s*(...):
    for a uniform state the mass flux is rho*(Uhat) with Uhat = mt + m.u."""
    P = np.array([1.3, 0.4, -0.2, 0.1, 0.9])
    m = np.array([0.8, 0.1, -0.3, -0.25])
    F, _ = O.hllc(P, P, m)
    Uh = m[3] + m[:3] @ P[1:4]
    assert F[0] == pytest.approx(P[0] * Uh, rel=1e-13)


# ------------------------------------------------------------------ MP limiter (P6)
def test_limiter_accepts_smooth_monotone_data():
    """App. E, E.1: for smooth monotone data the unlimited value lies between W_i and W^MP."""
    x = np.arange(-8, 9, dtype=float) * 0.1
    f = np.tanh(x) + 2.0
    d = O.line_op("D2", f)
    Lf = O.line_op("Lft", f)
    mm = lambda a, b: 0.5 * (np.sign(a) + np.sign(b)) * min(abs(a), abs(b))
    for i in range(6, 11):
        v, fl = O.mp_limit(Lf[i], f[i], f[i - 1], f[i + 1], mm(d[i], d[i + 1]), mm(d[i - 1], d[i]))
        assert fl == 0 and v == Lf[i]


def test_limiter_bounds_at_isolated_step():
    """step data: result within [min,max] of (W_i, W_{i+1}) -- no new extrema (Suresh-Huynh property)."""
    f = np.where(np.arange(20) < 10, 1.0, 0.0)
    d = O.line_op("D2", f)
    Lf = O.line_op("Lft", f)
    mm = lambda a, b: 0.5 * (np.sign(a) + np.sign(b)) * min(abs(a), abs(b))
    n_lim = 0
    for i in range(6, 14):
        v, fl = O.mp_limit(Lf[i], f[i], f[i - 1], f[i + 1], mm(d[i], d[i + 1]), mm(d[i - 1], d[i]))
        n_lim += fl
        assert min(f[i], f[i + 1]) - 1e-14 <= v <= max(f[i], f[i + 1]) + 1e-14
    assert n_lim > 0


def test_limiter_large_alpha_never_limits_monotone():
    v, fl = O.mp_limit(1.7, 1.0, 0.5, 2.0, 0.0, 0.0, alpha=1e9)
    assert fl == 0 and v == 1.7


def test_limiter_formulae_on_hand_computed_case():
    """E.2-E.4 evaluated by hand: c0=1, cm=0, cp=1.5, alpha=4, dM_near=0.2, dM_far=-0.1, w=2:
    WMP = 1 + minmod(0.5, 4) = 1.5; (2-1)(2-1.5) > 0 -> limit.  WMD = 1.25-0.1 = 1.15; WUL = 5;
    WLC = 1.5 + 4/3*(-0.1) = 1.3666..; Wmin = max(min(1,1.5,1.15), min(1,5,1.3667)) = 1;
    Wmax = min(max(1,1.5,1.15), max(1,5,1.3667)) = 1.5; result = 2 + minmod(-1,-0.5) = 1.5."""
    v, fl = O.mp_limit(2.0, 1.0, 0.0, 1.5, 0.2, -0.1, alpha=4.0)
    assert fl == 1 and v == pytest.approx(1.5, abs=1e-15)


def test_limiter_hand_computed_cases_where_WMD_and_WLC_bind():
    """E.3-E.4 by hand, alpha = 4, chosen so that the median (W^MD) and the large-curvature (W^LC)
    bounds are the ones that decide -- the first hand-computed case is decided by c_p alone.
    A: c0=1, cm=0.5, cp=1.2, dM_near=-0.4, dM_far=0.3, w=1.5: WMP = 1 + minmod(0.2, 2) = 1.2, (0.5)(0.3) > 0 -> limit;
       WMD = 1.1 + 0.2 = 1.3, WUL = 3, WLC = 1.25 + 0.4 = 1.65; Wmin = max(1, 1) = 1, Wmax = min(1.3, 3) = 1.3;
       result = 1.5 + minmod(-0.5, -0.2) = 1.3                                          (W^MD binds).
    B: c0=1, cm=1.1, cp=1.5, dM_near=0.1, dM_far=0.15, w=1.4: WMP = 1 + minmod(0.5, -0.4) = 1, (0.4)(0.4) > 0 -> limit;
       WMD = 1.25 - 0.05 = 1.2, WUL = 0.6, WLC = 0.95 + 4/3 0.15 = 1.15; Wmin = max(1, 0.6) = 1,
       Wmax = min(1.5, max(1, 0.6, 1.15)) = 1.15; result = 1.4 + minmod(-0.4, -0.25) = 1.15   (W^LC with its 4/3 binds).
    The limiter is odd: negating every argument negates the result (W^min and W^max swap roles)."""
    for args, want in (((1.5, 1.0, 0.5, 1.2, -0.4, 0.3), 1.3), ((1.4, 1.0, 1.1, 1.5, 0.1, 0.15), 1.15)):
        v, fl = O.mp_limit(*args, alpha=4.0)
        assert fl == 1 and v == pytest.approx(want, abs=1e-15)
        v, fl = O.mp_limit(*(-a for a in args), alpha=4.0)
        assert fl == 1 and v == pytest.approx(-want, abs=1e-15)


# ------------------------------------------------------------------ full inviscid interface (O3)
def test_inviscid_face_uniform_state_returns_exact_flux():
    P = np.array([1.2, 0.3, -0.1, 0.2, 0.8])
    m = np.array([0.7, -0.2, 0.4, 0.15])
    F = O.inviscid_face(np.tile(P, (4, 1)), np.zeros((2, 5)), np.zeros((4, 5)), m)
    assert np.allclose(F, flux_of_state(P, m), rtol=1e-12, atol=1e-13)


@pytest.mark.parametrize("rough", [0, 1, 2, 3, 4, 5])
def test_inviscid_face_mirror_symmetry_L_R(rough):
    """R8: the right state is the mirror image of the left one: reflecting the data about the interface
    (cells reversed, normal velocity and gradients' sign flipped) must flip mass/energy flux and keep the
    normal momentum flux.  rough > 0: seeded cell-to-cell noise on every field, so that both states are limited with
    all of d^M_near, d^M_far of E.3 non-zero and different on the two sides."""
    rng = np.random.default_rng(3 + rough)
    x = np.arange(-6, 6) + 0.5          # cell centres; interface at 0 between index 5 and 6
    P = np.stack([1 + 0.2 * np.sin(0.4 * x + 1), 0.3 + 0.2 * np.cos(0.3 * x), 0.1 * np.sin(0.5 * x),
                  0.05 * x, 1 + 0.1 * np.cos(0.45 * x + 2)], axis=1)
    # add a kink so that the limiter is active on some component
    P[7:, 0] += 0.4
    if rough:
        P += 0.08 * rng.standard_normal(P.shape)

    def face(Pa):
        g1 = np.stack([O.line_op("D1", Pa[:, f]) for f in range(5)], axis=1)
        g2 = np.stack([O.line_op("D2", Pa[:, f]) for f in range(5)], axis=1)
        return O.inviscid_face(Pa[4:8], g1[5:7], g2[4:8], [1.0, 0.0, 0.0, 0.0])
    F = face(P)
    Pm = P[::-1].copy()
    Pm[:, 1] *= -1.0
    Fm = face(Pm)
    assert np.allclose(Fm, F * np.array([-1, 1, -1, -1, -1]), rtol=1e-12, atol=1e-13)


def test_inviscid_face_linear_advection_limit_is_upwind_fourth_order():
    """Smooth density wave carried by a uniform supersonic stream (u > a): HLLC returns F(P^L) and the
    left state is Eq. 21 applied component-wise (the characteristic projection is linear and frozen), so
    the mass flux equals u * Lft[rho]."""
    x = np.arange(-6, 6) + 0.5
    rho = 1 + 0.1 * np.sin(0.3 * x)
    P = np.stack([rho, 3.0 + 0 * x, 0 * x, 0 * x, 1.0 + 0 * x], axis=1)
    g1 = np.stack([O.line_op("D1", P[:, f]) for f in range(5)], axis=1)
    g2 = np.stack([O.line_op("D2", P[:, f]) for f in range(5)], axis=1)
    F = O.inviscid_face(P[4:8], g1[5:7], g2[4:8], [1.0, 0.0, 0.0, 0.0])
    lft = O.line_op("Lft", rho)[5]
    assert F[0] == pytest.approx(3.0 * lft, rel=1e-13)


# ------------------------------------------------------------------ viscous interface (O4)
CFG = dict(gamma=1.4, r_gas=1.0, prandtl=0.71, mu_ref=0.01, t_ref=1.0, s_suth=-1.0, viscous=1)


def test_viscous_face_pure_shear():
    """u = s*y on a Cartesian grid (spacing h): tau_xy = mu s; eta-interface flux = (0, h^2 mu s, 0, 0, h^2 u mu s)."""
    h, s, mu = 0.5, 2.0, 0.01
    mh = np.diag([h * h] * 3).reshape(9)        # hatted metrics of a uniform grid: (dy dz, ...) ; 1/J = h^3
    rj = h ** 3
    # eta-interface between cells j, j+1 at y = 0: cell values u = s*(-h/2), s*(h/2); gradient per index = s*h
    phi = np.array([[-s * h / 2, 0, 0, 1.0], [s * h / 2, 0, 0, 1.0]])
    g = np.zeros((2, 3, 4))
    g[:, 1, 0] = s * h
    Fv = O.viscous_face(1, phi, g, mh, rj, CFG)
    assert np.allclose(Fv, [0, h * h * mu * s, 0, 0, 0], atol=1e-15)


def test_viscous_face_stokes_hypothesis_and_heat_flux():
    """isotropic dilatation u_x=v_y=w_z=d: tau_ii = 2 mu d - 2/3 mu 3d = 0; T gradient gives
    kappa T_x with kappa = mu gamma R/((gamma-1) Pr)."""
    h, d, mu = 1.0, 0.3, 0.01
    mh = np.eye(3).reshape(9)
    phi = np.array([[-d / 2, 0, 0, 1.0], [d / 2, 0, 0, 1.2]])
    g = np.zeros((2, 3, 4))
    g[:, 0, 0] = d
    g[:, 1, 1] = d
    g[:, 2, 2] = d
    g[:, 0, 3] = 0.2
    Fv = O.viscous_face(0, phi, g, mh, 1.0, CFG)
    kap = mu * 1.4 * 1.0 / (0.4 * 0.71)
    assert np.allclose(Fv[:4], 0.0, atol=1e-16)
    assert Fv[4] == pytest.approx(kap * 0.2, rel=1e-13)   # u = 0 at the interface


def test_viscous_face_damping_term_only_on_normal_direction():
    """Eq. 29: with zero cell gradients and a jump in u across a xi-interface the interface
    gradient is alpha^D/2 * (uR - uL) = 2*jump along xi only."""
    mh = np.eye(3).reshape(9)
    phi = np.array([[0.0, 0, 0, 1.0], [0.1, 0, 0, 1.0]])
    g = np.zeros((2, 3, 4))
    Fv = O.viscous_face(0, phi, g, mh, 1.0, CFG)
    ux = 2.0 * 0.1
    txx = 2 * 0.01 * ux - 2.0 / 3.0 * 0.01 * ux
    assert Fv[1] == pytest.approx(txx, rel=1e-13)
    assert Fv[4] == pytest.approx(0.05 * txx, rel=1e-13)


def test_viscous_face_normal_gradient_is_the_P4_stencil_and_differences_to_D2():
    """P4 through the function the right-hand side calls (not the line-operator restatement): on unit Cartesian metrics
    with a velocity u(xi) alone, F_v[1] = (2 mu + lambda) u_xi = 4/3 mu g_{i+1/2}.  The interface gradient of Eq. 29-31
    (alpha^D = 4, beta^D = 0) has the stencil (1/120, -1/15, 3/10, -13/8, 13/8, -3/10, 1/15, -1/120) on
    i-3..i+4 and consecutive interface gradients differ by Eq. 19's D2 exactly (fourth order)."""
    mh = np.eye(3).reshape(9)
    mu = CFG["mu_ref"]

    def iface_grad(f):
        d1 = O.line_op("D1", f)
        out = np.full(f.size, np.nan)
        for i in range(3, f.size - 4):
            phi = np.array([[f[i], 0, 0, 1.0], [f[i + 1], 0, 0, 1.0]])
            g = np.zeros((2, 3, 4))
            g[0, 0, 0], g[1, 0, 0] = d1[i], d1[i + 1]
            out[i] = O.viscous_face(0, phi, g, mh, 1.0, CFG)[1] / (4.0 / 3.0 * mu)
        return out
    imp = np.zeros(21)
    imp[10] = 1.0
    r = iface_grad(imp)
    want = [1 / 120, -1 / 15, 3 / 10, -13 / 8, 13 / 8, -3 / 10, 1 / 15, -1 / 120]
    # response at interface i+1/2 to an impulse at cell 10 = stencil weight of offset 10 - i
    assert np.allclose([r[10 - m] for m in range(-3, 5)], want, atol=1e-14)
    f = np.random.default_rng(3).standard_normal(40)
    g = iface_grad(f)
    d2 = O.line_op("D2", f)
    for i in range(6, 32):
        assert g[i] - g[i - 1] == pytest.approx(d2[i], abs=5e-14)


def test_sutherland():
    cfg = dict(CFG, s_suth=110.4 / 293.0, mu_ref=2.0)
    assert O.sutherland(cfg, 1.0) == pytest.approx(2.0)
    T = 1.7
    S = 110.4 / 293.0
    assert O.sutherland(cfg, T) == pytest.approx(2.0 * T ** 1.5 * (1 + S) / (T + S), rel=1e-14)
