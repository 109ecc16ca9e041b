"""Pins for the CPU oracle: every check here compares oracle/sledge_oracle.cpp with something OTHER than
itself -- closed forms, textbook routines, invariants, brute force, or values printed in the paper
(tests/golden/).  CPU only.  SURVEY.md section 8(c) "What pins each part"; DESIGN.md "Oracle pins"."""
import math
import os

import numpy as np
import pytest

from oracle.oracle import Oracle, OracleError, plaquette_winding
from paper_2404_02950_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def single(n, **kw):
    return Oracle(n, **kw)


def coords(shape):
    z, y, x = np.meshgrid(*[np.arange(s, dtype=np.float64) for s in shape], indexing="ij")
    return x, y, z


# ------------------------------------------------------------------------------------------------
# O2 Laplacian
# ------------------------------------------------------------------------------------------------


@pytest.mark.parametrize("order,deg", [(1, 2), (1, 3), (2, 4), (2, 5), (3, 6), (3, 7)])
def test_laplacian_exact_on_polynomials(order, deg):
    """Central 3-point (5-, 7-point) second differences are exact on cubics (quintics, septics) per axis.  Ghosts
    are filled analytically on a NON-periodic box, so a wrong coefficient, sign or axis shows up directly."""
    g = 3 if order == 3 else 2
    n = (8, 16, 24)  # x, y, z -- all different to catch a transposed index
    h = 0.37
    o = Oracle(n, nghost=g, blocking_factor=8, lap_order=order, h0=h, lam=0.0)
    zz, yy, xx = np.meshgrid(*[(np.arange(-g, s + g) + 0.5) * h for s in n[::-1]], indexing="ij")
    rng = np.random.default_rng(7)
    cx, cy, cz = rng.uniform(-1, 1, size=(3, deg + 1))

    def poly(c, t):
        return sum(c[m] * t ** m for m in range(deg + 1))

    def d2poly(c, t):
        return sum(m * (m - 1) * c[m] * t ** (m - 2) for m in range(2, deg + 1))

    # separable sum + a cross term that every axis-wise second difference treats exactly
    u1 = poly(cx, xx) + poly(cy, yy) + poly(cz, zz) + 0.3 * xx * yy * zz
    lap1 = d2poly(cx, xx) + d2poly(cy, yy) + d2poly(cz, zz)
    u2 = 2.0 * poly(cz, xx) - poly(cx, yy) + 0.5 * poly(cy, zz)
    lap2 = 2.0 * d2poly(cz, xx) - d2poly(cx, yy) + 0.5 * d2poly(cy, zz)
    o.set_raw(0, 0, u1)
    o.set_raw(0, 1, u2)
    k = o.eval_rhs(0, eta=1.0, fill=False)[0]
    v = slice(g, -g)
    scale = np.abs(u1).max() / h ** 2
    assert np.abs(k[2] - lap1[v, v, v]).max() < 1e-12 * scale
    assert np.abs(k[3] - lap2[v, v, v]).max() < 1e-12 * scale
    # k_psi = Pi (Eq.10): Pi was zero
    assert np.all(k[0] == 0) and np.all(k[1] == 0)


def test_laplacian_order1_not_exact_on_quartic():
    """Sanity of the pin above: the 3-point stencil must NOT be exact on x^4 (error h^2/12 * 24)."""
    g, n, h = 1, (8, 8, 8), 0.5
    o = Oracle(n, nghost=g, lap_order=1, h0=h, lam=0.0)
    zz, yy, xx = np.meshgrid(*[(np.arange(-g, s + g) + 0.5) * h for s in n], indexing="ij")
    o.set_raw(0, 0, xx ** 4)
    k = o.eval_rhs(0, 1.0, fill=False)[0]
    err = k[2] - 12 * xx[1:-1, 1:-1, 1:-1] ** 2
    assert np.allclose(err, 2 * h ** 2, rtol=1e-9)


def test_laplacian_order2_not_exact_on_sextic():
    """The 5-point stencil must NOT be exact on x^6: its error is -(h^4/90) u^(6) = -8 h^4, which the 7-point stencil
    of order 3 removes (separates the two on the same data)."""
    g, n, h = 3, (8, 8, 8), 0.5
    zz, yy, xx = np.meshgrid(*[(np.arange(-g, s + g) + 0.5) * h for s in n], indexing="ij")
    v = slice(g, -g)
    exact = 30 * xx[v, v, v] ** 4
    res = {}
    for order in (2, 3):
        o = Oracle(n, nghost=g, lap_order=order, h0=h, lam=0.0)
        o.set_raw(0, 0, xx ** 6)
        res[order] = o.eval_rhs(0, 1.0, fill=False)[0][2] - exact
    assert np.allclose(res[2], -8 * h ** 4, rtol=1e-8)
    assert np.abs(res[3]).max() < 1e-9


@pytest.mark.parametrize("order", [1, 2, 3])
def test_laplacian_symbol_on_plane_waves(order):
    """exp(i k.x) is an eigenvector of the periodic discrete Laplacian with eigenvalue
    -(1/h^2) sum_i 4 sin^2(k_i h/2)                                                   (order 1)
    -(1/h^2) sum_i [16/3 sin^2(k_i h/2) - 1/3 sin^2(k_i h)]                           (order 2)
    -(1/h^2) sum_i [6 sin^2(k_i h/2) - 3/5 sin^2(k_i h) + 2/45 sin^2(3 k_i h/2)]      (order 3)."""
    n = (16, 24, 32)
    h = 0.8
    o = Oracle(n, nghost=3, lap_order=order, h0=h, lam=0.0)
    x, y, z = coords(n[::-1])
    m = (3, 2, 5)  # mode numbers per axis
    kh = [2 * math.pi * m[d] / n[d] for d in range(3)]
    ph = kh[0] * x + kh[1] * y + kh[2] * z
    o.set_state(0, 0, np.cos(ph))
    o.set_state(0, 1, np.sin(ph))
    k = o.eval_rhs(0, 1.0)[0]
    if order == 1:
        ev = -sum(4 * math.sin(a / 2) ** 2 for a in kh) / h ** 2
    elif order == 2:
        ev = -sum(16 / 3 * math.sin(a / 2) ** 2 - 1 / 3 * math.sin(a) ** 2 for a in kh) / h ** 2
    else:
        ev = -sum(6 * math.sin(a / 2) ** 2 - 0.6 * math.sin(a) ** 2 + 2 / 45 * math.sin(1.5 * a) ** 2 for a in kh) / h ** 2
    assert np.abs(k[2] - ev * np.cos(ph)).max() < 1e-12 * abs(ev)
    assert np.abs(k[3] - ev * np.sin(ph)).max() < 1e-12 * abs(ev)


# ------------------------------------------------------------------------------------------------
# O10 Kreiss-Oliger dissipation (Eq.7; dissipation_order r in {2,3} = ghost cells, p = 2r - 1, L751)
# ------------------------------------------------------------------------------------------------

KO_EPS = (0.013, 0.021, 0.034, 0.055)  # all different: a swapped component index shows up


@pytest.mark.parametrize("r", [2, 3])
def test_ko_annihilates_low_degree_and_is_exact_on_the_leading_monomial(r):
    """Eq.7 applied to a monomial, by hand: Q x^m = 0 for m <= 2r - 1 = p, and for u = (x/h)^(2r) the (p+1)-st
    derivative is (2r)!/h^(2r), so Q u = (-1)^((p+3)/2) eps h^p / 2^(p+1) * (2r)!/h^(2r)
    = -1.5 eps/h (r = 2) and +11.25 eps/h (r = 3), the same for every cell.  The (2r+1)-point central difference is
    exact on both, so sign, normalisation, power of h and the axis sum are all pinned; ghosts are analytic on a
    non-periodic box; lambda = 0 and Laplacian<1> of the same data is subtracted analytically."""
    g, n, h = r, (8, 16, 24), 0.37
    o = Oracle(n, nghost=g, lap_order=1, h0=h, lam=0.0, ko_order=r, ko_strength=KO_EPS)
    kk, jj, ii = np.meshgrid(*[np.arange(-g, s + g, dtype=np.float64) for s in n[::-1]], indexing="ij")
    v = slice(g, -g)
    # degree <= p per axis (plus a cross term): Q vanishes on every component
    rng = np.random.default_rng(3)
    co = rng.uniform(-1, 1, size=(4, 3, 2 * r))
    lowdeg = [sum(co[c, 0, m] * (ii / 8) ** m + co[c, 1, m] * (jj / 8) ** m + co[c, 2, m] * (kk / 8) ** m
                  for m in range(2 * r)) + 0.1 * (ii * jj * kk) / 512 for c in range(4)]
    for c in range(4):
        o.set_raw(0, c, lowdeg[c])
    k = o.eval_rhs(0, eta=1.0, fill=False)[0]
    assert np.abs(k[0] - lowdeg[2][v, v, v]).max() < 1e-12  # k_psi = Pi + 0
    assert np.abs(k[1] - lowdeg[3][v, v, v]).max() < 1e-12
    # leading monomials: psi1 = i^(2r), psi2 = j^(2r) + 2 k^(2r), Pi1 = k^(2r), Pi2 = -i^(2r)
    lead = math.factorial(2 * r) / 2 ** (2 * r) / h * (-1 if r == 2 else 1)
    assert lead == (-1.5 / h if r == 2 else 11.25 / h)
    u = [ii ** (2 * r), jj ** (2 * r) + 2 * kk ** (2 * r), kk ** (2 * r), -(ii ** (2 * r))]
    for c in range(4):
        o.set_raw(0, c, u[c])
    k = o.eval_rhs(0, eta=1.0, fill=False)[0]
    want = [KO_EPS[0] * lead, KO_EPS[1] * 3 * lead, KO_EPS[2] * lead, -KO_EPS[3] * lead]
    scale = float(max(n) + g) ** (2 * r)
    assert np.abs(k[0] - (u[2][v, v, v] + want[0])).max() < 1e-13 * scale
    assert np.abs(k[1] - (u[3][v, v, v] + want[1])).max() < 1e-13 * scale
    # k_Pi = Lap<1> psi + Q Pi; second difference of i^(2r) along x, analytic
    d2 = lambda t: ((t + 1) ** (2 * r) - 2 * t ** (2 * r) + (t - 1) ** (2 * r)) / h ** 2
    lap1 = d2(ii)
    lap2 = d2(jj) + 2 * d2(kk)
    assert np.abs(k[2] - (lap1[v, v, v] + want[2])).max() < 1e-13 * scale / h ** 2
    assert np.abs(k[3] - (lap2[v, v, v] + want[3])).max() < 1e-13 * scale / h ** 2


def ko_symbol(r, eps, kh, h):
    """Eq.7 on exp(i k.x) with the derivative as the (2r+1)-point central difference delta^(2r) = (-4 sin^2(kh/2))^r:
    eigenvalue -(eps/h) sum_d sin^(2r)(k_d h/2), never positive: the term only damps."""
    return -(eps / h) * sum(math.sin(a / 2) ** (2 * r) for a in kh)


@pytest.mark.parametrize("r", [2, 3])
def test_ko_symbol_on_plane_waves(r):
    n, h = (16, 24, 32), 0.8
    o = Oracle(n, nghost=3, lap_order=2, h0=h, lam=0.0, ko_order=r, ko_strength=KO_EPS)
    x, y, z = coords(n[::-1])
    m = (3, 2, 5)
    kh = [2 * math.pi * m[d] / n[d] for d in range(3)]
    ph = kh[0] * x + kh[1] * y + kh[2] * z
    amp = (1.0, 0.6, -0.4, 0.9)
    wave = [np.cos(ph), np.sin(ph), np.cos(ph), np.sin(ph)]
    for c in range(4):
        o.set_state(0, c, amp[c] * wave[c])
    k = o.eval_rhs(0, 1.0)[0]
    lap = -sum(16 / 3 * math.sin(a / 2) ** 2 - 1 / 3 * math.sin(a) ** 2 for a in kh) / h ** 2
    q = [ko_symbol(r, KO_EPS[c], kh, h) for c in range(4)]
    for c in range(2):
        assert np.abs(k[c] - (amp[c + 2] + q[c] * amp[c]) * wave[c]).max() < 1e-14
        assert np.abs(k[c + 2] - (lap * amp[c] + q[c + 2] * amp[c + 2]) * wave[c]).max() < 1e-13 * abs(lap)
    # the Nyquist checkerboard is damped at the largest rate, -3 eps/h
    cb = (-1.0) ** (x + y + z)
    o.set_state(0, 0, cb)
    o.set_state(0, 2, 0 * cb)
    k = o.eval_rhs(0, 1.0)[0]
    assert np.abs(k[0] + 3 * KO_EPS[0] / h * cb).max() < 1e-14


@pytest.mark.parametrize("r", [2, 3])
def test_ko_inside_rk4_matches_the_damped_amplification_matrix(r):
    """lambda = 0 with dissipation: a plane wave evolves by R(dt A)^n with A = [[q_psi, 1], [-w^2, q_Pi]]: the term
    is evaluated at every stage state, on psi and Pi, with the level's h."""
    n, h = (16, 8, 24), 0.5
    eps = (0.2, 0.3, 0.5, 0.7)  # large on purpose: the damping is far above the 1e-13 tolerance
    o = Oracle(n, nghost=3, lap_order=1, h0=h, lam=0.0, ko_order=r, ko_strength=eps)
    x, y, z = coords(n[::-1])
    m = (1, 2, 3)
    kh = [2 * math.pi * m[d] / n[d] for d in range(3)]
    ph = kh[0] * x + kh[1] * y + kh[2] * z
    w2 = sum(4 * math.sin(a / 2) ** 2 for a in kh) / h ** 2
    A0, B0 = 0.7, -0.4
    o.set_state(0, 0, A0 * np.cos(ph))
    o.set_state(0, 2, B0 * np.cos(ph))
    o.set_state(0, 1, 2 * A0 * np.sin(ph))
    o.set_state(0, 3, -B0 * np.sin(ph))
    dt, steps = 0.2 * h, 25
    eta = 3.0
    for _ in range(steps):
        o.rk_step(dt, eta)
        eta += dt
    out = []
    for c in range(2):
        Z = dt * np.array([[ko_symbol(r, eps[c], kh, h), 1.0], [-w2, ko_symbol(r, eps[c + 2], kh, h)]])
        R = np.eye(2) + Z + Z @ Z / 2 + Z @ Z @ Z / 6 + Z @ Z @ Z @ Z / 24
        out.append(np.linalg.matrix_power(R, steps) @ (np.array([A0, B0]) if c == 0 else np.array([2 * A0, -B0])))
    assert np.abs(o.get_state(0, 0) - out[0][0] * np.cos(ph)).max() < 1e-13
    assert np.abs(o.get_state(0, 2) - out[0][1] * np.cos(ph)).max() < 1e-12
    assert np.abs(o.get_state(0, 1) - out[1][0] * np.sin(ph)).max() < 1e-13
    assert np.abs(o.get_state(0, 3) - out[1][1] * np.sin(ph)).max() < 1e-12
    # and the damping is really there: without the term the same run differs by far more than the tolerance
    o2 = Oracle(n, nghost=3, lap_order=1, h0=h, lam=0.0)
    o2.set_state(0, 0, A0 * np.cos(ph))
    o2.set_state(0, 2, B0 * np.cos(ph))
    eta = 3.0
    for _ in range(steps):
        o2.rk_step(dt, eta)
        eta += dt
    assert np.abs(o2.get_state(0, 0) - o.get_state(0, 0)).max() > 1e-3


def test_ko_validation_and_off_switch():
    with pytest.raises(OracleError):
        Oracle(16, nghost=2, lap_order=1, ko_order=3, ko_strength=0.01)  # needs 3 ghost cells (L751)
    with pytest.raises(OracleError):
        Oracle(16, nghost=3, lap_order=1, ko_order=1, ko_strength=0.01)  # order is 2 or 3 (L751)
    with pytest.raises(OracleError):
        Oracle(16, nghost=3, lap_order=1, ko_order=2, ko_strength=-0.01)
    Oracle(16, nghost=1, lap_order=1, ko_order=0, ko_strength=0.0)  # strength 0 removes the term (L749)


# ------------------------------------------------------------------------------------------------
# O3 + O4: potential, friction, eta handling and the RK4 tableau against a textbook scalar ODE solve
# ------------------------------------------------------------------------------------------------


def scalar_rk4(y, eta, dt, lam, a, kappa, eta_fixed=None):
    """Textbook RK4 for the 4-variable ODE obtained from Eq.10-11 with a spatially constant field."""

    def f(y, e):
        e = eta_fixed if eta_fixed is not None else e
        p1, p2, q1, q2 = y
        pot = lam * e * e * (p1 * p1 + p2 * p2 - 1.0) + a
        fr = kappa / e if kappa != 0 else 0.0
        return np.array([q1, q2, -p1 * pot - fr * q1, -p2 * pot - fr * q2])

    k1 = f(y, eta)
    k2 = f(y + 0.5 * dt * k1, eta + 0.5 * dt)
    k3 = f(y + 0.5 * dt * k2, eta + 0.5 * dt)
    k4 = f(y + dt * k3, eta + dt)
    return y + dt / 6.0 * (k1 + 2 * k2 + 2 * k3 + k4)


@pytest.mark.parametrize("order", [1, 2])
@pytest.mark.parametrize("eta_fixed", [False, True])
def test_constant_field_equals_scalar_ode(order, eta_fixed):
    n = 8
    lam, a, kappa = 1.3, 0.56233, 2.0  # a: the listing's constant (L214), kappa = 2: Eq.11
    o = Oracle(n, nghost=2, lap_order=order, h0=0.7, lam=lam, a_mass=a, friction=kappa, eta_fixed=eta_fixed)
    y = np.array([0.3, -0.8, 0.1, 0.25])
    for c in range(4):
        o.set_state(0, c, np.full((n, n, n), y[c]))
    eta, dt = 1.5, 0.05
    for _ in range(20):
        o.rk_step(dt, eta)
        y = scalar_rk4(y, eta, dt, lam, a, kappa, eta_fixed=eta if eta_fixed else None)
        eta += dt
    for c in range(4):
        got = o.get_state(0, c)
        assert np.all(got == got.flat[0]), "a constant field must stay constant (difference-form stencil)"
        assert abs(got.flat[0] - y[c]) <= 64 * np.finfo(float).eps * max(1.0, abs(y[c]))


@pytest.mark.parametrize("order", [1, 2, 3])
def test_linear_plane_wave_matches_rk4_amplification_matrix(order):
    """lambda = 0: a lattice plane wave evolves by R(dt A)^n exactly, A = [[0,1],[-w^2,0]],
    R(z) = 1 + z + z^2/2 + z^3/6 + z^4/24, w^2 = lattice symbol (BASELINE.json 'discrete-dispersion plane
    wave' for the 2nd-order stencil; the 13-point symbol for order 2)."""
    n = (16, 8, 24)
    h = 0.5
    o = Oracle(n, nghost=3, lap_order=order, h0=h, lam=0.0)
    x, y, z = coords(n[::-1])
    m = (1, 2, 3)
    kh = [2 * math.pi * m[d] / n[d] for d in range(3)]
    ph = kh[0] * x + kh[1] * y + kh[2] * z
    if order == 1:
        w2 = sum(4 * math.sin(a / 2) ** 2 for a in kh) / h ** 2
    elif order == 2:
        w2 = sum(16 / 3 * math.sin(a / 2) ** 2 - 1 / 3 * math.sin(a) ** 2 for a in kh) / h ** 2
    else:
        w2 = sum(6 * math.sin(a / 2) ** 2 - 0.6 * math.sin(a) ** 2 + 2 / 45 * math.sin(1.5 * a) ** 2 for a in kh) / h ** 2
    A0, B0 = 0.7, -0.4  # psi1 = A cos, Pi1 = B cos ; psi2 = 2A sin, Pi2 = -B sin
    o.set_state(0, 0, A0 * np.cos(ph))
    o.set_state(0, 2, B0 * np.cos(ph))
    o.set_state(0, 1, 2 * A0 * np.sin(ph))
    o.set_state(0, 3, -B0 * np.sin(ph))
    dt, steps = 0.2 * h, 25
    Z = dt * np.array([[0.0, 1.0], [-w2, 0.0]])
    R = np.eye(2) + Z + Z @ Z / 2 + Z @ Z @ Z / 6 + Z @ Z @ Z @ Z / 24
    Rn = np.linalg.matrix_power(R, steps)
    eta = 3.0
    for _ in range(steps):
        o.rk_step(dt, eta)
        eta += dt
    a1, b1 = Rn @ np.array([A0, B0])
    a2, b2 = Rn @ np.array([2 * A0, -B0])
    assert np.abs(o.get_state(0, 0) - a1 * np.cos(ph)).max() < 1e-13
    assert np.abs(o.get_state(0, 2) - b1 * np.cos(ph)).max() < 1e-12
    assert np.abs(o.get_state(0, 1) - a2 * np.sin(ph)).max() < 1e-13
    assert np.abs(o.get_state(0, 3) - b2 * np.sin(ph)).max() < 1e-12


def test_energy_conservation_minkowski_is_fourth_order():
    """Constant-eta variant: E = sum[1/2 Pi^2 - 1/2 psi.L psi + lambda eta^2/4 (|psi|^2-1)^2] h^3 is conserved
    by the semi-discrete system; RK4 drifts as O(dt^4): halving dt must cut the drift by >= 14."""
    n, h, eta = 16, 1.0, 1.2
    psi1 = inputs.grf(n, 0.5, 11).numpy()
    psi2 = inputs.grf(n, 0.5, 12).numpy()

    def drift(dt, steps):
        o = Oracle(n, nghost=1, lap_order=1, h0=h, lam=1.0, eta_fixed=True)
        o.set_state(0, 0, 0.6 * psi1)
        o.set_state(0, 1, 0.6 * psi2)
        e0 = o.energy(eta)[:3].sum()
        for _ in range(steps):
            o.rk_step(dt, eta)
        return abs(o.energy(eta)[:3].sum() - e0) / abs(e0)

    d1 = drift(0.2, 20)
    d2 = drift(0.1, 40)
    assert d1 < 1e-3
    assert d1 / d2 > 14.0, (d1, d2)


# ------------------------------------------------------------------------------------------------
# Paper Appendix B (golden fixture): plane wave, 13-point Laplacian, RK4, dt = 0.32 dx
# ------------------------------------------------------------------------------------------------


def read_golden(name):
    out = {}
    for line in open(os.path.join(GOLD, name)):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split("=")
            out[k.strip()] = float(v)
    return out


def plane_wave_energy_error(N, gold, periods):
    L = gold["L_over_sqrt5"] * math.sqrt(5.0)
    h = L / N
    m = (gold["wavelengths_x"], gold["wavelengths_y"], -gold["wavelengths_z"])  # reading G6: k = pi(8,5,-6)/(5 sqrt5)
    kvec = [2 * math.pi * mm / L for mm in m]
    omega = gold["omega_over_pi"] * math.pi
    o = Oracle(N, nghost=2, lap_order=int(gold["laplacian_order"]), h0=h, lam=0.0)
    x, y, z = coords((N, N, N))
    ph = kvec[0] * (x + 0.5) * h + kvec[1] * (y + 0.5) * h + kvec[2] * (z + 0.5) * h
    o.set_state(0, 0, gold["A"] * np.cos(ph))  # u(x,0)
    o.set_state(0, 2, -gold["A"] * omega * np.sin(ph))  # du/dt(x,0), Eq.B2
    t_end = periods * 2 * math.pi / omega
    dt0 = gold["cfl"] * h
    steps = int(math.ceil(t_end / dt0 - 1e-9))
    dt = t_end / steps
    t = 0.0
    for _ in range(steps):
        o.rk_step(dt, t + 1.0)  # eta is irrelevant for lambda = 0, friction = 0
        t += dt
    e = o.energy(1.0)
    E = (e[0] + e[3]) / L ** 3  # mean of u_t^2/2 + (grad u)^2/2, L678
    return E - gold["E_exact_over_pi2"] * math.pi ** 2, kvec


def test_appendix_b_wavevector_reading():
    """Reading G6: |k| must equal omega/c = pi for Eq.B2 to solve Eq.B1; the printed L = 10 sqrt5 then holds
    exactly 8, 5, 6 wavelengths."""
    g = read_golden("appendix_b_plane_wave.txt")
    th = math.atan(g["tan_theta"])
    phi = math.asin(g["sin_phi"])
    k = math.pi * np.array([math.cos(th) * math.cos(phi), math.sin(th), -math.cos(th) * math.sin(phi)])
    assert abs(np.linalg.norm(k) - math.pi) < 1e-14
    L = g["L_over_sqrt5"] * math.sqrt(5)
    waves = np.abs(k) * L / (2 * math.pi)
    assert np.allclose(waves, [g["wavelengths_x"], g["wavelengths_y"], g["wavelengths_z"]], atol=1e-12)


def test_appendix_b_energy_converges_at_fourth_order():
    """Delta E -> 0 as a power law in N with index 'roughly -p or better' (paper fit for RK4: -4.7)."""
    g = read_golden("appendix_b_plane_wave.txt")
    periods = 10  # the paper runs 100 periods; the index does not depend on it, the CPU time does
    d32, _ = plane_wave_energy_error(32, g, periods)
    d64, _ = plane_wave_energy_error(64, g, periods)
    idx = math.log(abs(d64) / abs(d32)) / math.log(2.0)
    assert abs(d32) < 0.3 * math.pi ** 2 / 2  # converged regime (the paper excludes Delta E ~ O(1))
    assert -6.5 < idx < -3.7, idx
    assert abs(idx - g["rk4_power_law_index"]) < 1.5


# ------------------------------------------------------------------------------------------------
# O1/O5: periodic fill and same-level copies
# ------------------------------------------------------------------------------------------------


def run_single(n, boxes, psi, pi, steps, dt, eta0, **kw):
    o = Oracle(n, boxes=boxes, **kw)
    for ib, (l, lo, hi) in enumerate(o.boxes):
        sl = (slice(lo[2], hi[2] + 1), slice(lo[1], hi[1] + 1), slice(lo[0], hi[0] + 1))
        o.set_state(ib, 0, psi[0][sl])
        o.set_state(ib, 1, psi[1][sl])
        o.set_state(ib, 2, pi[0][sl])
        o.set_state(ib, 3, pi[1][sl])
    eta = eta0
    for _ in range(steps):
        o.rk_step(dt, eta)
        eta += dt
    out = np.zeros((4,) + psi[0].shape)
    for ib, (l, lo, hi) in enumerate(o.boxes):
        sl = (slice(lo[2], hi[2] + 1), slice(lo[1], hi[1] + 1), slice(lo[0], hi[0] + 1))
        for c in range(4):
            out[c][sl] = o.get_state(ib, c)
    return out


@pytest.mark.parametrize("order,g", [(1, 1), (2, 2), (2, 3)])
def test_translation_invariance_bit_for_bit(order, g):
    n = 16
    psi = [inputs.grf(n, 0.5, s).numpy() for s in (21, 22)]
    pi = [0.1 * inputs.grf(n, 0.5, s).numpy() for s in (23, 24)]
    kw = dict(nghost=g, lap_order=order, h0=1.0, lam=1.0)
    a = run_single(n, None, psi, pi, 3, 0.2, 1.0, **kw)
    sh = (5, -3, 9)  # z, y, x
    psi_s = [np.roll(p, sh, axis=(0, 1, 2)) for p in psi]
    pi_s = [np.roll(p, sh, axis=(0, 1, 2)) for p in pi]
    b = run_single(n, None, psi_s, pi_s, 3, 0.2, 1.0, **kw)
    assert np.array_equal(np.roll(a, sh, axis=(1, 2, 3)), b)


@pytest.mark.parametrize("order,g", [(1, 1), (2, 3)])
def test_multibox_level_equals_single_box_bit_for_bit(order, g):
    """Same-level ghost copies (incl. edges/corners across the periodic seam) must make a tiled level 0
    indistinguishable from one big box."""
    n = 16
    psi = [inputs.grf(n, 0.5, s).numpy() for s in (31, 32)]
    pi = [0.1 * inputs.grf(n, 0.5, s).numpy() for s in (33, 34)]
    kw = dict(nghost=g, lap_order=order, h0=0.5, lam=1.0)
    a = run_single(n, None, psi, pi, 3, 0.1, 1.0, **kw)
    b = run_single(n, inputs.split_level0(n, 8), psi, pi, 3, 0.1, 1.0, **kw)
    assert np.array_equal(a, b)
    # non-uniform split: boxes of 8 and 16 cells
    boxes = [(0, (0, 0, 0), (7, 15, 15)), (0, (8, 0, 0), (15, 7, 15)), (0, (8, 8, 0), (15, 15, 7)),
             (0, (8, 8, 8), (15, 15, 15))]
    c = run_single(n, boxes, psi, pi, 3, 0.1, 1.0, **kw)
    assert np.array_equal(a, c)


# ------------------------------------------------------------------------------------------------
# O5: coarse->fine trilinear + linear-in-time interpolation;  O7: average-down
# ------------------------------------------------------------------------------------------------


def two_level(n0=16, g=3, order=2, lo=(8, 16, 8), hi=(23, 23, 15), **kw):
    """Level 0: one box; level 1: one box lo..hi (fine indices), properly nested."""
    boxes = [(0, (0, 0, 0), (n0 - 1, n0 - 1, n0 - 1)), (1, lo, hi)]
    return Oracle(n0, boxes=boxes, n_levels=2, nghost=g, lap_order=order, **kw)


def affine(level_h, shape, lo, coef, g=0):
    zz, yy, xx = np.meshgrid(*[(np.arange(l - g, l + s + g) + 0.5) * level_h for l, s in zip(lo[::-1], shape)],
                             indexing="ij")
    return coef[0] + coef[1] * xx + coef[2] * yy + coef[3] * zz


def test_trilinear_reproduces_affine_data_in_space():
    h0 = 0.5
    o = two_level(h0=h0, lam=0.0)
    coefs = [(0.3, 1.0, -2.0, 0.5), (-1.0, 0.25, 0.75, -1.5), (0.1, -1.0, 1.0, 1.0), (2.0, 0.5, 0.5, 0.5)]
    for c in range(4):
        o.set_state(0, c, affine(h0, (16, 16, 16), (0, 0, 0), coefs[c]))
    o.fill_ghosts(1, 0.0)
    g = 3
    lo = (8, 16, 8)
    shp = o.box_shape(1)
    for c in range(4):
        raw = o.get_raw(1, c)
        want = affine(h0 / 2, shp, lo, coefs[c], g=g)
        ghost = np.ones_like(raw, dtype=bool)
        ghost[g:-g, g:-g, g:-g] = False
        assert np.abs(raw - want)[ghost].max() < 1e-13
        assert np.all(raw[g:-g, g:-g, g:-g] == 0.0)  # valid cells are never touched by a fill


@pytest.mark.parametrize("order,integrator", [(1, 4), (2, 4), (2, 10)])
def test_time_interpolation_is_linear_between_coarse_old_and_new(order, integrator):
    """lambda = 0 and psi = b + c t (Pi = c, spatially constant) is an exact solution that RK4 (and SSPRK3, whose
    stage times are t, t + dt, t + dt/2: alpha in {0, 1/2, 1/4} and {1/2, 1, 3/4}) reproduces
    exactly; during the fine substeps the ghosts must then carry b + c t_s for alpha in {0, 1/4, 1/2, 3/4, 1}.
    The fine interior sees a ghost value consistent with its own only if alpha is right; any wrong alpha
    puts a kink at the box edge that the Laplacian turns into a non-zero k_Pi."""
    h0 = 1.0
    o = two_level(h0=h0, lam=0.0, order=order, integrator=integrator)
    b, c = 0.25, 0.5
    for ib in (0, 1):
        shp = o.box_shape(ib)
        o.set_state(ib, 0, np.full(shp, b))
        o.set_state(ib, 1, np.full(shp, -b))
        o.set_state(ib, 2, np.full(shp, c))
        o.set_state(ib, 3, np.full(shp, 2 * c))
    t, dt = 2.0, 0.5  # exactly representable: alpha is exact
    for _ in range(2):
        o.rk_step(dt, t)
        t += dt
    for ib in (0, 1):
        assert np.abs(o.get_state(ib, 0) - (b + c * (t - 2.0))).max() < 1e-14
        assert np.abs(o.get_state(ib, 1) - (-b + 2 * c * (t - 2.0))).max() < 1e-14
        assert np.abs(o.get_state(ib, 2) - c).max() < 1e-14


def test_ghosts_at_sync_use_new_coarse_state_only():
    """After a coarse step (alpha = 1) fine ghosts equal the interpolated CURRENT coarse state."""
    o = two_level(h0=1.0, lam=0.0)
    coef = (0.3, 1.0, -2.0, 0.5)
    a = affine(1.0, (16, 16, 16), (0, 0, 0), coef)
    o.set_state(0, 0, a)
    o.set_state(1, 0, affine(0.5, o.box_shape(1), (8, 16, 8), coef))
    o.rk_step(0.25, 1.0)  # psi is affine and Pi = 0, lambda = 0: interior stays put
    o.set_state(0, 0, 2 * a)  # change the current coarse state by hand
    o.fill_ghosts(1, 1.25)
    raw = o.get_raw(1, 0)
    want = 2 * affine(0.5, o.box_shape(1), (8, 16, 8), coef, g=3)
    # ghosts not adjacent to the periodic seam are affine-exact
    assert abs(raw[0, 5, 5] - want[0, 5, 5]) < 1e-13
    assert abs(raw[5, -1, 7] - want[5, -1, 7]) < 1e-13


def test_average_down_affine_and_mean_preserving():
    h0 = 1.0
    o = two_level(h0=h0, lam=0.0)
    coef = (0.3, 1.0, -2.0, 0.5)
    rng = np.random.default_rng(5)
    fine = [rng.normal(size=o.box_shape(1)) for _ in range(4)]
    fine[0] = affine(h0 / 2, o.box_shape(1), (8, 16, 8), coef)
    for c in range(4):
        o.set_state(0, c, np.full((16, 16, 16), 7.0))
        o.set_state(1, c, fine[c])
    o.average_down(1)
    cov = (slice(4, 8), slice(8, 12), slice(4, 12))  # z, y, x coarse footprint
    for c in range(4):
        got = o.get_state(0, c)
        mask = np.ones_like(got, dtype=bool)
        mask[cov] = False
        assert np.all(got[mask] == 7.0)  # uncovered cells untouched
        f = fine[c]
        want = f.reshape(4, 2, 4, 2, 8, 2).mean(axis=(1, 3, 5))
        assert np.abs(got[cov] - want).max() < 1e-14
        assert abs(got[cov].sum() - f.sum() / 8) < 1e-11
    want0 = affine(h0, (4, 4, 8), (4, 8, 4), coef)
    assert np.abs(o.get_state(0, 0)[cov] - want0).max() < 1e-13


# ------------------------------------------------------------------------------------------------
# O9: truncation-error tags at synchronisation (L82-111 Eq.5-6, L373-380 Eq.12)
# ------------------------------------------------------------------------------------------------


def test_tee_is_zero_when_coarse_is_the_mean_of_its_children():
    """Exactly representable affine data whose coarse values are the children's means: Delta = 0, and Eq.12 is a
    strict inequality, so nothing is tagged even for eps = 0; a second synchronisation sees coarse == mean too."""
    o = two_level(h0=1.0, lam=0.0)
    coef = (0.5, 1.0, -2.0, 0.25)
    for c in range(4):
        o.set_state(0, c, affine(1.0, (16, 16, 16), (0, 0, 0), coef))
        o.set_state(1, c, affine(0.5, o.box_shape(1), (8, 16, 8), coef))
    o.tee_enable(1, 0.0, 0.0)
    for _ in range(2):
        o.average_down(1)
        tags, counts = o.tee_tags(1)
        assert not tags[0].any() and not counts.any()


def test_tee_tags_equal_the_prescribed_offsets_exactly():
    """fine = 1 everywhere (mean exactly 1), coarse = 1 + delta(C) with dyadic offsets: Delta = |delta| exactly, so
    the tags are (|delta| > eps) per component, copied to the 8 children, and the block counts are 8 x the number
    of tagged coarse cells in the block -- all computed here independently of the oracle."""
    o = two_level(n0=32, lo=(8, 24, 16), hi=(39, 47, 47), h0=1.0, lam=0.0)  # fine box straddles 32-blocks
    rng = np.random.default_rng(9)
    d = [rng.integers(-8, 9, size=(32, 32, 32)) / 64.0 for _ in range(4)]  # multiples of 1/64 in [-1/8, 1/8]
    for c in range(4):
        o.set_state(0, c, 1.0 + d[c])
        o.set_state(1, c, np.ones(o.box_shape(1)))
    # one threshold per component, momenta included (te_crit_$ScalarField, L781-782; Scalar::Pi1, L202)
    eps = (3 / 64.0, 5 / 64.0, 6 / 64.0, 2 / 64.0)
    o.tee_enable(1, *eps)
    o.average_down(1)
    tags, counts = o.tee_tags(1)
    cov = (slice(8, 24), slice(12, 24), slice(4, 20))  # z, y, x coarse footprint of the fine box
    want_c = np.zeros(d[0][cov].shape, dtype=np.uint8)
    for c in range(4):
        want_c |= (np.abs(d[c][cov]) > eps[c]).astype(np.uint8) << c
    assert all(((want_c >> c) & 1).any() and not ((want_c >> c) & 1).all() for c in range(4))
    assert want_c.any() and not want_c.all()
    want_f = want_c.repeat(2, axis=0).repeat(2, axis=1).repeat(2, axis=2)
    assert np.array_equal(tags[0], want_f)
    # a value exactly at the threshold is NOT tagged (strict >)
    at = np.abs(d[0][cov]) == eps[0]
    assert at.any() and not (want_c[at] & 1).any()
    want_counts = np.zeros_like(counts)
    zz, yy, xx = np.nonzero(want_f)
    np.add.at(want_counts, ((zz + 16) // 32, (yy + 24) // 32, (xx + 8) // 32), 1)
    assert np.array_equal(counts, want_counts) and counts.sum() == 8 * np.count_nonzero(want_c)
    # the synchronisation itself is unchanged: covered coarse cells now hold the children's mean
    assert np.all(o.get_state(0, 0)[cov] == 1.0)
    # the default threshold (DBL_MAX, L781) switches a component off: psi-only thresholds give bits 0, 1 only
    for c in range(4):
        o.set_state(0, c, 1.0 + d[c])
    o.tee_enable(1, eps[0], eps[1])
    o.average_down(1)
    tags2, _ = o.tee_tags(1)
    assert np.array_equal(tags2[0], want_f & 3)


def test_tee_inside_rk_step_shrinks_with_resolution():
    """Self-shadow estimate on a smooth standing wave (lambda = 0): the largest |coarse - fine| at the sync inside
    rk_step, found by bisecting eps on the tag output, drops by more than 4x when h and dt are halved (one step of
    length dt ~ h times a spatial error of at least O(h^2), the trilinear ghosts at the fine boundary, L100), i.e.
    the tags respond to convergence as L98 describes."""
    def max_tee(n0):
        h0 = 1.0 / n0
        lo = (n0 // 2,) * 3                # fine indices: the fine box refines coarse cells [n0/4, 3 n0/4)
        hi = (3 * n0 // 2 - 1,) * 3
        def run(eps):
            o = Oracle(n0, boxes=[(0, (0, 0, 0), (n0 - 1,) * 3), (1, lo, hi)], n_levels=2, nghost=2, blocking_factor=4,
                       lap_order=2, h0=h0, lam=0.0)
            for l, ib in ((0, 0), (1, 1)):
                hl = h0 / (1 << l)
                blo = (0, 0, 0) if l == 0 else lo
                z, y, x = coords(o.box_shape(ib))
                X = (x + blo[0] + 0.5) * hl
                Yc = (y + blo[1] + 0.5) * hl
                Z = (z + blo[2] + 0.5) * hl
                o.set_state(ib, 0, np.cos(2 * np.pi * X) * np.cos(2 * np.pi * Yc) * np.cos(2 * np.pi * Z))
                o.set_state(ib, 1, np.sin(2 * np.pi * X) + 0 * Yc + 0 * Z)
            o.average_down(1)  # start from identical states: coarse = mean of its children (Eq.5 "identical states")
            o.tee_enable(1, eps, 1e30)
            o.rk_step(0.25 * h0, 1.0)
            return o.tee_tags(1)[0][0].any()
        lo_e, hi_e = 0.0, 1.0
        assert run(lo_e) and not run(hi_e)
        for _ in range(24):
            mid = 0.5 * (lo_e + hi_e)
            if run(mid):
                lo_e = mid
            else:
                hi_e = mid
        return hi_e
    e8, e16 = max_tee(8), max_tee(16)
    assert e8 > 0 and e16 < e8 / 4.0


# ------------------------------------------------------------------------------------------------
# O6: subcycling bookkeeping
# ------------------------------------------------------------------------------------------------


@pytest.mark.parametrize("order,g,ko,integrator", [(1, 1, 0, 4), (2, 2, 0, 4), (1, 2, 2, 4), (2, 3, 3, 4), (2, 2, 0, 10)])
def test_fully_covered_level1_equals_uniform_fine_run(order, g, ko, integrator):
    """A hierarchy whose level 1 covers 100 % of the domain never interpolates: level 1 must reproduce the
    single-level 2N run with dt/2 bit-for-bit, and level 0 must equal its average.  With Kreiss-Oliger dissipation
    on (ko = dissipation order) this also pins that Q_l uses the level's own spacing (Eq.7: Delta x_l)."""
    kw = dict(ko_order=ko, ko_strength=(0.02, 0.03, 0.05, 0.07)) if ko else {}
    kw["integrator"] = integrator
    n0, h0, dt, eta0 = 8, 1.0, 0.25, 1.0  # binary fractions: both runs see identical stage times
    nf = 2 * n0
    psi = [inputs.grf(nf, 0.5, s).numpy() for s in (41, 42)]
    pi = [0.1 * inputs.grf(nf, 0.5, s).numpy() for s in (43, 44)]
    ref = run_single(nf, None, psi, pi, 4, dt / 2, eta0, nghost=g, lap_order=order, h0=h0 / 2, lam=1.0, **kw)
    boxes = [(0, (0, 0, 0), (n0 - 1,) * 3), (1, (0, 0, 0), (nf - 1,) * 3)]
    o = Oracle(n0, boxes=boxes, n_levels=2, nghost=g, lap_order=order, h0=h0, lam=1.0, **kw)
    for c, a in enumerate(psi + pi):
        o.set_state(1, c, a)
    o.average_down(1)
    eta = eta0
    for _ in range(2):
        o.rk_step(dt, eta)
        eta += dt
    for c in range(4):
        f = o.get_state(1, c)
        assert np.array_equal(f, ref[c])
        want = f.reshape(n0, 2, n0, 2, n0, 2).sum(axis=5).sum(axis=3).sum(axis=1) * 0.125
        assert np.abs(o.get_state(0, c) - want).max() < 4e-15  # summation order only


def test_constant_field_on_three_levels_follows_scalar_ode_per_level():
    """Each level integrates the scalar ODE with ITS OWN dt (dt/2^l, 2^l times); after synchronisation the
    covered coarse cells carry the fine value (L74), uncovered ones the coarse value."""
    n0 = 16
    boxes = [(0, (0, 0, 0), (15, 15, 15)), (1, (8, 8, 8), (23, 23, 23)), (2, (24, 24, 24), (39, 39, 39))]
    lam = 1.0
    o = Oracle(n0, boxes=boxes, n_levels=3, nghost=2, lap_order=2, h0=1.0, lam=lam, friction=2.0)
    y0 = np.array([0.4, 0.3, -0.2, 0.1])
    for ib in range(3):
        for c in range(4):
            o.set_state(ib, c, np.full(o.box_shape(ib), y0[c]))
    eta, dt = 1.0, 0.1
    o.rk_step(dt, eta)
    ys = []
    for l in range(3):
        y, e = y0.copy(), eta
        for _ in range(1 << l):
            y = scalar_rk4(y, e, dt / (1 << l), lam, 0.0, 2.0)
            e += dt / (1 << l)
        ys.append(y)
    # Ghost cells of a fine level carry the coarse solution interpolated LINEARLY in time (error ~dt^2 psi''/8
    # ~1e-3 at mid-step); it leaks into uncovered level-1 cells (all within 4 cells of the patch edge) but
    # reaches the level-2 centre only at high order in dt.
    assert 1e-7 < np.abs(ys[1] - ys[0]).max() < 1e-3
    for c in range(4):
        f2 = o.get_state(2, c)
        assert abs(f2[8, 8, 8] - ys[2][c]) < 1e-13
        f1 = o.get_state(1, c)
        assert abs(f1[0, 0, 0] - ys[1][c]) < 5e-3 and abs(f1[1, 8, 1] - ys[1][c]) < 5e-3
        f0 = o.get_state(0, c)
        assert abs(f0[0, 0, 0] - ys[0][c]) < 1e-14
        assert abs(f0[8, 8, 8] - f1[8:10, 8:10, 8:10].mean()) < 1e-15  # covered by level 1 -> average of children
        assert abs(f1[8, 8, 8] - f2[8:10, 8:10, 8:10].mean()) < 1e-15


def amr_wave_error(n0):
    """Long-wavelength linear wave (one wavelength per box length L = 16) crossing a refined patch."""
    L = 16.0
    h0 = L / n0
    q = n0 // 4
    boxes = [(0, (0, 0, 0), (n0 - 1,) * 3), (1, (2 * q,) * 3, (6 * q - 1,) * 3)]
    o = Oracle(n0, boxes=boxes, n_levels=2, nghost=2, lap_order=2, h0=h0, lam=0.0)
    kx = 2 * math.pi / L
    w = kx

    def exact(level, lo, shp, t):
        h = h0 / (1 << level)
        x = (np.arange(lo[0], lo[0] + shp[2]) + 0.5) * h
        u = np.cos(kx * x - w * t)
        ut = w * np.sin(kx * x - w * t)
        return np.broadcast_to(u[None, None, :], shp), np.broadcast_to(ut[None, None, :], shp)

    for ib, (l, lo, hi) in enumerate(o.boxes):
        u, ut = exact(l, lo, o.box_shape(ib), 0.0)
        o.set_state(ib, 0, u)
        o.set_state(ib, 2, ut)
    t, dt = 0.0, 0.25 * h0
    for _ in range(int(round(4.0 / dt))):
        o.rk_step(dt, t + 1.0)
        t += dt
    err = 0.0
    for ib, (l, lo, hi) in enumerate(o.boxes):
        u, _ = exact(l, lo, o.box_shape(ib), t)
        err = max(err, np.abs(o.get_state(ib, 0) - u).max())
    return err


def test_amr_smooth_wave_converges():
    """End-to-end sanity for the hierarchy: a smooth wave crossing a refined patch.  Trilinear ghosts carry an
    O(h^2) error that the Laplacian divides by h^2, so the scheme BASELINE.json prescribes is first-order at
    the patch edge (the reason the paper defaults to quartic interpolation, L70/L780): halving h must cut the
    error by ~2.  A wrong ghost offset, weight or alpha makes it grow or stall instead."""
    e16 = amr_wave_error(16)
    e32 = amr_wave_error(32)
    assert e16 < 0.1
    assert e32 < e16 / 1.8, (e16, e32)


# ------------------------------------------------------------------------------------------------
# O8: string tags
# ------------------------------------------------------------------------------------------------


def atan2_winding(A, B, C, D):
    """Textbook definition: sum of principal-value phase differences around the loop / 2 pi."""
    z = [complex(*A), complex(*B), complex(*C), complex(*D)]
    tot = 0.0
    for a, b in zip(z, z[1:] + z[:1]):
        tot += np.angle(b / a)
    return int(round(tot / (2 * math.pi)))


def brute_tags(psi1, psi2):
    """Pure-Python tags of a periodic single-level grid from the atan2 definition."""
    n = psi1.shape
    tags = np.zeros(n, dtype=np.uint8)
    P = lambda k, j, i: (psi1[k % n[0], j % n[1], i % n[2]], psi2[k % n[0], j % n[1], i % n[2]])
    for k in range(n[0]):
        for j in range(n[1]):
            for i in range(n[2]):
                t = 0
                if atan2_winding(P(k, j, i), P(k, j, i + 1), P(k, j + 1, i + 1), P(k, j + 1, i)):
                    t |= 1  # xy
                if atan2_winding(P(k, j, i), P(k, j + 1, i), P(k + 1, j + 1, i), P(k + 1, j, i)):
                    t |= 2  # yz
                if atan2_winding(P(k, j, i), P(k + 1, j, i), P(k + 1, j, i + 1), P(k, j, i + 1)):
                    t |= 4  # zx
                tags[k, j, i] = t
    return tags


def test_plaquette_winding_matches_atan2_definition_on_random_corners():
    rng = np.random.default_rng(3)
    seen = set()
    for _ in range(20000):
        v = rng.normal(size=(4, 2))
        w = plaquette_winding(*v)
        assert w == atan2_winding(*v)
        seen.add(w)
    assert seen == {-1, 0, 1}
    # hand-made cases: CCW loop around the origin, CW loop, loop that misses it
    sq = np.array([[1, 1], [-1, 1], [-1, -1], [1, -1]], dtype=float)
    assert plaquette_winding(*sq) == 1
    assert plaquette_winding(*sq[::-1]) == -1
    assert plaquette_winding(*(sq + 3.0)) == 0


def test_straight_string_tags_exactly_four_columns():
    """psi = (x - x0) + i (y - y0), x0, y0 half-integers, periodic N grid: xy-plaquettes wind at
    (floor x0, floor y0) [+1], (N-1, floor y0) [-1], (floor x0, N-1) [-1], (N-1, N-1) [+1] for every z,
    and no yz / zx plaquette winds."""
    n = 16
    x0, y0 = 5.5, 9.5
    psi1, psi2 = inputs.straight_string(n, x0, y0)
    o = Oracle(n, nghost=1, lap_order=1)
    o.set_state(0, 0, psi1)
    o.set_state(0, 1, psi2)
    tags, counts = o.tag_strings(0)
    want = np.zeros((n, n, n), dtype=np.uint8)
    for (j, i) in [(9, 5), (9, n - 1), (n - 1, 5), (n - 1, n - 1)]:
        want[:, j, i] = 1
    assert np.array_equal(tags[0], want)
    assert counts.shape == (1, 1, 1) and counts[0, 0, 0] == 4 * n
    # signs of the four windings
    P = lambda j, i: (psi1[0, j % n, i % n], psi2[0, j % n, i % n])
    W = lambda j, i: plaquette_winding(P(j, i), P(j, i + 1), P(j + 1, i + 1), P(j + 1, i))
    assert (W(9, 5), W(9, n - 1), W(n - 1, 5), W(n - 1, n - 1)) == (1, -1, -1, 1)


def test_tags_match_brute_force_and_torus_identity():
    n = 8
    psi1 = inputs.grf(n, 0.9, 51).numpy()
    psi2 = inputs.grf(n, 0.9, 52).numpy()
    o = Oracle(n, nghost=1, lap_order=1)
    o.set_state(0, 0, psi1)
    o.set_state(0, 1, psi2)
    tags, counts = o.tag_strings(0)
    want = brute_tags(psi1, psi2)
    assert want.any(), "test field should contain strings"
    assert np.array_equal(tags[0], want)
    assert counts[0, 0, 0] == np.count_nonzero(want)
    # torus identity: the windings of all xy plaquettes of one z-slice sum to zero
    P = lambda k, j, i: (psi1[k % n, j % n, i % n], psi2[k % n, j % n, i % n])
    for k in range(n):
        tot = sum(plaquette_winding(P(k, j, i), P(k, j, i + 1), P(k, j + 1, i + 1), P(k, j + 1, i))
                  for j in range(n) for i in range(n))
        assert tot == 0


def test_tags_invariant_under_global_phase_rotation():
    n = 16
    psi1 = inputs.grf(n, 0.6, 61).numpy()
    psi2 = inputs.grf(n, 0.6, 62).numpy()
    o = Oracle(n, nghost=1, lap_order=1)
    o.set_state(0, 0, psi1)
    o.set_state(0, 1, psi2)
    t0, _ = o.tag_strings(0)
    ph = 1.2345
    o.set_state(0, 0, math.cos(ph) * psi1 - math.sin(ph) * psi2)
    o.set_state(0, 1, math.sin(ph) * psi1 + math.cos(ph) * psi2)
    t1, _ = o.tag_strings(0)
    assert t0[0].any()
    assert np.array_equal(t0[0], t1[0])


def test_tags_on_multibox_and_flag_block_counts():
    """Tags of a tiled level equal the single-box tags (ghost +1 neighbours incl. edge ghosts), and counts
    are accumulated per aligned 32^3 block of the level index space."""
    n = 64
    psi1 = inputs.grf(n, 0.3, 71).numpy()
    psi2 = inputs.grf(n, 0.3, 72).numpy()
    o = Oracle(n, nghost=1, lap_order=1)
    o.set_state(0, 0, psi1)
    o.set_state(0, 1, psi2)
    t_single, c_single = o.tag_strings(0)
    boxes = inputs.split_level0(n, 16)
    om = Oracle(n, boxes=boxes, nghost=1, lap_order=1)
    full = np.zeros((n, n, n), dtype=np.uint8)
    for ib, (l, lo, hi) in enumerate(boxes):
        sl = (slice(lo[2], hi[2] + 1), slice(lo[1], hi[1] + 1), slice(lo[0], hi[0] + 1))
        om.set_state(ib, 0, psi1[sl])
        om.set_state(ib, 1, psi2[sl])
    t_multi, c_multi = om.tag_strings(0)
    for ib, (l, lo, hi) in enumerate(boxes):
        sl = (slice(lo[2], hi[2] + 1), slice(lo[1], hi[1] + 1), slice(lo[0], hi[0] + 1))
        full[sl] = t_multi[ib]
    assert np.array_equal(full, t_single[0])
    assert np.array_equal(c_multi, c_single)
    want = (t_single[0] != 0).reshape(2, 32, 2, 32, 2, 32).sum(axis=(1, 3, 5))
    assert np.array_equal(c_single, want.astype(np.uint32))


# ------------------------------------------------------------------------------------------------
# O1: validation of box lists
# ------------------------------------------------------------------------------------------------


def test_box_list_validation():
    ok = [(0, (0, 0, 0), (15, 15, 15)), (1, (8, 8, 8), (23, 23, 23))]
    Oracle(16, boxes=ok, n_levels=2, nghost=2, lap_order=2)
    with pytest.raises(OracleError, match="overlap"):
        Oracle(16, boxes=ok + [(1, (16, 16, 16), (31, 31, 31))], n_levels=2, nghost=2, lap_order=2)
    with pytest.raises(OracleError, match="aligned"):
        Oracle(16, boxes=[ok[0], (1, (4, 8, 8), (19, 23, 23))], n_levels=2, nghost=2, lap_order=2)
    with pytest.raises(OracleError, match="cover"):
        Oracle(16, boxes=[(0, (0, 0, 0), (7, 15, 15))], nghost=1)
    with pytest.raises(OracleError, match="nghost"):
        Oracle(16, nghost=8, blocking_factor=8)
    with pytest.raises(OracleError, match="lap_order"):
        Oracle(16, nghost=1, lap_order=2)
    # level 2 box whose grown region leaves level 1 -> nesting violation
    bad = [(0, (0, 0, 0), (15, 15, 15)), (1, (8, 8, 8), (23, 23, 23)), (2, (16, 16, 16), (31, 31, 31))]
    with pytest.raises(OracleError, match="nesting"):
        Oracle(16, boxes=bad, n_levels=3, nghost=2, lap_order=2)
    good = [(0, (0, 0, 0), (15, 15, 15)), (1, (8, 8, 8), (23, 23, 23)), (2, (24, 24, 24), (39, 39, 39))]
    Oracle(16, boxes=good, n_levels=3, nghost=2, lap_order=2)


# ------------------------------------------------------------------------------------------------
# BASELINE.json config 1 as printed is outside the RK4 stability region (reading R12)
# ------------------------------------------------------------------------------------------------


def test_c1_literal_parameters_blow_up():
    """h = 1, dt = 0.25, lambda = 1, eta 1 -> 3.5 on a unit-variance GRF: where |psi| > 1 the local frequency
    sqrt(12/h^2 + lambda eta^2 (3|psi|^2 - 1)) * dt exceeds the RK4 stability limit 2.83 (at eta = 3, |psi| = 2:
    sqrt(12 + 99) * 0.25 = 2.63; |psi| = 2.5: 3.3) and the run diverges; with dt = 0.0625 it stays bounded.
    Documented so that the GPU parity test's treatment of C1 (absolute bar while bounded) is checkable here."""
    cfg = inputs.CONFIGS["C1"]

    def run(dt, steps):
        o = Oracle(cfg.n0, nghost=1, lap_order=1, h0=cfg.h0, lam=cfg.lam)
        for c, s in enumerate(cfg.seeds):
            o.set_state(0, c, inputs.grf(cfg.n0, cfg.grf_f, s).numpy())
        eta, peak = cfg.eta0, []
        for _ in range(steps):
            o.rk_step(dt, eta)
            eta += dt
            with np.errstate(invalid="ignore"):
                peak.append(max(float(np.abs(o.get_state(0, c)).max()) for c in range(2)))
        return peak

    lit = run(cfg.dt, 10)
    assert max(lit[:7]) < 4.0            # bounded for the first 7 steps (eta <= 2.75)
    assert lit[7] > 1e2 and not lit[9] < 1e100
    stab = run(0.0625, 40)
    assert max(stab) < 4.5 and max(stab[20:]) < 3.0  # the initial GRF peaks at ~4 sigma, then relaxes

# ------------------------------------------------------------------------------------------------
# O11 SSPRK3 (integrator.type 3 / 10, L808)
# ------------------------------------------------------------------------------------------------


def scalar_ssprk3_butcher(y, eta, dt, lam, a, kappa):
    """SSPRK3 in BUTCHER form (the oracle is written in Shu-Osher form): c = (0, 1, 1/2), a21 = 1,
    a31 = a32 = 1/4, b = (1/6, 1/6, 2/3), for the 4-variable ODE of a spatially constant field."""

    def f(y, e):
        p1, p2, q1, q2 = y
        pot = lam * e * e * (p1 * p1 + p2 * p2 - 1.0) + a
        fr = kappa / e if kappa != 0 else 0.0
        return np.array([q1, q2, -p1 * pot - fr * q1, -p2 * pot - fr * q2])

    k1 = f(y, eta)
    k2 = f(y + dt * k1, eta + dt)
    k3 = f(y + 0.25 * dt * (k1 + k2), eta + 0.5 * dt)
    return y + dt * (k1 / 6.0 + k2 / 6.0 + 2.0 * k3 / 3.0)


@pytest.mark.parametrize("integrator", [3, 10])
def test_ssprk3_constant_field_equals_butcher_form_scalar_ode(integrator):
    n = 8
    lam, a, kappa = 1.3, 0.56233, 2.0
    o = Oracle(n, nghost=2, lap_order=2, h0=0.7, lam=lam, a_mass=a, friction=kappa, integrator=integrator)
    y = np.array([0.3, -0.8, 0.1, 0.25])
    for c in range(4):
        o.set_state(0, c, np.full((n, n, n), y[c]))
    eta, dt = 1.5, 0.05
    for _ in range(20):
        o.rk_step(dt, eta)
        y = scalar_ssprk3_butcher(y, eta, dt, lam, a, kappa)
        eta += dt
    for c in range(4):
        got = o.get_state(0, c)
        assert np.all(got == got.flat[0])
        assert abs(got.flat[0] - y[c]) <= 256 * np.finfo(float).eps * max(1.0, abs(y[c]))
    # and it is NOT RK4: the two schemes differ at O(dt^4) per step, far above that tolerance
    o4 = Oracle(n, nghost=2, lap_order=2, h0=0.7, lam=lam, a_mass=a, friction=kappa)
    y0 = np.array([0.3, -0.8, 0.1, 0.25])
    for c in range(4):
        o4.set_state(0, c, np.full((n, n, n), y0[c]))
    eta = 1.5
    for _ in range(20):
        o4.rk_step(dt, eta)
        eta += dt
    assert abs(o4.get_state(0, 2).flat[0] - y[2]) > 1e-7


def test_ssprk3_linear_plane_wave_matches_cubic_amplification_matrix():
    """lambda = 0: every 3-stage third-order scheme has R(z) = 1 + z + z^2/2 + z^3/6 on linear problems."""
    n, h = (16, 8, 24), 0.5
    o = Oracle(n, nghost=2, lap_order=2, h0=h, lam=0.0, integrator=10)
    x, y, z = coords(n[::-1])
    m = (1, 2, 3)
    kh = [2 * math.pi * m[d] / n[d] for d in range(3)]
    ph = kh[0] * x + kh[1] * y + kh[2] * z
    w2 = sum(16 / 3 * math.sin(a / 2) ** 2 - 1 / 3 * math.sin(a) ** 2 for a in kh) / h ** 2
    A0, B0 = 0.7, -0.4
    o.set_state(0, 0, A0 * np.cos(ph))
    o.set_state(0, 2, B0 * np.cos(ph))
    o.set_state(0, 1, 2 * A0 * np.sin(ph))
    o.set_state(0, 3, -B0 * np.sin(ph))
    dt, steps = 0.2 * h, 25
    Z = dt * np.array([[0.0, 1.0], [-w2, 0.0]])
    R = np.eye(2) + Z + Z @ Z / 2 + Z @ Z @ Z / 6
    Rn = np.linalg.matrix_power(R, steps)
    eta = 3.0
    for _ in range(steps):
        o.rk_step(dt, eta)
        eta += dt
    a1, b1 = Rn @ np.array([A0, B0])
    a2, b2 = Rn @ np.array([2 * A0, -B0])
    assert np.abs(o.get_state(0, 0) - a1 * np.cos(ph)).max() < 1e-13
    assert np.abs(o.get_state(0, 2) - b1 * np.cos(ph)).max() < 1e-12
    assert np.abs(o.get_state(0, 1) - a2 * np.sin(ph)).max() < 1e-13
    assert np.abs(o.get_state(0, 3) - b2 * np.sin(ph)).max() < 1e-12


def test_ssprk3_is_third_order_on_the_nonlinear_problem():
    """error against a fine-dt RK4 run of the same semi-discrete system drops by ~8 when dt is halved"""
    n, T = 16, 0.4
    psi = [inputs.grf(n, 0.5, s).numpy() for s in (61, 62)]
    pi = [0.1 * inputs.grf(n, 0.5, s).numpy() for s in (63, 64)]
    kw = dict(nghost=2, lap_order=2, h0=0.5, lam=1.0)
    ref = run_single(n, None, psi, pi, 128, T / 128, 1.0, **kw)
    err = []
    for steps in (8, 16, 32):
        got = run_single(n, None, psi, pi, steps, T / steps, 1.0, integrator=10, **kw)
        err.append(np.abs(got - ref).max())
    assert 6.5 < err[0] / err[1] < 9.5 and 6.5 < err[1] / err[2] < 9.5, err


# ------------------------------------------------------------------------------------------------
# O12 quartic polynomial conservative coarse->fine interpolation (amr.interpolation_type 4, L70, L780)
# ------------------------------------------------------------------------------------------------


def _cell_avg_monomial(p, lo, hi):
    """exact average of x^p over [lo, hi] (arrays allowed)"""
    return (hi ** (p + 1) - lo ** (p + 1)) / ((p + 1) * (hi - lo))


def _poly_cell_averages(level_h, shape, lo, coefs, g=0):
    """cell averages of sum_t a_t x^px y^py z^pz over the cells of an index range (z, y, x array)"""
    ax = []
    for l, s in zip(lo[::-1], shape):  # z, y, x
        idx = np.arange(l - g, l + s + g, dtype=np.float64)
        ax.append((idx * level_h, (idx + 1) * level_h))
    out = 0.0
    for a, (px, py, pz) in coefs:
        Z = _cell_avg_monomial(pz, *ax[0])[:, None, None]
        Y = _cell_avg_monomial(py, *ax[1])[None, :, None]
        X = _cell_avg_monomial(px, *ax[2])[None, None, :]
        out = out + a * Z * Y * X
    return out


def test_quartic_interpolation_reproduces_cell_averages_of_quartic_polynomials():
    """The defining property (L780 "quartic polynomial conservative"): if the coarse values are the cell averages of a
    polynomial of degree <= 4 per axis, every interpolated fine ghost cell is that polynomial's average over the fine
    cell.  Distinct powers per axis catch a swapped axis or a mirrored left/right child; degree 5 is NOT reproduced."""
    h0 = 1.0 / 16  # coordinates in [0, 1): keeps the monomials O(1)
    o = two_level(h0=h0, lam=0.0, interp=4)
    coefs = [(0.7, (4, 0, 0)), (-1.1, (0, 4, 0)), (0.9, (0, 0, 4)), (1.3, (3, 2, 1)), (-0.8, (1, 4, 2)), (0.5, (2, 1, 4)),
             (2.0, (4, 4, 4)), (0.25, (0, 0, 0)), (-0.6, (1, 0, 3))]
    o.set_state(0, 0, _poly_cell_averages(h0, (16, 16, 16), (0, 0, 0), coefs))
    o.fill_ghosts(1, 0.0)
    raw = o.get_raw(1, 0)
    want = _poly_cell_averages(h0 / 2, o.box_shape(1), (8, 16, 8), coefs, g=3)
    ghost = np.ones(raw.shape, dtype=bool)
    ghost[3:-3, 3:-3, 3:-3] = False
    assert np.abs(raw - want)[ghost].max() < 2e-15
    # a quintic is not reproduced (the scheme is exactly quartic), and trilinear does not reproduce the quartic
    o.set_state(0, 0, _poly_cell_averages(h0, (16, 16, 16), (0, 0, 0), [(1.0, (5, 0, 0))]))
    o.fill_ghosts(1, 0.0)
    want5 = _poly_cell_averages(h0 / 2, o.box_shape(1), (8, 16, 8), [(1.0, (5, 0, 0))], g=3)
    assert 1e-9 < np.abs(o.get_raw(1, 0) - want5)[ghost].max() < 1e-5
    o1 = two_level(h0=h0, lam=0.0)
    o1.set_state(0, 0, _poly_cell_averages(h0, (16, 16, 16), (0, 0, 0), coefs))
    o1.fill_ghosts(1, 0.0)
    assert np.abs(o1.get_raw(1, 0) - want)[ghost].max() > 1e-4


def test_quartic_interpolation_is_conservative_and_matches_a_numerical_polynomial_fit():
    rng = np.random.default_rng(12)
    g = 2  # two ghost layers = one whole coarse cell per face: every coarse cell in the shell has all 8 children there
    o = two_level(g=g, h0=1.0, lam=0.0, interp=4)
    coarse = [rng.normal(size=(16, 16, 16)) for _ in range(4)]
    for c in range(4):
        o.set_state(0, c, coarse[c])
    o.fill_ghosts(1, 0.0)
    lo = (8, 16, 8)  # fine lo (x, y, z); raw index (kz, jy, ix) <-> fine index lo - g + index
    for c in range(4):
        raw = o.get_raw(1, c)
        nz, ny, nx = raw.shape
        blocks = raw.reshape(nz // 2, 2, ny // 2, 2, nx // 2, 2).mean(axis=(1, 3, 5))
        cz0, cy0, cx0 = (lo[2] - g) // 2, (lo[1] - g) // 2, (lo[0] - g) // 2
        par = coarse[c][cz0:cz0 + nz // 2, cy0:cy0 + ny // 2, cx0:cx0 + nx // 2]
        shell = np.ones(par.shape, dtype=bool)
        shell[1:-1, 1:-1, 1:-1] = False
        assert np.abs(blocks - par)[shell].max() < 4e-15  # conservative: the 8 children average to their parent
    # data varying along ONE axis: the ghost value is the fine-cell average of the quartic fitted, numerically, to
    # the five coarse cell averages around the parent (no weights typed in)
    for axis in range(3):  # 0 = x
        prof = rng.normal(size=16)
        shape = [1, 1, 1]
        shape[2 - axis] = 16
        o.set_state(0, 0, np.broadcast_to(prof.reshape(shape), (16, 16, 16)).copy())
        o.fill_ghosts(1, 0.0)
        raw = o.get_raw(1, 0)
        for fidx in (lo[axis] - 2, lo[axis] - 1):  # the two low-side ghost layers along this axis
            c0, r = fidx // 2, fidx % 2
            edges = np.arange(-2.5, 3.0, 1.0)
            A = np.array([[_cell_avg_monomial(p, edges[m], edges[m + 1]) for p in range(5)] for m in range(5)])
            coef = np.linalg.solve(A, prof[c0 - 2:c0 + 3])
            a, b = (-0.5, 0.0) if r == 0 else (0.0, 0.5)
            want = sum(coef[p] * _cell_avg_monomial(p, a, b) for p in range(5))
            sl = [slice(g, g + 1)] * 3
            sl[2 - axis] = slice(fidx - (lo[axis] - g), fidx - (lo[axis] - g) + 1)
            assert abs(raw[tuple(sl)].item() - want) < 1e-13


def test_quartic_interpolation_in_time_and_validation():
    """same linear-in-time rule as the trilinear fill (L72): psi = b + c t stays exact through two coarse steps"""
    o = two_level(h0=1.0, lam=0.0, order=2, interp=4)
    b, c = 0.25, 0.5
    for ib in (0, 1):
        shp = o.box_shape(ib)
        o.set_state(ib, 0, np.full(shp, b))
        o.set_state(ib, 2, np.full(shp, c))
    t, dt = 2.0, 0.5
    for _ in range(2):
        o.rk_step(dt, t)
        t += dt
    for ib in (0, 1):
        assert np.abs(o.get_state(ib, 0) - (b + c * (t - 2.0))).max() < 1e-14
    with pytest.raises(OracleError):
        Oracle(16, interp=2)  # only trilinear (0) and quartic conservative (4) are built
