"""Pins for the oracle parts added in round 2: gravitational-wave auxiliary fields (O13, Eq.16),
the user-defined Runge-Kutta-Nystrom integrator (O14, L808-815) and the level-0 shadow level (O15, L98).
As in test_oracle_pins.py every check compares oracle/sledge_oracle.cpp with something OTHER than itself: closed
forms, independently written scalar solvers, numpy, or the oracle's own already pinned RK4 path.  CPU only."""
import math

import numpy as np
import pytest

from oracle.oracle import Oracle, OracleError
from paper_2404_02950_b200 import inputs

GW_IJ = [(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)]  # xx, yy, zz, xy, xz, yz (L436)
U0, DU0 = 4, 10


def coords(shape):
    z, y, x = np.meshgrid(*[np.arange(s, dtype=np.float64) for s in shape], indexing="ij")
    return x, y, z


# ------------------------------------------------------------------------------------------------
# O13 gravitational-wave auxiliary fields
# ------------------------------------------------------------------------------------------------


@pytest.mark.parametrize("order", [1, 2, 3])
def test_gw_source_is_the_outer_product_of_exact_gradients_on_polynomials(order):
    """Gradient<order> is exact on polynomials of degree 2 / 4 / 6 per axis (analytic ghosts on a NON-periodic box),
    so k_du_ij = c_gw sum_c d_i psi_c d_j psi_c must equal the analytic outer product in every cell and for each of
    the six components in the paper's order xx, yy, zz, xy, xz, yz.  Distinct polynomials per axis and per field
    component catch a wrong index pair, a missing field component, a wrong coefficient or a wrong power of h."""
    g, deg = order, 2 * order
    n = (8, 16, 24)
    h, cgw = 0.37, 1.7
    o = Oracle(n, nghost=g, blocking_factor=8, lap_order=order, h0=h, lam=0.0, gw=True, gw_coupling=cgw)
    zz, yy, xx = np.meshgrid(*[(np.arange(-g, s + g) + 0.5) * h for s in n[::-1]], indexing="ij")
    rng = np.random.default_rng(11)
    co = rng.uniform(-1, 1, size=(2, 3, deg + 1))
    ax = (xx, yy, zz)

    def poly(c, t):
        return sum(c[m] * t ** m for m in range(deg + 1))

    def dpoly(c, t):
        return sum(m * c[m] * t ** (m - 1) for m in range(1, deg + 1))

    grads = []
    for c in range(2):
        o.set_raw(0, c, sum(poly(co[c, d], ax[d]) for d in range(3)))
        grads.append([dpoly(co[c, d], ax[d]) for d in range(3)])
    k = o.eval_rhs(0, eta=1.0, fill=False)[0]
    v = slice(g, -g)
    for m, (i, j) in enumerate(GW_IJ):
        want = cgw * (grads[0][i] * grads[0][j] + grads[1][i] * grads[1][j])[v, v, v]
        assert np.abs(k[DU0 + m] - want).max() < 1e-11 * max(1.0, np.abs(want).max()), (m, i, j)
        assert np.abs(k[U0 + m]).max() == 0.0  # k_u = du = 0


def test_gw_gradient_order1_is_not_exact_on_a_cubic():
    """Negative control: the 3-point gradient has the error h^2 u'''/6 on x^3, which the source must show."""
    g, n, h = 1, (8, 8, 8), 0.5
    o = Oracle(n, nghost=g, blocking_factor=8, lap_order=1, h0=h, lam=0.0, gw=True, gw_coupling=1.0)
    zz, yy, xx = np.meshgrid(*[(np.arange(-g, s + g) + 0.5) * h for s in n[::-1]], indexing="ij")
    o.set_raw(0, 0, xx ** 3)
    k = o.eval_rhs(0, eta=1.0, fill=False)[0]
    v = slice(g, -g)
    want = (3 * xx ** 2 + h * h) ** 2  # (u(x+h) - u(x-h)) / 2h = 3x^2 + h^2 exactly
    assert np.abs(k[DU0 + 0] - want[v, v, v]).max() < 1e-11 * want.max()


@pytest.mark.parametrize("order", [1, 2, 3])
def test_gw_source_on_plane_waves_uses_the_gradient_symbol(order):
    """psi1 = sin(k.x), psi2 = cos(q.x) on the periodic lattice: D_d psi1 = s(k_d) cos(k.x), D_d psi2 = -s(q_d)
    sin(q.x) with the stencil's symbol s, so T_ij is a closed-form quadratic form (VERDICT: "plane-wave source")."""
    n, h, cgw = (16, 8, 24), 0.5, 0.9
    o = Oracle(n, nghost=3, lap_order=order, h0=h, lam=0.0, gw=True, gw_coupling=cgw)
    x, y, z = coords(n[::-1])
    mk, mq = (1, 2, 3), (2, -1, 1)
    kh = [2 * math.pi * mk[d] / n[d] for d in range(3)]
    qh = [2 * math.pi * mq[d] / n[d] for d in range(3)]
    pk = kh[0] * x + kh[1] * y + kh[2] * z
    pq = qh[0] * x + qh[1] * y + qh[2] * z

    def sym(a):
        if order == 1:
            return math.sin(a) / h
        if order == 2:
            return (8 * math.sin(a) - math.sin(2 * a)) / (6 * h)
        return (45 * math.sin(a) - 9 * math.sin(2 * a) + math.sin(3 * a)) / (30 * h)

    o.set_state(0, 0, np.sin(pk))
    o.set_state(0, 1, np.cos(pq))
    k = o.eval_rhs(0, eta=2.0)[0]
    for m, (i, j) in enumerate(GW_IJ):
        want = cgw * (sym(kh[i]) * sym(kh[j]) * np.cos(pk) ** 2 + sym(qh[i]) * sym(qh[j]) * np.sin(pq) ** 2)
        assert np.abs(k[DU0 + m] - want).max() < 1e-12 * max(1.0, np.abs(want).max())


def test_gw_free_field_obeys_the_rk4_amplification_matrix_with_friction_off_and_scalar_ode_with_it_on():
    """c_gw = 0: every u_ij is a free wave, R(dt A)^n with the lattice symbol (the pin of O4, applied to each of the six
    components with its own amplitude); with a spatially constant u and kappa_u != 0, du' = -(kappa_u/eta) du is a
    scalar ODE integrated by an independently written RK4 (stage times included)."""
    n, h = (8, 16, 8), 0.5
    o = Oracle(n, nghost=2, lap_order=2, h0=h, lam=0.0, gw=True, gw_coupling=0.0)
    x, y, z = coords(n[::-1])
    kh = [2 * math.pi * m / s for m, s in zip((1, 3, 2), n)]
    ph = kh[0] * x + kh[1] * y + kh[2] * z
    w2 = sum(16 / 3 * math.sin(a / 2) ** 2 - 1 / 3 * math.sin(a) ** 2 for a in kh) / h ** 2
    amp = [(0.3 + 0.1 * m, -0.2 + 0.05 * m) for m in range(6)]
    for m, (A, B) in enumerate(amp):
        o.set_state(0, U0 + m, A * np.cos(ph))
        o.set_state(0, DU0 + m, B * np.cos(ph))
    dt, steps, eta = 0.1, 15, 1.0
    Z = dt * np.array([[0.0, 1.0], [-w2, 0.0]])
    R = np.eye(2) + Z + Z @ Z / 2 + Z @ Z @ Z / 6 + Z @ Z @ Z @ Z / 24
    Rn = np.linalg.matrix_power(R, steps)
    for _ in range(steps):
        o.rk_step(dt, eta)
        eta += dt
    for m, (A, B) in enumerate(amp):
        a1, b1 = Rn @ np.array([A, B])
        assert np.abs(o.get_state(0, U0 + m) - a1 * np.cos(ph)).max() < 1e-13
        assert np.abs(o.get_state(0, DU0 + m) - b1 * np.cos(ph)).max() < 1e-12
    # friction: constant fields
    ku = 3.0
    o = Oracle(8, nghost=1, lap_order=1, h0=1.0, lam=0.0, gw=True, gw_coupling=5.0, gw_friction=ku)
    yv = np.array([[0.1 * (m + 1), 0.3 - 0.1 * m] for m in range(6)])  # (u, du) per component
    for m in range(6):
        o.set_state(0, U0 + m, np.full((8, 8, 8), yv[m, 0]))
        o.set_state(0, DU0 + m, np.full((8, 8, 8), yv[m, 1]))
    f = lambda v, e: np.stack([v[:, 1], -(ku / e) * v[:, 1]], axis=1)
    eta, dt = 1.5, 0.05
    for _ in range(10):
        o.rk_step(dt, eta)
        k1 = f(yv, eta)
        k2 = f(yv + 0.5 * dt * k1, eta + 0.5 * dt)
        k3 = f(yv + 0.5 * dt * k2, eta + 0.5 * dt)
        k4 = f(yv + dt * k3, eta + dt)
        yv = yv + dt / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
        eta += dt
    for m in range(6):
        assert abs(o.get_state(0, U0 + m).flat[0] - yv[m, 0]) < 1e-14
        assert abs(o.get_state(0, DU0 + m).flat[7] - yv[m, 1]) < 1e-14


def test_gw_leaves_the_scalar_field_untouched_and_is_linear_in_the_coupling():
    """The scalar components must evolve exactly as without the auxiliary fields (bit for bit); the auxiliary fields
    are linear in c_gw, exactly so for a factor that is a power of two; and the source does not change when the two
    scalar components are exchanged."""
    n, kw = 16, dict(nghost=2, lap_order=2, h0=0.5, lam=1.0)
    psi = [inputs.grf(n, 0.5, s).numpy() for s in (71, 72)]
    a = Oracle(n, **kw)
    b = Oracle(n, gw=True, gw_coupling=1.0, **kw)
    c = Oracle(n, gw=True, gw_coupling=4.0, **kw)
    for o in (a, b, c):
        for q in range(2):
            o.set_state(0, q, psi[q])
    eta, dt = 1.0, 0.05
    for _ in range(5):
        for o in (a, b, c):
            o.rk_step(dt, eta)
        eta += dt
    for q in range(4):
        assert np.array_equal(a.get_state(0, q), b.get_state(0, q))
    for m in range(6):
        ub, uc = b.get_state(0, U0 + m), c.get_state(0, U0 + m)
        assert np.abs(ub).max() > 1e-6
        assert np.array_equal(4.0 * ub, uc)
    # the source is symmetric under exchanging the two scalar components: sum_c d_i psi_c d_j psi_c
    d = Oracle(n, gw=True, gw_coupling=1.0, **kw)
    e = Oracle(n, gw=True, gw_coupling=1.0, **kw)
    for q in range(2):
        d.set_state(0, q, psi[1 - q])
        e.set_state(0, q, psi[q])
    kd, ke = d.eval_rhs(0, 1.0)[0], e.eval_rhs(0, 1.0)[0]
    for m in range(6):
        assert np.abs(ke[DU0 + m] - kd[DU0 + m]).max() < 1e-12 * max(1.0, np.abs(ke[DU0 + m]).max())


def test_gw_fully_covered_level1_equals_uniform_fine_run():
    """AMR plumbing of the 12 extra components (ghost fill, subcycling, average-down): a level 1 that covers the whole
    domain reproduces the uniform fine run bit for bit, auxiliary fields included."""
    n0, h0, dt, eta0, g, order = 8, 1.0, 0.25, 1.0, 2, 2
    nf = 2 * n0
    kw = dict(nghost=g, lap_order=order, lam=1.0, gw=True, gw_coupling=0.5, gw_friction=1.0)
    fields = [inputs.grf(nf, 0.5, 80 + s).numpy() * (1.0 if s < 2 else 0.1) for s in range(16)]
    ref = Oracle(nf, h0=h0 / 2, **kw)
    for c, a in enumerate(fields):
        ref.set_state(0, c, a)
    eta = eta0
    for _ in range(4):
        ref.rk_step(dt / 2, eta)
        eta += dt / 2
    boxes = [(0, (0, 0, 0), (n0 - 1,) * 3), (1, (0, 0, 0), (nf - 1,) * 3)]
    o = Oracle(n0, boxes=boxes, n_levels=2, h0=h0, **kw)
    for c, a in enumerate(fields):
        o.set_state(1, c, a)
    o.average_down(1)
    eta = eta0
    for _ in range(2):
        o.rk_step(dt, eta)
        eta += dt
    for c in range(16):
        f = o.get_state(1, c)
        assert np.array_equal(f, ref.get_state(0, c)), c
        want = f.reshape(n0, 2, n0, 2, n0, 2).sum(axis=5).sum(axis=3).sum(axis=1) * 0.125
        assert np.abs(o.get_state(0, c) - want).max() < 4e-15


# ------------------------------------------------------------------------------------------------
# O14 user-defined Runge-Kutta-Nystrom tableau (integrator.type 20)
# ------------------------------------------------------------------------------------------------

# Nystrom's classical three-stage fourth-order scheme (Hairer, Norsett, Wanner I, sect. II.14): test data, passed to
# the oracle exactly as a user would pass rkn.nodes / rkn.weights_b / rkn.weights_bar_b / rkn.tableau (L812-815)
RKN4 = dict(nodes=[0.0, 0.5, 1.0], weights_b=[1 / 6, 4 / 6, 1 / 6], weights_bar_b=[1 / 6, 1 / 3, 0.0],
            tableau=[0.0, 1 / 8, 0.0, 0.0, 0.5, 0.0])
# classic RK4 applied to (psi, Pi) with psi'' = f(psi) IS the four-stage RKN scheme
#   c = (0, 1/2, 1/2, 1), a31 = 1/4, a42 = 1/2, bbar = (1/6, 1/6, 1/6, 0), b = (1/6, 1/3, 1/3, 1/6)
RK4_AS_RKN = dict(nodes=[0.0, 0.5, 0.5, 1.0], weights_b=[1 / 6, 1 / 3, 1 / 3, 1 / 6], weights_bar_b=[1 / 6, 1 / 6, 1 / 6, 0.0],
                  tableau=[0.0, 0.0, 0.0, 0.25, 0.0, 0.0, 0.0, 0.5, 0.0, 0.0])


def scalar_rkn(y, v, eta, dt, lam, a, tab):
    """Independent scalar Nystrom step for psi_c'' = -psi_c (lam eta^2 (psi1^2 + psi2^2 - 1) + a), c = 1, 2."""
    c, b, bb = tab["nodes"], tab["weights_b"], tab["weights_bar_b"]
    s = len(c)
    A = np.zeros((s, s))
    q = 0
    for i in range(s):
        for j in range(i + 1):
            A[i, j] = tab["tableau"][q]
            q += 1
    fs = []
    for i in range(s):
        Y = y + c[i] * dt * v + dt * dt * sum(A[i, j] * fs[j] for j in range(i))
        e = eta + c[i] * dt
        fs.append(-Y * (lam * e * e * (Y[0] ** 2 + Y[1] ** 2 - 1.0) + a))
    return (y + dt * v + dt * dt * sum(bb[i] * fs[i] for i in range(s)), v + dt * sum(b[i] * fs[i] for i in range(s)))


@pytest.mark.parametrize("tab", [RKN4, RK4_AS_RKN], ids=["nystrom4", "rk4-as-rkn"])
def test_rkn_constant_field_equals_scalar_nystrom_solve(tab):
    n, lam, a = 8, 1.3, 0.56233
    o = Oracle(n, nghost=2, lap_order=2, h0=0.7, lam=lam, a_mass=a, integrator=20, rkn=tab)
    y, v = np.array([0.3, -0.8]), np.array([0.1, 0.25])
    for c in range(2):
        o.set_state(0, c, np.full((n, n, n), y[c]))
        o.set_state(0, 2 + c, np.full((n, n, n), v[c]))
    eta, dt = 1.5, 0.05
    for _ in range(20):
        o.rk_step(dt, eta)
        y, v = scalar_rkn(y, v, eta, dt, lam, a, tab)
        eta += dt
    for c in range(2):
        assert abs(o.get_state(0, c).flat[3] - y[c]) < 1e-14
        assert abs(o.get_state(0, 2 + c).flat[3] - v[c]) < 1e-14
        assert np.all(o.get_state(0, c) == o.get_state(0, c).flat[0])


def test_rkn_with_the_rk4_tableau_reproduces_the_rk4_run():
    """Structural pin against the already pinned RK4 path: with friction 0 classic RK4 is a four-stage Nystrom scheme,
    so the two integrators must agree to rounding on a nonlinear multi-box run with ghosts -- stage times, the
    flattened lower-triangular tableau, b and bar-b each show up at O(dt^2) or larger if misread."""
    n = 16
    boxes = inputs.split_level0(n, 8)
    kw = dict(boxes=boxes, nghost=2, lap_order=2, h0=0.5, lam=1.0, a_mass=0.2)
    psi = [inputs.grf(n, 0.5, s).numpy() for s in (61, 62)]
    pi = [0.3 * inputs.grf(n, 0.5, s).numpy() for s in (63, 64)]
    a = Oracle(n, integrator=4, **kw)
    b = Oracle(n, integrator=20, rkn=RK4_AS_RKN, **kw)
    for o in (a, b):
        for ib, (_, lo, hi) in enumerate(boxes):
            sl = tuple(slice(lo[d], hi[d] + 1) for d in (2, 1, 0))
            for c in range(2):
                o.set_state(ib, c, psi[c][sl])
                o.set_state(ib, 2 + c, pi[c][sl])
    eta, dt = 1.0, 0.05
    for _ in range(10):
        a.rk_step(dt, eta)
        b.rk_step(dt, eta)
        eta += dt
    for ib in range(len(boxes)):
        for c in range(4):
            assert np.abs(a.get_state(ib, c) - b.get_state(ib, c)).max() < 2e-13


def test_rkn4_is_fourth_order_and_differs_from_rk4():
    n, kw = 16, dict(nghost=2, lap_order=2, h0=0.5, lam=1.0)
    psi = [inputs.grf(n, 0.5, s).numpy() for s in (65, 66)]

    def run(dt, steps, **ikw):
        o = Oracle(n, **kw, **ikw)
        for c in range(2):
            o.set_state(0, c, psi[c])
        eta = 1.0
        for _ in range(steps):
            o.rk_step(dt, eta)
            eta += dt
        return np.stack([o.get_state(0, c) for c in range(4)])

    ref = run(0.2 / 64, 64 * 4, integrator=20, rkn=RKN4)
    errs = [np.abs(run(0.2 / m, 4 * m, integrator=20, rkn=RKN4) - ref).max() for m in (1, 2, 4)]
    assert 11 < errs[0] / errs[1] < 22 and 11 < errs[1] / errs[2] < 22, errs
    assert np.abs(run(0.2, 4, integrator=20, rkn=RKN4) - run(0.2, 4, integrator=4)).max() > 1e-8


def test_rkn_fully_covered_level1_equals_uniform_fine_run_and_validation():
    n0, h0, dt, eta0 = 8, 1.0, 0.25, 1.0
    nf = 2 * n0
    kw = dict(nghost=2, lap_order=2, lam=1.0, integrator=20, rkn=RKN4)
    psi = [inputs.grf(nf, 0.5, s).numpy() for s in (41, 42)]
    pi = [0.1 * inputs.grf(nf, 0.5, s).numpy() for s in (43, 44)]
    ref = Oracle(nf, h0=h0 / 2, **kw)
    for c, a in enumerate(psi + pi):
        ref.set_state(0, c, a)
    eta = eta0
    for _ in range(4):
        ref.rk_step(dt / 2, eta)
        eta += dt / 2
    boxes = [(0, (0, 0, 0), (n0 - 1,) * 3), (1, (0, 0, 0), (nf - 1,) * 3)]
    o = Oracle(n0, boxes=boxes, n_levels=2, h0=h0, **kw)
    for c, a in enumerate(psi + pi):
        o.set_state(1, c, a)
    o.average_down(1)
    eta = eta0
    for _ in range(2):
        o.rk_step(dt, eta)
        eta += dt
    for c in range(4):
        assert np.array_equal(o.get_state(1, c), ref.get_state(0, c))
    with pytest.raises(OracleError):
        Oracle(8, nghost=1, integrator=20, rkn=RKN4, friction=2.0)  # psi'' = f(psi) only
    bad = dict(RKN4, tableau=[0.0, 1 / 8, 0.1, 0.0, 0.5, 0.0])
    with pytest.raises(OracleError):
        Oracle(8, nghost=1, integrator=20, rkn=bad)  # implicit diagonal entry
    with pytest.raises(OracleError):
        Oracle(8, nghost=1, integrator=20)  # no tableau


# ------------------------------------------------------------------------------------------------
# O15 shadow level (L98)
# ------------------------------------------------------------------------------------------------


def rk4_scalar(y, eta, dt, lam):
    def f(y, e):
        p1, p2, q1, q2 = y
        pot = lam * e * e * (p1 * p1 + p2 * p2 - 1.0)
        return np.array([q1, q2, -p1 * pot, -p2 * pot])
    k1 = f(y, eta)
    k2 = f(y + 0.5 * dt * k1, eta + 0.5 * dt)
    k3 = f(y + 0.5 * dt * k2, eta + 0.5 * dt)
    k4 = f(y + dt * k3, eta + dt)
    return y + dt / 6.0 * (k1 + 2 * k2 + 2 * k3 + k4)


def test_shadow_tags_on_a_constant_field_equal_the_scalar_step_doubling_error():
    """Spatially constant field: the shadow level takes ONE RK4 step of 2 dt, level 0 two of dt; Delta_c is the
    step-doubling difference of the scalar ODE, computed independently.  Thresholds just below / above it flip every
    tag (strict >), per component."""
    n, lam, eta, dt = 8, 1.0, 1.5, 0.2
    y0 = np.array([0.3, -0.8, 0.1, 0.25])
    big = rk4_scalar(y0, eta, 2 * dt, lam)
    two = rk4_scalar(rk4_scalar(y0, eta, dt, lam), eta + dt, dt, lam)
    delta = np.abs(big - two)
    assert delta.min() > 1e-7
    for c in range(4):
        for scale, hit in ((0.99, True), (1.01, False)):
            o = Oracle(n, nghost=2, lap_order=2, h0=0.5, lam=lam, blocking_factor=4)
            for q in range(4):
                o.set_state(0, q, np.full((n, n, n), y0[q]))
            eps = [np.inf] * 4
            eps[c] = scale * delta[c]
            tags, counts = o.shadow_tee(dt, eta, *eps)
            assert np.all(tags[0] == ((1 << c) if hit else 0))
            assert counts.sum() == (n ** 3 if hit else 0)
            # the hierarchy itself has taken the two steps of dt
            for q in range(4):
                assert abs(o.get_state(0, q).flat[5] - two[q]) < 1e-14


def test_shadow_level_equals_a_hand_built_coarse_run():
    """Independent reconstruction with numpy and the already pinned single-level path: coarsen by block means, run ONE
    box of n/2 cells at spacing 2h for one step of 2 dt, compare with the block means of the fine run after two steps."""
    n, h, lam, eta, dt = 16, 0.5, 1.0, 1.0, 0.05
    boxes = inputs.split_level0(n, 8)
    psi = [inputs.grf(n, 0.4, s).numpy() for s in (91, 92)]
    pi = [0.5 * inputs.grf(n, 0.4, s).numpy() for s in (93, 94)]
    blockmean = lambda a: a.reshape(n // 2, 2, n // 2, 2, n // 2, 2).sum(axis=5).sum(axis=3).sum(axis=1) * 0.125
    coarse = Oracle(n // 2, nghost=2, lap_order=2, h0=2 * h, lam=lam, blocking_factor=8)
    fine = Oracle(n, boxes=boxes, nghost=2, lap_order=2, h0=h, lam=lam)
    sh = Oracle(n, boxes=boxes, nghost=2, lap_order=2, h0=h, lam=lam)
    for c, a in enumerate(psi + pi):
        coarse.set_state(0, c, blockmean(a))
        for o in (fine, sh):
            for ib, (_, lo, hi) in enumerate(boxes):
                o.set_state(ib, c, a[lo[2]:hi[2] + 1, lo[1]:hi[1] + 1, lo[0]:hi[0] + 1])
    coarse.rk_step(2 * dt, eta)
    fine.rk_step(dt, eta)
    fine.rk_step(dt, eta + dt)

    def assemble(o, c):
        out = np.empty((n, n, n))
        for ib, (_, lo, hi) in enumerate(boxes):
            out[lo[2]:hi[2] + 1, lo[1]:hi[1] + 1, lo[0]:hi[0] + 1] = o.get_state(ib, c)
        return out

    delta = [np.abs(coarse.get_state(0, c) - blockmean(assemble(fine, c))) for c in range(4)]
    eps = [float(np.median(d)) for d in delta]  # half of the parents above, half below
    tags, counts = sh.shadow_tee(dt, eta, *eps)
    want = np.zeros((n // 2,) * 3, dtype=np.uint8)
    for c in range(4):
        want |= (delta[c] > eps[c]).astype(np.uint8) << c
    # cells whose Delta is within rounding of the threshold may fall either way in the two evaluations
    sure = np.ones_like(want, dtype=bool)
    for c in range(4):
        sure &= np.abs(delta[c] - eps[c]) > 1e-13
    got = np.empty((n, n, n), dtype=np.uint8)
    for ib, (_, lo, hi) in enumerate(boxes):
        got[lo[2]:hi[2] + 1, lo[1]:hi[1] + 1, lo[0]:hi[0] + 1] = tags[ib]
    up = np.repeat(np.repeat(np.repeat(want, 2, axis=0), 2, axis=1), 2, axis=2)
    sure8 = np.repeat(np.repeat(np.repeat(sure, 2, axis=0), 2, axis=1), 2, axis=2)
    assert sure.mean() > 0.99
    assert np.array_equal(got[sure8], up[sure8])
    assert 0.2 < (got != 0).mean() < 1.0
    assert counts.sum() == (got != 0).sum()
    for c in range(4):  # the hierarchy ends where two plain steps end
        assert np.array_equal(assemble(sh, c), assemble(fine, c))


def test_shadow_error_shrinks_with_resolution():
    """Smooth data: halving h and dt cuts the largest level-0 truncation-error estimate by > 4 (the pair shadow / level 0
    differs at O(h^2) of the smoothed field; measured by bisection through the tag output)."""
    def max_delta(n):
        h, dt, eta = 8.0 / n, 0.4 / n, 1.0
        x = (np.arange(n) + 0.5) * h
        zz, yy, xx = np.meshgrid(x, x, x, indexing="ij")
        k = 2 * math.pi / 8.0
        psi1 = 0.5 * np.sin(k * xx) * np.cos(k * yy) + 0.2 * np.cos(k * zz)
        psi2 = 0.3 * np.cos(k * xx + 0.3) * np.sin(k * zz)
        lo, hi = 0.0, 1.0
        for _ in range(30):
            mid = 0.5 * (lo + hi)
            o = Oracle(n, nghost=2, lap_order=2, h0=h, lam=1.0)
            o.set_state(0, 0, psi1)
            o.set_state(0, 1, psi2)
            tags, _ = o.shadow_tee(dt, eta, mid, np.inf)
            if tags[0].any():
                lo = mid
            else:
                hi = mid
        return hi

    d16, d32 = max_delta(16), max_delta(32)
    assert d16 > 1e-6 and d16 / d32 > 4.0, (d16, d32)
