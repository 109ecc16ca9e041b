"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Bars (BASELINE.json north_star): fp64 max abs field error <= 1e-11 after the configured number of steps;
fp32 max relative error <= 2e-5; string tags and box counts bit-exact when both sides tag the same state.
Sizes: small enough for the oracle to finish in seconds, large enough to span several K1 tiles
(32 x 8 x 64 cells fp64, 64 x 8 x 64 fp32) and ragged tails."""
import numpy as np
import pytest
import torch

from paper_2404_02950_b200 import inputs

pytestmark = pytest.mark.gpu

F64_TOL = 1e-11
F32_TOL = 2e-5


def _pair():
    import _pair as P  # tests/ is on sys.path (pytest rootdir conftest)
    return P


def _compare_tags(o, s, level):
    P = _pair()
    P.upload_oracle_state(o, s)
    ot, oc = o.tag_strings(level)
    gt, gc = s.tag_strings(level)
    s.synchronize()
    gts = s.split_tags(level, gt)
    for a, b in zip(ot, gts):
        assert np.array_equal(a, b.cpu().numpy())
    assert np.array_equal(oc.astype(np.int64), gc.cpu().numpy().astype(np.int64))
    return sum(int((a != 0).sum()) for a in ot)


# ---- C1: the small BASELINE.json config, full length -------------------------------------------------
# DESIGN.md reading R12: with the literal C1 numbers (h = 1, dt = 0.25, unit-variance GRF, eta up to 3.5) classic
# RK4 is unstable -- the local frequency sqrt(12/h^2 + lambda eta^2 (3|psi|^2 - 1)) dt passes the RK4 limit
# 2.83 where |psi| > 1 -- and the fields reach 1e2 at step 8, 1e22 at step 9 and overflow at step 10 IN THE ORACLE
# (tests/test_oracle_pins.py::test_c1_literal_parameters_blow_up).  The literal run therefore carries the
# 1e-11 absolute bar while the oracle state is bounded (max |u| <= 20, the same bound the stable run asserts);
# once the instability has taken off the cubic term multiplies RELATIVE rounding differences by ~3 per RHS
# evaluation, so no fixed bar holds: there the test only checks that the CUDA path diverges the same way
# (agreement to 1e-6 of the largest oracle value while finite, non-finite at the same step).  The stabilised
# variant C1s (same grid, fields, eta range; dt = 0.0625, 40 steps) carries 1e-11 absolute over the whole run.

def _c1_run(flow, dt, steps, literal):
    P = _pair()
    cfg = inputs.CONFIGS["C1"]
    o, s = P.make_pair(cfg.n0, nghost=cfg.nghost, lap_order=cfg.lap_order, h0=cfg.h0, lam=cfg.lam, rk_dataflow=flow)
    P.init_grf(o, s, cfg.n0, cfg.grf_f, cfg.seeds)
    eta = cfg.eta0
    n_tagged = 0
    bounded_steps = 0
    for step in range(steps):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
        big = max(float(np.abs(o.get_state(0, c)).max()) for c in range(4))
        if not np.isfinite(big):
            assert literal
            gbig = max(float(s.get_state(0, c).abs().max()) for c in range(4))
            assert not np.isfinite(gbig) or gbig > 1e100  # the CUDA path blew up at the same step
            break
        if not literal:
            assert big < 20.0
        if big <= 20.0:
            assert P.max_err(o, s) <= F64_TOL, f"step {step}"
            bounded_steps += 1
        else:  # diverging run (R12): same blow-up, no fixed bar
            assert P.max_err(o, s) <= 1e-6 * big, f"step {step}"
        # free-running tags: both sides tag their own state; identical while the states agree to the last bits
        ot, oc = o.tag_strings(0)
        gt, gc = s.tag_strings(0)
        if big < 1e3:
            assert np.array_equal(ot[0], s.split_tags(0, gt)[0].cpu().numpy())
            assert np.array_equal(oc.astype(np.int64), gc.cpu().numpy().astype(np.int64))
        n_tagged += int((ot[0] != 0).sum())
    assert n_tagged > 0  # the GRF does contain strings
    assert bounded_steps >= (5 if literal else steps)
    s.synchronize()
    return eta


@pytest.mark.parametrize("flow", ["lean", "classic", "fused"])
def test_c1_literal_32cubed_10_steps_with_tags(flow):
    _c1_run(flow, dt=inputs.CONFIGS["C1"].dt, steps=10, literal=True)


@pytest.mark.parametrize("flow", ["lean", "classic", "fused", "fused3"])
def test_c1s_stabilised_32cubed_eta_1_to_3p5_with_tags(flow):
    eta = _c1_run(flow, dt=0.0625, steps=40, literal=False)
    assert eta == pytest.approx(3.5)


# ---- ragged single-level grids, several boxes, both stencils, friction and mass terms -----------------

def _ragged_boxes():
    # 40 x 24 x 72 domain cut into boxes of different sizes (bf = 8): exercises partial K1 tiles in x and y,
    # same-level ghost copies across box faces/edges/corners and the periodic wrap, and two z chunks.
    return [
        (0, (0, 0, 0), (31, 15, 71)),
        (0, (32, 0, 0), (39, 15, 71)),
        (0, (0, 16, 0), (39, 23, 39)),
        (0, (0, 16, 40), (15, 23, 71)),
        (0, (16, 16, 40), (39, 23, 71)),
    ]


@pytest.mark.parametrize("order,g", [(1, 1), (1, 3), (2, 2), (2, 3), (3, 3), (3, 5)])
@pytest.mark.parametrize("flow", ["lean", "classic", "fused", "fused3"])
def test_ragged_multibox_fp64(order, g, flow):
    P = _pair()
    n0 = (40, 24, 72)
    o, s = P.make_pair(n0, boxes=_ragged_boxes(), nghost=g, lap_order=order, h0=0.5, lam=0.7, a_mass=0.3,
                       friction=2.0, rk_dataflow=flow)
    P.init_smooth(o, s, n0, seed=11)
    eta, dt = 1.5, 0.1
    for _ in range(4):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
    assert P.max_err(o, s) <= F64_TOL
    _compare_tags(o, s, 0)


# ---- Kreiss-Oliger dissipation (Eq.7; S8(f) NEXT-2) inside K1 ---------------------------------

KO_EPS = (0.02, 0.03, 0.05, 0.07)  # per component, all different (L750)


@pytest.mark.parametrize("order,ko,g", [(1, 2, 2), (2, 2, 3), (3, 2, 3), (1, 3, 3), (2, 3, 3), (3, 3, 5)])
@pytest.mark.parametrize("flow", ["lean", "classic", "fused"])
def test_kreiss_oliger_ragged_multibox_fp64(order, ko, g, flow):
    """Every (Laplacian order, dissipation order) pair: the z-window radius is the larger of the two, Pi is differenced
    too; `fused` must fall back to the staged sweeps (k_psi is no longer pointwise)."""
    P = _pair()
    n0 = (40, 24, 72)
    o, s = P.make_pair(n0, boxes=_ragged_boxes(), nghost=g, lap_order=order, h0=0.5, lam=0.7, a_mass=0.3,
                       friction=2.0, rk_dataflow=flow, ko_order=ko, ko_strength=KO_EPS)
    P.init_smooth(o, s, n0, seed=13)
    # grid-scale noise on top, so that the dissipation term is far above the tolerance
    rng = np.random.default_rng(5)
    for ib, (l, lo, hi) in enumerate(s.boxes):
        for c in range(4):
            a = o.get_state(ib, c)
            P.set_both(o, s, ib, c, a + 0.05 * rng.standard_normal(a.shape))
    eta, dt = 1.5, 0.1
    for _ in range(4):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
    assert P.max_err(o, s) <= F64_TOL
    _compare_tags(o, s, 0)


def test_kreiss_oliger_changes_the_result():
    """guards the test above against a silently ignored parameter: with and without the term the GPU runs differ"""
    P = _pair()
    n = 32
    out = []
    for eps in (0.0, 0.05):
        o, s = P.make_pair(n, nghost=3, lap_order=2, h0=0.5, ko_order=3 if eps else 0, ko_strength=eps)
        P.init_grf(o, s, n, 0.9, (81, 82))
        s.rk_step(0.1, 1.0)
        out.append(s.get_state(0, 0).cpu().numpy())
    assert np.abs(out[0] - out[1]).max() > 1e-4


@pytest.mark.parametrize("ko", [2, 3])
@pytest.mark.parametrize("flow", ["lean", "fused"])
def test_kreiss_oliger_two_level_subcycled(ko, flow):
    """Pi ghosts of the fine level come from the time-interpolated coarse state at every stage (L72), h_l per level"""
    P = _pair()
    n0 = 32
    boxes = P.two_level_boxes(n0)
    o, s = P.make_pair(n0, boxes=boxes, n_levels=2, nghost=3, lap_order=2, h0=0.5, rk_dataflow=flow, ko_order=ko,
                       ko_strength=KO_EPS)
    P.init_smooth(o, s, n0, seed=9)
    eta, dt = 2.0, 0.1
    for _ in range(3):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
    assert P.max_err(o, s) <= F64_TOL
    for l in (0, 1):
        _compare_tags(o, s, l)


@pytest.mark.parametrize("ko", [2, 3])
def test_kreiss_oliger_fp32(ko):
    P = _pair()
    n = 64
    o, s = P.make_pair(n, nghost=3, lap_order=2, h0=0.125, dtype="f32", ko_order=ko, ko_strength=0.05)
    P.init_grf(o, s, n, 0.25, (71, 72))
    eta, dt = 1.0, 0.03125
    for _ in range(20):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
    assert P.max_err(o, s, relative=True) <= F32_TOL


# ---- SSPRK3 (integrator.type 3 / 10, L808; S8(f) NEXT-2) ------------------------------------------------


@pytest.mark.parametrize("order,g,ko", [(1, 1, 0), (2, 2, 0), (3, 3, 0), (2, 3, 3), (1, 2, 2)])
@pytest.mark.parametrize("integrator", [3, 10])
def test_ssprk3_ragged_multibox_fp64(order, g, ko, integrator):
    P = _pair()
    n0 = (40, 24, 72)
    o, s = P.make_pair(n0, boxes=_ragged_boxes(), nghost=g, lap_order=order, h0=0.5, lam=0.7, a_mass=0.3,
                       friction=2.0, rk_dataflow="fused", integrator=integrator, ko_order=ko,
                       ko_strength=KO_EPS if ko else 0.0)
    P.init_smooth(o, s, n0, seed=17)
    eta, dt = 1.5, 0.1
    for _ in range(4):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
    assert P.max_err(o, s) <= F64_TOL
    _compare_tags(o, s, 0)


def test_ssprk3_is_not_rk4_on_the_gpu():
    P = _pair()
    n = 32
    out = []
    for integ in (4, 10):
        o, s = P.make_pair(n, nghost=2, lap_order=2, h0=0.5, integrator=integ)
        P.init_grf(o, s, n, 0.5, (81, 82))
        for q in range(3):
            s.rk_step(0.1, 1.0 + 0.1 * q)
        out.append(s.get_state(0, 0).cpu().numpy())
    assert np.abs(out[0] - out[1]).max() > 1e-7


def test_ssprk3_three_level_subcycled():
    """stage times t, t + dt, t + dt/2 in the coarse->fine ghost interpolation (L72), average-down"""
    P = _pair()
    n0 = 32
    _, boxes, _ = _ring_hierarchy(n0)
    o, s = P.make_pair(n0, boxes=boxes, n_levels=3, nghost=3, lap_order=2, h0=0.5, integrator=10)
    P.init_smooth(o, s, n0, seed=23)
    eta, dt = 2.0, 0.1
    for _ in range(2):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
    assert P.max_err(o, s) <= F64_TOL
    for l in range(3):
        _compare_tags(o, s, l)


def test_ssprk3_fp32():
    P = _pair()
    n = 64
    o, s = P.make_pair(n, nghost=2, lap_order=2, h0=0.125, dtype="f32", integrator=10)
    P.init_grf(o, s, n, 0.25, (71, 72))
    eta, dt = 1.0, 0.03125
    for _ in range(20):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
    assert P.max_err(o, s, relative=True) <= F32_TOL


def _bf4_boxes():
    # 44 x 36 x 40 domain, blocking factor 4: tile heights that are not multiples of the K1 tile (4, 12, 20, 24
    # rows), box corners that are not multiples of 32 (a tagging warp straddles two count blocks in x)
    return [
        (0, (0, 0, 0), (27, 11, 39)),
        (0, (28, 0, 0), (43, 11, 39)),
        (0, (0, 12, 0), (43, 35, 19)),
        (0, (0, 12, 20), (19, 35, 39)),
        (0, (20, 12, 20), (43, 31, 39)),
        (0, (20, 32, 20), (43, 35, 39)),
    ]


@pytest.mark.parametrize("order,g", [(1, 1), (2, 2), (2, 3), (3, 3)])
@pytest.mark.parametrize("flow", ["lean", "fused"])
def test_ragged_blocking_factor_4(order, g, flow):
    P = _pair()
    n0 = (44, 36, 40)
    o, s = P.make_pair(n0, boxes=_bf4_boxes(), nghost=g, blocking_factor=4, lap_order=order, h0=0.5, lam=1.0,
                       rk_dataflow=flow)
    P.init_smooth(o, s, n0, seed=12)
    eta, dt = 1.2, 0.1
    for _ in range(3):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
    assert P.max_err(o, s) <= F64_TOL
    _compare_tags(o, s, 0)


def test_blocking_factor_2_rows_of_one_warp_straddle_two_count_blocks():
    # box 2 starts at y = 30: the four rows of a tagging warp (30..33) fall into two 32-blocks
    P = _pair()
    n0 = (34, 38, 36)
    boxes = [(0, (0, 0, 0), (33, 29, 35)), (0, (0, 30, 0), (17, 37, 35)), (0, (18, 30, 0), (33, 37, 35))]
    o, s = P.make_pair(n0, boxes=boxes, nghost=1, blocking_factor=2, lap_order=1, h0=0.5, lam=1.0, rk_dataflow="fused")
    P.init_smooth(o, s, n0, seed=13)
    eta, dt = 1.0, 0.1
    for _ in range(3):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
    assert P.max_err(o, s) <= F64_TOL
    _compare_tags(o, s, 0)


def test_eta_fixed_minkowski_variant():
    P = _pair()
    o, s = P.make_pair(16, nghost=2, lap_order=2, h0=0.25, eta_fixed=True)
    P.init_smooth(o, s, 16, seed=5)
    for q in range(3):
        o.rk_step(0.05, 2.0)
        s.rk_step(0.05, 2.0)
    assert P.max_err(o, s) <= F64_TOL


@pytest.mark.parametrize("order,g", [(1, 1), (2, 2), (3, 3)])
def test_fp32_relative_error(order, g):
    P = _pair()
    n = 64
    o, s = P.make_pair(n, nghost=g, lap_order=order, h0=0.125, dtype="f32")
    P.init_grf(o, s, n, 0.25, (71, 72))
    eta, dt = 1.0, 0.03125
    for _ in range(20):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
    assert P.max_err(o, s, relative=True) <= F32_TOL
    # tags on the same (fp32-representable) state are bit-exact
    assert _compare_tags(o, s, 0) > 0


# ---- ghost fill ------------------------------------------------------------------------------------

@pytest.mark.parametrize("g", [1, 2, 3])
def test_ghost_fill_two_levels_matches_oracle_bitwise(g):
    """Periodic wrap, same-level copy and coarse->fine trilinear interpolation (no time interpolation yet:
    the coarse level has not stepped).  Same arithmetic order on both sides -> identical bits."""
    P = _pair()
    n0 = 32
    boxes = P.two_level_boxes(n0)
    o, s = P.make_pair(n0, boxes=boxes, n_levels=2, nghost=g, lap_order=1, h0=1.0)
    P.init_smooth(o, s, n0, seed=3)
    for l in (0, 1):
        o.fill_ghosts(l, 0.0)
        s.fill_ghosts(l, 0.0)
    s.synchronize()
    for ib in range(len(boxes)):
        for c in range(4):
            a = o.get_raw(ib, c)
            b = s.get_ghosted(ib, c).cpu().numpy()
            assert np.array_equal(a, b), (ib, c)


def test_ghost_fill_time_interpolation():
    """After a coarse step the fine ghosts at an intermediate time are (1-alpha) old + alpha new (L72)."""
    P = _pair()
    n0 = 32
    boxes = P.two_level_boxes(n0)
    o, s = P.make_pair(n0, boxes=boxes, n_levels=2, nghost=2, lap_order=2, h0=0.5)
    P.init_smooth(o, s, n0, seed=4)
    o.rk_step(0.1, 1.0)
    s.rk_step(0.1, 1.0)
    for time in (1.0, 1.025, 1.05, 1.1):
        o.fill_ghosts(1, time)
        s.fill_ghosts(1, time)
        for ib in s.level_boxes(1):
            for c in range(4):
                a = o.get_raw(ib, c)
                b = s.get_ghosted(ib, c).cpu().numpy()
                assert np.abs(a - b).max() <= F64_TOL, (time, ib, c)
    s.synchronize()


# ---- quartic polynomial conservative coarse->fine interpolation (amr.interpolation_type 4, L780; S8(f) NEXT-3) -----


@pytest.mark.parametrize("g", [1, 2, 3])
def test_quartic_ghost_fill_two_levels_matches_oracle_bitwise(g):
    """5^3 parents per ghost cell.  g = 1: per-cell entries (fast: window inside one coarse box; slow: periodic /
    multi-box), same summation order and individually rounded operations on both sides -> identical bits.  g >= 2: by
    coarse parent through the coarse boxes' ghost cells, evaluated separably (x, y, z passes): equal
    to the oracle's direct triple sum up to rounding order -> a few ulp of values of order 1, far inside the 1e-11 bar
    of BASELINE.json's north_star."""
    P = _pair()
    n0 = 32
    boxes = P.two_level_boxes(n0)
    o, s = P.make_pair(n0, boxes=boxes, n_levels=2, nghost=g, lap_order=1, h0=1.0, interp=4)
    P.init_smooth(o, s, n0, seed=3)
    for l in (0, 1):
        o.fill_ghosts(l, 0.0)
        s.fill_ghosts(l, 0.0)
    s.synchronize()
    for ib in range(len(boxes)):
        for c in range(4):
            a = o.get_raw(ib, c)
            b = s.get_ghosted(ib, c).cpu().numpy()
            if g == 1:
                assert np.array_equal(a, b), (ib, c)
            else:
                assert np.abs(a - b).max() <= 1e-14 * max(1.0, float(np.abs(a).max())), (ib, c)


def test_quartic_differs_from_trilinear_on_the_gpu():
    P = _pair()
    n0 = 32
    boxes = P.two_level_boxes(n0)
    out = []
    for interp in (0, 4):
        o, s = P.make_pair(n0, boxes=boxes, n_levels=2, nghost=2, lap_order=1, h0=1.0, interp=interp)
        P.init_smooth(o, s, n0, seed=3)
        s.fill_ghosts(1, 0.0)
        out.append(s.get_ghosted(1, 0).cpu().numpy())
    assert np.abs(out[0] - out[1]).max() > 1e-4


def test_quartic_ghost_fill_multibox_coarse_level_and_time_interpolation():
    """coarse level cut into 8^3 boxes: every 5-cell window straddles boxes (slow entries only); then alpha in (0, 1)"""
    P = _pair()
    n0 = 32
    boxes = [(0, lo, hi) for _, lo, hi in inputs.split_level0(n0, 8)] + P.two_level_boxes(n0)[1:]
    o, s = P.make_pair(n0, boxes=boxes, n_levels=2, nghost=3, lap_order=2, h0=0.5, interp=4)
    P.init_smooth(o, s, n0, seed=4)
    o.rk_step(0.1, 1.0)
    s.rk_step(0.1, 1.0)
    for time in (1.0, 1.025, 1.05, 1.1):
        o.fill_ghosts(1, time)
        s.fill_ghosts(1, time)
        for ib in s.level_boxes(1):
            for c in range(4):
                a = o.get_raw(ib, c)
                b = s.get_ghosted(ib, c).cpu().numpy()
                assert np.abs(a - b).max() <= F64_TOL, (time, ib, c)
    s.synchronize()


@pytest.mark.parametrize("flow,integrator", [("fused", 4), ("lean", 4), ("lean", 10)])
def test_quartic_three_level_subcycled(flow, integrator):
    P = _pair()
    n0 = 32
    rings, boxes, _ = _ring_hierarchy(n0)
    o, s = P.make_pair(n0, boxes=boxes, n_levels=3, nghost=3, lap_order=2, h0=0.25, rk_dataflow=flow,
                       integrator=integrator, interp=4)
    for ib, (l, lo, hi) in enumerate(boxes):
        re, im = inputs.ring_field(rings, l, lo, hi)
        P.set_both(o, s, ib, 0, re.numpy())
        P.set_both(o, s, ib, 1, im.numpy())
    eta, dt = 2.0, 0.0625
    for _ in range(2):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
    assert P.max_err(o, s) <= F64_TOL
    for l in range(3):
        _compare_tags(o, s, l)


def test_quartic_fp32_two_level():
    P = _pair()
    n0 = 32
    boxes = P.two_level_boxes(n0)
    o, s = P.make_pair(n0, boxes=boxes, n_levels=2, nghost=3, lap_order=2, h0=0.5, dtype="f32", interp=4)
    P.init_smooth(o, s, n0, seed=9, comps=(0, 1))
    eta, dt = 2.0, 0.1
    for _ in range(3):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
    assert P.max_err(o, s, relative=True) <= F32_TOL


# ---- average-down ------------------------------------------------------------------------------------

def test_average_down_matches_oracle_bitwise():
    P = _pair()
    n0 = 32
    boxes = P.two_level_boxes(n0)
    o, s = P.make_pair(n0, boxes=boxes, n_levels=2, nghost=1, h0=1.0)
    P.init_smooth(o, s, n0, seed=8)
    o.average_down(1)
    s.average_down(1)
    s.synchronize()
    for c in range(4):
        a = o.get_state(0, c)
        b = s.get_state(0, c).cpu().numpy()
        assert np.array_equal(a, b)
    # something was actually overwritten
    assert not np.array_equal(o.get_state(0, 0), P.smooth_field(((0, 0, 0), (31, 31, 31)), 0, (32,) * 3, 80))


# ---- AMR with subcycling ---------------------------------------------------------------------------------

# ---- truncation-error tags fused into the synchronisation (S8(f) NEXT-1) ----------------------------------

def _tee_compare(o, s, level):
    ot, oc = o.tee_tags(level)
    gt, gc = s._tee[level]
    s.synchronize()
    for a, b in zip(ot, s.split_tags(level, gt)):
        assert np.array_equal(a, b.cpu().numpy())
    assert np.array_equal(oc.astype(np.int64), gc.cpu().numpy().astype(np.int64))
    return sum(int((a != 0).sum()) for a in ot)


def test_tee_tags_at_explicit_average_down_match_oracle_bitwise():
    """Same input state on both sides (independent smooth fields on the two levels, so that Delta is O(1e-2) and the
    thresholds cut through its distribution): tags, 32^3 counts and the synchronised coarse state are bit-exact."""
    P = _pair()
    n0 = 32
    boxes = P.two_level_boxes(n0)
    o, s = P.make_pair(n0, boxes=boxes, n_levels=2, nghost=2, lap_order=2, h0=1.0)
    P.init_smooth(o, s, n0, seed=21)
    eps = (0.004, 0.009, 0.006, 0.012)  # psi1, psi2, Pi1, Pi2 (L781-782)
    o.tee_enable(1, *eps)
    s.tee_enable(1, *eps)
    o.average_down(1)
    s.average_down(1)
    ntag = _tee_compare(o, s, 1)
    bits = np.concatenate([t.ravel() for t in o.tee_tags(1)[0]])
    assert all(0 < int(((bits >> c) & 1).sum()) < bits.size for c in range(4))  # every component's bit is exercised
    ncell = sum(int(np.prod(o.box_shape(ib))) for ib in o.level_boxes(1))
    assert 0 < ntag < ncell
    assert P.max_err(o, s) == 0.0
    # second synchronisation: coarse already equals the mean -> Delta = 0, nothing tagged on either side
    o.average_down(1)
    s.average_down(1)
    assert _tee_compare(o, s, 1) == 0


def test_tee_tags_inside_rk_step_three_levels():
    """TEE enabled on levels 1 and 2 of a ring hierarchy: after a coarse step the buffers hold the tags of each
    level's LAST synchronisation.  Free-running states agree to <= 1e-11, so the comparison is restricted to cells
    whose Delta is not within 1e-9 of the threshold: run both sides with eps*(1 -+ 1e-6) on the oracle and require
    oracle(eps+) <= gpu(eps) <= oracle(eps-) cell by cell."""
    P = _pair()
    n0 = 32
    rings, boxes, _ = _ring_hierarchy(n0)
    kw = dict(boxes=boxes, n_levels=3, nghost=3, lap_order=2, h0=0.25, lam=1.0)
    eps = 2e-4
    runs = []
    for scale in (1.0 + 1e-6, 1.0 - 1e-6):
        o, s = P.make_pair(n0, **kw)
        for ib, (l, lo, hi) in enumerate(boxes):
            re, im = inputs.ring_field(rings, l, lo, hi)
            P.set_both(o, s, ib, 0, re.numpy())
            P.set_both(o, s, ib, 1, im.numpy())
        for l in (1, 2):
            o.tee_enable(l, eps * scale, eps * scale, 4 * eps * scale, 4 * eps * scale)
            s.tee_enable(l, eps, eps, 4 * eps, 4 * eps)
        o.rk_step(0.0625, 2.0)
        s.rk_step(0.0625, 2.0)
        s.synchronize()
        assert P.max_err(o, s) <= F64_TOL
        runs.append((o, s))
    (o_hi, s), (o_lo, _) = runs
    total = 0
    for l in (1, 2):
        t_hi, _ = o_hi.tee_tags(l)
        t_lo, _ = o_lo.tee_tags(l)
        g = [b.cpu().numpy() for b in s.split_tags(l, s._tee[l][0])]
        for a, b, c in zip(t_hi, g, t_lo):
            assert np.all((a & ~b) == 0) and np.all((b & ~c) == 0)
            total += int((b != 0).sum())
    assert total > 0


@pytest.mark.parametrize("flow", ["lean", "classic", "fused", "fused3"])
@pytest.mark.parametrize("order", [2, 3])
def test_two_level_subcycled_steps(flow, order):
    P = _pair()
    n0 = 32
    boxes = P.two_level_boxes(n0)
    o, s = P.make_pair(n0, boxes=boxes, n_levels=2, nghost=3, lap_order=order, h0=0.5, rk_dataflow=flow)
    P.init_smooth(o, s, n0, seed=9, comps=(0, 1))
    eta, dt = 2.0, 0.1
    for _ in range(3):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
    assert P.max_err(o, s) <= F64_TOL
    for l in (0, 1):
        _compare_tags(o, s, l)


def _ring_hierarchy(n0=32, box=16, n_levels=3):
    rings = inputs.make_rings(n0, 2, 5.0, 9.0, 1.5, seed=77)
    boxes, cover = inputs.amr_boxes_for_rings(rings, n_levels=n_levels, box=box, r1=3.0, r2=1.0, blocking_factor=8)
    return rings, boxes, cover


def test_three_level_ring_hierarchy_like_c5():
    """Small version of BASELINE.json config 5: vortex rings, 3 levels, boxes of one size placed around the
    ring curves, 13-point stencil, 3 ghost cells, subcycling 1/2/4, average-down after every fine pair."""
    P = _pair()
    n0 = 32
    rings, boxes, cover = _ring_hierarchy(n0)
    assert 0 < cover[2] < cover[1] < 1
    o, s = P.make_pair(n0, boxes=boxes, n_levels=3, nghost=3, lap_order=2, h0=0.25)
    for ib, (l, lo, hi) in enumerate(boxes):
        re, im = inputs.ring_field(rings, l, lo, hi)
        P.set_both(o, s, ib, 0, re.numpy())
        P.set_both(o, s, ib, 1, im.numpy())
    eta, dt = 2.0, 0.0625
    for _ in range(2):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
    s.synchronize()
    assert P.max_err(o, s) <= F64_TOL
    total = 0
    for l in range(3):
        total += _compare_tags(o, s, l)
    assert total > 0


def test_fully_covered_level1_equals_uniform_fine_run_on_gpu():
    """Bookkeeping identity: a hierarchy whose level 1 covers the whole domain reproduces on
    level 1 the single-level 2N run with dt/2, bit for bit -- GPU against GPU, no oracle involved."""
    from paper_2404_02950_b200.sledge import Sledge
    P = _pair()
    n0, g = 16, 2
    boxes = [(0, (0, 0, 0), (15, 15, 15)), (1, (0, 0, 0), (31, 31, 31))]
    two = Sledge(n0, boxes=boxes, n_levels=2, nghost=g, lap_order=2, h0=0.5)
    one = Sledge(2 * n0, nghost=g, lap_order=2, h0=0.25)
    for c in range(2):
        fine = torch.from_numpy(P.smooth_field(((0, 0, 0), (31, 31, 31)), 1, (n0,) * 3, 40 + c)).cuda().contiguous()
        coarse = torch.nn.functional.avg_pool3d(fine[None, None], 2)[0, 0].contiguous()
        two.set_state(0, c, coarse)
        two.set_state(1, c, fine)
        one.set_state(0, c, fine)
    eta, dt = 1.0, 0.1
    two.rk_step(dt, eta)
    one.rk_step(dt / 2, eta)
    one.rk_step(dt / 2, eta + dt / 2)
    for c in range(4):
        assert torch.equal(two.get_state(1, c), one.get_state(0, c))
    two.synchronize()
    one.synchronize()


# ---- hooks and error paths -----------------------------------------------------------------------------

def test_rk_stage_hook_equals_rk_step():
    from paper_2404_02950_b200.sledge import Sledge
    P = _pair()
    a = Sledge(16, nghost=1, lap_order=1, h0=0.5)
    b = Sledge(16, nghost=1, lap_order=1, h0=0.5)
    for c in range(4):
        f = torch.from_numpy(P.smooth_field(((0, 0, 0), (15, 15, 15)), 0, (16,) * 3, 60 + c)).cuda().contiguous()
        a.set_state(0, c, f)
        b.set_state(0, c, f)
    a.rk_step(0.05, 1.0)
    for st in range(4):
        b.rk_stage(0, st, 0.05, 1.0)
    for c in range(4):
        assert torch.equal(a.get_state(0, c), b.get_state(0, c))
    assert a.launch_count() > 0


def test_host_buffer_roundtrip_and_profile_counters():
    from paper_2404_02950_b200.sledge import Sledge, KIND_STAGE, KIND_GHOST
    s = Sledge(16, nghost=1)
    src = torch.randn(16, 16, 16, dtype=torch.float64).pin_memory()
    dst = torch.empty(16, 16, 16, dtype=torch.float64).pin_memory()
    s.set_state_host(0, 1, src)
    s.get_state_host(0, 1, dst)
    s.synchronize()
    assert torch.equal(src, dst)
    s.profile_enable(True)
    s.rk_step(0.01, 1.0)
    n, ms = s.profile_read(KIND_STAGE)
    assert n == 4 and ms > 0
    n, ms = s.profile_read(KIND_GHOST)
    assert n == 4
    s.profile_enable(False)


def test_create_rejects_bad_arena():
    import ctypes as C
    from paper_2404_02950_b200 import sledge as S
    p, arr, boxes, _ = S._marshal(16, None, 1, 1, 8, "f64", 1, 1.0, 1.0, 0.0, 0.0, False, "lean")
    h = C.c_void_p()
    buf = torch.empty(1024, dtype=torch.uint8, device="cuda")
    rc = S.lib().sledge_create(C.byref(h), C.byref(p), arr, 1, buf.data_ptr(), 1024, None)
    assert rc == -2 and b"arena" in S.lib().sledge_last_error(None)


def test_c1_run_as_one_cuda_graph_replays_bit_for_bit():
    """C1 additionally under CUDA Graph replay.  The stabilised C1 run (dt = 0.0625) captured into one
    graph (restore + 10 x (rk_step + tag_strings)) reproduces the eager run bit for bit, fields and tags."""
    import bench
    cfg = inputs.CONFIGS["C1"]
    for flow in ("fused", "lean"):
        r = bench.graph_leg(cfg, "cuda:0", flow, replays=3, dt=0.0625)
        assert r["replay_equals_eager_bitwise"], flow
        assert r["launches_per_run"] >= 4 + 3 * cfg.steps
        assert r["ms_per_step_graph"] > 0

