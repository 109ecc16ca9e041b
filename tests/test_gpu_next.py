"""GPU parity of the rows added in round 2: gravitational-wave auxiliary fields (NEXT-4), the
user-defined Runge-Kutta-Nystrom integrator (NEXT-2) and the level-0 shadow level (NEXT-1), each against the CPU oracle
on the same seeded inputs.  Bars as everywhere: fp64 <= 1e-11 absolute, fp32 <= 2e-5 relative, tags bit-exact where
the decision is not within rounding of the threshold."""
import numpy as np
import pytest
import torch

from paper_2404_02950_b200 import inputs

pytestmark = pytest.mark.gpu

F64_TOL = 1e-11
F32_TOL = 2e-5

RKN4 = dict(nodes=[0.0, 0.5, 1.0], weights_b=[1 / 6, 4 / 6, 1 / 6], weights_bar_b=[1 / 6, 1 / 3, 0.0],
            tableau=[0.0, 1 / 8, 0.0, 0.0, 0.5, 0.0])
RK4_AS_RKN = dict(nodes=[0.0, 0.5, 0.5, 1.0], weights_b=[1 / 6, 1 / 3, 1 / 3, 1 / 6], weights_bar_b=[1 / 6, 1 / 6, 1 / 6, 0.0],
                  tableau=[0.0, 0.0, 0.0, 0.25, 0.0, 0.0, 0.0, 0.5, 0.0, 0.0])
# a five-stage tableau with every entry non-zero (consistency is irrelevant here: both sides must compute the same thing)
RKN5_DENSE = dict(nodes=[0.0, 0.2, 0.5, 0.7, 1.0], weights_b=[0.1, 0.3, 0.2, 0.3, 0.1], weights_bar_b=[0.1, 0.15, 0.1, 0.1, 0.05],
                  tableau=[0.0, 0.02, 0.0, 0.05, 0.075, 0.0, 0.06, 0.085, 0.1, 0.0, 0.1, 0.12, 0.14, 0.14, 0.0])


def _pair():
    import _pair as P
    return P


def _ring_hierarchy(n0=32, box=16, n_levels=3):
    """the three-level hierarchy of test_gpu_parity.py: boxes of 16^3 around two seeded vortex rings"""
    rings = inputs.make_rings(n0, 2, 5.0, 9.0, 1.5, seed=77)
    boxes, _ = inputs.amr_boxes_for_rings(rings, n_levels=n_levels, box=box, r1=3.0, r2=1.0, blocking_factor=8)
    return boxes


def _ragged_boxes():
    """40 x 24 x 72 periodic level 0 in boxes of different shapes: partial K1 tiles in x and y, several boxes in z."""
    return [(0, (0, 0, 0), (23, 23, 39)), (0, (24, 0, 0), (39, 23, 39)), (0, (0, 0, 40), (39, 7, 71)),
            (0, (0, 8, 40), (39, 23, 71))]


# ---- NEXT-4: gravitational-wave auxiliary fields (Eq.16) ------------------------------------------------

@pytest.mark.parametrize("order,g", [(1, 1), (2, 2), (2, 3), (3, 3)])
def test_gw_ragged_multibox_fp64(order, g):
    P = _pair()
    n0 = (40, 24, 72)
    o, s = P.make_pair(n0, boxes=_ragged_boxes(), nghost=g, blocking_factor=8, lap_order=order, h0=0.5, lam=0.7,
                       a_mass=0.3, friction=2.0, gw=True, gw_coupling=0.8, gw_friction=3.0)
    P.init_smooth(o, s, n0, 5, comps=range(16), amp=0.5)
    eta, dt = 1.5, 0.05
    for _ in range(3):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
    s.synchronize()
    assert P.max_err(o, s, comps=range(16)) <= F64_TOL
    # the auxiliary fields must actually have been sourced
    assert max(float(np.abs(o.get_state(0, c)).max()) for c in range(4, 10)) > 1e-3


def test_gw_classic_dataflow_and_fp32():
    P = _pair()
    n0 = (40, 24, 72)
    o, s = P.make_pair(n0, boxes=_ragged_boxes(), nghost=2, lap_order=2, h0=0.5, lam=1.0, gw=True, gw_coupling=1.0,
                       rk_dataflow="classic")
    P.init_smooth(o, s, n0, 6, comps=range(16), amp=0.5)
    o32, s32 = P.make_pair(n0, boxes=_ragged_boxes(), nghost=2, lap_order=2, h0=0.5, lam=1.0, gw=True, gw_coupling=1.0,
                           dtype="f32", rk_dataflow="fused")  # fused is not applicable with gw: staged sweeps run
    P.init_smooth(o32, s32, n0, 6, comps=range(16), amp=0.5)
    eta, dt = 1.0, 0.05
    for _ in range(3):
        for a in (o, s, o32, s32):
            a.rk_step(dt, eta)
        eta += dt
    assert P.max_err(o, s, comps=range(16)) <= F64_TOL
    assert P.max_err(o32, s32, comps=range(16), relative=True) <= F32_TOL


def test_gw_three_levels_subcycled_with_average_down():
    """16 components through the whole AMR path: per-stage ghost fills (same-level + trilinear coarse->fine, linear
    in time), subcycling and average-down."""
    P = _pair()
    n0 = 32
    boxes = _ring_hierarchy(n0)
    o, s = P.make_pair(n0, boxes=boxes, n_levels=3, nghost=2, lap_order=2, h0=0.5, lam=1.0, gw=True, gw_coupling=0.5,
                       gw_friction=1.0)
    P.init_smooth(o, s, n0, 7, comps=range(16), amp=0.5)
    for l in (2, 1):
        o.average_down(l)
        s.average_down(l)
    eta, dt = 1.0, 0.1
    for _ in range(2):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
    assert P.max_err(o, s, comps=range(16)) <= F64_TOL
    # ghosts of the auxiliary fields after an explicit fill
    o.fill_ghosts(1, eta)
    s.fill_ghosts(1, eta)
    for ib in s.level_boxes(1):
        for c in (4, 9, 15):
            a = o.get_raw(ib, c)
            b = s.get_ghosted(ib, c).cpu().numpy()
            assert np.abs(a - b).max() <= F64_TOL


# ---- NEXT-2: user-defined Runge-Kutta-Nystrom tableau (integrator.type 20) ------------------------------

@pytest.mark.parametrize("tab", [RKN4, RK4_AS_RKN, RKN5_DENSE], ids=["nystrom4", "rk4-as-rkn", "dense5"])
@pytest.mark.parametrize("order,g", [(1, 1), (2, 2), (3, 3)])
def test_rkn_ragged_multibox_fp64(tab, order, g):
    P = _pair()
    n0 = (40, 24, 72)
    o, s = P.make_pair(n0, boxes=_ragged_boxes(), nghost=g, lap_order=order, h0=0.5, lam=0.7, a_mass=0.3,
                       integrator=20, rkn=tab)
    P.init_smooth(o, s, n0, 8, amp=0.5)
    eta, dt = 1.5, 0.05
    for _ in range(4):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
    assert P.max_err(o, s) <= F64_TOL


@pytest.mark.parametrize("interp", [0, 4])
def test_rkn_three_levels_subcycled_and_fp32(interp):
    P = _pair()
    n0 = 32
    boxes = _ring_hierarchy(n0)
    kw = dict(boxes=boxes, n_levels=3, nghost=2, lap_order=2, h0=0.5, lam=1.0, integrator=20, rkn=RKN4, interp=interp)
    o, s = P.make_pair(n0, **kw)
    o32, s32 = P.make_pair(n0, dtype="f32", **kw)
    for a, b in ((o, s), (o32, s32)):
        P.init_smooth(a, b, n0, 9, amp=0.5)
        for l in (2, 1):
            a.average_down(l)
            b.average_down(l)
    eta, dt = 1.0, 0.1
    for _ in range(3):
        for a in (o, s, o32, s32):
            a.rk_step(dt, eta)
        eta += dt
    assert P.max_err(o, s) <= F64_TOL
    assert P.max_err(o32, s32, relative=True) <= F32_TOL


# ---- NEXT-1: the shadow level of level 0 (L98) ------------------------------------------------------------

@pytest.mark.parametrize("flow,nlev", [("fused", 1), ("lean", 1), ("fused", 2)])
def test_shadow_level_tags_of_level0(flow, nlev):
    """sledge_shadow_tee against the oracle: same final state (two coarse steps), and the same level-0 tags wherever
    the oracle's decision does not change when its thresholds move by 1e-6 relative (the two sides' Delta differ by
    rounding, 1e-13, against thresholds of 1e-4 .. 1e-2)."""
    P = _pair()
    n0 = 32
    boxes = inputs.split_level0(n0, 16) if nlev == 1 else P.two_level_boxes(n0, 8)
    kw = dict(boxes=boxes, n_levels=nlev, nghost=2, lap_order=2, h0=0.5, lam=1.0)
    eta, dt = 1.0, 0.1

    def fresh():
        o, s = P.make_pair(n0, rk_dataflow=flow, shadow_level=True, **kw)
        P.init_smooth(o, s, n0, 3, amp=0.6)
        if nlev == 2:
            o.average_down(1)
            s.average_down(1)
        return o, s

    # thresholds at the median of the level-0 Delta of each component: found by bisection on the oracle
    eps = []
    for c in range(4):
        lo, hi = 0.0, 1.0
        for _ in range(16):
            mid = 0.5 * (lo + hi)
            o, _ = fresh()
            e = [np.inf] * 4
            e[c] = mid
            t, _ = o.shadow_tee(dt, eta, *e)
            frac = np.mean([float((a != 0).mean()) for a in t])
            if frac > 0.5:
                lo = mid
            else:
                hi = mid
        eps.append(hi)
    assert all(1e-9 < e < 1.0 for e in eps), eps
    o, s = fresh()
    ot, oc = o.shadow_tee(dt, eta, *eps)
    gt, gc = s.shadow_tee(dt, eta, *eps)
    s.synchronize()
    assert P.max_err(o, s) <= F64_TOL
    lo_t = fresh()[0].shadow_tee(dt, eta, *[e * (1 - 1e-6) for e in eps])[0]
    hi_t = fresh()[0].shadow_tee(dt, eta, *[e * (1 + 1e-6) for e in eps])[0]
    gts = s.split_tags(0, gt)
    n_sure = n_all = n_tagged = 0
    for a, b, l_, h_ in zip(ot, gts, lo_t, hi_t):
        sure = l_ == h_
        n_sure += int(sure.sum())
        n_all += sure.size
        n_tagged += int((a != 0).sum())
        assert np.array_equal(a[sure], b.cpu().numpy()[sure])
    assert n_sure > 0.999 * n_all and 0.2 * n_all < n_tagged < n_all
    # counts: equal up to the cells that are not sure (8 per parent)
    assert np.abs(oc.astype(np.int64) - gc.cpu().numpy().astype(np.int64)).sum() <= 8 * (n_all - n_sure)
    # a context without the shadow level refuses
    _, s2 = P.make_pair(n0, **kw)
    with pytest.raises(Exception):
        s2.shadow_tee(dt, eta, 1.0, 1.0)


# ---- bookkeeping: which data-flow a level runs ---------------------------------------------------------------

def test_level_dataflow_reports_launches_and_words():
    import os
    from paper_2404_02950_b200.sledge import Sledge
    if any(os.environ.get(k) == "0" for k in ("SLEDGE_K1_TMA", "SLEDGE_K2_PATCHES", "SLEDGE_FINE_FUSED")):
        pytest.skip("a diagnostic switch turns the fused sweeps of the finer levels off")
    n0 = 32
    boxes = _ring_hierarchy(n0)
    kw = dict(boxes=boxes, n_levels=3, nghost=3, lap_order=2, h0=0.5)
    s = Sledge(n0, rk_dataflow="fused", **kw)
    assert [s.level_dataflow(l) for l in range(3)] == [(2, 20)] * 3      # FUSED on every level (velocity ghosts)
    s = Sledge(n0, rk_dataflow="fused", interp=4, **kw)
    assert [s.level_dataflow(l) for l in range(3)] == [(2, 20)] * 3      # quartic by coarse parent
    s = Sledge(n0, rk_dataflow="lean", **kw)
    assert s.level_dataflow(1) == (4, 52)
    s = Sledge(n0, rk_dataflow="classic", **kw)
    assert s.level_dataflow(2) == (4, 64)
    s = Sledge(n0, rk_dataflow="fused", integrator=10, **kw)
    assert s.level_dataflow(0) == (3, 32)
    s = Sledge(n0, rk_dataflow="fused", integrator=20, rkn=RKN4, **kw)
    assert s.level_dataflow(0) == (3, 8 + 12 + 14)
    s = Sledge(n0, rk_dataflow="fused", gw=True, **kw)
    assert s.level_dataflow(1) == (8, 52 + 164)
    s = Sledge(n0, rk_dataflow="fused", ko_order=2, ko_strength=0.01, **kw)
    assert s.level_dataflow(0) == (4, 52)


def test_fused_on_fine_levels_matches_the_oracle_with_moving_coarse_data():
    """The velocity ghosts (K2) must make the two-stage sweeps of a fine level see the coarse state at t + dt/2 and
    t + dt: a hierarchy with large coarse time derivatives (Pi of order 1), five coarse steps, friction and mass on."""
    P = _pair()
    n0 = 32
    boxes = _ring_hierarchy(n0)
    for interp in (0, 4):
        o, s = P.make_pair(n0, boxes=boxes, n_levels=3, nghost=3, lap_order=2, h0=0.5, lam=0.7, a_mass=0.3,
                           friction=2.0, rk_dataflow="fused", interp=interp)
        P.init_smooth(o, s, n0, 13, amp=0.8)
        for l in (2, 1):
            o.average_down(l)
            s.average_down(l)
        eta, dt = 1.5, 0.1
        for _ in range(5):
            o.rk_step(dt, eta)
            s.rk_step(dt, eta)
            eta += dt
        assert P.max_err(o, s) <= F64_TOL


def test_fused_on_fine_levels_fp32():
    P = _pair()
    n0 = 32
    boxes = _ring_hierarchy(n0)
    o, s = P.make_pair(n0, boxes=boxes, n_levels=3, nghost=3, lap_order=2, h0=0.5, lam=1.0, rk_dataflow="fused", dtype="f32")
    P.init_smooth(o, s, n0, 14, amp=0.8)
    for l in (2, 1):
        o.average_down(l)
        s.average_down(l)
    eta, dt = 1.5, 0.1
    for _ in range(4):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
    assert P.max_err(o, s, relative=True) <= F32_TOL


def test_host_buffer_copies_are_pipelined_but_ordered():
    """sledge_set_state_host / sledge_get_state_host run on the library's own copy streams through two staging slots
    per direction: many back-to-back copies of different boxes and components, a step in between, and a second round
    that overwrites the first must behave exactly like the device-buffer calls."""
    from paper_2404_02950_b200.sledge import Sledge
    n0 = (40, 24, 72)
    boxes = _ragged_boxes()
    kw = dict(boxes=boxes, nghost=2, lap_order=2, h0=0.5, lam=1.0, rk_dataflow="fused")
    a, b = Sledge(n0, **kw), Sledge(n0, **kw)
    rng = np.random.default_rng(5)
    for rnd in range(2):
        host = {}
        for ib in range(len(boxes)):
            for c in range(4):
                t = torch.from_numpy(rng.normal(size=a.box_shape(ib)) * (0.5 if c < 2 else 0.1)).pin_memory()
                host[(ib, c)] = t
                a.set_state_host(ib, c, t)
                b.set_state(ib, c, t.cuda())
        a.rk_step(0.05, 1.0)
        b.rk_step(0.05, 1.0)
        outs = {k: torch.empty_like(v).pin_memory() for k, v in host.items()}
        for (ib, c), o in outs.items():
            a.get_state_host(ib, c, o)
        a.synchronize()
        for (ib, c), o in outs.items():
            assert torch.equal(o, b.get_state(ib, c).cpu()), (rnd, ib, c)
    # join: work enqueued on the context stream afterwards sees the downloads done
    o2 = torch.empty(a.box_shape(0), dtype=torch.float64).pin_memory()
    a.get_state_host(0, 0, o2)
    a.host_copies_join()
    torch.cuda.current_stream().synchronize()
    assert torch.equal(o2, b.get_state(0, 0).cpu())


# ---- patches and velocity ghosts on other shapes: small blocking factors, non-cubic domains ------------------------

@pytest.mark.parametrize("bf,g,order", [(4, 2, 2), (4, 3, 3), (2, 1, 1), (8, 3, 2)])
@pytest.mark.parametrize("interp", [0, 4])
def test_fused_multilevel_small_blocking_factors_and_noncubic_domain(bf, g, order, interp):
    """Level 1 made of boxes of different shapes on a 24 x 16 x 32 periodic domain, level 2 inside it; the fills before
    the sweeps go by patch (bf x bf x R pieces), the sweeps are FUSED on every level where the library allows it."""
    P = _pair()
    if interp == 4 and (g + 1) // 2 + 2 > bf // 2:
        pytest.skip("quartic window leaves the nesting gap for this blocking factor (L70)")
    n0 = (24, 16, 32)
    m = max(bf, 4)  # fine boxes are multiples of 2 bf so that level 2 can nest with a gap of one blocking factor
    boxes = [(0, (0, 0, 0), (n0[0] - 1, n0[1] - 1, n0[2] - 1))]
    # level 1 (index space 48 x 32 x 64): an L of three boxes around the middle, wrapping around the periodic z seam
    boxes += [(1, (8, 8, 56), (8 + 4 * m - 1, 8 + 2 * m - 1, 63)), (1, (8, 8, 0), (8 + 4 * m - 1, 8 + 2 * m - 1, 2 * m - 1)),
              (1, (8, 8 + 2 * m, 0), (8 + 2 * m - 1, 8 + 4 * m - 1 if 8 + 4 * m <= 32 else 31, 2 * m - 1))]
    boxes = [b for b in boxes if all(b[2][d] < (n0[d] << b[0]) for d in range(3))]
    nlev = 2
    if bf <= 4:  # level 2 (index space 96 x 64 x 128) inside the first level-1 boxes, gap >= bf fine cells
        boxes.append((2, (24, 20, 4), (24 + 2 * bf - 1, 20 + 2 * bf - 1, 4 + 2 * bf - 1)))
        nlev = 3
    from paper_2404_02950_b200 import sledge as S
    try:
        S.sledge_arena_bytes(n0, boxes=boxes, n_levels=nlev, nghost=g, blocking_factor=bf, lap_order=order, interp=interp)
    except S.SledgeError as e:
        pytest.skip(f"hierarchy not valid for this case: {e}")
    o, s = P.make_pair(n0, boxes=boxes, n_levels=nlev, nghost=g, blocking_factor=bf, lap_order=order, h0=0.5, lam=0.8,
                       a_mass=0.2, rk_dataflow="fused", interp=interp)
    P.init_smooth(o, s, n0, 21, amp=0.7)
    for l in range(nlev - 1, 0, -1):
        o.average_down(l)
        s.average_down(l)
    eta, dt = 1.2, 0.08
    for _ in range(3):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
    assert P.max_err(o, s) <= F64_TOL
    for l in range(nlev):
        P.upload_oracle_state(o, s) if l == 0 else None
        ot, oc = o.tag_strings(l)
        gt, gc = s.tag_strings(l)
        s.synchronize()
        for a, b in zip(ot, s.split_tags(l, gt)):
            assert np.array_equal(a, b.cpu().numpy())
        assert np.array_equal(oc.astype(np.int64), gc.cpu().numpy().astype(np.int64))


def test_shadow_level_with_auxiliary_fields():
    P = _pair()
    n0 = 32
    boxes = inputs.split_level0(n0, 16)
    o, s = P.make_pair(n0, boxes=boxes, nghost=2, lap_order=2, h0=0.5, lam=1.0, gw=True, gw_coupling=0.7, shadow_level=True)
    P.init_smooth(o, s, n0, 4, comps=range(16), amp=0.5)
    o.shadow_tee(0.1, 1.0, 1e-3, 1e-3)
    s.shadow_tee(0.1, 1.0, 1e-3, 1e-3)
    s.synchronize()
    assert P.max_err(o, s, comps=range(16)) <= F64_TOL


# ---- storage boxes: the caller's boxes coalesced into larger rectangles --------------------------------------

def _run_hierarchy(monkeypatch, coalesce, dtype, flow, interp, ragged):
    """three coarse steps + tags + truncation-error tags on a multi-box hierarchy; returns everything a caller can see"""
    from paper_2404_02950_b200.sledge import Sledge
    P = _pair()
    if coalesce is None:
        monkeypatch.delenv("SLEDGE_COALESCE", raising=False)
    else:
        monkeypatch.setenv("SLEDGE_COALESCE", coalesce)
    if ragged:
        n0, boxes, nl = (40, 24, 72), _ragged_boxes(), 1
    else:
        n0, boxes, nl = 32, _ring_hierarchy(32), 3
    s = Sledge(n0, boxes=boxes, n_levels=nl, nghost=3, lap_order=2, h0=0.5, lam=0.7, a_mass=0.3, friction=2.0,
               rk_dataflow=flow, interp=interp, dtype=dtype)
    n03 = (n0,) * 3 if isinstance(n0, int) else n0
    for ib, (lvl, lo, hi) in enumerate(boxes):
        for c in range(4):
            f = P.smooth_field((lo, hi), lvl, n03, 31 + c, amp=0.8)
            s.set_state(ib, c, torch.from_numpy(np.ascontiguousarray(f)).to(s.tdtype).cuda().contiguous())
    for l in range(nl - 1, 0, -1):
        s.average_down(l)
    out = {"storage": [s.level_storage(l) for l in range(nl)]}
    tee = None
    if nl > 1:
        tee = s.tee_enable(1, 1e-4, 1e-4, 1e-3, 1e-3)
    eta, dt = 1.5, 0.1
    for _ in range(3):
        s.rk_step(dt, eta)
        eta += dt
    out["state"] = [s.get_state(ib, c).cpu() for ib in range(len(boxes)) for c in range(4)]
    out["tags"] = [tuple(t.cpu() for t in s.tag_strings(l)) for l in range(nl)]
    if tee is not None:
        s.synchronize()
        out["tee"] = tuple(t.cpu() for t in tee)
    s.fill_ghosts(nl - 1, eta)
    out["ghosted"] = [s.get_ghosted(ib, c).cpu() for ib in s.level_boxes(nl - 1) for c in (0, 3)]
    return out


@pytest.mark.parametrize("dtype,flow,interp,ragged", [("f64", "fused", 0, False), ("f64", "lean", 4, False),
                                                      ("f32", "fused", 4, False), ("f64", "fused", 0, True),
                                                      ("f32", "classic", 0, True)])
def test_coalesced_storage_gives_the_same_bits(monkeypatch, dtype, flow, interp, ragged):
    """Merging boxes that share a face removes ghost cells, never changes a result: states, string tags + counts,
    truncation-error tags and ghosted copies are bit-identical with SLEDGE_COALESCE=0, the default order and zyx."""
    ref = _run_hierarchy(monkeypatch, "0", dtype, flow, interp, ragged)
    nbox = [len([b for b in (_ragged_boxes() if ragged else _ring_hierarchy(32)) if b[0] == l]) for l in range(len(ref["storage"]))]
    assert [n for n, _ in ref["storage"]] == nbox
    for mode in (None, "zyx"):
        got = _run_hierarchy(monkeypatch, mode, dtype, flow, interp, ragged)
        assert got["storage"][0][0] == 1          # level 0 covers the domain: one rectangle (the ragged list too)
        assert all(g[0] <= r[0] and g[1] <= r[1] for g, r in zip(got["storage"], ref["storage"]))
        for key in ("state", "ghosted"):
            for a, b in zip(ref[key], got[key]):
                assert torch.equal(a, b), key
        for (ta, ca), (tb, cb) in zip(ref["tags"], got["tags"]):
            assert torch.equal(ta, tb) and torch.equal(ca, cb)
        if "tee" in ref:
            for a, b in zip(ref["tee"], got["tee"]):
                assert torch.equal(a, b)
