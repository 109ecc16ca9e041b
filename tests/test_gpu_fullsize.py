"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.

The oracle cannot step a 512^3 or 1024^3 grid in seconds, but the path is periodic and translation invariant
(pinned for the oracle in test_oracle_pins.py::test_translation_invariance_bit_for_bit): a field
that repeats with period P cells evolves into a field that repeats with period P, and every one of its periods
equals the run on the P^3 periodic grid.  So the full-size GPU run started from a P^3 seeded GRF tiled N/P times
per axis (inputs.tile_periodic) is compared, at EVERY cell, with the tiled result of the P^3 oracle run: same
parameters, same step count as the config, all of the full-size grid's K1 tiles, z chunks and ghost wraps.
Tags and per-32^3 block counts are compared bit for bit on the uploaded oracle state (R19).
"""
import numpy as np
import pytest
import torch

from paper_2404_02950_b200 import inputs

pytestmark = pytest.mark.gpu

F64_TOL = 1e-11
F32_TOL = 2e-5


def _run_tiled(name, period, flow, steps=None, check_tags=False):
    from oracle.oracle import Oracle
    from paper_2404_02950_b200.sledge import Sledge
    cfg = inputs.CONFIGS[name]
    steps = cfg.steps if steps is None else steps
    reps = cfg.n0 // period
    tdt = torch.float64 if cfg.dtype == "f64" else torch.float32
    o = Oracle(period, nghost=cfg.nghost, lap_order=cfg.lap_order, h0=cfg.h0, lam=cfg.lam)
    s = Sledge(cfg.n0, nghost=cfg.nghost, lap_order=cfg.lap_order, h0=cfg.h0, lam=cfg.lam, dtype=cfg.dtype,
               rk_dataflow=flow)
    # the band limit is a fraction of k_Nyquist = pi/h, the same on the small and on the full grid
    for c, seed in enumerate(cfg.seeds):
        small = inputs.grf(period, cfg.grf_f, seed).to(tdt)
        o.set_state(0, c, small.to(torch.float64).numpy())
        s.set_state(0, c, inputs.tile_periodic(small.cuda(), reps).contiguous())
    eta = cfg.eta0
    for _ in range(steps):
        o.rk_step(cfg.dt, eta)
        s.rk_step(cfg.dt, eta)
        eta += cfg.dt
    s.synchronize()
    worst = 0.0
    for c in range(4):
        ref = torch.from_numpy(o.get_state(0, c)).cuda()
        got = s.get_state(0, c).to(torch.float64)
        err = float((got.view(reps, period, reps, period, reps, period) - ref[None, :, None, :, None, :]).abs().max())
        scale = float(ref.abs().max()) if cfg.dtype == "f32" else 1.0
        worst = max(worst, err / scale if scale > 0 else err)
        del got, ref
    assert worst <= (F64_TOL if cfg.dtype == "f64" else F32_TOL), worst
    if check_tags:
        for c in range(4):
            ref = torch.from_numpy(o.get_state(0, c)).to(tdt).cuda()
            s.set_state(0, c, inputs.tile_periodic(ref, reps).contiguous())
        ot, oc = o.tag_strings(0)
        gt, gc = s.tag_strings(0)
        s.synchronize()
        want = inputs.tile_periodic(torch.from_numpy(ot[0]).cuda(), reps)
        assert torch.equal(s.split_tags(0, gt)[0], want)
        wantc = inputs.tile_periodic(torch.from_numpy(oc.astype(np.int32)).cuda(), reps)
        assert torch.equal(gc, wantc)
        assert int((ot[0] != 0).sum()) > 0
    s.close()
    return worst


@pytest.mark.parametrize("flow", ["fused", "lean"])
def test_c3_512cubed_fp64_13pt_50_steps_all_cells_and_tags(flow):
    _run_tiled("C3", 64, flow, check_tags=True)


def test_c2_256cubed_fp64_7pt_100_steps_all_cells():
    _run_tiled("C2", 64, "fused")


def test_c4_1024cubed_fp32_7pt_20_steps_all_cells_and_tags():
    free, _ = torch.cuda.mem_get_info()
    if free < 90e9:
        pytest.skip("needs ~80 GB of free HBM")
    _run_tiled("C4", 64, "fused", check_tags=True)


# ---- C5 at full size: a property that holds at any size ------------------------------------------------------------

@pytest.mark.parametrize("interp,extra", [(0, {}), (4, {}),
                                          (4, dict(integrator=10, ko_order=3, ko_strength=(0.02, 0.03, 0.05, 0.07)))])
def test_c5_full_hierarchy_reproduces_an_affine_linear_in_time_solution(interp, extra):
    """The oracle cannot step the 2,067-box C5 hierarchy in seconds, but with lambda = 0 the field
    psi_c = a_c . x + b_c + v_c t, Pi_c = v_c solves Eq.10-11 exactly, and every piece of the path reproduces it exactly
    (up to rounding): the central Laplacians vanish on affine data, RK4 is exact for a solution linear in time, trilinear
    and quartic interpolation reproduce affine data, linear-in-time ghosts are exact, the mean of 8 children of an affine
    field is its value at the parent's centre.  Any wrong ghost source, parent, time weight or box offset anywhere in
    the full hierarchy shows up as a non-zero Laplacian.  The periodic wrap breaks the affine field at the domain
    faces; that disturbance travels at most lap_order cells per stage, so cells further than 12 coarse cells from a face
    must hold the exact solution after one coarse step, in the launch configuration bench.py times.  The third variant
    runs SSPRK3 with the order-3 Kreiss-Oliger term, which vanishes on affine data as well (at most 3 cells per stage)."""
    import bench
    from paper_2404_02950_b200.sledge import Sledge
    cfg = inputs.CONFIGS["C5"]
    rings, boxes, cover = bench.hierarchy(cfg)
    s = Sledge(cfg.n0, boxes=boxes, n_levels=cfg.n_levels, nghost=cfg.nghost, blocking_factor=cfg.blocking_factor,
               dtype="f64", lap_order=cfg.lap_order, h0=cfg.h0, lam=0.0, rk_dataflow="fused", interp=interp, **extra)
    A = torch.tensor([[0.01, 0.02, -0.015], [-0.02, 0.005, 0.01]], dtype=torch.float64, device="cuda")  # per comp: x, y, z
    B = (0.3, -0.8)
    V = (0.1, 0.25)

    def coords(l, lo, hi):
        h = cfg.h0 / (1 << l)
        ax = [(torch.arange(lo[d], hi[d] + 1, dtype=torch.float64, device="cuda") + 0.5) * h for d in range(3)]
        return ax[0][None, None, :], ax[1][None, :, None], ax[2][:, None, None]

    for ib, (l, lo, hi) in enumerate(boxes):
        X, Y, Z = coords(l, lo, hi)
        for c in range(2):
            s.set_state(ib, c, (A[c, 0] * X + A[c, 1] * Y + A[c, 2] * Z + B[c]).contiguous())
            s.set_state(ib, c + 2, torch.full(s.box_shape(ib), V[c], dtype=torch.float64, device="cuda"))
    s.rk_step(cfg.dt, cfg.eta0)
    s.synchronize()
    L = cfg.n0 * cfg.h0
    margin = 12 * cfg.h0
    worst, checked = 0.0, 0
    for ib, (l, lo, hi) in enumerate(boxes):
        X, Y, Z = coords(l, lo, hi)
        inner = ((X > margin) & (X < L - margin)) & ((Y > margin) & (Y < L - margin)) & ((Z > margin) & (Z < L - margin))
        if not bool(inner.any()):
            continue
        for c in range(2):
            want = A[c, 0] * X + A[c, 1] * Y + A[c, 2] * Z + (B[c] + V[c] * cfg.dt)
            worst = max(worst, float(((s.get_state(ib, c) - want).abs() * inner).max()))
            worst = max(worst, float(((s.get_state(ib, c + 2) - V[c]).abs() * inner).max()))
        checked += int(inner.sum())
    assert checked > 0.5 * sum(int(np.prod(s.box_shape(ib))) for ib in range(len(boxes)))
    assert worst <= F64_TOL, worst
    s.close()


# ---- C5 against the oracle in its own shape (BASELINE.json config 5; section II.A, Fig.2 L88) -------------

def _host_ram_free_gb():
    import psutil
    return psutil.virtual_memory().available / 1e9


def _ring_pair(cfg, rings, boxes, flow="fused", interp=0):
    """Oracle + CUDA context for a ring hierarchy with C5's parameters, both fed the same arrays (evaluated once, on
    the GPU, and copied to the host for the oracle)."""
    from oracle.oracle import Oracle
    from paper_2404_02950_b200.sledge import Sledge
    kw = dict(boxes=boxes, n_levels=cfg.n_levels, nghost=cfg.nghost, blocking_factor=cfg.blocking_factor,
              lap_order=cfg.lap_order, h0=cfg.h0, lam=cfg.lam, interp=interp)
    o = Oracle(rings.n0, **kw)
    s = Sledge(rings.n0, dtype="f64", rk_dataflow=flow, **kw)
    for ib, (l, lo, hi) in enumerate(boxes):
        re, im = inputs.ring_field(rings, l, lo, hi, device="cuda")
        for c, t in enumerate((re, im)):
            t = t.contiguous()
            s.set_state(ib, c, t)
            o.set_state(ib, c, t.cpu().numpy())
    return o, s


def _max_err_all_boxes(o, s):
    worst = 0.0
    for ib in range(len(s.boxes)):
        for c in range(4):
            worst = max(worst, float(np.abs(o.get_state(ib, c) - s.get_state(ib, c).cpu().numpy()).max()))
    return worst


def _tags_on_oracle_state(o, s, n_levels):
    """bit-exact tags + 32^3 counts on every level, both sides tagging the oracle's state (R19)"""
    for ib in range(len(s.boxes)):
        for c in range(4):
            s.set_state(ib, c, torch.from_numpy(o.get_state(ib, c)).cuda().contiguous())
    total = 0
    for l in range(n_levels):
        ot, oc = o.tag_strings(l)
        gt, gc = s.tag_strings(l)
        s.synchronize()
        for a, b in zip(ot, s.split_tags(l, gt)):
            assert np.array_equal(a, b.cpu().numpy()), f"tags differ on level {l}"
        assert np.array_equal(oc.astype(np.int64), gc.cpu().numpy().astype(np.int64)), f"counts differ on level {l}"
        total += sum(int((a != 0).sum()) for a in ot)
    return total


def test_c5_real_hierarchy_one_coarse_step_every_cell_against_the_oracle():
    """The configuration `bench.py --workload C5` times: the 2,067-box hierarchy (512 + 843 + 712 boxes of 32^3, g = 3,
    13-point, lambda = 1, ring IC), FUSED sweeps on level 0, LEAN on levels 1 and 2, packed star lists, subcycling
    1/2/4 with trilinear + linear-in-time ghosts and two average-downs -- ONE coarse step compared with the oracle at
    every cell of every box, then tags and 32^3 counts bit for bit on all three levels."""
    import bench
    need = 34.0
    if _host_ram_free_gb() < need:
        pytest.skip(f"the oracle needs ~{need:.0f} GB of host RAM for 2,067 boxes x 7 states; "
                    f"{_host_ram_free_gb():.0f} GB free")
    cfg = inputs.CONFIGS["C5"]
    rings, boxes, cover = bench.hierarchy(cfg)
    assert len(boxes) == 2067 and all(hi[0] - lo[0] == 31 for _, lo, hi in boxes)
    o, s = _ring_pair(cfg, rings, boxes)
    o.rk_step(cfg.dt, cfg.eta0)
    s.rk_step(cfg.dt, cfg.eta0)
    s.synchronize()
    assert _max_err_all_boxes(o, s) <= F64_TOL
    assert _tags_on_oracle_state(o, s, cfg.n_levels) > 0
    s.close()


@pytest.mark.parametrize("interp,steps", [(0, 20), (4, 4)])
def test_c5_recipe_at_base_128_with_32cubed_boxes_20_coarse_steps(interp, steps):
    """C5's own box size (32^3), ghost width, stencil, time step and the configured 20 coarse steps, on a 128^3 base so
    that the oracle finishes in about a minute: every cell of every box, then tags on all levels.  The quartic
    interpolation variant (not C5's; the oracle's 5^3-point fill is slow) runs 4 coarse steps."""
    cfg = inputs.CONFIGS["C5"]
    ex = cfg.extra
    rings = inputs.make_rings(128, 4, 12.0, 30.0, ex["core_w"], cfg.seeds[0] + 1)
    boxes, cover = inputs.amr_boxes_for_rings(rings, n_levels=3, box=32, r1=ex["r1"], r2=ex["r2"],
                                              blocking_factor=cfg.blocking_factor)
    assert 0 < cover[2] < cover[1] < 1
    o, s = _ring_pair(cfg, rings, boxes, interp=interp)
    assert steps == cfg.steps or interp != 0
    eta = cfg.eta0
    for _ in range(steps):
        o.rk_step(cfg.dt, eta)
        s.rk_step(cfg.dt, eta)
        eta += cfg.dt
    s.synchronize()
    assert _max_err_all_boxes(o, s) <= F64_TOL
    assert _tags_on_oracle_state(o, s, 3) > 0
    s.close()


# ---- sizes incommensurate with every tile of the kernels -------------------------------------------------------------
# The tiled-IC runs above repeat with period 64, a multiple of K1's 32 x 8 column tile, a divisor of its 128-plane z
# chunk and two 32-blocks of the count reduction: a CTA that took its halo, z-window or wrapped address from the wrong
# tile at an offset that is a multiple of 64 would go unseen.  Here nothing repeats: one periodic box of 392^3 = (8 x 49)^3
# -- 12.25 x tiles, 3.06 z chunks, 12.25 count blocks -- with a real, untiled GRF; the oracle runs the same field cut
# into 56^3 boxes (bitwise equal to one box: test_oracle_pins.py::test_multibox_level_equals_single_box_bitwise).

def _untiled(n, oracle_box, flow, steps, f, seeds, cfg):
    from oracle.oracle import Oracle
    from paper_2404_02950_b200.sledge import Sledge
    oboxes = inputs.split_level0(n, oracle_box)
    o = Oracle(n, boxes=oboxes, nghost=cfg.nghost, lap_order=cfg.lap_order, h0=cfg.h0, lam=cfg.lam)
    s = Sledge(n, nghost=cfg.nghost, lap_order=cfg.lap_order, h0=cfg.h0, lam=cfg.lam, dtype="f64", rk_dataflow=flow)

    def scatter(c, full):  # full: numpy [z, y, x]
        for ib, (_, lo, hi) in enumerate(oboxes):
            o.set_state(ib, c, full[lo[2]:hi[2] + 1, lo[1]:hi[1] + 1, lo[0]:hi[0] + 1])

    def gather(c):
        full = np.empty((n, n, n))
        for ib, (_, lo, hi) in enumerate(oboxes):
            full[lo[2]:hi[2] + 1, lo[1]:hi[1] + 1, lo[0]:hi[0] + 1] = o.get_state(ib, c)
        return full

    for c, seed in enumerate(seeds):
        a = inputs.grf(n, f, seed)
        scatter(c, a.numpy())
        s.set_state(0, c, a.cuda().contiguous())
        del a
    eta = cfg.eta0
    for _ in range(steps):
        o.rk_step(cfg.dt, eta)
        s.rk_step(cfg.dt, eta)
        eta += cfg.dt
    s.synchronize()
    worst = 0.0
    state = []
    for c in range(4):
        ref = torch.from_numpy(gather(c)).cuda()
        worst = max(worst, float((s.get_state(0, c) - ref).abs().max()))
        state.append(ref)
    assert worst <= F64_TOL, worst
    for c in range(4):
        s.set_state(0, c, state[c].contiguous())
    del state
    ot, oc = o.tag_strings(0)
    gt, gc = s.tag_strings(0)
    s.synchronize()
    got = s.split_tags(0, gt)[0]
    ntag = 0
    for ib, (_, lo, hi) in enumerate(oboxes):
        assert np.array_equal(ot[ib], got[lo[2]:hi[2] + 1, lo[1]:hi[1] + 1, lo[0]:hi[0] + 1].cpu().numpy())
        ntag += int((ot[ib] != 0).sum())
    assert np.array_equal(oc.astype(np.int64), gc.cpu().numpy().astype(np.int64))
    assert ntag > 0
    s.close()


@pytest.mark.parametrize("flow", ["fused", "lean"])
def test_untiled_392cubed_incommensurate_with_the_tiles(flow):
    need = 22.0
    if _host_ram_free_gb() < need:
        pytest.skip(f"the oracle needs ~{need:.0f} GB of host RAM; {_host_ram_free_gb():.0f} GB free")
    _untiled(392, 56, flow, 3, 0.1, (3921, 3922), inputs.CONFIGS["C3"])


def test_c3_real_untiled_initial_data_two_steps():
    """C3's own initial data (seeds 3001 / 3002 at 512^3, NOT tiled), two steps of the flow bench.py times."""
    need = 48.0
    if _host_ram_free_gb() < need:
        pytest.skip(f"the oracle needs ~{need:.0f} GB of host RAM for 512^3 in 64^3 boxes; {_host_ram_free_gb():.0f} GB free")
    cfg = inputs.CONFIGS["C3"]
    _untiled(cfg.n0, 64, "fused", 2, cfg.grf_f, cfg.seeds, cfg)


# ---- round-2 rows at bench size: the workloads bench.py --gw / --integrator 20 time --------------------------------

def _tiled_extra(n_full, period, steps, **kw):
    """C2-sized periodic box, period-`period` seeded data (every component), GPU against the tiled oracle run."""
    from oracle.oracle import Oracle
    from paper_2404_02950_b200.sledge import Sledge
    cfg = inputs.CONFIGS["C2"]
    reps = n_full // period
    okw = dict(nghost=2, lap_order=2, h0=cfg.h0, lam=cfg.lam)
    o = Oracle(period, **okw, **kw)
    s = Sledge(n_full, rk_dataflow="fused", **okw, **kw)
    ncomp = 16 if kw.get("gw") else 4
    for c in range(ncomp):
        amp = 1.0 if c < 2 else 0.1
        small = amp * inputs.grf(period, 0.2, 7000 + c).to(torch.float64)
        o.set_state(0, c, small.numpy())
        s.set_state(0, c, inputs.tile_periodic(small.cuda(), reps).contiguous())
    eta = cfg.eta0
    for _ in range(steps):
        o.rk_step(cfg.dt, eta)
        s.rk_step(cfg.dt, eta)
        eta += cfg.dt
    s.synchronize()
    worst = 0.0
    for c in range(ncomp):
        ref = torch.from_numpy(o.get_state(0, c)).cuda()
        got = s.get_state(0, c)
        worst = max(worst, float((got.view(reps, period, reps, period, reps, period) - ref[None, :, None, :, None, :]).abs().max()))
        del got, ref
    s.close()
    return worst


def test_gw_256cubed_all_16_components():
    assert _tiled_extra(256, 64, 5, gw=True, gw_coupling=1.0, gw_friction=2.0) <= F64_TOL


def test_rkn_256cubed_nystrom4():
    rkn4 = dict(nodes=[0.0, 0.5, 1.0], weights_b=[1 / 6, 4 / 6, 1 / 6], weights_bar_b=[1 / 6, 1 / 3, 0.0],
                tableau=[0.0, 1 / 8, 0.0, 0.0, 0.5, 0.0])
    assert _tiled_extra(256, 64, 20, integrator=20, rkn=rkn4) <= F64_TOL
