"""GPU parity on seeded RANDOM hierarchies (paper_2404_02950_b200/inputs.py::random_hierarchy): boxes of mixed sizes on
every level, many sharing faces (coalesced into storage boxes by the library) and many not,
level-1 / level-2 sets with holes, single blocking cells and boxes touching the periodic seam.  Everything a caller can
see is compared with the CPU oracle: states after subcycled coarse steps (fp64 <= 1e-11, fp32 <= 2e-5 relative), ghost
cells after an explicit fill on every level, string tags + 32^3 counts bit-exact on the same state (PAPER.md L23,
L66-76, L80-96)."""
import numpy as np
import pytest
import torch

from paper_2404_02950_b200 import inputs

pytestmark = pytest.mark.gpu

F64_TOL = 1e-11
F32_TOL = 2e-5


def _pair():
    import _pair as P
    return P


CASES = [
    # n0, blocking factor, levels, ghosts, order, flow, interp, dtype
    ((32, 24, 40), 8, 3, 3, 2, "fused", 0, "f64"),
    ((32, 24, 40), 8, 3, 2, 2, "lean", 4, "f64"),
    ((16, 16, 16), 4, 3, 2, 2, "fused", 0, "f64"),
    ((24, 16, 8), 8, 2, 1, 1, "classic", 0, "f64"),
    ((32, 24, 40), 8, 3, 3, 2, "fused", 4, "f32"),
    ((16, 24, 16), 2, 2, 1, 1, "fused", 0, "f64"),
]


@pytest.mark.parametrize("seed", [0, 1, 2, 3])
@pytest.mark.parametrize("case", CASES, ids=lambda c: f"{c[0][0]}x{c[0][1]}x{c[0][2]}-bf{c[1]}-L{c[2]}-g{c[3]}-{c[5]}-i{c[6]}-{c[7]}")
def test_random_hierarchy_matches_the_oracle(case, seed):
    P = _pair()
    n0, bf, nl, g, order, flow, interp, dtype = case
    boxes = inputs.random_hierarchy(n0, nl, bf, 100 * seed + bf + nl)
    nl_eff = 1 + max(b[0] for b in boxes)
    assert nl_eff == nl
    o, s = P.make_pair(n0, boxes=boxes, n_levels=nl, nghost=g, blocking_factor=bf, lap_order=order, h0=0.5, lam=0.7,
                       a_mass=0.3, friction=2.0, rk_dataflow=flow, interp=interp, dtype=dtype)
    # fewer storage boxes than caller's boxes wherever two of them share a face (level 0 always merges to one)
    assert s.level_storage(0)[0] == 1
    assert all(s.level_storage(l)[0] <= len(s.level_boxes(l)) for l in range(nl))
    P.init_smooth(o, s, n0, 17 + seed, amp=0.8)
    for l in range(nl - 1, 0, -1):
        o.average_down(l)
        s.average_down(l)
    eta, dt = 1.5, 0.1
    for _ in range(2):
        o.rk_step(dt, eta)
        s.rk_step(dt, eta)
        eta += dt
    if dtype == "f64":
        assert P.max_err(o, s) <= F64_TOL
    else:
        assert P.max_err(o, s, relative=True) <= F32_TOL
    # same state on both sides from here on: ghosts and tags are then bit-level statements
    P.upload_oracle_state(o, s)
    if dtype == "f32":  # the oracle continues from the fp32-rounded state (R15)
        for ib in range(len(boxes)):
            for c in range(4):
                o.set_state(ib, c, s.get_state(ib, c).to(torch.float64).cpu().numpy())
    for l in range(nl):
        o.fill_ghosts(l, eta)
        s.fill_ghosts(l, eta)
        for ib in s.level_boxes(l)[:: max(1, len(s.level_boxes(l)) // 12)]:
            for c in (0, 3):
                a = o.get_raw(ib, c)
                b = s.get_ghosted(ib, c).to(torch.float64).cpu().numpy()
                tol = F64_TOL if dtype == "f64" else F32_TOL * max(1.0, float(np.abs(a).max()))
                assert np.abs(a - b).max() <= tol, (l, ib, c)
    for l in range(nl):
        ot, oc = o.tag_strings(l)
        gt, gc = s.tag_strings(l)
        s.synchronize()
        for a, b in zip(ot, s.split_tags(l, gt)):
            assert np.array_equal(a, b.cpu().numpy())
        assert np.array_equal(oc.astype(np.int64), gc.cpu().numpy().astype(np.int64))
