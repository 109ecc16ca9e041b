"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/sledge.h declares; host-side validation (sledge_arena_bytes needs no GPU) rejects what the
paper's grid rules forbid; the product path fails loudly without a GPU; the product never imports the
oracle."""
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))

from paper_2404_02950_b200 import build as sbuild
from paper_2404_02950_b200 import inputs
from paper_2404_02950_b200 import sledge as S


@pytest.fixture(scope="module", autouse=True)
def built():
    sbuild.build()


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "sledge.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(sledge_[a-z_]+)\s*\(", hdr)))
    assert len(declared) >= 19
    out = subprocess.run(["nm", "-D", "--defined-only", S.LIB_PATH], capture_output=True, text=True, check=True).stdout
    exported = set(re.findall(r" T (sledge_[a-z_]+)", out))
    assert set(declared) <= exported, set(declared) - exported
    assert set(declared) == set(S.SYMBOLS)
    L = S.lib()
    for name in declared:
        assert hasattr(L, name)


def test_library_is_compiled_for_sm_100a():
    out = subprocess.run(["cuobjdump", "-lelf", S.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_arena_bytes_matches_hand_count_single_box():
    # 32^3, g = 1, fp64: pair = 16 B, rows padded to 8 + 32 + 8 = 48 pairs, 34 rows, 34 planes
    n = S.sledge_arena_bytes(32, nghost=1, dtype="f64")
    plane = 48 * 34 * 34 * 16
    # + six staging slots (2 in, 4 out) of one ghosted box component for the host-buffer copies + the descriptor tables
    assert n >= 8 * plane + 6 * 34 ** 3 * 8 and n < 8 * plane + 6 * 34 ** 3 * 8 + 256 * 1024
    # fp32 pairs are 8 B: 16 + 32 + 16 = 64 pairs per row
    n32 = S.sledge_arena_bytes(32, nghost=1, dtype="f32")
    assert n32 >= 8 * 64 * 34 * 34 * 8


def test_coalescing_removes_the_ghost_cells_between_boxes(monkeypatch):
    """Storage boxes (include/sledge.h, sledge_level_storage): 8 boxes of 16^3 covering a 32^3 level are stored as one
    32^3 rectangle -- the arena is that of the one-box layout (plus descriptor tables), and smaller than with
    SLEDGE_COALESCE=0 (8 x (16 + 2g)^3 against (32 + 2g)^3 stored cells per plane)."""
    split = inputs.split_level0(32, 16)
    kw = dict(nghost=2, blocking_factor=8, lap_order=2)
    monkeypatch.delenv("SLEDGE_COALESCE", raising=False)
    one = S.sledge_arena_bytes(32, **kw)
    merged = S.sledge_arena_bytes(32, boxes=split, **kw)
    monkeypatch.setenv("SLEDGE_COALESCE", "0")
    apart = S.sledge_arena_bytes(32, boxes=split, **kw)
    # staging slots are sized by the largest caller's box: smaller for the split list
    assert merged <= one + 64 * 1024
    plane_one = 48 * 36 * 36 * 16          # 8 + 32 + 8 pairs per row
    plane_apart = 8 * 32 * 20 * 20 * 16    # 8 + 16 + 8 pairs per row
    assert apart - merged >= 8 * (plane_apart - plane_one) - 64 * 1024
    assert apart > merged


@pytest.mark.parametrize("seed", [0, 1, 2, 3, 4, 5])
def test_random_hierarchies_validate_and_coalescing_never_costs_memory(monkeypatch, seed):
    """host logic only (no GPU): the seeded random hierarchies of the GPU parity tests pass the library's validation
    (alignment, disjointness, level 0 covering the domain, proper nesting: L39, L70, L137) with and without the
    storage-box coalescing, in any merge order, and merged storage never needs more arena than separate boxes"""
    for n0, bf, nl, g in (((32, 24, 40), 8, 3, 3), ((16, 16, 16), 4, 3, 2), ((16, 24, 16), 2, 2, 1)):
        boxes = inputs.random_hierarchy(n0, nl, bf, 100 * seed + bf + nl)
        kw = dict(boxes=boxes, n_levels=nl, nghost=g, blocking_factor=bf, lap_order=min(g, 2))
        sizes = {}
        for mode in ("0", None, "zyx", "yxz"):
            if mode is None:
                monkeypatch.delenv("SLEDGE_COALESCE", raising=False)
            else:
                monkeypatch.setenv("SLEDGE_COALESCE", mode)
            sizes[mode] = S.sledge_arena_bytes(n0, **kw)
        assert all(sizes[m] <= sizes["0"] for m in (None, "zyx", "yxz")), sizes
        # a box list that violates nesting is still rejected when boxes are merged: drop a level-1 box under a level-2 one
        if nl == 3:
            monkeypatch.delenv("SLEDGE_COALESCE", raising=False)
            l2 = [b for b in boxes if b[0] == 2]
            if l2:
                lo = tuple(v // 2 for v in l2[0][1])
                bad = [b for b in boxes if not (b[0] == 1 and all(b[1][d] <= lo[d] <= b[2][d] for d in range(3)))]
                if len(bad) < len(boxes):
                    with pytest.raises(S.SledgeError):
                        S.sledge_arena_bytes(n0, **dict(kw, boxes=bad))


RKN4 = dict(nodes=[0.0, 0.5, 1.0], weights_b=[1 / 6, 4 / 6, 1 / 6], weights_bar_b=[1 / 6, 1 / 3, 0.0],
            tableau=[0.0, 1 / 8, 0.0, 0.0, 0.5, 0.0])


def test_validation_rules_from_the_paper():
    ok = dict(n_levels=1, nghost=2, blocking_factor=8, lap_order=2)
    S.sledge_arena_bytes(32, **ok)
    bad = [
        dict(ok, lap_order=3),                     # the 19-point stencil needs 3 ghost layers: lap_order <= nghost (L240)
        dict(ok, nghost=1),                        # lap_order <= nghost (L240)
        dict(ok, nghost=8),                        # nghost < blocking_factor (L772)
        dict(ok, blocking_factor=12),              # power of 2 (L39)
        dict(ok, h0=0.0),
        dict(ok, ko_order=3, ko_strength=0.01),    # dissipation order = ghost cells needed (L751): 3 > nghost
        dict(ok, ko_order=1, ko_strength=0.01),    # order is 2 or 3 (L751)
        dict(ok, interp=2),                        # only trilinear (0) and quartic conservative (4, L780)
        dict(ok, n_levels=2, nghost=5, lap_order=2, interp=4,  # ceil(5/2) + 2 > 8/2: window leaves the nesting gap (L70)
             boxes=[(0, (0, 0, 0), (31, 31, 31)), (1, (16, 16, 16), (47, 47, 47))]),
        dict(ok, integrator=21),                   # the RKN4 / RKN5 tableaux (types 21, 22) are not printed in the paper: unavailable
        dict(ok, integrator=20),                   # type 20 needs the user's tableau (L812-815)
        dict(ok, integrator=20, rkn=RKN4, friction=2.0),         # a Nystrom scheme integrates psi'' = f(psi) only
        dict(ok, integrator=20, rkn=RKN4, ko_order=2, ko_strength=0.01),
        dict(ok, integrator=20, rkn=dict(RKN4, tableau=[0.0, 1 / 8, 0.1, 0.0, 0.5, 0.0])),  # implicit diagonal entry (L815)
        dict(ok, integrator=20, rkn=dict(RKN4, nodes=[0.1, 0.5, 1.0])),                      # first stage = the state
        dict(ok, integrator=20, rkn=RKN4, gw=True),
        dict(ok, gw=True, integrator=10),          # auxiliary fields: classic RK4 only
        dict(ok, gw=True, interp=4, n_levels=2, nghost=3,
             boxes=[(0, (0, 0, 0), (31, 31, 31)), (1, (16, 16, 16), (47, 47, 47))]),
        dict(ok, ko_order=2, ko_strength=(0.0, -0.1, 0.0, 0.0)),  # strength in R+ (L749)
    ]
    S.sledge_arena_bytes(32, **dict(ok, ko_order=2, ko_strength=(0.0, 0.0, 0.02, 0.0)))
    S.sledge_arena_bytes(32, **dict(ok, integrator=10))
    S.sledge_arena_bytes(32, **dict(ok, integrator=20, rkn=RKN4))
    # the auxiliary fields add six pair planes per state buffer: 4x the state
    assert S.sledge_arena_bytes(32, **dict(ok, gw=True)) > 3.2 * S.sledge_arena_bytes(32, **ok)
    # shadow level (L98): level 0 coarsened by 2 in one box; n0 must be even and the coarsened grid valid
    assert S.sledge_arena_bytes(32, **dict(ok, shadow_level=True)) > S.sledge_arena_bytes(32, **ok)
    with pytest.raises(S.SledgeError, match="shadow"):
        S.sledge_arena_bytes(8, **dict(ok, shadow_level=True, nghost=4))  # 4^3 cells cannot carry 4 ghost layers (L772)
    S.sledge_arena_bytes(32, **dict(ok, n_levels=2, nghost=3, interp=4,
                                    boxes=[(0, (0, 0, 0), (31, 31, 31)), (1, (16, 16, 16), (47, 47, 47))]))
    S.sledge_arena_bytes(32, **dict(ok, ko_order=7, ko_strength=0.0))  # strength 0 removes the term, order unused
    for kw in bad:
        with pytest.raises(S.SledgeError):
            S.sledge_arena_bytes(32, **kw)
    with pytest.raises(S.SledgeError):            # n0 multiple of the blocking factor
        S.sledge_arena_bytes(36, **ok)
    full = (0, (0, 0, 0), (31, 31, 31))
    with pytest.raises(S.SledgeError, match="cover"):
        S.sledge_arena_bytes(32, boxes=[(0, (0, 0, 0), (31, 31, 15))], **ok)
    with pytest.raises(S.SledgeError, match="overlap"):
        S.sledge_arena_bytes(32, boxes=[full, (0, (8, 8, 8), (15, 15, 15))], **ok)
    with pytest.raises(S.SledgeError, match="aligned"):
        S.sledge_arena_bytes(32, boxes=[(0, (0, 0, 0), (31, 31, 27)), (0, (0, 0, 28), (31, 31, 31))], **ok)
    # nesting (L70, L137): a level-2 box needs a gap of one blocking factor to the level-1 boundary
    l1 = (1, (16, 16, 16), (47, 47, 47))
    S.sledge_arena_bytes(32, boxes=[full, l1, (2, (48, 48, 48), (63, 63, 63))], **dict(ok, n_levels=3))
    with pytest.raises(S.SledgeError, match="nesting"):
        S.sledge_arena_bytes(32, boxes=[full, l1, (2, (32, 48, 48), (47, 63, 63))], **dict(ok, n_levels=3))
    with pytest.raises(S.SledgeError, match="no boxes"):
        S.sledge_arena_bytes(32, boxes=[full], **dict(ok, n_levels=2))
    # a fine level may wrap around the periodic boundary as long as level 0 is everywhere
    S.sledge_arena_bytes(32, boxes=[full, (1, (0, 0, 0), (15, 15, 15)), (1, (48, 0, 0), (63, 15, 15))],
                         **dict(ok, n_levels=2))


def test_config5_generator_produces_a_valid_nested_hierarchy():
    """The C5 recipe (DESIGN.md input recipe) at reduced size passes the library's own nesting check and the
    oracle's, and reaches coverage fractions in the intended range."""
    from oracle.oracle import Oracle
    rings = inputs.make_rings(64, 3, 8.0, 16.0, 2.0, seed=5000)
    boxes, cover = inputs.amr_boxes_for_rings(rings, n_levels=3, box=16, r1=4.0, r2=1.0, blocking_factor=8)
    assert 0.0 < cover[2] < cover[1] < 0.6
    S.sledge_arena_bytes(64, boxes=boxes, n_levels=3, nghost=3, blocking_factor=8, lap_order=2)
    Oracle(64, boxes=boxes, n_levels=3, nghost=3, blocking_factor=8, lap_order=2)


def test_test_hierarchies_are_valid_without_a_gpu():
    import _pair as P
    from test_gpu_parity import _ragged_boxes, _ring_hierarchy
    S.sledge_arena_bytes(32, boxes=P.two_level_boxes(32), n_levels=2, nghost=3, lap_order=2)
    S.sledge_arena_bytes((40, 24, 72), boxes=_ragged_boxes(), nghost=3, lap_order=2)
    _, boxes, _ = _ring_hierarchy()
    S.sledge_arena_bytes(32, boxes=boxes, n_levels=3, nghost=3, lap_order=2)


def test_no_cpu_fallback_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(S.SledgeError, match="no CUDA device"):
        S.Sledge(16)
    # the C entry point itself refuses as well (an arena pointer that looks valid but no device)
    import ctypes as C
    p, arr, boxes, _ = S._marshal(16, None, 1, 1, 8, "f64", 1, 1.0, 1.0, 0.0, 0.0, False, "lean")
    need = S.sledge_arena_bytes(16)
    h = C.c_void_p()
    rc = S.lib().sledge_create(C.byref(h), C.byref(p), arr, 1, 256, need, None)
    assert rc == -3 and b"no CPU fallback" in S.lib().sledge_last_error(None)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2404_02950_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("the oracle", "").replace("oracle rounding", "") or f == "inputs.py", f
    hdr = open(os.path.join(ROOT, "include", "sledge.h")).read()
    assert "oracle" not in hdr
