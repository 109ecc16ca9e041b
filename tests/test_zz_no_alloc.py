"""sledge_tag_strings_static (include/sledge.h): the string-tagging pass with NO allocation -- no context, no arena; its
scratch (packed pair plane + box / tile tables) is a file-scope static __device__ array of 8 MiB inside libsledge.so.

Checked against the existing path (sledge_create + sledge_set_state + sledge_tag_strings on a one-box periodic level 0)
on the same seeded input: tag bytes and 32^3 block counts are integer work, so the bar is bit-exact, as everywhere in
tests/.  Two calls in a row of different sizes and dtypes share the array: the second must not see the first one's
leftovers, and repeating the first must reproduce it.  The file sorts last on purpose (the suite runs with pytest -x)
and passes both alone in a fresh process and after every other test."""
import pytest
import torch

from paper_2404_02950_b200 import inputs
from paper_2404_02950_b200 import sledge as S


def _fields(shape_zyx, dtype, seed):
    """two band-limited Gaussian random components on a 48^3 periodic grid (strings: lines where both vanish), repeated twice per axis and cropped
    to shape_zyx -- the crop's seam is not periodic, which only adds plaquettes with winding there"""
    nz, ny, nx = shape_zyx
    p1 = inputs.tile_periodic(inputs.grf(48, 0.25, seed, device="cuda"), 2)[:nz, :ny, :nx].to(dtype).contiguous()
    p2 = inputs.tile_periodic(inputs.grf(48, 0.25, seed + 1, device="cuda"), 2)[:nz, :ny, :nx].to(dtype).contiguous()
    return p1, p2


def _existing_path(p1, p2):
    nz, ny, nx = p1.shape
    s = S.Sledge((nx, ny, nz), nghost=1, blocking_factor=4, dtype="f64" if p1.dtype == torch.float64 else "f32")
    s.set_state(0, 0, p1)
    s.set_state(0, 1, p2)
    tags, counts = s.tag_strings(0)
    s.synchronize()
    out = tags.clone().view(nz, ny, nx), counts.clone()
    s.close()
    return out


@pytest.mark.gpu
def test_static_tagging_matches_the_context_path_on_calls_in_a_row():
    cases = [((48, 48, 48), torch.float64, 11), ((36, 24, 40), torch.float32, 23), ((72, 72, 72), torch.float64, 37),
             ((8, 52, 44), torch.float64, 41), ((48, 48, 48), torch.float64, 11)]
    want = [_existing_path(*_fields(shp, dt, seed)) for shp, dt, seed in cases]
    assert int((want[0][0] != 0).sum()) > 0 and int(want[0][1].sum()) > 0  # the fields do contain strings
    got = []
    for shp, dt, seed in cases:  # back to back on one stream, outputs preallocated by the caller
        p1, p2 = _fields(shp, dt, seed)
        nb = tuple((v + 31) // 32 for v in shp)
        tags = torch.full(shp, 255, dtype=torch.uint8, device="cuda")
        counts = torch.full(nb, -1, dtype=torch.int32, device="cuda")
        t, c = S.tag_strings_static(p1, p2, tags, counts)
        assert t.data_ptr() == tags.data_ptr() and c.data_ptr() == counts.data_ptr()
        got.append((tags, counts))
    torch.cuda.synchronize()
    for (wt, wc), (gt, gc) in zip(want, got):
        assert torch.equal(wt, gt)
        assert torch.equal(wc, gc)
    assert torch.equal(got[0][0], got[-1][0]) and torch.equal(got[0][1], got[-1][1])


@pytest.mark.gpu
def test_static_tagging_straight_string_exact_tags():
    """psi = (x - x0) + i (y - y0) with the zero inside a plaquette: exactly that xy plaquette column is tagged (plus the
    columns the periodic seam creates, which the context path sees identically)"""
    n = 16
    p1n, p2n = inputs.straight_string(n, 5.5, 9.5)
    p1 = torch.from_numpy(p1n).cuda().contiguous()
    p2 = torch.from_numpy(p2n).cuda().contiguous()
    tags, counts = S.tag_strings_static(p1, p2)
    wt, wc = _existing_path(p1, p2)
    torch.cuda.synchronize()
    assert torch.equal(tags, wt) and torch.equal(counts, wc)
    assert bool((tags[:, 9, 5] & 1).all())  # the plaquette whose lowest corner is (x, y) = (5, 9), every z


def test_static_tagging_rejects_what_does_not_fit():
    """the size check comes before any CUDA call: needs no GPU.  80^3 fp64 and 128^3 fp32 exceed the 8 MiB array."""
    import ctypes as C
    L = S.lib()
    fake = C.c_void_p(256)
    for n, dt in (((80, 80, 80), S.SLEDGE_F64), ((128, 128, 128), S.SLEDGE_F32)):
        rc = L.sledge_tag_strings_static(fake, fake, (C.c_int * 3)(*n), dt, None, None, None)
        assert rc == -1
        msg = L.sledge_last_error(None).decode()
        assert "static array holds 8388608" in msg and "SLEDGE_STATIC_SCRATCH_BYTES" in msg
    assert L.sledge_tag_strings_static(fake, fake, (C.c_int * 3)(1, 8, 8), S.SLEDGE_F64, None, None, None) == -1
    assert L.sledge_tag_strings_static(None, fake, (C.c_int * 3)(8, 8, 8), S.SLEDGE_F64, None, None, None) == -1
    assert L.sledge_tag_strings_static(fake, fake, (C.c_int * 3)(8, 8, 8), 7, None, None, None) == -1
