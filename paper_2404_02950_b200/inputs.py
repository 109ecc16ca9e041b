"""Seeded synthetic inputs shared by the CUDA path and the oracle's tests.

This module holds NONE of the method's arithmetic (no Laplacian, RHS, integrator, ghost fill, tagging
or averaging) -- only the recipes that manufacture initial data, box lists and run parameters with
the shapes / value distributions of the five BASELINE.json configs.  It imports neither the CUDA
binding nor the oracle, so both sides can be fed the very same arrays.

The paper's own initial states are HDF5 files that are not available; these
generators stand in for them.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np
import torch

# ---------------------------------------------------------------------------------------------
# run parameters of the five configs (BASELINE.json `configs`, SURVEY.md section 8(d) readings G12/G13)
# ---------------------------------------------------------------------------------------------


@dataclass
class Config:
    name: str
    n0: int
    dtype: str  # "f64" | "f32"
    h0: float
    lap_order: int  # paper's `order`: 1 -> 7-point, 2 -> 13-point
    dt: float
    eta0: float
    steps: int
    nghost: int
    grf_f: float = 0.0  # band limit as a fraction of k_Nyquist
    seeds: tuple = (0, 0)
    n_levels: int = 1
    blocking_factor: int = 8
    lam: float = 1.0
    tags_every_step: bool = False
    extra: dict = field(default_factory=dict)


CONFIGS = {
    # C1: h = 1, dt = 0.25, eta 1 -> 3.5
    "C1": Config("C1", 32, "f64", 1.0, 1, 0.25, 1.0, 10, 1, 0.25, (1001, 1002), tags_every_step=True),
    # C2: h = 0.125 (reading G12), dt = 0.25 h
    "C2": Config("C2", 256, "f64", 0.125, 1, 0.03125, 1.0, 100, 1, 0.1, (2001, 2002)),
    # C3: 13-point, dt = 0.2 h, tags + per-32^3 counts after every step
    "C3": Config("C3", 512, "f64", 0.125, 2, 0.025, 2.0, 50, 2, 0.1, (3001, 3002), tags_every_step=True),
    # C4: fp32, 1024^3
    "C4": Config("C4", 1024, "f32", 0.125, 1, 0.03125, 1.0, 20, 1, 0.05, (4001, 4002)),
    # C5: 3-level AMR, base 256^3, 32^3 boxes, blocking factor 8, 3 ghost cells, 13-point (reading G13)
    "C5": Config("C5", 256, "f64", 0.25, 2, 0.0625, 2.0, 20, 3, 0.0, (5000, 5000), n_levels=3,
                 extra=dict(n_rings=8, rmin=20.0, rmax=60.0, core_w=3.0, box=32, r1=8.0, r2=2.0)),
}


# ---------------------------------------------------------------------------------------------
# band-limited Gaussian random field (reading G17)
# ---------------------------------------------------------------------------------------------


def grf(n: int, f: float, seed: int, device: str = "cpu", dtype=torch.float64) -> torch.Tensor:
    """White N(0,1) noise (seeded) -> rfftn -> zero every mode with |k| >= f*k_Nyquist and the DC mode
    -> irfftn -> divide by the grid standard deviation.  Returned as [z, y, x]."""
    gen = torch.Generator(device="cpu")
    gen.manual_seed(int(seed))
    work = torch.float64 if dtype == torch.float64 else torch.float32
    if n <= 512:
        noise = torch.randn((n, n, n), generator=gen, dtype=work).to(device)
    else:  # large grids: generate plane by plane to bound host memory
        noise = torch.empty((n, n, n), dtype=work, device=device)
        for z in range(n):
            noise[z] = torch.randn((n, n), generator=gen, dtype=work).to(device)
    spec = torch.fft.rfftn(noise)
    del noise
    k1 = torch.fft.fftfreq(n, d=1.0 / n).to(device)  # integer mode numbers
    kx = torch.fft.rfftfreq(n, d=1.0 / n).to(device)
    kcut2 = (f * (n / 2.0)) ** 2
    for z in range(n):  # plane by plane: avoids a full-size |k|^2 temporary
        k2 = (k1[z] ** 2 + k1[:, None] ** 2) + kx[None, :] ** 2
        spec[z] = torch.where(k2 < kcut2, spec[z], torch.zeros((), dtype=spec.dtype, device=device))
    spec[0, 0, 0] = 0
    out = torch.fft.irfftn(spec, s=(n, n, n))
    del spec
    out = out / out.std(unbiased=False)
    return out.to(dtype)


def tile_periodic(a: torch.Tensor, reps: int) -> torch.Tensor:
    """Repeat a periodic cube `reps` times along every axis."""
    return a.repeat(reps, reps, reps)


def straight_string(n: int, x0: float, y0: float):
    """psi = (x - x0) + i (y - y0) on cell indices x, y in [0, n); returns (psi1, psi2) as [z, y, x] float64."""
    idx = np.arange(n, dtype=np.float64)
    psi1 = np.broadcast_to((idx - x0)[None, None, :], (n, n, n)).copy()
    psi2 = np.broadcast_to((idx - y0)[None, :, None], (n, n, n)).copy()
    return psi1, psi2


# ---------------------------------------------------------------------------------------------
# vortex rings (reading G14) and the box layout placed around them (BASELINE.json config 5)
# ---------------------------------------------------------------------------------------------


@dataclass
class Rings:
    centre: np.ndarray  # [n, 3] in coarse cells, (x, y, z)
    normal: np.ndarray  # [n, 3] unit vectors
    radius: np.ndarray  # [n] in coarse cells
    core_w: float  # core width in coarse cells
    n0: int


def make_rings(n0: int, n_rings: int, rmin: float, rmax: float, core_w: float, seed: int) -> Rings:
    rng = np.random.default_rng(seed)
    centre = rng.uniform(0.0, n0, size=(n_rings, 3))
    radius = rng.uniform(rmin, rmax, size=n_rings)
    v = rng.normal(size=(n_rings, 3))
    normal = v / np.linalg.norm(v, axis=1, keepdims=True)
    return Rings(centre, normal, radius, core_w, n0)


def ring_field(rings: Rings, level: int, lo, hi, device: str = "cpu"):
    """psi = prod_rings tanh(r/w) exp(i theta), theta = atan2(z, rho-R) - atan2(z, rho+R), evaluated at the
    cell centres of the inclusive index range lo..hi (x, y, z) of `level`.  Lengths are in coarse cells,
    displacements use the minimum image.  Returns (psi1, psi2) float64 tensors [z, y, x]."""
    s = 1.0 / (1 << level)
    ax = [(torch.arange(lo[d], hi[d] + 1, dtype=torch.float64, device=device) + 0.5) * s for d in range(3)]
    X = ax[0][None, None, :]
    Y = ax[1][None, :, None]
    Z = ax[2][:, None, None]
    L = float(rings.n0)
    re = torch.ones((ax[2].numel(), ax[1].numel(), ax[0].numel()), dtype=torch.float64, device=device)
    im = torch.zeros_like(re)
    for c, nrm, R in zip(rings.centre, rings.normal, rings.radius):
        dx = X - float(c[0])
        dy = Y - float(c[1])
        dz = Z - float(c[2])
        dx = dx - L * torch.round(dx / L)
        dy = dy - L * torch.round(dy / L)
        dz = dz - L * torch.round(dz / L)
        zeta = dx * float(nrm[0]) + dy * float(nrm[1]) + dz * float(nrm[2])
        px = dx - zeta * float(nrm[0])
        py = dy - zeta * float(nrm[1])
        pz = dz - zeta * float(nrm[2])
        rho = torch.sqrt(px * px + py * py + pz * pz)
        theta = torch.atan2(zeta, rho - float(R)) - torch.atan2(zeta, rho + float(R))
        r = torch.sqrt((rho - float(R)) ** 2 + zeta * zeta)
        mod = torch.tanh(r / rings.core_w)
        a = mod * torch.cos(theta)
        b = mod * torch.sin(theta)
        re, im = re * a - im * b, re * b + im * a
    return re, im


def _ring_points(rings: Rings, per_cell: float = 2.0):
    pts = []
    for c, nrm, R in zip(rings.centre, rings.normal, rings.radius):
        t = np.array([1.0, 0.0, 0.0]) if abs(nrm[0]) < 0.9 else np.array([0.0, 1.0, 0.0])
        e1 = np.cross(nrm, t)
        e1 /= np.linalg.norm(e1)
        e2 = np.cross(nrm, e1)
        m = max(16, int(math.ceil(2 * math.pi * R * per_cell)))
        ph = np.arange(m) * (2 * math.pi / m)
        pts.append(c[None, :] + R * (np.cos(ph)[:, None] * e1[None, :] + np.sin(ph)[:, None] * e2[None, :]))
    return np.concatenate(pts, axis=0)


def _tiles_near(points_lvl: np.ndarray, n_lvl: int, tile: int, r: float) -> np.ndarray:
    """Boolean [tz, ty, tx] map of aligned tiles whose box lies within distance r (level cells) of a point."""
    nt = n_lvl // tile
    near = np.zeros((nt, nt, nt), dtype=bool)
    for p in points_lvl:
        lo = np.floor((p - r) / tile).astype(int)
        hi = np.floor((p + r) / tile).astype(int)
        for tz in range(lo[2], hi[2] + 1):
            for ty in range(lo[1], hi[1] + 1):
                for tx in range(lo[0], hi[0] + 1):
                    t = np.array([tx, ty, tz])
                    blo = t * tile
                    d = np.maximum(np.maximum(blo - p, p - (blo + tile)), 0.0)
                    if float(np.sqrt((d * d).sum())) <= r:
                        near[tz % nt, ty % nt, tx % nt] = True
    return near


def _grow_tiles(mask: np.ndarray) -> np.ndarray:
    """Tiles touching a marked tile (26-neighbourhood, periodic)."""
    out = mask.copy()
    for dz in (-1, 0, 1):
        for dy in (-1, 0, 1):
            for dx in (-1, 0, 1):
                out |= np.roll(mask, (dz, dy, dx), axis=(0, 1, 2))
    return out


def amr_boxes_for_rings(rings: Rings, n_levels: int = 3, box: int = 32, r1: float = 8.0, r2: float = 2.0,
                        blocking_factor: int = 8, split0: bool = True):
    """Box list (level, lo, hi) for a hierarchy refined around the ring curves: level 0 = the whole domain
    (aligned `box`^3 tiles if split0, else one box); level l>0 = aligned `box`^3 tiles within r_l coarse cells of a ring curve.  Level l is then
    enlarged to contain every level l+1 tile grown by one blocking factor of fine cells, so that the list
    satisfies proper nesting.  Returns (boxes, coverage fractions per level)."""
    n0 = rings.n0
    pts = _ring_points(rings)
    radii = {1: r1, 2: r2}
    masks = {}
    for l in range(1, n_levels):
        r = radii.get(l, r2)
        masks[l] = _tiles_near(pts * (1 << l), n0 << l, box, r * (1 << l))
    for l in range(n_levels - 2, 0, -1):
        fine = masks[l + 1]
        # a fine tile grown by bf fine cells (= bf/2 cells of level l) touches at most the 26 neighbours of
        # its parent tile when bf/2 <= box; mark every level-l tile that such a grown fine tile overlaps.
        nt_f = fine.shape[0]
        need = np.zeros_like(masks[l])
        nt_c = need.shape[0]
        grow = blocking_factor // 2
        for tz, ty, tx in zip(*np.nonzero(fine)):
            lo = (np.array([tx, ty, tz]) * box) // 2 - grow
            hi = ((np.array([tx, ty, tz]) + 1) * box - 1) // 2 + grow
            for cz in range(lo[2] // box, hi[2] // box + 1):
                for cy in range(lo[1] // box, hi[1] // box + 1):
                    for cx in range(lo[0] // box, hi[0] // box + 1):
                        need[cz % nt_c, cy % nt_c, cx % nt_c] = True
        del nt_f
        masks[l] = masks[l] | need
    boxes = split_level0(n0, box) if split0 else [(0, (0, 0, 0), (n0 - 1, n0 - 1, n0 - 1))]
    cover = [1.0]
    for l in range(1, n_levels):
        m = masks[l]
        for tz, ty, tx in zip(*np.nonzero(m)):
            lo = (int(tx) * box, int(ty) * box, int(tz) * box)
            boxes.append((l, lo, (lo[0] + box - 1, lo[1] + box - 1, lo[2] + box - 1)))
        cover.append(float(m.mean()))
    return boxes, cover


def split_level0(n0: int, box: int):
    """Level-0 box list made of aligned box^3 tiles (exercises same-level ghost copies)."""
    out = []
    for z in range(0, n0, box):
        for y in range(0, n0, box):
            for x in range(0, n0, box):
                out.append((0, (x, y, z), (x + box - 1, y + box - 1, z + box - 1)))
    return out


# ---------------------------------------------------------------------------------------------
# seeded random hierarchies (tests): boxes of mixed sizes on every level, properly nested
# ---------------------------------------------------------------------------------------------


def _random_partition(rng, lo, hi, unit, min_units=1, p_stop=0.3):
    """Recursive bisection of the index range [lo, hi) (x, y, z; multiples of `unit`) into rectangles whose sides are
    multiples of `unit`: at every node either stop (probability p_stop) or cut a random axis at a random multiple."""
    ext = [(hi[d] - lo[d]) // unit for d in range(3)]
    axes = [d for d in range(3) if ext[d] >= 2 * min_units]
    if not axes or rng.random() < p_stop:
        return [(tuple(lo), tuple(hi))]
    d = int(rng.choice(axes))
    cut = lo[d] + unit * int(rng.integers(min_units, ext[d] - min_units + 1))
    hi1 = list(hi)
    hi1[d] = cut
    lo2 = list(lo)
    lo2[d] = cut
    return (_random_partition(rng, list(lo), hi1, unit, min_units, p_stop)
            + _random_partition(rng, lo2, list(hi), unit, min_units, p_stop))


def random_hierarchy(n0, n_levels: int, blocking_factor: int, seed: int, fill: float = 0.35):
    """Box list (level, lo, hi) of a random, valid hierarchy on the periodic domain n0 (int or (nx, ny, nz)):
    level 0 = a random partition of the whole domain; level l > 0 = a random set of blocking-factor cells (probability
    `fill`, grown so that it is not empty) cut down to proper nesting -- every cell of it, grown by one blocking factor,
    lies on level l-1 -- and then cut into rectangles by random bisection of its bounding boxes.
    Boxes of a level are disjoint; many share faces (the storage-box coalescing of the library) and many do not."""
    rng = np.random.default_rng(seed)
    n0 = (n0,) * 3 if isinstance(n0, int) else tuple(n0)
    bf = blocking_factor
    boxes = [(0, lo, tuple(h - 1 for h in hi)) for lo, hi in _random_partition(rng, [0, 0, 0], list(n0), bf, 1, 0.25)]
    prev = np.ones(tuple(n0[d] // bf for d in (2, 1, 0)), dtype=bool)  # [z, y, x] blocking cells of level l-1 that exist
    for l in range(1, n_levels):
        shape = tuple(2 * s for s in prev.shape)
        # fine blocking cells whose parent region grown by one fine blocking factor (= half a coarse blocking cell:
        # the parent cell and, on the side the child sits, its neighbour) is covered by level l-1
        ok = np.ones(shape, dtype=bool)
        up = np.repeat(np.repeat(np.repeat(prev, 2, 0), 2, 1), 2, 2)
        ok &= up
        for ax in range(3):
            for sh in (-1, 1):
                ok &= np.roll(up, sh, axis=ax)  # the neighbour fine cells' parents cover the grown region
        # corners: a grown box also touches the diagonal neighbours
        for dz in (-1, 0, 1):
            for dy in (-1, 0, 1):
                for dx in (-1, 0, 1):
                    ok &= np.roll(up, (dz, dy, dx), axis=(0, 1, 2))
        want = rng.random(shape) < fill
        # smooth the random set a little so that boxes larger than one cell appear
        want |= np.roll(want, 1, axis=int(rng.integers(0, 3)))
        mask = want & ok
        if not mask.any():
            idx = np.argwhere(ok)
            if len(idx) == 0:
                break
            z, y, x = idx[int(rng.integers(0, len(idx)))]
            mask[z, y, x] = True
        # cut the mask into rectangles: random bisection of the domain, keep leaves that are fully inside the mask,
        # recurse to single cells otherwise
        def emit(lo, hi):
            sub = mask[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]]
            if not sub.any():
                return []
            if sub.all() and rng.random() < 0.7:
                return [(l, tuple(bf * v for v in lo), tuple(bf * v - 1 for v in hi))]
            ext = [hi[d] - lo[d] for d in range(3)]
            axes = [d for d in range(3) if ext[d] >= 2]
            if not axes:
                return [(l, tuple(bf * v for v in lo), tuple(bf * v - 1 for v in hi))]
            d = int(rng.choice(axes))
            cut = lo[d] + int(rng.integers(1, ext[d]))
            hi1 = list(hi)
            hi1[d] = cut
            lo2 = list(lo)
            lo2[d] = cut
            return emit(list(lo), hi1) + emit(lo2, list(hi))
        boxes += emit([0, 0, 0], [shape[2], shape[1], shape[0]])
        prev = mask
    return boxes
