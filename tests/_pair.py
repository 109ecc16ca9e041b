"""Test helper: build the CPU oracle and the CUDA context for the same hierarchy and feed both the same
seeded initial data.  The two sides share nothing but these input arrays."""
import numpy as np
import torch

from oracle.oracle import Oracle
from paper_2404_02950_b200 import inputs
from paper_2404_02950_b200.sledge import Sledge


def make_pair(n0, boxes=None, n_levels=1, nghost=1, blocking_factor=8, lap_order=1, h0=1.0, lam=1.0, a_mass=0.0,
              friction=0.0, eta_fixed=False, dtype="f64", rk_dataflow="lean", ko_order=0, ko_strength=0.0,
              integrator=4, interp=0, gw=False, gw_coupling=0.0, gw_friction=0.0, rkn=None, shadow_level=False):
    o = Oracle(n0, boxes=boxes, n_levels=n_levels, nghost=nghost, blocking_factor=blocking_factor,
               lap_order=lap_order, h0=h0, lam=lam, a_mass=a_mass, friction=friction, eta_fixed=eta_fixed,
               ko_order=ko_order, ko_strength=ko_strength, integrator=integrator, interp=interp, gw=gw,
               gw_coupling=gw_coupling, gw_friction=gw_friction, rkn=rkn)
    s = Sledge(n0, boxes=boxes, n_levels=n_levels, nghost=nghost, blocking_factor=blocking_factor, dtype=dtype,
               lap_order=lap_order, h0=h0, lam=lam, a_mass=a_mass, friction=friction, eta_fixed=eta_fixed,
               rk_dataflow=rk_dataflow, ko_order=ko_order, ko_strength=ko_strength, integrator=integrator,
               interp=interp, gw=gw, gw_coupling=gw_coupling, gw_friction=gw_friction, rkn=rkn,
               shadow_level=shadow_level)
    return o, s


def set_both(o, s, ib, comp, arr):
    """arr: numpy float64 [z,y,x].  For an fp32 context the oracle starts from the fp32-rounded values
    (R15)."""
    t = torch.from_numpy(np.ascontiguousarray(arr)).to(s.tdtype)
    o.set_state(ib, comp, t.to(torch.float64).numpy())
    s.set_state(ib, comp, t.cuda().contiguous())


def smooth_field(shape_xyz_lo_hi, level, n0, seed, amp=1.0):
    """Smooth periodic test field evaluated at the cell centres of an index range of `level`: a few
    low Fourier modes with seeded amplitudes and phases (exactly periodic over the level-0 domain)."""
    lo, hi = shape_xyz_lo_hi
    rng = np.random.default_rng(seed)
    s = 1.0 / (1 << level)
    ax = [(np.arange(lo[d], hi[d] + 1) + 0.5) * s / n0[d] * 2 * np.pi for d in range(3)]
    X, Y, Z = ax[0][None, None, :], ax[1][None, :, None], ax[2][:, None, None]
    out = np.zeros((ax[2].size, ax[1].size, ax[0].size))
    for _ in range(6):
        k = rng.integers(-2, 3, size=3)
        a, ph = rng.normal(), rng.uniform(0, 2 * np.pi)
        out = out + a * np.cos(k[0] * X + k[1] * Y + k[2] * Z + ph)
    return amp * out


def init_smooth(o, s, n0, seed, comps=(0, 1, 2, 3), amp=1.0):
    if isinstance(n0, int):
        n0 = (n0,) * 3
    for ib, (l, lo, hi) in enumerate(s.boxes):
        for c in comps:
            set_both(o, s, ib, c, smooth_field((lo, hi), l, n0, seed * 10 + c, amp))


def init_grf(o, s, n, f, seeds):
    """Single-box level 0: psi1, psi2 band-limited GRFs (reading R17), Pi = 0."""
    for c, seed in enumerate(seeds):
        a = inputs.grf(n, f, seed).numpy()
        set_both(o, s, 0, c, a)
    z = np.zeros((n, n, n))
    set_both(o, s, 0, 2, z)
    set_both(o, s, 0, 3, z)


def max_err(o, s, comps=(0, 1, 2, 3), relative=False):
    """max over boxes/cells of |gpu - oracle| per component (relative: divided by max |oracle| of the comp)."""
    errs = []
    for c in comps:
        e, m = 0.0, 0.0
        for ib in range(len(s.boxes)):
            a = o.get_state(ib, c)
            b = s.get_state(ib, c).to(torch.float64).cpu().numpy()
            e = max(e, float(np.abs(a - b).max()))
            m = max(m, float(np.abs(a).max()))
        errs.append(e / m if relative and m > 0 else e)
    return max(errs)


def upload_oracle_state(o, s):
    """Make the GPU state a copy of the oracle's (for bit-exact tag comparison on the same input, R19)."""
    for ib in range(len(s.boxes)):
        for c in range(4):
            s.set_state(ib, c, torch.from_numpy(o.get_state(ib, c)).to(s.tdtype).cuda().contiguous())


def two_level_boxes(n0=32, bf=8):
    """Level 0: one box; level 1: an L-shaped set of boxes around the domain centre, nested with a gap of bf."""
    b = [(0, (0, 0, 0), (n0 - 1, n0 - 1, n0 - 1))]
    lo = n0 // 2  # fine index space is 2*n0; fine boxes between n0/2 and 3*n0/2
    b.append((1, (lo, lo, lo), (lo + 2 * bf - 1, lo + 2 * bf - 1, lo + bf - 1)))
    b.append((1, (lo + 2 * bf, lo, lo), (lo + 3 * bf - 1, lo + bf - 1, lo + bf - 1)))
    b.append((1, (lo, lo, lo + bf), (lo + bf - 1, lo + 2 * bf - 1, lo + 3 * bf - 1)))
    return b
