"""ctypes loader for the CPU oracle (oracle/sledge_oracle.cpp) -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from paper_2404_02950_b200 and shares no code with the
CUDA path.  All arithmetic lives in the C++ file; this module only marshals numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sledge_oracle.cpp")
_LIB = os.path.join(_HERE, "libsledge_oracle.so")

FLAG_BLOCK = 32
COMPS = ("psi1", "psi2", "pi1", "pi2")
GW_COMPS = tuple(f"u_{ij}" for ij in ("xx", "yy", "zz", "xy", "xz", "yz")) + \
    tuple(f"du_{ij}" for ij in ("xx", "yy", "zz", "xy", "xz", "yz"))  # components 4..15 (L436)


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (no FMA contraction, OpenMP on outer loops)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


class _Params(C.Structure):
    _fields_ = [
        ("n_levels", C.c_int32),
        ("n0", C.c_int32 * 3),
        ("nghost", C.c_int32),
        ("blocking_factor", C.c_int32),
        ("lap_order", C.c_int32),
        ("eta_fixed", C.c_int32),
        ("h0", C.c_double),
        ("lam", C.c_double),
        ("a_mass", C.c_double),
        ("friction", C.c_double),
        ("ko_strength", C.c_double * 4),
        ("ko_order", C.c_int32),
        ("integrator", C.c_int32),
        ("interp", C.c_int32),
        ("gw", C.c_int32),
        ("gw_coupling", C.c_double),
        ("gw_friction", C.c_double),
        ("rkn_stages", C.c_int32),
        ("pad_", C.c_int32),
        ("rkn_c", C.c_double * 6),
        ("rkn_b", C.c_double * 6),
        ("rkn_bbar", C.c_double * 6),
        ("rkn_a", C.c_double * 21),
    ]


class _Box(C.Structure):
    _fields_ = [("level", C.c_int32), ("lo", C.c_int32 * 3), ("hi", C.c_int32 * 3)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.POINTER(_Params), C.POINTER(_Box), C.c_int]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_last_error.restype = C.c_char_p
        L.orc_last_error.argtypes = [C.c_void_p]
        dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
        L.orc_set_state.argtypes = [C.c_void_p, C.c_int, C.c_int, dp]
        L.orc_get_state.argtypes = [C.c_void_p, C.c_int, C.c_int, dp]
        L.orc_set_raw.argtypes = [C.c_void_p, C.c_int, C.c_int, dp]
        L.orc_get_raw.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, dp]
        L.orc_fill_ghosts.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.orc_eval_rhs.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_int]
        L.orc_rk_step.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.orc_average_down.argtypes = [C.c_void_p, C.c_int]
        L.orc_shadow_tee.argtypes = [C.c_void_p, C.c_double, C.c_double, C.POINTER(C.c_double), C.c_void_p, C.c_void_p]
        L.orc_tee_enable.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_double), C.c_void_p, C.c_void_p]
        L.orc_tag_strings.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.orc_plaquette_winding.argtypes = [dp, dp, dp, dp]
        L.orc_energy.argtypes = [C.c_void_p, C.c_double, dp]
        L.orc_omp_threads.restype = C.c_int
        L.orc_set_threads.argtypes = [C.c_int]
        _lib = L
    return _lib


def omp_threads() -> int:
    return int(lib().orc_omp_threads())


def set_threads(n: int) -> None:
    """OpenMP threads for the oracle's loops over boxes (timing only; results do not depend on it)."""
    lib().orc_set_threads(int(n))


def plaquette_winding(A, B, Cc, D) -> int:
    f = lambda v: np.ascontiguousarray(v, dtype=np.float64)
    return int(lib().orc_plaquette_winding(f(A), f(B), f(Cc), f(D)))


class OracleError(RuntimeError):
    pass


class Oracle:
    """The CPU oracle for one box hierarchy.

    boxes: sequence of (level, (lo_x, lo_y, lo_z), (hi_x, hi_y, hi_z)), inclusive cell ranges in the
    level's index space.  Arrays passed in/out are indexed [z, y, x] (x fastest), float64.
    """

    def __init__(self, n0, boxes=None, n_levels=1, nghost=1, blocking_factor=8, lap_order=1,
                 h0=1.0, lam=1.0, a_mass=0.0, friction=0.0, eta_fixed=False, ko_order=0, ko_strength=0.0,
                 integrator=4, interp=0, gw=False, gw_coupling=0.0, gw_friction=0.0, rkn=None):
        """rkn: for integrator 20, the user's Runge-Kutta-Nystrom tableau as a dict with `nodes` (c), `weights_b`,
        `weights_bar_b` (length s) and `tableau` (flattened lower triangle INCLUDING the diagonal, s(s+1)/2 values),
        the four arrays of Table V (L812-815)."""
        if np.isscalar(n0):
            n0 = (int(n0),) * 3
        if boxes is None:
            boxes = [(0, (0, 0, 0), (n0[0] - 1, n0[1] - 1, n0[2] - 1))]
        self.n0 = tuple(int(v) for v in n0)
        self.boxes = [(int(l), tuple(int(v) for v in lo), tuple(int(v) for v in hi)) for l, lo, hi in boxes]
        self.n_levels = int(n_levels)
        self.nghost = int(nghost)
        self.h0 = float(h0)
        p = _Params()
        p.n_levels = n_levels
        p.n0[:] = self.n0
        p.nghost = nghost
        p.blocking_factor = blocking_factor
        p.lap_order = lap_order
        p.eta_fixed = 1 if eta_fixed else 0
        p.h0 = h0
        p.lam = lam
        p.a_mass = a_mass
        p.friction = friction
        ks = (ko_strength,) * 4 if np.isscalar(ko_strength) else tuple(ko_strength)
        p.ko_strength[:] = [float(v) for v in ks]
        p.ko_order = ko_order
        p.integrator = integrator
        p.interp = interp
        p.gw = 1 if gw else 0
        p.gw_coupling = gw_coupling
        p.gw_friction = gw_friction
        self.ncomp = 16 if gw else 4
        if rkn is not None:
            st = len(rkn["nodes"])
            assert len(rkn["weights_b"]) == st and len(rkn["weights_bar_b"]) == st and len(rkn["tableau"]) == st * (st + 1) // 2
            p.rkn_stages = st
            p.rkn_c[:st] = [float(v) for v in rkn["nodes"]]
            p.rkn_b[:st] = [float(v) for v in rkn["weights_b"]]
            p.rkn_bbar[:st] = [float(v) for v in rkn["weights_bar_b"]]
            p.rkn_a[:st * (st + 1) // 2] = [float(v) for v in rkn["tableau"]]
        arr = (_Box * len(self.boxes))()
        for q, (l, lo, hi) in enumerate(self.boxes):
            arr[q].level = l
            arr[q].lo[:] = lo
            arr[q].hi[:] = hi
        self._h = lib().orc_create(C.byref(p), arr, len(self.boxes))
        if not self._h:
            raise OracleError(lib().orc_last_error(None).decode())

    def __del__(self):
        h = getattr(self, "_h", None)
        if h:
            lib().orc_destroy(h)
            self._h = None

    def _chk(self, rc):
        if rc != 0:
            raise OracleError(lib().orc_last_error(self._h).decode())

    def box_shape(self, ib):
        _, lo, hi = self.boxes[ib]
        return (hi[2] - lo[2] + 1, hi[1] - lo[1] + 1, hi[0] - lo[0] + 1)

    def level_boxes(self, level):
        return [q for q, b in enumerate(self.boxes) if b[0] == level]

    def set_state(self, ib, comp, arr):
        a = np.ascontiguousarray(arr, dtype=np.float64)
        assert a.shape == self.box_shape(ib), (a.shape, self.box_shape(ib))
        self._chk(lib().orc_set_state(self._h, ib, comp, a))

    def get_state(self, ib, comp):
        out = np.empty(self.box_shape(ib), dtype=np.float64)
        self._chk(lib().orc_get_state(self._h, ib, comp, out))
        return out

    def set_raw(self, ib, comp, arr):
        g = self.nghost
        shp = tuple(s + 2 * g for s in self.box_shape(ib))
        a = np.ascontiguousarray(arr, dtype=np.float64)
        assert a.shape == shp
        self._chk(lib().orc_set_raw(self._h, ib, comp, a))

    def get_raw(self, ib, comp, which=0):
        g = self.nghost
        shp = tuple(s + 2 * g for s in self.box_shape(ib))
        out = np.empty(shp, dtype=np.float64)
        self._chk(lib().orc_get_raw(self._h, ib, comp, which, out))
        return out

    def fill_ghosts(self, level, time=0.0):
        self._chk(lib().orc_fill_ghosts(self._h, level, time))

    def eval_rhs(self, level, eta, fill=True):
        """k = f(Y, eta); returns [k_psi1, k_psi2, k_pi1, k_pi2 (, k_u_xx .. k_du_yz)] for each box of the level
        (valid cells)."""
        self._chk(lib().orc_eval_rhs(self._h, level, eta, 1 if fill else 0))
        g = self.nghost
        out = []
        for ib in self.level_boxes(level):
            ks = []
            for c in range(self.ncomp):
                r = self.get_raw(ib, c, which=1)
                ks.append(r[g:-g, g:-g, g:-g].copy())
            out.append(ks)
        return out

    def rk_step(self, dt, eta):
        self._chk(lib().orc_rk_step(self._h, dt, eta))

    def average_down(self, fine_level):
        self._chk(lib().orc_average_down(self._h, fine_level))

    def tee_enable(self, fine_level, eps_psi1, eps_psi2, eps_pi1=np.inf, eps_pi2=np.inf):
        """O9: every later synchronisation of `fine_level` (average_down, also inside rk_step) writes truncation-error
        tags; read them with tee_tags(fine_level)."""
        ibs = self.level_boxes(fine_level)
        n = sum(int(np.prod(self.box_shape(ib))) for ib in ibs)
        if not hasattr(self, "_tee"):
            self._tee = {}
        tags = np.zeros(n, dtype=np.uint8)
        counts = np.zeros(self.count_shape(fine_level), dtype=np.uint32)
        self._tee[fine_level] = (tags, counts)
        eps = (C.c_double * 4)(eps_psi1, eps_psi2, eps_pi1, eps_pi2)
        self._chk(lib().orc_tee_enable(self._h, fine_level, eps, tags.ctypes.data, counts.ctypes.data))

    def shadow_tee(self, dt, eta, eps_psi1, eps_psi2, eps_pi1=np.inf, eps_pi2=np.inf):
        """O15 (L98): level-0 truncation-error tags against the shadow level.  Advances the hierarchy by TWO coarse
        steps of dt; returns (list of uint8 tag arrays [z,y,x], one per level-0 box; uint32 counts [bz,by,bx])."""
        ibs = self.level_boxes(0)
        sizes = [int(np.prod(self.box_shape(ib))) for ib in ibs]
        tags = np.zeros(sum(sizes), dtype=np.uint8)
        counts = np.zeros(self.count_shape(0), dtype=np.uint32)
        eps = (C.c_double * 4)(eps_psi1, eps_psi2, eps_pi1, eps_pi2)
        self._chk(lib().orc_shadow_tee(self._h, dt, eta, eps, tags.ctypes.data, counts.ctypes.data))
        out, off = [], 0
        for ib, s in zip(ibs, sizes):
            out.append(tags[off:off + s].reshape(self.box_shape(ib)).copy())
            off += s
        return out, counts

    def tee_tags(self, fine_level):
        """(list of uint8 tag arrays [z,y,x], one per box of the level; uint32 counts [bz,by,bx]) of the last sync."""
        tags, counts = self._tee[fine_level]
        out, off = [], 0
        for ib in self.level_boxes(fine_level):
            s = int(np.prod(self.box_shape(ib)))
            out.append(tags[off:off + s].reshape(self.box_shape(ib)).copy())
            off += s
        return out, counts.copy()

    def count_shape(self, level):
        return tuple((self.n0[d] * (1 << level) + FLAG_BLOCK - 1) // FLAG_BLOCK for d in (2, 1, 0))

    def tag_strings(self, level):
        """Returns (list of uint8 tag arrays [z,y,x], one per box of the level; uint32 counts [bz,by,bx])."""
        ibs = self.level_boxes(level)
        sizes = [int(np.prod(self.box_shape(ib))) for ib in ibs]
        tags = np.zeros(sum(sizes), dtype=np.uint8)
        counts = np.zeros(self.count_shape(level), dtype=np.uint32)
        self._chk(lib().orc_tag_strings(self._h, level, tags.ctypes.data, counts.ctypes.data))
        out, off = [], 0
        for ib, s in zip(ibs, sizes):
            out.append(tags[off:off + s].reshape(self.box_shape(ib)))
            off += s
        return out, counts

    def energy(self, eta):
        """Level-0 energies (kinetic, conserved-gradient, potential, Gradient<order>-gradient)."""
        out = np.zeros(4, dtype=np.float64)
        self._chk(lib().orc_energy(self._h, eta, out))
        return out
