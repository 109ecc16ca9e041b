"""ctypes binding of libsledge.so (include/sledge.h) -- argument marshalling only.

Every step of the path (ghost fill, fused Laplacian + potential + RK stage, string tagging, box-flag
reduction, average-down) runs in the CUDA kernels of the library.  PyTorch is used for device memory (the
arena and the dense in/out arrays) and for the stream.  There is NO CPU fallback: loading fails loudly
if libsledge.so is missing, and `Sledge(...)` fails if no CUDA device is present.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libsledge.so")

SLEDGE_F32, SLEDGE_F64 = 0, 1
SLEDGE_RK_LEAN, SLEDGE_RK_CLASSIC, SLEDGE_RK_FUSED, SLEDGE_RK_FUSED3 = 0, 1, 2, 3
KIND_STAGE, KIND_GHOST, KIND_TAG, KIND_AVG = 0, 1, 2, 3
COUNT_BLOCK = 32

SYMBOLS = [
    "sledge_arena_bytes", "sledge_create", "sledge_destroy", "sledge_set_state", "sledge_get_state",
    "sledge_set_state_host", "sledge_get_state_host", "sledge_host_copies_join", "sledge_get_ghosted", "sledge_fill_ghosts",
    "sledge_rk_stage", "sledge_rk_step", "sledge_tag_strings", "sledge_average_down", "sledge_tee_enable",
    "sledge_shadow_tee", "sledge_level_cells", "sledge_level_storage", "sledge_level_dataflow", "sledge_tag_strings_static",
    "sledge_launch_count", "sledge_synchronize", "sledge_profile_enable", "sledge_profile_read",
    "sledge_last_error",
]


class SledgeError(RuntimeError):
    pass


class sledge_box(C.Structure):
    _fields_ = [("level", C.c_int32), ("lo", C.c_int32 * 3), ("hi", C.c_int32 * 3)]


class sledge_params(C.Structure):
    _fields_ = [
        ("n_levels", C.c_int32), ("n0", C.c_int32 * 3), ("nghost", C.c_int32), ("blocking_factor", C.c_int32),
        ("dtype", C.c_int32), ("lap_order", C.c_int32), ("eta_fixed", C.c_int32), ("rk_dataflow", C.c_int32),
        ("h0", C.c_double), ("lam", C.c_double), ("a_mass", C.c_double), ("friction", C.c_double),
        ("ko_strength", C.c_double * 4), ("ko_order", C.c_int32), ("integrator", C.c_int32),
        ("interp", C.c_int32), ("shadow_level", C.c_int32), ("gw", C.c_int32), ("rkn_stages", C.c_int32),
        ("gw_coupling", C.c_double), ("gw_friction", C.c_double),
        ("rkn_nodes", C.c_double * 6), ("rkn_weights_b", C.c_double * 6), ("rkn_weights_bar_b", C.c_double * 6),
        ("rkn_tableau", C.c_double * 21),
    ]


_lib = None


def lib():
    """Load libsledge.so (built in-tree by paper_2404_02950_b200.build); never falls back to anything else."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise SledgeError(f"{LIB_PATH} is missing: run `python -m paper_2404_02950_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i, d = C.c_void_p, C.c_int, C.c_double
        L.sledge_arena_bytes.argtypes = [C.POINTER(sledge_params), C.POINTER(sledge_box), i, C.POINTER(C.c_size_t)]
        L.sledge_create.argtypes = [C.POINTER(vp), C.POINTER(sledge_params), C.POINTER(sledge_box), i, vp, C.c_size_t, vp]
        L.sledge_destroy.argtypes = [vp]
        for name in ("sledge_set_state", "sledge_get_state", "sledge_set_state_host", "sledge_get_state_host",
                     "sledge_get_ghosted"):
            getattr(L, name).argtypes = [vp, i, i, vp]
        L.sledge_host_copies_join.argtypes = [vp]
        L.sledge_fill_ghosts.argtypes = [vp, i, d]
        L.sledge_rk_stage.argtypes = [vp, i, i, d, d]
        L.sledge_rk_step.argtypes = [vp, d, d]
        L.sledge_tag_strings.argtypes = [vp, i, vp, vp]
        L.sledge_tag_strings_static.argtypes = [vp, vp, C.POINTER(C.c_int), i, vp, vp, vp]
        L.sledge_average_down.argtypes = [vp, i]
        L.sledge_tee_enable.argtypes = [vp, i, C.POINTER(C.c_double), vp, vp]
        L.sledge_shadow_tee.argtypes = [vp, d, d, C.POINTER(C.c_double), vp, vp]
        L.sledge_level_cells.argtypes = [vp, i, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        L.sledge_level_storage.argtypes = [vp, i, C.POINTER(C.c_int), C.POINTER(C.c_int64)]
        L.sledge_level_dataflow.argtypes = [vp, i, C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.sledge_launch_count.argtypes = [vp]
        L.sledge_launch_count.restype = C.c_int64
        L.sledge_synchronize.argtypes = [vp]
        L.sledge_profile_enable.argtypes = [vp, i]
        L.sledge_profile_read.argtypes = [vp, i, C.POINTER(C.c_int64), C.POINTER(d)]
        L.sledge_last_error.argtypes = [vp]
        L.sledge_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def _marshal(n0, boxes, n_levels, nghost, blocking_factor, dtype, lap_order, h0, lam, a_mass, friction, eta_fixed,
             rk_dataflow, ko_order=0, ko_strength=0.0, integrator=4, interp=0, shadow_level=False, gw=False,
             gw_coupling=0.0, gw_friction=0.0, rkn=None):
    if isinstance(n0, int):
        n0 = (n0,) * 3
    if boxes is None:
        boxes = [(0, (0, 0, 0), (n0[0] - 1, n0[1] - 1, n0[2] - 1))]
    p = sledge_params()
    p.n_levels = n_levels
    p.n0[:] = [int(v) for v in n0]
    p.nghost = nghost
    p.blocking_factor = blocking_factor
    p.dtype = {"f32": SLEDGE_F32, "f64": SLEDGE_F64}[dtype]
    p.lap_order = lap_order
    p.eta_fixed = 1 if eta_fixed else 0
    p.rk_dataflow = {"lean": SLEDGE_RK_LEAN, "classic": SLEDGE_RK_CLASSIC, "fused": SLEDGE_RK_FUSED,
                     "fused3": SLEDGE_RK_FUSED3}[rk_dataflow]
    p.h0, p.lam, p.a_mass, p.friction = h0, lam, a_mass, friction
    ks = (ko_strength,) * 4 if isinstance(ko_strength, (int, float)) else tuple(ko_strength)
    p.ko_strength[:] = [float(v) for v in ks]
    p.ko_order = ko_order
    p.integrator = integrator
    p.interp = interp
    p.shadow_level = 1 if shadow_level else 0
    p.gw = 1 if gw else 0
    p.gw_coupling, p.gw_friction = float(gw_coupling), float(gw_friction)
    if rkn is not None:  # the four arrays of Table V (L812-815), passed through unchanged
        st = len(rkn["nodes"])
        p.rkn_stages = st
        p.rkn_nodes[:st] = [float(v) for v in rkn["nodes"]]
        p.rkn_weights_b[:st] = [float(v) for v in rkn["weights_b"]]
        p.rkn_weights_bar_b[:st] = [float(v) for v in rkn["weights_bar_b"]]
        p.rkn_tableau[:len(rkn["tableau"])] = [float(v) for v in rkn["tableau"]]
    arr = (sledge_box * len(boxes))()
    for q, (l, lo, hi) in enumerate(boxes):
        arr[q].level = int(l)
        arr[q].lo[:] = [int(v) for v in lo]
        arr[q].hi[:] = [int(v) for v in hi]
    return p, arr, list(boxes), tuple(int(v) for v in n0)


def sledge_arena_bytes(n0, boxes=None, n_levels=1, nghost=1, blocking_factor=8, dtype="f64", lap_order=1, h0=1.0,
                       lam=1.0, a_mass=0.0, friction=0.0, eta_fixed=False, rk_dataflow="lean", ko_order=0,
                       ko_strength=0.0, integrator=4, interp=0, shadow_level=False, gw=False, gw_coupling=0.0,
                       gw_friction=0.0, rkn=None) -> int:
    """Host-only: validates the parameters and the box list and returns the arena size (needs no GPU)."""
    p, arr, boxes, _ = _marshal(n0, boxes, n_levels, nghost, blocking_factor, dtype, lap_order, h0, lam, a_mass,
                                friction, eta_fixed, rk_dataflow, ko_order, ko_strength, integrator, interp,
                                shadow_level, gw, gw_coupling, gw_friction, rkn)
    out = C.c_size_t(0)
    rc = lib().sledge_arena_bytes(C.byref(p), arr, len(boxes), C.byref(out))
    if rc != 0:
        raise SledgeError(f"sledge_arena_bytes: {rc}: {lib().sledge_last_error(None).decode()}")
    return int(out.value)


STATIC_SCRATCH_BYTES = 8 << 20  # SLEDGE_STATIC_SCRATCH_BYTES of include/sledge.h


def tag_strings_static(psi1: torch.Tensor, psi2: torch.Tensor, tags: torch.Tensor | None = None,
                       counts: torch.Tensor | None = None, stream=None):
    """sledge_tag_strings_static: string tags of ONE periodic box given as two dense CUDA tensors [z, y, x] (fp32 or
    fp64), with no context and no arena -- the library allocates nothing (its scratch is a static device array of
    8 MiB: up to 72^3 in fp64, 88^3 in fp32).  Pass `tags` (uint8 [z, y, x]) and `counts` (int32 [bz, by, bx], 32^3
    blocks) to keep this call free of allocations too; tensors created here are the binding's, not the library's.
    Calls that may overlap on the GPU share the scratch array and race: keep them on one stream."""
    if psi1.shape != psi2.shape or psi1.dim() != 3 or psi1.dtype != psi2.dtype or not psi1.is_cuda or not psi2.is_cuda:
        raise SledgeError("tag_strings_static: psi1, psi2 must be CUDA tensors [z, y, x] of the same shape and dtype")
    if not (psi1.is_contiguous() and psi2.is_contiguous()):
        raise SledgeError("tag_strings_static: dense contiguous tensors expected")
    if psi1.dtype not in (torch.float32, torch.float64):
        raise SledgeError("tag_strings_static: fp32 or fp64 only")
    nz, ny, nx = (int(v) for v in psi1.shape)
    nb = tuple((v + COUNT_BLOCK - 1) // COUNT_BLOCK for v in (nz, ny, nx))
    if tags is None:
        tags = torch.empty((nz, ny, nx), dtype=torch.uint8, device=psi1.device)
    if counts is None:
        counts = torch.empty(nb, dtype=torch.int32, device=psi1.device)
    if tags.numel() != nz * ny * nx or tags.dtype != torch.uint8 or counts.numel() != nb[0] * nb[1] * nb[2] \
            or counts.dtype != torch.int32 or not tags.is_contiguous() or not counts.is_contiguous():
        raise SledgeError("tag_strings_static: tags must be uint8 [z, y, x], counts int32 [ceil(n/32)] per axis")
    n = (C.c_int * 3)(nx, ny, nz)
    st = torch.cuda.current_stream(psi1.device) if stream is None else stream
    rc = lib().sledge_tag_strings_static(psi1.data_ptr(), psi2.data_ptr(), n,
                                         SLEDGE_F64 if psi1.dtype == torch.float64 else SLEDGE_F32,
                                         tags.data_ptr(), counts.data_ptr(), st.cuda_stream)
    if rc != 0:
        raise SledgeError(f"sledge_tag_strings_static: {rc}: {lib().sledge_last_error(None).decode()}")
    return tags, counts


class Sledge:
    """One context = one box hierarchy on one GPU.  Method names follow the C ABI (sledge_<name>).

    boxes: sequence of (level, (lo_x, lo_y, lo_z), (hi_x, hi_y, hi_z)), inclusive, level index space.
    Dense arrays are torch CUDA tensors indexed [z, y, x] (x fastest) of the context's dtype.
    """

    def __init__(self, n0, boxes=None, n_levels=1, nghost=1, blocking_factor=8, dtype="f64", lap_order=1, h0=1.0,
                 lam=1.0, a_mass=0.0, friction=0.0, eta_fixed=False, rk_dataflow="lean", ko_order=0, ko_strength=0.0,
                 integrator=4, interp=0, shadow_level=False, gw=False, gw_coupling=0.0, gw_friction=0.0, rkn=None,
                 device="cuda:0"):
        self._h = None
        L = lib()
        if not torch.cuda.is_available():
            raise SledgeError("no CUDA device: the sledge path has no CPU fallback")
        p, arr, self.boxes, self.n0 = _marshal(n0, boxes, n_levels, nghost, blocking_factor, dtype, lap_order, h0, lam,
                                               a_mass, friction, eta_fixed, rk_dataflow, ko_order, ko_strength,
                                               integrator, interp, shadow_level, gw, gw_coupling, gw_friction, rkn)
        self.n_levels, self.nghost, self.dtype = n_levels, nghost, dtype
        self.ncomp = 16 if gw else 4
        self.tdtype = torch.float64 if dtype == "f64" else torch.float32
        self.device = torch.device(device)
        nbytes = C.c_size_t(0)
        rc = L.sledge_arena_bytes(C.byref(p), arr, len(self.boxes), C.byref(nbytes))
        if rc != 0:
            raise SledgeError(f"sledge_arena_bytes: {rc}: {L.sledge_last_error(None).decode()}")
        self.arena_bytes = int(nbytes.value)
        torch.cuda.set_device(self.device)
        self.arena = torch.empty(self.arena_bytes + 256, dtype=torch.uint8, device=self.device)
        base = self.arena.data_ptr()
        self._arena_ptr = (base + 255) // 256 * 256
        self.stream = torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        rc = L.sledge_create(C.byref(h), C.byref(p), arr, len(self.boxes), self._arena_ptr, self.arena_bytes,
                             self.stream.cuda_stream)
        if rc != 0:
            raise SledgeError(f"sledge_create: {rc}: {L.sledge_last_error(None).decode()}")
        self._h = h

    # -- helpers ---------------------------------------------------------------------------------
    def _chk(self, rc, what):
        if rc != 0:
            raise SledgeError(f"{what}: {rc}: {lib().sledge_last_error(self._h).decode()}")

    def close(self):
        if self._h is not None:
            lib().sledge_destroy(self._h)
            self._h = None
            self.arena = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def box_shape(self, ib, ghosts=False):
        _, lo, hi = self.boxes[ib]
        e = 2 * self.nghost if ghosts else 0
        return (hi[2] - lo[2] + 1 + e, hi[1] - lo[1] + 1 + e, hi[0] - lo[0] + 1 + e)

    def level_boxes(self, level):
        return [q for q, b in enumerate(self.boxes) if b[0] == level]

    def level_cells(self, level):
        v, b = C.c_int64(0), C.c_int64(0)
        self._chk(lib().sledge_level_cells(self._h, level, C.byref(v), C.byref(b)), "sledge_level_cells")
        return int(v.value), int(b.value)

    def level_storage(self, level):
        """(storage boxes the level's caller boxes were coalesced into, stored cells per plane of one state buffer)"""
        n, w = C.c_int(0), C.c_int64(0)
        self._chk(lib().sledge_level_storage(self._h, level, C.byref(n), C.byref(w)), "sledge_level_storage")
        return int(n.value), int(w.value)

    def level_dataflow(self, level):
        """(K1 launches per step of the level, algorithmic words per cell-step of those launches)"""
        n, w = C.c_int(0), C.c_int(0)
        self._chk(lib().sledge_level_dataflow(self._h, level, C.byref(n), C.byref(w)), "sledge_level_dataflow")
        return int(n.value), int(w.value)

    def count_shape(self, level):
        return tuple((self.n0[d] * (1 << level) + COUNT_BLOCK - 1) // COUNT_BLOCK for d in (2, 1, 0))

    # -- the ABI ----------------------------------------------------------------------------------
    def set_state(self, ib, comp, t: torch.Tensor):
        assert t.is_cuda and t.dtype == self.tdtype and t.is_contiguous() and tuple(t.shape) == self.box_shape(ib)
        self._chk(lib().sledge_set_state(self._h, ib, comp, t.data_ptr()), "sledge_set_state")

    def get_state(self, ib, comp) -> torch.Tensor:
        out = torch.empty(self.box_shape(ib), dtype=self.tdtype, device=self.device)
        self._chk(lib().sledge_get_state(self._h, ib, comp, out.data_ptr()), "sledge_get_state")
        return out

    def set_state_host(self, ib, comp, t: torch.Tensor):
        assert (not t.is_cuda) and t.dtype == self.tdtype and t.is_contiguous() and tuple(t.shape) == self.box_shape(ib)
        self._chk(lib().sledge_set_state_host(self._h, ib, comp, t.data_ptr()), "sledge_set_state_host")

    def get_state_host(self, ib, comp, out: torch.Tensor):
        assert (not out.is_cuda) and out.dtype == self.tdtype and out.is_contiguous()
        assert tuple(out.shape) == self.box_shape(ib)
        self._chk(lib().sledge_get_state_host(self._h, ib, comp, out.data_ptr()), "sledge_get_state_host")
        return out

    def host_copies_join(self):
        self._chk(lib().sledge_host_copies_join(self._h), "sledge_host_copies_join")

    def get_ghosted(self, ib, comp) -> torch.Tensor:
        out = torch.empty(self.box_shape(ib, ghosts=True), dtype=self.tdtype, device=self.device)
        self._chk(lib().sledge_get_ghosted(self._h, ib, comp, out.data_ptr()), "sledge_get_ghosted")
        return out

    def fill_ghosts(self, level, time=0.0):
        self._chk(lib().sledge_fill_ghosts(self._h, level, float(time)), "sledge_fill_ghosts")

    def rk_stage(self, level, stage, dt, eta):
        self._chk(lib().sledge_rk_stage(self._h, level, stage, float(dt), float(eta)), "sledge_rk_stage")

    def rk_step(self, dt, eta):
        self._chk(lib().sledge_rk_step(self._h, float(dt), float(eta)), "sledge_rk_step")

    def tag_strings(self, level, tags: torch.Tensor | None = None, counts: torch.Tensor | None = None,
                    want_tags=True, want_counts=True):
        """Returns (tags uint8 [valid cells of the level, boxes back to back], counts int32 [bz, by, bx])."""
        ncell, _ = self.level_cells(level)
        if tags is None and want_tags:
            tags = torch.empty(ncell, dtype=torch.uint8, device=self.device)
        if counts is None and want_counts:
            counts = torch.empty(self.count_shape(level), dtype=torch.int32, device=self.device)
        self._chk(lib().sledge_tag_strings(self._h, level, tags.data_ptr() if tags is not None else None,
                                           counts.data_ptr() if counts is not None else None), "sledge_tag_strings")
        return tags, counts

    def split_tags(self, level, tags: torch.Tensor):
        out, off = [], 0
        for ib in self.level_boxes(level):
            shp = self.box_shape(ib)
            n = shp[0] * shp[1] * shp[2]
            out.append(tags[off:off + n].view(shp))
            off += n
        return out

    def average_down(self, fine_level):
        self._chk(lib().sledge_average_down(self._h, fine_level), "sledge_average_down")

    def tee_enable(self, fine_level, eps_psi1, eps_psi2, eps_pi1=float("inf"), eps_pi2=float("inf"),
                   tags: torch.Tensor | None = None, counts: torch.Tensor | None = None):
        """sledge_tee_enable: every later synchronisation of `fine_level` writes truncation-error tags into the
        returned (tags uint8 [valid cells of the level], counts int32 [bz, by, bx]) tensors, which this object
        keeps alive."""
        ncell, _ = self.level_cells(fine_level)
        if tags is None:
            tags = torch.zeros(ncell, dtype=torch.uint8, device=self.device)
        if counts is None:
            counts = torch.zeros(self.count_shape(fine_level), dtype=torch.int32, device=self.device)
        eps = (C.c_double * 4)(float(eps_psi1), float(eps_psi2), float(eps_pi1), float(eps_pi2))
        self._chk(lib().sledge_tee_enable(self._h, fine_level, eps, tags.data_ptr(), counts.data_ptr()),
                  "sledge_tee_enable")
        if not hasattr(self, "_tee"):
            self._tee = {}
        self._tee[fine_level] = (tags, counts)
        return tags, counts

    def shadow_tee(self, dt, eta, eps_psi1, eps_psi2, eps_pi1=float("inf"), eps_pi2=float("inf"),
                   tags: torch.Tensor | None = None, counts: torch.Tensor | None = None):
        """sledge_shadow_tee: level-0 truncation-error tags through the shadow level (L98); advances the hierarchy by
        two coarse steps of dt.  Returns (tags uint8 [valid level-0 cells], counts int32 [bz, by, bx])."""
        ncell, _ = self.level_cells(0)
        if tags is None:
            tags = torch.zeros(ncell, dtype=torch.uint8, device=self.device)
        if counts is None:
            counts = torch.zeros(self.count_shape(0), dtype=torch.int32, device=self.device)
        eps = (C.c_double * 4)(float(eps_psi1), float(eps_psi2), float(eps_pi1), float(eps_pi2))
        self._chk(lib().sledge_shadow_tee(self._h, float(dt), float(eta), eps, tags.data_ptr(), counts.data_ptr()),
                  "sledge_shadow_tee")
        return tags, counts

    def synchronize(self):
        self._chk(lib().sledge_synchronize(self._h), "sledge_synchronize")

    def launch_count(self) -> int:
        return int(lib().sledge_launch_count(self._h))

    def profile_enable(self, on=True):
        self._chk(lib().sledge_profile_enable(self._h, 1 if on else 0), "sledge_profile_enable")

    def profile_read(self, kind):
        n, ms = C.c_int64(0), C.c_double(0.0)
        self._chk(lib().sledge_profile_read(self._h, kind, C.byref(n), C.byref(ms)), "sledge_profile_read")
        return int(n.value), float(ms.value)
