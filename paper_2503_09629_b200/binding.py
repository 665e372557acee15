"""Thin ctypes binding of libsubcycle.so — same names as include/subcycle.h, argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels; PyTorch is used for the device arena,
the stream and (by the callers) pinned host buffers. There is no CPU fallback: creating a hierarchy
without a usable GPU, or importing without a built library, fails loudly.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsubcycle.so")

SC_OK, SC_ERR_INVALID_ARG, SC_ERR_NESTING, SC_ERR_UNSUPPORTED, SC_ERR_OOM, SC_ERR_CUDA = 0, -1, -2, -3, -4, -5

EXPORTS = ["sc_arena_bytes", "sc_create_hierarchy", "sc_set_state", "sc_step", "sc_read_level", "sc_time",
           "sc_launch_count", "sc_debug_ghost_map", "sc_debug_read_padded", "sc_debug_read_slot", "sc_destroy",
           "sc_last_error", "sc_profile", "sc_profile_read", "sc_debug_max_abs", "sc_debug_graph_stats", "sc_debug_stream",
           "sc_max_abs_noalloc", "sc_debug_interp_weights"]


class sc_box(C.Structure):
    _fields_ = [("level", C.c_int32), ("lo", C.c_int32 * 3), ("n", C.c_int32 * 3)]


class sc_hierarchy_desc(C.Structure):
    _fields_ = [("nlevels", C.c_int32), ("nboxes", C.c_int32), ("boxes", C.POINTER(sc_box)),
                ("ref_ratio", C.c_int32), ("ghost", C.c_int32), ("nfields", C.c_int32),
                ("domain_cells", C.c_int32 * 3), ("xlo", C.c_double * 3), ("xhi", C.c_double * 3),
                ("coupling", C.POINTER(C.c_double)), ("arena", C.c_void_p), ("arena_bytes", C.c_uint64),
                ("cuda_stream", C.c_void_p), ("ko_sigma", C.c_double), ("fd_order", C.c_int32),
                ("ko_order", C.c_int32), ("integrator", C.c_int32), ("outer_bc", C.c_int32),
                ("interp_order", C.c_int32), ("centering", C.c_int32)]


class SubcycleError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libsubcycle error {code}: {msg}")
        self.code = code


_lib = None


def lib():
    """Load libsubcycle.so (built in-tree by paper_2503_09629_b200.build). Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2503_09629_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        H, dp = C.c_void_p, C.c_void_p  # data pointers are passed as raw addresses (host or device)
        L.sc_last_error.restype = C.c_char_p
        L.sc_arena_bytes.restype = C.c_uint64
        L.sc_arena_bytes.argtypes = [C.POINTER(sc_hierarchy_desc)]
        L.sc_create_hierarchy.restype = C.c_int32
        L.sc_create_hierarchy.argtypes = [C.POINTER(sc_hierarchy_desc), C.POINTER(H)]
        L.sc_set_state.restype = C.c_int32
        L.sc_set_state.argtypes = [H, C.c_int32, C.c_int32, C.c_int32, dp, C.c_int32]
        L.sc_step.restype = C.c_int32
        L.sc_step.argtypes = [H, C.c_double, C.c_int32]
        L.sc_read_level.restype = C.c_int32
        L.sc_read_level.argtypes = [H, C.c_int32, C.c_int32, C.c_int32, dp, C.c_int32]
        L.sc_time.restype = C.c_double
        L.sc_time.argtypes = [H]
        L.sc_launch_count.restype = C.c_uint64
        L.sc_launch_count.argtypes = [H]
        L.sc_debug_ghost_map.restype = C.c_int64
        L.sc_debug_ghost_map.argtypes = [H, C.c_int32, C.c_int32, C.c_void_p, C.c_uint64]
        L.sc_debug_read_padded.restype = C.c_int32
        L.sc_debug_read_padded.argtypes = [H, C.c_int32, C.c_int32, C.c_int32, dp]
        L.sc_debug_read_slot.restype = C.c_int32
        L.sc_debug_read_slot.argtypes = [H, C.c_int32, C.c_int32, C.c_int32, C.c_int32, dp]
        L.sc_debug_max_abs.restype = C.c_int32
        L.sc_debug_max_abs.argtypes = [H, C.c_int32, C.c_int32, C.c_int32, C.POINTER(C.c_double)]
        L.sc_debug_graph_stats.restype = C.c_int32
        L.sc_debug_graph_stats.argtypes = [H] + [C.POINTER(C.c_uint64)] * 4
        L.sc_debug_stream.restype = C.c_int32
        L.sc_debug_stream.argtypes = [H, C.c_int32, C.c_int32, C.c_uint64, C.POINTER(C.c_double)]
        L.sc_max_abs_noalloc.restype = C.c_int32
        L.sc_max_abs_noalloc.argtypes = [dp, C.c_uint64, dp, C.c_void_p]
        L.sc_debug_interp_weights.restype = C.c_int32
        L.sc_debug_interp_weights.argtypes = [C.c_int32, C.c_int32, C.POINTER(C.c_int32), C.POINTER(C.c_int32), dp, dp,
                                              C.POINTER(C.c_int32), C.POINTER(C.c_int32), dp]
        L.sc_destroy.restype = C.c_int32
        L.sc_destroy.argtypes = [H]
        L.sc_profile.restype = C.c_int32
        L.sc_profile.argtypes = [H, C.c_int32]
        L.sc_profile_read.restype = C.c_int32
        L.sc_profile_read.argtypes = [H, C.c_int32, C.POINTER(C.c_uint64), C.POINTER(C.c_double),
                                      C.POINTER(C.c_double)]
        _lib = L
    return _lib


def _check(rc: int):
    if rc < 0:
        raise SubcycleError(int(rc), lib().sc_last_error().decode())
    return rc


def make_desc(boxes, domain_cells, nfields=1, ghost=3, xlo=(-1.0, -1.0, -1.0), xhi=(1.0, 1.0, 1.0),
              coupling: Optional[np.ndarray] = None, ref_ratio: int = 2, nlevels: Optional[int] = None,
              ko_sigma: float = 0.0, fd_order: int = 4, ko_order: int = 0, integrator: int = 4, outer_bc: int = 0,
              interp: int = 0, vertex: int = 0):
    """Marshal a box list into an sc_hierarchy_desc. Returns (desc, keepalive)."""
    arr = (sc_box * len(boxes))()
    for i, b in enumerate(boxes):
        arr[i].level = b.level
        arr[i].lo[:] = list(b.lo)
        arr[i].n[:] = list(b.n)
    d = sc_hierarchy_desc()
    d.nlevels = (max(b.level for b in boxes) + 1) if nlevels is None else nlevels
    d.nboxes = len(boxes)
    d.boxes = arr
    d.ref_ratio, d.ghost, d.nfields = ref_ratio, ghost, nfields
    d.domain_cells[:] = list(domain_cells)
    d.xlo[:] = list(xlo)
    d.xhi[:] = list(xhi)
    d.ko_sigma = float(ko_sigma)
    d.fd_order = int(fd_order)
    d.ko_order, d.integrator, d.outer_bc = int(ko_order), int(integrator), int(outer_bc)
    d.interp_order, d.centering = int(interp), int(vertex)
    keep = [arr]
    if coupling is not None:
        cm = np.ascontiguousarray(coupling, dtype=np.float64)
        keep.append(cm)
        d.coupling = cm.ctypes.data_as(C.POINTER(C.c_double))
    return d, keep


def sc_arena_bytes(desc: sc_hierarchy_desc) -> int:
    n = lib().sc_arena_bytes(C.byref(desc))
    if n == 0:
        raise SubcycleError(SC_ERR_INVALID_ARG, lib().sc_last_error().decode())
    return int(n)


SC_NOALLOC_MAX_DOUBLES = 1 << 26


def sc_max_abs_noalloc(x, out, stream=None) -> None:
    """max |x| of a contiguous fp64 CUDA tensor into the one-element fp64 CUDA tensor `out`, NaN / inf reported as by
    Hierarchy.sc_debug_max_abs — but without a hierarchy and without any device allocation, for programs whose memory
    pool already owns the whole GPU or whose time loop cannot take cudaMalloc's device-wide synchronisation
    (include/subcycle.h). Asynchronous on `stream` (default: torch's current stream on x's device); at most
    SC_NOALLOC_MAX_DOUBLES elements; calls that may overlap on one GPU race on the library's built-in scratch array."""
    import torch

    assert x.is_cuda and out.is_cuda and x.device == out.device
    assert x.dtype == torch.float64 and out.dtype == torch.float64 and x.is_contiguous() and out.numel() == 1
    with torch.cuda.device(x.device):
        st = torch.cuda.current_stream() if stream is None else stream
        _check(lib().sc_max_abs_noalloc(x.data_ptr(), x.numel(), out.data_ptr(), st.cuda_stream))


def sc_debug_interp_weights(interp: int = 0, vertex: int = 0) -> dict:
    """The library's 1-D prolongation / restriction operators for these options (host only; include/subcycle.h)."""
    n = [C.c_int32() for _ in range(4)]
    w0, w1, r = (np.zeros(10) for _ in range(3))
    _check(lib().sc_debug_interp_weights(int(interp), int(vertex), C.byref(n[0]), C.byref(n[1]), w0.ctypes.data,
                                         w1.ctypes.data, C.byref(n[2]), C.byref(n[3]), r.ctypes.data))
    npts, pmin, nr, rmin = (int(x.value) for x in n)
    return {"np": npts, "pmin": pmin, "w": (w0[:npts].copy(), w1[:npts].copy()), "nr": nr, "rmin": rmin, "r": r[:nr].copy(),
            "tail": np.concatenate([w0[npts:], w1[npts:], r[nr:]])}


class Hierarchy:
    """A device-resident AMR hierarchy. Methods mirror the C calls one to one."""

    def __init__(self, boxes, domain_cells, nfields=1, ghost=3, xlo=(-1.0, -1.0, -1.0), xhi=(1.0, 1.0, 1.0),
                 coupling: Optional[np.ndarray] = None, device: str = "cuda:0", use_torch_arena: bool = True,
                 ko_sigma: float = 0.0, fd_order: int = 4, ko_order: int = 0, integrator: int = 4, outer_bc: int = 0,
                 interp: int = 0, vertex: int = 0):
        import torch  # device memory + stream only

        self._h = C.c_void_p()
        self.boxes = list(boxes)
        self.nfields, self.ghost = nfields, ghost
        desc, keep = make_desc(boxes, domain_cells, nfields, ghost, xlo, xhi, coupling, ko_sigma=ko_sigma, fd_order=fd_order,
                               ko_order=ko_order, integrator=integrator, outer_bc=outer_bc, interp=interp, vertex=vertex)
        self.nlevels = desc.nlevels
        self.arena_bytes = sc_arena_bytes(desc)
        if not torch.cuda.is_available():
            raise SubcycleError(SC_ERR_CUDA, "no CUDA device: libsubcycle has no CPU fallback")
        self._dev = torch.device(device)
        torch.cuda.set_device(self._dev)
        self._stream = torch.cuda.Stream(device=self._dev)
        self._arena = None
        if use_torch_arena:
            self._arena = torch.empty(self.arena_bytes + 256, dtype=torch.uint8, device=self._dev)
            ptr = (self._arena.data_ptr() + 255) // 256 * 256
            desc.arena, desc.arena_bytes = ptr, self.arena_bytes
        desc.cuda_stream = self._stream.cuda_stream
        _check(lib().sc_create_hierarchy(C.byref(desc), C.byref(self._h)))
        del keep

    @classmethod
    def from_workload(cls, w, **kw) -> "Hierarchy":
        kw.setdefault("ko_sigma", getattr(w, "ko_sigma", 0.0))
        kw.setdefault("fd_order", getattr(w, "fd_order", 4))
        for opt, default in (("ko_order", 0), ("integrator", 4), ("outer_bc", 0), ("interp", 0), ("vertex", 0)):
            kw.setdefault(opt, int(getattr(w, opt, default)))
        h = cls(w.boxes, w.domain_cells, w.nfields, w.ghost, w.xlo, w.xhi, w.coupling, **kw)
        for l in range(w.nlevels):
            for ib in range(len(w.level_boxes(l))):
                for c in range(w.ncomp):
                    h.sc_set_state(l, ib, c, w.initial_state(l, ib, c))
        return h

    # -- helpers ---------------------------------------------------------------------------------
    def _box(self, level: int, ibox: int):
        lb = [b for b in self.boxes if b.level == level]
        if not 0 <= ibox < len(lb):
            raise SubcycleError(SC_ERR_INVALID_ARG, f"no box {ibox} on level {level}")
        return lb[ibox]

    @property
    def stream(self):
        return self._stream

    @staticmethod
    def _ptr(a):
        """(address, on_device) of a numpy array or a torch tensor."""
        if isinstance(a, np.ndarray):
            assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
            return a.ctypes.data, 0
        assert a.dtype.is_floating_point and a.element_size() == 8 and a.is_contiguous()
        return a.data_ptr(), int(a.is_cuda)

    # -- the C calls -----------------------------------------------------------------------------
    def sc_set_state(self, level: int, ibox: int, comp: int, src) -> None:
        b = self._box(level, ibox)
        if isinstance(src, np.ndarray):
            src = np.ascontiguousarray(src, dtype=np.float64)
        nel = src.size if isinstance(src, np.ndarray) else src.numel()
        if nel != b.n[0] * b.n[1] * b.n[2]:
            raise ValueError("sc_set_state: src must hold n[0]*n[1]*n[2] doubles")
        p, dev = self._ptr(src)
        if dev:
            # device source: the copy kernel runs on the hierarchy's stream. Order it after the work that produced
            # `src` on the caller's current stream, and keep `src`'s memory from being recycled until it has run
            # (include/subcycle.h, sc_set_state: ordering contract for device pointers).
            import torch
            self._stream.wait_stream(torch.cuda.current_stream(self._dev))
        _check(lib().sc_set_state(self._h, level, ibox, comp, p, dev))
        if dev:
            src.record_stream(self._stream)

    def sc_step(self, dt_coarse: float, subcycling: bool = True) -> None:
        _check(lib().sc_step(self._h, float(dt_coarse), int(bool(subcycling))))

    def sc_read_level(self, level: int, ibox: int, comp: int, out=None):
        b = self._box(level, ibox)
        if out is None:
            out = np.empty((b.n[2], b.n[1], b.n[0]), dtype=np.float64)
        p, dev = self._ptr(out)
        if dev:  # `out` may still be in use on the caller's stream (sc_read_level itself synchronises ours)
            import torch
            self._stream.wait_stream(torch.cuda.current_stream(self._dev))
        _check(lib().sc_read_level(self._h, level, ibox, comp, p, dev))
        return out

    def sc_time(self) -> float:
        return lib().sc_time(self._h)

    def sc_launch_count(self) -> int:
        return int(lib().sc_launch_count(self._h))

    def sc_debug_ghost_map(self, level: int, ibox: int) -> np.ndarray:
        n = _check(lib().sc_debug_ghost_map(self._h, level, ibox, None, 0))
        out = np.empty((n, 7), dtype=np.int32)
        _check(lib().sc_debug_ghost_map(self._h, level, ibox, out.ctypes.data, out.size))
        return out

    def sc_debug_read_padded(self, level: int, ibox: int, comp: int) -> np.ndarray:
        b, g = self._box(level, ibox), self.ghost
        out = np.empty((b.n[2] + 2 * g, b.n[1] + 2 * g, b.n[0] + 2 * g), dtype=np.float64)
        _check(lib().sc_debug_read_padded(self._h, level, ibox, comp, out.ctypes.data))
        return out

    def sc_debug_max_abs(self, level: int, ibox: int, comp: int) -> float:
        out = C.c_double(0.0)
        _check(lib().sc_debug_max_abs(self._h, level, ibox, comp, C.byref(out)))
        return out.value

    def sc_debug_read_slot(self, level: int, ibox: int, slot: int, comp: int) -> np.ndarray:
        b = self._box(level, ibox)
        out = np.empty((b.n[2], b.n[1], b.n[0]), dtype=np.float64)
        _check(lib().sc_debug_read_slot(self._h, level, ibox, slot, comp, out.ctypes.data))
        return out

    def sc_debug_graph_stats(self) -> dict:
        v = [C.c_uint64() for _ in range(4)]
        _check(lib().sc_debug_graph_stats(self._h, *[C.byref(x) for x in v]))
        return dict(zip(("captures", "instantiations", "updates", "cached"), (int(x.value) for x in v)))

    def sc_debug_stream(self, nread: int, nwrite: int, ndoubles: int) -> float:
        """GB/s of a plain streaming kernel with `nread` arrays read and `nwrite` written (include/subcycle.h)."""
        out = C.c_double(0.0)
        _check(lib().sc_debug_stream(self._h, nread, nwrite, ndoubles, C.byref(out)))
        return out.value

    KERNEL_KINDS = ("rk_stage", "ghost_dense_prolong", "periodic_fill", "restrict")

    def sc_profile(self, enable: bool) -> None:
        _check(lib().sc_profile(self._h, int(bool(enable))))

    def sc_profile_read(self, kind: int):
        """(launches, total ms, total algorithmic bytes) of one kernel kind since sc_profile(True)."""
        n, ms, by = C.c_uint64(), C.c_double(), C.c_double()
        _check(lib().sc_profile_read(self._h, kind, C.byref(n), C.byref(ms), C.byref(by)))
        return int(n.value), float(ms.value), float(by.value)

    def synchronize(self) -> None:
        self._stream.synchronize()

    def sc_destroy(self) -> None:
        if getattr(self, "_h", None) and self._h.value:
            lib().sc_destroy(self._h)
            self._h = C.c_void_p()
        self._arena = None

    close = sc_destroy

    def __del__(self):
        try:
            self.sc_destroy()
        except Exception:
            pass
