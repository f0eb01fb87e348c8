"""Thin ctypes binding over the C-ABI library libqld.so (include/qld.h).

Argument marshalling only: every step of the hot path (tables, ingest, sums, finalise) runs in the CUDA
kernels behind the C calls.  PyTorch is used for device memory (the workspace, map views), pinned host
buffers and stream handles.  There is no CPU fallback: importing this module without the built library,
or creating a context without a CUDA device, raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

_PKG = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_PKG, "libqld.so")

QLD_U8, QLD_U16, QLD_U16_BE = 0, 1, 2
QLD_OK, QLD_E_INVAL, QLD_E_NOMEM, QLD_E_CUDA, QLD_E_STATE, QLD_E_OVERRUN, QLD_E_UNSUPPORTED = 0, -1, -2, -3, -4, -5, -6
QLD_ACC_AUTO, QLD_ACC_FP32, QLD_ACC_INT_BINS, QLD_ACC_FIXED, QLD_ACC_INT_REFS = 0, 1, 2, 3, 4
QLD_NORM_PAPER, QLD_NORM_AMPLITUDE = 0, 1
QLD_WHOLE, QLD_SLIDE = 0, 1
QLD_MAP_I, QLD_MAP_Q, QLD_MAP_AMP, QLD_MAP_PHASE, QLD_MAP_ALL, QLD_MAP_SUMS_I64 = 1, 2, 4, 8, 15, 16
_STATUS = {0: "QLD_OK", -1: "QLD_E_INVAL", -2: "QLD_E_NOMEM", -3: "QLD_E_CUDA", -4: "QLD_E_STATE", -5: "QLD_E_OVERRUN",
           -6: "QLD_E_UNSUPPORTED"}

# every symbol include/qld.h declares (tests check that the library exports each of them)
EXPORTS = ["qld_workspace_bytes", "qld_create", "qld_push_frames", "qld_push_frames_device", "qld_attach_frames_device",
           "qld_commit_frames", "qld_push_done", "qld_demod", "qld_get_maps", "qld_get_bins", "qld_read_map", "qld_read_ref_table", "qld_set_ref_tables",
           "qld_set_ref_table_fixed", "qld_read_ref_table_fixed", "qld_get_sums_i64", "qld_counters", "qld_sync", "qld_reset", "qld_destroy", "qld_last_error", "qld_kernel_launches", "qld_accum_mode", "qld_last_kernel", "qld_debug_set_tile",
           "qld_cnr", "qld_dominant_bin", "qld_dominant_bin_static", "qld_dominant_bin_static_bytes", "qld_dominant_bin_static_error",
           "qld_display_map", "qld_synth_fill", "qld_probe_read"]


class qld_ref(C.Structure):
    _fields_ = [("nu", C.c_double), ("phase", C.c_double), ("num", C.c_int64), ("den", C.c_int64),
                ("phase_quarter", C.c_int32), ("reserved", C.c_int32)]


class qld_config(C.Structure):
    _fields_ = [("H", C.c_int32), ("W", C.c_int32), ("dtype", C.c_int32), ("N", C.c_int32), ("K", C.c_int32),
                ("refs", C.POINTER(qld_ref)), ("ring_frames", C.c_int32), ("accum", C.c_int32), ("norm", C.c_int32),
                ("maps", C.c_int32), ("max_value", C.c_uint32), ("resync_hops", C.c_int32), ("external_store", C.c_int32),
                ("slide_hop", C.c_int32), ("window_relative", C.c_int32), ("reserved2", C.c_int32), ("ref_tables_supplied", C.c_int32),
                ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
                ("compute_stream", C.c_void_p), ("copy_stream", C.c_void_p)]


class qld_synth_scene(C.Structure):
    _fields_ = [("H", C.c_int32), ("W", C.c_int32), ("dtype", C.c_int32), ("maxval", C.c_uint32), ("key", C.c_uint64),
                ("n_terms", C.c_int32), ("has_disk", C.c_int32), ("base", C.c_void_p), ("weights", C.c_void_p),
                ("mods", C.c_void_p), ("mod_stride", C.c_int64), ("noise_a", C.c_double), ("noise_b", C.c_double),
                ("disk_x0", C.c_int32), ("disk_cy", C.c_int32), ("disk_radius", C.c_int32), ("reserved", C.c_int32),
                ("disk_amp", C.c_double), ("disk_mod", C.c_void_p)]


class QLDError(RuntimeError):
    def __init__(self, status: int, text: str = ""):
        self.status = status
        super().__init__(f"{_STATUS.get(status, status)}: {text}")


_lib = None


def load_library():
    """Load libqld.so; raises (never falls back) when it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(f"{_LIB_PATH} is missing: build it with `python -m paper_1511_03390_b200.build` "
                          "(nvcc, sm_100a). There is no CPU fallback.")
    l = C.CDLL(_LIB_PATH)
    vp, i, i64 = C.c_void_p, C.c_int, C.c_int64
    pf = C.POINTER(C.c_void_p)
    l.qld_workspace_bytes.argtypes = [C.POINTER(qld_config), C.POINTER(C.c_size_t)]
    l.qld_create.argtypes = [C.POINTER(qld_config), C.POINTER(vp)]
    l.qld_push_frames.argtypes = [vp, vp, i]
    l.qld_push_frames_device.argtypes = [vp, vp, i]
    l.qld_attach_frames_device.argtypes = [vp, vp]
    l.qld_commit_frames.argtypes = [vp, i, vp]
    l.qld_push_done.argtypes = [vp, i]
    l.qld_demod.argtypes = [vp, i, i]
    l.qld_get_maps.argtypes = [vp, i, pf, pf, pf, pf]
    l.qld_get_bins.argtypes = [vp, i, pf, C.POINTER(C.c_int)]
    l.qld_read_map.argtypes = [vp, i, i, vp]
    l.qld_read_ref_table.argtypes = [vp, i, i64, i, vp, vp]
    l.qld_set_ref_tables.argtypes = [vp, i, vp, vp, i64]
    l.qld_set_ref_table_fixed.argtypes = [vp, i, vp, vp, i]
    l.qld_read_ref_table_fixed.argtypes = [vp, i, vp, vp]
    l.qld_get_sums_i64.argtypes = [vp, i, pf, pf]
    l.qld_counters.argtypes = [vp, C.POINTER(i64), C.POINTER(i64)]
    l.qld_sync.argtypes = [vp]
    l.qld_reset.argtypes = [vp]
    l.qld_destroy.argtypes = [vp]
    l.qld_destroy.restype = None
    l.qld_last_error.argtypes = [vp]
    l.qld_last_error.restype = C.c_char_p
    l.qld_kernel_launches.argtypes = [vp]
    l.qld_kernel_launches.restype = i64
    l.qld_accum_mode.argtypes = [vp]
    l.qld_last_kernel.argtypes = [vp]
    l.qld_last_kernel.restype = C.c_char_p
    l.qld_debug_set_tile.argtypes = [vp, i, i, i, i]
    l.qld_cnr.argtypes = [vp, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, vp, vp]
    l.qld_dominant_bin.argtypes = [vp, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, vp, vp, vp]
    l.qld_probe_read.argtypes = [vp, C.c_int64, vp, vp]
    l.qld_dominant_bin_static.argtypes = [vp, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, vp, vp, vp]
    l.qld_dominant_bin_static_bytes.argtypes = [C.c_int32, C.c_int32, C.c_int32]
    l.qld_dominant_bin_static_bytes.restype = C.c_int64
    l.qld_dominant_bin_static_error.argtypes = []
    l.qld_dominant_bin_static_error.restype = C.c_char_p
    l.qld_display_map.argtypes = [vp, C.c_int64, vp, vp, vp, vp]
    l.qld_synth_fill.argtypes = [C.POINTER(qld_synth_scene), i64, i, vp, vp]
    _lib = l
    return l


def make_refs(refs: Sequence[dict]):
    arr = (qld_ref * len(refs))()
    for k, r in enumerate(refs):
        arr[k].nu = float(r.get("nu", 0.0) or 0.0)
        arr[k].phase = float(r.get("phase", 0.0))
        arr[k].num = int(r.get("num", 0) or 0)
        arr[k].den = int(r.get("den", 0) or 0)
        arr[k].phase_quarter = int(r.get("phase_quarter", 0))
    return arr


class QLD:
    """One QLD context (qld_create .. qld_destroy).  Methods carry the names of the C calls."""

    def __init__(self, H: int, W: int, dtype, N: int, refs: Sequence[dict], ring_frames: int = 0,
                 accum: int = QLD_ACC_AUTO, norm: int = QLD_NORM_PAPER, maps: int = QLD_MAP_ALL, max_value: int = 0,
                 resync_hops: int = 0, device=None, copy_stream=None, torch_workspace: bool = True,
                 external_store: bool = False, slide_hop: int = 0, debug_tile=None,
                 ref_tables_supplied: bool = False, window_relative: bool = False):
        import torch
        self._torch = torch
        self.lib = load_library()
        self.H, self.W, self.N, self.K = int(H), int(W), int(N), len(refs)
        self.dtype = QLD_U8 if str(dtype) in ("u8", "uint8", "torch.uint8", "0") else (QLD_U16_BE if str(dtype) in ("u16be", "2") else QLD_U16)
        self._refs = make_refs(refs)
        cfg = qld_config()
        cfg.H, cfg.W, cfg.dtype, cfg.N, cfg.K = self.H, self.W, self.dtype, self.N, self.K
        cfg.refs = C.cast(self._refs, C.POINTER(qld_ref))
        cfg.ring_frames, cfg.accum, cfg.norm, cfg.maps = int(ring_frames), int(accum), int(norm), int(maps)
        cfg.max_value, cfg.resync_hops, cfg.external_store = int(max_value), int(resync_hops), int(bool(external_store))
        cfg.slide_hop = int(slide_hop)
        cfg.ref_tables_supplied = int(bool(ref_tables_supplied))
        cfg.window_relative = int(bool(window_relative))
        self._ctx = C.c_void_p()
        nbytes = C.c_size_t()
        rc = self.lib.qld_workspace_bytes(C.byref(cfg), C.byref(nbytes))
        if rc != QLD_OK:
            raise QLDError(rc, self.lib.qld_last_error(None).decode())
        self.workspace_bytes = nbytes.value
        self._ws = None
        self._copy_stream = copy_stream
        if torch.cuda.is_available():
            self.device = torch.device(device if device is not None else f"cuda:{torch.cuda.current_device()}")
            with torch.cuda.device(self.device):
                if torch_workspace:
                    self._ws = torch.empty(nbytes.value + 256, dtype=torch.uint8, device=self.device)
                    ptr = (self._ws.data_ptr() + 255) & ~255
                    cfg.workspace, cfg.workspace_bytes = ptr, nbytes.value
                # torch's legacy default stream has handle 0, which the C API reads as "create one": pass
                # cudaStreamLegacy (0x1) so kernels stay ordered with torch work on that stream
                cfg.compute_stream = torch.cuda.current_stream(self.device).cuda_stream or 1
                if copy_stream is None:
                    self._copy_stream = torch.cuda.Stream(device=self.device)
                cfg.copy_stream = self._copy_stream.cuda_stream
                rc = self.lib.qld_create(C.byref(cfg), C.byref(self._ctx))
        else:
            self.device = None
            rc = self.lib.qld_create(C.byref(cfg), C.byref(self._ctx))   # fails loudly: QLD_E_CUDA
        if rc != QLD_OK:
            raise QLDError(rc, self.lib.qld_last_error(None).decode())
        if debug_tile:
            self.debug_set_tile(*debug_tile)

    # -- helpers -------------------------------------------------------------------------------
    def _check(self, rc: int):
        if rc != QLD_OK:
            raise QLDError(rc, self.lib.qld_last_error(self._ctx).decode())

    def _view(self, ptr: int, shape, dtype):
        """Zero-copy torch view of library-owned device memory."""
        torch = self._torch
        n = 1
        for s in shape:
            n *= s
        itemsize = torch.empty((), dtype=dtype).element_size()
        if self._ws is not None:
            off = ptr - self._ws.data_ptr()
            return self._ws[off:off + n * itemsize].view(dtype).view(*shape)
        iface = {"shape": tuple(shape), "typestr": {torch.float32: "<f4", torch.int32: "<i4", torch.int64: "<i8"}[dtype], "data": (ptr, False), "version": 2}
        holder = type("_Dev", (), {"__cuda_array_interface__": iface})()
        return torch.as_tensor(holder, device=self.device)

    # -- the C calls ---------------------------------------------------------------------------
    def push_frames(self, frames) -> None:
        """qld_push_frames (host tensor / numpy array) or qld_push_frames_device (CUDA tensor)."""
        torch = self._torch
        if isinstance(frames, torch.Tensor) and frames.is_cuda:
            assert frames.is_contiguous()
            self._check(self.lib.qld_push_frames_device(self._ctx, frames.data_ptr(), int(frames.shape[0])))
            self._keep = frames
        elif isinstance(frames, torch.Tensor):
            assert frames.is_contiguous()
            self._check(self.lib.qld_push_frames(self._ctx, frames.data_ptr(), int(frames.shape[0])))
            self._keep = frames
        else:
            import numpy as np
            a = np.ascontiguousarray(frames)
            self._check(self.lib.qld_push_frames(self._ctx, a.ctypes.data, int(a.shape[0])))
            self._keep = a

    def attach_frames_device(self, frames) -> None:
        assert frames.is_cuda and frames.is_contiguous()
        self._check(self.lib.qld_attach_frames_device(self._ctx, frames.data_ptr()))
        self._attached = frames

    def commit_frames(self, n_frames: int, producer_stream=None) -> None:
        """qld_commit_frames: n more frames were written in place into the attached store (zero-copy ingest)."""
        h = 0 if producer_stream is None else (producer_stream.cuda_stream or 1)
        self._check(self.lib.qld_commit_frames(self._ctx, int(n_frames), h))

    def push_done(self, block: bool = False) -> bool:
        rc = self.lib.qld_push_done(self._ctx, int(block))
        if rc == QLD_E_STATE:
            return False
        self._check(rc)
        return True

    def demod(self, mode: int = QLD_WHOLE, hop: int = 0) -> None:
        self._check(self.lib.qld_demod(self._ctx, int(mode), int(hop)))

    def get_maps(self, k: int = 0):
        """Device views (I, Q, amplitude, phase) of reference k, each [H, W] float32 or None."""
        p = [C.c_void_p() for _ in range(4)]
        self._check(self.lib.qld_get_maps(self._ctx, int(k), *[C.byref(x) for x in p]))
        return tuple(self._view(x.value, (self.H, self.W), self._torch.float32) if x.value else None for x in p)

    def get_bins(self, k: int = 0):
        p, n = C.c_void_p(), C.c_int()
        self._check(self.lib.qld_get_bins(self._ctx, int(k), C.byref(p), C.byref(n)))
        return self._view(p.value, (n.value, self.H, self.W), self._torch.int32)

    def read_map(self, k: int, which: int, host_dst) -> None:
        self._check(self.lib.qld_read_map(self._ctx, int(k), int(which), host_dst.data_ptr()))

    def read_ref_table(self, k: int, s_first: int, n: int):
        import numpy as np
        sn = np.empty(n, dtype=np.float32)
        cs = np.empty(n, dtype=np.float32)
        self._check(self.lib.qld_read_ref_table(self._ctx, int(k), int(s_first), int(n), sn.ctypes.data, cs.ctypes.data))
        return sn, cs

    def set_ref_tables(self, k: int, sin_tab, cos_tab) -> None:
        import numpy as np
        a = np.ascontiguousarray(sin_tab, dtype=np.float64)
        b = np.ascontiguousarray(cos_tab, dtype=np.float64)
        assert a.size == b.size
        self._check(self.lib.qld_set_ref_tables(self._ctx, int(k), a.ctypes.data, b.ctypes.data, int(a.size)))

    def set_ref_table_fixed(self, k: int, sin_q30, cos_q30) -> None:
        import numpy as np
        a = np.ascontiguousarray(sin_q30, dtype=np.int32)
        b = np.ascontiguousarray(cos_q30, dtype=np.int32)
        self._check(self.lib.qld_set_ref_table_fixed(self._ctx, int(k), a.ctypes.data, b.ctypes.data, int(a.size)))

    def read_ref_table_fixed(self, k: int):
        import numpy as np
        a = np.empty(self.N, dtype=np.int32)
        b = np.empty(self.N, dtype=np.int32)
        self._check(self.lib.qld_read_ref_table_fixed(self._ctx, int(k), a.ctypes.data, b.ctypes.data))
        return a, b

    def get_sums_i64(self, k: int = 0):
        p, q = C.c_void_p(), C.c_void_p()
        self._check(self.lib.qld_get_sums_i64(self._ctx, int(k), C.byref(p), C.byref(q)))
        return (self._view(p.value, (self.H, self.W), self._torch.int64), self._view(q.value, (self.H, self.W), self._torch.int64))

    def counters(self):
        a, b = C.c_int64(), C.c_int64()
        self._check(self.lib.qld_counters(self._ctx, C.byref(a), C.byref(b)))
        return a.value, b.value

    def sync(self) -> None:
        self._check(self.lib.qld_sync(self._ctx))

    def reset(self) -> None:
        self._check(self.lib.qld_reset(self._ctx))

    def kernel_launches(self) -> int:
        return int(self.lib.qld_kernel_launches(self._ctx))

    def accum_mode(self) -> int:
        return int(self.lib.qld_accum_mode(self._ctx))

    def accum_name(self) -> str:
        return {QLD_ACC_FP32: "FP32", QLD_ACC_INT_BINS: "INT_BINS", QLD_ACC_FIXED: "FIXED", QLD_ACC_INT_REFS: "INT_REFS"}[self.accum_mode()]

    def debug_set_tile(self, which, a: int = 0, b: int = 0, c: int = 0) -> None:
        """qld_debug_set_tile: which = "stream" (SEG, KC), "tc" (T, STAGES, KC) or "slide" (1 = always k_slide_bulk, 2 = never)."""
        w = {"stream": 0, "tc": 1, "slide": 2}.get(which, which)
        self._check(self.lib.qld_debug_set_tile(self._ctx, int(w), int(a), int(b), int(c)))

    def last_kernel(self) -> str:
        return self.lib.qld_last_kernel(self._ctx).decode()

    def destroy(self) -> None:
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self.lib.qld_destroy(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def cnr(image, y0: int, x0: int, m: int):
    """qld_cnr on a CUDA float32 map [H, W]: returns a CUDA tensor of 4 doubles {CNR, mean_s, mean_surr, rms}
    (Eq. (1)), enqueued on torch's current stream."""
    import torch
    lib = load_library()
    assert image.is_cuda and image.dtype == torch.float32 and image.is_contiguous() and image.dim() == 2
    out = torch.empty(4, dtype=torch.float64, device=image.device)
    rc = lib.qld_cnr(image.data_ptr(), int(image.shape[0]), int(image.shape[1]), int(y0), int(x0), int(m), out.data_ptr(),
                     torch.cuda.current_stream(image.device).cuda_stream or 1)
    if rc != QLD_OK:
        raise QLDError(rc, "qld_cnr")
    return out


def display_map(image):
    """qld_display_map on a CUDA float32 map: returns (u8 image of the same shape, range tensor {lo, hi})."""
    import torch
    lib = load_library()
    assert image.is_cuda and image.dtype == torch.float32 and image.is_contiguous()
    out = torch.empty(image.shape, dtype=torch.uint8, device=image.device)
    rng = torch.empty(2, dtype=torch.float32, device=image.device)
    scratch = torch.empty(2, dtype=torch.int32, device=image.device)
    rc = lib.qld_display_map(image.data_ptr(), int(image.numel()), out.data_ptr(), rng.data_ptr(), scratch.data_ptr(),
                             torch.cuda.current_stream(image.device).cuda_stream or 1)
    if rc != QLD_OK:
        raise QLDError(rc, "qld_display_map")
    return out, rng


def dominant_bin(frames, q_lo: int, q_hi: int):
    """qld_dominant_bin on a CUDA stack [N, H, W] (uint8 / uint16 / int16 view): returns (amp_max [H, W] float32,
    bin [H, W] int32) -- the largest amplitude over the DFT bins q_lo..q_hi and where it sits."""
    import torch
    lib = load_library()
    assert frames.is_cuda and frames.is_contiguous() and frames.dim() == 3
    N, H, W = (int(x) for x in frames.shape)
    dtype = QLD_U8 if frames.element_size() == 1 else QLD_U16
    amp = torch.empty((H, W), dtype=torch.float32, device=frames.device)
    bins = torch.empty((H, W), dtype=torch.int32, device=frames.device)
    rc = lib.qld_dominant_bin(frames.data_ptr(), dtype, H, W, N, int(q_lo), int(q_hi), amp.data_ptr(), bins.data_ptr(),
                              torch.cuda.current_stream(frames.device).cuda_stream or 1)
    if rc != QLD_OK:
        raise QLDError(rc, lib.qld_last_error(None).decode())
    return amp, bins


QLD_SEARCH_STATIC_BYTES = 4 << 20
QLD_PROBE_OUT_WORDS = 4096


def probe_read(buf, out=None):
    """qld_probe_read: one read-only pass over the CUDA tensor `buf` on torch's current stream (the read
    ceiling); returns the per-CTA checksum words (uint32 viewed as int32, [QLD_PROBE_OUT_WORDS]; unused words keep their contents)."""
    import torch
    lib = load_library()
    assert buf.is_cuda and buf.is_contiguous()
    if out is None:
        out = torch.zeros(QLD_PROBE_OUT_WORDS, dtype=torch.int32, device=buf.device)
    rc = lib.qld_probe_read(buf.data_ptr(), buf.numel() * buf.element_size(), out.data_ptr(), torch.cuda.current_stream(buf.device).cuda_stream or 1)
    if rc != QLD_OK:
        raise QLDError(rc, "qld_probe_read")
    return out


def dominant_bin_static(frames, q_lo: int, q_hi: int, amp=None, bins=None):
    """qld_dominant_bin_static: the search of dominant_bin() without any device allocation inside the library, for callers
    that cannot afford one (a live acquisition loop, a process whose HBM is already spoken for): the scratch is a fixed
    4 MiB array in the library, so the search must fit it (QLDError with QLD_E_NOMEM otherwise) and the frames must be a
    multiple of 16 bytes.  Pass preallocated `amp` [H, W] float32 and `bins` [H, W] int32 to keep this wrapper from
    allocating too.  One search at a time per device: overlapping calls share the scratch and race."""
    import torch
    lib = load_library()
    assert frames.is_cuda and frames.is_contiguous() and frames.dim() == 3
    N, H, W = (int(x) for x in frames.shape)
    dtype = QLD_U8 if frames.element_size() == 1 else QLD_U16
    if amp is None:
        amp = torch.empty((H, W), dtype=torch.float32, device=frames.device)
    if bins is None:
        bins = torch.empty((H, W), dtype=torch.int32, device=frames.device)
    assert amp.is_contiguous() and bins.is_contiguous() and amp.dtype == torch.float32 and bins.dtype == torch.int32
    with torch.cuda.device(frames.device):
        rc = lib.qld_dominant_bin_static(frames.data_ptr(), dtype, H, W, N, int(q_lo), int(q_hi), amp.data_ptr(), bins.data_ptr(),
                                         torch.cuda.current_stream(frames.device).cuda_stream or 1)
    if rc != QLD_OK:
        raise QLDError(rc, lib.qld_dominant_bin_static_error().decode())
    return amp, bins


def synth_fill(scene, s_first: int, n_frames: int, out=None, device="cuda"):
    """Fill frames s_first .. s_first+n-1 of a synth.Scene into a CUDA tensor [n, H, W] (qld_synth_fill)."""
    import numpy as np
    import torch
    lib = load_library()
    dev = torch.device(device)
    tdt = torch.uint8 if scene.dtype == "u8" else torch.uint16
    if out is None:
        out = torch.empty((n_frames, scene.H, scene.W), dtype=tdt, device=dev)
    cache = scene.meta.setdefault("_dev", {})
    if "base" not in cache:
        cache["base"] = torch.from_numpy(np.ascontiguousarray(scene.base)).to(dev)
        cache["weights"] = torch.from_numpy(np.ascontiguousarray(scene.weights)).to(dev) if scene.weights.shape[0] else torch.zeros(1, device=dev)
        cache["mods"] = torch.from_numpy(np.ascontiguousarray(scene.mods)).to(dev) if scene.mods.shape[0] else torch.zeros(1, dtype=torch.float64, device=dev)
        cache["disk_mod"] = torch.from_numpy(np.ascontiguousarray(scene.disk.mod)).to(dev) if scene.disk is not None else torch.zeros(1, dtype=torch.float64, device=dev)
    sc = qld_synth_scene()
    sc.H, sc.W, sc.dtype, sc.maxval, sc.key = scene.H, scene.W, (QLD_U8 if scene.dtype == "u8" else QLD_U16), scene.maxval, int(scene.key)
    sc.n_terms, sc.has_disk = int(scene.weights.shape[0]), int(scene.disk is not None)
    sc.base, sc.weights, sc.mods = cache["base"].data_ptr(), cache["weights"].data_ptr(), cache["mods"].data_ptr()
    sc.mod_stride = int(scene.mods.shape[1]) if scene.mods.shape[0] else 0
    sc.noise_a, sc.noise_b = float(scene.noise_a), float(scene.noise_b)
    if scene.disk is not None:
        d = scene.disk
        sc.disk_x0, sc.disk_cy, sc.disk_radius, sc.disk_amp = int(d.x0), int(d.cy), int(d.radius), float(d.amp)
    sc.disk_mod = cache["disk_mod"].data_ptr()
    rc = lib.qld_synth_fill(C.byref(sc), int(s_first), int(n_frames), out.data_ptr(), torch.cuda.current_stream(dev).cuda_stream or 1)
    if rc != QLD_OK:
        raise QLDError(rc, "qld_synth_fill")
    return out
