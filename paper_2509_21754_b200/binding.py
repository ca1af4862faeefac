"""ctypes binding of include/fitrig.h.  Same names as the C ABI, minus the fitrig_ prefix, as methods
of `Context`.  No arithmetic of the method happens here; there is no CPU fallback: if libfitrig.so is
missing or no CUDA device is present every compute call raises."""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import List, Optional, Sequence, Tuple

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))

OK, ERR_INVALID_ARG, ERR_CUDA, ERR_NOMEM, ERR_STATE, ERR_CAPACITY = 0, -1, -2, -3, -4, -5
REF_ABS, REF_LITERAL, REF_FLOOR = 0, 1, 2
BRANCH_IMAGE, BRANCH_FREQUENCY = 0, 1


class FitrigError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"fitrig error {code}: {msg}")
        self.code = code


class _Params(ctypes.Structure):
    _fields_ = [("tile", ctypes.c_int32), ("C", ctypes.c_float), ("ref_mode", ctypes.c_int32),
                ("M_override", ctypes.c_float), ("branch", ctypes.c_int32), ("strip_rows", ctypes.c_int32),
                ("device", ctypes.c_int32), ("row_offset", ctypes.c_int32), ("accumulate", ctypes.c_int32), ("harmonics", ctypes.c_int32), ("stride", ctypes.c_int32), ("batch", ctypes.c_int32), ("reserved", ctypes.c_int32 * 4)]


class _Candidate(ctypes.Structure):
    _fields_ = [("x", ctypes.c_int32), ("y", ctypes.c_int32), ("snapshot", ctypes.c_int32),
                ("score", ctypes.c_float)]


class _Plan(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in
                ("units", "Ty", "Tx", "path", "units_per_cta", "box_tiles", "warps_per_cta", "stages", "grid",
                 "smem_bytes", "strip_rows", "n_strips", "n_strip_buffers", "reserved")] + \
               [("strip_buffer_bytes", ctypes.c_int64), ("workspace_bytes", ctypes.c_int64)]


POSITION_DTYPE = np.dtype([("x", np.float64), ("y", np.float64), ("value", np.float64)])
INTERP_BILINEAR, INTERP_BICUBIC, INTERP_SPLINE, INTERP_MAKIMA = 0, 1, 2, 3
CANDIDATE_DTYPE = np.dtype([("x", np.int32), ("y", np.int32), ("snapshot", np.int32), ("score", np.float32)])


@dataclass
class Candidate:
    x: int
    y: int
    snapshot: int
    score: float


@dataclass
class Plan:
    units: int
    Ty: int
    Tx: int
    path: int
    units_per_cta: int
    box_tiles: int
    warps_per_cta: int
    stages: int
    grid: int
    smem_bytes: int
    strip_rows: int
    n_strips: int
    n_strip_buffers: int
    strip_buffer_bytes: int
    workspace_bytes: int


_lib = None


def lib_path() -> str:
    return os.path.join(_PKG, "libfitrig.so")


def load_library(build_if_missing: bool = True) -> ctypes.CDLL:
    """dlopen the in-tree libfitrig.so (building it with nvcc first if it is missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if build_if_missing:
        from . import build as _b
        if _b.stale():
            _b.build()
    if not os.path.exists(path):
        raise FitrigError(ERR_CUDA, f"{path} not found: run `python -m paper_2509_21754_b200.build`")
    L = ctypes.CDLL(path)
    vp, i32, i64, f32 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_float
    P = ctypes.POINTER
    L.fitrig_plan_query.argtypes = [i32, i32, i32, P(_Params), i32, P(_Plan)]
    L.fitrig_create.argtypes = [i32, i32, i32, P(_Params), P(vp)]
    L.fitrig_destroy.argtypes = [vp]
    L.fitrig_map_dims.argtypes = [vp, P(i32), P(i32), P(i32)]
    L.fitrig_tlisi.argtypes = [vp, vp, vp, vp]
    L.fitrig_tlisi_batch.argtypes = [vp, P(vp), vp, vp]
    L.fitrig_detect.argtypes = [vp, f32, vp, i64, P(i64), vp]
    L.fitrig_detect_batch.argtypes = [vp, f32, vp, i64, P(i64), vp, vp]
    L.fitrig_detect_launch.argtypes = [vp, f32, i64, vp]
    L.fitrig_detect_fetch.argtypes = [vp, vp, P(i64), vp]
    L.fitrig_shard_export_eta.argtypes = [vp, vp, vp]
    L.fitrig_shard_import_eta.argtypes = [vp, vp, i32, vp]
    L.fitrig_stream.argtypes = [vp, P(vp), vp, vp]
    L.fitrig_push.argtypes = [vp, vp, f32, vp, vp, i64, P(i64), P(i64), vp]
    L.fitrig_push_reset.argtypes = [vp]
    L.fitrig_shard_export.argtypes = [vp, vp, vp]
    L.fitrig_shard_import.argtypes = [vp, vp, i32, vp, vp]
    L.fitrig_get_stats.argtypes = [vp, P(f32), vp, vp]
    L.fitrig_get_map.argtypes = [vp, i32, vp]
    L.fitrig_get_raw.argtypes = [vp, vp, vp, vp, vp, vp]
    L.fitrig_profile.argtypes = [vp, i32]
    L.fitrig_last_timing.argtypes = [vp, P(f32), P(i32), P(f32), P(i32)]
    L.fitrig_localise.argtypes = [vp, vp, i64, i32, i32, vp, vp, vp]
    L.fitrig_stream_timeline.argtypes = [vp, vp, i32, P(i32)]
    L.fitrig_launch_count.argtypes = [vp, P(i64)]
    L.fitrig_copy_count.argtypes = [vp, P(i64)]
    L.fitrig_probe_read_bandwidth.argtypes = [vp, vp, i64, i32, P(f32), vp]
    L.fitrig_choose_accumulate.argtypes = [vp, i32, i32, i32, f32, i32, i32, P(i32), vp, P(i32), vp]
    L.fitrig_choose_accumulate_static.argtypes = [vp, i32, i32, i32, f32, i32, i32, P(i32), vp, P(i32), vp]
    for n in ("fitrig_plan_query", "fitrig_create", "fitrig_destroy", "fitrig_map_dims", "fitrig_tlisi",
              "fitrig_tlisi_batch", "fitrig_detect_batch", "fitrig_detect_launch", "fitrig_detect_fetch", "fitrig_shard_export_eta", "fitrig_shard_import_eta",
              "fitrig_detect", "fitrig_stream", "fitrig_push", "fitrig_push_reset", "fitrig_shard_export", "fitrig_shard_import", "fitrig_get_stats", "fitrig_get_map", "fitrig_get_raw",
              "fitrig_profile", "fitrig_last_timing", "fitrig_launch_count", "fitrig_copy_count", "fitrig_localise", "fitrig_stream_timeline", "fitrig_probe_read_bandwidth", "fitrig_choose_accumulate",
              "fitrig_choose_accumulate_static"):
        getattr(L, n).restype = ctypes.c_int
    L.fitrig_last_error.restype = ctypes.c_char_p
    L.fitrig_version.restype = ctypes.c_char_p
    _lib = L
    return L


def exported_symbols() -> List[str]:
    """Names include/fitrig.h declares (parsed from the header)."""
    import re
    hdr = os.path.join(os.path.dirname(_PKG), "include", "fitrig.h")
    with open(hdr) as f:
        txt = f.read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(fitrig_[a-z_]+)\s*\(", txt)))


def last_error() -> str:
    return load_library().fitrig_last_error().decode()


def version() -> str:
    return load_library().fitrig_version().decode()


def _check(rc: int, allow: Tuple[int, ...] = ()) -> int:
    if rc != OK and rc not in allow:
        raise FitrigError(rc, last_error())
    return rc


def _make_params(tile=0, C=0.0, ref_mode=REF_ABS, M_override=0.0, branch=BRANCH_IMAGE, strip_rows=0, device=0,
                 row_offset=0, accumulate=0, harmonics=0, stride=0, batch=0):
    p = _Params()
    p.tile, p.C, p.ref_mode, p.M_override = int(tile), float(C), int(ref_mode), float(M_override)
    p.branch, p.strip_rows, p.device = int(branch), int(strip_rows), int(device)
    p.row_offset = int(row_offset)
    p.accumulate = int(accumulate)
    p.harmonics = int(harmonics)
    p.stride = int(stride)
    p.batch = int(batch)
    return p


def plan_query(H: int, W: int, n_snapshots: int, num_sms: int = 0, **params) -> Plan:
    """fitrig_plan_query: host-only, works without a GPU."""
    L = load_library()
    p = _make_params(**params)
    out = _Plan()
    _check(L.fitrig_plan_query(H, W, n_snapshots, ctypes.byref(p), num_sms, ctypes.byref(out)))
    return Plan(**{f: getattr(out, f) for f in Plan.__dataclass_fields__})


def choose_accumulate(d_stack, eps: float, g_max: int = 32, stream=None):
    """fitrig_choose_accumulate on a [L, H, W] CUDA tensor: (g, [contrast of g = 1, 2, 4, .. up to the chosen level])."""
    L = load_library()
    if not (d_stack.is_cuda and d_stack.is_contiguous() and d_stack.dim() == 3 and d_stack.dtype.is_floating_point and d_stack.element_size() == 4):
        raise ValueError("choose_accumulate: need a contiguous [L, H, W] fp32 CUDA tensor")
    n, H, W = d_stack.shape
    g, nl = ctypes.c_int32(), ctypes.c_int32()
    d = (ctypes.c_double * 6)()
    _check(L.fitrig_choose_accumulate(_dev_ptr(d_stack), H, W, n, float(eps), int(g_max), d_stack.device.index or 0,
                                      ctypes.byref(g), ctypes.cast(d, ctypes.c_void_p), ctypes.byref(nl), _stream_ptr(stream)))
    return g.value, [d[i] for i in range(nl.value)]


STATIC_ACCUM_MAX_PARTIALS = 8192  # FITRIG_STATIC_ACCUM_MAX_PARTIALS of include/fitrig.h


def choose_accumulate_static(d_stack, eps: float, g_max: int = 32, stream=None):
    """fitrig_choose_accumulate_static: `choose_accumulate` for callers that must not allocate device memory -- a
    real-time loop whose copy / compute overlap a cudaMalloc or cudaFree would stall, or a process whose device memory
    is already held by another allocator.  Same arguments and the same (bit-identical) result; the scratch is a fixed
    array inside the library (room for STATIC_ACCUM_MAX_PARTIALS partial sums: every image size on one B200), shared by
    all calls on the device, so calls whose GPU work overlaps race.  The first call on a device does a one-time
    set-up; make it before any stream capture on that device."""
    L = load_library()
    if not (d_stack.is_cuda and d_stack.is_contiguous() and d_stack.dim() == 3 and d_stack.dtype.is_floating_point and d_stack.element_size() == 4):
        raise ValueError("choose_accumulate_static: need a contiguous [L, H, W] fp32 CUDA tensor")
    n, H, W = d_stack.shape
    g, nl = ctypes.c_int32(), ctypes.c_int32()
    d = (ctypes.c_double * 6)()
    _check(L.fitrig_choose_accumulate_static(_dev_ptr(d_stack), H, W, n, float(eps), int(g_max), d_stack.device.index or 0,
                                             ctypes.byref(g), ctypes.cast(d, ctypes.c_void_p), ctypes.byref(nl), _stream_ptr(stream)))
    return g.value, [d[i] for i in range(nl.value)]


def _dev_ptr(t) -> int:
    """Device pointer of a torch CUDA tensor (or a raw integer address)."""
    if t is None:
        return 0
    if isinstance(t, int):
        return t
    assert t.is_cuda and t.is_contiguous() and str(t.dtype) == "torch.float32", "need a contiguous CUDA fp32 tensor"
    return t.data_ptr()


def _stream_ptr(stream) -> int:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


class Context:
    """fitrig_ctx.  Methods mirror the C ABI: tlisi, detect, stream, get_stats, get_map, get_raw, ..."""

    def __init__(self, H: int, W: int, n_snapshots: int, **params):
        self._L = load_library()
        self._h = ctypes.c_void_p()
        p = _make_params(**params)
        _check(self._L.fitrig_create(H, W, n_snapshots, ctypes.byref(p), ctypes.byref(self._h)))
        self.H, self.W, self.L = H, W, n_snapshots
        u, ty, tx = ctypes.c_int32(), ctypes.c_int32(), ctypes.c_int32()
        _check(self._L.fitrig_map_dims(self._h, ctypes.byref(u), ctypes.byref(ty), ctypes.byref(tx)))
        self.units, self.Ty, self.Tx = u.value, ty.value, tx.value
        self.branch = int(params.get("branch", BRANCH_IMAGE))
        self.tile = int(params.get("tile", 0)) or 32
        self.batch = int(params.get("batch", 0)) or 1
        self._launch_caps: List[int] = []  # capacities of the detect_launch calls that have not been fetched yet

    def map_dims(self) -> Tuple[int, int, int]:
        return self.units, self.Ty, self.Tx

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._L.fitrig_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # ---- compute calls ----
    def tlisi(self, d_stack, d_tlisi=None, stream=None) -> None:
        _check(self._L.fitrig_tlisi(self._h, _dev_ptr(d_stack), _dev_ptr(d_tlisi), _stream_ptr(stream)))

    def tlisi_batch(self, d_stacks: Sequence, d_tlisi=None, stream=None) -> None:
        """d_stacks: B CUDA tensors [L, H, W] (params.batch = B); d_tlisi: [B, U, Ty, Tx] or None."""
        assert len(d_stacks) == self.batch
        arr = (ctypes.c_void_p * self.batch)(*[_dev_ptr(t) for t in d_stacks])
        _check(self._L.fitrig_tlisi_batch(self._h, arr, _dev_ptr(d_tlisi), _stream_ptr(stream)))

    def detect_batch(self, sigma_threshold: float, capacity: int = 1 << 16, stream=None, out: Optional[np.ndarray] = None):
        """Returns (candidates of stack 0, then stack 1, ..; n_found; per-stack totals [B])."""
        if out is None:
            out = np.zeros(max(capacity, 1), dtype=CANDIDATE_DTYPE)
        n = ctypes.c_int64(0)
        per = np.zeros(self.batch, dtype=np.int64)
        _check(self._L.fitrig_detect_batch(self._h, float(sigma_threshold), out.ctypes.data, int(capacity), ctypes.byref(n),
                                           per.ctypes.data, _stream_ptr(stream)), allow=(ERR_CAPACITY,))
        return out[: min(n.value, capacity)], n.value, per

    def detect(self, sigma_threshold: float, capacity: int = 1 << 16, stream=None, out: Optional[np.ndarray] = None):
        """Returns (structured array of candidates actually written, n_found).  Raises on errors other than
        FITRIG_ERR_CAPACITY (then n_found > len(result))."""
        if out is None:
            out = np.zeros(max(capacity, 1), dtype=CANDIDATE_DTYPE)
        n = ctypes.c_int64(0)
        _check(self._L.fitrig_detect(self._h, float(sigma_threshold), out.ctypes.data, int(capacity), ctypes.byref(n),
                                     _stream_ptr(stream)), allow=(ERR_CAPACITY,))
        return out[: min(n.value, capacity)], n.value

    def detect_launch(self, sigma_threshold: float, capacity: int = 1 << 16, stream=None) -> None:
        """Enqueue the detection of the current map (at most two may be in flight); see detect_fetch."""
        _check(self._L.fitrig_detect_launch(self._h, float(sigma_threshold), int(capacity), _stream_ptr(stream)))
        self._launch_caps.append(int(capacity))  # the library copies up to this many records into detect_fetch's array

    def detect_fetch(self, out: np.ndarray):
        """Wait for the oldest unfetched detect_launch and return (candidates, n_found, per-stack totals); `out` must
        hold the capacity given to that launch (checked here: the library would write past a shorter array)."""
        cap = self._launch_caps[0] if self._launch_caps else 0
        if out.dtype != CANDIDATE_DTYPE or not out.flags["C_CONTIGUOUS"] or len(out) < cap:
            raise ValueError(f"detect_fetch: need a contiguous candidate array of at least {cap} records (the capacity of the launch)")
        n = ctypes.c_int64(0)
        per = np.zeros(self.batch, dtype=np.int64)
        rc = self._L.fitrig_detect_fetch(self._h, out.ctypes.data, ctypes.byref(n), per.ctypes.data)
        if self._launch_caps and rc in (OK, ERR_CAPACITY):
            self._launch_caps.pop(0)
        _check(rc, allow=(ERR_CAPACITY,))
        return out[: min(n.value, cap)], n.value, per

    def stream(self, h_snapshots: Sequence, h_tlisi=None, stream=None) -> None:
        """h_snapshots: L host tensors/arrays of [H, W] fp32 (pinned for overlap)."""
        arr = (ctypes.c_void_p * self.L)()
        assert len(h_snapshots) == self.L
        for i, s in enumerate(h_snapshots):
            arr[i] = s.data_ptr() if hasattr(s, "data_ptr") else s.ctypes.data
        out = 0
        if h_tlisi is not None:
            out = h_tlisi.data_ptr() if hasattr(h_tlisi, "data_ptr") else h_tlisi.ctypes.data
        _check(self._L.fitrig_stream(self._h, arr, out, _stream_ptr(stream)))

    def localise(self, cands: np.ndarray, method: int = INTERP_SPLINE, oversample: int = 1, eta: Optional[np.ndarray] = None,
                 stream=None) -> np.ndarray:
        """fitrig_localise: sub-tile positions (structured array x, y, value) of frequency-branch candidates; `eta`
        (fp32 [Ty, Tx]) replaces the context's own spectrum matrix when given."""
        cands = np.ascontiguousarray(cands, dtype=CANDIDATE_DTYPE)
        out = np.zeros(len(cands), dtype=POSITION_DTYPE)
        e = None
        if eta is not None:
            e = np.ascontiguousarray(eta, dtype=np.float32)
            assert e.shape == (self.Ty, self.Tx)
        _check(self._L.fitrig_localise(self._h, cands.ctypes.data, len(cands), int(method), int(oversample),
                                       e.ctypes.data if e is not None else None, out.ctypes.data, _stream_ptr(stream)))
        return out

    # ---- real-time mode ----
    def push(self, snapshot, sigma_threshold: float, d_tlisi=None, capacity: int = 1 << 16, stream=None,
             out: Optional[np.ndarray] = None):
        """snapshot: [H, W] fp32 host (pinned) or CUDA tensor, or None to flush.  Returns (unit, candidates, n_found);
        unit = -1 while fewer than three snapshots had been pushed before this call."""
        ptr = 0
        if snapshot is not None:
            ptr = snapshot.data_ptr() if hasattr(snapshot, "data_ptr") else snapshot.ctypes.data
        if out is None:
            out = np.zeros(max(capacity, 1), dtype=CANDIDATE_DTYPE)
        n, u = ctypes.c_int64(0), ctypes.c_int64(-1)
        _check(self._L.fitrig_push(self._h, ptr, float(sigma_threshold), _dev_ptr(d_tlisi), out.ctypes.data,
                                   int(capacity), ctypes.byref(n), ctypes.byref(u), _stream_ptr(stream)),
               allow=(ERR_CAPACITY,))
        return u.value, out[: min(n.value, capacity)], n.value

    def push_reset(self) -> None:
        _check(self._L.fitrig_push_reset(self._h))

    # ---- row shards ----
    def shard_export(self, d_out, stream=None) -> None:
        """d_out: CUDA float64 tensor of 2 + 2U elements."""
        assert d_out.is_cuda and d_out.is_contiguous() and str(d_out.dtype) == "torch.float64"
        assert d_out.numel() >= 2 + 2 * self.units
        _check(self._L.fitrig_shard_export(self._h, d_out.data_ptr(), _stream_ptr(stream)))

    def shard_import(self, d_all, world: int, d_tlisi=None, stream=None) -> None:
        """d_all: CUDA float64 tensor [world, 2 + 2U] (the all-gathered export vectors, in shard order)."""
        assert d_all.is_cuda and d_all.is_contiguous() and str(d_all.dtype) == "torch.float64"
        assert d_all.numel() >= world * (2 + 2 * self.units)
        _check(self._L.fitrig_shard_import(self._h, d_all.data_ptr(), int(world), _dev_ptr(d_tlisi),
                                           _stream_ptr(stream)))

    def shard_export_eta(self, d_out, stream=None) -> None:
        """d_out: CUDA float64 tensor of 3 elements (frequency branch, after shard_import)."""
        assert d_out.is_cuda and d_out.is_contiguous() and str(d_out.dtype) == "torch.float64" and d_out.numel() >= 3
        _check(self._L.fitrig_shard_export_eta(self._h, d_out.data_ptr(), _stream_ptr(stream)))

    def shard_import_eta(self, d_all, world: int, stream=None) -> None:
        """d_all: CUDA float64 tensor [world, 3]."""
        assert d_all.is_cuda and d_all.is_contiguous() and str(d_all.dtype) == "torch.float64"
        assert d_all.numel() >= 3 * world
        _check(self._L.fitrig_shard_import_eta(self._h, d_all.data_ptr(), int(world), _stream_ptr(stream)))

    # ---- getters ----
    def get_stats(self):
        """(M, mu, sigma): B = 1: M a float, mu / sigma [U]; B > 1: M [B], mu / sigma [B, U]."""
        B = self.batch
        M = np.zeros(B, dtype=np.float32)
        mu = np.zeros(B * self.units)
        sd = np.zeros(B * self.units)
        _check(self._L.fitrig_get_stats(self._h, M.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), mu.ctypes.data,
                                        sd.ctypes.data))
        if B == 1:
            return float(M[0]), mu, sd
        return M, mu.reshape(B, self.units), sd.reshape(B, self.units)

    def _bshape(self, *shape):
        return shape if self.batch == 1 else (self.batch,) + shape

    def get_map(self, which: int = 0) -> np.ndarray:
        shape = self._bshape(self.units, self.Ty, self.Tx) if which in (0, 1) else self._bshape(self.Ty, self.Tx)
        out = np.zeros(shape, dtype=np.float32)
        _check(self._L.fitrig_get_map(self._h, int(which), out.ctypes.data))
        return out

    def get_raw(self):
        shape = self._bshape(self.units, self.Ty, self.Tx)
        sd, md, sr = (np.zeros(shape, np.float32) for _ in range(3))
        ax, ay = (np.zeros(shape, np.int32) for _ in range(2))
        _check(self._L.fitrig_get_raw(self._h, sd.ctypes.data, md.ctypes.data, sr.ctypes.data, ax.ctypes.data,
                                      ay.ctypes.data))
        return sd, md, sr, ax, ay

    def profile(self, enable: bool = True) -> None:
        _check(self._L.fitrig_profile(self._h, int(bool(enable))))

    def last_timing(self):
        """(main kernel ms, launches, finalise ms, launches), summed since profiling was enabled or last read."""
        a, n, b, m = ctypes.c_float(), ctypes.c_int32(), ctypes.c_float(), ctypes.c_int32()
        _check(self._L.fitrig_last_timing(self._h, ctypes.byref(a), ctypes.byref(n), ctypes.byref(b), ctypes.byref(m)))
        return a.value, n.value, b.value, m.value

    def probe_read_bandwidth(self, d_tensor, reps: int = 5, stream=None) -> float:
        """GB/s of a plain read-only pass over `d_tensor` (calibration for roofline fractions)."""
        g = ctypes.c_float()
        nbytes = d_tensor.numel() * d_tensor.element_size()
        _check(self._L.fitrig_probe_read_bandwidth(self._h, d_tensor.data_ptr(), nbytes, int(reps), ctypes.byref(g),
                                                   _stream_ptr(stream)))
        return g.value

    def stream_timeline(self, max_strips: int = 4096) -> np.ndarray:
        """[n_strips, 4] ms since the first copy started: copy start, copy end, kernel start, kernel end of every strip
        of the last stream() that ran under profile(True)."""
        out = np.zeros((max_strips, 4), dtype=np.float32)
        n = ctypes.c_int32()
        _check(self._L.fitrig_stream_timeline(self._h, out.ctypes.data, max_strips, ctypes.byref(n)))
        return out[: min(n.value, max_strips)]

    def copy_count(self) -> int:
        n = ctypes.c_int64()
        _check(self._L.fitrig_copy_count(self._h, ctypes.byref(n)))
        return n.value

    def launch_count(self) -> int:
        n = ctypes.c_int64()
        _check(self._L.fitrig_launch_count(self._h, ctypes.byref(n)))
        return n.value
