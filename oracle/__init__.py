"""ctypes front end of the CPU fp64 oracle (oracle/fitrig_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It does not
import, link or read anything of the CUDA path (paper_2509_21754_b200).

The per-pixel, per-tile and spectral arithmetic lives in the C file; this module marshals numpy arrays and holds
the steps that are plain numpy one-liners: the fp64 sums of snapshot accumulation (`accumulate`), the
maximum of the accumulated images (`_tlisi_f64`), the running maximum of the real-time forms
(`run_realtime`, `run_realtime_frequency`), and the accumulation rule (`accumulation_contrast`, `choose_accumulate`:
means of absolute values).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fitrig_oracle.c")
_LIB = os.path.join(_HERE, "libfitrig_oracle.so")

REF_ABS, REF_LITERAL, REF_FLOOR = 0, 1, 2
INTERP_BILINEAR, INTERP_BICUBIC, INTERP_SPLINE, INTERP_MAKIMA = 0, 1, 2, 3


def build(force: bool = False) -> str:
    """gcc -O2 (no fast-math) -fopenmp; rebuilt when the source is newer than the library."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.run(["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"],
                       check=True)
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        c_f32pp = ctypes.POINTER(ctypes.c_void_p)
        dp, ip64, ip32 = ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p
        L.fitrig_oracle_num_threads.restype = ctypes.c_int
        L.fitrig_oracle_set_threads.argtypes = [ctypes.c_int]
        L.fitrig_oracle_global_max.restype = ctypes.c_double
        L.fitrig_oracle_global_max.argtypes = [c_f32pp, ctypes.c_int, ctypes.c_int64, ctypes.c_int64, ctypes.c_double]
        L.fitrig_oracle_tlisi.restype = ctypes.c_int
        L.fitrig_oracle_tlisi.argtypes = [c_f32pp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                          ctypes.c_double, ctypes.c_int, ctypes.c_double,
                                          dp, dp, dp, ip64, dp, dp]
        L.fitrig_oracle_tlisi_windows.restype = ctypes.c_int
        L.fitrig_oracle_tlisi_windows.argtypes = [c_f32pp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                                  ctypes.c_int, ctypes.c_double, ctypes.c_int, ctypes.c_double,
                                                  dp, dp, dp, ip64, dp, dp]
        L.fitrig_oracle_n_windows.restype = ctypes.c_int
        L.fitrig_oracle_n_windows.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int]
        L.fitrig_oracle_tlisi_f64.restype = ctypes.c_int
        L.fitrig_oracle_tlisi_f64.argtypes = L.fitrig_oracle_tlisi.argtypes
        L.fitrig_oracle_zscore.restype = None
        L.fitrig_oracle_zscore.argtypes = [dp, ctypes.c_int, ctypes.c_int64, dp, dp, dp]
        L.fitrig_oracle_select.restype = ctypes.c_int64
        L.fitrig_oracle_select.argtypes = [dp, ip64, ctypes.c_int, ctypes.c_int64, ctypes.c_int, ctypes.c_double,
                                           ip32, ip32, ip32, ip64, dp, ctypes.c_int64]
        L.fitrig_oracle_spectrum.restype = None
        L.fitrig_oracle_spectrum.argtypes = [dp, ctypes.c_int, ctypes.c_int64, dp, ip32]
        L.fitrig_oracle_spectrum_hsum.restype = None
        L.fitrig_oracle_spectrum_hsum.argtypes = [dp, ctypes.c_int, ctypes.c_int64, ctypes.c_int, dp, ip32, dp]
        L.fitrig_oracle_select_spectrum.restype = ctypes.c_int64
        L.fitrig_oracle_select_spectrum.argtypes = [dp, ip32, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                                    ctypes.c_int, ctypes.c_double, ip32, ip32, ip32, ip64, dp,
                                                    ctypes.c_int64]
        L.fitrig_oracle_interp_eval.restype = ctypes.c_int
        L.fitrig_oracle_interp_eval.argtypes = [dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp, ctypes.c_int64, dp]
        L.fitrig_oracle_localise.restype = ctypes.c_int
        L.fitrig_oracle_localise.argtypes = [dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                             ip64, ctypes.c_int64, dp, dp, dp]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().fitrig_oracle_num_threads())


def set_threads(n: int) -> None:
    lib().fitrig_oracle_set_threads(int(n))


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _snap_ptrs(snaps: Sequence[np.ndarray], H: int, W: int):
    keep = []
    arr = (ctypes.c_void_p * len(snaps))()
    for i, s in enumerate(snaps):
        s = np.ascontiguousarray(s, dtype=np.float32)
        assert s.shape == (H, W), (s.shape, H, W)
        keep.append(s)
        arr[i] = s.ctypes.data
    return arr, keep


def as_snapshots(stack) -> List[np.ndarray]:
    """[L,H,W] array (numpy or CPU torch) or a list of [H,W] arrays -> list of fp32 numpy views."""
    if hasattr(stack, "detach"):
        stack = stack.detach().cpu().numpy()
    if isinstance(stack, np.ndarray):
        assert stack.ndim == 3
        return [stack[i] for i in range(stack.shape[0])]
    return [s.detach().cpu().numpy() if hasattr(s, "detach") else np.asarray(s) for s in stack]


def global_max(stack, C: float = 1e-6) -> float:
    snaps = as_snapshots(stack)
    H, W = snaps[0].shape
    arr, keep = _snap_ptrs(snaps, H, W)
    return float(lib().fitrig_oracle_global_max(arr, len(snaps), H, W, float(C)))


@dataclass
class TlisiResult:
    M: float
    U: int
    Ty: int
    Tx: int
    sumD: np.ndarray  # [U,Ty,Tx] float64
    maxD: np.ndarray
    sumR: np.ndarray
    argmax: np.ndarray  # [U,Ty,Tx] int64, y*W + x
    q: np.ndarray
    tlisi: np.ndarray


def accumulate(stack, g: int) -> List[np.ndarray]:
    """Snapshot accumulation, PAPER.md:497 (section 3.3.2) and Fig. 16 ("adding the two snapshots together and
    outputting their sum", applied progressively): A_j = x_{gj} + x_{gj+1} + ... + x_{gj+g-1}, j = 0 .. L//g - 1,
    summed in fp64 in snapshot order.  Reading R25: g is any integer >= 1 (the figure's pairwise tree
    gives g = 2^m); the trailing L mod g snapshots do not form a complete group and are left out."""
    snaps = as_snapshots(stack)
    if g < 1:
        raise ValueError("accumulate: g >= 1")
    out = []
    for j in range(len(snaps) // g):
        a = np.zeros(snaps[0].shape, dtype=np.float64)
        for i in range(g):
            a += snaps[g * j + i].astype(np.float64)
        out.append(a)
    return out


def accumulation_contrast(stack, g: int) -> float:
    """How different adjacent g-accumulated snapshots are (reading R30): the mean over adjacent pairs and
    pixels of the paper's own difference image |A_{j+1} - A_j| (Eq. 3, on accumulated snapshots), relative
    to the mean over accumulated snapshots and pixels of the intensity level |A_j| (the quantity Eq. 4 normalises by,
    PAPER.md:171, 201).  0 for identical (or all-zero) snapshots.  Needs at least two accumulated snapshots."""
    A = accumulate(stack, g)
    if len(A) < 2:
        raise ValueError("accumulation_contrast: need at least two accumulated snapshots")
    num = float(np.mean([np.mean(np.abs(A[j + 1] - A[j])) for j in range(len(A) - 1)]))
    den = float(np.mean([np.mean(np.abs(a)) for a in A]))
    return num / den if den > 0.0 else 0.0


def choose_accumulate(stack, eps: float, g_max: int = 32):
    """PAPER.md:497 (section 3.3.2): "Snapshots can be combined progressively until there is enough difference between
    adjacent accumulated snapshots."  The paper gives neither the measure nor the threshold; reading R30:
    combine progressively as in Fig. 16 -- g = 1, 2, 4, ... while g <= g_max and at least 3 accumulated snapshots remain
     -- and stop at the FIRST g whose accumulation_contrast reaches eps; if none does, take the largest
    admissible g.  Returns (g, [(g_level, contrast), ...] for the levels that were looked at)."""
    snaps = as_snapshots(stack)
    if len(snaps) < 3 or g_max < 1:
        raise ValueError("choose_accumulate: need L >= 3 and g_max >= 1")
    levels, g, last = [], 1, 1
    while g <= g_max and len(snaps) // g >= 3:
        d = accumulation_contrast(snaps, g)
        levels.append((g, d))
        last = g
        if d >= eps:
            break
        g *= 2
    return last, levels


def tlisi_windows(stack, tile: int, stride: int, C: float = 1e-6, ref_mode: int = REF_ABS,
                  M: Optional[float] = None) -> TlisiResult:
    """Eq. 2-6 on overlapping windows of `tile` pixels every `stride` pixels (reading R27, an extension)."""
    snaps = as_snapshots(stack)
    L = len(snaps)
    H, W = snaps[0].shape
    arr, keep = _snap_ptrs(snaps, H, W)
    if M is None:
        M = float(lib().fitrig_oracle_global_max(arr, L, H, W, float(C)))
    if L < 3 or stride < 1 or tile % stride:
        raise ValueError("need L >= 3 and a stride that divides the tile")
    U = L - 2
    Ty, Tx = lib().fitrig_oracle_n_windows(H, tile, stride), lib().fitrig_oracle_n_windows(W, tile, stride)
    shp = (U, Ty, Tx)
    out = [np.zeros(shp, dtype=np.float64) for _ in range(5)]
    arg = np.zeros(shp, dtype=np.int64)
    rc = lib().fitrig_oracle_tlisi_windows(arr, L, H, W, int(tile), int(stride), float(C), int(ref_mode), float(M),
                                           _ptr(out[0]), _ptr(out[1]), _ptr(out[2]), _ptr(arg), _ptr(out[3]),
                                           _ptr(out[4]))
    if rc != 0:
        raise ValueError("fitrig_oracle_tlisi_windows: bad arguments")
    return TlisiResult(M, U, Ty, Tx, out[0], out[1], out[2], arg, out[3], out[4])


def tlisi(stack, tile: int = 32, C: float = 1e-6, ref_mode: int = REF_ABS, M: Optional[float] = None,
          accumulate_g: int = 1) -> TlisiResult:
    """Eq. 2-6 for every unit and tile.  M=None -> O1 global max of the images tLISI assesses (floored at C).
    accumulate_g > 1: the images are the accumulated snapshots A_j, in fp64."""
    if accumulate_g > 1:
        return _tlisi_f64(accumulate(stack, accumulate_g), tile, C, ref_mode, M)
    snaps = as_snapshots(stack)
    L = len(snaps)
    H, W = snaps[0].shape
    arr, keep = _snap_ptrs(snaps, H, W)
    if M is None:
        M = float(lib().fitrig_oracle_global_max(arr, L, H, W, float(C)))
    U = L - 2
    if U < 1:
        raise ValueError("need L >= 3 snapshots (PAPER.md:155)")
    Ty, Tx = -(-H // tile), -(-W // tile)
    shp = (U, Ty, Tx)
    out = [np.zeros(shp, dtype=np.float64) for _ in range(5)]
    arg = np.zeros(shp, dtype=np.int64)
    rc = lib().fitrig_oracle_tlisi(arr, L, H, W, int(tile), float(C), int(ref_mode), float(M),
                                   _ptr(out[0]), _ptr(out[1]), _ptr(out[2]), _ptr(arg), _ptr(out[3]), _ptr(out[4]))
    if rc != 0:
        raise ValueError("fitrig_oracle_tlisi: bad arguments")
    return TlisiResult(M, U, Ty, Tx, out[0], out[1], out[2], arg, out[3], out[4])


def _tlisi_f64(imgs: Sequence[np.ndarray], tile: int, C: float, ref_mode: int, M: Optional[float]) -> TlisiResult:
    """O1-O5 on fp64 images (accumulated snapshots)."""
    L = len(imgs)
    if L < 3:
        raise ValueError("need at least 3 (accumulated) snapshots (PAPER.md:155)")
    H, W = imgs[0].shape
    keep = [np.ascontiguousarray(a, dtype=np.float64) for a in imgs]
    arr = (ctypes.c_void_p * L)(*[a.ctypes.data for a in keep])
    if M is None:
        M = max(max(float(a.max()) for a in keep), float(C))  # O1 on the accumulated images
    U = L - 2
    Ty, Tx = -(-H // tile), -(-W // tile)
    shp = (U, Ty, Tx)
    out = [np.zeros(shp, dtype=np.float64) for _ in range(5)]
    arg = np.zeros(shp, dtype=np.int64)
    rc = lib().fitrig_oracle_tlisi_f64(arr, L, H, W, int(tile), float(C), int(ref_mode), float(M),
                                       _ptr(out[0]), _ptr(out[1]), _ptr(out[2]), _ptr(arg), _ptr(out[3]), _ptr(out[4]))
    if rc != 0:
        raise ValueError("fitrig_oracle_tlisi_f64: bad arguments")
    return TlisiResult(M, U, Ty, Tx, out[0], out[1], out[2], arg, out[3], out[4])


def zscore(v: np.ndarray):
    """Eq. 8 / Eq. 11 over the last axes of v[U, ...] -> (mu[U], sigma[U], z like v)."""
    v = np.ascontiguousarray(v, dtype=np.float64)
    U = v.shape[0]
    n = int(np.prod(v.shape[1:]))
    mu = np.zeros(U)
    sd = np.zeros(U)
    z = np.zeros_like(v)
    lib().fitrig_oracle_zscore(_ptr(v), U, n, _ptr(mu), _ptr(sd), _ptr(z))
    return mu, sd, z


@dataclass
class Candidates:
    x: np.ndarray
    y: np.ndarray
    snapshot: np.ndarray  # unit index u (branch 0) or peak bin k* (branch 1)
    tile: np.ndarray  # ty*Tx + tx
    score: np.ndarray
    n_found: int


def select(z: np.ndarray, argmax: np.ndarray, W: int, tau: float, capacity: int = 1 << 22) -> Candidates:
    """Eq. 9: { t | z > tau } in (u, ty, tx) order."""
    z = np.ascontiguousarray(z, dtype=np.float64)
    argmax = np.ascontiguousarray(argmax, dtype=np.int64)
    U = z.shape[0]
    n = int(np.prod(z.shape[1:]))
    x = np.zeros(capacity, np.int32)
    y = np.zeros(capacity, np.int32)
    u = np.zeros(capacity, np.int32)
    t = np.zeros(capacity, np.int64)
    sc = np.zeros(capacity, np.float64)
    k = int(lib().fitrig_oracle_select(_ptr(z), _ptr(argmax), U, n, int(W), float(tau),
                                       _ptr(x), _ptr(y), _ptr(u), _ptr(t), _ptr(sc), capacity))
    m = min(k, capacity)
    return Candidates(x[:m], y[:m], u[:m], t[:m], sc[:m], k)


def spectrum(q: np.ndarray):
    """Eq. 10 with h = max magnitude: (eta[Ty,Tx], kstar[Ty,Tx]) from q[U,Ty,Tx]."""
    q = np.ascontiguousarray(q, dtype=np.float64)
    U = q.shape[0]
    n = int(np.prod(q.shape[1:]))
    eta = np.zeros(q.shape[1:], np.float64)
    ks = np.zeros(q.shape[1:], np.int32)
    lib().fitrig_oracle_spectrum(_ptr(q), U, n, _ptr(eta), _ptr(ks))
    return eta, ks


def spectrum_hsum(q: np.ndarray, harmonics: int, want_mag: bool = False):
    """Eq. 10 with h = harmonic summing over 1, 2, 4, .., `harmonics` harmonics (reading R26):
    (eta[Ty,Tx], kstar[Ty,Tx]) and, on request, the magnitude spectrum m[K, Ty, Tx]."""
    q = np.ascontiguousarray(q, dtype=np.float64)
    U = q.shape[0]
    n = int(np.prod(q.shape[1:]))
    eta = np.zeros(q.shape[1:], np.float64)
    ks = np.zeros(q.shape[1:], np.int32)
    mag = np.zeros((U // 2,) + q.shape[1:], np.float64) if want_mag else None
    lib().fitrig_oracle_spectrum_hsum(_ptr(q), U, n, int(harmonics), _ptr(eta), _ptr(ks), _ptr(mag))
    return (eta, ks, mag) if want_mag else (eta, ks)


def select_spectrum(z: np.ndarray, kstar: np.ndarray, H: int, W: int, tile: int, tau: float,
                    capacity: int = 1 << 22) -> Candidates:
    """Eq. 12 on the eta z-scores; record = (tile centre, k*, z), R18."""
    z = np.ascontiguousarray(z, dtype=np.float64)
    kstar = np.ascontiguousarray(kstar, dtype=np.int32)
    Ty, Tx = z.shape[-2], z.shape[-1]
    x = np.zeros(capacity, np.int32)
    y = np.zeros(capacity, np.int32)
    kk = np.zeros(capacity, np.int32)
    t = np.zeros(capacity, np.int64)
    sc = np.zeros(capacity, np.float64)
    k = int(lib().fitrig_oracle_select_spectrum(_ptr(z), _ptr(kstar), Ty, Tx, int(H), int(W), int(tile), float(tau),
                                                _ptr(x), _ptr(y), _ptr(kk), _ptr(t), _ptr(sc), capacity))
    m = min(k, capacity)
    return Candidates(x[:m], y[:m], kk[:m], t[:m], sc[:m], k)


@dataclass
class DetectResult:
    res: TlisiResult
    mu: np.ndarray
    sigma: np.ndarray
    z: np.ndarray
    cands: Candidates
    eta: Optional[np.ndarray] = None
    kstar: Optional[np.ndarray] = None


def run(stack, tile: int = 32, C: float = 1e-6, ref_mode: int = REF_ABS, M: Optional[float] = None,
        tau: float = 5.0, branch: int = 0, accumulate_g: int = 1, harmonics: int = 1,
        stride: int = 0) -> DetectResult:
    """Whole path on one stack: O1..O7 (branch 0) or O1..O5 + O8 (branch 1); accumulate_g > 1 first combines
    groups of g snapshots."""
    snaps = as_snapshots(stack)
    H, W = snaps[0].shape
    if stride and stride != tile:
        if branch != 0 or accumulate_g != 1:
            raise ValueError("overlapping windows: image branch, no accumulation")
        res = tlisi_windows(snaps, tile, stride, C, ref_mode, M)
    else:
        res = tlisi(snaps, tile, C, ref_mode, M, accumulate_g)
    if branch == 0:
        mu, sd, z = zscore(res.q)
        c = select(z, res.argmax, W, tau)
        return DetectResult(res, mu, sd, z, c)
    eta, ks = spectrum(res.q) if harmonics <= 1 else spectrum_hsum(res.q, harmonics)
    mu, sd, z = zscore(eta[None])
    c = select_spectrum(z[0], ks, H, W, tile, tau)
    return DetectResult(res, mu, sd, z[0], c, eta, ks)


def run_realtime(stack, tile: int = 32, C: float = 1e-6, ref_mode: int = REF_ABS, tau: float = 5.0) -> List[DetectResult]:
    """Real-time (snapshot-by-snapshot) form of the image branch, one DetectResult per unit n = 0..L-3.

    PAPER.md:189 (section 2.2.3): "For real-time processing, this maximum can be estimated from at least three
    past snapshots"; PAPER.md:457 (section 3.2, Fig. 14): unit n is computed as soon as x_n, x_{n+1}, x_{n+2} are
    on the device.  Reading (R24): the normaliser of unit n is the running maximum of everything
    seen when the unit is computed, M_n = max(max pixel of x_0 .. x_{n+2}, C) -- at least three snapshots, the
    same rule as the batch M (R2, R14) restricted to the past.  Everything else is O2-O7 on the three
    snapshots of the unit; candidate.snapshot = n.
    """
    snaps = as_snapshots(stack)
    L = len(snaps)
    if L < 3:
        raise ValueError("need L >= 3 snapshots (PAPER.md:155)")
    H, W = snaps[0].shape
    out = []
    running = max(float(np.max(snaps[0])), float(np.max(snaps[1])))
    for n in range(L - 2):
        running = max(running, float(np.max(snaps[n + 2])))  # x_{n+2} has just arrived
        res = tlisi(snaps[n:n + 3], tile, C, ref_mode, M=max(running, C))
        mu, sd, z = zscore(res.q)
        c = select(z, res.argmax, W, tau)
        c.snapshot[:] = n
        out.append(DetectResult(res, mu, sd, z, c))
    return out


def interp_eval(eta: np.ndarray, method: int, u, v) -> np.ndarray:
    """The interpolated eta surface of reading R28 at index coordinates (u, v) (tile centres at integers)."""
    eta = np.ascontiguousarray(eta, dtype=np.float64)
    Ty, Tx = eta.shape
    u, v = np.broadcast_arrays(np.asarray(u, dtype=np.float64), np.asarray(v, dtype=np.float64))
    u, v = np.ascontiguousarray(u).reshape(-1), np.ascontiguousarray(v).reshape(-1)
    assert u.shape == v.shape
    out = np.zeros(u.shape, dtype=np.float64)
    rc = lib().fitrig_oracle_interp_eval(_ptr(eta), Ty, Tx, int(method), _ptr(u), _ptr(v), len(u), _ptr(out))
    if rc != 0:
        raise ValueError("fitrig_oracle_interp_eval: bad arguments")
    return out


@dataclass
class Positions:
    x: np.ndarray  # pixels, pixel centres at integers
    y: np.ndarray
    value: np.ndarray  # the interpolated surface at (x, y)


def localise(eta: np.ndarray, tile: int, cand_tiles, method: int = INTERP_SPLINE, oversample: int = 1) -> Positions:
    """O9 (reading R28): the maximum of the interpolated eta surface within one tile of the
    centre of each selected tile (cand_tiles = ty * Tx + tx)."""
    eta = np.ascontiguousarray(eta, dtype=np.float64)
    Ty, Tx = eta.shape
    t = np.ascontiguousarray(cand_tiles, dtype=np.int64).reshape(-1)
    x, y, val = np.zeros(len(t)), np.zeros(len(t)), np.zeros(len(t))
    rc = lib().fitrig_oracle_localise(_ptr(eta), Ty, Tx, int(tile), int(method), int(oversample), _ptr(t), len(t),
                                      _ptr(x), _ptr(y), _ptr(val))
    if rc != 0:
        raise ValueError("fitrig_oracle_localise: bad arguments")
    return Positions(x, y, val)


def run_realtime_frequency(stack, window: int, tile: int = 32, C: float = 1e-6, ref_mode: int = REF_ABS,
                           tau: float = 5.0, harmonics: int = 1) -> List[Optional[DetectResult]]:
    """Real-time form of the image-frequency branch: one entry per unit n = 0..L-3, None while fewer than
    `window` - 2 units exist.

    PAPER.md:453 (section 3.2): "In image-frequency domain FITrig, a set of time-sequential snapshots needs to be
    loaded onto the device.  Rather than loading all snapshots at once ..." with the timeline of Fig. 14
    (PAPER.md:457-467), and the tLISI cube of PAPER.md:341.  Reading R29: snapshots arrive one at a time;
    once unit n is computed, Eq. 10-12 run over the cube of the LAST U_w = window - 2 units, n - U_w + 1 .. n, i.e.
    over snapshots x_{n-U_w+1} .. x_{n+2}; every tile matrix of that cube is normalised by the running maximum
    M_n = max(largest pixel of x_0 .. x_{n+2}, C) (R24).  eta scales with 1/M^2, z (Eq. 11) does not, so the
    candidates are those of the batch branch on the same `window` snapshots.
    """
    snaps = as_snapshots(stack)
    L = len(snaps)
    if L < 3 or window < 3:
        raise ValueError("need L >= 3 snapshots and a window of at least 3 snapshots (PAPER.md:155)")
    Uw = window - 2
    out: List[Optional[DetectResult]] = []
    running = max(float(np.max(snaps[0])), float(np.max(snaps[1])))
    for n in range(L - 2):
        running = max(running, float(np.max(snaps[n + 2])))  # x_{n+2} has just arrived
        if n < Uw - 1:
            out.append(None)
            continue
        out.append(run(snaps[n - Uw + 1:n + 3], tile=tile, C=C, ref_mode=ref_mode, M=max(running, C), tau=tau,
                       branch=1, harmonics=harmonics))
    return out
