"""Thin ctypes binding of libbluebild_b200.so (include/bluebild.h). Argument marshalling only:
every step of the path runs in the library's CUDA kernels; there is no CPU fallback, and a missing
library or a missing GPU raises.

Matrices are column-major. Host arguments are numpy arrays (converted to Fortran
order if needed). Device arguments are ``DeviceMatrix`` objects (a torch CUDA tensor holding the
column-major data) — torch is used for device memory and streams only.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbluebild_b200.so")

BB_OK = 0
VARIANT_FP32 = 0
VARIANT_TF32X3 = 1
VARIANT_FP16X3 = 2
VARIANT_FP16_FP8 = 3
FILTERS = {"lsq": 0, "std": 1}
GRAM_MODES = {"sinc": 0, "identity": 1}
_VARIANTS = {"fp32": VARIANT_FP32, "tf32x3": VARIANT_TF32X3, "fp16x3": VARIANT_FP16X3, "fp16fp8": VARIANT_FP16_FP8, 0: 0, 1: 1, 2: 2, 3: 3}

EXPORTS = ["bb_ctx_create", "bb_ctx_destroy", "bb_synth_create", "bb_synth_destroy", "bb_synth_reset",
           "bb_synth_collect", "bb_synth_collect_ex", "bb_synth_collect_batch", "bb_synth_collect_eig", "bb_synth_flush", "bb_synth_get", "bb_synth_timings",
           "bb_synth_status", "bb_synth_launches", "bb_eig", "bb_level_weights", "bb_uvgrid_create", "bb_uvgrid_add",
           "bb_uvgrid_destroy", "bb_synth_set_weighting", "bb_estimate_n_eig", "bb_kmeans_levels", "bb_kmeans_levels_static", "bb_status_string", "bb_version",
           "bb_plan_collect_split", "bb_nufft_plan", "bb_nufft_create", "bb_nufft_destroy", "bb_nufft_collect_eig", "bb_nufft_collect", "bb_nufft_get", "bb_nufft_stats"]

_lib = None


class BluebildError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        msg = _lib.bb_status_string(code).decode() if _lib is not None else "?"
        super().__init__("%s failed: [%d] %s" % (where, code, msg))


def load_library(path: str = LIB_PATH):
    """Load the C-ABI library; raises if it has not been built (python -m paper_2310_09200_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(path):
        raise ImportError("CUDA extension %s is missing: run `python -m paper_2310_09200_b200.build` "
                          "(there is no CPU fallback)" % path)
    lib = ctypes.CDLL(path)
    vp, i32, i64, f64 = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_double
    pp = ctypes.POINTER(ctypes.c_void_p)
    pd = ctypes.POINTER(ctypes.c_double)
    sig = {
        "bb_ctx_create": ([i32, vp, pp], i32),
        "bb_ctx_destroy": ([vp], i32),
        "bb_synth_create": ([vp, i64, vp, i64, i32, i32, pp], i32),
        "bb_synth_destroy": ([vp], i32),
        "bb_synth_reset": ([vp], i32),
        "bb_synth_collect": ([vp, i32, i32, i32, f64, vp, i32, vp, i32, vp, i32, vp, i32], i32),
        "bb_synth_collect_ex": ([vp, i32, i32, i32, f64, vp, i32, vp, i32, vp, i32, vp, i32, i32, vp, i32], i32),
        "bb_synth_collect_batch": ([vp, i32, i32, i32, i32, vp, vp, i32, i64, vp, i32, i64, vp, i32, i64, vp, i32], i32),
        "bb_synth_collect_eig": ([vp, i32, i32, f64, vp, i32, vp, i32, vp, i32], i32),
        "bb_synth_flush": ([vp], i32),
        "bb_synth_get": ([vp, i32, vp], i32),
        "bb_synth_timings": ([vp, pd, pd, pd, pd], i32),
        "bb_synth_launches": ([vp], i64),
        "bb_eig": ([vp, i32, i32, i32, f64, vp, i32, vp, i32, vp, i32, vp, vp, i32], i32),
        "bb_estimate_n_eig": ([vp, vp, i32, f64, ctypes.POINTER(ctypes.c_int)], i32),
        "bb_kmeans_levels": ([vp, vp, i32, i32, i32, vp, i32], i32),
        "bb_kmeans_levels_static": ([i32, vp, vp, i32, i32, i32, vp, i32, vp], i32),
        "bb_synth_status": ([vp], i32),
        "bb_level_weights": ([vp, vp, i32, vp, i32, i32, i32, vp, vp, i32], i32),
        "bb_uvgrid_create": ([vp, f64, vp, vp, f64, pp], i32),
        "bb_uvgrid_add": ([vp, i32, f64, vp, i32], i32),
        "bb_uvgrid_destroy": ([vp], i32),
        "bb_synth_set_weighting": ([vp, vp], i32),
        "bb_plan_collect_split": ([i32, i64, i32, i32, i32, i32, i32], i32),
        "bb_nufft_plan": ([i64, vp, i64, i32, vp, i32, f64, f64, i32, i32, ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_int64), pd, pd], i32),
        "bb_nufft_create": ([vp, i64, vp, i64, i32, f64, i32, i32, pp], i32),
        "bb_nufft_destroy": ([vp], i32),
        "bb_nufft_collect_eig": ([vp, i32, i32, f64, vp, i32, vp, i32, vp, i32], i32),
        "bb_nufft_collect": ([vp, i32, i32, i32, f64, vp, i32, vp, i32, vp, i32, vp, i32, i32, vp], i32),
        "bb_nufft_get": ([vp, i32, vp], i32),
        "bb_nufft_stats": ([vp, ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_int64)], i32),
        "bb_status_string": ([i32], ctypes.c_char_p),
        "bb_version": ([], ctypes.c_char_p),
    }
    for name, (args, res) in sig.items():
        fn = getattr(lib, name)
        fn.argtypes, fn.restype = args, res
    _lib = lib
    return lib


def _check(code, where):
    if code != BB_OK:
        raise BluebildError(code, where)


class DeviceMatrix:
    """A column-major (rows x cols) matrix in device memory, backed by a torch CUDA tensor of shape
    (cols, rows) (its row-major storage is the column-major matrix; ld = rows)."""

    def __init__(self, tensor, rows, cols):
        assert tensor.is_cuda and tensor.is_contiguous()
        self.tensor, self.rows, self.cols, self.ld = tensor, rows, cols, rows

    @classmethod
    def from_numpy(cls, a, dtype, device="cuda:0"):
        import torch
        a = np.asarray(a, dtype=dtype)
        if a.ndim == 1:
            a = a[:, None]
        t = torch.from_numpy(np.ascontiguousarray(a.T)).to(device)
        return cls(t, a.shape[0], a.shape[1])

    @property
    def ptr(self):
        return self.tensor.data_ptr()


def _marshal(a, dtype, keep):
    """-> (pointer as int, rows, cols, ld). numpy -> Fortran-ordered host buffer (kept alive in `keep`)."""
    if a is None:
        return None, 0, 0, 1
    if isinstance(a, DeviceMatrix):
        return a.ptr, a.rows, a.cols, a.ld
    arr = np.asarray(a, dtype=dtype)
    if arr.ndim == 1:
        arr = arr[:, None]
    arr = np.asfortranarray(arr)
    keep.append(arr)
    return arr.ctypes.data, arr.shape[0], arr.shape[1], max(arr.shape[0], 1)


class Context:
    """bb_ctx: device + stream + library handles (PAPER.md:262 'Context')."""

    def __init__(self, device: int = 0, stream=None):
        lib = load_library()
        h = ctypes.c_void_p()
        sp = None
        if stream is not None:
            sp = ctypes.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))
        _check(lib.bb_ctx_create(int(device), sp, ctypes.byref(h)), "bb_ctx_create")
        self._h, self._stream, self.device = h, stream, device
        self._children = []                      # weak references to the imaging handles created from this context

    def close(self):
        """Destroys the context; imaging handles created from it are closed first (bb_ctx_destroy refuses while any is alive)."""
        if getattr(self, "_h", None) and _lib is not None:
            for ref in self._children:
                child = ref()
                if child is not None:
                    child.close()
            self._children = []
            _lib.bb_ctx_destroy(self._h)
            self._h = None

    __del__ = close

    def estimate_n_eig(self, lam, energy_fraction: float) -> int:
        """number of leading eigenvalues holding `energy_fraction` of the total energy."""
        lam = np.ascontiguousarray(lam, dtype=np.float64)
        out = ctypes.c_int()
        _check(_lib.bb_estimate_n_eig(self._h, lam.ctypes.data, lam.size, float(energy_fraction), ctypes.byref(out)),
               "bb_estimate_n_eig")
        return out.value

    def kmeans_levels(self, lam, n_levels: int, log_domain: bool = True):
        """level intervals (n_levels, 2) from exact 1-D k-means of the eigenvalues."""
        lam = np.ascontiguousarray(lam, dtype=np.float64)
        iv = np.zeros((n_levels, 2), dtype=np.float64, order="F")
        _check(_lib.bb_kmeans_levels(self._h, lam.ctypes.data, lam.size, int(n_levels), int(bool(log_domain)),
                                     iv.ctypes.data, n_levels), "bb_kmeans_levels")
        return iv

    def level_weights(self, lam, intervals, filters=None):
        """Alg. 1 l.7-8: D (n_levels, n_eig) float32 from eigenvalues and closed intervals (the library's own kernel)."""
        lam = np.ascontiguousarray(lam, dtype=np.float64)
        iv = np.asfortranarray(np.asarray(intervals, dtype=np.float64).reshape(-1, 2))
        kinds = [FILTERS[f] for f in (filters or ["lsq"])]
        arr = (ctypes.c_int * len(kinds))(*kinds)
        L = iv.shape[0] * len(kinds)
        D = np.zeros((L, lam.size), dtype=np.float32, order="F")
        _check(_lib.bb_level_weights(self._h, lam.ctypes.data, lam.size, iv.ctypes.data, iv.shape[0], iv.shape[0], len(kinds),
                                     ctypes.cast(arr, ctypes.c_void_p), D.ctypes.data, L), "bb_level_weights")
        return D

    def eig(self, S, W, xyz, wavelength, n_eig, want_B=True):
        """Alg. 1 lines 2-4: (lambda desc float64 (n_eig,), B complex64 (n_ant, n_eig))."""
        keep = []
        Sp, n_beam, _, lds = _marshal(S, np.complex64, keep)
        Wp, _, _, ldw = _marshal(W, np.complex64, keep)
        Xp, n_ant, _, ldx = _marshal(xyz, np.float64, keep)
        lam = np.zeros(n_eig, dtype=np.float64)
        B = np.zeros((n_ant, n_eig), dtype=np.complex64, order="F") if want_B else None
        _check(_lib.bb_eig(self._h, n_ant, n_beam, n_eig, float(wavelength), Wp, ldw, Sp, lds, Xp, ldx,
                           lam.ctypes.data, B.ctypes.data if want_B else None, max(n_ant, 1)), "bb_eig")
        return lam, B


class UVGrid:
    """bb_uvgrid: sampling density on a uv grid of cell 1/FoV for "uniform" weighting (Section 3.5)."""

    def __init__(self, ctx: Context, cell: float, e_u, e_v, max_uv: float):
        eu = np.ascontiguousarray(e_u, dtype=np.float64)
        ev = np.ascontiguousarray(e_v, dtype=np.float64)
        h = ctypes.c_void_p()
        _check(_lib.bb_uvgrid_create(ctx._h, float(cell), eu.ctypes.data, ev.ctypes.data, float(max_uv), ctypes.byref(h)), "bb_uvgrid_create")
        self._h, self.ctx = h, ctx

    def add(self, xyz, wavelength):
        keep = []
        Xp, n_ant, _, ldx = _marshal(xyz, np.float64, keep)
        _check(_lib.bb_uvgrid_add(self._h, n_ant, float(wavelength), Xp, ldx), "bb_uvgrid_add")

    def close(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.bb_uvgrid_destroy(self._h)
            self._h = None

    __del__ = close


class StandardSynthesis:
    """bb_synth: the imaging handle (Algorithm 1)."""

    def __init__(self, ctx: Context, pix, n_levels: int, variant="fp32"):
        keep = []
        Pp, n_pix, c, ld = _marshal(pix, np.float64, keep)
        assert c == 3, "pix must be (n_pix, 3)"
        h = ctypes.c_void_p()
        _check(_lib.bb_synth_create(ctx._h, n_pix, Pp, ld, int(n_levels), _VARIANTS[variant], ctypes.byref(h)),
               "bb_synth_create")
        self._h, self.ctx, self.n_pix, self.n_levels = h, ctx, n_pix, n_levels
        import weakref
        ctx._children.append(weakref.ref(self))

    def close(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.bb_synth_destroy(self._h)
            self._h = None

    __del__ = close

    def reset(self):
        _check(_lib.bb_synth_reset(self._h), "bb_synth_reset")

    def set_weighting(self, grid):
        """Uniform weighting (Section 3.5) from a UVGrid for the collects made from now on; None = natural."""
        _check(_lib.bb_synth_set_weighting(self._h, None if grid is None else grid._h), "bb_synth_set_weighting")
        self._weighting = grid                                 # keep the grid alive while the handle refers to it

    def collect(self, S, W, xyz, wavelength, n_eig, intervals, filters=None, gram="sinc"):
        """Algorithm 1. filters: None (one LSQ filter) or a sequence of "lsq" / "std"; the handle's n_levels must be
        len(filters) * len(intervals) and image f * n_intervals + i belongs to (filter f, interval i).
        gram: "sinc" (Eq. 11) or "identity" (dirty-image eigendecomposition)."""
        keep = []
        Sp, n_beam, _, lds = _marshal(S, np.complex64, keep)
        Wp, _, _, ldw = _marshal(W, np.complex64, keep)
        Xp, n_ant, _, ldx = _marshal(xyz, np.float64, keep)
        Ip, _, _, ldi = _marshal(intervals, np.float64, keep)
        if filters is None and gram == "sinc":
            _check(_lib.bb_synth_collect(self._h, n_ant, n_beam, int(n_eig), float(wavelength), Wp, ldw, Sp, lds, Xp, ldx,
                                         Ip, ldi), "bb_synth_collect")
            return
        kinds = [FILTERS[f] for f in (filters or ["lsq"])]
        arr = (ctypes.c_int * len(kinds))(*kinds)
        _check(_lib.bb_synth_collect_ex(self._h, n_ant, n_beam, int(n_eig), float(wavelength), Wp, ldw, Sp, lds, Xp, ldx,
                                        Ip, ldi, len(kinds), ctypes.cast(arr, ctypes.c_void_p), GRAM_MODES[gram]),
               "bb_synth_collect_ex")

    def collect_batch(self, S, W, xyz, wavelengths, n_eig, intervals):
        """Algorithm 1 for several collects with batched device eigensolves. S: (T, n_beam, n_beam) complex64,
        xyz: (T, n_ant, 3) float64, W: None, (n_ant, n_beam) shared, or (T, n_ant, n_beam); numpy arrays."""
        S = np.ascontiguousarray(np.transpose(np.asarray(S, dtype=np.complex64), (0, 2, 1)))      # column-major slices
        X = np.ascontiguousarray(np.transpose(np.asarray(xyz, dtype=np.float64), (0, 2, 1)))
        T, n_beam = S.shape[0], S.shape[1]
        n_ant = X.shape[2]
        wl = np.ascontiguousarray(np.broadcast_to(np.asarray(wavelengths, dtype=np.float64), (T,)))
        Wp, ldw, sw = None, 0, 0
        if W is not None:
            W = np.asarray(W, dtype=np.complex64)
            if W.ndim == 2:
                W = np.ascontiguousarray(W.T)
            else:
                W = np.ascontiguousarray(np.transpose(W, (0, 2, 1)))
                sw = n_ant * n_beam
            Wp, ldw = W.ctypes.data, n_ant
        keep = []
        Ip, _, _, ldi = _marshal(intervals, np.float64, keep)
        _check(_lib.bb_synth_collect_batch(self._h, T, n_ant, n_beam, int(n_eig), wl.ctypes.data, Wp, ldw, sw, S.ctypes.data, n_beam,
                                           n_beam * n_beam, X.ctypes.data, n_ant, 3 * n_ant, Ip, ldi), "bb_synth_collect_batch")

    def collect_eig(self, B, D, xyz, wavelength):
        keep = []
        Bp, n_ant, n_eig, ldb = _marshal(B, np.complex64, keep)
        Dp, _, _, ldd = _marshal(D, np.float32, keep)
        Xp, _, _, ldx = _marshal(xyz, np.float64, keep)
        _check(_lib.bb_synth_collect_eig(self._h, n_ant, n_eig, float(wavelength), Bp, ldb, Dp, ldd, Xp, ldx),
               "bb_synth_collect_eig")

    def flush(self):
        _check(_lib.bb_synth_flush(self._h), "bb_synth_flush")

    def status(self):
        """Flush, synchronise and raise if a collect was dropped on the device (Gram not positive definite,
        eigensolver failure, coordinates beyond the phase generator's range)."""
        _check(_lib.bb_synth_status(self._h), "bb_synth_status")

    def get(self, level: int, out=None):
        """Level image as float32 (n_pix,). `out` may be a numpy array or a torch CUDA tensor."""
        if out is None:
            out = np.empty(self.n_pix, dtype=np.float32)
        ptr = out.data_ptr() if hasattr(out, "data_ptr") else out.ctypes.data
        _check(_lib.bb_synth_get(self._h, int(level), ptr), "bb_synth_get")
        return out

    def images(self):
        return np.stack([self.get(l) for l in range(self.n_levels)])

    def timings(self):
        v = [ctypes.c_double() for _ in range(4)]
        _check(_lib.bb_synth_timings(self._h, *[ctypes.byref(x) for x in v]), "bb_synth_timings")
        return dict(gram_ms=v[0].value, eig_ms=v[1].value, prep_ms=v[2].value, synth_ms=v[3].value)

    def launches(self) -> int:
        return int(_lib.bb_synth_launches(self._h))


KMEANS_STATIC_MAX_N = 1024   # BB_KMEANS_STATIC_MAX_N


def kmeans_levels_static(device: int, stream: int, lambda_ptr: int, n: int, n_levels: int, log_domain: bool,
                         intervals_ptr: int, ld_int: int, status_ptr: int) -> None:
    """bb_kmeans_levels_static: PAPER.md:164 level intervals for callers that must not allocate GPU memory at call
    time (fixed memory plan, a framework pool that owns HBM, latency-bound loops that cannot afford cudaMalloc's
    device-wide stall). Everything is the caller's and on the device: `lambda_ptr` n float64 values, `intervals_ptr`
    n_levels x 2 float64 column-major with leading dimension ld_int, `status_ptr` one int32 (0 = written, 1 = fewer
    positive eigenvalues than levels); `stream` is a cudaStream_t as an integer (0 = default stream). Enqueues and
    returns without synchronising and without allocating here either: pass raw addresses (tensor.data_ptr()).
    n above KMEANS_STATIC_MAX_N raises BluebildError code 7. The first call on a device does a one-time address
    look-up: make it before any stream capture. Calls that overlap on one GPU share the scratch and race."""
    load_library()
    code = _lib.bb_kmeans_levels_static(int(device), stream or None, lambda_ptr, int(n), int(n_levels), int(bool(log_domain)),
                                        intervals_ptr, int(ld_int), status_ptr)
    if code == 7:
        raise BluebildError(code, "bb_kmeans_levels_static (n = %d, limit %d eigenvalues)" % (n, KMEANS_STATIC_MAX_N))
    _check(code, "bb_kmeans_levels_static")


def plan_collect_split(variant, n_pix, n_ant, n_eig, n_levels, n_collects, sm_count=148) -> int:
    """How many collect ranges a launch over n_collects queued collects is split into (host-only query, no device needed)."""
    load_library()
    return int(_lib.bb_plan_collect_split(_VARIANTS[variant], int(n_pix), int(n_ant), int(n_eig), int(n_levels), int(n_collects), int(sm_count)))


def nufft_plan(pix, xyz, wavelength, eps=1e-6, n_part_in=1, n_part_out=1):
    """Host-only (Section 3.4.1): transforms, largest / summed fine-grid points and non-empty input-cell fraction of one collect."""
    load_library()
    P = np.asfortranarray(np.asarray(pix, dtype=np.float64)); X = np.asfortranarray(np.asarray(xyz, dtype=np.float64))
    nt, mx, sm, ne = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_double(), ctypes.c_double()
    _check(_lib.bb_nufft_plan(P.shape[0], P.ctypes.data, P.shape[0], X.shape[0], X.ctypes.data, X.shape[0], float(wavelength), float(eps),
                              int(n_part_in), int(n_part_out), ctypes.byref(nt), ctypes.byref(mx), ctypes.byref(sm), ctypes.byref(ne)), "bb_nufft_plan")
    return dict(n_transforms=nt.value, max_grid_points=mx.value, sum_grid_points=sm.value, nonempty_input_cells=ne.value)


class NufftSynthesis:
    """bb_nufft: NUFFT Synthesis (Section 3.4, Algorithm 3) — the same level images as StandardSynthesis.collect_eig up to
    `eps`, through Gram-corrected visibilities per level and a partitioned 3-D type-3 NUFFT."""

    def __init__(self, ctx: Context, pix, n_levels: int, eps: float = 1e-6, n_part_in: int = 1, n_part_out: int = 1):
        keep = []
        Pp, n_pix, c, ld = _marshal(pix, np.float64, keep)
        assert c == 3, "pix must be (n_pix, 3)"
        h = ctypes.c_void_p()
        _check(_lib.bb_nufft_create(ctx._h, n_pix, Pp, ld, int(n_levels), float(eps), int(n_part_in), int(n_part_out),
                                    ctypes.byref(h)), "bb_nufft_create")
        self._h, self.ctx, self.n_pix, self.n_levels = h, ctx, n_pix, n_levels
        import weakref
        ctx._children.append(weakref.ref(self))

    def close(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.bb_nufft_destroy(self._h)
            self._h = None

    __del__ = close

    def collect_eig(self, B, D, xyz, wavelength):
        keep = []
        Bp, n_ant, n_eig, ldb = _marshal(B, np.complex64, keep)
        Dp, _, _, ldd = _marshal(D, np.float32, keep)
        Xp, _, _, ldx = _marshal(xyz, np.float64, keep)
        _check(_lib.bb_nufft_collect_eig(self._h, n_ant, n_eig, float(wavelength), Bp, ldb, Dp, ldd, Xp, ldx), "bb_nufft_collect_eig")

    def collect(self, S, W, xyz, wavelength, n_eig, intervals, filters=None):
        """Algorithm 3 from S, W, xyz and the intervals; filters as StandardSynthesis.collect."""
        keep = []
        Sp, n_beam, _, lds = _marshal(S, np.complex64, keep)
        Wp, _, _, ldw = _marshal(W, np.complex64, keep)
        Xp, n_ant, _, ldx = _marshal(xyz, np.float64, keep)
        Ip, _, _, ldi = _marshal(intervals, np.float64, keep)
        kinds = [FILTERS[f] for f in (filters or ["lsq"])]
        arr = (ctypes.c_int * len(kinds))(*kinds)
        _check(_lib.bb_nufft_collect(self._h, n_ant, n_beam, int(n_eig), float(wavelength), Wp, ldw, Sp, lds, Xp, ldx, Ip, ldi,
                                     len(kinds), ctypes.cast(arr, ctypes.c_void_p)), "bb_nufft_collect")

    def images(self):
        out = np.empty((self.n_levels, self.n_pix), dtype=np.float32)
        for l in range(self.n_levels):
            _check(_lib.bb_nufft_get(self._h, l, out[l].ctypes.data), "bb_nufft_get")
        return out

    def stats(self):
        a, b = ctypes.c_int64(), ctypes.c_int64()
        _check(_lib.bb_nufft_stats(self._h, ctypes.byref(a), ctypes.byref(b)), "bb_nufft_stats")
        return dict(n_transforms=a.value, max_grid_points=b.value)
