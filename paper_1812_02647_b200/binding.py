"""Thin ctypes binding of include/hs.h: same names, argument marshalling only.

Every step of the path runs in libhs.so's CUDA kernels; PyTorch supplies device memory and streams.  There is no
fallback: if libhs.so is missing (run `python -m paper_1812_02647_b200.build`) importing this module raises.
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
# The binding reads no environment variable.  A program that wants another build of the same sources in this directory
# (libhs_tuning.so: the -DHS_TUNING build of the builder's sweeps and of the forced-timeout test) says so in code, before
# the first import of this module:  import paper_1812_02647_b200 as pkg; pkg.LIBRARY = "libhs_tuning.so"
import paper_1812_02647_b200 as _pkg

LIB_PATH = os.path.join(_HERE, os.path.basename(_pkg.__dict__.get("LIBRARY", "libhs.so")))

HS_STANDARD, HS_MAX, HS_FREQBIN, HS_GREEDY = 0, 1, 2, 3
HS_OUT_FULL, HS_OUT_REDUCED, HS_OUT_BOTH = 1, 2, 3
HS_ALGO_AUTO, HS_ALGO_DIRECT, HS_ALGO_TILED, HS_ALGO_TWOPHASE, HS_ALGO_GATHER, HS_ALGO_GROUPED, HS_ALGO_GENERAL = 0, 1, 2, 3, 4, 5, 6
HS_LEVELS_DYADIC, HS_LEVELS_ALL = 0, 1
HS_WINDOW_C2, HS_WINDOW_PRINTED, HS_TERM_INTERP = 0, 1, 2
LEVELS = {"dyadic": HS_LEVELS_DYADIC, "all": HS_LEVELS_ALL}
WINDOWS = {"c2": HS_WINDOW_C2, "printed": HS_WINDOW_PRINTED, "interp": HS_TERM_INTERP}
(HS_OK, HS_ERR_INVALID_ARG, HS_ERR_NULL_POINTER, HS_ERR_MISALIGNED, HS_ERR_UNSUPPORTED, HS_ERR_WORKSPACE, HS_ERR_CUDA,
 HS_ERR_DEVICE_TIMEOUT) = range(8)
HS_ERR_SCRATCH_LIMIT = 8
VARIANTS = {"standard": HS_STANDARD, "max": HS_MAX, "freqbin": HS_FREQBIN, "greedy": HS_GREEDY}
OUT_MODES = {"full": HS_OUT_FULL, "reduced": HS_OUT_REDUCED, "both": HS_OUT_BOTH}
ALGOS = {"auto": HS_ALGO_AUTO, "direct": HS_ALGO_DIRECT, "tiled": HS_ALGO_TILED, "twophase": HS_ALGO_TWOPHASE,
         "gather": HS_ALGO_GATHER, "grouped": HS_ALGO_GROUPED}

if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build the CUDA library with `python -m paper_1812_02647_b200.build` "
                      "(there is no CPU fallback)")

lib = ctypes.CDLL(LIB_PATH)
_i64, _p, _int, _sz = ctypes.c_int64, ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t
_SIGS = {
    "hs_plan_create": ([_i64, _i64, _int, _int, _int], _p),
    "hs_plan_create_ex": ([_i64, _i64, _int, _int, _int, _int, _int], _p),
    "hs_plan_create_2d": ([_i64, _i64, _i64, _int, _int, _int], _p),
    "hs_execute": ([_p, _p, _p, _p, _p, _p], _int),
    "hs_execute_complex": ([_p, _p, ctypes.c_float, _p, _p, _p, _p], _int),
    "hs_destroy": ([_p], _int),
    "hs_last_error": ([], _int),
    "hs_error_string": ([_int], ctypes.c_char_p),
    "hs_version": ([], ctypes.c_char_p),
    "hs_plan_levels": ([_p], _int),
    "hs_plan_set_algo": ([_p, _int], _int),
    "hs_plan_algo": ([_p], _int),
    "hs_plan_workspace_bytes": ([_p], _sz),
    "hs_plan_set_workspace": ([_p, _p, _sz], _int),
    "hs_plan_launches": ([_p], _int),
    "hs_plan_device_status": ([_p, _p], _int),
    "hs_execute_host": ([_p, _p, _p, _p, _p, _p], _int),
    "hs_plan_host_staging_bytes": ([_p, _i64], _sz),
    "hs_plan_set_host_staging": ([_p, _p, _sz, _i64], _int),
    "hs_debug_greedy_paths": ([_p, _p, _p, _p], _int),
    "hs_execute_candidates": ([_p, _p, ctypes.c_float, _p, _i64, _p, _p], _int),
    "hs_execute_static": ([_p, _p, _p, _p, _p, _p], _int),
    "hs_static_scratch_bytes": ([], _sz),
}
for _name, (_args, _res) in _SIGS.items():
    _f = getattr(lib, _name)
    _f.argtypes, _f.restype = _args, _res


class HsError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {lib.hs_error_string(code).decode()} (hs_status {code})")


def _check(code: int, where: str):
    if code != HS_OK:
        raise HsError(code, where)


def _ptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _stream(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def hs_plan_create(nbins: int, batch: int, Hmax: int, variant, out_mode):
    v = VARIANTS[variant] if isinstance(variant, str) else int(variant)
    o = OUT_MODES[out_mode] if isinstance(out_mode, str) else int(out_mode)
    h = lib.hs_plan_create(int(nbins), int(batch), int(Hmax), v, o)
    if not h:
        raise HsError(lib.hs_last_error(), "hs_plan_create")
    return Plan(h, int(nbins), int(batch), int(Hmax), v, o)


def hs_plan_create_ex(nbins: int, batch: int, Hmax: int, variant, out_mode, levels="dyadic", window="c2"):
    v = VARIANTS[variant] if isinstance(variant, str) else int(variant)
    o = OUT_MODES[out_mode] if isinstance(out_mode, str) else int(out_mode)
    lv = LEVELS[levels] if isinstance(levels, str) else int(levels)
    w = WINDOWS[window] if isinstance(window, str) else int(window)
    h = lib.hs_plan_create_ex(int(nbins), int(batch), int(Hmax), v, o, lv, w)
    if not h:
        raise HsError(lib.hs_last_error(), "hs_plan_create_ex")
    return Plan(h, int(nbins), int(batch), int(Hmax), v, o)


def hs_plan_create_2d(nbins: int, nz: int, batch: int, Hmax: int, variant, out_mode):
    v = VARIANTS[variant] if isinstance(variant, str) else int(variant)
    o = OUT_MODES[out_mode] if isinstance(out_mode, str) else int(out_mode)
    h = lib.hs_plan_create_2d(int(nbins), int(nz), int(batch), int(Hmax), v, o)
    if not h:
        raise HsError(lib.hs_last_error(), "hs_plan_create_2d")
    return Plan(h, int(nbins), int(batch), int(Hmax), v, o, nz=int(nz))


class Plan:
    """Owns one hs_plan handle plus the torch tensors lent to it as workspace/staging."""

    def __init__(self, handle, nbins, batch, Hmax, variant, out_mode, nz=1):
        self.handle = ctypes.c_void_p(handle)
        self.nbins, self.batch, self.Hmax, self.variant, self.out_mode = nbins, batch, Hmax, variant, out_mode
        self.nz = nz
        self.levels = lib.hs_plan_levels(self.handle)
        self._ws = None
        self._staging = None

    # -- thin wrappers, one per C function ---------------------------------------------------------------------
    def set_algo(self, algo):
        a = ALGOS[algo] if isinstance(algo, str) else int(algo)
        _check(lib.hs_plan_set_algo(self.handle, a), "hs_plan_set_algo")
        self._ws = None
        return self

    @property
    def algo(self) -> int:
        return lib.hs_plan_algo(self.handle)

    def workspace_bytes(self) -> int:
        return lib.hs_plan_workspace_bytes(self.handle)

    def set_workspace(self, ws):
        """ws: a torch uint8 CUDA tensor (kept alive by the plan) or None when no workspace is needed."""
        nbytes = 0 if ws is None else ws.numel() * ws.element_size()
        _check(lib.hs_plan_set_workspace(self.handle, _ptr(ws), nbytes), "hs_plan_set_workspace")
        self._ws = ws
        return self

    def ensure_workspace(self, device=None):
        """Allocate (with torch) and set the workspace the resolved algorithm needs."""
        import torch
        need = self.workspace_bytes()
        if need and (self._ws is None or self._ws.numel() < need):
            self.set_workspace(torch.empty(need, dtype=torch.uint8, device=device or "cuda"))
        return self

    def launches(self) -> int:
        return lib.hs_plan_launches(self.handle)

    def device_status(self, stream=None) -> int:
        """hs_plan_device_status: synchronises the stream; raises HsError(HS_ERR_DEVICE_TIMEOUT) if a kernel gave up a wait."""
        _check(lib.hs_plan_device_status(self.handle, _stream(stream)), "hs_plan_device_status")
        return HS_OK

    def hs_execute(self, d_x, d_sums=None, d_max=None, d_argmax=None, stream=None):
        _check(lib.hs_execute(self.handle, _ptr(d_x), _ptr(d_sums), _ptr(d_max), _ptr(d_argmax), _stream(stream)),
               "hs_execute")

    def hs_execute_static(self, d_x, d_sums=None, d_max=None, d_argmax=None, stream=None):
        """eqs. 2-3 through the library's built-in scratch array, for callers that cannot allocate device memory (see
        include/hs.h): the caller passes inputs and outputs only; no workspace is set, taken or allocated.  Raises
        HsError(HS_ERR_SCRATCH_LIMIT) when one spectrum's arrays exceed hs_static_scratch_bytes().  Calls share the one
        array: do not let two of them overlap on the GPU."""
        _check(lib.hs_execute_static(self.handle, _ptr(d_x), _ptr(d_sums), _ptr(d_max), _ptr(d_argmax), _stream(stream)),
               "hs_execute_static")

    def hs_execute_complex(self, d_F, scale, d_sums=None, d_max=None, d_argmax=None, stream=None):
        """d_F: complex64 (or float32 [..., 2]) CUDA tensor [batch][nbins]; x = |F|^2 * scale - 1 is formed inside the kernels."""
        _check(lib.hs_execute_complex(self.handle, _ptr(d_F), ctypes.c_float(scale), _ptr(d_sums), _ptr(d_max),
                                      _ptr(d_argmax), _stream(stream)), "hs_execute_complex")

    def run_complex(self, d_F, scale, stream=None):
        """Allocate the outputs, execute on the complex series, return (sums, max, argmax)."""
        import torch
        assert d_F.is_cuda and d_F.is_contiguous() and tuple(d_F.shape[:2]) == (self.batch, self.nbins)
        sums = vmax = amax = None
        if self.out_mode & HS_OUT_FULL:
            sums = torch.empty((self.batch, self.levels, self.nbins), dtype=torch.float32, device=d_F.device)
        if self.out_mode & HS_OUT_REDUCED:
            vmax = torch.empty((self.batch, self.nbins), dtype=torch.float32, device=d_F.device)
            amax = torch.empty((self.batch, self.nbins), dtype=torch.uint8, device=d_F.device)
        self.ensure_workspace(d_F.device)
        self.hs_execute_complex(d_F, scale, sums, vmax, amax, stream)
        return sums, vmax, amax

    def host_staging_bytes(self, slab_spectra: int) -> int:
        return lib.hs_plan_host_staging_bytes(self.handle, int(slab_spectra))

    def set_host_staging(self, staging, slab_spectra: int):
        _check(lib.hs_plan_set_host_staging(self.handle, _ptr(staging), staging.numel() * staging.element_size(),
                                            int(slab_spectra)), "hs_plan_set_host_staging")
        self._staging = staging
        return self

    def hs_execute_host(self, h_x, h_sums=None, h_max=None, h_argmax=None, stream=None):
        _check(lib.hs_execute_host(self.handle, _ptr(h_x), _ptr(h_sums), _ptr(h_max), _ptr(h_argmax), _stream(stream)),
               "hs_execute_host")

    def hs_debug_greedy_paths(self, d_x, d_j, stream=None):
        _check(lib.hs_debug_greedy_paths(self.handle, _ptr(d_x), _ptr(d_j), _stream(stream)), "hs_debug_greedy_paths")

    def hs_execute_candidates(self, d_x, threshold, d_cand, capacity, d_count, stream=None):
        """d_cand: int32 CUDA tensor [capacity][4] (records spectrum, bin, value bits, level); d_count: int64 CUDA tensor [1]."""
        _check(lib.hs_execute_candidates(self.handle, _ptr(d_x), ctypes.c_float(threshold), _ptr(d_cand), int(capacity),
                                         _ptr(d_count), _stream(stream)), "hs_execute_candidates")

    def hs_destroy(self):
        if self.handle:
            lib.hs_destroy(self.handle)
            self.handle = ctypes.c_void_p(None)

    def __del__(self):
        try:
            self.hs_destroy()
        except Exception:
            pass

    # -- convenience: allocate outputs with torch and run ------------------------------------------------------
    def run(self, d_x, stream=None):
        """Allocate the outputs the plan's out_mode asks for, execute, return (sums, max, argmax) (None if absent)."""
        import torch
        assert d_x.is_cuda and d_x.dtype == torch.float32 and d_x.is_contiguous()
        row = (self.nbins,) if self.nz == 1 else (self.nz, self.nbins)     # one batch entry: a spectrum or a plane
        assert tuple(d_x.shape) == (self.batch,) + row
        sums = vmax = amax = None
        if self.out_mode & HS_OUT_FULL:
            sums = torch.empty((self.batch, self.levels) + row, dtype=torch.float32, device=d_x.device)
        if self.out_mode & HS_OUT_REDUCED:
            vmax = torch.empty((self.batch,) + row, dtype=torch.float32, device=d_x.device)
            amax = torch.empty((self.batch,) + row, dtype=torch.uint8, device=d_x.device)
        self.ensure_workspace(d_x.device)
        self.hs_execute(d_x, sums, vmax, amax, stream)
        return sums, vmax, amax

    def run_candidates(self, d_x, threshold, capacity=1 << 20, stream=None):
        """Allocate the candidate buffer, execute, return (count, records) with records = dict of torch tensors
        (spectrum, bin, level: int32; value: float32), the first min(count, capacity) appended records, any order."""
        import torch
        cand = torch.empty((max(1, capacity), 4), dtype=torch.int32, device=d_x.device)
        count = torch.zeros(1, dtype=torch.int64, device=d_x.device)
        self.ensure_workspace(d_x.device)
        self.hs_execute_candidates(d_x, threshold, cand, capacity, count, stream)
        torch.cuda.synchronize()
        n = int(count.item())
        rec = cand[:min(n, capacity)]
        return n, {"spectrum": rec[:, 0], "bin": rec[:, 1], "value": rec[:, 2].view(torch.float32), "level": rec[:, 3]}
