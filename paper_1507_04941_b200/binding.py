"""Thin ctypes binding of libpgsf.so (include/pgsf.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; torch is used for device memory and
streams.  There is no CPU fallback: if the library is missing or no sm_100 device is present the
calls raise.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpgsf.so")

PGSF_OK, PGSF_ERR_INVALID_ARG, PGSF_ERR_UNSUPPORTED, PGSF_ERR_OOM, PGSF_ERR_CUDA = range(5)
PGSF_FLAG_FORCE_GENERIC = 0x1
PGSF_FLAG_DRY_RUN = 0x4
PGSF_FLAG_TENSOR_ZPASS = 0x8
PGSF_OPT_GROUP_CUBES, PGSF_OPT_HOST_SECTION_PLANES, PGSF_OPT_HOST_DEVICE_BUDGET, PGSF_OPT_TUNE = 1, 2, 3, 4
PGSF_WEIGHTED_AS_PRINTED = 0
PGSF_WEIGHTED_NORMALISED = 1
PGSF_DIRECT_FP64_ACCUM = 0x1
PGSF_MAX_SCALES = 8
PGSF_MAX_RADIUS = 96
_STATUS = {0: "PGSF_OK", 1: "PGSF_ERR_INVALID_ARG", 2: "PGSF_ERR_UNSUPPORTED", 3: "PGSF_ERR_OOM",
           4: "PGSF_ERR_CUDA"}

EXPORTS = ["pgsf_plan_create", "pgsf_plan_destroy", "pgsf_plan_set_option", "pgsf_plan_path",
           "pgsf_plan_workspace_bytes", "pgsf_last_error",
           "pgsf_plan_get_taps", "pgsf_filter3d", "pgsf_filter3d_weighted", "pgsf_filter3d_direct", "pgsf_local_threshold", "pgsf_find_multiscale",
           "pgsf_find_multiscale_host", "pgsf_label_objects", "pgsf_filter3d_noalloc", "pgsf_plan_launch_count", "pgsf_plan_set_profiling",
           "pgsf_plan_profile_collect", "pgsf_plan_profile_entry"]


class PgsfError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__(f"{_STATUS.get(status, status)}: {text}")
        self.status = status


class _Desc(ctypes.Structure):
    _fields_ = [("nx", ctypes.c_int32), ("ny", ctypes.c_int32), ("nz", ctypes.c_int32),
                ("batch", ctypes.c_int32), ("halo", ctypes.c_int32 * 3), ("n_scales", ctypes.c_int32),
                ("sigmas", ctypes.POINTER(ctypes.c_double)), ("truncate", ctypes.c_double),
                ("box_half", ctypes.c_int32 * 3), ("k", ctypes.c_double), ("flags", ctypes.c_uint32)]


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen libpgsf.so (built in-tree by paper_1507_04941_b200.build); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(
                f"{LIB_PATH} not built; run `python -m paper_1507_04941_b200.build` "
                "(there is no CPU fallback)")
        lib = ctypes.CDLL(LIB_PATH)
        vp, i, u64p = ctypes.c_void_p, ctypes.c_int, ctypes.POINTER(ctypes.c_ulonglong)
        lib.pgsf_plan_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(_Desc), i]
        lib.pgsf_plan_create.restype = i
        lib.pgsf_plan_destroy.argtypes = [vp]
        lib.pgsf_plan_destroy.restype = i
        lib.pgsf_plan_set_option.argtypes = [vp, i, ctypes.c_longlong]
        lib.pgsf_plan_set_option.restype = i
        lib.pgsf_plan_path.argtypes = [vp, ctypes.c_char_p, i]
        lib.pgsf_plan_path.restype = i
        lib.pgsf_plan_workspace_bytes.argtypes = [vp]
        lib.pgsf_plan_workspace_bytes.restype = ctypes.c_size_t
        lib.pgsf_last_error.argtypes = [vp]
        lib.pgsf_last_error.restype = ctypes.c_char_p
        lib.pgsf_plan_get_taps.argtypes = [vp, i, i, ctypes.POINTER(ctypes.c_float), i, ctypes.POINTER(i)]
        lib.pgsf_plan_get_taps.restype = i
        lib.pgsf_filter3d.argtypes = [vp, i, vp, vp, vp, vp]
        lib.pgsf_filter3d.restype = i
        lib.pgsf_filter3d_weighted.argtypes = [vp, i, vp, vp, vp, i, vp, vp]
        lib.pgsf_filter3d_weighted.restype = i
        lib.pgsf_filter3d_direct.argtypes = [vp, vp, i, i, i, vp, vp, ctypes.c_uint, vp]
        lib.pgsf_filter3d_direct.restype = i
        lib.pgsf_label_objects.argtypes = [vp, vp, vp, vp, vp]
        lib.pgsf_label_objects.restype = i
        lib.pgsf_filter3d_noalloc.argtypes = [vp, vp, i, i, i, ctypes.POINTER(ctypes.c_double), ctypes.c_double, vp,
                                              ctypes.c_char_p, i]
        lib.pgsf_filter3d_noalloc.restype = i
        lib.pgsf_local_threshold.argtypes = [vp, vp, vp, i, vp, vp, vp, vp, vp]
        lib.pgsf_local_threshold.restype = i
        lib.pgsf_find_multiscale.argtypes = [vp, vp, ctypes.POINTER(vp), vp, vp, vp, vp]
        lib.pgsf_find_multiscale.restype = i
        lib.pgsf_find_multiscale_host.argtypes = [vp, vp, ctypes.POINTER(vp), vp, u64p]
        lib.pgsf_find_multiscale_host.restype = i
        lib.pgsf_plan_launch_count.argtypes = [vp]
        lib.pgsf_plan_launch_count.restype = ctypes.c_ulonglong
        lib.pgsf_plan_set_profiling.argtypes = [vp, i]
        lib.pgsf_plan_set_profiling.restype = i
        lib.pgsf_plan_profile_collect.argtypes = [vp, ctypes.POINTER(i)]
        lib.pgsf_plan_profile_collect.restype = i
        lib.pgsf_plan_profile_entry.argtypes = [vp, i, ctypes.c_char_p, i, u64p, ctypes.POINTER(ctypes.c_double)]
        lib.pgsf_plan_profile_entry.restype = i
        _lib = lib
    return _lib


def _ptr(t: Optional[torch.Tensor]):
    return ctypes.c_void_p(t.data_ptr()) if t is not None else None


def _stream_ptr(stream) -> ctypes.c_void_p:
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


class Plan:
    """pgsf_plan: cube geometry + filter bank + statistics window + threshold (include/pgsf.h)."""

    def __init__(self, dims_xyz: Sequence[int], sigmas: Sequence[Sequence[float]], box_half: Sequence[int],
                 k: float, batch: int = 1, halo: Sequence[int] = (0, 0, 0), truncate: float = 3.0,
                 flags: int = 0, device: int = 0):
        self._lib = load_library()
        self._h = ctypes.c_void_p()
        self.dims = tuple(int(v) for v in dims_xyz)
        self.batch = int(batch)
        self.n_scales = len(sigmas)
        self.sigmas = [tuple(float(v) for v in s) for s in sigmas]
        self.box_half = tuple(int(v) for v in box_half)
        self.halo = tuple(int(v) for v in halo)
        self.k = float(k)
        self.device = int(device)
        flat = (ctypes.c_double * (3 * max(1, self.n_scales)))(*[v for s in self.sigmas for v in s])
        d = _Desc(self.dims[0], self.dims[1], self.dims[2], self.batch,
                  (ctypes.c_int32 * 3)(*self.halo), self.n_scales, flat, float(truncate),
                  (ctypes.c_int32 * 3)(*self.box_half), self.k, int(flags))
        st = self._lib.pgsf_plan_create(ctypes.byref(self._h), ctypes.byref(d), self.device)
        if st != PGSF_OK:
            self._h = ctypes.c_void_p()
            raise PgsfError(st, self._lib.pgsf_last_error(None).decode())
        self._ws = None

    # ------------------------------------------------------------------ plumbing
    def _check(self, st: int):
        if st != PGSF_OK:
            raise PgsfError(st, self._lib.pgsf_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            self._lib.pgsf_plan_destroy(self._h)
            self._h = ctypes.c_void_p()
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    @property
    def voxels(self) -> int:
        return self.dims[0] * self.dims[1] * self.dims[2] * self.batch

    def pgsf_plan_workspace_bytes(self) -> int:
        return int(self._lib.pgsf_plan_workspace_bytes(self._h))

    def pgsf_plan_set_option(self, option: int, value: int) -> None:
        self._check(self._lib.pgsf_plan_set_option(self._h, int(option), int(value)))

    def pgsf_plan_path(self):
        """(all_tiled: bool, text) -- which kernels the plan runs and why."""
        buf = ctypes.create_string_buffer(512)
        rc = self._lib.pgsf_plan_path(self._h, buf, 512)
        if rc < 0:
            raise PgsfError(PGSF_ERR_INVALID_ARG, "pgsf_plan_path")
        return bool(rc), buf.value.decode()

    def pgsf_plan_launch_count(self) -> int:
        return int(self._lib.pgsf_plan_launch_count(self._h))

    def pgsf_plan_set_profiling(self, enable: bool) -> None:
        self._check(self._lib.pgsf_plan_set_profiling(self._h, int(bool(enable))))

    def pgsf_plan_profile(self) -> dict:
        """{kernel name: (launches, total ms)} of the launches since profiling was switched on
        (synchronises with them)."""
        n = ctypes.c_int(0)
        self._check(self._lib.pgsf_plan_profile_collect(self._h, ctypes.byref(n)))
        out = {}
        for idx in range(n.value):
            name = ctypes.create_string_buffer(64)
            cnt, ms = ctypes.c_ulonglong(0), ctypes.c_double(0.0)
            self._check(self._lib.pgsf_plan_profile_entry(self._h, idx, name, 64, ctypes.byref(cnt), ctypes.byref(ms)))
            out[name.value.decode()] = (int(cnt.value), float(ms.value))
        return out

    def workspace(self) -> Optional[torch.Tensor]:
        """A torch-owned device buffer of pgsf_plan_workspace_bytes() (allocated once)."""
        n = self.pgsf_plan_workspace_bytes()
        if n == 0:
            return None
        if self._ws is None or self._ws.numel() < n:
            self._ws = torch.empty(n, dtype=torch.uint8, device=f"cuda:{self.device}")
        return self._ws

    def pgsf_plan_get_taps(self, scale: int, axis: int):
        buf = (ctypes.c_float * (2 * PGSF_MAX_RADIUS + 1))()
        r = ctypes.c_int()
        self._check(self._lib.pgsf_plan_get_taps(self._h, scale, axis, buf, len(buf), ctypes.byref(r)))
        return [buf[i] for i in range(2 * r.value + 1)]

    def _shape(self):
        return (self.batch, self.dims[2], self.dims[1], self.dims[0])

    def _check_cube(self, t: torch.Tensor, dtype, name: str):
        if not t.is_cuda or t.dtype != dtype or not t.is_contiguous() or t.numel() != self.voxels:
            raise ValueError(f"{name}: need a contiguous cuda {dtype} tensor of {self.voxels} elements "
                             f"([batch,] nz, ny, nx)")

    # ------------------------------------------------------------------ the C-ABI calls
    def pgsf_filter3d(self, scale: int, d_in: torch.Tensor, d_out: Optional[torch.Tensor] = None,
                      stream=None) -> torch.Tensor:
        self._check_cube(d_in, torch.float32, "d_in")
        if d_out is None:
            d_out = torch.empty_like(d_in)
        self._check_cube(d_out, torch.float32, "d_out")
        ws = self.workspace()
        self._check(self._lib.pgsf_filter3d(self._h, int(scale), _ptr(d_in), _ptr(d_out), _ptr(ws),
                                            _stream_ptr(stream)))
        return d_out

    def pgsf_filter3d_weighted(self, scale: int, d_in: torch.Tensor, d_w: torch.Tensor, mode: int = 0,
                               d_out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
        """Eq. 1 of the paper (weighted convolution); mode: PGSF_WEIGHTED_AS_PRINTED / _NORMALISED."""
        self._check_cube(d_in, torch.float32, "d_in")
        self._check_cube(d_w, torch.float32, "d_w")
        if d_out is None:
            d_out = torch.empty_like(d_in)
        self._check_cube(d_out, torch.float32, "d_out")
        ws = self.workspace()
        self._check(self._lib.pgsf_filter3d_weighted(self._h, int(scale), _ptr(d_in), _ptr(d_w), _ptr(d_out),
                                                     int(mode), _ptr(ws), _stream_ptr(stream)))
        return d_out

    def pgsf_filter3d_direct(self, d_filter: torch.Tensor, d_in: torch.Tensor, fp64_accum: bool = False,
                             d_out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
        """Eq. 2 for an arbitrary filter array d_filter[fz, fy, fx] (odd extents, fp32, on the device)."""
        self._check_cube(d_in, torch.float32, "d_in")
        if d_filter.dtype != torch.float32 or d_filter.dim() != 3 or not d_filter.is_contiguous() or \
                any(n % 2 == 0 for n in d_filter.shape) or d_filter.device != d_in.device:
            raise ValueError("d_filter: contiguous fp32 [fz, fy, fx] with odd extents on the cube's device")
        if d_out is None:
            d_out = torch.empty_like(d_in)
        self._check_cube(d_out, torch.float32, "d_out")
        rz, ry, rx = [(n - 1) // 2 for n in d_filter.shape]
        self._check(self._lib.pgsf_filter3d_direct(self._h, _ptr(d_filter), rx, ry, rz, _ptr(d_in), _ptr(d_out),
                                                   PGSF_DIRECT_FP64_ACCUM if fp64_accum else 0, _stream_ptr(stream)))
        return d_out

    def pgsf_label_objects(self, d_mask: torch.Tensor, d_labels: Optional[torch.Tensor] = None, stream=None):
        """NEXT-4: connected components (26-connectivity) of the mask.  Returns (labels int32 tensor holding the uint32
        labels, count tensor); label = 1 + smallest linear index of the component inside its cube, 0 = background."""
        self._check_cube(d_mask, torch.uint8, "d_mask")
        if d_labels is None:
            d_labels = torch.empty(d_mask.shape, dtype=torch.int32, device=d_mask.device)
        self._check_cube(d_labels, torch.int32, "d_labels")
        cnt = torch.zeros(1, dtype=torch.int64, device=d_mask.device)
        self._check(self._lib.pgsf_label_objects(self._h, _ptr(d_mask), _ptr(d_labels), _ptr(cnt), _stream_ptr(stream)))
        return d_labels, cnt

    def pgsf_local_threshold(self, d_filtered: torch.Tensor, d_mask: Optional[torch.Tensor] = None,
                             or_into: bool = False, want_stats: bool = False, want_count: bool = True,
                             stream=None):
        """Returns (mask, count_tensor_or_None, mean_or_None, std_or_None); count is a 1-element
        int64 device tensor, valid after the stream is synchronised."""
        self._check_cube(d_filtered, torch.float32, "d_filtered")
        if d_mask is None:
            d_mask = torch.zeros(d_filtered.shape, dtype=torch.uint8, device=d_filtered.device)
        self._check_cube(d_mask, torch.uint8, "d_mask")
        mean = torch.empty_like(d_filtered) if want_stats else None
        std = torch.empty_like(d_filtered) if want_stats else None
        cnt = torch.zeros(1, dtype=torch.int64, device=d_filtered.device) if want_count else None
        ws = self.workspace()
        self._check(self._lib.pgsf_local_threshold(self._h, _ptr(d_filtered), _ptr(d_mask), int(bool(or_into)),
                                                   _ptr(mean), _ptr(std), _ptr(cnt), _ptr(ws),
                                                   _stream_ptr(stream)))
        return d_mask, cnt, mean, std

    def pgsf_find_multiscale(self, d_in: torch.Tensor, keep_filtered: bool = False,
                             d_filtered: Optional[Sequence[Optional[torch.Tensor]]] = None,
                             d_mask: Optional[torch.Tensor] = None,
                             d_count: Optional[torch.Tensor] = None, stream=None):
        """Returns (mask, count_tensor, filtered_list_or_None)."""
        self._check_cube(d_in, torch.float32, "d_in")
        if d_mask is None:
            d_mask = torch.empty(d_in.shape, dtype=torch.uint8, device=d_in.device)
        self._check_cube(d_mask, torch.uint8, "d_mask")
        if d_count is None:
            d_count = torch.zeros(1, dtype=torch.int64, device=d_in.device)
        if keep_filtered and d_filtered is None:
            d_filtered = [torch.empty_like(d_in) for _ in range(self.n_scales)]
        arr = None
        if d_filtered is not None:
            arr = (ctypes.c_void_p * self.n_scales)()
            for s, t in enumerate(d_filtered):
                if t is not None:
                    self._check_cube(t, torch.float32, f"d_filtered[{s}]")
                    arr[s] = t.data_ptr()
        ws = self.workspace()
        self._check(self._lib.pgsf_find_multiscale(self._h, _ptr(d_in), arr, _ptr(d_mask), _ptr(d_count),
                                                   _ptr(ws), _stream_ptr(stream)))
        return d_mask, d_count, d_filtered

    def pgsf_find_multiscale_host(self, h_in: torch.Tensor, h_mask: Optional[torch.Tensor] = None,
                                  h_filtered: Optional[Sequence[Optional[torch.Tensor]]] = None):
        """Host-buffer entry point: CPU tensors in, CPU tensors out (synchronises).  Returns
        (mask, count:int)."""
        if h_in.is_cuda or h_in.dtype != torch.float32 or not h_in.is_contiguous() or h_in.numel() != self.voxels:
            raise ValueError("h_in: need a contiguous CPU float32 tensor of the plan's size")
        if h_mask is None:
            h_mask = torch.empty(h_in.shape, dtype=torch.uint8)
        arr = None
        if h_filtered is not None:
            arr = (ctypes.c_void_p * self.n_scales)()
            for s, t in enumerate(h_filtered):
                if t is not None:
                    arr[s] = t.data_ptr()
        cnt = ctypes.c_ulonglong(0)
        self._check(self._lib.pgsf_find_multiscale_host(self._h, _ptr(h_in), arr, _ptr(h_mask),
                                                        ctypes.byref(cnt)))
        return h_mask, int(cnt.value)


PGSF_NOALLOC_MAX_VOXELS = 1 << 21


def pgsf_filter3d_noalloc(d_in: torch.Tensor, sigma_xyz: Sequence[float], truncate: float = 3.0,
                          d_out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """pgsf_filter3d for one cube [nz, ny, nx] without a plan or workspace: the library's static device scratch holds
    the intermediates (at most PGSF_NOALLOC_MAX_VOXELS voxels; calls on one device must not overlap on the GPU).
    The library call itself allocates nothing; pass d_out to keep this wrapper from allocating the output."""
    lib = load_library()
    if not d_in.is_cuda or d_in.dtype != torch.float32 or d_in.dim() != 3 or not d_in.is_contiguous():
        raise ValueError("d_in: need a contiguous cuda float32 tensor [nz, ny, nx]")
    if d_out is None:
        d_out = torch.empty_like(d_in)
    if d_out.shape != d_in.shape or d_out.dtype != torch.float32 or not d_out.is_contiguous() or d_out.device != d_in.device:
        raise ValueError("d_out: need a contiguous cuda float32 tensor of d_in's shape on its device")
    nz, ny, nx = d_in.shape
    sig = (ctypes.c_double * 3)(*[float(s) for s in sigma_xyz])
    err = ctypes.create_string_buffer(384)
    with torch.cuda.device(d_in.device):
        st = lib.pgsf_filter3d_noalloc(_ptr(d_in), _ptr(d_out), nx, ny, nz, sig, float(truncate), _stream_ptr(stream),
                                       err, len(err))
    if st != PGSF_OK:
        raise PgsfError(st, err.value.decode())
    return d_out
