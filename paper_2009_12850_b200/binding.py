"""Thin ctypes binding of include/monc_adv.h -- argument marshalling only.

Every step of the hot path runs inside libmonc_adv.so (hand-written sm_100a
kernels).  PyTorch tensors are used here only as owners of device / pinned
host memory and for stream handles.  There is no fallback: if the library is
missing or a call fails, a `MoncAdvError` is raised.

Names mirror the C ABI: create -> MoncAdv(...), monc_adv_momentum -> .momentum,
monc_adv_scalars -> .scalars, monc_adv_step_async -> .step_async, ...
"""
from __future__ import annotations

import ctypes as C
import os

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libmonc_adv.so")
LIB_PATH_CHECKED = os.path.join(HERE, "libmonc_adv_checked.so")  # -DMONC_ADV_CHECKED=1 (tests/test_gpu_checked.py)

F64, F32 = 0, 1
FORM_FLUX, FORM_PW_SKEW = 0, 1
OK, EINVAL, ECUDA, ENOMEM, ENOWIND, EBUSY = 0, -1, -2, -3, -4, -5
MAX_SCALARS = 64
NOALLOC_MAX_BYTES = 16 << 20  # MONC_ADV_NOALLOC_MAX_BYTES

# every symbol include/monc_adv.h declares (tests check the .so exports them all)
SYMBOLS = [
    "monc_adv_create", "monc_adv_destroy", "monc_adv_momentum", "monc_adv_bind_wind",
    "monc_adv_scalars", "monc_adv_tendencies", "monc_adv_set_fuse", "monc_adv_step_async", "monc_adv_step_inputs_consumed",
    "monc_adv_step_wait_chunk", "monc_adv_step_wait", "monc_adv_step_chunk_range", "monc_adv_step_chunk_count", "monc_adv_step_noalloc", "monc_adv_plan_chunks", "monc_adv_plan_describe",
    "monc_adv_step_times_ms", "monc_adv_set_chunks", "monc_adv_set_overlap",
    "monc_adv_set_form", "monc_adv_set_accumulate", "monc_adv_set_pdl", "monc_adv_set_variant",
    "monc_adv_set_tuning", "monc_adv_get_coefficients", "monc_adv_launch_count",
    "monc_adv_describe_plan", "monc_adv_last_error", "monc_adv_version", "monc_adv_set_work_scale",
    "monc_adv_set_cluster", "monc_adv_set_l2_hint", "monc_adv_set_graph", "monc_adv_graph_state",
]


def plan_chunks(nx, ny, nz, halo, dtype, nfields_in, nfields_out) -> int:
    """The chunk count an automatic hybrid step would take (no handle, no GPU)."""
    dt = {"f64": F64, "f32": F32}.get(dtype, dtype)
    n = load().monc_adv_plan_chunks(int(nx), int(ny), int(nz), int(halo), int(dt), int(nfields_in), int(nfields_out))
    if n < 1:
        raise MoncAdvError(n, "plan_chunks: bad argument")
    return n


def plan_describe(nx, ny, nz, halo, dtype, nq, fused=True, sm_count=148, smem_optin=232448) -> str:
    """The launch geometry the library's planners choose for this shape (no handle, no GPU)."""
    dt = {"f64": F64, "f32": F32}.get(dtype, dtype)
    buf = C.create_string_buffer(640)
    rc = load().monc_adv_plan_describe(int(nx), int(ny), int(nz), int(halo), int(dt), int(nq), int(bool(fused)),
                                       int(sm_count), int(smem_optin), buf, len(buf))
    if rc != OK:
        raise MoncAdvError(rc, "plan_describe: bad argument")
    return buf.value.decode()


class MoncAdvError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"monc_adv error {code}: {msg}")
        self.code = code


_lib = None
_libs = {}
_path = LIB_PATH


def select_build(checked: bool) -> None:
    """Handles created from now on come from the checked build (poisoned ring slots,
    jittered schedule; same ABI, same results) or from the normal one."""
    global _lib, _path
    _path = LIB_PATH_CHECKED if checked else LIB_PATH
    _lib = None


def load():
    """Open libmonc_adv.so (built by paper_2009_12850_b200.build). Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    if _path in _libs:
        _lib = _libs[_path]
        return _lib
    if not os.path.exists(_path):
        raise MoncAdvError(ECUDA, f"{_path} not built: run `python -m paper_2009_12850_b200.build`"
                           " (there is no CPU fallback)")
    lib = C.CDLL(_path)
    vp, dp, ci = C.c_void_p, C.POINTER(C.c_double), C.c_int
    lib.monc_adv_create.argtypes = [C.POINTER(vp), ci, ci, ci, ci, C.c_double, C.c_double] + [dp] * 8 + [ci]
    lib.monc_adv_create.restype = ci
    lib.monc_adv_destroy.argtypes = [vp]
    lib.monc_adv_destroy.restype = None
    lib.monc_adv_momentum.argtypes = [vp] * 8
    lib.monc_adv_momentum.restype = ci
    lib.monc_adv_bind_wind.argtypes = [vp] * 4
    lib.monc_adv_bind_wind.restype = ci
    lib.monc_adv_scalars.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), ci, vp]
    lib.monc_adv_scalars.restype = ci
    lib.monc_adv_tendencies.argtypes = [vp] * 7 + [C.POINTER(vp), C.POINTER(vp), ci, vp]
    lib.monc_adv_tendencies.restype = ci
    lib.monc_adv_step_async.argtypes = [vp, vp, vp, vp, C.POINTER(vp), ci, vp, vp, vp, C.POINTER(vp), vp]
    lib.monc_adv_step_async.restype = ci
    lib.monc_adv_step_noalloc.argtypes = [vp] * 8
    lib.monc_adv_step_noalloc.restype = ci
    for name in ("monc_adv_step_inputs_consumed", "monc_adv_step_wait"):
        getattr(lib, name).argtypes = [vp]
        getattr(lib, name).restype = ci
    lib.monc_adv_step_wait_chunk.argtypes = [vp, ci]
    lib.monc_adv_step_wait_chunk.restype = ci
    lib.monc_adv_step_chunk_range.argtypes = [vp, ci, C.POINTER(ci), C.POINTER(ci)]
    lib.monc_adv_step_chunk_range.restype = ci
    lib.monc_adv_graph_state.argtypes = [vp]
    lib.monc_adv_graph_state.restype = ci
    lib.monc_adv_plan_describe.argtypes = [ci] * 9 + [C.c_char_p, ci]
    lib.monc_adv_plan_describe.restype = ci
    lib.monc_adv_plan_chunks.argtypes = [ci] * 7
    lib.monc_adv_plan_chunks.restype = ci
    lib.monc_adv_step_chunk_count.argtypes = [vp]
    lib.monc_adv_step_chunk_count.restype = ci
    lib.monc_adv_step_times_ms.argtypes = [vp, C.POINTER(C.c_float)]
    lib.monc_adv_step_times_ms.restype = ci
    for name in ("monc_adv_set_chunks", "monc_adv_set_overlap", "monc_adv_set_form",
                 "monc_adv_set_accumulate", "monc_adv_set_pdl", "monc_adv_set_variant",
                 "monc_adv_set_fuse", "monc_adv_set_work_scale", "monc_adv_set_cluster", "monc_adv_set_l2_hint",
                 "monc_adv_set_graph"):
        getattr(lib, name).argtypes = [vp, ci]
        getattr(lib, name).restype = ci
    lib.monc_adv_set_tuning.argtypes = [vp, ci, ci, ci, ci, ci, ci, ci]
    lib.monc_adv_set_tuning.restype = ci
    lib.monc_adv_get_coefficients.argtypes = [vp] + [dp] * 4
    lib.monc_adv_get_coefficients.restype = ci
    lib.monc_adv_launch_count.argtypes = [vp]
    lib.monc_adv_launch_count.restype = C.c_long
    lib.monc_adv_describe_plan.argtypes = [vp]
    lib.monc_adv_describe_plan.restype = C.c_char_p
    lib.monc_adv_last_error.argtypes = [vp]
    lib.monc_adv_last_error.restype = C.c_char_p
    lib.monc_adv_version.argtypes = []
    lib.monc_adv_version.restype = C.c_char_p
    _libs[_path] = lib
    _lib = lib
    return lib


def version() -> str:
    return load().monc_adv_version().decode()


def _dptr(a):
    """double* of a float64 numpy array / sequence, or NULL."""
    if a is None:
        return None, None
    import numpy as np
    arr = np.ascontiguousarray(a, dtype=np.float64)
    return arr, arr.ctypes.data_as(C.POINTER(C.c_double))


def _stream_ptr(stream):
    if stream is None:
        return None
    if isinstance(stream, torch.cuda.Stream):
        return C.c_void_p(stream.cuda_stream)
    return C.c_void_p(int(stream))


class MoncAdv:
    """One advection problem on the current CUDA device (monc_adv_create)."""

    def __init__(self, nx, ny, nz, halo, dx, dy, dz=None, dzn=None, rho=None, rhon=None,
                 tzc1=None, tzc2=None, tzd1=None, tzd2=None, dtype="f64"):
        self._lib = load()
        self._h = C.c_void_p()
        self.nx, self.ny, self.nz, self.halo = int(nx), int(ny), int(nz), int(halo)
        self.dtype = {"f64": F64, "f32": F32}[dtype] if isinstance(dtype, str) else int(dtype)
        self.torch_dtype = torch.float64 if self.dtype == F64 else torch.float32
        self.shape = (self.nx + 2 * self.halo, self.ny + 2 * self.halo, self.nz)
        keep = [_dptr(a) for a in (dz, dzn, rho, rhon, tzc1, tzc2, tzd1, tzd2)]
        rc = self._lib.monc_adv_create(C.byref(self._h), self.nx, self.ny, self.nz, self.halo,
                                       float(dx), float(dy), *[k[1] for k in keep], self.dtype)
        if rc != OK:
            msg = self._lib.monc_adv_last_error(None).decode()
            self._h = C.c_void_p()
            raise MoncAdvError(rc, msg)
        self._wind_keepalive = None

    # -- plumbing ----------------------------------------------------------
    def _check(self, rc):
        if rc != OK:
            raise MoncAdvError(rc, self._lib.monc_adv_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            self._lib.monc_adv_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _dev(self, t, name):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == self.torch_dtype
                and t.is_contiguous() and tuple(t.shape) == self.shape):
            raise MoncAdvError(EINVAL, f"{name}: need a contiguous CUDA tensor of shape {self.shape}"
                               f" and dtype {self.torch_dtype}")
        return C.c_void_p(t.data_ptr())

    def _host(self, t, name):
        if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == self.torch_dtype
                and t.is_contiguous() and tuple(t.shape) == self.shape and t.is_pinned()):
            raise MoncAdvError(EINVAL, f"{name}: need a contiguous PINNED host tensor of shape"
                               f" {self.shape} and dtype {self.torch_dtype}")
        return C.c_void_p(t.data_ptr())

    @staticmethod
    def _table(ptrs):
        arr = (C.c_void_p * max(len(ptrs), 1))(*ptrs)
        return arr

    # -- compute calls -----------------------------------------------------
    def momentum(self, u, v, w, su, sv, sw, stream=None):
        args = [self._dev(t, n) for t, n in zip((u, v, w, su, sv, sw), ("u", "v", "w", "su", "sv", "sw"))]
        self._wind_keepalive = (u, v, w)
        self._check(self._lib.monc_adv_momentum(self._h, *args, _stream_ptr(stream)))

    def bind_wind(self, u, v, w):
        args = [self._dev(t, n) for t, n in zip((u, v, w), "uvw")]
        self._wind_keepalive = (u, v, w)
        self._check(self._lib.monc_adv_bind_wind(self._h, *args))

    def scalars(self, q, sq, stream=None):
        if len(q) != len(sq):
            raise MoncAdvError(EINVAL, "scalars: len(q) != len(sq)")
        qp = self._table([self._dev(t, f"q[{n}]") for n, t in enumerate(q)])
        sp = self._table([self._dev(t, f"sq[{n}]") for n, t in enumerate(sq)])
        self._check(self._lib.monc_adv_scalars(self._h, qp, sp, len(q), _stream_ptr(stream)))

    def tendencies(self, u, v, w, su, sv, sw, q, sq, stream=None):
        if len(q) != len(sq):
            raise MoncAdvError(EINVAL, "tendencies: len(q) != len(sq)")
        args = [self._dev(t, n) for t, n in zip((u, v, w, su, sv, sw), ("u", "v", "w", "su", "sv", "sw"))]
        qp = self._table([self._dev(t, f"q[{n}]") for n, t in enumerate(q)])
        sp = self._table([self._dev(t, f"sq[{n}]") for n, t in enumerate(sq)])
        self._wind_keepalive = (u, v, w)
        self._check(self._lib.monc_adv_tendencies(self._h, *args, qp, sp, len(q), _stream_ptr(stream)))

    def step_async(self, hu, hv, hw, hq, hsu, hsv, hsw, hsq, stream=None):
        hq, hsq = list(hq or []), list(hsq or [])
        if len(hq) != len(hsq):
            raise MoncAdvError(EINVAL, "step_async: len(hq) != len(hsq)")
        ins = [self._host(t, n) for t, n in zip((hu, hv, hw), ("hu", "hv", "hw"))]
        if hsu is None and hsv is None and hsw is None:
            outs = [None, None, None]
        else:
            outs = [self._host(t, n) for t, n in zip((hsu, hsv, hsw), ("hsu", "hsv", "hsw"))]
        qp = self._table([self._host(t, f"hq[{n}]") for n, t in enumerate(hq)])
        sp = self._table([self._host(t, f"hsq[{n}]") for n, t in enumerate(hsq)])
        self._step_keepalive = (hu, hv, hw, hq, hsu, hsv, hsw, hsq)
        self._check(self._lib.monc_adv_step_async(self._h, *ins, qp, len(hq), *outs, sp,
                                                  _stream_ptr(stream)))

    def step_noalloc(self, hu, hv, hw, hsu, hsv, hsw, stream=None):
        """Momentum step from pinned host tensors; device staging in the library's static scratch
        (no device allocation of any kind; limits and sharing rules: include/monc_adv.h)."""
        ins = [self._host(t, n) for t, n in zip((hu, hv, hw), ("hu", "hv", "hw"))]
        outs = [self._host(t, n) for t, n in zip((hsu, hsv, hsw), ("hsu", "hsv", "hsw"))]
        self._noalloc_keepalive = (hu, hv, hw, hsu, hsv, hsw)
        self._check(self._lib.monc_adv_step_noalloc(self._h, *ins, *outs, _stream_ptr(stream)))

    def step_inputs_consumed(self):
        self._check(self._lib.monc_adv_step_inputs_consumed(self._h))

    def step_wait_chunk(self, c):
        self._check(self._lib.monc_adv_step_wait_chunk(self._h, int(c)))

    def step_wait(self):
        self._check(self._lib.monc_adv_step_wait(self._h))

    def step_chunk_range(self, c):
        a, b = C.c_int(), C.c_int()
        self._check(self._lib.monc_adv_step_chunk_range(self._h, int(c), C.byref(a), C.byref(b)))
        return a.value, b.value

    def step_times_ms(self):
        out = (C.c_float * 4)()
        self._check(self._lib.monc_adv_step_times_ms(self._h, out))
        return dict(h2d=out[0], kernels=out[1], d2h=out[2], total=out[3])

    # -- settings ----------------------------------------------------------
    def step_chunk_count(self) -> int:
        return int(self._lib.monc_adv_step_chunk_count(self._h))

    def set_chunks(self, n):
        self._check(self._lib.monc_adv_set_chunks(self._h, int(n)))

    def set_overlap(self, on):
        self._check(self._lib.monc_adv_set_overlap(self._h, int(bool(on))))

    def set_form(self, form):
        form = {"flux": FORM_FLUX, "pw_skew": FORM_PW_SKEW}.get(form, form)
        self._check(self._lib.monc_adv_set_form(self._h, int(form)))

    def set_accumulate(self, on):
        self._check(self._lib.monc_adv_set_accumulate(self._h, int(bool(on))))

    def set_pdl(self, on):
        self._check(self._lib.monc_adv_set_pdl(self._h, int(bool(on))))

    def graph_state(self) -> int:
        return int(self._lib.monc_adv_graph_state(self._h))

    def set_graph(self, on):
        self._check(self._lib.monc_adv_set_graph(self._h, int(bool(on))))

    def set_l2_hint(self, hint):
        self._check(self._lib.monc_adv_set_l2_hint(self._h, int(hint)))

    def set_cluster(self, n):
        self._check(self._lib.monc_adv_set_cluster(self._h, int(n)))

    def set_work_scale(self, n):
        self._check(self._lib.monc_adv_set_work_scale(self._h, int(n)))

    def set_fuse(self, on):
        self._check(self._lib.monc_adv_set_fuse(self._h, int(bool(on))))

    def set_variant(self, variant):
        variant = {"auto": 0, "generic": 1, "march": 2, "tma": 3}.get(variant, variant)
        self._check(self._lib.monc_adv_set_variant(self._h, int(variant)))

    def set_tuning(self, xchunk=0, group=0, prefetch=0, warps=0, stages=0, tile_y=0, split=0):
        self._check(self._lib.monc_adv_set_tuning(self._h, int(xchunk), int(group), int(prefetch),
                                                  int(warps), int(stages), int(tile_y), int(split)))

    def get_coefficients(self):
        import numpy as np
        outs = [np.zeros(self.nz) for _ in range(4)]
        self._check(self._lib.monc_adv_get_coefficients(
            self._h, *[o.ctypes.data_as(C.POINTER(C.c_double)) for o in outs]))
        return tuple(outs)

    def describe_plan(self) -> str:
        return self._lib.monc_adv_describe_plan(self._h).decode()

    def launch_count(self) -> int:
        return int(self._lib.monc_adv_launch_count(self._h))
