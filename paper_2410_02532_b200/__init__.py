"""Python binding of libopo (include/opo.h): argument marshalling only.

Every step of the hot path -- FFTs, dispersion multiply, RK4, cavity boundary -- runs in the
hand-written sm_100a kernels behind the C ABI.  PyTorch supplies device memory and streams, nothing
else.  There is no CPU fallback: if libopo.so is missing or no B200 is present, calls raise.

The functions carry the names of the C entry points (opo_create, opo_set_pump, opo_propagate,
opo_roundtrips, opo_get_fields, ...); `Opo` is a small object wrapper over the same calls.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libopo.so")

OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_ALLOC, ERR_CUDA, ERR_STATE, ERR_NONFINITE = range(7)
PRECISION_C64, PRECISION_C128 = 0, 1
PARAM_DK, PARAM_DELTA_T, PARAM_DELTA_RAD, PARAM_GDD = 0, 1, 2, 3
WHICH_CURRENT, WHICH_EXIT = 0, 1
DOMAIN_TIME, DOMAIN_FREQ = 0, 1
ENGINE_AUTO, ENGINE_RESIDENT, ENGINE_STREAMING, ENGINE_LARGE, ENGINE_CUFFT, ENGINE_SOLO, ENGINE_WIDE = 0, 1, 2, 3, 4, 5, 6
OPT_ENGINE = 0
OPT_WIDE_SUBBLOCKS = 2
OPT_SPLITTING = 1
SPLITTING_LNL, SPLITTING_NLN = 0, 1
INFO_ENGINE, INFO_LAUNCHES, INFO_N, INFO_BATCH, INFO_SM_COUNT, INFO_SLOTS, INFO_WIDE_SUBBLOCKS = 0, 1, 2, 3, 4, 5, 6

_D3 = ctypes.c_double * 3
_I3 = ctypes.c_int * 3


class opo_crystal(ctypes.Structure):
    _fields_ = [("length_m", ctypes.c_double), ("dk_per_m", ctypes.c_double), ("d_eff_m_per_V", ctypes.c_double)]


class opo_fields(ctypes.Structure):
    _fields_ = [("n_fields", ctypes.c_int), ("lambda_m", _D3), ("n", _D3), ("beta1_s_per_m", _D3),
                ("beta2_s2_per_m", _D3), ("alpha_per_m", _D3), ("ref_field", ctypes.c_int),
                ("resonant", _I3), ("R", _D3), ("delta_rad", _D3), ("delta_T_s", _D3), ("gdd_s2", _D3)]


class opo_grid(ctypes.Structure):
    _fields_ = [("log2_n", ctypes.c_int), ("window_s", ctypes.c_double), ("nz_per_pass", ctypes.c_int),
                ("precision", ctypes.c_int), ("batch", ctypes.c_int)]


class opo_segment(ctypes.Structure):
    _fields_ = [("length_m", ctypes.c_double), ("dk_per_m", ctypes.c_double), ("d_eff_m_per_V", ctypes.c_double), ("nz", ctypes.c_int)]


class OpoError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"libopo status {status}: {message}")
        self.status = status


_lib = None


def lib() -> ctypes.CDLL:
    """Load libopo.so (built in-tree by paper_2410_02532_b200.build).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2410_02532_b200.build` "
                              "(there is no fallback path)")
        L = ctypes.CDLL(LIB_PATH)
        vp, ci = ctypes.c_void_p, ctypes.c_int
        L.opo_create.argtypes = [ctypes.POINTER(opo_crystal), ctypes.POINTER(opo_fields),
                                 ctypes.POINTER(opo_grid), ctypes.POINTER(vp)]
        L.opo_destroy.argtypes = [vp]
        L.opo_set_stream.argtypes = [vp, vp]
        L.opo_set_batch_param.argtypes = [vp, ci, ci, ctypes.POINTER(ctypes.c_double), ci]
        L.opo_set_eom.argtypes = [vp, ci, ctypes.c_double, ctypes.c_double]
        L.opo_set_beta3.argtypes = [vp, ci, ctypes.c_double]
        L.opo_set_pump.argtypes = [vp, vp, ci]
        L.opo_set_pump_host.argtypes = [vp, vp, ci]
        L.opo_set_field.argtypes = [vp, ci, vp]
        L.opo_set_field_host.argtypes = [vp, ci, vp]
        L.opo_propagate.argtypes = [vp, ci]
        L.opo_roundtrips.argtypes = [vp, ci]
        L.opo_roundtrips_train.argtypes = [vp, ci, vp, ci, vp, ci]
        L.opo_get_fields.argtypes = [vp, ci, ci, ci, vp]
        L.opo_get_fields_host.argtypes = [vp, ci, ci, ci, vp]
        L.opo_sync.argtypes = [vp]
        L.opo_check_finite.argtypes = [vp]
        L.opo_get_z_steps.argtypes = [vp, ctypes.POINTER(ci)]
        L.opo_set_option.argtypes = [vp, ci, ci]
        L.opo_get_info.argtypes = [vp, ci, ctypes.POINTER(ctypes.c_longlong)]
        L.opo_set_segments.argtypes = [vp, ci, ctypes.POINTER(opo_segment)]
        L.opo_selftest_peak.argtypes = [ci, ctypes.POINTER(ctypes.c_double)]
        L.opo_spectrum_noalloc.argtypes = [vp, vp, ci, ci, ci, vp]
        L.opo_last_error.argtypes = [vp]
        L.opo_last_error.restype = ctypes.c_char_p
        for name in EXPORTS:
            if name != "opo_last_error":
                getattr(L, name).restype = ci
        _lib = L
    return _lib


EXPORTS = ["opo_create", "opo_destroy", "opo_set_stream", "opo_set_batch_param", "opo_set_eom", "opo_set_beta3", "opo_set_pump",
           "opo_set_pump_host", "opo_set_field", "opo_set_field_host", "opo_propagate", "opo_roundtrips", "opo_roundtrips_train",
           "opo_get_fields", "opo_get_fields_host", "opo_sync", "opo_check_finite", "opo_get_z_steps",
           "opo_set_option", "opo_get_info", "opo_selftest_peak", "opo_set_segments", "opo_spectrum_noalloc", "opo_last_error"]


def _check(handle, status: int):
    if status != OK:
        msg = lib().opo_last_error(handle)
        raise OpoError(status, msg.decode() if msg else "")


def _d3(v: Optional[Sequence[float]]):
    a = _D3()
    for i, x in enumerate(v or ()):
        a[i] = float(x)
    return a


def _i3(v: Optional[Sequence[int]]):
    a = _I3()
    for i, x in enumerate(v or ()):
        a[i] = int(x)
    return a


# ---- the C calls, one to one ---------------------------------------------------------------------------

def opo_create(crystal: opo_crystal, fields: opo_fields, grid: opo_grid) -> ctypes.c_void_p:
    h = ctypes.c_void_p()
    st = lib().opo_create(ctypes.byref(crystal), ctypes.byref(fields), ctypes.byref(grid), ctypes.byref(h))
    _check(None, st)
    return h


def opo_destroy(h):
    _check(None, lib().opo_destroy(h))


def opo_set_stream(h, cuda_stream: int):
    _check(h, lib().opo_set_stream(h, ctypes.c_void_p(cuda_stream)))


def opo_set_batch_param(h, param: int, field: int, values):
    v = np.ascontiguousarray(values, dtype=np.float64)
    _check(h, lib().opo_set_batch_param(h, param, field, v.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), v.size))


def opo_set_segments(h, segments):
    """segments: sequence of (length_m, dk_per_m, d_eff_m_per_V, nz); empty restores the crystal of opo_create."""
    n = len(segments)
    arr = (opo_segment * max(n, 1))()
    for j, sg in enumerate(segments):
        arr[j].length_m, arr[j].dk_per_m, arr[j].d_eff_m_per_V, arr[j].nz = float(sg[0]), float(sg[1]), float(sg[2]), int(sg[3])
    _check(h, lib().opo_set_segments(h, n, arr))


def opo_set_beta3(h, field: int, beta3_s3_per_m: float):
    _check(h, lib().opo_set_beta3(h, int(field), float(beta3_s3_per_m)))


def opo_set_eom(h, field: int, beta_rad: float, f_mod_hz: float):
    _check(h, lib().opo_set_eom(h, int(field), float(beta_rad), float(f_mod_hz)))


def opo_set_pump(h, dev_ptr: int, per_instance: bool):
    _check(h, lib().opo_set_pump(h, ctypes.c_void_p(dev_ptr), int(per_instance)))


def opo_set_pump_host(h, host_ptr: int, per_instance: bool):
    _check(h, lib().opo_set_pump_host(h, ctypes.c_void_p(host_ptr), int(per_instance)))


def opo_set_field(h, field: int, dev_ptr: int):
    _check(h, lib().opo_set_field(h, field, ctypes.c_void_p(dev_ptr)))


def opo_set_field_host(h, field: int, host_ptr: int):
    _check(h, lib().opo_set_field_host(h, field, ctypes.c_void_p(host_ptr)))


def opo_propagate(h, nz: int):
    _check(h, lib().opo_propagate(h, int(nz)))


def opo_roundtrips(h, n: int):
    _check(h, lib().opo_roundtrips(h, int(n)))


def opo_roundtrips_train(h, n: int, dev_pump_train: int, per_instance: bool, dev_out_train: int, out_field: int):
    _check(h, lib().opo_roundtrips_train(h, int(n), ctypes.c_void_p(dev_pump_train), int(per_instance),
                                         ctypes.c_void_p(dev_out_train) if dev_out_train else None, int(out_field)))


def opo_get_fields(h, field: int, which: int, domain: int, dev_ptr: int):
    _check(h, lib().opo_get_fields(h, field, which, domain, ctypes.c_void_p(dev_ptr)))


def opo_get_fields_host(h, field: int, which: int, domain: int, host_ptr: int):
    _check(h, lib().opo_get_fields_host(h, field, which, domain, ctypes.c_void_p(host_ptr)))


def opo_sync(h):
    _check(h, lib().opo_sync(h))


def opo_check_finite(h):
    _check(h, lib().opo_check_finite(h))


def opo_get_z_steps(h) -> int:
    out = ctypes.c_int()
    _check(h, lib().opo_get_z_steps(h, ctypes.byref(out)))
    return out.value


def opo_set_option(h, option: int, value: int):
    _check(h, lib().opo_set_option(h, option, value))


PEAK_FP32_FMA, PEAK_FP64_FMA, PEAK_SMEM, PEAK_TMEM_LD, PEAK_TMEM_ST, PEAK_DSMEM = 0, 1, 2, 3, 4, 5


def opo_selftest_peak(what: int) -> float:
    """Device peak measured by the library's own micro-benchmark kernels (TFLOP/s or GB/s, see include/opo.h)."""
    out = ctypes.c_double()
    _check(None, lib().opo_selftest_peak(what, ctypes.byref(out)))
    return out.value


def opo_spectrum_noalloc(dev_in: int, dev_out: int, log2_n: int, batch: int, precision: int, cuda_stream: int = 0):
    """Forward DFT of [batch][2^log2_n] rows the caller owns, with no handle and no device allocation inside the library
    (include/opo.h: for callers whose memory pool owns all of HBM, or whose loop cannot take cudaMalloc's device-wide
    synchronisation).  Pointers are raw device addresses (tensor.data_ptr()); the tables live in a fixed 192 KiB array
    inside libopo.so, so rows are limited to 2^14 points (complex64) / 2^13 (complex128)."""
    _check(None, lib().opo_spectrum_noalloc(ctypes.c_void_p(dev_in), ctypes.c_void_p(dev_out), int(log2_n), int(batch), int(precision),
                                            ctypes.c_void_p(cuda_stream) if cuda_stream else None))


def opo_get_info(h, what: int) -> int:
    out = ctypes.c_longlong()
    _check(h, lib().opo_get_info(h, what, ctypes.byref(out)))
    return out.value


# ---- object wrapper (marshalling of torch tensors) -------------------------------------------------------

class Opo:
    """One handle.  Tensors are torch complex64/complex128 on the current CUDA device (or pinned
    host tensors for the *_host calls); the library works on the current torch stream."""

    def __init__(self, *, n_fields, log2_n, window_s, nz_per_pass, length_m, dk_per_m, d_eff_m_per_V,
                 lambda_m, n_index, beta1_s_per_m, beta2_s2_per_m, alpha_per_m=None, ref_field=1,
                 resonant=None, R=None, delta_rad=None, delta_T_s=None, gdd_s2=None,
                 precision="c64", batch=1, engine=ENGINE_AUTO):
        import torch
        self._torch = torch
        c = opo_crystal(float(length_m), float(dk_per_m), float(d_eff_m_per_V))
        f = opo_fields(int(n_fields), _d3(lambda_m), _d3(n_index), _d3(beta1_s_per_m), _d3(beta2_s2_per_m),
                       _d3(alpha_per_m), int(ref_field), _i3(resonant), _d3(R), _d3(delta_rad),
                       _d3(delta_T_s), _d3(gdd_s2))
        g = opo_grid(int(log2_n), float(window_s), int(nz_per_pass),
                     PRECISION_C128 if precision == "c128" else PRECISION_C64, int(batch))
        self.n_fields, self.n, self.batch = int(n_fields), 1 << int(log2_n), int(batch)
        self.dtype = torch.complex128 if precision == "c128" else torch.complex64
        self._h = opo_create(c, f, g)
        self.use_current_stream()
        if engine != ENGINE_AUTO:
            opo_set_option(self._h, OPT_ENGINE, engine)

    def close(self):
        if getattr(self, "_h", None):
            opo_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def use_current_stream(self):
        opo_set_stream(self._h, self._torch.cuda.current_stream().cuda_stream)

    def _dev(self, t, shape):
        assert t.is_cuda and t.dtype == self.dtype and t.is_contiguous() and tuple(t.shape) == tuple(shape), \
            (t.device, t.dtype, tuple(t.shape), shape)
        return t.data_ptr()

    def _host(self, t, shape):
        assert (not t.is_cuda) and t.dtype == self.dtype and t.is_contiguous() and tuple(t.shape) == tuple(shape)
        return t.data_ptr()

    def set_batch_param(self, param, field, values):
        opo_set_batch_param(self._h, param, field, values)

    def set_segments(self, segments):
        opo_set_segments(self._h, segments)

    def set_beta3(self, field, beta3_s3_per_m):
        opo_set_beta3(self._h, field, beta3_s3_per_m)

    def set_eom(self, field, beta_rad, f_mod_hz):
        opo_set_eom(self._h, field, beta_rad, f_mod_hz)

    def set_pump(self, pump):
        per = pump.dim() == 2 and pump.shape[0] == self.batch and self.batch > 1
        shape = (self.batch, self.n) if per else tuple(pump.shape)
        assert pump.numel() == (self.batch * self.n if per else self.n)
        if pump.is_cuda:
            opo_set_pump(self._h, self._dev(pump, shape), per)
        else:
            opo_set_pump_host(self._h, self._host(pump, shape), per)

    def set_field(self, field, data):
        if data.is_cuda:
            opo_set_field(self._h, field, self._dev(data, (self.batch, self.n)))
        else:
            opo_set_field_host(self._h, field, self._host(data, (self.batch, self.n)))

    def propagate(self, nz):
        opo_propagate(self._h, nz)

    def roundtrips(self, n):
        opo_roundtrips(self._h, n)

    def roundtrips_train(self, pump_train, out_field=None):
        """pump_train: CUDA tensor [n][N] or [n][batch][N]; returns the exit field `out_field` of every round trip,
        [n][batch][N], or None (nanosecond regime)."""
        torch = self._torch
        assert pump_train.is_cuda and pump_train.dtype == self.dtype
        n = pump_train.shape[0]
        per = pump_train.dim() == 3
        assert tuple(pump_train.shape[1:]) == ((self.batch, self.n) if per else (self.n,))
        pump_train = pump_train.contiguous()
        out = torch.empty((n, self.batch, self.n), dtype=self.dtype, device="cuda") if out_field is not None else None
        opo_roundtrips_train(self._h, n, pump_train.data_ptr(), per, out.data_ptr() if out is not None else 0,
                             out_field if out_field is not None else 0)
        return out

    def get_fields(self, field, which=WHICH_CURRENT, domain=DOMAIN_TIME, out=None):
        torch = self._torch
        if out is None:
            out = torch.empty((self.batch, self.n), dtype=self.dtype, device="cuda")
        if out.is_cuda:
            opo_get_fields(self._h, field, which, domain, self._dev(out, (self.batch, self.n)))
        else:
            opo_get_fields_host(self._h, field, which, domain, self._host(out, (self.batch, self.n)))
        return out

    def sync(self):
        opo_sync(self._h)

    def check_finite(self):
        opo_check_finite(self._h)

    @property
    def z_steps(self):
        return opo_get_z_steps(self._h)

    @property
    def engine(self):
        return opo_get_info(self._h, INFO_ENGINE)

    @property
    def launches(self):
        return opo_get_info(self._h, INFO_LAUNCHES)

    def set_engine(self, engine):
        opo_set_option(self._h, OPT_ENGINE, engine)


def from_workload(w, engine=ENGINE_AUTO, host_inputs=False) -> Opo:
    """Marshal an opo_workloads.Workload (seeded synthetic inputs) into a handle with pump and seeds loaded."""
    import torch
    o = Opo(n_fields=w.n_fields, log2_n=w.log2_n, window_s=w.window_s, nz_per_pass=w.nz_per_pass,
            length_m=w.length_m, dk_per_m=float(w.dk_per_m[0]), d_eff_m_per_V=w.d_eff_m_per_V,
            lambda_m=w.lambda_m, n_index=w.n_index, beta1_s_per_m=w.beta1_s_per_m,
            beta2_s2_per_m=w.beta2_s2_per_m, alpha_per_m=w.alpha_per_m, ref_field=w.ref_field,
            resonant=w.resonant, R=w.R, delta_rad=w.delta_rad, delta_T_s=w.delta_T_s, gdd_s2=w.gdd_s2,
            precision=w.precision, batch=w.batch, engine=engine)
    if getattr(w, "segments", None):
        o.set_segments(w.segments)          # before the per-instance dk sweep, which acts on the first segment
    if len(w.dk_per_m) > 1:
        o.set_batch_param(PARAM_DK, 0, w.dk_per_m)
    if w.delta_T_signal_s is not None:
        o.set_batch_param(PARAM_DELTA_T, 1, w.delta_T_signal_s)
    for x in range(w.n_fields):
        if w.eom_beta_rad[x] != 0.0:
            o.set_eom(x, w.eom_beta_rad[x], w.eom_f_hz[x])
        if w.beta3_s3_per_m[x] != 0.0:
            o.set_beta3(x, w.beta3_s3_per_m[x])
    if w.splitting:
        opo_set_option(o._h, OPT_SPLITTING, int(w.splitting))
    load_inputs(o, w, host_inputs)
    return o


def load_inputs(o: Opo, w, host_inputs=False):
    import torch
    dev = "cpu" if host_inputs else "cuda"
    pump = torch.from_numpy(np.ascontiguousarray(w.pump)).to(o.dtype)
    pump = pump if pump.shape[0] > 1 else pump[0]
    o.set_pump(pump.contiguous().to(dev))
    for x in range(1, w.n_fields):
        o.set_field(x, torch.from_numpy(np.ascontiguousarray(w.seeds[x])).to(o.dtype).contiguous().to(dev))
    o.sync()
