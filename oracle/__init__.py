"""ORACLE -- test infrastructure only (see oracle/opo_oracle.cpp header).

ctypes wrapper around the plain fp64 C++ oracle.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It imports nothing from
the CUDA package (paper_2410_02532_b200) and shares no code with it.
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor
from typing import Dict, List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "opo_oracle.cpp")
_SO = os.path.join(_HERE, "libopo_oracle.so")

_lib = None

_DP = ctypes.POINTER(ctypes.c_double)
_IP = ctypes.POINTER(ctypes.c_int)


def build(force: bool = False) -> str:
    """Compile the oracle with g++ -O2 (building the checker is not using it)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-ffp-contract=off", "-o", _SO, _SRC]
        subprocess.check_call(cmd)
    return _SO


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_SO)
        L.opo_oracle_create.restype = ctypes.c_void_p
        L.opo_oracle_create.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_int,
                                        ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                        _DP, _DP, _DP, _DP, _DP, ctypes.c_int, _IP, _DP, _DP, _DP, _DP,
                                        ctypes.c_int]
        L.opo_oracle_destroy.argtypes = [ctypes.c_void_p]
        L.opo_oracle_set_field.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, _DP]
        L.opo_oracle_set_eom.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_double]
        L.opo_oracle_set_beta3.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_double]
        L.opo_oracle_set_splitting.argtypes = [ctypes.c_void_p, ctypes.c_int]
        L.opo_oracle_set_segments.argtypes = [ctypes.c_void_p, ctypes.c_int, _DP, _DP, _DP, _IP]
        L.opo_oracle_set_segments.restype = ctypes.c_int
        L.opo_oracle_propagate.argtypes = [ctypes.c_void_p, ctypes.c_int]
        L.opo_oracle_propagate.restype = ctypes.c_int
        L.opo_oracle_roundtrips.argtypes = [ctypes.c_void_p, ctypes.c_int]
        L.opo_oracle_roundtrips.restype = ctypes.c_int
        L.opo_oracle_get_field.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, _DP]
        L.opo_oracle_kappa.argtypes = [ctypes.c_void_p, ctypes.c_int]
        L.opo_oracle_kappa.restype = ctypes.c_double
        L.opo_oracle_z.argtypes = [ctypes.c_void_p]
        L.opo_oracle_z.restype = ctypes.c_double
        L.opo_oracle_fft.argtypes = [ctypes.c_int, ctypes.c_int, _DP]
        _lib = L
    return _lib


def _darr(v: Sequence[float], n: int = 3):
    a = (ctypes.c_double * n)()
    for i, x in enumerate(v):
        a[i] = float(x)
    return a


def _iarr(v: Sequence[int], n: int = 3):
    a = (ctypes.c_int * n)()
    for i, x in enumerate(v):
        a[i] = int(x)
    return a


def fft(x: np.ndarray, inverse: bool = False) -> np.ndarray:
    """The oracle's own radix-2 transform (forward unnormalised, inverse 1/N)."""
    x = np.ascontiguousarray(x, dtype=np.complex128).copy()
    n = x.shape[0]
    log2n = n.bit_length() - 1
    assert 1 << log2n == n
    lib().opo_oracle_fft(log2n, int(inverse), x.view(np.float64).ctypes.data_as(_DP))
    return x


CURRENT, EXIT = 0, 1
TIME, FREQ = 0, 1


class OracleOpo:
    """One OPO instance.  Arguments are SI, named as in include/opo.h."""

    def __init__(self, *, n_fields, log2_n, window_s, nz_per_pass, length_m, dk_per_m, d_eff_m_per_V,
                 lambda_m, n_index, beta1_s_per_m, beta2_s2_per_m, alpha_per_m=None, ref_field=1,
                 resonant=None, R=None, delta_rad=None, delta_T_s=None, gdd_s2=None,
                 use_float=False):
        F = n_fields
        z3 = [0.0] * 3
        self.n_fields = F
        self.n = 1 << log2_n
        self._h = lib().opo_oracle_create(
            F, log2_n, float(window_s), int(nz_per_pass), float(length_m), float(dk_per_m),
            float(d_eff_m_per_V), _darr(lambda_m), _darr(n_index), _darr(beta1_s_per_m),
            _darr(beta2_s2_per_m), _darr(alpha_per_m or z3), int(ref_field),
            _iarr(resonant or [0, 0, 0]), _darr(R or z3), _darr(delta_rad or z3),
            _darr(delta_T_s or z3), _darr(gdd_s2 or z3), int(bool(use_float)))
        if not self._h:
            raise ValueError("opo_oracle_create rejected the parameters")

    def __del__(self):
        h = getattr(self, "_h", None)
        if h and _lib is not None:
            _lib.opo_oracle_destroy(h)
            self._h = None

    def set_field(self, field: int, data: np.ndarray, which: str = "both"):
        """which: 'state' (current field only), 'input' (stored S_x only) or 'both'."""
        d = np.ascontiguousarray(data, dtype=np.complex128)
        assert d.shape == (self.n,)
        code = {"state": 0, "input": 1, "both": 2}[which]
        lib().opo_oracle_set_field(self._h, field, code, d.view(np.float64).ctypes.data_as(_DP))

    def set_splitting(self, splitting: int):
        """0: L/2 - N - L/2 (default); 1: N/2 - L - N/2, the order of the paper's Eq. 10-11."""
        lib().opo_oracle_set_splitting(self._h, int(splitting))

    def set_beta3(self, field: int, beta3_s3_per_m: float):
        """Third-order dispersion of a field (Eq. 5 in the reading R7)."""
        lib().opo_oracle_set_beta3(self._h, int(field), float(beta3_s3_per_m))

    def set_segments(self, segments) -> int:
        """Crystal segments in series (reading R25): a list of (length_m, dk_per_m, d_eff_m_per_V, nz);
        an empty list restores the single crystal of the constructor.  Only at the start of a pass."""
        n = len(segments)
        return lib().opo_oracle_set_segments(self._h, n, _darr([s[0] for s in segments], max(n, 1)), _darr([s[1] for s in segments], max(n, 1)),
                                             _darr([s[2] for s in segments], max(n, 1)), _iarr([s[3] for s in segments], max(n, 1)))

    def set_eom(self, field: int, beta_rad: float, f_hz: float):
        """Intracavity phase modulator on a resonant field; beta = 0 switches it off."""
        lib().opo_oracle_set_eom(self._h, int(field), float(beta_rad), float(f_hz))

    def propagate(self, nz: int) -> int:
        return lib().opo_oracle_propagate(self._h, int(nz))

    def roundtrips(self, n: int) -> int:
        return lib().opo_oracle_roundtrips(self._h, int(n))

    def get_field(self, field: int, which: int = CURRENT, domain: int = TIME) -> np.ndarray:
        out = np.empty(self.n, dtype=np.complex128)
        lib().opo_oracle_get_field(self._h, field, which, domain, out.view(np.float64).ctypes.data_as(_DP))
        return out

    def kappa(self, field: int) -> float:
        return lib().opo_oracle_kappa(self._h, field)

    @property
    def z(self) -> float:
        return lib().opo_oracle_z(self._h)


def from_workload(w, b: int = 0, use_float: bool = False) -> OracleOpo:
    """Build instance b of an opo_workloads.Workload and load its pump and seeds (m = 0: all fields = S_x)."""
    dT = [w.delta_T_of(b, x) for x in range(w.n_fields)]
    o = OracleOpo(n_fields=w.n_fields, log2_n=w.log2_n, window_s=w.window_s, nz_per_pass=w.nz_per_pass,
                  length_m=w.length_m, dk_per_m=w.dk_of(b), d_eff_m_per_V=w.d_eff_m_per_V,
                  lambda_m=w.lambda_m, n_index=w.n_index, beta1_s_per_m=w.beta1_s_per_m,
                  beta2_s2_per_m=w.beta2_s2_per_m, alpha_per_m=w.alpha_per_m, ref_field=w.ref_field,
                  resonant=w.resonant, R=w.R, delta_rad=w.delta_rad, delta_T_s=dT, gdd_s2=w.gdd_s2,
                  use_float=use_float)
    o.set_field(0, w.pump_of(b))
    if w.resonant[0]:
        # resonant pump (reading R24): at m = 0 the cavity holds what the input coupler transmits, sqrt(1 - R_p) S_p
        o.set_field(0, math.sqrt(1.0 - w.R[0]) * w.pump_of(b), which="state")
    for x in range(1, w.n_fields):
        o.set_field(x, w.seeds[x][b])
    for x in range(w.n_fields):
        if w.eom_beta_rad[x] != 0.0:
            o.set_eom(x, w.eom_beta_rad[x], w.eom_f_hz[x])
        if w.beta3_s3_per_m[x] != 0.0:
            o.set_beta3(x, w.beta3_s3_per_m[x])
    if w.splitting:
        o.set_splitting(w.splitting)
    if getattr(w, "segments", None):
        # per-instance dk sweeps apply to the first segment (include/opo.h, OPO_PARAM_DK)
        segs = [tuple(sg) for sg in w.segments]
        if len(w.dk_per_m) > 1:
            segs[0] = (segs[0][0], w.dk_of(b), segs[0][2], segs[0][3])
        assert o.set_segments(segs) == 0
    return o


def run_workload(w, n_roundtrips: Optional[int] = None, instances: Optional[Sequence[int]] = None,
                 use_float: bool = False, threads: int = 1) -> Dict[str, np.ndarray]:
    """Run round trips for the listed instances; returns current and exit fields [len(instances)][F][N]."""
    inst = list(range(w.batch)) if instances is None else list(instances)
    nrt = w.n_roundtrips if n_roundtrips is None else n_roundtrips

    def one(b):
        o = from_workload(w, b, use_float)
        rc = o.roundtrips(nrt)
        assert rc == 0, rc
        cur = np.stack([o.get_field(x, CURRENT) for x in range(w.n_fields)])
        ex = np.stack([o.get_field(x, EXIT) for x in range(w.n_fields)])
        return cur, ex

    if threads > 1 and len(inst) > 1:
        with ThreadPoolExecutor(max_workers=threads) as ex:
            res = list(ex.map(one, inst))      # ctypes releases the GIL during the C call
    else:
        res = [one(b) for b in inst]
    return {"current": np.stack([r[0] for r in res]), "exit": np.stack([r[1] for r in res])}
