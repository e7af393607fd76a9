"""The C-ABI library loads and exports every symbol include/opo.h declares (no compute calls: no GPU here)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "opo.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(opo_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = declared_symbols()
    for must in ("opo_create", "opo_set_pump", "opo_propagate", "opo_roundtrips", "opo_get_fields", "opo_destroy"):
        assert must in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2410_02532_b200 import build as b
    path = b.build()
    lib = ctypes.CDLL(path)
    for name in declared_symbols():
        assert hasattr(lib, name), f"libopo.so does not export {name}"
    import paper_2410_02532_b200 as P
    assert sorted(P.EXPORTS) == declared_symbols()
    P.lib()


def test_create_fails_loudly_without_a_gpu_and_reports_why():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import paper_2410_02532_b200 as P
    import opo_workloads as W
    with pytest.raises(P.OpoError) as e:
        P.Opo(n_fields=2, log2_n=8, window_s=1e-11, nz_per_pass=4, length_m=5e-3, dk_per_m=0.0, d_eff_m_per_V=14e-12,
              lambda_m=[532e-9, 1064e-9], n_index=[2.23, 2.16], beta1_s_per_m=[0, 0], beta2_s2_per_m=[0, 0],
              resonant=[0, 1], R=[0, 0.98])
    assert e.value.status == P.ERR_CUDA          # no CPU fallback


def test_invalid_arguments_are_rejected_before_touching_the_device():
    import paper_2410_02532_b200 as P
    kw = dict(n_fields=2, log2_n=8, window_s=1e-11, nz_per_pass=4, length_m=5e-3, dk_per_m=0.0, d_eff_m_per_V=14e-12,
              lambda_m=[532e-9, 1064e-9], n_index=[2.23, 2.16], beta1_s_per_m=[0, 0], beta2_s2_per_m=[0, 0],
              resonant=[0, 1], R=[0, 0.98])
    for bad, status in ((dict(n_fields=4), P.ERR_INVALID_ARG), (dict(log2_n=30), P.ERR_INVALID_ARG),
                        (dict(nz_per_pass=0), P.ERR_INVALID_ARG), (dict(R=[0, 1.5]), P.ERR_INVALID_ARG),
                        (dict(resonant=[1, 1], log2_n=16), P.ERR_UNSUPPORTED)):      # resonant pump: not on the large-N engine
        with pytest.raises(P.OpoError) as e:
            P.Opo(**{**kw, **bad})
        assert e.value.status == status, bad
