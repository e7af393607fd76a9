#!/usr/bin/env python
"""Writes the stored expected values of the config-length parity tests (tests/test_gpu_config_length.py).

    python tests/golden/make_long_run_goldens.py [--only C1,C2,C3,C3s,C3full,C4] [--threads 8] [--no-float]

Calls ONLY oracle/ (the plain fp64 CPU implementation written from the paper) and opo_workloads (seeded inputs);
nothing here touches the CUDA path.  Each file name carries a hash of the workload's inputs and parameters, so a
changed input recipe cannot silently be compared against stale values.

Files (numpy .npz, under tests/golden/):
  c3_20rt_<hash>.npz          C3 (N = 2^18, nz = 500), exit pump and signal after 20 round trips, complex64
                              (the rounding of the stored value, 6e-8, is far below the 1e-4 tolerance)
  c3s_20rt_<hash>.npz         C3 on N = 2^15 (the smallest grid of the large-N engine), 20 round trips = 10^4 z-steps: exit
                              fields of the fp64 oracle and (pin P12) the field error of the oracle run in `float`
  c1_1000rt_<hash>.npz        long noise-seeded runs (BASELINE.json north_star: <= 1e-3 on output signal power and on
  c2_500rt_<hash>.npz         the power spectrum, not phase; reading R21): per instance the output signal power
  c4_300rt_sub16_<hash>.npz   (1 - R_s) mean|exit_s|^2 (R16), the pump depletion 1 - mean|exit_p|^2 / mean|S_p|^2, the
                              power spectrum |DFT(exit_s)|^2 (float32) -- from the fp64 oracle, and (pin P12, reported,
                              not asserted) the same three numbers' deviation when the oracle runs in `float`.
  c3_200rt_<hash>.npz         C3 at its full length (200 round trips = 10^5 z-steps on N = 2^18), same three numbers + P12
Oracle cost (8 cores): C3 ~ 6 min, C1 ~ 10 + 10 min, C2 ~ 20 + 20 min, C4 ~ 6 + 6 min; C3full ~ 70 min (one instance: the fp64
and the float run take one core each, side by side).
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import sys
import time
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import numpy as np

import opo_workloads as W
import oracle


def workload_hash(w) -> str:
    """Hash of everything the oracle is fed with for this workload."""
    h = hashlib.sha1()
    scalars = [w.length_m, w.d_eff_m_per_V, w.n_fields, w.ref_field, w.log2_n, w.window_s, w.nz_per_pass, w.batch, w.n_roundtrips,
               w.precision, w.splitting]
    h.update(repr(scalars).encode())
    for v in (w.lambda_m, w.n_index, w.beta1_s_per_m, w.beta2_s2_per_m, w.alpha_per_m, w.resonant, w.R, w.delta_rad, w.delta_T_s,
              w.gdd_s2, w.eom_beta_rad, w.eom_f_hz, w.beta3_s3_per_m):
        h.update(repr([float(x) for x in v]).encode())
    h.update(np.ascontiguousarray(w.dk_per_m, dtype=np.float64).tobytes())
    if w.delta_T_signal_s is not None:
        h.update(np.ascontiguousarray(w.delta_T_signal_s, dtype=np.float64).tobytes())
    h.update(np.ascontiguousarray(w.pump).tobytes())
    for s in w.seeds:
        if s is not None:
            h.update(np.ascontiguousarray(s).tobytes())
    return h.hexdigest()[:12]


C4_SUBSET = [0, 15, 240, 255, 17, 34, 51, 68, 85, 102, 119, 136, 153, 170, 187, 204]     # the 4 sweep corners + the diagonal


def long_run_workloads():
    return {"C1": ("c1_1000rt", W.config1()),
            "C2": ("c2_500rt", W.config2()),
            "C4": ("c4_300rt_sub16", W.config4().subset(C4_SUBSET))}


def summarise(w, ex):
    """Harness arithmetic on the exit fields (readings R16, R21): output signal power, pump depletion, power spectrum."""
    R_s = w.R[1]
    p_out = (1.0 - R_s) * np.mean(np.abs(ex[:, 1]) ** 2, axis=1)
    p_in = np.array([np.mean(np.abs(w.pump_of(b)) ** 2) for b in range(w.batch)])
    depletion = 1.0 - np.mean(np.abs(ex[:, 0]) ** 2, axis=1) / p_in
    spec = np.abs(np.fft.fft(ex[:, 1], axis=1)) ** 2
    return p_out, depletion, spec


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--only", default="C3,C3s,C4,C1,C2,C3full")
    ap.add_argument("--threads", type=int, default=os.cpu_count() or 1)
    ap.add_argument("--no-float", action="store_true", help="skip the float instantiation of the oracle (pin P12)")
    args = ap.parse_args()
    only = set(args.only.split(","))
    oracle.build()
    report = {}
    if "C3" in only:
        w = W.config3().truncated(20)
        name = f"c3_20rt_{workload_hash(w)}.npz"
        t0 = time.time()
        res = oracle.run_workload(w, threads=1)
        np.savez_compressed(os.path.join(HERE, name), exit_pump=res["exit"][0, 0].astype(np.complex64),
                            exit_signal=res["exit"][0, 1].astype(np.complex64), n_roundtrips=20)
        print(f"{name}: {time.time() - t0:.0f} s", flush=True)
    if "C3s" in only:
        w = W.config3(20, 15)
        name = f"c3s_20rt_{workload_hash(w)}.npz"
        t0 = time.time()
        res = oracle.run_workload(w, threads=1)
        out = {"exit_pump": res["exit"][0, 0].astype(np.complex64), "exit_signal": res["exit"][0, 1].astype(np.complex64), "n_roundtrips": 20}
        if not args.no_float:
            resf = oracle.run_workload(w, threads=1, use_float=True)
            fe = [float(np.linalg.norm(resf["exit"][0, x] - res["exit"][0, x]) / np.linalg.norm(res["exit"][0, x])) for x in range(2)]
            out["float_field_rel_l2"] = np.array(fe)
            report["C3s"] = {"p12_float_vs_fp64_field_rel_l2_pump": fe[0], "p12_float_vs_fp64_field_rel_l2_signal": fe[1]}
        np.savez_compressed(os.path.join(HERE, name), **out)
        print(f"{name}: {time.time() - t0:.0f} s {json.dumps(report.get('C3s', {}))}", flush=True)
    if "C3full" in only:
        # BASELINE.json configs[3] at its own length: one instance, so the fp64 and the float run go side by side
        w = W.config3()
        name = f"c3_200rt_{workload_hash(w)}.npz"
        t0 = time.time()
        with ThreadPoolExecutor(max_workers=2) as pool:      # ctypes releases the GIL during the C call
            f64 = pool.submit(oracle.run_workload, w, threads=1)
            f32 = None if args.no_float else pool.submit(oracle.run_workload, w, threads=1, use_float=True)
            res = f64.result()
            resf = f32.result() if f32 else None
        p_out, depl, spec = summarise(w, res["exit"])
        out = {"p_out": p_out, "depletion": depl, "spectrum": spec.astype(np.float32), "n_roundtrips": w.n_roundtrips}
        if resf is not None:
            pf, df, sf = summarise(w, resf["exit"])
            out["float_p_out"] = pf
            out["float_depletion"] = df
            out["float_spectrum_rel_l2"] = np.array([np.linalg.norm(sf[0] - spec[0]) / np.linalg.norm(spec[0])])
            out["float_field_rel_l2"] = np.array([np.linalg.norm(resf["exit"][0, 1] - res["exit"][0, 1]) / np.linalg.norm(res["exit"][0, 1])])
            report["C3"] = {"p12_float_vs_fp64_power_rel_err_max": float(np.max(np.abs(pf - p_out) / p_out)),
                            "p12_float_vs_fp64_spectrum_rel_l2_max": float(out["float_spectrum_rel_l2"][0]),
                            "p12_float_vs_fp64_field_rel_l2_max": float(out["float_field_rel_l2"][0])}
        np.savez_compressed(os.path.join(HERE, name), **out)
        print(f"{name}: {time.time() - t0:.0f} s; depletion {np.round(depl, 4).tolist()} {json.dumps(report.get('C3', {}))}", flush=True)
    for key, (stem, w) in long_run_workloads().items():
        if key not in only:
            continue
        name = f"{stem}_{workload_hash(w)}.npz"
        t0 = time.time()
        res = oracle.run_workload(w, threads=args.threads)
        p_out, depl, spec = summarise(w, res["exit"])
        out = {"p_out": p_out, "depletion": depl, "spectrum": spec.astype(np.float32), "n_roundtrips": w.n_roundtrips}
        t1 = time.time()
        if not args.no_float:
            resf = oracle.run_workload(w, threads=args.threads, use_float=True)
            pf, df, sf = summarise(w, resf["exit"])
            out["float_p_out"] = pf
            out["float_depletion"] = df
            out["float_spectrum_rel_l2"] = np.array([np.linalg.norm(sf[b] - spec[b]) / np.linalg.norm(spec[b]) for b in range(w.batch)])
            out["float_field_rel_l2"] = np.array([np.linalg.norm(resf["exit"][b, 1] - res["exit"][b, 1]) / np.linalg.norm(res["exit"][b, 1])
                                                  for b in range(w.batch)])
            report[key] = {"p12_float_vs_fp64_power_rel_err_max": float(np.max(np.abs(pf - p_out) / p_out)),
                           "p12_float_vs_fp64_spectrum_rel_l2_max": float(np.max(out["float_spectrum_rel_l2"])),
                           "p12_float_vs_fp64_field_rel_l2_max": float(np.max(out["float_field_rel_l2"]))}
        np.savez_compressed(os.path.join(HERE, name), **out)
        print(f"{name}: fp64 {t1 - t0:.0f} s, float {time.time() - t1:.0f} s; depletion {np.round(depl, 4).tolist()[:4]}.. "
              f"{json.dumps(report.get(key, {}))}", flush=True)
    if report:
        path = os.path.join(HERE, "p12_float_oracle_report.json")
        old = json.load(open(path)) if os.path.exists(path) else {}
        old.update(report)
        json.dump(old, open(path, "w"), indent=1, sort_keys=True)


if __name__ == "__main__":
    main()
