"""The seeded input generators: shapes, determinism, and the input scaling of SURVEY.md section 8(d)."""
import numpy as np

import opo_workloads as W


def test_config0_numbers():
    w = W.config0()
    assert w.n == 1024 and w.n_fields == 2 and w.precision == "c128" and w.nz_per_pass == 20
    k = w.kappa()
    assert abs(k[0] / 7.4147e-5 - 1) < 1e-4 and abs(k[1] / 3.8275e-5 - 1) < 1e-4
    a_p = w.pump[0, 0].real
    assert abs(a_p / 7.4647e4 - 1) < 1e-4
    assert w.seeds[1].shape == (1, 1024)
    rms = np.sqrt(np.mean(np.abs(w.seeds[1]) ** 2))
    assert abs(rms / (1e-6 * a_p) - 1) < 0.1


def test_config1_numbers_and_rounding():
    w = W.config1()
    assert w.n == 16384 and w.n_fields == 3 and w.precision == "c64" and w.nz_per_pass == 100
    assert abs(w.lambda_m[2] / 1136.752e-9 - 1) < 1e-6
    k = w.kappa()
    # n_p k_p = n_s k_s + n_i k_i (energy conservation with G1's indices)
    assert abs(w.n_index[0] * k[0] - w.n_index[1] * k[1] - w.n_index[2] * k[2]) / (w.n_index[0] * k[0]) < 1e-12
    assert abs(w.pump[0, 0].real / 3.2206e5 - 1) < 1e-4
    # inputs are exactly representable in fp32 (rounded once, fed identically to both sides)
    for a in (w.pump, w.seeds[1], w.seeds[2]):
        assert np.array_equal(a.astype(np.complex64).astype(np.complex128), a)
    # relative group delays: reference = signal (R10)
    db1 = [b - w.beta1_s_per_m[w.ref_field] for b in w.beta1_s_per_m]
    assert np.allclose(np.array(db1) / W.FS_PER_UM, [0.28, 0.0, -0.17])


def test_generators_are_deterministic():
    a, b = W.config4(batch_side=4), W.config4(batch_side=4)
    assert a.batch == 16
    assert np.array_equal(a.seeds[1], b.seeds[1]) and np.array_equal(a.pump, b.pump)
    assert len(np.unique(a.dk_per_m)) == 4
    assert not np.array_equal(a.seeds[1][0], a.seeds[1][1])


def test_config2_and_3_shapes():
    w2 = W.config2()
    assert w2.batch == 11 and w2.gdd_s2[1] == -500e-30 and w2.nz_per_pass == 200
    assert abs(w2.delta_T_signal_s[0] + 20e-15) < 1e-27 and abs(w2.delta_T_signal_s[-1] - 20e-15) < 1e-27
    p = np.abs(w2.pump[0]) ** 2
    half = np.where(p >= p.max() / 2)[0]
    assert abs((half[-1] - half[0] + 1) * w2.dt / 200e-15 - 1) < 0.02      # 200 fs FWHM
    w3 = W.config3(log2_n=12)
    assert w3.n == 4096 and w3.nz_per_pass == 500
    p = np.abs(w3.pump[0]) ** 2
    half = np.where(p >= p.max() / 2)[0]
    assert abs((half[-1] - half[0] + 1) * w3.dt / 500e-12 - 1) < 0.02      # 500 ps FWHM


def test_subset_and_truncate():
    w = W.config4(batch_side=4).truncated(3).subset([0, 5, 15])
    assert w.batch == 3 and w.n_roundtrips == 3 and w.pump.shape[0] == 3 and len(w.dk_per_m) == 3
