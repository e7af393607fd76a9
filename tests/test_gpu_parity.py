"""Parity of the CUDA path (through the C ABI) against the fp64 oracle, element by element, on the
same seeded inputs.  Tolerances are those of BASELINE.json:north_star: complex128 rel. L2 <= 1e-10,
complex64 rel. L2 <= 1e-4 (single pass and <= 20 round trips).  Run with -m gpu on a B200."""
import math

import numpy as np
import pytest

import opo_workloads as W

pytestmark = pytest.mark.gpu

TOL = {"c128": 1e-10, "c64": 1e-4}
_ORACLE_CACHE = {}      # oracle results shared by the engine parametrisations of one test


def _gpu():
    import torch
    import paper_2410_02532_b200 as P
    return torch, P


def rel_l2(a, b):
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def small_workload(log2_n, n_fields, precision, nz=6, batch=1, dk=0.0, seed=7, gdd_dt2=0.0, drad=0.0,
                   strong=True, alpha=0.0):
    """A short synthetic OPO with all effects switched on and every field O(1) populated, so that a
    wrong sign / index / table anywhere shows up at O(1)."""
    base = W.config1() if n_fields == 3 else W.config0()
    w = W.Workload(
        name=f"small{n_fields}w_2^{log2_n}_{precision}", length_m=base.length_m, d_eff_m_per_V=base.d_eff_m_per_V,
        n_fields=n_fields, lambda_m=list(base.lambda_m), n_index=list(base.n_index),
        beta1_s_per_m=list(base.beta1_s_per_m), beta2_s2_per_m=list(base.beta2_s2_per_m),
        alpha_per_m=[alpha * (x + 1) for x in range(n_fields)], ref_field=1,
        resonant=[0, 1, 1][:n_fields] if n_fields == 3 else [0, 1], R=[0.0, 0.9, 0.7][:n_fields],
        delta_rad=[0.0, drad, -0.5 * drad][:n_fields], delta_T_s=[0.0, 0.0, 0.0][:n_fields],
        gdd_s2=[0.0, 0.0, 0.0][:n_fields], log2_n=log2_n, window_s=base.window_s * (1 << log2_n) / base.n,
        nz_per_pass=nz, precision=precision, batch=batch, n_roundtrips=2,
        dk_per_m=np.full(batch, dk) + (np.arange(batch) % 16 * 7.0 if batch > 1 else 0.0))
    n = w.n
    k = w.kappa()
    # GDD in units of dt^2: spectral phase (gdd/2) Omega^2 reaches gdd_dt2 * pi^2 / 2 at the band edge
    w.gdd_s2 = [0.0, gdd_dt2 * w.dt ** 2, 0.5 * gdd_dt2 * w.dt ** 2][:n_fields]
    # pump strong enough for visible gain and depletion within one pass
    g_target = 1.5 if strong else 0.3
    a_p = g_target / (math.sqrt(k[1] * k[-1]) * w.length_m)
    rng = np.random.default_rng(seed)
    tau = w.tau / (w.window_s / 8)
    pump = a_p * (0.6 + 0.4 * np.exp(-tau ** 2)) * np.exp(1j * 0.3 * np.sin(2 * np.pi * np.arange(n) / n))
    pumps = np.stack([pump * (1.0 + 0.1 * (b % 8)) for b in range(batch)])
    w.pump = W._round_to_precision(pumps, precision)
    seeds = [None]
    for x in range(1, n_fields):
        s = np.stack([W.complex_gaussian_noise(seed * 100 + 10 * x + b, n, 0.2 * a_p) for b in range(batch)])
        # band-limit the seed a little so the spectrum is not flat white (closer to a real field)
        sf = np.fft.fft(s, axis=1) * np.exp(-(np.fft.fftfreq(n) * 6) ** 2)[None, :]
        seeds.append(W._round_to_precision(np.fft.ifft(sf, axis=1), precision))
    w.seeds = seeds
    return w


def run_gpu(w, engine, n_roundtrips=None, propagate=None, calls=1):
    torch, P = _gpu()
    o = P.from_workload(w, engine=engine)
    if propagate is not None:
        for nzp in propagate:
            o.propagate(nzp)
    else:
        nrt = w.n_roundtrips if n_roundtrips is None else n_roundtrips
        per = nrt // calls
        for c in range(calls):
            o.roundtrips(per if c < calls - 1 else nrt - per * (calls - 1))
    o.sync()
    cur = np.stack([o.get_fields(x, P.WHICH_CURRENT).cpu().numpy().astype(np.complex128) for x in range(w.n_fields)], axis=1)
    ex = np.stack([o.get_fields(x, P.WHICH_EXIT).cpu().numpy().astype(np.complex128) for x in range(w.n_fields)], axis=1)
    eng = o.engine
    o.close()
    return cur, ex, eng


def run_oracle(w, n_roundtrips=None, propagate=None):
    import oracle
    cur, ex = [], []
    for b in range(w.batch):
        o = oracle.from_workload(w, b)
        if propagate is not None:
            for nzp in propagate:
                assert o.propagate(nzp) == 0
        else:
            assert o.roundtrips(w.n_roundtrips if n_roundtrips is None else n_roundtrips) == 0
        cur.append(np.stack([o.get_field(x, oracle.CURRENT) for x in range(w.n_fields)]))
        ex.append(np.stack([o.get_field(x, oracle.EXIT) for x in range(w.n_fields)]))
    return np.stack(cur), np.stack(ex)


def engines():
    """streaming (unfused internal baseline), resident (cluster per instance), solo (one CTA per instance, TMEM),
    wide (a cluster of 4 F CTAs per instance, fields split over four SMs; N = 2^12 .. 2^14 only)"""
    import paper_2410_02532_b200 as P
    return [P.ENGINE_STREAMING, P.ENGINE_RESIDENT, P.ENGINE_SOLO, P.ENGINE_WIDE]


ENGINE_IDX = [0, 1, 2, 3]


def _engine_or_skip(w, engine):
    torch, P = _gpu()
    if engine in (P.ENGINE_RESIDENT, P.ENGINE_SOLO, P.ENGINE_WIDE):
        o = P.from_workload(w, engine=P.ENGINE_AUTO)
        try:
            o.set_engine(engine)
            ok = o.engine == engine
        except P.OpoError:
            ok = False
        o.close()
        if not ok:
            pytest.skip("engine not available for this size on this device")


def assert_close(got, ref, tol, what):
    worst = 0.0
    assert np.isfinite(got).all(), f"{what}: non-finite values in the CUDA result"
    for b in range(ref.shape[0]):
        for x in range(ref.shape[1]):
            if np.linalg.norm(ref[b, x]) == 0.0:
                assert np.linalg.norm(got[b, x]) == 0.0
                continue
            worst = max(worst, rel_l2(got[b, x], ref[b, x]))
    assert worst <= tol, f"{what}: worst rel L2 {worst:.3e} > {tol:.1e}"
    return worst


# ---------------------------------------------------------------------------------------------------------
# FFT read-out: opo_get_fields(FREQ) against the oracle's own transform, every supported size
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision,log2_n", [("c64", l) for l in range(4, 15)] + [("c128", l) for l in range(4, 14)])
def test_frequency_readout_matches_oracle_fft(precision, log2_n):
    import oracle
    torch, P = _gpu()
    w = small_workload(log2_n, 2, precision, batch=2)
    o = P.from_workload(w)
    got = o.get_fields(1, P.WHICH_CURRENT, P.DOMAIN_FREQ).cpu().numpy().astype(np.complex128)
    o.close()
    for b in range(2):
        ref = oracle.fft(w.seeds[1][b])
        assert rel_l2(got[b], ref) <= (1e-13 if precision == "c128" else 2e-6)


# ---------------------------------------------------------------------------------------------------------
# single crystal pass, every size (several tiles, ragged radix plans), both engines, dk != 0
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("engine_idx", ENGINE_IDX)
@pytest.mark.parametrize("precision,log2_n,n_fields", [
    ("c128", 4, 3), ("c128", 5, 2), ("c64", 4, 2), ("c64", 5, 3),          # the smallest grids of the ABI: N = 16, 32
    ("c128", 6, 2), ("c128", 7, 3), ("c128", 9, 3), ("c128", 10, 2), ("c128", 11, 3), ("c128", 13, 3),
    ("c64", 6, 3), ("c64", 8, 2), ("c64", 9, 3), ("c64", 10, 3), ("c64", 11, 2), ("c64", 12, 3), ("c64", 13, 3),
    ("c64", 14, 3), ("c64", 14, 2)])
def test_single_pass_matches_oracle(precision, log2_n, n_fields, engine_idx):
    engine = engines()[engine_idx]
    w = small_workload(log2_n, n_fields, precision, nz=5, dk=35.0, alpha=3.0)
    _engine_or_skip(w, engine)
    cur, _, eng = run_gpu(w, engine, propagate=[5])
    assert eng == engine
    ref, _ = run_oracle(w, propagate=[5])
    assert_close(cur, ref, TOL[precision] if precision == "c128" else 2e-5, w.name)


@pytest.mark.parametrize("engine_idx", ENGINE_IDX)
def test_partial_passes_continue_dk_phase(engine_idx):
    engine = engines()[engine_idx]
    w = small_workload(9, 3, "c128", nz=7, dk=120.0)
    _engine_or_skip(w, engine)
    cur, _, _ = run_gpu(w, engine, propagate=[2, 1, 4])
    ref, _ = run_oracle(w, propagate=[7])
    assert_close(cur, ref, 1e-10, "partial passes")


# ---------------------------------------------------------------------------------------------------------
# round trips with the full boundary operator: mirror, carrier phase, GDD, group-delay detuning,
# per-instance sweeps; one call (half-steps merged across the boundary) and call-by-call
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("engine_idx", ENGINE_IDX)
@pytest.mark.parametrize("precision,log2_n,n_fields,calls", [
    ("c128", 4, 3, 1), ("c64", 5, 2, 3), ("c128", 8, 3, 1), ("c128", 8, 3, 3), ("c128", 10, 2, 1), ("c64", 11, 3, 1), ("c64", 12, 2, 3)])
def test_roundtrips_with_boundary(precision, log2_n, n_fields, calls, engine_idx):
    engine = engines()[engine_idx]
    torch, P = _gpu()
    w = small_workload(log2_n, n_fields, precision, nz=4, batch=3, dk=-20.0, gdd_dt2=-1.7, drad=0.4, strong=False)
    # per-instance group-delay detuning of the signal in units of the grid step
    w.delta_T_signal_s = np.array([-2.5, 0.0, 1.25]) * w.dt
    _engine_or_skip(w, engine)
    cur, ex, _ = run_gpu(w, engine, n_roundtrips=3, calls=calls)
    rcur, rex = run_oracle(w, n_roundtrips=3)
    tol = TOL[precision] if precision == "c128" else 3e-5
    assert_close(cur, rcur, tol, "current")
    assert_close(ex, rex, tol, "exit")


@pytest.mark.parametrize("engine_idx", ENGINE_IDX)
def test_boundary_without_transform_and_nonresonant_restart(engine_idx):
    engine = engines()[engine_idx]
    w = small_workload(9, 3, "c128", nz=3, batch=2, dk=10.0, drad=-0.7, strong=False)
    w.resonant = [0, 1, 0]          # idler restarts from its seed every round trip (R12)
    _engine_or_skip(w, engine)
    cur, ex, _ = run_gpu(w, engine, n_roundtrips=4)
    rcur, rex = run_oracle(w, n_roundtrips=4)
    assert_close(cur, rcur, 1e-10, "current")
    assert_close(ex, rex, 1e-10, "exit")
    assert np.array_equal(cur[:, 0], w.pump) and np.array_equal(cur[:, 2], w.seeds[2])


# ---------------------------------------------------------------------------------------------------------
# resonant pump (input coupler, reading R24) and several crystals in series (reading R25)
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("engine_idx", ENGINE_IDX)
@pytest.mark.parametrize("precision,log2_n,n_fields,calls,eom", [
    ("c128", 9, 3, 1, False), ("c128", 10, 2, 2, True), ("c64", 12, 3, 1, False), ("c64", 14, 3, 2, False), ("c64", 8, 2, 1, True)])
def test_resonant_pump_matches_oracle(precision, log2_n, n_fields, calls, eom, engine_idx):
    """Doubly / triply resonant cavity: the pump is mirrored like the other resonant fields (own R_p, carrier phase, GDD)
    and the input coupler adds sqrt(1 - R_p) S_p at every boundary; inside the on-chip kernels that is t SH_p added after
    the merged boundary operator.  4 round trips in one call and split over two calls (the un-merged boundary of the
    call's last round trip), per-instance detuning of the pump, a modulator on the pump before the coupler."""
    engine = engines()[engine_idx]
    w = small_workload(log2_n, n_fields, precision, nz=4, batch=3, dk=-20.0, gdd_dt2=-1.3, drad=0.4, strong=False)
    w.resonant = [1, 1, 1][:n_fields]
    w.R = [0.6, 0.9, 0.7][:n_fields]
    w.delta_rad = [0.35, 0.4, -0.2][:n_fields]
    w.gdd_s2 = [0.8 * w.dt ** 2] + list(w.gdd_s2[1:])
    if eom:
        w.eom_beta_rad = [0.5, 0.0, 0.0]
        w.eom_f_hz = [2.0 / w.window_s, 0.0, 0.0]
    _engine_or_skip(w, engine)
    cur, ex, eng = run_gpu(w, engine, n_roundtrips=4, calls=calls)
    assert eng == engine
    rcur, rex = run_oracle(w, n_roundtrips=4)
    tol = TOL[precision] if precision == "c128" else 3e-5
    assert_close(cur, rcur, tol, "current")
    assert_close(ex, rex, tol, "exit")
    # the cavity really stored pump light: the intracavity pump differs from what a single-pass pump would be
    assert rel_l2(cur[0, 0], np.sqrt(1 - 0.6) * w.pump[0]) > 0.05


@pytest.mark.parametrize("engine_idx", ENGINE_IDX[:3])
def test_resonant_pump_input_changed_between_calls_keeps_the_stored_light(engine_idx):
    """A pump ramp on a triply resonant cavity: two round trips, opo_set_pump with 1.5 x the input, two more.  The second
    opo_set_pump finds the handle at z = 0 with light stored in the cavity and must change the input only (oracle pin
    P19, pump input changed mid-run); before round 3 it re-initialised the intracavity pump to sqrt(1 - R_p) S_p."""
    import oracle
    torch, P = _gpu()
    engine = engines()[engine_idx]
    w = small_workload(10, 3, "c128", nz=4, batch=2, dk=-20.0, gdd_dt2=-1.3, drad=0.4, strong=False)
    w.resonant, w.R, w.delta_rad = [1, 1, 1], [0.6, 0.9, 0.7], [0.35, 0.4, -0.2]
    _engine_or_skip(w, engine)
    o = P.from_workload(w, engine=engine)
    o.roundtrips(2)
    o.set_pump(torch.from_numpy(1.5 * w.pump).to(o.dtype).cuda().contiguous())
    o.roundtrips(2)
    o.sync()
    cur = np.stack([o.get_fields(x, P.WHICH_CURRENT).cpu().numpy() for x in range(3)], axis=1)
    o.close()
    ref = []
    for b in range(w.batch):
        r = oracle.from_workload(w, b)
        assert r.roundtrips(2) == 0
        r.set_field(0, 1.5 * w.pump_of(b), which="input")
        assert r.roundtrips(2) == 0
        ref.append(np.stack([r.get_field(x) for x in range(3)]))
    assert_close(cur, np.stack(ref), 1e-10, "pump input changed between calls")


def test_resonant_pump_builds_up_in_a_cold_cavity():
    """Airy build-up measured on the CUDA path alone (no oracle): coupling off, CW pump on resonance, after many round
    trips the intracavity pump power is (1 - R) / (1 - sqrt(R))^2 times the input."""
    torch, P = _gpu()
    w = small_workload(10, 2, "c128", nz=2, batch=1, strong=False)
    w.d_eff_m_per_V = 0.0
    w.resonant, w.R, w.delta_rad, w.gdd_s2 = [1, 0], [0.5, 0.0], [0.0, 0.0], [0.0, 0.0]
    w.beta1_s_per_m, w.beta2_s2_per_m = [0.0, 0.0], [0.0, 0.0]
    w.pump = np.ones((1, w.n), dtype=np.complex128)
    for engine in (P.ENGINE_RESIDENT, P.ENGINE_SOLO, P.ENGINE_STREAMING):
        cur, _, _ = run_gpu(w, engine, n_roundtrips=120)
        assert abs(np.mean(np.abs(cur[0, 0]) ** 2) / ((1 - 0.5) / (1 - np.sqrt(0.5)) ** 2) - 1) < 1e-10


@pytest.mark.parametrize("precision,log2_n,n_fields,splitting", [("c128", 9, 3, 0), ("c64", 12, 3, 0), ("c64", 14, 2, 0), ("c128", 8, 2, 1), ("c64", 11, 3, 1)])
def test_crystal_segments_match_oracle(precision, log2_n, n_fields, splitting):
    """Three crystals in series with different length, step size, dk and d_eff (the last one reversed): partial passes
    that stop inside the second crystal, then round trips with the boundary merged across the last and first crystal's
    half-steps; per-instance dk on the first crystal.  Runs on the host-sequenced streaming engine (AUTO picks it)."""
    torch, P = _gpu()
    w = small_workload(log2_n, n_fields, precision, nz=9, batch=2, dk=30.0, gdd_dt2=-0.9, drad=0.3, strong=False)
    L = w.length_m
    w.segments = [(0.5 * L, 30.0, w.d_eff_m_per_V, 4), (0.2 * L, -90.0, 0.6 * w.d_eff_m_per_V, 2), (0.3 * L, 10.0, -w.d_eff_m_per_V, 3)]
    w.splitting = splitting
    cur, _, eng = run_gpu(w, P.ENGINE_AUTO, propagate=[5, 1, 3])
    assert eng == P.ENGINE_STREAMING
    ref, _ = run_oracle(w, propagate=[9])
    tol = TOL[precision] if precision == "c128" else 3e-5
    assert_close(cur, ref, tol, "single pass through three crystals")
    cur, ex, _ = run_gpu(w, P.ENGINE_AUTO, n_roundtrips=3)
    rcur, rex = run_oracle(w, n_roundtrips=3)
    assert_close(cur, rcur, tol, "current")
    assert_close(ex, rex, tol, "exit")
    # and the ABI's own rules
    o = P.from_workload(w)
    o.propagate(2)
    with pytest.raises(P.OpoError) as e:
        o.set_segments([(L, 0.0, 1e-12, 5)])
    assert e.value.status == P.ERR_STATE
    with pytest.raises(P.OpoError) as e:
        o.propagate(8)                      # 2 + 8 > 9 steps per pass
    assert e.value.status == P.ERR_STATE
    o.close()


# ---------------------------------------------------------------------------------------------------------
# wide engine (a cluster of 4 F CTAs per instance): every size it serves, full boundary operator with per-instance
# sweeps, non-resonant restart, several calls, more instances than co-resident clusters
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision,log2_n,n_fields,calls,batch", [
    ("c64", 12, 3, 1, 3), ("c64", 12, 2, 2, 3), ("c64", 13, 2, 1, 3), ("c64", 13, 3, 3, 2), ("c64", 14, 3, 1, 3), ("c64", 14, 2, 2, 2),
    ("c128", 12, 2, 1, 3), ("c128", 12, 3, 3, 2), ("c128", 13, 3, 1, 2), ("c128", 13, 2, 2, 3), ("c64", 12, 3, 1, 37)])
def test_wide_engine_roundtrips_with_boundary(precision, log2_n, n_fields, calls, batch):
    torch, P = _gpu()
    w = small_workload(log2_n, n_fields, precision, nz=4, batch=batch, dk=-20.0, gdd_dt2=-1.7, drad=0.4, strong=False)
    w.delta_T_signal_s = (np.arange(batch) % 5 - 2.0) * 1.25 * w.dt
    if n_fields == 3:
        w.resonant = [0, 1, 0]      # the idler restarts from its seed every round trip (R12)
    _engine_or_skip(w, P.ENGINE_WIDE)
    cur, ex, eng = run_gpu(w, P.ENGINE_WIDE, n_roundtrips=3, calls=calls)
    assert eng == P.ENGINE_WIDE
    rcur, rex = run_oracle(w, n_roundtrips=3)
    tol = TOL[precision] if precision == "c128" else 3e-5
    assert_close(cur, rcur, tol, "current")
    assert_close(ex, rex, tol, "exit")
    # the same workload on the cluster engine: both follow the same factorisation, so they agree to rounding
    cur2, ex2, eng2 = run_gpu(w, P.ENGINE_RESIDENT, n_roundtrips=3, calls=calls)
    assert eng2 == P.ENGINE_RESIDENT
    assert_close(ex, ex2, 1e-12 if precision == "c128" else 1e-5, "wide vs cluster engine")


@pytest.mark.parametrize("precision,log2_n,n_fields,batch", [("c64", 12, 3, 61), ("c64", 13, 2, 45), ("c64", 14, 3, 15), ("c128", 12, 3, 23)])
def test_wide_engine_many_instances_bitwise_repeatable(precision, log2_n, n_fields, batch):
    """Several instances per cluster, several round trips per instance, every cluster of the GPU busy: two runs must agree bit
    for bit (every value crosses the SM-to-SM network asynchronously: a missing wait would show as a difference between runs),
    and with the cluster engine to rounding."""
    torch, P = _gpu()
    w = small_workload(log2_n, n_fields, precision, nz=5, batch=batch, dk=15.0, gdd_dt2=-0.9, drad=0.2, strong=False)
    w.delta_T_signal_s = (np.arange(batch) % 7 - 3.0) * 0.75 * w.dt
    if n_fields == 3:
        w.resonant = [0, 1, 0]
    _engine_or_skip(w, P.ENGINE_WIDE)
    runs = [run_gpu(w, P.ENGINE_WIDE, n_roundtrips=6, calls=2) for _ in range(3)]
    for cur, ex, eng in runs[1:]:
        assert eng == P.ENGINE_WIDE
        assert np.array_equal(cur, runs[0][0]) and np.array_equal(ex, runs[0][1])
    cur2, ex2, _ = run_gpu(w, P.ENGINE_RESIDENT, n_roundtrips=6, calls=2)
    assert_close(runs[0][1], ex2, 1e-12 if precision == "c128" else 1e-5, "wide vs cluster engine, exit")
    assert_close(runs[0][0], cur2, 1e-12 if precision == "c128" else 1e-5, "wide vs cluster engine, current")


@pytest.mark.parametrize("precision,log2_n,n_fields,batch", [("c64", 12, 3, 5), ("c64", 13, 2, 4), ("c64", 14, 3, 3), ("c128", 13, 3, 2), ("c64", 12, 3, 61)])
def test_wide_engine_two_subblocks_per_cta_is_bitwise_the_same(precision, log2_n, n_fields, batch):
    """OPO_OPT_WIDE_SUBBLOCKS = 2 (clusters of 2 F CTAs, two virtual ranks per CTA) performs exactly the arithmetic of the
    clusters of 4 F CTAs, thread for thread: the results agree bit for bit; and AUTO picks it where it finishes sooner."""
    torch, P = _gpu()
    w = small_workload(log2_n, n_fields, precision, nz=4, batch=batch, dk=-20.0, gdd_dt2=-1.7, drad=0.4, strong=False)
    w.delta_T_signal_s = (np.arange(batch) % 5 - 2.0) * 1.25 * w.dt
    if n_fields == 3:
        w.resonant = [0, 1, 0]
    if log2_n == 13:        # with a phase modulator on the signal: the crossing runs the in-place pass-0 phases
        w.eom_beta_rad = [0.0, 0.8, 0.0][:n_fields]
        w.eom_f_hz = [0.0, 2.0 / w.window_s, 0.0][:n_fields]
    _engine_or_skip(w, P.ENGINE_WIDE)
    res = {}
    for g in (1, 2):
        o = P.from_workload(w, engine=P.ENGINE_WIDE)
        P.opo_set_option(o._h, P.OPT_WIDE_SUBBLOCKS, g)
        slots = int(P.opo_get_info(o._h, P.INFO_SLOTS))
        o.roundtrips(3)
        o.sync()
        res[g] = (np.stack([o.get_fields(x, P.WHICH_EXIT).cpu().numpy() for x in range(n_fields)]),
                  np.stack([o.get_fields(x, P.WHICH_CURRENT).cpu().numpy() for x in range(n_fields)]), slots)
        o.close()
    assert np.array_equal(res[1][0], res[2][0]) and np.array_equal(res[1][1], res[2][1])
    assert res[2][2] >= res[1][2]               # more instances at once
    if batch == 61:
        assert res[2][2] >= 2 * res[1][2]


def test_wide_engine_is_what_auto_picks_for_a_single_instance_and_falls_back():
    torch, P = _gpu()
    w = W.config1().truncated(1)
    o = P.from_workload(w)
    assert o.engine == P.ENGINE_WIDE and int(P.opo_get_info(o._h, P.INFO_SLOTS)) == 1
    o.close()
    w4 = W.config4().truncated(1)
    o = P.from_workload(w4)
    assert o.engine == P.ENGINE_SOLO        # a batch that fills the GPU stays on the solo engine
    o.set_engine(P.ENGINE_WIDE)
    assert o.engine == P.ENGINE_WIDE        # ... unless the caller insists
    o.close()
    ws = small_workload(9, 3, "c64")
    o = P.from_workload(ws)
    with pytest.raises(P.OpoError):
        o.set_engine(P.ENGINE_WIDE)         # N = 2^9: not a size of the wide engine
    assert o.engine != P.ENGINE_WIDE
    o.close()


# ---------------------------------------------------------------------------------------------------------
# the five configurations of BASELINE.json (truncated to <= 20 round trips where they are longer)
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("engine_idx", ENGINE_IDX)
def test_config0_full_c128(engine_idx):
    engine = engines()[engine_idx]
    w = W.config0()
    _engine_or_skip(w, engine)
    cur, ex, _ = run_gpu(w, engine)
    rcur, rex = run_oracle(w)
    e1 = assert_close(cur, rcur, 1e-10, "C0 current")
    e2 = assert_close(ex, rex, 1e-10, "C0 exit")
    print(f"C0 engine {engine}: rel L2 current {e1:.3e} exit {e2:.3e}")


@pytest.mark.parametrize("engine_idx", ENGINE_IDX)
@pytest.mark.parametrize("nrt", [1, 20])
def test_config1_c64(nrt, engine_idx):
    engine = engines()[engine_idx]
    w = W.config1().truncated(nrt)
    _engine_or_skip(w, engine)
    cur, ex, _ = run_gpu(w, engine)
    rcur, rex = run_oracle(w)
    e1 = assert_close(cur, rcur, 1e-4, "C1 current")
    e2 = assert_close(ex, rex, 1e-4, "C1 exit")
    print(f"C1 {nrt} RT engine {engine}: rel L2 current {e1:.3e} exit {e2:.3e}")


@pytest.mark.parametrize("engine_idx", ENGINE_IDX)
def test_config2_subset_c64(engine_idx):
    engine = engines()[engine_idx]
    w = W.config2().truncated(5).subset([0, 5, 10])
    _engine_or_skip(w, engine)
    cur, ex, _ = run_gpu(w, engine)
    rcur, rex = run_oracle(w)
    e1 = assert_close(cur, rcur, 1e-4, "C2 current")
    e2 = assert_close(ex, rex, 1e-4, "C2 exit")
    print(f"C2 5 RT engine {engine}: rel L2 current {e1:.3e} exit {e2:.3e}")


@pytest.mark.parametrize("engine_idx", ENGINE_IDX)
def test_config4_corners_c64(engine_idx):
    engine = engines()[engine_idx]
    w = W.config4(batch_side=16).truncated(5).subset([0, 15, 240, 255, 100])
    _engine_or_skip(w, engine)
    cur, ex, _ = run_gpu(w, engine)
    rcur, rex = run_oracle(w)
    e1 = assert_close(cur, rcur, 1e-4, "C4 current")
    e2 = assert_close(ex, rex, 1e-4, "C4 exit")
    print(f"C4 5 RT engine {engine}: rel L2 current {e1:.3e} exit {e2:.3e}")


def _slots(o):
    """co-resident work slots (clusters / CTAs) the next roundtrips call deals its work to"""
    torch, P = _gpu()
    return int(P.opo_get_info(o._h, P.INFO_SLOTS))


def _fields(o, which, n_fields):
    torch, P = _gpu()
    return np.stack([o.get_fields(x, which).cpu().numpy().astype(np.complex128) for x in range(n_fields)], axis=1)


@pytest.mark.parametrize("engine_name", ["auto", "resident"])
def test_config4_full_batch_in_bench_launch_configuration(engine_name):
    """All 256 instances of C4 in ONE launch -- the configuration bench.py times (AUTO: the solo engine, 148 CTAs looping
    over 1.73 waves of instances; the cluster engine: 45 clusters, 5.7 waves) -- compared on sampled instances the oracle can
    compute one by one: first and last instance of the first wave, first of the second wave, one in the middle, the last."""
    import os
    import oracle
    torch, P = _gpu()
    w = W.config4().truncated(2)
    o = P.from_workload(w, engine=P.ENGINE_AUTO if engine_name == "auto" else P.ENGINE_RESIDENT)
    assert o.engine == (P.ENGINE_SOLO if engine_name == "auto" else P.ENGINE_RESIDENT)
    slots = _slots(o)
    assert 1 < slots < w.batch
    o.roundtrips(w.n_roundtrips)
    o.sync()
    sample = sorted({0, slots - 1, slots, 137, min(5 * slots, w.batch - 2), w.batch - 1})
    cur = _fields(o, P.WHICH_CURRENT, w.n_fields)[sample]
    ex = _fields(o, P.WHICH_EXIT, w.n_fields)[sample]
    o.check_finite()
    o.close()
    ref = oracle.run_workload(w, instances=sample, threads=min(len(sample), os.cpu_count() or 1))
    e1 = assert_close(cur, ref["current"], 1e-4, "C4 full batch current")
    e2 = assert_close(ex, ref["exit"], 1e-4, "C4 full batch exit")
    print(f"C4 full batch ({engine_name}, {slots} slots), 2 RT, sampled {sample}: rel L2 current {e1:.3e} exit {e2:.3e}")


def _split_instances(batch, steps, slots):
    """instances cut by a range boundary of the round-trip split schedule (batch x steps units in `slots` equal ranges)"""
    quota = -(-batch * steps // slots)
    cut = set()
    for c in range(1, slots):
        u = c * quota
        if u < batch * steps and u % steps != 0:
            cut.add(u // steps)
    return sorted(cut)


@pytest.mark.parametrize("engine_name", ["auto", "resident"])
def test_config4_full_batch_with_round_trip_split_schedule(engine_name):
    """256 instances are not a whole number of waves of clusters / CTAs, so the on-chip engines deal round trips, not
    instances: an instance cut by a range boundary runs its first round trips on one cluster and the rest on the next,
    handed over through HBM and a release / acquire flag.  Sampled instances, split and unsplit (derived from the number
    of slots the library reports), against the oracle; and the result must not depend on the schedule: one launch per
    round trip (no split possible) gives the same fields to rounding."""
    import os
    import oracle
    torch, P = _gpu()
    w = W.config4().truncated(5)
    engine = P.ENGINE_AUTO if engine_name == "auto" else P.ENGINE_RESIDENT
    o = P.from_workload(w, engine=engine)
    assert o.engine == (P.ENGINE_SOLO if engine_name == "auto" else P.ENGINE_RESIDENT)
    slots = _slots(o)
    cut = _split_instances(w.batch, 5, slots)
    assert len(cut) >= 3, "the schedule must cut instances, else the test shows nothing"
    o.roundtrips(5)
    o.sync()
    o.check_finite()
    sample = sorted(set([0, 137, w.batch - 1] + cut[:2] + cut[-2:]))
    cur = _fields(o, P.WHICH_CURRENT, w.n_fields)
    ex = _fields(o, P.WHICH_EXIT, w.n_fields)
    o.close()
    ref = oracle.run_workload(w, instances=sample, threads=min(len(sample), os.cpu_count() or 1))
    e1 = assert_close(cur[sample], ref["current"], 1e-4, "C4 split schedule current")
    e2 = assert_close(ex[sample], ref["exit"], 1e-4, "C4 split schedule exit")
    o = P.from_workload(w, engine=engine)
    for _ in range(5):
        o.roundtrips(1)
    o.sync()
    cur1 = _fields(o, P.WHICH_CURRENT, w.n_fields)
    o.close()
    worst = max(rel_l2(cur[b, x], cur1[b, x]) for b in range(w.batch) for x in range(1, w.n_fields))
    assert worst < 2e-5, worst
    print(f"C4 full batch ({engine_name}, {slots} slots, cut instances {cut[:4]}..), 5 RT, split schedule: rel L2 vs oracle current {e1:.3e} "
          f"exit {e2:.3e}; vs call-by-call {worst:.3e}")


@pytest.mark.parametrize("engine_name", ["solo", "resident"])
@pytest.mark.parametrize("precision,log2_n,n_fields,dk,eom,per_inst", [
    ("c64", 13, 3, 25.0, False, False),     # two CTAs per SM (cluster engine), split
    ("c64", 12, 2, 0.0, False, True),       # dk = 0 kernel variant, F = 2, per-instance boundary tables
    ("c64", 10, 3, -30.0, True, False),     # modulator inside the split launch, small N (cluster-barrier path)
    ("c128", 11, 3, 12.0, False, True),     # complex128
    ("c128", 13, 2, 0.0, True, False)])
def test_large_batch_split_and_unsplit(precision, log2_n, n_fields, dk, eom, per_inst, engine_name):
    """Batches much larger than the number of co-resident clusters / CTAs at N <= 2^13 (several CTAs per SM), for the
    combinations the C4 tests do not reach: F = 2 and 3, both precisions, dk = 0 and != 0, a modulator, per-instance
    delta_T (boundary tables with an instance stride).  One launch for all round trips (split schedule when the batch
    is not a whole number of waves) against the oracle on sampled instances, and against one launch per round trip
    (never split) on the full batch."""
    import os
    import oracle
    torch, P = _gpu()
    engine = P.ENGINE_SOLO if engine_name == "solo" else P.ENGINE_RESIDENT
    nrt = 3
    probe = small_workload(log2_n, n_fields, precision, nz=3, batch=1, dk=dk, strong=False)
    _engine_or_skip(probe, engine)
    o = P.from_workload(probe, engine=engine)
    slots1 = _slots(o)            # = 1 for batch 1; the device-wide number comes from a big batch below
    o.close()
    batch = 700 if log2_n <= 11 else 331
    w = small_workload(log2_n, n_fields, precision, nz=3, batch=batch, dk=dk, gdd_dt2=-1.1 if per_inst else 0.0, drad=0.3, strong=False)
    if dk == 0.0:
        w.dk_per_m = np.zeros(batch)
    if per_inst:
        w.delta_T_signal_s = np.linspace(-2.0, 2.0, batch) * w.dt
    if eom:
        w.eom_beta_rad = [0.0, 0.8, 0.0][:n_fields] + [0.0] * (3 - n_fields)
        w.eom_f_hz = [0.0, 2.0 / w.window_s, 0.0]
    w.n_roundtrips = nrt
    o = P.from_workload(w, engine=engine)
    assert o.engine == engine
    slots = _slots(o)
    cut = _split_instances(batch, nrt, slots) if batch % slots else []
    o.roundtrips(nrt)
    o.sync()
    o.check_finite()
    cur = _fields(o, P.WHICH_CURRENT, n_fields)
    ex = _fields(o, P.WHICH_EXIT, n_fields)
    o.close()
    sample = sorted(set([0, min(slots, batch - 1), batch // 2, batch - 1] + cut[:2] + cut[-1:]))
    ref = oracle.run_workload(w, instances=sample, threads=min(len(sample), os.cpu_count() or 1))
    tol = TOL[precision] if precision == "c128" else 3e-5
    e1 = assert_close(cur[sample], ref["current"], tol, "current")
    e2 = assert_close(ex[sample], ref["exit"], tol, "exit")
    o = P.from_workload(w, engine=engine)
    for _ in range(nrt):
        o.roundtrips(1)
    o.sync()
    cur1 = _fields(o, P.WHICH_CURRENT, n_fields)
    o.close()
    worst = max(rel_l2(cur[b, x], cur1[b, x]) for b in range(batch) for x in range(n_fields) if np.linalg.norm(cur1[b, x]) > 0)
    assert worst < (1e-12 if precision == "c128" else 2e-5), worst
    print(f"batch {batch} x 2^{log2_n} x {n_fields} {precision} ({engine_name}, {slots} slots, {len(cut)} cut instances): vs oracle {e1:.3e} / {e2:.3e}; "
          f"vs call-by-call {worst:.3e}")


@pytest.mark.parametrize("engine_name", ["solo", "resident"])
def test_resident_engine_is_bitwise_reproducible(engine_name):
    """The on-chip kernels synchronise with class-granular mbarriers instead of block / cluster barriers; a missing
    dependency would be a data race, and a race shows up as run-to-run differences.  Two runs of the full C4 batch must
    agree bit for bit; a run split into one call per round trip (un-merged boundary, state through HBM) must agree to
    rounding."""
    torch, P = _gpu()
    w = W.config4().truncated(3)
    engine = P.ENGINE_SOLO if engine_name == "solo" else P.ENGINE_RESIDENT
    outs = []
    for calls in (1, 1, 3):
        o = P.from_workload(w, engine=engine)
        for _ in range(calls):
            o.roundtrips(w.n_roundtrips // calls)
        o.sync()
        outs.append([o.get_fields(x, which).clone() for x in range(w.n_fields) for which in (P.WHICH_CURRENT, P.WHICH_EXIT)])
        o.close()
    for a, b in zip(outs[0], outs[1]):
        assert torch.equal(a.view(torch.float32), b.view(torch.float32)), "two identical launches differ: data race"
    # one launch per round trip takes the un-merged boundary path: equal to rounding, not bit for bit
    for a, b in zip(outs[0], outs[2]):
        d = (a - b).abs().max().item() / a.abs().max().item()
        assert d < 1e-5, d


@pytest.mark.parametrize("engine_idx", ENGINE_IDX)
def test_long_noise_seeded_run_power_and_spectrum(engine_idx):
    """BASELINE.json:north_star, long noise-seeded runs: relative error <= 1e-3 on output signal power and on the power
    spectrum (not phase; reading R21).  A three-wave singly resonant OPO as C1 but N = 2^12, nz = 50, pumped at 6.25x
    threshold from a 1e-2 noise seed, 200 round trips: the signal grows by ~5 orders of magnitude in power and
    saturates (pump depletion 85 %), so 10 000 z-steps of fp32 rounding pass through the gain before they are compared."""
    engine = engines()[engine_idx]
    base = W.config1()
    k = base.kappa()
    log2_n, nz, nrt = 12, 50, 200
    w = W.Workload(
        name="long_sro_2^12", length_m=base.length_m, d_eff_m_per_V=base.d_eff_m_per_V, n_fields=3,
        lambda_m=list(base.lambda_m), n_index=list(base.n_index), beta1_s_per_m=list(base.beta1_s_per_m),
        beta2_s2_per_m=list(base.beta2_s2_per_m), alpha_per_m=[0.0, 0.0, 0.0], ref_field=1, resonant=[0, 1, 0],
        R=[0.0, 0.98, 0.0], delta_rad=[0.0, 0.0, 0.0], delta_T_s=[0.0, 0.0, 0.0], gdd_s2=[0.0, 0.0, 0.0],
        log2_n=log2_n, window_s=base.window_s * (1 << log2_n) / base.n, nz_per_pass=nz, precision="c64", batch=1,
        n_roundtrips=nrt, dk_per_m=np.zeros(1))
    a_th = math.acosh(1.0 / math.sqrt(0.98)) / (math.sqrt(k[1] * k[2]) * w.length_m)     # reading R18 (SRO)
    a_p = 2.5 * a_th                                                                     # 6.25x threshold in power
    w.pump = W._round_to_precision(np.full((1, w.n), a_p, dtype=np.complex128), "c64")
    w.seeds = [None] + [W._round_to_precision(W.complex_gaussian_noise(900 + x, w.n, 1e-2 * a_p)[None, :], "c64") for x in (1, 2)]
    _engine_or_skip(w, engine)
    cur, ex, _ = run_gpu(w, engine)
    if "long" not in _ORACLE_CACHE:
        _ORACLE_CACHE["long"] = run_oracle(w)
    rcur, rex = _ORACLE_CACHE["long"]
    # output signal power (reading R16): (1 - R_s) mean |exit_s|^2 of the last round trip
    p_gpu = (1.0 - 0.98) * np.mean(np.abs(ex[0, 1]) ** 2)
    p_ref = (1.0 - 0.98) * np.mean(np.abs(rex[0, 1]) ** 2)
    assert 1.0 - np.mean(np.abs(rex[0, 0]) ** 2) / a_p ** 2 > 0.5, "the run must have reached saturation, else the test shows nothing"
    err_p = abs(p_gpu - p_ref) / p_ref
    s_gpu = np.abs(np.fft.fft(ex[0, 1])) ** 2
    s_ref = np.abs(np.fft.fft(rex[0, 1])) ** 2
    err_s = rel_l2(s_gpu, s_ref)
    # pump depletion as a second scalar
    d_gpu = 1.0 - np.mean(np.abs(ex[0, 0]) ** 2) / a_p ** 2
    d_ref = 1.0 - np.mean(np.abs(rex[0, 0]) ** 2) / a_p ** 2
    print(f"long run engine {engine}: signal power rel err {err_p:.3e}, power spectrum rel L2 {err_s:.3e}, "
          f"pump depletion {d_gpu:.4f} vs {d_ref:.4f}, field rel L2 {rel_l2(ex[0, 1], rex[0, 1]):.3e}")
    assert err_p <= 1e-3, err_p
    assert err_s <= 1e-3, err_s
    assert abs(d_gpu - d_ref) <= 1e-3


# ---------------------------------------------------------------------------------------------------------
# large-N engine (four-step decomposition, N = 2^15 .. 2^18; complex128 also 2^14): SURVEY 8(a) S7
# ---------------------------------------------------------------------------------------------------------
LARGE_SIZES = [("c64", l) for l in range(15, 19)] + [("c128", l) for l in range(14, 19)]


@pytest.mark.parametrize("precision,log2_n", LARGE_SIZES)
def test_large_frequency_readout_matches_oracle_fft(precision, log2_n):
    import oracle
    torch, P = _gpu()
    w = small_workload(log2_n, 2, precision, batch=2)
    o = P.from_workload(w)
    assert o.engine == P.ENGINE_LARGE
    got = o.get_fields(1, P.WHICH_CURRENT, P.DOMAIN_FREQ).cpu().numpy().astype(np.complex128)
    back = o.get_fields(1, P.WHICH_CURRENT, P.DOMAIN_TIME).cpu().numpy().astype(np.complex128)
    o.close()
    for b in range(2):
        ref = oracle.fft(w.seeds[1][b])
        assert rel_l2(got[b], ref) <= (1e-13 if precision == "c128" else 2e-6)
        assert np.array_equal(back[b], w.seeds[1][b])       # the read-out does not disturb the state


@pytest.mark.parametrize("precision,log2_n,n_fields", [
    ("c64", 15, 3), ("c64", 16, 2), ("c64", 17, 3), ("c64", 18, 2), ("c64", 18, 3),
    ("c128", 14, 3), ("c128", 15, 2), ("c128", 16, 3), ("c128", 17, 2), ("c128", 18, 2)])
def test_large_single_pass_matches_oracle(precision, log2_n, n_fields):
    torch, P = _gpu()
    w = small_workload(log2_n, n_fields, precision, nz=4, dk=35.0, alpha=3.0)
    cur, _, eng = run_gpu(w, P.ENGINE_AUTO, propagate=[1, 3])
    assert eng == P.ENGINE_LARGE
    ref, _ = run_oracle(w, propagate=[4])
    assert_close(cur, ref, TOL[precision] if precision == "c128" else 2e-5, w.name)


@pytest.mark.parametrize("precision,log2_n,n_fields,calls", [
    ("c128", 14, 3, 1), ("c128", 15, 2, 3), ("c64", 15, 3, 1), ("c64", 16, 2, 3)])
def test_large_roundtrips_with_boundary(precision, log2_n, n_fields, calls):
    torch, P = _gpu()
    w = small_workload(log2_n, n_fields, precision, nz=3, batch=3, dk=-20.0, gdd_dt2=-1.7, drad=0.4, strong=False)
    w.delta_T_signal_s = np.array([-2.5, 0.0, 1.25]) * w.dt
    cur, ex, eng = run_gpu(w, P.ENGINE_AUTO, n_roundtrips=3, calls=calls)
    assert eng == P.ENGINE_LARGE
    rcur, rex = run_oracle(w, n_roundtrips=3)
    tol = TOL[precision] if precision == "c128" else 3e-5
    assert_close(cur, rcur, tol, "current")
    assert_close(ex, rex, tol, "exit")


def test_large_boundary_without_transform_and_nonresonant_restart():
    torch, P = _gpu()
    w = small_workload(15, 3, "c128", nz=3, batch=2, dk=10.0, drad=-0.7, strong=False)
    w.resonant = [0, 1, 0]
    cur, ex, _ = run_gpu(w, P.ENGINE_AUTO, n_roundtrips=4)
    rcur, rex = run_oracle(w, n_roundtrips=4)
    assert_close(cur, rcur, 1e-10, "current")
    assert_close(ex, rex, 1e-10, "exit")
    assert np.array_equal(cur[:, 0], w.pump) and np.array_equal(cur[:, 2], w.seeds[2])


def test_config3_one_roundtrip_c64():
    """BASELINE.json configs[3] at its full grid (N = 2^18, nz = 500), one round trip (the oracle needs
    ~20 s for it; 20 round trips are compared against the cached oracle result in
    tests/test_gpu_config_length.py::test_config3_golden_20rt)."""
    torch, P = _gpu()
    w = W.config3().truncated(1)
    cur, ex, eng = run_gpu(w, P.ENGINE_AUTO)
    assert eng == P.ENGINE_LARGE
    rcur, rex = run_oracle(w)
    e1 = assert_close(cur, rcur, 1e-4, "C3 current")
    e2 = assert_close(ex, rex, 1e-4, "C3 exit")
    print(f"C3 1 RT: rel L2 current {e1:.3e} exit {e2:.3e}")


# ---------------------------------------------------------------------------------------------------------
# boundary behaviour of the ABI itself
# ---------------------------------------------------------------------------------------------------------
# ---------------------------------------------------------------------------------------------------------
# intracavity phase modulator (Listing 3)
# ---------------------------------------------------------------------------------------------------------
def _with_eom(w):
    """Modulator on every resonant field: depth ~1 rad, frequency = a few free spectral ranges of the time window
    (the paper: 'on the order of the cavity free-spectral range'), not an integer multiple so nothing is periodic."""
    w.eom_beta_rad = [0.0, 0.0, 0.0]
    w.eom_f_hz = [0.0, 0.0, 0.0]
    for x in range(w.n_fields):
        if w.resonant[x]:
            w.eom_beta_rad[x] = 0.9 + 0.4 * x
            w.eom_f_hz[x] = (2.3 + x) / w.window_s
    return w


@pytest.mark.parametrize("engine_idx", ENGINE_IDX)
@pytest.mark.parametrize("precision,log2_n,n_fields,gdd", [("c128", 10, 2, 0.0), ("c64", 12, 3, 0.0), ("c64", 9, 3, 0.7),
                                                           ("c64", 14, 3, 0.7), ("c128", 8, 3, 0.7)])
def test_eom_roundtrips_match_oracle(precision, log2_n, n_fields, gdd, engine_idx):
    """Round trips with the modulator as last boundary element, with and without the spectral-phase transform in the
    boundary, across a call boundary (3 = 2 + 1 round trips), both engines."""
    engine = engines()[engine_idx]
    w = _with_eom(small_workload(log2_n, n_fields, precision, nz=5, batch=2, dk=11.0, gdd_dt2=gdd, drad=0.3))
    _engine_or_skip(w, engine)
    cur, ex, _ = run_gpu(w, engine, n_roundtrips=3, calls=2)
    rcur, rex = run_oracle(w, n_roundtrips=3)
    e1 = assert_close(cur, rcur, TOL[precision], "EOM current")
    e2 = assert_close(ex, rex, TOL[precision], "EOM exit")
    # the modulator must have done something: without it the result differs at O(1)
    w0 = small_workload(log2_n, n_fields, precision, nz=5, batch=2, dk=11.0, gdd_dt2=gdd, drad=0.3)
    c0, _ = run_oracle(w0, n_roundtrips=3)
    assert rel_l2(c0[0, 1], rcur[0, 1]) > 0.1
    print(f"EOM {precision} 2^{log2_n} F={n_fields} engine {engine}: rel L2 current {e1:.3e} exit {e2:.3e}")


def test_eom_large_engine_matches_oracle():
    w = _with_eom(small_workload(15, 2, "c64", nz=4, batch=1, dk=5.0, gdd_dt2=0.7, drad=0.3))
    torch, P = _gpu()
    cur, ex, eng = run_gpu(w, P.ENGINE_AUTO, n_roundtrips=2)
    assert eng == P.ENGINE_LARGE
    rcur, rex = run_oracle(w, n_roundtrips=2)
    e1 = assert_close(cur, rcur, 1e-4, "EOM large current")
    e2 = assert_close(ex, rex, 1e-4, "EOM large exit")
    print(f"EOM large engine 2^15: rel L2 current {e1:.3e} exit {e2:.3e}")


def test_eom_config1_20_roundtrips_and_abi_errors():
    """C1 (N = 2^14, 100 z-steps) with a modulator on the signal at ~3 free spectral ranges, 20 round trips; the call
    rejects non-resonant fields and beta = 0 removes the modulator again."""
    torch, P = _gpu()
    w = W.config1().truncated(20)
    w.eom_beta_rad = [0.0, 1.2, 0.0]
    w.eom_f_hz = [0.0, 3.0 / w.window_s, 0.0]
    rcur, rex = run_oracle(w)
    for engine, expect in ((P.ENGINE_AUTO, P.ENGINE_WIDE), (P.ENGINE_RESIDENT, P.ENGINE_RESIDENT), (P.ENGINE_SOLO, P.ENGINE_SOLO)):
        cur, ex, eng = run_gpu(w, engine)
        assert eng == expect               # AUTO: one instance goes to the wide engine, modulator or not
        e1 = assert_close(cur, rcur, 1e-4, "C1+EOM current")
        e2 = assert_close(ex, rex, 1e-4, "C1+EOM exit")
        print(f"C1 + EOM, 20 RT, engine {eng}: rel L2 current {e1:.3e} exit {e2:.3e}")
    o = P.from_workload(w)
    with pytest.raises(P.OpoError) as ei:
        o.set_eom(0, 1.0, 1e11)                # the pump is not resonant
    assert ei.value.status == P.ERR_INVALID_ARG
    with pytest.raises(P.OpoError):
        o.set_eom(5, 1.0, 1e11)
    o.set_eom(1, 0.0, 0.0)                      # removed again: plain C1
    o.roundtrips(2)
    o.sync()
    got = o.get_fields(1, P.WHICH_CURRENT).cpu().numpy().astype(np.complex128)
    o.close()
    w2 = W.config1().truncated(2)
    rc2, _ = run_oracle(w2)
    assert rel_l2(got[0], rc2[0, 1]) <= 1e-4


# ---------------------------------------------------------------------------------------------------------
# nanosecond regime: pump train in, round-trip train out
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("engine_idx", ENGINE_IDX)
@pytest.mark.parametrize("precision,log2_n,n_fields", [("c64", 12, 2), ("c128", 9, 3)])
def test_pump_train_matches_oracle_loop(precision, log2_n, n_fields, engine_idx):
    """A pump pulse 6 windows long (Gaussian envelope sampled across the train, as the paper's ns pulse across many
    round trips): round trip m is pumped by slice m; the signal leaving the crystal in every round trip is recorded.
    The oracle side is the definition written out: set the pump slice, one round trip, read the exit field."""
    import oracle
    torch, P = _gpu()
    engine = engines()[engine_idx]
    w = small_workload(log2_n, n_fields, precision, nz=5, batch=2, dk=9.0, gdd_dt2=0.5, drad=0.2)
    _engine_or_skip(w, engine)
    n_rt, n = 6, w.n
    g = np.arange(n_rt * n) / (n_rt * n) - 0.5
    env = np.exp(-(g / 0.22) ** 2) * np.exp(1j * 2.0 * g)                       # long pulse with a slow chirp
    a_p = np.abs(w.pump[0]).max()
    train = W._round_to_precision((a_p * env).reshape(n_rt, n), precision)        # [n_rt][N], same for both instances
    o = P.from_workload(w, engine=engine)
    tt = torch.from_numpy(train).to(o.dtype).cuda()
    out = o.roundtrips_train(tt, out_field=1)
    o.sync()
    got_out = out.cpu().numpy().astype(np.complex128)
    got_cur = np.stack([o.get_fields(x, P.WHICH_CURRENT).cpu().numpy().astype(np.complex128) for x in range(w.n_fields)], axis=1)
    o.close()
    tol = TOL[precision]
    for b in range(w.batch):
        ro = oracle.from_workload(w, b)
        for m in range(n_rt):
            ro.set_field(0, train[m])
            assert ro.roundtrips(1) == 0
            ref = ro.get_field(1, oracle.EXIT)
            assert rel_l2(got_out[m, b], ref) <= tol, (m, b, rel_l2(got_out[m, b], ref))
        for x in range(w.n_fields):
            ref = ro.get_field(x, oracle.CURRENT)
            assert rel_l2(got_cur[b, x], ref) <= tol
    # the pump is re-injected from the last slice
    assert rel_l2(got_cur[0, 0], train[-1]) == 0.0


@pytest.mark.parametrize("precision,log2_n,n_fields,batch,out_field,idler_resonant,gdd", [
    ("c64", 10, 3, 331, 1, False, 0.5),       # more instances than CTAs and not a multiple: round trips dealt to the CTAs, slices by absolute index
    ("c64", 11, 3, 5, 2, False, 0.0),         # the recorded field is the non-resonant idler; mirror without a transform
    ("c128", 10, 2, 3, 0, False, 0.5),        # the recorded field is the pump itself
    ("c64", 12, 3, 4, 1, True, 0.0)])
def test_pump_train_inside_the_solo_launch(precision, log2_n, n_fields, batch, out_field, idler_resonant, gdd):
    """The solo engine takes the whole train in ONE launch (slices read and exit fields written at the round-trip crossings
    inside the kernel), with a per-instance train.  Reference: the host-sequenced streaming engine driven slice by slice
    (itself checked against the oracle loop above), and the oracle loop on sampled instances."""
    import oracle
    torch, P = _gpu()
    w = small_workload(log2_n, n_fields, precision, nz=4, batch=batch, dk=9.0, gdd_dt2=gdd, drad=0.2, strong=False)
    if n_fields == 3:
        w.resonant = [0, 1, 1 if idler_resonant else 0]
    _engine_or_skip(w, P.ENGINE_SOLO)
    n_rt, n = 5, w.n
    g = np.arange(n_rt * n) / (n_rt * n) - 0.5
    env = np.exp(-(g / 0.22) ** 2) * np.exp(1j * 2.0 * g)
    a_p = np.abs(w.pump[0]).max()
    base = (a_p * env).reshape(n_rt, 1, n)
    train = W._round_to_precision(base * (1.0 + 0.05 * (np.arange(batch) % 9))[None, :, None], precision)      # [n_rt][B][N]
    res = {}
    for engine in (P.ENGINE_SOLO, P.ENGINE_STREAMING):
        o = P.from_workload(w, engine=engine)
        l0 = o.launches
        out = o.roundtrips_train(torch.from_numpy(train).to(o.dtype).cuda(), out_field=out_field)
        o.sync()
        res[engine] = (out.cpu().numpy().astype(np.complex128),
                       np.stack([o.get_fields(x, P.WHICH_CURRENT).cpu().numpy().astype(np.complex128) for x in range(w.n_fields)], axis=1),
                       np.stack([o.get_fields(x, P.WHICH_EXIT).cpu().numpy().astype(np.complex128) for x in range(w.n_fields)], axis=1),
                       o.launches - l0)
        o.close()
    assert res[P.ENGINE_SOLO][3] <= 3, "the solo engine runs the train in one kernel launch (plus the pump broadcast)"
    tol = 1e-12 if precision == "c128" else 2e-5
    for k, what in ((0, "train of exit fields"), (1, "current"), (2, "exit")):
        a, bb = res[P.ENGINE_SOLO][k], res[P.ENGINE_STREAMING][k]
        assert np.isfinite(a).all()
        flat_a, flat_b = a.reshape(-1, n), bb.reshape(-1, n)
        worst = max(rel_l2(flat_a[i], flat_b[i]) for i in range(flat_a.shape[0]) if np.linalg.norm(flat_b[i]) > 0)
        assert worst <= tol, (what, worst)
    for b in sorted({0, batch // 2, batch - 1}):
        ro = oracle.from_workload(w, b)
        for m in range(n_rt):
            ro.set_field(0, train[m, b])
            assert ro.roundtrips(1) == 0
            assert rel_l2(res[P.ENGINE_SOLO][0][m, b], ro.get_field(out_field, oracle.EXIT)) <= TOL[precision]
    assert np.array_equal(res[P.ENGINE_SOLO][1][:, 0], train[-1].astype(np.complex128))      # the pump is re-injected from the last slice


# ---------------------------------------------------------------------------------------------------------
# third-order dispersion (Eq. 5 in the reading R7): tables only
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("engine_idx", ENGINE_IDX)
@pytest.mark.parametrize("precision,log2_n,n_fields", [("c64", 12, 3), ("c128", 10, 2), ("c64", 14, 3)])
def test_third_order_dispersion_matches_oracle(precision, log2_n, n_fields, engine_idx):
    engine = engines()[engine_idx]
    w = small_workload(log2_n, n_fields, precision, nz=5, batch=2, dk=7.0, gdd_dt2=0.5, drad=0.2)
    # beta3 L / 6 * Omega_max^3 of a few radians at the band edge: clearly visible, well resolved
    om_max = math.pi / w.dt
    w.beta3_s3_per_m = [(1.5 + x) * 6.0 * 3.0 / (om_max ** 3 * w.length_m) for x in range(n_fields)] + [0.0] * (3 - n_fields)
    _engine_or_skip(w, engine)
    cur, ex, _ = run_gpu(w, engine, n_roundtrips=2)
    rcur, rex = run_oracle(w, n_roundtrips=2)
    e1 = assert_close(cur, rcur, TOL[precision], "TOD current")
    e2 = assert_close(ex, rex, TOL[precision], "TOD exit")
    w0 = small_workload(log2_n, n_fields, precision, nz=5, batch=2, dk=7.0, gdd_dt2=0.5, drad=0.2)
    c0, _ = run_oracle(w0, n_roundtrips=2)
    assert rel_l2(c0[0, 1], rcur[0, 1]) > 0.05          # the term does something
    print(f"TOD {precision} 2^{log2_n} engine {engine}: rel L2 current {e1:.3e} exit {e2:.3e}")


def test_third_order_dispersion_large_engine():
    torch, P = _gpu()
    w = small_workload(15, 2, "c64", nz=4, batch=1, dk=5.0, gdd_dt2=0.5, drad=0.2)
    om_max = math.pi / w.dt
    w.beta3_s3_per_m = [2.0 * 18.0 / (om_max ** 3 * w.length_m), -1.0 * 18.0 / (om_max ** 3 * w.length_m), 0.0]
    cur, ex, eng = run_gpu(w, P.ENGINE_AUTO, n_roundtrips=2)
    assert eng == P.ENGINE_LARGE
    rcur, rex = run_oracle(w, n_roundtrips=2)
    assert_close(cur, rcur, 1e-4, "TOD large current")
    assert_close(ex, rex, 1e-4, "TOD large exit")


# ---------------------------------------------------------------------------------------------------------
# the paper's own operator order N/2 - L - N/2 (Eq. 10-11)
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("engine_idx", ENGINE_IDX)
@pytest.mark.parametrize("precision,log2_n,n_fields", [("c64", 12, 3), ("c128", 10, 2), ("c64", 14, 3), ("c64", 8, 2), ("c128", 13, 3)])
def test_nln_ordering_matches_oracle(precision, log2_n, n_fields, engine_idx):
    """Partial passes (2 + 3 z-steps), then full round trips with the boundary (spectral phase, mirror, modulator),
    all in the N/2 - L - N/2 order, against the oracle in the same order; the result must differ from the L/2 - N - L/2
    result by more than the tolerance (else the switch would not be tested)."""
    engine = engines()[engine_idx]
    w = _with_eom(small_workload(log2_n, n_fields, precision, nz=5, batch=2, dk=23.0, gdd_dt2=0.6, drad=0.3))
    w.splitting = 1
    _engine_or_skip(w, engine)
    cur, _, _ = run_gpu(w, engine, propagate=[2, 3])
    rcur, _ = run_oracle(w, propagate=[2, 3])
    e0 = assert_close(cur, rcur, TOL[precision], "NLN propagate")
    cur, ex, _ = run_gpu(w, engine, n_roundtrips=3, calls=2)
    rcur, rex = run_oracle(w, n_roundtrips=3)
    e1 = assert_close(cur, rcur, TOL[precision], "NLN current")
    e2 = assert_close(ex, rex, TOL[precision], "NLN exit")
    w.splitting = 0
    c0, _ = run_oracle(w, n_roundtrips=3)
    assert rel_l2(c0[0, 1], rcur[0, 1]) > 20 * TOL[precision]
    print(f"NLN {precision} 2^{log2_n} F={n_fields} engine {engine}: rel L2 propagate {e0:.3e} current {e1:.3e} exit {e2:.3e}")


def test_nln_ordering_config1_and_large_engine():
    torch, P = _gpu()
    w = W.config1().truncated(3)
    w.splitting = 1
    cur, ex, eng = run_gpu(w, P.ENGINE_AUTO)
    assert eng == P.ENGINE_RESIDENT
    rcur, rex = run_oracle(w)
    e1 = assert_close(cur, rcur, 1e-4, "C1 NLN current")
    e2 = assert_close(ex, rex, 1e-4, "C1 NLN exit")
    print(f"C1 in the N/2-L-N/2 order, 3 RT: rel L2 current {e1:.3e} exit {e2:.3e}")
    # large-N engine in the same order, with the boundary transform and the modulator
    wl = _with_eom(small_workload(15, 2, "c64", nz=4, batch=1, dk=9.0, gdd_dt2=0.6, drad=0.3))
    wl.splitting = 1
    cur, _, eng = run_gpu(wl, P.ENGINE_AUTO, propagate=[1, 3])
    assert eng == P.ENGINE_LARGE
    rcur, _ = run_oracle(wl, propagate=[1, 3])
    e0 = assert_close(cur, rcur, 1e-4, "large NLN propagate")
    cur, ex, _ = run_gpu(wl, P.ENGINE_AUTO, n_roundtrips=2)
    rcur, rex = run_oracle(wl, n_roundtrips=2)
    e1 = assert_close(cur, rcur, 1e-4, "large NLN current")
    e2 = assert_close(ex, rex, 1e-4, "large NLN exit")
    print(f"large-N engine in the N/2-L-N/2 order: rel L2 propagate {e0:.3e} current {e1:.3e} exit {e2:.3e}")
    # the splitting can only change at z = 0
    o = P.from_workload(W.config0())
    o.propagate(1)
    with pytest.raises(P.OpoError) as ei:
        P.opo_set_option(o._h, P.OPT_SPLITTING, P.SPLITTING_NLN)
    assert ei.value.status == P.ERR_STATE
    o.close()


# ---------------------------------------------------------------------------------------------------------
# internal baseline: cuFFT + separate elementwise kernels (BASELINE.json north_star item (d))
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision,log2_n,n_fields,splitting", [("c64", 12, 3, 0), ("c128", 10, 2, 0), ("c64", 14, 3, 0), ("c64", 9, 3, 1)])
def test_cufft_baseline_engine_matches_oracle(precision, log2_n, n_fields, splitting):
    torch, P = _gpu()
    w = _with_eom(small_workload(log2_n, n_fields, precision, nz=5, batch=3, dk=13.0, gdd_dt2=0.6, drad=0.3))
    w.delta_T_signal_s = np.array([-2.0, 0.0, 3.0]) * w.dt          # per-instance boundary table
    w.splitting = splitting
    cur, ex, eng = run_gpu(w, P.ENGINE_CUFFT, n_roundtrips=3, calls=2)
    assert eng == P.ENGINE_CUFFT
    rcur, rex = run_oracle(w, n_roundtrips=3)
    e1 = assert_close(cur, rcur, TOL[precision], "cuFFT baseline current")
    e2 = assert_close(ex, rex, TOL[precision], "cuFFT baseline exit")
    print(f"cuFFT baseline {precision} 2^{log2_n}: rel L2 current {e1:.3e} exit {e2:.3e}")


def test_abi_errors_and_state():
    torch, P = _gpu()
    w = small_workload(8, 2, "c64", nz=4)
    o = P.from_workload(w)
    o.propagate(3)
    assert o.z_steps == 3
    with pytest.raises(P.OpoError) as e:
        o.propagate(2)                       # would pass z = L
    assert e.value.status == P.ERR_STATE
    with pytest.raises(P.OpoError) as e:
        o.roundtrips(1)                      # z != 0
    assert e.value.status == P.ERR_STATE
    with pytest.raises(P.OpoError) as e:
        o.set_batch_param(P.PARAM_DK, 0, [1.0, 2.0])     # count != batch
    assert e.value.status == P.ERR_INVALID_ARG
    o.check_finite()
    o.close()
    with pytest.raises(P.OpoError) as e:
        bad = small_workload(16, 2, "c64")
        bad.resonant = [1, 1]               # a resonant pump is not available on the large-N engine
        P.from_workload(bad)
    assert e.value.status == P.ERR_UNSUPPORTED
    for bad_log2 in (3, 19):                 # N outside [2^4, 2^18]
        with pytest.raises(P.OpoError) as e:
            P.Opo(n_fields=2, log2_n=bad_log2, window_s=1e-11, nz_per_pass=4, length_m=5e-3, dk_per_m=0.0, d_eff_m_per_V=14e-12,
                  lambda_m=[532e-9, 1064e-9], n_index=[2.23, 2.16], beta1_s_per_m=[0.0, 0.0], beta2_s2_per_m=[0.0, 0.0],
                  alpha_per_m=[0.0, 0.0], ref_field=1, resonant=[0, 1], R=[0.0, 0.9], delta_rad=[0.0, 0.0], delta_T_s=[0.0, 0.0],
                  gdd_s2=[0.0, 0.0])
        assert e.value.status == P.ERR_INVALID_ARG
    with pytest.raises(P.OpoError) as e:
        bad = small_workload(8, 2, "c64")
        bad.R = [0.0, 1.5]
        P.from_workload(bad)
    assert e.value.status == P.ERR_INVALID_ARG


def test_nonfinite_is_reported_when_dz_too_coarse():
    """too coarse a dz makes the fields blow up to NaN; the ABI reports it."""
    torch, P = _gpu()
    w = small_workload(8, 2, "c64", nz=1)
    w.pump = w.pump * 1e4
    w.length_m *= 50
    o = P.from_workload(w)
    o.roundtrips(30)
    with pytest.raises(P.OpoError) as e:
        o.check_finite()
    assert e.value.status == P.ERR_NONFINITE
    o.close()


def test_host_buffer_calls_match_device_calls():
    torch, P = _gpu()
    w = small_workload(10, 3, "c64", nz=4, batch=2)
    a = P.from_workload(w)
    b = P.from_workload(w, host_inputs=True)
    a.roundtrips(2)
    b.roundtrips(2)
    for x in range(3):
        da = a.get_fields(x).cpu()
        hb = torch.empty((2, w.n), dtype=torch.complex64).pin_memory()
        b.get_fields(x, out=hb)
        assert torch.equal(da, hb)
    a.close()
    b.close()
