"""Pins for the CPU oracle (oracle/opo_oracle.cpp) -- none of them re-uses the oracle's own code.

Each test checks the oracle against something the paper or the mathematics fixes: an O(N^2) DFT, a
library FFT, closed forms, conservation laws, a library ODE integrator, the phases the paper prints.
Numbering P1..P12 follows SURVEY.md section 8(c); citations are PAPER.md lines.
"""
import math
import os

import numpy as np
import pytest

import oracle
from oracle import OracleOpo, CURRENT, EXIT, TIME, FREQ

FS, PS, UM, NM = 1e-15, 1e-12, 1e-6, 1e-9
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_printed_values.txt")


def golden():
    vals = {}
    with open(GOLDEN) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if "=" in line:
                k, v = line.split("=")
                vals[k.strip()] = float(v)
    return vals


def make(n_fields=3, log2_n=8, window_s=10 * PS, nz=20, length=5e-3, dk=0.0, d_eff=14e-12,
         beta1=(0, 0, 0), beta2=(0, 0, 0), resonant=(0, 0, 0), R=(0, 0, 0), delta_rad=(0, 0, 0),
         delta_T=(0, 0, 0), gdd=(0, 0, 0), alpha=(0, 0, 0), use_float=False, ref_field=1,
         lam=None, nidx=None):
    if lam is None:
        lam = [532 * NM, 1000 * NM, 1.0 / (1 / (532 * NM) - 1 / (1000 * NM))] if n_fields == 3 \
            else [532 * NM, 1064 * NM]
    if nidx is None:
        nidx = [2.23, 2.16, 2.15][:n_fields]
    return OracleOpo(n_fields=n_fields, log2_n=log2_n, window_s=window_s, nz_per_pass=nz,
                     length_m=length, dk_per_m=dk, d_eff_m_per_V=d_eff, lambda_m=list(lam),
                     n_index=list(nidx), beta1_s_per_m=list(beta1), beta2_s2_per_m=list(beta2),
                     alpha_per_m=list(alpha), ref_field=ref_field, resonant=list(resonant), R=list(R),
                     delta_rad=list(delta_rad), delta_T_s=list(delta_T), gdd_s2=list(gdd),
                     use_float=use_float)


def rel_l2(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


# ---------------------------------------------------------------------------------------------
# P1  the oracle's own radix-2 FFT
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("n", [2, 4, 8, 16, 64, 256])
def test_p1_fft_matches_naive_dft(n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    k = np.arange(n)
    # X[k] = sum_n x[n] exp(-2 pi i k n / N): forward sign and no normalisation (reading R8)
    W = np.exp(-2j * np.pi * np.outer(k, k) / n)
    assert rel_l2(oracle.fft(x), W @ x) < 1e-13
    # inverse carries 1/N
    assert rel_l2(oracle.fft(x, inverse=True), (np.conj(W) @ x) / n) < 1e-13
    assert rel_l2(oracle.fft(oracle.fft(x), inverse=True), x) < 1e-13


@pytest.mark.parametrize("log2n", [10, 14])
def test_p1_fft_matches_library_and_parseval(log2n):
    n = 1 << log2n
    rng = np.random.default_rng(7)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    X = oracle.fft(x)
    assert rel_l2(X, np.fft.fft(x)) < 1e-13
    assert abs(np.sum(np.abs(X) ** 2) / n - np.sum(np.abs(x) ** 2)) / np.sum(np.abs(x) ** 2) < 1e-13


def test_p1_single_exponential_lands_in_one_bin():
    n, k0 = 128, 37
    x = np.exp(2j * np.pi * k0 * np.arange(n) / n)
    X = oracle.fft(x)
    assert abs(X[k0] - n) < 1e-10
    X[k0] = 0
    assert np.abs(X).max() < 1e-10


def test_get_field_frequency_domain_is_unnormalised_forward_dft():
    o = make(n_fields=2, log2_n=6)
    rng = np.random.default_rng(3)
    a = rng.standard_normal(64) + 1j * rng.standard_normal(64)
    o.set_field(1, a)
    assert rel_l2(o.get_field(1, CURRENT, FREQ), np.fft.fft(a)) < 1e-13


# ---------------------------------------------------------------------------------------------
# P2  Gaussian pulse under GVD, coupling off: closed form derived from Eq. 5's GVD term
#     A(z,t) = T0/sqrt(T0^2 - i b2 z) exp(-t^2 / (2 (T0^2 - i b2 z)))
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("b2_fs2_per_um", [0.35, -0.2])
def test_p2_gaussian_gvd_closed_form(b2_fs2_per_um):
    log2n, T, L = 10, 10 * PS, 5e-3
    n = 1 << log2n
    b2 = b2_fs2_per_um * FS * FS / UM
    T0 = 100 * FS
    tau = (np.arange(n) - n // 2) * (T / n)
    o = make(n_fields=2, log2_n=log2n, window_s=T, nz=20, length=L, d_eff=0.0, beta2=(0.0, b2))
    o.set_field(1, np.exp(-tau ** 2 / (2 * T0 ** 2)).astype(complex))
    assert o.propagate(20) == 0
    q = T0 ** 2 - 1j * b2 * L
    expect = T0 / np.sqrt(q) * np.exp(-tau ** 2 / (2 * q))
    assert rel_l2(o.get_field(1), expect) < 1e-12


# ---------------------------------------------------------------------------------------------
# P3  group-velocity mismatch: Delta beta1 * L = m dt  ==>  circular shift by +m samples
#     (a slower field, larger beta1, arrives later; reading R7)
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("m", [7, -3])
def test_p3_gvm_integer_shift(m):
    log2n, T, L = 8, 10 * PS, 5e-3
    n = 1 << log2n
    dt = T / n
    rng = np.random.default_rng(11)
    a = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    # pump slower than the reference (signal) by m*dt over the crystal
    o = make(n_fields=2, log2_n=log2n, window_s=T, nz=10, length=L, d_eff=0.0,
             beta1=(m * dt / L, 0.0), ref_field=1)
    o.set_field(0, a)
    o.set_field(1, a)
    assert o.propagate(10) == 0
    assert rel_l2(o.get_field(0), np.roll(a, m)) < 1e-12     # pump delayed by m samples
    assert rel_l2(o.get_field(1), a) < 1e-13                 # reference frame: signal does not move


# ---------------------------------------------------------------------------------------------
# P4  undepleted-pump parametric gain, CW, three waves
#     dk = 0 : |A_s(L)|^2/|A_s(0)|^2 = cosh^2(gL),  g = sqrt(k_s k_i)|A_p|
#     dk != 0: 1 + (g/G)^2 sinh^2(G L),  G^2 = g^2 - (dk/2)^2   (sin form when negative)
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("dk", [0.0, 150.0, 600.0])
def test_p4_undepleted_gain(dk):
    L, nz = 5e-3, 200
    o = make(n_fields=3, log2_n=4, nz=nz, length=L, dk=dk)
    ks, ki = o.kappa(1), o.kappa(2)
    Ap = 0.3 / (math.sqrt(ks * ki) * L) * 1000.0 / 1000.0      # g L = 0.3 ... scaled below
    Ap = 1.2 / (math.sqrt(ks * ki) * L)                        # g L = 1.2
    g = math.sqrt(ks * ki) * Ap
    a0 = 1e-9 * Ap                                             # depletion ~ 1e-18
    n = 16
    o.set_field(0, np.full(n, Ap, complex))
    o.set_field(1, np.full(n, a0 * np.exp(0.3j), complex))
    o.set_field(2, np.zeros(n, complex))
    assert o.propagate(nz) == 0
    gain = np.abs(o.get_field(1)[0]) ** 2 / a0 ** 2
    G2 = g * g - (dk / 2) ** 2
    if G2 > 0:
        G = math.sqrt(G2)
        expect = 1 + (g / G) ** 2 * math.sinh(G * L) ** 2
    else:
        G = math.sqrt(-G2)
        expect = 1 + (g / G) ** 2 * math.sin(G * L) ** 2
    assert abs(gain / expect - 1) < 1e-8
    # idler generated with |A_i|^2/k_i = (|A_s|^2 - |A_s0|^2)/k_s  (Manley-Rowe)
    ai2 = np.abs(o.get_field(2)[0]) ** 2
    assert abs(ai2 / ki / ((gain - 1) * a0 ** 2 / ks) - 1) < 1e-8


# ---------------------------------------------------------------------------------------------
# P5  degenerate OPO, real positive CW pump: a seed at phase pi/4 (or -3pi/4) is amplified by
#     e^{2gL} in power, a seed at -pi/4 is de-amplified by e^{-2gL}; g = k_s |A_p|.
#     The two amplified phases are the ones the paper prints.
# ---------------------------------------------------------------------------------------------

def test_p5_degenerate_phase_sensitive_gain_matches_printed_phases():
    gv = golden()
    L, nz = 5e-3, 200
    o = make(n_fields=2, log2_n=4)
    ks = o.kappa(1)
    Ap = 0.8 / (ks * L)
    g = ks * Ap
    for phase_over_pi, sign in [(gv["degenerate_signal_phase_a_over_pi"], +1),
                                (gv["degenerate_signal_phase_b_over_pi"], +1),
                                (-0.25, -1), (0.75, -1)]:
        o = make(n_fields=2, log2_n=4, nz=nz, length=L)
        a0 = 1e-9 * Ap
        o.set_field(0, np.full(16, Ap, complex))
        o.set_field(1, np.full(16, a0 * np.exp(1j * np.pi * phase_over_pi), complex))
        assert o.propagate(nz) == 0
        out = o.get_field(1)[0]
        gain = abs(out) ** 2 / a0 ** 2
        assert abs(gain / math.exp(sign * 2 * g * L) - 1) < 1e-8
        # the amplified/de-amplified quadratures keep their phase
        assert abs(np.angle(out * np.exp(-1j * np.pi * phase_over_pi))) < 1e-8

    # a seed at an arbitrary phase is pulled towards the printed phases (pi/4 here)
    o = make(n_fields=2, log2_n=4, nz=400, length=4 * L)
    o.set_field(0, np.full(16, Ap, complex))
    o.set_field(1, np.full(16, 1e-12 * Ap * np.exp(0.1j), complex))
    o.propagate(400)
    ph = np.angle(o.get_field(1)[0]) / np.pi
    assert min(abs(ph - gv["degenerate_signal_phase_a_over_pi"]),
               abs(ph - gv["degenerate_signal_phase_b_over_pi"])) < 2e-3


# ---------------------------------------------------------------------------------------------
# P11 pump depletion against the pumping level N = P_p / P_th ("maximum pump depletion is
#     achieved at N = 4").  A plane-wave degenerate CW oscillator, signal resonant with R_s = 0.98 (the value the
#     paper prints), run to its steady state; in the low-loss limit the steady-state depletion of a single-pass
#     pump is 4 (sqrt(N) - 1) / N, which is 1 at N = 4 and smaller on either side.  Pins the whole loop at once:
#     coupling constants (R5's factor 1/2: with kappa_p not halved the maximum moves to another N), the mirror,
#     the re-injection of the pump (R11) and the threshold scaling of the input generator.
# ---------------------------------------------------------------------------------------------

def test_p11_pump_depletion_is_largest_at_the_printed_pumping_level():
    import opo_workloads as W
    gv = golden()
    L, nz, R = 5e-3, 10, gv["mirror_reflectivity_signal"]
    ks = make(n_fields=2, log2_n=4, nz=nz, length=L, resonant=(0, 1), R=(0, R)).kappa(1)
    a_th = W.threshold_amplitude_degenerate(ks, L, R)
    levels = [3.0, 3.5, 4.0, 4.5, 5.0, 6.25]
    depletion = []
    for N in levels:
        o = make(n_fields=2, log2_n=4, nz=nz, length=L, resonant=(0, 1), R=(0, R))
        a_p = math.sqrt(N) * a_th
        o.set_field(0, np.full(16, a_p, complex))
        o.set_field(1, np.full(16, 1e-3 * a_p * np.exp(1j * np.pi * gv["degenerate_signal_phase_a_over_pi"]), complex))
        assert o.roundtrips(2000) == 0
        d1 = 1 - np.mean(np.abs(o.get_field(0, EXIT)) ** 2) / a_p ** 2
        assert o.roundtrips(200) == 0
        d2 = 1 - np.mean(np.abs(o.get_field(0, EXIT)) ** 2) / a_p ** 2
        assert abs(d2 - d1) < 1e-5                       # steady state
        assert abs(d2 - 4 * (math.sqrt(N) - 1) / N) < 2e-3
        depletion.append(d2)
    assert levels[int(np.argmax(depletion))] == gv["pump_depletion_max_at_pumping_level"]
    assert max(depletion) > 0.9999


# ---------------------------------------------------------------------------------------------
# P6  Manley-Rowe and total energy through a lossless crystal (omega_p = omega_s + omega_i,
#     PAPER.md:L80).  The linear half-steps are unitary, so the drift is RK4's: ~h^4.
# ---------------------------------------------------------------------------------------------

def _invariants(o, F):
    k = [o.kappa(x) for x in range(F)]
    P = [np.sum(np.abs(o.get_field(x)) ** 2) for x in range(F)]
    if F == 3:
        return (P[0] / k[0] + P[1] / k[1], P[1] / k[1] - P[2] / k[2],
                P[0] / k[0] + P[2] / k[2])
    # degenerate (reading R5): photon flux |A_p|^2/(k_p/2) ... 2 signal photons per pump photon
    return (2 * P[0] / k[0] + P[1] / k[1],)


@pytest.mark.parametrize("F", [3, 2])
def test_p6_manley_rowe_and_energy(F):
    log2n, L = 7, 5e-3
    n = 1 << log2n
    rng = np.random.default_rng(5)

    def run(nz):
        o = make(n_fields=F, log2_n=log2n, nz=nz, length=L, dk=80.0,
                 beta1=(0.3 * FS / UM, 0.0, -0.17 * FS / UM)[:F] + (0,) * (3 - F),
                 beta2=(0.35 * FS * FS / UM, 0.1 * FS * FS / UM, 0.05 * FS * FS / UM))
        ks = o.kappa(1)
        amp = 1.5 / (ks * L)                    # strong coupling: k A L ~ 1.5, heavy depletion
        rs = np.random.default_rng(5)
        for x in range(F):
            o.set_field(x, amp * (0.6 + 0.4 * (rs.standard_normal(n) + 1j * rs.standard_normal(n))))
        i0 = _invariants(o, F)
        nidx = [2.23, 2.16, 2.15][:F]
        e0 = sum(nidx[x] * np.sum(np.abs(o.get_field(x)) ** 2) for x in range(F))
        p0 = np.sum(np.abs(o.get_field(0)) ** 2)
        assert o.propagate(nz) == 0
        i1 = _invariants(o, F)
        e1 = sum(nidx[x] * np.sum(np.abs(o.get_field(x)) ** 2) for x in range(F))
        p1 = np.sum(np.abs(o.get_field(0)) ** 2)
        assert abs(p1 / p0 - 1) > 0.05          # the pump really exchanged energy
        scale = abs(i0[0])
        return max(abs(a - b) / scale for a, b in zip(i0, i1)), abs(e1 - e0) / e0

    # (the summed drift changes sign at coarse h, so the ratio is taken in the asymptotic range)
    d1, e1 = run(160)
    d2, e2 = run(320)
    # total energy sum n_x |A_x|^2 (F = 2: conserved only with the 1/2 of reading R5, because
    # n_p (k_p/2) = n_s k_s when lambda_s = 2 lambda_p)
    assert d1 < 1e-9 and e1 < 1e-9
    assert 8 < d1 / d2 < 32                    # ~ h^4
    assert 8 < e1 / e2 < 32


# ---------------------------------------------------------------------------------------------
# P7  strongly depleted closed form (second-harmonic direction of the two-wave system):
#     A_p(0) = 0, A_s(0) = a, dk = 0, no dispersion:
#     |A_s(L)|^2 = a^2 sech^2(G L), |A_p(L)|^2 = (k_p/(2k_s)) a^2 tanh^2(G L), G = a sqrt(k_p k_s/2)
# ---------------------------------------------------------------------------------------------

def test_p7_depleted_shg_closed_form():
    L, nz = 5e-3, 400
    o = make(n_fields=2, log2_n=4, nz=nz, length=L)
    kp, ks = o.kappa(0), o.kappa(1)
    a = 1.3 / (math.sqrt(kp * ks / 2) * L)
    G = a * math.sqrt(kp * ks / 2)
    o.set_field(0, np.zeros(16, complex))
    o.set_field(1, np.full(16, a * np.exp(0.7j), complex))
    assert o.propagate(nz) == 0
    s2 = abs(o.get_field(1)[0]) ** 2
    p2 = abs(o.get_field(0)[0]) ** 2
    assert abs(s2 / (a * a / math.cosh(G * L) ** 2) - 1) < 1e-9
    assert abs(p2 / (kp / (2 * ks) * a * a * math.tanh(G * L) ** 2) - 1) < 1e-9


# ---------------------------------------------------------------------------------------------
# RK4 + all signs/conjugates/dk direction against a library ODE integrator (CW => the PDE is an ODE)
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("F", [3, 2])
def test_rk4_step_against_library_ode(F):
    from scipy.integrate import solve_ivp
    L, nz, dk = 5e-3, 400, 230.0
    o = make(n_fields=F, log2_n=4, nz=nz, length=L, dk=dk)
    k = [o.kappa(x) for x in range(F)]
    s = 1.1 / (k[1] * L)
    y0 = np.array([s * (0.9 + 0.2j), s * (0.3 - 0.5j), s * (-0.2 + 0.4j)][:F])
    for x in range(F):
        o.set_field(x, np.full(16, y0[x], complex))
    assert o.propagate(nz) == 0

    def f(z, y):
        em, ep = np.exp(-1j * dk * z), np.exp(1j * dk * z)
        if F == 3:
            return [1j * k[0] * y[1] * y[2] * em, 1j * k[1] * y[0] * np.conj(y[2]) * ep,
                    1j * k[2] * y[0] * np.conj(y[1]) * ep]
        return [0.5j * k[0] * y[1] ** 2 * em, 1j * k[1] * y[0] * np.conj(y[1]) * ep]

    sol = solve_ivp(f, (0, L), y0, method="DOP853", rtol=1e-13, atol=1e-13 * s)
    for x in range(F):
        assert abs(o.get_field(x)[0] - sol.y[x, -1]) / s < 1e-9


# ---------------------------------------------------------------------------------------------
# P8  global second-order convergence of the symmetric splitting
# ---------------------------------------------------------------------------------------------

def test_p8_second_order_convergence():
    gv = golden()
    log2n, L = 7, 5e-3
    n = 1 << log2n
    tau = (np.arange(n) - n // 2) * (10 * PS / n)

    def run(nz):
        o = make(n_fields=3, log2_n=log2n, nz=nz, length=L, dk=40.0,
                 beta1=(0.3 * FS / UM, 0.0, -0.2 * FS / UM),
                 beta2=(35 * FS * FS / UM, 12 * FS * FS / UM, 5 * FS * FS / UM))
        ks = o.kappa(1)
        amp = 1.0 / (ks * L)
        o.set_field(0, amp * np.exp(-(tau / (0.8 * PS)) ** 2).astype(complex))
        o.set_field(1, 0.3 * amp * np.exp(-((tau - 0.5 * PS) / (0.6 * PS)) ** 2) * np.exp(2j * np.pi * tau / (3 * PS)))
        o.set_field(2, 0.2 * amp * np.exp(-((tau + 0.4 * PS) / (0.7 * PS)) ** 2).astype(complex))
        assert o.propagate(nz) == 0
        return np.concatenate([o.get_field(x) for x in range(3)])

    ref = run(16 * 32)
    e1 = np.linalg.norm(run(16) - ref)
    e2 = np.linalg.norm(run(32) - ref)
    e3 = np.linalg.norm(run(64) - ref)
    order = gv["symmetrized_ssfm_local_error_order"] - 1
    assert abs(e1 / e2 - 2 ** order) < 0.1
    assert abs(e2 / e3 - 2 ** order) < 0.1


# ---------------------------------------------------------------------------------------------
# P9  cold cavity (pump = 0): after m round trips
#     A~_s^(m)[k] = A~_s^(0)[k] * ( sqrt(R) e^{i delta} G_s[k] e^{i D_s(Omega_k) L} )^m
# ---------------------------------------------------------------------------------------------

def test_p9_cold_cavity_closed_form():
    log2n, T, L, nz, m = 8, 10 * PS, 5e-3, 10, 7
    n = 1 << log2n
    dt = T / n
    b1s, b2s = 0.02 * FS / UM, 0.4 * FS * FS / UM
    R, delta, gdd, dT = 0.9, 0.37, -900 * FS * FS, 13 * FS
    o = make(n_fields=3, log2_n=log2n, window_s=T, nz=nz, length=L, ref_field=0,
             beta1=(0.0, b1s, 0.0), beta2=(0.0, b2s, 0.0), resonant=(0, 1, 0), R=(0, R, 0),
             delta_rad=(0, delta, 0), delta_T=(0, dT, 0), gdd=(0, gdd, 0))
    rng = np.random.default_rng(2)
    a = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    o.set_field(0, np.zeros(n, complex))
    o.set_field(1, a)
    o.set_field(2, np.zeros(n, complex))
    assert o.roundtrips(m) == 0
    kk = np.fft.fftfreq(n, d=1.0 / n)               # natural order, Nyquist negative (R9)
    om = 2 * np.pi * kk / (n * dt)
    per_trip = math.sqrt(R) * np.exp(1j * delta) * np.exp(1j * (gdd / 2) * om ** 2 - 1j * om * dT) \
        * np.exp(1j * (-b1s * om + b2s / 2 * om ** 2) * L)
    expect = np.fft.ifft(np.fft.fft(a) * per_trip ** m)
    assert rel_l2(o.get_field(1), expect) < 1e-11
    # exit field = pre-mirror field of the last pass
    expect_exit = np.fft.ifft(np.fft.fft(a) * per_trip ** (m - 1) * np.exp(1j * (-b1s * om + b2s / 2 * om ** 2) * L))
    assert rel_l2(o.get_field(1, EXIT), expect_exit) < 1e-11
    # non-resonant fields restart from their stored input (R11, R12)
    assert np.abs(o.get_field(0)).max() == 0 and np.abs(o.get_field(2)).max() == 0


def test_p9_boundary_signs_gdd_compensates_gvd_and_detuning_delays():
    """Independent sign pins for the boundary: GDD = -beta2 L undoes the crystal's GVD (same sign
    convention, reading R14); a positive Delta T = m dt delays the field by m samples (R13)."""
    log2n, T, L = 8, 10 * PS, 5e-3
    n = 1 << log2n
    dt = T / n
    b2s = 0.4 * FS * FS / UM
    rng = np.random.default_rng(4)
    a = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    o = make(n_fields=2, log2_n=log2n, window_s=T, nz=10, length=L, d_eff=0.0, beta2=(0.0, b2s),
             resonant=(0, 1), R=(0, 1.0), gdd=(0, -b2s * L), delta_T=(0, 5 * dt))
    o.set_field(0, np.zeros(n, complex))
    o.set_field(1, a)
    assert o.roundtrips(1) == 0
    assert rel_l2(o.get_field(1), np.roll(a, 5)) < 1e-12


# ---------------------------------------------------------------------------------------------
# P10  linear-regime growth per round trip of a single-mode seed: R cosh^2(sqrt(X) g_th L) (SRO),
#      R e^{2 sqrt(X) g_th L} (degenerate, amplified quadrature); exactly 1 at X = 1  (R18)
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("X", [1.0, 3.0])
def test_p10_threshold_growth_sro(X):
    from opo_workloads import threshold_amplitude_sro
    L, nz, R = 20e-3, 100, 0.98
    o = make(n_fields=3, log2_n=4, nz=nz, length=L, resonant=(0, 1, 0), R=(0, R, 0))
    ks, ki = o.kappa(1), o.kappa(2)
    a_th = threshold_amplitude_sro(ks, ki, L, R)
    Ap = math.sqrt(X) * a_th
    a0 = 1e-10 * Ap
    o.set_field(0, np.full(16, Ap, complex))
    o.set_field(1, np.full(16, a0, complex))
    o.set_field(2, np.zeros(16, complex))
    trips = 5
    assert o.roundtrips(trips) == 0
    growth = (abs(o.get_field(1)[0]) ** 2 / a0 ** 2) ** (1.0 / trips)
    expect = R * math.cosh(math.sqrt(X) * math.sqrt(ks * ki) * a_th * L) ** 2
    assert abs(growth / expect - 1) < 1e-9
    if X == 1.0:
        assert abs(growth - 1) < 1e-9


@pytest.mark.parametrize("X", [1.0, 2.0])
def test_p10_threshold_growth_degenerate(X):
    from opo_workloads import threshold_amplitude_degenerate
    L, nz, R = 5e-3, 20, 0.98
    o = make(n_fields=2, log2_n=4, nz=nz, length=L, resonant=(0, 1), R=(0, R))
    ks = o.kappa(1)
    a_th = threshold_amplitude_degenerate(ks, L, R)
    Ap = math.sqrt(X) * a_th
    a0 = 1e-10 * Ap
    o.set_field(0, np.full(16, Ap, complex))
    o.set_field(1, np.full(16, a0 * np.exp(0.25j * np.pi), complex))
    trips = 5
    assert o.roundtrips(trips) == 0
    growth = (abs(o.get_field(1)[0]) ** 2 / a0 ** 2) ** (1.0 / trips)
    expect = R * math.exp(2 * math.sqrt(X) * ks * a_th * L)
    assert abs(growth / expect - 1) < 1e-9
    if X == 1.0:
        assert abs(growth - 1) < 1e-9


# ---------------------------------------------------------------------------------------------
# error convention: partial passes accumulate z (R20); roundtrips needs z = 0; no stepping past L
# ---------------------------------------------------------------------------------------------

def test_state_conventions():
    o = make(n_fields=2, log2_n=4, nz=10)
    o.set_field(0, np.ones(16, complex))
    o.set_field(1, np.ones(16, complex))
    assert o.propagate(4) == 0
    assert abs(o.z - 4 * 5e-3 / 10) < 1e-15
    assert o.roundtrips(1) == 5          # STATE: z != 0
    assert o.propagate(7) == 5           # STATE: would pass z = L
    assert o.propagate(6) == 0


def test_dk_phase_continues_across_partial_passes():
    a = make(n_fields=3, log2_n=4, nz=40, dk=300.0)
    b = make(n_fields=3, log2_n=4, nz=40, dk=300.0)
    ks = a.kappa(1)
    s = 1.0 / (ks * 5e-3)
    for o in (a, b):
        o.set_field(0, np.full(16, s, complex))
        o.set_field(1, np.full(16, 0.2 * s, complex))
        o.set_field(2, np.full(16, 0.1j * s, complex))
    a.propagate(40)
    b.propagate(13)
    b.propagate(27)
    for x in range(3):
        assert rel_l2(b.get_field(x), a.get_field(x)) < 1e-14


def test_nan_when_dz_too_coarse():
    """'when the value of dz is not small enough ... the code returns NaN values'."""
    o = make(n_fields=2, log2_n=4, nz=1, length=5e-3)
    ks = o.kappa(1)
    o.set_field(0, np.full(16, 1e6 / (ks * 5e-3), complex))     # kappa A_p dz = 1e6 >> 1
    o.set_field(1, np.full(16, 1.0 + 1j, complex))
    for _ in range(60):
        o.propagate(1)
        o2 = o.get_field(1)
        if not np.all(np.isfinite(o2)):
            break
        # restart the pass to keep stepping (z is reset by a boundary with nothing resonant)
        o.roundtrips(0)
        break
    # one RK4 step with |kappa A dz| = 1e6 amplifies by ~ (1e6)^4/24 per step; 60 steps overflow fp64
    o = make(n_fields=2, log2_n=4, nz=60, length=5e-3 * 60)
    o.set_field(0, np.full(16, 1e6 / (ks * 5e-3), complex))
    o.set_field(1, np.full(16, 1.0 + 1j, complex))
    o.propagate(60)
    assert not np.all(np.isfinite(o.get_field(1)))


# ---------------------------------------------------------------------------------------------
# P13  intracavity EOM (Listing 3)
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("beta,q", [(0.8, 1), (2.4048, 3), (-1.3, 2)])
def test_p13_eom_sidebands_are_bessel_functions(beta, q):
    """A CW field through a cold cavity with only the modulator: exp(i beta sin(theta)) = sum_m J_m(beta)
    e^{i m theta} (Jacobi-Anger).  With f_pm = q / T_win, theta_n = 2 pi q (n - N/2) / N, so bin m q of the
    unnormalised forward DFT holds N J_m(beta) (-1)^{m q} and every other bin is empty.  Pins the form of the
    modulator, the sign of beta, the time origin (R19) and the 2 pi in the argument."""
    from scipy.special import jv
    log2n, T = 8, 10 * PS
    n = 1 << log2n
    o = make(n_fields=3, log2_n=log2n, window_s=T, nz=4, length=5e-3, resonant=(0, 1, 0), R=(0, 1.0, 0))
    o.set_eom(1, beta, q / T)
    o.set_field(0, np.zeros(n, complex))
    o.set_field(1, np.ones(n, complex))
    o.set_field(2, np.zeros(n, complex))
    assert o.roundtrips(1) == 0
    spec = o.get_field(1, CURRENT, FREQ)
    expect = np.zeros(n, complex)
    for m in range(-40, 41):
        expect[(m * q) % n] += n * jv(m, beta) * (-1.0) ** (m * q)
    assert np.abs(spec - expect).max() < 1e-10 * n
    # beta = 2.4048 is the first zero of J_0: the carrier is (almost) extinguished
    if abs(beta - 2.4048) < 1e-9:
        assert abs(spec[0]) < 1e-4 * n
    # a pure phase modulation leaves |A| untouched
    assert np.abs(np.abs(o.get_field(1)) - 1.0).max() < 1e-13


def test_p13_eom_acts_after_gdd_and_mirror_on_resonant_fields_only():
    """Order of the boundary elements (Listing 3; R15): spectral phase, mirror, then the modulator, which
    does not commute with the spectral phase.  Checked against the same chain written with the library FFT; the
    swapped order must differ.  A non-resonant field ignores its modulator (it restarts from S_x)."""
    log2n, T = 8, 10 * PS
    n = 1 << log2n
    dt = T / n
    R, delta, gdd, dT, beta, f = 0.81, 0.2, -4000 * FS * FS, 25 * FS, 1.1, 3 / T
    o = make(n_fields=3, log2_n=log2n, window_s=T, nz=4, length=5e-3, resonant=(0, 1, 0), R=(0, R, 0),
             delta_rad=(0, delta, 0), delta_T=(0, dT, 0), gdd=(0, gdd, 0))
    o.set_eom(1, beta, f)
    o.set_eom(2, 0.7, f)            # idler is not resonant: no effect
    rng = np.random.default_rng(5)
    a = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    s2 = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    o.set_field(0, np.zeros(n, complex))
    o.set_field(1, a)
    o.set_field(2, s2)
    assert o.roundtrips(1) == 0
    om = 2 * np.pi * np.fft.fftfreq(n, d=1.0 / n) / (n * dt)
    G = np.exp(1j * (gdd / 2) * om ** 2 - 1j * om * dT)
    tau = (np.arange(n) - n // 2) * dt
    E = np.exp(1j * beta * np.sin(2 * np.pi * f * tau))
    m = math.sqrt(R) * np.exp(1j * delta)
    right = m * np.fft.ifft(G * np.fft.fft(a)) * E
    wrong = m * np.fft.ifft(G * np.fft.fft(a * E))
    got = o.get_field(1)
    assert rel_l2(got, right) < 1e-12
    assert rel_l2(got, wrong) > 1e-2
    assert rel_l2(o.get_field(2), s2) < 1e-15      # pump = 0, so the idler seed passes unchanged and is re-injected
    # the exit field is taken before the boundary: no modulator on it
    assert rel_l2(o.get_field(1, EXIT), a) < 1e-12


# ---------------------------------------------------------------------------------------------
# P14  third-order dispersion (Eq. 5 in the reading R7)
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("b3_fs3_per_um,w0", [(40.0, 0.0), (-25.0, 0.12e15), (60.0, -0.05e15)])
def test_p14_tod_group_delay_of_an_offset_gaussian(b3_fs3_per_um, w0):
    """Pure third-order dispersion, no coupling.  For dA/dz = +(beta3/6) d^3A/dtau^3 a spectral component at physical
    offset w (field ~ e^{-i w tau}) acquires the phase -(beta3/6)(-w)^3 ... in the bin convention of R8 the multiplier is
    exp(-i (beta3/6) Omega_k^3 z).  The centroid of |A|^2 moves by the power-weighted mean group delay, in closed form
    for a Gaussian spectrum centred on Omega_0 with power-spectrum variance s^2:  <tau> = (beta3 z / 2)(Omega_0^2 + s^2),
    independent of the sign of Omega_0 (even in Omega) and odd in beta3.  Pins sign, the 1/6 and the Omega^3."""
    log2n, T, L, nz = 10, 20 * PS, 5e-3, 10
    n = 1 << log2n
    dt = T / n
    b3 = b3_fs3_per_um * FS ** 3 / UM
    T0 = 150 * FS
    o = make(n_fields=2, log2_n=log2n, window_s=T, nz=nz, length=L, d_eff=0.0)
    o.set_beta3(1, b3)
    tau = (np.arange(n) - n // 2) * dt
    # carrier offset chosen on the bin grid so that the field is periodic on the window
    kbin = round(w0 * n * dt / (2 * np.pi))
    om0 = 2 * np.pi * kbin / (n * dt)
    a = np.exp(-tau ** 2 / (2 * T0 ** 2)) * np.exp(1j * om0 * tau)     # spectrum centred on bin +kbin (Omega_k = om0)
    o.set_field(0, np.zeros(n, complex))
    o.set_field(1, a)
    assert o.propagate(nz) == 0
    out = o.get_field(1)
    p = np.abs(out) ** 2
    centroid = np.sum(tau * p) / np.sum(p)
    s2 = 1.0 / (2 * T0 ** 2)                       # variance of |A~|^2 for A = exp(-tau^2 / 2 T0^2)
    # group delay under R8: multiplier exp(i D z), D = -(beta3/6) Omega^3, delay = -dD/dOmega ... z = (beta3/2) Omega^2 z
    expect = 0.5 * b3 * L * (om0 ** 2 + s2)
    assert abs(centroid - expect) < 2e-4 * max(abs(expect), T0), (centroid, expect)
    assert abs(np.sum(p) / np.sum(np.abs(a) ** 2) - 1.0) < 1e-12     # a pure phase: energy conserved
    # exact spectral check against the closed-form multiplier with the library FFT
    om = 2 * np.pi * np.fft.fftfreq(n, d=1.0 / n) / (n * dt)
    ref = np.fft.ifft(np.fft.fft(a) * np.exp(-1j * (b3 / 6.0) * om ** 3 * L))
    assert rel_l2(out, ref) < 1e-11


# ---------------------------------------------------------------------------------------------
# P15  the paper's own operator order N/2 - L - N/2 (Eq. 10-11)
# ---------------------------------------------------------------------------------------------

def _p15_run(nz, splitting, beta=True, d_eff=14e-12):
    log2n, L = 7, 5e-3
    n = 1 << log2n
    tau = (np.arange(n) - n // 2) * (10 * PS / n)
    o = make(n_fields=3, log2_n=log2n, nz=nz, length=L, dk=40.0, d_eff=d_eff,
             beta1=(0.3 * FS / UM, 0.0, -0.2 * FS / UM) if beta else (0, 0, 0),
             beta2=(35 * FS * FS / UM, 12 * FS * FS / UM, 5 * FS * FS / UM) if beta else (0, 0, 0))
    o.set_splitting(splitting)
    ks = 2 * np.pi * 14e-12 / (2.16 * 1000 * NM)
    amp = 1.0 / (ks * L)
    o.set_field(0, amp * np.exp(-(tau / (0.8 * PS)) ** 2).astype(complex))
    o.set_field(1, 0.3 * amp * np.exp(-((tau - 0.5 * PS) / (0.6 * PS)) ** 2) * np.exp(2j * np.pi * tau / (3 * PS)))
    o.set_field(2, 0.2 * amp * np.exp(-((tau + 0.4 * PS) / (0.7 * PS)) ** 2).astype(complex))
    assert o.propagate(nz) == 0
    return np.concatenate([o.get_field(x) for x in range(3)])


def test_p15_nln_ordering_is_second_order_and_agrees_with_lnl_to_second_order():
    gv = golden()
    order = gv["symmetrized_ssfm_local_error_order"] - 1            # printed: local error O(dz^3) (L131)
    ref = _p15_run(16 * 32, 1)
    e = [np.linalg.norm(_p15_run(nz, 1) - ref) for nz in (16, 32, 64)]
    assert abs(e[0] / e[1] - 2 ** order) < 0.1 and abs(e[1] / e[2] - 2 ** order) < 0.1
    # "equivalent to its counterpart L/2 - N - L/2, since both lead to the same solution" (L133): same limit, and
    # the two orders differ from each other by O(h^2) -- not bit for bit
    d = [np.linalg.norm(_p15_run(nz, 1) - _p15_run(nz, 0)) for nz in (16, 32, 64)]
    assert d[0] > 0 and abs(d[0] / d[1] - 4.0) < 0.2 and abs(d[1] / d[2] - 4.0) < 0.2
    d512 = np.linalg.norm(ref - _p15_run(16 * 32, 0))
    assert abs(d512 / (d[2] / 64.0) - 1.0) < 0.05               # still falling as h^2: the limits coincide


def test_p15_nln_ordering_special_cases():
    # no coupling: both orders are the same product of linear multipliers, H.H = exp(D h)
    a = _p15_run(10, 1, d_eff=0.0)
    b = _p15_run(10, 0, d_eff=0.0)
    assert rel_l2(a, b) < 1e-13
    # no dispersion: N/2 - L - N/2 is plain RK4 with step h/2 (2 nz steps), L/2 - N - L/2 is RK4 with step h:
    # the N/2-L-N/2 run with nz steps must equal the L/2-N-L/2 run with 2 nz steps
    a = _p15_run(10, 1, beta=False)
    b = _p15_run(20, 0, beta=False)
    assert rel_l2(a, b) < 1e-13
    assert rel_l2(a, _p15_run(10, 0, beta=False)) > 1e-9          # and not the h-step result


# ---------------------------------------------------------------------------------------------
# P16  loss: Eq. 5 carries -(alpha_x/2) A_x on the AMPLITUDE, so power falls as e^{-alpha_x z}
# ---------------------------------------------------------------------------------------------

def test_p16_loss_is_alpha_over_two_on_the_amplitude():
    """Coupling off, dispersion on, alpha_x different per field: sum|A_x(L)|^2 / sum|A_x(0)|^2 = exp(-alpha_x L)
    (alpha is the POWER attenuation: the amplitude factor is exp(-alpha_x L / 2)), and the loss is a pure scale:
    the output equals the lossless output times exp(-alpha_x L / 2), spectral phase untouched.  A factor alpha
    instead of alpha/2 (or a dropped term) fails both."""
    log2n, T, L, nz = 8, 10 * PS, 5e-3, 20
    n = 1 << log2n
    alpha = (37.0, 110.0, 5.5)            # 1/m; alpha L = 0.185, 0.55, 0.0275
    b1 = (0.3 * FS / UM, 0.0, -0.17 * FS / UM)
    b2 = (0.35 * FS * FS / UM, 0.12 * FS * FS / UM, 0.05 * FS * FS / UM)
    rng = np.random.default_rng(16)
    a = [rng.standard_normal(n) + 1j * rng.standard_normal(n) for _ in range(3)]
    out = {}
    for al in (alpha, (0.0, 0.0, 0.0)):
        o = make(n_fields=3, log2_n=log2n, window_s=T, nz=nz, length=L, d_eff=0.0, beta1=b1, beta2=b2, alpha=al)
        for x in range(3):
            o.set_field(x, a[x])
        assert o.propagate(nz) == 0
        out[al] = [o.get_field(x) for x in range(3)]
    for x in range(3):
        lossy, lossless = out[alpha][x], out[(0.0, 0.0, 0.0)][x]
        p_ratio = np.sum(np.abs(lossy) ** 2) / np.sum(np.abs(a[x]) ** 2)
        assert abs(p_ratio / math.exp(-alpha[x] * L) - 1) < 1e-13
        assert rel_l2(lossy, lossless * math.exp(-0.5 * alpha[x] * L)) < 1e-13
        assert abs(np.sum(np.abs(lossless) ** 2) / np.sum(np.abs(a[x]) ** 2) - 1) < 1e-13   # dispersion alone is unitary
    # a partial pass: z = 7 h
    o = make(n_fields=2, log2_n=log2n, window_s=T, nz=nz, length=L, d_eff=0.0, alpha=(0.0, 64.0))
    o.set_field(1, a[1])
    assert o.propagate(7) == 0
    assert abs(np.sum(np.abs(o.get_field(1)) ** 2) / np.sum(np.abs(a[1]) ** 2) / math.exp(-64.0 * L * 7 / nz) - 1) < 1e-13


def test_p16_loss_enters_the_cold_cavity_round_trip_factor():
    """Cold cavity with loss: per round trip the power falls by R exp(-alpha_s L)."""
    log2n, L, nz, R, al, m = 6, 5e-3, 10, 0.9, 48.0, 5
    n = 1 << log2n
    o = make(n_fields=2, log2_n=log2n, nz=nz, length=L, d_eff=0.0, resonant=(0, 1), R=(0, R), alpha=(0.0, al),
             beta2=(0.0, 0.2 * FS * FS / UM))
    rng = np.random.default_rng(17)
    a = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    o.set_field(0, np.zeros(n, complex))
    o.set_field(1, a)
    assert o.roundtrips(m) == 0
    assert abs(np.sum(np.abs(o.get_field(1)) ** 2) / np.sum(np.abs(a) ** 2) / (R * math.exp(-al * L)) ** m - 1) < 1e-12


# ---------------------------------------------------------------------------------------------
# P17  pump re-injection at the boundary (ReadPump; readings R11, R12): every round trip starts
#      from the stored pump input S_p, whatever the crystal did to the pump in the pass before
# ---------------------------------------------------------------------------------------------

def _mirror(a, R, delta=0.0):
    return math.sqrt(R) * np.exp(1j * delta) * a


def test_p17_depleted_pump_is_replaced_by_the_stored_input_every_round_trip():
    log2n, L, nz, R = 6, 5e-3, 40, 0.7
    n = 1 << log2n
    kw = dict(n_fields=3, log2_n=log2n, nz=nz, length=L, dk=60.0, resonant=(0, 1, 0), R=(0, R, 0),
              beta1=(0.3 * FS / UM, 0.0, -0.17 * FS / UM),
              beta2=(0.35 * FS * FS / UM, 0.12 * FS * FS / UM, 0.05 * FS * FS / UM))
    o = make(**kw)
    ks = o.kappa(1)
    amp = 1.5 / (ks * L)                              # kappa A L ~ 1.5: heavy depletion in a single pass (as in P6)
    rng = np.random.default_rng(170)
    Sp = amp * (0.8 + 0.2 * (rng.standard_normal(n) + 1j * rng.standard_normal(n)))
    Ss = 0.5 * amp * (0.7 + 0.3 * (rng.standard_normal(n) + 1j * rng.standard_normal(n)))
    Si = 0.2 * amp * (rng.standard_normal(n) + 1j * rng.standard_normal(n))
    for x, s in enumerate((Sp, Ss, Si)):
        o.set_field(x, s)
    assert o.roundtrips(1) == 0
    # after the boundary the current pump IS the stored input, bit for bit; the pump that left the crystal is not
    assert np.array_equal(o.get_field(0, CURRENT), Sp)
    ex_p = o.get_field(0, EXIT)
    assert abs(np.sum(np.abs(ex_p) ** 2) / np.sum(np.abs(Sp) ** 2) - 1) > 0.05
    assert rel_l2(ex_p, Sp) > 0.05
    assert np.array_equal(o.get_field(2, CURRENT), Si)              # R12: the non-resonant idler restarts too
    ex_s1 = o.get_field(1, EXIT)
    assert o.roundtrips(1) == 0
    # round trip 2, composed by hand from single passes only: fresh pump, mirrored signal, fresh idler, z = 0
    c = make(**kw)
    c.set_field(0, Sp)
    c.set_field(1, _mirror(ex_s1, R))
    c.set_field(2, Si)
    assert c.propagate(nz) == 0
    for x in range(3):
        assert rel_l2(o.get_field(x, EXIT), c.get_field(x)) < 1e-13
    # ... and NOT what a pass fed with the depleted pump would give
    d = make(**kw)
    d.set_field(0, ex_p)
    d.set_field(1, _mirror(ex_s1, R))
    d.set_field(2, Si)
    assert d.propagate(nz) == 0
    assert rel_l2(o.get_field(1, EXIT), d.get_field(1)) > 1e-2


def test_p17_set_field_input_only_changes_the_next_injection():
    """The stored input can be replaced between round trips (a pump train): the new S_p is what the next
    boundary injects, the current state is untouched."""
    log2n, nz = 5, 10
    n = 1 << log2n
    o = make(n_fields=2, log2_n=log2n, nz=nz, resonant=(0, 1), R=(0, 0.9))
    ks = o.kappa(1)
    amp = 0.7 / (ks * 5e-3)
    o.set_field(0, np.full(n, amp, complex))
    o.set_field(1, np.full(n, 0.3 * amp * np.exp(0.4j), complex))
    new_pump = np.full(n, 0.5 * amp * np.exp(0.2j), complex)
    o.set_field(0, new_pump, which="input")
    assert np.array_equal(o.get_field(0, CURRENT), np.full(n, amp, complex))
    assert o.roundtrips(1) == 0
    assert np.array_equal(o.get_field(0, CURRENT), new_pump)


# ---------------------------------------------------------------------------------------------
# P18  z is measured from the crystal entrance and starts again at 0 in every pass (reading R4): with dk != 0 the
#      phase e^{-/+ i dk z} of Eqs 2-4 must not run on across round trips
# ---------------------------------------------------------------------------------------------

def test_p18_dk_phase_restarts_at_the_crystal_entrance_every_round_trip():
    log2n, L, nz, R, delta, trips = 5, 5e-3, 25, 0.8, 0.3, 3
    n = 1 << log2n
    dk = 2.0 / L                                       # dk L = 2: a phase error of 2 rad per missed reset
    kw = dict(n_fields=2, log2_n=log2n, nz=nz, length=L, dk=dk, resonant=(0, 1), R=(0, R), delta_rad=(0, delta),
              beta1=(0.3 * FS / UM, 0.0), beta2=(0.35 * FS * FS / UM, 0.10 * FS * FS / UM))
    o = make(**kw)
    ks = o.kappa(1)
    amp = 0.9 / (ks * L)                               # degenerate two-wave: the gain depends on the relative phase
    rng = np.random.default_rng(18)
    Sp = amp * (0.9 + 0.1 * (rng.standard_normal(n) + 1j * rng.standard_normal(n)))
    Ss = 0.3 * amp * (rng.standard_normal(n) + 1j * rng.standard_normal(n))
    o.set_field(0, Sp)
    o.set_field(1, Ss)
    assert o.roundtrips(trips) == 0
    assert o.z == 0.0
    # the same three passes on fresh oracles (each starts at z = 0), boundary applied in numpy
    sig = Ss
    for m in range(trips):
        c = make(**kw)
        c.set_field(0, Sp)
        c.set_field(1, sig)
        assert c.propagate(nz) == 0
        ex = [c.get_field(0), c.get_field(1)]
        sig = _mirror(ex[1], R, delta)
    for x in range(2):
        assert rel_l2(o.get_field(x, EXIT), ex[x]) < 1e-13
    assert rel_l2(o.get_field(1, CURRENT), sig) < 1e-13
    # a crystal three times as long walked in three pieces has z running on: must NOT be what roundtrips() does
    kw3 = dict(kw, nz=trips * nz, length=trips * L)
    r = make(**kw3)
    r.set_field(0, Sp)
    r.set_field(1, Ss)
    for m in range(trips):
        assert r.propagate(nz) == 0
        exr = [r.get_field(0), r.get_field(1)]
        r.set_field(0, Sp, which="state")
        r.set_field(1, _mirror(exr[1], R, delta), which="state")
    assert rel_l2(exr[1], ex[1]) > 1e-2
    # three-wave as well (C4 sweeps dk over +-50 1/m for 300 round trips)
    kw = dict(n_fields=3, log2_n=log2n, nz=nz, length=L, dk=-1.3 / L, resonant=(0, 1, 0), R=(0, R, 0))
    o = make(**kw)
    Si = 0.2 * amp * (rng.standard_normal(n) + 1j * rng.standard_normal(n))
    for x, s in enumerate((Sp, Ss, Si)):
        o.set_field(x, s)
    assert o.roundtrips(2) == 0
    sig = Ss
    for m in range(2):
        c = make(**kw)
        for x, s in enumerate((Sp, sig, Si)):
            c.set_field(x, s)
        assert c.propagate(nz) == 0
        ex = [c.get_field(x) for x in range(3)]
        sig = _mirror(ex[1], R)
    for x in range(3):
        assert rel_l2(o.get_field(x, EXIT), ex[x]) < 1e-13


# ---------------------------------------------------------------------------------------------
# P19  resonant pump (reading R24: the paper names triply resonant oscillators, without an
#      injection rule): A_p <- sqrt(R_p) e^{i delta_p} IDFT(G_p DFT(A_p(L))) + sqrt(1 - R_p) S_p at every boundary
# ---------------------------------------------------------------------------------------------

def test_p19_cold_cavity_pump_builds_up_to_the_airy_steady_state():
    """Coupling off (d_eff = 0): the intracavity pump after m boundaries, started from the transmitted input t S_p, is
    the geometric partial sum  t S~[k] (1 - rho_k^{m+1}) / (1 - rho_k),  rho_k = sqrt(R) e^{i delta} G[k] e^{i D(Omega_k) L},
    and converges to the Airy steady state  t S~[k] / (1 - rho_k)  per bin.  On resonance (delta = 0, bin 0) the
    intracavity power is enhanced by (1 - R) / (1 - sqrt(R))^2."""
    log2n, T, L, nz = 7, 10 * PS, 5e-3, 8
    n = 1 << log2n
    dt = T / n
    Rp, delta, gdd, dT = 0.6, 0.4, 300 * FS * FS, -7 * FS
    b1p, b2p = 0.05 * FS / UM, 0.35 * FS * FS / UM
    o = make(n_fields=2, log2_n=log2n, window_s=T, nz=nz, length=L, d_eff=0.0, resonant=(1, 0), R=(Rp, 0),
             delta_rad=(delta, 0), delta_T=(dT, 0), gdd=(gdd, 0), beta1=(b1p, 0.0), beta2=(b2p, 0.0), ref_field=1)
    rng = np.random.default_rng(19)
    S = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    t = math.sqrt(1 - Rp)
    o.set_field(0, S, which="input")
    o.set_field(0, t * S, which="state")
    om = 2 * np.pi * np.fft.fftfreq(n, d=1.0 / n) / (n * dt)
    rho = math.sqrt(Rp) * np.exp(1j * delta) * np.exp(1j * (gdd / 2) * om ** 2 - 1j * om * dT) * np.exp(1j * (-b1p * om + b2p / 2 * om ** 2) * L)
    Sf = np.fft.fft(S)
    done = 0
    for m in (1, 2, 5, 40):
        assert o.roundtrips(m - done) == 0
        done = m
        expect = np.fft.ifft(t * Sf * (1 - rho ** (m + 1)) / (1 - rho))
        assert rel_l2(o.get_field(0), expect) < 1e-12
    assert o.roundtrips(200) == 0                       # 0.6^120 ~ 1e-27: converged
    airy = np.fft.ifft(t * Sf / (1 - rho))
    assert rel_l2(o.get_field(0), airy) < 1e-12
    # on resonance, CW input: power enhancement (1 - R) / (1 - sqrt(R))^2
    o = make(n_fields=2, log2_n=4, nz=4, d_eff=0.0, resonant=(1, 0), R=(Rp, 0))
    o.set_field(0, np.ones(16, complex), which="input")
    o.set_field(0, t * np.ones(16, complex), which="state")
    assert o.roundtrips(300) == 0
    assert abs(abs(o.get_field(0)[0]) ** 2 / ((1 - Rp) / (1 - math.sqrt(Rp)) ** 2) - 1) < 1e-12


def test_p19_pump_input_changed_mid_run_leaves_the_stored_light_alone():
    """Cold cavity again: m1 round trips with input S1, then the input (not the state) becomes S2 for m2 more.  Per bin
    A = rho^m2 [t S1~ (1 - rho^(m1+1)) / (1 - rho)] + t S2~ (1 - rho^m2) / (1 - rho): the light built up from S1 decays
    geometrically while S2 is injected from the next boundary on.  (What opo_set_pump does on a running resonant pump.)"""
    log2n, T, L, nz = 6, 10 * PS, 5e-3, 4
    n = 1 << log2n
    dt = T / n
    Rp, delta, gdd = 0.7, -0.3, 200 * FS * FS
    b2p = 0.35 * FS * FS / UM
    o = make(n_fields=2, log2_n=log2n, window_s=T, nz=nz, length=L, d_eff=0.0, resonant=(1, 0), R=(Rp, 0),
             delta_rad=(delta, 0), gdd=(gdd, 0), beta2=(b2p, 0.0), ref_field=1)
    rng = np.random.default_rng(193)
    S1 = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    S2 = 1.5 * (rng.standard_normal(n) + 1j * rng.standard_normal(n))
    t = math.sqrt(1 - Rp)
    o.set_field(0, S1, which="input")
    o.set_field(0, t * S1, which="state")
    om = 2 * np.pi * np.fft.fftfreq(n, d=1.0 / n) / (n * dt)
    rho = math.sqrt(Rp) * np.exp(1j * delta) * np.exp(1j * (gdd / 2) * om ** 2) * np.exp(1j * (b2p / 2 * om ** 2) * L)
    m1, m2 = 3, 4
    assert o.roundtrips(m1) == 0
    o.set_field(0, S2, which="input")
    assert o.roundtrips(m2) == 0
    a1 = t * np.fft.fft(S1) * (1 - rho ** (m1 + 1)) / (1 - rho)
    expect = np.fft.ifft(rho ** m2 * a1 + t * np.fft.fft(S2) * (1 - rho ** m2) / (1 - rho))
    assert rel_l2(o.get_field(0), expect) < 1e-12
    # had the change reset the cavity to t S2 (an empty-cavity start), the result would differ at O(1)
    wrong = np.fft.ifft(t * np.fft.fft(S2) * (1 - rho ** (m2 + 1)) / (1 - rho))
    assert rel_l2(wrong, expect) > 0.1


def test_p19_single_pass_pump_is_the_r_equals_zero_case_and_signal_gets_no_injection():
    """R_p = 0 with the pump flagged resonant gives exactly the single-pass rule A_p <- S_p (R11); the injection acts on
    the pump only: a resonant signal is not topped up from its seed."""
    log2n, nz = 5, 10
    n = 1 << log2n
    kw = dict(n_fields=3, log2_n=log2n, nz=nz, dk=30.0, beta2=(0.35 * FS * FS / UM, 0.12 * FS * FS / UM, 0.05 * FS * FS / UM))
    a = make(resonant=(1, 1, 0), R=(0.0, 0.9, 0), **kw)
    b = make(resonant=(0, 1, 0), R=(0.0, 0.9, 0), **kw)
    ks = a.kappa(1)
    amp = 0.8 / (ks * 5e-3)
    rng = np.random.default_rng(191)
    f = [amp * (0.7 + 0.3 * (rng.standard_normal(n) + 1j * rng.standard_normal(n))) for _ in range(3)]
    for o in (a, b):
        for x in range(3):
            o.set_field(x, f[x] * (1.0, 0.2, 0.1)[x])
        assert o.roundtrips(3) == 0
    for x in range(3):
        assert rel_l2(a.get_field(x), b.get_field(x)) < 1e-14
        assert rel_l2(a.get_field(x, EXIT), b.get_field(x, EXIT)) < 1e-14
    # cold cavity, signal resonant: pure decay, no source term
    c = make(n_fields=2, log2_n=4, nz=4, d_eff=0.0, resonant=(0, 1), R=(0, 0.5))
    c.set_field(0, np.zeros(16, complex))
    c.set_field(1, np.ones(16, complex))
    assert c.roundtrips(4) == 0
    assert abs(abs(c.get_field(1)[0]) ** 2 - 0.5 ** 4) < 1e-14


def test_p19_resonant_pump_with_coupling_composes_from_single_passes():
    """Round trip 2 of a doubly resonant pump + signal equals a single pass fed by hand with
    sqrt(R_p) e^{i delta_p} exit_p + sqrt(1 - R_p) S_p and sqrt(R_s) exit_s."""
    log2n, nz, L = 5, 30, 5e-3
    n = 1 << log2n
    Rp, Rs, dp = 0.5, 0.8, 0.6
    kw = dict(n_fields=2, log2_n=log2n, nz=nz, length=L, dk=40.0, resonant=(1, 1), R=(Rp, Rs), delta_rad=(dp, 0.0),
              beta1=(0.3 * FS / UM, 0.0), beta2=(0.35 * FS * FS / UM, 0.10 * FS * FS / UM))
    o = make(**kw)
    ks = o.kappa(1)
    amp = 1.0 / (ks * L)
    rng = np.random.default_rng(192)
    Sp = amp * (0.9 + 0.1 * (rng.standard_normal(n) + 1j * rng.standard_normal(n)))
    Ss = 0.3 * amp * (rng.standard_normal(n) + 1j * rng.standard_normal(n))
    o.set_field(0, Sp, which="input")
    o.set_field(0, math.sqrt(1 - Rp) * Sp, which="state")
    o.set_field(1, Ss)
    assert o.roundtrips(1) == 0
    ex = [o.get_field(x, EXIT) for x in range(2)]
    nxt_p = _mirror(ex[0], Rp, dp) + math.sqrt(1 - Rp) * Sp
    assert rel_l2(o.get_field(0), nxt_p) < 1e-14
    assert o.roundtrips(1) == 0
    c = make(**kw)
    c.set_field(0, nxt_p)
    c.set_field(1, _mirror(ex[1], Rs))
    assert c.propagate(nz) == 0
    for x in range(2):
        assert rel_l2(o.get_field(x, EXIT), c.get_field(x)) < 1e-13


# ---------------------------------------------------------------------------------------------
# P20  several crystals in series ("one or more nonlinear media"; reading R25)
# ---------------------------------------------------------------------------------------------

def _p20_fields(n, amp, seed=20):
    rng = np.random.default_rng(seed)
    return [amp * s * (0.7 + 0.3 * (rng.standard_normal(n) + 1j * rng.standard_normal(n))) for s in (1.0, 0.4, 0.2)]


def test_p20_a_crystal_cut_in_two_is_the_same_crystal_when_dk_is_zero():
    """Two segments with the parameters of the whole crystal and dk = 0 are the uncut crystal step for step."""
    log2n, L, nz = 6, 5e-3, 24
    n = 1 << log2n
    kw = dict(n_fields=3, log2_n=log2n, nz=nz, length=L, dk=0.0, beta1=(0.3 * FS / UM, 0.0, -0.17 * FS / UM),
              beta2=(0.35 * FS * FS / UM, 0.12 * FS * FS / UM, 0.05 * FS * FS / UM), resonant=(0, 1, 0), R=(0, 0.9, 0))
    a, b = make(**kw), make(**kw)
    assert b.set_segments([(L * 10 / 24, 0.0, 14e-12, 10), (L * 14 / 24, 0.0, 14e-12, 14)]) == 0
    amp = 1.2 / (a.kappa(1) * L)
    for o in (a, b):
        for x, f in enumerate(_p20_fields(n, amp)):
            o.set_field(x, f)
        assert o.roundtrips(2) == 0
    for x in range(3):
        assert rel_l2(b.get_field(x, EXIT), a.get_field(x, EXIT)) < 1e-13
        assert rel_l2(b.get_field(x), a.get_field(x)) < 1e-13


def test_p20_segments_equal_single_passes_chained_by_hand():
    """Different length, step size, dk and d_eff per segment: the pass equals one single-crystal oracle per segment,
    each started at z = 0 of its own crystal, fed with the previous one's output; z does NOT run on across segments."""
    log2n = 6
    n = 1 << log2n
    segs = [(3e-3, 150.0, 14e-12, 12), (1e-3, -400.0, 9e-12, 7), (2e-3, 60.0, -14e-12, 10)]
    kw = dict(n_fields=3, log2_n=log2n, beta1=(0.3 * FS / UM, 0.0, -0.17 * FS / UM),
              beta2=(0.35 * FS * FS / UM, 0.12 * FS * FS / UM, 0.05 * FS * FS / UM), alpha=(2.0, 5.0, 1.0))
    o = make(nz=29, length=6e-3, **kw)
    assert o.set_segments(segs) == 0
    amp = 1.0 / (2 * np.pi * 14e-12 / (2.16 * 1000 * NM) * 6e-3)
    f = _p20_fields(n, amp, seed=21)
    for x in range(3):
        o.set_field(x, f[x])
    assert o.propagate(12 + 3) == 0                # stops inside the second crystal
    assert abs(o.z - 3 * 1e-3 / 7) < 1e-18          # z counts from that crystal's entrance
    assert o.propagate(29 - 15) == 0
    assert o.propagate(1) == 5                      # the pass is complete
    cur = f
    for (ln, dk, deff, nz) in segs:
        c = make(nz=nz, length=ln, dk=dk, d_eff=deff, **kw)
        for x in range(3):
            c.set_field(x, cur[x])
        assert c.propagate(nz) == 0
        cur = [c.get_field(x) for x in range(3)]
    for x in range(3):
        assert rel_l2(o.get_field(x), cur[x]) < 1e-13
    # one crystal of the total length with the first segment's parameters is something else
    w = make(nz=29, length=6e-3, dk=150.0, **kw)
    for x in range(3):
        w.set_field(x, f[x])
    w.propagate(29)
    assert rel_l2(w.get_field(1), cur[1]) > 1e-2


def test_p20_a_reversed_second_crystal_undoes_the_first():
    """Dispersion off, dk = 0: the coupled-wave equations with d_eff -> -d_eff are the same equations
    run backwards in z, so crystal + its reversed copy returns the input up to the RK4 truncation error, which falls as
    h^4; and round trips restart from segment 0."""
    log2n, L = 4, 5e-3
    n = 1 << log2n
    errs = []
    for nz in (20, 40):
        o = make(n_fields=3, log2_n=log2n, nz=2 * nz, length=2 * L, resonant=(0, 1, 0), R=(0, 1.0, 0))
        assert o.set_segments([(L, 0.0, 14e-12, nz), (L, 0.0, -14e-12, nz)]) == 0
        amp = 1.3 / (o.kappa(1) * L)
        f = _p20_fields(n, amp, seed=22)
        for x in range(3):
            o.set_field(x, f[x])
        assert o.propagate(nz) == 0
        assert abs(np.sum(np.abs(o.get_field(0)) ** 2) / np.sum(np.abs(f[0]) ** 2) - 1) > 0.05      # the first crystal did something
        assert o.propagate(nz) == 0
        errs.append(max(rel_l2(o.get_field(x), f[x]) for x in range(3)))
    assert errs[0] < 1e-6 and 8 < errs[0] / errs[1] < 32
    o = make(n_fields=3, log2_n=log2n, nz=40, length=2 * L, resonant=(0, 1, 0), R=(0, 1.0, 0))
    o.set_segments([(L, 0.0, 14e-12, 20), (L, 0.0, -14e-12, 20)])
    for x in range(3):
        o.set_field(x, f[x])
    assert o.roundtrips(3) == 0                      # R = 1, everything undone each pass: still the input
    assert rel_l2(o.get_field(1), f[1]) < 1e-5
    assert o.kappa(1) > 0                            # back in segment 0 after the boundary
