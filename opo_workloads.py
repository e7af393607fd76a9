"""Seeded synthetic inputs for the OPO hot path (shared by the oracle tests and the CUDA tests).

This module holds NONE of the method's arithmetic: no FFT, no dispersion operator, no RK4, no
boundary operator.  It only turns the five workloads of BASELINE.json:configs[0..4] (concretised
in SURVEY.md section 8(d), recipe restated in DESIGN.md) into plain parameter records and numpy
arrays: the pump envelope, and the noise seeds for signal/idler.  The only physics here is the
input *scaling* (how many V/m "X times threshold" is, reading R18), which is harness arithmetic
(Eq. 12 region) and is never used by either implementation.

Everything is SI at this level (metres, seconds, V/m), as at the C ABI (include/opo.h).
The paper ships no data set (outputs are .dat files), so these synthetic inputs
stand in for its cw / pulsed workloads (sizes 2^10..2^15 L180;
50-250 z points L162; R = 0.98 L348).
"""
from __future__ import annotations

import copy
import math
from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

FS = 1e-15
PS = 1e-12
UM = 1e-6
NM = 1e-9
# fs/um and fs^2/um in SI
FS_PER_UM = FS / UM
FS2_PER_UM = FS * FS / UM

PUMP, SIGNAL, IDLER = 0, 1, 2


@dataclass
class Workload:
    """One batch of independent OPO instances with identical crystal/grid and per-instance sweeps."""

    name: str
    # crystal
    length_m: float
    d_eff_m_per_V: float
    # fields (index 0 pump, 1 signal, 2 idler); lists of length n_fields
    n_fields: int
    lambda_m: List[float]
    n_index: List[float]
    beta1_s_per_m: List[float]      # group delay per metre relative to an arbitrary origin
    beta2_s2_per_m: List[float]
    alpha_per_m: List[float]
    ref_field: int
    resonant: List[int]
    R: List[float]
    delta_rad: List[float]
    delta_T_s: List[float]
    gdd_s2: List[float]
    # grid
    log2_n: int
    window_s: float
    nz_per_pass: int
    precision: str                   # "c64" | "c128"
    batch: int
    n_roundtrips: int
    # per-instance sweeps (length batch) -- None means "same for all instances"
    dk_per_m: np.ndarray = field(default_factory=lambda: np.zeros(1))
    delta_T_signal_s: Optional[np.ndarray] = None
    # inputs, complex128 arrays, already rounded to the grid precision
    pump: np.ndarray = None          # [batch or 1][N]
    seeds: List[Optional[np.ndarray]] = None   # per field: None (pump) or [batch][N]
    notes: str = ""
    # intracavity phase modulator per field: depth [rad] (0 = none) and frequency [Hz]
    eom_beta_rad: List[float] = field(default_factory=lambda: [0.0, 0.0, 0.0])
    eom_f_hz: List[float] = field(default_factory=lambda: [0.0, 0.0, 0.0])
    # third-order dispersion per field [s^3/m] (Eq. 5, reading R7); 0 = none
    beta3_s3_per_m: List[float] = field(default_factory=lambda: [0.0, 0.0, 0.0])
    # operator splitting: 0 = L/2 - N - L/2 (default), 1 = N/2 - L - N/2 (the paper's Eq. 10-11)
    splitting: int = 0
    # several crystals in series (reading R25): list of (length_m, dk_per_m, d_eff_m_per_V, nz) or None for
    # the single crystal (length_m, dk_per_m, d_eff_m_per_V, nz_per_pass); nz_per_pass must then be the sum of the nz
    segments: Optional[list] = None

    @property
    def n(self) -> int:
        return 1 << self.log2_n

    @property
    def dt(self) -> float:
        return self.window_s / self.n

    @property
    def tau(self) -> np.ndarray:
        """Time axis, reading R19: tau_n = (n - N/2) dt."""
        return (np.arange(self.n) - self.n // 2) * self.dt

    def kappa(self) -> List[float]:
        """kappa_x = 2 pi d_eff / (n_x lambda_x) -- used here only to scale inputs."""
        return [2.0 * math.pi * self.d_eff_m_per_V / (self.n_index[x] * self.lambda_m[x])
                for x in range(self.n_fields)]

    def dk_of(self, b: int) -> float:
        return float(self.dk_per_m[b if len(self.dk_per_m) > 1 else 0])

    def delta_T_of(self, b: int, x: int) -> float:
        if x == SIGNAL and self.delta_T_signal_s is not None:
            return float(self.delta_T_signal_s[b])
        return float(self.delta_T_s[x])

    def pump_of(self, b: int) -> np.ndarray:
        return self.pump[b if self.pump.shape[0] > 1 else 0]

    def truncated(self, n_roundtrips: int) -> "Workload":
        w = copy.copy(self)
        w.n_roundtrips = int(n_roundtrips)
        w.name = f"{self.name}[rt={n_roundtrips}]"
        return w

    def subset(self, instances) -> "Workload":
        """Keep only the listed batch instances (parity on a subset of a large sweep)."""
        idx = np.asarray(list(instances), dtype=np.int64)
        w = copy.copy(self)
        w.batch = len(idx)
        w.dk_per_m = self.dk_per_m[idx] if len(self.dk_per_m) > 1 else self.dk_per_m
        if self.delta_T_signal_s is not None:
            w.delta_T_signal_s = self.delta_T_signal_s[idx]
        w.pump = self.pump[idx] if self.pump.shape[0] > 1 else self.pump
        w.seeds = [None if s is None else s[idx] for s in self.seeds]
        w.name = f"{self.name}[subset {len(idx)}]"
        return w


# ----------------------------------------------------------------------------------------------
# helpers (input scaling and random draws only)
# ----------------------------------------------------------------------------------------------

def _round_to_precision(a: np.ndarray, precision: str) -> np.ndarray:
    """Round inputs once to the grid precision so both sides are fed identical numbers."""
    if precision == "c64":
        return a.astype(np.complex64).astype(np.complex128)
    return a.astype(np.complex128)


def complex_gaussian_noise(seed: int, n: int, rms: float) -> np.ndarray:
    """Circular complex Gaussian, E|A|^2 = rms^2 (reading R17; PAPER.md:L340 'random amplitude and phase')."""
    rng = np.random.default_rng(int(seed))
    re = rng.standard_normal(n)
    im = rng.standard_normal(n)
    return (re + 1j * im) * (rms / math.sqrt(2.0))


def splitmix64(master: int, index: int) -> int:
    """Counter-based seed derivation for the batched sweep (C4): one 64-bit seed per instance."""
    mask = (1 << 64) - 1
    z = (master * 0x9E3779B97F4A7C15 + (index + 1) * 0x9E3779B97F4A7C15) & mask
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & mask
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & mask
    return (z ^ (z >> 31)) & mask


def threshold_amplitude_degenerate(kappa_s: float, length: float, R_s: float) -> float:
    """Reading R18: plane-wave dispersionless degenerate threshold  sqrt(R) exp(kappa_s A_th L) = 1."""
    return -math.log(R_s) / (2.0 * kappa_s * length)


def threshold_amplitude_sro(kappa_s: float, kappa_i: float, length: float, R_s: float) -> float:
    """Reading R18: singly resonant threshold  R_s cosh^2(sqrt(kappa_s kappa_i) A_th L) = 1."""
    return math.acosh(1.0 / math.sqrt(R_s)) / (math.sqrt(kappa_s * kappa_i) * length)


# ----------------------------------------------------------------------------------------------
# the five workloads
# ----------------------------------------------------------------------------------------------

def _degenerate_base(name, log2_n, window_s, nz, precision, n_rt) -> Workload:
    return Workload(
        name=name, length_m=5e-3, d_eff_m_per_V=14e-12, n_fields=2,
        lambda_m=[532 * NM, 1064 * NM], n_index=[2.23, 2.16],
        # beta1_s - beta1_p = -0.30 fs/um  (configs[0]); origin chosen at the signal (R10)
        beta1_s_per_m=[0.30 * FS_PER_UM, 0.0],
        beta2_s2_per_m=[0.35 * FS2_PER_UM, 0.10 * FS2_PER_UM],
        alpha_per_m=[0.0, 0.0], ref_field=SIGNAL, resonant=[0, 1], R=[0.0, 0.98],
        delta_rad=[0.0, 0.0], delta_T_s=[0.0, 0.0], gdd_s2=[0.0, 0.0],
        log2_n=log2_n, window_s=window_s, nz_per_pass=nz, precision=precision, batch=1,
        n_roundtrips=n_rt, dk_per_m=np.zeros(1))


def config0(n_roundtrips: int = 20) -> Workload:
    """C0: degenerate two-wave CW OPO, N = 2^10, complex128 (BASELINE.json:configs[0])."""
    w = _degenerate_base("C0", 10, 10 * PS, 20, "c128", n_roundtrips)
    k = w.kappa()
    a_th = threshold_amplitude_degenerate(k[SIGNAL], w.length_m, w.R[SIGNAL])
    a_p = math.sqrt(2.0) * a_th                       # 2x threshold intensity
    w.pump = _round_to_precision(np.full((1, w.n), a_p, dtype=np.complex128), w.precision)
    w.seeds = [None, _round_to_precision(complex_gaussian_noise(0, w.n, 1e-6 * a_p)[None, :], w.precision)]
    w.notes = f"A_th={a_th:.6e} V/m, A_p={a_p:.6e} V/m"
    return w


def _nondegenerate_base(name, nz, n_rt, batch) -> Workload:
    lam_p, lam_s = 532 * NM, 1000 * NM
    lam_i = 1.0 / (1.0 / lam_p - 1.0 / lam_s)           # energy conservation
    return Workload(
        name=name, length_m=20e-3, d_eff_m_per_V=14e-12, n_fields=3,
        lambda_m=[lam_p, lam_s, lam_i], n_index=[2.23, 2.16, 2.15],          # G1
        # offsets relative to the pump: -0.28 (signal), -0.45 (idler) fs/um (configs[1])
        beta1_s_per_m=[0.0, -0.28 * FS_PER_UM, -0.45 * FS_PER_UM],
        beta2_s2_per_m=[0.35 * FS2_PER_UM, 0.12 * FS2_PER_UM, 0.05 * FS2_PER_UM],
        alpha_per_m=[0.0, 0.0, 0.0], ref_field=SIGNAL, resonant=[0, 1, 0], R=[0.0, 0.98, 0.0],
        delta_rad=[0.0] * 3, delta_T_s=[0.0] * 3, gdd_s2=[0.0] * 3,
        log2_n=14, window_s=10 * PS, nz_per_pass=nz, precision="c64", batch=batch,       # G2
        n_roundtrips=n_rt, dk_per_m=np.zeros(1))


def _sro_threshold(w: Workload) -> float:
    k = w.kappa()
    return threshold_amplitude_sro(k[SIGNAL], k[IDLER], w.length_m, w.R[SIGNAL])


def config1(n_roundtrips: int = 1000) -> Workload:
    """C1: three-wave singly resonant CW OPO, N = 2^14, complex64 (BASELINE.json:configs[1])."""
    w = _nondegenerate_base("C1", 100, n_roundtrips, 1)
    a_th = _sro_threshold(w)
    a_p = math.sqrt(3.0) * a_th
    w.pump = _round_to_precision(np.full((1, w.n), a_p, dtype=np.complex128), w.precision)
    w.seeds = [None,
               _round_to_precision(complex_gaussian_noise(1, w.n, 1e-6 * a_p)[None, :], w.precision),
               _round_to_precision(complex_gaussian_noise(2, w.n, 1e-6 * a_p)[None, :], w.precision)]
    w.notes = f"A_th={a_th:.6e} V/m, A_p={a_p:.6e} V/m"
    return w


def config2(n_roundtrips: int = 500) -> Workload:
    """C2: synchronously pumped fs OPO, sech pump, GDD -500 fs^2, 11 detunings (configs[2])."""
    w = _nondegenerate_base("C2", 200, n_roundtrips, 11)
    a_pk = math.sqrt(3.0) * _sro_threshold(w)             # G3
    t0 = 200 * FS / (2.0 * math.acosh(math.sqrt(2.0)))    # sech^2 intensity FWHM = 1.7627 T0
    pump = a_pk / np.cosh(w.tau / t0)
    w.pump = _round_to_precision(pump[None, :].astype(np.complex128), w.precision)
    w.gdd_s2 = [0.0, -500 * FS * FS, 0.0]
    w.delta_T_signal_s = np.linspace(-20 * FS, 20 * FS, 11)
    sig = np.stack([complex_gaussian_noise(10 + b, w.n, 1e-6 * a_pk) for b in range(w.batch)])
    idl = np.stack([complex_gaussian_noise(1000 + 10 + b, w.n, 1e-6 * a_pk) for b in range(w.batch)])
    w.seeds = [None, _round_to_precision(sig, w.precision), _round_to_precision(idl, w.precision)]
    w.notes = f"A_pk={a_pk:.6e} V/m, T0={t0:.6e} s"
    return w


def config3(n_roundtrips: int = 200, log2_n: int = 18) -> Workload:
    """C3: long-window degenerate OPO, N = 2^18 over 2 ns, Gaussian pump 500 ps FWHM (configs[3])."""
    w = _degenerate_base("C3", log2_n, 2000 * PS, 500, "c64", n_roundtrips)
    k = w.kappa()
    a_th = threshold_amplitude_degenerate(k[SIGNAL], w.length_m, w.R[SIGNAL])
    a_pk = 2.0 * a_th                                     # 4x threshold intensity
    fwhm = 500 * PS
    sigma_i = fwhm / (2.0 * math.sqrt(2.0 * math.log(2.0)))      # intensity std-dev
    pump = a_pk * np.exp(-w.tau ** 2 / (4.0 * sigma_i ** 2))     # amplitude = sqrt(intensity)
    w.pump = _round_to_precision(pump[None, :].astype(np.complex128), w.precision)
    w.seeds = [None, _round_to_precision(complex_gaussian_noise(3, w.n, 1e-6 * a_pk)[None, :], w.precision)]
    w.notes = f"A_th={a_th:.6e} V/m, A_pk={a_pk:.6e} V/m"
    return w


def config4(n_roundtrips: int = 300, batch_side: int = 16) -> Workload:
    """C4: batched sweep, 16 pump levels x 16 phase mismatches = 256 instances of C1 (configs[4])."""
    b_total = batch_side * batch_side
    w = _nondegenerate_base("C4", 100, n_roundtrips, b_total)
    a_th = _sro_threshold(w)
    levels = np.linspace(1.0, 5.0, batch_side)
    dks = np.linspace(-50.0, 50.0, batch_side)
    pump = np.empty((b_total, w.n), dtype=np.complex128)
    dk = np.empty(b_total)
    sig = np.empty((b_total, w.n), dtype=np.complex128)
    idl = np.empty((b_total, w.n), dtype=np.complex128)
    for b in range(b_total):
        ip, ik = divmod(b, batch_side)
        a_p = math.sqrt(levels[ip]) * a_th
        pump[b, :] = a_p
        dk[b] = dks[ik]
        sig[b] = complex_gaussian_noise(splitmix64(4, 2 * b), w.n, 1e-6 * a_p)
        idl[b] = complex_gaussian_noise(splitmix64(4, 2 * b + 1), w.n, 1e-6 * a_p)
    w.dk_per_m = dk
    w.pump = _round_to_precision(pump, w.precision)
    w.seeds = [None, _round_to_precision(sig, w.precision), _round_to_precision(idl, w.precision)]
    w.notes = f"A_th={a_th:.6e} V/m, X in [1,5] x dk in [-50,50] 1/m"
    return w


ALL_CONFIGS = {"C0": config0, "C1": config1, "C2": config2, "C3": config3, "C4": config4}
