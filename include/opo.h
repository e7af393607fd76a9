/*
 * opo.h -- C ABI of libopo: split-step Fourier propagation of the chi(2) coupled-wave equations
 * through a crystal inside a ring cavity, on one NVIDIA B200 (sm_100a).
 *
 * What the library computes is the hot path of arxiv 2410.02532 ("CUDA-based optical parametric
 * oscillator simulator"; text at PAPER.md).  Citations are PAPER.md lines; "R<n>" are the readings
 * of the paper listed in DESIGN.md (and SURVEY.md section 8(c)).
 *
 *   z-step  (Eqs 10-11, order L/2 - N - L/2 of L133, reading R2), h = L/nz:
 *       A_x <- IDFT( H_x .* DFT(A_x) ),  H_x[k] = exp((-alpha_x/2 + i D_x(Omega_k)) h/2)
 *              D_x(Omega) = -(beta1_x - beta1_ref) Omega + (beta2_x/2) Omega^2    (L99 Eq. 5; R7, R8)
 *       one classic RK4 step of size h of the coupling terms of Eqs 2-4 (L86-95), pointwise in
 *              tau, stage abscissae z, z+h/2, z+h/2, z+h for exp(-/+ i dk z)      (L115; R3, R4)
 *              three-wave:  dA_p = i k_p A_s A_i e^{-i dk z}, dA_s = i k_s A_p A_i^* e^{+i dk z},
 *                           dA_i = i k_i A_p A_s^* e^{+i dk z}
 *              two-wave (degenerate, L164, R5): dA_p = i (k_p/2) A_s^2 e^{-i dk z},
 *                           dA_s = i k_s A_p A_s^* e^{+i dk z}
 *              k_x = 2 pi d_eff / (n_x lambda_x)                                   (L97)
 *       A_x <- IDFT( H_x .* DFT(A_x) );  z += h
 *   cavity boundary, once per round trip (L105-109 Eq. 6, Listing 3):
 *       exit_x <- A_x                                  (fields at z = L, before the mirror)
 *       resonant x:      A_x <- sqrt(R_x) e^{i delta_x} IDFT( G_x .* DFT(A_x) ),
 *                        G_x[k] = exp(i (gdd_x/2) Omega_k^2 - i Omega_k delta_T_x)  (R13-R15)
 *       non-resonant x:  A_x <- S_x   (stored input: fresh pump / frozen seed)      (R11, R12)
 *       resonant pump (x = 0; PAPER.md:L311 names doubly / triply resonant oscillators without an injection rule; reading
 *                        R24): the input coupler of power reflectivity R_p adds the external pump,
 *                        A_p <- sqrt(R_p) e^{i delta_p} IDFT( G_p .* DFT(A_p) ) [x modulator] + sqrt(1 - R_p) S_p;
 *                        R_p = 0 is the single-pass rule above.  Not on the large-N engine.
 *
 * Grid (L175-178; R8, R9, R19): N = 2^log2_n points, dt = window/N, tau_n = (n - N/2) dt,
 * Omega_k = 2 pi k'/(N dt), k' = k (k < N/2) or k - N.  DFT: X[k] = sum_n x[n] e^{-2 pi i k n/N},
 * unnormalised; the inverse carries 1/N.  Frequency-domain outputs are in natural FFT order.
 *
 * The implementation merges adjacent linear half-steps (H.H = one transform pair, an algebraic
 * identity) and keeps the fields on chip where they fit; results agree with the step-by-step
 * definition above to rounding.  See DESIGN.md.
 *
 * Conventions
 *   - SI units everywhere (m, s, V/m, rad).
 *   - Field buffers are contiguous [batch][N] interleaved (re, im): float2 (precision 0) or
 *     double2 (precision 1), 16-byte aligned.  "dev" pointers are CUDA device pointers on the
 *     current device, "host" pointers are ordinary (preferably pinned) host memory.
 *   - The caller owns every buffer it passes; the library copies out of / into it on the handle's
 *     stream and never frees or keeps it.  The handle owns its state and tables.
 *   - Every call returns an opo_status.  No exceptions, no global state.  Handles are independent;
 *     one handle must not be used from two threads at once.
 *   - A run may be cut into opo_propagate / opo_roundtrips calls in any way (z-step by z-step as in the paper's own loop,
 *     PAPER.md:L266-297): the result is the same to rounding.  In complex64 the kernels cycle through several roundings of
 *     the dispersion tables and apply constant corrections at every 8th operator; both follow the handle's running count
 *     of operators since opo_create, which no call resets.  Hence two handles driven by the same sequence of calls agree
 *     bit for bit, while a second run on a REUSED handle differs from the first at rounding level (1e-7 relative).
 *   - Calls enqueue work on the handle's stream and return; asynchronous faults surface at
 *     opo_sync or at the next call (OPO_ERR_CUDA).  The CUDA error state of the calling thread is shared with the rest
 *     of the process: the library looks at it (cudaPeekAtLastError) and clears it only after a failed call of its own,
 *     so an error that PyTorch or another library raised makes opo calls fail until its owner has dealt with it.  There is no CPU fallback of any kind: without
 *     a usable sm_100 device opo_create fails with OPO_ERR_CUDA.
 */
#ifndef OPO_H_
#define OPO_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct opo_handle opo_handle;

typedef enum {
    OPO_OK = 0,
    OPO_ERR_INVALID_ARG = 1, /* null pointer, N not a supported power of two, n_fields not 2|3, R outside [0,1], nz <= 0 ... */
    OPO_ERR_UNSUPPORTED = 2, /* precision/size/engine combination (e.g. a resonant pump or several crystals at N > 2^14) */
    OPO_ERR_ALLOC = 3,
    OPO_ERR_CUDA = 4,        /* message from the CUDA runtime in opo_last_error */
    OPO_ERR_STATE = 5,       /* propagate past z = L, roundtrips at z != 0 */
    OPO_ERR_NONFINITE = 6    /* opo_check_finite found NaN/Inf (the too-coarse-dz case of PAPER.md:L162) */
} opo_status;

/* crystal: PAPER.md:L97 (d_eff), L82 Eq. 1 (dk, the residual after quasi-phase-matching), L115 (L_cr) */
typedef struct {
    double length_m;
    double dk_per_m;      /* default for all batch instances; per-instance via opo_set_batch_param */
    double d_eff_m_per_V;
} opo_crystal;

/* fields: index 0 = pump, 1 = signal, 2 = idler (three-wave only).  PAPER.md:L99 Eq. 5, L105-109 Eq. 6,
 * L145 (GDD), L316-320 (resonance flags). */
typedef struct {
    int n_fields;              /* 2 (degenerate, signal = idler) or 3 */
    double lambda_m[3];
    double n[3];               /* refractive indices n_x */
    double beta1_s_per_m[3];   /* 1/v_x, any common origin; only differences to ref_field are used */
    double beta2_s2_per_m[3];  /* k''_x */
    double alpha_per_m[3];     /* power attenuation alpha_x */
    int ref_field;             /* co-moving frame (paper: the signal, L101) */
    int resonant[3];           /* a resonant pump (reading R24) re-enters through an input coupler, see below */
    double R[3];               /* power reflectivity 1 - theta_x, resonant fields */
    double delta_rad[3];       /* carrier detuning phase delta_x of Eq. 6 */
    double delta_T_s[3];       /* group-delay detuning: A(tau) -> A(tau - delta_T), circular (R13) */
    double gdd_s2[3];          /* gamma_x of L145: spectral phase (gamma/2) Omega^2 (R14) */
} opo_fields;

#define OPO_PRECISION_C64 0
#define OPO_PRECISION_C128 1

/* grid: PAPER.md:L175-178 (dt = t_rt/n), L162 (nz), L193 (precision) */
typedef struct {
    int log2_n;        /* 4 .. 18 */
    double window_s;   /* N dt, the round-trip window t_rt */
    int nz_per_pass;   /* z-steps per crystal pass; h = length_m / nz_per_pass */
    int precision;     /* OPO_PRECISION_C64 | OPO_PRECISION_C128 */
    int batch;         /* independent OPO instances sharing crystal, fields and grid */
} opo_grid;

/* Create a handle: validates, builds the fp64 host tables, allocates device state (zeroed) and
 * uploads the tables on the default stream.  *out is untouched on failure. */
int opo_create(const opo_crystal* crystal, const opo_fields* fields, const opo_grid* grid, opo_handle** out);
int opo_destroy(opo_handle* h);

/* All later work is enqueued on this stream (a cudaStream_t cast to void*; NULL = default stream).
 * The caller owns the stream and keeps it alive while the handle uses it. */
int opo_set_stream(opo_handle* h, void* cuda_stream);

/* Per-instance sweep parameters (BASELINE.json configs[2] detuning sweep, configs[4] dk sweep).
 * host_vals has `count` doubles and count must equal batch.  `field` is ignored for OPO_PARAM_DK. */
#define OPO_PARAM_DK 0
#define OPO_PARAM_DELTA_T 1
#define OPO_PARAM_DELTA_RAD 2
#define OPO_PARAM_GDD 3
int opo_set_batch_param(opo_handle* h, int param, int field, const double* host_vals, int count);

/* Several crystals in series inside one pass ("incorporation of one or more nonlinear media"; SURVEY 8(f) N4;
 * reading R25): segment j is walked in nz fixed steps h_j = length_m / nz with its own kappa_x = 2 pi d_eff / (n_x lambda_x)
 * and its own dk, z counted from that crystal's entrance; the fields' dispersion and loss are those of opo_fields for
 * every segment.  Replaces the crystal of opo_create (n = 0 restores it); afterwards a pass has sum(nz) z-steps, which
 * is what opo_propagate counts.  Per-instance OPO_PARAM_DK values act on the first segment and are reset by this call.
 * Only at z = 0 (OPO_ERR_STATE otherwise).  With n > 1 the host-sequenced STREAMING engine runs the pass (AUTO picks it);
 * OPO_ERR_UNSUPPORTED on the large-N engine and the cuFFT baseline. */
typedef struct {
    double length_m;
    double dk_per_m;
    double d_eff_m_per_V;
    int nz;
} opo_segment;
int opo_set_segments(opo_handle* h, int n, const opo_segment* segs);

/* Third-order dispersion of field `field` [s^3/m] (Eq. 5; reading R7 of DESIGN.md: the physical form
 * dA/dz = +(beta3/6) d^3A/dtau^3, i.e. D_x(Omega) gains the term -(beta3_x/6) Omega^3; the term as printed would be a
 * gain).  0 removes it.  Only the fp64 host tables change (rebuilt before the next propagate / roundtrips call). */
int opo_set_beta3(opo_handle* h, int field, double beta3_s3_per_m);

/* Intracavity electro-optic phase modulator on a resonant field, the last element of the cavity boundary
 * ("A(tau) -> A(tau) exp(i beta sin(2 pi f_pm tau))"; Listing 3
 * PhaseModulatorIntraCavity, after AddGDD and AddPhase): every round trip, after the spectral phase and the
 * mirror factor, A_x[n] *= exp(i beta sin(2 pi f_pm tau_n)), tau_n = (n - N/2) dt.  beta_rad = 0 removes it.
 * Same modulator for every instance.  OPO_ERR_INVALID_ARG for a non-resonant field (it restarts from its
 * stored input every round trip, so a modulator on it would never act).  The table is built in fp64 on the
 * host.  The on-chip engines (solo, wide, cluster) keep a whole opo_roundtrips call in one launch with a modulator
 * present: at a crossing they apply the table H G m, go to the time domain for the modulator and come back for the first
 * half-step H of the next pass (the boundary is then not merged into that half-step).  The large-N and streaming engines
 * run one launch sequence per round trip. */
int opo_set_eom(opo_handle* h, int field, double beta_rad, double f_mod_hz);

/* Pump input S_p (PAPER.md:L268 ReadPump): time-domain complex [N] (per_instance = 0, broadcast to
 * all instances) or [batch][N].  Copied into the handle; re-injected at every round-trip boundary.  Single-pass pump: when
 * z = 0 the current pump field becomes S_p as well, so the new input drives the next pass.  Resonant pump (reading R24):
 * before the handle has taken its first z-step the current pump field becomes sqrt(1 - R_p) S_p, what the input coupler
 * lets into an empty cavity; once the run is under way only S_p changes -- the light stored in the cavity stays, and the
 * boundary of the next round trip injects the new input (a pump ramp between opo_roundtrips calls).  To start over on
 * the same handle, set the intracavity pump yourself with opo_set_field(h, 0, ..) and then the input with this call. */
int opo_set_pump(opo_handle* h, const void* dev_pump, int per_instance);
int opo_set_pump_host(opo_handle* h, const void* host_pump, int per_instance);

/* Signal / idler (or pump) seed, [batch][N]: sets the current field and the stored input S_x
 * (noise seed).  Resets nothing else; allowed at any z. */
int opo_set_field(opo_handle* h, int field, const void* dev_data);
int opo_set_field_host(opo_handle* h, int field, const void* host_data);

/* nz fixed z-steps from the current z; no boundary operator.  OPO_ERR_STATE if it would pass z = L. */
int opo_propagate(opo_handle* h, int nz);

/* n x (full crystal pass + cavity boundary).  Requires z = 0.  Afterwards the current fields are
 * those at z = 0 of the next round trip and the exit buffer holds the fields at z = L of the last
 * pass (before the mirror). */
int opo_roundtrips(opo_handle* h, int n);

/* Nanosecond regime (PAPER.md:L228 NS_OPO, L302, L322-335): the pump pulse is much longer than a round trip, so
 * it is a long vector of n consecutive windows; round trip m is pumped by slice m (ReadPump, L268) and the field
 * that leaves the crystal in round trip m is appended to a long output vector (SaveRoundTrip, L272).
 *   dev_pump_train: [n][N] (per_instance = 0, every instance sees the same train) or [n][batch][N], time domain;
 *   dev_out_train : NULL, or [n][batch][N]: exit field `out_field` (z = L, before the mirror) of every round trip.
 * Equivalent to n x { opo_set_pump(slice m); opo_roundtrips(1); copy of OPO_WHICH_EXIT } with everything staying
 * on the device and on the handle's stream (the SOLO engine does the whole train in one launch, reading the slices and
 * writing the exit fields at the round-trip crossings inside the kernel).  Afterwards the stored pump input is the last slice.
 * OPO_ERR_UNSUPPORTED for a resonant pump, OPO_ERR_STATE unless z = 0. */
int opo_roundtrips_train(opo_handle* h, int n, const void* dev_pump_train, int per_instance, void* dev_out_train, int out_field);

#define OPO_WHICH_CURRENT 0
#define OPO_WHICH_EXIT 1
#define OPO_DOMAIN_TIME 0
#define OPO_DOMAIN_FREQ 1
/* Copy field `field` of every instance, [batch][N], into the caller's buffer.  FREQ = unnormalised
 * forward DFT, natural order, no fftshift. */
int opo_get_fields(opo_handle* h, int field, int which, int domain, void* dev_out);
int opo_get_fields_host(opo_handle* h, int field, int which, int domain, void* host_out);

/* Wait for the stream; reports asynchronous faults. */
int opo_sync(opo_handle* h);
/* Synchronises, then scans the current fields: OPO_ERR_NONFINITE if any NaN/Inf. */
int opo_check_finite(opo_handle* h);
/* Position inside the crystal in z-steps taken since the entrance (0 .. nz_per_pass). */
int opo_get_z_steps(const opo_handle* h, int* out_steps);

/* Execution engine.  AUTO picks RESIDENT or SOLO (see below) where one field fits one SM's shared memory (N <= 2^14 c64,
 * N <= 2^13 c128), else LARGE.
 *   RESIDENT : one thread-block cluster per instance, one CTA per field, fields stay in shared
 *              memory across z-steps and round trips; one launch per opo_propagate/opo_roundtrips.
 *   STREAMING: fields live in HBM/L2; one fused FFT-multiply-IFFT kernel and one RK4 kernel per z-step
 *              (same sizes as RESIDENT; the unfused internal baseline).
 *   LARGE    : N = 2^15 .. 2^18 (c128: 2^14 .. 2^18): four-step decomposition N = N1 x N2 in one
 *              persistent cooperative kernel, two L2-resident memory passes per z-step with RK4 fused
 *              into the column pass; one launch per opo_propagate/opo_roundtrips (plus the boundary
 *              of the last round trip). */
#define OPO_ENGINE_AUTO 0
#define OPO_ENGINE_RESIDENT 1
#define OPO_ENGINE_STREAMING 2
#define OPO_ENGINE_LARGE 3
/* Internal baseline, not the product (BASELINE.json north_star item (d)): cuFFT C2C over the batch + separate
 * elementwise kernels (table multiply, RK4, mirror), the structure of the paper's own program (PAPER.md:L248,
 * L286-287).  Never chosen by AUTO; libcufft is loaded on request.  Sizes of the streaming engine. */
#define OPO_ENGINE_CUFFT 4
/* SOLO: one CTA (one SM) per instance, same sizes as RESIDENT: one field in shared memory, the other fields in the SM's
 * tensor memory (TMEM), so the RK4 step of the coupling terms finds all fields of a grid point on
 * one SM and nothing crosses the SM-to-SM link; one launch per opo_propagate / opo_roundtrips.  AUTO picks it for
 * batches that keep (nearly) every SM busy (BASELINE.json configs[4]), RESIDENT for few instances (lowest latency per
 * instance).  The N/2 - L - N/2 ordering runs on RESIDENT. */
#define OPO_ENGINE_SOLO 5
/* WIDE: one thread-block cluster of 4 F CTAs per instance (N = 2^12 .. 2^14; c128: 2^12, 2^13): every field is split
 * over four SMs along the radix-4 first pass of the transform, the pass that crosses the split (fused with the RK4
 * step) exchanges its operands over distributed shared memory; one launch per opo_propagate /
 * opo_roundtrips.  The lowest latency per z-step: AUTO picks it when the whole batch fits the co-resident clusters in
 * one wave (the paper's own workload, one OPO followed for thousands of round trips; BASELINE.json
 * configs[1], [2]).  Not with the N/2 - L - N/2 ordering or a resonant pump: those run on RESIDENT (a request for WIDE is
 * then served by RESIDENT / SOLO as AUTO would). */
#define OPO_ENGINE_WIDE 6
#define OPO_OPT_ENGINE 0
/* Operator splitting of a z-step.  LNL (default, BASELINE.json north_star): linear half-step,
 * one RK4 step h, linear half-step.  NLN: the order the paper implements, Eq. 10-11: one RK4 step of h/2, the full
 * linear step, one RK4 step of h/2 (stage abscissae z, z+h/4, z+h/2 and z+h/2, z+3h/4, z+h).  Both are second
 * order and differ by O(h^2).  Can change at z = 0 only.  With NLN the resident and large-N engines run one launch
 * per round trip. */
#define OPO_OPT_SPLITTING 1
/* WIDE engine only: sub-blocks of a field per CTA.  1: clusters of 4 F CTAs (lowest latency per instance, 7 clusters of 12 CTAs
 * co-resident on a B200); 2: clusters of 2 F CTAs (22 co-resident, each ~1.4x slower per z-step); 0 (default): whichever
 * finishes the batch sooner. */
#define OPO_OPT_WIDE_SUBBLOCKS 2
#define OPO_SPLITTING_LNL 0
#define OPO_SPLITTING_NLN 1
int opo_set_option(opo_handle* h, int option, int value);

#define OPO_INFO_ENGINE 0        /* engine the next propagate/roundtrips call will use */
#define OPO_INFO_LAUNCHES 1      /* kernels launched by this handle so far */
#define OPO_INFO_N 2
#define OPO_INFO_BATCH 3
#define OPO_INFO_SM_COUNT 4
#define OPO_INFO_SLOTS 5           /* co-resident work slots (clusters / CTAs) the next roundtrips call deals its work to */
#define OPO_INFO_WIDE_SUBBLOCKS 6  /* sub-blocks of a field per CTA the WIDE engine will use (1 | 2; see OPO_OPT_WIDE_SUBBLOCKS), 0 on other engines */
int opo_get_info(const opo_handle* h, int what, long long* out);

/* Device peaks measured on the spot with the library's own micro-benchmark kernels, the roofline denominators bench.py
 * reports against; independent of any handle, runs on the default stream of the current device
 * and takes ~0.1 s.  FP32 / FP64: independent FMA chains on every SM [TFLOP/s]; SMEM: conflict-free 16-byte shared-memory
 * loads + stores on every SM [GB/s]; TMEM_LD / TMEM_ST: tcgen05.ld / tcgen05.st of a thread's own columns [GB/s];
 * DSMEM: 16-byte stores into the shared memory of the next CTA of a cluster of 4, all co-resident clusters at once:
 * bytes SENT per SM [GB/s per SM]; every SM receives the same amount at the same time. */
#define OPO_PEAK_FP32_FMA 0
#define OPO_PEAK_FP64_FMA 1
#define OPO_PEAK_SMEM 2
#define OPO_PEAK_TMEM_LD 3
#define OPO_PEAK_TMEM_ST 4
#define OPO_PEAK_DSMEM 5
int opo_selftest_peak(int what, double* out_value);

/* Forward DFT of caller-owned rows WITHOUT a handle and without any device-memory allocation: the frequency read-out
 * of opo_get_fields(.., OPO_DOMAIN_FREQ, ..) (same kernel, same tables, bit-identical result) for callers that cannot
 * afford, or are not allowed, to call cudaMalloc.  Who that is: (1) a process whose framework allocator (PyTorch's caching
 * allocator, an RMM pool, a lab control program's arena) has already taken the whole of HBM, so that a cudaMalloc of the
 * library's own would fail although the caller has plenty of room inside its pool; (2) a measurement or feedback loop
 * that looks at the spectrum every few round trips (PAPER.md:L449 writes spectra out; Listing 3 L279-297 is such a loop)
 * and cannot take the device-wide synchronisation that cudaMalloc / cudaFree imply; (3) code that must prove, for a
 * long unattended run, that its device footprint does not grow.  opo_create, by contrast, allocates state and tables.
 *     dev_in, dev_out : device pointers on the current device, [batch][N] interleaved (re, im), float2 (precision 0) or
 *                       double2 (precision 1), 16-byte aligned, N = 2^log2_n; both stay the caller's; they may be the
 *                       same buffer (each row is read completely before it is written).
 *     result          : dev_out[b][k] = sum_n dev_in[b][n] exp(-2 pi i k n / N), unnormalised, natural order (see "Grid").
 *     cuda_stream     : a cudaStream_t cast to void* (NULL = default stream); the launch is enqueued there.
 * Limit: log2_n in 4 .. 14 for complex64, 4 .. 13 for complex128; anything longer returns OPO_ERR_UNSUPPORTED with a
 * message naming the limit (use a handle for those).  batch is any positive int.
 * Where the tables live instead: in a 192 KiB array that is part of the library image (a file-scope __device__ array
 * in opo_api.cu).  Every GPU on which a CUDA context loads libopo.so carries these 192 KiB until the process exits,
 * whether or not this function is ever called.
 * First call on each device: looks up that device's address of the array and writes the tables (two host-to-device
 * copies on cuda_stream followed by a wait for that stream).  Make this first call during start-up, before any stream
 * capture is begun.  The same copy + wait happens again whenever (log2_n, precision) differ from the previous call on
 * that device, because the array holds the tables of one size at a time and keeps them between calls.
 * Concurrency: all calls on a device share the one array.  Calls with the same (log2_n, precision) only read it and
 * may overlap freely.  A call with a different size rewrites it in the order of ITS stream only: if work from an
 * earlier call with another size is still running on a different stream, the two race and that earlier result is
 * garbage.  Keep such calls on one stream or put an event between them.  Host threads may call concurrently (the
 * bookkeeping is under a mutex); the rule above is about what overlaps on the GPU.
 * Calls no cudaMalloc / cudaFree / cuFFT.  Errors: status code, text via opo_last_error(NULL) of the calling thread. */
int opo_spectrum_noalloc(const void* dev_in, void* dev_out, int log2_n, int batch, int precision, void* cuda_stream);

/* Last error text of this handle (or of the failed opo_create when h is NULL).  Never NULL. */
const char* opo_last_error(const opo_handle* h);

#ifdef __cplusplus
}
#endif
#endif /* OPO_H_ */
