// =================================================================================================
// ORACLE -- TEST INFRASTRUCTURE ONLY.  Not part of the product.
//
// A plain, slow, obviously-correct CPU implementation of the hot path of arxiv 2410.02532
// ("CUDA-based optical parametric oscillator simulator"): fixed-step symmetric split-step Fourier
// propagation of the two-/three-wave chi(2) coupled-wave equations through a crystal, repeated
// over cavity round trips.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may build, load or call this file.  It shares no code with the CUDA path
// (paper_2410_02532_b200/csrc): own radix-2 FFT, own tables, own RK4.
//
// It follows the algorithm step by step in the paper's order and notation, in fp64 (the `float`
// instantiation exists only to measure the fp32 error floor, pin P12).  No blocking, fusion,
// half-step merging or reordering.  Readings R1..R21 are those of SURVEY.md section 8(c), listed
// again in DESIGN.md.
//
//   z-step  ("L/2 - N - L/2", reading R2):
//        A_x <- IDFT( H_x .* DFT(A_x) )                        (Eq. 5; R7, R8)
//        (A_p, A_s[, A_i])[n] <- one classic RK4 step of size h of the coupling terms of
//                                Eqs 2-4, abscissae z, z+h/2, z+h/2, z+h (R3, R4)
//        A_x <- IDFT( H_x .* DFT(A_x) );  z += h
//        (optional: the paper's own order N/2 - L - N/2 of Eq. 10-11, two RK4 half-steps around one full linear step)
//        (optional third-order dispersion: D_x -= (beta3_x/6) Omega^3, reading R7)
//   pass    = nz z-steps from z = 0
//   boundary (Eq. 6, Listing 3; R11-R15):
//        exit_x <- A_x
//        resonant x:     A_x <- sqrt(R_x) e^{i delta_x} IDFT( G_x .* DFT(A_x) )
//                        A_x[n] <- A_x[n] exp(i beta_x sin(2 pi f_x tau_n))   intracavity EOM, last element
//                                  (Listing 3; off when beta_x = 0)
//        non-resonant x: A_x <- S_x   (stored input: fresh pump / frozen seed)
//        resonant pump (x = 0, reading R24): the input coupler adds the external pump,
//                        A_p <- [boundary of a resonant field] + sqrt(1 - R_p) S_p     (R_p = 0 is the single-pass rule above)
//   several crystals in series ("one or more nonlinear media", reading R25): a pass is a
//        sequence of segments (length L_j, dk_j, d_eff_j, nz_j); each is walked with its own h_j = L_j / nz_j,
//        kappa_x = 2 pi d_eff_j / (n_x lambda_x) and dk_j, z measured from the segment's own entrance
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): P1 naive DFT, P2 Gaussian GVD closed form, P3 GVM
// integer shift, P4 cosh^2 gain (+dk), P5 degenerate phase-sensitive gain (paper's pi/4, -3pi/4,
// PAPER.md:L400), P6 Manley-Rowe, P7 depleted SHG closed form, P8 2nd-order convergence, P9 cold
// cavity, P10 threshold growth, P11 steady-state pump depletion 4 (sqrt(N) - 1) / N, largest at the printed N = 4,
// P13 EOM sidebands = Bessel J_m(beta) (Jacobi-Anger) and element order,
// P14 third-order dispersion: centroid delay (beta3 z/2)(Omega_0^2 + s^2) of an offset Gaussian, P15 N/2-L-N/2 ordering:
// second-order convergence, O(h^2) agreement with L/2-N-L/2, exact agreement when the operators commute,
// P16 loss: power falls as exp(-alpha_x z), a pure scale (alpha/2 on the amplitude, Eq. 5), P17 pump re-injection: after
// the boundary the pump is the stored input bit for bit and round trip 2 equals a hand-composed single pass (L268, R11),
// P18 z restarts at the crystal entrance every pass with dk != 0 (R4): round trips = passes on fresh oracles,
// P19 resonant pump: cold-cavity build-up to the closed-form Airy steady state sqrt(1-R) S / (1 - sqrt(R) e^{i delta} G e^{i D L})
// per bin, geometric partial sums on the way, R_p = 0 equals the single-pass rule, the input changed mid-run leaves the stored light alone,
// P20 crystal segments: a crystal cut in two equal-parameter segments with dk = 0 equals the uncut crystal; with dk != 0 it
// equals two single passes chained by hand; a second segment with d_eff -> -d_eff undoes the first one (dispersion off).
// Parity unpinned: reading R12 (non-resonant fields restart from
// S_x) is a convention with no physical pin; the paper's P_th values (L348) and Figs 3-5.
// =================================================================================================
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

constexpr double kPi = 3.14159265358979323846264338327950288;

// ---- own FFT: iterative radix-2 decimation in time, bit-reversal first ---------------------------
// X[k] = sum_n x[n] exp(-2 pi i k n / N)   (forward, unnormalised);  inverse carries 1/N  (R8).
// Twiddles are evaluated per index in fp64 (no recurrence), then rounded to R.
template <class R>
struct Fft {
    int n = 0, log2n = 0;
    std::vector<std::complex<R>> w;   // w[j] = exp(-2 pi i j / N), j < N/2
    std::vector<uint32_t> rev;

    void init(int log2n_) {
        log2n = log2n_;
        n = 1 << log2n;
        w.resize(n / 2 > 0 ? n / 2 : 1);
        for (int j = 0; j < n / 2; ++j) {
            double ang = -2.0 * kPi * (double)j / (double)n;
            w[j] = std::complex<R>((R)std::cos(ang), (R)std::sin(ang));
        }
        rev.resize(n);
        for (int i = 0; i < n; ++i) {
            uint32_t r = 0;
            for (int b = 0; b < log2n; ++b)
                if (i & (1 << b)) r |= 1u << (log2n - 1 - b);
            rev[i] = r;
        }
    }

    void transform(std::complex<R>* x, bool inverse) const {
        for (int i = 0; i < n; ++i) {
            int r = (int)rev[i];
            if (r > i) std::swap(x[i], x[r]);
        }
        for (int len = 2; len <= n; len <<= 1) {
            int half = len >> 1;
            int step = n / len;
            for (int base = 0; base < n; base += len) {
                for (int j = 0; j < half; ++j) {
                    std::complex<R> tw = w[j * step];
                    if (inverse) tw = std::conj(tw);
                    std::complex<R> u = x[base + j];
                    std::complex<R> v = x[base + j + half];
                    // explicit complex product (no library special-casing)
                    std::complex<R> t(v.real() * tw.real() - v.imag() * tw.imag(),
                                      v.real() * tw.imag() + v.imag() * tw.real());
                    x[base + j] = u + t;
                    x[base + j + half] = u - t;
                }
            }
        }
        if (inverse) {
            R s = (R)1 / (R)n;
            for (int i = 0; i < n; ++i) x[i] *= s;
        }
    }
};

struct Params {
    int n_fields, log2n, nz, ref_field;
    double window_s, length_m, dk_per_m, d_eff;
    double lambda_m[3], n_index[3], beta1[3], beta2[3], alpha[3];
    int resonant[3];
    double R[3], delta_rad[3], delta_T[3], gdd[3];
    int splitting;                  // 0: L/2 - N - L/2 (north_star, default); 1: N/2 - L - N/2 (the paper's Eq. 10-11)
    double beta3[3];                // third-order dispersion of field x [s^3/m] (Eq. 5; reading R7), 0 unless set
    double eom_beta[3], eom_f[3];   // intracavity phase modulator: depth [rad], frequency [Hz]
    // crystal segments in series (reading R25); n_seg = 0 means the single crystal (length_m, dk_per_m, d_eff, nz)
    int n_seg;
    double seg_len[8], seg_dk[8], seg_deff[8];
    int seg_nz[8];
};

template <class R>
struct Oracle {
    using C = std::complex<R>;
    Params p;
    int N, F;
    double h;       // dz = L / nz of the current segment
    double z;       // position inside the current crystal segment, 0 at its entrance (R4, R20, R25)
    double kappa[3];            // of the current segment
    int K;                      // number of segments
    int seg, seg_step;          // current segment and z-steps taken inside it
    double seg_h[8], seg_kappa[8][3];
    Fft<R> fft;
    std::vector<C> A[3], S[3], EX[3], G[3];
    std::vector<C> Hs[8][3], HFs[8][3];     // half-step / full-step multipliers per segment
    bool boundary_needs_transform[3];

    double seg_len(int j) const { return p.n_seg ? p.seg_len[j] : p.length_m; }
    double seg_dk(int j) const { return p.n_seg ? p.seg_dk[j] : p.dk_per_m; }
    double seg_deff(int j) const { return p.n_seg ? p.seg_deff[j] : p.d_eff; }
    int seg_nz(int j) const { return p.n_seg ? p.seg_nz[j] : p.nz; }
    int steps_per_pass() const { int t = 0; for (int j = 0; j < K; ++j) t += seg_nz(j); return t; }
    void enter_segment(int j) {
        seg = j; seg_step = 0; z = 0.0; h = seg_h[j];
        for (int x = 0; x < F; ++x) kappa[x] = seg_kappa[j][x];
    }

    // Omega_k = 2 pi k' / (N dt), natural FFT order, Nyquist bin negative (R9)
    double omega(int k) const {
        int kp = (k < N / 2) ? k : k - N;
        double dt = p.window_s / (double)N;
        return 2.0 * kPi * (double)kp / ((double)N * dt);
    }

    void init(const Params& pp) {
        p = pp;
        F = p.n_fields;
        N = 1 << p.log2n;
        seg = 0; seg_step = 0; z = 0.0;
        fft.init(p.log2n);
        for (int x = 0; x < F; ++x) {
            A[x].assign(N, C(0, 0));
            S[x].assign(N, C(0, 0));
            EX[x].assign(N, C(0, 0));
        }
        build_tables();
    }

    void build_tables() {
        K = p.n_seg ? p.n_seg : 1;
        for (int j = 0; j < K; ++j) {
            seg_h[j] = seg_len(j) / (double)seg_nz(j);             // dz = L_j / nz_j
            // kappa_x = 2 pi d_eff / (n_x lambda_x)
            for (int x = 0; x < F; ++x) seg_kappa[j][x] = 2.0 * kPi * seg_deff(j) / (p.n_index[x] * p.lambda_m[x]);
        }
        for (int j = 0; j < K; ++j)
        for (int x = 0; x < F; ++x) {
            std::vector<C>& H = Hs[j][x];
            std::vector<C>& HF = HFs[j][x];
            const double h = seg_h[j];
            H.resize(N);
            HF.resize(N);
            G[x].resize(N);
            double db1 = p.beta1[x] - p.beta1[p.ref_field];       // Delta beta1_x (R7, R10)
            for (int k = 0; k < N; ++k) {
                double om = omega(k);
                // D_x(Omega) = -Delta beta1_x Omega + (beta2_x / 2) Omega^2          Eq. 5, R7/R8
                //              - (beta3_x / 6) Omega^3      third-order dispersion in its physical form +(beta3/6) d^3/dtau^3
                //                (R7: the term as printed in Eq. 5 would be a gain, not a phase)
                double D = -db1 * om + 0.5 * p.beta2[x] * om * om - p.beta3[x] / 6.0 * om * om * om;
                // H_x = exp( (-alpha_x/2 + i D_x) h/2 )                              half step
                std::complex<double> e = std::exp(std::complex<double>(-0.5 * p.alpha[x], D) * (0.5 * h));
                H[k] = C((R)e.real(), (R)e.imag());
                // full step exp( (-alpha_x/2 + i D_x) h ), used by the N/2 - L - N/2 ordering (Eq. 11)
                std::complex<double> ef = std::exp(std::complex<double>(-0.5 * p.alpha[x], D) * h);
                HF[k] = C((R)ef.real(), (R)ef.imag());
                // G_x = exp( i (gamma_x/2) Omega^2 - i Omega DeltaT_x )              L145, R13, R14
                double ph = 0.5 * p.gdd[x] * om * om - om * p.delta_T[x];
                G[x][k] = C((R)std::cos(ph), (R)std::sin(ph));
            }
            boundary_needs_transform[x] = (p.gdd[x] != 0.0) || (p.delta_T[x] != 0.0);   // L284
        }
        // the position inside the pass is kept; step size and couplings are those of the current segment
        h = seg_h[seg];
        for (int x = 0; x < F; ++x) kappa[x] = seg_kappa[seg][x];
    }

    void linear_half_step() {
        for (int x = 0; x < F; ++x) {
            fft.transform(A[x].data(), false);
            for (int k = 0; k < N; ++k) A[x][k] = A[x][k] * Hs[seg][x][k];
            fft.transform(A[x].data(), true);
        }
    }

    // right-hand side of Eqs 2-4 without L, at position zz
    void rhs(double zz, const C* y, C* f) const {
        double ph = seg_dk(seg) * zz;                  // dk of the current crystal segment, z from its entrance
        C em((R)std::cos(ph), (R)(-std::sin(ph)));    // e^{-i dk z}
        C ep((R)std::cos(ph), (R)(std::sin(ph)));     // e^{+i dk z}
        const C I(0, 1);
        if (F == 3) {
            f[0] = I * (R)kappa[0] * y[1] * y[2] * em;
            f[1] = I * (R)kappa[1] * y[0] * std::conj(y[2]) * ep;
            f[2] = I * (R)kappa[2] * y[0] * std::conj(y[1]) * ep;
        } else {
            // degenerate (reading R5): dA_p/dz = i (kappa_p/2) A_s^2 e^{-i dk z};
            //                          dA_s/dz = i kappa_s A_p A_s^* e^{+i dk z}
            f[0] = I * (R)(0.5 * kappa[0]) * y[1] * y[1] * em;
            f[1] = I * (R)kappa[1] * y[0] * std::conj(y[1]) * ep;
        }
    }

    void linear_full_step() {
        for (int x = 0; x < F; ++x) {
            fft.transform(A[x].data(), false);
            for (int k = 0; k < N; ++k) A[x][k] = A[x][k] * HFs[seg][x][k];
            fft.transform(A[x].data(), true);
        }
    }

    // one classic RK4 step of size hstep of the coupling terms, from position z0 (R3, R4)
    void nonlinear_step(double z0, double hstep) {
        const R hh = (R)hstep;
        const double z = z0, h = hstep;
        for (int n = 0; n < N; ++n) {
            C y[3], k1[3], k2[3], k3[3], k4[3], t[3];
            for (int x = 0; x < F; ++x) y[x] = A[x][n];
            rhs(z, y, k1);
            for (int x = 0; x < F; ++x) t[x] = y[x] + (R)0.5 * hh * k1[x];
            rhs(z + 0.5 * h, t, k2);
            for (int x = 0; x < F; ++x) t[x] = y[x] + (R)0.5 * hh * k2[x];
            rhs(z + 0.5 * h, t, k3);
            for (int x = 0; x < F; ++x) t[x] = y[x] + hh * k3[x];
            rhs(z + h, t, k4);
            for (int x = 0; x < F; ++x)
                A[x][n] = y[x] + (hh / (R)6) * (k1[x] + (R)2 * k2[x] + (R)2 * k3[x] + k4[x]);
        }
    }

    void z_step() {
        if (p.splitting == 0) {          // L/2 - N - L/2 ("its counterpart"; north_star; R2)
            linear_half_step();
            nonlinear_step(z, h);
            linear_half_step();
        } else {                          // N/2 - L - N/2, the order the paper implements (Eq. 10-11)
            nonlinear_step(z, 0.5 * h);
            linear_full_step();
            nonlinear_step(z + 0.5 * h, 0.5 * h);
        }
        z += h;
        ++seg_step;
    }

    bool at_pass_start() const { return seg == 0 && seg_step == 0; }
    // one z-step of the pass; moves on to the next crystal segment when the current one is finished.
    // false if the pass is already complete
    bool pass_step() {
        while (seg_step >= seg_nz(seg)) {
            if (seg + 1 >= K) return false;
            enter_segment(seg + 1);
        }
        z_step();
        return true;
    }

    int steps_done() const {
        int t = seg_step;
        for (int j = 0; j < seg; ++j) t += seg_nz(j);
        return t;
    }

    int propagate(int nsteps) {
        if (nsteps < 0) return 1;
        // error if it would pass the end of the last crystal
        if (steps_done() + nsteps > steps_per_pass()) return 5;
        for (int s = 0; s < nsteps; ++s) pass_step();
        return 0;
    }

    void boundary() {
        for (int x = 0; x < F; ++x) {
            EX[x] = A[x];
            if (p.resonant[x]) {
                if (boundary_needs_transform[x]) {
                    fft.transform(A[x].data(), false);
                    for (int k = 0; k < N; ++k) A[x][k] = A[x][k] * G[x][k];
                    fft.transform(A[x].data(), true);
                }
                double r = std::sqrt(p.R[x]);
                C m((R)(r * std::cos(p.delta_rad[x])), (R)(r * std::sin(p.delta_rad[x])));
                for (int n = 0; n < N; ++n) A[x][n] = A[x][n] * m;
                // intracavity EOM, last element of the boundary (Listing 3, after AddGDD and AddPhase):
                // A(tau) -> A(tau) exp(i beta sin(2 pi f_pm tau))          PAPER.md:L149-154; tau_n = (n - N/2) dt (R19)
                if (p.eom_beta[x] != 0.0) {
                    double dt = p.window_s / (double)N;
                    for (int n = 0; n < N; ++n) {
                        double tau = (double)(n - N / 2) * dt;
                        double ph = p.eom_beta[x] * std::sin(2.0 * kPi * p.eom_f[x] * tau);
                        A[x][n] = A[x][n] * C((R)std::cos(ph), (R)std::sin(ph));
                    }
                }
                // resonant pump (reading R24): the input coupler of power reflectivity R_p transmits the external pump S_p
                if (x == 0) {
                    R t = (R)std::sqrt(1.0 - p.R[x]);
                    for (int n = 0; n < N; ++n) A[x][n] = A[x][n] + t * S[x][n];
                }
            } else {
                A[x] = S[x];
            }
        }
        enter_segment(0);
        z = 0.0;
    }

    int roundtrips(int n) {
        if (n < 0) return 1;
        if (!at_pass_start()) return 5;
        for (int m = 0; m < n; ++m) {
            enter_segment(0);
            z = 0.0;
            while (pass_step()) {}
            boundary();
        }
        return 0;
    }
};

struct Handle {
    bool is_float;
    Oracle<double>* d;
    Oracle<float>* f;
};

template <class R>
void set_vec(std::vector<std::complex<R>>& v, const double* reim) {
    for (size_t i = 0; i < v.size(); ++i) v[i] = std::complex<R>((R)reim[2 * i], (R)reim[2 * i + 1]);
}
template <class R>
void get_vec(const std::vector<std::complex<R>>& v, double* reim) {
    for (size_t i = 0; i < v.size(); ++i) {
        reim[2 * i] = (double)v[i].real();
        reim[2 * i + 1] = (double)v[i].imag();
    }
}

}  // namespace

extern "C" {

void* opo_oracle_create(int n_fields, int log2n, double window_s, int nz, double length_m,
                        double dk_per_m, double d_eff, const double* lambda_m, const double* n_index,
                        const double* beta1, const double* beta2, const double* alpha, int ref_field,
                        const int* resonant, const double* R, const double* delta_rad,
                        const double* delta_T, const double* gdd, int use_float) {
    if (n_fields < 2 || n_fields > 3 || log2n < 1 || log2n > 24 || nz <= 0) return nullptr;
    Params p;
    std::memset(&p, 0, sizeof(p));
    p.n_fields = n_fields; p.log2n = log2n; p.nz = nz; p.ref_field = ref_field;
    p.window_s = window_s; p.length_m = length_m; p.dk_per_m = dk_per_m; p.d_eff = d_eff;
    for (int x = 0; x < n_fields; ++x) {
        p.lambda_m[x] = lambda_m[x]; p.n_index[x] = n_index[x]; p.beta1[x] = beta1[x];
        p.beta2[x] = beta2[x]; p.alpha[x] = alpha[x]; p.resonant[x] = resonant[x]; p.R[x] = R[x];
        p.delta_rad[x] = delta_rad[x]; p.delta_T[x] = delta_T[x]; p.gdd[x] = gdd[x];
    }
    Handle* hnd = new Handle{use_float != 0, nullptr, nullptr};
    if (use_float) { hnd->f = new Oracle<float>(); hnd->f->init(p); }
    else           { hnd->d = new Oracle<double>(); hnd->d->init(p); }
    return hnd;
}

void opo_oracle_destroy(void* h) {
    Handle* hnd = (Handle*)h;
    if (!hnd) return;
    delete hnd->d; delete hnd->f; delete hnd;
}

// which: 0 = current state only, 1 = stored input S_x only, 2 = both
void opo_oracle_set_field(void* h, int field, int which, const double* reim) {
    Handle* hnd = (Handle*)h;
    if (hnd->is_float) {
        if (which != 1) set_vec(hnd->f->A[field], reim);
        if (which != 0) set_vec(hnd->f->S[field], reim);
    } else {
        if (which != 1) set_vec(hnd->d->A[field], reim);
        if (which != 0) set_vec(hnd->d->S[field], reim);
    }
}

// 0: L/2 - N - L/2 (default), 1: N/2 - L - N/2 (Eq. 10-11)
void opo_oracle_set_splitting(void* h, int splitting) {
    Handle* hnd = (Handle*)h;
    if (hnd->is_float) hnd->f->p.splitting = splitting;
    else               hnd->d->p.splitting = splitting;
}

// third-order dispersion of field x; rebuilds the multiplier tables
void opo_oracle_set_beta3(void* h, int field, double beta3_s3_per_m) {
    Handle* hnd = (Handle*)h;
    if (hnd->is_float) { hnd->f->p.beta3[field] = beta3_s3_per_m; hnd->f->build_tables(); }
    else               { hnd->d->p.beta3[field] = beta3_s3_per_m; hnd->d->build_tables(); }
}

// crystal segments in series (reading R25); n = 0 restores the single crystal of opo_oracle_create.  Only at the start of a pass.
int opo_oracle_set_segments(void* h, int n, const double* len, const double* dk, const double* deff, const int* nz) {
    Handle* hnd = (Handle*)h;
    if (n < 0 || n > 8) return 1;
    for (int j = 0; j < n; ++j) if (!(len[j] > 0.0) || nz[j] <= 0) return 1;
    auto apply = [&](Params& p) {
        p.n_seg = n;
        for (int j = 0; j < n; ++j) { p.seg_len[j] = len[j]; p.seg_dk[j] = dk[j]; p.seg_deff[j] = deff[j]; p.seg_nz[j] = nz[j]; }
    };
    if (hnd->is_float) { if (!hnd->f->at_pass_start()) return 5; apply(hnd->f->p); hnd->f->build_tables(); }
    else               { if (!hnd->d->at_pass_start()) return 5; apply(hnd->d->p); hnd->d->build_tables(); }
    return 0;
}

// intracavity phase modulator on (resonant) field x; beta = 0 switches it off
void opo_oracle_set_eom(void* h, int field, double beta_rad, double f_hz) {
    Handle* hnd = (Handle*)h;
    if (hnd->is_float) { hnd->f->p.eom_beta[field] = beta_rad; hnd->f->p.eom_f[field] = f_hz; }
    else               { hnd->d->p.eom_beta[field] = beta_rad; hnd->d->p.eom_f[field] = f_hz; }
}

int opo_oracle_propagate(void* h, int nz) {
    Handle* hnd = (Handle*)h;
    return hnd->is_float ? hnd->f->propagate(nz) : hnd->d->propagate(nz);
}

int opo_oracle_roundtrips(void* h, int n) {
    Handle* hnd = (Handle*)h;
    return hnd->is_float ? hnd->f->roundtrips(n) : hnd->d->roundtrips(n);
}

// which: 0 = current, 1 = exit (z = L of the last pass, pre-mirror); domain: 0 = time, 1 = frequency
void opo_oracle_get_field(void* h, int field, int which, int domain, double* reim) {
    Handle* hnd = (Handle*)h;
    if (hnd->is_float) {
        std::vector<std::complex<float>> v = which ? hnd->f->EX[field] : hnd->f->A[field];
        if (domain) hnd->f->fft.transform(v.data(), false);
        get_vec(v, reim);
    } else {
        std::vector<std::complex<double>> v = which ? hnd->d->EX[field] : hnd->d->A[field];
        if (domain) hnd->d->fft.transform(v.data(), false);
        get_vec(v, reim);
    }
}

double opo_oracle_kappa(void* h, int field) {
    Handle* hnd = (Handle*)h;
    return hnd->is_float ? hnd->f->kappa[field] : hnd->d->kappa[field];
}

double opo_oracle_z(void* h) {
    Handle* hnd = (Handle*)h;
    return hnd->is_float ? hnd->f->z : hnd->d->z;
}

// standalone transform of the oracle's own FFT (pin P1)
void opo_oracle_fft(int log2n, int inverse, double* reim) {
    Fft<double> f;
    f.init(log2n);
    std::vector<std::complex<double>> v((size_t)1 << log2n);
    set_vec(v, reim);
    f.transform(v.data(), inverse != 0);
    get_vec(v, reim);
}

}  // extern "C"
