// opo_api.cu -- the C ABI of include/opo.h: handle, fp64 host tables, engine selection, launches.
//
// Everything numerical on the path runs in the kernels of opo_kernels.cuh / opo_resident.cuh /
// opo_large.cuh; the host only builds constant tables in fp64 (dispersion multipliers, boundary
// multipliers, FFT twiddles, dk phases) and sequences launches.  There is no CPU fallback.
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include <cuda_runtime.h>
#include <dlfcn.h>

#include "../../include/opo.h"
#include "opo_internal.h"

namespace {

using cd = std::complex<double>;
constexpr double kPi = 3.14159265358979323846264338327950288;

thread_local std::string g_create_error;

// ---- radix plan on the host (mirror of opo::plan<L> in opo_fft.cuh) ------------------------------------
struct HostPlan {
    int L = 0, P = 0;
    int rbits[8] = {0}, sbits[8] = {0}, tw_offset[9] = {0};
    int tw_total = 0;
    explicit HostPlan(int L_) : L(L_) {
        // pass 0: radix 4; the remaining L - 2 bits: radix 16 as often as possible, then 8 / 4
        const int L1 = L - 2;
        const int rem = L1 % 4;
        const int n16 = (rem == 1) ? (L1 / 4 - 1) : (L1 / 4);
        P = 1 + n16 + (rem == 0 ? 0 : (rem == 1 ? 2 : 1));
        int used = 0, off = 0;
        for (int p = 0; p < P; ++p) {
            int rb;
            const int q = p - 1;
            if (p == 0) rb = 2;
            else if (q < n16) rb = 4;
            else if (rem == 1) rb = (q == n16) ? 3 : 2;
            else if (rem == 2) rb = 2;
            else rb = 3;
            rbits[p] = rb;
            used += rb;
            sbits[p] = L - used;
            tw_offset[p] = off;
            off += ((1 << rb) - 1) << sbits[p];
        }
        tw_offset[P] = off;
        tw_total = off;
    }
    // position after all forward passes -> frequency index:  pos = sum_p k_p S_p,  k = sum_p k_p R_1..R_{p-1}
    int freq_of_pos(int pos) const {
        int k = 0, mult = 1;
        for (int p = 0; p < P; ++p) {
            const int kp = (pos >> sbits[p]) & ((1 << rbits[p]) - 1);
            k += kp * mult;
            mult <<= rbits[p];
        }
        return k;
    }
};

// (c, s) on the unit circle -> floats bracketing the exact values, chosen so that c^2 + s^2 is
// closest to 1: twiddle *magnitude* error is what accumulates over z-steps (see opo_fft.cuh).
void round_unit(double c, double s, float* cf, float* sf) {
    float cc[2] = {(float)c, (float)c}, ss[2] = {(float)s, (float)s};
    if ((double)cc[0] != c) cc[1] = std::nextafterf(cc[0], (double)cc[0] < c ? INFINITY : -INFINITY);
    if ((double)ss[0] != s) ss[1] = std::nextafterf(ss[0], (double)ss[0] < s ? INFINITY : -INFINITY);
    double best = 1e300;
    for (int i = 0; i < 2; ++i)
        for (int j = 0; j < 2; ++j) {
            double e = std::fabs((double)cc[i] * cc[i] + (double)ss[j] * ss[j] - 1.0);
            if (e < best) { best = e; *cf = cc[i]; *sf = ss[j]; }
        }
}

}  // namespace

struct opo_handle {
    opo_crystal crystal{};
    opo_fields fields{};
    opo_grid grid{};
    int N = 0, L = 0, F = 0, B = 0, nz = 0;
    bool dbl = false;
    size_t esz = 8;            // bytes per complex element
    double h = 0.0;
    double kappa[3] = {0, 0, 0};
    cudaStream_t stream = nullptr;
    int sm_count = 0;

    // per-instance parameters
    std::vector<double> dk;                 // [B]
    std::vector<double> dT[3], drad[3], gdd[3];
    bool per_inst_boundary[3] = {false, false, false};
    bool tables_dirty = true, phase_dirty = true;

    // device state
    void* cur[3] = {nullptr, nullptr, nullptr};
    void* S[3] = {nullptr, nullptr, nullptr};
    void* exitb[3] = {nullptr, nullptr, nullptr};
    void* SH[3] = {nullptr, nullptr, nullptr};
    void* scratch = nullptr;
    // device tables
    void* tw = nullptr;
    int* perm = nullptr;
    void* tabH[3] = {nullptr, nullptr, nullptr};
    void* tabH2[3] = {nullptr, nullptr, nullptr};
    void* tabGM[3] = {nullptr, nullptr, nullptr};
    void* tabHB[3] = {nullptr, nullptr, nullptr};
    void* tabHG[3] = {nullptr, nullptr, nullptr};      // H G m / N: last half-step + boundary, when a modulator follows
    size_t tabB_count[3] = {0, 0, 0};      // instances allocated for GM / HB (1 or B)
    void* mirror[3] = {nullptr, nullptr, nullptr};
    void* eom[3] = {nullptr, nullptr, nullptr};       // [N] exp(i beta sin(2 pi f tau_n)) or null
    double eom_beta[3] = {0, 0, 0}, eom_f[3] = {0, 0, 0};
    double beta3[3] = {0, 0, 0};                      // third-order dispersion [s^3/m] (opo_set_beta3)
    int splitting = 0;                                // OPO_OPT_SPLITTING
    int* rt_flags = nullptr;                          // resident engine, split launches: [B][F] round trips done
    // cuFFT baseline engine: plan over [B][N] and natural-order tables (H, H^2, G m; all with 1/N folded in)
    int cufft_plan = -1;
    void* natH[3] = {nullptr, nullptr, nullptr};
    void* natH2[3] = {nullptr, nullptr, nullptr};
    void* natGM[3] = {nullptr, nullptr, nullptr};
    size_t natGM_count[3] = {0, 0, 0};
    bool boundary_fft[3] = {false, false, false};
    void* phase = nullptr;
    int* flag = nullptr;

    // large-N engine (four-step decomposition N = N1 x N2, opo_large.cuh)
    bool large = false;
    int L1 = 0, L2 = 0;
    void* tw2 = nullptr;
    void* wlo = nullptr;
    void* whi = nullptr;
    int* perm2 = nullptr;
    void* scratch2 = nullptr;
    unsigned long long* barrier = nullptr;
    opo::LargeInfo linfo{};
    std::vector<int> host_perm1, host_perm2;
    size_t tab_esz = 8;        // bytes per table entry (large engine, c64: hi + lo = 16)

    int z_steps = 0;
    bool run_started = false;       // a z-step has been taken since opo_create (opo_set_pump: empty-cavity start of a resonant pump)
    size_t phase_bytes = 0;         // capacity of `phase`
    int engine_opt = OPO_ENGINE_AUTO;
    bool resident_ok = false;
    opo::ResidentInfo rinfo{};
    // crystal segments in series (opo_set_segments, reading R25).  n_seg = 1: the crystal of opo_create.
    // nz is the number of z-steps of a whole pass; h and kappa above are those of segment 0.
    struct Segment { double len = 0, dk = 0, deff = 0, hstep = 0, kappa[3] = {0, 0, 0}; int nz = 0; };
    int n_seg = 1;
    Segment seg[8];
    void* segH[8][3] = {};                            // per-segment tables, allocated when n_seg > 1 (streaming engine):
    void* segH2[8][3] = {};                           //   half step H_j / N, full step H_j^2 / N,
    void* segHX[8][3] = {};                           //   H_j H_{j+1} / N across the junction of two crystals
    bool solo_ok = false;                             // solo engine (one CTA per instance, fields in shared + tensor memory)
    opo::ResidentInfo sinfo{};                        // max_clusters = co-resident CTAs on the device
    int tab_cycle = 1;                                // roundings of H and of H^2 cycled through by the on-chip engines (fp32: 16; build_tables)
    // Linear operators / half-step tables / full-step tables applied by this handle since opo_create (kept modulo 2^20, a
    // multiple of every cycle length).  They go into every launch (ResidentArgs::op0, hq0, fq0; LargeArgs::op0) so that the
    // table cycles and the bunched constant corrections continue across calls instead of restarting at each call's first
    // operator: accuracy then does not depend on how a run is cut into opo_propagate / opo_roundtrips calls.  Never reset;
    // two handles driven by the same sequence of calls give bitwise the same fields.
    int op_count = 0, hq_count = 0, fq_count = 0;
    bool wide_ok = false;                             // wide engine (a cluster of 4 F CTAs per instance)
    opo::ResidentInfo winfo{};                        // max_clusters = co-resident clusters of 4 F CTAs
    int wide_g_opt = 0;                               // OPO_OPT_WIDE_SUBBLOCKS: 0 = AUTO, 1 | 2 = sub-blocks per CTA
    opo::ResidentInfo winfo2{};                       // ... of 2 F CTAs holding two sub-blocks each (0: that variant is unavailable)
    int device = 0;
    long long launches = 0;
    std::string err;
    std::vector<int> host_perm;

    size_t field_bytes() const { return (size_t)B * N * esz; }
};

namespace {


// ---- cuFFT, for the internal baseline engine only (BASELINE.json north_star item (d): "a cuFFT + separate
// elementwise-kernel pipeline kept as an internal baseline, not the product").  Loaded with dlopen on first use so
// that libopo.so itself has no dependency on it.
typedef int cufftHandle_t;
struct CufftApi {
    void* lib = nullptr;
    int (*PlanMany)(cufftHandle_t*, int, int*, int*, int, int, int*, int, int, int, int) = nullptr;
    int (*SetStream)(cufftHandle_t, cudaStream_t) = nullptr;
    int (*ExecC2C)(cufftHandle_t, void*, void*, int) = nullptr;
    int (*ExecZ2Z)(cufftHandle_t, void*, void*, int) = nullptr;
    int (*Destroy)(cufftHandle_t) = nullptr;
    bool ok = false;
};
CufftApi& cufft_api() {
    static CufftApi api;
    static bool tried = false;
    if (!tried) {
        tried = true;
        const char* names[] = {"libcufft.so.11", "libcufft.so", "/usr/local/cuda/lib64/libcufft.so.11", "/usr/local/cuda/lib64/libcufft.so"};
        for (const char* n : names) { api.lib = dlopen(n, RTLD_NOW | RTLD_LOCAL); if (api.lib) break; }
        if (api.lib) {
            api.PlanMany = (decltype(api.PlanMany))dlsym(api.lib, "cufftPlanMany");
            api.SetStream = (decltype(api.SetStream))dlsym(api.lib, "cufftSetStream");
            api.ExecC2C = (decltype(api.ExecC2C))dlsym(api.lib, "cufftExecC2C");
            api.ExecZ2Z = (decltype(api.ExecZ2Z))dlsym(api.lib, "cufftExecZ2Z");
            api.Destroy = (decltype(api.Destroy))dlsym(api.lib, "cufftDestroy");
            api.ok = api.PlanMany && api.SetStream && api.ExecC2C && api.ExecZ2Z && api.Destroy;
        }
    }
    return api;
}
constexpr int kCufftC2C = 0x29, kCufftZ2Z = 0x69, kCufftForward = -1, kCufftInverse = 1;

int fail(opo_handle* h, int code, const std::string& msg) {
    if (h) h->err = msg; else g_create_error = msg;
    return code;
}

#define OPO_CUDA(h, call)                                                                  \
    do {                                                                                   \
        cudaError_t e_ = (call);                                                           \
        if (e_ != cudaSuccess)                                                             \
            return fail((h), OPO_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
    } while (0)

// upload complex<double> values as float2 / double2
int upload_complex(opo_handle* h, void* dst, const cd* src, size_t count, bool unit_twiddles = false) {
    if (h->dbl) {
        OPO_CUDA(h, cudaMemcpyAsync(dst, src, count * sizeof(cd), cudaMemcpyHostToDevice, h->stream));
        OPO_CUDA(h, cudaStreamSynchronize(h->stream));
    } else {
        std::vector<float> tmp(2 * count);
        for (size_t i = 0; i < count; ++i) {
            if (unit_twiddles) round_unit(src[i].real(), src[i].imag(), &tmp[2 * i], &tmp[2 * i + 1]);
            else { tmp[2 * i] = (float)src[i].real(); tmp[2 * i + 1] = (float)src[i].imag(); }
        }
        OPO_CUDA(h, cudaMemcpyAsync(dst, tmp.data(), tmp.size() * sizeof(float), cudaMemcpyHostToDevice, h->stream));
        OPO_CUDA(h, cudaStreamSynchronize(h->stream));
    }
    return OPO_OK;
}

// upload table values in the entry format of the engine: plain complex, or (large engine, c64) hi + lo
int upload_table(opo_handle* h, void* dst, const cd* src, size_t count) {
    if (!(h->large && !h->dbl)) return upload_complex(h, dst, src, count);
    std::vector<float> tmp(4 * count);
    for (size_t i = 0; i < count; ++i) {
        const float hr = (float)src[i].real(), hi = (float)src[i].imag();
        tmp[4 * i] = hr;
        tmp[4 * i + 1] = hi;
        tmp[4 * i + 2] = (float)(src[i].real() - (double)hr);
        tmp[4 * i + 3] = (float)(src[i].imag() - (double)hi);
    }
    OPO_CUDA(h, cudaMemcpyAsync(dst, tmp.data(), tmp.size() * sizeof(float), cudaMemcpyHostToDevice, h->stream));
    OPO_CUDA(h, cudaStreamSynchronize(h->stream));
    return OPO_OK;
}

// Omega_k = 2 pi k' / (N dt), natural FFT order, Nyquist bin negative (R9)
double omega_of(const opo_handle* h, int k) {
    const int kp = (k < h->N / 2) ? k : k - h->N;
    return 2.0 * kPi * (double)kp / h->grid.window_s;
}

// natural-order frequency multiplier -> register layout of mid_pass_smem: tab[kk * NBF + u] = M[freq(u R + kk)]
void to_mid_layout(const opo_handle* h, const HostPlan& pl, const cd* M, cd* out) {
    const int R = 1 << pl.rbits[pl.P - 1];
    const int NBF = h->N / R;
    for (int u = 0; u < NBF; ++u)
        for (int kk = 0; kk < R; ++kk) out[(size_t)kk * NBF + u] = M[h->host_perm[u * R + kk]];
}

// natural-order frequency multiplier -> layout of the large engine's row pass: row r holds k1 = perm1[r],
// inside the row the mid-pass layout of the row plan: out[r N2 + kk NBF + u] = M[k1 + N1 perm2[u R + kk]]
void to_large_layout(const opo_handle* h, const HostPlan& pl2, const cd* M, cd* out) {
    const int N1 = 1 << h->L1, N2 = 1 << h->L2;
    const int R = 1 << pl2.rbits[pl2.P - 1];
    const int NBF = N2 / R;
    for (int r = 0; r < N1; ++r) {
        const int k1 = h->host_perm1[r];
        for (int u = 0; u < NBF; ++u)
            for (int kk = 0; kk < R; ++kk)
                out[(size_t)r * N2 + (size_t)kk * NBF + u] = M[(size_t)k1 + (size_t)N1 * h->host_perm2[u * R + kk]];
    }
}

void to_engine_layout(const opo_handle* h, const HostPlan& pl, const cd* M, cd* out) {
    if (h->large) to_large_layout(h, pl, M, out);
    else to_mid_layout(h, pl, M, out);
}

}  // namespace

namespace {

// ---- tables ----------------------------------------------------------------------------------------------
// H_x[k]  = exp((-alpha_x/2 + i D_x(Omega_k)) h/2),  D_x = -(beta1_x - beta1_ref) Omega + (beta2_x/2) Omega^2
//           (Eq. 5 with readings R7, R8, R10)
// G_x[k]  = exp(i (gdd_x/2) Omega_k^2 - i Omega_k delta_T_x)     (R13, R14)
// m_x     = sqrt(R_x) exp(i delta_x)                              (Eq. 6)
// Device tables carry the 1/N of the inverse transform and are stored in mid-pass layout:
//   tabH = H/N, tabH2 = H^2/N, tabGM = G m/N, tabHB = H^2 G m/N (half-steps merged across the boundary).
int build_tables(opo_handle* h) {
    const int N = h->N, F = h->F, B = h->B, K = h->n_seg;
    HostPlan pl(h->large ? h->L2 : h->L);
    const double invN = 1.0 / (double)N;
    const double h0 = h->seg[0].hstep, hl = h->seg[K - 1].hstep;      // first and last step size of a pass
    std::vector<cd> Hh(N), M(N), lay(N), Dx(N);
    // fp32, on-chip engines: a cycle of roundings of a table M (H^2, and likewise H) with error feedback.  One rounded table
    // T = fl(M) puts the same 3e-8 of error per bin into every application (coherent: 3e4 z-steps of C4 turn it into ~5e-4).
    // Here table j of the cycle is T_j = fl(M / r_{j-1}), r_j = r_{j-1} T_j / M the relative error of the product applied so
    // far, so after any number of applications the product of the tables is M^n to ONE rounding, and the drift per
    // application falls by the cycle length.  Copy 0 is fl(M) itself (the host-sequenced baseline engines, which do not
    // cycle, use it).  The kernels pick the copy by the handle's running count of uses (op_count / hq_count / fq_count).
    auto upload_cycle = [&](void* dst, const std::vector<cd>& Mt) -> int {
        if (h->tab_cycle <= 1) return OPO_OK;
        std::vector<cd> ratio(N, cd(1.0, 0.0));
        for (int j = 0; j < h->tab_cycle; ++j) {
            for (int k = 0; k < N; ++k) {
                const cd want = Mt[k] / ratio[k];
                const cd t((double)(float)want.real(), (double)(float)want.imag());
                Hh[k] = t;
                if (Mt[k] != cd(0.0, 0.0)) ratio[k] *= t / Mt[k];
            }
            to_engine_layout(h, pl, Hh.data(), lay.data());
            if (int rc = upload_table(h, (char*)dst + (size_t)j * N * h->tab_esz, lay.data(), N)) return rc;
        }
        return OPO_OK;
    };
    for (int x = 0; x < F; ++x) {
        const double db1 = h->fields.beta1_s_per_m[x] - h->fields.beta1_s_per_m[h->fields.ref_field];
        const double b2 = h->fields.beta2_s2_per_m[x], al = h->fields.alpha_per_m[x];
        const double b3 = h->beta3[x] / 6.0;            // D_x -= (beta3_x/6) Omega^3   (reading R7)
        for (int k = 0; k < N; ++k) {
            const double om = omega_of(h, k);
            Dx[k] = cd(-0.5 * al, -db1 * om + 0.5 * b2 * om * om - b3 * om * om * om);      // -alpha_x/2 + i D_x(Omega_k)
        }
        // first linear operator of a pass / of a call: half step of segment 0
        for (int k = 0; k < N; ++k) M[k] = std::exp(Dx[k] * (0.5 * h0)) * invN;
        to_engine_layout(h, pl, M.data(), lay.data());
        if (int rc = upload_table(h, h->tabH[x], lay.data(), N)) return rc;
        if (int rc = upload_cycle(h->tabH[x], M)) return rc;       // (the half-steps at the ends of every call: z-step-by-z-step
                                                                   //  driving applies nothing else)
        if (h->natH[x]) if (int rc = upload_complex(h, h->natH[x], M.data(), N)) return rc;        // cuFFT baseline: natural order
        for (int k = 0; k < N; ++k) M[k] = std::exp(Dx[k] * h0) * invN;                            // H^2 evaluated directly in fp64
        to_engine_layout(h, pl, M.data(), lay.data());
        if (int rc = upload_table(h, h->tabH2[x], lay.data(), N)) return rc;
        if (int rc = upload_cycle(h->tabH2[x], M)) return rc;
        if (h->natH2[x]) if (int rc = upload_complex(h, h->natH2[x], M.data(), N)) return rc;
        if (K > 1) {
            // several crystals: per segment the half step, the full step and the junction H_j H_{j+1}
            for (int j = 0; j < K; ++j) {
                const double hj = h->seg[j].hstep;
                for (int v = 0; v < 3; ++v) {
                    if (v == 2 && j == K - 1) continue;
                    const double len = v == 0 ? 0.5 * hj : (v == 1 ? hj : 0.5 * (hj + h->seg[j + 1].hstep));
                    void** dst = v == 0 ? &h->segH[j][x] : (v == 1 ? &h->segH2[j][x] : &h->segHX[j][x]);
                    if (!*dst && cudaMalloc(dst, (size_t)N * h->tab_esz) != cudaSuccess) { cudaGetLastError(); return fail(h, OPO_ERR_ALLOC, "cudaMalloc of segment tables failed"); }
                    for (int k = 0; k < N; ++k) M[k] = std::exp(Dx[k] * len) * invN;
                    to_engine_layout(h, pl, M.data(), lay.data());
                    if (int rc = upload_table(h, *dst, lay.data(), N)) return rc;
                }
            }
        }

        if (!h->fields.resonant[x]) continue;
        // boundary tables, shared or per instance
        const size_t need = h->per_inst_boundary[x] ? (size_t)B : 1;
        if (h->tabB_count[x] != need) {
            if (h->tabGM[x]) cudaFree(h->tabGM[x]);
            if (h->tabHB[x]) cudaFree(h->tabHB[x]);
            if (h->tabHG[x]) cudaFree(h->tabHG[x]);
            h->tabGM[x] = h->tabHB[x] = h->tabHG[x] = nullptr;
            if (cudaMalloc(&h->tabGM[x], need * N * h->tab_esz) != cudaSuccess ||
                cudaMalloc(&h->tabHB[x], need * N * h->tab_esz) != cudaSuccess ||
                cudaMalloc(&h->tabHG[x], need * N * h->tab_esz) != cudaSuccess)
            { cudaGetLastError(); return fail(h, OPO_ERR_ALLOC, "cudaMalloc of boundary tables failed"); }
            h->tabB_count[x] = need;
        }
        bool any_fft = false;
        std::vector<cd> mir(B);
        for (int b = 0; b < B; ++b) {
            if (h->gdd[x][b] != 0.0 || h->dT[x][b] != 0.0) any_fft = true;
            mir[b] = std::sqrt(h->fields.R[x]) * cd(std::cos(h->drad[x][b]), std::sin(h->drad[x][b]));
        }
        h->boundary_fft[x] = any_fft;
        if (int rc = upload_complex(h, h->mirror[x], mir.data(), B)) return rc;
        for (size_t b = 0; b < need; ++b) {
            for (int k = 0; k < N; ++k) {
                const double om = omega_of(h, k);
                const double ph = 0.5 * h->gdd[x][b] * om * om - om * h->dT[x][b];
                const cd gm = cd(std::cos(ph), std::sin(ph)) * mir[b];
                M[k] = gm * invN;
                // last half-step of the pass, boundary, first half-step of the next pass
                Hh[k] = std::exp(Dx[k] * (0.5 * (hl + h0))) * gm * invN;
            }
            to_engine_layout(h, pl, M.data(), lay.data());
            if (int rc = upload_table(h, (char*)h->tabGM[x] + b * N * h->tab_esz, lay.data(), N)) return rc;
            if (h->natH[x]) {      // cuFFT baseline
                if (h->natGM_count[x] != need) {
                    if (h->natGM[x]) cudaFree(h->natGM[x]);
                    h->natGM[x] = nullptr;
                    if (cudaMalloc(&h->natGM[x], need * N * h->esz) != cudaSuccess) { cudaGetLastError(); return fail(h, OPO_ERR_ALLOC, "cudaMalloc of baseline tables failed"); }
                    h->natGM_count[x] = need;
                }
                if (int rc = upload_complex(h, (char*)h->natGM[x] + b * N * h->esz, M.data(), N)) return rc;
            }
            to_engine_layout(h, pl, Hh.data(), lay.data());
            if (int rc = upload_table(h, (char*)h->tabHB[x] + b * N * h->tab_esz, lay.data(), N)) return rc;
            // H G m: the last half-step of a pass and the boundary, the modulator and the next half-step follow separately
            for (int k = 0; k < N; ++k) Hh[k] = std::exp(Dx[k] * (0.5 * hl)) * M[k];
            to_engine_layout(h, pl, Hh.data(), lay.data());
            if (int rc = upload_table(h, (char*)h->tabHG[x] + b * N * h->tab_esz, lay.data(), N)) return rc;
        }
    }
    h->tables_dirty = false;
    return OPO_OK;
}

// index of the first phase-table entry of z-step s (counted from the start of the pass): the table of an instance is the
// concatenation of one table per crystal segment, [q nz_j + 1] entries exp(i dk_j i h_j / q), q = 2 (4: N/2 - L - N/2),
// because z restarts at every crystal entrance (readings R4, R25)
int segment_of_step(const opo_handle* h, int s) {
    int j = 0, first = 0;
    while (j + 1 < h->n_seg && s >= first + h->seg[j].nz) { first += h->seg[j].nz; ++j; }
    return j;
}

// phase[b][j] = exp(i dk_b j h/2), j = 0 .. 2 nz   (R4: z from the crystal entrance)
int phase_stride(const opo_handle* h) { return (h->splitting ? 4 : 2) * h->nz + h->n_seg; }

// N/2 - L - N/2 (OPO_SPLITTING_NLN): the RK4 steps have size h/2, so the table runs in steps of h/4, j = 0 .. 4 nz
int build_phase(opo_handle* h) {
    const int stride = phase_stride(h), q = h->splitting ? 4 : 2;
    std::vector<cd> ph((size_t)h->B * stride);
    for (int b = 0; b < h->B; ++b) {
        size_t at = (size_t)b * stride;
        for (int j = 0; j < h->n_seg; ++j) {
            const double dk = j == 0 ? h->dk[b] : h->seg[j].dk;        // per-instance sweeps act on the first crystal
            const double dz = h->seg[j].hstep / (double)q;
            for (int i = 0; i <= q * h->seg[j].nz; ++i) {
                const double a = dk * dz * (double)i;
                ph[at++] = cd(std::cos(a), std::sin(a));
            }
        }
    }
    if (int rc = upload_complex(h, h->phase, ph.data(), ph.size())) return rc;
    h->phase_dirty = false;
    return OPO_OK;
}

std::vector<cd> pass_twiddles(const HostPlan& pl) {
    std::vector<cd> tw((size_t)std::max(pl.tw_total, 1));
    for (int p = 0; p < pl.P; ++p) {
        const int R = 1 << pl.rbits[p], S = 1 << pl.sbits[p];
        const double M = (double)R * (double)S;
        for (int k = 1; k < R; ++k)
            for (int t = 0; t < S; ++t) {
                const double a = -2.0 * kPi * (double)k * (double)t / M;
                tw[(size_t)pl.tw_offset[p] + (size_t)(k - 1) * S + t] = cd(std::cos(a), std::sin(a));
            }
    }
    return tw;
}

int upload_twiddles(opo_handle* h, void** dst, const std::vector<cd>& tw) {
    if (cudaMalloc(dst, tw.size() * h->esz) != cudaSuccess) return fail(h, OPO_ERR_ALLOC, "cudaMalloc(twiddles)");
    return upload_complex(h, *dst, tw.data(), tw.size(), /*unit_twiddles=*/true);
}

int upload_perm(opo_handle* h, int** dst, const std::vector<int>& perm) {
    if (cudaMalloc((void**)dst, perm.size() * sizeof(int)) != cudaSuccess) return fail(h, OPO_ERR_ALLOC, "cudaMalloc(perm)");
    OPO_CUDA(h, cudaMemcpy(*dst, perm.data(), perm.size() * sizeof(int), cudaMemcpyHostToDevice));
    return OPO_OK;
}

int build_fft_tables(opo_handle* h) {
    if (!h->large) {
        HostPlan pl(h->L);
        if (int rc = upload_twiddles(h, &h->tw, pass_twiddles(pl))) return rc;
        h->host_perm.resize(h->N);
        for (int pos = 0; pos < h->N; ++pos) h->host_perm[pos] = pl.freq_of_pos(pos);
        return upload_perm(h, &h->perm, h->host_perm);
    }
    // large engine: column plan (L1), row plan (L2), the two factors of W_N^{n2 k1}
    HostPlan pl1(h->L1), pl2(h->L2);
    const int N1 = 1 << h->L1, N2 = 1 << h->L2;
    if (int rc = upload_twiddles(h, &h->tw, pass_twiddles(pl1))) return rc;
    if (int rc = upload_twiddles(h, &h->tw2, pass_twiddles(pl2))) return rc;
    std::vector<cd> wlo(N1), whi(N2);
    for (int j = 0; j < N1; ++j) {
        const double a = -2.0 * kPi * (double)j / (double)h->N;
        wlo[j] = cd(std::cos(a), std::sin(a));
    }
    for (int j = 0; j < N2; ++j) {
        const double a = -2.0 * kPi * (double)j / (double)N2;      // W_N^{j N1} = W_N2^j
        whi[j] = cd(std::cos(a), std::sin(a));
    }
    if (int rc = upload_twiddles(h, &h->wlo, wlo)) return rc;
    if (int rc = upload_twiddles(h, &h->whi, whi)) return rc;
    h->host_perm1.resize(N1);
    h->host_perm2.resize(N2);
    for (int pos = 0; pos < N1; ++pos) h->host_perm1[pos] = pl1.freq_of_pos(pos);
    for (int pos = 0; pos < N2; ++pos) h->host_perm2[pos] = pl2.freq_of_pos(pos);
    if (int rc = upload_perm(h, &h->perm, h->host_perm1)) return rc;
    return upload_perm(h, &h->perm2, h->host_perm2);
}

int ensure_tables(opo_handle* h) {
    if (h->tables_dirty) if (int rc = build_tables(h)) return rc;
    if (h->phase_dirty) if (int rc = build_phase(h)) return rc;
    return OPO_OK;
}

void free_all(opo_handle* h) {
    for (int x = 0; x < 3; ++x) {
        void* ptrs[] = {h->cur[x], h->S[x], h->exitb[x], h->SH[x], h->tabH[x], h->tabH2[x], h->tabGM[x], h->tabHB[x], h->tabHG[x], h->mirror[x], h->eom[x], h->natH[x], h->natH2[x], h->natGM[x]};
        for (void* p : ptrs) if (p) cudaFree(p);
    }
    for (int j = 0; j < 8; ++j)
        for (int x = 0; x < 3; ++x) {
            void* ptrs[] = {h->segH[j][x], h->segH2[j][x], h->segHX[j][x]};
            for (void* p : ptrs) if (p) cudaFree(p);
        }
    if (h->cufft_plan >= 0 && cufft_api().ok) cufft_api().Destroy(h->cufft_plan);
    if (h->rt_flags) cudaFree(h->rt_flags);
    void* more[] = {h->scratch, h->tw, h->perm, h->phase, h->flag, h->tw2, h->wlo, h->whi, h->perm2, h->scratch2, h->barrier};
    for (void* p : more) if (p) cudaFree(p);
}

}  // namespace

extern "C" {

const char* opo_last_error(const opo_handle* h) { return h ? h->err.c_str() : g_create_error.c_str(); }

int opo_create(const opo_crystal* c, const opo_fields* f, const opo_grid* g, opo_handle** out) {
    if (!c || !f || !g || !out) return fail(nullptr, OPO_ERR_INVALID_ARG, "null argument");
    if (f->n_fields != 2 && f->n_fields != 3) return fail(nullptr, OPO_ERR_INVALID_ARG, "n_fields must be 2 or 3");
    if (g->precision != OPO_PRECISION_C64 && g->precision != OPO_PRECISION_C128)
        return fail(nullptr, OPO_ERR_INVALID_ARG, "precision must be 0 (c64) or 1 (c128)");
    if (g->log2_n < 4 || g->log2_n > 18) return fail(nullptr, OPO_ERR_INVALID_ARG, "log2_n outside [4, 18]");
    if (g->nz_per_pass <= 0 || g->batch <= 0 || !(g->window_s > 0.0) || !(c->length_m > 0.0))
        return fail(nullptr, OPO_ERR_INVALID_ARG, "nz_per_pass, batch, window_s and length_m must be positive");
    if (f->ref_field < 0 || f->ref_field >= f->n_fields) return fail(nullptr, OPO_ERR_INVALID_ARG, "ref_field out of range");
    for (int x = 0; x < f->n_fields; ++x) {
        if (!(f->lambda_m[x] > 0.0) || !(f->n[x] > 0.0)) return fail(nullptr, OPO_ERR_INVALID_ARG, "lambda and n must be positive");
        if (f->resonant[x] && !(f->R[x] >= 0.0 && f->R[x] <= 1.0)) return fail(nullptr, OPO_ERR_INVALID_ARG, "R outside [0, 1]");
    }
    const int maxL = (g->precision == OPO_PRECISION_C64) ? opo::kMaxLog2Smem : opo::kMaxLog2Smem - 1;
    if (g->log2_n < opo::kMinLog2 || g->log2_n > opo::kMaxLog2)
        return fail(nullptr, OPO_ERR_UNSUPPORTED, "grid size not supported (2^4 .. 2^18)");
    if (f->resonant[0] && g->log2_n > maxL)
        return fail(nullptr, OPO_ERR_UNSUPPORTED, "resonant pump: not on the large-N engine (N > 2^14, c128: > 2^13)");

    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess)
        return fail(nullptr, OPO_ERR_CUDA, std::string("no usable CUDA device: ") + cudaGetErrorString(cudaGetLastError()));
    if (prop.major != 10)
        return fail(nullptr, OPO_ERR_CUDA, "libopo is built for sm_100a only; device is sm_" + std::to_string(prop.major) + std::to_string(prop.minor));

    opo_handle* h = new opo_handle();
    h->crystal = *c; h->fields = *f; h->grid = *g;
    h->L = g->log2_n; h->N = 1 << g->log2_n; h->F = f->n_fields; h->B = g->batch; h->nz = g->nz_per_pass;
    h->dbl = (g->precision == OPO_PRECISION_C128);
    h->esz = h->dbl ? 16 : 8;
    h->large = h->L > maxL;
    h->L1 = h->L / 2;
    h->L2 = h->L - h->L1;
    h->tab_esz = h->large ? 16 : h->esz;
    h->tab_cycle = (!h->large && !h->dbl) ? 16 : 1;       // (a power of two: the kernels index with a mask)
    h->h = c->length_m / (double)g->nz_per_pass;
    h->sm_count = prop.multiProcessorCount;
    h->device = dev;
    for (int x = 0; x < h->F; ++x) h->kappa[x] = 2.0 * kPi * c->d_eff_m_per_V / (f->n[x] * f->lambda_m[x]);
    if (h->F == 2) h->kappa[0] *= 0.5;                                                                         // reading R5
    h->n_seg = 1;
    h->seg[0].len = c->length_m; h->seg[0].dk = c->dk_per_m; h->seg[0].deff = c->d_eff_m_per_V; h->seg[0].nz = h->nz; h->seg[0].hstep = h->h;
    for (int x = 0; x < 3; ++x) h->seg[0].kappa[x] = h->kappa[x];
    h->dk.assign(h->B, c->dk_per_m);
    for (int x = 0; x < 3; ++x) {
        h->dT[x].assign(h->B, x < h->F ? f->delta_T_s[x] : 0.0);
        h->drad[x].assign(h->B, x < h->F ? f->delta_rad[x] : 0.0);
        h->gdd[x].assign(h->B, x < h->F ? f->gdd_s2[x] : 0.0);
    }
    auto bail = [&](int code, const std::string& msg) { free_all(h); delete h; return fail(nullptr, code, msg); };
    const size_t fb = h->field_bytes();
    for (int x = 0; x < h->F; ++x) {
        void** arrs[] = {&h->cur[x], &h->S[x], &h->exitb[x], &h->SH[x]};
        for (void** p : arrs) {
            if (cudaMalloc(p, fb) != cudaSuccess) return bail(OPO_ERR_ALLOC, "cudaMalloc of field state failed");
            cudaMemset(*p, 0, fb);
        }
        if (cudaMalloc(&h->tabH[x], (size_t)h->tab_cycle * h->N * h->tab_esz) != cudaSuccess ||
            cudaMalloc(&h->tabH2[x], (size_t)h->tab_cycle * h->N * h->tab_esz) != cudaSuccess ||
            cudaMalloc(&h->mirror[x], (size_t)h->B * h->esz) != cudaSuccess)
            return bail(OPO_ERR_ALLOC, "cudaMalloc of tables failed");
    }
    h->phase_bytes = (size_t)h->B * (4 * (size_t)h->nz + 8) * h->esz;
    if (cudaMalloc(&h->scratch, fb) != cudaSuccess || cudaMalloc(&h->phase, h->phase_bytes) != cudaSuccess ||
        cudaMalloc((void**)&h->flag, sizeof(int)) != cudaSuccess)
        return bail(OPO_ERR_ALLOC, "cudaMalloc of scratch failed");
    if (int rc = build_fft_tables(h)) { std::string m = h->err; return bail(rc, m); }
    if (int rc = ensure_tables(h)) { std::string m = h->err; return bail(rc, m); }
    if (h->large) {
        if (cudaMalloc(&h->scratch2, fb) != cudaSuccess || cudaMalloc((void**)&h->barrier, sizeof(unsigned long long)) != cudaSuccess)
            return bail(OPO_ERR_ALLOC, "cudaMalloc of large-engine scratch failed");
        cudaError_t e = h->dbl ? opo::large_info_f64(h->L, h->F, h->B, h->sm_count, &h->linfo)
                               : opo::large_info_f32(h->L, h->F, h->B, h->sm_count, &h->linfo);
        if (e != cudaSuccess || h->linfo.grid <= 0) {
            cudaGetLastError();
            return bail(OPO_ERR_UNSUPPORTED, std::string("large-N engine unavailable for this size/precision: ") + cudaGetErrorString(e));
        }
    } else {
        // resident engine availability
        cudaError_t e = h->dbl ? opo::resident_info_f64(h->L, h->F, &h->rinfo) : opo::resident_info_f32(h->L, h->F, &h->rinfo);
        h->resident_ok = (e == cudaSuccess && h->rinfo.max_clusters > 0);
        if (e != cudaSuccess) cudaGetLastError();
        e = h->dbl ? opo::solo_info_f64(h->L, h->F, &h->sinfo) : opo::solo_info_f32(h->L, h->F, &h->sinfo);
        h->solo_ok = (e == cudaSuccess && h->sinfo.max_clusters > 0);
        if (e != cudaSuccess) cudaGetLastError();
        e = h->dbl ? opo::wide_info_f64(h->L, h->F, 1, &h->winfo) : opo::wide_info_f32(h->L, h->F, 1, &h->winfo);
        h->wide_ok = (e == cudaSuccess && h->winfo.max_clusters > 0);
        if (e != cudaSuccess) cudaGetLastError();
        e = h->dbl ? opo::wide_info_f64(h->L, h->F, 2, &h->winfo2) : opo::wide_info_f32(h->L, h->F, 2, &h->winfo2);
        if (e != cudaSuccess) { cudaGetLastError(); h->winfo2.max_clusters = 0; }
    }
    if (cudaDeviceSynchronize() != cudaSuccess) return bail(OPO_ERR_CUDA, cudaGetErrorString(cudaGetLastError()));
    *out = h;
    return OPO_OK;
}

int opo_destroy(opo_handle* h) {
    if (!h) return OPO_ERR_INVALID_ARG;
    cudaStreamSynchronize(h->stream);
    free_all(h);
    delete h;
    return OPO_OK;
}

int opo_set_stream(opo_handle* h, void* s) {
    if (!h) return OPO_ERR_INVALID_ARG;
    h->stream = (cudaStream_t)s;
    if (h->cufft_plan >= 0) cufft_api().SetStream(h->cufft_plan, h->stream);
    return OPO_OK;
}

int opo_set_batch_param(opo_handle* h, int param, int field, const double* v, int count) {
    if (!h || !v) return fail(h, OPO_ERR_INVALID_ARG, "null argument");
    if (count != h->B) return fail(h, OPO_ERR_INVALID_ARG, "count must equal batch");
    if (param == OPO_PARAM_DK) {
        h->dk.assign(v, v + count);
        h->phase_dirty = true;
        return OPO_OK;
    }
    if (field < 0 || field >= h->F) return fail(h, OPO_ERR_INVALID_ARG, "field out of range");
    std::vector<double>* dst = nullptr;
    if (param == OPO_PARAM_DELTA_T) dst = &h->dT[field];
    else if (param == OPO_PARAM_DELTA_RAD) dst = &h->drad[field];
    else if (param == OPO_PARAM_GDD) dst = &h->gdd[field];
    else return fail(h, OPO_ERR_INVALID_ARG, "unknown param");
    dst->assign(v, v + count);
    bool uniform = true;
    for (int x = 0; x < h->F; ++x) {
        bool u = true;
        for (int b = 1; b < h->B; ++b)
            if (h->dT[x][b] != h->dT[x][0] || h->gdd[x][b] != h->gdd[x][0] || h->drad[x][b] != h->drad[x][0]) u = false;
        h->per_inst_boundary[x] = !u;
        uniform = uniform && u;
    }
    (void)uniform;
    h->tables_dirty = true;
    return OPO_OK;
}

}  // extern "C"

namespace {

#define OPO_LAUNCH(h, call)                                                                \
    do {                                                                                   \
        cudaError_t e_ = (call);                                                           \
        if (e_ != cudaSuccess)                                                             \
            return fail((h), OPO_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
        ++(h)->launches;                                                                   \
    } while (0)

// Surface an error left by earlier asynchronous work without synchronising.  The CUDA "last error" is per host thread and
// shared with everything else in the process (PyTorch, other handles): it is only looked at here (cudaPeekAtLastError), never
// cleared, so that whoever raised it still finds it.  The library clears the error state only right after a call of its own
// has failed (the cudaGetLastError() next to those calls).  A sticky error (a device fault) keeps coming back by itself.
int check_async(opo_handle* h) {
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) return fail(h, OPO_ERR_CUDA, std::string("earlier asynchronous fault: ") + cudaGetErrorString(e));
    return OPO_OK;
}

// AUTO between the two on-chip engines: the cluster engine gives an instance F SMs (lowest latency per instance,
// rinfo.max_clusters instances at a time), the solo engine one SM (no SM-to-SM exchange, every SM busy, sinfo.max_clusters
// instances at a time).  Per z-step an instance takes ~2.6x longer on one SM than on a cluster of three (measured on C4 /
// C1), so solo wins once the batch keeps more than ~2.6x as many CTAs busy as there are clusters.
bool prefer_solo(const opo_handle* h) {
    if (!h->solo_ok || h->splitting) return false;      // the N/2 - L - N/2 ordering runs on the cluster engine
    if (!h->resident_ok) return true;
    const double solo_slots = (double)std::min(h->B, h->sinfo.max_clusters);
    const double cluster_slots = (double)std::min(h->B, h->rinfo.max_clusters);
    return solo_slots > 2.6 * cluster_slots;
}

// The wide engine serves the default ordering without a resonant pump (opo_wide.cuh).
bool wide_serves(const opo_handle* h) {
    return h->wide_ok && !h->splitting && h->n_seg == 1 && !h->fields.resonant[0];
}

// Time of the batch on the wide engine in units of the cluster engine's time per instance: clusters of 4 F CTAs take 1 / 2.9
// of it per instance (measured on C1: 5.4 vs 15.9 us per z-step) but only winfo.max_clusters of them are co-resident (7 of 12
// CTAs on a B200); clusters of 2 F CTAs with two sub-blocks per CTA take 1 / 1.4 of it (11.3 us: every SM then moves twice the
// bytes over the SM-to-SM link, which is what bounds this engine) and 22 are co-resident: they win for 15 .. 22 instances.
constexpr double kWide1 = 2.9, kWide2 = 1.4;
int wide_group(const opo_handle* h, double* cost = nullptr) {
    const int w1 = (h->B + h->winfo.max_clusters - 1) / h->winfo.max_clusters;
    double c1 = (double)w1 / kWide1, c2 = 1e300;
    if (h->winfo2.max_clusters > 0) c2 = (double)((h->B + h->winfo2.max_clusters - 1) / h->winfo2.max_clusters) / kWide2;
    if (h->wide_g_opt == 1) c2 = 1e300;
    if (h->wide_g_opt == 2 && c2 < 1e300) c1 = 1e300;
    if (cost) *cost = std::min(c1, c2);
    return c2 < c1 ? 2 : 1;
}

// AUTO takes the wide engine when it finishes the batch sooner than the cluster engine.
bool prefer_wide(const opo_handle* h) {
    if (!wide_serves(h)) return false;
    if (!h->resident_ok) return true;
    double cost = 0.0;
    wide_group(h, &cost);
    const int waves_r = (h->B + h->rinfo.max_clusters - 1) / h->rinfo.max_clusters;
    return cost < (double)waves_r;
}

int engine_in_use(const opo_handle* h) {
    if (h->large) return OPO_ENGINE_LARGE;
    if (h->n_seg > 1) return OPO_ENGINE_STREAMING;       // several crystals in series: host-sequenced engine only
    if (h->engine_opt == OPO_ENGINE_STREAMING) return OPO_ENGINE_STREAMING;
    if (h->engine_opt == OPO_ENGINE_CUFFT) return OPO_ENGINE_CUFFT;
    if (h->engine_opt == OPO_ENGINE_WIDE && wide_serves(h)) return OPO_ENGINE_WIDE;
    if (h->engine_opt == OPO_ENGINE_SOLO && h->solo_ok && !h->splitting) return OPO_ENGINE_SOLO;
    if (h->engine_opt == OPO_ENGINE_RESIDENT && h->resident_ok) return OPO_ENGINE_RESIDENT;
    if (prefer_solo(h)) return OPO_ENGINE_SOLO;                 // a batch that fills the GPU
    if (h->engine_opt == OPO_ENGINE_AUTO && prefer_wide(h)) return OPO_ENGINE_WIDE;
    return h->resident_ok ? OPO_ENGINE_RESIDENT : OPO_ENGINE_STREAMING;
}

bool on_chip_engine(const opo_handle* h) {
    const int e = engine_in_use(h);
    return e == OPO_ENGINE_RESIDENT || e == OPO_ENGINE_SOLO || e == OPO_ENGINE_WIDE;
}

// ---- streaming engine ------------------------------------------------------------------------------------------
// which linear operator: half step of crystal segment j, its full step, or the junction H_j H_{j+1} of two crystals
enum TableKind { TAB_H, TAB_H2, TAB_HX };

// cuFFT baseline: A <- IDFT(tab .* DFT(A)) as three launches per field (forward C2C over the batch, table multiply, inverse C2C)
int cufft_linear(opo_handle* h, int x, const void* tab, long long tab_stride) {
    CufftApi& cf = cufft_api();
    const int rc1 = h->dbl ? cf.ExecZ2Z(h->cufft_plan, h->cur[x], h->cur[x], kCufftForward) : cf.ExecC2C(h->cufft_plan, h->cur[x], h->cur[x], kCufftForward);
    if (rc1 != 0) return fail(h, OPO_ERR_CUDA, "cufftExec (forward) failed");
    opo::MulTabArgs m{h->cur[x], tab, h->B, h->N, tab_stride};
    OPO_LAUNCH(h, h->dbl ? opo::launch_multab_f64(m, h->stream) : opo::launch_multab_f32(m, h->stream));
    const int rc2 = h->dbl ? cf.ExecZ2Z(h->cufft_plan, h->cur[x], h->cur[x], kCufftInverse) : cf.ExecC2C(h->cufft_plan, h->cur[x], h->cur[x], kCufftInverse);
    if (rc2 != 0) return fail(h, OPO_ERR_CUDA, "cufftExec (inverse) failed");
    h->launches += 2;
    return OPO_OK;
}

int stream_linear_all(opo_handle* h, TableKind kind, int j, bool to_exit) {
    if (engine_in_use(h) == OPO_ENGINE_CUFFT) {          // single crystal only (engine_in_use)
        for (int x = 0; x < h->F; ++x) {
            if (int rc = cufft_linear(h, x, kind == TAB_H ? h->natH[x] : h->natH2[x], 0)) return rc;
            if (to_exit) OPO_CUDA(h, cudaMemcpyAsync(h->exitb[x], h->cur[x], h->field_bytes(), cudaMemcpyDeviceToDevice, h->stream));
        }
        return OPO_OK;
    }
    opo::LinArgs a{};
    a.n_slots = h->F; a.batch = h->B; a.tw = h->tw;
    for (int x = 0; x < h->F; ++x) {
        a.slot[x].src = h->cur[x]; a.slot[x].dst = h->cur[x];
        a.slot[x].dst2 = to_exit ? h->exitb[x] : nullptr;
        if (h->n_seg == 1) a.slot[x].tab = (kind == TAB_H) ? h->tabH[x] : h->tabH2[x];
        else a.slot[x].tab = kind == TAB_H ? h->segH[j][x] : (kind == TAB_H2 ? h->segH2[j][x] : h->segHX[j][x]);
        a.slot[x].tab_stride = 0;
    }
    OPO_LAUNCH(h, h->dbl ? opo::launch_linear_f64(h->L, a, h->stream) : opo::launch_linear_f32(h->L, a, h->stream));
    return OPO_OK;
}

// one RK4 step of the coupling terms of z-step `step` (counted from the start of the pass), with the couplings, step size
// and dk of the crystal segment it lies in; half = -1: the full step h; half = 0 | 1: first / second half step h/2 of the
// N/2 - L - N/2 ordering (phase table in steps of h/4)
int stream_rk4(opo_handle* h, int step, int half = -1) {
    const int j = segment_of_step(h, step);
    const opo_handle::Segment& sg = h->seg[j];
    opo::Rk4Args a{};
    for (int x = 0; x < h->F; ++x) { a.A[x] = h->cur[x]; a.kappa[x] = sg.kappa[x]; }
    a.n_fields = h->F; a.batch = h->B; a.n = h->N; a.h = half < 0 ? sg.hstep : 0.5 * sg.hstep;
    a.phase = h->phase; a.phase_stride = phase_stride(h); a.step = step;
    // entry of the concatenated per-segment tables (segment_of_step): q s + j, q = 2 | 4
    a.phase_index = half < 0 ? 2 * step + j : 4 * step + j + 2 * half;
    OPO_LAUNCH(h, h->dbl ? opo::launch_rk4_f64(a, h->stream) : opo::launch_rk4_f32(a, h->stream));
    return OPO_OK;
}

// nsteps z-steps from step index z0, half-steps merged:  H, N, H^2, N, ..., N, H; at the junction of two crystals the
// merged operator is H_j H_{j+1}
int stream_steps(opo_handle* h, int z0, int nsteps, bool to_exit) {
    if (nsteps <= 0) return OPO_OK;
    if (h->splitting) {      // N/2 - L - N/2 (Eq. 10-11), un-merged: two RK4 half-steps around one full linear step
        for (int s = z0; s < z0 + nsteps; ++s) {
            if (int rc = stream_rk4(h, s, 0)) return rc;
            if (int rc = stream_linear_all(h, TAB_H2, segment_of_step(h, s), false)) return rc;
            if (int rc = stream_rk4(h, s, 1)) return rc;
        }
        if (to_exit)
            for (int x = 0; x < h->F; ++x)
                OPO_CUDA(h, cudaMemcpyAsync(h->exitb[x], h->cur[x], h->field_bytes(), cudaMemcpyDeviceToDevice, h->stream));
        return OPO_OK;
    }
    if (int rc = stream_linear_all(h, TAB_H, segment_of_step(h, z0), false)) return rc;
    for (int s = 0; s < nsteps; ++s) {
        if (int rc = stream_rk4(h, z0 + s)) return rc;
        if (s + 1 < nsteps) {
            const int j = segment_of_step(h, z0 + s), jn = segment_of_step(h, z0 + s + 1);
            if (int rc = stream_linear_all(h, j == jn ? TAB_H2 : TAB_HX, j, false)) return rc;
        }
    }
    return stream_linear_all(h, TAB_H, segment_of_step(h, z0 + nsteps - 1), to_exit);
}

// A <- (accumulate ? A : 0) + c S  (input coupler of a resonant pump, reading R24)
int stream_axpy(opo_handle* h, void* A, const void* S, double c, bool accumulate) {
    OPO_LAUNCH(h, h->dbl ? opo::launch_axpy_f64(A, S, c, accumulate ? 1 : 0, (long long)h->B * h->N, h->stream)
                         : opo::launch_axpy_f32(A, S, c, accumulate ? 1 : 0, (long long)h->B * h->N, h->stream));
    return OPO_OK;
}
double pump_inject(const opo_handle* h) { return h->fields.resonant[0] ? std::sqrt(1.0 - h->fields.R[0]) : 0.0; }

// cavity boundary on the fields at z = L (readings R11-R15)
int stream_boundary(opo_handle* h) {
    opo::LinArgs a{};
    a.batch = h->B; a.tw = h->tw;
    for (int x = 0; x < h->F; ++x) {
        if (!h->fields.resonant[x]) {
            OPO_CUDA(h, cudaMemcpyAsync(h->cur[x], h->S[x], h->field_bytes(), cudaMemcpyDeviceToDevice, h->stream));
        } else if (h->boundary_fft[x] && engine_in_use(h) == OPO_ENGINE_CUFFT) {
            if (int rc = cufft_linear(h, x, h->natGM[x], h->per_inst_boundary[x] ? h->N : 0)) return rc;
        } else if (h->boundary_fft[x]) {
            opo::LinSlot& sl = a.slot[a.n_slots++];
            sl.src = h->cur[x]; sl.dst = h->cur[x]; sl.dst2 = nullptr;
            sl.tab = h->tabGM[x]; sl.tab_stride = h->per_inst_boundary[x] ? h->N : 0;
        } else {
            opo::ScaleArgs sc{h->cur[x], h->mirror[x], h->B, h->N};
            OPO_LAUNCH(h, h->dbl ? opo::launch_scale_f64(sc, h->stream) : opo::launch_scale_f32(sc, h->stream));
        }
    }
    if (a.n_slots > 0)
        OPO_LAUNCH(h, h->dbl ? opo::launch_linear_f64(h->L, a, h->stream) : opo::launch_linear_f32(h->L, a, h->stream));
    // resonant pump: the input coupler adds sqrt(1 - R_p) S_p (reading R24; with a modulator on the pump it acts before the
    // injection, as in the oracle)
    if (h->fields.resonant[0] && !h->eom[0]) return stream_axpy(h, h->cur[0], h->S[0], pump_inject(h), true);
    return OPO_OK;
}

// intracavity phase modulator after the boundary (Listing 3), streaming / large engines
bool any_eom(const opo_handle* h) {
    for (int x = 0; x < h->F; ++x) if (h->eom[x]) return true;
    return false;
}
int apply_eom(opo_handle* h) {
    for (int x = 0; x < h->F; ++x) {
        if (!h->eom[x]) continue;
        opo::MulTabArgs m{h->cur[x], h->eom[x], h->B, h->N, 0};
        OPO_LAUNCH(h, h->dbl ? opo::launch_multab_f64(m, h->stream) : opo::launch_multab_f32(m, h->stream));
        if (x == 0 && h->fields.resonant[0])        // the input coupler comes after the pump's own modulator (stream_boundary)
            if (int rc = stream_axpy(h, h->cur[0], h->S[0], pump_inject(h), true)) return rc;
    }
    return OPO_OK;
}

// ---- resident engine ---------------------------------------------------------------------------------------------
// pump train handled inside the launch (solo engine): slices in, exit fields of `out_field` out
struct TrainArgs {
    const void* pump = nullptr;
    bool per_instance = false;
    void* out = nullptr;
    int out_field = 0;
};

void advance_counts(opo_handle* h, long long ops, long long half_uses, long long full_uses) {
    constexpr long long kWrap = 1 << 20;
    h->op_count = (int)((h->op_count + ops) % kWrap);
    h->hq_count = (int)((h->hq_count + half_uses) % kWrap);
    h->fq_count = (int)((h->fq_count + full_uses) % kWrap);
}

int resident_run(opo_handle* h, int mode, int z0, int steps, const TrainArgs* train = nullptr) {
    opo::ResidentArgs a{};
    if (train) {
        a.train = train->pump;
        a.train_stride = (long long)h->N * (train->per_instance ? h->B : 1);
        a.train_inst_stride = train->per_instance ? h->N : 0;
        a.out_train = train->out;
        a.out_field = train->out_field;
    }
    for (int x = 0; x < h->F; ++x) {
        a.cur[x] = h->cur[x]; a.S[x] = h->S[x]; a.exitb[x] = h->exitb[x]; a.SH[x] = h->SH[x];
        a.tabH[x] = h->tabH[x]; a.tabH2[x] = h->tabH2[x]; a.tabHB[x] = h->tabHB[x]; a.tabGM[x] = h->tabGM[x]; a.tabHG[x] = h->tabHG[x];
        a.tab_stride[x] = h->per_inst_boundary[x] ? h->N : 0;
        a.mirror[x] = h->mirror[x];
        a.eom[x] = h->eom[x];
        a.boundary_fft[x] = h->boundary_fft[x] ? 1 : 0;
        a.resonant[x] = h->fields.resonant[x] ? 1 : 0;
        a.kappa[x] = h->kappa[x];
    }
    a.inject = pump_inject(h);
    a.tw = h->tw; a.phase = h->phase; a.phase_stride = phase_stride(h);
    a.h = h->h; a.n_fields = h->F; a.batch = h->B; a.nz = h->nz;
    a.mode = mode; a.z0 = z0; a.steps = steps; a.nln = h->splitting;
    a.tab_cycle_mask = h->tab_cycle - 1;
    a.op0 = h->op_count; a.hq0 = h->hq_count; a.fq0 = h->fq_count;
    a.dk0 = !h->splitting;
    for (int b = 0; b < h->B; ++b) if (h->dk[b] != 0.0) a.dk0 = 0;
    const bool solo = engine_in_use(h) == OPO_ENGINE_SOLO, wide = engine_in_use(h) == OPO_ENGINE_WIDE;
    a.wide_g = wide ? wide_group(h) : 1;
    const int n_clusters = std::min(h->B, wide ? (a.wide_g == 2 ? h->winfo2.max_clusters : h->winfo.max_clusters) : solo ? h->sinfo.max_clusters : h->rinfo.max_clusters);
    // more instances than clusters and not a multiple: deal round trips instead of instances (see the kernel)
    a.split = 0; a.flags = nullptr;
    if (mode == 1 && !wide && !h->splitting && steps > 1 && h->B > n_clusters && h->B % n_clusters != 0) {
        if (!h->rt_flags && cudaMalloc((void**)&h->rt_flags, (size_t)h->B * 3 * sizeof(int)) != cudaSuccess) {
            cudaGetLastError();
            return fail(h, OPO_ERR_ALLOC, "cudaMalloc of the round-trip flags failed");
        }
        OPO_CUDA(h, cudaMemsetAsync(h->rt_flags, 0, (size_t)h->B * 3 * sizeof(int), h->stream));
        a.split = 1; a.flags = h->rt_flags;
    }
    auto launch = [&]() {
        if (wide) return h->dbl ? opo::launch_wide_f64(h->L, a, n_clusters, h->stream) : opo::launch_wide_f32(h->L, a, n_clusters, h->stream);
        if (solo) return h->dbl ? opo::launch_solo_f64(h->L, a, n_clusters, h->stream) : opo::launch_solo_f32(h->L, a, n_clusters, h->stream);
        return h->dbl ? opo::launch_resident_f64(h->L, a, n_clusters, h->stream) : opo::launch_resident_f32(h->L, a, n_clusters, h->stream);
    };
    cudaError_t e = launch();
    if (e != cudaSuccess && a.split) {
        // the split schedule needs every cluster / CTA of the grid resident (cooperative launch); if the device cannot
        // promise that right now, deal whole instances instead -- slower by the ragged last wave, never a hang
        cudaGetLastError();
        a.split = 0; a.flags = nullptr;
        e = launch();
    }
    if (e != cudaSuccess) return fail(h, OPO_ERR_CUDA, std::string("launch of the on-chip kernel: ") + cudaGetErrorString(e));
    ++h->launches;
    // what an (uncut) instance has applied in this launch: the operators q = 0 .. total, of which the first and the last are
    // half-steps and the boundary crossings use tables of their own; N/2 - L - N/2: full steps only
    const long long passes = mode == 1 ? steps : 1, per_pass = mode == 1 ? h->nz : steps;
    advance_counts(h, h->splitting ? passes * per_pass : passes * per_pass + 1, h->splitting ? 0 : 2,
                   h->splitting ? passes * per_pass : passes * (per_pass - 1));
    return OPO_OK;
}

// ---- large-N engine -----------------------------------------------------------------------------------------------
void large_common(const opo_handle* h, opo::LargeArgs& a) {
    for (int x = 0; x < h->F; ++x) {
        a.cur[x] = h->cur[x]; a.SH[x] = h->SH[x];
        a.tabH[x] = h->tabH[x]; a.tabH2[x] = h->tabH2[x]; a.tabHB[x] = h->tabHB[x];
        a.tabHB_stride[x] = h->per_inst_boundary[x] ? h->N : 0;
        a.resonant[x] = h->fields.resonant[x] ? 1 : 0;
        a.kappa[x] = h->kappa[x];
    }
    a.tw1 = h->tw; a.tw2 = h->tw2; a.wlo = h->wlo; a.whi = h->whi; a.perm1 = h->perm; a.perm2 = h->perm2;
    a.phase = h->phase; a.phase_stride = phase_stride(h); a.nln = h->splitting;
    a.h = h->h; a.n_fields = h->F; a.batch = h->B; a.nz = h->nz;
    a.field_mask = (1 << h->F) - 1;
    a.barrier = h->barrier; a.barrier_base = 0;
    a.op0 = h->op_count;
}

int large_launch(opo_handle* h, const opo::LargeArgs& a) {
    OPO_CUDA(h, cudaMemsetAsync(h->barrier, 0, sizeof(unsigned long long), h->stream));
    OPO_LAUNCH(h, h->dbl ? opo::launch_large_f64(h->L, a, h->linfo.grid, h->stream)
                         : opo::launch_large_f32(h->L, a, h->linfo.grid, h->stream));
    if (a.mode != 2) {      // linear operators of this launch (the read-out applies none)
        const long long total = a.mode == 1 ? (long long)a.steps * a.nz : a.steps;
        advance_counts(h, a.nln ? total : total + 1, 0, 0);
    }
    return OPO_OK;
}

// mode 0: `steps` z-steps from step index z0.  mode 1: `steps` round trips; the kernel leaves the fields
// at z = L of the last pass, the boundary of that last pass follows here.
int large_run(opo_handle* h, int mode, int z0, int steps) {
    opo::LargeArgs a{};
    large_common(h, a);
    a.mode = mode; a.z0 = z0; a.steps = steps;
    if (int rc = large_launch(h, a)) return rc;
    if (mode == 0) return OPO_OK;
    int fft_mask = 0;
    for (int x = 0; x < h->F; ++x) {
        OPO_CUDA(h, cudaMemcpyAsync(h->exitb[x], h->cur[x], h->field_bytes(), cudaMemcpyDeviceToDevice, h->stream));
        if (!h->fields.resonant[x]) {
            OPO_CUDA(h, cudaMemcpyAsync(h->cur[x], h->S[x], h->field_bytes(), cudaMemcpyDeviceToDevice, h->stream));
        } else if (h->boundary_fft[x]) {
            fft_mask |= 1 << x;
        } else {
            opo::ScaleArgs sc{h->cur[x], h->mirror[x], h->B, h->N};
            OPO_LAUNCH(h, h->dbl ? opo::launch_scale_f64(sc, h->stream) : opo::launch_scale_f32(sc, h->stream));
        }
    }
    if (fft_mask) {
        opo::LargeArgs g{};
        large_common(h, g);
        g.mode = 0; g.z0 = 0; g.steps = 0; g.field_mask = fft_mask; g.nln = 0;     // one linear operator, whatever the splitting
        for (int x = 0; x < h->F; ++x) {
            g.tabH[x] = h->tabGM[x];
            g.tabH_stride[x] = h->per_inst_boundary[x] ? h->N : 0;
        }
        if (int rc = large_launch(h, g)) return rc;
    }
    return OPO_OK;
}

// out[b][k] = DFT(src[b])[k], natural order (dst may be the handle's own scratch)
int large_freq(opo_handle* h, const void* src, void* dst) {
    opo::LargeArgs a{};
    large_common(h, a);
    a.mode = 2; a.field_mask = 1;
    a.cur[0] = h->scratch2; a.src_override[0] = const_cast<void*>(src); a.out[0] = dst;
    return large_launch(h, a);
}

int copy_in(opo_handle* h, void* dst_field, const void* src, bool per_instance, cudaMemcpyKind kind) {
    const size_t one = (size_t)h->N * h->esz;
    if (per_instance) {
        OPO_CUDA(h, cudaMemcpyAsync(dst_field, src, one * h->B, kind, h->stream));
    } else {
        // one slice in, one kernel replicates it to every instance
        OPO_CUDA(h, cudaMemcpyAsync(dst_field, src, one, kind, h->stream));
        if (h->B > 1)
            OPO_LAUNCH(h, h->dbl ? opo::launch_broadcast_f64(dst_field, h->B, h->N, h->stream) : opo::launch_broadcast_f32(dst_field, h->B, h->N, h->stream));
    }
    return OPO_OK;
}

int set_pump_impl(opo_handle* h, const void* p, int per_instance, cudaMemcpyKind kind) {
    if (!h || !p) return fail(h, OPO_ERR_INVALID_ARG, "null argument");
    if (int rc = check_async(h)) return rc;
    if (int rc = copy_in(h, h->S[0], p, per_instance != 0, kind)) return rc;
    if (h->z_steps == 0) {
        // what the boundary injects into an empty cavity: S_p for a single-pass pump, sqrt(1 - R_p) S_p through the
        // input coupler of a resonant one (reading R24).  A resonant pump that has been running holds stored light, which a
        // new input must not wipe out (a power ramp between opo_roundtrips calls): then only S_p changes and the boundary of
        // the next round trip injects it, as in the oracle, where the input and the state of a field are set separately.
        if (h->fields.resonant[0]) return h->run_started ? OPO_OK : stream_axpy(h, h->cur[0], h->S[0], pump_inject(h), false);
        OPO_CUDA(h, cudaMemcpyAsync(h->cur[0], h->S[0], h->field_bytes(), cudaMemcpyDeviceToDevice, h->stream));
    }
    return OPO_OK;
}

int set_field_impl(opo_handle* h, int field, const void* p, cudaMemcpyKind kind) {
    if (!h || !p) return fail(h, OPO_ERR_INVALID_ARG, "null argument");
    if (field < 0 || field >= h->F) return fail(h, OPO_ERR_INVALID_ARG, "field out of range");
    if (int rc = check_async(h)) return rc;
    if (int rc = copy_in(h, h->S[field], p, true, kind)) return rc;
    OPO_CUDA(h, cudaMemcpyAsync(h->cur[field], h->S[field], h->field_bytes(), cudaMemcpyDeviceToDevice, h->stream));
    return OPO_OK;
}

int get_fields_impl(opo_handle* h, int field, int which, int domain, void* out, bool host) {
    if (!h || !out) return fail(h, OPO_ERR_INVALID_ARG, "null argument");
    if (field < 0 || field >= h->F) return fail(h, OPO_ERR_INVALID_ARG, "field out of range");
    if (which != OPO_WHICH_CURRENT && which != OPO_WHICH_EXIT) return fail(h, OPO_ERR_INVALID_ARG, "which must be CURRENT or EXIT");
    if (domain != OPO_DOMAIN_TIME && domain != OPO_DOMAIN_FREQ) return fail(h, OPO_ERR_INVALID_ARG, "domain must be TIME or FREQ");
    if (int rc = check_async(h)) return rc;
    const void* src = (which == OPO_WHICH_CURRENT) ? h->cur[field] : h->exitb[field];
    if (domain == OPO_DOMAIN_FREQ) {
        if (h->large) {
            if (int rc = large_freq(h, src, host ? h->scratch : out)) return rc;
        } else {
            opo::FreqArgs a{src, host ? h->scratch : out, h->perm, h->tw, h->B};
            OPO_LAUNCH(h, h->dbl ? opo::launch_freq_f64(h->L, a, h->stream) : opo::launch_freq_f32(h->L, a, h->stream));
        }
        if (!host) return OPO_OK;
        src = h->scratch;
    }
    OPO_CUDA(h, cudaMemcpyAsync(out, src, h->field_bytes(), host ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, h->stream));
    if (host) OPO_CUDA(h, cudaStreamSynchronize(h->stream));
    return OPO_OK;
}

}  // namespace

extern "C" {

int opo_set_pump(opo_handle* h, const void* dev_pump, int per_instance) { return set_pump_impl(h, dev_pump, per_instance, cudaMemcpyDeviceToDevice); }
int opo_set_pump_host(opo_handle* h, const void* host_pump, int per_instance) { return set_pump_impl(h, host_pump, per_instance, cudaMemcpyHostToDevice); }
int opo_set_field(opo_handle* h, int field, const void* dev_data) { return set_field_impl(h, field, dev_data, cudaMemcpyDeviceToDevice); }
int opo_set_field_host(opo_handle* h, int field, const void* host_data) { return set_field_impl(h, field, host_data, cudaMemcpyHostToDevice); }
int opo_get_fields(opo_handle* h, int field, int which, int domain, void* dev_out) { return get_fields_impl(h, field, which, domain, dev_out, false); }
int opo_get_fields_host(opo_handle* h, int field, int which, int domain, void* host_out) { return get_fields_impl(h, field, which, domain, host_out, true); }

int opo_propagate(opo_handle* h, int nz) {
    if (!h) return OPO_ERR_INVALID_ARG;
    if (nz < 0) return fail(h, OPO_ERR_INVALID_ARG, "nz must be >= 0");
    if (h->z_steps + nz > h->nz) return fail(h, OPO_ERR_STATE, "propagate would pass z = L");
    if (nz == 0) return OPO_OK;
    if (int rc = check_async(h)) return rc;
    if (int rc = ensure_tables(h)) return rc;
    int rc;
    if (h->large) rc = large_run(h, 0, h->z_steps, nz);
    else if (on_chip_engine(h)) rc = resident_run(h, 0, h->z_steps, nz);
    else rc = stream_steps(h, h->z_steps, nz, false);
    if (rc) return rc;
    h->z_steps += nz;
    h->run_started = true;
    return OPO_OK;
}

int opo_roundtrips(opo_handle* h, int n) {
    if (!h) return OPO_ERR_INVALID_ARG;
    if (n < 0) return fail(h, OPO_ERR_INVALID_ARG, "n must be >= 0");
    if (h->z_steps != 0) return fail(h, OPO_ERR_STATE, "roundtrips requires z = 0");
    if (n == 0) return OPO_OK;
    if (int rc = check_async(h)) return rc;
    if (int rc = ensure_tables(h)) return rc;
    h->run_started = true;
    // a phase modulator acts in the time domain between the boundary's spectral phase and the next pass, so the
    // boundary cannot be merged into the neighbouring half-steps: one launch per round trip then
    const bool eom = any_eom(h);
    if (h->large) {
        if (!eom && !h->splitting) return large_run(h, 1, 0, n);
        for (int m = 0; m < n; ++m) {
            if (int rc = large_run(h, 1, 0, 1)) return rc;
            if (int rc = apply_eom(h)) return rc;
        }
        return OPO_OK;
    }
    if (on_chip_engine(h)) {
        // a modulator is applied inside the kernel (between two linear cores at a crossing, with the last store at the
        // end of a call); only the N/2 - L - N/2 ordering runs one pass per launch
        if (!h->splitting) return resident_run(h, 1, 0, n);
        for (int m = 0; m < n; ++m)
            if (int rc = resident_run(h, 1, 0, 1)) return rc;
        return OPO_OK;
    }
    for (int m = 0; m < n; ++m) {
        if (int rc = stream_steps(h, 0, h->nz, true)) return rc;
        if (int rc = stream_boundary(h)) return rc;
        if (eom) if (int rc = apply_eom(h)) return rc;
    }
    return OPO_OK;
}

int opo_roundtrips_train(opo_handle* h, int n, const void* dev_pump_train, int per_instance, void* dev_out_train, int out_field) {
    if (!h || !dev_pump_train) return fail(h, OPO_ERR_INVALID_ARG, "null argument");
    if (n < 0) return fail(h, OPO_ERR_INVALID_ARG, "n must be >= 0");
    if (dev_out_train && (out_field < 0 || out_field >= h->F)) return fail(h, OPO_ERR_INVALID_ARG, "out_field out of range");
    if (h->fields.resonant[0]) return fail(h, OPO_ERR_UNSUPPORTED, "a pump train needs a single-pass (non-resonant) pump");
    if (h->z_steps != 0) return fail(h, OPO_ERR_STATE, "roundtrips requires z = 0");
    const size_t slice = (size_t)h->N * h->esz * (per_instance ? (size_t)h->B : 1);
    if (n > 0 && engine_in_use(h) == OPO_ENGINE_SOLO && !h->splitting && !any_eom(h)) {
        // one launch for the whole train: the kernel reads slice m at the crossing into round trip m and writes the exit field
        // of every round trip (opo_solo.cuh, TRAIN); the stored pump input ends up as the last slice, as in the loop below
        if (int rc = set_pump_impl(h, (const char*)dev_pump_train + (size_t)(n - 1) * slice, per_instance, cudaMemcpyDeviceToDevice)) return rc;
        if (int rc = ensure_tables(h)) return rc;
        TrainArgs t;
        t.pump = dev_pump_train; t.per_instance = per_instance != 0; t.out = dev_out_train; t.out_field = dev_out_train ? out_field : 0;
        return resident_run(h, 1, 0, n, &t);
    }
    for (int m = 0; m < n; ++m) {
        // ReadPump: the m-th slice of the long pump vector becomes the intracavity pump
        if (int rc = set_pump_impl(h, (const char*)dev_pump_train + (size_t)m * slice, per_instance, cudaMemcpyDeviceToDevice)) return rc;
        if (int rc = opo_roundtrips(h, 1)) return rc;
        // SaveRoundTrip: the field leaving the crystal in this round trip
        if (dev_out_train)
            OPO_CUDA(h, cudaMemcpyAsync((char*)dev_out_train + (size_t)m * h->field_bytes(), h->exitb[out_field], h->field_bytes(),
                                        cudaMemcpyDeviceToDevice, h->stream));
    }
    return OPO_OK;
}

int opo_set_segments(opo_handle* h, int n, const opo_segment* segs) {
    if (!h) return OPO_ERR_INVALID_ARG;
    if (n < 0 || n > 8 || (n > 0 && !segs)) return fail(h, OPO_ERR_INVALID_ARG, "0 .. 8 segments");
    if (h->z_steps != 0) return fail(h, OPO_ERR_STATE, "the crystal segments can only change at z = 0");
    if (h->large && n > 1) return fail(h, OPO_ERR_UNSUPPORTED, "several crystals: not on the large-N engine (N > 2^14, c128: > 2^13)");
    if (n > 1 && h->engine_opt == OPO_ENGINE_CUFFT) return fail(h, OPO_ERR_UNSUPPORTED, "several crystals: not on the cuFFT baseline engine");
    long long total = 0;
    for (int j = 0; j < n; ++j) {
        if (!(segs[j].length_m > 0.0) || segs[j].nz <= 0 || !std::isfinite(segs[j].dk_per_m) || !std::isfinite(segs[j].d_eff_m_per_V))
            return fail(h, OPO_ERR_INVALID_ARG, "segment length and nz must be positive, dk and d_eff finite");
        total += segs[j].nz;
    }
    if (int rc = check_async(h)) return rc;
    // everything that can fail comes first, so that a failure leaves the handle as it was: a larger phase table (the old
    // one is kept when it is large enough) and the wait for work that still reads the old one
    const long long new_nz = n == 0 ? h->grid.nz_per_pass : total;
    const size_t need = (size_t)h->B * (4 * (size_t)new_nz + 8) * h->esz;
    void* new_phase = nullptr;
    if (need > h->phase_bytes && cudaMalloc(&new_phase, need) != cudaSuccess) {
        cudaGetLastError();
        return fail(h, OPO_ERR_ALLOC, "cudaMalloc of the phase table failed");
    }
    {
        const cudaError_t e = cudaStreamSynchronize(h->stream);
        if (e != cudaSuccess) {
            if (new_phase) cudaFree(new_phase);
            return fail(h, OPO_ERR_CUDA, std::string("cudaStreamSynchronize: ") + cudaGetErrorString(e));
        }
    }
    if (new_phase) { cudaFree(h->phase); h->phase = new_phase; h->phase_bytes = need; }
    if (n == 0) {       // back to the crystal of opo_create
        h->n_seg = 1;
        h->seg[0].len = h->crystal.length_m; h->seg[0].dk = h->crystal.dk_per_m; h->seg[0].deff = h->crystal.d_eff_m_per_V;
        h->seg[0].nz = h->grid.nz_per_pass;
    } else {
        h->n_seg = n;
        for (int j = 0; j < n; ++j) { h->seg[j].len = segs[j].length_m; h->seg[j].dk = segs[j].dk_per_m; h->seg[j].deff = segs[j].d_eff_m_per_V; h->seg[j].nz = segs[j].nz; }
    }
    h->nz = 0;
    for (int j = 0; j < h->n_seg; ++j) {
        opo_handle::Segment& sg = h->seg[j];
        sg.hstep = sg.len / (double)sg.nz;
        for (int x = 0; x < h->F; ++x) sg.kappa[x] = 2.0 * kPi * sg.deff / (h->fields.n[x] * h->fields.lambda_m[x]);
        if (h->F == 2) sg.kappa[0] *= 0.5;                                                                               // reading R5
        h->nz += sg.nz;
    }
    h->h = h->seg[0].hstep;
    for (int x = 0; x < 3; ++x) h->kappa[x] = h->seg[0].kappa[x];
    // per-instance dk sweeps act on the first crystal; a new segment list resets them to its dk
    h->dk.assign(h->B, h->seg[0].dk);
    if (h->n_seg == 1)      // a single crystal uses tabH / tabH2: give the per-segment tables back (the stream is idle)
        for (int j = 0; j < 8; ++j)
            for (int x = 0; x < 3; ++x) {
                void** ptrs[] = {&h->segH[j][x], &h->segH2[j][x], &h->segHX[j][x]};
                for (void** p : ptrs) if (*p) { cudaFree(*p); *p = nullptr; }
            }
    h->tables_dirty = true;
    h->phase_dirty = true;
    return OPO_OK;
}

int opo_set_beta3(opo_handle* h, int field, double beta3_s3_per_m) {
    if (!h) return OPO_ERR_INVALID_ARG;
    if (field < 0 || field >= h->F) return fail(h, OPO_ERR_INVALID_ARG, "field out of range");
    if (!std::isfinite(beta3_s3_per_m)) return fail(h, OPO_ERR_INVALID_ARG, "non-finite beta3");
    h->beta3[field] = beta3_s3_per_m;
    h->tables_dirty = true;
    return OPO_OK;
}

int opo_set_eom(opo_handle* h, int field, double beta_rad, double f_mod_hz) {
    if (!h) return OPO_ERR_INVALID_ARG;
    if (field < 0 || field >= h->F) return fail(h, OPO_ERR_INVALID_ARG, "field out of range");
    if (!h->fields.resonant[field]) return fail(h, OPO_ERR_INVALID_ARG, "a phase modulator acts on resonant fields only");
    if (!std::isfinite(beta_rad) || !std::isfinite(f_mod_hz)) return fail(h, OPO_ERR_INVALID_ARG, "non-finite modulator parameter");
    if (int rc = check_async(h)) return rc;
    h->eom_beta[field] = beta_rad; h->eom_f[field] = f_mod_hz;
    if (beta_rad == 0.0) {
        if (h->eom[field]) { OPO_CUDA(h, cudaStreamSynchronize(h->stream)); cudaFree(h->eom[field]); h->eom[field] = nullptr; }
        return OPO_OK;
    }
    if (!h->eom[field] && cudaMalloc(&h->eom[field], (size_t)h->N * h->esz) != cudaSuccess) {
        cudaGetLastError();
        return fail(h, OPO_ERR_ALLOC, "cudaMalloc of the modulator table failed");
    }
    std::vector<cd> E(h->N);
    const double dt = h->grid.window_s / (double)h->N;
    for (int n = 0; n < h->N; ++n) {
        const double tau = (double)(n - h->N / 2) * dt;                       // reading R19
        const double ph = beta_rad * std::sin(2.0 * kPi * f_mod_hz * tau);
        E[n] = cd(std::cos(ph), std::sin(ph));
    }
    return upload_complex(h, h->eom[field], E.data(), (size_t)h->N, true);
}

int opo_sync(opo_handle* h) {
    if (!h) return OPO_ERR_INVALID_ARG;
    OPO_CUDA(h, cudaStreamSynchronize(h->stream));
    return check_async(h);
}

int opo_check_finite(opo_handle* h) {
    if (!h) return OPO_ERR_INVALID_ARG;
    OPO_CUDA(h, cudaMemsetAsync(h->flag, 0, sizeof(int), h->stream));
    for (int x = 0; x < h->F; ++x) {
        const long long count = 2LL * h->B * h->N;
        OPO_LAUNCH(h, h->dbl ? opo::launch_finite_f64(h->cur[x], count, h->flag, h->stream)
                             : opo::launch_finite_f32(h->cur[x], count, h->flag, h->stream));
    }
    int flag = 0;
    OPO_CUDA(h, cudaMemcpyAsync(&flag, h->flag, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    OPO_CUDA(h, cudaStreamSynchronize(h->stream));
    if (flag) return fail(h, OPO_ERR_NONFINITE, "non-finite field values (dz too coarse? PAPER.md:L162)");
    return OPO_OK;
}

int opo_get_z_steps(const opo_handle* h, int* out) {
    if (!h || !out) return OPO_ERR_INVALID_ARG;
    *out = h->z_steps;
    return OPO_OK;
}

int opo_set_option(opo_handle* h, int option, int value) {
    if (!h) return OPO_ERR_INVALID_ARG;
    if (option == OPO_OPT_SPLITTING) {
        if (value != OPO_SPLITTING_LNL && value != OPO_SPLITTING_NLN) return fail(h, OPO_ERR_INVALID_ARG, "unknown splitting");
        if (h->z_steps != 0) return fail(h, OPO_ERR_STATE, "the splitting can only change at z = 0");
        if (value != h->splitting) { h->splitting = value; h->phase_dirty = true; }
        return OPO_OK;
    }
    if (option == OPO_OPT_WIDE_SUBBLOCKS) {
        if (value < 0 || value > 2) return fail(h, OPO_ERR_INVALID_ARG, "sub-blocks per CTA: 0 (AUTO), 1 or 2");
        if (value == 2 && h->winfo2.max_clusters <= 0) return fail(h, OPO_ERR_UNSUPPORTED, "two sub-blocks per CTA: unavailable for this size/precision");
        h->wide_g_opt = value;
        return OPO_OK;
    }
    if (option != OPO_OPT_ENGINE) return fail(h, OPO_ERR_INVALID_ARG, "unknown option");
    if (value != OPO_ENGINE_AUTO && value != OPO_ENGINE_RESIDENT && value != OPO_ENGINE_STREAMING && value != OPO_ENGINE_LARGE &&
        value != OPO_ENGINE_CUFFT && value != OPO_ENGINE_SOLO && value != OPO_ENGINE_WIDE)
        return fail(h, OPO_ERR_INVALID_ARG, "unknown engine");
    if (value == OPO_ENGINE_CUFFT) {
        if (h->large) return fail(h, OPO_ERR_UNSUPPORTED, "the cuFFT baseline serves the sizes of the streaming engine");
        CufftApi& cf = cufft_api();
        if (!cf.ok) return fail(h, OPO_ERR_UNSUPPORTED, "libcufft could not be loaded");
        if (h->cufft_plan < 0) {
            int n[1] = {h->N};
            cufftHandle_t plan;
            if (cf.PlanMany(&plan, 1, n, nullptr, 1, h->N, nullptr, 1, h->N, h->dbl ? kCufftZ2Z : kCufftC2C, h->B) != 0)
                return fail(h, OPO_ERR_CUDA, "cufftPlanMany failed");
            h->cufft_plan = plan;
            for (int x = 0; x < h->F; ++x)
                if (cudaMalloc(&h->natH[x], (size_t)h->N * h->esz) != cudaSuccess || cudaMalloc(&h->natH2[x], (size_t)h->N * h->esz) != cudaSuccess)
                    return fail(h, OPO_ERR_ALLOC, "cudaMalloc of baseline tables failed");
            h->tables_dirty = true;
        }
        cf.SetStream(h->cufft_plan, h->stream);
    }
    if (h->large && value != OPO_ENGINE_AUTO && value != OPO_ENGINE_LARGE)
        return fail(h, OPO_ERR_UNSUPPORTED, "N > 2^14 (c128: > 2^13) runs on the large-N engine only");
    if (!h->large && value == OPO_ENGINE_LARGE)
        return fail(h, OPO_ERR_UNSUPPORTED, "the large-N engine serves N > 2^14 (c128: > 2^13) only");
    if (value == OPO_ENGINE_RESIDENT && !h->resident_ok)
        return fail(h, OPO_ERR_UNSUPPORTED, "resident engine unavailable for this size/precision on this device");
    if (value == OPO_ENGINE_SOLO && !h->solo_ok)
        return fail(h, OPO_ERR_UNSUPPORTED, "solo engine unavailable for this size/precision on this device");
    if (value == OPO_ENGINE_WIDE && !h->wide_ok)
        return fail(h, OPO_ERR_UNSUPPORTED, "wide engine unavailable for this size/precision on this device (N = 2^12 .. 2^14; c128: 2^12, 2^13)");
    h->engine_opt = value;
    return OPO_OK;
}

int opo_get_info(const opo_handle* h, int what, long long* out) {
    if (!h || !out) return OPO_ERR_INVALID_ARG;
    switch (what) {
        case OPO_INFO_ENGINE: *out = engine_in_use(h); return OPO_OK;
        case OPO_INFO_LAUNCHES: *out = h->launches; return OPO_OK;
        case OPO_INFO_N: *out = h->N; return OPO_OK;
        case OPO_INFO_BATCH: *out = h->B; return OPO_OK;
        case OPO_INFO_SM_COUNT: *out = h->sm_count; return OPO_OK;
        case OPO_INFO_SLOTS: {
            const int e = engine_in_use(h);
            if (e == OPO_ENGINE_SOLO) *out = std::min(h->B, h->sinfo.max_clusters);
            else if (e == OPO_ENGINE_WIDE) *out = std::min(h->B, wide_group(h) == 2 ? h->winfo2.max_clusters : h->winfo.max_clusters);
            else if (e == OPO_ENGINE_RESIDENT) *out = std::min(h->B, h->rinfo.max_clusters);
            else if (e == OPO_ENGINE_LARGE) *out = h->linfo.grid;
            else *out = (long long)h->B * h->F;
            return OPO_OK;
        }
        case OPO_INFO_WIDE_SUBBLOCKS: *out = engine_in_use(h) == OPO_ENGINE_WIDE ? wide_group(h) : 0; return OPO_OK;
        default: return OPO_ERR_INVALID_ARG;
    }
}

}  // extern "C"

// ---- opo_spectrum_noalloc: the frequency read-out for callers that must not allocate device memory -------------------
// The read-out kernel (k_freq, opo_kernels.cuh) needs two tables next to its input and output: the pass twiddles of the
// transform and the map from the transform's digit-reversed positions to frequency indices.  A handle keeps them in
// cudaMalloc'ed memory.  This entry point keeps them in the fixed array below instead, which is part of the library image:
// the driver places it when the library is loaded on a GPU and takes it back at process exit, so no call here ever asks
// the allocator for anything.
//
//   bytes [0, 128 KiB)         : pass twiddles, N - 1 entries of float2 (N <= 2^14) or double2 (N <= 2^13)
//   bytes [128 KiB, 192 KiB)   : int32 position -> frequency index, N entries
namespace {

constexpr int kNoAllocMaxLog2C64 = 14, kNoAllocMaxLog2C128 = 13;
constexpr size_t kNoAllocTwBytes = (size_t)8 << kNoAllocMaxLog2C64;       // = 16 << kNoAllocMaxLog2C128
constexpr size_t kNoAllocPermBytes = (size_t)4 << kNoAllocMaxLog2C64;
constexpr size_t kNoAllocBytes = kNoAllocTwBytes + kNoAllocPermBytes;     // 192 KiB on every GPU that loads libopo.so

static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocBytes];

// Host view of the array, one entry per device.  `base` is what cudaGetSymbolAddress returned with that device current: the
// name g_noalloc_scratch itself means nothing to a kernel when it is written in host code.
struct NoAllocDevice {
    unsigned char* base = nullptr;
    int log2_n = -1, precision = -1;      // which tables the array holds now (-1: none yet)
};
constexpr int kNoAllocMaxDevices = 64;
NoAllocDevice g_noalloc_dev[kNoAllocMaxDevices];
std::mutex g_noalloc_mutex;               // host bookkeeping only; it orders nothing on the GPU

}  // namespace

extern "C" int opo_spectrum_noalloc(const void* dev_in, void* dev_out, int log2_n, int batch, int precision, void* cuda_stream) {
    if (!dev_in || !dev_out) return fail(nullptr, OPO_ERR_INVALID_ARG, "opo_spectrum_noalloc: null buffer");
    if (precision != OPO_PRECISION_C64 && precision != OPO_PRECISION_C128)
        return fail(nullptr, OPO_ERR_INVALID_ARG, "opo_spectrum_noalloc: precision must be 0 (c64) or 1 (c128)");
    if (batch <= 0) return fail(nullptr, OPO_ERR_INVALID_ARG, "opo_spectrum_noalloc: batch must be positive");
    if (log2_n < opo::kMinLog2) return fail(nullptr, OPO_ERR_INVALID_ARG, "opo_spectrum_noalloc: log2_n below 4");
    const bool dbl = precision == OPO_PRECISION_C128;
    const int max_log2 = dbl ? kNoAllocMaxLog2C128 : kNoAllocMaxLog2C64;
    if (log2_n > max_log2)
        return fail(nullptr, OPO_ERR_UNSUPPORTED, "opo_spectrum_noalloc: N = 2^" + std::to_string(log2_n) + " does not fit the built-in table space (limit 2^" +
                                                      std::to_string(max_log2) + " points per row at this precision); use a handle and opo_get_fields for longer rows");
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return fail(nullptr, OPO_ERR_CUDA, std::string("opo_spectrum_noalloc: no usable CUDA device: ") + cudaGetErrorString(cudaGetLastError()));
    if (dev < 0 || dev >= kNoAllocMaxDevices) return fail(nullptr, OPO_ERR_UNSUPPORTED, "opo_spectrum_noalloc: device ordinal above 63");

    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    NoAllocDevice& d = g_noalloc_dev[dev];
    if (!d.base) {
        // set-up, once per device, with that device current: ask the runtime where this GPU's copy of the array lives
        int major = 0;
        if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess || major != 10)
            return fail(nullptr, OPO_ERR_CUDA, "opo_spectrum_noalloc: libopo is built for sm_100a only");
        unsigned char* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return fail(nullptr, OPO_ERR_CUDA, std::string("opo_spectrum_noalloc: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
        }
        d.base = p;
    }
    const int N = 1 << log2_n;
    if (d.log2_n != log2_n || d.precision != precision) {
        // The array still holds the tables of the last call on this device; they serve only that size and precision.
        // Overwrite them in stream order (earlier launches on `stream` finish reading first); launches on OTHER streams
        // that are still reading them are not waited for -- see the header.
        d.log2_n = d.precision = -1;
        const HostPlan pl(log2_n);
        const std::vector<cd> tw = pass_twiddles(pl);
        std::vector<int> perm((size_t)N);
        for (int pos = 0; pos < N; ++pos) perm[pos] = pl.freq_of_pos(pos);
        cudaError_t e;
        if (dbl) {
            e = cudaMemcpyAsync(d.base, tw.data(), tw.size() * sizeof(cd), cudaMemcpyHostToDevice, stream);
        } else {
            std::vector<float> tmp(2 * tw.size());
            for (size_t i = 0; i < tw.size(); ++i) round_unit(tw[i].real(), tw[i].imag(), &tmp[2 * i], &tmp[2 * i + 1]);
            e = cudaMemcpyAsync(d.base, tmp.data(), tmp.size() * sizeof(float), cudaMemcpyHostToDevice, stream);
        }
        if (e == cudaSuccess) e = cudaMemcpyAsync(d.base + kNoAllocTwBytes, perm.data(), perm.size() * sizeof(int), cudaMemcpyHostToDevice, stream);
        // the sources are pageable temporaries: wait until the copies have left them
        if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
        if (e != cudaSuccess) return fail(nullptr, OPO_ERR_CUDA, std::string("opo_spectrum_noalloc: table upload: ") + cudaGetErrorString(e));
        d.log2_n = log2_n;
        d.precision = precision;
    }
    const opo::FreqArgs a{dev_in, dev_out, reinterpret_cast<const int*>(d.base + kNoAllocTwBytes), d.base, batch};
    const cudaError_t e = dbl ? opo::launch_freq_f64(log2_n, a, stream) : opo::launch_freq_f32(log2_n, a, stream);
    if (e != cudaSuccess) return fail(nullptr, e == cudaErrorNotSupported ? OPO_ERR_UNSUPPORTED : OPO_ERR_CUDA, std::string("opo_spectrum_noalloc: launch: ") + cudaGetErrorString(e));
    return OPO_OK;
}
