// opo_internal.h -- plain-C++ interface between the host library (opo_api.cu) and the templated
// kernel launchers (opo_inst.cu, opo_inst_solo.cu, opo_inst_wide.cu, opo_inst_large.cu, one object per precision and size,
// routed by opo_dispatch.cu).  No CUDA templates leak through here.
#pragma once
#include <cuda_runtime.h>

namespace opo {

constexpr int kMinLog2 = 4;
constexpr int kMaxLog2Smem = 14;   // one field in one SM's shared memory (fp32); fp64: 13
constexpr int kMaxLog2 = 18;       // large-N engine above kMaxLog2Smem

// ---- streaming engine ------------------------------------------------------------------------------
// One CTA per (slot, instance): dst[b] = IDFT( tab[b?] .* DFT(src[b]) ), optionally also to dst2.
struct LinSlot {
    const void* src;       // [B][N]
    void* dst;             // [B][N]
    void* dst2;            // optional second destination (exit buffer), may be null
    const void* tab;       // mid-pass table, [N] or [B][N] in the layout of mid_pass_smem
    long long tab_stride;  // elements between instances (0 = shared)
};
struct LinArgs {
    LinSlot slot[3];
    int n_slots;
    int batch;
    const void* tw;        // pass twiddles
};

struct Rk4Args {
    void* A[3];            // current fields, [B][N]
    int n_fields;          // 2 | 3
    int batch;
    int n;                 // N
    double kappa[3];       // coupling of each equation (two-wave: kappa[0] already halved, reading R5)
    double h;
    const void* phase;     // [B][2 nz + 1] complex: exp(i dk_b * j * h/2)
    int phase_stride;      // 2 nz + 1
    int step;              // z-step index s: stage phases at 2s, 2s+1, 2s+2 (phase_index < 0)
    int phase_index;       // >= 0: stage phases at phase_index, +1, +2 instead (N/2 - L - N/2: steps of h/4)
};

// A[b][n] *= E[n]  (intracavity phase modulator exp(i beta sin(2 pi f tau_n)); also the
// frequency-domain table multiply of the cuFFT baseline engine)
struct MulTabArgs {
    void* A;
    const void* E;         // [N] complex, or [B][N] with tab_stride = N
    int batch, n;
    long long tab_stride;  // elements between instances (0 = shared)
};

// A[b][n] *= m[b]  (mirror sqrt(R) e^{i delta}, Eq. 6)
struct ScaleArgs {
    void* A;
    const void* m;         // [B] complex
    int batch, n;
};

// out[b][perm[pos]] = DFT(src[b])[pos]  (frequency-domain read-out, natural order)
struct FreqArgs {
    const void* src;
    void* dst;
    const int* perm;       // digit-reversed position -> frequency index
    const void* tw;
    int batch;
};

// ---- resident (cluster) engine and solo engine ---------------------------------------------------------
// Cluster engine: one thread-block cluster per instance, CTA rank = field (opo_resident.cuh).
// Solo engine: one CTA per instance, one field in shared memory, the others in tensor memory (opo_solo.cuh).
// Wide engine: one cluster of 4 F CTAs per instance, every field split over four CTAs (opo_wide.cuh).
struct ResidentArgs {
    void* cur[3];          // [B][N] current fields (read at start, written at end)
    const void* S[3];      // stored inputs (non-resonant fields restart from these)
    void* exitb[3];        // exit fields (z = L of the last pass), written when write_exit
    void* SH[3];           // scratch [B][N]: IDFT(H DFT(S_x)) of non-resonant fields
    const void* tabH[3];   // half step            (shared): [tab_cycle_mask + 1][N], cycled like tabH2 (copy 0 = the plain rounding)
    const void* tabH2[3];  // merged full step     (shared): [tab_cycle_mask + 1][N], a cycle of roundings with error feedback
                           //   (opo_api.cu build_tables); the k-th full step the handle applies uses copy k & tab_cycle_mask
    const void* tabHB[3];  // H G m H merged across the boundary (resonant; maybe per instance)
    const void* tabGM[3];  // G m / N, un-merged boundary       (resonant; maybe per instance)
    const void* tabHG[3];  // H G m / N: last half-step + boundary, used when a modulator (eom) follows
    long long tab_stride[3];   // instance stride of HB / GM (0 = shared)
    const void* mirror[3]; // [B] complex sqrt(R) e^{i delta} (used when the boundary has no G)
    const void* eom[3];    // [N] complex exp(i beta sin(2 pi f tau_n)) applied after the boundary of the call's last
                           // round trip, or null
    int boundary_fft[3];   // resonant field needs the transform pair at the boundary
    int resonant[3];
    double inject;         // resonant pump (field 0): sqrt(1 - R_p), the input coupler adds inject * S_p at every boundary (R24); else 0
    const void* tw;
    const void* phase;     // as Rk4Args
    int phase_stride;
    double kappa[3];
    double h;
    int n_fields, batch, nz;   // nz = steps per pass
    int tab_cycle_mask;    // see tabH2
    // What the handle has applied before this call (opo_api.cu advances them after every launch), so that neither cycle of
    // roundings nor the bunched constant correction restarts with the call: z-step-by-z-step driving (PAPER.md:L266-297,
    // Listing 3 is such a loop) then sees the same sequence of tables and corrections as one long call.
    int op0;               //   linear-operator applications (selects the applications that carry kConstBunch low parts)
    int hq0;               //   uses of the half-step table (copy (hq0 + k) & tab_cycle_mask of tabH is used next)
    int fq0;               //   uses of the full-step table (likewise for tabH2)
    int wide_g;            // wide engine: sub-blocks per CTA (1: clusters of 4 F CTAs, 2: clusters of 2 F CTAs)
    int mode;              // 0 = propagate `steps` z-steps from step index z0; 1 = `steps` round trips
    int split;             // 1 (mode 1 only): work is dealt to the clusters in round trips, not instances (opo_resident.cuh)
    int* flags;            // [B][F] round trips completed per (instance, field), zeroed before a split launch
    // pump train inside the launch (solo engine, mode 1): round trip r of the call is pumped by
    // slice r, and the exit field `out_field` of round trip r goes to out_train[r]
    const void* train;     // [steps][N] (train_inst_stride = 0) or [steps][B][N] (train_inst_stride = N); null: no train
    long long train_stride;        // elements between slices
    long long train_inst_stride;
    void* out_train;       // [steps][B][N] or null
    int out_field;
    int dk0;               // 1: dk = 0 for every instance (and nln = 0): the kernel variant without stage phases
    int nln;               // 1: order N/2 - L - N/2 (Eq. 10-11); phase table then has stride 4 nz + 1 (steps of h/4)
                           //    and mode 1 takes steps = 1
    int z0;
    int steps;
};

struct ResidentInfo {
    int threads;
    size_t smem_bytes;
    int max_clusters;      // co-resident clusters (0 = cannot launch)
};

// ---- large-N engine ------------------------------------------------------------------------------------
// One persistent cooperative kernel, four-step decomposition N = N1 x N2.  See opo_large.cuh.
struct LargeArgs {
    void* cur[3];              // [B][N] fields, transformed in place (mode 2: the scratch the column pass writes)
    void* src_override[3];     // mode 2: where the column pass reads instead of cur (may be null)
    void* out[3];              // mode 2: natural-order frequency-domain destination
    void* SH[3];               // scratch [B][N]: row-domain image of IDFT(H DFT(S_x)) of non-resonant fields
    const void* tabH[3];       // first / last operator of the call (half step; or G m for the boundary-only call)
    long long tabH_stride[3];  // instance stride of tabH in table elements (0 = shared)
    const void* tabH2[3];      // merged full step
    const void* tabHB[3];      // merged across the boundary (resonant fields)
    long long tabHB_stride[3];
    const void* tw1;           // pass twiddles of the column transform (plan<L1>)
    const void* tw2;           // pass twiddles of the row transform (plan<L2>)
    const void* wlo;           // W_N^j, j < N1
    const void* whi;           // W_N^{j N1}, j < N2
    const int* perm1;          // row index -> k1 (digit reversal of the column transform)
    const int* perm2;          // position in a transformed row -> k2
    const void* phase;         // as Rk4Args
    int phase_stride;
    double kappa[3];
    double h;
    int resonant[3];
    int field_mask;            // bit x set: field x takes part
    int n_fields, batch, nz;
    int mode;                  // 0 = `steps` z-steps from step index z0 (steps = 0: one linear operator with tabH);
                               // 1 = `steps` round trips; 2 = forward DFT read-out
    int z0;
    int steps;
    int nln;                   // 1: order N/2 - L - N/2; phase table in steps of h/4; mode 1 takes steps = 1
    int op0;                   // linear operators the handle has applied before this launch (the every-FIX_EVERY-th twiddle defect
                               // correction is keyed on op0 + q, not on the call's own q)
    unsigned long long* barrier;        // zeroed by the host before the launch
    unsigned long long barrier_base;    // counter value at launch (0)
};

struct LargeInfo {
    int threads;
    size_t smem_bytes;
    int max_ctas;          // co-resident CTAs on the device
    int grid;              // CTAs to launch for this batch
    int n1, n2;
};

#define OPO_DECLARE_LAUNCHERS(SUFFIX)                                                   \
    cudaError_t launch_linear_##SUFFIX(int log2n, const LinArgs& a, cudaStream_t s);    \
    cudaError_t launch_rk4_##SUFFIX(const Rk4Args& a, cudaStream_t s);                  \
    cudaError_t launch_scale_##SUFFIX(const ScaleArgs& a, cudaStream_t s);              \
    cudaError_t launch_multab_##SUFFIX(const MulTabArgs& a, cudaStream_t s);            \
    cudaError_t launch_freq_##SUFFIX(int log2n, const FreqArgs& a, cudaStream_t s);     \
    cudaError_t launch_finite_##SUFFIX(const void* A, long long count, int* flag, cudaStream_t s); \
    cudaError_t launch_broadcast_##SUFFIX(void* dst, int batch, int n, cudaStream_t s); \
    cudaError_t launch_axpy_##SUFFIX(void* A, const void* S, double c, int accumulate, long long count, cudaStream_t s); \
    cudaError_t resident_info_##SUFFIX(int log2n, int n_fields, ResidentInfo* out);     \
    cudaError_t launch_resident_##SUFFIX(int log2n, const ResidentArgs& a, int n_clusters, cudaStream_t s); \
    cudaError_t solo_info_##SUFFIX(int log2n, int n_fields, ResidentInfo* out);         \
    cudaError_t launch_solo_##SUFFIX(int log2n, const ResidentArgs& a, int n_ctas, cudaStream_t s); \
    cudaError_t wide_info_##SUFFIX(int log2n, int n_fields, int g, ResidentInfo* out);  \
    cudaError_t launch_wide_##SUFFIX(int log2n, const ResidentArgs& a, int n_clusters, cudaStream_t s); \
    cudaError_t large_info_##SUFFIX(int log2n, int n_fields, int batch, int sm_count, LargeInfo* out);       \
    cudaError_t launch_large_##SUFFIX(int log2n, const LargeArgs& a, int grid, cudaStream_t s);

OPO_DECLARE_LAUNCHERS(f32)
OPO_DECLARE_LAUNCHERS(f64)

}  // namespace opo
