// opo_large.cuh -- large-N engine (N = 2^15 .. 2^18; complex128 also 2^14): one field no longer
// fits one SM's shared memory (BASELINE.json configs[3]), so the transform is the four-step
// decomposition N = N1 x N2 executed by ONE persistent kernel whose CTAs meet at a grid barrier
// between memory passes.  The fields live in global memory and stay in the 126 MB L2 (4 MB of
// state at N = 2^18, two fields); HBM sees them only at the ends of a call.
//
// Index split: n = n1 N2 + n2, k = k1 + N1 k2.
//     X[k1 + N1 k2] = sum_n2 W_N2^{n2 k2} [ W_N^{n2 k1} sum_n1 x[n1 N2 + n2] W_N1^{n1 k1} ]
// A z-step (order L/2 - N - L/2, adjacent half-steps merged as in the resident engine)
// is two memory passes:
//
//   row pass    (one row k1 = N2 contiguous elements per team): W_N^{n2 k1} . DFT_N2 . table .
//               IDFT_N2 . conj W_N^{n2 k1} -- the frequency-domain part of the linear operator
//               (Eq. 5, L135 Eq. 11; boundary factors of Eq. 6 / L145 merged into the
//               table at a round-trip crossing);
//   column pass (a tile of TC adjacent columns n2, all F fields): IDFT_N1 . RK4 . DFT_N1.  The RK4
//               step of the coupling terms is pointwise in n and is fused
//               between inverse and forward radix-4 pass 0 exactly as in opo_resident.cuh.
//
// Every transform is the shared-memory machinery of opo_fft.cuh run by a *team* of N/16 threads
// (several teams per CTA); digit-reversed orders are absorbed by the host tables (perm1: row index
// -> k1; the row table is stored per row in mid-pass layout).  W_N^{n2 k1} is the product of two
// small shared-memory tables, W_N^{p} = W_N^{(p >> L1) << L1} . W_N^{p & (N1-1)}.
//
// fp32: the frequency-domain table is carried as hi + lo (tabx<float>, opo_fft.cuh): at 10^4..10^5
// z-steps the rounding of a single-float table entry is a coherent per-bin drift above tolerance.
#pragma once
#include "opo_kernels.cuh"

namespace opo {

#ifndef OPO_LARGE_TC
#define OPO_LARGE_TC 4
#endif

template <class T> struct large_tab { using type = cplx<T>; };
template <> struct large_tab<float> { using type = tabx<float>; };

template <class T, int L, int F> struct large_cfg {
    static constexpr int L1 = L / 2, L2 = L - L1;
    static constexpr int N1 = 1 << L1, N2 = 1 << L2, N = 1 << L;
    static constexpr int TC = OPO_LARGE_TC;            // columns per tile
    // Points per thread of a transform.  8 points per thread (twice the warps, teams of two warps with named barriers) was
    // measured SLOWER on C3 (17.0 vs 14.8 us per z-step): the compute phases are ~54 % issue-bound already, the radix-16
    // pass then runs on half a team and every thread repeats the index arithmetic.
#ifdef OPO_LARGE_PT
    static constexpr int PT = OPO_LARGE_PT;
#else
    static constexpr int PT = 16;
#endif
    static constexpr int TT1 = N1 / PT, TT2 = N2 / PT; // threads per column / row transform (a "team")
    // barrier of a team between passes: teams of <= 32 threads never span warps (pass_sync in opo_fft.cuh)
    static constexpr int SY1 = TT1 <= 32 ? 1 : TT1, SY2 = TT2 <= 32 ? 1 : TT2;
    static constexpr int NT = F * TC * TT1;            // one team per (field, column)
    static constexpr int ROWS = NT / TT2;              // rows per chunk in the row pass
    static constexpr int SKEW = (128 / (int)sizeof(cplx<T>)) / TC;   // makes the transposing tile load conflict-free
    static constexpr int CSTRIDE = padded_len<T>(N1) + SKEW;
    static constexpr int RSTRIDE = padded_len<T>(N2);
    static constexpr int FIELD_ELEMS = (F * TC * CSTRIDE > ROWS * RSTRIDE) ? F * TC * CSTRIDE : ROWS * RSTRIDE;
    static constexpr int TW1 = plan<L1>::tw_total, TW2 = plan<L2>::tw_total;
    static constexpr int SMEM_ELEMS = FIELD_ELEMS + TW1 + TW2 + N1 + N2;
    static constexpr size_t BASE_BYTES = (size_t)SMEM_ELEMS * sizeof(cplx<T>);
    // Per-CTA caches of what a row team needs at EVERY z-step when the CTA keeps the same rows for the whole launch (one
    // chunk per CTA: C3): the rows' slice of the merged full-step table H2 (fp32: hi + lo, 16 B per entry -- 8 MB per
    // z-step out of L2 otherwise, which is what the row pass was waiting for), and (fp32) the rows' four-step twiddles
    // W_N^{n2 k1} with their magnitude defects; plus (fp32) the defects of the pass twiddles.
    static constexpr size_t TABC_BYTES = (size_t)ROWS * N2 * sizeof(typename large_tab<T>::type);
    static constexpr size_t WC_BYTES = sizeof(T) == 4 ? (size_t)ROWS * N2 * (sizeof(cplx<T>) + sizeof(float)) : 0;
    static constexpr size_t DTW_BYTES = sizeof(T) == 4 ? (size_t)(TW1 + TW2) * sizeof(float) : 0;
    static constexpr size_t CACHE_OFFSET = (BASE_BYTES + 15) / 16 * 16;
    static constexpr bool CACHE = CACHE_OFFSET + TABC_BYTES + WC_BYTES + DTW_BYTES <= 232448;
    static constexpr size_t SMEM_BYTES = CACHE ? CACHE_OFFSET + TABC_BYTES + WC_BYTES + DTW_BYTES : CACHE_OFFSET + DTW_BYTES;
    static constexpr int TILES_PER_INST = N2 / TC;
    static constexpr int CHUNKS_PER_FIELD = (N1 + ROWS - 1) / ROWS;
    static_assert(ROWS >= 1, "a CTA must hold at least one row");
    static_assert((TT1 <= 32 || F * TC <= 15) && (TT2 <= 32 || ROWS <= 15), "one named barrier per team");
};

// coherent (L2) load of field data written by other SMs earlier in the same launch
__device__ __forceinline__ cplx<float> ldcg(const cplx<float>* p) {
    float2 v = __ldcg(reinterpret_cast<const float2*>(p));
    return {v.x, v.y};
}
__device__ __forceinline__ cplx<double> ldcg(const cplx<double>* p) {
    double2 v = __ldcg(reinterpret_cast<const double2*>(p));
    return {v.x, v.y};
}

// All CTAs of the (cooperatively launched, hence co-resident) grid meet here.  Monotone counter:
// barrier number j completes when the counter reaches j * gridDim.x.
__device__ __forceinline__ void grid_barrier(unsigned long long* ctr, unsigned long long& target) {
    target += gridDim.x;
    __syncthreads();
    if (threadIdx.x == 0) {
        // arrive: the release orders this CTA's global stores (made visible to this thread by the __syncthreads) before
        // the increment; wait: relaxed polls (no cache invalidation per poll), one acquire fence at the end
        asm volatile("red.release.gpu.global.add.u64 [%0], 1;" ::"l"(ctr) : "memory");
        unsigned long long v;
        do {
            asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(ctr) : "memory");
        } while (v < target);
        asm volatile("fence.acq_rel.gpu;" ::: "memory");
    }
    __syncthreads();
}

// inverse pass 0 -> RK4 -> forward pass 0 for butterfly t of all F fields held in local shared memory
template <class T, int L, int F>
__device__ __forceinline__ void pass0_rk4_local(cplx<T>* const* fld, int t, const cplx<T>* __restrict__ tw0s,
                                                cplx<T> e0, cplx<T> e1, cplx<T> e2, const T* kap, T h,
                                                bool two = false, cplx<T> e3 = cplx<T>{}, cplx<T> e4 = cplx<T>{},
                                                const float* __restrict__ dtw0 = nullptr) {
    constexpr int RB = 2, R = 4, SB = L - 2, S = 1 << SB;
    cplx<T> w[R - 1];
#pragma unroll
    for (int k = 0; k < R - 1; ++k) w[k] = tw0s[k * S + t];
    const int p0 = elem_base<T, RB, SB>(0, t);
    cplx<T> v[F][R];
#pragma unroll
    for (int x = 0; x < F; ++x)
#pragma unroll
        for (int k = 0; k < R; ++k) v[x][k] = fld[x][p0 + elem_off<T, RB, SB>(k)];
    // dtw0 (fp32): the magnitude defects to take out of the twiddles in this application (cmulc_unit); null: plain multiply
    if (sizeof(T) == 4 && dtw0 != nullptr) {
        float wd[R - 1];
#pragma unroll
        for (int k = 0; k < R - 1; ++k) wd[k] = dtw0[k * S + t];
#pragma unroll
        for (int x = 0; x < F; ++x)
#pragma unroll
            for (int k = 1; k < R; ++k) v[x][k] = cmulc_unit(v[x][k], w[k - 1], wd[k - 1]);
    } else {
#pragma unroll
        for (int x = 0; x < F; ++x)
#pragma unroll
            for (int k = 1; k < R; ++k) v[x][k] = cmulc(v[x][k], w[k - 1]);
    }
#pragma unroll
    for (int x = 0; x < F; ++x) dit_inv<T, R>::run(v[x]);
#pragma unroll
    for (int j = 0; j < R; ++j) {
        cplx<T> y[F];
#pragma unroll
        for (int x = 0; x < F; ++x) y[x] = v[x][j];
        Rk4<T, F>::step(y, e0, e1, e2, kap, h);
        if (two) Rk4<T, F>::step(y, e2, e3, e4, kap, h);      // N/2 - L - N/2: two half-steps meet here
#pragma unroll
        for (int x = 0; x < F; ++x) v[x][j] = y[x];
    }
#pragma unroll
    for (int x = 0; x < F; ++x) {
        dif<T, R>::run(v[x]);
#pragma unroll
        for (int k = 1; k < R; ++k) v[x][k] = cmul(v[x][k], w[k - 1]);
    }
#pragma unroll
    for (int x = 0; x < F; ++x)
#pragma unroll
        for (int k = 0; k < R; ++k) fld[x][p0 + elem_off<T, RB, SB>(k)] = v[x][k];
}

// COL_NFWD / COL_INVN (N/2 - L - N/2 ordering): an RK4 half-step in the time domain before the forward / after the
// inverse column transform; COL_RK4 then takes two half-steps
enum { COL_FWD = 0, COL_RK4 = 1, COL_INV = 2, COL_NFWD = 3, COL_INVN = 4 };
enum { ROW_LINEAR = 0, ROW_RELOAD = 1, ROW_FREQ = 2 };

// Diagnostic build (-DOPO_LARGE_TIMING; OPO_EXTRA_NVCC_FLAGS of build.py): thread 0 of a CTA accumulates clock64 stamps per
// phase of a z-step, two CTAs print their per-z-step averages when the launch ends (profiles/r02f_large_kernel.md).
#ifdef OPO_LARGE_TIMING
#define OPO_TSTAMP(eng, i) do { if (threadIdx.x == 0) { const long long t_ = clock64(); (eng).t_acc[i] += t_ - (eng).t_last; (eng).t_last = t_; } } while (0)
#else
#define OPO_TSTAMP(eng, i) do {} while (0)
#endif

template <class T, int L, int F> struct LargeEngine {
#ifdef OPO_LARGE_TIMING
    long long t_acc[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    long long t_last = 0;
#endif
    using C = large_cfg<T, L, F>;
    using TAB = typename large_tab<T>::type;
    using P1 = plan<C::L1>;
    using P2 = plan<C::L2>;

    cplx<T>* sm;            // tile / rows
    const cplx<T>* tw1;     // shared-memory copies
    const cplx<T>* tw2;
    const cplx<T>* wlo;     // W_N^j, j < N1
    const cplx<T>* whi;     // W_N^{j N1}, j < N2
    int tid;
    // Magnitude defects of the pass twiddles (fp32; cmulc_unit in opo_fft.cuh), indexed as tw1 / tw2.  The correction is
    // applied at every FIX_EVERY-th z-step only, FIX_EVERY times as large: the tables hold FIX_EVERY (|w|^2 - 1) and the
    // kernel sets `fix` for those z-steps (13 instructions per inverse twiddle were 19 % of the instructions of a z-step).
    // The defect operator does not commute with the dispersion step U, so bunching K corrections leaves K/2 |U - 1| of the
    // defect behind: with 8 that is a third at the band edge of C3 (0.085 rad per z-step) and a few per cent where the
    // signal lives; measured on C3 x 20 RT: 6.8e-5 with K = 1, 8 and 16 alike.
    static constexpr int FIX_EVERY = 8;
    const float* dtw1 = nullptr;
    const float* dtw2 = nullptr;
    bool fix = false;               // this z-step takes the accumulated defects out
    // row caches (large_cfg::CACHE): valid for rows of `cache_tab` handled by this CTA's teams
    const void* cache_src = nullptr;        // the global table the cached slice was copied from (null: no cache)
    const TAB* cache_tab = nullptr;         // [ROWS][N2] in mid-pass layout
    const cplx<T>* cache_w = nullptr;       // [ROWS][N2] four-step twiddles of the rows
    const float* cache_wd = nullptr;        // [ROWS][N2] their defects

    __device__ __forceinline__ cplx<T> big_twiddle(int k1, int n2) const {
        const int p = k1 * n2;
        return cmul(whi[p >> C::L1], wlo[p & (C::N1 - 1)]);
    }
    // (the row pass multiplies by w = big_twiddle on the way in and by conj(w) on the way out; in fp32 the rounded product has
    // |w|^2 = 1 + d, d ~ 1e-7, the same at every z-step: cmulc_unit takes it out, opo_fft.cuh)

    // ---- column pass over this CTA's tiles ----------------------------------------------------------
    // src/dst: per-field base pointers ([B][N]); fields outside `mask` are neither read nor written.
    template <int MODE>
    __device__ __forceinline__ void col_pass(cplx<T>* const* src, cplx<T>* const* dst, int mask, int batch,
                                             const cplx<T>* phase, int phase_stride, int pidx, const T* kap, T h, bool two = false) {
        const int n_tiles = batch * C::TILES_PER_INST;
        const int team = tid / C::TT1, lt = tid % C::TT1;
        cplx<T>* smt = sm + team * C::CSTRIDE;
#pragma unroll 1
        for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            const int b = tile / C::TILES_PER_INST, c0 = (tile % C::TILES_PER_INST) * C::TC;
            {   // all loads of the tile are in flight before the first one is consumed (the pass is latency-bound)
                constexpr int CNT = (C::N1 * C::TC + C::NT - 1) / C::NT;
                cplx<T> r[F][CNT];
#pragma unroll
                for (int x = 0; x < F; ++x) {
                    if (!((mask >> x) & 1)) continue;
                    const cplx<T>* g = src[x] + (size_t)b * C::N + c0;
#pragma unroll
                    for (int j = 0; j < CNT; ++j) {
                        const int i = tid + j * C::NT;
                        if (i < C::N1 * C::TC) r[x][j] = ldcg(g + (size_t)(i / C::TC) * C::N2 + (i % C::TC));
                    }
                }
#pragma unroll
                for (int x = 0; x < F; ++x) {
                    if (!((mask >> x) & 1)) continue;
#pragma unroll
                    for (int j = 0; j < CNT; ++j) {
                        const int i = tid + j * C::NT;
                        if (i < C::N1 * C::TC) sm[(x * C::TC + i % C::TC) * C::CSTRIDE + phys<T>(i / C::TC)] = r[x][j];
                    }
                }
            }
            // pointwise RK4 half-step on the tile in the time domain (Eq. 10-11)
            auto rk4_tile = [&]() {
                __syncthreads();
                const cplx<T>* ph = phase + (size_t)b * phase_stride + pidx;
                const cplx<T> e0 = ldg(ph), e1 = ldg(ph + 1), e2 = ldg(ph + 2);
#pragma unroll 1
                for (int it = tid; it < C::TC * C::N1; it += C::NT) {
                    const int c = it / C::N1, n1 = it % C::N1;
                    cplx<T> y[F];
#pragma unroll
                    for (int x = 0; x < F; ++x) y[x] = sm[(x * C::TC + c) * C::CSTRIDE + phys<T>(n1)];
                    Rk4<T, F>::step(y, e0, e1, e2, kap, h);
#pragma unroll
                    for (int x = 0; x < F; ++x) sm[(x * C::TC + c) * C::CSTRIDE + phys<T>(n1)] = y[x];
                }
            };
#ifdef OPO_LARGE_TIMING
            __syncthreads();
            OPO_TSTAMP(*this, 0);                           // column tile loaded
#endif
            if constexpr (MODE == COL_NFWD) rk4_tile();
            if constexpr (MODE != COL_FWD && MODE != COL_NFWD) {
                __syncthreads();
                inv_pass_smem<T, C::L1, P1::P - 1, C::TT1, true>(smt, tw1, lt);
                inv_passes<T, C::L1, C::TT1, true, ((MODE == COL_INV || MODE == COL_INVN) ? 0 : 1), C::SY1, true>(smt, tw1, lt, 1 + team, fix ? dtw1 : nullptr);
            }
            if constexpr (MODE == COL_INVN) rk4_tile();
            if constexpr (MODE == COL_RK4) {
                __syncthreads();
                const cplx<T>* ph = phase + (size_t)b * phase_stride + pidx;
                const cplx<T> e0 = ldg(ph), e1 = ldg(ph + 1), e2 = ldg(ph + 2);
                const cplx<T> e3 = two ? ldg(ph + 3) : e2, e4 = two ? ldg(ph + 4) : e2;
                constexpr int S = C::N1 / 4;
#pragma unroll 1
                for (int it = tid; it < C::TC * S; it += C::NT) {
                    const int c = it / S, t = it % S;
                    cplx<T>* fld[F];
#pragma unroll
                    for (int x = 0; x < F; ++x) fld[x] = sm + (x * C::TC + c) * C::CSTRIDE;
                    pass0_rk4_local<T, C::L1, F>(fld, t, tw1 + P1::tw_offset(0), e0, e1, e2, kap, h, two, e3, e4,
                                                 (fix && dtw1 != nullptr) ? dtw1 + P1::tw_offset(0) : nullptr);
                }
            }
            if constexpr (MODE != COL_INV && MODE != COL_INVN) {
                __syncthreads();
                fwd_passes<T, C::L1, C::TT1, true, ((MODE == COL_FWD || MODE == COL_NFWD) ? 0 : 1), C::SY1>(smt, tw1, lt, 1 + team);
                fwd_pass_smem<T, C::L1, P1::P - 1, C::TT1, true>(smt, tw1, lt);
            }
            __syncthreads();
            OPO_TSTAMP(*this, 1);                           // column transforms + RK4
#pragma unroll
            for (int x = 0; x < F; ++x) {
                if (!((mask >> x) & 1)) continue;
                cplx<T>* g = dst[x] + (size_t)b * C::N + c0;
#pragma unroll 4
                for (int i = tid; i < C::N1 * C::TC; i += C::NT) {
                    const int n1 = i / C::TC, c = i % C::TC;
                    g[(size_t)n1 * C::N2 + c] = sm[(x * C::TC + c) * C::CSTRIDE + phys<T>(n1)];
                }
            }
            __syncthreads();
            OPO_TSTAMP(*this, 2);                           // column tile stored
        }
    }

    // ---- row pass over this CTA's chunks of ROWS rows ----------------------------------------------------
    struct RowOp {
        int kind[3];              // ROW_LINEAR / ROW_RELOAD / ROW_FREQ per field; -1 = skip the field
        const TAB* tab[3];        // ROW_LINEAR: table of the field, [N] or per instance
        long long tab_stride[3];
        cplx<T>* sh_store[3];     // ROW_LINEAR: also store the result here (may be null)
        const cplx<T>* aux[3];    // ROW_RELOAD: source (SH); ROW_FREQ: unused
        cplx<T>* out[3];          // ROW_FREQ: natural-order destination
    };

    // The row pass begins with the grid barrier that separates it from the column pass before it: everything that does not
    // depend on the fields (multiplier table entries from L2, the row's twiddles) is requested BEFORE that barrier, so its
    // latency is spent while the CTA waits for the slowest column tile anyway.
    // element x of a per-field array by a chain of selects: the arrays of RowOp stay in registers (indexed with a runtime x
    // they went to local memory, and every row pass began with a chain of dependent local loads: 1.5 k cycles)
    template <class A> static __device__ __forceinline__ A pick(const A* arr, int x) {
        A v = arr[0];
#pragma unroll
        for (int f = 1; f < F; ++f) v = (x == f) ? arr[f] : v;
        return v;
    }

    __device__ __forceinline__ void row_pass(cplx<T>* const* data, const RowOp& op, int batch, const int* __restrict__ perm1,
                                             const int* __restrict__ perm2, unsigned long long* bar_ctr, unsigned long long& bar_target) {
        const int n_chunks = batch * F * C::CHUNKS_PER_FIELD;
        const int team = tid / C::TT2, lt = tid % C::TT2;
        cplx<T>* smt = sm + team * C::RSTRIDE;
        bool synced = false;        // uniform over the CTA
        auto sync_once = [&]() {
            if (!synced) { grid_barrier(bar_ctr, bar_target); synced = true; }
        };
#pragma unroll 1
        for (int chunk = blockIdx.x; chunk < n_chunks; chunk += gridDim.x) {
            const int b = chunk / (F * C::CHUNKS_PER_FIELD);
            const int rem = chunk % (F * C::CHUNKS_PER_FIELD);
            const int x = rem / C::CHUNKS_PER_FIELD;
            const int r = (rem % C::CHUNKS_PER_FIELD) * C::ROWS + team;
            const int kind = pick(op.kind, x);
            if (kind < 0) continue;                                 // uniform over the CTA
            const bool active = r < C::N1;
            const size_t off = (size_t)b * C::N + (size_t)(active ? r : 0) * C::N2;
            cplx<T>* g = pick(data, x) + off;
            if (kind == ROW_RELOAD) {
                sync_once();
                if (active) {
                    const cplx<T>* __restrict__ a = pick(op.aux, x) + off;
#pragma unroll 4
                    for (int i = lt; i < C::N2; i += C::TT2) g[i] = ldcg(a + i);
                }
                continue;
            }
            // this CTA's rows of this table are in shared memory (merged full step H2: every z-step but the ends of a pass)
            const bool cached = kind == ROW_LINEAR && cache_src != nullptr && cache_src == (const void*)pick(op.tab, x) && pick(op.tab_stride, x) == 0;
            const int k1 = (cached && sizeof(T) == 4) ? 0 : __ldg(&perm1[active ? r : 0]);      // (the cached twiddles need no k1)
            // A row is one team's business from its first load to its last store: every barrier of the row pass is the
            // team's own (a __syncwarp, or a named barrier when the team has two warps), the teams of a CTA drift apart and
            // one row's loads run under another row's arithmetic.  All loads of the row -- data and multiplier table -- are in flight
            // before the first one is consumed (the pass is bound by latency, not by bandwidth).
            constexpr int CNT = C::N2 / C::TT2;
            constexpr int RM = 1 << P2::rbits(P2::P - 1), NBM = C::N2 / RM, NIT = NBM / C::TT2;
            static_assert(NBM % C::TT2 == 0, "whole iterations of the middle pass per team");
            cplx<T> rv[CNT];
            if (kind == ROW_FREQ) {
                sync_once();
                if (active) {
#pragma unroll
                    for (int j = 0; j < CNT; ++j) rv[j] = ldcg(g + lt + j * C::TT2);
                }
                if (active) {
#pragma unroll
                    for (int j = 0; j < CNT; ++j) smt[phys<T>(lt + j * C::TT2)] = cmul(rv[j], big_twiddle(k1, lt + j * C::TT2));
                }
                pass_sync<C::SY2>(1 + team);
                fwd_passes<T, C::L2, C::TT2, true, 0, C::SY2>(smt, tw2, lt, 1 + team);
                fwd_pass_smem<T, C::L2, P2::P - 1, C::TT2, true>(smt, tw2, lt);
                pass_sync<C::SY2>(1 + team);
                if (active) {
                    cplx<T>* o = pick(op.out, x) + (size_t)b * C::N + k1;
#pragma unroll 4
                    for (int i = lt; i < C::N2; i += C::TT2) o[(size_t)__ldg(&perm2[i]) * C::N1] = smt[phys<T>(i)];
                }
            } else {
                const TAB* tab = pick(op.tab, x) + (size_t)b * pick(op.tab_stride, x) + (size_t)(active ? r : 0) * C::N2;
                TAB hh[NIT][RM];
                cplx<T> w[CNT];
                float wd[CNT];
                if (!cached) {
#pragma unroll
                    for (int it = 0; it < NIT; ++it)
#pragma unroll
                        for (int k = 0; k < RM; ++k) hh[it][k] = ldg(&tab[k * NBM + lt + it * C::TT2]);
#pragma unroll
                    for (int j = 0; j < CNT; ++j) {
                        w[j] = big_twiddle(k1, lt + j * C::TT2);
                        if constexpr (sizeof(T) == 4) wd[j] = fix ? (float)FIX_EVERY * unit_defect(w[j]) : 0.0f;
                        else wd[j] = 0.0f;
                    }
                }
                OPO_TSTAMP(*this, 3);                       // row prologue
                sync_once();
                OPO_TSTAMP(*this, 4);                       // grid barrier after the column pass
                if (active) {
#pragma unroll
                    for (int j = 0; j < CNT; ++j) rv[j] = ldcg(g + lt + j * C::TT2);
                }
                if (cached) {
                    if constexpr (sizeof(T) == 4) {
#pragma unroll
                        for (int j = 0; j < CNT; ++j) {
                            w[j] = cache_w[team * C::N2 + lt + j * C::TT2];
                            wd[j] = fix ? cache_wd[team * C::N2 + lt + j * C::TT2] : 0.0f;
                        }
                    } else {
#pragma unroll
                        for (int j = 0; j < CNT; ++j) { w[j] = big_twiddle(k1, lt + j * C::TT2); wd[j] = 0.0f; }
                    }
                }
                if (active) {
#pragma unroll
                    for (int j = 0; j < CNT; ++j) smt[phys<T>(lt + j * C::TT2)] = cmul(rv[j], w[j]);
                }
                pass_sync<C::SY2>(1 + team);
                OPO_TSTAMP(*this, 5);                       // row loaded (team 0)
                fwd_passes<T, C::L2, C::TT2, true, 0, C::SY2>(smt, tw2, lt, 1 + team);
                if (cached) {
                    const TAB* ct = cache_tab + team * C::N2;
#pragma unroll
                    for (int it = 0; it < NIT; ++it)
#pragma unroll
                        for (int k = 0; k < RM; ++k) hh[it][k] = ct[k * NBM + lt + it * C::TT2];
                }
#pragma unroll
                for (int it = 0; it < NIT; ++it) mid_bf<T, C::L2, TAB>(smt, hh[it], lt + it * C::TT2);
                inv_passes<T, C::L2, C::TT2, true, 0, C::SY2, true>(smt, tw2, lt, 1 + team, fix ? dtw2 : nullptr);
                pass_sync<C::SY2>(1 + team);
                OPO_TSTAMP(*this, 6);                       // row transforms (team 0)
                if (active) {
                    cplx<T>* sh = pick(op.sh_store, x) ? pick(op.sh_store, x) + off : nullptr;
                    if (sizeof(T) == 4 && fix) {
#pragma unroll
                        for (int j = 0; j < CNT; ++j) {
                            const int i = lt + j * C::TT2;
                            const cplx<T> v = cmulc_unit(smt[phys<T>(i)], w[j], wd[j]);
                            g[i] = v;
                            if (sh) sh[i] = v;
                        }
                    } else {
#pragma unroll
                        for (int j = 0; j < CNT; ++j) {
                            const int i = lt + j * C::TT2;
                            const cplx<T> v = cmulc(smt[phys<T>(i)], w[j]);
                            g[i] = v;
                            if (sh) sh[i] = v;
                        }
                    }
                }
            }
            pass_sync<C::SY2>(1 + team);
        }
        sync_once();        // a CTA without a row of its own still takes part in the barrier
    }
};

template <class T, int L, int F>
__global__ void __launch_bounds__(large_cfg<T, L, F>::NT, 1) k_large(LargeArgs a) {
    using C = large_cfg<T, L, F>;
    using E = LargeEngine<T, L, F>;
    using TAB = typename E::TAB;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
    const int tid = threadIdx.x;

    E e;
    e.sm = sm;
    e.tid = tid;
    {
        cplx<T>* p = sm + C::FIELD_ELEMS;
        auto copy = [&](const void* srcv, int count) {
            const cplx<T>* src = reinterpret_cast<const cplx<T>*>(srcv);
            for (int i = tid; i < count; i += C::NT) p[i] = ldg(&src[i]);
            const cplx<T>* r = p;
            p += count;
            return r;
        };
        e.tw1 = copy(a.tw1, C::TW1);
        e.tw2 = copy(a.tw2, C::TW2);
        e.wlo = copy(a.wlo, C::N1);
        e.whi = copy(a.whi, C::N2);
    }
    __syncthreads();
    if constexpr (sizeof(T) == 4) {     // magnitude defects of the pass twiddles
        float* d = reinterpret_cast<float*>(smem_raw + C::CACHE_OFFSET + (C::CACHE ? C::TABC_BYTES + C::WC_BYTES : 0));
        for (int i = tid; i < C::TW1; i += C::NT) d[i] = (float)E::FIX_EVERY * unit_defect(e.tw1[i]);
        for (int i = tid; i < C::TW2; i += C::NT) d[C::TW1 + i] = (float)E::FIX_EVERY * unit_defect(e.tw2[i]);
        e.dtw1 = d;
        e.dtw2 = d + C::TW1;
    }
    if constexpr (C::CACHE) {
        // one chunk of rows per CTA for the whole launch: keep the rows' slice of H2 and their four-step twiddles on chip
        const int n_chunks = a.batch * F * C::CHUNKS_PER_FIELD;
        if (a.mode != 2 && n_chunks <= (int)gridDim.x && (int)blockIdx.x < n_chunks) {
            const int rem = blockIdx.x % (F * C::CHUNKS_PER_FIELD);
            const int x = rem / C::CHUNKS_PER_FIELD, r0 = (rem % C::CHUNKS_PER_FIELD) * C::ROWS;
            if ((a.field_mask >> x) & 1) {
                const TAB* src = reinterpret_cast<const TAB*>(a.tabH2[x]);
                TAB* ct = reinterpret_cast<TAB*>(smem_raw + C::CACHE_OFFSET);
                for (int i = tid; i < C::ROWS * C::N2; i += C::NT) {
                    const int rr = r0 + i / C::N2;
                    if (rr < C::N1) ct[i] = ldg(&src[(size_t)rr * C::N2 + i % C::N2]);
                }
                e.cache_src = src;
                e.cache_tab = ct;
                if constexpr (sizeof(T) == 4) {
                    cplx<T>* cw = reinterpret_cast<cplx<T>*>(smem_raw + C::CACHE_OFFSET + C::TABC_BYTES);
                    float* cd = reinterpret_cast<float*>(smem_raw + C::CACHE_OFFSET + C::TABC_BYTES + (size_t)C::ROWS * C::N2 * sizeof(cplx<T>));
                    for (int i = tid; i < C::ROWS * C::N2; i += C::NT) {
                        const int rr = r0 + i / C::N2;
                        if (rr < C::N1) {
                            const cplx<T> w = e.big_twiddle(__ldg(&a.perm1[rr]), i % C::N2);
                            cw[i] = w;
                            cd[i] = (float)E::FIX_EVERY * unit_defect(w);
                        }
                    }
                    e.cache_w = cw;
                    e.cache_wd = cd;
                }
            }
        }
    }
    __syncthreads();

    cplx<T>* cur[F];
    cplx<T>* srcp[F];
    cplx<T>* dstp[F];
#pragma unroll
    for (int x = 0; x < F; ++x) {
        cur[x] = reinterpret_cast<cplx<T>*>(a.cur[x]);
        srcp[x] = a.src_override[x] ? reinterpret_cast<cplx<T>*>(a.src_override[x]) : cur[x];
        dstp[x] = cur[x];
    }
    const cplx<T>* phase = reinterpret_cast<const cplx<T>*>(a.phase);
    T kap[3] = {(T)a.kappa[0], (T)a.kappa[1], (T)a.kappa[2]};
    const T h = (T)a.h;
    const int nz = a.nz, batch = a.batch, mask = a.field_mask;
    unsigned long long target = a.barrier_base;
    typename E::RowOp op;

    if (a.mode == 2) {
        // frequency read-out: column transforms src -> cur slot (scratch), rows -> natural order
        e.template col_pass<COL_FWD>(srcp, dstp, mask, batch, phase, a.phase_stride, 0, kap, h);
#pragma unroll
        for (int x = 0; x < F; ++x) {
            op.kind[x] = ((mask >> x) & 1) ? ROW_FREQ : -1;
            op.out[x] = reinterpret_cast<cplx<T>*>(a.out[x]);
        }
        e.row_pass(cur, op, batch, a.perm1, a.perm2, a.barrier, target);
        return;
    }

    const bool rt_mode = a.mode == 1;
    const int total = rt_mode ? a.steps * nz : a.steps;

    if (a.nln) {
        // N/2 - L - N/2 (Eq. 10-11): [N/2] (L [N/2 N/2])^(n-1) L [N/2]; every L a full step (table H2),
        // every RK4 step of size h/2, phase table in steps of h/4; one pass per launch (mode 1: steps = 1)
        const int zs = rt_mode ? 0 : a.z0, nsteps = rt_mode ? nz : a.steps;
        const T hh = (T)0.5 * h;
        e.template col_pass<COL_NFWD>(cur, cur, mask, batch, phase, a.phase_stride, 4 * zs, kap, hh);
#pragma unroll
        for (int x = 0; x < F; ++x) {
            op.sh_store[x] = nullptr; op.aux[x] = nullptr; op.out[x] = nullptr; op.tab_stride[x] = 0;
            op.kind[x] = ((mask >> x) & 1) ? ROW_LINEAR : -1;
            op.tab[x] = reinterpret_cast<const TAB*>(a.tabH2[x]);
        }
#pragma unroll 1
        for (int q = 0; q < nsteps; ++q) {
            e.fix = ((a.op0 + q) % E::FIX_EVERY) == 0;
            e.row_pass(cur, op, batch, a.perm1, a.perm2, a.barrier, target);      // (begins with the grid barrier)
            grid_barrier(a.barrier, target);
            if (q + 1 < nsteps) e.template col_pass<COL_RK4>(cur, cur, mask, batch, phase, a.phase_stride, 4 * (zs + q) + 2, kap, hh, true);
        }
        e.template col_pass<COL_INVN>(cur, cur, mask, batch, phase, a.phase_stride, 4 * (zs + nsteps - 1) + 2, kap, hh);
        return;
    }

    e.template col_pass<COL_FWD>(cur, cur, mask, batch, phase, a.phase_stride, 0, kap, h);
    int s = rt_mode ? 0 : a.z0;        // index of the RK4 step that follows the operator q: q mod nz / z0 + q
#pragma unroll 1
    for (int q = 0; q <= total; ++q, s = (rt_mode && s + 1 == nz) ? 0 : s + 1) {
        const bool crossing = rt_mode && q > 0 && q < total && s == 0;
#pragma unroll
        for (int x = 0; x < F; ++x) {
            const bool res = a.resonant[x] != 0;
            op.sh_store[x] = nullptr;
            op.aux[x] = nullptr;
            op.out[x] = nullptr;
            op.tab_stride[x] = 0;
            if (!((mask >> x) & 1)) { op.kind[x] = -1; continue; }
            if (crossing && !res) {
                op.kind[x] = ROW_RELOAD;
                op.aux[x] = reinterpret_cast<const cplx<T>*>(a.SH[x]);
            } else {
                op.kind[x] = ROW_LINEAR;
                if (q == 0 || q == total) op.tab[x] = reinterpret_cast<const TAB*>(a.tabH[x]);
                else if (crossing) { op.tab[x] = reinterpret_cast<const TAB*>(a.tabHB[x]); op.tab_stride[x] = a.tabHB_stride[x]; }
                else op.tab[x] = reinterpret_cast<const TAB*>(a.tabH2[x]);
                if ((q == 0 || q == total) && a.tabH_stride[x]) op.tab_stride[x] = a.tabH_stride[x];
                if (rt_mode && q == 0 && !res && a.steps > 1) op.sh_store[x] = reinterpret_cast<cplx<T>*>(a.SH[x]);
            }
        }
        e.fix = ((a.op0 + q) % E::FIX_EVERY) == 0;        // (row pass and the column pass that follows)
        e.row_pass(cur, op, batch, a.perm1, a.perm2, a.barrier, target);          // (begins with the grid barrier)
        OPO_TSTAMP(e, 7);                                   // row stored
        grid_barrier(a.barrier, target);
        OPO_TSTAMP(e, 8);                                   // grid barrier after the row pass
        if (q == total) break;
        e.template col_pass<COL_RK4>(cur, cur, mask, batch, phase, a.phase_stride, 2 * s, kap, h);
    }
    e.fix = false;
    e.template col_pass<COL_INV>(cur, cur, mask, batch, phase, a.phase_stride, 0, kap, h);
#ifdef OPO_LARGE_TIMING
    // (the first column-load interval of a launch starts at t = 0 and is left out: divide the rest by the z-steps timed)
    if (threadIdx.x == 0 && (blockIdx.x == 0 || blockIdx.x == gridDim.x / 2) && total >= 100)
        printf("k_large cta %d, cycles per z-step (%d z-steps): col compute %lld store %lld | row prologue %lld barrier %lld load %lld "
               "compute %lld store %lld barrier %lld | next col load = z-step time minus these\n", (int)blockIdx.x, total, e.t_acc[1] / total,
               e.t_acc[2] / total, e.t_acc[3] / total, e.t_acc[4] / total, e.t_acc[5] / total, e.t_acc[6] / total, e.t_acc[7] / total, e.t_acc[8] / total);
#endif
}

template <class T, int L, int F> cudaError_t large_setup() {
    static device_once once;
    return once.run([&] { return cudaFuncSetAttribute(k_large<T, L, F>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                      (int)large_cfg<T, L, F>::SMEM_BYTES); });
}

template <class T, int L, int F> cudaError_t large_info_LF(int batch, int sm_count, LargeInfo* out) {
    using C = large_cfg<T, L, F>;
    cudaError_t e = large_setup<T, L, F>();
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_large<T, L, F>, C::NT, C::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    const long long tiles = (long long)batch * C::TILES_PER_INST;
    const long long chunks = (long long)batch * F * C::CHUNKS_PER_FIELD;
    long long want = tiles > chunks ? tiles : chunks;
    const long long cap = (long long)per_sm * sm_count;
    out->threads = C::NT;
    out->smem_bytes = C::SMEM_BYTES;
    out->max_ctas = (int)cap;
    out->grid = (int)(want < cap ? want : cap);
    out->n1 = C::N1;
    out->n2 = C::N2;
    return cudaSuccess;
}

template <class T, int L, int F> cudaError_t launch_large_LF(const LargeArgs& a, int grid, cudaStream_t s) {
    using C = large_cfg<T, L, F>;
    cudaError_t e = large_setup<T, L, F>();
    if (e != cudaSuccess) return e;
    LargeArgs copy = a;
    void* params[] = {&copy};
    return cudaLaunchCooperativeKernel((const void*)k_large<T, L, F>, dim3((unsigned)grid), dim3(C::NT), params, C::SMEM_BYTES, s);
}

template <class T, int L> cudaError_t large_info_L(int n_fields, int batch, int sm_count, LargeInfo* out) {
    return n_fields == 3 ? large_info_LF<T, L, 3>(batch, sm_count, out) : large_info_LF<T, L, 2>(batch, sm_count, out);
}
template <class T, int L> cudaError_t launch_large_L(const LargeArgs& a, int grid, cudaStream_t s) {
    return a.n_fields == 3 ? launch_large_LF<T, L, 3>(a, grid, s) : launch_large_LF<T, L, 2>(a, grid, s);
}

}  // namespace opo
