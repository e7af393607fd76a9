// opo_solo.cuh -- solo engine: ONE CTA (one SM) per OPO instance, all F coupled fields on chip:
// one field in (padded) shared memory, the other F - 1 in TENSOR MEMORY (TMEM, 256 KB per SM on sm_100a).
//
// Why.  The cluster engine (opo_resident.cuh) gives every field its own SM, so the RK4 step of the coupling terms
// (PAPER.md:L86-95, L115), which needs all F fields at the same grid points, moves 2/3 of the state over the
// SM-to-SM link in each direction every z-step -- at a measured ~16 B/clk per SM (profiles/r01d) -- and clusters of
// 3 place on 135 of the 148 SMs only.  3 x 128 KB (N = 2^14, complex64) does not fit one SM's 227 KB of shared
// memory, but it does fit shared memory PLUS tensor memory: tcgen05.st / tcgen05.ld move registers to / from TMEM at
// ~500-650 B/clk per SM (measured, profiles/r02a), five times the shared-memory crossbar, with no MMA involved.
// TMEM is lane-private (a warp reaches the 32 lanes of its quarter, a thread its own lane), which is exactly what
// the pass-0 / RK4 phase needs: a thread meets the same radix-4 butterflies t (elements t + j N/4) at every z-step.
//
// Layout.  The linear core (forward passes 1..P-1, table, inverse passes P-1..1; opo_fft.cuh) works on the field
// that is in shared memory; the other fields wait in TMEM in "butterfly layout": thread (warp w, lane l) keeps the
// four elements of its i-th butterfly t = (w + NW i) 32 + l of field slot s in the W = 8 (complex64) or 16
// (complex128) consecutive 32-bit columns  s COLS + (w >> 2) MAXT W + i W  of lane 32 (w & 3) + l.
//
// A z-step (order L/2 - N - L/2, adjacent half-steps merged exactly as in the cluster engine):
//     core(field 0) | swap 0 | core(field 1) | swap 1 | ... | core(field F-1) | fused
//   swap k : thread-private exchange  shared memory (field k) <-> TMEM slot k (field k + 1)
//   fused  : inverse pass 0 -> RK4 -> forward pass 0 on registers: field F-1 from shared memory, fields 0..F-2 from
//            TMEM slots 0..F-2; results: field 0 -> shared memory, field x -> slot x - 1.
// No data ever leaves the SM between the ends of a call; there is no cluster, no distributed shared memory and no
// cluster barrier.  Synchronisation is the class-granular mbarrier flow of opo_fft.cuh inside the CTA (N >= 2^12) or
// __syncthreads (smaller N).  The pass-0 twiddles (3 per butterfly) stream from L2, one tile ahead.
//
// Everything else (merged tables H, H2, HB = H2 G m, stored inputs SH of non-resonant fields, intracavity modulator
// at a crossing, round-trip split schedule over the CTAs) is the cluster engine's logic, field by field.
#pragma once
#include "opo_resident.cuh"

namespace opo {

// ---- tensor memory as lane-private storage ------------------------------------------------------------------
__device__ __forceinline__ void tmem_alloc(uint32_t smem_dst, int cols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t base, int cols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(base), "r"(cols) : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// one butterfly (4 complex values) of one field <-> consecutive columns of the calling thread's lane
__device__ __forceinline__ void tmem_ld4(uint32_t addr, cplx<float>* v) {
    uint32_t r[8];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(addr) : "memory");
    // the destination registers are defined only after tcgen05.wait::ld: the caller waits before touching v
#pragma unroll
    for (int k = 0; k < 4; ++k) { v[k].re = __uint_as_float(r[2 * k]); v[k].im = __uint_as_float(r[2 * k + 1]); }
}
__device__ __forceinline__ void tmem_st4(uint32_t addr, const cplx<float>* v) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(addr),
                 "r"(__float_as_uint(v[0].re)), "r"(__float_as_uint(v[0].im)), "r"(__float_as_uint(v[1].re)), "r"(__float_as_uint(v[1].im)),
                 "r"(__float_as_uint(v[2].re)), "r"(__float_as_uint(v[2].im)), "r"(__float_as_uint(v[3].re)), "r"(__float_as_uint(v[3].im))
                 : "memory");
}
__device__ __forceinline__ void tmem_ld4(uint32_t addr, cplx<double>* v) {
    uint32_t r[16];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                   "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                 : "r"(addr) : "memory");
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        v[k].re = __hiloint2double((int)r[4 * k + 1], (int)r[4 * k]);
        v[k].im = __hiloint2double((int)r[4 * k + 3], (int)r[4 * k + 2]);
    }
}
__device__ __forceinline__ void tmem_st4(uint32_t addr, const cplx<double>* v) {
    uint32_t r[16];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        r[4 * k] = (uint32_t)__double2loint(v[k].re); r[4 * k + 1] = (uint32_t)__double2hiint(v[k].re);
        r[4 * k + 2] = (uint32_t)__double2loint(v[k].im); r[4 * k + 3] = (uint32_t)__double2hiint(v[k].im);
    }
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(addr),
                 "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
                 "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]) : "memory");
}

template <class T, int L, int F> struct solo_layout {
    static constexpr int NT = cta_threads<T, L>::value;
    static constexpr int S = 1 << (L - 2), NTILES = (S + 31) / 32, NW = NT / 32;
    static constexpr int MAXT = (NTILES + NW - 1) / NW;                 // tiles (of 32 pass-0 butterflies) per warp
    static constexpr int W = 4 * (int)sizeof(cplx<T>) / 4;               // 32-bit words of one butterfly of one field
    static constexpr int QW = (NW + 3) / 4;                              // warps per TMEM lane quarter
    static constexpr int cols_per_slot = QW * MAXT * W;
    static constexpr int cols_needed = (F - 1) * cols_per_slot;
    static constexpr int cols_alloc = cols_needed <= 32 ? 32 : cols_needed <= 64 ? 64 : cols_needed <= 128 ? 128 : cols_needed <= 256 ? 256 : 512;
    static constexpr bool fits = cols_needed <= 512;
    using FC = flow_cfg<T, L, NT>;
    static constexpr int NCLS1 = FC::NCLS > 0 ? FC::NCLS : 1;
    static constexpr bool flow = FC::ok && NW % NCLS1 == 0 && NW <= NTILES && S >= 32;
    static constexpr size_t mbar_offset = (smem_layout<T, L>::total + 15) / 16 * 16;
    static constexpr size_t tmem_word_offset = mbar_offset + 16 * (size_t)NCLS1;      // ready[NCLS], done[NCLS]
    static constexpr size_t total = tmem_word_offset + 16;
    static constexpr int ready_count = FC::G;                            // one warp per group after its inverse pass 1 of the class
    static constexpr int done_count = flow ? NW / NCLS1 : 0;             // the warps that own tiles of the class
    // CTAs per SM: shared memory (plus 1 KB of system reservation each), TMEM columns, registers
    static constexpr int by_smem = (int)(233472 / (total + 1024));
    static constexpr int by_tmem = 512 / cols_alloc;
    static constexpr int by_regs = 65536 / (NT * 128);
    static constexpr int ctas_per_sm_raw = by_smem < by_tmem ? (by_smem < by_regs ? by_smem : by_regs) : (by_tmem < by_regs ? by_tmem : by_regs);
    static constexpr int ctas_per_sm = ctas_per_sm_raw < 1 ? 1 : (ctas_per_sm_raw > 4 ? 4 : ctas_per_sm_raw);
};

// TRAIN: the pump-train instantiation (nanosecond regime; objects of its own so that the default
// kernel's code is untouched): at every round-trip crossing the pump is the next slice of a long pump vector (loaded in the
// time domain, forward pass 0 and its first half-step follow), and the field `out_field` is taken out at z = L -- last
// half-step, inverse pass 0, store, then the boundary and the next half-step as one operator -- instead of crossing merged.
template <class T, int L, int F, bool DK0 = false, bool TRAIN = false>
__global__ void __launch_bounds__(cta_threads<T, L>::value, solo_layout<T, L, F>::ctas_per_sm) k_solo(ResidentArgs a) {
    constexpr int N = 1 << L, NT = cta_threads<T, L>::value;
    using PL = plan<L>;
    using SL = smem_layout<T, L>;
    using SO = solo_layout<T, L, F>;
    using FC = flow_cfg<T, L, NT>;
    static_assert(SO::fits, "the fields of one instance must fit shared memory + tensor memory of one SM");
    static_assert(PL::rbits(0) == 2, "pass 0 must be radix 4");
    constexpr bool FLOW = SO::flow;
    constexpr int RB = 2, R = 4, SB = L - 2, S = 1 << SB;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
    const int cid = blockIdx.x, n_ctas = gridDim.x;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    const cplx<T>* tw = reinterpret_cast<const cplx<T>*>(a.tw);
    {   // shared-memory copy of the twiddles of the local passes
        cplx<T>* twl = reinterpret_cast<cplx<T>*>(smem_raw + SL::field_bytes);
        for (int i = tid; i < PL::tw_local_count; i += NT) twl[i] = ldg(&tw[PL::tw_local_begin + i]);
    }
    const uint32_t mb = (uint32_t)__cvta_generic_to_shared(smem_raw + SO::mbar_offset);
    if constexpr (FLOW) {
        if (tid == 0) {
            for (int c = 0; c < FC::NCLS; ++c) {
                mbar_init(mb + 8 * c, SO::ready_count);
                mbar_init(mb + 8 * (FC::NCLS + c), SO::done_count);
            }
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");      // (the only scope this fence has)
        }
    }
    // tensor memory: (F - 1) field slots
    uint32_t* tmem_word = reinterpret_cast<uint32_t*>(smem_raw + SO::tmem_word_offset);
    if (warp == 0) tmem_alloc((uint32_t)__cvta_generic_to_shared(tmem_word), SO::cols_alloc);
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = *tmem_word;
    // this thread's columns of slot 0, tile 0
    const uint32_t tm0 = tmem_base + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * SO::MAXT * SO::W);
    auto tmem_at = [&](int slot, int i) -> uint32_t { return tm0 + (uint32_t)(slot * SO::cols_per_slot + i * SO::W); };

    uint32_t fz = 0;        // transitions (swap / fused) executed so far: mbarrier phase parity
    const int wg = (tid % FC::NTG) >> 5;
    const int cls = FLOW ? warp % SO::NCLS1 : 0;       // all tiles of a warp belong to one class (NW is a multiple of NCLS)
    auto flow_wait_done_all = [&](uint32_t parity) {
        if constexpr (FLOW)
            for (int it = 0; it < FC::NIT; ++it) mbar_wait_cta(mb + 8 * (FC::NCLS + wg + FC::NWG * it), parity);
    };
    auto flow_arrive_ready_all = [&]() {
        if constexpr (FLOW)
            for (int it = 0; it < FC::NIT; ++it) mbar_arrive_cta(mb + 8 * (wg + FC::NWG * it), lane);
    };
    T kap[3] = {(T)a.kappa[0], (T)a.kappa[1], (T)a.kappa[2]};
    const T h = (T)a.h;
    const int nz = a.nz;
    const bool rt_mode = a.mode != 0;

    // ---- thread-private moves between shared memory and a TMEM slot -------------------------------------------
    auto s2t = [&](int slot) {          // shared memory -> slot
        int i = 0;
#pragma unroll 1
        for (int tile = warp; tile < SO::NTILES; tile += SO::NW, ++i) {
            const int t = tile * 32 + lane;
            const int p0 = elem_base<T, RB, SB>(0, (S >= 32 || t < S) ? t : 0);
            cplx<T> v[R];
#pragma unroll
            for (int k = 0; k < R; ++k) v[k] = sm[p0 + elem_off<T, RB, SB>(k)];
            tmem_st4(tmem_at(slot, i), v);
        }
        tmem_wait_st();
    };
    auto t2s = [&](int slot) {          // slot -> shared memory
        int i = 0;
#pragma unroll 1
        for (int tile = warp; tile < SO::NTILES; tile += SO::NW, ++i) {
            const int t = tile * 32 + lane;
            cplx<T> v[R];
            tmem_ld4(tmem_at(slot, i), v);
            tmem_wait_ld();
            if (S >= 32 || t < S) {
                const int p0 = elem_base<T, RB, SB>(0, t);
#pragma unroll
                for (int k = 0; k < R; ++k) sm[p0 + elem_off<T, RB, SB>(k)] = v[k];
            }
        }
    };
    // swap k: field k (shared memory) <-> field k + 1 (slot k)
    auto swap_fields = [&](int slot) {
        if constexpr (FLOW) mbar_wait_cta(mb + 8 * cls, fz & 1);         // ready[cls]: inverse pass 1 of my class is done in all groups
        else __syncthreads();
        int i = 0;
#pragma unroll 1
        for (int tile = warp; tile < SO::NTILES; tile += SO::NW, ++i) {
            const int t = tile * 32 + lane;
            const bool active = S >= 32 || t < S;
            const int p0 = elem_base<T, RB, SB>(0, active ? t : 0);
            cplx<T> in[R], out[R];
            tmem_ld4(tmem_at(slot, i), in);
#pragma unroll
            for (int k = 0; k < R; ++k) out[k] = sm[p0 + elem_off<T, RB, SB>(k)];
            tmem_wait_ld();
            if (active) {
#pragma unroll
                for (int k = 0; k < R; ++k) sm[p0 + elem_off<T, RB, SB>(k)] = in[k];
            }
            tmem_st4(tmem_at(slot, i), out);
        }
        tmem_wait_st();
        if constexpr (FLOW) mbar_arrive_cta(mb + 8 * (FC::NCLS + cls), lane);    // done[cls]
        else __syncthreads();
        ++fz;
    };
    // fused: inverse pass 0 -> RK4 -> forward pass 0; field F-1 in shared memory, field x < F-1 in slot x;
    // afterwards field 0 in shared memory, field x >= 1 in slot x - 1
    auto fused = [&](cplx<T> e0, cplx<T> e1, cplx<T> e2) {
        if constexpr (FLOW) mbar_wait_cta(mb + 8 * cls, fz & 1);
        else __syncthreads();
        cplx<T> wn[R - 1];
        auto load_tw = [&](int tile) {
            const int t = tile * 32 + lane;
            const int tt = (S >= 32 || t < S) ? t : 0;
#pragma unroll
            for (int k = 0; k < R - 1; ++k) wn[k] = ldg(&tw[k * S + tt]);
        };
        load_tw(warp);
        int i = 0;
#pragma unroll 1
        for (int tile = warp; tile < SO::NTILES; tile += SO::NW, ++i) {
            const int t = tile * 32 + lane;
            const bool active = S >= 32 || t < S;
            const int p0 = elem_base<T, RB, SB>(0, active ? t : 0);
            cplx<T> v[F][R], w[R - 1];
#pragma unroll
            for (int x = 0; x < F - 1; ++x) tmem_ld4(tmem_at(x, i), v[x]);
#pragma unroll
            for (int k = 0; k < R; ++k) v[F - 1][k] = sm[p0 + elem_off<T, RB, SB>(k)];
#pragma unroll
            for (int k = 0; k < R - 1; ++k) w[k] = wn[k];
            if (tile + SO::NW < SO::NTILES) load_tw(tile + SO::NW);
            tmem_wait_ld();
#pragma unroll
            for (int x = 0; x < F; ++x) {
#pragma unroll
                for (int k = 1; k < R; ++k) v[x][k] = cmulc(v[x][k], w[k - 1]);
                dit_inv<T, R>::run(v[x]);
            }
#pragma unroll
            for (int j = 0; j < R; ++j) {
                cplx<T> y[F];
#pragma unroll
                for (int x = 0; x < F; ++x) y[x] = v[x][j];
                Rk4<T, F>::template step<DK0>(y, e0, e1, e2, kap, h);
#pragma unroll
                for (int x = 0; x < F; ++x) v[x][j] = y[x];
            }
#pragma unroll
            for (int x = 0; x < F; ++x) {
                dif<T, R>::run(v[x]);
#pragma unroll
                for (int k = 1; k < R; ++k) v[x][k] = cmul(v[x][k], w[k - 1]);
            }
            if (active) {
#pragma unroll
                for (int k = 0; k < R; ++k) sm[p0 + elem_off<T, RB, SB>(k)] = v[0][k];
            }
#pragma unroll
            for (int x = 1; x < F; ++x) tmem_st4(tmem_at(x - 1, i), v[x]);
        }
        tmem_wait_st();
        if constexpr (FLOW) mbar_arrive_cta(mb + 8 * (FC::NCLS + cls), lane);
        else __syncthreads();
        ++fz;
    };
    // bunch: this application carries the low parts of the butterflies' compile-time constants for kConstBunch applications
    // (kconst in opo_fft.cuh; fp32 with the flow synchronisation, i.e. N >= 2^12): the other kConstBunch - 1 use the high
    // parts alone, one instruction per constant product instead of two
    auto core = [&](const cplx<T>* tab, bool wait_in, bool arrive_out, bool bunch = false) {
        if constexpr (FLOW) {
            FlowArgs fa;
            fa.mb = mb; fa.nf = 1;
            fa.wait_in = wait_in; fa.par_done = (fz - 1) & 1;
            fa.arrive_out = arrive_out;
            if constexpr (sizeof(T) == 4) {
                if (bunch) linear_core_smem<T, L, NT, true, true, 2>(tab, tid, fa);
                else linear_core_smem<T, L, NT, true, true, 1>(tab, tid, fa);
            } else {
                linear_core_smem<T, L, NT, true, true>(tab, tid, fa);
            }
        } else {
            linear_core_smem<T, L, NT>(tab, tid);
        }
    };

    // Work list of this CTA: whole instances b = cid, cid + n_ctas, ...; with a.split (round-trip mode) contiguous ranges of
    // (instance, round trip) units, walked backwards, state handed over through `cur` (see opo_resident.cuh).  The launch
    // is cooperative when a.split, so every CTA is resident and the wait below cannot deadlock.
    const long long units = (long long)a.batch * a.steps;
    const long long quota = (units + n_ctas - 1) / n_ctas;
    const long long u_lo = a.split ? (long long)cid * quota : 0;
    long long u_hi = a.split ? (u_lo + quota < units ? u_lo + quota : units) : 0;
    int b = cid;
    while (true) {
        int steps_l = a.steps, rt0 = 0;
        if (a.split) {
            if (u_hi <= u_lo) break;
            b = (int)((u_hi - 1) / a.steps);
            const long long seg_lo = u_lo > (long long)b * a.steps ? u_lo : (long long)b * a.steps;
            rt0 = (int)(seg_lo - (long long)b * a.steps);
            steps_l = (int)(u_hi - seg_lo);
            u_hi = seg_lo;
        } else if (b >= a.batch) {
            break;
        }
        const int total = rt_mode ? steps_l * nz : steps_l;
        const cplx<T>* ph = reinterpret_cast<const cplx<T>*>(a.phase) + (size_t)b * a.phase_stride;
        // where this piece stands in the handle's count of operators / table uses (ResidentArgs::op0, hq0, fq0): an instance
        // cut into pieces by the split schedule applies two half-steps more per cut
        const int cuts = (a.split && rt0 > 0) ? (int)(((long long)b * a.steps + rt0) / quota - ((long long)b * a.steps) / quota) : 0;
        const int op_base = a.op0 + (rt_mode ? rt0 * nz : 0) + cuts;
        const int hq_base = a.hq0 + 2 * cuts;
        int fq = a.fq0 + (rt_mode ? rt0 * (nz - 1) : 0);       // full steps applied before the next one (counted, not divided out:
                                                               // the table address is on the critical path of every z-step)

        auto load = [&](const cplx<T>* __restrict__ g) {
#pragma unroll 4
            for (int i = tid; i < N; i += NT) sm[phys<T>(i)] = g[i];
        };
        auto store = [&](cplx<T>* __restrict__ g) {
#pragma unroll 4
            for (int i = tid; i < N; i += NT) g[i] = sm[phys<T>(i)];
        };

        // resonant pump (reading R24): the input coupler adds t S_p at every boundary, and the first half-step of the next
        // pass acts on the sum: SH_p <- IDFT(H DFT(S_p)) (up to its inverse pass 0) once per piece of work, t SH_p is added
        // after the merged boundary operator at every crossing
        const T tinj = (T)a.inject;
        const bool inj_any = tinj != (T)0 && a.resonant[0] != 0;
        if (inj_any && rt_mode && steps_l > 1) {
            load(reinterpret_cast<const cplx<T>*>(a.S[0]) + (size_t)b * N);
            __syncthreads();
            pass0_local<T, L, NT>(tw, tid, false);
            __syncthreads();
            linear_core_smem<T, L, NT>(reinterpret_cast<const cplx<T>*>(a.tabH[0]), tid);
            __syncthreads();
            store(reinterpret_cast<cplx<T>*>(a.SH[0]) + (size_t)b * N);
            __syncthreads();
        }

        // ---- bring the instance on chip: every field through shared memory and forward pass 0; fields 1.. park in TMEM
        if (a.split && rt0 > 0) {       // the earlier round trips of this instance ran on another CTA
            if (tid == 0) {
                for (int x = 0; x < F; ++x) {
                    const int* flag = a.flags + (size_t)b * F + x;
                    int v;
                    do { asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(flag) : "memory"); } while (v < rt0);
                }
            }
            __syncthreads();
        }
#pragma unroll 1
        for (int xi = 0; xi < F; ++xi) {
            const int x = (xi + 1) % F;         // 1, 2, .., F-1, 0: field 0 stays in shared memory
            const cplx<T>* cur = reinterpret_cast<const cplx<T>*>(a.cur[x]) + (size_t)b * N;
            if (TRAIN && x == 0) {              // ReadPump: the slice of this piece's first round trip
                load(reinterpret_cast<const cplx<T>*>(a.train) + (size_t)rt0 * a.train_stride + (size_t)b * a.train_inst_stride);
            } else if (a.split && rt0 > 0) {
#pragma unroll 4
                for (int i = tid; i < N; i += NT) sm[phys<T>(i)] = ldcg_c(cur + i);
            } else {
                load(cur);
            }
            __syncthreads();
            pass0_local<T, L, NT>(tw, tid, false);
            __syncthreads();
            if (x != 0) { s2t(x - 1); __syncthreads(); }
        }

        // q counts linear operators: q = 0 first half-step, q = total last half-step, between them the merged full
        // steps; in round-trip mode q = m nz + s and s = 0 (m > 0) crosses the boundary
#pragma unroll 1
        for (int q = 0; q <= total; ++q) {
            const int s = rt_mode ? q % nz : a.z0 + q;
            const bool crossing = rt_mode && q > 0 && q < total && s == 0;
            const bool bunch = ((op_base + q) & (kConstBunch - 1)) == 0;
#pragma unroll
            for (int x = 0; x < F; ++x) {
                const bool resonant = a.resonant[x] != 0;
                const bool keep = rt_mode && q == 0 && !resonant && steps_l > 1 && !(TRAIN && x == 0);     // SH <- first half-stepped input
                const bool first_core = q == 0 && x == 0;                             // no transition precedes
                const bool last_core = q == total && x == F - 1;                      // no transition follows
                const bool inj = x == 0 && crossing && inj_any;                       // input coupler of a resonant pump
                const cplx<T>* tabH = reinterpret_cast<const cplx<T>*>(a.tabH[x]);
                cplx<T>* SH = reinterpret_cast<cplx<T>*>(a.SH[x]) + (size_t)b * N;
                const int rt_done = rt0 + q / (nz > 0 ? nz : 1);      // round trips of the instance completed at a crossing
                if (TRAIN && crossing && (x == 0 || (x == a.out_field && a.out_train != nullptr))) {
                    if (x == a.out_field && a.out_train != nullptr) {
                        // SaveRoundTrip: the field at z = L of the round trip just finished, before the mirror
                        core(tabH, true, false, bunch);
                        __syncthreads();
                        pass0_local<T, L, NT>(tw, tid, true);
                        __syncthreads();
                        cplx<T>* __restrict__ o = reinterpret_cast<cplx<T>*>(a.out_train) + ((size_t)(rt_done - 1) * a.batch + b) * N;
                        const cplx<T> mf = (resonant && !a.boundary_fft[x]) ? ldg(reinterpret_cast<const cplx<T>*>(a.mirror[x]) + b) : cplx<T>{(T)1, (T)0};
#pragma unroll 4
                        for (int i = tid; i < N; i += NT) { const cplx<T> v = sm[phys<T>(i)]; o[i] = v; sm[phys<T>(i)] = cmul(v, mf); }
                        __syncthreads();
                    } else {
                        if constexpr (FLOW) { flow_wait_done_all((fz - 1) & 1); }
                        __syncthreads();
                    }
                    if (x == 0) {                    // ReadPump: the slice of the round trip that begins (the pump is single-pass)
                        load(reinterpret_cast<const cplx<T>*>(a.train) + (size_t)rt_done * a.train_stride + (size_t)b * a.train_inst_stride);
                        __syncthreads();
                    } else if (!resonant) {          // a non-resonant field restarts from its stored input (R12)
                        load(reinterpret_cast<const cplx<T>*>(a.S[x]) + (size_t)b * N);
                        __syncthreads();
                    }
                    pass0_local<T, L, NT>(tw, tid, false);
                    __syncthreads();
                    // the boundary (spectral phase and mirror: G m, or the mirror alone, applied above) and the first half-step
                    core((resonant && a.boundary_fft[x]) ? reinterpret_cast<const cplx<T>*>(a.tabHG[x]) + (size_t)b * a.tab_stride[x] : tabH, false, true);
                } else if (crossing && !resonant) {
                    if constexpr (FLOW) { flow_wait_done_all((fz - 1) & 1); __syncthreads(); }
                    load(SH);                                        // fresh pump / frozen seed, already half-stepped
                    if constexpr (FLOW) { __syncthreads(); flow_arrive_ready_all(); }
                } else if (crossing && a.eom[x] != nullptr) {
                    // resonant field with an intracavity modulator:
                    //   core(H G m) -> inverse pass 0 -> x E[n] -> forward pass 0 -> core(H)
                    const cplx<T>* tabHG = reinterpret_cast<const cplx<T>*>(a.tabHG[x]) + (size_t)b * a.tab_stride[x];
                    const cplx<T>* __restrict__ E = reinterpret_cast<const cplx<T>*>(a.eom[x]);
                    core(tabHG, true, false, bunch);
                    __syncthreads();
                    pass0_local<T, L, NT>(tw, tid, true);
                    __syncthreads();
#pragma unroll 4
                    for (int i = tid; i < N; i += NT) sm[phys<T>(i)] = cmul(sm[phys<T>(i)], ldg(&E[i]));
                    __syncthreads();
                    pass0_local<T, L, NT>(tw, tid, false);
                    __syncthreads();
                    core(tabH, false, !inj);
                } else {
                    const cplx<T>* tab = tabH + (size_t)((hq_base + (q == 0 ? 0 : 1)) & a.tab_cycle_mask) * N;
                    if (q != 0 && q != total)
                        tab = crossing ? reinterpret_cast<const cplx<T>*>(a.tabHB[x]) + (size_t)b * a.tab_stride[x]
                                       : reinterpret_cast<const cplx<T>*>(a.tabH2[x]) + (size_t)(fq & a.tab_cycle_mask) * N;
                    core(tab, !first_core, !last_core && !keep && !inj, bunch);
                }
                if (inj) {
                    __syncthreads();
                    const cplx<T>* __restrict__ g = SH;
#pragma unroll 4
                    for (int i = tid; i < N; i += NT) {
                        const cplx<T> v = sm[phys<T>(i)], sv = g[i];
                        sm[phys<T>(i)] = {v.re + tinj * sv.re, v.im + tinj * sv.im};
                    }
                    if constexpr (FLOW) { __syncthreads(); flow_arrive_ready_all(); }
                }
                if (keep) {   // keep it for the later round trips
                    __syncthreads();
                    store(SH);
                    if constexpr (FLOW) { __syncthreads(); flow_arrive_ready_all(); }
                }
                if (x < F - 1) {
                    swap_fields(x);
                } else if (q < total) {
                    if (q > 0 && !crossing) ++fq;
                    const cplx<T> e0 = ldg(ph + 2 * s), e1 = ldg(ph + 2 * s + 1), e2 = ldg(ph + 2 * s + 2);
                    fused(e0, e1, e2);
                }
            }
        }

        // ---- leave the chip: field F-1 is in shared memory, field x < F-1 in slot x, all before their inverse pass 0
#pragma unroll 1
        for (int xi = 0; xi < F; ++xi) {
            const int x = F - 1 - xi;
            __syncthreads();
            if (xi > 0) { t2s(x); __syncthreads(); }
            pass0_local<T, L, NT>(tw, tid, true);
            __syncthreads();
            cplx<T>* cur = reinterpret_cast<cplx<T>*>(a.cur[x]) + (size_t)b * N;
            if (!rt_mode) {
                store(cur);
            } else {
                store(reinterpret_cast<cplx<T>*>(a.exitb[x]) + (size_t)b * N);     // fields at z = L of the last pass
                if (TRAIN && x == a.out_field && a.out_train != nullptr)
                    store(reinterpret_cast<cplx<T>*>(a.out_train) + ((size_t)(rt0 + steps_l - 1) * a.batch + b) * N);
                if (a.resonant[x]) {
                    // mirror, spectral phase and phase modulator of the last round trip of the call
                    const cplx<T>* __restrict__ E = reinterpret_cast<const cplx<T>*>(a.eom[x]);
                    cplx<T> mf = {(T)1, (T)0};
                    if (a.boundary_fft[x]) {
                        const cplx<T>* tabGM = reinterpret_cast<const cplx<T>*>(a.tabGM[x]) + (size_t)b * a.tab_stride[x];
                        __syncthreads();
                        pass0_local<T, L, NT>(tw, tid, false);
                        __syncthreads();
                        linear_core_smem<T, L, NT>(tabGM, tid);
                        __syncthreads();
                        pass0_local<T, L, NT>(tw, tid, true);
                        __syncthreads();
                    } else {
                        mf = ldg(reinterpret_cast<const cplx<T>*>(a.mirror[x]) + b);
                    }
                    if (E != nullptr) {
#pragma unroll 4
                        for (int i = tid; i < N; i += NT) cur[i] = cmul(cmul(sm[phys<T>(i)], mf), ldg(&E[i]));
                    } else {
#pragma unroll 4
                        for (int i = tid; i < N; i += NT) cur[i] = cmul(sm[phys<T>(i)], mf);
                    }
                    if (x == 0 && inj_any) {     // input coupler (reading R24)
                        const cplx<T>* __restrict__ Sp = reinterpret_cast<const cplx<T>*>(a.S[0]) + (size_t)b * N;
#pragma unroll 4
                        for (int i = tid; i < N; i += NT) { const cplx<T> v = cur[i], sv = Sp[i]; cur[i] = {v.re + tinj * sv.re, v.im + tinj * sv.im}; }
                    }
                } else {
                    const cplx<T>* __restrict__ Sx = reinterpret_cast<const cplx<T>*>(a.S[x]) + (size_t)b * N;
#pragma unroll 4
                    for (int i = tid; i < N; i += NT) cur[i] = Sx[i];
                }
            }
        }
        __syncthreads();
        if (a.split) {
            if (rt0 + steps_l < a.steps && tid == 0) {      // hand the instance over: its state is in `cur`
                __threadfence();
                for (int x = 0; x < F; ++x)
                    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(a.flags + (size_t)b * F + x), "r"(rt0 + steps_l) : "memory");
            }
        } else {
            b += n_ctas;
        }
    }
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem_base, SO::cols_alloc);
}

template <class T, int L, int F, bool DK0, bool TRAIN = false> cudaError_t solo_setup() {
    static device_once once;
    return once.run([&] { return cudaFuncSetAttribute(k_solo<T, L, F, DK0, TRAIN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)solo_layout<T, L, F>::total); });
}

template <class T, int L, int F> cudaError_t solo_info_LF(ResidentInfo* out) {
    using SO = solo_layout<T, L, F>;
    if constexpr (!SO::fits) {
        return cudaErrorNotSupported;
    } else {
        cudaError_t e = solo_setup<T, L, F, false>();
        if (e != cudaSuccess) return e;
        int per_sm = 0, dev = 0, sms = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_solo<T, L, F, false>, SO::NT, SO::total);
        if (e != cudaSuccess) return e;
        if (per_sm > SO::by_tmem) per_sm = SO::by_tmem;      // the occupancy calculator does not know about tensor memory
        e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return e;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        out->threads = SO::NT;
        out->smem_bytes = SO::total;
        out->max_clusters = per_sm * sms;
        return cudaSuccess;
    }
}
template <class T, int L> cudaError_t solo_info_L(int n_fields, ResidentInfo* out) {
    return n_fields == 3 ? solo_info_LF<T, L, 3>(out) : solo_info_LF<T, L, 2>(out);
}

template <class T, int L, int F, bool DK0, bool TRAIN = false> cudaError_t launch_solo_LF(const ResidentArgs& a, int n_ctas, cudaStream_t s) {
    using SO = solo_layout<T, L, F>;
    if constexpr (!SO::fits) {
        return cudaErrorNotSupported;
    } else {
        cudaError_t e = solo_setup<T, L, F, DK0, TRAIN>();
        if (e != cudaSuccess) return e;
        cudaLaunchConfig_t cfg{};
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeCooperative;      // co-residency of all CTAs is what makes the split schedule's wait safe
        attr[0].val.cooperative = a.split ? 1 : 0;
        cfg.gridDim = dim3((unsigned)n_ctas, 1, 1);
        cfg.blockDim = dim3(SO::NT, 1, 1);
        cfg.dynamicSmemBytes = SO::total;
        cfg.stream = s;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        return cudaLaunchKernelEx(&cfg, k_solo<T, L, F, DK0, TRAIN>, a);
    }
}
template <class T, int L, bool DK0, bool TRAIN = false> cudaError_t launch_solo_L(const ResidentArgs& a, int n_ctas, cudaStream_t s) {
    return a.n_fields == 3 ? launch_solo_LF<T, L, 3, DK0, TRAIN>(a, n_ctas, s) : launch_solo_LF<T, L, 2, DK0, TRAIN>(a, n_ctas, s);
}

}  // namespace opo
