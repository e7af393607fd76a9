// opo_wide.cuh -- wide engine: ONE OPO instance on a thread-block cluster of 4 F CTAs, every field split over four SMs,
// the FFT stages that cross the split exchanged over distributed shared memory (BASELINE.json north_star item (a)).
//
// Why.  The paper's own workload is a single OPO followed for 10^3 .. 10^4 round trips ("massive and
// sequential simulations", L252), i.e. BASELINE.json configs[1] and [2]: nothing to batch, and z-steps are strictly
// sequential.  The cluster engine (opo_resident.cuh) gives such an instance F SMs, and each of them has to issue the
// whole 2^14-point transform pair of its field: ~16 us per z-step on 3 of 148 SMs.  Here the instance gets 4 F SMs.
//
// Decomposition.  The radix-4 pass 0 (decimation in frequency, butterflies over x[t + j N/4], j = 0..3) leaves four
// independent sub-transforms of S = N/4 points.  CTA rank 4 x + j of the cluster holds sub-block j of field x -- logical
// indices [j S, (j + 1) S), the same index range before and after pass 0 -- in (padded) shared memory for the whole call.
//
//   core  : CTA-local.  Forward passes 1..P-1, table multiply, inverse passes P-1..1 of the sub-block (opo_fft.cuh), one
//           radix-16 butterfly per thread and pass (N = 2^14: 256 threads).
//   fused : inverse pass 0 -> RK4 of the coupling terms -> forward pass 0, on registers.  The
//           butterfly t needs element t of all four sub-blocks of all F fields: 4 F CTAs.  The S butterflies are dealt
//           to the warps of the cluster in tiles of 32; a thread finds the 4 F operands of its butterfly in its warp's
//           staging buffer (see "push"), integrates, and sends the 4 F results to the CTAs that own them.
//   sync  : no cluster-wide barrier inside the z-step loop.  The pass-1 butterfly t' touches the elements t' + (S/16) k,
//           so the tiles of class c = (tile mod S/512) depend exactly on the pass-1 butterflies of warp c of every CTA, and
//           vice versa: warp c of each of the 4 F CTAs forms a ring of its own.  The 16 tiles of a class are dealt to the 4 F
//           warps of its ring (rotated by the class so that every CTA gets the same number of tiles): two tiles per warp
//           with two fields; with three fields 12 warps would share 16 tiles, so the four left over per class go to
//           HELPER warps -- up to three extra warps per CTA that take no part in the core and integrate one tile each.
//   push  : all traffic between the SMs is asynchronous stores (st.async ... mbarrier::complete_tx::bytes).  The inverse
//           pass 1 does not write its 16 results back in place: it sends each one to the staging buffer of the warp that
//           owns its tile; that warp waits on a local mbarrier (ready[c], armed with the bytes it expects), reads its 4 F
//           operands per butterfly from LOCAL shared memory, integrates, and sends every result to its owner's field, where
//           the forward pass 1 waits on done[c] the same way.  No remote load, no release fence and no arrival message is
//           ever waited for: a z-step was 7.2 us with remote loads + release/acquire arrivals (the top stalls were the
//           long scoreboard of the remote loads and the membar of the releases), 5.5 us this way.  The waits acquire at CTA
//           scope: the bytes counted on a barrier are visible to its waiter, and a cluster-scope acquire would make
//           ptxas invalidate L1 (CCTL.IVALL) at every wait.  The pass-0 phases at the two ends of a call (no RK4) read
//           and write the fields in place through ld / st.shared::cluster between cluster barriers.
//
// Everything else (merged tables H, H2, HB = H2 G m across the cavity boundary; stored
// inputs SH of non-resonant fields re-injected every round trip, L268; mirror / spectral phase / modulator of the
// call's last round trip) is the cluster engine's logic on sub-blocks.  Not served here (the host keeps those on the
// cluster engine): the N/2 - L - N/2 ordering and a resonant pump.  A phase modulator acts at a crossing
// between two in-place pass-0 phases of the modulated field, as in the cluster engine.
#pragma once
#include "opo_resident.cuh"

namespace opo {

// G: sub-blocks ("virtual ranks") per CTA.  G = 1: a cluster of 4 F CTAs, the lowest latency for one instance (7 such
// clusters of 12 are co-resident on a B200).  G = 2: a cluster of 2 F CTAs with two groups of threads, each group the
// complete machinery of one virtual rank -- its own sub-block, staging slots, barriers and named CTA barrier -- so three
// times as many instances run at once (22 clusters of 6, a portable cluster size), each a little slower: the engine of
// sweeps of a dozen instances (BASELINE.json configs[2]).
template <class T, int L, int F, int G = 1> struct wide_layout {
    using PL = plan<L>;
    static constexpr int C = 4;                              // sub-blocks left by the radix-4 pass 0 = virtual ranks per field
    static constexpr int NV = C * F;                         // virtual ranks of an instance
    static constexpr int NCTA = NV / G;                      // cluster size: 8 / 12 (G = 1; 12 is a non-portable size), 4 / 6 (G = 2)
    static constexpr int S = 1 << (L - 2);                   // points of a sub-block = number of pass-0 butterflies
    static constexpr int NT = S / 16;                        // threads of a group: one radix-16 pass-1 butterfly per thread
    static constexpr int NW = NT / 32;                       // warps of a group = classes
    static constexpr int TPC = 16;                           // tiles (of 32 pass-0 butterflies) per class: S / 32 / NW
    // G = 1: core warps own TPC / NV tiles each (rounded down); the EX tiles left over go to NH helper warps per CTA, one each.
    // G = 2: no helpers (the registers of 512 core threads are all there is); a warp owns up to ceil(TPC / NV) tiles.
    static constexpr bool HELP = G == 1;
    static constexpr int MAXT = HELP ? TPC / NV : (TPC + NV - 1) / NV;      // tiles per core warp
    static constexpr int EX = HELP ? (TPC - MAXT * NV) * NW : 0;            // tiles of the cluster no core warp owns
    static constexpr int NH = (EX + NCTA - 1) / NCTA;        // helper warps per CTA
    static constexpr int NCORE = G * NT;                     // core threads per CTA
    static constexpr int NTH = NCORE + 32 * NH;              // threads per CTA
    static constexpr int NSLOT = G * NW * MAXT + NH;         // staging slots (one per owned tile)
    static constexpr bool ok = PL::P == 4 && PL::rbits(0) == 2 && PL::rbits(1) == 4 && NT >= 32 && NV % G == 0 && C % G == 0;
    static constexpr size_t field_bytes = (size_t)padded_len<T>(S) * sizeof(cplx<T>);       // one sub-block
    static constexpr size_t tw_offset_bytes = (size_t)G * field_bytes;
    static constexpr size_t tw_bytes = (size_t)PL::tw_local_count * sizeof(cplx<T>);
    static constexpr int NQ = NV;                            // operands of a pass-0 butterfly over all fields
    // staging buffer of the fused phase: [slot][field, sub-block][lane]; slot = (group NW + warp) MAXT + tile (core warps),
    // G NW MAXT + h (helpers)
    static constexpr size_t stage_offset = (tw_offset_bytes + tw_bytes + 15) / 16 * 16;
    static constexpr size_t stage_bytes = (size_t)(NSLOT > 0 ? NSLOT : 1) * NQ * 32 * sizeof(cplx<T>);
    static constexpr size_t mbar_offset = stage_offset + stage_bytes;           // per group ready[NW], done[NW]; then helper_ready[NH]
    static constexpr size_t total = mbar_offset + 8 * (size_t)(G * 2 * NW + NH) + 8;
    static constexpr uint32_t done_bytes = TPC * 32 * (uint32_t)sizeof(cplx<T>);      // results per class and phase arriving in a sub-block
};

// distributed shared memory through 32-bit shared::cluster addresses (half the address registers of generic pointers)
__device__ __forceinline__ uint32_t dsmem_addr(uint32_t local_addr, int rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local_addr), "r"(rank));
    return r;
}
__device__ __forceinline__ cplx<float> dsmem_ld(uint32_t addr, cplx<float>) {
    cplx<float> v;
    asm volatile("ld.shared::cluster.v2.f32 {%0, %1}, [%2];" : "=f"(v.re), "=f"(v.im) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ cplx<double> dsmem_ld(uint32_t addr, cplx<double>) {
    cplx<double> v;
    asm volatile("ld.shared::cluster.v2.f64 {%0, %1}, [%2];" : "=d"(v.re), "=d"(v.im) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void dsmem_st(uint32_t addr, cplx<float> v) {
    asm volatile("st.shared::cluster.v2.f32 [%0], {%1, %2};" ::"r"(addr), "f"(v.re), "f"(v.im) : "memory");
}
__device__ __forceinline__ void dsmem_st(uint32_t addr, cplx<double> v) {
    asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};" ::"r"(addr), "d"(v.re), "d"(v.im) : "memory");
}

// asynchronous store into a CTA of the cluster; its bytes are counted on the mbarrier `mbar` OF THAT CTA (complete_tx),
// which is what orders the data before the waiter's reads: no fence, no arrival message
__device__ __forceinline__ void st_async(uint32_t addr, cplx<float> v, uint32_t mbar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f32 [%0], {%1, %2}, [%3];" ::"r"(addr), "f"(v.re), "f"(v.im), "r"(mbar) : "memory");
}
__device__ __forceinline__ void st_async(uint32_t addr, cplx<double> v, uint32_t mbar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1, %2}, [%3];" ::"r"(addr), "d"(v.re), "d"(v.im), "r"(mbar) : "memory");
}
// one thread arms a barrier of its own CTA for the next phase: its single arrival plus the bytes that phase will bring
__device__ __forceinline__ void mbar_arm(uint32_t addr, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.release.cta.shared::cta.b64 _, [%0], %1;" ::"r"(addr), "r"(bytes) : "memory");
}

struct WideFlow {
    uint32_t mb;         // shared address of my group's ready[0]; done[c] = mb + 8 (NW + c)
    uint32_t mb0;        // shared address of the CTA's first barrier (group 0)
    uint32_t stage;      // shared address of the CTA's staging buffer
    int q_me;            // my virtual rank 4 x + j = my operand slot in a staged butterfly
    int wait_in;         // forward pass 1 waits for done[warp] (a fused phase precedes)
    int push_out;        // inverse pass 1 sends its results to the owners of their tiles (a fused phase follows); else in place
    uint32_t par_done;
};

// The 16 values v[m] = elements t' + (S/16) m of this thread's pass-1 butterfly t' (class c = its warp inside the group) go to
// the warps that own the tiles c + NW m.  m < MAXT NV: warp c of virtual rank (m + 4 c) mod NV -- CTA vr / G, group vr mod G --
// its tile m / NV; the others (G = 1): tile number e = (m - MAXT NV) NW + c of the left-over tiles, helper e / NV of CTA
// e mod NV.  Operand slot q_me, lane t' mod 32.
template <class T, int NW, int NV, int G, int MAXT, int NQ>
__device__ __forceinline__ void wide_push16(const cplx<T>* v, const WideFlow& fa, int c, int lane) {
    constexpr uint32_t SLOT = (uint32_t)(NQ * 32 * sizeof(cplx<T>));
    const uint32_t base = fa.stage + (uint32_t)(fa.q_me * 32 + lane) * (uint32_t)sizeof(cplx<T>);
#pragma unroll
    for (int m = 0; m < 16; ++m) {
        if (m < MAXT * NV) {
            const int vo = (m + 4 * c) % NV, cta = vo / G, go = vo % G;
            st_async(dsmem_addr(base + (uint32_t)((go * NW + c) * MAXT + m / NV) * SLOT, cta), v[m], dsmem_addr(fa.mb0 + 8 * (go * 2 * NW + c), cta));
        } else {
            const int e = (m - MAXT * NV) * NW + c, owner = e % NV, hlp = e / NV;
            st_async(dsmem_addr(base + (uint32_t)(NW * MAXT + hlp) * SLOT, owner), v[m], dsmem_addr(fa.mb0 + 8 * (2 * NW + hlp), owner));
        }
    }
}

// The linear core of one sub-block.  smv is the "virtual" base of the field: logical index i lives at smv[phys(i)], and
// this CTA holds i in [j S, (j + 1) S) only; the butterfly and table indices are the global ones of plan<L>.
// sh_keep (may be null): the results of the inverse pass 1 are also stored there (the half-stepped input of a non-resonant
// field, kept for the later round trips).
// KM: constant mode of the butterflies (kconst in opo_fft.cuh; fp32: the z-step loop runs kConstBunch - 1 applications with
// the high parts of the compile-time roots alone and one that carries kConstBunch low parts)
// tid: index inside the group; bar_id: the group's named CTA barrier
template <class T, int L, int NT, int NV, int G, int MAXT, int NQ, int KM = 0>
__device__ __noinline__ void wide_core(cplx<T>* smv, const cplx<T>* twl, const cplx<T>* __restrict__ tab, int j, int tid, WideFlow fa,
                                       cplx<T>* __restrict__ sh_keep, int bar_id) {
    using PL = plan<L>;
    constexpr int NW = NT / 32, S = 1 << (L - 2);
    constexpr int RBL = PL::rbits(3), R = 1 << RBL, NBF = (1 << L) >> RBL, NBL = S >> RBL;
    constexpr int NB2 = S >> PL::rbits(2);
    constexpr bool chain = PL::rbits(2) == RBL && NBL % NT == 0;     // N = 2^14: passes 2, 3, 2 stay inside a warp's blocks
    const int warp = tid >> 5, lane = tid & 31;
    auto core_bar = [bar_id] { asm volatile("bar.sync %0, %1;" ::"r"(bar_id), "n"(NT) : "memory"); };      // the threads of this group only
    if (fa.wait_in) {
        mbar_wait_cta(fa.mb + 8 * (NW + warp), fa.par_done);      // (acquire at CTA scope: the bytes counted on the barrier are visible, and L1 is left alone)
        if (lane == 0) mbar_arm(fa.mb + 8 * (NW + warp), 16u * 32u * (uint32_t)sizeof(cplx<T>));       // the results of the next fused phase
    }
    fwd_bf<T, L, 1, KM>(smv, twl, j * NT + tid);
    core_bar();
    if constexpr (chain) {
#pragma unroll 1
        for (int ul = tid; ul < NBL; ul += NT) {
            const int u = j * NBL + ul;
            cplx<T> h[R];
#pragma unroll
            for (int k = 0; k < R; ++k) h[k] = ldg(&tab[k * NBF + u]);
            fwd_bf<T, L, 2, KM>(smv, twl, u);
            __syncwarp();
            mid_bf<T, L, cplx<T>, KM>(smv, h, u);
            __syncwarp();
            inv_bf<T, L, 2, KM>(smv, twl, u);
        }
    } else {
#pragma unroll 1
        for (int ul = tid; ul < NB2; ul += NT) fwd_bf<T, L, 2, KM>(smv, twl, j * NB2 + ul);
        core_bar();
#pragma unroll 1
        for (int ul = tid; ul < NBL; ul += NT) {
            const int u = j * NBL + ul;
            cplx<T> h[R];
#pragma unroll
            for (int k = 0; k < R; ++k) h[k] = ldg(&tab[k * NBF + u]);
            mid_bf<T, L, cplx<T>, KM>(smv, h, u);
        }
        core_bar();
#pragma unroll 1
        for (int ul = tid; ul < NB2; ul += NT) inv_bf<T, L, 2, KM>(smv, twl, j * NB2 + ul);
    }
    core_bar();
    if (!fa.push_out) {
        inv_bf<T, L, 1, KM>(smv, twl, j * NT + tid);
    } else {
        // inverse pass 1 with its results sent to the owners of their tiles
        constexpr int RB = PL::rbits(1), R1 = 1 << RB, SB = PL::sbits(1);
        static_assert(R1 == 16 && (1 << SB) == NT, "one radix-16 pass-1 butterfly per thread");
        const cplx<T>* __restrict__ w = twl + PL::tw_offset(1);
        const cplx<T>* __restrict__ p = smv + elem_base<T, RB, SB>(j, tid);
        cplx<T> v[R1];
#pragma unroll
        for (int k = 0; k < R1; ++k) v[k] = p[elem_off<T, RB, SB>(k)];
#pragma unroll
        for (int k = 1; k < R1; ++k) v[k] = cmulc(v[k], w[((k - 1) << SB) + tid]);
        dit_inv<T, R1, KM>::run(v);
        wide_push16<T, NW, NV, G, MAXT, NQ>(v, fa, warp, lane);
        if (sh_keep != nullptr) {
#pragma unroll
            for (int m = 0; m < R1; ++m) sh_keep[tid + NT * m] = v[m];
        }
    }
}

enum { WIDE_RK4 = 0, WIDE_FWD0 = 1, WIDE_INV0 = 2 };

template <class T, int L, int F, bool DK0 = false, int G = 1>
__global__ void __launch_bounds__(wide_layout<T, L, F, G>::NTH, 1) k_wide(ResidentArgs a) {
    using WL = wide_layout<T, L, F, G>;
    using PL = plan<L>;
    static_assert(WL::ok, "wide engine: N = 4 . 16 . r . r'");
    constexpr int N = 1 << L, S = WL::S, NT = WL::NT, NW = WL::NW, NCTA = WL::NCTA, NV = WL::NV, R = 4;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank();
    const int cid = blockIdx.x / NCTA, n_clusters = gridDim.x / NCTA;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    // a core warp belongs to group grp = one virtual rank: one pass-1 butterfly per thread, up to MAXT tiles; the warps behind
    // the groups are helpers (G = 1): one tile each, no part in the core
    const bool core = warp < G * NW;
    const int grp = (G > 1 && core) ? warp / NW : 0, wc = core ? warp - grp * NW : 0, tid_g = tid - grp * NT;
    const int vr = rank * G + grp;                               // my virtual rank
    const int x = vr / WL::C, j = vr % WL::C;                    // my field (the same for every group of a CTA), my sub-block
    cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw + (size_t)grp * WL::field_bytes);       // my sub-block: local index i at sm[phys(i)]

    // sub-block k of field f, wherever it lives in the cluster: CTA (4 f + k) / G, group (4 f + k) mod G (one mapa where it is
    // used: twelve addresses kept in registers cost the two-group variant, which has 128 registers per thread, more in spills)
    const uint32_t smem0 = (uint32_t)__cvta_generic_to_shared(smem_raw);
    auto fld = [smem0](int f, int k) -> uint32_t {
        return dsmem_addr(smem0 + (uint32_t)(((f * WL::C + k) % G) * WL::field_bytes), (f * WL::C + k) / G);
    };
    cplx<T>* const smv = sm - phys<T>(j * S);                    // phys(j S + i) = phys(j S) + phys(i): S is a multiple of the pad period

    const cplx<T>* tw = reinterpret_cast<const cplx<T>*>(a.tw);
    {   // shared-memory copy of the twiddles of the local passes, addressed as the global table is
        cplx<T>* d = reinterpret_cast<cplx<T>*>(smem_raw + WL::tw_offset_bytes);
        for (int i = tid; i < PL::tw_local_count; i += WL::NTH) d[i] = ldg(&tw[PL::tw_local_begin + i]);
    }
    const cplx<T>* twl = reinterpret_cast<const cplx<T>*>(smem_raw + WL::tw_offset_bytes) - PL::tw_local_begin;
    const uint32_t mb0 = (uint32_t)__cvta_generic_to_shared(smem_raw + WL::mbar_offset);
    const uint32_t mb = mb0 + 8 * (grp * 2 * NW);                // my group's ready[0]
    if (tid == 0) {
        for (int c = 0; c < G * 2 * NW; ++c) mbar_init(mb0 + 8 * c, 1);
        // per group ready[c]: the operands of warp c's tiles have arrived in its staging slots; done[c]: the results of all tiles
        // of class c have arrived in the group's sub-block
        for (int hh = 0; hh < WL::NH; ++hh) mbar_init(mb0 + 8 * (G * 2 * NW + hh), 1);      // the operands of helper hh's tile have arrived
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    cluster.sync();       // every CTA's barriers exist (and its twiddle copy is complete) before anybody sends to them

    // this thread's pass-0 butterflies -- the same at every z-step -- and their twiddles
    int nt_own = 0;
    int cls = wc;                                 // class of my tiles
    int p_own[WL::MAXT];
    cplx<T> w0[WL::MAXT][R - 1];
    {
        int m = ((vr - 4 * wc) % NV + NV) % NV;                  // tile m < MAXT NV of class c goes to virtual rank (m + 4 c) mod NV
        int n_mine = WL::MAXT;
        if (!core) {                                             // (G = 1) left-over tile e = hlp NV + rank: class e mod NW
            const int e = (warp - NW) * NV + rank;
            cls = e % NW;
            m = WL::MAXT * NV + e / NW;
            n_mine = e < WL::EX ? 1 : 0;
        }
#pragma unroll
        for (int i = 0; i < WL::MAXT; ++i, m += NV) {
            p_own[i] = 0;
#pragma unroll
            for (int k = 0; k < R - 1; ++k) w0[i][k] = cplx<T>{(T)1, (T)0};
            if (i < n_mine && m < WL::TPC) {
                const int t = (cls + NW * m) * 32 + lane;
                p_own[i] = phys<T>(t) * (int)sizeof(cplx<T>);       // byte offset inside a sub-block
#pragma unroll
                for (int k = 0; k < R - 1; ++k) w0[i][k] = ldg(&tw[k * S + t]);
                nt_own = i + 1;
            }
        }
    }

    // Every phase of a barrier has ONE arrival -- its own warp's, which also announces the bytes the phase will bring
    // (mbar_arm) -- and completes when those bytes have landed.  A warp arms the next phase right after its wait; bytes that
    // arrive before the arming leave the count negative for a moment, which the barrier allows.
    const uint32_t ready_bytes = (uint32_t)nt_own * WL::NQ * 32 * (uint32_t)sizeof(cplx<T>);
    const uint32_t my_ready = core ? mb + 8 * wc : mb0 + 8 * (G * 2 * NW + (warp - G * NW));
    if (lane == 0) {
        if (nt_own > 0) mbar_arm(my_ready, ready_bytes);
        if (core) mbar_arm(mb + 8 * (NW + wc), WL::done_bytes);
    }
    WideFlow fb;
    fb.mb = mb;
    fb.mb0 = mb0;
    fb.stage = (uint32_t)__cvta_generic_to_shared(smem_raw + WL::stage_offset);
    fb.q_me = vr;
    fb.wait_in = 0; fb.push_out = 0; fb.par_done = 0;
    const cplx<T>* stg = reinterpret_cast<const cplx<T>*>(smem_raw + WL::stage_offset) +
                         (size_t)(core ? (grp * NW + wc) * WL::MAXT : G * NW * WL::MAXT + (warp - G * NW)) * WL::NQ * 32 + lane;       // my staging slot(s)

    T kap[3] = {(T)a.kappa[0], (T)a.kappa[1], (T)a.kappa[2]};
    const T h = (T)a.h;
    const int nz = a.nz;
    const bool rt_mode = a.mode != 0;
    const bool resonant = a.resonant[x] != 0;
    const cplx<T>* tabH = reinterpret_cast<const cplx<T>*>(a.tabH[x]);
    const cplx<T>* tabH2 = reinterpret_cast<const cplx<T>*>(a.tabH2[x]);
    uint32_t fz = 0;          // fused phases executed so far (mbarrier phase parity)
    int mask_eom = 0;         // resonant fields with an intracavity phase modulator
#pragma unroll
    for (int f = 0; f < F; ++f)
        if (a.eom[f] != nullptr && a.resonant[f]) mask_eom |= 1 << f;
    const bool my_eom = (mask_eom >> x) & 1;

    // pass-0 butterflies of this thread's tiles: MODE = WIDE_RK4: inverse pass 0 -> RK4 -> forward pass 0 (all fields);
    // WIDE_FWD0 / WIDE_INV0: the pass alone, on the fields of `mask`
    auto tiles = [&](auto mode_tag, int mask, cplx<T> e0, cplx<T> e1, cplx<T> e2) {
        constexpr int MODE = decltype(mode_tag)::value;
        cplx<T> v[WL::MAXT][F][R];
        if constexpr (MODE != WIDE_RK4) {
#pragma unroll
            for (int i = 0; i < WL::MAXT; ++i) {        // remote loads: all of them in flight before the first is consumed
                if (i < nt_own) {
#pragma unroll
                    for (int f = 0; f < F; ++f) {
                        if (!((mask >> f) & 1)) continue;
#pragma unroll
                        for (int k = 0; k < R; ++k) v[i][f][k] = dsmem_ld(fld(f, k) + p_own[i], cplx<T>{});
                    }
                }
            }
        }
#pragma unroll
        for (int i = 0; i < WL::MAXT; ++i) {
            if (i < nt_own) {
                if constexpr (MODE == WIDE_RK4) {       // operands staged in local shared memory by the owners' inverse pass 1
#pragma unroll
                    for (int f = 0; f < F; ++f)
#pragma unroll
                        for (int k = 0; k < R; ++k) v[i][f][k] = stg[(i * WL::NQ + f * WL::C + k) * 32];
                }
#pragma unroll
                for (int f = 0; f < F; ++f) {
                    if (MODE != WIDE_RK4 && !((mask >> f) & 1)) continue;
                    if constexpr (MODE != WIDE_FWD0) {
#pragma unroll
                        for (int k = 1; k < R; ++k) v[i][f][k] = cmulc(v[i][f][k], w0[i][k - 1]);
                        dit_inv<T, R>::run(v[i][f]);
                    }
                }
                if constexpr (MODE == WIDE_RK4) {
#pragma unroll
                    for (int q = 0; q < R; ++q) {
                        cplx<T> y[F];
#pragma unroll
                        for (int f = 0; f < F; ++f) y[f] = v[i][f][q];
                        Rk4<T, F>::template step<DK0>(y, e0, e1, e2, kap, h);
#pragma unroll
                        for (int f = 0; f < F; ++f) v[i][f][q] = y[f];
                    }
                }
#pragma unroll
                for (int f = 0; f < F; ++f) {
                    if (MODE != WIDE_RK4 && !((mask >> f) & 1)) continue;
                    if constexpr (MODE != WIDE_INV0) {
                        dif<T, R>::run(v[i][f]);
#pragma unroll
                        for (int k = 1; k < R; ++k) v[i][f][k] = cmul(v[i][f][k], w0[i][k - 1]);
                    }
#pragma unroll
                    for (int k = 0; k < R; ++k) {
                        if constexpr (MODE == WIDE_RK4) {
                            // counted on done[class] of the owner: its group go = (4 f + k) mod G of its CTA
                            const uint32_t dst = fld(f, k);
                            st_async(dst + p_own[i], v[i][f][k],
                                     dst + (uint32_t)(WL::mbar_offset - ((f * WL::C + k) % G) * WL::field_bytes + 8 * (((f * WL::C + k) % G) * 2 * NW + NW + cls)));
                        } else {
                            dsmem_st(fld(f, k) + p_own[i], v[i][f][k]);
                        }
                    }
                }
            }
        }
    };
    using tag_rk4 = std::integral_constant<int, WIDE_RK4>;
    using tag_fwd0 = std::integral_constant<int, WIDE_FWD0>;
    using tag_inv0 = std::integral_constant<int, WIDE_INV0>;
    const cplx<T> one = {(T)1, (T)0};
    auto cluster_bar = [&]() { cluster_arrive(); cluster_wait(); };

    // a cluster loops over instances b = cid, cid + n_clusters, ...
#pragma unroll 1
    for (int b = cid; b < a.batch; b += n_clusters) {
        const int steps_l = a.steps;
        const int total = rt_mode ? steps_l * nz : steps_l;     // RK4 steps of this call
        const size_t off = (size_t)b * N + (size_t)j * S;       // my sub-block inside [B][N]
        cplx<T>* cur = reinterpret_cast<cplx<T>*>(a.cur[x]) + off;
        const cplx<T>* ph = reinterpret_cast<const cplx<T>*>(a.phase) + (size_t)b * a.phase_stride;
        const cplx<T>* tabHB = reinterpret_cast<const cplx<T>*>(a.tabHB[x]) + (size_t)b * a.tab_stride[x];
        cplx<T>* SH = reinterpret_cast<cplx<T>*>(a.SH[x]) + off;

        if (core) {
            const cplx<T>* __restrict__ g = cur;
#pragma unroll 4
            for (int i = tid_g; i < S; i += NT) sm[phys<T>(i)] = g[i];
        }
        cluster_bar();                                    // every sub-block of the instance is on chip
        tiles(tag_fwd0{}, (1 << F) - 1, one, one, one);
        cluster_bar();

        // q counts linear operators: q = 0 first half-step, q = total last half-step, between them the merged full steps;
        // in round-trip mode q = m nz + s and s = 0 (m > 0) crosses the cavity boundary
        int fq = a.fq0;                                         // full steps applied before the next one (ResidentArgs::fq0)
#pragma unroll 1
        for (int q = 0; q <= total; ++q) {
            const int s = rt_mode ? q % nz : a.z0 + q;          // index of the RK4 step that follows
            const bool crossing = rt_mode && q > 0 && q < total && s == 0;
            const bool keep = rt_mode && q == 0 && !resonant && steps_l > 1;      // SH <- first half-stepped input
            cplx<T> e0 = one, e1 = one, e2 = one;
            if constexpr (!DK0) {
                if (q < total) { e0 = ldg(ph + 2 * s); e1 = ldg(ph + 2 * s + 1); e2 = ldg(ph + 2 * s + 2); }
            }
            if (!core) {
                // a helper warp has no part in the linear core
            } else if (crossing && my_eom) {
                // the modulator acts in the time domain between the boundary's spectral factor and the next pass: last
                // half-step and boundary in place (table H G m), the rest below
                WideFlow fa = fb;
                fa.wait_in = 1; fa.par_done = (fz - 1) & 1;
                fa.push_out = 0;
                wide_core<T, L, NT, NV, G, WL::MAXT, WL::NQ>(smv, twl, reinterpret_cast<const cplx<T>*>(a.tabHG[x]) + (size_t)b * a.tab_stride[x], j, tid_g, fa, nullptr, 1 + grp);
            } else if (crossing && !resonant) {
                // fresh pump / frozen seed, already half-stepped: a thread sends the elements of its own pass-1
                // butterfly, i.e. of its class, to the tiles' owners as an inverse pass 1 would
                mbar_wait_cta(mb + 8 * (NW + wc), (fz - 1) & 1);
                if (lane == 0) mbar_arm(mb + 8 * (NW + wc), WL::done_bytes);
                const cplx<T>* __restrict__ g = SH;
                cplx<T> v[16];
#pragma unroll
                for (int k = 0; k < 16; ++k) v[k] = g[tid_g + NT * k];
                wide_push16<T, NW, NV, G, WL::MAXT, WL::NQ>(v, fb, wc, lane);
            } else {
                const cplx<T>* tab = (q == 0 || q == total) ? tabH + (size_t)((a.hq0 + (q == 0 ? 0 : 1)) & a.tab_cycle_mask) * N
                                                            : (crossing ? tabHB : tabH2 + (size_t)(fq & a.tab_cycle_mask) * N);
                WideFlow fa = fb;
                fa.wait_in = q > 0; fa.par_done = (fz - 1) & 1;
                fa.push_out = q < total;
                if constexpr (sizeof(T) == 4) {
                    if (((a.op0 + q) & (kConstBunch - 1)) == 0) wide_core<T, L, NT, NV, G, WL::MAXT, WL::NQ, 2>(smv, twl, tab, j, tid_g, fa, keep ? SH : nullptr, 1 + grp);
                    else wide_core<T, L, NT, NV, G, WL::MAXT, WL::NQ, 1>(smv, twl, tab, j, tid_g, fa, keep ? SH : nullptr, 1 + grp);
                } else {
                    wide_core<T, L, NT, NV, G, WL::MAXT, WL::NQ>(smv, twl, tab, j, tid_g, fa, keep ? SH : nullptr, 1 + grp);
                }
            }
            if (crossing && mask_eom) {         // uniform over the cluster
                // inverse pass 0 -> x E[n] -> forward pass 0 -> first half-step of the next pass, for the modulated fields; the
                // other fields have sent their operands already and their owners' tiles simply wait for these
                cluster_bar();
                tiles(tag_inv0{}, mask_eom, one, one, one);
                cluster_bar();
                if (core && my_eom) {
                    const cplx<T>* __restrict__ E = reinterpret_cast<const cplx<T>*>(a.eom[x]) + (size_t)j * S;
#pragma unroll 4
                    for (int i = tid_g; i < S; i += NT) sm[phys<T>(i)] = cmul(sm[phys<T>(i)], ldg(&E[i]));
                }
                cluster_bar();
                tiles(tag_fwd0{}, mask_eom, one, one, one);
                cluster_bar();
                if (core && my_eom) {
                    WideFlow fa = fb;
                    fa.wait_in = 0; fa.push_out = 1;
                    wide_core<T, L, NT, NV, G, WL::MAXT, WL::NQ>(smv, twl, tabH, j, tid_g, fa, nullptr, 1 + grp);
                }
            }
            if (q == total) break;
            if (q > 0 && !crossing) ++fq;
            if (nt_own > 0) {
                mbar_wait_cta(my_ready, fz & 1);                // the operands of my tiles are in my staging buffer
                if (lane == 0) mbar_arm(my_ready, ready_bytes);
                tiles(tag_rk4{}, (1 << F) - 1, e0, e1, e2);
            }
            ++fz;
        }
        cluster_bar();                                    // every field is ready for its inverse pass 0
        tiles(tag_inv0{}, (1 << F) - 1, one, one, one);
        cluster_bar();

        if (!rt_mode) {
            if (core) {
                cplx<T>* __restrict__ g = cur;
#pragma unroll 4
                for (int i = tid_g; i < S; i += NT) g[i] = sm[phys<T>(i)];
            }
        } else {
            if (core) {   // fields at z = L of the last pass
                cplx<T>* __restrict__ g = reinterpret_cast<cplx<T>*>(a.exitb[x]) + off;
#pragma unroll 4
                for (int i = tid_g; i < S; i += NT) g[i] = sm[phys<T>(i)];
            }
            // mirror, spectral phase and phase modulator of the call's last round trip
            int maskb = 0;
#pragma unroll
            for (int f = 0; f < F; ++f)
                if (a.resonant[f] && a.boundary_fft[f]) maskb |= 1 << f;
            if (maskb) {        // uniform over the cluster
                cluster_bar();                            // nobody writes into a field whose owner still stores its exit copy
                tiles(tag_fwd0{}, maskb, one, one, one);
                cluster_bar();
                if (core && ((maskb >> x) & 1)) {
                    const cplx<T>* tabGM = reinterpret_cast<const cplx<T>*>(a.tabGM[x]) + (size_t)b * a.tab_stride[x];
                    wide_core<T, L, NT, NV, G, WL::MAXT, WL::NQ>(smv, twl, tabGM, j, tid_g, fb, nullptr, 1 + grp);
                }
                cluster_bar();
                tiles(tag_inv0{}, maskb, one, one, one);
                cluster_bar();
            }
            if (!core) {
                // (helpers hold no field)
            } else if (resonant) {
                const cplx<T>* __restrict__ E = reinterpret_cast<const cplx<T>*>(a.eom[x]);
                cplx<T> mf = one;
                if (!a.boundary_fft[x]) mf = ldg(reinterpret_cast<const cplx<T>*>(a.mirror[x]) + b);
                if (E != nullptr) {
#pragma unroll 4
                    for (int i = tid_g; i < S; i += NT) cur[i] = cmul(cmul(sm[phys<T>(i)], mf), ldg(&E[j * S + i]));
                } else {
#pragma unroll 4
                    for (int i = tid_g; i < S; i += NT) cur[i] = cmul(sm[phys<T>(i)], mf);
                }
            } else {
                const cplx<T>* __restrict__ Sx = reinterpret_cast<const cplx<T>*>(a.S[x]) + off;
#pragma unroll 4
                for (int i = tid_g; i < S; i += NT) cur[i] = Sx[i];
            }
        }
        // the next instance's load overwrites shared memory that only this CTA reads from here on: all foreign
        // accesses of this instance ended at the last cluster barrier
        __syncthreads();
    }
    cluster.sync();     // keep shared memory alive until every peer has left its last tile phase
}

template <class T, int L, int F, bool DK0, int G> cudaError_t wide_cfg(cudaLaunchConfig_t* cfg, cudaLaunchAttribute* attr, int n_clusters, cudaStream_t s) {
    using WL = wide_layout<T, L, F, G>;
    static device_once once;
    cudaError_t e0 = once.run([&] {
        cudaError_t e = cudaFuncSetAttribute(k_wide<T, L, F, DK0, G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)WL::total);
        if (e != cudaSuccess) return e;
        if (WL::NCTA > 8) e = cudaFuncSetAttribute(k_wide<T, L, F, DK0, G>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        return e;
    });
    if (e0 != cudaSuccess) return e0;
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = WL::NCTA;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg->gridDim = dim3((unsigned)(n_clusters * WL::NCTA), 1, 1);
    cfg->blockDim = dim3(WL::NTH, 1, 1);
    cfg->dynamicSmemBytes = WL::total;
    cfg->stream = s;
    cfg->attrs = attr;
    cfg->numAttrs = 1;
    return cudaSuccess;
}

template <class T, int L, int F, int G> cudaError_t wide_info_LF(ResidentInfo* out) {
    if constexpr (!wide_layout<T, L, F, G>::ok || wide_layout<T, L, F, G>::total > 232448) {
        return cudaErrorNotSupported;
    } else {
        cudaLaunchConfig_t cfg{};
        cudaLaunchAttribute attr[1];
        cudaError_t e = wide_cfg<T, L, F, false, G>(&cfg, attr, 1, nullptr);
        if (e != cudaSuccess) return e;
        int n = 0;
        e = cudaOccupancyMaxActiveClusters(&n, k_wide<T, L, F, false, G>, &cfg);
        if (e != cudaSuccess) return e;
        out->threads = wide_layout<T, L, F, G>::NTH;
        out->smem_bytes = cfg.dynamicSmemBytes;
        out->max_clusters = n;
        return cudaSuccess;
    }
}
// g: sub-blocks per CTA (1: clusters of 4 F CTAs, 2: clusters of 2 F CTAs)
template <class T, int L> cudaError_t wide_info_L(int n_fields, int g, ResidentInfo* out) {
    if (g == 2) return n_fields == 3 ? wide_info_LF<T, L, 3, 2>(out) : wide_info_LF<T, L, 2, 2>(out);
    return n_fields == 3 ? wide_info_LF<T, L, 3, 1>(out) : wide_info_LF<T, L, 2, 1>(out);
}

template <class T, int L, int F, bool DK0, int G> cudaError_t launch_wide_LF(const ResidentArgs& a, int n_clusters, cudaStream_t s) {
    if constexpr (!wide_layout<T, L, F, G>::ok || wide_layout<T, L, F, G>::total > 232448) {
        return cudaErrorNotSupported;
    } else {
        cudaLaunchConfig_t cfg{};
        cudaLaunchAttribute attr[1];
        cudaError_t e = wide_cfg<T, L, F, DK0, G>(&cfg, attr, n_clusters, s);
        if (e != cudaSuccess) return e;
        return cudaLaunchKernelEx(&cfg, k_wide<T, L, F, DK0, G>, a);
    }
}
template <class T, int L, bool DK0> cudaError_t launch_wide_L(const ResidentArgs& a, int n_clusters, cudaStream_t s) {
    if (a.wide_g == 2) return a.n_fields == 3 ? launch_wide_LF<T, L, 3, DK0, 2>(a, n_clusters, s) : launch_wide_LF<T, L, 2, DK0, 2>(a, n_clusters, s);
    return a.n_fields == 3 ? launch_wide_LF<T, L, 3, DK0, 1>(a, n_clusters, s) : launch_wide_LF<T, L, 2, DK0, 1>(a, n_clusters, s);
}

}  // namespace opo
