// opo_resident.cuh -- resident engine: one thread-block cluster per OPO instance, CTA rank = field.
//
// Each CTA keeps its field in (padded) shared memory for the whole call -- every z-step of every
// round trip -- so HBM is touched only at the ends of the call and, per round trip, for the
// re-injected non-resonant inputs; the constant tables stream from L2.
//
// A z-step (order L/2 - N - L/2, adjacent half-steps merged) is two phases:
//
//   core   : CTA-local.  Forward passes 1..P-2, [last forward pass . table . first inverse pass] in
//            registers, inverse passes P-2..1 (opo_fft.cuh), twiddles from a shared-memory copy.
//   fused  : inverse pass 0 -> RK4 -> forward pass 0, in registers.  Pass 0 is a radix-4 butterfly
//            over x[t + j N/4], j = 0..3; the RK4 step of the coupling terms
//            needs all F fields at those four grid points.  The butterflies t are dealt to the F
//            CTAs in tiles of 32; a CTA reads its own field locally and the foreign fields through
//            distributed shared memory, transforms, integrates, transforms back and writes all F
//            fields back.  The loop over a warp's tiles is software-pipelined: the DSMEM loads of the
//            next tile are in flight under the arithmetic of the current one (the SM-to-SM link moves
//            ~16 B/clk per SM, measured; 2/3 of the state crosses it in each direction per z-step).
//   sync   : N >= 2^12: class-granular mbarriers (flow_cfg in opo_fft.cuh), no cluster-wide barrier;
//            smaller N: one cluster barrier before and one after the fused phase.
//
// Variants: the paper's order N/2 - L - N/2 (Eq. 10-11) is the instantiation NLN = true (two RK4
// half-steps in the fused phase, one pass per launch); the intracavity phase modulator (L149-154)
// rides on the last store of a call.
//
// Merged tables: H.H = H2 between RK4 steps; H . G m . H = HB across the cavity boundary for a
// resonant field; a non-resonant field restarts every round trip
// from IDFT(H DFT(S_x)) (kept, up to its inverse pass 0, in the scratch buffer SH).
//
// A cluster loops over instances b = cluster_id, cluster_id + n_clusters, ... (batched mode,
// BASELINE.json configs[4]); instances are independent, there is no inter-cluster communication.
#pragma once
#include <cooperative_groups.h>

#include "opo_kernels.cuh"

namespace opo {

namespace cg = cooperative_groups;

// cluster barrier, split so that independent work can sit between arrive and wait.  release / acquire
// at cluster scope: the distributed-shared-memory stores of the fused phase are visible to their
// owner after the wait.
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

// Shared memory of the resident engine: smem_layout (field + twiddles of the local passes), then this
// thread's pass-0 twiddles.  A thread handles the same pass-0 butterflies t at every z-step, so
// their three twiddles are read from L2 once per launch: tw0s[(i * 3 + k) * NT + tid] for its i-th tile.
template <class T, int L, int F> struct res_layout {
    static constexpr int NT = cta_threads<T, L>::value;
    static constexpr int S = 1 << (L - 2), NTILES = (S + 31) / 32, NW = NT / 32;
    static constexpr int MAXT = (NTILES + F * NW - 1) / (F * NW);          // tiles per warp
    static constexpr size_t tw0_offset = (smem_layout<T, L>::total + 15) / 16 * 16;
    static constexpr size_t tw0_bytes = (size_t)MAXT * 3 * NT * sizeof(cplx<T>);
    static constexpr bool tw0_smem = tw0_offset + tw0_bytes <= 232448;    // 227 KB per CTA
    static constexpr size_t data_end = tw0_smem ? tw0_offset + tw0_bytes : smem_layout<T, L>::total;
    // flow synchronisation (opo_fft.cuh): ready[NCLS], done[NCLS] mbarriers
    using FC = flow_cfg<T, L, NT>;
    static constexpr bool flow = FC::ok && (F * FC::NW) % (FC::NCLS > 0 ? FC::NCLS : 1) == 0 && NTILES % 1 == 0 && S >= 32 &&
                                 F * NW <= NTILES;      // every warp owns at least one tile
    static constexpr size_t mbar_offset = (data_end + 15) / 16 * 16;
    static constexpr size_t total = flow ? mbar_offset + 16 * (size_t)(FC::NCLS > 0 ? FC::NCLS : 1) : data_end;
    static constexpr int done_count = flow ? F * FC::NW / FC::NCLS : 0;
    static constexpr int ready_count = FC::G * F;
    // two clusters' CTAs share an SM when shared memory (plus 1 KB of system reservation each) and registers allow it:
    // the exchange of one instance then runs under the arithmetic of another
    static constexpr int ctas_per_sm = (2 * (total + 1024) <= 233472 && 2 * NT * 128 <= 65536) ? 2 : 1;
};

// inverse pass 0 -> RK4 -> forward pass 0 on this CTA's share of the radix-4 butterflies.
// Software-pipelined over the warp's tiles: the distributed-shared-memory loads of the next tile's
// foreign fields are issued before the arithmetic of the current one (the link moves ~16 B/clk per
// SM, so the exchange takes about as long as the arithmetic and has to run under it).  RANK is a
// template parameter so that "foreign" is a compile-time property of the field index.
template <class T, int L, int F, int NT, int RANK, bool NLN, bool DK0 = false>
__device__ __forceinline__ void fused_pass0_rk4(cplx<T>* const* fld, int tid, const cplx<T>* __restrict__ tw0,
                                                const cplx<T>* __restrict__ tw0s, cplx<T> e0, cplx<T> e1, cplx<T> e2,
                                                cplx<T> e3, cplx<T> e4, int halves, T pre, T post, const T* kap, T h, uint32_t mb, uint32_t parity) {
    static_assert(plan<L>::rbits(0) == 2, "pass 0 must be radix 4");
    using RL = res_layout<T, L, F>;
    constexpr int RB = 2, R = 4, SB = L - 2, S = 1 << SB;
    constexpr int NTILES = (S + 31) / 32, NW = NT / 32;
    constexpr bool TWS = res_layout<T, L, F>::tw0_smem;
    const int warp = tid >> 5, lane = tid & 31;
    cplx<T> nv[F][R];                       // foreign fields of the next tile (slot RANK unused)
    auto prefetch = [&](int tile) {
        const int t = tile * 32 + lane;
        if (S >= 32 || t < S) {
            const int p0 = elem_base<T, RB, SB>(0, t);
#pragma unroll
            for (int x = 0; x < F; ++x)
                if (x != RANK) {
#pragma unroll
                    for (int k = 0; k < R; ++k) nv[x][k] = fld[x][p0 + elem_off<T, RB, SB>(k)];
                }
        }
    };
    int tile = RANK + F * warp, i = 0;
    // all tiles of a warp belong to one class (F NW is a multiple of NCLS)
    const int cls = RL::flow ? tile % (RL::FC::NCLS > 0 ? RL::FC::NCLS : 1) : 0;
    if constexpr (RL::flow) mbar_wait(mb + 8 * cls, parity);      // ready[cls]: every field's inverse pass 1 of my class
    if (tile < NTILES) prefetch(tile);
#pragma unroll 1
    for (; tile < NTILES; tile += F * NW, ++i) {
        const int t = tile * 32 + lane;
        const bool active = S >= 32 || t < S;
        const int p0 = elem_base<T, RB, SB>(0, t);
        cplx<T> w[R - 1];
        cplx<T> v[F][R];
        if (active) {
#pragma unroll
            for (int k = 0; k < R - 1; ++k) {
                if constexpr (TWS) w[k] = tw0s[(i * 3 + k) * NT + tid];
                else w[k] = ldg(&tw0[k * S + t]);
            }
#pragma unroll
            for (int k = 0; k < R; ++k) v[RANK][k] = fld[RANK][p0 + elem_off<T, RB, SB>(k)];
#pragma unroll
            for (int x = 0; x < F; ++x)
                if (x != RANK) {
#pragma unroll
                    for (int k = 0; k < R; ++k) v[x][k] = nv[x][k];
                }
        }
        if (tile + F * NW < NTILES) prefetch(tile + F * NW);
        if (active) {
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
                if constexpr (NLN) {      // a pass-0 pair with no table between (first / last half-step) carries its own 1/4
#pragma unroll
                    for (int x = 0; x < F; ++x) y[x] = {y[x].re * pre, y[x].im * pre};
                }
                Rk4<T, F>::template step<DK0>(y, e0, e1, e2, kap, h);
                if constexpr (NLN) {      // N/2 - L - N/2: two half-steps meet between two linear operators
                    if (halves == 2) Rk4<T, F>::step(y, e2, e3, e4, kap, h);
#pragma unroll
                    for (int x = 0; x < F; ++x) y[x] = {y[x].re * post, y[x].im * post};
                }
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
    }
    if constexpr (RL::flow) mbar_arrive_cluster(mb + 8 * (RL::FC::NCLS + cls), lane, F);   // done[cls] in every CTA
}

// stand-alone pass 0 on the CTA's own field (the first and last linear operator of a call)
template <class T, int L, int NT>
__device__ __noinline__ void pass0_local(const cplx<T>* tw, int tid, bool inverse) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
    if (inverse) inv_pass_smem<T, L, 0, NT, false>(sm, tw, tid);
    else fwd_pass_smem<T, L, 0, NT, false>(sm, tw, tid);
}

// NLN: the N/2 - L - N/2 ordering is a separate instantiation, so that the default kernel carries none of its code
// DK0: every instance has dk = 0 (BASELINE.json configs[0..3]): the RK4 stage phases are skipped; again its own instantiation
template <class T, int L, int F, bool NLN = false, bool DK0 = false>
__global__ void __launch_bounds__(cta_threads<T, L>::value, res_layout<T, L, F>::ctas_per_sm) k_resident(ResidentArgs a) {
    constexpr int N = 1 << L, NT = cta_threads<T, L>::value;
    using PL = plan<L>;
    using SL = smem_layout<T, L>;
    using RL = res_layout<T, L, F>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
    cg::cluster_group cluster = cg::this_cluster();
    const int x = (int)cluster.block_rank();            // my field
    const int cid = blockIdx.x / F, n_clusters = gridDim.x / F;
    const int tid = threadIdx.x;

    cplx<T>* fld[F];
#pragma unroll
    for (int f = 0; f < F; ++f) fld[f] = cluster.map_shared_rank(sm, f);

    const cplx<T>* tw = reinterpret_cast<const cplx<T>*>(a.tw);
    {   // shared-memory copy of the twiddles of the local passes
        cplx<T>* twl = reinterpret_cast<cplx<T>*>(smem_raw + SL::field_bytes);
        for (int i = tid; i < PL::tw_local_count; i += NT) twl[i] = ldg(&tw[PL::tw_local_begin + i]);
    }
    const cplx<T>* tw0s = reinterpret_cast<const cplx<T>*>(smem_raw + RL::tw0_offset);
    if constexpr (RL::tw0_smem) {   // this thread's pass-0 twiddles (see res_layout)
        cplx<T>* d = reinterpret_cast<cplx<T>*>(smem_raw + RL::tw0_offset);
        constexpr int S = 1 << (L - 2);
        int i = 0;
        for (int tile = x + F * (tid >> 5); tile < RL::NTILES; tile += F * RL::NW, ++i) {
            const int t = tile * 32 + (tid & 31);
            if (t < S)
                for (int k = 0; k < 3; ++k) d[(i * 3 + k) * NT + tid] = ldg(&tw[k * S + t]);
        }
    }
    constexpr bool FLOW = RL::flow;
    using FC = flow_cfg<T, L, NT>;
    const uint32_t mb = (uint32_t)__cvta_generic_to_shared(smem_raw + RL::mbar_offset);
    if constexpr (FLOW) {
        if (tid == 0) {
            for (int c = 0; c < FC::NCLS; ++c) {
                mbar_init(mb + 8 * c, RL::ready_count);
                mbar_init(mb + 8 * (FC::NCLS + c), RL::done_count);
            }
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        cluster.sync();     // every CTA's barriers exist before anybody arrives on them
    }
    uint32_t fz = 0;        // fused phases executed so far by this cluster (mbarrier phase parity)
    // this warp's classes in pass 1 (as in group_fwd / group_inv)
    const int wg = (tid % FC::NTG) >> 5, lane = tid & 31;
    auto flow_wait_done_all = [&](uint32_t parity) {      // the previous fused phase has released all of my field
        if constexpr (FLOW)
            for (int it = 0; it < FC::NIT; ++it) mbar_wait(mb + 8 * (FC::NCLS + wg + FC::NWG * it), parity);
    };
    auto flow_arrive_ready_all = [&]() {                   // stands in for the arrivals of an inverse pass 1
        if constexpr (FLOW)
            for (int it = 0; it < FC::NIT; ++it) mbar_arrive_cluster(mb + 8 * (wg + FC::NWG * it), lane, F);
    };
    const cplx<T>* tabH = reinterpret_cast<const cplx<T>*>(a.tabH[x]);
    const cplx<T>* tabH2 = reinterpret_cast<const cplx<T>*>(a.tabH2[x]);
    const bool resonant = a.resonant[x] != 0;
    T kap[3] = {(T)a.kappa[0], (T)a.kappa[1], (T)a.kappa[2]};
    const T h = (T)a.h;
    const int nz = a.nz;
    const bool rt_mode = a.mode != 0;

    // Work list of this cluster.  Default: whole instances b = cid, cid + n_clusters, ...  With a.split (round-trip mode,
    // batch >= clusters) the unit of work is one round trip of one instance: the batch x steps units are cut into
    // n_clusters equal contiguous ranges (McNaughton's wrap-around rule), so that 256 instances on 45 clusters take
    // 5.69 instead of 6 instance-times.  An instance cut by a range boundary runs its early round trips on cluster c
    // and the late ones on cluster c + 1; each cluster walks its range backwards, so the early piece is the first thing
    // cluster c does and the late piece the last thing cluster c + 1 does; the state passes through HBM (`cur`) and a
    // per-(instance, field) flag with release / acquire at gpu scope.  All clusters are co-resident (grid <= max
    // active clusters), so the wait cannot deadlock.
    const long long units = (long long)a.batch * a.steps;
    const long long quota = (units + n_clusters - 1) / n_clusters;
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
        const int total = rt_mode ? steps_l * nz : steps_l;     // RK4 steps of this piece of work
        // where this piece stands in the handle's count of table uses (ResidentArgs::hq0, fq0): an instance cut into pieces
        // by the split schedule applies two half-steps more per cut
        const int cuts = (a.split && rt0 > 0) ? (int)(((long long)b * a.steps + rt0) / quota - ((long long)b * a.steps) / quota) : 0;
        const int hq_base = a.hq0 + 2 * cuts;
        int fq = a.fq0 + (rt_mode ? rt0 * (nz - 1) : 0);       // full steps applied before the next one
        int* const flag = a.flags ? a.flags + (size_t)b * F + x : nullptr;
        cplx<T>* cur = reinterpret_cast<cplx<T>*>(a.cur[x]) + (size_t)b * N;
        const cplx<T>* ph = reinterpret_cast<const cplx<T>*>(a.phase) + (size_t)b * a.phase_stride;
        const cplx<T>* tabHB = reinterpret_cast<const cplx<T>*>(a.tabHB[x]) + (size_t)b * a.tab_stride[x];
        cplx<T>* SH = reinterpret_cast<cplx<T>*>(a.SH[x]) + (size_t)b * N;

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
        const bool inj_any = x == 0 && tinj != (T)0 && resonant;
        if (inj_any && rt_mode && steps_l > 1 && !NLN) {
            load(reinterpret_cast<const cplx<T>*>(a.S[x]) + (size_t)b * N);
            __syncthreads();
            pass0_local<T, L, NT>(tw, tid, false);
            __syncthreads();
            linear_core_smem<T, L, NT>(tabH, tid);
            __syncthreads();
            store(SH);
            __syncthreads();
        }
        if (a.split && rt0 > 0) {       // the earlier round trips of this instance ran on another cluster
            if (tid == 0) {
                int v;
                do { asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(flag) : "memory"); } while (v < rt0);
            }
            __syncthreads();
#pragma unroll 4
            for (int i = tid; i < N; i += NT) sm[phys<T>(i)] = ldcg_c(cur + i);
        } else {
            load(cur);
        }
        __syncthreads();
        pass0_local<T, L, NT>(tw, tid, false);
        __syncthreads();

        if constexpr (NLN) {
            // inverse pass 0 -> RK4 -> forward pass 0 over the cluster, with the synchronisation around it
            auto run_fused = [&](cplx<T> e0, cplx<T> e1, cplx<T> e2, cplx<T> e3, cplx<T> e4, int halves, T hstep, T pre, T post) {
                if constexpr (!FLOW) { cluster_arrive(); cluster_wait(); }      // every field is ready for its inverse pass 0
                if (x == 0) fused_pass0_rk4<T, L, F, NT, 0, true>(fld, tid, tw, tw0s, e0, e1, e2, e3, e4, halves, pre, post, kap, hstep, mb, fz & 1);
                else if (F == 2 || x == 1) fused_pass0_rk4<T, L, F, NT, 1, true>(fld, tid, tw, tw0s, e0, e1, e2, e3, e4, halves, pre, post, kap, hstep, mb, fz & 1);
                else fused_pass0_rk4<T, L, F, NT, F - 1, true>(fld, tid, tw, tw0s, e0, e1, e2, e3, e4, halves, pre, post, kap, hstep, mb, fz & 1);
                ++fz;
                if constexpr (!FLOW) { cluster_arrive(); cluster_wait(); }      // every result has landed in its owner's shared memory
            };
            // the paper's own order N/2 - L - N/2 (Eq. 10-11), adjacent half-steps NOT merged into one
            // RK4 step (they are two RK4 steps of h/2): [N/2] (L [N/2 N/2])^(n-1) L [N/2], every L a full step (table H2).
            // The tables carry the 1/N of one forward + inverse transform; the first and the last half-step sit between a
            // forward and an inverse pass 0 with no table, hence their own exact factor 1/4.
            // phase table: exp(i dk j h/4).  One pass per launch (the host loops over round trips).
            const int zs = rt_mode ? 0 : a.z0, nsteps = rt_mode ? nz : a.steps;
            const T hh = (T)0.5 * h;
            if constexpr (FLOW) flow_arrive_ready_all();
            {
                const cplx<T>* p = ph + 4 * zs;
                run_fused(ldg(p), ldg(p + 1), ldg(p + 2), ldg(p + 2), ldg(p + 2), 1, hh, (T)0.25, (T)1);
            }
#pragma unroll 1
            for (int q = 0; q < nsteps; ++q) {
                if constexpr (FLOW) {
                    FlowArgs fa;
                    fa.mb = mb; fa.nf = F;
                    fa.wait_in = 1; fa.par_done = (fz - 1) & 1;
                    fa.arrive_out = 1;
                    linear_core_smem<T, L, NT, true>(tabH2 + (size_t)((a.fq0 + q) & a.tab_cycle_mask) * N, tid, fa);
                } else {
                    linear_core_smem<T, L, NT>(tabH2 + (size_t)((a.fq0 + q) & a.tab_cycle_mask) * N, tid);
                }
                const cplx<T>* p = ph + 4 * (zs + q) + 2;
                if (q + 1 < nsteps) run_fused(ldg(p), ldg(p + 1), ldg(p + 2), ldg(p + 3), ldg(p + 4), 2, hh, (T)1, (T)1);
                else run_fused(ldg(p), ldg(p + 1), ldg(p + 2), ldg(p + 2), ldg(p + 2), 1, hh, (T)1, (T)0.25);
            }
            if constexpr (FLOW) flow_wait_done_all((fz - 1) & 1);     // the last half-step has landed in my field
        } else {
        // q counts linear operators: q = 0 first half-step, q = total last half-step, between them the
        // merged full steps; in round-trip mode q = m nz + s and s = 0 (m > 0) crosses the boundary
#pragma unroll 1
        for (int q = 0; q <= total; ++q) {
            const int s = rt_mode ? q % nz : a.z0 + q;          // index of the RK4 step that follows
            const bool crossing = rt_mode && q > 0 && q < total && s == 0;
            const bool keep = rt_mode && q == 0 && !resonant && steps_l > 1;   // SH <- first half-stepped input
            const bool inj = crossing && inj_any;                               // input coupler of a resonant pump
            if (crossing && !resonant) {
                if constexpr (FLOW) { flow_wait_done_all((fz - 1) & 1); __syncthreads(); }
                load(SH);                                        // fresh pump / frozen seed, already half-stepped
                if constexpr (FLOW) { __syncthreads(); flow_arrive_ready_all(); }
            } else if (crossing && a.eom[x] != nullptr) {
                // resonant field with an intracavity modulator: the modulator acts in the time domain
                // between the boundary's spectral factor and the next pass, so the crossing is
                //   core(H G m) -> inverse pass 0 -> x E[n] -> forward pass 0 -> core(H)
                const cplx<T>* tabHG = reinterpret_cast<const cplx<T>*>(a.tabHG[x]) + (size_t)b * a.tab_stride[x];
                const cplx<T>* __restrict__ E = reinterpret_cast<const cplx<T>*>(a.eom[x]);
                if constexpr (FLOW) {
                    FlowArgs fa;
                    fa.mb = mb; fa.nf = F;
                    fa.wait_in = 1; fa.par_done = (fz - 1) & 1;
                    fa.arrive_out = 0;
                    linear_core_smem<T, L, NT, true>(tabHG, tid, fa);
                } else {
                    linear_core_smem<T, L, NT>(tabHG, tid);
                }
                __syncthreads();
                pass0_local<T, L, NT>(tw, tid, true);
                __syncthreads();
#pragma unroll 4
                for (int i = tid; i < N; i += NT) sm[phys<T>(i)] = cmul(sm[phys<T>(i)], ldg(&E[i]));
                __syncthreads();
                pass0_local<T, L, NT>(tw, tid, false);
                __syncthreads();
                if constexpr (FLOW) {
                    FlowArgs fa;
                    fa.mb = mb; fa.nf = F;
                    fa.wait_in = 0; fa.par_done = 0;
                    fa.arrive_out = !inj;
                    linear_core_smem<T, L, NT, true>(tabH, tid, fa);
                } else {
                    linear_core_smem<T, L, NT>(tabH, tid);
                }
            } else {
                const cplx<T>* tab = (q == 0 || q == total) ? tabH + (size_t)((hq_base + (q == 0 ? 0 : 1)) & a.tab_cycle_mask) * N
                                                            : (crossing ? tabHB : tabH2 + (size_t)(fq & a.tab_cycle_mask) * N);
                if constexpr (FLOW) {
                    FlowArgs fa;
                    fa.mb = mb; fa.nf = F;
                    fa.wait_in = q > 0; fa.par_done = (fz - 1) & 1;
                    fa.arrive_out = (q < total) && !keep && !inj;
                    linear_core_smem<T, L, NT, true>(tab, tid, fa);
                } else {
                    linear_core_smem<T, L, NT>(tab, tid);
                }
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
                if constexpr (FLOW) { __syncthreads(); flow_arrive_ready_all(); }   // only now may the peers write into my field
            }
            if (q == total) break;
            if (q > 0 && !crossing) ++fq;
            if constexpr (!FLOW) cluster_arrive();   // my field is ready for its inverse pass 0
            const cplx<T> e0 = ldg(ph + 2 * s), e1 = ldg(ph + 2 * s + 1), e2 = ldg(ph + 2 * s + 2);
            if constexpr (!FLOW) cluster_wait();     // ... and so is every other field
            if (x == 0) fused_pass0_rk4<T, L, F, NT, 0, false, DK0>(fld, tid, tw, tw0s, e0, e1, e2, e2, e2, 1, (T)1, (T)1, kap, h, mb, fz & 1);
            else if (F == 2 || x == 1) fused_pass0_rk4<T, L, F, NT, 1, false, DK0>(fld, tid, tw, tw0s, e0, e1, e2, e2, e2, 1, (T)1, (T)1, kap, h, mb, fz & 1);
            else fused_pass0_rk4<T, L, F, NT, F - 1, false, DK0>(fld, tid, tw, tw0s, e0, e1, e2, e2, e2, 1, (T)1, (T)1, kap, h, mb, fz & 1);
            ++fz;
            if constexpr (!FLOW) {
                cluster_arrive();
                cluster_wait();     // every result has landed in its owner's shared memory
            }
        }
        }   // L/2 - N - L/2
        __syncthreads();
        pass0_local<T, L, NT>(tw, tid, true);
        __syncthreads();

        if (!rt_mode) {
            store(cur);
        } else {
            store(reinterpret_cast<cplx<T>*>(a.exitb[x]) + (size_t)b * N);     // fields at z = L of the last pass
            if (resonant) {
                // intracavity phase modulator, last element of the boundary (Listing 3)
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
                if (inj_any) {     // input coupler (reading R24)
                    const cplx<T>* __restrict__ Sp = reinterpret_cast<const cplx<T>*>(a.S[x]) + (size_t)b * N;
#pragma unroll 4
                    for (int i = tid; i < N; i += NT) { const cplx<T> v = cur[i], sv = Sp[i]; cur[i] = {v.re + tinj * sv.re, v.im + tinj * sv.im}; }
                }
            } else {
                const cplx<T>* __restrict__ S = reinterpret_cast<const cplx<T>*>(a.S[x]) + (size_t)b * N;
#pragma unroll 4
                for (int i = tid; i < N; i += NT) cur[i] = S[i];
            }
        }
        // nobody reloads its shared memory for the next instance while it still stores from it; all
        // foreign accesses of this instance ended at the last cluster barrier
        __syncthreads();
        if (a.split) {
            if (rt0 + steps_l < a.steps && tid == 0) {      // hand the instance over: my field's state is in `cur`
                __threadfence();
                asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(flag), "r"(rt0 + steps_l) : "memory");
            }
        } else {
            b += n_clusters;
        }
    }
    cluster.sync();     // keep shared memory alive until every peer has left its last fused phase
}

template <class T, int L, int F> cudaError_t resident_cfg(cudaLaunchConfig_t* cfg, cudaLaunchAttribute* attr, int n_clusters, cudaStream_t s) {
    constexpr int NT = cta_threads<T, L>::value;
    const size_t smem = res_layout<T, L, F>::total;
    static device_once once;
    cudaError_t e0 = once.run([&] { return cudaFuncSetAttribute(k_resident<T, L, F, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); });
    if (e0 != cudaSuccess) return e0;
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = F;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg->gridDim = dim3((unsigned)(n_clusters * F), 1, 1);
    cfg->blockDim = dim3(NT, 1, 1);
    cfg->dynamicSmemBytes = smem;
    cfg->stream = s;
    cfg->attrs = attr;
    cfg->numAttrs = 1;
    return cudaSuccess;
}

template <class T, int L, int F> cudaError_t resident_info_LF(ResidentInfo* out) {
    cudaLaunchConfig_t cfg{};
    cudaLaunchAttribute attr[2];
    cudaError_t e = resident_cfg<T, L, F>(&cfg, attr, 1, nullptr);
    if (e != cudaSuccess) return e;
    int n = 0;
    e = cudaOccupancyMaxActiveClusters(&n, k_resident<T, L, F>, &cfg);
    if (e != cudaSuccess) return e;
    out->threads = cta_threads<T, L>::value;
    out->smem_bytes = cfg.dynamicSmemBytes;
    out->max_clusters = n;
    return cudaSuccess;
}

template <class T, int L> cudaError_t resident_info_L(int n_fields, ResidentInfo* out) {
    return n_fields == 3 ? resident_info_LF<T, L, 3>(out) : resident_info_LF<T, L, 2>(out);
}

// NLN = true and DK0 = true are instantiated in their own objects (opo_inst.cu with -DOPO_NLN / -DOPO_DK0): the default
// kernel's object code stays byte for byte what it is without the N/2 - L - N/2 ordering.
// With a.split the launch is cooperative: the round-trip split schedule spins on a flag another cluster sets, which is
// safe only if every cluster of the grid is resident; a cooperative launch fails (cudaErrorCooperativeLaunchTooLarge)
// instead of hanging when that cannot be guaranteed, and the host then launches without the split.
template <class T, int L, int F, bool NLN, bool DK0 = false> cudaError_t launch_resident_LF(const ResidentArgs& a, int n_clusters, cudaStream_t s) {
    cudaLaunchConfig_t cfg{};
    cudaLaunchAttribute attr[2];
    cudaError_t e = resident_cfg<T, L, F>(&cfg, attr, n_clusters, s);
    if (e != cudaSuccess) return e;
    if constexpr (NLN || DK0) {
        static device_once once;
        e = once.run([&] { return cudaFuncSetAttribute(k_resident<T, L, F, NLN, DK0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.dynamicSmemBytes); });
        if (e != cudaSuccess) return e;
    }
    if (a.split) {
        attr[1].id = cudaLaunchAttributeCooperative;
        attr[1].val.cooperative = 1;
        cfg.numAttrs = 2;
    }
    return cudaLaunchKernelEx(&cfg, k_resident<T, L, F, NLN, DK0>, a);
}

template <class T, int L, bool NLN, bool DK0 = false> cudaError_t launch_resident_L(const ResidentArgs& a, int n_clusters, cudaStream_t s) {
    return a.n_fields == 3 ? launch_resident_LF<T, L, 3, NLN, DK0>(a, n_clusters, s) : launch_resident_LF<T, L, 2, NLN, DK0>(a, n_clusters, s);
}

}  // namespace opo
