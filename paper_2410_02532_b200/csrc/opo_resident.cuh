// opo_resident.cuh -- resident engine: one thread-block cluster per OPO instance, CTA rank = field.
//
// Each CTA keeps its field in (padded) shared memory for the whole call -- every z-step of every
// round trip -- so HBM is touched only at the ends of the call and, per round trip, for the
// re-injected non-resonant inputs and the constant tables (L2-resident).
//
//   linear step  : CTA-local FFT . table . IFFT on its own field (opo_fft.cuh); adjacent half-steps
//                  are merged (H.H = H2) and, between round trips, merged across the cavity
//                  boundary (H . G m . H = HB), so a z-step costs one transform pair per field.
//   nonlinear    : RK4 needs all F fields at the same tau.  The grid points are dealt to the F
//                  CTAs in tiles of 32; a CTA reads the two foreign fields of its tiles through
//                  distributed shared memory, integrates, and writes all F results back.
//   two cluster barriers per z-step order the two phases.
//
// A cluster loops over instances b = cluster_id, cluster_id + n_clusters, ... (batched mode,
// BASELINE.json configs[4]); instances are independent, there is no inter-cluster communication.
#pragma once
#include <cooperative_groups.h>

#include "opo_kernels.cuh"

namespace opo {

namespace cg = cooperative_groups;

template <class T, int L, int F, int NT>
__device__ __forceinline__ void resident_rk4(cplx<T>* const* fld, int rank, int tid, cplx<T> e0, cplx<T> e1, cplx<T> e2,
                                             const T* kap, T h) {
    constexpr int N = 1 << L, NTILES = N / 32, NW = NT / 32;
    const int warp = tid >> 5, lane = tid & 31;
    // tiles tau = rank + F * j, j = warp, warp + NW, ...   two tiles in flight per iteration
    for (int j = warp; rank + F * j < NTILES; j += 2 * NW) {
        const int t0 = rank + F * j, t1 = rank + F * (j + NW);
        const bool has1 = t1 < NTILES;
        const int i0 = phys<T>(t0 * 32 + lane), i1 = phys<T>((has1 ? t1 : t0) * 32 + lane);
        cplx<T> y0[F], y1[F];
#pragma unroll
        for (int x = 0; x < F; ++x) { y0[x] = fld[x][i0]; y1[x] = fld[x][i1]; }
        Rk4<T, F>::step(y0, e0, e1, e2, kap, h);
        Rk4<T, F>::step(y1, e0, e1, e2, kap, h);
#pragma unroll
        for (int x = 0; x < F; ++x) {
            fld[x][i0] = y0[x];
            if (has1) fld[x][i1] = y1[x];
        }
    }
}

template <class T, int L, int F>
__global__ void __launch_bounds__(cta_threads<T, L>::value, 1) k_resident(ResidentArgs a) {
    constexpr int N = 1 << L, NT = cta_threads<T, L>::value;
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
    const cplx<T>* tabH = reinterpret_cast<const cplx<T>*>(a.tabH[x]);
    const cplx<T>* tabH2 = reinterpret_cast<const cplx<T>*>(a.tabH2[x]);
    const bool resonant = a.resonant[x] != 0;
    T kap[3] = {(T)a.kappa[0], (T)a.kappa[1], (T)a.kappa[2]};
    const T h = (T)a.h;

    for (int b = cid; b < a.batch; b += n_clusters) {
        cplx<T>* cur = reinterpret_cast<cplx<T>*>(a.cur[x]) + (size_t)b * N;
        const cplx<T>* ph = reinterpret_cast<const cplx<T>*>(a.phase) + (size_t)b * a.phase_stride;

        auto load = [&](const cplx<T>* __restrict__ g) {
#pragma unroll 4
            for (int i = tid; i < N; i += NT) sm[phys<T>(i)] = g[i];
        };
        auto store = [&](cplx<T>* __restrict__ g) {
#pragma unroll 4
            for (int i = tid; i < N; i += NT) g[i] = sm[phys<T>(i)];
        };
        auto nonlinear = [&](int s) {
            cluster.sync();     // every field has finished its linear step
            const cplx<T> e0 = ldg(ph + 2 * s), e1 = ldg(ph + 2 * s + 1), e2 = ldg(ph + 2 * s + 2);
            resident_rk4<T, L, F, NT>(fld, x, tid, e0, e1, e2, kap, h);
            cluster.sync();     // every RK4 result has landed in its owner's shared memory
        };

        load(cur);
        __syncthreads();

        if (a.mode == 0) {
            // `steps` z-steps from step index z0:  H, N, H2, N, ..., N, H
            linear_op_smem<T, L, NT>(sm, tw, tabH, tid);
            for (int s = 0; s < a.steps; ++s) {
                nonlinear(a.z0 + s);
                if (s + 1 < a.steps) linear_op_smem<T, L, NT>(sm, tw, tabH2, tid);
            }
            linear_op_smem<T, L, NT>(sm, tw, tabH, tid);
            __syncthreads();
            store(cur);
        } else {
            const cplx<T>* tabHB = reinterpret_cast<const cplx<T>*>(a.tabHB[x]) + (size_t)b * a.tab_stride[x];
            const cplx<T>* tabGM = reinterpret_cast<const cplx<T>*>(a.tabGM[x]) + (size_t)b * a.tab_stride[x];
            cplx<T>* SH = reinterpret_cast<cplx<T>*>(a.SH[x]) + (size_t)b * N;
            for (int m = 0; m < a.steps; ++m) {
                const bool first = (m == 0), last = (m == a.steps - 1);
                if (first) {
                    linear_op_smem<T, L, NT>(sm, tw, tabH, tid);
                    if (!resonant && a.steps > 1) {       // keep IDFT(H DFT(S_x)) for the later round trips
                        __syncthreads();
                        store(SH);
                    }
                } else if (resonant) {
                    linear_op_smem<T, L, NT>(sm, tw, tabHB, tid);   // H . G m . H across the boundary
                } else {
                    load(SH);                                        // fresh pump / frozen seed, already half-stepped
                }
                for (int s = 0; s < a.nz; ++s) {
                    nonlinear(s);
                    if (s + 1 < a.nz) linear_op_smem<T, L, NT>(sm, tw, tabH2, tid);
                }
                if (last) {
                    linear_op_smem<T, L, NT>(sm, tw, tabH, tid);
                    __syncthreads();
                    store(reinterpret_cast<cplx<T>*>(a.exitb[x]) + (size_t)b * N);     // fields at z = L
                    if (resonant) {
                        if (a.boundary_fft[x]) {
                            linear_op_smem<T, L, NT>(sm, tw, tabGM, tid);
                            __syncthreads();
                            store(cur);
                        } else {
                            const cplx<T> mf = ldg(reinterpret_cast<const cplx<T>*>(a.mirror[x]) + b);
#pragma unroll 4
                            for (int i = tid; i < N; i += NT) cur[i] = cmul(sm[phys<T>(i)], mf);
                        }
                    } else {
                        const cplx<T>* __restrict__ S = reinterpret_cast<const cplx<T>*>(a.S[x]) + (size_t)b * N;
#pragma unroll 4
                        for (int i = tid; i < N; i += NT) cur[i] = S[i];
                    }
                }
            }
        }
        // all foreign reads/writes of this instance are fenced by the last nonlinear(); make sure
        // nobody reloads its shared memory for the next instance while a peer still stores from it
        __syncthreads();
    }
    cluster.sync();     // keep shared memory alive until every peer has left its last RK4
}

template <class T, int L, int F> cudaError_t resident_cfg(cudaLaunchConfig_t* cfg, cudaLaunchAttribute* attr, int n_clusters, cudaStream_t s) {
    constexpr int NT = cta_threads<T, L>::value;
    const size_t smem = (size_t)padded_len<T>(1 << L) * sizeof(cplx<T>);
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(k_resident<T, L, F>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured = true;
    }
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
    cudaLaunchAttribute attr[1];
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

template <class T, int L, int F> cudaError_t launch_resident_LF(const ResidentArgs& a, int n_clusters, cudaStream_t s) {
    cudaLaunchConfig_t cfg{};
    cudaLaunchAttribute attr[1];
    cudaError_t e = resident_cfg<T, L, F>(&cfg, attr, n_clusters, s);
    if (e != cudaSuccess) return e;
    return cudaLaunchKernelEx(&cfg, k_resident<T, L, F>, a);
}

template <class T, int L> cudaError_t launch_resident_L(const ResidentArgs& a, int n_clusters, cudaStream_t s) {
    return a.n_fields == 3 ? launch_resident_LF<T, L, 3>(a, n_clusters, s) : launch_resident_LF<T, L, 2>(a, n_clusters, s);
}

}  // namespace opo
