// opo_selftest.cu -- device peaks measured on the box, the roofline denominators bench.py reports against
// ("nominal peaks to be measured by a micro-benchmark on the box").  Not on the hot path.
//
//   OPO_PEAK_FP32_FMA   : independent FFMA chains on every SM (8 per thread, 512 threads x 2 CTAs per SM)   -> TFLOP/s
//   OPO_PEAK_FP64_FMA   : the same with DFMA                                                               -> TFLOP/s
//   OPO_PEAK_SMEM       : conflict-free 16-byte shared-memory loads + stores, every SM                     -> GB/s
//   OPO_PEAK_TMEM_LD/ST : tcgen05.ld / tcgen05.st 32x32b.x8 of a thread's own columns, every SM            -> GB/s
//   OPO_PEAK_DSMEM      : 16-byte stores into the shared memory of the next CTA of a cluster of 4, on as many clusters as
//                         are co-resident: bytes SENT per SM (every SM receives as much at the same time)   -> GB/s per SM
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cuda_runtime.h>

#include "../../include/opo.h"

namespace {

template <class T>
__global__ void __launch_bounds__(512, 2) k_peak_fma(int iters, T* sink) {
    T a[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) a[j] = (T)(threadIdx.x + j) * (T)1e-3;
    const T m = (T)0.999, c = (T)1e-4;
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 16; ++r)
#pragma unroll
            for (int j = 0; j < 8; ++j) a[j] = a[j] * m + c;       // one FMA each, 8 independent chains
    }
    T s = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) s += a[j];
    if (s == (T)123456.789) sink[0] = s;
}

__global__ void __launch_bounds__(512, 1) k_peak_smem(int iters, float* sink) {
    extern __shared__ float4 sm4[];
    const int tid = threadIdx.x;
    for (int i = tid; i < 4096; i += 512) sm4[i] = make_float4((float)i, 1.f, 2.f, 3.f);
    __syncthreads();
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(sm4) + 16u * tid;
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            float4 v;                                             // consecutive threads, consecutive 16 B: conflict-free
            asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(base + 8192u * r) : "memory");
            acc.x += v.x; acc.y += v.y;
            asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(base + 8192u * ((r + 1) & 7)), "f"(acc.x), "f"(acc.y), "f"(acc.z), "f"(acc.w) : "memory");
        }
    }
    if (acc.x == 123456.789f) sink[0] = acc.x + acc.y;
}

__global__ void __launch_bounds__(512, 1) k_peak_tmem(int iters, int store, float* sink) {
    __shared__ uint32_t base_s;
    const int warp = threadIdx.x >> 5;
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"((uint32_t)__cvta_generic_to_shared(&base_s)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t my = base_s + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)(128 * (warp >> 2));
    uint32_t v[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = threadIdx.x + j;
    for (int g = 0; g < 16; ++g)
        asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(my + 8 * g), "r"(v[0]), "r"(v[1]), "r"(v[2]),
                     "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]) : "memory");
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    uint32_t acc = 0;
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int g = 0; g < 16; ++g) {
            if (store) {
                v[0] = it + g;
                asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(my + 8 * g), "r"(v[0]), "r"(v[1]),
                             "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]) : "memory");
            } else {
                asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];" : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]),
                             "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]) : "r"(my + 8 * g) : "memory");
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                acc += v[g & 7];
            }
        }
        if (store) asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    }
    if (acc == 0xdeadbeefu) sink[0] = (float)acc;
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(base_s) : "memory");
}

// every CTA of a cluster streams into the shared memory of its successor (the traffic pattern of the wide engine's pushes,
// opo_wide.cuh: every SM sends and receives at once)
__global__ void __cluster_dims__(4, 1, 1) __launch_bounds__(512, 1) k_peak_dsmem(int iters, float* sink) {
    extern __shared__ float4 sm4[];
    const int tid = threadIdx.x;
    uint32_t rank;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
    for (int i = tid; i < 4096; i += 512) sm4[i] = make_float4((float)i, 1.f, 2.f, 3.f);
    const uint32_t local = (uint32_t)__cvta_generic_to_shared(sm4) + 16u * tid;
    uint32_t remote;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(local), "r"((rank + 1u) & 3u));
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");   // every peer is resident
    float4 v = make_float4((float)tid, 1.f, 2.f, 3.f);
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
            asm volatile("st.shared::cluster.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(remote + 8192u * r), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
        v.x += 1.f;
    }
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");   // nobody exits while a peer still writes into it
    if (sm4[tid].x == 123456.789f) sink[0] = sm4[tid].y;
}

template <class F> int timed(F&& launch, double* ms_out) {
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return OPO_ERR_CUDA;
    launch();                                   // warm-up (clocks, instruction cache)
    float best = 1e30f;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(e0, 0);
        launch();
        cudaEventRecord(e1, 0);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); cudaGetLastError(); return OPO_ERR_CUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *ms_out = best;
    return OPO_OK;
}

}  // namespace

extern "C" int opo_selftest_peak(int what, double* out_value) {
    if (!out_value) return OPO_ERR_INVALID_ARG;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return OPO_ERR_CUDA;
    float* sink = nullptr;
    if (cudaMalloc(&sink, 64) != cudaSuccess) return OPO_ERR_ALLOC;
    double ms = 0.0;
    int rc = OPO_OK;
    if (what == OPO_PEAK_FP32_FMA || what == OPO_PEAK_FP64_FMA) {
        const bool dbl = what == OPO_PEAK_FP64_FMA;
        const int iters = dbl ? 2000 : 20000, grid = 2 * sms;
        rc = timed([&] { if (dbl) k_peak_fma<double><<<grid, 512>>>(iters, (double*)sink); else k_peak_fma<float><<<grid, 512>>>(iters, sink); }, &ms);
        const double flops = 2.0 * 128.0 * (double)iters * 512.0 * (double)grid;       // 16 x 8 FMAs per thread and iteration
        *out_value = flops / (ms * 1e-3) / 1e12;
    } else if (what == OPO_PEAK_SMEM) {
        const int iters = 20000;
        if (cudaFuncSetAttribute(k_peak_smem, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536) != cudaSuccess) { cudaFree(sink); cudaGetLastError(); return OPO_ERR_CUDA; }
        rc = timed([&] { k_peak_smem<<<sms, 512, 65536>>>(iters, sink); }, &ms);
        const double bytes = 2.0 * 8.0 * 16.0 * 512.0 * (double)iters * (double)sms;   // 8 loads + 8 stores of 16 B per thread and iteration
        *out_value = bytes / (ms * 1e-3) / 1e9;
    } else if (what == OPO_PEAK_TMEM_LD || what == OPO_PEAK_TMEM_ST) {
        const int iters = 20000;
        const int store = what == OPO_PEAK_TMEM_ST;
        rc = timed([&] { k_peak_tmem<<<sms, 512>>>(iters, store, sink); }, &ms);
        const double bytes = 16.0 * 32.0 * 512.0 * (double)iters * (double)sms;        // 16 x (8 columns x 4 B) per thread and iteration
        *out_value = bytes / (ms * 1e-3) / 1e9;
    } else if (what == OPO_PEAK_DSMEM) {
        const int iters = 20000;
        constexpr int kSmem = 120 * 1024;       // more than half of an SM's shared memory: one CTA per SM, so "per CTA" is "per SM"
        if (cudaFuncSetAttribute(k_peak_dsmem, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmem) != cudaSuccess) { cudaFree(sink); cudaGetLastError(); return OPO_ERR_CUDA; }
        // as many clusters as run at once: a second wave would be timed as if it were part of the first
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(4 * (unsigned)sms, 1, 1);
        cfg.blockDim = dim3(512, 1, 1);
        cfg.dynamicSmemBytes = kSmem;
        int clusters = 0;
        if (cudaOccupancyMaxActiveClusters(&clusters, k_peak_dsmem, &cfg) != cudaSuccess || clusters <= 0) { cudaFree(sink); cudaGetLastError(); return OPO_ERR_CUDA; }
        if (4 * clusters > sms) clusters = sms / 4;
        rc = timed([&] { k_peak_dsmem<<<4 * clusters, 512, kSmem>>>(iters, sink); }, &ms);
        if (getenv("OPO_SELFTEST_VERBOSE")) fprintf(stderr, "k_peak_dsmem: %d clusters of 4 on %d SMs, %.3f ms\n", clusters, sms, ms);
        const double bytes_per_sm = 8.0 * 16.0 * 512.0 * (double)iters;                 // 8 stores of 16 B per thread and iteration
        *out_value = bytes_per_sm / (ms * 1e-3) / 1e9;
    } else {
        rc = OPO_ERR_INVALID_ARG;
    }
    cudaFree(sink);
    if (rc == OPO_OK && cudaGetLastError() != cudaSuccess) rc = OPO_ERR_CUDA;
    return rc;
}
