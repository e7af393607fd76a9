// DSMEM bandwidth microbenchmark: cluster of 3, 512 threads, each CTA accesses rank+1's shared memory
#include <cooperative_groups.h>
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
namespace cg = cooperative_groups;
constexpr int NT = 512, BYTES = 128 * 1024;
__device__ __forceinline__ uint32_t mapa(uint32_t a, uint32_t r) { uint32_t o; asm volatile("mapa.shared::cluster.u32 %0,%1,%2;" : "=r"(o) : "r"(a), "r"(r)); return o; }

template <int MODE> __global__ void __cluster_dims__(3, 1, 1) __launch_bounds__(NT, 1) k(long long* out, int iters) {
    extern __shared__ __align__(128) unsigned char sm[];
    __shared__ uint64_t bar;
    cg::cluster_group c = cg::this_cluster();
    const uint32_t rank = c.block_rank(), peer = (rank + 1) % 3;
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(sm);
    const uint32_t rbase = mapa(base, peer);
    for (int i = threadIdx.x; i < BYTES / 4; i += NT) ((float*)sm)[i] = i;
    if (threadIdx.x == 0) { asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"((uint32_t)__cvta_generic_to_shared(&bar))); }
    c.sync();
    float acc = 0;
    long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
        if constexpr (MODE == 0) {          // remote read 8 B / lane
#pragma unroll 8
            for (int i = threadIdx.x; i < BYTES / 8; i += NT) { float a, b; asm volatile("ld.shared::cluster.v2.f32 {%0,%1}, [%2];" : "=f"(a), "=f"(b) : "r"(rbase + i * 8)); acc += a + b; }
        } else if constexpr (MODE == 1) {   // remote read 16 B / lane
#pragma unroll 8
            for (int i = threadIdx.x; i < BYTES / 16; i += NT) { float a, b, cc, d; asm volatile("ld.shared::cluster.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(a), "=f"(b), "=f"(cc), "=f"(d) : "r"(rbase + i * 16)); acc += a + b + cc + d; }
        } else if constexpr (MODE == 2) {   // remote write 8 B
#pragma unroll 8
            for (int i = threadIdx.x; i < BYTES / 8; i += NT) asm volatile("st.shared::cluster.v2.f32 [%0], {%1,%2};" ::"r"(rbase + i * 8), "f"(acc), "f"(1.f));
        } else if constexpr (MODE == 3) {   // remote write 16 B
#pragma unroll 8
            for (int i = threadIdx.x; i < BYTES / 16; i += NT) asm volatile("st.shared::cluster.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(rbase + i * 16), "f"(acc), "f"(1.f), "f"(2.f), "f"(3.f));
        } else if constexpr (MODE == 4) {   // read 8 B + write 8 B (half each)
#pragma unroll 8
            for (int i = threadIdx.x; i < BYTES / 16; i += NT) { float a, b; asm volatile("ld.shared::cluster.v2.f32 {%0,%1}, [%2];" : "=f"(a), "=f"(b) : "r"(rbase + i * 8)); acc += a + b;
                asm volatile("st.shared::cluster.v2.f32 [%0], {%1,%2};" ::"r"(rbase + BYTES / 2 + i * 8), "f"(1.f), "f"(2.f)); }
        } else if constexpr (MODE >= 5) {   // bulk push local -> remote, chunk = 272 B (5), 4 KB (6), 32 KB (7); completes on the REMOTE mbarrier
            constexpr int CH = MODE == 5 ? 272 : (MODE == 6 ? 4096 : 32768);
            constexpr int NCH = BYTES / CH;
            const uint32_t lbar = (uint32_t)__cvta_generic_to_shared(&bar), rbar = mapa(lbar, peer);
            if (threadIdx.x == 0) asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(lbar), "r"(NCH * CH) : "memory");
            c.sync();
            for (int ch = threadIdx.x; ch < NCH; ch += NT)
                asm volatile("cp.async.bulk.shared::cluster.shared::cta.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(rbase + ch * CH), "r"(base + ch * CH), "r"(CH), "r"(rbar) : "memory");
            uint32_t ok = 0;
            while (!ok) asm volatile("{ .reg .pred q; mbarrier.try_wait.parity.shared::cta.b64 q, [%1], %2; selp.u32 %0,1,0,q; }" : "=r"(ok) : "r"(lbar), "r"(it & 1) : "memory");
        }
    }
    long long t1 = clock64();
    c.sync();
    if (acc == 123.456f) out[100] = 1;
    if (threadIdx.x == 0) out[blockIdx.x] = t1 - t0;
}
template <int MODE> void run(const char* name, int grid, int iters, double bytes_per_iter) {
    long long* d; cudaMalloc(&d, 4096 * 8); cudaMemset(d, 0, 4096 * 8);
    cudaFuncSetAttribute(k<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, BYTES);
    k<MODE><<<grid, NT, BYTES>>>(d, iters);
    cudaError_t e = cudaDeviceSynchronize();
    long long h[512]; cudaMemcpy(h, d, grid * 8, cudaMemcpyDeviceToHost);
    double mx = 0, av = 0; for (int i = 0; i < grid; ++i) { av += h[i]; if (h[i] > mx) mx = h[i]; } av /= grid;
    printf("%-28s grid %3d: %s  avg %.1f B/clk/SM  (slowest CTA %.1f)\n", name, grid, cudaGetErrorString(e), bytes_per_iter * iters / av, bytes_per_iter * iters / mx);
    cudaFree(d);
}
int main() {
    for (int grid : {3, 135}) {
        run<0>("remote ld 8B", grid, 50, BYTES);
        run<1>("remote ld 16B", grid, 50, BYTES);
        run<2>("remote st 8B", grid, 50, BYTES);
        run<3>("remote st 16B", grid, 50, BYTES);
        run<4>("remote ld 8B + st 8B", grid, 50, BYTES);
        run<5>("bulk push 272 B", grid, 50, 272.0 * (BYTES / 272));
        run<6>("bulk push 4 KB", grid, 50, BYTES);
        run<7>("bulk push 32 KB", grid, 50, BYTES);
    }
    return 0;
}
