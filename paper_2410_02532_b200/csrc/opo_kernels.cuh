// opo_kernels.cuh -- streaming-engine kernels (fields in HBM/L2) and the shared RK4 device code.
//
//   k_linear : one CTA per (field, instance): global -> smem, FFT . table . IFFT, smem -> global
//              (Eq. 11, linear part; steps S1-S3/S5 of SURVEY.md section 8(a)).
//   k_rk4    : pointwise classic RK4 of the coupling terms of Eqs 2-4 (S4).
//   k_scale  : mirror factor sqrt(R) e^{i delta} (Eq. 6; S6 without GDD).
//   k_freq   : forward DFT into natural order for opo_get_fields(FREQ).
#pragma once
#include "opo_fft.cuh"
#include "opo_internal.h"

namespace opo {

// ---- RK4 of the nonlinear operator at one grid point ---------------------------------------------------
// e0, e1, e2 = exp(i dk z) at z, z + h/2, z + h.  kap[x] real couplings.  Readings R3, R4, R5.
template <class T, int F> struct Rk4 {
    // g = N(y) / (i kappa) at phase e: the complex products of Eqs 2-4 without the factor i kappa_x,
    // which step() folds into its update constants (y + c i kappa g costs one FMA per component)
    // DK0: dk = 0 for every instance of the launch, all stage phases are exactly 1 and their products are skipped
    template <bool DK0 = false>
    static __device__ __forceinline__ void rhs(const cplx<T>* y, cplx<T> e, cplx<T>* g) {
        if constexpr (DK0) {
            if constexpr (F == 3) {
                g[0] = cmul(y[1], y[2]);
                g[1] = cmulc(y[0], y[2]);
                g[2] = cmulc(y[0], y[1]);
            } else {
                g[0] = cmul(y[1], y[1]);
                g[1] = cmulc(y[0], y[1]);
            }
        } else if constexpr (F == 3) {
            // dA_p = i k_p A_s A_i e^{-i dk z}
            g[0] = cmulc(cmul(y[1], y[2]), e);
            // dA_s = i k_s A_p A_i^* e^{+i dk z},  dA_i = i k_i A_p A_s^* e^{+i dk z}
            const cplx<T> pe = cmul(y[0], e);
            g[1] = cmulc(pe, y[2]);
            g[2] = cmulc(pe, y[1]);
        } else {
            // dA_p = i (k_p/2) A_s^2 e^{-i dk z}   (kap[0] holds k_p/2),  dA_s = i k_s A_p A_s^* e^{+i dk z}
            g[0] = cmulc(cmul(y[1], y[1]), e);
            g[1] = cmulc(cmul(y[0], e), y[1]);
        }
    }
    // a + c * (i g)
    static __device__ __forceinline__ cplx<T> axpy_i(cplx<T> a, T c, cplx<T> g) { return {a.re - c * g.im, a.im + c * g.re}; }
    template <bool DK0 = false>
    static __device__ __forceinline__ void step(cplx<T>* y, cplx<T> e0, cplx<T> e1, cplx<T> e2, const T* kap, T h) {
        cplx<T> g[F], t[F], acc[F];
        T c2[F], c3[F], c6[F], c1[F];
#pragma unroll
        for (int x = 0; x < F; ++x) {
            c1[x] = h * kap[x];
            c2[x] = (T)0.5 * c1[x];
            c3[x] = c1[x] / (T)3;
            c6[x] = c1[x] / (T)6;
        }
        rhs<DK0>(y, e0, g);
#pragma unroll
        for (int x = 0; x < F; ++x) { acc[x] = axpy_i(y[x], c6[x], g[x]); t[x] = axpy_i(y[x], c2[x], g[x]); }
        rhs<DK0>(t, e1, g);
#pragma unroll
        for (int x = 0; x < F; ++x) { acc[x] = axpy_i(acc[x], c3[x], g[x]); t[x] = axpy_i(y[x], c2[x], g[x]); }
        rhs<DK0>(t, e1, g);
#pragma unroll
        for (int x = 0; x < F; ++x) { acc[x] = axpy_i(acc[x], c3[x], g[x]); t[x] = axpy_i(y[x], c1[x], g[x]); }
        rhs<DK0>(t, e2, g);
#pragma unroll
        for (int x = 0; x < F; ++x) y[x] = axpy_i(acc[x], c6[x], g[x]);
    }
};

// ---- k_linear ---------------------------------------------------------------------------------------------
template <class T, int L>
__global__ void __launch_bounds__(cta_threads<T, L>::value) k_linear(LinArgs a) {
    constexpr int N = 1 << L, NT = cta_threads<T, L>::value;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
    const int slot = blockIdx.x % a.n_slots, b = blockIdx.x / a.n_slots;
    const LinSlot& sl = a.slot[slot];
    const cplx<T>* __restrict__ src = reinterpret_cast<const cplx<T>*>(sl.src) + (size_t)b * N;
    cplx<T>* __restrict__ dst = reinterpret_cast<cplx<T>*>(sl.dst) + (size_t)b * N;
    const cplx<T>* tab = reinterpret_cast<const cplx<T>*>(sl.tab) + (size_t)b * sl.tab_stride;
    const cplx<T>* tw = reinterpret_cast<const cplx<T>*>(a.tw);
    const int tid = threadIdx.x;
#pragma unroll 4
    for (int i = tid; i < N; i += NT) sm[phys<T>(i)] = src[i];
    __syncthreads();
    linear_op_smem<T, L, NT>(sm, tw, tab, tid);
    __syncthreads();
    if (sl.dst2 != nullptr) {
        cplx<T>* __restrict__ d2 = reinterpret_cast<cplx<T>*>(sl.dst2) + (size_t)b * N;
#pragma unroll 4
        for (int i = tid; i < N; i += NT) { cplx<T> v = sm[phys<T>(i)]; dst[i] = v; d2[i] = v; }
    } else {
#pragma unroll 4
        for (int i = tid; i < N; i += NT) dst[i] = sm[phys<T>(i)];
    }
}

// ---- k_rk4 -------------------------------------------------------------------------------------------------
template <class T, int F>
__global__ void __launch_bounds__(256) k_rk4(Rk4Args a) {
    const int n = a.n;
    const long long total = (long long)a.batch * n;
    T kap[3] = {(T)a.kappa[0], (T)a.kappa[1], (T)a.kappa[2]};
    const T h = (T)a.h;
    const cplx<T>* ph = reinterpret_cast<const cplx<T>*>(a.phase);
    cplx<T>* A[F];
#pragma unroll
    for (int x = 0; x < F; ++x) A[x] = reinterpret_cast<cplx<T>*>(a.A[x]);
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const int b = (int)(i / n);
        const cplx<T>* p = ph + (size_t)b * a.phase_stride + (a.phase_index >= 0 ? a.phase_index : 2 * a.step);
        const cplx<T> e0 = ldg(p), e1 = ldg(p + 1), e2 = ldg(p + 2);
        cplx<T> y[F];
#pragma unroll
        for (int x = 0; x < F; ++x) y[x] = A[x][i];
        Rk4<T, F>::step(y, e0, e1, e2, kap, h);
#pragma unroll
        for (int x = 0; x < F; ++x) A[x][i] = y[x];
    }
}

template <class T>
__global__ void __launch_bounds__(256) k_scale(ScaleArgs a) {
    const long long total = (long long)a.batch * a.n;
    cplx<T>* A = reinterpret_cast<cplx<T>*>(a.A);
    const cplx<T>* m = reinterpret_cast<const cplx<T>*>(a.m);
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const int b = (int)(i / a.n);
        A[i] = cmul(A[i], ldg(&m[b]));
    }
}

// intracavity phase modulator: A[b][n] *= E[n]
template <class T>
__global__ void __launch_bounds__(256) k_multab(MulTabArgs a) {
    const long long total = (long long)a.batch * a.n;
    cplx<T>* A = reinterpret_cast<cplx<T>*>(a.A);
    const cplx<T>* E = reinterpret_cast<const cplx<T>*>(a.E);
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x)
        A[i] = cmul(A[i], ldg(&E[(i / a.n) * a.tab_stride + (i % a.n)]));
}

template <class T, int L>
__global__ void __launch_bounds__(cta_threads<T, L>::value) k_freq(FreqArgs a) {
    constexpr int N = 1 << L, NT = cta_threads<T, L>::value;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
    const int b = blockIdx.x, tid = threadIdx.x;
    const cplx<T>* __restrict__ src = reinterpret_cast<const cplx<T>*>(a.src) + (size_t)b * N;
    cplx<T>* __restrict__ dst = reinterpret_cast<cplx<T>*>(a.dst) + (size_t)b * N;
    for (int i = tid; i < N; i += NT) sm[phys<T>(i)] = src[i];
    __syncthreads();
    forward_only_smem<T, L, NT>(sm, reinterpret_cast<const cplx<T>*>(a.tw), tid);
    __syncthreads();
    for (int i = tid; i < N; i += NT) dst[__ldg(&a.perm[i])] = sm[phys<T>(i)];
}

// dst[b][i] = dst[0][i], b = 1 .. batch-1 (one input broadcast to every instance: opo_set_pump with per_instance = 0)
template <class T>
__global__ void __launch_bounds__(256) k_broadcast(cplx<T>* dst, int batch, int n) {
    const long long total = (long long)(batch - 1) * n;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x)
        dst[n + i] = dst[i % n];
}

// A[i] = (accumulate ? A[i] : 0) + c S[i]   (input coupler of a resonant pump, reading R24 of DESIGN.md)
template <class T>
__global__ void __launch_bounds__(256) k_axpy(cplx<T>* A, const cplx<T>* __restrict__ S, T c, int accumulate, long long count) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (long long)gridDim.x * blockDim.x) {
        const cplx<T> s = S[i];
        cplx<T> a = accumulate ? A[i] : cplx<T>{(T)0, (T)0};
        A[i] = {a.re + c * s.re, a.im + c * s.im};
    }
}

template <class T>
__global__ void __launch_bounds__(256) k_finite(const T* A, long long count, int* flag) {
    int bad = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (long long)gridDim.x * blockDim.x) {
        T v = A[i];
        if (!(v - v == (T)0)) bad = 1;   // NaN or Inf
    }
    if (bad) atomicExch(flag, 1);
}

// ---- launch helpers ------------------------------------------------------------------------------------------
template <class T, int L> cudaError_t launch_linear_L(const LinArgs& a, cudaStream_t s) {
    constexpr int NT = cta_threads<T, L>::value;
    const size_t smem = (size_t)padded_len<T>(1 << L) * sizeof(cplx<T>);
    static device_once once;
    cudaError_t e = once.run([&] { return cudaFuncSetAttribute(k_linear<T, L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); });
    if (e != cudaSuccess) return e;
    k_linear<T, L><<<a.n_slots * a.batch, NT, smem, s>>>(a);
    return cudaGetLastError();
}
template <class T, int L> cudaError_t launch_freq_L(const FreqArgs& a, cudaStream_t s) {
    constexpr int NT = cta_threads<T, L>::value;
    const size_t smem = (size_t)padded_len<T>(1 << L) * sizeof(cplx<T>);
    static device_once once;
    cudaError_t e = once.run([&] { return cudaFuncSetAttribute(k_freq<T, L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); });
    if (e != cudaSuccess) return e;
    k_freq<T, L><<<a.batch, NT, smem, s>>>(a);
    return cudaGetLastError();
}

// grid of a grid-stride pointwise kernel: enough CTAs for 16 per SM of the current device
inline int grid_for(long long total, int block) {
    static int sms[64] = {};
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64) dev = 0;
    if (sms[dev] == 0 && cudaDeviceGetAttribute(&sms[dev], cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) sms[dev] = 148;
    long long g = (total + block - 1) / block;
    const long long cap = (long long)sms[dev] * 16;
    return (int)(g < 1 ? 1 : (g > cap ? cap : g));
}

template <class T> cudaError_t launch_rk4_T(const Rk4Args& a, cudaStream_t s) {
    const int g = grid_for((long long)a.batch * a.n, 256);
    if (a.n_fields == 3) k_rk4<T, 3><<<g, 256, 0, s>>>(a);
    else k_rk4<T, 2><<<g, 256, 0, s>>>(a);
    return cudaGetLastError();
}
template <class T> cudaError_t launch_scale_T(const ScaleArgs& a, cudaStream_t s) {
    k_scale<T><<<grid_for((long long)a.batch * a.n, 256), 256, 0, s>>>(a);
    return cudaGetLastError();
}
template <class T> cudaError_t launch_multab_T(const MulTabArgs& a, cudaStream_t s) {
    k_multab<T><<<grid_for((long long)a.batch * a.n, 256), 256, 0, s>>>(a);
    return cudaGetLastError();
}
template <class T> cudaError_t launch_broadcast_T(void* dst, int batch, int n, cudaStream_t s) {
    if (batch <= 1) return cudaSuccess;
    k_broadcast<T><<<grid_for((long long)(batch - 1) * n, 256), 256, 0, s>>>(reinterpret_cast<cplx<T>*>(dst), batch, n);
    return cudaGetLastError();
}
template <class T> cudaError_t launch_axpy_T(void* A, const void* S, double c, int accumulate, long long count, cudaStream_t s) {
    k_axpy<T><<<grid_for(count, 256), 256, 0, s>>>(reinterpret_cast<cplx<T>*>(A), reinterpret_cast<const cplx<T>*>(S), (T)c, accumulate, count);
    return cudaGetLastError();
}
template <class T> cudaError_t launch_finite_T(const void* A, long long count, int* flag, cudaStream_t s) {
    k_finite<T><<<grid_for(count, 256), 256, 0, s>>>(reinterpret_cast<const T*>(A), count, flag);
    return cudaGetLastError();
}

}  // namespace opo
