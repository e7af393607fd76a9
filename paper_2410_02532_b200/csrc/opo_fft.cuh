// opo_fft.cuh -- in-place shared-memory complex FFT building blocks for sm_100a.
//
// The linear half-step of the split-step method (Eq. 11) is
//     A <- IDFT( H .* DFT(A) ).
// This file provides it as ONE pass structure over a field held in shared memory:
//
//   forward  : decimation-in-frequency passes p = 0..P-1 (radix R_p, N = R_0 ... R_{P-1}); natural
//              order in, digit-reversed order out, so no reordering pass is ever executed;
//   multiply : in registers, against a table that the host stored in the digit-reversed order;
//   inverse  : the exact adjoint factorisation (decimation-in-time, passes P-1..0, conjugate
//              twiddles), digit-reversed in, natural order out.
//
// Pass 0 has radix 4 and is special: its butterflies touch x[t + j N/4], j = 0..3, and nothing else,
// in both directions.  The resident engine (opo_resident.cuh) therefore runs "inverse pass 0 -> RK4
// on those four grid points -> forward pass 0" on registers, for all coupled fields at once -- the
// nonlinear step costs no shared-memory pass of its own.  Passes 1..P-2 are radix-16 (8/4 for the
// remainder) shared-memory passes; the last forward pass, the table multiply and the first inverse
// pass ("mid") also run on registers without touching shared memory in between.
//
// Because the inverse is the adjoint of the forward factorisation using the *same* rounded
// twiddles, twiddle phase rounding cancels between the two transforms and does not accumulate
// over thousands of z-steps; only twiddle magnitude rounding can, and the host picks table
// roundings that minimise | |w| - 1 | ("fp32 error budget").
//
// Shared-memory layout: element i lives at i + (i >> PADSH) (one pad element per 16 float2 / per
// 8 double2, i.e. per 128 bytes), which makes every pass -- including the unit-stride last one --
// bank-conflict free.  All element addresses of a butterfly are one runtime base plus
// compile-time offsets (elem_addr below).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <utility>

namespace opo {

template <class T>
struct alignas(2 * sizeof(T)) cplx {
    T re, im;
};

template <class T> __device__ __forceinline__ cplx<T> operator+(cplx<T> a, cplx<T> b) { return {a.re + b.re, a.im + b.im}; }
template <class T> __device__ __forceinline__ cplx<T> operator-(cplx<T> a, cplx<T> b) { return {a.re - b.re, a.im - b.im}; }
// fp32: complex add / subtract as ONE packed instruction (FADD2 on sm_100: two lanes of the FP32 pipe for two
// cycles, but a single issue slot -- the kernels are issue-bound, the FP32 pipe is ~55 % busy)
__device__ __forceinline__ unsigned long long pack2(cplx<float> a) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a.re), "f"(a.im));
    return r;
}
__device__ __forceinline__ cplx<float> unpack2(unsigned long long v) {
    cplx<float> r;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(r.re), "=f"(r.im) : "l"(v));
    return r;
}
template <> __device__ __forceinline__ cplx<float> operator+(cplx<float> a, cplx<float> b) {
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pack2(a)), "l"(pack2(b)));
    return unpack2(r);
}
template <> __device__ __forceinline__ cplx<float> operator-(cplx<float> a, cplx<float> b) {
    unsigned long long r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pack2(a)), "l"(pack2(b)));
    return unpack2(r);
}
// a * b
template <class T> __device__ __forceinline__ cplx<T> cmul(cplx<T> a, cplx<T> b) {
    return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re};
}
// a * conj(b)
template <class T> __device__ __forceinline__ cplx<T> cmulc(cplx<T> a, cplx<T> b) {
    return {a.re * b.re + a.im * b.im, a.im * b.re - a.re * b.im};
}

// a * conj(b) / |b|^2 to first order, for a rounded unit-modulus b.  A forward pass multiplies by the rounded twiddle w and
// the inverse pass by conj(w), so the pair scales its butterfly leg by |w|^2 = 1 + d, d ~ 3e-8 rms in fp32 -- the same d at
// every z-step.  Twiddle *phase* rounding is a similarity transform of the step and does not accumulate; this magnitude
// defect does, linearly in the number of z-steps, while the data rounding errors add up as a random walk (measured on
// IDFT(DFT(A)) alone: 3.5e-8 per z-step, 3.5e-4 after the 10^4 z-steps of C3 x 20 round trips; with the defect taken out
// the same loop grows as sqrt(n)).  No choice of float pair near the unit circle helps (for small angles the granularity
// of cos alone is 1.2e-7 in |w|^2).  d is evaluated without cancellation error -- the larger component has a^2 >= 1/2, so
// a^2 - 1 is exact, and an FMA recovers the rounding of a^2 -- and the correction -d a conj(b), which is smaller than
// half an ulp of the result, enters the sum BEFORE its single rounding (applied after the rounding it would be rounded
// away again, every time).  fp64: d ~ 1e-16, nothing to do.
__device__ __forceinline__ float unit_defect(cplx<float> w) {
    const float ar = fabsf(w.re), ai = fabsf(w.im);
    const float a = fmaxf(ar, ai), b = fminf(ar, ai);
    const float p = a * a;
    const float e = __fmaf_rn(a, a, -p);
    return __fmaf_rn(b, b, p - 1.0f) + e;
}
// d = |b|^2 - 1 supplied by the caller
__device__ __forceinline__ cplx<float> cmulc_unit(cplx<float> a, cplx<float> b, float d) {
    const float re0 = __fmaf_rn(a.re, b.re, a.im * b.im), im0 = __fmaf_rn(a.im, b.re, -(a.re * b.im));
    const float sr = -d * re0, si = -d * im0;
    return {__fmaf_rn(a.re, b.re, __fmaf_rn(a.im, b.im, sr)), __fmaf_rn(a.im, b.re, __fmaf_rn(-a.re, b.im, si))};
}
__device__ __forceinline__ cplx<double> cmulc_unit(cplx<double> a, cplx<double> b, float) { return cmulc(a, b); }
template <class T> __device__ __forceinline__ cplx<T> cmulc_unit(cplx<T> a, cplx<T> b) {
    if constexpr (sizeof(T) == 4) return cmulc_unit(a, b, unit_defect(b));
    else return cmulc(a, b);
}

// read-only (non-coherent) global load of one complex value
__device__ __forceinline__ cplx<float> ldg(const cplx<float>* p) {
    float2 v = __ldg(reinterpret_cast<const float2*>(p));
    return {v.x, v.y};
}
__device__ __forceinline__ cplx<double> ldg(const cplx<double>* p) {
    double2 v = __ldg(reinterpret_cast<const double2*>(p));
    return {v.x, v.y};
}
// L2-coherent load (data another SM wrote earlier in the same launch)
__device__ __forceinline__ cplx<float> ldcg_c(const cplx<float>* p) {
    float2 v = __ldcg(reinterpret_cast<const float2*>(p));
    return {v.x, v.y};
}
__device__ __forceinline__ cplx<double> ldcg_c(const cplx<double>* p) {
    double2 v = __ldcg(reinterpret_cast<const double2*>(p));
    return {v.x, v.y};
}
// twiddle fetch: SMEM = plain load from a shared-memory copy, otherwise read-only global load
template <bool SMEM, class T> __device__ __forceinline__ cplx<T> ldtw(const cplx<T>* p) {
    if constexpr (SMEM) return *p;
    else return ldg(p);
}

template <class T> struct pad_shift;
template <> struct pad_shift<float> { static constexpr int value = 4; };
template <> struct pad_shift<double> { static constexpr int value = 3; };

template <class T> __host__ __device__ __forceinline__ constexpr int phys(int i) { return i + (i >> pad_shift<T>::value); }
template <class T> __host__ __device__ constexpr int padded_len(int n) { return n + (n >> pad_shift<T>::value); }

// ---- compile-time roots of unity for the register butterflies -----------------------------------
// cos(2 pi m / 32), m = 0..8
__host__ __device__ constexpr double cos32(int m) {
    constexpr double c[9] = {1.0,
                             0.98078528040323044912618223613424,
                             0.92387953251128675612818318939679,
                             0.83146961230254523707878837761791,
                             0.70710678118654752440084436210485,
                             0.55557023301960222474283081394853,
                             0.38268343236508977172845998403040,
                             0.19509032201612826784828486847702,
                             0.0};
    return c[m];
}
// w_R^J = exp(-2 pi i J / R) for 0 <= J < R/2, R <= 32: (wr, wi) with wi <= 0
template <int R, int J> struct root {
    static constexpr int m = J * (32 / R);   // angle 2 pi m / 32, m in [0, 16)
    static constexpr double c = (m <= 8) ? cos32(m) : -cos32(16 - m);
    static constexpr double s = (m <= 8) ? cos32(8 - m) : cos32(m - 8);   // sin >= 0
};

// x * c for a compile-time constant c.  fp32: c is carried as hi + lo so that the product has no
// systematic (constant-rounding) bias -- a biased |w| != 1 inside every butterfly would change the
// field amplitude by ~1e-8 per transform, coherently, and thousands of z-steps add up.
// KM (fp32 only), the "constant mode": 0 = hi + lo at every application (exact to 1e-15);  1 = hi alone (one instruction
// instead of two);  2 = hi + kConstBunch lo.  A caller that applies the same butterflies at every z-step may use mode 1 at
// kConstBunch - 1 of every kConstBunch z-steps and mode 2 at the remaining one: the rounding of hi is a defect of ~3e-8, so
// the uncorrected steps deviate by (1 + d)^(K-1) = 1 + (K - 1) d to 1e-13 and the corrected one takes exactly that out
// (solo engine; the lo terms are 8 % of the FP32-pipe work of a z-step).
constexpr int kConstBunch = 8;
template <class T> struct kconst;
template <> struct kconst<double> {
    template <int KM, class C> static __device__ __forceinline__ double mul(double x, C) { return x * C::value; }
    // x * C1 + y * C2
    template <int KM, class C1, class C2> static __device__ __forceinline__ double dot(double x, C1, double y, C2) {
        return x * C1::value + y * C2::value;
    }
};
template <> struct kconst<float> {
    template <int KM, class C> static __device__ __forceinline__ float mul(float x, C) {
        constexpr float hi = (float)C::value;
        if constexpr (KM == 1) {
            return x * hi;
        } else {
            constexpr float lo = (float)((KM == 2 ? (double)kConstBunch : 1.0) * (C::value - (double)hi));
            return __fmaf_rn(x, hi, x * lo);
        }
    }
    template <int KM, class C1, class C2> static __device__ __forceinline__ float dot(float x, C1, float y, C2) {
        constexpr float h1 = (float)C1::value, h2 = (float)C2::value;
        if constexpr (KM == 1) {
            return __fmaf_rn(y, h2, x * h1);
        } else {
            constexpr double k = KM == 2 ? (double)kConstBunch : 1.0;
            constexpr float l1 = (float)(k * (C1::value - (double)h1)), l2 = (float)(k * (C2::value - (double)h2));
            float t = x * l1;
            t = __fmaf_rn(y, l2, t);
            t = __fmaf_rn(x, h1, t);
            return __fmaf_rn(y, h2, t);
        }
    }
};
struct c_sqrt_half { static constexpr double value = 0.70710678118654752440084436210485; };
template <int R, int J, bool NEG> struct c_cos { static constexpr double value = NEG ? -root<R, J>::c : root<R, J>::c; };
template <int R, int J, bool NEG> struct c_sin { static constexpr double value = NEG ? -root<R, J>::s : root<R, J>::s; };

// a * w_R^J (forward) or a * conj(w_R^J) (INV)
template <class T, int R, int J, bool INV, int KM = 0>
__device__ __forceinline__ cplx<T> mul_root(cplx<T> a) {
    using K = kconst<T>;
    if constexpr (J == 0) {
        return a;
    } else if constexpr (4 * J == R) {            // w = -i
        if constexpr (INV) return {-a.im, a.re};
        else return {a.im, -a.re};
    } else if constexpr (8 * J == R) {            // w = (1 - i)/sqrt2
        if constexpr (INV) return {K::template mul<KM>(a.re - a.im, c_sqrt_half{}), K::template mul<KM>(a.re + a.im, c_sqrt_half{})};
        else return {K::template mul<KM>(a.re + a.im, c_sqrt_half{}), K::template mul<KM>(a.im - a.re, c_sqrt_half{})};
    } else if constexpr (8 * J == 3 * R) {        // w = (-1 - i)/sqrt2
        if constexpr (INV) return {K::template mul<KM>(-a.re - a.im, c_sqrt_half{}), K::template mul<KM>(a.re - a.im, c_sqrt_half{})};
        else return {K::template mul<KM>(a.im - a.re, c_sqrt_half{}), K::template mul<KM>(-a.re - a.im, c_sqrt_half{})};
    } else {
        // forward: w = c - i s ; inverse: conj(w) = c + i s
        if constexpr (INV)
            return {K::template dot<KM>(a.re, c_cos<R, J, false>{}, a.im, c_sin<R, J, true>{}),
                    K::template dot<KM>(a.im, c_cos<R, J, false>{}, a.re, c_sin<R, J, false>{})};
        else
            return {K::template dot<KM>(a.re, c_cos<R, J, false>{}, a.im, c_sin<R, J, false>{}),
                    K::template dot<KM>(a.im, c_cos<R, J, false>{}, a.re, c_sin<R, J, true>{})};
    }
}

// ---- register DFT of size R, natural order in and out ---------------------------------------------
// Forward: decimation in frequency.  v[j] -> sum_j v[j] w_R^{jk}.
template <class T, int R, int KM = 0> struct dif {
    template <int J>
    static __device__ __forceinline__ void bf(cplx<T>* v) {
        cplx<T> a = v[J], b = v[J + R / 2];
        v[J] = a + b;
        v[J + R / 2] = mul_root<T, R, J, false, KM>(a - b);
    }
    template <int... J>
    static __device__ __forceinline__ void stage(cplx<T>* v, std::integer_sequence<int, J...>) {
        (bf<J>(v), ...);
    }
    static __device__ __forceinline__ void run(cplx<T>* v) {
        stage(v, std::make_integer_sequence<int, R / 2>{});
        dif<T, R / 2, KM>::run(v);
        dif<T, R / 2, KM>::run(v + R / 2);
        // X[2m] = first half [m], X[2m+1] = second half [m]
        cplx<T> t[R];
#pragma unroll
        for (int m = 0; m < R / 2; ++m) { t[2 * m] = v[m]; t[2 * m + 1] = v[m + R / 2]; }
#pragma unroll
        for (int m = 0; m < R; ++m) v[m] = t[m];
    }
};
template <class T, int KM> struct dif<T, 1, KM> { static __device__ __forceinline__ void run(cplx<T>*) {} };

// Inverse (unnormalised): decimation in time with conjugate roots -- the adjoint of dif<T,R>.
template <class T, int R, int KM = 0> struct dit_inv {
    template <int J>
    static __device__ __forceinline__ void bf(cplx<T>* v) {
        cplx<T> a = v[J], b = mul_root<T, R, J, true, KM>(v[J + R / 2]);
        v[J] = a + b;
        v[J + R / 2] = a - b;
    }
    template <int... J>
    static __device__ __forceinline__ void stage(cplx<T>* v, std::integer_sequence<int, J...>) {
        (bf<J>(v), ...);
    }
    static __device__ __forceinline__ void run(cplx<T>* v) {
        cplx<T> t[R];
#pragma unroll
        for (int m = 0; m < R / 2; ++m) { t[m] = v[2 * m]; t[m + R / 2] = v[2 * m + 1]; }
#pragma unroll
        for (int m = 0; m < R; ++m) v[m] = t[m];
        dit_inv<T, R / 2, KM>::run(v);
        dit_inv<T, R / 2, KM>::run(v + R / 2);
        stage(v, std::make_integer_sequence<int, R / 2>{});
    }
};
template <class T, int KM> struct dit_inv<T, 1, KM> { static __device__ __forceinline__ void run(cplx<T>*) {} };

// ---- radix plan ------------------------------------------------------------------------------------
// N = 2^L: pass 0 has radix 4 (the RK4-fused exchange pass); the remaining L - 2 bits are split into
// radix-16 passes (as many as possible) then 8 / 4, never radix 2:
//   (L-2)%4 == 0: 16..16 | 1: 16..16,8,4 | 2: 16..16,4 | 3: 16..16,8
template <int L> struct plan {
    static_assert(L >= 4 && L <= 14, "shared-memory FFT supports 2^4 .. 2^14");
    static constexpr int L1 = L - 2;
    static constexpr int rem = L1 % 4;
    static constexpr int n16 = (rem == 1) ? (L1 / 4 - 1) : (L1 / 4);
    static constexpr int P = 1 + n16 + (rem == 0 ? 0 : (rem == 1 ? 2 : 1));
    __host__ __device__ static constexpr int rbits(int p) {   // p = 0 .. P-1
        if (p == 0) return 2;
        const int q = p - 1;
        if (q < n16) return 4;
        if (rem == 1) return (q == n16) ? 3 : 2;
        if (rem == 2) return 2;
        return 3;   // rem == 3
    }
    // log2 of S_p = M_p / R_p (stride between the R_p inputs of a butterfly)
    __host__ __device__ static constexpr int sbits(int p) {
        int used = 0;
        for (int q = 0; q <= p; ++q) used += rbits(q);
        return L - used;
    }
    // offset (in complex elements) of pass p's twiddle block W_p[k-1][t] inside the twiddle table
    __host__ __device__ static constexpr int tw_offset(int p) {
        int off = 0;
        for (int q = 0; q < p; ++q) off += ((1 << rbits(q)) - 1) << sbits(q);
        return off;
    }
    static constexpr int tw_total = tw_offset(P);
    // twiddles of the shared-memory passes 1 .. P-2 (the last pass has none): one contiguous block
    static constexpr int tw_local_begin = tw_offset(1);
    static constexpr int tw_local_count = tw_offset(P - 1) - tw_offset(1);
};

// Address (in elements of the padded array) of butterfly input j, j = 0..R-1, of the butterfly
// (b, t) of a pass with R = 2^RB, S = 2^SB: logical index (b << (SB+RB)) + (j << SB) + t.
// Returns the runtime part; elem_off<..>(j) is the compile-time part.
template <class T, int RB, int SB>
__device__ __forceinline__ int elem_base(int b, int t) {
    constexpr int PS = pad_shift<T>::value;
    const int base = (b << (SB + RB)) + t;
    if constexpr (SB >= PS) return base + (base >> PS);
    else if constexpr (SB + RB >= PS) return base + (b << (SB + RB - PS));
    else return base + (b >> (PS - SB - RB));
}
template <class T, int RB, int SB>
__device__ __forceinline__ constexpr int elem_off(int j) {
    constexpr int PS = pad_shift<T>::value;
    if constexpr (SB >= PS) return j * ((1 << SB) + (1 << (SB - PS)));
    else if constexpr (SB + RB >= PS) return (j << SB) + (j >> (PS - SB));
    else return j << SB;
}

// ---- one forward (DIF) pass over shared memory -------------------------------------------------------
// butterflies u = tid, tid + NT, ...;  b = u >> sbits, t = u & (S-1); element j at b*M + j*S + t.
template <class T, int L, int PASS, int NT, bool TWS>
__device__ __forceinline__ void fwd_pass_smem(cplx<T>* __restrict__ sm, const cplx<T>* __restrict__ tw, int tid) {
    using PL = plan<L>;
    constexpr int RB = PL::rbits(PASS), R = 1 << RB, SB = PL::sbits(PASS), S = 1 << SB;
    constexpr int NBF = (1 << L) / R;
    const cplx<T>* __restrict__ w = tw + PL::tw_offset(PASS);
#pragma unroll 1
    for (int u = tid; u < NBF; u += NT) {
        const int b = u >> SB, t = u & (S - 1);
        cplx<T>* __restrict__ p = sm + elem_base<T, RB, SB>(b, t);
        cplx<T> v[R];
#pragma unroll
        for (int j = 0; j < R; ++j) v[j] = p[elem_off<T, RB, SB>(j)];
        dif<T, R>::run(v);
        if constexpr (SB > 0) {
#pragma unroll
            for (int k = 1; k < R; ++k) v[k] = cmul(v[k], ldtw<TWS>(&w[((k - 1) << SB) + t]));
        }
#pragma unroll
        for (int k = 0; k < R; ++k) p[elem_off<T, RB, SB>(k)] = v[k];
    }
}

// ---- one inverse (DIT) pass over shared memory ---------------------------------------------------------
// UF: the twiddle multiply can take the twiddles' magnitude defect out (cmulc_unit).  dtw (fp32): the defects to remove,
// tabulated with the index of the twiddle table -- a multiple K (|w|^2 - 1) when the caller corrects only every K-th
// application (the defect is ~3e-8: K uncorrected pairs make (1 + d)^K = 1 + K d to 1e-13, and one corrected multiply
// takes all of it out); null: this application is a plain multiply
template <class T, int L, int PASS, int NT, bool TWS, bool UF = false>
__device__ __forceinline__ void inv_pass_smem(cplx<T>* __restrict__ sm, const cplx<T>* __restrict__ tw, int tid, const float* __restrict__ dtw = nullptr) {
    using PL = plan<L>;
    constexpr int RB = PL::rbits(PASS), R = 1 << RB, SB = PL::sbits(PASS), S = 1 << SB;
    constexpr int NBF = (1 << L) / R;
    const cplx<T>* __restrict__ w = tw + PL::tw_offset(PASS);
#pragma unroll 1
    for (int u = tid; u < NBF; u += NT) {
        const int b = u >> SB, t = u & (S - 1);
        cplx<T>* __restrict__ p = sm + elem_base<T, RB, SB>(b, t);
        cplx<T> v[R];
#pragma unroll
        for (int k = 0; k < R; ++k) v[k] = p[elem_off<T, RB, SB>(k)];
        if constexpr (SB > 0) {
            bool plain = true;
            if constexpr (UF && sizeof(T) == 4) {
                if (dtw != nullptr) {       // uniform over the launch at this point of the program
                    plain = false;
#pragma unroll
                    for (int k = 1; k < R; ++k)
                        v[k] = cmulc_unit(v[k], ldtw<TWS>(&w[((k - 1) << SB) + t]), dtw[PL::tw_offset(PASS) + ((k - 1) << SB) + t]);
                }
            }
            if (plain) {
#pragma unroll
                for (int k = 1; k < R; ++k) v[k] = cmulc(v[k], ldtw<TWS>(&w[((k - 1) << SB) + t]));
            }
        }
        dit_inv<T, R>::run(v);
#pragma unroll
        for (int j = 0; j < R; ++j) p[elem_off<T, RB, SB>(j)] = v[j];
    }
}

// ---- multiplier tables --------------------------------------------------------------------------------
// A table entry is either one complex value (cplx<T>) or, for long fp32 runs, a two-float value
// hi + lo (tabx<float>): the frequency-domain multiplier acts on the same bin at every z-step, so
// the rounding of the *table* (3e-8 in modulus and phase) accumulates coherently over 10^4..10^5
// steps; hi + lo carries the fp64 table value to ~1e-15 and leaves only data rounding.
template <class T> struct alignas(4 * sizeof(T)) tabx { cplx<T> hi, lo; };

__device__ __forceinline__ tabx<float> ldg(const tabx<float>* p) {
    float4 v = __ldg(reinterpret_cast<const float4*>(p));
    return {{v.x, v.y}, {v.z, v.w}};
}
template <class T> __device__ __forceinline__ cplx<T> tab_mul(cplx<T> v, cplx<T> h) { return cmul(v, h); }
__device__ __forceinline__ cplx<float> tab_mul(cplx<float> v, tabx<float> h) {
    float re = v.re * h.lo.re;
    re = __fmaf_rn(-v.im, h.lo.im, re);
    re = __fmaf_rn(-v.im, h.hi.im, re);
    re = __fmaf_rn(v.re, h.hi.re, re);
    float im = v.re * h.lo.im;
    im = __fmaf_rn(v.im, h.lo.re, im);
    im = __fmaf_rn(v.im, h.hi.re, im);
    im = __fmaf_rn(v.re, h.hi.im, im);
    return {re, im};
}

// ---- the fused middle: last forward pass, table multiply, first inverse pass, all in registers ----------
// The last pass has S = 1: butterfly u owns positions u*R .. u*R + R-1.  The table is stored as
// tab[k * (N/R) + u] so that consecutive threads read consecutive addresses; it streams from L2 and
// its loads are issued before the shared-memory loads of the same butterfly.
template <class T, int L, int NT, class TAB = cplx<T>>
__device__ __forceinline__ void mid_pass_smem(cplx<T>* __restrict__ sm, const TAB* __restrict__ tab, int tid) {
    using PL = plan<L>;
    constexpr int PASS = PL::P - 1;
    constexpr int RB = PL::rbits(PASS), R = 1 << RB;
    static_assert(PL::sbits(PASS) == 0, "last pass must have unit stride");
    constexpr int NBF = (1 << L) / R;
#pragma unroll 1
    for (int u = tid; u < NBF; u += NT) {
        TAB h[R];
#pragma unroll
        for (int k = 0; k < R; ++k) h[k] = ldg(&tab[k * NBF + u]);
        cplx<T>* __restrict__ p = sm + elem_base<T, RB, 0>(u, 0);
        cplx<T> v[R];
#pragma unroll
        for (int j = 0; j < R; ++j) v[j] = p[elem_off<T, RB, 0>(j)];
        dif<T, R>::run(v);
#pragma unroll
        for (int k = 0; k < R; ++k) v[k] = tab_mul(v[k], h[k]);
        dit_inv<T, R>::run(v);
#pragma unroll
        for (int j = 0; j < R; ++j) p[elem_off<T, RB, 0>(j)] = v[j];
    }
}

// barrier between two shared-memory passes of a transform run by a team of threads.  SY = 0: the team is the CTA; 1..32: the
// team never spans warps, a __syncwarp will do; > 32: a named barrier of SY threads, id `bar` (1..15)
template <int SY> __device__ __forceinline__ void pass_sync(int bar = 0) {
    if constexpr (SY == 0) __syncthreads();
    else if constexpr (SY <= 32) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(bar), "n"(SY) : "memory");
}
// forward passes FIRST .. P-2 (everything before the fused middle), with the barriers between them
template <class T, int L, int NT, bool TWS, int PASS, int SY = 0>
__device__ __forceinline__ void fwd_passes(cplx<T>* sm, const cplx<T>* tw, int tid, int bar = 0) {
    if constexpr (PASS < plan<L>::P - 1) {
        fwd_pass_smem<T, L, PASS, NT, TWS>(sm, tw, tid);
        pass_sync<SY>(bar);
        fwd_passes<T, L, NT, TWS, PASS + 1, SY>(sm, tw, tid, bar);
    }
}
// inverse passes P-2 .. LAST
template <class T, int L, int NT, bool TWS, int LAST, int SY = 0, bool UF = false, int PASS = plan<L>::P - 2>
__device__ __forceinline__ void inv_passes(cplx<T>* sm, const cplx<T>* tw, int tid, int bar = 0, const float* dtw = nullptr) {
    if constexpr (PASS >= LAST) {
        pass_sync<SY>(bar);
        inv_pass_smem<T, L, PASS, NT, TWS, UF>(sm, tw, tid, dtw);
        inv_passes<T, L, NT, TWS, LAST, SY, UF, PASS - 1>(sm, tw, tid, bar, dtw);
    }
}

// A <- IDFT( tab .* DFT(A) ) on a field in (padded) shared memory, twiddles from global memory.
// Caller guarantees the field is visible to all threads on entry (barrier) and must barrier before
// reading the result.
template <class T, int L, int NT>
__device__ __forceinline__ void linear_op_smem(cplx<T>* sm, const cplx<T>* tw, const cplx<T>* tab, int tid) {
    fwd_passes<T, L, NT, false, 0>(sm, tw, tid);
    mid_pass_smem<T, L, NT>(sm, tab, tid);
    inv_passes<T, L, NT, false, 0>(sm, tw, tid);
}

// Shared-memory layout of the resident engine: the padded field, then a copy of the twiddles of the
// local passes 1..P-2.
template <class T, int L> struct smem_layout {
    static constexpr size_t field_bytes = (size_t)padded_len<T>(1 << L) * sizeof(cplx<T>);
    static constexpr size_t tw_bytes = (size_t)plan<L>::tw_local_count * sizeof(cplx<T>);
    static constexpr size_t total = field_bytes + (tw_bytes ? tw_bytes : 16);
};

// ---- the linear core of the resident engine ----------------------------------------------------------------
// The part of the linear operator between the two pass-0 halves: forward passes 1..P-2, middle,
// inverse passes P-2..1, on the field at the start of dynamic shared memory with the twiddles of
// the local passes behind it (smem_layout).  Input: the field after forward pass 0; output: the
// field before inverse pass 0.
//
// After the radix-4 pass 0 the field is four independent sub-transforms of N/4 points, so the CTA
// works as G = 4 thread groups (one sub-block each, NT/4 threads) that synchronise with their own
// named barrier instead of __syncthreads: the groups drift apart, and while one waits at a barrier
// or on shared memory the warps of the others keep the issue slots busy.  When the last two passes
// have the same radix R (N = 2^14: 16 . 16; N = 2^10: 16 . 16) the chain
//     forward pass P-2  ->  [last forward pass . table . first inverse pass]  ->  inverse pass P-2
// stays inside blocks of R^2 points that one warp owns completely (two blocks per warp and
// iteration), so it needs __syncwarp only, and the table entries of an iteration are requested from
// L2 before its first butterfly.
template <class T, int L, int NT> struct core_groups {
    using PL = plan<L>;
    static constexpr int G = (NT >= 128) ? 4 : 1;
    static constexpr int NTG = NT / G;
    static constexpr int RBL = PL::rbits(PL::P - 1);
    static constexpr int NBL = ((1 << L) / G) >> RBL;     // butterflies of the last pass per group
    static constexpr bool chain = PL::P >= 3 && PL::rbits(PL::P - 2) == RBL && NTG >= 32 && NBL % NTG == 0;
    // early table request costs 2 R registers on top of the butterfly: fp32 only
    static constexpr bool early_tab = sizeof(T) == 4;
};

// ---- class-granular cluster synchronisation ("flow") ------------------------------------------------------
// Pass 1 has stride S1 inside a sub-block; its butterfly t' touches the elements t' + S1 k and the
// pass-0 butterflies t (fused with RK4 in the resident engine, shared out over the cluster in tiles
// of 32) touch one element t of every sub-block.  So the tiles of *class* c = (t mod S1) / 32 depend
// only on the pass-1 butterflies of class c of every field, and vice versa: the two cluster-wide
// barriers of a z-step become 2 NCLS mbarriers per CTA,
//     ready[c]: every field's inverse pass 1 of class c is done   (G F arrivals: one warp per group and CTA)
//     done[c] : every tile of class c is integrated and written    (F NW / NCLS arrivals: the warps owning them)
// A warp waits only for the classes it touches; a warp that is half a phase late delays nobody.
template <class T, int L, int NT> struct flow_cfg {
    using PL = plan<L>;
    static constexpr int G = (NT >= 128) ? 4 : 1, NTG = NT / G, NWG = NTG / 32, NW = NT / 32;
    static constexpr int S1 = (PL::P >= 3) ? (1 << PL::sbits(PL::P >= 3 ? 1 : 0)) : 0;
    static constexpr int NCLS = S1 / 32;
    static constexpr int NB1 = (PL::P >= 3) ? (((1 << L) / G) >> PL::rbits(1)) : 0;
    static constexpr int NIT = (NTG > 0 && NB1 > 0) ? NB1 / NTG : 0;
    // pass 1 exists, is a shared-memory pass of its own, whole warps per class, every warp NIT classes
    static constexpr bool ok = G == 4 && PL::P >= 4 && NCLS >= 1 && NB1 % NTG == 0 && NIT * NWG == NCLS;
};

__device__ __forceinline__ void mbar_init(uint32_t addr, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(addr), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t addr, uint32_t parity) {
    asm volatile(
        "{\n.reg .pred P1;\nLAB_WAIT:\n"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\nbra LAB_WAIT;\nDONE:\n}" ::"r"(addr), "r"(parity)
        : "memory");
}
// the same with acquire at CTA scope: all producers are threads of this CTA (solo engine), no cache invalidation needed
__device__ __forceinline__ void mbar_wait_cta(uint32_t addr, uint32_t parity) {
    asm volatile(
        "{\n.reg .pred P1;\nLAB_WAIT:\n"
        "mbarrier.try_wait.parity.acquire.cta.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\nbra LAB_WAIT;\nDONE:\n}" ::"r"(addr), "r"(parity)
        : "memory");
}
// arrive on a barrier of this CTA; release at CTA scope after a __syncwarp that orders the other lanes' writes before it
__device__ __forceinline__ void mbar_arrive_cta(uint32_t addr, int lane) {
    __syncwarp();
    if (lane == 0) asm volatile("mbarrier.arrive.release.cta.shared::cta.b64 _, [%0];" ::"r"(addr) : "memory");
}
// lanes 0 .. nf-1 of a converged warp arrive on the barrier at local address `addr` in CTA `lane`;
// release at cluster scope, after a __syncwarp that orders the other lanes' writes before it
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t addr, int lane, int nf) {
    __syncwarp();
    if (lane < nf) {
        uint32_t remote;
        asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(addr), "r"(lane));
        asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(remote) : "memory");
    }
}
// runtime description of the synchronisation around one linear core
struct FlowArgs {
    uint32_t mb;        // shared address of ready[0]; done[c] = mb + 8 (NCLS + c)
    int nf;             // CTAs in the cluster
    int wait_in;        // forward pass 1 waits for done[class] (a fused phase precedes)
    int arrive_out;     // inverse pass 1 arrives on ready[class] (a fused phase follows)
    uint32_t par_done;  // parity of the done phase to wait for
};

template <int G, int NTG> __device__ __forceinline__ void group_bar(int g) {
    if constexpr (G == 1) __syncthreads();
    else asm volatile("bar.sync %0, %1;" ::"r"(g + 1), "n"(NTG) : "memory");
}

// one forward butterfly u of pass PASS (twiddles from shared memory)
template <class T, int L, int PASS, int KM = 0>
__device__ __forceinline__ void fwd_bf(cplx<T>* __restrict__ sm, const cplx<T>* __restrict__ tw, int u) {
    using PL = plan<L>;
    constexpr int RB = PL::rbits(PASS), R = 1 << RB, SB = PL::sbits(PASS), S = 1 << SB;
    const cplx<T>* __restrict__ w = tw + PL::tw_offset(PASS);
    const int b = u >> SB, t = u & (S - 1);
    cplx<T>* __restrict__ p = sm + elem_base<T, RB, SB>(b, t);
    cplx<T> v[R];
#pragma unroll
    for (int j = 0; j < R; ++j) v[j] = p[elem_off<T, RB, SB>(j)];
    dif<T, R, KM>::run(v);
    if constexpr (SB > 0) {
#pragma unroll
        for (int k = 1; k < R; ++k) v[k] = cmul(v[k], w[((k - 1) << SB) + t]);
    }
#pragma unroll
    for (int k = 0; k < R; ++k) p[elem_off<T, RB, SB>(k)] = v[k];
}
template <class T, int L, int PASS, int KM = 0>
__device__ __forceinline__ void inv_bf(cplx<T>* __restrict__ sm, const cplx<T>* __restrict__ tw, int u) {
    using PL = plan<L>;
    constexpr int RB = PL::rbits(PASS), R = 1 << RB, SB = PL::sbits(PASS), S = 1 << SB;
    const cplx<T>* __restrict__ w = tw + PL::tw_offset(PASS);
    const int b = u >> SB, t = u & (S - 1);
    cplx<T>* __restrict__ p = sm + elem_base<T, RB, SB>(b, t);
    cplx<T> v[R];
#pragma unroll
    for (int k = 0; k < R; ++k) v[k] = p[elem_off<T, RB, SB>(k)];
    if constexpr (SB > 0) {
#pragma unroll
        for (int k = 1; k < R; ++k) v[k] = cmulc(v[k], w[((k - 1) << SB) + t]);
    }
    dit_inv<T, R, KM>::run(v);
#pragma unroll
    for (int j = 0; j < R; ++j) p[elem_off<T, RB, SB>(j)] = v[j];
}
// the fused middle on butterfly u with its table entries already in registers
template <class T, int L, class TAB, int KM = 0>
__device__ __forceinline__ void mid_bf(cplx<T>* __restrict__ sm, const TAB* h, int u) {
    using PL = plan<L>;
    constexpr int RB = PL::rbits(PL::P - 1), R = 1 << RB;
    cplx<T>* __restrict__ p = sm + elem_base<T, RB, 0>(u, 0);
    cplx<T> v[R];
#pragma unroll
    for (int j = 0; j < R; ++j) v[j] = p[elem_off<T, RB, 0>(j)];
    dif<T, R, KM>::run(v);
#pragma unroll
    for (int k = 0; k < R; ++k) v[k] = tab_mul(v[k], h[k]);
    dit_inv<T, R, KM>::run(v);
#pragma unroll
    for (int j = 0; j < R; ++j) p[elem_off<T, RB, 0>(j)] = v[j];
}

// forward passes PASS .. LASTF of one group, a group barrier after each
template <class T, int L, int NT, int PASS, int LASTF, bool FLOW, bool CTA = false, int KM = 0>
__device__ __forceinline__ void group_fwd(cplx<T>* sm, const cplx<T>* twl, int g, int tg, const FlowArgs& fa) {
    using CG = core_groups<T, L, NT>;
    if constexpr (PASS <= LASTF) {
        constexpr int NB = ((1 << L) / CG::G) >> plan<L>::rbits(PASS);
        if constexpr (FLOW && PASS == 1) {
            using FC = flow_cfg<T, L, NT>;
#pragma unroll 1
            for (int it = 0; it < FC::NIT; ++it) {
                if (fa.wait_in) {
                    if constexpr (CTA) mbar_wait_cta(fa.mb + 8 * (FC::NCLS + (tg >> 5) + FC::NWG * it), fa.par_done);
                    else mbar_wait(fa.mb + 8 * (FC::NCLS + (tg >> 5) + FC::NWG * it), fa.par_done);
                }
                fwd_bf<T, L, PASS, KM>(sm, twl, g * NB + tg + CG::NTG * it);
            }
        } else {
#pragma unroll 1
            for (int ul = tg; ul < NB; ul += CG::NTG) fwd_bf<T, L, PASS, KM>(sm, twl, g * NB + ul);
        }
        group_bar<CG::G, CG::NTG>(g);
        group_fwd<T, L, NT, PASS + 1, LASTF, FLOW, CTA, KM>(sm, twl, g, tg, fa);
    }
}
// inverse passes PASS .. 1 of one group, a group barrier before each
template <class T, int L, int NT, int PASS, bool FLOW, bool CTA = false, int KM = 0>
__device__ __forceinline__ void group_inv(cplx<T>* sm, const cplx<T>* twl, int g, int tg, const FlowArgs& fa) {
    using CG = core_groups<T, L, NT>;
    if constexpr (PASS >= 1) {
        constexpr int NB = ((1 << L) / CG::G) >> plan<L>::rbits(PASS);
        group_bar<CG::G, CG::NTG>(g);
        if constexpr (FLOW && PASS == 1) {
            using FC = flow_cfg<T, L, NT>;
#pragma unroll 1
            for (int it = 0; it < FC::NIT; ++it) {
                inv_bf<T, L, PASS, KM>(sm, twl, g * NB + tg + CG::NTG * it);
                if (fa.arrive_out) {
                    if constexpr (CTA) mbar_arrive_cta(fa.mb + 8 * ((tg >> 5) + FC::NWG * it), tg & 31);
                    else mbar_arrive_cluster(fa.mb + 8 * ((tg >> 5) + FC::NWG * it), tg & 31, fa.nf);
                }
            }
        } else {
#pragma unroll 1
            for (int ul = tg; ul < NB; ul += CG::NTG) inv_bf<T, L, PASS, KM>(sm, twl, g * NB + ul);
        }
        group_inv<T, L, NT, PASS - 1, FLOW, CTA, KM>(sm, twl, g, tg, fa);
    }
}

// Caller guarantees the field is visible to all threads on entry (barrier) and must barrier before
// reading the result.  Not inlined: one copy serves every call site of a kernel.
// CTA: the flow barriers are used by threads of this CTA only (solo engine): acquire / release at CTA scope
// KM: constant mode of the butterflies (kconst)
template <class T, int L, int NT, bool FLOW = false, bool CTA = false, int KM = 0>
__device__ __noinline__ void linear_core_smem(const cplx<T>* __restrict__ tab, int tid, FlowArgs fa = FlowArgs{}) {
    using PL = plan<L>;
    using CG = core_groups<T, L, NT>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
    // addressed as the global table is: twl[tw_offset(p) + ...]
    const cplx<T>* twl = reinterpret_cast<const cplx<T>*>(smem_raw + smem_layout<T, L>::field_bytes) - PL::tw_local_begin;
    const int g = (CG::G == 1) ? 0 : tid / CG::NTG, tg = (CG::G == 1) ? tid : tid % CG::NTG;
    constexpr int R = 1 << CG::RBL, NBF = (1 << L) >> CG::RBL;
    if constexpr (CG::chain) {
        group_fwd<T, L, NT, 1, PL::P - 3, FLOW, CTA, KM>(sm, twl, g, tg, fa);
#pragma unroll 1
        for (int ul = tg; ul < CG::NBL; ul += CG::NTG) {
            const int u = g * CG::NBL + ul;
            cplx<T> h[R];
            if constexpr (CG::early_tab) {
#pragma unroll
                for (int k = 0; k < R; ++k) h[k] = ldg(&tab[k * NBF + u]);
            }
            fwd_bf<T, L, PL::P - 2, KM>(sm, twl, u);
            __syncwarp();
            if constexpr (!CG::early_tab) {
#pragma unroll
                for (int k = 0; k < R; ++k) h[k] = ldg(&tab[k * NBF + u]);
            }
            mid_bf<T, L, cplx<T>, KM>(sm, h, u);
            __syncwarp();
            inv_bf<T, L, PL::P - 2, KM>(sm, twl, u);
        }
        group_inv<T, L, NT, PL::P - 3, FLOW, CTA, KM>(sm, twl, g, tg, fa);
    } else {
        group_fwd<T, L, NT, 1, PL::P - 2, FLOW, CTA, KM>(sm, twl, g, tg, fa);
#pragma unroll 1
        for (int ul = tg; ul < CG::NBL; ul += CG::NTG) {
            const int u = g * CG::NBL + ul;
            cplx<T> h[R];
#pragma unroll
            for (int k = 0; k < R; ++k) h[k] = ldg(&tab[k * NBF + u]);
            mid_bf<T, L, cplx<T>, KM>(sm, h, u);
        }
        group_inv<T, L, NT, PL::P - 2, FLOW, CTA, KM>(sm, twl, g, tg, fa);
    }
}

// forward transform only (for frequency-domain output): result in digit-reversed order in smem
template <class T, int L, int NT>
__device__ __forceinline__ void forward_only_smem(cplx<T>* sm, const cplx<T>* tw, int tid) {
    fwd_passes<T, L, NT, false, 0>(sm, tw, tid);
    fwd_pass_smem<T, L, plan<L>::P - 1, NT, false>(sm, tw, tid);
}

// cudaFuncSetAttribute is per device: remember per (function, device) that it has been done
struct device_once {
    bool done[64] = {};
    // true if `set` still has to run for the current device (and marks it done when `set` succeeds)
    template <class F> cudaError_t run(F&& set) {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64 && done[dev]) return cudaSuccess;
        e = set();
        if (e == cudaSuccess && dev >= 0 && dev < 64) done[dev] = true;
        return e;
    }
};

// threads per CTA for a 2^L-point field: 32 points per thread for large fields (keeps the register
// budget at 128+/thread for the radix-16 butterflies), 16 for small ones
template <class T, int L> struct cta_threads {
    static constexpr int per = (L >= 11) ? 32 : 16;
    static constexpr int raw = (1 << L) / per;
    static constexpr int value = raw < 32 ? 32 : raw;
};

}  // namespace opo
