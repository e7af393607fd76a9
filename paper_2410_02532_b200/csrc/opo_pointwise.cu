// opo_pointwise.cu -- the size-independent kernels of the streaming engine (RK4, mirror scale,
// phase-modulator table, finite check) for both precisions.
#include "opo_kernels.cuh"

namespace opo {

cudaError_t launch_rk4_f32(const Rk4Args& a, cudaStream_t s) { return launch_rk4_T<float>(a, s); }
cudaError_t launch_rk4_f64(const Rk4Args& a, cudaStream_t s) { return launch_rk4_T<double>(a, s); }
cudaError_t launch_scale_f32(const ScaleArgs& a, cudaStream_t s) { return launch_scale_T<float>(a, s); }
cudaError_t launch_scale_f64(const ScaleArgs& a, cudaStream_t s) { return launch_scale_T<double>(a, s); }
cudaError_t launch_multab_f32(const MulTabArgs& a, cudaStream_t s) { return launch_multab_T<float>(a, s); }
cudaError_t launch_multab_f64(const MulTabArgs& a, cudaStream_t s) { return launch_multab_T<double>(a, s); }
cudaError_t launch_broadcast_f32(void* dst, int batch, int n, cudaStream_t s) { return launch_broadcast_T<float>(dst, batch, n, s); }
cudaError_t launch_broadcast_f64(void* dst, int batch, int n, cudaStream_t s) { return launch_broadcast_T<double>(dst, batch, n, s); }
cudaError_t launch_axpy_f32(void* A, const void* S, double c, int acc, long long n, cudaStream_t s) { return launch_axpy_T<float>(A, S, c, acc, n, s); }
cudaError_t launch_axpy_f64(void* A, const void* S, double c, int acc, long long n, cudaStream_t s) { return launch_axpy_T<double>(A, S, c, acc, n, s); }
cudaError_t launch_finite_f32(const void* A, long long count, int* flag, cudaStream_t s) { return launch_finite_T<float>(A, count, flag, s); }
cudaError_t launch_finite_f64(const void* A, long long count, int* flag, cudaStream_t s) { return launch_finite_T<double>(A, count, flag, s); }

}  // namespace opo
