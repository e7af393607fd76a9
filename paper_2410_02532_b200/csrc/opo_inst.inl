// opo_inst.inl -- included by opo_inst_f32.cu / opo_inst_f64.cu with OPO_T, OPO_SUFFIX, OPO_MAXL defined.
#include "opo_kernels.cuh"
#include "opo_resident.cuh"

namespace opo {

#define OPO_CAT2(a, b) a##b
#define OPO_CAT(a, b) OPO_CAT2(a, b)

#define OPO_CASE(LL, CALL)          \
    case LL:                        \
        if constexpr (LL <= OPO_MAXL) { constexpr int L = LL; return CALL; } \
        else return cudaErrorNotSupported;

#define OPO_SWITCH_L(log2n, CALL)   \
    switch (log2n) {                \
        OPO_CASE(6, CALL)           \
        OPO_CASE(7, CALL)           \
        OPO_CASE(8, CALL)           \
        OPO_CASE(9, CALL)           \
        OPO_CASE(10, CALL)          \
        OPO_CASE(11, CALL)          \
        OPO_CASE(12, CALL)          \
        OPO_CASE(13, CALL)          \
        OPO_CASE(14, CALL)          \
        default: return cudaErrorNotSupported; \
    }

cudaError_t OPO_CAT(launch_linear_, OPO_SUFFIX)(int log2n, const LinArgs& a, cudaStream_t s) {
    OPO_SWITCH_L(log2n, (launch_linear_L<OPO_T, L>(a, s)))
}
cudaError_t OPO_CAT(launch_freq_, OPO_SUFFIX)(int log2n, const FreqArgs& a, cudaStream_t s) {
    OPO_SWITCH_L(log2n, (launch_freq_L<OPO_T, L>(a, s)))
}
cudaError_t OPO_CAT(launch_rk4_, OPO_SUFFIX)(const Rk4Args& a, cudaStream_t s) { return launch_rk4_T<OPO_T>(a, s); }
cudaError_t OPO_CAT(launch_scale_, OPO_SUFFIX)(const ScaleArgs& a, cudaStream_t s) { return launch_scale_T<OPO_T>(a, s); }
cudaError_t OPO_CAT(launch_finite_, OPO_SUFFIX)(const void* A, long long count, int* flag, cudaStream_t s) {
    return launch_finite_T<OPO_T>(A, count, flag, s);
}
cudaError_t OPO_CAT(resident_info_, OPO_SUFFIX)(int log2n, int n_fields, ResidentInfo* out) {
    OPO_SWITCH_L(log2n, (resident_info_L<OPO_T, L>(n_fields, out)))
}
cudaError_t OPO_CAT(launch_resident_, OPO_SUFFIX)(int log2n, const ResidentArgs& a, int n_clusters, cudaStream_t s) {
    OPO_SWITCH_L(log2n, (launch_resident_L<OPO_T, L>(a, n_clusters, s)))
}

}  // namespace opo
