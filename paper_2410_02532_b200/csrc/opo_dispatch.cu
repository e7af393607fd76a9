// opo_dispatch.cu -- routes the size-templated launchers to the per-(precision, log2 N) translation
// units (opo_inst.cu).  The instances are declared weak: a size that was not built simply reports
// cudaErrorNotSupported (opo_create turns that into OPO_ERR_UNSUPPORTED).
#include "opo_internal.h"

namespace opo {

#define OPO_DECL(SUF, LL)                                                                                     \
    cudaError_t launch_linear_##SUF##_L##LL(const LinArgs&, cudaStream_t) __attribute__((weak));              \
    cudaError_t launch_freq_##SUF##_L##LL(const FreqArgs&, cudaStream_t) __attribute__((weak));               \
    cudaError_t resident_info_##SUF##_L##LL(int, ResidentInfo*) __attribute__((weak));                        \
    cudaError_t launch_resident_##SUF##_L##LL(const ResidentArgs&, int, cudaStream_t) __attribute__((weak));     \
    cudaError_t launch_resident_nln_##SUF##_L##LL(const ResidentArgs&, int, cudaStream_t) __attribute__((weak)); \
    cudaError_t launch_resident_dk0_##SUF##_L##LL(const ResidentArgs&, int, cudaStream_t) __attribute__((weak)); \
    cudaError_t solo_info_##SUF##_L##LL(int, ResidentInfo*) __attribute__((weak));                            \
    cudaError_t launch_solo_##SUF##_L##LL(const ResidentArgs&, int, cudaStream_t) __attribute__((weak));      \
    cudaError_t launch_solo_dk0_##SUF##_L##LL(const ResidentArgs&, int, cudaStream_t) __attribute__((weak)); \
    cudaError_t launch_solo_train_##SUF##_L##LL(const ResidentArgs&, int, cudaStream_t) __attribute__((weak)); \
    cudaError_t wide_info_##SUF##_L##LL(int, int, ResidentInfo*) __attribute__((weak));                       \
    cudaError_t launch_wide_##SUF##_L##LL(const ResidentArgs&, int, cudaStream_t) __attribute__((weak));      \
    cudaError_t launch_wide_dk0_##SUF##_L##LL(const ResidentArgs&, int, cudaStream_t) __attribute__((weak));

#define OPO_DECL_ALL(SUF) \
    OPO_DECL(SUF, 4) OPO_DECL(SUF, 5) OPO_DECL(SUF, 6) OPO_DECL(SUF, 7) OPO_DECL(SUF, 8) OPO_DECL(SUF, 9) OPO_DECL(SUF, 10) OPO_DECL(SUF, 11) \
    OPO_DECL(SUF, 12) OPO_DECL(SUF, 13) OPO_DECL(SUF, 14)

OPO_DECL_ALL(f32)
OPO_DECL_ALL(f64)

#define OPO_DECL_LARGE(SUF, LL)                                                                               \
    cudaError_t large_info_##SUF##_L##LL(int, int, int, LargeInfo*) __attribute__((weak));                    \
    cudaError_t launch_large_##SUF##_L##LL(const LargeArgs&, int, cudaStream_t) __attribute__((weak));
OPO_DECL_LARGE(f32, 15) OPO_DECL_LARGE(f32, 16) OPO_DECL_LARGE(f32, 17) OPO_DECL_LARGE(f32, 18)
OPO_DECL_LARGE(f64, 14) OPO_DECL_LARGE(f64, 15) OPO_DECL_LARGE(f64, 16) OPO_DECL_LARGE(f64, 17) OPO_DECL_LARGE(f64, 18)

#define OPO_CASE(FN, SUF, LL, ...) \
    case LL: return FN##SUF##_L##LL ? FN##SUF##_L##LL(__VA_ARGS__) : cudaErrorNotSupported;

#define OPO_SWITCH(FN, SUF, log2n, ...)                                                            \
    switch (log2n) {                                                                               \
        OPO_CASE(FN, SUF, 4, __VA_ARGS__) OPO_CASE(FN, SUF, 5, __VA_ARGS__)                                      \
        OPO_CASE(FN, SUF, 6, __VA_ARGS__) OPO_CASE(FN, SUF, 7, __VA_ARGS__) OPO_CASE(FN, SUF, 8, __VA_ARGS__)    \
        OPO_CASE(FN, SUF, 9, __VA_ARGS__) OPO_CASE(FN, SUF, 10, __VA_ARGS__) OPO_CASE(FN, SUF, 11, __VA_ARGS__)  \
        OPO_CASE(FN, SUF, 12, __VA_ARGS__) OPO_CASE(FN, SUF, 13, __VA_ARGS__) OPO_CASE(FN, SUF, 14, __VA_ARGS__) \
        default: return cudaErrorNotSupported;                                                     \
    }

#define OPO_DISPATCHERS(SUF)                                                                                      \
    cudaError_t launch_linear_##SUF(int log2n, const LinArgs& a, cudaStream_t s) { OPO_SWITCH(launch_linear_, SUF, log2n, a, s) } \
    cudaError_t launch_freq_##SUF(int log2n, const FreqArgs& a, cudaStream_t s) { OPO_SWITCH(launch_freq_, SUF, log2n, a, s) }   \
    cudaError_t resident_info_##SUF(int log2n, int n_fields, ResidentInfo* out) { OPO_SWITCH(resident_info_, SUF, log2n, n_fields, out) } \
    cudaError_t launch_resident_##SUF(int log2n, const ResidentArgs& a, int n_clusters, cudaStream_t s) {        \
        if (a.nln) { OPO_SWITCH(launch_resident_nln_, SUF, log2n, a, n_clusters, s) }                             \
        if (a.dk0) { OPO_SWITCH(launch_resident_dk0_, SUF, log2n, a, n_clusters, s) }                             \
        OPO_SWITCH(launch_resident_, SUF, log2n, a, n_clusters, s)                                                \
    }                                                                                                             \
    cudaError_t solo_info_##SUF(int log2n, int n_fields, ResidentInfo* out) { OPO_SWITCH(solo_info_, SUF, log2n, n_fields, out) } \
    cudaError_t launch_solo_##SUF(int log2n, const ResidentArgs& a, int n_ctas, cudaStream_t s) {                 \
        if (a.train) { OPO_SWITCH(launch_solo_train_, SUF, log2n, a, n_ctas, s) }                                 \
        if (a.dk0) { OPO_SWITCH(launch_solo_dk0_, SUF, log2n, a, n_ctas, s) }                                     \
        OPO_SWITCH(launch_solo_, SUF, log2n, a, n_ctas, s)                                                        \
    }                                                                                                             \
    cudaError_t wide_info_##SUF(int log2n, int n_fields, int g, ResidentInfo* out) { OPO_SWITCH(wide_info_, SUF, log2n, n_fields, g, out) } \
    cudaError_t launch_wide_##SUF(int log2n, const ResidentArgs& a, int n_clusters, cudaStream_t s) {             \
        if (a.dk0) { OPO_SWITCH(launch_wide_dk0_, SUF, log2n, a, n_clusters, s) }                                 \
        OPO_SWITCH(launch_wide_, SUF, log2n, a, n_clusters, s)                                                    \
    }

OPO_DISPATCHERS(f32)
OPO_DISPATCHERS(f64)

cudaError_t large_info_f32(int log2n, int n_fields, int batch, int sm_count, LargeInfo* out) {
    switch (log2n) {
        OPO_CASE(large_info_, f32, 15, n_fields, batch, sm_count, out) OPO_CASE(large_info_, f32, 16, n_fields, batch, sm_count, out)
        OPO_CASE(large_info_, f32, 17, n_fields, batch, sm_count, out) OPO_CASE(large_info_, f32, 18, n_fields, batch, sm_count, out)
        default: return cudaErrorNotSupported;
    }
}
cudaError_t large_info_f64(int log2n, int n_fields, int batch, int sm_count, LargeInfo* out) {
    switch (log2n) {
        OPO_CASE(large_info_, f64, 14, n_fields, batch, sm_count, out) OPO_CASE(large_info_, f64, 15, n_fields, batch, sm_count, out)
        OPO_CASE(large_info_, f64, 16, n_fields, batch, sm_count, out) OPO_CASE(large_info_, f64, 17, n_fields, batch, sm_count, out)
        OPO_CASE(large_info_, f64, 18, n_fields, batch, sm_count, out)
        default: return cudaErrorNotSupported;
    }
}
cudaError_t launch_large_f32(int log2n, const LargeArgs& a, int grid, cudaStream_t s) {
    switch (log2n) {
        OPO_CASE(launch_large_, f32, 15, a, grid, s) OPO_CASE(launch_large_, f32, 16, a, grid, s)
        OPO_CASE(launch_large_, f32, 17, a, grid, s) OPO_CASE(launch_large_, f32, 18, a, grid, s)
        default: return cudaErrorNotSupported;
    }
}
cudaError_t launch_large_f64(int log2n, const LargeArgs& a, int grid, cudaStream_t s) {
    switch (log2n) {
        OPO_CASE(launch_large_, f64, 14, a, grid, s) OPO_CASE(launch_large_, f64, 15, a, grid, s)
        OPO_CASE(launch_large_, f64, 16, a, grid, s) OPO_CASE(launch_large_, f64, 17, a, grid, s)
        OPO_CASE(launch_large_, f64, 18, a, grid, s)
        default: return cudaErrorNotSupported;
    }
}

}  // namespace opo
