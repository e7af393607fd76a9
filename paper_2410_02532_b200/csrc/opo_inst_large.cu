// opo_inst_large.cu -- one translation unit per (precision, log2 N) of the large-N engine: compiled by
// build.py with -DOPO_T=float|double -DOPO_SUFFIX=f32|f64 -DOPO_L=<15..18 | 14..18>.
#include "opo_large.cuh"

#if !defined(OPO_T) || !defined(OPO_SUFFIX) || !defined(OPO_L)
#error "compile with -DOPO_T=.. -DOPO_SUFFIX=.. -DOPO_L=.."
#endif

namespace opo {

#define OPO_CAT3_(a, b, c) a##b##_L##c
#define OPO_CAT3(a, b, c) OPO_CAT3_(a, b, c)
#define OPO_NAME(base) OPO_CAT3(base, OPO_SUFFIX, OPO_L)

cudaError_t OPO_NAME(large_info_)(int n_fields, int batch, int sm_count, LargeInfo* out) {
    return large_info_L<OPO_T, OPO_L>(n_fields, batch, sm_count, out);
}
cudaError_t OPO_NAME(launch_large_)(const LargeArgs& a, int grid, cudaStream_t s) { return launch_large_L<OPO_T, OPO_L>(a, grid, s); }

}  // namespace opo
