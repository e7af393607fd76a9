// opo_inst_wide.cu -- one translation unit per (precision, log2 N, dk variant) of the wide engine (opo_wide.cuh): compiled
// by build.py with -DOPO_T=float|double -DOPO_SUFFIX=f32|f64 -DOPO_L=<12..14> and, for the dk = 0 instantiation, -DOPO_DK0.
#include "opo_wide.cuh"

#if !defined(OPO_T) || !defined(OPO_SUFFIX) || !defined(OPO_L)
#error "compile with -DOPO_T=.. -DOPO_SUFFIX=.. -DOPO_L=.."
#endif

namespace opo {

#define OPO_CAT3_(a, b, c) a##b##_L##c
#define OPO_CAT3(a, b, c) OPO_CAT3_(a, b, c)
#define OPO_NAME(base) OPO_CAT3(base, OPO_SUFFIX, OPO_L)

#if defined(OPO_DK0)
cudaError_t OPO_NAME(launch_wide_dk0_)(const ResidentArgs& a, int n_clusters, cudaStream_t s) { return launch_wide_L<OPO_T, OPO_L, true>(a, n_clusters, s); }
#else
cudaError_t OPO_NAME(wide_info_)(int n_fields, int g, ResidentInfo* out) { return wide_info_L<OPO_T, OPO_L>(n_fields, g, out); }
cudaError_t OPO_NAME(launch_wide_)(const ResidentArgs& a, int n_clusters, cudaStream_t s) { return launch_wide_L<OPO_T, OPO_L, false>(a, n_clusters, s); }
#endif

}  // namespace opo
