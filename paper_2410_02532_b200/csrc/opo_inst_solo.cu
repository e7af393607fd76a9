// opo_inst_solo.cu -- one translation unit per (precision, log2 N, dk variant) of the solo engine (opo_solo.cuh): compiled
// by build.py with -DOPO_T=float|double -DOPO_SUFFIX=f32|f64 -DOPO_L=<4..14> and, for the dk = 0 instantiation, -DOPO_DK0; for
// the pump-train instantiation, -DOPO_TRAIN.
#include "opo_solo.cuh"

#if !defined(OPO_T) || !defined(OPO_SUFFIX) || !defined(OPO_L)
#error "compile with -DOPO_T=.. -DOPO_SUFFIX=.. -DOPO_L=.."
#endif

namespace opo {

#define OPO_CAT3_(a, b, c) a##b##_L##c
#define OPO_CAT3(a, b, c) OPO_CAT3_(a, b, c)
#define OPO_NAME(base) OPO_CAT3(base, OPO_SUFFIX, OPO_L)

#if defined(OPO_TRAIN)
cudaError_t OPO_NAME(launch_solo_train_)(const ResidentArgs& a, int n_ctas, cudaStream_t s) { return launch_solo_L<OPO_T, OPO_L, false, true>(a, n_ctas, s); }
#elif defined(OPO_DK0)
cudaError_t OPO_NAME(launch_solo_dk0_)(const ResidentArgs& a, int n_ctas, cudaStream_t s) { return launch_solo_L<OPO_T, OPO_L, true>(a, n_ctas, s); }
#else
cudaError_t OPO_NAME(solo_info_)(int n_fields, ResidentInfo* out) { return solo_info_L<OPO_T, OPO_L>(n_fields, out); }
cudaError_t OPO_NAME(launch_solo_)(const ResidentArgs& a, int n_ctas, cudaStream_t s) { return launch_solo_L<OPO_T, OPO_L, false>(a, n_ctas, s); }
#endif

}  // namespace opo
