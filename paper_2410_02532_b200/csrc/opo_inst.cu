// opo_inst.cu -- one translation unit per (precision, log2 N): compiled by build.py with
//   -DOPO_T=float|double -DOPO_SUFFIX=f32|f64 -DOPO_L=<6..14>
// so that the size-specialised kernels build in parallel.  opo_dispatch.cu routes to whichever
// instances were linked in.
#include "opo_kernels.cuh"
#include "opo_resident.cuh"

#if !defined(OPO_T) || !defined(OPO_SUFFIX) || !defined(OPO_L)
#error "compile with -DOPO_T=.. -DOPO_SUFFIX=.. -DOPO_L=.."
#endif

namespace opo {

#define OPO_CAT3_(a, b, c) a##b##_L##c
#define OPO_CAT3(a, b, c) OPO_CAT3_(a, b, c)
#define OPO_NAME(base) OPO_CAT3(base, OPO_SUFFIX, OPO_L)

#ifndef OPO_NLN
cudaError_t OPO_NAME(launch_linear_)(const LinArgs& a, cudaStream_t s) { return launch_linear_L<OPO_T, OPO_L>(a, s); }
cudaError_t OPO_NAME(launch_freq_)(const FreqArgs& a, cudaStream_t s) { return launch_freq_L<OPO_T, OPO_L>(a, s); }
cudaError_t OPO_NAME(resident_info_)(int n_fields, ResidentInfo* out) { return resident_info_L<OPO_T, OPO_L>(n_fields, out); }
#endif
#if defined(OPO_DK0)
// the dk = 0 instantiation of the resident kernel only (build.py: -DOPO_NLN -DOPO_DK0 selects this branch)
cudaError_t OPO_NAME(launch_resident_dk0_)(const ResidentArgs& a, int n_clusters, cudaStream_t s) {
    return launch_resident_L<OPO_T, OPO_L, false, true>(a, n_clusters, s);
}
#elif defined(OPO_NLN)
// the N/2 - L - N/2 instantiation of the resident kernel only (build.py compiles this file a second time with -DOPO_NLN)
cudaError_t OPO_NAME(launch_resident_nln_)(const ResidentArgs& a, int n_clusters, cudaStream_t s) {
    return launch_resident_L<OPO_T, OPO_L, true>(a, n_clusters, s);
}
#else
cudaError_t OPO_NAME(launch_resident_)(const ResidentArgs& a, int n_clusters, cudaStream_t s) {
    return launch_resident_L<OPO_T, OPO_L, false>(a, n_clusters, s);
}
#endif

}  // namespace opo
