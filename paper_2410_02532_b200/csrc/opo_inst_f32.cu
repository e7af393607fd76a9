// fp32 (complex64) instantiations of every kernel, N = 2^6 .. 2^14.
#define OPO_T float
#define OPO_SUFFIX f32
#define OPO_MAXL 14
#include "opo_inst.inl"
