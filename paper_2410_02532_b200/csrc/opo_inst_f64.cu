// fp64 (complex128) instantiations of every kernel, N = 2^6 .. 2^13 (one field per SM's shared memory).
#define OPO_T double
#define OPO_SUFFIX f64
#define OPO_MAXL 13
#include "opo_inst.inl"
