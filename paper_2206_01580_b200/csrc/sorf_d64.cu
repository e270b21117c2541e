// sorf_d64.cu -- instantiates the fused SORF kernels for descriptor length 64 (E = 64 elements per lane,
// P = 1 lanes per vector); see sorf_kernels.cuh.
#include "sorf_kernels.cuh"
namespace qmll {
QMLL_DEFINE_SORF_SHAPE(d64, 64, 1)
}
