// sorf_d16.cu -- instantiates the fused SORF kernels for descriptor length 16 (E = 16 elements per lane,
// P = 1 lanes per vector); see sorf_kernels.cuh.
#include "sorf_kernels.cuh"
namespace qmll {
QMLL_DEFINE_SORF_SHAPE(d16, 16, 1)
}
