// sorf_d256.cu -- instantiates the fused SORF kernels for descriptor length 256 (E = 128 elements per lane,
// P = 2 lanes per vector); see sorf_kernels.cuh.
#include "sorf_kernels.cuh"
namespace qmll {
QMLL_DEFINE_SORF_SHAPE(d256, 128, 2)
}
