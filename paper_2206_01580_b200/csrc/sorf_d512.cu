// sorf_d512.cu -- instantiates the fused SORF kernels for descriptor length 512 (E = 128 elements per lane,
// P = 4 lanes per vector); see sorf_kernels.cuh.
#include "sorf_kernels.cuh"
namespace qmll {
QMLL_DEFINE_SORF_SHAPE(d512, 128, 4)
}
