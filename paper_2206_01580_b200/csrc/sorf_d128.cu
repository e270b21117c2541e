// sorf_d128.cu -- instantiates the fused SORF kernels for descriptor length 128 (E = 128 elements per lane,
// P = 1 lanes per vector); see sorf_kernels.cuh.
#include "sorf_kernels.cuh"
namespace qmll {
QMLL_DEFINE_SORF_SHAPE(d128, 128, 1)
}
