// sorf_d32.cu -- instantiates the fused SORF kernels for descriptor length 32 (E = 32 elements per lane,
// P = 1 lanes per vector); see sorf_kernels.cuh.
#include "sorf_kernels.cuh"
namespace qmll {
QMLL_DEFINE_SORF_SHAPE(d32, 32, 1)
}
