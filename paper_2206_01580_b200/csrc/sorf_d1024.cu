// sorf_d1024.cu -- instantiates the fused SORF kernels for descriptor length 1024 (E = 128 elements per lane,
// P = 8 lanes per vector); see sorf_kernels.cuh.
#include "sorf_kernels.cuh"
namespace qmll {
QMLL_DEFINE_SORF_SHAPE(d1024, 128, 8)
}
