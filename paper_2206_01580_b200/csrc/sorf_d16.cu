// sorf_d16.cu -- instantiates the fused SORF kernels for descriptor length 16; see sorf_kernels.cuh.
#include "sorf_kernels.cuh"
namespace qmll {
QMLL_DEFINE_SORF_SHAPE_D(d16, 16)
}
