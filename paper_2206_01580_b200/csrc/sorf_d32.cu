// sorf_d32.cu -- instantiates the fused SORF kernels for descriptor length 32; see sorf_kernels.cuh.
#include "sorf_kernels.cuh"
namespace qmll {
QMLL_DEFINE_SORF_SHAPE_D(d32, 32)
}
