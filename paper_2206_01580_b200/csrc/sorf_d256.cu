// sorf_d256.cu -- instantiates the fused SORF kernels for descriptor length 256; see sorf_kernels.cuh.
#include "sorf_kernels.cuh"
namespace qmll {
QMLL_DEFINE_SORF_SHAPE_D(d256, 256)
}
