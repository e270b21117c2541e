// sorf_d1024.cu -- instantiates the fused SORF kernels for descriptor length 1024; see sorf_kernels.cuh.
#include "sorf_kernels.cuh"
namespace qmll {
QMLL_DEFINE_SORF_SHAPE_D(d1024, 1024)
}
