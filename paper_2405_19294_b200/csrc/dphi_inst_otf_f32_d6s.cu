// Dphi kernels for d_R = 6, two-index symmetric representation applied on the fly from fundamental links, f32.
#include "dphi_launch.cuh"
namespace hr { HR_DPHI_INSTANCE(float, 6, 2) }
