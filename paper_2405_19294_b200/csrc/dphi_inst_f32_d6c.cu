// Dphi kernels for d_R = 6, complex links, f32.
#include "dphi_launch.cuh"
namespace hr { HR_DPHI_INSTANCE(float, 6, 0) }
