// Dphi kernels for d_R = 2, complex links, f32.
#include "dphi_launch.cuh"
namespace hr { HR_DPHI_INSTANCE(float, 2, 0) }
