// Dphi kernels for d_R = 3, complex links, f32.
#include "dphi_launch.cuh"
namespace hr { HR_DPHI_INSTANCE(float, 3, 0) }
