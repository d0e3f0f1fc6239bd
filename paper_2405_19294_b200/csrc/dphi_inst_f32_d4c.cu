// Dphi kernels for d_R = 4, complex links, f32.
#include "dphi_launch.cuh"
namespace hr { HR_DPHI_INSTANCE(float, 4, 0) }
