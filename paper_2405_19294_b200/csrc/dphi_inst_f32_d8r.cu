// Dphi kernels for d_R = 8, real (adjoint) links, f32.
#include "dphi_launch.cuh"
namespace hr { HR_DPHI_INSTANCE(float, 8, 1) }
