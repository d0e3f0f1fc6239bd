// Dphi kernels for d_R = 3, real (adjoint) links, f64.
#include "dphi_launch.cuh"
namespace hr { HR_DPHI_INSTANCE(double, 3, 1) }
