// Dphi kernels for d_R = 2, complex links, f64.
#include "dphi_launch.cuh"
namespace hr { HR_DPHI_INSTANCE(double, 2, 0) }
