// Dphi kernels for d_R = 6, complex links, f64.
#include "dphi_launch.cuh"
namespace hr { HR_DPHI_INSTANCE(double, 6, 0) }
