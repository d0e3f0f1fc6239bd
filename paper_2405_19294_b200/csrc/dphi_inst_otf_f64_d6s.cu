// Dphi kernels for d_R = 6, two-index symmetric representation applied on the fly from fundamental links, f64.
#include "dphi_launch.cuh"
namespace hr { HR_DPHI_INSTANCE(double, 6, 2) }
