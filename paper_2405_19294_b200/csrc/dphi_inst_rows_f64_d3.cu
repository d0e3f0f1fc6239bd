// Dphi kernels for d_R = 3 reading the fundamental link as its first N-1 rows (link kind 4), f64.
#include "dphi_launch.cuh"
namespace hr { HR_DPHI_INSTANCE(double, 3, 4) }
