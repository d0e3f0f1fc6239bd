// Dphi kernels for d_R = 3 reading the fundamental link as its first N-1 rows (link kind 5), f32.
#include "dphi_launch.cuh"
namespace hr { HR_DPHI_INSTANCE(float, 3, 5) }
