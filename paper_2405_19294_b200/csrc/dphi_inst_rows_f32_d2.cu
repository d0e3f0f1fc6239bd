// Dphi kernels for d_R = 2 reading the fundamental link as its first N-1 rows (link kind 4), f32.
#include "dphi_launch.cuh"
namespace hr { HR_DPHI_INSTANCE(float, 2, 4) }
