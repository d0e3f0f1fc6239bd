// Dphi kernels for d_R = 10 (SU(4) two-index symmetric), complex links, f32: colour-parallel kernel + the one-thread-per-site kernel for comparison.
#include "dphi_launch.cuh"
namespace hr { HR_DPHI_INSTANCE(float, 10, 0) }
