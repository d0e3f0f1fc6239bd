// Dphi kernels for d_R = 15 (SU(4) adjoint), real links, f32: colour-parallel kernel + the one-thread-per-site kernel for comparison.
#include "dphi_launch.cuh"
namespace hr { HR_DPHI_INSTANCE(float, 15, 1) }
