// Dphi kernels for d_R = 3, two-index antisymmetric representation applied on the fly from fundamental links, f32.
#include "dphi_launch.cuh"
namespace hr { HR_DPHI_INSTANCE(float, 3, 3) }
