// Dphi kernels for d_R = 3, two-index antisymmetric representation applied on the fly from fundamental links, f64.
#include "dphi_launch.cuh"
namespace hr { HR_DPHI_INSTANCE(double, 3, 3) }
