// Dphi kernels for the SU(3) adjoint (d_R = 8) applied on the fly from fundamental links (link kind 6), f64.
#include "dphi_launch.cuh"
namespace hr { HR_DPHI_INSTANCE(double, 8, 6) }
