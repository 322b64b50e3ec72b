// vg_bool_k3.cu -- boolean distance kernels with operand A of kind kCone against every kind of B (see vg_bool.cuh)
#include "vg_bool.cuh"

namespace vg {
VG_BOOL_DEFINE_DIST(kCone)
}
