// vg_bool_k4.cu -- boolean distance kernels with operand A of kind kTrd against every kind of B (see vg_bool.cuh)
#include "vg_bool.cuh"

namespace vg {
VG_BOOL_DEFINE_DIST(kTrd)
}
