// vg_bool_k1.cu -- boolean distance kernels with operand A of kind kOrb against every kind of B (see vg_bool.cuh)
#include "vg_bool.cuh"

namespace vg {
VG_BOOL_DEFINE_DIST(kOrb)
}
