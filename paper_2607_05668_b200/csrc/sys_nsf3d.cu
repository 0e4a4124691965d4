// sys_nsf3d.cu -- kernel instantiations of the nsf3d system (see systems.cuh, ops_impl.cuh).
#include "ops_impl.cuh"

namespace lbmk {
const SysOps* ops_nsf3d() { return Ops<SysNsf3D>::get(); }
}  // namespace lbmk
