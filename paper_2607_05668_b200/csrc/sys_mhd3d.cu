// sys_mhd3d.cu -- kernel instantiations of the mhd3d system (see systems.cuh, ops_impl.cuh).
#include "ops_impl.cuh"

namespace lbmk {
const SysOps* ops_mhd3d() { return Ops<SysMhd3D>::get(); }
}  // namespace lbmk
