// sys_hcnsf3d.cu -- kernel instantiations of the hcnsf3d system (see systems.cuh, ops_impl.cuh).
#include "ops_impl.cuh"

namespace lbmk {
const SysOps* ops_hcnsf3d() { return Ops<SysHcnsf3D>::get(); }
}  // namespace lbmk
