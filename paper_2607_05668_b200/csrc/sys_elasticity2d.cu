// sys_elasticity2d.cu -- kernel instantiations of the elasticity2d system (see systems.cuh, ops_impl.cuh).
#include "ops_impl.cuh"

namespace lbmk {
const SysOps* ops_elasticity2d() { return Ops<SysElasticity2D>::get(); }
}  // namespace lbmk
