// sys_burgers2d.cu -- kernel instantiations of the burgers2d system (see systems.cuh, ops_impl.cuh).
#include "ops_impl.cuh"

namespace lbmk {
const SysOps* ops_burgers2d() { return Ops<SysBurgers2D>::get(); }
}  // namespace lbmk
