// sys_advection2d.cu -- kernel instantiations of the advection2d system (see systems.cuh, ops_impl.cuh).
#include "ops_impl.cuh"

namespace lbmk {
const SysOps* ops_advection2d() { return Ops<SysAdvection2D>::get(); }
}  // namespace lbmk
