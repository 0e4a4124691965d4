// sys_urf2d.cu -- kernel instantiations of the urf2d system (see systems.cuh, ops_impl.cuh).
#include "ops_impl.cuh"

namespace lbmk {
const SysOps* ops_urf2d() { return Ops<SysUrf2D>::get(); }
}  // namespace lbmk
