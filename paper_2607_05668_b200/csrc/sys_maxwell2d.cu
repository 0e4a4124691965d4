// sys_maxwell2d.cu -- kernel instantiations of the maxwell2d system (see systems.cuh, ops_impl.cuh).
#include "ops_impl.cuh"

namespace lbmk {
const SysOps* ops_maxwell2d() { return Ops<SysMaxwell2D>::get(); }
}  // namespace lbmk
