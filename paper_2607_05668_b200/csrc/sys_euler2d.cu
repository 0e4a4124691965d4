// sys_euler2d.cu -- kernel instantiations of the euler2d system (see systems.cuh, ops_impl.cuh).
#include "ops_impl.cuh"

namespace lbmk {
const SysOps* ops_euler2d() { return Ops<SysEuler2D>::get(); }
}  // namespace lbmk
