// sys_inse2d.cu -- kernel instantiations of the inse2d system (see systems.cuh, ops_impl.cuh).
#include "ops_impl.cuh"

namespace lbmk {
const SysOps* ops_inse2d() { return Ops<SysInse2D>::get(); }
}  // namespace lbmk
