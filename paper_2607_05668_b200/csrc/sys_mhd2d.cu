// sys_mhd2d.cu -- kernel instantiations of the mhd2d system (see systems.cuh, ops_impl.cuh).
#include "ops_impl.cuh"

namespace lbmk {
const SysOps* ops_mhd2d() { return Ops<SysMhd2D>::get(); }
}  // namespace lbmk
