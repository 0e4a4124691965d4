// sys_swe2d.cu -- kernel instantiations of the swe2d system (see systems.cuh, ops_impl.cuh).
#include "ops_impl.cuh"

namespace lbmk {
const SysOps* ops_swe2d() { return Ops<SysSwe2D>::get(); }
}  // namespace lbmk
