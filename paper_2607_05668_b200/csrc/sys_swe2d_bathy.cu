// sys_swe2d_bathy.cu -- kernel instantiations of the swe2d_bathy system (see systems.cuh, ops_impl.cuh).
#include "ops_impl.cuh"

namespace lbmk {
const SysOps* ops_swe2d_bathy() { return Ops<SysSwe2DBathy>::get(); }
}  // namespace lbmk
