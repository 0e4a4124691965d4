// sys_adr2d.cu -- kernel instantiations of the adr2d system (see systems.cuh, ops_impl.cuh).
#include "ops_impl.cuh"

namespace lbmk {
const SysOps* ops_adr2d() { return Ops<SysAdr2D>::get(); }
}  // namespace lbmk
