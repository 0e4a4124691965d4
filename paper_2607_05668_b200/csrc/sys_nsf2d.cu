// sys_nsf2d.cu -- kernel instantiations of the nsf2d system (see systems.cuh, ops_impl.cuh).
#include "ops_impl.cuh"

namespace lbmk {
const SysOps* ops_nsf2d() { return Ops<SysNsf2D>::get(); }
}  // namespace lbmk
