// sys_allencahn2d.cu -- kernel instantiations of the allencahn2d system (see systems.cuh, ops_impl.cuh).
#include "ops_impl.cuh"

namespace lbmk {
const SysOps* ops_allencahn2d() { return Ops<SysAllenCahn2D>::get(); }
}  // namespace lbmk
