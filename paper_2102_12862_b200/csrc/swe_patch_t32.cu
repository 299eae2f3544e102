// k_patch2 instances with 32 threads per block (__launch_bounds__ minimum blocks per SM: 8)
#include "swe_patch_inst.cuh"

namespace swe {

PatchKernel patch_kernel_32(int B, int scalars, int self, int morph) {
  switch (B) {
    case 8: return patch_fn<32, 8>(scalars, self, morph);
    default: return nullptr;
  }
}

}  // namespace swe
