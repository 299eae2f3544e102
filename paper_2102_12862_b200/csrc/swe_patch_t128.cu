// k_patch2 instances with 128 threads per block (__launch_bounds__ minimum blocks per SM: 6, 4)
#include "swe_patch_inst.cuh"

namespace swe {

PatchKernel patch_kernel_128(int B, int scalars, int self, int morph) {
  switch (B) {
    case 6: return patch_fn<128, 6>(scalars, self, morph);
    case 4: return patch_fn<128, 4>(scalars, self, morph);
    default: return nullptr;
  }
}

}  // namespace swe
