// k_patch2 instances with 256 threads per block (__launch_bounds__ minimum blocks per SM: 4, 3, 2)
#include "swe_patch_inst.cuh"

namespace swe {

PatchKernel patch_kernel_256(int B, int scalars, int self, int morph) {
  switch (B) {
    case 4: return patch_fn<256, 4>(scalars, self, morph);
    case 3: return patch_fn<256, 3>(scalars, self, morph);
    case 2: return patch_fn<256, 2>(scalars, self, morph);
    default: return nullptr;
  }
}

}  // namespace swe
