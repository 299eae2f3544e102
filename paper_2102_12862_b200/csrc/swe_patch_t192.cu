// k_patch2 instances with 192 threads per block (__launch_bounds__ minimum blocks per SM: 5, 4, 3)
#include "swe_patch_inst.cuh"

namespace swe {

PatchKernel patch_kernel_192(int B, int scalars, int self, int morph) {
  switch (B) {
    case 5: return patch_fn<192, 5>(scalars, self, morph);
    case 4: return patch_fn<192, 4>(scalars, self, morph);
    case 3: return patch_fn<192, 3>(scalars, self, morph);
    default: return nullptr;
  }
}

}  // namespace swe
