// k_patch2 instances with 512 threads per block (__launch_bounds__ minimum blocks per SM: 2, 1)
#include "swe_patch_inst.cuh"

namespace swe {

PatchKernel patch_kernel_512(int B, int scalars, int self, int morph) {
  switch (B) {
    case 2: return patch_fn<512, 2>(scalars, self, morph);
    case 1: return patch_fn<512, 1>(scalars, self, morph);
    default: return nullptr;
  }
}

}  // namespace swe
