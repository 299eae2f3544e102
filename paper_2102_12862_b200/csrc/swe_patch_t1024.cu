// k_patch2 instances with 1024 threads per block (__launch_bounds__ minimum blocks per SM: 1)
#include "swe_patch_inst.cuh"

namespace swe {

PatchKernel patch_kernel_1024(int B, int scalars, int self, int morph) {
  switch (B) {
    case 1: return patch_fn<1024, 1>(scalars, self, morph);
    default: return nullptr;
  }
}

}  // namespace swe
