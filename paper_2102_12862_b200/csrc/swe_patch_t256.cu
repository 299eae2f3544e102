// k_patch2 instances with 256 threads per block (__launch_bounds__ minimum blocks per SM: 4, 3, 2; single precision
// also 6 and 5: its kernel needs 40 / 48 registers there and 34 KB of shared memory per block)
#include "swe_patch_inst.cuh"

namespace swe {

PatchKernel patch_kernel_256(int B, int scalars, int self, int morph) {
  switch (B) {
    case 6: return (self == 4 && !scalars && !morph) ? (PatchKernel)k_patch2<256, 6, false, false, false, float> : nullptr;
    case 5: return (self == 4 && !scalars && !morph) ? (PatchKernel)k_patch2<256, 5, false, false, false, float> : nullptr;
    case 4: return patch_fn<256, 4>(scalars, self, morph);
    case 3: return patch_fn<256, 3>(scalars, self, morph);
    case 2: return patch_fn<256, 2>(scalars, self, morph);
    default: return nullptr;
  }
}

}  // namespace swe
