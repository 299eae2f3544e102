// Instances of the fused patch kernel, one translation unit per block size (swe_patch_t*.cu), so that the library builds
// in parallel: the kernel is ~5000 SASS instructions and there are ~50 instances.
#pragma once
#include "swe_patch2_kernel.cuh"

namespace swe {

typedef void (*PatchKernel)(Control *, Patch2Args);

// the instance of k_patch2<T, B, ...> for (scalar species on board, self-controlled step, mobile bed); the self-controlled
// step (small meshes; self = 4 asks for the single-precision instance instead) is built for the plain hydrodynamic step only: nullptr otherwise
template <int T, int B>
inline PatchKernel patch_fn(int scalars, int self, int morph) {
  if (self == 4)    // single precision (R-21): plain hydrodynamics behind k_step_control
    return (scalars || morph) ? nullptr : (PatchKernel)k_patch2<T, B, false, false, false, float>;
  if (self) return (scalars || morph) ? nullptr : (PatchKernel)k_patch2<T, B, false, true, false>;
  if (scalars) return morph ? (PatchKernel)k_patch2<T, B, true, false, true> : (PatchKernel)k_patch2<T, B, true, false, false>;
  return morph ? (PatchKernel)k_patch2<T, B, false, false, true> : (PatchKernel)k_patch2<T, B, false, false, false>;
}

// defined in swe_patch_t<T>.cu: nullptr for a (T, B) pair that is not built
PatchKernel patch_kernel_32(int B, int scalars, int self, int morph);
PatchKernel patch_kernel_64(int B, int scalars, int self, int morph);
PatchKernel patch_kernel_128(int B, int scalars, int self, int morph);
PatchKernel patch_kernel_192(int B, int scalars, int self, int morph);
PatchKernel patch_kernel_256(int B, int scalars, int self, int morph);
PatchKernel patch_kernel_384(int B, int scalars, int self, int morph);
PatchKernel patch_kernel_512(int B, int scalars, int self, int morph);
PatchKernel patch_kernel_1024(int B, int scalars, int self, int morph);

}  // namespace swe
