// swe_state_summary_static (include/swe.h): the reductions of swe_step_info -- water volume sum_i h_i |Omega_i|, cells
// with h > h_dry, non-finite check; the k_info kernel of swe_kernels.cuh -- for callers that may not allocate: code
// under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  k_info keeps one partial result
// per thread block and a ticket in scratch memory carved from the context's workspace; this variant keeps them in a
// file-scope __device__ array of fixed size, so the call needs no context, no workspace and no allocation.  Every GPU
// that loads the library holds the array (kScratchBytes = 98,560 bytes) until the process exits.
//
// The array's name is a device symbol: in HOST code it is a host-side stand-in, not a device address.  The address the
// kernel is given comes from cudaGetSymbolAddress, taken once per device with that device current (scratch_of below).
//
// All calls share the array.  It keeps the last call's contents: the ticket is cleared on the stream before every
// launch, the partials of the blocks a launch uses are overwritten before they are read.  Two calls that overlap on the
// GPU (different streams, or two host threads) race on it -- the caller serialises them.
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <mutex>

#include "../../include/swe.h"

namespace swe {
void set_thread_error(const char *msg);     // swe_abi.cu: what swe_last_error(NULL) returns on this thread
}

namespace {

constexpr int kThreads = 256;
constexpr int kCellsPerThread = 16;
constexpr int kChunk = kThreads * kCellsPerThread;                       // cells one block reduces: 4096
constexpr int64_t kMaxCells = SWE_SUMMARY_STATIC_MAX_CELLS;              // 2^24
constexpr int kMaxBlocks = (int)(kMaxCells / kChunk);                    // 4096 partials
static_assert((int64_t)kMaxBlocks * kChunk == kMaxCells, "the maximum is a whole number of chunks");

struct Partial { double vol; long long wet; int bad; int pad_; };        // 24 bytes
struct Scratch {
  Partial part[kMaxBlocks];                                              // 98,304 bytes
  unsigned int ticket;                                                   // blocks that have stored their partial
  unsigned int pad_[63];                                                 // 256 bytes: the ticket's own line
};
constexpr size_t kScratchBytes = sizeof(Scratch);                        // 98,560
static_assert(kScratchBytes == 98560, "stated in include/swe.h and README.md");

static __device__ __align__(256) unsigned char g_scratch[kScratchBytes];

// One block per chunk of kChunk consecutive cells; thread t takes cells chunk0 + t, + kThreads, ... in that order.  The
// block that stores its partial last adds all partials: thread t those with index t, t + kThreads, ... in ascending
// order, then a fixed pairwise tree -- the result does not depend on which block comes last.
__global__ void __launch_bounds__(kThreads)
k_info_static(const double *__restrict__ h, const double *__restrict__ hu, const double *__restrict__ hv,
              const double *__restrict__ area, long long n_cells, double h_dry, Scratch *scratch, swe_state_summary *out) {
  __shared__ double s_vol[kThreads];
  __shared__ long long s_wet[kThreads];
  __shared__ int s_bad[kThreads];
  __shared__ bool s_last;
  const int t = threadIdx.x;
  auto block_sum = [&](double &vol, long long &wet, int &bad) {          // fixed tree over the block; result in thread 0
    s_vol[t] = vol; s_wet[t] = wet; s_bad[t] = bad;
    __syncthreads();
    for (int s = kThreads / 2; s > 0; s >>= 1) {
      if (t < s) { s_vol[t] = s_vol[t] + s_vol[t + s]; s_wet[t] += s_wet[t + s]; s_bad[t] |= s_bad[t + s]; }
      __syncthreads();
    }
    vol = s_vol[0]; wet = s_wet[0]; bad = s_bad[0];
    __syncthreads();
  };
  double vol = 0.0;
  long long wet = 0;
  int bad = 0;
  const long long c0 = (long long)blockIdx.x * kChunk;
#pragma unroll 4
  for (int k = 0; k < kCellsPerThread; ++k) {
    const long long i = c0 + (long long)k * kThreads + t;
    if (i < n_cells) {
      const double hi = h[i];
      vol += hi * area[i];
      wet += (hi > h_dry);
      bad |= !(isfinite(hi) && isfinite(hu[i]) && isfinite(hv[i]));
    }
  }
  block_sum(vol, wet, bad);
  if (t == 0) {
    Partial p; p.vol = vol; p.wet = wet; p.bad = bad; p.pad_ = 0;
    scratch->part[blockIdx.x] = p;
    __threadfence();
    s_last = (atomicAdd(&scratch->ticket, 1u) == gridDim.x - 1);
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  vol = 0.0; wet = 0; bad = 0;
  for (unsigned k = t; k < gridDim.x; k += kThreads) {
    const Partial p = scratch->part[k];
    vol += p.vol; wet += p.wet; bad |= p.bad;
  }
  block_sum(vol, wet, bad);
  if (t == 0) {
    swe_state_summary r; r.vol = vol; r.n_wet = wet; r.nonfinite = bad ? 1 : 0; r.pad_ = 0;
    *out = r;
    scratch->ticket = 0u;
  }
}

// Device address of g_scratch on the current device, resolved once per device (set-up: no allocation, no launch).
constexpr int kMaxDevices = 64;
std::mutex g_mu;
Scratch *g_addr[kMaxDevices] = {nullptr};

int scratch_of(Scratch **out, char *why, size_t why_cap) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { std::snprintf(why, why_cap, "swe_state_summary_static: cudaGetDevice: %s", cudaGetErrorString(e)); return SWE_ECUDA; }
  if (dev < 0 || dev >= kMaxDevices) { std::snprintf(why, why_cap, "swe_state_summary_static: device ordinal %d not supported", dev); return SWE_EINVAL; }
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_addr[dev]) {
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, g_scratch);          // with device `dev` current: ITS copy of the array
    if (e != cudaSuccess || !p) {
      std::snprintf(why, why_cap, "swe_state_summary_static: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
      return SWE_ECUDA;
    }
    g_addr[dev] = reinterpret_cast<Scratch *>(p);
  }
  *out = g_addr[dev];
  return SWE_OK;
}

}  // namespace

extern "C" int swe_state_summary_static(const double *h, const double *hu, const double *hv, const double *area,
                                        int64_t n_cells, double h_dry, void *cuda_stream, swe_state_summary *out) {
  char why[256];
  if (!h || !hu || !hv || !area || !out) { swe::set_thread_error("swe_state_summary_static: null pointer"); return SWE_EINVAL; }
  if (n_cells < 1 || n_cells > kMaxCells) {
    std::snprintf(why, sizeof why, "swe_state_summary_static: n_cells = %lld is outside 1 .. %lld (SWE_SUMMARY_STATIC_MAX_CELLS: "
                  "the static scratch array holds one partial per %d cells)", (long long)n_cells, (long long)kMaxCells, kChunk);
    swe::set_thread_error(why);
    return SWE_EINVAL;
  }
  if (!(h_dry >= 0.0)) { swe::set_thread_error("swe_state_summary_static: h_dry must be >= 0"); return SWE_EINVAL; }
  Scratch *scratch = nullptr;
  int rc = scratch_of(&scratch, why, sizeof why);
  if (rc != SWE_OK) { swe::set_thread_error(why); return rc; }
  cudaStream_t s = (cudaStream_t)cuda_stream;
  // what must start at zero: the ticket (a launch that was aborted would leave it behind).  The partials need no
  // clearing: every block of this launch stores its own before the last block reads them.
  cudaError_t e = cudaMemsetAsync(&scratch->ticket, 0, sizeof(unsigned int), s);
  if (e == cudaSuccess) {
    const int grid = (int)((n_cells + kChunk - 1) / kChunk);
    k_info_static<<<grid, kThreads, 0, s>>>(h, hu, hv, area, (long long)n_cells, h_dry, scratch, out);
    e = cudaGetLastError();
  }
  if (e != cudaSuccess) {
    std::snprintf(why, sizeof why, "swe_state_summary_static: %s", cudaGetErrorString(e));
    swe::set_thread_error(why);
    return SWE_ECUDA;
  }
  return SWE_OK;
}
