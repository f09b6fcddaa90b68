// Flag census without any allocation: mhd_flag_census_static (include/mhd.h). Same result as the census inside mhd_patch_status (flag bits of
// PAPER.md App. D, l.1151-1162: atmosphere reset, eps clamps, velocity cap, Ye clamp, fatal, no convergence, M1 fix-up), for callers that cannot
// call cudaMalloc (stream capture, tight serving loops, harnesses that forbid it) and do not own an mhd_patch (whose create call allocates).
//
// The scratch of the census, one partial count per CTA and flag bit, lives in a file-scope __device__ array of fixed size: every GPU that loads the
// library holds these 128 KB until exit. In host code the NAME of that array is a host-side stand-in, not a device address (a kernel handed it faults, or
// silently uses the wrong memory where the GPU can reach host memory): the device address comes from cudaGetSymbolAddress, asked once per device with that
// device current, and it is that pointer the kernels receive. All calls share the array and it keeps the last call's contents. Nothing in it has to start
// at zero: every CTA of the first kernel overwrites its own eight words before the second kernel reads exactly those. Two calls that overlap on the GPU
// (different streams, or one device driven from two threads) race on it; calls on one stream are ordered.
#include "mhd_internal.cuh"

namespace mhd {
namespace {

constexpr int CENSUS_CHUNK = 65536;                            // flags per CTA (a partial count fits 32 bits)
constexpr int CENSUS_MAX_CTAS = (int)(MHD_CENSUS_MAX_POINTS / CENSUS_CHUNK);
static_assert((long long)CENSUS_MAX_CTAS * CENSUS_CHUNK == MHD_CENSUS_MAX_POINTS, "MHD_CENSUS_MAX_POINTS must be a multiple of the chunk");

static __device__ __align__(256) unsigned int g_census_partial[CENSUS_MAX_CTAS * 8];   // 4096 x 8 x 4 B = 128 KB

// CTA b counts the flags [b CHUNK, min(n, (b + 1) CHUNK)) and writes its eight partial counts (plain stores: no word of the scratch is accumulated into)
__global__ void __launch_bounds__(256) k_census_partial(long long n, const uint8_t* __restrict__ flags, unsigned int* __restrict__ partial) {
  __shared__ unsigned int sh[8];
  if (threadIdx.x < 8) sh[threadIdx.x] = 0;
  __syncthreads();
  const long long lo = (long long)blockIdx.x * CENSUS_CHUNK, hi = min(n, lo + CENSUS_CHUNK);
  unsigned int loc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  for (long long t = lo + threadIdx.x; t < hi; t += blockDim.x) {
    const unsigned int f = flags[t];
#pragma unroll
    for (int b = 0; b < 8; ++b) loc[b] += (f >> b) & 1u;
  }
#pragma unroll
  for (int b = 0; b < 8; ++b) {
    unsigned int v = loc[b];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0 && v) atomicAdd(&sh[b], v);
  }
  __syncthreads();
  if (threadIdx.x < 8) partial[blockIdx.x * 8 + threadIdx.x] = sh[threadIdx.x];
}

// one CTA of eight warps: warp b sums the partial counts of bit b over the CTAs of the first kernel; out[0] = n, out[1 + b] = points with bit b set
__global__ void __launch_bounds__(256) k_census_total(long long n, int nctas, const unsigned int* __restrict__ partial, unsigned long long* __restrict__ out) {
  const int b = threadIdx.x >> 5, lane = threadIdx.x & 31;
  unsigned long long v = 0;
  for (int c = lane; c < nctas; c += 32) v += partial[c * 8 + b];
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  if (lane == 0) out[1 + b] = v;
  if (threadIdx.x == 0) out[0] = (unsigned long long)n;
}

// device address of the scratch array on the current device, asked once per device
cudaError_t census_scratch(unsigned int** out) {
  static unsigned int* addr[64] = {};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
  if (!addr[dev]) {
    unsigned int* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_census_partial);   // `dev` is current: the address is that of this device's copy
    if (e != cudaSuccess) return e;
    addr[dev] = p;
  }
  *out = addr[dev];
  return cudaSuccess;
}

}  // namespace
}  // namespace mhd

extern "C" int mhd_flag_census_static(const uint8_t* d_flags, long long n_points, unsigned long long* d_counts, void* cuda_stream) {
  using namespace mhd;
  if (!d_flags || !d_counts || n_points < 1) return MHD_E_ARG;
  if (n_points > MHD_CENSUS_MAX_POINTS) return MHD_E_TOO_LARGE;
  unsigned int* scratch = nullptr;
  if (census_scratch(&scratch) != cudaSuccess) return MHD_E_CUDA;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const int nctas = (int)((n_points + CENSUS_CHUNK - 1) / CENSUS_CHUNK);
  k_census_partial<<<nctas, 256, 0, s>>>(n_points, d_flags, scratch);
  k_census_total<<<1, 256, 0, s>>>(n_points, nctas, scratch, d_counts);
  return cudaGetLastError() == cudaSuccess ? MHD_OK : MHD_E_CUDA;
}
