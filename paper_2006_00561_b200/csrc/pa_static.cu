// pa_static.cu -- pa_overlap_hist_static: the order-parameter histogram (D1, reading G28) for
// callers that must not allocate.
//
// Who this is for.  Everything else in this library works inside a workspace the caller allocates up front and needs a
// pa_ctx, whose creation pins host memory.  Some users cannot do either at the moment they want the histogram: an
// analysis hook that runs while another component (a framework's caching allocator, a second simulation) already owns
// all of the GPU's memory and a cudaMalloc would fail or force that component to give memory back; a monitoring loop
// that must not stall, where cudaMalloc / cudaFree would synchronise the whole device under the running sweeps; code
// that is only handed a device pointer and a stream and has no permission to create CUDA resources.  For them this
// file offers ONE call that creates nothing: the caller passes the packed lattices and the output array, and the
// histogram's 64-bit accumulation bins -- the scratch memory the context path keeps in its workspace -- live in a
// fixed array that is part of the library image.
//
// What that costs.  The array below is (128*128 + 1) 64-bit counters, rounded up to a multiple of 256 bytes =
// 131 328 bytes.  Every GPU on which the library's device code gets loaded carries it from then until the process ends,
// whether or not this call is ever made.  It fixes the largest lattice: L <= PA_STATIC_MAX_L = 128 (the largest L
// the library supports anyway); a larger L is refused with PA_EINVAL, never truncated.
//
// Sharing.  There is one array per GPU, not per call or per stream.  Each call first clears the bins it will use (the
// array still holds the previous call's counts) and then accumulates into them, all on the caller's stream.  Two calls
// whose GPU work can overlap -- different streams, or different host threads without an ordering between their streams
// -- clear and add to the same bins and both results are garbage.  Calls on one stream, or calls separated by a
// synchronisation, are safe.
//
// Set-up.  In host code `g_ovl_bins` is only a handle for the array, not its address on a GPU; passing it to a kernel
// would hand the kernel a host address.  The device address is looked up with cudaGetSymbolAddress the first time
// the call runs on a given GPU (with that GPU current) and remembered per device ordinal.  That first call may make the
// CUDA runtime load this library's device code, so make it once, early, outside any stream capture; later calls on
// the same GPU only read the remembered pointer.
//
// The kernel is a variant of k_overlap_hist (pa_observe.cuh): the same pair loop and the same block-level histogram in
// shared memory, but R and the lattice pointer come as arguments instead of from a context's device state.  The
// existing path (pa_overlap_hist) is untouched.
#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

#include "../../include/pa_b200.h"

namespace {

constexpr int SOVL_MAX_N = PA_STATIC_MAX_L * PA_STATIC_MAX_L;
constexpr int SOVL_BINS = SOVL_MAX_N + 1;
constexpr int SOVL_BINS_PADDED = (SOVL_BINS + 31) / 32 * 32;  // whole 256-byte lines
constexpr int SOVL_THREADS = 256;
constexpr int SOVL_SMEM_BINS = 4097;  // L <= 64 keeps a block-level histogram in shared memory
constexpr int SOVL_MAX_DEVICES = 64;

// the scratch: accumulation bins of the histogram, one array per GPU that loads the library
static __device__ __align__(256) unsigned long long g_ovl_bins[SOVL_BINS_PADDED];

// overlap q = N - 2 popc(a xor b) of replica j and replica j + floor(R/2); bins[(q + N) / 2] += 1 for every j < floor(R/2).
// One warp per pair; lanes stride over the words of the two lattices.
__global__ void __launch_bounds__(SOVL_THREADS)
k_overlap_hist_static(const uint32_t* __restrict__ spins, const unsigned long long R, unsigned long long* __restrict__ bins,
                      const int N) {
  __shared__ unsigned s_hist[SOVL_SMEM_BINS];
  const bool use_smem = N + 1 <= SOVL_SMEM_BINS;
  if (use_smem)
    for (int i = threadIdx.x; i <= N; i += SOVL_THREADS) s_hist[i] = 0u;
  __syncthreads();
  const unsigned long long half = R / 2ull;
  const int wrep = N / 32, lane = threadIdx.x & 31;
  const unsigned long long warps = (unsigned long long)gridDim.x * (SOVL_THREADS / 32);
  for (unsigned long long j = (unsigned long long)blockIdx.x * (SOVL_THREADS / 32) + (threadIdx.x >> 5); j < half; j += warps) {
    const uint32_t* a = spins + j * wrep;
    const uint32_t* b = spins + (j + half) * wrep;
    int diff = 0;
    if ((wrep & 127) == 0) {  // L >= 64: 128-bit loads
      const uint4* a4 = reinterpret_cast<const uint4*>(a);
      const uint4* b4 = reinterpret_cast<const uint4*>(b);
      for (int w = lane; w < wrep / 4; w += 32) {
        const uint4 x = __ldg(a4 + w), y = __ldg(b4 + w);
        diff += __popc(x.x ^ y.x) + __popc(x.y ^ y.y) + __popc(x.z ^ y.z) + __popc(x.w ^ y.w);
      }
    } else {
      for (int w = lane; w < wrep; w += 32) diff += __popc(__ldg(a + w) ^ __ldg(b + w));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) diff += __shfl_xor_sync(0xffffffffu, diff, o);
    if (lane == 0) {
      const int bin = N - diff;
      if (use_smem) atomicAdd(&s_hist[bin], 1u);
      else atomicAdd(&bins[bin], 1ull);
    }
  }
  __syncthreads();
  if (use_smem)
    for (int i = threadIdx.x; i <= N; i += SOVL_THREADS)
      if (s_hist[i]) atomicAdd(&bins[i], (unsigned long long)s_hist[i]);
}

// ---- host side: no heap, no CUDA resource is created anywhere below ------------------------------------
thread_local char t_err[256] = "";

int sfail(int code, const char* what, const char* detail = nullptr) {
  if (detail) std::snprintf(t_err, sizeof t_err, "pa_overlap_hist_static: %s: %s", what, detail);
  else std::snprintf(t_err, sizeof t_err, "pa_overlap_hist_static: %s", what);
  return code;
}

std::mutex g_mu;
unsigned long long* g_bins_on[SOVL_MAX_DEVICES] = {};  // device address of g_ovl_bins, per device ordinal

// once per GPU, with that GPU current: turn the host-side handle g_ovl_bins into the array's address on this GPU
int bins_of_current_device(int dev, unsigned long long** out) {
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_bins_on[dev]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_ovl_bins);
    if (e != cudaSuccess || !p) return sfail(PA_ECUDA, "cudaGetSymbolAddress", cudaGetErrorString(e));
    g_bins_on[dev] = static_cast<unsigned long long*>(p);
  }
  *out = g_bins_on[dev];
  return PA_OK;
}

}  // namespace

extern "C" {

int pa_overlap_hist_static(const uint32_t* spins, int32_t L, int64_t R, uint64_t* hist, int hist_on_device, void* stream) {
  t_err[0] = 0;
  if (L > PA_STATIC_MAX_L) {
    char d[128];
    std::snprintf(d, sizeof d, "L = %d needs %lld bins, the built-in scratch array holds %d (L <= %d)", (int)L,
                  (long long)L * L + 1, SOVL_BINS, PA_STATIC_MAX_L);
    return sfail(PA_EINVAL, "lattice too large for the static scratch", d);
  }
  if (L != 8 && L != 16 && L != 32 && L != 64 && L != 128) return sfail(PA_EINVAL, "L must be 8, 16, 32, 64 or 128");
  if (R < 0 || R >= (int64_t)1 << 31) return sfail(PA_EINVAL, "R must be in [0, 2^31)");
  if (!hist || (!spins && R > 0)) return sfail(PA_EINVAL, "null pointer");
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return sfail(PA_ECUDA, "cudaGetDevice", cudaGetErrorString(e));
  if (dev < 0 || dev >= SOVL_MAX_DEVICES) return sfail(PA_EINVAL, "device ordinal beyond the 64 this call keeps a pointer for");
  if (R > 0) {  // the lattices must live on the GPU whose copy of the scratch array is about to be used
    cudaPointerAttributes at;
    e = cudaPointerGetAttributes(&at, spins);
    if (e != cudaSuccess) return sfail(PA_ECUDA, "cudaPointerGetAttributes(spins)", cudaGetErrorString(e));
    if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)
      return sfail(PA_EINVAL, "spins is not a device pointer");
    if (at.type == cudaMemoryTypeDevice && at.device != dev)
      return sfail(PA_EINVAL, "spins lives on another GPU than the current one");
  }
  unsigned long long* bins = nullptr;
  if (int rc = bins_of_current_device(dev, &bins)) return rc;

  const int N = L * L;
  const size_t bytes = ((size_t)N + 1) * 8;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  // the array keeps the last call's counts: clear the bins of this call
  e = cudaMemsetAsync(bins, 0, bytes, s);
  if (e != cudaSuccess) return sfail(PA_ECUDA, "cudaMemsetAsync(scratch)", cudaGetErrorString(e));
  const int64_t pairs = R / 2;
  if (pairs > 0) {
    const int64_t want = (pairs + 63) / 64;
    const unsigned grid = (unsigned)(want > 148 * 8 ? 148 * 8 : want);
    k_overlap_hist_static<<<grid, SOVL_THREADS, 0, s>>>(spins, (unsigned long long)R, bins, N);
    e = cudaGetLastError();
    if (e != cudaSuccess) return sfail(PA_ECUDA, "kernel launch", cudaGetErrorString(e));
  }
  e = cudaMemcpyAsync(hist, bins, bytes, hist_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, s);
  if (e != cudaSuccess) return sfail(PA_ECUDA, "cudaMemcpyAsync(hist)", cudaGetErrorString(e));
  if (!hist_on_device) {
    e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return sfail(PA_ECUDA, "cudaStreamSynchronize", cudaGetErrorString(e));
  }
  return PA_OK;
}

const char* pa_static_last_error(void) { return t_err; }

}  // extern "C"
