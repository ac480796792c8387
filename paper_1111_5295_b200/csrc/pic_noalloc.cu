// pic_noalloc.cu — pic_kinetic_energy_noalloc (include/pic.h): the kinetic-energy diagnostic for
// callers that must not allocate device memory while the time loop runs.
//
// Who that is.  pic_kinetic_energy() is what an implicit-PIC run calls every time step to check
// the energy identity (pin P-9), and it does a cudaMalloc and a cudaFree of a few bytes per call
// for its accumulators.  That is harmless in a test and a problem in three kinds of host program:
//   * one whose own memory pool has already taken (nearly) all of the GPU's memory at start-up --
//     a torch caching allocator grown to the card's size around a 1e8-particle state, a solver
//     that sub-allocates one big slab -- so that a cudaMalloc of even 16 bytes can fail in step
//     40,000 of a run;
//   * one that runs several streams or several handles (replicas, a field solve next to the
//     particle push): cudaFree waits for the WHOLE device, so a per-step diagnostic stalls
//     everything else that was in flight;
//   * one whose time loop runs under a "no allocation after set-up" rule (fixed memory budget,
//     fragmentation-free long runs) that is enforced by hooks on the allocator.
// For them the accumulators live in a file-scope device array that is part of the loaded library
// image: its memory is reserved on every GPU that loads libpic_b200.so, from load until the
// process ends, whether this entry point is ever called or not (kKeMaxSpecies * kKeBlocks doubles
// = 64 KiB).
//
// What it computes.  Same quantity as pic_kinetic_energy: per species sum_p w_m v_p^2 / 2 with
// w_m = w_q / (q/m), summed in fp64.  The existing kernel adds one fp64 atomic per block into a
// freshly allocated accumulator; this variant writes one partial sum per block into the static
// scratch and a second, single-block kernel adds those partials in a fixed order, so the result
// is also reproducible bit for bit from call to call (the atomic version is reproducible only to
// rounding order).
//
// Sharing rules.  There is ONE scratch array per GPU, shared by every handle, stream and thread
// of the process, and it keeps whatever the previous call left in it.  Nothing in it has to start
// at zero: a call overwrites every slot it later reads (block b of species s owns slot
// s * kKeBlocks + b, the finishing kernel reads exactly the slots of the blocks that were
// launched), so stale contents are never summed.  Two calls whose GPU work overlaps -- different
// streams, or different host threads on streams that do not order with each other -- write the
// same slots and race; the caller has to order them (same stream, an event, or a host lock held
// until the first call's stream work is complete).
//
// Set-up.  In host code the name of a __device__ array is only a stand-in that the runtime knows
// the symbol by; it is not an address the GPU can use.  The device address comes from
// cudaGetSymbolAddress, asked once per device with that device current, on the first call made
// on that device (the lookup also makes the runtime load this file's kernels onto the device).
// Make that first call during set-up, before any stream capture is started on the device.
// After it, a call issues two or more kernel launches and, for a host result pointer, one small
// device-to-host copy; it never calls cudaMalloc, cudaFree or any routine that allocates.
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

#include "pic_internal.h"

namespace {
constexpr int kKeMaxSpecies = PIC_KE_NOALLOC_MAX_SPECIES;   // species per handle accepted (pic.h)
constexpr int kKeBlocks = 1024;       // partial sums (= blocks) per species, at most
constexpr int kKeThreads = 256;
constexpr int kMaxDevices = 64;
}  // namespace

// The scratch, at file scope: [kKeMaxSpecies][kKeBlocks] block sums, then kKeMaxSpecies results
// (staging of the result for callers that pass a host pointer).  64 KiB + 64 B per GPU.
static __device__ __align__(256) double g_ke_scratch[kKeMaxSpecies * kKeBlocks + kKeMaxSpecies];

namespace picb200 {
namespace {

struct KePlan {                       // by-value kernel argument of the finishing kernel
  int n_species;
  int blocks[kKeMaxSpecies];          // partial sums written for species s (0: no particles)
  double half_w_m[kKeMaxSpecies];     // w_q / (q/m) / 2
};

// Stage 1: block b's share of sum_p v_p^2 -> part[b] (grid-stride, fixed assignment of particles
// to threads, fixed reduction tree: the value depends only on v, n and the launch shape).
template <typename T>
__global__ void __launch_bounds__(kKeThreads)
ke_partial_kernel(long long n, const T* __restrict__ v, double* part) {
  __shared__ double red[kKeThreads / 32];
  double s = 0.0;
  for (long long i = blockIdx.x * (long long)kKeThreads + threadIdx.x; i < n;
       i += (long long)gridDim.x * kKeThreads) {
    const double t = (double)v[i];
    s += t * t;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
#pragma unroll
    for (int w = 0; w < kKeThreads / 32; ++w) t += red[w];
    part[blockIdx.x] = t;             // plain store: the slot is overwritten, never accumulated
  }
}

// Stage 2 (one block): per species the partials in a fixed order, times w_m / 2.  Thread t adds
// slots t, t + 256, ...; then the same shuffle tree and warp order as above.
__global__ void __launch_bounds__(kKeThreads)
ke_finish_kernel(KePlan plan, const double* part, double* ke_out) {
  __shared__ double red[kKeThreads / 32];
  for (int s = 0; s < plan.n_species; ++s) {
    double a = 0.0;
    for (int b = threadIdx.x; b < plan.blocks[s]; b += kKeThreads) a += part[s * kKeBlocks + b];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = a;
    __syncthreads();
    if (threadIdx.x == 0) {
      double t = 0.0;
#pragma unroll
      for (int w = 0; w < kKeThreads / 32; ++w) t += red[w];
      ke_out[s] = t * plan.half_w_m[s];
    }
    __syncthreads();
  }
}

// Device address of g_ke_scratch on the current device, looked up once per device.
std::mutex g_setup_lock;
double* g_scratch_addr[kMaxDevices] = {};

cudaError_t scratch_on_current_device(int* dev_out, double** ptr_out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> hold(g_setup_lock);
  if (!g_scratch_addr[dev]) {
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_ke_scratch);   // host code: never pass g_ke_scratch itself
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    g_scratch_addr[dev] = p;
  }
  *dev_out = dev;
  *ptr_out = g_scratch_addr[dev];
  return cudaSuccess;
}

}  // namespace
}  // namespace picb200

using namespace picb200;

extern "C" int pic_kinetic_energy_noalloc(pic_handle* h, int which, double* ke_out) {
  if (!h || !ke_out) return PIC_ERR_ARG;
  if (which != PIC_STATE_N && which != PIC_STATE_NP1)
    return set_err(h, PIC_ERR_ARG, "pic_kinetic_energy_noalloc: which must be PIC_STATE_N or PIC_STATE_NP1");
  if (which == PIC_STATE_NP1 && !h->have_np1)
    return set_err(h, PIC_ERR_STATE, "pic_kinetic_energy_noalloc: no state n+1");
  const int ns = (int)h->sp.size();
  if (ns > kKeMaxSpecies)
    return set_err(h, PIC_ERR_UNSUPPORTED,
                   "pic_kinetic_energy_noalloc: more than PIC_KE_NOALLOC_MAX_SPECIES (8) species: "
                   "the static scratch holds 8 rows of block sums; use pic_kinetic_energy");
  static_assert(PIC_KE_NOALLOC_MAX_SPECIES == 8, "keep the message above in step with pic.h");
  int dev = -1;
  double* scratch = nullptr;
  cudaError_t e = scratch_on_current_device(&dev, &scratch);
  if (e != cudaSuccess)
    return set_err(h, PIC_ERR_CUDA, "pic_kinetic_energy_noalloc: cudaGetSymbolAddress(g_ke_scratch)", e);
  const int b = which == PIC_STATE_N ? h->cur : 1 - h->cur;
  KePlan plan{};
  plan.n_species = ns;
  for (int s = 0; s < ns; ++s) {
    const SpeciesState& S = h->sp[s];
    plan.half_w_m[s] = 0.5 * S.w_q / S.q_over_m;
    plan.blocks[s] = 0;
    if (S.n == 0) continue;
    // the scratch of THIS device is the one the kernels get: the state must live here too
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, S.v[b]) != cudaSuccess || at.device != dev) {
      cudaGetLastError();
      return set_err(h, PIC_ERR_ARG,
                     "pic_kinetic_energy_noalloc: the handle was created on another device than "
                     "the current one");
    }
    const long long want = (S.n + kKeThreads - 1) / kKeThreads;
    const int blocks = (int)(want < kKeBlocks ? want : kKeBlocks);
    plan.blocks[s] = blocks;
    double* part = scratch + (size_t)s * kKeBlocks;
    if (h->elem == 4)
      ke_partial_kernel<float><<<blocks, kKeThreads, 0, h->stream>>>(S.n, (const float*)S.v[b], part);
    else
      ke_partial_kernel<double><<<blocks, kKeThreads, 0, h->stream>>>(S.n, (const double*)S.v[b], part);
    h->launches++;
  }
  const bool dev_out = is_device_ptr(ke_out);
  double* result = dev_out ? ke_out : scratch + (size_t)kKeMaxSpecies * kKeBlocks;
  ke_finish_kernel<<<1, kKeThreads, 0, h->stream>>>(plan, scratch, result);
  h->launches++;
  PIC_CUDA(h, cudaGetLastError());
  if (!dev_out) {
    PIC_CUDA(h, cudaMemcpyAsync(ke_out, result, sizeof(double) * ns, cudaMemcpyDeviceToHost, h->stream));
    PIC_CUDA(h, cudaStreamSynchronize(h->stream));
  }
  return PIC_OK;
}
