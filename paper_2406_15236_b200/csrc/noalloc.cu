// noalloc.cu -- mpc_velocity_profile_noalloc: the layer-averaged velocity profile (the shear-profile binning of
// PAPER.md:212, the same quantity mpc_observables returns in profile_host) for callers that have no device memory to give.
//
// Every other entry point of this library works in a workspace the caller allocates and hands to mpc_bind. That is no
// use to a caller that cannot allocate: an analysis or monitoring hook that another program calls from inside its time
// loop, where that program's caching allocator already holds nearly all of the GPU's memory (a direct cudaMalloc then
// fails, or, when it succeeds, stalls every stream of the device while it runs) or where the rule is simply "no
// allocation after start-up"; or a caller that only ever sees pointers it was given by another runtime and has no
// allocator of its own. For these the accumulation buffer of the profile kernel lives in the library image itself: a
// file-scope __device__ array of fixed size, which every GPU that loads the library holds until the process exits
// (32 KiB: MPC_PROFILE_NOALLOC_MAX_LAYERS layers x (one 64-bit velocity sum + one 64-bit count)).
//
// The kernel is k_obs_profile of observe.cu with that array as its scratch and a small second kernel that turns the sums
// into the averages on the device (mpc_observables does that on the host, after a copy). Sums are 64-bit fixed point, so
// the result does not depend on the order of the particles and is the same, bit for bit, as mpc_observables' profile of
// the same particles.
//
// The array's name means something only in device code. In host code it is a stand-in object in host memory: its address
// must never reach a kernel. The device address comes from cudaGetSymbolAddress, asked once per device (with that device
// current) the first time the entry point runs there; the kernels get that pointer.
#include <mutex>

#include "internal.cuh"

namespace mpc {

static __device__ __align__(256) u64 g_profile_scratch[2 * MPC_PROFILE_NOALLOC_MAX_LAYERS];

// scratch[0, nb): sums of v_f in units of 2^-28 u (int64); scratch[nb, 2 nb): particle counts. Both start at zero.
__global__ void __launch_bounds__(256) k_profile_noalloc(float inv_a, double fx, size_t n, int nb, const float* __restrict__ rp,
                                                         const float* __restrict__ vf, u64* __restrict__ scratch) {
  extern __shared__ u64 bins[];   // the CTA's own 2 nb words, flushed once at the end
  for (int b = threadIdx.x; b < 2 * nb; b += blockDim.x) bins[b] = 0ull;
  __syncthreads();
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  const size_t i0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  for (size_t base = i0 - (threadIdx.x & 31); base < n; base += stride) {   // whole warps iterate together
    const size_t i = base + (threadIdx.x & 31);
    int b = -1;
    long long q = 0;
    if (i < n) {
      b = max(0, min((int)floorf(rp[i] * inv_a), nb - 1));
      q = __double2ll_rn((double)vf[i] * fx);
    }
    // neighbouring particles mostly share a layer: one shared atomic per (warp, layer present in it) and quantity
    unsigned todo = __ballot_sync(0xffffffffu, b >= 0);
    while (todo) {
      const int lead = __ffs((int)todo) - 1;
      const int bl = __shfl_sync(0xffffffffu, b, lead);
      const bool mine = (b == bl);
      const unsigned grp = __ballot_sync(0xffffffffu, mine);
      long long s = mine ? q : 0ll;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
      if ((int)(threadIdx.x & 31) == lead) {
        atomicAdd(&bins[bl], (u64)s);
        atomicAdd(&bins[nb + bl], (u64)__popc(grp));
      }
      todo &= ~grp;
    }
  }
  __syncthreads();
  for (int b = threadIdx.x; b < 2 * nb; b += blockDim.x) if (bins[b] != 0ull) atomicAdd(&scratch[b], bins[b]);
}
// the averages, with the operations (and their order) of mpc_observables' host code: sum * 2^-28 u / count, then to float
__global__ void __launch_bounds__(256) k_profile_noalloc_finish(int nb, double fxi, const u64* __restrict__ scratch,
                                                                float* __restrict__ profile, u64* __restrict__ counts) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= nb) return;
  const long long s = (long long)scratch[b];
  const u64 k = scratch[nb + b];
  profile[b] = k > 0 ? (float)((double)s * fxi / (double)k) : 0.0f;
  if (counts) counts[b] = k;
}

}  // namespace mpc

using namespace mpc;

namespace {

constexpr int MAX_DEVICES = 64;
std::mutex g_setup_mutex;
u64* g_scratch_dev[MAX_DEVICES];   // device address of g_profile_scratch on each device, nullptr = not asked yet

// One-time set-up on the current device `dev`: the device address of the static array. No allocation: the array is
// part of the loaded module.
cudaError_t scratch_on_current_device(int dev, u64** out) {
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  if (!g_scratch_dev[dev]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_profile_scratch);
    if (e != cudaSuccess) return e;
    g_scratch_dev[dev] = static_cast<u64*>(p);
  }
  *out = g_scratch_dev[dev];
  return cudaSuccess;
}

}  // namespace

extern "C" int mpc_velocity_profile_noalloc(mpc_ctx* c, unsigned long long n, const float* r_w, const float* v_f, int n_layers,
                                            float* profile, unsigned long long* counts, void* cuda_stream) {
  if (!c) return MPC_EINVAL;
  if (c->sticky) return MPC_ECUDA;
  if (n_layers < 1) return fail(c, MPC_EINVAL, "mpc_velocity_profile_noalloc: n_layers must be at least 1");
  if (n_layers > MPC_PROFILE_NOALLOC_MAX_LAYERS)
    return fail(c, MPC_EINVAL, "mpc_velocity_profile_noalloc: n_layers exceeds MPC_PROFILE_NOALLOC_MAX_LAYERS (2048), the size of the "
                               "library's built-in scratch array; use mpc_observables with a bound workspace instead");
  if (!profile || (n && (!r_w || !v_f))) return fail(c, MPC_EINVAL, "mpc_velocity_profile_noalloc: NULL array");
  int dev = -1;
  CU(cudaGetDevice(&dev));
  if (dev < 0 || dev >= MAX_DEVICES) return fail(c, MPC_EINVAL, "mpc_velocity_profile_noalloc: device ordinal beyond 63");
  u64* scratch = nullptr;
  CU(scratch_on_current_device(dev, &scratch));
  cudaStream_t stream = (cudaStream_t)cuda_stream;
  const Geo& G = c->G;
  const int nb = n_layers;
  // the array still holds the previous call's sums: the part this call uses starts at zero
  CU(cudaMemsetAsync(scratch, 0, (size_t)2 * nb * sizeof(u64), stream));
  if (n) {
    const unsigned grid = (unsigned)(n < (unsigned long long)OBS_BLOCKS * 256ull ? (n + 255ull) / 256ull : (unsigned long long)OBS_BLOCKS);
    k_profile_noalloc<<<grid, 256, (size_t)2 * nb * sizeof(u64), stream>>>(G.inv_a, (double)G.fxv * 64.0, (size_t)n, nb, r_w, v_f, scratch);
    LAUNCH_CHECK("k_profile_noalloc");
  }
  k_profile_noalloc_finish<<<nblk((size_t)nb, 256), 256, 0, stream>>>(nb, G.fxv_inv / 64.0, scratch, profile, counts);
  LAUNCH_CHECK("k_profile_noalloc_finish");
  return MPC_OK;
}
