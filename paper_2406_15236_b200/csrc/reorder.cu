// reorder.cu -- REORDER: counting sort of the particles by (cell key, id). Counts come from the
// cell sums (no separate histogram), an exclusive scan gives the cell offsets, a scatter gives the
// permutation; the gather is folded into the next step's sweep or done property-wise through one
// temporary array in the compact workspace.
#include "internal.cuh"

namespace mpc {

// ---- exclusive scan of the per-cell counts (three kernels; tile = 2048) ----------------------------
// `in` is read with a stride in 32-bit words: the count is the low 16 bits of word 0 of a cell's sums.
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t& total) {
  __shared__ uint32_t wsum[33];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  uint32_t inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) wsum[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    const uint32_t w = lane < nw ? wsum[lane] : 0u;
    uint32_t winc = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, winc, o);
      if (lane >= o) winc += t;
    }
    wsum[lane] = winc - w;            // exclusive offset of every warp
    if (lane == 31) wsum[32] = winc;  // block total
  }
  __syncthreads();
  const uint32_t res = wsum[warp] + inc - v;
  total = wsum[32];
  __syncthreads();                    // wsum is reused by the caller's next round
  return res;
}
__global__ void __launch_bounds__(SCAN_T) k_scan_reduce(const uint32_t* __restrict__ in, int stride, size_t n, uint32_t* __restrict__ bsum) {
  const size_t base = (size_t)blockIdx.x * SCAN_TILE;
  uint32_t s = 0;
#pragma unroll
  for (int j = 0; j < SCAN_PER; ++j) {
    const size_t i = base + (size_t)j * SCAN_T + threadIdx.x;
    if (i < n) s += in[i * stride] & 0xffffu;
  }
  __shared__ uint32_t red[SCAN_T / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t t = 0;
    for (int w = 0; w < SCAN_T / 32; ++w) t += red[w];
    bsum[blockIdx.x] = t;
  }
}
__global__ void __launch_bounds__(1024) k_scan_top(uint32_t* __restrict__ bsum, size_t nb) {
  uint32_t carry = 0;
  for (size_t base = 0; base < nb; base += 1024) {
    const size_t i = base + threadIdx.x;
    const uint32_t v = i < nb ? bsum[i] : 0u;
    uint32_t total;
    const uint32_t ex = block_exclusive_scan(v, total);
    if (i < nb) bsum[i] = carry + ex;
    carry += total;
  }
}
__global__ void __launch_bounds__(SCAN_T) k_scan_apply(const uint32_t* __restrict__ in, int stride, size_t n,
                                                       const uint32_t* __restrict__ bsum, uint32_t* __restrict__ out) {
  const size_t base = (size_t)blockIdx.x * SCAN_TILE + (size_t)threadIdx.x * SCAN_PER;
  uint32_t v[SCAN_PER], s = 0;
#pragma unroll
  for (int j = 0; j < SCAN_PER; ++j) {
    v[j] = (base + j < n) ? (in[(base + j) * stride] & 0xffffu) : 0u;
    s += v[j];
  }
  uint32_t total;
  uint32_t ex = block_exclusive_scan(s, total) + bsum[blockIdx.x];
#pragma unroll
  for (int j = 0; j < SCAN_PER; ++j) {
    if (base + j < n) out[base + j] = ex;
    ex += v[j];
  }
  if (blockIdx.x == gridDim.x - 1 && threadIdx.x == SCAN_T - 1) out[n] = ex;   // grand total
}

// ---- scatter --------------------------------------------------------------------------------------
// lane-spread order inside a group of 32 cells: spread_slot (internal.cuh)
__device__ __forceinline__ uint32_t spread_key(const uint32_t* __restrict__ offset, uint32_t k, uint32_t slot, int spread) {
  if (!spread) return slot;
  const uint32_t kg = k & ~((1u << spread) - 1u);
  return spread_slot(slot, offset[kg], offset[kg + (1u << spread)]);
}

// Lanes of a warp that hold the same key as their neighbours form runs (the array is still nearly sorted):
// one cursor atomic per run. Returns the first slot of this lane within its cell segment's arrival order.
// (match.any would also merge non-adjacent lanes but runs at a fraction of the rate: measured 72 % pipe busy.)
__device__ __forceinline__ uint32_t run_slot(uint32_t k, uint32_t* __restrict__ cursor) {
  const unsigned lane = threadIdx.x & 31u;
  const unsigned act = __activemask();                      // a prefix of the warp (i < n)
  const uint32_t kprev = __shfl_up_sync(act, k, 1);
  const unsigned heads = __ballot_sync(act, lane == 0u || kprev != k);
  const unsigned le = 0xffffffffu >> (31u - lane);          // lanes <= lane
  const int leader = 31 - __clz((int)(heads & le));
  const unsigned above = heads & ~le;
  const int end = above ? (__ffs((int)above) - 1) : __popc(act);
  uint32_t base = 0;
  if ((int)lane == leader) base = atomicAdd(&cursor[k], (uint32_t)(end - leader));
  base = __shfl_sync(act, base, leader);
  return base + (lane - (unsigned)leader);
}
// Canonical path, step 1: every particle takes a slot of its cell segment in arrival order
__global__ void __launch_bounds__(256) k_scatter_slots(size_t n, const uint32_t* __restrict__ key, const uint32_t* __restrict__ id,
                                                       const uint32_t* __restrict__ offset, uint32_t* __restrict__ cursor,
                                                       uint2* __restrict__ slot) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t k = key[i];
  const uint32_t s = offset[k] + run_slot(k, cursor);
  slot[s] = make_uint2(id[i], (uint32_t)i);   // one 8-byte store: (id, source index)
}
// Canonical path, step 2, one thread per slot: rank of the slot's particle inside its cell = number of cell mates
// with a smaller id (U4); perm[first slot of the cell + rank] = source index.
__global__ void __launch_bounds__(256) k_rank(size_t n, const uint32_t* __restrict__ key, const uint32_t* __restrict__ offset,
                                              const uint2* __restrict__ slot, uint32_t* __restrict__ perm) {
  const size_t s = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n) return;
  const uint2 me = slot[s];
  const uint32_t k = key[me.y];
  const uint32_t b = offset[k], e = offset[k + 1];
  uint32_t r = 0;
  for (uint32_t j = b; j < e; ++j) r += (slot[j].x < me.x) ? 1u : 0u;
  perm[b + r] = me.y;
}
// Hot-path variant (SRD) when no order is known yet: the order inside a cell does not enter the physics (integer
// cell sums), so the reorder only groups the particles by key: perm[slot] = source index, slots in arrival order
// from one cursor atomic per run of equal keys. Four independent particles per thread: the kernel is bound by the
// latency of the chain key load -> cursor atomic (with return) -> store.
constexpr int SCAT_U = 4;
__global__ void __launch_bounds__(256) k_scatter_src(size_t n, const uint32_t* __restrict__ key, const uint32_t* __restrict__ offset,
                                                     uint32_t* __restrict__ cursor, uint32_t* __restrict__ perm, int spread) {
  const size_t base = (size_t)blockIdx.x * (256 * SCAT_U) + threadIdx.x;
  const unsigned lane = threadIdx.x & 31u, le = 0xffffffffu >> (31u - lane);
  uint32_t k[SCAT_U], slot[SCAT_U];
  bool ok[SCAT_U];
  int leader[SCAT_U], len[SCAT_U];
#pragma unroll
  for (int j = 0; j < SCAT_U; ++j) {
    const size_t i = base + (size_t)j * 256;
    ok[j] = i < n;
    k[j] = ok[j] ? key[i] : 0u;
  }
#pragma unroll
  for (int j = 0; j < SCAT_U; ++j) {   // runs of equal keys among neighbouring lanes (run_slot, all 32 lanes take part)
    const uint32_t kprev = __shfl_up_sync(0xffffffffu, k[j], 1);
    const int okprev = __shfl_up_sync(0xffffffffu, (int)ok[j], 1);
    const unsigned heads = __ballot_sync(0xffffffffu, lane == 0u || kprev != k[j] || okprev != (int)ok[j]);
    leader[j] = 31 - __clz((int)(heads & le));
    const unsigned above = heads & ~le;
    len[j] = (above ? (__ffs((int)above) - 1) : 32) - leader[j];
  }
#pragma unroll
  for (int j = 0; j < SCAT_U; ++j) {
    slot[j] = 0;
    if (ok[j] && (int)lane == leader[j]) slot[j] = atomicAdd(&cursor[k[j]], (uint32_t)len[j]);
  }
  uint32_t off[SCAT_U];
#pragma unroll
  for (int j = 0; j < SCAT_U; ++j) off[j] = ok[j] ? offset[k[j]] : 0u;
#pragma unroll
  for (int j = 0; j < SCAT_U; ++j) {
    const uint32_t b = __shfl_sync(0xffffffffu, slot[j], leader[j]);
    if (ok[j]) perm[spread_key(offset, k[j], off[j] + b + (lane - (unsigned)leader[j]), spread)] = (uint32_t)(base + (size_t)j * 256);
  }
}

// The same, moving the particles at once (non-compact workspace): instead of a permutation for a 7-fold random 4-byte
// gather (k_gather<7>: 4.5 sectors of traffic per useful one, 208 ms at config 5), every particle is read where it is
// (coalesced) and written as ONE 32-byte record {r, v, id, 0} at its slot of the staging buffer (a full sector);
// k_unstage then copies the records back into the SoA arrays (coalesced both ways).
struct Soa7 { const uint32_t* p[7]; };
__global__ void __launch_bounds__(256) k_scatter_rec(size_t n, const uint32_t* __restrict__ key, const uint32_t* __restrict__ offset,
                                                     uint32_t* __restrict__ cursor, Soa7 src, float* __restrict__ aos, int spread) {
  const size_t base = (size_t)blockIdx.x * (256 * SCAT_U) + threadIdx.x;
  const unsigned lane = threadIdx.x & 31u, le = 0xffffffffu >> (31u - lane);
  uint32_t k[SCAT_U], slot[SCAT_U];
  bool ok[SCAT_U];
  int leader[SCAT_U], len[SCAT_U];
#pragma unroll
  for (int j = 0; j < SCAT_U; ++j) {
    const size_t i = base + (size_t)j * 256;
    ok[j] = i < n;
    k[j] = ok[j] ? key[i] : 0u;
  }
#pragma unroll
  for (int j = 0; j < SCAT_U; ++j) {   // runs of equal keys among neighbouring lanes (as in k_scatter_src)
    const uint32_t kprev = __shfl_up_sync(0xffffffffu, k[j], 1);
    const int okprev = __shfl_up_sync(0xffffffffu, (int)ok[j], 1);
    const unsigned heads = __ballot_sync(0xffffffffu, lane == 0u || kprev != k[j] || okprev != (int)ok[j]);
    leader[j] = 31 - __clz((int)(heads & le));
    const unsigned above = heads & ~le;
    len[j] = (above ? (__ffs((int)above) - 1) : 32) - leader[j];
  }
#pragma unroll
  for (int j = 0; j < SCAT_U; ++j) {
    slot[j] = 0;
    if (ok[j] && (int)lane == leader[j]) slot[j] = atomicAdd(&cursor[k[j]], (uint32_t)len[j]);
  }
  uint32_t off[SCAT_U];
#pragma unroll
  for (int j = 0; j < SCAT_U; ++j) off[j] = ok[j] ? offset[k[j]] : 0u;
#pragma unroll
  for (int j = 0; j < SCAT_U; ++j) {
    const uint32_t b = __shfl_sync(0xffffffffu, slot[j], leader[j]);
    if (!ok[j]) continue;
    const size_t i = base + (size_t)j * 256;
    const uint32_t d = spread_key(offset, k[j], off[j] + b + (lane - (unsigned)leader[j]), spread);
    const uint4 lo = make_uint4(src.p[0][i], src.p[1][i], src.p[2][i], src.p[3][i]);
    const uint4 hi = make_uint4(src.p[4][i], src.p[5][i], src.p[6][i], 0u);
    uint4* o = reinterpret_cast<uint4*>(aos + (size_t)d * 8);
    o[0] = lo; o[1] = hi;
  }
}
struct Soa7w { uint32_t* p[7]; };
__global__ void __launch_bounds__(256) k_unstage(size_t n, const float* __restrict__ aos, Soa7w dst) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint4* r = reinterpret_cast<const uint4*>(aos + i * 8);
  const uint4 lo = r[0], hi = r[1];
  dst.p[0][i] = lo.x; dst.p[1][i] = lo.y; dst.p[2][i] = lo.z; dst.p[3][i] = lo.w;
  dst.p[4][i] = hi.x; dst.p[5][i] = hi.y; dst.p[6][i] = hi.z;
}

// brick ranges of the old order, saved before the scan of a folded reorder overwrites the offsets: the scatter pass
// (k_sweep<.., IO_SCATTER>) still walks the old order
__global__ void __launch_bounds__(256) k_save_chunks(const uint32_t* __restrict__ offset, int bvol_shift, uint32_t nbricks,
                                                     uint32_t n, uint32_t* __restrict__ chunk0) {
  const uint32_t b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b < nbricks) chunk0[b] = offset[(size_t)b << bvol_shift];
  if (b == nbricks) chunk0[b] = n;
}
// one thread per cell: the particles of segment [offset[k], offset[k+1]) ranked by id
// (spread: the cell's particles sit at spread_slot() of the segment's positions)
__global__ void __launch_bounds__(256) k_rank_cells(size_t nkeys, const uint32_t* __restrict__ offset, const uint32_t* __restrict__ id,
                                                    uint32_t* __restrict__ perm, int spread, int inverse) {
  const size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= nkeys) return;
  const uint32_t b = offset[k], e = offset[k + 1];
  if (b == e) return;
  uint32_t g0 = 0, g1 = 0;               // R = 0: spread_slot is the identity
  if (spread) { const size_t kg = k & ~(((size_t)1 << spread) - 1); g0 = offset[kg]; g1 = offset[kg + ((size_t)1 << spread)]; }
  for (uint32_t j = b; j < e; ++j) {
    const uint32_t pj = spread_slot(j, g0, g1), me = id[pj];
    uint32_t r = 0;
    for (uint32_t m = b; m < e; ++m) r += (id[spread_slot(m, g0, g1)] < me) ? 1u : 0u;
    if (inverse) perm[pj] = b + r;      // where the particle at pj goes
    else perm[b + r] = pj;              // which particle comes to b + r
  }
}
// particle i goes to slot dest[i]: read where it is (coalesced), written as one 32-byte record (see k_scatter_rec)
__global__ void __launch_bounds__(256) k_move_rec(size_t n, const uint32_t* __restrict__ dest, Soa7 src, float* __restrict__ aos) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint4 lo = make_uint4(src.p[0][i], src.p[1][i], src.p[2][i], src.p[3][i]);
  const uint4 hi = make_uint4(src.p[4][i], src.p[5][i], src.p[6][i], 0u);
  uint4* o = reinterpret_cast<uint4*>(aos + (size_t)dest[i] * 8);
  o[0] = lo; o[1] = hi;
}
struct Arrays8 { void* p[8]; };
template <int NA>
__global__ void __launch_bounds__(256) k_gather(size_t n, const uint32_t* __restrict__ perm, Arrays8 src, Arrays8 dst) {
  const size_t d = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (d >= n) return;
  const uint32_t s = perm[d];
  uint32_t v[NA];
#pragma unroll
  for (int a = 0; a < NA; ++a) v[a] = ((const uint32_t*)src.p[a])[s];
#pragma unroll
  for (int a = 0; a < NA; ++a) ((uint32_t*)dst.p[a])[d] = v[a];
}

// Property-wise gather of the compact workspace when the particles already have an order: the particles
// that land in a group of 2^gsh consecutive keys (a brick or an aligned part of one) come almost all from the same group's range of
// the PREVIOUS order (old0, saved before the scan; a particle moves a fraction of a cell between two reorders). k_gather<1>
// asks L2 for one 32-byte sector per 4-byte element and is bound by that request rate; here a CTA reads its group's old range
// coalesced into shared memory once and gathers from there; the few sources outside the window are read from global memory.
// The window is brought in by the TMA engine (cp.async.bulk global -> shared, completion on an mbarrier; SASS: UBLKCP): no
// registers and no load instructions are spent on it, and with two CTAs per SM one CTA's copy runs under the other's gather.
// Bulk copies want 16-byte aligned addresses and sizes: the window starts at the old range's start rounded down to 4 elements and
// ends rounded up (the extra elements are particles of the neighbouring groups: valid sources like any other; the arrays are
// padded to 256 bytes and followed by the next array of the workspace, so reading up to 12 bytes past n is safe).
constexpr int GWIN_T = 512;
constexpr uint32_t GWIN_CHUNK = 32768;   // bytes per bulk copy
__global__ void __launch_bounds__(GWIN_T) k_gather_win(const uint32_t* __restrict__ perm, const uint32_t* __restrict__ src, uint32_t* __restrict__ dst,
                                                       const uint32_t* __restrict__ old0, const uint32_t* __restrict__ offset, int gsh, uint32_t cap) {
  extern __shared__ __align__(16) uint32_t win[];
  __shared__ __align__(8) unsigned long long bar;
  const uint32_t g = blockIdx.x;
  const uint32_t w0 = old0[g] & ~3u;
  const uint32_t wl = min((old0[g + 1] - w0 + 3u) & ~3u, cap & ~3u);
  const uint32_t bar_a = (uint32_t)__cvta_generic_to_shared(&bar), win_a = (uint32_t)__cvta_generic_to_shared(win);
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_a));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if (wl) {
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar_a), "r"(wl * 4u) : "memory");
      for (uint32_t o = 0; o < wl * 4u; o += GWIN_CHUNK) {
        const uint32_t bytes = min(GWIN_CHUNK, wl * 4u - o);
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"(win_a + o), "l"(reinterpret_cast<const char*>(src + w0) + o), "r"(bytes), "r"(bar_a) : "memory");
      }
    }
  }
  __syncthreads();   // the barrier is initialised (and armed) before anyone waits on it
  const uint32_t d0 = offset[(size_t)g << gsh], d1 = offset[((size_t)g + 1) << gsh];
  // GWIN_U independent index loads in flight per thread (one at a time left the kernel waiting on the latency of perm: 1024
  // threads x 4 bytes per SM against the ~35 KB the DRAM pipe wants); the first batch is on its way while the window arrives
  constexpr int GWIN_U = 8;
  uint32_t base = d0 + threadIdx.x;
  uint32_t sidx[GWIN_U];
#pragma unroll
  for (int k = 0; k < GWIN_U; ++k) { const uint32_t d = base + k * GWIN_T; sidx[k] = d < d1 ? perm[d] : 0u; }
  if (wl) {
    uint32_t done;
    do {
      asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\nselp.u32 %0, 1, 0, p;\n}" : "=r"(done) : "r"(bar_a) : "memory");
    } while (!done);
  }
  for (; base < d1; base += GWIN_U * GWIN_T) {
    uint32_t snext[GWIN_U];
    const uint32_t nb = base + GWIN_U * GWIN_T;
#pragma unroll
    for (int k = 0; k < GWIN_U; ++k) { const uint32_t d = nb + k * GWIN_T; snext[k] = d < d1 ? perm[d] : 0u; }
#pragma unroll
    for (int k = 0; k < GWIN_U; ++k) {
      const uint32_t d = base + k * GWIN_T;
      if (d < d1) {
        const uint32_t u = sidx[k] - w0;
        dst[d] = (u < wl) ? win[u] : src[sidx[k]];
      }
    }
#pragma unroll
    for (int k = 0; k < GWIN_U; ++k) sidx[k] = snext[k];
  }
}

__global__ void __launch_bounds__(256) k_iota(size_t n, uint32_t* __restrict__ id) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) id[i] = (uint32_t)i;
}

}  // namespace mpc

using namespace mpc;

int launch_iota(mpc_ctx* c) {
  k_iota<<<nblk(c->n_max ? c->n_max : 1, 256), 256, 0, c->stream>>>(c->n_max, c->A[6]);
  LAUNCH_CHECK("k_iota");
  return MPC_OK;
}

namespace {

// particle arrays gathered through c->perm: new[i] = old[perm[i]]
int apply_perm(mpc_ctx* c, bool windowed = false) {
  const size_t n = c->n;
  FamilyTimer ftg(c, F_GATHER);
  if (!c->compact) {
    Arrays8 src, dst;
    for (int a = 0; a < 7; ++a) { src.p[a] = c->A[a]; dst.p[a] = c->Bf[a]; }
    src.p[7] = dst.p[7] = nullptr;
    k_gather<7><<<nblk(n, 256), 256, 0, c->stream>>>(n, c->perm, src, dst);
    LAUNCH_CHECK("k_gather");
    for (int a = 0; a < 7; ++a) { uint32_t* t = c->A[a]; c->A[a] = c->Bf[a]; c->Bf[a] = t; }
  } else {
    // property-wise through one temporary array: each property is gathered into the spare array,
    // which then takes its place; the array it came from is the spare for the next property (no copy back)
    Arrays8 src, dst;
    for (int a = 0; a < 7; ++a) {
      uint32_t*& arr = c->A[a];
      src.p[0] = arr; dst.p[0] = c->Bf[0];
      if (windowed) {   // c->chunk0: the group ranges of the previous order (do_reorder), c->offset: those of the new one
        const size_t bytes = (size_t)c->gwin_cap * 4;
        if (a == 0) CU(cudaFuncSetAttribute(k_gather_win, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
        k_gather_win<<<c->G.nkeys >> c->gwin_shift, GWIN_T, bytes, c->stream>>>(c->perm, arr, c->Bf[0], c->chunk0, c->offset, c->gwin_shift, c->gwin_cap);
        LAUNCH_CHECK("k_gather_win");
      } else {
        k_gather<1><<<nblk(n, 256), 256, 0, c->stream>>>(n, c->perm, src, dst);
        LAUNCH_CHECK("k_gather");
      }
      uint32_t* t = arr; arr = c->Bf[0];
      for (int b = 0; b < 7; ++b) c->Bf[b] = t;     // compact mode: all seven alias the one spare array
    }
  }
  return MPC_OK;
}

}  // namespace

// counting-sort reorder by (key, id); counts = low word of word 0 of the sums
// folded: the sweep of this step was the rank pass (IO_RANK): only the scan is done here, the next two sweeps move the
//         particles (IO_SCATTER, IO_AOS_IN); otherwise c->key holds the keys and scatter + gather kernels run now
// canonical: rank the particles of a cell by id now (needed by MPC-AT); otherwise group by key only
int do_reorder(mpc_ctx* c, bool folded, bool canonical, bool counts_in_cursor) {
  const size_t n = c->n, nk = c->G.nkeys, nb = (nk + SCAN_TILE - 1) / SCAN_TILE;
  // counts_in_cursor: compact counts written by k_cell into c->cursor (the sums are already cleared); otherwise the low
  // 16 bits of word 0 of the sums
  const uint32_t* cnt = counts_in_cursor ? c->cursor : reinterpret_cast<const uint32_t*>(c->sums);
  const int stride = counts_in_cursor ? 1 : c->G.sw * 2;
  if (folded && !counts_in_cursor) return fail(c, MPC_ESTATE, "internal: folded reorder without compact counts");
  const int bvs = c->G.bs[0] + c->G.bs[1] + c->G.bs[2];
  if (folded && canonical) return fail(c, MPC_ESTATE, "internal: folded reorder cannot rank by id");
  // lane-spread order inside every group of 32 keys: hot path only, bricks of whole groups (spread_slot)
  const int gs = SPREAD_GROUP_SHIFT;
  const int spread = (!canonical && bvs >= gs && !(c->debug & MPC_DEBUG_NO_LANE_SPREAD)) ? gs : 0;
  if (folded) {   // the brick ranges of the old order, before the scan overwrites the offsets
    FamilyTimer ft(c, F_SCAN);
    k_save_chunks<<<nblk((size_t)c->nbricks + 1, 256), 256, 0, c->stream>>>(c->offset, bvs, c->nbricks, (uint32_t)n, c->chunk0);
    LAUNCH_CHECK("k_save_chunks");
  }
  // compact workspace with a previous order: the gather goes through shared-memory windows (k_gather_win) and needs the
  // previous order's group ranges (MPC_DEBUG_NO_FUSE_GATHER: the plain element-wise gather, same result)
  const bool windowed = c->compact && !folded && !canonical && c->have_order && c->chunk0 && c->gwin_shift > 0 && n != 0 &&
                        !(c->debug & MPC_DEBUG_NO_FUSE_GATHER);
  if (windowed) {
    FamilyTimer ft(c, F_SCAN);
    const uint32_t ng = c->G.nkeys >> c->gwin_shift;
    k_save_chunks<<<nblk((size_t)ng + 1, 256), 256, 0, c->stream>>>(c->offset, c->gwin_shift, ng, (uint32_t)n, c->chunk0);
    LAUNCH_CHECK("k_save_chunks");
  }
  {
    FamilyTimer ft(c, F_SCAN);
    k_scan_reduce<<<(unsigned)nb, SCAN_T, 0, c->stream>>>(cnt, stride, nk, c->bsum);
    LAUNCH_CHECK("k_scan_reduce");
    k_scan_top<<<1, 1024, 0, c->stream>>>(c->bsum, nb);
    LAUNCH_CHECK("k_scan_top");
    k_scan_apply<<<(unsigned)nb, SCAN_T, 0, c->stream>>>(cnt, stride, nk, c->bsum, c->offset);
    LAUNCH_CHECK("k_scan_apply");
  }
  if (!folded && n == 0) {   // a slab rank without particles: the offsets (all zero) are what its neighbours and its next reorder need
    c->have_order = true;
    c->order_canonical = canonical;
    c->order_spread = spread;
    return MPC_OK;
  }
  if (!folded) {
    { FamilyTimer ft(c, F_MEMSET); CU(cudaMemsetAsync(c->cursor, 0, nk * 4, c->stream)); }
    if (canonical) {
      uint2* slot2 = reinterpret_cast<uint2*>(c->compact ? c->slot_id : c->Bf[0]);
      {
        FamilyTimer ft(c, F_SCATTER);
        k_scatter_slots<<<nblk(n, 256), 256, 0, c->stream>>>(n, c->key, c->A[6], c->offset, c->cursor, slot2);
        LAUNCH_CHECK("k_scatter_slots");
      }
      FamilyTimer ft(c, F_RANK);
      k_rank<<<nblk(n, 256), 256, 0, c->stream>>>(n, c->key, c->offset, slot2, c->perm);
      LAUNCH_CHECK("k_rank");
    } else if (!c->compact) {   // group by key and move at once, through 32-byte records
      {
        FamilyTimer ft(c, F_SCATTER);
        Soa7 src;
        for (int a = 0; a < 7; ++a) src.p[a] = c->A[a];
        k_scatter_rec<<<nblk(n, 256 * SCAT_U), 256, 0, c->stream>>>(n, c->key, c->offset, c->cursor, src, aos_base(c), spread);
        LAUNCH_CHECK("k_scatter_rec");
      }
      FamilyTimer ft(c, F_GATHER);
      Soa7w dst;
      for (int a = 0; a < 7; ++a) dst.p[a] = c->A[a];
      k_unstage<<<nblk(n, 256), 256, 0, c->stream>>>(n, aos_base(c), dst);
      LAUNCH_CHECK("k_unstage");
      c->have_order = true;
      c->order_canonical = false;
      c->order_spread = spread;
      return MPC_OK;
    } else {
      FamilyTimer ft(c, F_SCATTER);
      k_scatter_src<<<nblk(n, 256 * SCAT_U), 256, 0, c->stream>>>(n, c->key, c->offset, c->cursor, c->perm, spread);
      LAUNCH_CHECK("k_scatter_src");
    }
  }
  c->have_order = true;
  c->order_canonical = canonical;
  c->order_spread = spread;
  if (folded) { c->reorder_stage = 1; return MPC_OK; }
  return apply_perm(c, windowed);
}

// restore the canonical (key, id) order inside the cell segments of the last reorder (U4); called
// before the state is read when the hot path has left the particles grouped by key only
int canonicalise(mpc_ctx* c) {
  if (!c->have_order || c->order_canonical || c->n == 0) return MPC_OK;
  {
    FamilyTimer ft(c, F_RANK);
    k_rank_cells<<<nblk(c->G.nkeys, 256), 256, 0, c->stream>>>(c->G.nkeys, c->offset, c->A[6], c->perm, c->order_spread, c->compact ? 0 : 1);
    LAUNCH_CHECK("k_rank_cells");
  }
  int rc = MPC_OK;
  if (c->compact) rc = apply_perm(c);
  else {   // through 32-byte records instead of a 7-fold random gather
    FamilyTimer ftg(c, F_GATHER);
    Soa7 src; Soa7w dst;
    for (int a = 0; a < 7; ++a) { src.p[a] = c->A[a]; dst.p[a] = c->A[a]; }
    k_move_rec<<<nblk(c->n, 256), 256, 0, c->stream>>>(c->n, c->perm, src, aos_base(c));
    LAUNCH_CHECK("k_move_rec");
    k_unstage<<<nblk(c->n, 256), 256, 0, c->stream>>>(c->n, aos_base(c), dst);
    LAUNCH_CHECK("k_unstage");
  }
  if (rc == MPC_OK) { c->order_canonical = true; c->order_spread = 0; }
  return rc;
}
