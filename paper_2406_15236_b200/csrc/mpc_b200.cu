// mpc_b200.cu -- B200 (sm_100a) implementation of the MPC fluid step behind include/mpc_b200.h.
//
// One CUDA stream, no host synchronisation inside mpc_step. Kernel families:
//   k_stream_key   MOVE + shift + cell key (+ histogram on reorder steps)
//   k_scan_*       exclusive prefix sum of the per-cell histogram
//   k_scatter_ids / k_rank / k_gather   counting-sort reorder by (key, id)
//   k_accum        per-cell sums in 32-bit fixed point (order-independent)
//   k_cell         v_cm, axis, kappa, virtual wall particles
//   k_collide      rotation / MPC-AT applied to every particle                   Eqs. (2)-(5)
//   k_obs_*        observables
// Compile with --fmad=false: every multiply-add that must fuse is an explicit fmaf (U1).
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include <new>

#include "../../include/mpc_b200.h"
#include "philox.cuh"

namespace mpc {

// ------------------------------------------------------------------------------------------------
// fixed-point cell sums (the paper's reproducibility option): integer atomics make
// the sums independent of the order of arrival, so a run is bit-reproducible.
// Scales are powers of two relative to the thermal velocity u = 2^round(log2 sqrt(kT/m)), so the
// conversion is exact up to the final rounding and the precision does not depend on the unit system:
//   velocity sums : 2^20 / u    ->  |sum v_d|  < 2048 u      (resolution 9.5e-7 u)
//   energy sums   : 2^18 / u^2  ->  sum |v|^2  < 16384 u^2   (resolution 3.8e-6 u^2)
constexpr int SUMS_W = 8;                   // ints per cell (32 B, one sector)
constexpr int REC_W = 8;                    // floats per cell record (32 B, one sector)
constexpr int OBS_BLOCKS = 1184;            // 148 SMs x 8
constexpr int MAX_PROFILE = 2048;
constexpr size_t OBS_HOST_DOUBLES = (size_t)OBS_BLOCKS * 8 + 2 * MAX_PROFILE;

struct Geo {
  float L[3];
  float a, inv_a;
  int n[3];       // fluid cells
  int m[3];       // cell layers incl. wall layers
  int mb[3];      // bricks per axis
  int bshift;     // log2(brick edge)
  int bc[3];
  int wall;       // wall axis or -1
  float g[3];
  float dt;
  float s[3];     // lattice shift of this step
  uint32_t k0, k1, t;
  float cosa, sina;
  float kT, mass, sigma;   // sigma = sqrt(kT/m)
  float fxv, fxe;          // fixed-point scales (powers of two)
  double fxv_inv, fxe_inv;
  int nbar;
  int collision, thermostat;
  uint32_t nkeys;
};

// ---- geometry helpers ----------------------------------------------------------------------------
__device__ __forceinline__ uint32_t layout_key(const Geo& G, int ix, int iy, int iz) {
  const int b = G.bshift, mask = (1 << b) - 1;
  const uint32_t brick = ((uint32_t)(iz >> b) * (uint32_t)G.mb[1] + (uint32_t)(iy >> b)) * (uint32_t)G.mb[0] + (uint32_t)(ix >> b);
  const uint32_t local = ((((uint32_t)(iz & mask)) << b | (uint32_t)(iy & mask)) << b) | (uint32_t)(ix & mask);
  return (brick << (3 * b)) | local;
}
__device__ __forceinline__ void key_to_cell(const Geo& G, uint32_t key, int& ix, int& iy, int& iz) {
  const int b = G.bshift;
  const uint32_t mask = (1u << b) - 1u;
  const uint32_t local = key & ((1u << (3 * b)) - 1u), brick = key >> (3 * b);
  const uint32_t bx = brick % (uint32_t)G.mb[0], r = brick / (uint32_t)G.mb[0];
  const uint32_t by = r % (uint32_t)G.mb[1], bz = r / (uint32_t)G.mb[1];
  ix = (int)((bx << b) | (local & mask));
  iy = (int)((by << b) | ((local >> b) & mask));
  iz = (int)((bz << b) | (local >> (2 * b)));
}
__device__ __forceinline__ uint32_t canonical_id(const Geo& G, int ix, int iy, int iz) {
  return (uint32_t)ix + (uint32_t)G.m[0] * ((uint32_t)iy + (uint32_t)G.m[1] * (uint32_t)iz);
}
// cell coordinate along one axis; rho = cell-local coordinate in [0,1)
__device__ __forceinline__ int cell_coord(const Geo& G, int d, float r, float& rho) {
  const float q = (r + G.s[d]) * G.inv_a;
  const float f = floorf(q);
  int k = (int)f;
  if (G.bc[d] == 0) {
    if (k < 0) k += G.n[d];
    if (k >= G.n[d]) k -= G.n[d];
  } else {
    k += 1;
    k = max(0, min(k, G.n[d] + 1));
  }
  rho = q - f;
  return k;
}
__device__ __forceinline__ uint32_t key_of(const Geo& G, float x, float y, float z) {
  float r0, r1, r2;
  const int ix = cell_coord(G, 0, x, r0), iy = cell_coord(G, 1, y, r1), iz = cell_coord(G, 2, z, r2);
  return layout_key(G, ix, iy, iz);
}

// ---- MOVE ----------------------------------------------------------------------------------------
template <bool GRAV>
__device__ __forceinline__ void advance(const Geo& G, float (&r)[3], float (&v)[3], float tau) {
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    if (GRAV && G.g[d] != 0.0f) {
      const float vh = fmaf(0.5f * tau, G.g[d], v[d]);
      r[d] = fmaf(vh, tau, r[d]);
      v[d] = fmaf(tau, G.g[d], v[d]);
    } else {
      r[d] = fmaf(v[d], tau, r[d]);
    }
  }
}
template <bool WALL, bool GRAV>
__device__ __forceinline__ void stream_one(const Geo& G, float (&r)[3], float (&v)[3]) {
  bool bounced = false;
  if (WALL) {
    const int w = G.wall;
    const float rw = (w == 0) ? r[0] : (w == 1) ? r[1] : r[2];
    const float vw = (w == 0) ? v[0] : (w == 1) ? v[1] : v[2];
    const float Lw = (w == 0) ? G.L[0] : (w == 1) ? G.L[1] : G.L[2];
    const float z1 = fmaf(vw, G.dt, rw);
    if (z1 < 0.0f || z1 > Lw) {
      const float zw = (z1 < 0.0f) ? 0.0f : Lw;
      float tc = (zw - rw) / vw;
      tc = fminf(fmaxf(tc, 0.0f), G.dt);
      advance<GRAV>(G, r, v, tc);
      if (w == 0) r[0] = zw; else if (w == 1) r[1] = zw; else r[2] = zw;
      v[0] = -v[0]; v[1] = -v[1]; v[2] = -v[2];
      advance<GRAV>(G, r, v, G.dt - tc);
      if (w == 0) r[0] = fminf(fmaxf(r[0], 0.0f), Lw);
      else if (w == 1) r[1] = fminf(fmaxf(r[1], 0.0f), Lw);
      else r[2] = fminf(fmaxf(r[2], 0.0f), Lw);
      bounced = true;
    }
  }
  if (!bounced) advance<GRAV>(G, r, v, G.dt);
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    if (WALL && G.bc[d] != 0) continue;
    if (r[d] < 0.0f) r[d] += G.L[d];
    if (r[d] >= G.L[d]) r[d] -= G.L[d];
  }
}

template <bool WALL, bool GRAV>
__global__ void __launch_bounds__(256) k_stream_key(Geo G, size_t n, float* __restrict__ x, float* __restrict__ y,
                                                    float* __restrict__ z, float* __restrict__ vx, float* __restrict__ vy,
                                                    float* __restrict__ vz, uint32_t* __restrict__ key,
                                                    uint32_t* __restrict__ hist) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float r[3] = {x[i], y[i], z[i]}, v[3] = {vx[i], vy[i], vz[i]};
  stream_one<WALL, GRAV>(G, r, v);
  x[i] = r[0]; y[i] = r[1]; z[i] = r[2];
  if (WALL || GRAV) { vx[i] = v[0]; vy[i] = v[1]; vz[i] = v[2]; }
  const uint32_t k = key_of(G, r[0], r[1], r[2]);
  key[i] = k;
  if (hist) atomicAdd(&hist[k], 1u);
}

// ---- exclusive scan of uint32 (three kernels; tile = 2048) --------------------------------------
constexpr int SCAN_T = 256, SCAN_PER = 8, SCAN_TILE = SCAN_T * SCAN_PER;

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
    wsum[lane] = winc - w;          // exclusive offset of every warp
    if (lane == 31) wsum[32] = winc;  // block total
  }
  __syncthreads();
  const uint32_t res = wsum[warp] + inc - v;
  total = wsum[32];
  __syncthreads();                  // wsum is reused by the caller's next round
  return res;
}

__global__ void __launch_bounds__(SCAN_T) k_scan_reduce(const uint32_t* __restrict__ in, size_t n, uint32_t* __restrict__ bsum) {
  const size_t base = (size_t)blockIdx.x * SCAN_TILE;
  uint32_t s = 0;
#pragma unroll
  for (int j = 0; j < SCAN_PER; ++j) {
    const size_t i = base + (size_t)j * SCAN_T + threadIdx.x;
    if (i < n) s += in[i];
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
__global__ void __launch_bounds__(SCAN_T) k_scan_apply(const uint32_t* __restrict__ in, size_t n, const uint32_t* __restrict__ bsum,
                                                       uint32_t* __restrict__ out) {
  const size_t base = (size_t)blockIdx.x * SCAN_TILE + (size_t)threadIdx.x * SCAN_PER;
  uint32_t v[SCAN_PER], s = 0;
#pragma unroll
  for (int j = 0; j < SCAN_PER; ++j) {
    v[j] = (base + j < n) ? in[base + j] : 0u;
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

// ---- reorder by (key, id) -----------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_scatter_ids(size_t n, const uint32_t* __restrict__ key, const uint32_t* __restrict__ id,
                                                     const uint32_t* __restrict__ offset, uint32_t* __restrict__ cursor,
                                                     uint32_t* __restrict__ slot_id) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t k = key[i];
  const uint32_t s = offset[k] + atomicAdd(&cursor[k], 1u);
  slot_id[s] = id[i];
}
// rank of a particle inside its cell = number of cell mates with a smaller id (U4)
__global__ void __launch_bounds__(256) k_rank(size_t n, const uint32_t* __restrict__ key, const uint32_t* __restrict__ id,
                                              const uint32_t* __restrict__ offset, const uint32_t* __restrict__ slot_id,
                                              uint32_t* __restrict__ perm) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t k = key[i], me = id[i];
  const uint32_t b = offset[k], e = offset[k + 1];
  uint32_t r = 0;
  for (uint32_t j = b; j < e; ++j) r += (slot_id[j] < me) ? 1u : 0u;
  perm[b + r] = (uint32_t)i;
}
struct Arrays8 { void* p[8]; };
__global__ void __launch_bounds__(256) k_gather8(size_t n, const uint32_t* __restrict__ perm, Arrays8 src, Arrays8 dst) {
  const size_t d = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (d >= n) return;
  const uint32_t s = perm[d];
  uint32_t v[8];
#pragma unroll
  for (int a = 0; a < 8; ++a) v[a] = ((const uint32_t*)src.p[a])[s];
#pragma unroll
  for (int a = 0; a < 8; ++a) ((uint32_t*)dst.p[a])[d] = v[a];
}
__global__ void __launch_bounds__(256) k_gather1(size_t n, const uint32_t* __restrict__ perm, const uint32_t* __restrict__ src,
                                                 uint32_t* __restrict__ dst) {
  const size_t d = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (d >= n) return;
  dst[d] = src[perm[d]];
}
__global__ void __launch_bounds__(256) k_iota(size_t n, uint32_t* __restrict__ id) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) id[i] = (uint32_t)i;
}

// ---- PROCESS: per-cell sums ----------------------------------------------------------------------
// sums[key] = { N, Sx, Sy, Sz, E | R0, R1, R2 (MPC-AT) }
template <bool AT>
__global__ void __launch_bounds__(256) k_accum(Geo G, size_t n, const float* __restrict__ vx, const float* __restrict__ vy,
                                               const float* __restrict__ vz, const uint32_t* __restrict__ key,
                                               const uint32_t* __restrict__ offset, int* __restrict__ sums) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t k = key[i];
  const float a = vx[i], b = vy[i], c = vz[i];
  int* s = sums + (size_t)k * SUMS_W;
  atomicAdd((unsigned*)s, 1u);
  atomicAdd(s + 1, __float2int_rn(a * G.fxv));
  atomicAdd(s + 2, __float2int_rn(b * G.fxv));
  atomicAdd(s + 3, __float2int_rn(c * G.fxv));
  if (!AT) {
    const float e = fmaf(a, a, fmaf(b, b, c * c));
    atomicAdd((unsigned*)(s + 4), __float2uint_rn(e * G.fxe));
  } else {
    int ix, iy, iz;
    key_to_cell(G, k, ix, iy, iz);
    const uint32_t rank = (uint32_t)i - offset[k];
    const Block4 o = philox(canonical_id(G, ix, iy, iz), rank, G.t, TAG_AT, G.k0, G.k1);
    float g0, g1, g2;
    normals3(o, g0, g1, g2);
    atomicAdd(s + 5, __float2int_rn(G.sigma * g0 * G.fxv));
    atomicAdd(s + 6, __float2int_rn(G.sigma * g1 * G.fxv));
    atomicAdd(s + 7, __float2int_rn(G.sigma * g2 * G.fxv));
  }
}

// ---- PROCESS_CELLS -------------------------------------------------------------------------------
// E_k / k_BT ~ Gamma(3(Nc-1)/2, 1): floor(f/2) unit exponentials (+ half a squared normal if f is odd)
__device__ float mbs_energy(const Geo& G, uint32_t cid, uint32_t Nc) {
  const uint32_t f = 3u * (Nc - 1u), M = f >> 1, odd = f & 1u;
  const uint32_t need = M + 2u * odd;
  float e = 0.0f, lg = 0.0f, cs = 0.0f;
  uint32_t sub = 0;
  for (uint32_t base = 0; base < need; base += 4, ++sub) {
    const Block4 o = philox(cid, sub, G.t, TAG_MBS, G.k0, G.k1);
    const uint32_t w[4] = {o.a, o.b, o.c, o.d};
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const uint32_t pos = base + q;
      if (pos < M) e -= logf(u01_oc(w[q]));
      else if (odd && pos == M) lg = -logf(u01_oc(w[q]));
      else if (odd && pos == M + 1u) cs = cospif(2.0f * u01_co(w[q]));
    }
  }
  if (odd) e += lg * cs * cs;
  return e;
}

// rec[key] = SRD: { vcm.x, vcm.y, vcm.z, kappa, n.x, n.y, n.z, - }   AT: { (vcm - mean v_ran).xyz, ... }
__global__ void __launch_bounds__(128) k_cell(Geo G, const int* __restrict__ sums, float* __restrict__ rec) {
  const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= G.nkeys) return;
  const int4 s0 = reinterpret_cast<const int4*>(sums)[(size_t)k * 2];
  const uint32_t nreal = (uint32_t)s0.x;
  if (nreal == 0u) return;
  const int4 s1 = reinterpret_cast<const int4*>(sums)[(size_t)k * 2 + 1];
  int ix, iy, iz;
  key_to_cell(G, k, ix, iy, iz);
  const uint32_t cid = canonical_id(G, ix, iy, iz);
  double S0 = (double)s0.y * G.fxv_inv, S1 = (double)s0.z * G.fxv_inv, S2 = (double)s0.w * G.fxv_inv;
  float4 r0, r1;
  if (G.collision == 1) {
    const double inv = 1.0 / (double)nreal;
    r0.x = (float)((S0 - (double)s1.y * G.fxv_inv) * inv);
    r0.y = (float)((S1 - (double)s1.z * G.fxv_inv) * inv);
    r0.z = (float)((S2 - (double)s1.w * G.fxv_inv) * inv);
    r0.w = 1.0f;
    r1 = make_float4(0.f, 0.f, 0.f, 0.f);
  } else {
    double E = (double)(uint32_t)s1.x * G.fxe_inv;
    uint32_t Nc = nreal;
    if (G.wall >= 0) {
      // virtual wall particles fill wall-cut cells up to nbar (U8)
      const int w = G.wall;
      const int iw = (w == 0) ? ix : (w == 1) ? iy : iz;
      const float sw = (w == 0) ? G.s[0] : (w == 1) ? G.s[1] : G.s[2];
      const int nw = (w == 0) ? G.n[0] : (w == 1) ? G.n[1] : G.n[2];
      const bool cut = (sw > 0.0f) ? (iw == 1 || iw == nw + 1) : (sw < 0.0f) ? (iw == 0 || iw == nw) : false;
      if (cut && (int)nreal < G.nbar) {
        const uint32_t nv = (uint32_t)G.nbar - nreal;
        for (uint32_t j = 0; j < nv; ++j) {
          const Block4 o = philox(cid, j, G.t, TAG_WALL, G.k0, G.k1);
          float g0, g1, g2;
          normals3(o, g0, g1, g2);
          const double a = (double)(G.sigma * g0), b = (double)(G.sigma * g1), c = (double)(G.sigma * g2);
          S0 += a; S1 += b; S2 += c; E += a * a + b * b + c * c;
        }
        Nc += nv;
      }
    }
    const double inv = 1.0 / (double)Nc;
    r0.x = (float)(S0 * inv); r0.y = (float)(S1 * inv); r0.z = (float)(S2 * inv);
    float kappa = 1.0f;
    if (G.thermostat && Nc >= 2u) {
      const double W2 = E - (S0 * S0 + S1 * S1 + S2 * S2) * inv;   // sum |v - vcm|^2
      if (W2 > 0.0) {
        const float ek = G.kT * mbs_energy(G, cid, Nc);
        kappa = sqrtf(2.0f * ek / (G.mass * (float)W2));
      }
    }
    r0.w = kappa;
    const Block4 o = philox(cid, 0u, G.t, TAG_AXIS, G.k0, G.k1);
    const float zz = 2.0f * u01_co(o.a) - 1.0f;
    const float rr = sqrtf((1.0f - zz) * (1.0f + zz));
    float sp, cp;
    sincospif(2.0f * u01_co(o.b), &sp, &cp);
    r1 = make_float4(rr * cp, rr * sp, zz, 0.0f);
  }
  reinterpret_cast<float4*>(rec)[(size_t)k * 2] = r0;
  reinterpret_cast<float4*>(rec)[(size_t)k * 2 + 1] = r1;
}

// ---- ROTATE_VELOCITIES ---------------------------------------------------------------------------
template <bool AT>
__global__ void __launch_bounds__(256) k_collide(Geo G, size_t n, float* __restrict__ vx, float* __restrict__ vy,
                                                 float* __restrict__ vz, const uint32_t* __restrict__ key,
                                                 const uint32_t* __restrict__ offset, const float* __restrict__ rec) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t k = key[i];
  const float4 r0 = __ldg(reinterpret_cast<const float4*>(rec) + (size_t)k * 2);
  if (AT) {
    int ix, iy, iz;
    key_to_cell(G, k, ix, iy, iz);
    const uint32_t rank = (uint32_t)i - offset[k];
    const Block4 o = philox(canonical_id(G, ix, iy, iz), rank, G.t, TAG_AT, G.k0, G.k1);
    float g0, g1, g2;
    normals3(o, g0, g1, g2);
    vx[i] = r0.x + G.sigma * g0;
    vy[i] = r0.y + G.sigma * g1;
    vz[i] = r0.z + G.sigma * g2;
  } else {
    const float4 ax = __ldg(reinterpret_cast<const float4*>(rec) + (size_t)k * 2 + 1);
    const float w0 = vx[i] - r0.x, w1 = vy[i] - r0.y, w2 = vz[i] - r0.z;
    const float c = G.cosa, s = G.sina, omc = 1.0f - G.cosa;
    const float nd = fmaf(ax.x, w0, fmaf(ax.y, w1, ax.z * w2)) * omc;
    const float cx = fmaf(ax.y, w2, -(ax.z * w1)), cy = fmaf(ax.z, w0, -(ax.x * w2)), cz = fmaf(ax.x, w1, -(ax.y * w0));
    const float o0 = fmaf(w0, c, fmaf(cx, s, ax.x * nd));
    const float o1 = fmaf(w1, c, fmaf(cy, s, ax.y * nd));
    const float o2 = fmaf(w2, c, fmaf(cz, s, ax.z * nd));
    vx[i] = fmaf(r0.w, o0, r0.x);
    vy[i] = fmaf(r0.w, o1, r0.y);
    vz[i] = fmaf(r0.w, o2, r0.z);
  }
}

// ---- observables ---------------------------------------------------------------------------------
__device__ __forceinline__ double block_sum(double v, double* sh) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
  __syncthreads();
  double t = 0.0;
  if (threadIdx.x == 0) for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += sh[w];
  __syncthreads();
  return t;
}
__global__ void __launch_bounds__(256) k_obs_particles(size_t n, const float* __restrict__ vx, const float* __restrict__ vy,
                                                       const float* __restrict__ vz, double* __restrict__ part) {
  __shared__ double sh[8];
  double a = 0, b = 0, c = 0, e = 0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const double p = vx[i], q = vy[i], r = vz[i];
    a += p; b += q; c += r; e += p * p + q * q + r * r;
  }
  a = block_sum(a, sh); b = block_sum(b, sh); c = block_sum(c, sh); e = block_sum(e, sh);
  if (threadIdx.x == 0) { double* o = part + (size_t)blockIdx.x * 8; o[0] = a; o[1] = b; o[2] = c; o[3] = e; }
}
__global__ void __launch_bounds__(256) k_obs_cells(Geo G, const int* __restrict__ sums, double* __restrict__ part) {
  __shared__ double sh[8];
  __shared__ unsigned smax;
  if (threadIdx.x == 0) smax = 0;
  __syncthreads();
  double num = 0, den = 0;
  unsigned mx = 0;
  for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < G.nkeys; k += (size_t)gridDim.x * blockDim.x) {
    const int4 s0 = reinterpret_cast<const int4*>(sums)[k * 2];
    const unsigned nc = (unsigned)s0.x;
    mx = max(mx, nc);
    if (nc < 2u) continue;
    const unsigned e = (unsigned)sums[k * SUMS_W + 4];
    const double S0 = s0.y * G.fxv_inv, S1 = s0.z * G.fxv_inv, S2 = s0.w * G.fxv_inv;
    num += (double)G.mass * ((double)e * G.fxe_inv - (S0 * S0 + S1 * S1 + S2 * S2) / nc);
    den += 3.0 * (nc - 1u);
  }
  atomicMax(&smax, mx);
  num = block_sum(num, sh); den = block_sum(den, sh);
  if (threadIdx.x == 0) { double* o = part + (size_t)blockIdx.x * 8; o[4] = num; o[5] = den; o[6] = (double)smax; }
}
__global__ void __launch_bounds__(256) k_obs_profile(Geo G, size_t n, int pa, int nb, const float* __restrict__ rp,
                                                     const float* __restrict__ vf, double* __restrict__ prof) {
  extern __shared__ double bins[];   // nb sums, nb counts
  for (int b = threadIdx.x; b < 2 * nb; b += blockDim.x) bins[b] = 0.0;
  __syncthreads();
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    int b = (int)floorf(rp[i] * G.inv_a);
    b = max(0, min(b, nb - 1));
    atomicAdd(&bins[b], (double)vf[i]);
    atomicAdd(&bins[nb + b], 1.0);
  }
  __syncthreads();
  for (int b = threadIdx.x; b < 2 * nb; b += blockDim.x) if (bins[b] != 0.0) atomicAdd(&prof[b], bins[b]);
}
template <bool AT>
__global__ void __launch_bounds__(256) k_export_cells(Geo G, const int* __restrict__ sums, unsigned* __restrict__ count,
                                                      float* __restrict__ px, float* __restrict__ py, float* __restrict__ pz,
                                                      float* __restrict__ e2) {
  const size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= G.nkeys) return;
  const int* s = sums + k * SUMS_W;
  if (count) count[k] = (unsigned)s[0];
  if (px) px[k] = (float)((double)G.mass * s[1] * G.fxv_inv);
  if (py) py[k] = (float)((double)G.mass * s[2] * G.fxv_inv);
  if (pz) pz[k] = (float)((double)G.mass * s[3] * G.fxv_inv);
  if (e2) e2[k] = AT ? 0.0f : (float)((double)(unsigned)s[4] * G.fxe_inv);
}

}  // namespace mpc

// =================================================================================================
// host side
// =================================================================================================
using namespace mpc;

enum Family { F_STREAM = 0, F_SCAN, F_SCATTER, F_RANK, F_GATHER, F_ACCUM, F_CELL, F_COLLIDE, F_MEMSET, F_OBS, F_COUNT };
static const char* const FAMILY_NAMES[F_COUNT] = {"stream_key", "scan", "scatter_ids", "rank", "gather", "accum", "cell",
                                                  "collide", "memset", "observables"};
constexpr int PROF_MAX_PAIRS = 16384;

struct mpc_ctx {
  Geo G;
  mpc_params p;
  float box[3];
  int cells[3];
  unsigned long long seed;
  uint32_t t;
  size_t n, n_max;
  bool bound, have_state, have_cells, compact, sticky;
  cudaStream_t stream;
  char* ws;
  size_t ws_bytes;
  // device arrays
  uint32_t* A[8];   // x y z vx vy vz id key (current)
  uint32_t* Bf[8];  // second copy (non-compact) ; Bf[0] = 4-byte temp (compact)
  uint32_t *slot_id, *perm, *hist, *offset, *bsum;
  int* sums;
  float* rec;
  double* obs;      // OBS_BLOCKS*8 doubles + 2*MAX_PROFILE doubles
  double* hbuf;     // host staging for mpc_observables
  // optional per-family timing with CUDA events on the bound stream (mpc_profile_*)
  bool prof_on;
  cudaEvent_t* prof_ev;          // 2 * PROF_MAX_PAIRS events, created on first enable
  int* prof_fam;                 // family of every recorded pair
  int prof_pairs;
  double prof_ms[F_COUNT];
  unsigned long long prof_launches[F_COUNT];
  unsigned long long launches;
  char err[256];
};

namespace {

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Layout {
  size_t off_A[8], off_B[8], off_slot, off_perm, off_hist, off_offset, off_bsum, off_sums, off_rec, off_obs, total;
};
Layout make_layout(size_t n_max, size_t nkeys, bool compact) {
  Layout l;
  size_t o = 0;
  auto take = [&](size_t bytes) { const size_t r = o; o = align_up(o + bytes, 256); return r; };
  const size_t pn = (n_max ? n_max : 1) * 4;
  for (int a = 0; a < 8; ++a) l.off_A[a] = take(pn);
  if (compact) { l.off_B[0] = take(pn); for (int a = 1; a < 8; ++a) l.off_B[a] = l.off_B[0]; }
  else for (int a = 0; a < 8; ++a) l.off_B[a] = take(pn);
  l.off_slot = take(pn);
  l.off_perm = take(pn);
  l.off_hist = take(nkeys * 4);
  l.off_offset = take((nkeys + 1) * 4);
  l.off_bsum = take(((nkeys + SCAN_TILE - 1) / SCAN_TILE + 1) * 4);
  l.off_sums = take(nkeys * SUMS_W * 4);
  l.off_rec = take(nkeys * REC_W * 4);
  l.off_obs = take((size_t)OBS_BLOCKS * 8 * 8 + (size_t)2 * MAX_PROFILE * 8);
  l.total = o;
  return l;
}

int fail(mpc_ctx* c, int code, const char* msg) {
  if (c) snprintf(c->err, sizeof(c->err), "%s", msg);
  return code;
}
int cuda_fail(mpc_ctx* c, cudaError_t e, const char* where) {
  if (c) { snprintf(c->err, sizeof(c->err), "%s: %s", where, cudaGetErrorString(e)); c->sticky = true; }
  return MPC_ECUDA;
}
struct FamilyTimer {   // records an event pair around the launches of one kernel family
  mpc_ctx* c; int slot;
  FamilyTimer(mpc_ctx* c_, int fam) : c(c_), slot(-1) {
    if (!c->prof_on) return;
    c->prof_launches[fam]++;
    if (c->prof_pairs >= PROF_MAX_PAIRS) return;
    slot = c->prof_pairs++;
    c->prof_fam[slot] = fam;
    cudaEventRecord(c->prof_ev[2 * slot], c->stream);
  }
  ~FamilyTimer() { if (slot >= 0) cudaEventRecord(c->prof_ev[2 * slot + 1], c->stream); }
};
#define CU(call)                                                 \
  do {                                                           \
    cudaError_t e_ = (call);                                     \
    if (e_ != cudaSuccess) return cuda_fail(c, e_, #call);       \
  } while (0)
#define LAUNCH_CHECK(name)                                       \
  do {                                                           \
    c->launches++;                                               \
    cudaError_t e_ = cudaGetLastError();                         \
    if (e_ != cudaSuccess) return cuda_fail(c, e_, name);        \
  } while (0)

inline unsigned nblk(size_t n, int t) { return (unsigned)((n + t - 1) / t); }

void host_shift(const mpc_ctx* c, uint32_t t, float s[3]) {
  s[0] = s[1] = s[2] = 0.0f;
  if (!c->p.grid_shift) return;
  const Block4 o = philox(0u, 0u, t, TAG_SHIFT, c->G.k0, c->G.k1);
  s[0] = (u01_co(o.a) - 0.5f) * c->G.a;
  s[1] = (u01_co(o.b) - 0.5f) * c->G.a;
  s[2] = (u01_co(o.c) - 0.5f) * c->G.a;
}

int do_scan(mpc_ctx* c) {
  const size_t nk = c->G.nkeys, nb = (nk + SCAN_TILE - 1) / SCAN_TILE;
  FamilyTimer ft(c, F_SCAN);
  k_scan_reduce<<<(unsigned)nb, SCAN_T, 0, c->stream>>>(c->hist, nk, c->bsum);
  LAUNCH_CHECK("k_scan_reduce");
  k_scan_top<<<1, 1024, 0, c->stream>>>(c->bsum, nb);
  LAUNCH_CHECK("k_scan_top");
  k_scan_apply<<<(unsigned)nb, SCAN_T, 0, c->stream>>>(c->hist, nk, c->bsum, c->offset);
  LAUNCH_CHECK("k_scan_apply");
  return MPC_OK;
}

int do_reorder(mpc_ctx* c) {
  const size_t n = c->n;
  int rc = do_scan(c);
  if (rc) return rc;
  { FamilyTimer ft(c, F_MEMSET); CU(cudaMemsetAsync(c->hist, 0, (size_t)c->G.nkeys * 4, c->stream)); }   // reuse as cursor
  {
    FamilyTimer ft(c, F_SCATTER);
    k_scatter_ids<<<nblk(n, 256), 256, 0, c->stream>>>(n, c->A[7], c->A[6], c->offset, c->hist, c->slot_id);
    LAUNCH_CHECK("k_scatter_ids");
  }
  {
    FamilyTimer ft(c, F_RANK);
    k_rank<<<nblk(n, 256), 256, 0, c->stream>>>(n, c->A[7], c->A[6], c->offset, c->slot_id, c->perm);
    LAUNCH_CHECK("k_rank");
  }
  FamilyTimer ftg(c, F_GATHER);
  if (!c->compact) {
    Arrays8 src, dst;
    for (int a = 0; a < 8; ++a) { src.p[a] = c->A[a]; dst.p[a] = c->Bf[a]; }
    k_gather8<<<nblk(n, 256), 256, 0, c->stream>>>(n, c->perm, src, dst);
    LAUNCH_CHECK("k_gather8");
    for (int a = 0; a < 8; ++a) { uint32_t* t = c->A[a]; c->A[a] = c->Bf[a]; c->Bf[a] = t; }
  } else {
    // property-wise through one temporary array
    for (int a = 0; a < 8; ++a) {
      CU(cudaMemcpyAsync(c->Bf[0], c->A[a], n * 4, cudaMemcpyDeviceToDevice, c->stream));
      k_gather1<<<nblk(n, 256), 256, 0, c->stream>>>(n, c->perm, c->Bf[0], c->A[a]);
      LAUNCH_CHECK("k_gather1");
    }
  }
  return MPC_OK;
}

int one_step(mpc_ctx* c) {
  const size_t n = c->n;
  Geo& G = c->G;
  G.t = c->t;
  host_shift(c, c->t, G.s);
  const bool rebin = (c->t % (uint32_t)c->p.rebin_every) == 0u;
  float** F = reinterpret_cast<float**>(c->A);
  {
    FamilyTimer ft(c, F_MEMSET);
    CU(cudaMemsetAsync(c->sums, 0, (size_t)G.nkeys * SUMS_W * 4, c->stream));
    if (rebin) CU(cudaMemsetAsync(c->hist, 0, (size_t)G.nkeys * 4, c->stream));
  }
  if (n == 0) { c->t++; c->have_cells = true; return MPC_OK; }
  uint32_t* hist = rebin ? c->hist : nullptr;
  const bool wall = G.wall >= 0, grav = (G.g[0] != 0.f || G.g[1] != 0.f || G.g[2] != 0.f);
  const unsigned gb = nblk(n, 256);
  {
  FamilyTimer ft(c, F_STREAM);
  if (wall && grav) k_stream_key<true, true><<<gb, 256, 0, c->stream>>>(G, n, F[0], F[1], F[2], F[3], F[4], F[5], c->A[7], hist);
  else if (wall) k_stream_key<true, false><<<gb, 256, 0, c->stream>>>(G, n, F[0], F[1], F[2], F[3], F[4], F[5], c->A[7], hist);
  else if (grav) k_stream_key<false, true><<<gb, 256, 0, c->stream>>>(G, n, F[0], F[1], F[2], F[3], F[4], F[5], c->A[7], hist);
  else k_stream_key<false, false><<<gb, 256, 0, c->stream>>>(G, n, F[0], F[1], F[2], F[3], F[4], F[5], c->A[7], hist);
  LAUNCH_CHECK("k_stream_key");
  }
  if (rebin) {
    const int rc = do_reorder(c);
    if (rc) return rc;
    F = reinterpret_cast<float**>(c->A);
  }
  {
    FamilyTimer ft(c, F_ACCUM);
    if (G.collision == 1) k_accum<true><<<gb, 256, 0, c->stream>>>(G, n, F[3], F[4], F[5], c->A[7], c->offset, c->sums);
    else k_accum<false><<<gb, 256, 0, c->stream>>>(G, n, F[3], F[4], F[5], c->A[7], c->offset, c->sums);
    LAUNCH_CHECK("k_accum");
  }
  {
    FamilyTimer ft(c, F_CELL);
    k_cell<<<nblk(G.nkeys, 128), 128, 0, c->stream>>>(G, c->sums, c->rec);
    LAUNCH_CHECK("k_cell");
  }
  {
    FamilyTimer ft(c, F_COLLIDE);
    if (G.collision == 1) k_collide<true><<<gb, 256, 0, c->stream>>>(G, n, F[3], F[4], F[5], c->A[7], c->offset, c->rec);
    else k_collide<false><<<gb, 256, 0, c->stream>>>(G, n, F[3], F[4], F[5], c->A[7], c->offset, c->rec);
    LAUNCH_CHECK("k_collide");
  }
  c->t++;
  c->have_cells = true;
  return MPC_OK;
}

int set_state_impl(mpc_ctx* c, unsigned long long n, const float* const src[6], const unsigned* id, unsigned step,
                   cudaMemcpyKind kind) {
  if (!c) return MPC_EINVAL;
  if (c->sticky) return MPC_ECUDA;
  if (!c->bound) return fail(c, MPC_ESTATE, "mpc_set_state before mpc_bind");
  if (n > c->n_max) return fail(c, MPC_ENOMEM, "n exceeds the n_max given to mpc_bind");
  for (int a = 0; a < 6; ++a) if (n && !src[a]) return fail(c, MPC_EINVAL, "NULL state array");
  for (int a = 0; a < 6; ++a)
    if (n) CU(cudaMemcpyAsync(c->A[a], src[a], n * 4, kind, c->stream));
  if (n) {
    if (id) CU(cudaMemcpyAsync(c->A[6], id, n * 4, kind, c->stream));
    else { k_iota<<<nblk(n, 256), 256, 0, c->stream>>>(n, c->A[6]); LAUNCH_CHECK("k_iota"); }
  }
  c->n = n; c->t = step; c->have_state = true; c->have_cells = false;
  return MPC_OK;
}
int get_state_impl(mpc_ctx* c, float* const dst[6], unsigned* id, cudaMemcpyKind kind) {
  if (!c) return MPC_EINVAL;
  if (c->sticky) return MPC_ECUDA;
  if (!c->have_state) return fail(c, MPC_ESTATE, "mpc_get_state before mpc_set_state");
  for (int a = 0; a < 6; ++a)
    if (dst[a] && c->n) CU(cudaMemcpyAsync(dst[a], c->A[a], c->n * 4, kind, c->stream));
  if (id && c->n) CU(cudaMemcpyAsync(id, c->A[6], c->n * 4, kind, c->stream));
  if (kind == cudaMemcpyDeviceToHost) CU(cudaStreamSynchronize(c->stream));
  return MPC_OK;
}

}  // namespace

extern "C" {

int mpc_create(mpc_ctx** out, const float box[3], const int cells[3], float n_per_cell, const mpc_params* p,
               unsigned long long seed) {
  if (!out) return MPC_EINVAL;
  *out = nullptr;
  if (!box || !cells || !p) return MPC_EINVAL;
  for (int d = 0; d < 3; ++d) if (cells[d] < 1 || !(box[d] > 0.0f)) return MPC_EINVAL;
  const float a = box[0] / (float)cells[0];
  for (int d = 1; d < 3; ++d) if (box[d] / (float)cells[d] != a) return MPC_EINVAL;
  if (p->collision < 0 || p->collision > 1) return MPC_EINVAL;
  if (!(p->dt > 0.0f) || !(p->kT > 0.0f) || !(p->mass > 0.0f) || p->rebin_every < 1 || !(n_per_cell > 0.0f)) return MPC_EINVAL;
  if (p->brick < 1 || (p->brick & (p->brick - 1)) != 0 || p->brick > 64) return MPC_EINVAL;   // power of two
  int nwall = 0, wall = -1;
  for (int d = 0; d < 3; ++d) {
    if (p->bc[d] != 0 && p->bc[d] != 1) return MPC_EINVAL;
    if (p->bc[d] == 1) { nwall++; wall = d; if (p->g[d] != 0.0f) return MPC_EINVAL; }
  }
  if (nwall > 1) return MPC_EINVAL;
  if (nwall && (p->conserve_L || p->collision == 1)) return MPC_EINVAL;
  if (p->collision == 0 && p->conserve_L && p->thermostat) return MPC_EINVAL;
  if (p->collision == 1 && p->rebin_every != 1) return MPC_EINVAL;
  if (p->conserve_L) return MPC_EINVAL;   // +a: not built yet
  mpc_ctx* c = new (std::nothrow) mpc_ctx();   // value-initialised: all zero
  if (!c) return MPC_ENOMEM;
  c->p = *p; c->seed = seed;
  c->hbuf = new (std::nothrow) double[OBS_HOST_DOUBLES];
  if (!c->hbuf) { delete c; return MPC_ENOMEM; }
  Geo& G = c->G;
  int bs = 0;
  while ((1 << bs) < p->brick) ++bs;
  G.bshift = bs; G.a = a; G.inv_a = 1.0f / a; G.wall = wall;
  unsigned long long nk = 1;
  for (int d = 0; d < 3; ++d) {
    c->box[d] = box[d]; c->cells[d] = cells[d];
    G.L[d] = box[d]; G.n[d] = cells[d]; G.bc[d] = p->bc[d]; G.g[d] = p->g[d];
    G.m[d] = cells[d] + (p->bc[d] == 1 ? 2 : 0);
    G.mb[d] = (G.m[d] + p->brick - 1) >> bs;
    nk *= (unsigned long long)G.mb[d] << bs;
  }
  if (nk >= 0xffffffffull) { delete[] c->hbuf; delete c; return MPC_EINVAL; }
  G.nkeys = (uint32_t)nk;
  G.dt = p->dt; G.kT = p->kT; G.mass = p->mass;
  G.sigma = (float)sqrt((double)p->kT / (double)p->mass);
  G.cosa = (float)cos((double)p->alpha); G.sina = (float)sin((double)p->alpha);
  G.k0 = (uint32_t)(seed & 0xffffffffull); G.k1 = (uint32_t)(seed >> 32);
  G.nbar = (int)lround((double)n_per_cell);
  const int ue = (int)lround(log2((double)G.sigma));        // thermal velocity rounded to a power of two
  G.fxv = (float)ldexp(1.0, 20 - ue); G.fxv_inv = ldexp(1.0, ue - 20);
  G.fxe = (float)ldexp(1.0, 18 - 2 * ue); G.fxe_inv = ldexp(1.0, 2 * ue - 18);
  G.collision = p->collision; G.thermostat = p->thermostat;
  *out = c;
  return MPC_OK;
}

int mpc_num_keys(const mpc_ctx* c, unsigned long long* nkeys) {
  if (!c || !nkeys) return MPC_EINVAL;
  *nkeys = c->G.nkeys;
  return MPC_OK;
}

int mpc_workspace_bytes(const mpc_ctx* c, unsigned long long n_max, int compact, size_t* bytes) {
  if (!c || !bytes || n_max > 0xffffffffull) return MPC_EINVAL;
  *bytes = make_layout((size_t)n_max, c->G.nkeys, compact != 0).total;
  return MPC_OK;
}

int mpc_bind(mpc_ctx* c, void* workspace, size_t bytes, unsigned long long n_max, void* cuda_stream) {
  if (!c) return MPC_EINVAL;
  if (!workspace || ((uintptr_t)workspace & 255u) || n_max > 0xffffffffull) return fail(c, MPC_EINVAL, "workspace NULL, misaligned or n_max too large");
  Layout l = make_layout((size_t)n_max, c->G.nkeys, false);
  bool compact = false;
  if (bytes < l.total) { l = make_layout((size_t)n_max, c->G.nkeys, true); compact = true; }
  if (bytes < l.total) return fail(c, MPC_ENOMEM, "workspace smaller than mpc_workspace_bytes(n_max, compact=1)");
  c->ws = (char*)workspace; c->ws_bytes = bytes; c->n_max = (size_t)n_max; c->compact = compact;
  c->stream = (cudaStream_t)cuda_stream;
  for (int a = 0; a < 8; ++a) { c->A[a] = (uint32_t*)(c->ws + l.off_A[a]); c->Bf[a] = (uint32_t*)(c->ws + l.off_B[a]); }
  c->slot_id = (uint32_t*)(c->ws + l.off_slot); c->perm = (uint32_t*)(c->ws + l.off_perm);
  c->hist = (uint32_t*)(c->ws + l.off_hist); c->offset = (uint32_t*)(c->ws + l.off_offset);
  c->bsum = (uint32_t*)(c->ws + l.off_bsum);
  c->sums = (int*)(c->ws + l.off_sums); c->rec = (float*)(c->ws + l.off_rec); c->obs = (double*)(c->ws + l.off_obs);
  c->bound = true; c->have_state = false; c->have_cells = false; c->n = 0;
  return MPC_OK;
}

int mpc_set_state(mpc_ctx* c, unsigned long long n, const float* x, const float* y, const float* z, const float* vx,
                  const float* vy, const float* vz, const unsigned* id, unsigned step) {
  const float* const src[6] = {x, y, z, vx, vy, vz};
  return set_state_impl(c, n, src, id, step, cudaMemcpyDeviceToDevice);
}
int mpc_set_state_host(mpc_ctx* c, unsigned long long n, const float* x, const float* y, const float* z, const float* vx,
                       const float* vy, const float* vz, const unsigned* id, unsigned step) {
  const float* const src[6] = {x, y, z, vx, vy, vz};
  return set_state_impl(c, n, src, id, step, cudaMemcpyHostToDevice);
}

int mpc_step(mpc_ctx* c, int nsteps) {
  if (!c || nsteps < 0) return MPC_EINVAL;
  if (c->sticky) return MPC_ECUDA;
  if (!c->bound || !c->have_state) return fail(c, MPC_ESTATE, "mpc_step before mpc_bind / mpc_set_state");
  for (int k = 0; k < nsteps; ++k) {
    const int rc = one_step(c);
    if (rc) return rc;
  }
  return MPC_OK;
}

int mpc_get_state(mpc_ctx* c, float* x, float* y, float* z, float* vx, float* vy, float* vz, unsigned* id) {
  float* const dst[6] = {x, y, z, vx, vy, vz};
  return get_state_impl(c, dst, id, cudaMemcpyDeviceToDevice);
}
int mpc_get_state_host(mpc_ctx* c, float* x, float* y, float* z, float* vx, float* vy, float* vz, unsigned* id) {
  float* const dst[6] = {x, y, z, vx, vy, vz};
  return get_state_impl(c, dst, id, cudaMemcpyDeviceToHost);
}

int mpc_observables(mpc_ctx* c, mpc_obs* out, float* profile_host) {
  if (!c || !out) return MPC_EINVAL;
  if (c->sticky) return MPC_ECUDA;
  if (!c->have_state) return fail(c, MPC_ESTATE, "mpc_observables before mpc_set_state");
  memset(out, 0, sizeof(*out));
  const Geo& G = c->G;
  float** F = reinterpret_cast<float**>(c->A);
  const size_t n = c->n;
  double* part = c->obs;
  double* prof = c->obs + (size_t)OBS_BLOCKS * 8;
  int pa = 2, fa = 0;
  for (int d = 0; d < 3; ++d) if (G.bc[d] == 1) pa = d;
  for (int d = 2; d >= 0; --d) if (G.g[d] != 0.0f) fa = d;
  const int nb = G.n[pa];
  if (profile_host && nb > MAX_PROFILE) return fail(c, MPC_EINVAL, "profile axis longer than 2048 layers");
  CU(cudaMemsetAsync(c->obs, 0, ((size_t)OBS_BLOCKS * 8 + 2 * MAX_PROFILE) * 8, c->stream));
  if (n) {
    k_obs_particles<<<OBS_BLOCKS, 256, 0, c->stream>>>(n, F[3], F[4], F[5], part);
    LAUNCH_CHECK("k_obs_particles");
    if (profile_host) {
      k_obs_profile<<<OBS_BLOCKS, 256, (size_t)2 * nb * 8, c->stream>>>(G, n, pa, nb, F[pa], F[3 + fa], prof);
      LAUNCH_CHECK("k_obs_profile");
    }
  }
  if (c->have_cells) {   // MPC-AT keeps no energy sum: kT_cell is reported as 0 there
    k_obs_cells<<<OBS_BLOCKS, 256, 0, c->stream>>>(G, c->sums, part);
    LAUNCH_CHECK("k_obs_cells");
  }
  double* hbuf = c->hbuf;
  CU(cudaMemcpyAsync(hbuf, c->obs, OBS_HOST_DOUBLES * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  CU(cudaStreamSynchronize(c->stream));
  double P[3] = {0, 0, 0}, E = 0, num = 0, den = 0, mx = 0;
  for (int b = 0; b < OBS_BLOCKS; ++b) {
    const double* o = hbuf + (size_t)b * 8;
    P[0] += o[0]; P[1] += o[1]; P[2] += o[2]; E += o[3]; num += o[4]; den += o[5];
    if (o[6] > mx) mx = o[6];
  }
  const double m = G.mass;
  out->n = n; out->step = c->t;
  for (int d = 0; d < 3; ++d) out->P[d] = m * P[d];
  out->E_kin = 0.5 * m * E;
  out->kT_est = n > 1 ? m * (E - (P[0] * P[0] + P[1] * P[1] + P[2] * P[2]) / (double)n) / (3.0 * (double)(n - 1)) : 0.0;
  out->kT_cell = (G.collision == 0 && den > 0) ? num / den : 0.0;
  out->max_cell_count = (unsigned)mx;
  out->n_singular_cells = 0;
  if (profile_host) {
    const double* pr = hbuf + (size_t)OBS_BLOCKS * 8;
    for (int b = 0; b < nb; ++b) profile_host[b] = pr[nb + b] > 0 ? (float)(pr[b] / pr[nb + b]) : 0.0f;
  }
  return MPC_OK;
}

int mpc_get_cells(mpc_ctx* c, unsigned* count, float* px, float* py, float* pz, float* e2, unsigned* key) {
  if (!c) return MPC_EINVAL;
  if (c->sticky) return MPC_ECUDA;
  if (!c->have_cells) return fail(c, MPC_ESTATE, "mpc_get_cells before the first mpc_step");
  const Geo& G = c->G;
  if (G.collision == 1) k_export_cells<true><<<nblk(G.nkeys, 256), 256, 0, c->stream>>>(G, c->sums, count, px, py, pz, e2);
  else k_export_cells<false><<<nblk(G.nkeys, 256), 256, 0, c->stream>>>(G, c->sums, count, px, py, pz, e2);
  LAUNCH_CHECK("k_export_cells");
  if (key && c->n) CU(cudaMemcpyAsync(key, c->A[7], c->n * 4, cudaMemcpyDeviceToDevice, c->stream));
  return MPC_OK;
}

void mpc_philox4x32_10(const unsigned ctr[4], const unsigned key[2], unsigned out[4]) {
  const Block4 o = philox(ctr[0], ctr[1], ctr[2], ctr[3], key[0], key[1]);
  out[0] = o.a; out[1] = o.b; out[2] = o.c; out[3] = o.d;
}

unsigned long long mpc_launch_count(const mpc_ctx* c) { return c ? c->launches : 0ull; }

int mpc_profile_enable(mpc_ctx* c, int on) {
  if (!c) return MPC_EINVAL;
  if (c->sticky) return MPC_ECUDA;
  if (on && !c->prof_ev) {
    c->prof_ev = new (std::nothrow) cudaEvent_t[2 * PROF_MAX_PAIRS];
    c->prof_fam = new (std::nothrow) int[PROF_MAX_PAIRS];
    if (!c->prof_ev || !c->prof_fam) return fail(c, MPC_ENOMEM, "profile buffers");
    for (int i = 0; i < 2 * PROF_MAX_PAIRS; ++i) CU(cudaEventCreate(&c->prof_ev[i]));
  }
  c->prof_on = on != 0;
  return MPC_OK;
}

int mpc_profile_read(mpc_ctx* c, int* n_families, const char** names, double* total_ms, unsigned long long* launches) {
  if (!c || !n_families) return MPC_EINVAL;
  if (c->sticky) return MPC_ECUDA;
  if (c->prof_pairs) CU(cudaStreamSynchronize(c->stream));
  for (int i = 0; i < c->prof_pairs; ++i) {
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, c->prof_ev[2 * i], c->prof_ev[2 * i + 1]));
    c->prof_ms[c->prof_fam[i]] += ms;
  }
  c->prof_pairs = 0;
  *n_families = F_COUNT;
  for (int f = 0; f < F_COUNT; ++f) {
    if (names) names[f] = FAMILY_NAMES[f];
    if (total_ms) total_ms[f] = c->prof_ms[f];
    if (launches) launches[f] = c->prof_launches[f];
    c->prof_ms[f] = 0.0; c->prof_launches[f] = 0;
  }
  return MPC_OK;
}

const char* mpc_last_error(const mpc_ctx* c) { return c ? c->err : "null context"; }

int mpc_destroy(mpc_ctx* c) {
  if (c) {
    delete[] c->hbuf;
    if (c->prof_ev) for (int i = 0; i < 2 * PROF_MAX_PAIRS; ++i) cudaEventDestroy(c->prof_ev[i]);
    delete[] c->prof_ev;
    delete[] c->prof_fam;
  }
  delete c;
  return MPC_OK;
}

}  // extern "C"
