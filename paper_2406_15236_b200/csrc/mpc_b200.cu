// mpc_b200.cu -- B200 (sm_100a) implementation of the MPC fluid step behind include/mpc_b200.h.
//
// One CUDA stream, no host synchronisation inside mpc_step. Kernel families:
//   k_sweep        SRD hot path, ONE pass over the particles per step: collision of step t-1
//                  (Eqs. 2,5) fused with MOVE of step t (Eq. 1), shift + cell key, and the per-cell
//                  sums of step t accumulated in a shared-memory tile per brick of cells.
//                  PAPER.md:29-37,68,70,176
//   k_cell         PROCESS_CELLS: v_cm, axis, kappa, virtual wall particles
//   k_collide_pos  trailing collision of the last step of an mpc_step call       Eqs. (2),(5)
//                  Variants IO_AOS_OUT / IO_GATHER fold a reorder into the sweeps of its own and the
//                  next step through 32-byte staging records.
//   k_scan_* / k_scatter_src (hot path: group by key) / k_scatter_slots + k_rank (rank by id) /
//   k_rank_cells (lazy canonical order) / k_gather*   counting-sort reorder
//   k_stream_key / k_accum_at / k_accum_a / k_accum_seg / k_cell_a / k_collide_at / k_collide_a
//                  MPC-AT and +a path (needs the rank of a particle in its sorted cell segment or
//                  22 sums per cell: not fused; per-cell segmented sums when the order is fresh)
//   k_obs_*        observables
// Cell sums are 32-bit fixed point (the paper's reproducibility option), two per
// 64-bit word, added with integer atomics: order-independent, so a trajectory is bit-reproducible and
// does not depend on the memory order of the particles.
// Compile with --fmad=false: every multiply-add that must fuse is an explicit fmaf (U1).
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "../../include/mpc_b200.h"
#include "philox.cuh"

namespace mpc {

typedef unsigned long long u64;

// halo 1 instead of 2: 0.5 % of the particles (the ones that moved two cells since the reorder) take the global-atomic
// path, the tile shrinks from 96 to 65 KB and its flush by a third: sweep 12.34 -> 12.03 ms per step at config 5
#ifndef MPC_HALO
#define MPC_HALO 1
#endif
#ifndef MPC_SWEEP_T
#define MPC_SWEEP_T 512
#endif
#ifndef MPC_SWEEP_MINB
#define MPC_SWEEP_MINB 2
#endif
constexpr int HALO = MPC_HALO;        // tile halo in cells on every side of a brick
constexpr int SWEEP_T = MPC_SWEEP_T;  // threads per sweep CTA
constexpr int SWEEP_T3 = 384;         // ... of the steady-state sweep when three tiles fit in an SM's shared memory
constexpr int PF_DIST = 4;           // L2 prefetch distance of the sweep, in iterations of SWEEP_T particles
constexpr int TILE_W = 5;             // int32 words per tile cell: N, Sx, Sy, Sz, E
constexpr int REC_W = 8;              // floats per cell record (32 B, one sector)
constexpr int OBS_BLOCKS = 1184;      // 148 SMs x 8
constexpr int MAX_PROFILE = 2048;
constexpr size_t OBS_HOST_DOUBLES = (size_t)OBS_BLOCKS * 8 + 2 * MAX_PROFILE;
constexpr size_t MAX_TILE_BYTES = 110 * 1024;

struct Geo {
  float L[3];
  float a, inv_a;
  int n[3];       // fluid cells
  int m[3];       // cell layers incl. wall layers
  int mb[3];      // bricks per axis
  int bs[3];      // log2(brick dims)
  int bc[3];      // 0 periodic, 1 no-slip walls, 2 slip walls
  int wall;       // wall axis or -1
  int slip;       // 1: the walls reflect specularly and have no virtual particles (U20)
  float g[3];
  float dt;
  float s[3];     // lattice shift of this step
  uint32_t k0, k1, t;
  uint32_t rk[20];   // Philox round keys of (k0, k1), see philox_rk
  float cosa, sina;
  float kT, mass, sigma;   // sigma = sqrt(kT/m)
  // Fixed-point scales: powers of two relative to u = 2^round(log2 sigma), so precision does not
  // depend on the unit system: velocity sums 2^22/u in int32 (|sum_cell v_d| < 512 u); energy sums
  // 2^22/u^2, uint32 per tile (< 1024 u^2 per cell and CTA) and 48 bits in the global word.
  float fxv, fxe;
  double fxv_inv, fxe_inv;
  int nbar;
  int collision, thermostat, conserve_L;
  int generic;    // 1 = unfused path (MPC-AT and every +a variant), 0 = fused SRD sweep
  int sw;         // 64-bit words per cell in the global sums array (3 SRD, 4 MPC-AT, 10 with +a)
  int rw;         // floats per cell record (8, or 16 with +a)
  uint32_t nkeys;
};

// ---- packed sums ---------------------------------------------------------------------------------
// word0 = E << 16 | N (E: 48 bits, N: 16 bits, so at most 65535 particles per cell); word1 = (Sy, Sx); word2 = (R0, Sz); word3 = (R2, R1)  [AT: R = sum v_ran]
// +a adds, in cell-local coordinates rho in [0,1)^3 (U9), scale 2^20 for rho terms:
// word4 = (rho_y, rho_x); word5 = (Qxx, rho_z); word6 = (Qzz, Qyy); word7 = (Qxz, Qxy); word8 = (Lx, Qyz);
// word9 = (Lz, Ly)   with Q = sum rho rho^T, L = sum rho x u, u = v - D v (SRD) or v - v_ran (AT)
__device__ __forceinline__ u64 pack_ss(int lo, int hi) { return (u64)((long long)hi * 4294967296ll + (long long)lo); }
__device__ __forceinline__ void unpack_ss(u64 w, int& lo, int& hi) {
  lo = (int)(uint32_t)(w & 0xffffffffull);
  hi = (int)(((long long)w - (long long)lo) >> 32);
}

// ---- geometry helpers ----------------------------------------------------------------------------
__device__ __forceinline__ uint32_t layout_key(const Geo& G, int ix, int iy, int iz) {
  const int b0 = G.bs[0], b1 = G.bs[1], b2 = G.bs[2];
  const uint32_t brick = ((uint32_t)(iz >> b2) * (uint32_t)G.mb[1] + (uint32_t)(iy >> b1)) * (uint32_t)G.mb[0] + (uint32_t)(ix >> b0);
  const uint32_t local = ((((uint32_t)(iz & ((1 << b2) - 1))) << b1 | (uint32_t)(iy & ((1 << b1) - 1))) << b0) | (uint32_t)(ix & ((1 << b0) - 1));
  return (brick << (b0 + b1 + b2)) | local;
}
__device__ __forceinline__ void brick_to_origin(const Geo& G, uint32_t brick, int& ox, int& oy, int& oz) {
  const uint32_t bx = brick % (uint32_t)G.mb[0], r = brick / (uint32_t)G.mb[0];
  const uint32_t by = r % (uint32_t)G.mb[1], bz = r / (uint32_t)G.mb[1];
  ox = (int)(bx << G.bs[0]); oy = (int)(by << G.bs[1]); oz = (int)(bz << G.bs[2]);
}
__device__ __forceinline__ void key_to_cell(const Geo& G, uint32_t key, int& ix, int& iy, int& iz) {
  const int b0 = G.bs[0], b1 = G.bs[1], b2 = G.bs[2];
  const uint32_t local = key & ((1u << (b0 + b1 + b2)) - 1u), brick = key >> (b0 + b1 + b2);
  int ox, oy, oz;
  brick_to_origin(G, brick, ox, oy, oz);
  ix = ox + (int)(local & ((1u << b0) - 1u));
  iy = oy + (int)((local >> b0) & ((1u << b1) - 1u));
  iz = oz + (int)(local >> (b0 + b1));
}
__device__ __forceinline__ uint32_t canonical_id(const Geo& G, int ix, int iy, int iz) {
  return (uint32_t)ix + (uint32_t)G.m[0] * ((uint32_t)iy + (uint32_t)G.m[1] * (uint32_t)iz);
}
// cell coordinate of position r along axis d for lattice shift s
__device__ __forceinline__ int cell_coord(const Geo& G, int d, float r, float s) {
  const float q = (r + s) * G.inv_a;
  int k = (int)floorf(q);
  if (G.bc[d] == 0) {
    if (k < 0) k += G.n[d];
    if (k >= G.n[d]) k -= G.n[d];
  } else {
    k += 1;
    k = max(0, min(k, G.n[d] + 1));
  }
  return k;
}
__device__ __forceinline__ uint32_t key_of(const Geo& G, float x, float y, float z, float s0, float s1, float s2) {
  return layout_key(G, cell_coord(G, 0, x, s0), cell_coord(G, 1, y, s1), cell_coord(G, 2, z, s2));
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
      if (G.slip) {   // specular reflection: only the wall-normal component turns round
        if (w == 0) v[0] = -v[0]; else if (w == 1) v[1] = -v[1]; else v[2] = -v[2];
      } else { v[0] = -v[0]; v[1] = -v[1]; v[2] = -v[2]; }   // bounce-back
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

// 256-bit read-only load of one 32-byte cell record (sm_100: LDG.E.ENL2.256): one L1 request instead of two
__device__ __forceinline__ void load_rec(const float* __restrict__ rec, uint32_t key, float4& r0, float4& ax) {
  const float* p = rec + (size_t)key * REC_W;
  asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=f"(r0.x), "=f"(r0.y), "=f"(r0.z), "=f"(r0.w), "=f"(ax.x), "=f"(ax.y), "=f"(ax.z), "=f"(ax.w)
               : "l"(p));
}

// ---- SRD rotation with thermostat scaling: v' = vcm + kappa D(alpha) (v - vcm) ----------------------
__device__ __forceinline__ void srd_apply(const Geo& G, const float4 r0, const float4 ax, float (&v)[3]) {
  const float w0 = v[0] - r0.x, w1 = v[1] - r0.y, w2 = v[2] - r0.z;
  const float c = G.cosa, s = G.sina, omc = 1.0f - G.cosa;
  const float nd = fmaf(ax.x, w0, fmaf(ax.y, w1, ax.z * w2)) * omc;
  const float cx = fmaf(ax.y, w2, -(ax.z * w1)), cy = fmaf(ax.z, w0, -(ax.x * w2)), cz = fmaf(ax.x, w1, -(ax.y * w0));
  const float o0 = fmaf(w0, c, fmaf(cx, s, ax.x * nd));
  const float o1 = fmaf(w1, c, fmaf(cy, s, ax.y * nd));
  const float o2 = fmaf(w2, c, fmaf(cz, s, ax.z * nd));
  v[0] = fmaf(r0.w, o0, r0.x);
  v[1] = fmaf(r0.w, o1, r0.y);
  v[2] = fmaf(r0.w, o2, r0.z);
}

// ---- the fused sweep -----------------------------------------------------------------------------
// One CTA per brick of cells. Its particles are the contiguous range that was sorted into the brick at
// the last reorder (chunk[] = offset[] of the brick's first key); since then they have moved by a
// fraction of a cell and the lattice shift has changed by less than a cell, so nearly all of them fall
// into the brick's tile (brick + HALO cells on every side), held in shared memory as int32 sums. The
// rest (and everything, if no order is known yet) goes to the global sums directly.
// B0,B1,B2 = log2 of the brick dims at compile time (the {16,16,8} fast path), or -1: read from Geo.
template <int B0, int B1, int B2>
struct BrickShape {
  static constexpr bool fixed = B0 >= 0;
  __device__ __forceinline__ static int s0(const Geo& G) { return fixed ? B0 : G.bs[0]; }
  __device__ __forceinline__ static int s1(const Geo& G) { return fixed ? B1 : G.bs[1]; }
  __device__ __forceinline__ static int s2(const Geo& G) { return fixed ? B2 : G.bs[2]; }
  __device__ __forceinline__ static uint32_t key(const Geo& G, int ix, int iy, int iz) {
    const int b0 = s0(G), b1 = s1(G), b2 = s2(G);
    const uint32_t brick = ((uint32_t)(iz >> b2) * (uint32_t)G.mb[1] + (uint32_t)(iy >> b1)) * (uint32_t)G.mb[0] + (uint32_t)(ix >> b0);
    const uint32_t local = ((((uint32_t)(iz & ((1 << b2) - 1))) << b1 | (uint32_t)(iy & ((1 << b1) - 1))) << b0) | (uint32_t)(ix & ((1 << b0) - 1));
    return (brick << (b0 + b1 + b2)) | local;
  }
};
// floor index of a coordinate, not yet folded into [0, m)
__device__ __forceinline__ int cell_raw(const Geo& G, float r, float s) { return __float2int_rd((r + s) * G.inv_a); }
// fold an index known to lie in [-m, 2m) into [0, m)
__device__ __forceinline__ int fold(int k, int m) {
  k += (k < 0) ? m : 0;
  k -= (k >= m) ? m : 0;
  return k;
}

// Reorder folded into two consecutive sweeps (IO = 1 on the reorder step, IO = 2 on the step after it):
//   IO_AOS_OUT  the pass writes every particle as ONE 32-byte record {r, v, id, 0} into a staging buffer
//               instead of updating the SoA arrays in place;
//   IO_GATHER   particle i of the new order is read with one 256-bit load from staging[perm[i]] (a whole
//               sector, every byte used) and written to the SoA arrays at i.
// A gather of the SoA arrays themselves costs ~4.5 sectors of L2 traffic per useful one (measured).
enum { IO_PLAIN = 0, IO_AOS_OUT = 1, IO_GATHER = 2 };
struct SweepIO {
  const float* aos_in;      // IO_GATHER: staging records in the old order
  float* aos_out;           // IO_AOS_OUT
  const uint32_t* perm;     // IO_GATHER
  uint32_t* id;             // IO_AOS_OUT: read at i; IO_GATHER: written at i
};
__device__ __forceinline__ void ld256(const float* p, float (&a)[8]) {
  asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=f"(a[0]), "=f"(a[1]), "=f"(a[2]), "=f"(a[3]), "=f"(a[4]), "=f"(a[5]), "=f"(a[6]), "=f"(a[7]) : "l"(p));
}
__device__ __forceinline__ void st256(float* p, const float (&a)[8]) {
  asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
               :: "l"(p), "f"(a[0]), "f"(a[1]), "f"(a[2]), "f"(a[3]), "f"(a[4]), "f"(a[5]), "f"(a[6]), "f"(a[7]) : "memory");
}
// T = threads per CTA: 512 (2 CTAs per SM), or 384 (3 CTAs per SM at <= 56 registers: the steady-state sweep is
// 2 % faster that way, the staged reorder sweeps are not)
template <bool COLLIDE, bool WALL, bool GRAV, bool WKEY, class BS, int IO = IO_PLAIN, int T = SWEEP_T>
__global__ void __launch_bounds__(T, T <= 384 ? 3 : 2)
k_sweep(Geo G, float sp0, float sp1, float sp2, uint32_t n, float* __restrict__ x, float* __restrict__ y, float* __restrict__ z,
        float* __restrict__ vx, float* __restrict__ vy, float* __restrict__ vz, uint32_t* __restrict__ key_out,
        const uint32_t* __restrict__ chunk, uint32_t nbricks, const float* __restrict__ rec, u64* __restrict__ sums,
        SweepIO io) {
  extern __shared__ int tile[];
  const int T0 = (1 << BS::s0(G)) + 2 * HALO, T1 = (1 << BS::s1(G)) + 2 * HALO, T2 = (1 << BS::s2(G)) + 2 * HALO;
  const int tcells = T0 * T1 * T2;
  for (int i = threadIdx.x; i < tcells * TILE_W; i += T) tile[i] = 0;
  const uint32_t b = blockIdx.x;
  const int m0 = G.m[0], m1 = G.m[1], m2 = G.m[2];
  int ox, oy, oz;
  {
    const uint32_t bx = b % (uint32_t)G.mb[0], q = b / (uint32_t)G.mb[0];
    const uint32_t by = q % (uint32_t)G.mb[1], bz = q / (uint32_t)G.mb[1];
    ox = (int)(bx << BS::s0(G)) - HALO; oy = (int)(by << BS::s1(G)) - HALO; oz = (int)(bz << BS::s2(G)) - HALO;
  }
  uint32_t i0, i1;
  if (chunk) {
    const uint32_t bvol_shift = BS::s0(G) + BS::s1(G) + BS::s2(G);
    i0 = chunk[(size_t)b << bvol_shift];
    i1 = (b + 1 == nbricks) ? n : chunk[(size_t)(b + 1) << bvol_shift];
  } else {   // no order known: even split, (almost) everything takes the global path
    i0 = (uint32_t)((u64)n * b / nbricks);
    i1 = (uint32_t)((u64)n * (b + 1) / nbricks);
  }
  // index offsets added before the floor index is folded: +1 on a wall axis (layer 0 lies in the wall)
  // the CTA takes the 128-byte-aligned groups of 32 particles that START in its range: every group belongs to
  // exactly one CTA and every access of a warp is line-aligned (L1 tag requests per load 1.9 -> 1.0)
  i0 = (i0 + 31u) & ~31u;
  if (b + 1 != nbricks) i1 = min((i1 + 31u) & ~31u, n);   // trailing empty bricks: chunk = n, do not round past the end
  const int w0 = (WALL && G.bc[0]) ? 1 : 0, w1 = (WALL && G.bc[1]) ? 1 : 0, w2 = (WALL && G.bc[2]) ? 1 : 0;
  __syncthreads();
  // software pipeline: the loads of the next particle are in flight while this one is processed
  uint32_t i = i0 + threadIdx.x;
  float p0 = 0.f, p1 = 0.f, p2 = 0.f, p3 = 0.f, p4 = 0.f, p5 = 0.f;
  // IO_GATHER: source indices of the particles 1, 2 and 3 iterations ahead (the first feeds the register
  // prefetch, the second an L2 prefetch of its record, the third is in flight); pid = id of the particle in flight
  float pid = 0.f;
  uint32_t jn = 0, jn2 = 0, jn3 = 0;
  if (IO == IO_GATHER) {
    if (i < i1) {
      float q[8];
      ld256(io.aos_in + (size_t)io.perm[i] * 8, q);
      p0 = q[0]; p1 = q[1]; p2 = q[2]; p3 = q[3]; p4 = q[4]; p5 = q[5]; pid = q[6];
    }
    if (i + T < i1) jn = io.perm[i + T];
    if (i + 2 * T < i1) jn2 = io.perm[i + 2 * T];
    if (i + 3 * T < i1) jn3 = io.perm[i + 3 * T];
  } else if (i < i1) {
    p0 = x[i]; p1 = y[i]; p2 = z[i]; p3 = vx[i]; p4 = vy[i]; p5 = vz[i];
    if (IO == IO_AOS_OUT) pid = __uint_as_float(io.id[i]);
  }
  for (; i < i1; i += T) {
    float r[3] = {p0, p1, p2}, v[3] = {p3, p4, p5};
    const float idbits = pid;
    const uint32_t inext = i + T;
    if (IO == IO_GATHER) {
      io.id[i] = __float_as_uint(idbits);
      if (inext < i1) {
        float q[8];
        ld256(io.aos_in + (size_t)jn * 8, q);
        p0 = q[0]; p1 = q[1]; p2 = q[2]; p3 = q[3]; p4 = q[4]; p5 = q[5]; pid = q[6];
        jn = jn2; jn2 = jn3;
        if (i + 2 * T < i1) asm volatile("prefetch.global.L2 [%0];" ::"l"(io.aos_in + (size_t)jn * 8));
        if (i + 4 * T < i1) jn3 = io.perm[i + 4 * T];
      }
    } else if (inext < i1) {
      p0 = x[inext]; p1 = y[inext]; p2 = z[inext]; p3 = vx[inext]; p4 = vy[inext]; p5 = vz[inext];
      if (IO == IO_AOS_OUT) pid = __uint_as_float(io.id[inext]);
    }
    if (IO != IO_GATHER) {   // pull the lines of a later iteration into L2: the register prefetch above then pays L2, not DRAM, latency
      const uint32_t ifar = i + PF_DIST * T;
      if (ifar < i1) {
        asm volatile("prefetch.global.L2 [%0];" ::"l"(x + ifar));
        asm volatile("prefetch.global.L2 [%0];" ::"l"(y + ifar));
        asm volatile("prefetch.global.L2 [%0];" ::"l"(z + ifar));
        asm volatile("prefetch.global.L2 [%0];" ::"l"(vx + ifar));
        asm volatile("prefetch.global.L2 [%0];" ::"l"(vy + ifar));
        asm volatile("prefetch.global.L2 [%0];" ::"l"(vz + ifar));
      }
    }
    if (COLLIDE) {   // ROTATE_VELOCITIES of the previous step; its key is recomputed from r and that step's shift
      int kx = cell_raw(G, r[0], sp0) + w0, ky = cell_raw(G, r[1], sp1) + w1, kz = cell_raw(G, r[2], sp2) + w2;
      if (WALL) { kx = G.bc[0] ? max(0, min(kx, m0 - 1)) : fold(kx, m0); ky = G.bc[1] ? max(0, min(ky, m1 - 1)) : fold(ky, m1);
                  kz = G.bc[2] ? max(0, min(kz, m2 - 1)) : fold(kz, m2); }
      else { kx = fold(kx, m0); ky = fold(ky, m1); kz = fold(kz, m2); }
      const uint32_t kp = BS::key(G, kx, ky, kz);
      float4 r0, ax;
      load_rec(rec, kp, r0, ax);
      srd_apply(G, r0, ax, v);
    }
    stream_one<WALL, GRAV>(G, r, v);
    if (IO == IO_AOS_OUT) {
      const float q[8] = {r[0], r[1], r[2], v[0], v[1], v[2], idbits, 0.f};
      st256(io.aos_out + (size_t)i * 8, q);
    } else {
      x[i] = r[0]; y[i] = r[1]; z[i] = r[2];
      vx[i] = v[0]; vy[i] = v[1]; vz[i] = v[2];
    }
    int cx = cell_raw(G, r[0], G.s[0]) + w0, cy = cell_raw(G, r[1], G.s[1]) + w1, cz = cell_raw(G, r[2], G.s[2]) + w2;
    if (WALL) { if (G.bc[0]) cx = max(0, min(cx, m0 - 1)); if (G.bc[1]) cy = max(0, min(cy, m1 - 1)); if (G.bc[2]) cz = max(0, min(cz, m2 - 1)); }
    const int a0 = __float2int_rn(v[0] * G.fxv), a1 = __float2int_rn(v[1] * G.fxv), a2 = __float2int_rn(v[2] * G.fxv);
    const unsigned e = __float2uint_rn(fmaf(v[0], v[0], fmaf(v[1], v[1], v[2] * v[2])) * G.fxe);
    // tile coordinates: one fold takes care of the periodic image of the cell and of the tile origin
    const int l0 = fold(cx - ox, m0), l1 = fold(cy - oy, m1), l2 = fold(cz - oz, m2);
    const bool inside = (l0 < T0) & (l1 < T1) & (l2 < T2);
    if (inside) {
      int* s = tile + ((l2 * T1 + l1) * T0 + l0) * TILE_W;
      atomicAdd(s, 1); atomicAdd(s + 1, a0); atomicAdd(s + 2, a1); atomicAdd(s + 3, a2); atomicAdd((unsigned*)s + 4, e);
    }
    if (WKEY || !inside) {
      const uint32_t kc = BS::key(G, fold(cx, m0), fold(cy, m1), fold(cz, m2));
      if (WKEY) key_out[i] = kc;
      if (!inside) {
        u64* s = sums + (size_t)kc * G.sw;
        atomicAdd(s, ((u64)e << 16) | 1ull); atomicAdd(s + 1, pack_ss(a0, a1)); atomicAdd(s + 2, pack_ss(a2, 0));
      }
    }
  }
  __syncthreads();
  // flush the tile: one packed 64-bit reduction per pair of sums, empty cells skipped
  for (int c = threadIdx.x; c < tcells; c += T) {
    const int* s = tile + c * TILE_W;
    const int cnt = s[0];
    if (cnt == 0) continue;
    const int l0 = c % T0, q = c / T0, l1 = q % T1, l2 = q / T1;
    u64* g = sums + (size_t)BS::key(G, fold(ox + l0, m0), fold(oy + l1, m1), fold(oz + l2, m2)) * G.sw;
    atomicAdd(g, ((u64)(unsigned)s[4] << 16) | (u64)(unsigned)cnt);
    atomicAdd(g + 1, pack_ss(s[1], s[2]));
    atomicAdd(g + 2, pack_ss(s[3], 0));
  }
}

// trailing collision of the last step of a call (key recomputed from the position)
__global__ void __launch_bounds__(256) k_collide_pos(Geo G, size_t n, const float* __restrict__ x, const float* __restrict__ y,
                                                     const float* __restrict__ z, float* __restrict__ vx, float* __restrict__ vy,
                                                     float* __restrict__ vz, const float* __restrict__ rec) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t k = key_of(G, x[i], y[i], z[i], G.s[0], G.s[1], G.s[2]);
  float4 r0, ax;
  load_rec(rec, k, r0, ax);
  float v[3] = {vx[i], vy[i], vz[i]};
  srd_apply(G, r0, ax, v);
  vx[i] = v[0]; vy[i] = v[1]; vz[i] = v[2];
}

__global__ void __launch_bounds__(256) k_keys(Geo G, size_t n, const float* __restrict__ x, const float* __restrict__ y,
                                              const float* __restrict__ z, uint32_t* __restrict__ key) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) key[i] = key_of(G, x[i], y[i], z[i], G.s[0], G.s[1], G.s[2]);
}

// ---- MPC-AT path (unfused) -----------------------------------------------------------------------
template <bool WALL, bool GRAV>
__global__ void __launch_bounds__(256) k_stream_key(Geo G, size_t n, float* __restrict__ x, float* __restrict__ y,
                                                    float* __restrict__ z, float* __restrict__ vx, float* __restrict__ vy,
                                                    float* __restrict__ vz, uint32_t* __restrict__ key, u64* __restrict__ sums) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float r[3] = {x[i], y[i], z[i]}, v[3] = {vx[i], vy[i], vz[i]};
  stream_one<WALL, GRAV>(G, r, v);
  x[i] = r[0]; y[i] = r[1]; z[i] = r[2];
  if (WALL || GRAV) { vx[i] = v[0]; vy[i] = v[1]; vz[i] = v[2]; }
  const uint32_t k = key_of(G, r[0], r[1], r[2], G.s[0], G.s[1], G.s[2]);
  key[i] = k;
  atomicAdd(sums + (size_t)k * G.sw, 1ull);            // histogram = the count field of word 0
}
// needs the reordered arrays: rank = position of the particle in its (key, id)-sorted cell segment (U5)
__global__ void __launch_bounds__(256) k_accum_at(Geo G, size_t n, const float* __restrict__ vx, const float* __restrict__ vy,
                                                  const float* __restrict__ vz, const uint32_t* __restrict__ key,
                                                  const uint32_t* __restrict__ offset, u64* __restrict__ sums) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t k = key[i];
  int ix, iy, iz;
  key_to_cell(G, k, ix, iy, iz);
  const Block4 o = philox(canonical_id(G, ix, iy, iz), (uint32_t)i - offset[k], G.t, TAG_AT, G.k0, G.k1);
  float g0, g1, g2;
  normals3(o, g0, g1, g2);
  u64* s = sums + (size_t)k * G.sw;
  atomicAdd(s + 1, pack_ss(__float2int_rn(vx[i] * G.fxv), __float2int_rn(vy[i] * G.fxv)));
  atomicAdd(s + 2, pack_ss(__float2int_rn(vz[i] * G.fxv), __float2int_rn(G.sigma * g0 * G.fxv)));
  atomicAdd(s + 3, pack_ss(__float2int_rn(G.sigma * g1 * G.fxv), __float2int_rn(G.sigma * g2 * G.fxv)));
}
__global__ void __launch_bounds__(256) k_collide_at(Geo G, size_t n, float* __restrict__ vx, float* __restrict__ vy,
                                                    float* __restrict__ vz, const uint32_t* __restrict__ key,
                                                    const uint32_t* __restrict__ offset, const float* __restrict__ rec) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t k = key[i];
  const float4 r0 = __ldg(reinterpret_cast<const float4*>(rec) + (size_t)k * 2);
  int ix, iy, iz;
  key_to_cell(G, k, ix, iy, iz);
  const Block4 o = philox(canonical_id(G, ix, iy, iz), (uint32_t)i - offset[k], G.t, TAG_AT, G.k0, G.k1);
  float g0, g1, g2;
  normals3(o, g0, g1, g2);
  vx[i] = r0.x + G.sigma * g0;
  vy[i] = r0.y + G.sigma * g1;
  vz[i] = r0.z + G.sigma * g2;
}

// ---- +a variants (Eqs. 3-4; MPC-AT+a, U5): unfused path --------------------------------
constexpr float FX_RHO = 4194304.0f;            // 2^22 per unit of cell-local coordinate (products too): N_c < 512
constexpr double FX_RHO_INV = 1.0 / 4194304.0;

__device__ __forceinline__ void srd_axis(const Geo& G, uint32_t cid, float& ax, float& ay, float& az) {
  const Block4 o = philox(cid, 0u, G.t, TAG_AXIS, G.k0, G.k1);
  az = 2.0f * u01_co(o.a) - 1.0f;
  const float rr = sqrtf((1.0f - az) * (1.0f + az));
  float sp, cp;
  sincospif(2.0f * u01_co(o.b), &sp, &cp);
  ax = rr * cp; ay = rr * sp;
}
// D(alpha) w for unit axis n (Rodrigues, right-handed)
__device__ __forceinline__ void rotate(const Geo& G, float nx, float ny, float nz, const float (&w)[3], float (&o)[3]) {
  const float c = G.cosa, s = G.sina;
  const float nd = fmaf(nx, w[0], fmaf(ny, w[1], nz * w[2])) * (1.0f - c);
  const float cx = fmaf(ny, w[2], -(nz * w[1])), cy = fmaf(nz, w[0], -(nx * w[2])), cz = fmaf(nx, w[1], -(ny * w[0]));
  o[0] = fmaf(w[0], c, fmaf(cx, s, nx * nd));
  o[1] = fmaf(w[1], c, fmaf(cy, s, ny * nd));
  o[2] = fmaf(w[2], c, fmaf(cz, s, nz * nd));
}
__device__ __forceinline__ float cell_frac(const Geo& G, float r, float s) {
  const float q = (r + s) * G.inv_a;
  return q - floorf(q);
}

template <bool AT>
__global__ void __launch_bounds__(256) k_accum_a(Geo G, size_t n, const float* __restrict__ x, const float* __restrict__ y,
                                                 const float* __restrict__ z, const float* __restrict__ vx,
                                                 const float* __restrict__ vy, const float* __restrict__ vz,
                                                 const uint32_t* __restrict__ key, const uint32_t* __restrict__ offset,
                                                 u64* __restrict__ sums) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t k = key[i];
  int ix, iy, iz;
  key_to_cell(G, k, ix, iy, iz);
  const uint32_t cid = canonical_id(G, ix, iy, iz);
  const float v[3] = {vx[i], vy[i], vz[i]};
  const float r0 = cell_frac(G, x[i], G.s[0]), r1 = cell_frac(G, y[i], G.s[1]), r2 = cell_frac(G, z[i], G.s[2]);
  float u[3], g[3] = {0.f, 0.f, 0.f};
  if (AT) {
    const Block4 o = philox(cid, (uint32_t)i - offset[k], G.t, TAG_AT, G.k0, G.k1);
    normals3(o, g[0], g[1], g[2]);
    g[0] *= G.sigma; g[1] *= G.sigma; g[2] *= G.sigma;
    u[0] = v[0] - g[0]; u[1] = v[1] - g[1]; u[2] = v[2] - g[2];
  } else {
    float ax, ay, az, d[3];
    srd_axis(G, cid, ax, ay, az);
    rotate(G, ax, ay, az, v, d);
    u[0] = v[0] - d[0]; u[1] = v[1] - d[1]; u[2] = v[2] - d[2];
  }
  const float l0 = fmaf(r1, u[2], -(r2 * u[1])), l1 = fmaf(r2, u[0], -(r0 * u[2])), l2 = fmaf(r0, u[1], -(r1 * u[0]));
  u64* s = sums + (size_t)k * G.sw;
  auto fv = [&](float a) { return __float2int_rn(a * G.fxv); };
  auto fq = [&](float a) { return __float2int_rn(a * FX_RHO); };
  atomicAdd(s + 1, pack_ss(fv(v[0]), fv(v[1])));
  atomicAdd(s + 2, pack_ss(fv(v[2]), AT ? fv(g[0]) : 0));
  if (AT) atomicAdd(s + 3, pack_ss(fv(g[1]), fv(g[2])));
  atomicAdd(s + 4, pack_ss(fq(r0), fq(r1)));
  atomicAdd(s + 5, pack_ss(fq(r2), fq(r0 * r0)));
  atomicAdd(s + 6, pack_ss(fq(r1 * r1), fq(r2 * r2)));
  atomicAdd(s + 7, pack_ss(fq(r0 * r1), fq(r0 * r2)));
  atomicAdd(s + 8, pack_ss(fq(r1 * r2), fv(l0)));
  atomicAdd(s + 9, pack_ss(fv(l1), fv(l2)));
}

// Segmented variant of k_accum_at / k_accum_a for a step that has just reordered: the particles of cell k are
// the contiguous segment [offset[k], offset[k+1]) in (key, id) order, so one thread sums its cell in registers
// and stores the packed words: no atomics (the atomic versions are bound by ~190 G global atomics/s) and the same
// integers (two's-complement adds of the same addends, any order).
template <bool AT, bool PLUS_A>
__global__ void __launch_bounds__(128) k_accum_seg(Geo G, int cpb_shift, const float* __restrict__ x, const float* __restrict__ y,
                                                   const float* __restrict__ z, const float* __restrict__ vx,
                                                   const float* __restrict__ vy, const float* __restrict__ vz,
                                                   const uint32_t* __restrict__ offset, u64* __restrict__ sums) {
  const int b0 = G.bs[0], b1 = G.bs[1], b2 = G.bs[2];
  const uint32_t bx = blockIdx.x >> cpb_shift, by = blockIdx.y, bz = blockIdx.z;
  const uint32_t local = ((blockIdx.x & ((1u << cpb_shift) - 1u)) << 7) | threadIdx.x;
  if (local >= (1u << (b0 + b1 + b2))) return;
  const uint32_t brick = (bz * (uint32_t)G.mb[1] + by) * (uint32_t)G.mb[0] + bx;
  const uint32_t k = (brick << (b0 + b1 + b2)) | local;
  const uint32_t jb = offset[k], je = offset[k + 1];
  if (jb == je) return;
  const int ix = (int)((bx << b0) | (local & ((1u << b0) - 1u)));
  const int iy = (int)((by << b1) | ((local >> b0) & ((1u << b1) - 1u)));
  const int iz = (int)((bz << b2) | (local >> (b0 + b1)));
  const uint32_t cid = canonical_id(G, ix, iy, iz);
  float ax = 0.f, ay = 0.f, az = 0.f;
  if (!AT) srd_axis(G, cid, ax, ay, az);
  int S[18];
#pragma unroll
  for (int q = 0; q < 18; ++q) S[q] = 0;
  auto fv = [&](float a) { return __float2int_rn(a * G.fxv); };
  auto fq = [&](float a) { return __float2int_rn(a * FX_RHO); };
  for (uint32_t j = jb; j < je; ++j) {
    const float v[3] = {vx[j], vy[j], vz[j]};
    float u[3], g[3] = {0.f, 0.f, 0.f};
    if (AT) {
      const Block4 o = philox(cid, j - jb, G.t, TAG_AT, G.k0, G.k1);
      normals3(o, g[0], g[1], g[2]);
      g[0] *= G.sigma; g[1] *= G.sigma; g[2] *= G.sigma;
      u[0] = v[0] - g[0]; u[1] = v[1] - g[1]; u[2] = v[2] - g[2];
    } else {
      float d[3];
      rotate(G, ax, ay, az, v, d);
      u[0] = v[0] - d[0]; u[1] = v[1] - d[1]; u[2] = v[2] - d[2];
    }
    S[0] += fv(v[0]); S[1] += fv(v[1]); S[2] += fv(v[2]);
    if (AT) { S[3] += fv(g[0]); S[4] += fv(g[1]); S[5] += fv(g[2]); }
    if (PLUS_A) {
      const float r0 = cell_frac(G, x[j], G.s[0]), r1 = cell_frac(G, y[j], G.s[1]), r2 = cell_frac(G, z[j], G.s[2]);
      const float l0 = fmaf(r1, u[2], -(r2 * u[1])), l1 = fmaf(r2, u[0], -(r0 * u[2])), l2 = fmaf(r0, u[1], -(r1 * u[0]));
      S[6] += fq(r0); S[7] += fq(r1); S[8] += fq(r2); S[9] += fq(r0 * r0); S[10] += fq(r1 * r1); S[11] += fq(r2 * r2);
      S[12] += fq(r0 * r1); S[13] += fq(r0 * r2); S[14] += fq(r1 * r2); S[15] += fv(l0); S[16] += fv(l1); S[17] += fv(l2);
    }
  }
  u64* s = sums + (size_t)k * G.sw;
  s[1] = pack_ss(S[0], S[1]);
  s[2] = pack_ss(S[2], S[3]);
  if (AT) s[3] = pack_ss(S[4], S[5]);
  if (PLUS_A) {
    s[4] = pack_ss(S[6], S[7]); s[5] = pack_ss(S[8], S[9]); s[6] = pack_ss(S[10], S[11]);
    s[7] = pack_ss(S[12], S[13]); s[8] = pack_ss(S[14], S[15]); s[9] = pack_ss(S[16], S[17]);
  }
}

// rec[key] (16 floats) = { base.xyz, 1 | axis.xyz, - | omega.xyz, - | rho_cm.xyz, - }
//   SRD+a: base = v_cm ; AT+a: base = v_cm - mean(v_ran)
template <bool AT>
__global__ void __launch_bounds__(128) k_cell_a(Geo G, int cpb_shift, const u64* __restrict__ sums, float* __restrict__ rec,
                                                u64* __restrict__ nsing) {
  const int b0 = G.bs[0], b1 = G.bs[1], b2 = G.bs[2];
  const uint32_t bx = blockIdx.x >> cpb_shift, by = blockIdx.y, bz = blockIdx.z;
  const uint32_t local = ((blockIdx.x & ((1u << cpb_shift) - 1u)) << 7) | threadIdx.x;
  if (local >= (1u << (b0 + b1 + b2))) return;
  const uint32_t brick = (bz * (uint32_t)G.mb[1] + by) * (uint32_t)G.mb[0] + bx;
  const uint32_t k = (brick << (b0 + b1 + b2)) | local;
  const u64* s = sums + (size_t)k * G.sw;
  const uint32_t N = (uint32_t)(s[0] & 0xffffull);
  if (N == 0u) return;
  const int ix = (int)((bx << b0) | (local & ((1u << b0) - 1u)));
  const int iy = (int)((by << b1) | ((local >> b0) & ((1u << b1) - 1u)));
  const int iz = (int)((bz << b2) | (local >> (b0 + b1)));
  const uint32_t cid = canonical_id(G, ix, iy, iz);
  int i0, i1, i2, i3, i4, i5;
  unpack_ss(s[1], i0, i1); unpack_ss(s[2], i2, i3);
  const double inv = 1.0 / (double)N;
  const double S[3] = {i0 * G.fxv_inv, i1 * G.fxv_inv, i2 * G.fxv_inv};
  double R[3] = {i3 * G.fxv_inv, 0.0, 0.0};
  if (AT) { unpack_ss(s[3], i4, i5); R[1] = i4 * G.fxv_inv; R[2] = i5 * G.fxv_inv; }
  float ax = 0.f, ay = 0.f, az = 1.f;
  double Su[3];
  if (AT) { Su[0] = S[0] - R[0]; Su[1] = S[1] - R[1]; Su[2] = S[2] - R[2]; }
  else {
    srd_axis(G, cid, ax, ay, az);
    // (1 - D) S in double, with the fp32 axis and the fp32 cos/sin the particles used
    const double c = G.cosa, sn = G.sina, nx = ax, ny = ay, nz = az;
    const double nd = (nx * S[0] + ny * S[1] + nz * S[2]) * (1.0 - c);
    const double cx = ny * S[2] - nz * S[1], cy = nz * S[0] - nx * S[2], cz = nx * S[1] - ny * S[0];
    Su[0] = S[0] - (S[0] * c + cx * sn + nx * nd);
    Su[1] = S[1] - (S[1] * c + cy * sn + ny * nd);
    Su[2] = S[2] - (S[2] * c + cz * sn + nz * nd);
  }
  double om[3] = {0.0, 0.0, 0.0}, rcm[3] = {0.0, 0.0, 0.0};
  if (N >= 2u) {
    int q0, q1, q2, q3, q4, q5, q6, q7, q8, q9, q10, q11;
    unpack_ss(s[4], q0, q1); unpack_ss(s[5], q2, q3); unpack_ss(s[6], q4, q5);
    unpack_ss(s[7], q6, q7); unpack_ss(s[8], q8, q9); unpack_ss(s[9], q10, q11);
    rcm[0] = q0 * FX_RHO_INV * inv; rcm[1] = q1 * FX_RHO_INV * inv; rcm[2] = q2 * FX_RHO_INV * inv;
    const double a = G.a, m = G.mass, Nd = (double)N;
    // second moments about the centre of mass, in units of a^2
    const double Qxx = q3 * FX_RHO_INV - Nd * rcm[0] * rcm[0], Qyy = q4 * FX_RHO_INV - Nd * rcm[1] * rcm[1];
    const double Qzz = q5 * FX_RHO_INV - Nd * rcm[2] * rcm[2], Qxy = q6 * FX_RHO_INV - Nd * rcm[0] * rcm[1];
    const double Qxz = q7 * FX_RHO_INV - Nd * rcm[0] * rcm[2], Qyz = q8 * FX_RHO_INV - Nd * rcm[1] * rcm[2];
    const double Lr[3] = {q9 * G.fxv_inv, q10 * G.fxv_inv, q11 * G.fxv_inv};
    const double dL[3] = {m * a * (Lr[0] - (rcm[1] * Su[2] - rcm[2] * Su[1])),
                          m * a * (Lr[1] - (rcm[2] * Su[0] - rcm[0] * Su[2])),
                          m * a * (Lr[2] - (rcm[0] * Su[1] - rcm[1] * Su[0]))};
    const double R2 = a * a * (Qxx + Qyy + Qzz);
    if (N == 2u) {
      if (R2 > 0.0) { om[0] = dL[0] / (m * R2); om[1] = dL[1] / (m * R2); om[2] = dL[2] / (m * R2); }
    } else {
      const double f = m * a * a;
      const double xx = f * (Qyy + Qzz), yy = f * (Qxx + Qzz), zz = f * (Qxx + Qyy), xy = -f * Qxy, xz = -f * Qxz, yz = -f * Qyz;
      const double c00 = yy * zz - yz * yz, c01 = xz * yz - xy * zz, c02 = xy * yz - xz * yy;
      const double c11 = xx * zz - xz * xz, c12 = xy * xz - xx * yz, c22 = xx * yy - xy * xy;
      const double det = xx * c00 + xy * c01 + xz * c02, tr3 = (xx + yy + zz) / 3.0;
      if (det > 1e-6 * tr3 * tr3 * tr3) {
        om[0] = (c00 * dL[0] + c01 * dL[1] + c02 * dL[2]) / det;
        om[1] = (c01 * dL[0] + c11 * dL[1] + c12 * dL[2]) / det;
        om[2] = (c02 * dL[0] + c12 * dL[1] + c22 * dL[2]) / det;
      } else {
        atomicAdd(nsing, 1ull);     // rejected inertia tensor (U10): omega = 0
      }
    }
  }
  float4* o = reinterpret_cast<float4*>(rec) + (size_t)k * 4;
  if (AT) o[0] = make_float4((float)((S[0] - R[0]) * inv), (float)((S[1] - R[1]) * inv), (float)((S[2] - R[2]) * inv), 1.0f);
  else o[0] = make_float4((float)(S[0] * inv), (float)(S[1] * inv), (float)(S[2] * inv), 1.0f);
  o[1] = make_float4(ax, ay, az, 0.0f);
  o[2] = make_float4((float)om[0], (float)om[1], (float)om[2], 0.0f);
  o[3] = make_float4((float)rcm[0], (float)rcm[1], (float)rcm[2], 0.0f);
}

template <bool AT>
__global__ void __launch_bounds__(256) k_collide_a(Geo G, size_t n, const float* __restrict__ x, const float* __restrict__ y,
                                                   const float* __restrict__ z, float* __restrict__ vx, float* __restrict__ vy,
                                                   float* __restrict__ vz, const uint32_t* __restrict__ key,
                                                   const uint32_t* __restrict__ offset, const float* __restrict__ rec) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t k = key[i];
  const float4* rc = reinterpret_cast<const float4*>(rec) + (size_t)k * 4;
  const float4 base = __ldg(rc), axis = __ldg(rc + 1), om = __ldg(rc + 2), rcm = __ldg(rc + 3);
  float o[3];
  if (AT) {
    int ix, iy, iz;
    key_to_cell(G, k, ix, iy, iz);
    const Block4 b = philox(canonical_id(G, ix, iy, iz), (uint32_t)i - offset[k], G.t, TAG_AT, G.k0, G.k1);
    float g0, g1, g2;
    normals3(b, g0, g1, g2);
    o[0] = base.x + G.sigma * g0; o[1] = base.y + G.sigma * g1; o[2] = base.z + G.sigma * g2;
  } else {
    const float w[3] = {vx[i] - base.x, vy[i] - base.y, vz[i] - base.z};
    float d[3];
    rotate(G, axis.x, axis.y, axis.z, w, d);
    o[0] = base.x + d[0]; o[1] = base.y + d[1]; o[2] = base.z + d[2];
  }
  const float r0 = (cell_frac(G, x[i], G.s[0]) - rcm.x) * G.a, r1 = (cell_frac(G, y[i], G.s[1]) - rcm.y) * G.a,
              r2 = (cell_frac(G, z[i], G.s[2]) - rcm.z) * G.a;
  vx[i] = o[0] + fmaf(om.y, r2, -(om.z * r1));
  vy[i] = o[1] + fmaf(om.z, r0, -(om.x * r2));
  vz[i] = o[2] + fmaf(om.x, r1, -(om.y * r0));
}

// ---- exclusive scan of the per-cell counts (three kernels; tile = 2048) ----------------------------
// `in` is read with a stride in 32-bit words: the count is the low 16 bits of word 0 of a cell's sums.
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

// ---- reorder by (key, id) -----------------------------------------------------------------------
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
// Step 1: every particle takes a slot of its cell segment in arrival order. Particles of one cell are
// mostly lane neighbours (the array is still nearly sorted), so the lanes of a warp with the same key
// share ONE cursor atomic (match.any + leader), which is what bounds this kernel otherwise.
__global__ void __launch_bounds__(256) k_scatter_slots(size_t n, const uint32_t* __restrict__ key, const uint32_t* __restrict__ id,
                                                       const uint32_t* __restrict__ offset, uint32_t* __restrict__ cursor,
                                                       uint2* __restrict__ slot) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t k = key[i];
  const uint32_t s = offset[k] + run_slot(k, cursor);
  slot[s] = make_uint2(id[i], (uint32_t)i);   // one 8-byte store: (id, source index)
}
// Step 2, one thread per slot: rank of the slot's particle inside its cell = number of cell mates with a
// smaller id (U4); perm[first slot of the cell + rank] = source index. Reads and writes of a
// warp stay inside the few segments its 32 consecutive slots belong to.
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
// Hot-path variant (SRD): the order inside a cell does not enter the physics (integer cell sums), so the
// reorder only groups the particles by key: perm[slot] = source index, slots in arrival order. The canonical
// (key, id) order is restored by k_rank_cells + gather before the state is read (canonicalise()).
// Four independent particles per thread (block-strided): the kernel is bound by the latency of the chain
// key load -> cursor atomic (with return) -> store, so four chains in flight per thread pay for themselves.
constexpr int SCAT_U = 4;
__global__ void __launch_bounds__(256) k_scatter_src(size_t n, const uint32_t* __restrict__ key, const uint32_t* __restrict__ offset,
                                                     uint32_t* __restrict__ cursor, uint32_t* __restrict__ perm) {
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
    if (ok[j]) perm[off[j] + b + (lane - (unsigned)leader[j])] = (uint32_t)(base + (size_t)j * 256);
  }
}
// one thread per cell: the particles of segment [offset[k], offset[k+1]) ranked by id
__global__ void __launch_bounds__(256) k_rank_cells(size_t nkeys, const uint32_t* __restrict__ offset, const uint32_t* __restrict__ id,
                                                    uint32_t* __restrict__ perm) {
  const size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= nkeys) return;
  const uint32_t b = offset[k], e = offset[k + 1];
  for (uint32_t j = b; j < e; ++j) {
    const uint32_t me = id[j];
    uint32_t r = 0;
    for (uint32_t m = b; m < e; ++m) r += (id[m] < me) ? 1u : 0u;
    perm[b + r] = j;
  }
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
__global__ void __launch_bounds__(256) k_iota(size_t n, uint32_t* __restrict__ id) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) id[i] = (uint32_t)i;
}

// ---- PROCESS_CELLS -------------------------------------------------------------------------------
// E_k / k_BT ~ Gamma(3(Nc-1)/2, 1) (Eq. 7; U6): minus the log of a product of floor(f/2)
// uniforms (the product is renormalised with frexp so it never underflows: one log per cell instead
// of one per uniform), plus half a squared normal if f is odd.
__device__ __forceinline__ void renorm(float& p, int& ex) {   // p = m * 2^e with m in [0.5,1): keep m, bank e
  const int bits = __float_as_int(p);
  ex += (bits >> 23) - 126;
  p = __int_as_float((bits & 0x007fffff) | 0x3f000000);
}
// 2^24 * u01_oc(w): the power-of-two scale of every uniform is banked in the exponent instead (exact)
__device__ __forceinline__ float u24_oc(uint32_t w) { return (float)((w >> 8) + 1u); }
// wm, wa: words 2 and 3 of the cell's TAG_AXIS block, the two uniforms of the half squared normal (f odd)
__device__ float mbs_energy(const Geo& G, uint32_t cid, uint32_t Nc, uint32_t wm, uint32_t wa) {
  const uint32_t f = 3u * (Nc - 1u), M = f >> 1, odd = f & 1u;
  const uint32_t full = M >> 2, rem = M & 3u;    // blocks whose four uniforms all enter the product; uniforms of the last one
  float p = 1.0f;
  int ex = -24 * (int)M;                         // M uniforms enter the product, each carried as 2^24 u
  uint32_t sub = 0;
  for (; sub < full; ++sub) {
    const Block4 o = philox_rk(cid, sub, G.t, TAG_MBS, G.rk);
    p *= (u24_oc(o.a) * u24_oc(o.b)) * (u24_oc(o.c) * u24_oc(o.d));   // < 2^96: cannot overflow
    renorm(p, ex);
  }
  if (rem) {
    const Block4 o = philox_rk(cid, full, G.t, TAG_MBS, G.rk);
    float q = u24_oc(o.a);
    q *= (rem > 1u) ? u24_oc(o.b) : 1.0f;
    q *= (rem > 2u) ? u24_oc(o.c) : 1.0f;
    p *= q;
    renorm(p, ex);
  }
  float e = -(float)((double)logf(p) + (double)ex * 0.6931471805599453);
  if (odd) {
    const float cs = cospif(2.0f * u01_co(wa));
    e -= logf(u01_oc(wm)) * cs * cs;
  }
  return e;
}

// rec[key] = SRD: { vcm.x, vcm.y, vcm.z, kappa, n.x, n.y, n.z, - }   AT: { (vcm - mean v_ran).xyz, ... }
// grid = (mb0 * CTAs-per-brick, mb1, mb2): the brick coordinates come from blockIdx, no division
// zero != 0: the sums of a cell are cleared once read, which saves the memset before the next step's sweep
// one cell: (bx, by, bz) = brick coordinates, local = index of the cell inside its brick
__device__ __forceinline__ void cell_finalize(const Geo& G, uint32_t bx, uint32_t by, uint32_t bz, uint32_t local,
                                              u64* __restrict__ sums, float* __restrict__ rec, int zero) {
  const int b0 = G.bs[0], b1 = G.bs[1], b2 = G.bs[2];
  if (local >= (1u << (b0 + b1 + b2))) return;
  const uint32_t brick = (bz * (uint32_t)G.mb[1] + by) * (uint32_t)G.mb[0] + bx;
  const uint32_t k = (brick << (b0 + b1 + b2)) | local;
  u64* s = sums + (size_t)k * G.sw;
  const u64 w0 = s[0];
  const uint32_t nreal = (uint32_t)(w0 & 0xffffull);
  if (nreal == 0u) return;
  const int ix = (int)((bx << b0) | (local & ((1u << b0) - 1u)));
  const int iy = (int)((by << b1) | ((local >> b0) & ((1u << b1) - 1u)));
  const int iz = (int)((bz << b2) | (local >> (b0 + b1)));
  const uint32_t cid = canonical_id(G, ix, iy, iz);
  int sx, sy, sz, r0i;
  unpack_ss(s[1], sx, sy);
  unpack_ss(s[2], sz, r0i);
  if (zero) { s[0] = 0ull; s[1] = 0ull; s[2] = 0ull; }
  double S0 = (double)sx * G.fxv_inv, S1 = (double)sy * G.fxv_inv, S2 = (double)sz * G.fxv_inv;
  float4 r0, r1;
  if (G.collision == 1) {
    int r1i, r2i;
    unpack_ss(s[3], r1i, r2i);
    const double inv = 1.0 / (double)nreal;
    r0.x = (float)((S0 - (double)r0i * G.fxv_inv) * inv);
    r0.y = (float)((S1 - (double)r1i * G.fxv_inv) * inv);
    r0.z = (float)((S2 - (double)r2i * G.fxv_inv) * inv);
    r0.w = 1.0f;
    r1 = make_float4(0.f, 0.f, 0.f, 0.f);
  } else {
    double E = (double)(w0 >> 16) * G.fxe_inv;
    uint32_t Nc = nreal;
    if (G.wall >= 0 && !G.slip) {
      // virtual wall particles fill wall-cut cells up to nbar (U8)
      const int w = G.wall;
      const int iw = (w == 0) ? ix : (w == 1) ? iy : iz;
      const float sw = (w == 0) ? G.s[0] : (w == 1) ? G.s[1] : G.s[2];
      const int nw = (w == 0) ? G.n[0] : (w == 1) ? G.n[1] : G.n[2];
      const bool cut = (sw > 0.0f) ? (iw == 1 || iw == nw + 1) : (sw < 0.0f) ? (iw == 0 || iw == nw) : false;
      if (cut && (int)nreal < G.nbar) {
        const uint32_t nv = (uint32_t)G.nbar - nreal;
        for (uint32_t j = 0; j < nv; ++j) {
          const Block4 o = philox_rk(cid, j, G.t, TAG_WALL, G.rk);
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
    const Block4 o = philox_rk(cid, 0u, G.t, TAG_AXIS, G.rk);
    float kappa = 1.0f;
    if (G.thermostat && Nc >= 2u) {
      const double W2 = E - (S0 * S0 + S1 * S1 + S2 * S2) * inv;   // sum |v - vcm|^2
      if (W2 > 0.0) {
        const float ek = G.kT * mbs_energy(G, cid, Nc, o.c, o.d);
        kappa = sqrtf(2.0f * ek / (G.mass * (float)W2));
      }
    }
    r0.w = kappa;
    const float zz = 2.0f * u01_co(o.a) - 1.0f;
    const float rr = sqrtf((1.0f - zz) * (1.0f + zz));
    float sp, cp;
    sincospif(2.0f * u01_co(o.b), &sp, &cp);
    r1 = make_float4(rr * cp, rr * sp, zz, 0.0f);
  }
  reinterpret_cast<float4*>(rec)[(size_t)k * 2] = r0;
  reinterpret_cast<float4*>(rec)[(size_t)k * 2 + 1] = r1;
}
__global__ void __launch_bounds__(128) k_cell(Geo G, int cpb_shift, u64* __restrict__ sums, float* __restrict__ rec, int zero) {
  cell_finalize(G, blockIdx.x >> cpb_shift, blockIdx.y, blockIdx.z, ((blockIdx.x & ((1u << cpb_shift) - 1u)) << 7) | threadIdx.x,
                sums, rec, zero);
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
__global__ void __launch_bounds__(256) k_obs_cells(Geo G, const u64* __restrict__ sums, double* __restrict__ part) {
  __shared__ double sh[8];
  __shared__ unsigned smax;
  if (threadIdx.x == 0) smax = 0;
  __syncthreads();
  double num = 0, den = 0;
  unsigned mx = 0;
  for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < G.nkeys; k += (size_t)gridDim.x * blockDim.x) {
    const u64* s = sums + k * G.sw;
    const u64 w0 = s[0];
    const unsigned nc = (unsigned)(w0 & 0xffffull);
    mx = max(mx, nc);
    if (nc < 2u || G.generic) continue;
    int sx, sy, sz, sp;
    unpack_ss(s[1], sx, sy);
    unpack_ss(s[2], sz, sp);
    const double S0 = sx * G.fxv_inv, S1 = sy * G.fxv_inv, S2 = sz * G.fxv_inv;
    num += (double)G.mass * ((double)(w0 >> 16) * G.fxe_inv - (S0 * S0 + S1 * S1 + S2 * S2) / nc);
    den += 3.0 * (nc - 1u);
  }
  atomicMax(&smax, mx);
  num = block_sum(num, sh); den = block_sum(den, sh);
  if (threadIdx.x == 0) { double* o = part + (size_t)blockIdx.x * 8; o[4] = num; o[5] = den; o[6] = (double)smax; }
}
__global__ void __launch_bounds__(256) k_obs_profile(Geo G, size_t n, int nb, const float* __restrict__ rp,
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
__global__ void __launch_bounds__(256) k_export_cells(Geo G, const u64* __restrict__ sums, unsigned* __restrict__ count,
                                                      float* __restrict__ px, float* __restrict__ py, float* __restrict__ pz,
                                                      float* __restrict__ e2) {
  const size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= G.nkeys) return;
  const u64* s = sums + k * G.sw;
  int sx, sy, sz, sp;
  unpack_ss(s[1], sx, sy);
  unpack_ss(s[2], sz, sp);
  if (count) count[k] = (unsigned)(s[0] & 0xffffull);
  if (px) px[k] = (float)((double)G.mass * sx * G.fxv_inv);
  if (py) py[k] = (float)((double)G.mass * sy * G.fxv_inv);
  if (pz) pz[k] = (float)((double)G.mass * sz * G.fxv_inv);
  if (e2) e2[k] = G.generic ? 0.0f : (float)((double)(s[0] >> 16) * G.fxe_inv);
}

}  // namespace mpc

// =================================================================================================
// host side
// =================================================================================================
using namespace mpc;

enum Family { F_SWEEP = 0, F_CELL, F_COLLIDE, F_SCAN, F_SCATTER, F_RANK, F_GATHER, F_MEMSET, F_STREAM, F_ACCUM, F_OBS, F_SWEEPG, F_COUNT };
static const char* const FAMILY_NAMES[F_COUNT] = {"sweep", "cell", "collide", "scan", "scatter_slots", "rank", "gather", "memset",
                                                  "stream_key", "accum", "observables", "sweep_gather"};
constexpr int PROF_MAX_PAIRS = 16384;

struct mpc_ctx {
  Geo G;
  mpc_params p;
  unsigned long long seed;
  uint32_t t;
  size_t n, n_max;
  bool bound, have_state, have_cells, have_order, compact, sticky, fast_brick, sums_clean, gather_pending, no_fuse_gather, order_canonical, eager_canonical, three_ctas;
  cudaStream_t stream;
  cudaStream_t stream2;       // side stream: PROCESS_CELLS of a reorder step runs beside the reorder's scatter
  cudaEvent_t ev_scan, ev_cell;
  bool side_ready, no_overlap;
  char* ws;
  size_t ws_bytes;
  uint32_t nbricks;
  size_t tile_bytes;
  dim3 cell_grid;       // k_cell launch: (mb0 << cell_cpb_shift, mb1, mb2) CTAs of 128 cells
  int cell_cpb_shift;
  // device arrays
  uint32_t* A[7];   // x y z vx vy vz id (current)
  uint32_t* Bf[7];  // second copy (non-compact); Bf[0] = 4-byte temp (compact)
  uint32_t *key, *slot_id, *perm, *cursor, *offset, *bsum;
  u64* sums;
  float* rec;
  double* obs;      // OBS_BLOCKS*8 doubles + 2*MAX_PROFILE doubles
  u64* nsing;       // +a: number of rejected inertia tensors in the last step
  double* hbuf;     // host staging for mpc_observables
  // optional per-family timing with CUDA events on the bound stream (mpc_profile_*)
  bool prof_on;
  cudaEvent_t* prof_ev;
  int* prof_fam;
  int prof_pairs;
  double prof_ms[F_COUNT];
  unsigned long long prof_launches[F_COUNT];
  unsigned long long launches;
  char err[256];
};

namespace {

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Layout {
  size_t off_A[7], off_B[7], off_key, off_slot, off_perm, off_cursor, off_offset, off_bsum, off_sums, off_rec, off_obs, total;
};
Layout make_layout(size_t n_max, size_t nkeys, int sw, int rw, bool compact) {
  Layout l;
  size_t o = 0;
  auto take = [&](size_t bytes) { const size_t r = o; o = align_up(o + bytes, 256); return r; };
  const size_t pn = align_up((n_max ? n_max : 1) * 4, 256);   // whole 256-byte units: consecutive arrays are contiguous
  for (int a = 0; a < 7; ++a) l.off_A[a] = take(pn);
  // the slot array sits between the two particle copies: either copy plus it = 8 contiguous arrays (aos_base)
  l.off_slot = take(compact ? pn * 2 : pn);
  if (compact) { l.off_B[0] = take(pn); for (int a = 1; a < 7; ++a) l.off_B[a] = l.off_B[0]; }
  else for (int a = 0; a < 7; ++a) l.off_B[a] = take(pn);
  l.off_key = take(pn);
  // (the slot array holds (id, source index) pairs, 8 bytes each, in compact mode; with the second copy present
  // those live in its first two arrays and the slot array only receives the sorted keys of the unfused path)
  l.off_perm = take(pn);
  l.off_cursor = take(nkeys * 4);
  l.off_offset = take((nkeys + 1) * 4);
  l.off_bsum = take(((nkeys + SCAN_TILE - 1) / SCAN_TILE + 1) * 4);
  l.off_sums = take(nkeys * (size_t)sw * 8);
  l.off_rec = take(nkeys * (size_t)rw * 4);
  l.off_obs = take(OBS_HOST_DOUBLES * 8 + 256);
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
  mpc_ctx* c; int slot; cudaStream_t st;
  FamilyTimer(mpc_ctx* c_, int fam, cudaStream_t st_ = nullptr) : c(c_), slot(-1), st(st_ ? st_ : c_->stream) {
    if (!c->prof_on) return;
    c->prof_launches[fam]++;
    if (c->prof_pairs >= PROF_MAX_PAIRS) return;
    slot = c->prof_pairs++;
    c->prof_fam[slot] = fam;
    cudaEventRecord(c->prof_ev[2 * slot], st);
  }
  ~FamilyTimer() { if (slot >= 0) cudaEventRecord(c->prof_ev[2 * slot + 1], st); }
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

// particle arrays (and the keys, if asked) gathered through c->perm: new[i] = old[perm[i]]
int apply_perm(mpc_ctx* c, bool need_key) {
  const size_t n = c->n;
  FamilyTimer ftg(c, F_GATHER);
  if (!c->compact) {
    Arrays8 src, dst;
    for (int a = 0; a < 7; ++a) { src.p[a] = c->A[a]; dst.p[a] = c->Bf[a]; }
    src.p[7] = c->key; dst.p[7] = c->slot_id;
    if (need_key) k_gather<8><<<nblk(n, 256), 256, 0, c->stream>>>(n, c->perm, src, dst);
    else k_gather<7><<<nblk(n, 256), 256, 0, c->stream>>>(n, c->perm, src, dst);
    LAUNCH_CHECK("k_gather");
    for (int a = 0; a < 7; ++a) { uint32_t* t = c->A[a]; c->A[a] = c->Bf[a]; c->Bf[a] = t; }
    if (need_key) CU(cudaMemcpyAsync(c->key, c->slot_id, n * 4, cudaMemcpyDeviceToDevice, c->stream));
  } else {
    // property-wise through one temporary array: each property is gathered into the spare array,
    // which then takes its place; the array it came from is the spare for the next property (no copy back)
    Arrays8 src, dst;
    for (int a = 0; a < (need_key ? 8 : 7); ++a) {
      uint32_t*& arr = a < 7 ? c->A[a] : c->key;
      src.p[0] = arr; dst.p[0] = c->Bf[0];
      k_gather<1><<<nblk(n, 256), 256, 0, c->stream>>>(n, c->perm, src, dst);
      LAUNCH_CHECK("k_gather");
      uint32_t* t = arr; arr = c->Bf[0];
      for (int b = 0; b < 7; ++b) c->Bf[b] = t;     // compact mode: all seven alias the one spare array
    }
  }
  return MPC_OK;
}

// counting-sort reorder by (key, id); counts = low word of word 0 of the sums; c->key holds the keys
// defer_gather: leave the permutation in c->perm for the next sweep to apply (launch_sweep<.., GATHER>)
// canonical: rank the particles of a cell by id now (needed by MPC-AT); otherwise group by key only
// cell_zero >= 0: launch k_cell(zero = cell_zero) on the side stream once the counts have been scanned
int do_reorder(mpc_ctx* c, bool defer_gather, bool canonical, int cell_zero = -1) {
  const size_t n = c->n, nk = c->G.nkeys, nb = (nk + SCAN_TILE - 1) / SCAN_TILE;
  const uint32_t* cnt = reinterpret_cast<const uint32_t*>(c->sums);
  const int stride = c->G.sw * 2;
  {
    FamilyTimer ft(c, F_SCAN);
    k_scan_reduce<<<(unsigned)nb, SCAN_T, 0, c->stream>>>(cnt, stride, nk, c->bsum);
    LAUNCH_CHECK("k_scan_reduce");
    k_scan_top<<<1, 1024, 0, c->stream>>>(c->bsum, nb);
    LAUNCH_CHECK("k_scan_top");
    k_scan_apply<<<(unsigned)nb, SCAN_T, 0, c->stream>>>(cnt, stride, nk, c->bsum, c->offset);
    LAUNCH_CHECK("k_scan_apply");
  }
  if (cell_zero >= 0) {
    CU(cudaEventRecord(c->ev_scan, c->stream));
    CU(cudaStreamWaitEvent(c->stream2, c->ev_scan, 0));
    {
      FamilyTimer ft(c, F_CELL, c->stream2);
      k_cell<<<c->cell_grid, 128, 0, c->stream2>>>(c->G, c->cell_cpb_shift, c->sums, c->rec, cell_zero);
      LAUNCH_CHECK("k_cell");
    }
    CU(cudaEventRecord(c->ev_cell, c->stream2));
  }
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
  } else {
    FamilyTimer ft(c, F_SCATTER);
    k_scatter_src<<<nblk(n, 256 * SCAT_U), 256, 0, c->stream>>>(n, c->key, c->offset, c->cursor, c->perm);
    LAUNCH_CHECK("k_scatter_src");
  }
  c->have_order = true;
  c->order_canonical = canonical;
  int rc = MPC_OK;
  if (defer_gather) c->gather_pending = true;
  else rc = apply_perm(c, c->G.generic != 0);     // the unfused path reads the sorted keys afterwards
  if (cell_zero >= 0) CU(cudaStreamWaitEvent(c->stream, c->ev_cell, 0));
  return rc;
}

// restore the canonical (key, id) order inside the cell segments of the last reorder (U4); called
// before the state is read when the hot path has left the particles grouped by key only
int canonicalise(mpc_ctx* c) {
  if (!c->have_order || c->order_canonical || c->n == 0) return MPC_OK;
  {
    FamilyTimer ft(c, F_RANK);
    k_rank_cells<<<nblk(c->G.nkeys, 256), 256, 0, c->stream>>>(c->G.nkeys, c->offset, c->A[6], c->perm);
    LAUNCH_CHECK("k_rank_cells");
  }
  const int rc = apply_perm(c, false);
  if (rc == MPC_OK) c->order_canonical = true;
  return rc;
}

typedef BrickShape<-1, -1, -1> BSgeneric;
typedef BrickShape<4, 4, 3> BSfast;   // {16,16,8}

// staging buffer of the folded reorder (32 bytes per particle): the unused SoA copy plus the slot array, which
// the workspace layout places between the two copies so that either copy extends to 8 arrays
inline float* aos_base(const mpc_ctx* c) {
  return reinterpret_cast<float*>(c->A[0] < c->Bf[0] ? c->slot_id : c->Bf[0]);
}
template <bool COLLIDE, bool WKEY, class BS, int IO>
int launch_sweep_bs(mpc_ctx* c, const float sp[3]) {
  const Geo& G = c->G;
  float** F = reinterpret_cast<float**>(c->A);
  SweepIO io;
  io.aos_in = io.aos_out = aos_base(c);
  io.perm = c->perm; io.id = c->A[6];
  const uint32_t* chunk = c->have_order ? c->offset : nullptr;
  const bool wall = G.wall >= 0, grav = (G.g[0] != 0.f || G.g[1] != 0.f || G.g[2] != 0.f);
#define SWEEP_ARGS G, sp[0], sp[1], sp[2], (uint32_t)c->n, F[0], F[1], F[2], F[3], F[4], F[5], c->key, chunk, c->nbricks, c->rec, c->sums
  if (IO == IO_PLAIN && !WKEY && c->three_ctas) {   // steady-state sweep: 3 CTAs of 384 threads per SM
    if (wall && grav) k_sweep<COLLIDE, true, true, false, BS, IO_PLAIN, SWEEP_T3><<<c->nbricks, SWEEP_T3, c->tile_bytes, c->stream>>>(SWEEP_ARGS, io);
    else if (wall) k_sweep<COLLIDE, true, false, false, BS, IO_PLAIN, SWEEP_T3><<<c->nbricks, SWEEP_T3, c->tile_bytes, c->stream>>>(SWEEP_ARGS, io);
    else if (grav) k_sweep<COLLIDE, false, true, false, BS, IO_PLAIN, SWEEP_T3><<<c->nbricks, SWEEP_T3, c->tile_bytes, c->stream>>>(SWEEP_ARGS, io);
    else k_sweep<COLLIDE, false, false, false, BS, IO_PLAIN, SWEEP_T3><<<c->nbricks, SWEEP_T3, c->tile_bytes, c->stream>>>(SWEEP_ARGS, io);
  } else
  if (wall && grav) k_sweep<COLLIDE, true, true, WKEY, BS, IO><<<c->nbricks, SWEEP_T, c->tile_bytes, c->stream>>>(SWEEP_ARGS, io);
  else if (wall) k_sweep<COLLIDE, true, false, WKEY, BS, IO><<<c->nbricks, SWEEP_T, c->tile_bytes, c->stream>>>(SWEEP_ARGS, io);
  else if (grav) k_sweep<COLLIDE, false, true, WKEY, BS, IO><<<c->nbricks, SWEEP_T, c->tile_bytes, c->stream>>>(SWEEP_ARGS, io);
  else k_sweep<COLLIDE, false, false, WKEY, BS, IO><<<c->nbricks, SWEEP_T, c->tile_bytes, c->stream>>>(SWEEP_ARGS, io);
#undef SWEEP_ARGS
  LAUNCH_CHECK("k_sweep");
  if (IO == IO_GATHER) c->gather_pending = false;
  return MPC_OK;
}
template <bool COLLIDE, bool WKEY, int IO = IO_PLAIN>
int launch_sweep(mpc_ctx* c, const float sp[3]) {
  return c->fast_brick ? launch_sweep_bs<COLLIDE, WKEY, BSfast, IO>(c, sp) : launch_sweep_bs<COLLIDE, WKEY, BSgeneric, IO>(c, sp);
}

template <bool COLLIDE, bool WKEY, class BS>
cudaError_t sweep_attr_bs(size_t bytes) {
  cudaError_t e;
  if ((e = cudaFuncSetAttribute(k_sweep<COLLIDE, true, true, WKEY, BS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes))) return e;
  if ((e = cudaFuncSetAttribute(k_sweep<COLLIDE, true, false, WKEY, BS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes))) return e;
  if ((e = cudaFuncSetAttribute(k_sweep<COLLIDE, false, true, WKEY, BS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes))) return e;
  if ((e = cudaFuncSetAttribute(k_sweep<COLLIDE, false, false, WKEY, BS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes))) return e;
  if (!WKEY) {
    if ((e = cudaFuncSetAttribute(k_sweep<COLLIDE, true, true, false, BS, IO_PLAIN, SWEEP_T3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes))) return e;
    if ((e = cudaFuncSetAttribute(k_sweep<COLLIDE, true, false, false, BS, IO_PLAIN, SWEEP_T3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes))) return e;
    if ((e = cudaFuncSetAttribute(k_sweep<COLLIDE, false, true, false, BS, IO_PLAIN, SWEEP_T3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes))) return e;
    if ((e = cudaFuncSetAttribute(k_sweep<COLLIDE, false, false, false, BS, IO_PLAIN, SWEEP_T3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes))) return e;
  }
  constexpr int IOX = WKEY ? IO_AOS_OUT : (COLLIDE ? IO_GATHER : IO_PLAIN);   // the staged variant that exists for these flags
  if ((e = cudaFuncSetAttribute(k_sweep<COLLIDE, true, true, WKEY, BS, IOX>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes))) return e;
  if ((e = cudaFuncSetAttribute(k_sweep<COLLIDE, true, false, WKEY, BS, IOX>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes))) return e;
  if ((e = cudaFuncSetAttribute(k_sweep<COLLIDE, false, true, WKEY, BS, IOX>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes))) return e;
  if ((e = cudaFuncSetAttribute(k_sweep<COLLIDE, false, false, WKEY, BS, IOX>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes))) return e;
  return cudaSuccess;
}
template <bool COLLIDE, bool WKEY>
cudaError_t sweep_attr(size_t bytes) {
  cudaError_t e = sweep_attr_bs<COLLIDE, WKEY, BSgeneric>(bytes);
  return e ? e : sweep_attr_bs<COLLIDE, WKEY, BSfast>(bytes);
}

// SRD: n steps = sweep(no collide), cell, [sweep(collide t-1 + move t), cell] x (n-1), trailing collide
int steps_srd(mpc_ctx* c, int nsteps) {
  Geo& G = c->G;
  const size_t n = c->n;
  float sp[3] = {0.f, 0.f, 0.f};
  for (int k = 0; k < nsteps; ++k) {
    G.t = c->t;
    host_shift(c, c->t, G.s);
    const bool rebin = (c->t % (uint32_t)c->p.rebin_every) == 0u;
    if (!c->sums_clean) { FamilyTimer ft(c, F_MEMSET); CU(cudaMemsetAsync(c->sums, 0, (size_t)G.nkeys * G.sw * 8, c->stream)); }
    c->sums_clean = false;
    // reorder folded into this sweep (writes the 32-byte staging records) and the next one (reads them through
    // the permutation): needs a next step in this call, the second particle copy, and rebin_every >= 2
    const bool stage = rebin && !c->compact && !c->no_fuse_gather && !c->eager_canonical && k + 1 < nsteps && c->p.rebin_every >= 2;
    if (n) {
      {
        FamilyTimer ft(c, (c->gather_pending || stage) ? F_SWEEPG : F_SWEEP);
        int rc;
        if (c->gather_pending) rc = launch_sweep<true, false, IO_GATHER>(c, sp);      // stage implies rebin_every >= 2
        else if (stage) rc = (k == 0) ? launch_sweep<false, true, IO_AOS_OUT>(c, sp) : launch_sweep<true, true, IO_AOS_OUT>(c, sp);
        else if (k == 0) rc = rebin ? launch_sweep<false, true>(c, sp) : launch_sweep<false, false>(c, sp);
        else rc = rebin ? launch_sweep<true, true>(c, sp) : launch_sweep<true, false>(c, sp);
        if (rc) return rc;
      }
      // all but the last step of the call: k_cell clears the sums it has read (the last step's stay for
      // mpc_observables / mpc_get_cells)
      const int zero = (k + 1 < nsteps) ? 1 : 0;
      const bool overlap = rebin && c->side_ready && !c->no_overlap;
      // the gather of a reorder is folded into the next step's sweep when there is one in this call;
      // PROCESS_CELLS of a reorder step runs on the side stream beside the scatter (both wait for the scan)
      if (rebin) {
        const int rc = do_reorder(c, stage, c->eager_canonical, overlap ? zero : -1);
        if (rc) return rc;
      }
      if (!overlap) {
        FamilyTimer ft(c, F_CELL);
        k_cell<<<c->cell_grid, 128, 0, c->stream>>>(G, c->cell_cpb_shift, c->sums, c->rec, zero);
        LAUNCH_CHECK("k_cell");
      }
      c->sums_clean = zero != 0;
    }
    sp[0] = G.s[0]; sp[1] = G.s[1]; sp[2] = G.s[2];
    c->t++;
    c->have_cells = true;
  }
  if (nsteps > 0 && n) {
    float** F = reinterpret_cast<float**>(c->A);
    FamilyTimer ft(c, F_COLLIDE);
    k_collide_pos<<<nblk(n, 256), 256, 0, c->stream>>>(G, n, F[0], F[1], F[2], F[3], F[4], F[5], c->rec);
    LAUNCH_CHECK("k_collide_pos");
  }
  return MPC_OK;
}

// MPC-AT and every +a variant: stream+key, reorder when due, per-cell sums with global atomics, cell
// finalize, collide. MPC-AT needs the sorted segments (rank of a particle in its cell), so it reorders
// every step (rebin_every == 1 is enforced at create).
int steps_generic(mpc_ctx* c, int nsteps) {
  Geo& G = c->G;
  const size_t n = c->n;
  const bool at = G.collision == 1, plus_a = G.conserve_L != 0;
  for (int k = 0; k < nsteps; ++k) {
    G.t = c->t;
    host_shift(c, c->t, G.s);
    const bool rebin = (c->t % (uint32_t)c->p.rebin_every) == 0u;
    {
      FamilyTimer ft(c, F_MEMSET);
      CU(cudaMemsetAsync(c->sums, 0, (size_t)G.nkeys * G.sw * 8, c->stream));
      CU(cudaMemsetAsync(c->nsing, 0, 8, c->stream));
    }
    if (n) {
      float** F = reinterpret_cast<float**>(c->A);
      const unsigned gb = nblk(n, 256);
      const bool grav = (G.g[0] != 0.f || G.g[1] != 0.f || G.g[2] != 0.f);
      {
        FamilyTimer ft(c, F_STREAM);
        if (grav) k_stream_key<false, true><<<gb, 256, 0, c->stream>>>(G, n, F[0], F[1], F[2], F[3], F[4], F[5], c->key, c->sums);
        else k_stream_key<false, false><<<gb, 256, 0, c->stream>>>(G, n, F[0], F[1], F[2], F[3], F[4], F[5], c->key, c->sums);
        LAUNCH_CHECK("k_stream_key");
      }
      if (rebin) { const int rc = do_reorder(c, false, true); if (rc) return rc; }
      F = reinterpret_cast<float**>(c->A);
      {
        FamilyTimer ft(c, F_ACCUM);
        if (rebin) {   // fresh (key, id) order: per-cell segmented sums, no atomics
          if (plus_a && at) k_accum_seg<true, true><<<c->cell_grid, 128, 0, c->stream>>>(G, c->cell_cpb_shift, F[0], F[1], F[2], F[3], F[4], F[5], c->offset, c->sums);
          else if (plus_a) k_accum_seg<false, true><<<c->cell_grid, 128, 0, c->stream>>>(G, c->cell_cpb_shift, F[0], F[1], F[2], F[3], F[4], F[5], c->offset, c->sums);
          else k_accum_seg<true, false><<<c->cell_grid, 128, 0, c->stream>>>(G, c->cell_cpb_shift, F[0], F[1], F[2], F[3], F[4], F[5], c->offset, c->sums);
        } else
        if (plus_a && at) k_accum_a<true><<<gb, 256, 0, c->stream>>>(G, n, F[0], F[1], F[2], F[3], F[4], F[5], c->key, c->offset, c->sums);
        else if (plus_a) k_accum_a<false><<<gb, 256, 0, c->stream>>>(G, n, F[0], F[1], F[2], F[3], F[4], F[5], c->key, c->offset, c->sums);
        else k_accum_at<<<gb, 256, 0, c->stream>>>(G, n, F[3], F[4], F[5], c->key, c->offset, c->sums);
        LAUNCH_CHECK("k_accum");
      }
      {
        FamilyTimer ft(c, F_CELL);
        if (plus_a && at) k_cell_a<true><<<c->cell_grid, 128, 0, c->stream>>>(G, c->cell_cpb_shift, c->sums, c->rec, c->nsing);
        else if (plus_a) k_cell_a<false><<<c->cell_grid, 128, 0, c->stream>>>(G, c->cell_cpb_shift, c->sums, c->rec, c->nsing);
        else k_cell<<<c->cell_grid, 128, 0, c->stream>>>(G, c->cell_cpb_shift, c->sums, c->rec, 0);
        LAUNCH_CHECK("k_cell");
      }
      FamilyTimer ft(c, F_COLLIDE);
      if (plus_a && at) k_collide_a<true><<<gb, 256, 0, c->stream>>>(G, n, F[0], F[1], F[2], F[3], F[4], F[5], c->key, c->offset, c->rec);
      else if (plus_a) k_collide_a<false><<<gb, 256, 0, c->stream>>>(G, n, F[0], F[1], F[2], F[3], F[4], F[5], c->key, c->offset, c->rec);
      else k_collide_at<<<gb, 256, 0, c->stream>>>(G, n, F[3], F[4], F[5], c->key, c->offset, c->rec);
      LAUNCH_CHECK("k_collide");
    }
    c->t++;
    c->have_cells = true;
  }
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
  c->n = n; c->t = step; c->have_state = true; c->have_cells = false; c->have_order = false; c->gather_pending = false; c->order_canonical = true;
  return MPC_OK;
}
int get_state_impl(mpc_ctx* c, float* const dst[6], unsigned* id, cudaMemcpyKind kind) {
  if (!c) return MPC_EINVAL;
  if (c->sticky) return MPC_ECUDA;
  if (!c->have_state) return fail(c, MPC_ESTATE, "mpc_get_state before mpc_set_state");
  { const int rc = canonicalise(c); if (rc) return rc; }
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
  // >= 3 cells per axis: with fewer, a particle shares a collision cell with its own periodic image
  for (int d = 0; d < 3; ++d) if (cells[d] < 3 || !(box[d] > 0.0f)) return MPC_EINVAL;
  const float a = box[0] / (float)cells[0];
  for (int d = 1; d < 3; ++d) if (box[d] / (float)cells[d] != a) return MPC_EINVAL;
  if (p->collision < 0 || p->collision > 1) return MPC_EINVAL;
  if (!(p->dt > 0.0f) || !(p->kT > 0.0f) || !(p->mass > 0.0f) || p->rebin_every < 1 || !(n_per_cell > 0.0f)) return MPC_EINVAL;
  size_t tile_cells = 1;
  for (int d = 0; d < 3; ++d) {
    const int b = p->brick[d];
    if (b < 1 || (b & (b - 1)) != 0 || b > 64) return MPC_EINVAL;   // powers of two
    tile_cells *= (size_t)(b + 2 * HALO);
  }
  if (tile_cells * TILE_W * 4 > MAX_TILE_BYTES) return MPC_EINVAL;
  int nwall = 0, wall = -1;
  for (int d = 0; d < 3; ++d) {
    if (p->bc[d] < 0 || p->bc[d] > 2) return MPC_EINVAL;
    if (p->bc[d] != 0) { nwall++; wall = d; if (p->g[d] != 0.0f) return MPC_EINVAL; }
  }
  if (nwall > 1) return MPC_EINVAL;
  if (nwall && (p->conserve_L || p->collision == 1)) return MPC_EINVAL;
  if (p->collision == 0 && p->conserve_L && p->thermostat) return MPC_EINVAL;
  if (p->collision == 1 && p->rebin_every != 1) return MPC_EINVAL;
  mpc_ctx* c = new (std::nothrow) mpc_ctx();   // value-initialised: all zero
  if (!c) return MPC_ENOMEM;
  c->p = *p; c->seed = seed;
  c->hbuf = new (std::nothrow) double[OBS_HOST_DOUBLES];
  if (!c->hbuf) { delete c; return MPC_ENOMEM; }
  Geo& G = c->G;
  G.a = a; G.inv_a = 1.0f / a; G.wall = wall; G.slip = (wall >= 0 && p->bc[wall] == 2) ? 1 : 0;
  unsigned long long nk = 1, nbr = 1;
  for (int d = 0; d < 3; ++d) {
    int bs = 0;
    while ((1 << bs) < p->brick[d]) ++bs;
    G.bs[d] = bs;
    G.L[d] = box[d]; G.n[d] = cells[d]; G.bc[d] = p->bc[d]; G.g[d] = p->g[d];
    G.m[d] = cells[d] + (p->bc[d] != 0 ? 2 : 0);
    G.mb[d] = (G.m[d] + p->brick[d] - 1) >> bs;
    nk *= (unsigned long long)G.mb[d] << bs;
    nbr *= (unsigned long long)G.mb[d];
  }
  if (nk >= 0xffffffffull) { delete[] c->hbuf; delete c; return MPC_EINVAL; }
  G.nkeys = (uint32_t)nk;
  c->nbricks = (uint32_t)nbr;
  c->tile_bytes = tile_cells * TILE_W * 4;
  c->three_ctas = 3 * (c->tile_bytes + 1024) <= 227 * 1024 && !getenv("MPC_SWEEP_2CTA");
  c->fast_brick = (G.bs[0] == 4 && G.bs[1] == 4 && G.bs[2] == 3);
  { const char* e = getenv("MPC_NO_FUSE_GATHER"); c->no_fuse_gather = (e && e[0] == '1'); }
  { const char* e = getenv("MPC_EAGER_CANONICAL"); c->eager_canonical = (e && e[0] == '1'); }
  // measured: no gain (k_cell beside the scatter slows the scatter down by as much), so off unless asked for
  { const char* e = getenv("MPC_OVERLAP_CELL"); c->no_overlap = !(e && e[0] == '1'); }
  c->side_ready = false;
  {
    const int bvs = G.bs[0] + G.bs[1] + G.bs[2];
    c->cell_cpb_shift = bvs > 7 ? bvs - 7 : 0;
    c->cell_grid = dim3((unsigned)G.mb[0] << c->cell_cpb_shift, (unsigned)G.mb[1], (unsigned)G.mb[2]);
    if (G.mb[1] > 65535 || G.mb[2] > 65535) { delete[] c->hbuf; delete c; return MPC_EINVAL; }
  }
  G.dt = p->dt; G.kT = p->kT; G.mass = p->mass;
  G.sigma = (float)sqrt((double)p->kT / (double)p->mass);
  G.cosa = (float)cos((double)p->alpha); G.sina = (float)sin((double)p->alpha);
  G.k0 = (uint32_t)(seed & 0xffffffffull); G.k1 = (uint32_t)(seed >> 32);
  philox_round_keys(G.k0, G.k1, G.rk);
  G.nbar = (int)lround((double)n_per_cell);
  const int ue = (int)lround(log2((double)G.sigma));        // thermal velocity rounded to a power of two
  G.fxv = (float)ldexp(1.0, 22 - ue); G.fxv_inv = ldexp(1.0, ue - 22);
  G.fxe = (float)ldexp(1.0, 22 - 2 * ue); G.fxe_inv = ldexp(1.0, 2 * ue - 22);
  G.collision = p->collision; G.thermostat = p->thermostat; G.conserve_L = p->conserve_L;
  G.generic = (p->collision == 1 || p->conserve_L) ? 1 : 0;
  G.sw = p->conserve_L ? 10 : (p->collision == 1 ? 4 : 3);
  G.rw = p->conserve_L ? 16 : REC_W;
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
  *bytes = make_layout((size_t)n_max, c->G.nkeys, c->G.sw, c->G.rw, compact != 0).total;
  return MPC_OK;
}

int mpc_bind(mpc_ctx* c, void* workspace, size_t bytes, unsigned long long n_max, void* cuda_stream) {
  if (!c) return MPC_EINVAL;
  if (!workspace || ((uintptr_t)workspace & 255u) || n_max > 0xffffffffull) return fail(c, MPC_EINVAL, "workspace NULL, misaligned or n_max too large");
  Layout l = make_layout((size_t)n_max, c->G.nkeys, c->G.sw, c->G.rw, false);
  bool compact = false;
  if (bytes < l.total) { l = make_layout((size_t)n_max, c->G.nkeys, c->G.sw, c->G.rw, true); compact = true; }
  if (bytes < l.total) return fail(c, MPC_ENOMEM, "workspace smaller than mpc_workspace_bytes(n_max, compact=1)");
  c->ws = (char*)workspace; c->ws_bytes = bytes; c->n_max = (size_t)n_max; c->compact = compact;
  c->stream = (cudaStream_t)cuda_stream;
  for (int a = 0; a < 7; ++a) { c->A[a] = (uint32_t*)(c->ws + l.off_A[a]); c->Bf[a] = (uint32_t*)(c->ws + l.off_B[a]); }
  c->key = (uint32_t*)(c->ws + l.off_key);
  c->slot_id = (uint32_t*)(c->ws + l.off_slot); c->perm = (uint32_t*)(c->ws + l.off_perm);
  c->cursor = (uint32_t*)(c->ws + l.off_cursor); c->offset = (uint32_t*)(c->ws + l.off_offset);
  c->bsum = (uint32_t*)(c->ws + l.off_bsum);
  c->sums = (u64*)(c->ws + l.off_sums); c->rec = (float*)(c->ws + l.off_rec); c->obs = (double*)(c->ws + l.off_obs);
  c->nsing = (u64*)(c->ws + l.off_obs + OBS_HOST_DOUBLES * 8);
  if (!c->side_ready) {
    CU(cudaStreamCreateWithFlags(&c->stream2, cudaStreamNonBlocking));
    CU(cudaEventCreateWithFlags(&c->ev_scan, cudaEventDisableTiming));
    CU(cudaEventCreateWithFlags(&c->ev_cell, cudaEventDisableTiming));
    c->side_ready = true;
  }
  c->bound = true; c->have_state = false; c->have_cells = false; c->have_order = false; c->sums_clean = false; c->gather_pending = false; c->n = 0;
  if (c->tile_bytes > 48 * 1024) {
    cudaError_t e;
    if ((e = sweep_attr<false, false>(c->tile_bytes)) || (e = sweep_attr<false, true>(c->tile_bytes)) ||
        (e = sweep_attr<true, false>(c->tile_bytes)) || (e = sweep_attr<true, true>(c->tile_bytes)))
      return cuda_fail(c, e, "cudaFuncSetAttribute(k_sweep, MaxDynamicSharedMemorySize)");
  }
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
  return c->G.generic ? steps_generic(c, nsteps) : steps_srd(c, nsteps);
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
  for (int d = 0; d < 3; ++d) if (G.bc[d] != 0) pa = d;
  for (int d = 2; d >= 0; --d) if (G.g[d] != 0.0f) fa = d;
  const int nb = G.n[pa];
  if (profile_host && nb > MAX_PROFILE) return fail(c, MPC_EINVAL, "profile axis longer than 2048 layers");
  {
    FamilyTimer ft(c, F_OBS);
    CU(cudaMemsetAsync(c->obs, 0, OBS_HOST_DOUBLES * 8, c->stream));
    if (n) {
      k_obs_particles<<<OBS_BLOCKS, 256, 0, c->stream>>>(n, F[3], F[4], F[5], part);
      LAUNCH_CHECK("k_obs_particles");
      if (profile_host) {
        k_obs_profile<<<OBS_BLOCKS, 256, (size_t)2 * nb * 8, c->stream>>>(G, n, nb, F[pa], F[3 + fa], prof);
        LAUNCH_CHECK("k_obs_profile");
      }
    }
    if (c->have_cells) {   // MPC-AT keeps no energy sum: kT_cell is reported as 0 there
      k_obs_cells<<<OBS_BLOCKS, 256, 0, c->stream>>>(G, c->sums, part);
      LAUNCH_CHECK("k_obs_cells");
    }
  }
  double* hbuf = c->hbuf;
  unsigned long long nsing = 0;
  CU(cudaMemcpyAsync(hbuf, c->obs, OBS_HOST_DOUBLES * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  if (c->have_cells && G.conserve_L) CU(cudaMemcpyAsync(&nsing, c->nsing, 8, cudaMemcpyDeviceToHost, c->stream));
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
  out->kT_cell = (!G.generic && den > 0) ? num / den : 0.0;
  out->max_cell_count = (unsigned)mx;
  out->n_singular_cells = nsing;
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
  const Geo& G = c->G;   // G.s / G.t are still those of the last step
  k_export_cells<<<nblk(G.nkeys, 256), 256, 0, c->stream>>>(G, c->sums, count, px, py, pz, e2);
  LAUNCH_CHECK("k_export_cells");
  if (key && c->n) {
    float** F = reinterpret_cast<float**>(c->A);
    k_keys<<<nblk(c->n, 256), 256, 0, c->stream>>>(G, c->n, F[0], F[1], F[2], key);
    LAUNCH_CHECK("k_keys");
  }
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
    if (c->side_ready) { cudaStreamDestroy(c->stream2); cudaEventDestroy(c->ev_scan); cudaEventDestroy(c->ev_cell); }
    if (c->prof_ev) for (int i = 0; i < 2 * PROF_MAX_PAIRS; ++i) cudaEventDestroy(c->prof_ev[i]);
    delete[] c->prof_ev;
    delete[] c->prof_fam;
  }
  delete c;
  return MPC_OK;
}

}  // extern "C"
