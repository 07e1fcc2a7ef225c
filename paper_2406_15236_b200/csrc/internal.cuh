// internal.cuh -- shared by the translation units of libmpc_b200.so (not installed, not part of the C ABI).
//
// Kernel families, one .cu file each:
//   sweep.cu    k_sweep: SRD hot path, ONE pass over the particles per step: collision of step t-1 (Eqs. 2,5) fused
//               with MOVE of step t (Eq. 1), shift + cell key, per-cell sums of step t in a shared-memory tile per
//               brick of cells; k_collide_pos: the collision still pending when the
//               state is read
//   cell.cu     k_cell: PROCESS_CELLS: v_cm, axis, kappa, virtual wall particles
//   reorder.cu  counting-sort reorder (scan, scatter, rank, gather), folded into two sweeps
//   generic.cu  MPC-AT and every +a variant (stream+key, per-cell segment pass or atomics, collide) Eqs. (3),(4), U5
//   observe.cu  observables and the cell-sum test hook
//   abi.cu      the C ABI of include/mpc_b200.h and the step scheduler
// Cell sums are 32-bit fixed point (the paper's reproducibility option), two per 64-bit word,
// added with integer atomics: order-independent, so a trajectory is bit-reproducible and does not depend on the
// memory order of the particles.
// Compile with --fmad=false: every multiply-add that must fuse is an explicit fmaf (U1).
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "../../include/mpc_b200.h"
#include "philox.cuh"

namespace mpc {

typedef unsigned long long u64;

// tile halo 1: 0.5 % of the particles (the ones that moved two cells since the reorder) take the global-atomic
// path; the 16x16x8 brick's tile is 18x18x10 cells = 65 KB, three of them fit in an SM's shared memory
constexpr int HALO = 1;               // tile halo in cells on every side of a brick
constexpr int SWEEP_T = 512;          // threads per sweep CTA (2 CTAs per SM): first-step and staged reorder sweeps
constexpr int SWEEP_T3 = 384;         // ... of the steady-state sweep when three tiles fit in an SM's shared memory (320: +5 %, 448: +10 %, 512 x 2: +4 %)
constexpr int PF_DIST = 4;            // L2 prefetch distance of the sweep, in iterations of T particles (3..6 equal, 8: +2.5 %)
constexpr int TILE_W = 5;             // int32 words per tile cell: N, Sx, Sy, Sz, E
constexpr int REC_W = 8;              // floats per cell record (32 B, one sector)
constexpr int OBS_BLOCKS = 1184;      // 148 SMs x 8
constexpr int MAX_PROFILE = 2048;
constexpr int SPREAD_GROUP_SHIFT = 5;  // lane-spread order: groups of 32 cells (spread_slot); 64: equal, 128: sweep +4 % (gathered cell records spread over more lines)
constexpr int MT_TABLE = 64;          // thermostat draw: table of (c, k)(N_c) for N_c < 64 (cell.cuh)
constexpr size_t OBS_HOST_DOUBLES = (size_t)OBS_BLOCKS * 8 + 2 * MAX_PROFILE;
constexpr size_t MAX_TILE_BYTES = 110 * 1024;
constexpr int SCAN_T = 256, SCAN_PER = 8, SCAN_TILE = SCAN_T * SCAN_PER;
// A particle whose |v|^2 reaches 64 u^2 (u = the power of two next to sqrt(kT/m), so |v| >= 8 u ~ 6..11 thermal
// velocities) is outside the range the fixed-point sums are sized for: counted in n_range_overflows.
constexpr unsigned E_RANGE_LIMIT = 1u << 28;   // in units of the energy quantum 2^-22 u^2
// Shared-memory tile of the sweep: word 0 of a cell = count (low 11 bits) | sum of (e >> 21) (high 21 bits), word 4 = sum
// of (e & (2^21 - 1)). With e < 2^28 neither field overflows below 2048 particles per (CTA, cell); a cell total of 2048
// or more is counted as a range overflow by k_cell.
constexpr int TILE_N_BITS = 11, TILE_E_SHIFT = 21;
constexpr unsigned TILE_N_MASK = (1u << TILE_N_BITS) - 1u;
constexpr unsigned MAX_CELL_COUNT = 1u << TILE_N_BITS;

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
  // 2^22/u^2, uint32 per tile (carries go to the global word) and 48 bits in the global word.
  float fxv, fxe;
  double fxv_inv, fxe_inv;
  float vmax;     // 8 u: velocity components at or beyond it are counted as range overflows
  int nbar;
  int collision, thermostat, conserve_L;
  int generic;    // 1 = unfused path (MPC-AT and every +a variant), 0 = fused SRD sweep
  int sw;         // 64-bit words per cell in the global sums array (3 SRD, 4 MPC-AT, 10 with +a)
  int rw;         // floats per cell record (8, or 16 with +a)
  uint32_t nkeys;
  u64* nrange;    // device counter of range overflows since the last mpc_set_state
  int shear;      // Lees-Edwards shear along z, flow along x (U21)
  float le_u;     // velocity of the image above: shear_rate * L_z
  float le_d;     // x displacement of the image above at the time the positions of this step refer to
  int phantoms;        // explicit phantom particles in wall-cut cells (U22)
  uint32_t solute_id0; // particles with id >= solute_id0 have mass solute_mass (if > 0; U23)
  float solute_mass;
  float wall_u;        // moving no-slip walls: +wall_u along x at L, -wall_u at 0 (U24)
  const float* mt_c;   // device table of MT_TABLE float pairs: (c, k)(N_c) of the thermostat draw (cell.cuh)
  // Slab subdomain of a multi-GPU run: this context holds the cell layers
  // [sub_z0 - bz, sub_z0 + sub_nz + bz) of a periodic box of nzg layers (bz = brick size along z: one brick layer of halo on
  // either side); m[2] = local layers. Local layer = global layer - zoff (mod nzg). Cell sums of the four brick layers it
  // shares with its two neighbours are ALSO added into the neighbours' arrays (integer REDs over peer memory), so that after
  // a barrier every rank holds the complete sums of all its local cells.
  int sub;              // 1 = slab subdomain
  int zoff, nzg;        // first local layer (may be negative), global number of layers along z
  int nbz;              // local brick layers along z
  u64* peer[2];         // cell sums of the neighbour below / above (device pointers, peer memory)
  long long peer_koff[2];   // key of a shared cell in that neighbour's array = local key + peer_koff
  uint32_t* lcount;     // particle counts of THIS rank only, for the cells of the shared brick layers (indexed by local key)
  // hand-over of particles riding on the folded reorder (sweep.cu, IO_SCATTER): the neighbours' new cell offsets and staging
  // buffers (peer memory), and for every cell of this rank's halo layers the neighbour's own count of the cell at the reorder
  // step (the first slot, inside the cell's segment of the neighbour's new order, of the particles this rank hands over)
  const uint32_t* peer_offset[2];
  float* peer_aos[2];
  uint32_t* abase;
};

// ---- packed sums ---------------------------------------------------------------------------------
// word0 = E << 16 | N (E: 48 bits, N: 16 bits, so at most 65535 particles per cell); word1 = (Sy, Sx); word2 = (R0, Sz); word3 = (R2, R1)  [AT: R = sum v_ran]
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
// slab subdomain: the id of the cell in the whole box (every rank draws the same numbers for it); iz = local layer
__device__ __forceinline__ uint32_t canonical_id_sub(const Geo& G, int ix, int iy, int iz) {
  iz += G.zoff;
  iz += (iz < 0) ? G.nzg : 0;
  iz -= (iz >= G.nzg) ? G.nzg : 0;
  return canonical_id(G, ix, iy, iz);
}
// cell coordinate of position r along axis d for lattice shift s
__device__ __forceinline__ int cell_coord(const Geo& G, int d, float r, float s) {
  const float q = (r + s) * G.inv_a;
  int k = (int)floorf(q);
  if (d == 2 && G.sub) {   // slab subdomain: local layer (clamped; the sweep counts particles outside the slab)
    int t = k - G.zoff;
    t += (t < 0) ? G.nzg : 0;
    t -= (t >= G.nzg) ? G.nzg : 0;
    t -= (t >= G.nzg) ? G.nzg : 0;
    return min(t, G.m[2] - 1);
  }
  if (G.bc[d] == 0) {
    if (k < 0) k += G.n[d];
    if (k >= G.n[d]) k -= G.n[d];
  } else {
    k += 1;
    k = max(0, min(k, G.n[d] + 1));
  }
  return k;
}
// Lees-Edwards (U21): a particle whose shifted z leaves [0, L_z) collides as its periodic image, x -+ D
// (wrapped once) and v_x -+ U. Returns the x to bin with; vs = what is added to v_x for the collision (and taken off
// again afterwards).
__device__ __forceinline__ float le_image(const Geo& G, float x, float z, float sz, float D, float& vs) {
  vs = 0.0f;
  const int kz = __float2int_rd((z + sz) * G.inv_a);
  float xe = x;
  if (kz < 0) { xe = x + D; if (xe >= G.L[0]) xe -= G.L[0]; vs = G.le_u; }
  else if (kz >= G.n[2]) { xe = x - D; if (xe < 0.0f) xe += G.L[0]; vs = -G.le_u; }
  return xe;
}
// memory key of a position for lattice shift s (and the Lees-Edwards displacement G.le_d of the same step)
__device__ __forceinline__ uint32_t key_of(const Geo& G, float x, float y, float z, float s0, float s1, float s2, float* vs_out = nullptr) {
  float vs = 0.0f;
  if (G.shear) x = le_image(G, x, z, s2, G.le_d, vs);
  if (vs_out) *vs_out = vs;
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
template <bool WALL, bool GRAV, bool SHEAR = false>
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
      } else {                                                // bounce-back, in the frame of a moving wall (U24): v -> 2 u_wall - v
        v[0] = -v[0]; v[1] = -v[1]; v[2] = -v[2];
        if (G.wall_u != 0.0f) v[0] = fmaf(2.0f, (z1 < 0.0f) ? -G.wall_u : G.wall_u, v[0]);
      }
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
    if (SHEAR && d == 2) {   // crossing z = 0 / L_z enters the sheared image (U21)
      if (r[2] < 0.0f) { r[2] += G.L[2]; r[0] += G.le_d; if (r[0] >= G.L[0]) r[0] -= G.L[0]; v[0] += G.le_u; }
      if (r[2] >= G.L[2]) { r[2] -= G.L[2]; r[0] -= G.le_d; if (r[0] < 0.0f) r[0] += G.L[0]; v[0] -= G.le_u; }
      continue;
    }
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

// SRD rotation axis of cell cid at step G.t: uniform on the sphere (U11)
__device__ __forceinline__ void srd_axis(const Geo& G, uint32_t cid, float& ax, float& ay, float& az) {
  const Block4 o = philox_rk(cid, 0u, G.t, TAG_AXIS, G.rk);
  az = 2.0f * u01_co(o.a) - 1.0f;
  const float rr = sqrtf((1.0f - az) * (1.0f + az));
  float sp, cp;
  sincospif(2.0f * u01_co(o.b), &sp, &cp);
  ax = rr * cp; ay = rr * sp;
}

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
typedef BrickShape<-1, -1, -1> BSgeneric;
typedef BrickShape<4, 4, 3> BSfast;   // {16,16,8}

// floor index of a coordinate, not yet folded into [0, m)
__device__ __forceinline__ int cell_raw(const Geo& G, float r, float s) { return __float2int_rd((r + s) * G.inv_a); }
// Lane-spread order inside a group of 32 cells (hot path). The sweep's shared-memory atomics serialise on
// lanes of a warp that hit the same cell; in plain cell order a warp's 32 consecutive particles sit in ~3 cells. The
// hot-path reorder therefore stores the n_g particles of every aligned group of 32 keys (one contiguous range [g0, g1)
// of the counting sort, always inside one brick) TRANSPOSED: with R = n_g / 32, sorted position p < 32 R goes to row
// p % R, column p / R of an R x 32 matrix, so neighbouring lanes hold particles R ~ <N_c> sorted positions apart:
// (mostly) different cells. The tail p >= 32 R stays where it is. The brick ranges the sweep works on are unchanged; the
// order inside a cell does not enter the physics (integer sums); canonicalise() reads the cells back through the same map.
__device__ __forceinline__ uint32_t spread_slot(uint32_t slot, uint32_t g0, uint32_t g1) {
  const uint32_t R = (g1 - g0) >> 5, p = slot - g0;
  if (p >= (R << 5)) return slot;
  const uint32_t col = p / R, row = p - col * R;
  return g0 + (row << 5) + col;
}
// fold an index known to lie in [-m, 2m) into [0, m)
__device__ __forceinline__ int fold(int k, int m) {
  k += (k < 0) ? m : 0;
  k -= (k >= m) ? m : 0;
  return k;
}

// ---- slab subdomain (Geo::sub) ---------------------------------------------------------------------
// local layer of the global (unfolded, in [-1, nzg]) layer index kz; -1 if the layer is not held by this rank
__device__ __forceinline__ int sub_layer(const Geo& G, int kz) {
  int t = kz - G.zoff;
  t += (t < 0) ? G.nzg : 0;
  t -= (t >= G.nzg) ? G.nzg : 0;
  t -= (t >= G.nzg) ? G.nzg : 0;
  return (t < G.m[2]) ? t : -1;
}
// which neighbour shares the cell of local layer iz (0 below, 1 above, -1 none)
__device__ __forceinline__ int sub_shared(const Geo& G, int iz) {
  const int bl = iz >> G.bs[2];
  return (bl <= 1) ? 0 : (bl >= G.nbz - 2) ? 1 : -1;
}

}  // namespace mpc

// =================================================================================================
// host side
// =================================================================================================
enum Family { F_SWEEP = 0, F_CELL, F_COLLIDE, F_SCAN, F_SCATTER, F_RANK, F_GATHER, F_MEMSET, F_STREAM, F_ACCUM, F_OBS, F_SWEEPG, F_COUNT };
constexpr int PROF_MAX_PAIRS = 16384;

struct mpc_ctx {
  mpc::Geo G;
  mpc_params p;
  unsigned long long seed;
  uint32_t t;
  size_t n, n_max;
  bool bound, have_state, have_cells, have_order, compact, sticky, fast_brick, sums_clean, order_canonical, three_ctas;
  // the collision of the last step of an mpc_step call stays pending: the next call's first sweep
  // applies it; every call that reads particle velocities applies it first (flush_collide)
  bool collide_pending;
  bool pow2_cells;      // no walls and every m[d] a power of two: the sweep folds indices with a mask
  int order_spread;     // log2 of the cells per group whose particles are stored lane-spread (spread_slot); 0 = plain cell order
  bool sub_open;        // slab subdomain: mpc_sub_begin has run, mpc_sub_end has not
  bool sub_stage;       // ... and it started a folded reorder with hand-over (decided in mpc_sub_begin, used by mpc_sub_end)
  int sub_ahead;        // ... steps the caller has promised to run after the open one before it reads or replaces the state
  uint32_t sub_nn;      // ... particle count of this rank once the folded reorder in flight has handed particles over
  int reorder_stage;    // folded reorder: 0 none in flight, 1 the next sweep scatters into the new order, 2 the next sweep reads the staged records
  float le_dprev;       // Lees-Edwards displacement of the step whose collision is pending
  unsigned debug;       // MPC_DEBUG_* flags
  int device;           // CUDA device of the workspace
  cudaStream_t stream;
  char* ws;
  size_t ws_bytes;
  uint32_t nbricks;
  size_t tile_bytes;
  dim3 cell_grid;       // k_cell launch: (mb0 << cell_cpb_shift, mb1, mb2) CTAs of 256 cells
  int cell_cpb_shift;
  dim3 seg_grid;        // per-cell kernels of the generic path: CTAs of 128 cells
  int seg_cpb_shift;
  // device arrays
  uint32_t* A[7];   // x y z vx vy vz id (current)
  uint32_t* Bf[7];  // second copy (non-compact); Bf[0] = 4-byte temp (compact)
  uint32_t *key, *slot_id, *perm, *cursor, *offset, *bsum;
  uint32_t *tbase, *chunk0;   // staged reorder: per (brick, tile cell) first slot; brick ranges of the previous order
  int gwin_shift;             // compact workspace: log2 of the keys per shared-memory window of k_gather_win (0: not used); chunk0 then
  uint32_t gwin_cap;          // ... holds the previous order's ranges of these groups; gwin_cap = elements per window
  mpc::u64* sums;
  float* rec;
  double* obs;      // OBS_BLOCKS*8 doubles + 2*MAX_PROFILE doubles
  mpc::u64* nsing;  // +a: number of rejected inertia tensors in the last step
  mpc::u64* nrange; // range overflows since the last mpc_set_state
  double* hbuf;     // host staging for mpc_observables
  float mt_host[2 * mpc::MT_TABLE];   // host copy of the thermostat table: (c, k) per N_c
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

inline int fail(mpc_ctx* c, int code, const char* msg) {
  if (c) snprintf(c->err, sizeof(c->err), "%s", msg);
  return code;
}
inline int cuda_fail(mpc_ctx* c, cudaError_t e, const char* where) {
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
// staging buffer of the reorder (32 bytes per particle): the unused SoA copy plus the slot array, which the workspace
// layout places between the two copies so that either copy extends to 8 arrays (non-compact workspace only)
inline float* aos_base(const mpc_ctx* c) {
  return reinterpret_cast<float*>(c->A[0] < c->Bf[0] ? c->slot_id : c->Bf[0]);
}

// ---- entry points of the translation units ---------------------------------------------------------
// sweep.cu
enum { IO_PLAIN = 0, IO_RANK = 1, IO_SCATTER = 2, IO_AOS_IN = 3 };   // sweep.cu: the reorder folded into three sweeps
int launch_sweep(mpc_ctx* c, bool collide, bool wkey, int io, const float sp[3]);
int launch_sub_clear(mpc_ctx* c);
cudaError_t sweep_set_attributes(size_t tile_bytes);
int launch_collide_pos(mpc_ctx* c);
int launch_keys(mpc_ctx* c, uint32_t* key_out);
// cell.cu
int launch_cell(mpc_ctx* c, int zero, uint32_t* counts, bool handover = false);   // counts != nullptr: also writes the per-cell particle counts (one word per key)
void fill_mt_table(float* host);
// reorder.cu
int do_reorder(mpc_ctx* c, bool folded, bool canonical, bool counts_in_cursor);
int canonicalise(mpc_ctx* c);
int launch_iota(mpc_ctx* c);
// generic.cu
int steps_generic(mpc_ctx* c, int nsteps);
// observe.cu
int observables_impl(mpc_ctx* c, mpc_obs* out, float* profile_host, int n_profile);
int sub_pack_impl(mpc_ctx* c, float* const out[6], unsigned* id_out, unsigned long long counts[3]);
int get_cells_impl(mpc_ctx* c, unsigned* count, float* px, float* py, float* pz, float* e2, unsigned* key);
// abi.cu
int flush_collide(mpc_ctx* c);
