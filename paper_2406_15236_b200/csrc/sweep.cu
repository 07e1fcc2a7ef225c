// sweep.cu -- the fused SRD sweep: ROTATE_VELOCITIES of step t-1 (Eqs. 2,5) + MOVE of step t (Eq. 1, PAPER.md:31;
// gravity PAPER.md:70; walls PAPER.md:68) + lattice shift and cell index + the per-cell sums of
// step t, in ONE pass over the particles.
#include "internal.cuh"

namespace mpc {

// Reorder folded into three consecutive sweeps, IO = 1, 2, 3 on the reorder step t and the two after it:
//   IO_RANK     step t: the pass works in place as always and also writes one word per particle: its arrival rank
//               inside (this CTA, its cell), which the tile's count atomic returns (or bit 31 | its slot in the cell's
//               segment, from the returning global atomic, for the few particles outside the tile); the tile flush
//               uses the returning form of the count atomic: what it returns is the first slot of this CTA's particles
//               inside the cell's segment (tbase). A scan of the counts follows (reorder.cu).
//   IO_SCATTER  step t+1: still in the old order (coalesced SoA reads); the cell of step t is recomputed for the
//               collision anyway, so slot = offset[cell] + tbase[CTA, cell] + rank is known, and the particle
//               (after collision and MOVE) is written as ONE 32-byte record {r, v, id, 0} at its slot of the new
//               order in the staging buffer (a whole sector per store);
//   IO_AOS_IN   step t+2: in the new order; records read back with coalesced 256-bit loads, SoA arrays written at i.
// No permutation array, no scatter kernel, no random reads: 32 bytes per particle more than three plain sweeps.
// (A gather of the SoA arrays themselves costs ~4.5 sectors of L2 traffic per useful one.)
struct SweepIO {
  float* aos;               // IO_SCATTER: written at the slot; IO_AOS_IN: read at i
  uint32_t* id;             // IO_SCATTER: read at i; IO_AOS_IN: written at i
  uint32_t* tbase;          // IO_RANK: written by the flush; IO_SCATTER: read: first slot of this CTA's particles inside every tile cell's segment
  const uint32_t* offset;   // IO_SCATTER: cell offsets of the new order
  int spread;               // IO_SCATTER: log2 of the cells per group of the lane-spread order (spread_slot), 0 = plain cell order
  int chunk_shift;          // chunk[b << chunk_shift] = first particle of brick b
  float le_dprev;           // Lees-Edwards displacement of the previous step (for its collision)
};
__device__ __forceinline__ void ld256(const float* p, float (&a)[8]) {
  asm volatile("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=f"(a[0]), "=f"(a[1]), "=f"(a[2]), "=f"(a[3]), "=f"(a[4]), "=f"(a[5]), "=f"(a[6]), "=f"(a[7]) : "l"(p));
}
__device__ __forceinline__ void st256(float* p, const float (&a)[8]) {
  asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
               :: "l"(p), "f"(a[0]), "f"(a[1]), "f"(a[2]), "f"(a[3]), "f"(a[4]), "f"(a[5]), "f"(a[6]), "f"(a[7]) : "memory");
}

// One CTA per brick of cells. Its particles are the contiguous range that was sorted into the brick at
// the last reorder (chunk[] = offset[] of the brick's first key); since then they have moved by a
// fraction of a cell and the lattice shift has changed by less than a cell, so nearly all of them fall
// into the brick's tile (brick + HALO cells on every side), held in shared memory as int32 sums. The
// rest (and everything, if no order is known yet) goes to the global sums directly.
// The CTA takes the 128-byte-aligned groups of 32 particles that START in its range: every group belongs to
// exactly one CTA and every access of a warp is line-aligned (L1 tag requests per load 1.9 -> 1.0).
__device__ __forceinline__ void chunk_range(const uint32_t* __restrict__ chunk, uint32_t b, uint32_t nbricks, uint32_t n,
                                            int bvol_shift, uint32_t& i0, uint32_t& i1) {
  if (chunk) {
    i0 = chunk[(size_t)b << bvol_shift];
    i1 = (b + 1 == nbricks) ? n : chunk[(size_t)(b + 1) << bvol_shift];
  } else {   // no order known: even split, (almost) everything takes the global path
    i0 = (uint32_t)((u64)n * b / nbricks);
    i1 = (uint32_t)((u64)n * (b + 1) / nbricks);
  }
  i0 = (i0 + 31u) & ~31u;
  if (b + 1 != nbricks) i1 = min((i1 + 31u) & ~31u, n);   // trailing empty bricks: chunk = n, do not round past the end
}

// T = threads per CTA: 512 (2 CTAs per SM), or 384 (3 CTAs per SM at <= 56 registers: the steady-state sweep is
// 2 % faster that way, the staged reorder sweeps are not)
// P2: the cell-layer counts m[] are powers of two (and there are no walls): folding an index into [0, m) is one AND
template <bool P2>
__device__ __forceinline__ int foldp(int k, int m) { return P2 ? (k & (m - 1)) : fold(k, m); }

// SHEAR: Lees-Edwards boundary along z (U21); the few particles that collide as their image are binned at
// x -+ D, usually far from their brick: they take the global path
// SUB: slab subdomain of a multi-GPU run (Geo::sub): the z axis holds local layers and does not wrap; the sums of the cells
// shared with a neighbour are also added into the neighbour's array (peer memory)
template <bool COLLIDE, bool WALL, bool GRAV, bool WKEY, class BS, int IO, int T, bool P2, bool SHEAR, bool SUB = false>
__global__ void __launch_bounds__(T, T <= 384 ? 3 : 2)
k_sweep(Geo G, float sp0, float sp1, float sp2, uint32_t n, float* __restrict__ x, float* __restrict__ y, float* __restrict__ z,
        float* __restrict__ vx, float* __restrict__ vy, float* __restrict__ vz, uint32_t* __restrict__ key_out,
        const uint32_t* __restrict__ chunk, uint32_t nbricks, const float* __restrict__ rec, u64* __restrict__ sums,
        SweepIO io) {
  static_assert(IO != IO_SCATTER || COLLIDE, "the scatter pass sorts by the cell of the collision it applies");
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
  chunk_range(chunk, b, nbricks, n, io.chunk_shift, i0, i1);
  constexpr bool ranked = IO == IO_RANK;
  // index offsets added before the floor index is folded: +1 on a wall axis (layer 0 lies in the wall)
  const int w0 = (WALL && G.bc[0]) ? 1 : 0, w1 = (WALL && G.bc[1]) ? 1 : 0, w2 = (WALL && G.bc[2]) ? 1 : 0;
  unsigned nbad = 0;
  __syncthreads();
  // software pipeline: the loads of the next particle are in flight while this one is processed
  uint32_t i = i0 + threadIdx.x;
  float p0 = 0.f, p1 = 0.f, p2 = 0.f, p3 = 0.f, p4 = 0.f, p5 = 0.f;
  // pid = id of the particle in flight (IO_SCATTER, IO_AOS_IN), pw = its rank word (IO_SCATTER)
  float pid = 0.f;
  uint32_t pw = 0;
  if (IO == IO_AOS_IN) {
    if (i < i1) {
      float q[8];
      ld256(io.aos + (size_t)i * 8, q);
      p0 = q[0]; p1 = q[1]; p2 = q[2]; p3 = q[3]; p4 = q[4]; p5 = q[5]; pid = q[6];
    }
  } else if (i < i1) {
    p0 = x[i]; p1 = y[i]; p2 = z[i]; p3 = vx[i]; p4 = vy[i]; p5 = vz[i];
    if (IO == IO_SCATTER) { pid = __uint_as_float(io.id[i]); pw = key_out[i]; }
  }
  for (; i < i1; i += T) {
    float r[3] = {p0, p1, p2}, v[3] = {p3, p4, p5};
    const float idbits = pid;
    const uint32_t w = pw;
    const uint32_t inext = i + T;
    if (IO == IO_AOS_IN) {
      io.id[i] = __float_as_uint(idbits);
      if (inext < i1) {
        float q[8];
        ld256(io.aos + (size_t)inext * 8, q);
        p0 = q[0]; p1 = q[1]; p2 = q[2]; p3 = q[3]; p4 = q[4]; p5 = q[5]; pid = q[6];
      }
    } else if (inext < i1) {
      p0 = x[inext]; p1 = y[inext]; p2 = z[inext]; p3 = vx[inext]; p4 = vy[inext]; p5 = vz[inext];
      if (IO == IO_SCATTER) { pid = __uint_as_float(io.id[inext]); pw = key_out[inext]; }
    }
    if (threadIdx.x == 0) {
      // pull the lines of a later iteration into L2: the register prefetch above then pays L2, not DRAM, latency. ONE bulk
      // prefetch per array and CTA iteration (cp.async.bulk.prefetch.L2): a per-thread prefetch.global.L2 costs every warp
      // six more requests in the L1TEX pipe that bounds this kernel (sweep 15.0 -> 14.3 ms at config 5; none at all: 16.6)
      const uint32_t ifar = i + PF_DIST * T;
      if (ifar < i1) {
        const uint32_t bytes = (min((uint32_t)T, i1 - ifar) * 4u) & ~15u;
        if (bytes) {
          if (IO == IO_AOS_IN) {
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(io.aos + (size_t)ifar * 8), "r"(bytes * 8u));
          } else {
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(x + ifar), "r"(bytes));
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(y + ifar), "r"(bytes));
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(z + ifar), "r"(bytes));
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(vx + ifar), "r"(bytes));
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(vy + ifar), "r"(bytes));
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(vz + ifar), "r"(bytes));
            if (IO == IO_SCATTER) {
              asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(io.id + ifar), "r"(bytes));
              asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(key_out + ifar), "r"(bytes));
            }
          }
        }
      }
    }
    uint32_t slot = 0;   // IO_SCATTER: the particle's place in the new order
    int leave_side = -1; // ... of the neighbour below / above, if the particle changes owner (slab subdomains)
    if (COLLIDE) {   // ROTATE_VELOCITIES of the previous step; its key is recomputed from r and that step's shift
      float vsp = 0.0f;
      const float xp = SHEAR ? le_image(G, r[0], r[2], sp2, io.le_dprev, vsp) : r[0];
      int kx = cell_raw(G, xp, sp0) + w0, ky = cell_raw(G, r[1], sp1) + w1, kz = cell_raw(G, r[2], sp2) + w2;
      if (WALL) { kx = G.bc[0] ? max(0, min(kx, m0 - 1)) : foldp<P2>(kx, m0); ky = G.bc[1] ? max(0, min(ky, m1 - 1)) : foldp<P2>(ky, m1);
                  kz = G.bc[2] ? max(0, min(kz, m2 - 1)) : foldp<P2>(kz, m2); }
      else { kx = foldp<P2>(kx, m0); ky = foldp<P2>(ky, m1); kz = SUB ? max(sub_layer(G, kz), 0) : foldp<P2>(kz, m2); }
      const uint32_t kp = BS::key(G, kx, ky, kz);
      float4 r0, ax;
      load_rec(rec, kp, r0, ax);
      if (IO == IO_SCATTER) {   // kp is the cell the reorder sorts by: slot = cell offset + first slot of this CTA + arrival rank
        slot = io.offset[kp];
        if (w & 0x80000000u) slot += w & 0xffffu;
        else {
          const int l0 = foldp<P2>(kx - ox, m0), l1 = foldp<P2>(ky - oy, m1), l2 = SUB ? kz - oz : foldp<P2>(kz - oz, m2);
          slot += io.tbase[(size_t)b * tcells + (l2 * T1 + l1) * T0 + l0] + w;
        }
        if (io.spread) { const uint32_t kg = kp & ~((1u << io.spread) - 1u); slot = spread_slot(slot, io.offset[kg], io.offset[kg + (1u << io.spread)]); }
        if (SUB) {
          // hand-over riding on the reorder: a particle whose cell of the reorder step lies in a halo layer now
          // belongs to the neighbour that owns the layer. Its record goes straight into that neighbour's staging buffer
          // (peer memory), behind the neighbour's own particles of the cell: the neighbour's scan has left room for it
          // (its count of the cell is the complete one), and abase = that neighbour's own count = complete - this rank's
          const int bl = kz >> BS::s2(G);
          const int side = (bl == 0) ? 0 : (bl == G.nbz - 1) ? 1 : -1;
          if (side >= 0) {
            const uint32_t* poff = G.peer_offset[side];
            const uint32_t pk = (uint32_t)((long long)kp + G.peer_koff[side]);
            uint32_t r_in_cell;
            if (w & 0x80000000u) r_in_cell = w & 0xffffu;
            else {
              const int l0 = foldp<P2>(kx - ox, m0), l1 = foldp<P2>(ky - oy, m1), l2 = kz - oz;
              r_in_cell = io.tbase[(size_t)b * tcells + (l2 * T1 + l1) * T0 + l0] + w;
            }
            uint32_t ps = poff[pk] + G.abase[kp] + r_in_cell;
            if (io.spread) { const uint32_t kg = pk & ~((1u << io.spread) - 1u); ps = spread_slot(ps, poff[kg], poff[kg + (1u << io.spread)]); }
            slot = ps;
            leave_side = side;
          }
        }
      }
      if (SHEAR) v[0] += vsp;
      srd_apply(G, r0, ax, v);
      if (SHEAR) v[0] -= vsp;
    }
    stream_one<WALL, GRAV, SHEAR>(G, r, v);
    if (IO == IO_SCATTER) {
      const float q[8] = {r[0], r[1], r[2], v[0], v[1], v[2], idbits, 0.f};
      st256(((SUB && leave_side >= 0) ? G.peer_aos[leave_side] : io.aos) + (size_t)slot * 8, q);
    } else {
      x[i] = r[0]; y[i] = r[1]; z[i] = r[2];
      vx[i] = v[0]; vy[i] = v[1]; vz[i] = v[2];
    }
    float vsn = 0.0f;
    const float xn = SHEAR ? le_image(G, r[0], r[2], G.s[2], G.le_d, vsn) : r[0];
    if (SHEAR) v[0] += vsn;        // the sums are taken in the frame of the image (v is not stored after this point)
    int cx = cell_raw(G, xn, G.s[0]) + w0, cy = cell_raw(G, r[1], G.s[1]) + w1, cz = cell_raw(G, r[2], G.s[2]) + w2;
    if (WALL) { if (G.bc[0]) cx = max(0, min(cx, m0 - 1)); if (G.bc[1]) cy = max(0, min(cy, m1 - 1)); if (G.bc[2]) cz = max(0, min(cz, m2 - 1)); }
    if (SUB) {   // local layer; a particle outside the layers this rank holds invalidates the run (counted)
      cz = sub_layer(G, cz);
      if (cz < 0) { cz = 0; nbad++; }
    }
    const int a0 = __float2int_rn(v[0] * G.fxv), a1 = __float2int_rn(v[1] * G.fxv), a2 = __float2int_rn(v[2] * G.fxv);
    const unsigned e = __float2uint_rn(fmaf(v[0], v[0], fmaf(v[1], v[1], v[2] * v[2])) * G.fxe);
    nbad += (e >= E_RANGE_LIMIT) ? 1u : 0u;     // |v| >= 8 u: outside the range of the fixed-point sums
    // tile coordinates: one fold takes care of the periodic image of the cell and of the tile origin
    const int l0 = foldp<P2>(cx - ox, m0), l1 = foldp<P2>(cy - oy, m1), l2 = SUB ? cz - oz : foldp<P2>(cz - oz, m2);
    const bool inside = (l0 < T0) & (l1 < T1) & ((unsigned)l2 < (unsigned)T2);
    uint32_t word = 0;   // IO_RANK: rank word of the particle
    if (inside) {
      const int tc = (l2 * T1 + l1) * T0 + l0;
      int* s = tile + tc * TILE_W;
      // word 0 = count (11 bits) | sum of the energies' high parts e >> 21 (21 bits); word 4 = sum of their low 21 bits:
      // neither can overflow below 2048 particles per (CTA, cell) with e < 2^28 (U19)
      const int w0add = 1 + (int)((e >> TILE_E_SHIFT) << TILE_N_BITS);
      if (ranked) word = (uint32_t)atomicAdd(s, w0add) & TILE_N_MASK;   // arrival rank inside (CTA, cell)
      else atomicAdd(s, w0add);
      atomicAdd(s + 1, a0); atomicAdd(s + 2, a1); atomicAdd(s + 3, a2);
      atomicAdd((unsigned*)s + 4, e & ((1u << TILE_E_SHIFT) - 1u));
    }
    if (WKEY || !inside) {
      const uint32_t kc = BS::key(G, foldp<P2>(cx, m0), foldp<P2>(cy, m1), SUB ? cz : foldp<P2>(cz, m2));
      if (!inside) {
        u64* s = sums + (size_t)kc * G.sw;
        const int side = SUB ? sub_shared(G, cz) : -1;
        // (a shared cell's count word also receives the neighbour's particles: this rank's own count, which numbers
        // its particles inside the cell, is kept apart)
        if (SUB && side >= 0) {
          // a shared cell's words are added to by two GPUs at once (this rank here, the neighbour through its peer
          // mapping): both sides use system-scope reductions, the only scope at which atomicity across GPUs is defined
          atomicAdd_system(s, ((u64)e << 16) | 1ull); atomicAdd_system(s + 1, pack_ss(a0, a1)); atomicAdd_system(s + 2, pack_ss(a2, 0));
          u64* q = G.peer[side] + (size_t)((long long)kc + G.peer_koff[side]) * G.sw;
          atomicAdd_system(q, ((u64)e << 16) | 1ull); atomicAdd_system(q + 1, pack_ss(a0, a1)); atomicAdd_system(q + 2, pack_ss(a2, 0));
          if (ranked) word = 0x80000000u | (atomicAdd(G.lcount + kc, 1u) & 0xffffu);
          else atomicAdd(G.lcount + kc, 1u);
        } else {
          if (ranked) word = 0x80000000u | (uint32_t)(atomicAdd(s, ((u64)e << 16) | 1ull) & 0xffffull);
          else atomicAdd(s, ((u64)e << 16) | 1ull);
          atomicAdd(s + 1, pack_ss(a0, a1)); atomicAdd(s + 2, pack_ss(a2, 0));
        }
      }
      if (WKEY) key_out[i] = kc;
    }
    if (ranked) key_out[i] = word;
  }
  if (nbad) atomicAdd(G.nrange, (u64)nbad);
  __syncthreads();
  // flush the tile: one packed 64-bit reduction per pair of sums, empty cells skipped. The staging sweep of a ranked
  // reorder needs what the count atomic returns (the slots taken so far in the cell = the first slot of this CTA's
  // particles): FLUSH_U atomics are in flight per thread before the first return is used (one at a time cost 1.9 ms
  // per launch at config 5: the loop is in-order, every use waits a full L2 round trip)
  constexpr int FLUSH_U = 4;
  for (int c0 = threadIdx.x; c0 < tcells; c0 += FLUSH_U * T) {
    u64 old[FLUSH_U];
#pragma unroll
    for (int k = 0; k < FLUSH_U; ++k) {
      const int c = c0 + k * T;
      old[k] = ~0ull;
      if (c >= tcells) continue;
      const int* s = tile + c * TILE_W;
      const int cnt = (int)((unsigned)s[0] & TILE_N_MASK);
      if (cnt == 0) continue;
      const int l0 = c % T0, q = c / T0, l1 = q % T1, l2 = q / T1;
      const uint32_t kf = BS::key(G, foldp<P2>(ox + l0, m0), foldp<P2>(oy + l1, m1), SUB ? oz + l2 : foldp<P2>(oz + l2, m2));
      u64* g = sums + (size_t)kf * G.sw;
      const u64 etile = ((u64)((unsigned)s[0] >> TILE_N_BITS) << TILE_E_SHIFT) + (u64)(unsigned)s[4];
      const u64 w0 = (etile << 16) | (u64)(unsigned)cnt;
      const int side = SUB ? sub_shared(G, oz + l2) : -1;
      if (SUB && side >= 0) {   // the same sums into the neighbour that also holds this cell (integer adds commute: no staging, no ordering)
        // system scope on both copies: the neighbour's GPU adds into `g` at the same time as this one (see above)
        atomicAdd_system(g, w0); atomicAdd_system(g + 1, pack_ss(s[1], s[2])); atomicAdd_system(g + 2, pack_ss(s[3], 0));
        u64* pq = G.peer[side] + (size_t)((long long)kf + G.peer_koff[side]) * G.sw;
        atomicAdd_system(pq, w0); atomicAdd_system(pq + 1, pack_ss(s[1], s[2])); atomicAdd_system(pq + 2, pack_ss(s[3], 0));
        if (ranked) old[k] = (u64)atomicAdd(G.lcount + kf, (uint32_t)cnt);   // this rank's particles already numbered in the cell
        else atomicAdd(G.lcount + kf, (uint32_t)cnt);
      } else {
        if (ranked) old[k] = atomicAdd(g, w0);
        else atomicAdd(g, w0);
        atomicAdd(g + 1, pack_ss(s[1], s[2]));
        atomicAdd(g + 2, pack_ss(s[3], 0));
      }
      // partial momentum sums of >= 64 particles that come within a factor two of the int32 range
      if (cnt >= 64 && (abs(s[1]) >= (1 << 30) || abs(s[2]) >= (1 << 30) || abs(s[3]) >= (1 << 30))) atomicAdd(G.nrange, 1ull);
    }
    if (ranked) {
#pragma unroll
      for (int k = 0; k < FLUSH_U; ++k)
        if (old[k] != ~0ull) io.tbase[(size_t)b * tcells + c0 + k * T] = (uint32_t)(old[k] & 0xffffull);   // slots taken so far in this cell
    }
  }
}

// the collision of the last step, applied on its own when the state is read before the next step
// (key recomputed from the position and that step's shift, still in G.s)
__global__ void __launch_bounds__(256) k_collide_pos(Geo G, size_t n, const float* __restrict__ x, const float* __restrict__ y,
                                                     const float* __restrict__ z, float* __restrict__ vx, float* __restrict__ vy,
                                                     float* __restrict__ vz, const float* __restrict__ rec) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float vs;
  const uint32_t k = key_of(G, x[i], y[i], z[i], G.s[0], G.s[1], G.s[2], &vs);
  float4 r0, ax;
  load_rec(rec, k, r0, ax);
  float v[3] = {vx[i] + vs, vy[i], vz[i]};
  srd_apply(G, r0, ax, v);
  vx[i] = v[0] - vs; vy[i] = v[1]; vz[i] = v[2];
}

__global__ void __launch_bounds__(256) k_keys(Geo G, size_t n, const float* __restrict__ x, const float* __restrict__ y,
                                              const float* __restrict__ z, uint32_t* __restrict__ key) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) key[i] = key_of(G, x[i], y[i], z[i], G.s[0], G.s[1], G.s[2]);
}

}  // namespace mpc

using namespace mpc;

namespace {


// the instantiations that exist: (COLLIDE, WKEY, IO) in { (*,0,PLAIN) at 384 or 512 threads, (*,1,PLAIN), (*,0,RANK),
// (1,0,SCATTER), (1,0,AOS_IN) } x (WALL, GRAV) x brick shape
template <bool COLLIDE, bool WKEY, class BS, int IO, int T>
void* sweep_fn(bool wall, bool grav, bool p2, bool shear) {
  if (shear) return grav ? (void*)k_sweep<COLLIDE, false, true, WKEY, BS, IO, T, false, true> : (void*)k_sweep<COLLIDE, false, false, WKEY, BS, IO, T, false, true>;
  if (wall && grav) return (void*)k_sweep<COLLIDE, true, true, WKEY, BS, IO, T, false, false>;
  if (wall) return (void*)k_sweep<COLLIDE, true, false, WKEY, BS, IO, T, false, false>;
  if (p2) return grav ? (void*)k_sweep<COLLIDE, false, true, WKEY, BS, IO, T, true, false> : (void*)k_sweep<COLLIDE, false, false, WKEY, BS, IO, T, true, false>;
  if (grav) return (void*)k_sweep<COLLIDE, false, true, WKEY, BS, IO, T, false, false>;
  return (void*)k_sweep<COLLIDE, false, false, WKEY, BS, IO, T, false, false>;
}
// slab subdomains: periodic SRD without force
template <class BS, bool P2>
void* sweep_variant_sub2(bool collide, bool wkey, int io, bool three) {
  if (io == IO_AOS_IN) return (void*)k_sweep<true, false, false, false, BS, IO_AOS_IN, SWEEP_T, P2, false, true>;
  if (io == IO_SCATTER) return (void*)k_sweep<true, false, false, false, BS, IO_SCATTER, SWEEP_T, P2, false, true>;
  if (io == IO_RANK) return collide ? (void*)k_sweep<true, false, false, false, BS, IO_RANK, SWEEP_T, P2, false, true> : (void*)k_sweep<false, false, false, false, BS, IO_RANK, SWEEP_T, P2, false, true>;
  if (wkey) return collide ? (void*)k_sweep<true, false, false, true, BS, IO_PLAIN, SWEEP_T, P2, false, true> : (void*)k_sweep<false, false, false, true, BS, IO_PLAIN, SWEEP_T, P2, false, true>;
  if (three) return collide ? (void*)k_sweep<true, false, false, false, BS, IO_PLAIN, SWEEP_T3, P2, false, true> : (void*)k_sweep<false, false, false, false, BS, IO_PLAIN, SWEEP_T3, P2, false, true>;
  return collide ? (void*)k_sweep<true, false, false, false, BS, IO_PLAIN, SWEEP_T, P2, false, true> : (void*)k_sweep<false, false, false, false, BS, IO_PLAIN, SWEEP_T, P2, false, true>;
}
void* sweep_variant_sub(bool fast, bool collide, bool wkey, int io, bool three, bool p2) {
  if (!fast) return sweep_variant_sub2<BSgeneric, false>(collide, wkey, io, three);
  return p2 ? sweep_variant_sub2<BSfast, true>(collide, wkey, io, three) : sweep_variant_sub2<BSfast, false>(collide, wkey, io, three);
}
template <class BS>
void* sweep_variant(bool collide, bool wkey, int io, bool three, bool wall, bool grav, bool p2, bool shear) {
  if (io == IO_AOS_IN) return sweep_fn<true, false, BS, IO_AOS_IN, SWEEP_T>(wall, grav, p2, shear);   // 384 x 3: 15.8 instead of 14.4 ms
  if (io == IO_SCATTER) return sweep_fn<true, false, BS, IO_SCATTER, SWEEP_T>(wall, grav, p2, shear);
  if (io == IO_RANK) {
    if (three) return collide ? sweep_fn<true, false, BS, IO_RANK, SWEEP_T3>(wall, grav, p2, shear) : sweep_fn<false, false, BS, IO_RANK, SWEEP_T3>(wall, grav, p2, shear);
    return collide ? sweep_fn<true, false, BS, IO_RANK, SWEEP_T>(wall, grav, p2, shear) : sweep_fn<false, false, BS, IO_RANK, SWEEP_T>(wall, grav, p2, shear);
  }
  if (wkey) return collide ? sweep_fn<true, true, BS, IO_PLAIN, SWEEP_T>(wall, grav, p2, shear) : sweep_fn<false, true, BS, IO_PLAIN, SWEEP_T>(wall, grav, p2, shear);
  if (three) return collide ? sweep_fn<true, false, BS, IO_PLAIN, SWEEP_T3>(wall, grav, p2, shear) : sweep_fn<false, false, BS, IO_PLAIN, SWEEP_T3>(wall, grav, p2, shear);
  return collide ? sweep_fn<true, false, BS, IO_PLAIN, SWEEP_T>(wall, grav, p2, shear) : sweep_fn<false, false, BS, IO_PLAIN, SWEEP_T>(wall, grav, p2, shear);
}
// the power-of-two variants exist for the {16,16,8} brick only (the shape the large boxes use)
void* sweep_variant_any(bool fast, bool collide, bool wkey, int io, bool three, bool wall, bool grav, bool p2, bool shear) {
  return fast ? sweep_variant<BSfast>(collide, wkey, io, three, wall, grav, p2, shear) : sweep_variant<BSgeneric>(collide, wkey, io, three, wall, grav, false, shear);
}

}  // namespace

int launch_sweep(mpc_ctx* c, bool collide, bool wkey, int io, const float sp[3]) {
  Geo& G = c->G;
  float** F = reinterpret_cast<float**>(c->A);
  if (io == IO_SCATTER && !collide) return fail(c, MPC_ESTATE, "internal: scatter pass without a pending collision");
  SweepIO sio;
  sio.aos = aos_base(c);
  sio.id = c->A[6];
  sio.tbase = c->tbase;
  sio.offset = c->offset;
  sio.spread = c->order_spread;
  // the scatter pass still walks the old order: its brick ranges were saved before the scan overwrote the offsets
  const uint32_t* chunk = (io == IO_SCATTER) ? c->chunk0 : (c->have_order ? c->offset : nullptr);
  sio.chunk_shift = (io == IO_SCATTER) ? 0 : G.bs[0] + G.bs[1] + G.bs[2];
  const bool wall = G.wall >= 0, grav = (G.g[0] != 0.f || G.g[1] != 0.f || G.g[2] != 0.f);
  const bool three = ((io == IO_PLAIN && !wkey) || io == IO_RANK) && c->three_ctas;   // rank pass: 14.8 instead of 15.9 ms
  sio.le_dprev = c->le_dprev;
  void* fn = sweep_variant_any(c->fast_brick, collide, wkey && io == IO_PLAIN, io, three, wall, grav, c->pow2_cells, G.shear != 0);
  const bool three_sub = io == IO_PLAIN && !wkey && c->three_ctas;       // (the rank pass of a subdomain runs 2 x 512)
  if (G.sub) fn = sweep_variant_sub(c->fast_brick, collide, wkey && io == IO_PLAIN, io, three_sub, c->pow2_cells);
  float s0 = sp[0], s1 = sp[1], s2 = sp[2];
  uint32_t n = (uint32_t)c->n;
  void* args[] = {&G, &s0, &s1, &s2, &n, &F[0], &F[1], &F[2], &F[3], &F[4], &F[5], &c->key, &chunk, &c->nbricks, &c->rec, &c->sums, &sio};
  const int T = (G.sub ? three_sub : three) ? SWEEP_T3 : SWEEP_T;
  cudaLaunchKernel(fn, dim3(c->nbricks), dim3(T), args, c->tile_bytes, c->stream);
  LAUNCH_CHECK("k_sweep");
  return MPC_OK;
}

cudaError_t sweep_set_attributes(size_t bytes) {
  for (int m = 0; m < 8; ++m) {   // slab subdomain variants
    const bool fast = m & 1, collide = m & 2, p2 = m & 4;
    if (p2 && !fast) continue;
    const struct { bool wkey; int io; bool three; } v[] = {{false, IO_PLAIN, false}, {false, IO_PLAIN, true}, {true, IO_PLAIN, false},
                                                           {false, IO_RANK, false}, {false, IO_SCATTER, false}, {false, IO_AOS_IN, false}};
    for (const auto& q : v) {
      if (!collide && (q.io == IO_SCATTER || q.io == IO_AOS_IN)) continue;
      const cudaError_t e = cudaFuncSetAttribute(sweep_variant_sub(fast, collide, q.wkey, q.io, q.three, p2), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
      if (e != cudaSuccess) return e;
    }
  }
  for (int mode = 0; mode < 6; ++mode) {          // bit 0: {16,16,8} brick; modes 2,3: power-of-two variant; 4,5: Lees-Edwards
    const bool fast = (mode & 1) != 0, p2 = (mode >> 1) == 1, shear = (mode >> 1) == 2;
    for (int wall = 0; wall < 2; ++wall)
      for (int grav = 0; grav < 2; ++grav)
        for (int collide = 0; collide < 2; ++collide) {
          const struct { bool wkey; int io; bool three; } v[] = {{false, IO_PLAIN, false}, {false, IO_PLAIN, true}, {true, IO_PLAIN, false},
                                                                 {false, IO_RANK, false}, {false, IO_RANK, true}, {false, IO_SCATTER, false}, {false, IO_AOS_IN, false}};
          for (const auto& q : v) {
            if (!collide && (q.io == IO_SCATTER || q.io == IO_AOS_IN)) continue;
            const cudaError_t e = cudaFuncSetAttribute(sweep_variant_any(fast, collide != 0, q.wkey, q.io, q.three, wall != 0, grav != 0, p2, shear),
                                                       cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
            if (e != cudaSuccess) return e;
          }
        }
  }
  return cudaSuccess;
}

int launch_sub_clear(mpc_ctx* c) {   // slab subdomain, before the first step: sums (the neighbours add into them) and local counts
  if (cudaMemsetAsync(c->sums, 0, (size_t)c->G.nkeys * c->G.sw * 8, c->stream) != cudaSuccess ||
      cudaMemsetAsync(c->G.lcount, 0, (size_t)c->G.nkeys * 4, c->stream) != cudaSuccess) return cuda_fail(c, cudaGetLastError(), "cudaMemsetAsync");
  return MPC_OK;
}

int launch_collide_pos(mpc_ctx* c) {
  float** F = reinterpret_cast<float**>(c->A);
  k_collide_pos<<<nblk(c->n, 256), 256, 0, c->stream>>>(c->G, c->n, F[0], F[1], F[2], F[3], F[4], F[5], c->rec);
  LAUNCH_CHECK("k_collide_pos");
  return MPC_OK;
}

int launch_keys(mpc_ctx* c, uint32_t* key_out) {
  float** F = reinterpret_cast<float**>(c->A);
  k_keys<<<nblk(c->n, 256), 256, 0, c->stream>>>(c->G, c->n, F[0], F[1], F[2], key_out);
  LAUNCH_CHECK("k_keys");
  return MPC_OK;
}
