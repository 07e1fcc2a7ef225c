// generic.cu -- MPC-AT (U5) and every angular-momentum-conserving (+a) variant (Eqs. 3-4).
//
// These need the rank of a particle in its (key, id)-sorted cell segment (MPC-AT's random-number index) or ~20 sums
// per cell, so they do not go through the fused SRD sweep. A step is: k_stream_key (MOVE + cell key + count), the
// reorder when due, then
//   * fresh order (every MPC-AT step, every reorder step of SRD+a): k_cell_seg -- ONE thread owns a whole cell, whose
//     particles are the contiguous segment [offset[k], offset[k+1]): it accumulates all cell sums in double in
//     registers (the paper's precision for cell quantities), solves I omega = dL (U10) and
//     applies the collision to its particles. No atomics, no per-cell record, one Philox draw per particle
//     (MPC-AT parks sigma*g in the velocity array between the two passes over the segment);
//   * stale order (SRD+a between reorders): k_accum_a adds 64-bit fixed-point moments (2^40 per unit: the sums are
//     exact to ~1e-12, so the parallel-axis subtraction and I^-1 lose nothing) with global integer atomics,
//     k_cell_a finalises, k_collide_a applies.
#include "cell.cuh"

namespace mpc {

constexpr double FX40 = 1099511627776.0;            // 2^40 per unit of cell-local coordinate (and of u, for velocities)
constexpr double FX40_INV = 1.0 / 1099511627776.0;
// +a sums (16 words per cell): w0 = count; w1..3 = sum v (int64, 2^40/u); w4..6 = sum rho; w7..12 = sum rho rho^T
// (xx, yy, zz, xy, xz, yz); w13..15 = sum rho x (v - D v), in cell-local coordinates rho in [0,1)^3 (U9)

__device__ __forceinline__ float cell_frac(const Geo& G, float r, float s) {
  const float q = (r + s) * G.inv_a;
  return q - floorf(q);
}
// D(alpha) w for unit axis n (Rodrigues, right-handed), fp32: what the particles get
__device__ __forceinline__ void rotate(const Geo& G, float nx, float ny, float nz, const float (&w)[3], float (&o)[3]) {
  const float c = G.cosa, s = G.sina;
  const float nd = fmaf(nx, w[0], fmaf(ny, w[1], nz * w[2])) * (1.0f - c);
  const float cx = fmaf(ny, w[2], -(nz * w[1])), cy = fmaf(nz, w[0], -(nx * w[2])), cz = fmaf(nx, w[1], -(ny * w[0]));
  o[0] = fmaf(w[0], c, fmaf(cx, s, nx * nd));
  o[1] = fmaf(w[1], c, fmaf(cy, s, ny * nd));
  o[2] = fmaf(w[2], c, fmaf(cz, s, nz * nd));
}
// (1 - D(alpha)) w in double, with the fp32 axis and the fp32 cos/sin the particles use
__device__ __forceinline__ void one_minus_D(const Geo& G, double nx, double ny, double nz, const double (&w)[3], double (&u)[3]) {
  const double c = G.cosa, sn = G.sina;
  const double nd = (nx * w[0] + ny * w[1] + nz * w[2]) * (1.0 - c);
  const double cx = ny * w[2] - nz * w[1], cy = nz * w[0] - nx * w[2], cz = nx * w[1] - ny * w[0];
  u[0] = w[0] - (w[0] * c + cx * sn + nx * nd);
  u[1] = w[1] - (w[1] * c + cy * sn + ny * nd);
  u[2] = w[2] - (w[2] * c + cz * sn + nz * nd);
}

// omega = I^-1 dL from the raw moments about the cell corner (parallel-axis forms about rho_cm, U9),
// with the degenerate-cell rules of DESIGN.md U10. P = sum rho, Q = sum rho rho^T (xx,yy,zz,xy,xz,yz),
// Lr = sum rho x u, Su = sum u (all in double). Returns false if the inertia tensor was rejected.
__device__ __forceinline__ bool solve_omega(const Geo& G, uint32_t N, const double (&P)[3], const double (&Q)[6], const double (&Lr)[3],
                                            const double (&Su)[3], double (&rcm)[3], double (&om)[3]) {
  const double inv = 1.0 / (double)N, Nd = (double)N;
  rcm[0] = P[0] * inv; rcm[1] = P[1] * inv; rcm[2] = P[2] * inv;
  om[0] = om[1] = om[2] = 0.0;
  if (N < 2u) return true;
  const double a = G.a, m = G.mass;
  // second moments about the centre of mass, in units of a^2
  const double Qxx = Q[0] - Nd * rcm[0] * rcm[0], Qyy = Q[1] - Nd * rcm[1] * rcm[1], Qzz = Q[2] - Nd * rcm[2] * rcm[2];
  const double Qxy = Q[3] - Nd * rcm[0] * rcm[1], Qxz = Q[4] - Nd * rcm[0] * rcm[2], Qyz = Q[5] - Nd * rcm[1] * rcm[2];
  const double dL[3] = {m * a * (Lr[0] - (rcm[1] * Su[2] - rcm[2] * Su[1])),
                        m * a * (Lr[1] - (rcm[2] * Su[0] - rcm[0] * Su[2])),
                        m * a * (Lr[2] - (rcm[0] * Su[1] - rcm[1] * Su[0]))};
  const double R2 = a * a * (Qxx + Qyy + Qzz);
  if (N == 2u) {
    if (R2 > 0.0) { om[0] = dL[0] / (m * R2); om[1] = dL[1] / (m * R2); om[2] = dL[2] / (m * R2); }
    return true;
  }
  const double f = m * a * a;
  const double xx = f * (Qyy + Qzz), yy = f * (Qxx + Qzz), zz = f * (Qxx + Qyy), xy = -f * Qxy, xz = -f * Qxz, yz = -f * Qyz;
  const double c00 = yy * zz - yz * yz, c01 = xz * yz - xy * zz, c02 = xy * yz - xz * yy;
  const double c11 = xx * zz - xz * xz, c12 = xy * xz - xx * yz, c22 = xx * yy - xy * xy;
  const double det = xx * c00 + xy * c01 + xz * c02, tr3 = (xx + yy + zz) / 3.0;
  if (!(det > 1e-6 * tr3 * tr3 * tr3)) return false;     // rejected inertia tensor (U10): omega = 0
  om[0] = (c00 * dL[0] + c01 * dL[1] + c02 * dL[2]) / det;
  om[1] = (c01 * dL[0] + c11 * dL[1] + c12 * dL[2]) / det;
  om[2] = (c02 * dL[0] + c12 * dL[1] + c22 * dL[2]) / det;
  return true;
}

// MOVE + cell key + count (the count field of word 0 of the cell's sums)
template <bool WALL, bool GRAV>
__global__ void __launch_bounds__(256) k_stream_key(Geo G, size_t n, float* __restrict__ x, float* __restrict__ y,
                                                    float* __restrict__ z, float* __restrict__ vx, float* __restrict__ vy,
                                                    float* __restrict__ vz, uint32_t* __restrict__ key, u64* __restrict__ sums) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float r[3] = {x[i], y[i], z[i]}, v[3] = {vx[i], vy[i], vz[i]};
  if (!(fabsf(v[0]) < G.vmax && fabsf(v[1]) < G.vmax && fabsf(v[2]) < G.vmax)) atomicAdd(G.nrange, 1ull);
  stream_one<WALL, GRAV>(G, r, v);
  x[i] = r[0]; y[i] = r[1]; z[i] = r[2];
  if (WALL || GRAV) { vx[i] = v[0]; vy[i] = v[1]; vz[i] = v[2]; }
  const uint32_t k = key_of(G, r[0], r[1], r[2], G.s[0], G.s[1], G.s[2]);
  key[i] = k;
  atomicAdd(sums + (size_t)k * G.sw, 1ull);
}

// Fresh (key, id) order: one thread per cell does PROCESS, PROCESS_CELLS and ROTATE_VELOCITIES for its segment.
template <bool AT, bool PLUS_A>
__global__ void __launch_bounds__(128) k_cell_seg(Geo G, int cpb_shift, const float* __restrict__ x, const float* __restrict__ y,
                                                  const float* __restrict__ z, float* vx, float* vy, float* vz,
                                                  const uint32_t* __restrict__ offset, u64* __restrict__ sums, u64* __restrict__ nsing) {
  const int b0 = G.bs[0], b1 = G.bs[1], b2 = G.bs[2];
  const uint32_t bx = blockIdx.x >> cpb_shift, by = blockIdx.y, bz = blockIdx.z;
  const uint32_t brick = (bz * (uint32_t)G.mb[1] + by) * (uint32_t)G.mb[0] + bx;
  const uint32_t bvol = 1u << (b0 + b1 + b2);
  // neighbouring lanes own neighbouring cells, i.e. neighbouring segments: a warp's loads stay within a few lines
  // (assigning the cells to lanes in order of occupancy instead balances the loop lengths but scatters the accesses:
  // measured 2.3 ms against 0.69 ms at config 3)
  const uint32_t local = ((blockIdx.x & ((1u << cpb_shift) - 1u)) << 7) | threadIdx.x;
  if (local >= bvol) return;
  const uint32_t k = (brick << (b0 + b1 + b2)) | local;
  const uint32_t jb = offset[k], je = offset[k + 1];
  const uint32_t N = je - jb;
  if (N == 0u) return;
  const int ix = (int)((bx << b0) | (local & ((1u << b0) - 1u)));
  const int iy = (int)((by << b1) | ((local >> b0) & ((1u << b1) - 1u)));
  const int iz = (int)((bz << b2) | (local >> (b0 + b1)));
  const uint32_t cid = canonical_id(G, ix, iy, iz);
  float ax = 0.f, ay = 0.f, az = 1.f;
  if (!AT) srd_axis(G, cid, ax, ay, az);
  double S[3] = {0, 0, 0}, R[3] = {0, 0, 0}, P[3] = {0, 0, 0}, Q[6] = {0, 0, 0, 0, 0, 0}, Lr[3] = {0, 0, 0};
  for (uint32_t j = jb; j < je; ++j) {
    const float vf[3] = {vx[j], vy[j], vz[j]};
    const double v[3] = {vf[0], vf[1], vf[2]};
    double u[3];
    if (AT) {
      const Block4 o = philox_rk(cid, j - jb, G.t, TAG_AT, G.rk);
      float g0, g1, g2;
      normals3(o, g0, g1, g2);
      g0 *= G.sigma; g1 *= G.sigma; g2 *= G.sigma;
      if (N > 1u) { vx[j] = g0; vy[j] = g1; vz[j] = g2; }      // parked for the second pass
      R[0] += g0; R[1] += g1; R[2] += g2;
      u[0] = v[0] - g0; u[1] = v[1] - g1; u[2] = v[2] - g2;
    } else if (PLUS_A) {
      one_minus_D(G, ax, ay, az, v, u);
    }
    S[0] += v[0]; S[1] += v[1]; S[2] += v[2];
    if (PLUS_A) {
      const double r0 = cell_frac(G, x[j], G.s[0]), r1 = cell_frac(G, y[j], G.s[1]), r2 = cell_frac(G, z[j], G.s[2]);
      P[0] += r0; P[1] += r1; P[2] += r2;
      Q[0] += r0 * r0; Q[1] += r1 * r1; Q[2] += r2 * r2; Q[3] += r0 * r1; Q[4] += r0 * r2; Q[5] += r1 * r2;
      Lr[0] += r1 * u[2] - r2 * u[1]; Lr[1] += r2 * u[0] - r0 * u[2]; Lr[2] += r0 * u[1] - r1 * u[0];
    }
  }
  {   // pre-collision momentum sums for the observables / test hook, in the packed format of the SRD path
    u64* s = sums + (size_t)k * G.sw;
    s[1] = pack_ss(__double2int_rn(S[0] * (double)G.fxv), __double2int_rn(S[1] * (double)G.fxv));
    s[2] = pack_ss(__double2int_rn(S[2] * (double)G.fxv), 0);
  }
  if (N == 1u) return;                                   // a lone particle keeps its velocity
  const double inv = 1.0 / (double)N;
  const float base[3] = {(float)((S[0] - R[0]) * inv), (float)((S[1] - R[1]) * inv), (float)((S[2] - R[2]) * inv)};   // R = 0 for SRD
  double om[3] = {0, 0, 0}, rcm[3] = {0, 0, 0};
  if (PLUS_A) {
    double Su[3];
    if (AT) { Su[0] = S[0] - R[0]; Su[1] = S[1] - R[1]; Su[2] = S[2] - R[2]; }
    else one_minus_D(G, ax, ay, az, S, Su);
    if (!solve_omega(G, N, P, Q, Lr, Su, rcm, om)) atomicAdd(nsing, 1ull);
  }
  const float omf[3] = {(float)om[0], (float)om[1], (float)om[2]}, rcf[3] = {(float)rcm[0], (float)rcm[1], (float)rcm[2]};
  for (uint32_t j = jb; j < je; ++j) {
    float o[3];
    if (AT) {
      o[0] = base[0] + vx[j]; o[1] = base[1] + vy[j]; o[2] = base[2] + vz[j];
    } else {
      const float w[3] = {vx[j] - base[0], vy[j] - base[1], vz[j] - base[2]};
      float d[3];
      rotate(G, ax, ay, az, w, d);
      o[0] = base[0] + d[0]; o[1] = base[1] + d[1]; o[2] = base[2] + d[2];
    }
    if (PLUS_A) {
      const float r0 = (cell_frac(G, x[j], G.s[0]) - rcf[0]) * G.a, r1 = (cell_frac(G, y[j], G.s[1]) - rcf[1]) * G.a,
                  r2 = (cell_frac(G, z[j], G.s[2]) - rcf[2]) * G.a;
      o[0] += fmaf(omf[1], r2, -(omf[2] * r1));
      o[1] += fmaf(omf[2], r0, -(omf[0] * r2));
      o[2] += fmaf(omf[0], r1, -(omf[1] * r0));
    }
    vx[j] = o[0]; vy[j] = o[1]; vz[j] = o[2];
  }
}


// ---- extended per-cell pass: particle masses (embedded solutes, U23) and explicit phantom particles in
// wall-cut cells (U22) -------------------------------------------------------------
// omega from mass-weighted raw moments: Ms = sum m_i, P = sum m_i rho_i, Q = sum m_i rho_i rho_i^T, Lr = sum m_i rho_i x u_i,
// Su = sum m_i u_i; N = number of members (degenerate-cell rules of U10)
__device__ __forceinline__ bool solve_omega_m(const Geo& G, uint32_t N, double Ms, const double (&P)[3], const double (&Q)[6],
                                              const double (&Lr)[3], const double (&Su)[3], double (&rcm)[3], double (&om)[3]) {
  const double inv = 1.0 / Ms;
  rcm[0] = P[0] * inv; rcm[1] = P[1] * inv; rcm[2] = P[2] * inv;
  om[0] = om[1] = om[2] = 0.0;
  if (N < 2u) return true;
  const double a = G.a;
  const double Qxx = Q[0] - Ms * rcm[0] * rcm[0], Qyy = Q[1] - Ms * rcm[1] * rcm[1], Qzz = Q[2] - Ms * rcm[2] * rcm[2];
  const double Qxy = Q[3] - Ms * rcm[0] * rcm[1], Qxz = Q[4] - Ms * rcm[0] * rcm[2], Qyz = Q[5] - Ms * rcm[1] * rcm[2];
  const double dL[3] = {a * (Lr[0] - (rcm[1] * Su[2] - rcm[2] * Su[1])), a * (Lr[1] - (rcm[2] * Su[0] - rcm[0] * Su[2])),
                        a * (Lr[2] - (rcm[0] * Su[1] - rcm[1] * Su[0]))};
  const double R2 = a * a * (Qxx + Qyy + Qzz);
  if (N == 2u) {
    if (R2 > 0.0) { om[0] = dL[0] / R2; om[1] = dL[1] / R2; om[2] = dL[2] / R2; }
    return true;
  }
  const double f = a * a;
  const double xx = f * (Qyy + Qzz), yy = f * (Qxx + Qzz), zz = f * (Qxx + Qyy), xy = -f * Qxy, xz = -f * Qxz, yz = -f * Qyz;
  const double c00 = yy * zz - yz * yz, c01 = xz * yz - xy * zz, c02 = xy * yz - xz * yy;
  const double c11 = xx * zz - xz * xz, c12 = xy * xz - xx * yz, c22 = xx * yy - xy * xy;
  const double det = xx * c00 + xy * c01 + xz * c02, tr3 = (xx + yy + zz) / 3.0;
  if (!(det > 1e-6 * tr3 * tr3 * tr3)) return false;
  om[0] = (c00 * dL[0] + c01 * dL[1] + c02 * dL[2]) / det;
  om[1] = (c01 * dL[0] + c11 * dL[1] + c12 * dL[2]) / det;
  om[2] = (c02 * dL[0] + c12 * dL[1] + c22 * dL[2]) / det;
  return true;
}

// One thread owns a cell (fresh (key, id) order, as k_cell_seg). Members of the cell = its real particles in ascending
// id, then the phantoms of its wall part (regenerated from their Philox streams, never stored). Every sum carries the
// member's mass; SRD -a may use the cell thermostat (kappa from sum m_i |v_i - v_cm|^2 and f = 3 (members - 1)).
template <bool AT, bool PLUS_A>
__global__ void __launch_bounds__(128) k_cell_seg_ext(Geo G, int cpb_shift, const float* __restrict__ x, const float* __restrict__ y,
                                                      const float* __restrict__ z, float* vx, float* vy, float* vz,
                                                      const uint32_t* __restrict__ id, const uint32_t* __restrict__ offset,
                                                      u64* __restrict__ sums, u64* __restrict__ nsing) {
  const int b0 = G.bs[0], b1 = G.bs[1], b2 = G.bs[2];
  const uint32_t bx = blockIdx.x >> cpb_shift, by = blockIdx.y, bz = blockIdx.z;
  const uint32_t brick = (bz * (uint32_t)G.mb[1] + by) * (uint32_t)G.mb[0] + bx;
  const uint32_t bvol = 1u << (b0 + b1 + b2);
  const uint32_t local = ((blockIdx.x & ((1u << cpb_shift) - 1u)) << 7) | threadIdx.x;
  if (local >= bvol) return;
  const uint32_t k = (brick << (b0 + b1 + b2)) | local;
  const uint32_t jb = offset[k], je = offset[k + 1];
  const uint32_t nreal = je - jb;
  if (nreal == 0u) return;
  const int ix = (int)((bx << b0) | (local & ((1u << b0) - 1u)));
  const int iy = (int)((by << b1) | ((local >> b0) & ((1u << b1) - 1u)));
  const int iz = (int)((bz << b2) | (local >> (b0 + b1)));
  const uint32_t cid = canonical_id(G, ix, iy, iz);
  // ---- phantoms of this cell (U22): number, wall part [0, phi) (wall at 0) or [sp, 1) (wall at L) of the wall axis ----
  uint32_t nph = 0;
  bool top = false;
  float phi = 0.0f, sp = 0.0f;
  const int w = G.wall;
  if (G.phantoms && w >= 0) {
    const float sw = (w == 0) ? G.s[0] : (w == 1) ? G.s[1] : G.s[2];
    if (sw != 0.0f) {
      const int iw = (w == 0) ? ix : (w == 1) ? iy : iz;
      const int nw = (w == 0) ? G.n[0] : (w == 1) ? G.n[1] : G.n[2];
      const float sg = sw * G.inv_a;
      sp = (sg > 0.0f) ? sg : 1.0f + sg;
      const int lo = (sw > 0.0f) ? 1 : 0, hi = (sw > 0.0f) ? nw + 1 : nw;
      if (iw == lo) phi = sp;
      else if (iw == hi) { top = true; phi = 1.0f - sp; }
      if (phi > 0.0f) {
        const Block4 o = philox_rk(cid, 0u, G.t, TAG_PHANTOM, G.rk);
        nph = (uint32_t)(int)floorf(fmaf((float)G.nbar, phi, u01_co(o.a)));
      }
    }
  }
  const uint32_t N = nreal + nph;
  const Block4 oax = philox_rk(cid, 0u, G.t, TAG_AXIS, G.rk);
  float ax = 0.f, ay = 0.f, az = 1.f;
  if (!AT) {
    az = 2.0f * u01_co(oax.a) - 1.0f;
    const float rr = sqrtf((1.0f - az) * (1.0f + az));
    float sph, cph;
    sincospif(2.0f * u01_co(oax.b), &sph, &cph);
    ax = rr * cph; ay = rr * sph;
  }
  const double m0 = G.mass;
  const bool solutes = G.solute_mass > 0.0f;
  const float sig_sol = solutes ? (float)sqrt((double)G.kT / (double)G.solute_mass) : G.sigma;
  double Ms = 0.0, S[3] = {0, 0, 0}, R[3] = {0, 0, 0}, P[3] = {0, 0, 0}, Q[6] = {0, 0, 0, 0, 0, 0}, Lr[3] = {0, 0, 0}, E = 0.0;
  for (uint32_t j = 0; j < N; ++j) {
    double mi = m0, v[3], rho[3] = {0, 0, 0};
    float sgi = G.sigma;
    if (j < nreal) {
      const uint32_t i = jb + j;
      if (solutes && id[i] >= G.solute_id0) { mi = (double)G.solute_mass; sgi = sig_sol; }
      v[0] = vx[i]; v[1] = vy[i]; v[2] = vz[i];
      if (PLUS_A) { rho[0] = cell_frac(G, x[i], G.s[0]); rho[1] = cell_frac(G, y[i], G.s[1]); rho[2] = cell_frac(G, z[i], G.s[2]); }
    } else {
      const uint32_t q = j - nreal;
      const Block4 pp = philox_rk(cid, 1u + 2u * q, G.t, TAG_PHANTOM, G.rk);
      const Block4 pv = philox_rk(cid, 2u + 2u * q, G.t, TAG_PHANTOM, G.rk);
      const float ua = u01_co(pp.a), ub = u01_co(pp.b), zeta = u01_co(pp.c);
      const float rw = top ? fmaf(zeta, phi, sp) : zeta * phi;
      rho[0] = (w == 0) ? rw : ua;
      rho[1] = (w == 1) ? rw : ((w == 0) ? ua : ub);
      rho[2] = (w == 2) ? rw : ub;
      float g0, g1, g2;
      normals3(pv, g0, g1, g2);
      v[0] = (double)(G.sigma * g0) + (top ? (double)G.wall_u : -(double)G.wall_u);
      v[1] = (double)(G.sigma * g1); v[2] = (double)(G.sigma * g2);
    }
    double u[3] = {0, 0, 0};
    if (AT) {
      const Block4 o = philox_rk(cid, j, G.t, TAG_AT, G.rk);
      float g0, g1, g2;
      normals3(o, g0, g1, g2);
      g0 *= sgi; g1 *= sgi; g2 *= sgi;
      if (j < nreal && N > 1u) { vx[jb + j] = g0; vy[jb + j] = g1; vz[jb + j] = g2; }   // parked for the second pass
      R[0] += mi * g0; R[1] += mi * g1; R[2] += mi * g2;
      u[0] = v[0] - g0; u[1] = v[1] - g1; u[2] = v[2] - g2;
    } else if (PLUS_A) {
      one_minus_D(G, ax, ay, az, v, u);
    }
    Ms += mi;
    S[0] += mi * v[0]; S[1] += mi * v[1]; S[2] += mi * v[2];
    if (!AT && !PLUS_A) E += mi * (v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
    if (PLUS_A) {
      P[0] += mi * rho[0]; P[1] += mi * rho[1]; P[2] += mi * rho[2];
      Q[0] += mi * rho[0] * rho[0]; Q[1] += mi * rho[1] * rho[1]; Q[2] += mi * rho[2] * rho[2];
      Q[3] += mi * rho[0] * rho[1]; Q[4] += mi * rho[0] * rho[2]; Q[5] += mi * rho[1] * rho[2];
      Lr[0] += mi * (rho[1] * u[2] - rho[2] * u[1]); Lr[1] += mi * (rho[2] * u[0] - rho[0] * u[2]); Lr[2] += mi * (rho[0] * u[1] - rho[1] * u[0]);
    }
    if (j + 1 == nreal) {   // pre-collision momentum of the real particles (in units of the fluid-particle mass) for the test hook
      u64* sk = sums + (size_t)k * G.sw;
      const double f = (double)G.fxv / m0;
      sk[1] = pack_ss(__double2int_rn(S[0] * f), __double2int_rn(S[1] * f));
      sk[2] = pack_ss(__double2int_rn(S[2] * f), 0);
    }
  }
  if (N == 1u) return;                                   // a lone particle keeps its velocity
  const double inv = 1.0 / Ms;
  const float base[3] = {(float)((S[0] - R[0]) * inv), (float)((S[1] - R[1]) * inv), (float)((S[2] - R[2]) * inv)};   // R = 0 for SRD
  double om[3] = {0, 0, 0}, rcm[3] = {0, 0, 0};
  if (PLUS_A) {
    double Su[3];
    if (AT) { Su[0] = S[0] - R[0]; Su[1] = S[1] - R[1]; Su[2] = S[2] - R[2]; }
    else one_minus_D(G, ax, ay, az, S, Su);
    if (!solve_omega_m(G, N, Ms, P, Q, Lr, Su, rcm, om)) atomicAdd(nsing, 1ull);
  }
  float kappa = 1.0f;
  if (!AT && !PLUS_A && G.thermostat) {
    const double W2 = E - (S[0] * S[0] + S[1] * S[1] + S[2] * S[2]) * inv;   // sum m_i |v_i - v_cm|^2
    if (W2 > 0.0) kappa = mbs_kappa(G, cid, oax, N, (float)W2);
  }
  const float omf[3] = {(float)om[0], (float)om[1], (float)om[2]}, rcf[3] = {(float)rcm[0], (float)rcm[1], (float)rcm[2]};
  for (uint32_t j = jb; j < je; ++j) {
    float o[3];
    if (AT) {
      o[0] = base[0] + vx[j]; o[1] = base[1] + vy[j]; o[2] = base[2] + vz[j];
    } else {
      const float wv[3] = {vx[j] - base[0], vy[j] - base[1], vz[j] - base[2]};
      float d[3];
      rotate(G, ax, ay, az, wv, d);
      o[0] = fmaf(kappa, d[0], base[0]); o[1] = fmaf(kappa, d[1], base[1]); o[2] = fmaf(kappa, d[2], base[2]);
    }
    if (PLUS_A) {
      const float r0 = (cell_frac(G, x[j], G.s[0]) - rcf[0]) * G.a, r1 = (cell_frac(G, y[j], G.s[1]) - rcf[1]) * G.a,
                  r2 = (cell_frac(G, z[j], G.s[2]) - rcf[2]) * G.a;
      o[0] += fmaf(omf[1], r2, -(omf[2] * r1));
      o[1] += fmaf(omf[2], r0, -(omf[0] * r2));
      o[2] += fmaf(omf[0], r1, -(omf[1] * r0));
    }
    vx[j] = o[0]; vy[j] = o[1]; vz[j] = o[2];
  }
}

// ---- SRD+a on a stale order: 64-bit fixed-point moments with global atomics ---------------------------
__global__ void __launch_bounds__(256) k_accum_a(Geo G, size_t n, const float* __restrict__ x, const float* __restrict__ y,
                                                 const float* __restrict__ z, const float* __restrict__ vx,
                                                 const float* __restrict__ vy, const float* __restrict__ vz,
                                                 const uint32_t* __restrict__ key, u64* __restrict__ sums) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t k = key[i];
  int ix, iy, iz;
  key_to_cell(G, k, ix, iy, iz);
  const uint32_t cid = canonical_id(G, ix, iy, iz);
  const double v[3] = {vx[i], vy[i], vz[i]};
  const double r0 = cell_frac(G, x[i], G.s[0]), r1 = cell_frac(G, y[i], G.s[1]), r2 = cell_frac(G, z[i], G.s[2]);
  float ax, ay, az;
  srd_axis(G, cid, ax, ay, az);
  double u[3];
  one_minus_D(G, ax, ay, az, v, u);
  const double fv = (double)G.fxv * 262144.0;          // 2^40 / u
  u64* s = sums + (size_t)k * G.sw;
  auto add = [&](int w, double val, double scale) { atomicAdd(s + w, (u64)__double2ll_rn(val * scale)); };
  add(1, v[0], fv); add(2, v[1], fv); add(3, v[2], fv);
  add(4, r0, FX40); add(5, r1, FX40); add(6, r2, FX40);
  add(7, r0 * r0, FX40); add(8, r1 * r1, FX40); add(9, r2 * r2, FX40);
  add(10, r0 * r1, FX40); add(11, r0 * r2, FX40); add(12, r1 * r2, FX40);
  add(13, r1 * u[2] - r2 * u[1], fv); add(14, r2 * u[0] - r0 * u[2], fv); add(15, r0 * u[1] - r1 * u[0], fv);
}

// rec[key] (16 floats) = { v_cm.xyz, 1 | axis.xyz, - | omega.xyz, - | rho_cm.xyz, - }
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
  const double fvi = G.fxv_inv / 262144.0;
  auto get = [&](int w, double scale) { return (double)(long long)s[w] * scale; };
  const double S[3] = {get(1, fvi), get(2, fvi), get(3, fvi)};
  const double P[3] = {get(4, FX40_INV), get(5, FX40_INV), get(6, FX40_INV)};
  const double Q[6] = {get(7, FX40_INV), get(8, FX40_INV), get(9, FX40_INV), get(10, FX40_INV), get(11, FX40_INV), get(12, FX40_INV)};
  const double Lr[3] = {get(13, fvi), get(14, fvi), get(15, fvi)};
  float ax, ay, az;
  srd_axis(G, cid, ax, ay, az);
  double Su[3], om[3], rcm[3];
  one_minus_D(G, ax, ay, az, S, Su);
  if (!solve_omega(G, N, P, Q, Lr, Su, rcm, om)) atomicAdd(nsing, 1ull);
  const double inv = 1.0 / (double)N;
  float4* o = reinterpret_cast<float4*>(rec) + (size_t)k * 4;
  o[0] = make_float4((float)(S[0] * inv), (float)(S[1] * inv), (float)(S[2] * inv), 1.0f);
  o[1] = make_float4(ax, ay, az, 0.0f);
  o[2] = make_float4((float)om[0], (float)om[1], (float)om[2], 0.0f);
  o[3] = make_float4((float)rcm[0], (float)rcm[1], (float)rcm[2], 0.0f);
}

__global__ void __launch_bounds__(256) k_collide_a(Geo G, size_t n, const float* __restrict__ x, const float* __restrict__ y,
                                                   const float* __restrict__ z, float* __restrict__ vx, float* __restrict__ vy,
                                                   float* __restrict__ vz, const uint32_t* __restrict__ key, const float* __restrict__ rec) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t k = key[i];
  const float4* rc = reinterpret_cast<const float4*>(rec) + (size_t)k * 4;
  const float4 base = __ldg(rc), axis = __ldg(rc + 1), om = __ldg(rc + 2), rcm = __ldg(rc + 3);
  const float w[3] = {vx[i] - base.x, vy[i] - base.y, vz[i] - base.z};
  float d[3];
  rotate(G, axis.x, axis.y, axis.z, w, d);
  const float r0 = (cell_frac(G, x[i], G.s[0]) - rcm.x) * G.a, r1 = (cell_frac(G, y[i], G.s[1]) - rcm.y) * G.a,
              r2 = (cell_frac(G, z[i], G.s[2]) - rcm.z) * G.a;
  vx[i] = base.x + d[0] + fmaf(om.y, r2, -(om.z * r1));
  vy[i] = base.y + d[1] + fmaf(om.z, r0, -(om.x * r2));
  vz[i] = base.z + d[2] + fmaf(om.x, r1, -(om.y * r0));
}

// pre-collision momentum sums of the stale-order path, repacked for the observables / test hook
__global__ void __launch_bounds__(256) k_export_a(Geo G, u64* __restrict__ sums) {
  const size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= G.nkeys) return;
  u64* s = sums + k * G.sw;
  if ((s[0] & 0xffffull) == 0ull) return;
  const long long a = (long long)s[1], b = (long long)s[2], c = (long long)s[3];
  s[1] = pack_ss((int)((a + 131072) >> 18), (int)((b + 131072) >> 18));
  s[2] = pack_ss((int)((c + 131072) >> 18), 0);
}

}  // namespace mpc

using namespace mpc;

int steps_generic(mpc_ctx* c, int nsteps) {
  Geo& G = c->G;
  const size_t n = c->n;
  const bool at = G.collision == 1, plus_a = G.conserve_L != 0;
  for (int k = 0; k < nsteps; ++k) {
    G.t = c->t;
    {
      float s[3] = {0.f, 0.f, 0.f};
      if (c->p.grid_shift) {
        const Block4 o = philox(0u, 0u, c->t, TAG_SHIFT, G.k0, G.k1);
        s[0] = (u01_co(o.a) - 0.5f) * G.a; s[1] = (u01_co(o.b) - 0.5f) * G.a; s[2] = (u01_co(o.c) - 0.5f) * G.a;
      }
      G.s[0] = s[0]; G.s[1] = s[1]; G.s[2] = s[2];
    }
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
        const bool wall = G.wall >= 0;
        if (wall && grav) k_stream_key<true, true><<<gb, 256, 0, c->stream>>>(G, n, F[0], F[1], F[2], F[3], F[4], F[5], c->key, c->sums);
        else if (wall) k_stream_key<true, false><<<gb, 256, 0, c->stream>>>(G, n, F[0], F[1], F[2], F[3], F[4], F[5], c->key, c->sums);
        else if (grav) k_stream_key<false, true><<<gb, 256, 0, c->stream>>>(G, n, F[0], F[1], F[2], F[3], F[4], F[5], c->key, c->sums);
        else k_stream_key<false, false><<<gb, 256, 0, c->stream>>>(G, n, F[0], F[1], F[2], F[3], F[4], F[5], c->key, c->sums);
        LAUNCH_CHECK("k_stream_key");
      }
      if (rebin) {
        const int rc = do_reorder(c, false, true, false);
        if (rc) return rc;
        F = reinterpret_cast<float**>(c->A);
        FamilyTimer ft(c, F_CELL);
        if (G.phantoms || G.solute_mass > 0.0f) {     // particle masses / explicit phantoms (U22, U23): extended per-cell pass
#define EXT_ARGS c->seg_grid, 128, 0, c->stream>>>(G, c->seg_cpb_shift, F[0], F[1], F[2], F[3], F[4], F[5], c->A[6], c->offset, c->sums, c->nsing)
          if (plus_a && at) k_cell_seg_ext<true, true><<<EXT_ARGS;
          else if (plus_a) k_cell_seg_ext<false, true><<<EXT_ARGS;
          else if (at) k_cell_seg_ext<true, false><<<EXT_ARGS;
          else k_cell_seg_ext<false, false><<<EXT_ARGS;
#undef EXT_ARGS
        }
        else if (plus_a && at) k_cell_seg<true, true><<<c->seg_grid, 128, 0, c->stream>>>(G, c->seg_cpb_shift, F[0], F[1], F[2], F[3], F[4], F[5], c->offset, c->sums, c->nsing);
        else if (plus_a) k_cell_seg<false, true><<<c->seg_grid, 128, 0, c->stream>>>(G, c->seg_cpb_shift, F[0], F[1], F[2], F[3], F[4], F[5], c->offset, c->sums, c->nsing);
        else k_cell_seg<true, false><<<c->seg_grid, 128, 0, c->stream>>>(G, c->seg_cpb_shift, F[0], F[1], F[2], F[3], F[4], F[5], c->offset, c->sums, c->nsing);
        LAUNCH_CHECK("k_cell_seg");
      } else {   // SRD+a between reorders (MPC-AT reorders every step: enforced at create)
        {
          FamilyTimer ft(c, F_ACCUM);
          k_accum_a<<<gb, 256, 0, c->stream>>>(G, n, F[0], F[1], F[2], F[3], F[4], F[5], c->key, c->sums);
          LAUNCH_CHECK("k_accum_a");
        }
        {
          FamilyTimer ft(c, F_CELL);
          k_cell_a<<<c->seg_grid, 128, 0, c->stream>>>(G, c->seg_cpb_shift, c->sums, c->rec, c->nsing);
          LAUNCH_CHECK("k_cell_a");
        }
        FamilyTimer ft(c, F_COLLIDE);
        k_collide_a<<<gb, 256, 0, c->stream>>>(G, n, F[0], F[1], F[2], F[3], F[4], F[5], c->key, c->rec);
        LAUNCH_CHECK("k_collide_a");
        k_export_a<<<nblk(G.nkeys, 256), 256, 0, c->stream>>>(G, c->sums);
        LAUNCH_CHECK("k_export_a");
      }
    }
    c->t++;
    c->have_cells = true;
  }
  return MPC_OK;
}
