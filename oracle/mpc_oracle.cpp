// =====================================================================================
// oracle/mpc_oracle.cpp  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded CPU restatement of one multiparticle-collision-dynamics
// (MPC) time step as defined in /root/reference/PAPER.md (arXiv 2406.15236, "HTMPC"),
// Sec. II, with the readings U1..U24 listed in DESIGN.md ("Readings of the paper").
// It exists to check the CUDA library (paper_2406_15236_b200/csrc) element by element.
//
//   * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
//     legs may load this library. The product never calls it; there is no CPU fallback.
//   * It shares no code with the CUDA path: no header, helper, table or constant
//     generator is common. The Philox-4x32-10 stream *definition* is re-typed here.
//   * Per-particle state is fp32 (what decides a cell index is done in fp32 with explicit
//     fmaf, U1). Everything per cell (sums, centre of mass, rotation, thermostat,
//     inertia tensor) is done in double, the paper's own choice (III.G.1),
//     and cast to fp32 when written back to a particle.
//   * No blocking, fusion or reordering: the step is written in the paper's order
//     MOVE -> PROCESS -> PROCESS_CELLS -> ROTATE_VELOCITIES (Fig. 1c).
//
// Pins (tests/test_oracle_*.py): Philox known-answer vectors, the hand-computed SRD cell
// of DESIGN.md, exact per-cell momentum / energy / angular-momentum invariants,
// the thermostat's gamma sampler (restated with exact rational arithmetic, bit for bit; moments,
// KS, golden vector), Maxwell statistics, the analytic SRD viscosity from a forced Poiseuille
// profile and from the Lees-Edwards shear stress. Parity unpinned: none; U7/U8 (wall details)
// pinned by hand cases and statistically.
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -fPIC -shared  (see oracle/build.py)
// =====================================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <string>
#include <vector>

namespace {

// ---- parameter block (re-typed; layout mirrored by oracle/binding.py) --------------------
struct Params {
  int   collision;    // 0 = SRD (Eq. 2), 1 = MPC-AT (reading U5)
  int   conserve_L;   // 0 = -a, 1 = +a (Eqs. 3,4)
  int   thermostat;   // 0 = none, 1 = cell-level Maxwell-Boltzmann scaling (Eqs. 5-7)
  float alpha;        // SRD rotation angle [rad]
  float dt, kT, mass;
  float g[3];         // constant acceleration
  int   bc[3];        // 0 periodic, 1 no-slip walls at 0 and L (bounce-back + virtual wall particles), 2 slip walls
                      // (specular reflection, no virtual particles; reading U20)
  int   grid_shift;   // 1 = random lattice shift every step
  int   rebin_every;  // reorder interval
  int   brick[3];     // brick dims of the brick-major key layout ({1,1,1} = row-major); memory order only
  float shear_rate;   // Lees-Edwards shear ("shear flow can also be added", reading U21): d v_x / d z; 0 = off
  int   phantoms;     // 1 = explicit phantom-particle set in wall-cut cells (reading U22) instead of the
                      // velocity-only virtual particles of U8; needed for +a and MPC-AT at walls
  unsigned solute_id0;// embedded point-particle solutes (reading U23): particles with id >= solute_id0
  float solute_mass;  // ... have this mass instead of `mass` (0 = no solutes); they take part in the collision with their mass
  float wall_velocity;// moving no-slip walls (Couette; "no-slip (... also supporting shear flow)", reading U24):
                      // the wall at L moves with +wall_velocity along x, the wall at 0 with -wall_velocity
};

struct Obs {
  unsigned long long n;
  double P[3], E_kin, kT_est, kT_cell;
  unsigned max_cell_count;
  unsigned long long n_singular_cells, step;
};

enum { TAG_SHIFT = 0, TAG_AXIS = 1, TAG_MBS = 2, TAG_AT = 3, TAG_WALL = 4, TAG_PHANTOM = 5 };
enum { E_OK = 0, E_INVAL = -1, E_STATE = -2 };

struct Ctx {
  float L[3];
  int n[3];        // fluid cells per axis
  int m[3];        // collision-cell layers per axis (n, or n+2 on a wall axis, reading U8)
  int mb[3];       // bricks per axis
  int B[3];        // brick dims
  float a, inv_a;
  int nbar;        // round(n_per_cell): target occupancy of wall-cut cells
  Params p;
  uint64_t seed;
  uint32_t t;
  double cosa, sina;
  size_t nkeys;
  std::vector<float> x, y, z, vx, vy, vz;
  std::vector<uint32_t> id;
  bool have_state = false, have_cells = false;
  // bookkeeping of the last executed step (pre-collision, real particles only)
  std::vector<uint32_t> key;               // per particle, current order
  std::vector<float> rho[3];               // cell-local coordinate per particle (U9)
  std::vector<uint32_t> count;             // per key
  std::vector<double> sx, sy, sz, se;      // per key: sum v, sum |v|^2
  unsigned long long n_singular = 0;
  float last_shift[3] = {0, 0, 0};
  std::vector<signed char> img;            // Lees-Edwards: -1 / +1 if the particle collides as its image below / above (U21)
  std::string err;
};

// ---- Philox-4x32-10 (Salmon et al., SC'11); stream layout DESIGN.md "RNG" -----------------
inline void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    const uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += W0; k1 += W1;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

inline void draw(const Ctx& c, uint32_t index, uint32_t sub, uint32_t t, uint32_t tag, uint32_t out[4]) {
  const uint32_t ctr[4] = {index, sub, t, tag};
  const uint32_t key[2] = {(uint32_t)(c.seed & 0xffffffffu), (uint32_t)(c.seed >> 32)};
  philox4x32_10(ctr, key, out);
}

// uniform in [0,1) and in (0,1] from the top 24 bits; both exact in fp32 and in double
inline double u_co(uint32_t o) { return (double)(o >> 8) * (1.0 / 16777216.0); }
inline double u_oc(uint32_t o) { return (double)((o >> 8) + 1u) * (1.0 / 16777216.0); }

const double TWO_PI = 6.283185307179586476925286766559;

// Box-Muller on one Philox block: (o0,o1) -> n0,n1 ; (o2,o3) -> n2,n3 (n3 unused by callers)
inline void normals4(const uint32_t o[4], double nrm[4]) {
  const double r0 = std::sqrt(-2.0 * std::log(u_oc(o[0]))), a0 = TWO_PI * u_co(o[1]);
  const double r1 = std::sqrt(-2.0 * std::log(u_oc(o[2]))), a1 = TWO_PI * u_co(o[3]);
  nrm[0] = r0 * std::cos(a0); nrm[1] = r0 * std::sin(a0);
  nrm[2] = r1 * std::cos(a1); nrm[3] = r1 * std::sin(a1);
}

// ---- grid shift (reading U12): one draw per step, s_d in [-a/2, a/2) ---------
inline void grid_shift(const Ctx& c, uint32_t t, float s[3]) {
  s[0] = s[1] = s[2] = 0.0f;
  if (!c.p.grid_shift) return;
  uint32_t o[4];
  draw(c, 0u, 0u, t, TAG_SHIFT, o);
  for (int d = 0; d < 3; ++d) {
    const float u = (float)(o[d] >> 8) * 5.9604644775390625e-08f;  // 2^-24, exact
    s[d] = (u - 0.5f) * c.a;
  }
}

// ---- cell index of a position (readings U1,U3,U8) -------------------------
inline void cell_of(const Ctx& c, const float r[3], const float s[3], int i[3], float rho[3]) {
  for (int d = 0; d < 3; ++d) {
    const float q = (r[d] + s[d]) * c.inv_a;   // one fp32 add, one fp32 multiply
    const float f = floorf(q);
    int k = (int)f;
    if (c.p.bc[d] == 0) {
      if (k < 0) k += c.n[d];
      if (k >= c.n[d]) k -= c.n[d];
    } else {
      k += 1;                                   // layers 0 .. n+1, walls cut one layer each side
      if (k < 0) k = 0;
      if (k > c.n[d] + 1) k = c.n[d] + 1;
    }
    i[d] = k;
    rho[d] = q - f;
  }
}
// ---- Lees-Edwards sheared periodic boundary along z, flow along x (reading U21) ----------
// The periodic images of the box above / below are displaced by +-D(t) along x and move with +-U = +-gamma L_z.
// D is taken at the time the positions refer to: (t+1) h for the wrap after MOVE of step t and for its collision.
inline float le_velocity(const Ctx& c) { return (float)((double)c.p.shear_rate * (double)c.L[2]); }
inline float le_offset(const Ctx& c, uint32_t t) {
  const double Ud = (double)c.p.shear_rate * (double)c.L[2];
  double d = std::fmod(Ud * (double)c.p.dt * ((double)t + 1.0), (double)c.L[0]);
  if (d < 0.0) d += (double)c.L[0];
  return (float)d;
}
// cell of a position under Lees-Edwards: a particle whose shifted z leaves [0, L_z) collides as its periodic image:
// x -+ D (wrapped once), v_x -+ U. image = -1: image below the box top was used (particle above), +1: the reverse.
inline void cell_of_le(const Ctx& c, uint32_t t, const float r[3], const float s[3], int i[3], float rho[3], int* image) {
  float rr[3] = {r[0], r[1], r[2]};
  int im = 0;
  if (c.p.shear_rate != 0.0f) {
    const float qz = (r[2] + s[2]) * c.inv_a;
    const int kz = (int)floorf(qz);
    const float D = le_offset(c, t);
    if (kz < 0) { im = +1; rr[0] = r[0] + D; if (rr[0] >= c.L[0]) rr[0] -= c.L[0]; }
    else if (kz >= c.n[2]) { im = -1; rr[0] = r[0] - D; if (rr[0] < 0.0f) rr[0] += c.L[0]; }
  }
  cell_of(c, rr, s, i, rho);
  if (image) *image = im;
}
inline uint32_t canonical_id(const Ctx& c, const int i[3]) {
  return (uint32_t)i[0] + (uint32_t)c.m[0] * ((uint32_t)i[1] + (uint32_t)c.m[1] * (uint32_t)i[2]);
}
// memory-order key: brick-major over Bx*By*Bz bricks (B = {1,1,1}: identical to canonical_id)
inline uint32_t layout_key(const Ctx& c, const int i[3]) {
  const uint32_t bx = i[0] / c.B[0], by = i[1] / c.B[1], bz = i[2] / c.B[2];
  const uint32_t lx = i[0] % c.B[0], ly = i[1] % c.B[1], lz = i[2] % c.B[2];
  const uint32_t brick = (bz * (uint32_t)c.mb[1] + by) * (uint32_t)c.mb[0] + bx;
  return brick * (uint32_t)(c.B[0] * c.B[1] * c.B[2]) + (lz * c.B[1] + ly) * c.B[0] + lx;
}
inline void key_to_cell(const Ctx& c, uint32_t key, int i[3]) {
  const uint32_t B3 = c.B[0] * c.B[1] * c.B[2];
  const uint32_t brick = key / B3, l = key % B3;
  const uint32_t lx = l % c.B[0], ly = (l / c.B[0]) % c.B[1], lz = l / (c.B[0] * c.B[1]);
  const uint32_t bx = brick % c.mb[0], by = (brick / c.mb[0]) % c.mb[1], bz = brick / (c.mb[0] * c.mb[1]);
  i[0] = bx * c.B[0] + lx; i[1] = by * c.B[1] + ly; i[2] = bz * c.B[2] + lz;
}

// ---- streaming, Eq. (1) + gravity + bounce-back (U7)
inline void advance(const Ctx& c, float r[3], float v[3], float tau) {
  for (int d = 0; d < 3; ++d) {
    const float g = c.p.g[d];
    if (g != 0.0f) {
      const float vh = fmaf(0.5f * tau, g, v[d]);
      r[d] = fmaf(vh, tau, r[d]);
      v[d] = fmaf(tau, g, v[d]);
    } else {
      r[d] = fmaf(v[d], tau, r[d]);
    }
  }
}
inline void stream_one(const Ctx& c, float r[3], float v[3], uint32_t t) {
  const float h = c.p.dt;
  int w = -1;
  for (int d = 0; d < 3; ++d) if (c.p.bc[d] != 0) w = d;   // at most one wall axis (create checks)
  bool bounced = false;
  if (w >= 0) {
    const float z1 = fmaf(v[w], h, r[w]);
    if (z1 < 0.0f || z1 > c.L[w]) {
      const float zw = (z1 < 0.0f) ? 0.0f : c.L[w];
      float tc = (zw - r[w]) / v[w];
      if (tc < 0.0f) tc = 0.0f;
      if (tc > h) tc = h;
      advance(c, r, v, tc);
      r[w] = zw;
      if (c.p.bc[w] == 1) {                                                // no-slip, bounce-back: v -> -v in the frame of the wall
        v[0] = -v[0]; v[1] = -v[1]; v[2] = -v[2];
        if (c.p.wall_velocity != 0.0f) {                                   // moving wall (reading U24): v -> 2 u_wall - v
          const float uw = (z1 < 0.0f) ? -c.p.wall_velocity : c.p.wall_velocity;
          v[0] = fmaf(2.0f, uw, v[0]);
        }
      }
      else v[w] = -v[w];                                                   // slip, specular reflection
      const float tr = h - tc;
      advance(c, r, v, tr);
      if (r[w] < 0.0f) r[w] = 0.0f;
      if (r[w] > c.L[w]) r[w] = c.L[w];
      bounced = true;
    }
  }
  if (!bounced) advance(c, r, v, h);
  for (int d = 0; d < 3; ++d) {
    if (c.p.bc[d] != 0) continue;
    if (d == 2 && c.p.shear_rate != 0.0f) {                 // Lees-Edwards: crossing z = 0 / L_z enters the sheared image (U21)
      const float D = le_offset(c, t), U = le_velocity(c);
      if (r[2] < 0.0f) { r[2] += c.L[2]; r[0] += D; if (r[0] >= c.L[0]) r[0] -= c.L[0]; v[0] += U; }
      if (r[2] >= c.L[2]) { r[2] -= c.L[2]; r[0] -= D; if (r[0] < 0.0f) r[0] += c.L[0]; v[0] -= U; }
      continue;
    }
    if (r[d] < 0.0f) r[d] += c.L[d];                        // reading U2: this order, single wrap
    if (r[d] >= c.L[d]) r[d] -= c.L[d];
  }
}

// ---- random rotation axis, uniform on the unit sphere (reading U11) -----------
inline void srd_axis(const Ctx& c, uint32_t cid, uint32_t t, double n[3]) {
  uint32_t o[4];
  draw(c, cid, 0u, t, TAG_AXIS, o);
  const double zz = 2.0 * u_co(o[0]) - 1.0, phi = TWO_PI * u_co(o[1]);
  const double rr = std::sqrt((1.0 - zz) * (1.0 + zz));
  n[0] = rr * std::cos(phi); n[1] = rr * std::sin(phi); n[2] = zz;
}
// Rodrigues rotation of w by +alpha (right-handed) about unit axis n: D(alpha) w of Eq. (2)
inline void rotate(const double n[3], double ca, double sa, const double w[3], double out[3]) {
  const double nd = n[0] * w[0] + n[1] * w[1] + n[2] * w[2];
  const double cx = n[1] * w[2] - n[2] * w[1], cy = n[2] * w[0] - n[0] * w[2], cz = n[0] * w[1] - n[1] * w[0];
  out[0] = w[0] * ca + cx * sa + n[0] * nd * (1.0 - ca);
  out[1] = w[1] * ca + cy * sa + n[1] * nd * (1.0 - ca);
  out[2] = w[2] * ca + cz * sa + n[2] * nd * (1.0 - ca);
}

// ---- E_k / k_BT ~ Gamma(f/2, 1), f = 3(N_c-1): Eq. (7), sampler reading U6 ----------------------
// The paper gives only the density. Reading U6: the rejection sampler of Marsaglia & Tsang (ACM TOMS 26,
// 2000) for Gamma(a), a = f/2 >= 3/2: d = a - 1/3, c = 1/sqrt(9 d); draw x ~ N(0,1), U ~ U(0,1]; v = (1 + c x)^3;
// accept if v > 0 and ( U < 1 - k x^4  or  ln U < x^2/2 + d (1 - v + ln v) ); E_k / k_BT = d v (k: below).
// An accept/reject decision is an integer decided by floating point: both codes take it in the SAME arithmetic, fixed
// here operation by operation in IEEE binary32 (every operation rounded once, fmaf where written, no contraction;
// -ffp-contract=off), with the logarithm and the cosine defined by the short series below instead of libm, whose
// last bit differs between implementations. The sampler is exact up to those series' truncation (< 3e-9) and fp32
// rounding, far below the statistical meaning of one draw. Constants are the binary32 numbers nearest to the
// stated fractions, written as hexadecimal floats.
// Random words: attempt 0 takes the cell's TAG_AXIS block of the step (whose top 24 bits of words 0, 1 give the rotation
// axis): radius uniform = top 24 bits of word 2, angle = top 24 bits of word 3, acceptance uniform = the low bytes
// of words 0, 1, 2 (bits the other draws do not use); attempt j >= 1 takes words 0, 1, 2 (top 24 bits) of block j - 1
// of the cell's TAG_MBS stream. After 16 rejections (probability < 1e-20) E_k / k_BT = d.
namespace mt {
inline uint32_t f2u(float x) { uint32_t u; std::memcpy(&u, &x, 4); return u; }
inline float u2f(uint32_t u) { float x; std::memcpy(&x, &u, 4); return x; }
// ln x for a positive normal float: x = m 2^e with m in [sqrt(1/2), sqrt(2)); ln m = 2 atanh(s), s = (m-1)/(m+1),
// atanh series up to s^9 (|s| <= 0.1716: the first dropped term is 2 s^11 / 11 < 7e-10)
inline float rlog(float x) {
  const int32_t i = (int32_t)f2u(x);
  const int32_t e = (i - 0x3f3504f3) >> 23;                       // 0x3f3504f3 = bits of sqrt(1/2), arithmetic shift
  const float m = u2f((uint32_t)(i - e * 8388608));               // in [sqrt(1/2), sqrt(2))
  const float f = m - 1.0f;                                       // exact
  const float s = f / (2.0f + f);
  const float z = s * s;
  float p = std::fmaf(z, 0x1.c71c72p-3f, 0x1.24924ap-2f);             // 2/9, 2/7
  p = std::fmaf(z, p, 0x1.99999ap-2f);                              // 2/5
  p = std::fmaf(z, p, 0x1.555556p-1f);                              // 2/3
  p = std::fmaf(z, p, 2.0f);
  return std::fmaf((float)e, 0x1.62e43p-1f /* ln 2 */, s * p);
}
// cos(2 pi k / 2^24) for a 24-bit integer k: the angle is split exactly (integers) into a quarter turn q and
// y in [-pi/4, pi/4); Taylor series of sin and cos up to y^9 / y^10 (first dropped terms < 2e-9)
inline float rcos(uint32_t k) {
  const uint32_t kk = k + 2097152u;                               // + 1/8 turn
  const uint32_t q = (kk >> 22) & 3u;
  const int32_t r = (int32_t)(kk & 4194303u) - 2097152;           // in [-2^21, 2^21)
  const float y = (float)r * 0x1.921fb6p-22f;                     // (pi/2) / 2^22
  const float z = y * y;
  float sp = std::fmaf(z, 0x1.71de3ap-19f, -0x1.a01a02p-13f);     // 1/9!, -1/7!
  sp = std::fmaf(z, sp, 0x1.111112p-7f);                         // 1/5!
  sp = std::fmaf(z, sp, -0x1.555556p-3f);                        // -1/3!
  const float sn = std::fmaf(y * z, sp, y);
  float cp = std::fmaf(z, -0x1.27e4fcp-22f, 0x1.a01a02p-16f);     // -1/10!, 1/8!
  cp = std::fmaf(z, cp, -0x1.6c16c2p-10f);                        // -1/6!
  cp = std::fmaf(z, cp, 0x1.555556p-5f);                         // 1/4!
  const float cs = std::fmaf(z * z, cp, std::fmaf(-0.5f, z, 1.0f));
  return (q == 0u) ? cs : (q == 1u) ? -sn : (q == 2u) ? -cs : sn;
}
}  // namespace mt

inline double mbs_energy_over_kT(const Ctx& c, uint32_t cid, uint32_t t, unsigned Nc) {
  if (Nc < 2) return 0.0;
  const float a = 1.5f * (float)(Nc - 1u);
  const float d = a - 0x1.555556p-2f /* 1/3 */;
  const float cc = 1.0f / std::sqrt(9.0f * d);
  // squeeze U < 1 - k x^4: valid whenever k >= -g(x) / x^4 for every reachable x (|x| <= sqrt(48 ln 2) = 5.77 from a
  // 24-bit uniform), g(x) = x^2/2 + d (1 - v + ln v), because exp(g) >= 1 + g. Marsaglia and Tsang's k = 0.0331 holds for
  // every a >= 1; for N_c >= 7 the bound k = (0.0093 + 0.0145 / sqrt(d) + 0.06 / d) / d is 4..30 times tighter (the series
  // of g starts with -x^4 / (108 d) + x^5 / (405 d^1.5)); checked numerically in tests/test_oracle_collision.py
  const float kq = (Nc < 7u) ? 0x1.0f27bcp-5f /* 0.0331 */
                             : (0x1.30be0ep-7f /* 0.0093 */ + 0x1.db22d0p-7f /* 0.0145 */ / std::sqrt(d) + 0x1.eb851ep-5f /* 0.06 */ / d) / d;
  for (unsigned j = 0; j < 16u; ++j) {
    uint32_t o[4], wr, wa, wu;
    if (j == 0u) {
      draw(c, cid, 0u, t, TAG_AXIS, o);
      wr = o[2] >> 8; wa = o[3] >> 8;
      wu = ((o[0] & 0xffu) << 16) | ((o[1] & 0xffu) << 8) | (o[2] & 0xffu);
    } else {
      draw(c, cid, j - 1u, t, TAG_MBS, o);
      wr = o[0] >> 8; wa = o[1] >> 8; wu = o[2] >> 8;
    }
    const float Ur = (float)(wr + 1u) * 0x1p-24f;   // (0, 1], exact
    const float U = (float)(wu + 1u) * 0x1p-24f;
    const float x = std::sqrt(-2.0f * mt::rlog(Ur)) * mt::rcos(wa);
    const float v0 = std::fmaf(cc, x, 1.0f);
    if (!(v0 > 0x1p-20f)) continue;                    // v0 <= 2^-20, v <= 2^-60: never accepted by a 24-bit U
    const float v = (v0 * v0) * v0;
    const float x2 = x * x;
    bool ok = U < std::fmaf(-(kq * x2), x2, 1.0f);
    if (!ok) ok = mt::rlog(U) < std::fmaf(0.5f, x2, d * ((1.0f - v) + mt::rlog(v)));
    if (ok) return (double)(d * v);
  }
  return (double)d;
}

// 3x3 symmetric solve for omega = I^-1 dL with the degenerate-cell rules of reading U10
inline bool solve_inertia(const double I[6] /*xx,yy,zz,xy,xz,yz*/, const double dL[3], double w[3]) {
  const double xx = I[0], yy = I[1], zz = I[2], xy = I[3], xz = I[4], yz = I[5];
  const double c00 = yy * zz - yz * yz, c01 = xz * yz - xy * zz, c02 = xy * yz - xz * yy;
  const double c11 = xx * zz - xz * xz, c12 = xy * xz - xx * yz, c22 = xx * yy - xy * xy;
  const double det = xx * c00 + xy * c01 + xz * c02;
  const double tr3 = (xx + yy + zz) / 3.0;
  if (!(det > 1e-6 * tr3 * tr3 * tr3)) { w[0] = w[1] = w[2] = 0.0; return false; }
  w[0] = (c00 * dL[0] + c01 * dL[1] + c02 * dL[2]) / det;
  w[1] = (c01 * dL[0] + c11 * dL[1] + c12 * dL[2]) / det;
  w[2] = (c02 * dL[0] + c12 * dL[1] + c22 * dL[2]) / det;
  return true;
}

// ---- collision of ONE cell -------------------------------------------------------------------
// idx[0..n) = particle indices of the cell in ascending-id order (rank = position, U4/U5).
// ---- explicit phantom particles of a wall-cut cell (reading U22) ----------------------------
// "The part of these collision cells in walls ... are filled with uniformly distributed phantom particles, which are
// identical to MPC particles, such that the whole collision cell contains the same average number <N_c>", "created in
// the subdomain where they are to be processed while random shifts are taken into account". With sigma+ = the
// fractional part of s_w / a in (0,1): the wall occupies the cell-local range [0, sigma+) of the cut layer at the
// wall at 0 and [sigma+, 1) of the cut layer at the wall at L. Number of phantoms of a cut cell: the wall volume
// fraction phi times <N_c>, rounded stochastically (fp32: floorf(fmaf(nbar, phi, u))), positions uniform in the
// wall part, velocities Gaussian about the wall velocity.
struct Phantom { double rho[3], v[3]; };
inline float wall_fraction(const Ctx& c, int w, const int icell[3], const float s[3], bool* top) {
  if (c.p.bc[w] != 1 || s[w] == 0.0f) return 0.0f;
  const float sg = s[w] * c.inv_a;
  const float sp = (sg > 0.0f) ? sg : 1.0f + sg;
  const int lo = (s[w] > 0.0f) ? 1 : 0, hi = (s[w] > 0.0f) ? c.n[w] + 1 : c.n[w];
  if (icell[w] == lo) { *top = false; return sp; }
  if (icell[w] == hi) { *top = true; return 1.0f - sp; }
  return 0.0f;
}
void make_phantoms(const Ctx& c, uint32_t cid, const int icell[3], const float s[3], uint32_t t, std::vector<Phantom>& ph) {
  ph.clear();
  if (!c.p.phantoms) return;
  int w = -1;
  for (int d = 0; d < 3; ++d) if (c.p.bc[d] == 1) w = d;
  if (w < 0) return;
  bool top = false;
  const float phi = wall_fraction(c, w, icell, s, &top);
  if (!(phi > 0.0f)) return;
  uint32_t o[4];
  draw(c, cid, 0u, t, TAG_PHANTOM, o);
  const float u = (float)(o[0] >> 8) * 5.9604644775390625e-08f;
  const int nph = (int)floorf(fmaf((float)c.nbar, phi, u));
  const float sg = s[w] * c.inv_a, sp = (sg > 0.0f) ? sg : 1.0f + sg;
  const double sig = std::sqrt((double)c.p.kT / (double)c.p.mass);
  const double uw = (c.p.wall_velocity != 0.0f) ? (top ? (double)c.p.wall_velocity : -(double)c.p.wall_velocity) : 0.0;
  for (int k = 0; k < nph; ++k) {
    Phantom q;
    uint32_t P[4], V[4]; double g[4];
    draw(c, cid, 1u + 2u * (uint32_t)k, t, TAG_PHANTOM, P);
    draw(c, cid, 2u + 2u * (uint32_t)k, t, TAG_PHANTOM, V);
    const float ua = (float)(P[0] >> 8) * 5.9604644775390625e-08f, ub = (float)(P[1] >> 8) * 5.9604644775390625e-08f;
    const float zeta = (float)(P[2] >> 8) * 5.9604644775390625e-08f;
    const float rw = top ? fmaf(zeta, phi, sp) : zeta * phi;
    int e = 0;
    for (int d = 0; d < 3; ++d) q.rho[d] = (d == w) ? (double)rw : (double)((e++ == 0) ? ua : ub);
    normals4(V, g);
    for (int d = 0; d < 3; ++d) q.v[d] = sig * g[d] + (d == 0 ? uw : 0.0);
    ph.push_back(q);
  }
}

inline double particle_mass(const Ctx& c, uint32_t id) {
  return (c.p.solute_mass > 0.0f && id >= c.p.solute_id0) ? (double)c.p.solute_mass : (double)c.p.mass;
}

// ---- collision of ONE cell with particle masses (embedded solutes, reading U23) and explicit phantoms (U22) ----
// The same equations with every sum weighted by the particle mass: v_cm = sum m_i v_i / sum m_i,
// Eq. (2), Eqs. (3)-(4) with I = sum m_i (r^2 1 - r r^T) and r_cm mass-weighted, Eq. (6) with sum m_i v_ic^2 and
// f = 3 (N_c - 1); MPC-AT: v_ran,i ~ N(0, kT / m_i), v' = v_cm + v_ran,i - sum m_j v_ran,j / sum m_j (U5).
// Members = the real particles (ascending id) followed by the phantoms; phantoms are discarded afterwards.
void collide_cell_ext(Ctx& c, uint32_t cid, const int icell[3], const float s[3], uint32_t t,
                      const uint32_t* idx, unsigned n, const double* forced_axis, const double* forced_kappa) {
  std::vector<Phantom> ph;
  make_phantoms(c, cid, icell, s, t, ph);
  const unsigned N = n + (unsigned)ph.size();
  struct Mem { double m, v[3], rho[3]; };
  std::vector<Mem> mem(N);
  for (unsigned k = 0; k < n; ++k) {
    const uint32_t i = idx[k];
    mem[k].m = particle_mass(c, c.id[i]);
    mem[k].v[0] = c.vx[i]; mem[k].v[1] = c.vy[i]; mem[k].v[2] = c.vz[i];
    for (int d = 0; d < 3; ++d) mem[k].rho[d] = c.rho[d][i];
  }
  for (unsigned k = n; k < N; ++k) {
    mem[k].m = c.p.mass;
    for (int d = 0; d < 3; ++d) { mem[k].v[d] = ph[k - n].v[d]; mem[k].rho[d] = ph[k - n].rho[d]; }
  }
  if (N < 2) return;                                           // a lone particle keeps its velocity
  double Ms = 0.0, S[3] = {0, 0, 0};
  for (unsigned k = 0; k < N; ++k) { Ms += mem[k].m; for (int d = 0; d < 3; ++d) S[d] += mem[k].m * mem[k].v[d]; }
  const double vcm[3] = {S[0] / Ms, S[1] / Ms, S[2] / Ms};
  // velocity of every member after the collision rule without the +a term, relative to v_cm
  std::vector<double> vnew(3 * (size_t)N);
  double kappa = 1.0;
  if (c.p.collision == 0) {
    double axis[3];
    if (forced_axis) { axis[0] = forced_axis[0]; axis[1] = forced_axis[1]; axis[2] = forced_axis[2]; }
    else srd_axis(c, cid, t, axis);
    if (forced_kappa) kappa = *forced_kappa;
    else if (c.p.thermostat) {
      double W2 = 0.0;                                          // sum m_i |v_i - v_cm|^2 (Eq. 6)
      for (unsigned k = 0; k < N; ++k) for (int d = 0; d < 3; ++d) { const double w = mem[k].v[d] - vcm[d]; W2 += mem[k].m * w * w; }
      if (W2 > 0.0) kappa = std::sqrt(2.0 * (double)c.p.kT * mbs_energy_over_kT(c, cid, t, N) / W2);
    }
    for (unsigned k = 0; k < N; ++k) {
      const double w[3] = {mem[k].v[0] - vcm[0], mem[k].v[1] - vcm[1], mem[k].v[2] - vcm[2]};
      rotate(axis, c.cosa, c.sina, w, &vnew[3 * k]);
    }
  } else {
    double R[3] = {0, 0, 0};
    for (unsigned k = 0; k < N; ++k) {
      uint32_t o[4]; double g[4];
      draw(c, cid, k, t, TAG_AT, o);                            // k = rank among the members
      normals4(o, g);
      const double sg = std::sqrt((double)c.p.kT / mem[k].m);
      for (int d = 0; d < 3; ++d) { vnew[3 * k + d] = sg * g[d]; R[d] += mem[k].m * vnew[3 * k + d]; }
    }
    for (unsigned k = 0; k < N; ++k) for (int d = 0; d < 3; ++d) vnew[3 * k + d] -= R[d] / Ms;
  }
  double om[3] = {0, 0, 0};
  std::vector<double> rc;
  if (c.p.conserve_L) {
    double rcm[3] = {0, 0, 0};
    for (unsigned k = 0; k < N; ++k) for (int d = 0; d < 3; ++d) rcm[d] += mem[k].m * mem[k].rho[d];
    for (int d = 0; d < 3; ++d) rcm[d] /= Ms;
    rc.resize(3 * (size_t)N);
    double I[6] = {0, 0, 0, 0, 0, 0}, dL[3] = {0, 0, 0}, R2 = 0.0;
    for (unsigned k = 0; k < N; ++k) {
      double* r = &rc[3 * k];
      const double m = mem[k].m;
      for (int d = 0; d < 3; ++d) r[d] = (mem[k].rho[d] - rcm[d]) * (double)c.a;
      // change of the relative velocity by the collision rule without +a: (v - v_cm) - v_new
      const double dv[3] = {mem[k].v[0] - vcm[0] - vnew[3 * k], mem[k].v[1] - vcm[1] - vnew[3 * k + 1], mem[k].v[2] - vcm[2] - vnew[3 * k + 2]};
      dL[0] += m * (r[1] * dv[2] - r[2] * dv[1]);
      dL[1] += m * (r[2] * dv[0] - r[0] * dv[2]);
      dL[2] += m * (r[0] * dv[1] - r[1] * dv[0]);
      const double r2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
      R2 += m * r2;
      I[0] += m * (r2 - r[0] * r[0]); I[1] += m * (r2 - r[1] * r[1]); I[2] += m * (r2 - r[2] * r[2]);
      I[3] -= m * r[0] * r[1]; I[4] -= m * r[0] * r[2]; I[5] -= m * r[1] * r[2];
    }
    if (N == 2) {
      if (R2 > 0.0) for (int d = 0; d < 3; ++d) om[d] = dL[d] / R2;
    } else if (!solve_inertia(I, dL, om)) c.n_singular++;
  }
  for (unsigned k = 0; k < n; ++k) {                            // phantoms are discarded
    const uint32_t i = idx[k];
    double o3[3] = {vcm[0] + kappa * vnew[3 * k], vcm[1] + kappa * vnew[3 * k + 1], vcm[2] + kappa * vnew[3 * k + 2]};
    if (!rc.empty()) {
      const double* r = &rc[3 * k];
      o3[0] += om[1] * r[2] - om[2] * r[1];
      o3[1] += om[2] * r[0] - om[0] * r[2];
      o3[2] += om[0] * r[1] - om[1] * r[0];
    }
    c.vx[i] = (float)o3[0]; c.vy[i] = (float)o3[1]; c.vz[i] = (float)o3[2];
  }
}

void collide_cell(Ctx& c, uint32_t cid, const int icell[3], const float s[3], uint32_t t,
                  const uint32_t* idx, unsigned n, const double* forced_axis, const double* forced_kappa) {
  if (n == 0) return;
  if (c.p.phantoms || c.p.solute_mass > 0.0f) { collide_cell_ext(c, cid, icell, s, t, idx, n, forced_axis, forced_kappa); return; }
  const double m = c.p.mass, sig = std::sqrt((double)c.p.kT / (double)c.p.mass);
  // PROCESS: cell sums over real particles
  double S[3] = {0, 0, 0};
  for (unsigned k = 0; k < n; ++k) { const uint32_t i = idx[k]; S[0] += c.vx[i]; S[1] += c.vy[i]; S[2] += c.vz[i]; }
  unsigned Nc = n;
  // virtual wall particles in wall-cut layers (reading U8)
  std::vector<double> virt;   // 3 per virtual particle
  for (int d = 0; d < 3; ++d) {
    if (c.p.bc[d] != 1 || s[d] == 0.0f) continue;
    const bool cut = (s[d] > 0.0f) ? (icell[d] == 1 || icell[d] == c.n[d] + 1) : (icell[d] == 0 || icell[d] == c.n[d]);
    if (cut && (int)n < c.nbar) {
      const unsigned nv = (unsigned)c.nbar - n;
      for (unsigned k = 0; k < nv; ++k) {
        uint32_t o[4]; double g[4];
        draw(c, cid, k, t, TAG_WALL, o);
        normals4(o, g);
        // virtual particles of a moving wall are thermal about the wall velocity (reading U24)
        const double uw = (c.p.wall_velocity != 0.0f) ? ((icell[d] <= 1) ? -(double)c.p.wall_velocity : (double)c.p.wall_velocity) : 0.0;
        for (int e = 0; e < 3; ++e) { const double ve = sig * g[e] + (e == 0 ? uw : 0.0); virt.push_back(ve); S[e] += ve; }
      }
      Nc += nv;
    }
  }
  const double vcm[3] = {S[0] / Nc, S[1] / Nc, S[2] / Nc};

  if (c.p.collision == 0) {
    // ---------------- SRD: Eq. (2), optionally Eq. (3)-(4) and Eq. (5)-(7) -------------------
    double axis[3];
    if (forced_axis) { axis[0] = forced_axis[0]; axis[1] = forced_axis[1]; axis[2] = forced_axis[2]; }
    else srd_axis(c, cid, t, axis);
    double kappa = 1.0;
    if (forced_kappa) kappa = *forced_kappa;
    else if (c.p.thermostat && Nc >= 2) {
      double W2 = 0.0;   // sum over the cell of |v - v_cm|^2, before rotation
      for (unsigned k = 0; k < n; ++k) {
        const uint32_t i = idx[k];
        const double w0 = c.vx[i] - vcm[0], w1 = c.vy[i] - vcm[1], w2 = c.vz[i] - vcm[2];
        W2 += w0 * w0 + w1 * w1 + w2 * w2;
      }
      for (size_t k = 0; k < virt.size(); k += 3) {
        const double w0 = virt[k] - vcm[0], w1 = virt[k + 1] - vcm[1], w2 = virt[k + 2] - vcm[2];
        W2 += w0 * w0 + w1 * w1 + w2 * w2;
      }
      if (W2 > 0.0) {
        const double Ek = (double)c.p.kT * mbs_energy_over_kT(c, cid, t, Nc);
        kappa = std::sqrt(2.0 * Ek / (m * W2));                       // Eq. (6)
      }
    }
    std::vector<double> wrot(3 * (size_t)n);
    for (unsigned k = 0; k < n; ++k) {
      const uint32_t i = idx[k];
      const double w[3] = {c.vx[i] - vcm[0], c.vy[i] - vcm[1], c.vz[i] - vcm[2]};
      rotate(axis, c.cosa, c.sina, w, &wrot[3 * k]);
    }
    double om[3] = {0, 0, 0};
    std::vector<double> rc;
    if (c.p.conserve_L && n >= 2) {
      // Eq. (4): omega = m I^-1 sum r_ic x (v_ic - D v_ic); r_ic from cell-local coordinates (U9)
      double rcm[3] = {0, 0, 0};
      for (unsigned k = 0; k < n; ++k) for (int d = 0; d < 3; ++d) rcm[d] += c.rho[d][idx[k]];
      for (int d = 0; d < 3; ++d) rcm[d] /= n;
      rc.resize(3 * (size_t)n);
      double I[6] = {0, 0, 0, 0, 0, 0}, dL[3] = {0, 0, 0}, R2 = 0.0;
      for (unsigned k = 0; k < n; ++k) {
        const uint32_t i = idx[k];
        double* r = &rc[3 * k];
        for (int d = 0; d < 3; ++d) r[d] = ((double)c.rho[d][i] - rcm[d]) * (double)c.a;
        const double w[3] = {c.vx[i] - vcm[0], c.vy[i] - vcm[1], c.vz[i] - vcm[2]};
        const double dv[3] = {w[0] - wrot[3 * k], w[1] - wrot[3 * k + 1], w[2] - wrot[3 * k + 2]};
        dL[0] += m * (r[1] * dv[2] - r[2] * dv[1]);
        dL[1] += m * (r[2] * dv[0] - r[0] * dv[2]);
        dL[2] += m * (r[0] * dv[1] - r[1] * dv[0]);
        const double r2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
        R2 += r2;
        I[0] += m * (r2 - r[0] * r[0]); I[1] += m * (r2 - r[1] * r[1]); I[2] += m * (r2 - r[2] * r[2]);
        I[3] -= m * r[0] * r[1]; I[4] -= m * r[0] * r[2]; I[5] -= m * r[1] * r[2];
      }
      if (n == 2) {
        if (R2 > 0.0) for (int d = 0; d < 3; ++d) om[d] = dL[d] / (m * R2);
      } else if (!solve_inertia(I, dL, om)) c.n_singular++;
    }
    for (unsigned k = 0; k < n; ++k) {
      const uint32_t i = idx[k];
      double o3[3] = {vcm[0] + kappa * wrot[3 * k], vcm[1] + kappa * wrot[3 * k + 1], vcm[2] + kappa * wrot[3 * k + 2]};
      if (!rc.empty()) {
        const double* r = &rc[3 * k];
        o3[0] += om[1] * r[2] - om[2] * r[1];
        o3[1] += om[2] * r[0] - om[0] * r[2];
        o3[2] += om[0] * r[1] - om[1] * r[0];
      }
      c.vx[i] = (float)o3[0]; c.vy[i] = (float)o3[1]; c.vz[i] = (float)o3[2];
    }
  } else {
    // ---------------- MPC-AT (reading U5; refs [67],[70] of the paper) ----------------------
    std::vector<double> vr(3 * (size_t)n);
    double R[3] = {0, 0, 0};
    for (unsigned k = 0; k < n; ++k) {
      uint32_t o[4]; double g[4];
      draw(c, cid, k, t, TAG_AT, o);          // k = rank of the particle in (key,id) order
      normals4(o, g);
      for (int d = 0; d < 3; ++d) { vr[3 * k + d] = sig * g[d]; R[d] += vr[3 * k + d]; }
    }
    for (int d = 0; d < 3; ++d) R[d] /= n;
    double om[3] = {0, 0, 0};
    std::vector<double> rc;
    if (c.p.conserve_L && n >= 2) {
      double rcm[3] = {0, 0, 0};
      for (unsigned k = 0; k < n; ++k) for (int d = 0; d < 3; ++d) rcm[d] += c.rho[d][idx[k]];
      for (int d = 0; d < 3; ++d) rcm[d] /= n;
      rc.resize(3 * (size_t)n);
      double I[6] = {0, 0, 0, 0, 0, 0}, dL[3] = {0, 0, 0}, R2 = 0.0;
      for (unsigned k = 0; k < n; ++k) {
        const uint32_t i = idx[k];
        double* r = &rc[3 * k];
        for (int d = 0; d < 3; ++d) r[d] = ((double)c.rho[d][i] - rcm[d]) * (double)c.a;
        const double dv[3] = {c.vx[i] - vr[3 * k], c.vy[i] - vr[3 * k + 1], c.vz[i] - vr[3 * k + 2]};
        dL[0] += m * (r[1] * dv[2] - r[2] * dv[1]);
        dL[1] += m * (r[2] * dv[0] - r[0] * dv[2]);
        dL[2] += m * (r[0] * dv[1] - r[1] * dv[0]);
        const double r2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
        R2 += r2;
        I[0] += m * (r2 - r[0] * r[0]); I[1] += m * (r2 - r[1] * r[1]); I[2] += m * (r2 - r[2] * r[2]);
        I[3] -= m * r[0] * r[1]; I[4] -= m * r[0] * r[2]; I[5] -= m * r[1] * r[2];
      }
      if (n == 2) {
        if (R2 > 0.0) for (int d = 0; d < 3; ++d) om[d] = dL[d] / (m * R2);
      } else if (!solve_inertia(I, dL, om)) c.n_singular++;
    }
    for (unsigned k = 0; k < n; ++k) {
      const uint32_t i = idx[k];
      double o3[3] = {vcm[0] + vr[3 * k] - R[0], vcm[1] + vr[3 * k + 1] - R[1], vcm[2] + vr[3 * k + 2] - R[2]};
      if (n == 1) { o3[0] = c.vx[i]; o3[1] = c.vy[i]; o3[2] = c.vz[i]; }   // lone particle keeps its velocity
      if (!rc.empty()) {
        const double* r = &rc[3 * k];
        o3[0] += om[1] * r[2] - om[2] * r[1];
        o3[1] += om[2] * r[0] - om[0] * r[2];
        o3[2] += om[0] * r[1] - om[1] * r[0];
      }
      c.vx[i] = (float)o3[0]; c.vy[i] = (float)o3[1]; c.vz[i] = (float)o3[2];
    }
  }
}

template <class T>
void permute(std::vector<T>& a, const std::vector<uint32_t>& order) {
  std::vector<T> b(a.size());
  for (size_t k = 0; k < order.size(); ++k) b[k] = a[order[k]];
  a.swap(b);
}

void one_step(Ctx& c) {
  const size_t N = c.x.size();
  const uint32_t t = c.t;
  // 1. MOVE (Eq. 1)
  for (size_t i = 0; i < N; ++i) {
    float r[3] = {c.x[i], c.y[i], c.z[i]}, v[3] = {c.vx[i], c.vy[i], c.vz[i]};
    stream_one(c, r, v, t);
    c.x[i] = r[0]; c.y[i] = r[1]; c.z[i] = r[2];
    c.vx[i] = v[0]; c.vy[i] = v[1]; c.vz[i] = v[2];
  }
  // 2.-3. shift and cell index
  float s[3];
  grid_shift(c, t, s);
  for (int d = 0; d < 3; ++d) c.last_shift[d] = s[d];
  c.key.resize(N);
  for (int d = 0; d < 3; ++d) c.rho[d].resize(N);
  for (size_t i = 0; i < N; ++i) {
    const float r[3] = {c.x[i], c.y[i], c.z[i]};
    int ic[3]; float rho[3]; int im;
    cell_of_le(c, t, r, s, ic, rho, &im);
    c.key[i] = layout_key(c, ic);
    c.rho[0][i] = rho[0]; c.rho[1][i] = rho[1]; c.rho[2][i] = rho[2];
    if (c.p.shear_rate != 0.0f) {       // collide in the frame of the image: v_x -+ U, one fp32 add (undone after the collision)
      if (i == 0) c.img.assign(N, 0);
      c.img[i] = (signed char)im;
      if (im) c.vx[i] = c.vx[i] + (float)im * le_velocity(c);
    }
  }
  // 4. REORDER when due (readings U3,U4): ascending (key, id)
  if (t % (uint32_t)c.p.rebin_every == 0u) {
    std::vector<uint32_t> order(N);
    for (size_t i = 0; i < N; ++i) order[i] = (uint32_t)i;
    std::sort(order.begin(), order.end(), [&](uint32_t p, uint32_t q) {
      if (c.key[p] != c.key[q]) return c.key[p] < c.key[q];
      return c.id[p] < c.id[q];
    });
    permute(c.x, order); permute(c.y, order); permute(c.z, order);
    permute(c.vx, order); permute(c.vy, order); permute(c.vz, order);
    permute(c.id, order); permute(c.key, order);
    permute(c.rho[0], order); permute(c.rho[1], order); permute(c.rho[2], order);
    if (c.p.shear_rate != 0.0f) permute(c.img, order);
  }
  // members of every cell, in ascending id
  c.count.assign(c.nkeys, 0u);
  for (size_t i = 0; i < N; ++i) c.count[c.key[i]]++;
  std::vector<size_t> off(c.nkeys + 1, 0);
  for (size_t k = 0; k < c.nkeys; ++k) off[k + 1] = off[k] + c.count[k];
  std::vector<uint32_t> mem(N);
  {
    std::vector<size_t> cur(off.begin(), off.end() - 1);
    for (size_t i = 0; i < N; ++i) mem[cur[c.key[i]]++] = (uint32_t)i;
  }
  for (size_t k = 0; k < c.nkeys; ++k)
    std::sort(mem.begin() + off[k], mem.begin() + off[k + 1], [&](uint32_t p, uint32_t q) { return c.id[p] < c.id[q]; });
  // 5. bookkeeping of the pre-collision sums (real particles) for the parity tests
  c.sx.assign(c.nkeys, 0.0); c.sy.assign(c.nkeys, 0.0); c.sz.assign(c.nkeys, 0.0); c.se.assign(c.nkeys, 0.0);
  for (size_t i = 0; i < N; ++i) {
    const uint32_t k = c.key[i];
    const double a = c.vx[i], b = c.vy[i], d = c.vz[i];
    const double mr = particle_mass(c, c.id[i]) / (double)c.p.mass;     // 1 for a fluid particle (solutes: reading U23)
    c.sx[k] += mr * a; c.sy[k] += mr * b; c.sz[k] += mr * d; c.se[k] += mr * (a * a + b * b + d * d);
  }
  // 6.-7. PROCESS_CELLS + ROTATE_VELOCITIES
  c.n_singular = 0;
  for (size_t k = 0; k < c.nkeys; ++k) {
    if (c.count[k] == 0) continue;
    int ic[3];
    key_to_cell(c, (uint32_t)k, ic);
    collide_cell(c, canonical_id(c, ic), ic, s, t, &mem[off[k]], c.count[k], nullptr, nullptr);
  }
  if (c.p.shear_rate != 0.0f)
    for (size_t i = 0; i < N; ++i) if (c.img[i]) c.vx[i] = c.vx[i] - (float)c.img[i] * le_velocity(c);
  c.have_cells = true;
  c.t = t + 1u;
}

}  // namespace

// =================================== C ABI ====================================================
extern "C" {

int oracle_create(void** out, const float box[3], const int cells[3], float n_per_cell, const Params* p,
                  unsigned long long seed) {
  if (!out || !box || !cells || !p) return E_INVAL;
  *out = nullptr;
  for (int d = 0; d < 3; ++d) if (cells[d] < 1 || !(box[d] > 0.0f)) return E_INVAL;
  const float a = box[0] / (float)cells[0];
  for (int d = 1; d < 3; ++d) if (box[d] / (float)cells[d] != a) return E_INVAL;   // cubic cells only
  if (p->collision < 0 || p->collision > 1) return E_INVAL;
  if (!(p->dt > 0.0f) || !(p->kT > 0.0f) || !(p->mass > 0.0f) || p->rebin_every < 1) return E_INVAL;
  for (int d = 0; d < 3; ++d) if (p->brick[d] < 1) return E_INVAL;
  int nwall = 0;
  for (int d = 0; d < 3; ++d) {
    if (p->bc[d] < 0 || p->bc[d] > 2) return E_INVAL;
    if (p->bc[d] != 0) { nwall++; if (p->g[d] != 0.0f) return E_INVAL; }   // no force along the wall normal
  }
  if (nwall > 1) return E_INVAL;                                            // slit geometry only
  if (nwall && (p->conserve_L || p->collision == 1) && !p->phantoms) return E_INVAL;   // needs explicit phantom sets (U8, U22)
  bool noslip = false;
  for (int d = 0; d < 3; ++d) if (p->bc[d] == 1) noslip = true;
  if (p->phantoms < 0 || p->phantoms > 1 || (p->phantoms && !noslip)) return E_INVAL;   // phantoms fill no-slip walls (U20: none at slip walls)
  if (p->solute_mass < 0.0f) return E_INVAL;
  if (p->wall_velocity != 0.0f && (!nwall || p->bc[0] != 0)) return E_INVAL;            // moving walls: no-slip wall axis y or z, flow along x (U24)
  for (int d = 0; d < 3; ++d) if (p->wall_velocity != 0.0f && p->bc[d] == 2) return E_INVAL;
  if (p->collision == 0 && p->conserve_L && p->thermostat) return E_INVAL;  // ambiguous (U6)
  if (!(n_per_cell > 0.0f)) return E_INVAL;
  if (p->shear_rate != 0.0f && (nwall || p->collision == 1 || p->conserve_L)) return E_INVAL;   // Lees-Edwards: periodic SRD only (U21)
  Ctx* c = new Ctx();
  c->p = *p; c->seed = seed; c->t = 0; c->a = a; c->inv_a = 1.0f / a;
  c->nbar = (int)std::lround((double)n_per_cell);
  c->nkeys = 1;
  for (int d = 0; d < 3; ++d) {
    c->L[d] = box[d]; c->n[d] = cells[d];
    c->m[d] = cells[d] + (p->bc[d] != 0 ? 2 : 0);
    c->B[d] = p->brick[d];
    c->mb[d] = (c->m[d] + c->B[d] - 1) / c->B[d];
    c->nkeys *= (size_t)c->mb[d] * (size_t)c->B[d];
  }
  if (c->nkeys >= 0xffffffffull) { delete c; return E_INVAL; }
  c->cosa = std::cos((double)p->alpha); c->sina = std::sin((double)p->alpha);
  *out = c;
  return E_OK;
}

int oracle_destroy(void* h) { delete (Ctx*)h; return E_OK; }

int oracle_num_keys(void* h, unsigned long long* nkeys) {
  if (!h || !nkeys) return E_INVAL;
  *nkeys = ((Ctx*)h)->nkeys;
  return E_OK;
}

int oracle_set_state(void* h, unsigned long long n, const float* x, const float* y, const float* z, const float* vx,
                     const float* vy, const float* vz, const unsigned* id, unsigned step) {
  Ctx* c = (Ctx*)h;
  if (!c || (n && (!x || !y || !z || !vx || !vy || !vz)) || n > 0xffffffffull) return E_INVAL;
  c->x.assign(x, x + n); c->y.assign(y, y + n); c->z.assign(z, z + n);
  c->vx.assign(vx, vx + n); c->vy.assign(vy, vy + n); c->vz.assign(vz, vz + n);
  c->id.resize(n);
  for (size_t i = 0; i < n; ++i) c->id[i] = id ? id[i] : (uint32_t)i;
  c->t = step; c->have_state = true; c->have_cells = false;
  return E_OK;
}

int oracle_step(void* h, int nsteps) {
  Ctx* c = (Ctx*)h;
  if (!c || nsteps < 0) return E_INVAL;
  if (!c->have_state) return E_STATE;
  for (int k = 0; k < nsteps; ++k) one_step(*c);
  return E_OK;
}

int oracle_get_state(void* h, float* x, float* y, float* z, float* vx, float* vy, float* vz, unsigned* id) {
  Ctx* c = (Ctx*)h;
  if (!c) return E_INVAL;
  if (!c->have_state) return E_STATE;
  const size_t n = c->x.size(), b = n * sizeof(float);
  if (x) memcpy(x, c->x.data(), b);
  if (y) memcpy(y, c->y.data(), b);
  if (z) memcpy(z, c->z.data(), b);
  if (vx) memcpy(vx, c->vx.data(), b);
  if (vy) memcpy(vy, c->vy.data(), b);
  if (vz) memcpy(vz, c->vz.data(), b);
  if (id) memcpy(id, c->id.data(), n * sizeof(uint32_t));
  return E_OK;
}

// per-key pre-collision sums of the last step (real particles): count, m*sum v, sum |v|^2; per-particle key
int oracle_get_cells(void* h, unsigned* count, double* px, double* py, double* pz, double* e2, unsigned* key) {
  Ctx* c = (Ctx*)h;
  if (!c) return E_INVAL;
  if (!c->have_cells) return E_STATE;
  for (size_t k = 0; k < c->nkeys; ++k) {
    if (count) count[k] = c->count[k];
    if (px) px[k] = c->p.mass * c->sx[k];
    if (py) py[k] = c->p.mass * c->sy[k];
    if (pz) pz[k] = c->p.mass * c->sz[k];
    if (e2) e2[k] = c->se[k];
  }
  if (key) memcpy(key, c->key.data(), c->key.size() * sizeof(uint32_t));
  return E_OK;
}

int oracle_observables(void* h, Obs* o, float* profile) {
  Ctx* c = (Ctx*)h;
  if (!c || !o) return E_INVAL;
  if (!c->have_state) return E_STATE;
  const size_t N = c->x.size();
  const double m = c->p.mass;
  double P[3] = {0, 0, 0}, E = 0, Mr = 0;   // in units of the fluid-particle mass
  for (size_t i = 0; i < N; ++i) {
    const double a = c->vx[i], b = c->vy[i], d = c->vz[i];
    const double mr = particle_mass(*c, c->id[i]) / m;
    P[0] += mr * a; P[1] += mr * b; P[2] += mr * d; E += mr * (a * a + b * b + d * d); Mr += mr;
  }
  o->n = N; o->step = c->t;
  for (int d = 0; d < 3; ++d) o->P[d] = m * P[d];
  o->E_kin = 0.5 * m * E;
  // global estimate: sum m_i |v_i - <v>|^2 / (3 (N-1)), <v> = sum m_i v_i / sum m_i
  o->kT_est = (N > 1) ? m * (E - (P[0] * P[0] + P[1] * P[1] + P[2] * P[2]) / Mr) / (3.0 * (double)(N - 1)) : 0.0;
  // cell-level estimate from the last step's pre-collision sums: <m sum w^2> / <3 (N_c - 1)>
  o->kT_cell = 0.0; o->max_cell_count = 0; o->n_singular_cells = c->n_singular;
  if (c->have_cells) {
    double num = 0, den = 0;   // (with solutes the sums are mass-weighted and this estimate is not formed: 0)
    for (size_t k = 0; k < c->nkeys; ++k) {
      const unsigned nc = c->count[k];
      if (nc > o->max_cell_count) o->max_cell_count = nc;
      if (nc < 2 || c->p.solute_mass > 0.0f) continue;
      num += m * (c->se[k] - (c->sx[k] * c->sx[k] + c->sy[k] * c->sy[k] + c->sz[k] * c->sz[k]) / nc);
      den += 3.0 * (nc - 1);
    }
    o->kT_cell = den > 0 ? num / den : 0.0;
  }
  if (profile) {
    int pa = 2, fa = 0;
    for (int d = 0; d < 3; ++d) if (c->p.bc[d] != 0) pa = d;
    for (int d = 2; d >= 0; --d) if (c->p.g[d] != 0.0f) fa = d;
    const int nb = c->n[pa];
    std::vector<double> sv(nb, 0.0), cnt(nb, 0.0);
    const std::vector<float>* R[3] = {&c->x, &c->y, &c->z};
    const std::vector<float>* V[3] = {&c->vx, &c->vy, &c->vz};
    for (size_t i = 0; i < N; ++i) {
      int b = (int)floorf((*R[pa])[i] * c->inv_a);
      if (b < 0) b = 0;
      if (b >= nb) b = nb - 1;
      sv[b] += (*V[fa])[i]; cnt[b] += 1.0;
    }
    for (int b = 0; b < nb; ++b) profile[b] = cnt[b] > 0 ? (float)(sv[b] / cnt[b]) : 0.0f;
  }
  return E_OK;
}

// ------------------------------- hooks for hand checks ----------------------------------------
void oracle_philox4x32_10(const unsigned ctr[4], const unsigned key[2], unsigned out[4]) {
  philox4x32_10(ctr, key, out);
}
int oracle_grid_shift(void* h, unsigned t, float s[3]) {
  if (!h) return E_INVAL;
  grid_shift(*(Ctx*)h, t, s);
  return E_OK;
}
int oracle_srd_axis(void* h, unsigned cid, unsigned t, double n[3]) {
  if (!h) return E_INVAL;
  srd_axis(*(Ctx*)h, cid, t, n);
  return E_OK;
}
int oracle_mbs_energy(void* h, unsigned cid, unsigned t, unsigned Nc, double* e_over_kT) {
  if (!h || !e_over_kT) return E_INVAL;
  *e_over_kT = mbs_energy_over_kT(*(Ctx*)h, cid, t, Nc);
  return E_OK;
}
int oracle_normals(void* h, unsigned index, unsigned sub, unsigned t, unsigned tag, double g[4]) {
  if (!h) return E_INVAL;
  uint32_t o[4];
  draw(*(Ctx*)h, index, sub, t, tag, o);
  normals4(o, g);
  return E_OK;
}
// cell of a position for a given shift: ijk, canonical id, memory key, cell-local coordinate
int oracle_cell_of(void* h, const float r[3], const float s[3], int ijk[3], unsigned* cid, unsigned* key, float rho[3]) {
  if (!h) return E_INVAL;
  Ctx& c = *(Ctx*)h;
  int ic[3]; float rr[3];
  cell_of(c, r, s, ic, rr);
  for (int d = 0; d < 3; ++d) { if (ijk) ijk[d] = ic[d]; if (rho) rho[d] = rr[d]; }
  if (cid) *cid = canonical_id(c, ic);
  if (key) *key = layout_key(c, ic);
  return E_OK;
}
int oracle_stream_one(void* h, float r[3], float v[3]) {
  if (!h) return E_INVAL;
  stream_one(*(Ctx*)h, r, v, ((Ctx*)h)->t);
  return E_OK;
}
// Lees-Edwards hooks: MOVE of step t, and the cell (with the image used: -1, 0, +1) of a position at step t
int oracle_stream_one_at(void* h, unsigned t, float r[3], float v[3]) {
  if (!h) return E_INVAL;
  stream_one(*(Ctx*)h, r, v, t);
  return E_OK;
}
int oracle_cell_of_le(void* h, unsigned t, const float r[3], const float s[3], int ijk[3], unsigned* cid, unsigned* key, int* image) {
  if (!h) return E_INVAL;
  Ctx& c = *(Ctx*)h;
  int ic[3]; float rr[3];
  cell_of_le(c, t, r, s, ic, rr, image);
  for (int d = 0; d < 3; ++d) if (ijk) ijk[d] = ic[d];
  if (cid) *cid = canonical_id(c, ic);
  if (key) *key = layout_key(c, ic);
  return E_OK;
}
int oracle_le_offset(void* h, unsigned t, float* D, float* U) {
  if (!h) return E_INVAL;
  if (D) *D = le_offset(*(Ctx*)h, t);
  if (U) *U = le_velocity(*(Ctx*)h);
  return E_OK;
}
// explicit phantom particles (reading U22) of cell ijk for lattice shift s at step t: up to `cap` of them as
// rho[3k..3k+2] (cell-local coordinates) and v[3k..3k+2]; *n = their number
int oracle_phantoms(void* h, const int ijk[3], const float s[3], unsigned t, int cap, double* rho, double* v, int* n) {
  if (!h || !ijk || !s || !n) return E_INVAL;
  Ctx& c = *(Ctx*)h;
  std::vector<Phantom> ph;
  make_phantoms(c, canonical_id(c, ijk), ijk, s, t, ph);
  *n = (int)ph.size();
  for (int k = 0; k < (int)ph.size() && k < cap; ++k)
    for (int d = 0; d < 3; ++d) { if (rho) rho[3 * k + d] = ph[k].rho[d]; if (v) v[3 * k + d] = ph[k].v[d]; }
  return E_OK;
}
// Collide the whole current state as ONE cell (cell id `cid`, step t) with a prescribed axis and/or
// scaling factor: the hand-computed checks of DESIGN.md. rho = positions / a are used for +a.
int oracle_collide_one_cell(void* h, unsigned cid, unsigned t, const double* axis, const double* kappa) {
  Ctx* c = (Ctx*)h;
  if (!c) return E_INVAL;
  if (!c->have_state) return E_STATE;
  const size_t N = c->x.size();
  std::vector<uint32_t> idx(N);
  for (size_t i = 0; i < N; ++i) idx[i] = (uint32_t)i;
  std::sort(idx.begin(), idx.end(), [&](uint32_t p, uint32_t q) { return c->id[p] < c->id[q]; });
  for (int d = 0; d < 3; ++d) c->rho[d].resize(N);
  for (size_t i = 0; i < N; ++i) {
    c->rho[0][i] = c->x[i] * c->inv_a; c->rho[1][i] = c->y[i] * c->inv_a; c->rho[2][i] = c->z[i] * c->inv_a;
  }
  const int ic[3] = {0, 0, 0};
  const float s[3] = {0, 0, 0};
  c->n_singular = 0;
  collide_cell(*c, cid, ic, s, t, idx.data(), (unsigned)N, axis, kappa);
  return E_OK;
}

}  // extern "C"
