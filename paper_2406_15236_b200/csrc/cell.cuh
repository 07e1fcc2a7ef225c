// cell.cuh -- PROCESS_CELLS for a batch of cells: per cell v_cm, the SRD rotation axis, the
// thermostat factor kappa (Eqs. 5-7) and the virtual wall particles of wall-cut cells (U8).
// Used by k_cell (cell.cu) and by the sweep that finalises the previous step's cells itself (sweep.cu).
#pragma once
#include "internal.cuh"

namespace mpc {


// E_k / k_BT ~ Gamma(a, 1), a = 3 (N_c - 1) / 2 (Eq. 7; U6): Marsaglia-Tsang rejection from one
// normal x and one uniform U per attempt: d = a - 1/3, c = 1 / sqrt(9 d), v = (1 + c x)^3, accepted if v > 0 and
// (U < 1 - k x^4 or ln U < x^2 / 2 + d (1 - v + ln v)), k = 0.0331 for N_c < 7 and (0.0093 + 0.0145 / sqrt(d) + 0.06 / d) / d
// above; E_k / k_BT = d v. Whether an attempt is accepted decides
// which random words make E_k, so U6 fixes every operation up to that decision in binary32 (each rounded once: the _rn
// intrinsics below are never contracted or reassociated), with ln and cos given by short series instead of the
// hardware approximations. Attempt 0 uses the cell's TAG_AXIS block (radius: word 2, angle: word 3, top 24 bits each;
// U: the low bytes of words 0, 1, 2), attempt j >= 1 words 0, 1, 2 of block j - 1 of the cell's TAG_MBS stream.
// ln x, x a positive normal float: x = m 2^e, m in [sqrt(1/2), sqrt(2)), ln m = 2 atanh((m - 1) / (m + 1)) up to s^9
__device__ __forceinline__ float mt_log(float x) {
  const int i = __float_as_int(x);
  const int e = (i - 0x3f3504f3) >> 23;
  const float f = __fadd_rn(__int_as_float(i - (e << 23)), -1.0f);
  const float s = __fdiv_rn(f, __fadd_rn(2.0f, f));
  const float z = __fmul_rn(s, s);
  float p = __fmaf_rn(z, 0x1.c71c72p-3f, 0x1.24924ap-2f);   // 2/9, 2/7
  p = __fmaf_rn(z, p, 0x1.99999ap-2f);                      // 2/5
  p = __fmaf_rn(z, p, 0x1.555556p-1f);                      // 2/3
  p = __fmaf_rn(z, p, 2.0f);
  return __fmaf_rn((float)e, 0x1.62e43p-1f, __fmul_rn(s, p));
}
// cos(2 pi k / 2^24), k < 2^24: quarter turn q and y in [-pi/4, pi/4) split off exactly, Taylor series to y^9 / y^10
__device__ __forceinline__ float mt_cos(uint32_t k) {
  const uint32_t kk = k + 2097152u;
  const uint32_t q = (kk >> 22) & 3u;
  const int r = (int)(kk & 4194303u) - 2097152;
  const float y = __fmul_rn((float)r, 0x1.921fb6p-22f);     // (pi / 2) / 2^22
  const float z = __fmul_rn(y, y);
  float t;
  if (q & 1u) {                                             // -+ sin y
    t = __fmaf_rn(z, 0x1.71de3ap-19f, -0x1.a01a02p-13f);    // 1/9!, -1/7!
    t = __fmaf_rn(z, t, 0x1.111112p-7f);                    // 1/5!
    t = __fmaf_rn(z, t, -0x1.555556p-3f);                   // -1/3!
    t = __fmaf_rn(__fmul_rn(y, z), t, y);
    return (q == 1u) ? -t : t;
  }
  t = __fmaf_rn(z, -0x1.27e4fcp-22f, 0x1.a01a02p-16f);      // -1/10!, 1/8!
  t = __fmaf_rn(z, t, -0x1.6c16c2p-10f);                    // -1/6!
  t = __fmaf_rn(z, t, 0x1.555556p-5f);                      // 1/4!
  t = __fmaf_rn(__fmul_rn(z, z), t, __fmaf_rn(-0.5f, z, 1.0f));
  return (q == 0u) ? t : -t;
}
struct MtShape { float d, c, k; };   // d = a - 1/3, c = 1 / sqrt(9 d), k = constant of the squeeze U < 1 - k x^4 (U6)
// (c, k) for N_c < MT_TABLE come from a table made on the host with the same IEEE operations (mt_shape_host)
__host__ __device__ __forceinline__ float mt_d_of(uint32_t nc) {
#ifdef __CUDA_ARCH__
  return __fadd_rn(__fmul_rn(1.5f, (float)(nc - 1u)), -0x1.555556p-2f);
#else
  volatile float a = 1.5f * (float)(nc - 1u);      // volatile: every operation rounded to binary32 on the host as well
  volatile float d = a - 0x1.555556p-2f;
  return d;
#endif
}
inline void mt_shape_host(uint32_t nc, float& c_out, float& k_out) {
  const float d = mt_d_of(nc);
  volatile float t = 9.0f * d;
  volatile float r = sqrtf(t);
  volatile float c = 1.0f / r;
  c_out = c;
  if (nc < 7u) { k_out = 0x1.0f27bcp-5f; return; }              // 0.0331
  volatile float sd = sqrtf(d);
  volatile float q1 = 0x1.db22d0p-7f / sd;                       // 0.0145 / sqrt(d)
  volatile float q2 = 0x1.eb851ep-5f / d;                        // 0.06 / d
  volatile float s1 = 0x1.30be0ep-7f + q1;                       // 0.0093 + ...
  volatile float s2 = s1 + q2;
  volatile float k = s2 / d;
  k_out = k;
}
__device__ __forceinline__ MtShape mt_shape(const Geo& G, uint32_t nc) {
  MtShape s;
  s.d = mt_d_of(nc);
  if (nc < (uint32_t)MT_TABLE) {
    const float2 ck = __ldg(reinterpret_cast<const float2*>(G.mt_c) + nc);
    s.c = ck.x; s.k = ck.y;
  } else {
    s.c = __fdiv_rn(1.0f, __fsqrt_rn(__fmul_rn(9.0f, s.d)));
    s.k = __fdiv_rn(__fadd_rn(__fadd_rn(0x1.30be0ep-7f, __fdiv_rn(0x1.db22d0p-7f, __fsqrt_rn(s.d))), __fdiv_rn(0x1.eb851ep-5f, s.d)), s.d);
  }
  return s;
}
// one attempt from the 24-bit integers wr (radius), wa (angle), wu (acceptance); true: accepted, ek = E_k / k_BT
__device__ __forceinline__ bool mt_attempt(const MtShape sh, uint32_t wr, uint32_t wa, uint32_t wu, float& ek) {
  const float Ur = __fmul_rn((float)(wr + 1u), 0x1p-24f), U = __fmul_rn((float)(wu + 1u), 0x1p-24f);
  const float x = __fmul_rn(__fsqrt_rn(__fmul_rn(-2.0f, mt_log(Ur))), mt_cos(wa));
  const float v0 = __fmaf_rn(sh.c, x, 1.0f);
  if (!(v0 > 0x1p-20f)) return false;
  const float v = __fmul_rn(__fmul_rn(v0, v0), v0);
  const float x2 = __fmul_rn(x, x);
  ek = __fmul_rn(sh.d, v);
  if (U < __fmaf_rn(-__fmul_rn(sh.k, x2), x2, 1.0f)) return true;
  return mt_log(U) < __fmaf_rn(0.5f, x2, __fmul_rn(sh.d, __fadd_rn(__fadd_rn(1.0f, -v), mt_log(v))));
}
__device__ __forceinline__ bool mt_attempt0(const MtShape sh, const Block4& o, float& ek) {   // o = the cell's TAG_AXIS block
  return mt_attempt(sh, o.c >> 8, o.d >> 8, ((o.a & 0xffu) << 16) | ((o.b & 0xffu) << 8) | (o.c & 0xffu), ek);
}
// attempts 1, 2, ... (after a rejected attempt 0)
__device__ __forceinline__ float mt_retry(const Geo& G, uint32_t cid, const MtShape sh) {
  float ek;
  for (uint32_t j = 0; j < 15u; ++j) {
    const Block4 o = philox_rk(cid, j, G.t, TAG_MBS, G.rk);
    if (mt_attempt(sh, o.a >> 8, o.b >> 8, o.c >> 8, ek)) return ek;
  }
  return sh.d;
}
__device__ __forceinline__ float kappa_of(const Geo& G, float ek, float mw2) {   // Eq. (6)
  const float x = __fdividef(2.0f * (G.kT * ek), mw2);
  return x * rsqrtf(fmaxf(x, 1e-37f));
}
// kappa of Eq. (6) for a cell of nc >= 2 members with mw2 = sum m_i |v_i - v_cm|^2 > 0; o = the cell's TAG_AXIS block
__device__ __forceinline__ float mbs_kappa(const Geo& G, uint32_t cid, const Block4& o, uint32_t nc, float mw2) {
  const MtShape sh = mt_shape(G, nc);
  float ek;
  if (!mt_attempt0(sh, o, ek)) ek = mt_retry(G, cid, sh);
  return kappa_of(G, ek, mw2);
}

// rec[key] = { vcm.x, vcm.y, vcm.z, kappa, n.x, n.y, n.z, - }
// grid = (mb0 * CTAs-per-brick, mb1, mb2): the brick coordinates come from blockIdx, no division.
// zero != 0: the sums of a cell are cleared once read, which saves the memset before the next step's sweep.
// Thread t handles cell t of the CTA's CT cells: reads its sums (coalesced), v_cm, sum |v - v_cm|^2, N_c, the TAG_AXIS
// block (axis + first thermostat attempt) and writes one 32-byte record (coalesced). 0.3 % of the first attempts are
// rejected at <N_c> = 10; those lanes retry in place (8 % of the warps wait for one).
struct CellWork { float vx, vy, vz, w2; uint32_t cid, nc; };

// CT cells [lbase, lbase + CT) of brick (bx, by, bz), one per thread of the CTA (all CT threads must call)
template <bool SUB>
__device__ __forceinline__ void cell_batch(const Geo& G, uint32_t bx, uint32_t by, uint32_t bz, uint32_t lbase, u64* __restrict__ sums,
                                           float* __restrict__ rec, int zero, uint32_t* __restrict__ counts, int handover) {
  const unsigned tid = threadIdx.x;
  const int b0 = G.bs[0], b1 = G.bs[1], b2 = G.bs[2];
  const uint32_t local = lbase + tid;
  const bool valid = local < (1u << (b0 + b1 + b2));
  const uint32_t brick = (bz * (uint32_t)G.mb[1] + by) * (uint32_t)G.mb[0] + bx;
  const uint32_t kbase = (brick << (b0 + b1 + b2)) + lbase;
  u64* s = sums + (size_t)(kbase + tid) * G.sw;
  u64 w0 = 0ull;
  if (valid) w0 = s[0];
  const uint32_t nreal = (uint32_t)(w0 & 0xffffull);
  if (SUB && valid && sub_shared(G, (int)((bz << b2) | (local >> (b0 + b1)))) >= 0) {
    // slab subdomain: the count in the (now complete) sums of a shared cell includes the neighbour's particles.
    // Unfolded local reorder (handover = 0): every particle stays, the scan needs this rank's own count. Folded reorder
    // with hand-over (handover = 1): the particles in the halo layers leave (count 0; abase = the owner's own count, behind
    // which they are placed in the owner's new order), those of the neighbour in this rank's own layers arrive (complete count)
    const uint32_t mine = G.lcount[kbase + tid];
    const uint32_t bl = bz, nb = (uint32_t)G.nbz;
    if (counts) {
      if (!handover) counts[kbase + tid] = mine;
      else if (bl == 0u || bl == nb - 1u) { counts[kbase + tid] = 0u; G.abase[kbase + tid] = nreal - mine; }
      else counts[kbase + tid] = nreal;
    }
    if (zero && mine) G.lcount[kbase + tid] = 0u;
  } else
  if (counts && valid) counts[kbase + tid] = nreal;      // compact per-cell counts for the scan of a reorder
  CellWork cw = {0.f, 0.f, 0.f, 0.f, 0u, 0u};
  if (valid && nreal != 0u) {
    const int ix = (int)((bx << b0) | (local & ((1u << b0) - 1u)));
    const int iy = (int)((by << b1) | ((local >> b0) & ((1u << b1) - 1u)));
    const int iz = (int)((bz << b2) | (local >> (b0 + b1)));
    cw.cid = SUB ? canonical_id_sub(G, ix, iy, iz) : canonical_id(G, ix, iy, iz);
    int sx, sy, sz, pad;
    unpack_ss(s[1], sx, sy);
    unpack_ss(s[2], sz, pad);
    if (zero) { s[0] = 0ull; s[1] = 0ull; s[2] = 0ull; }
    double S0 = (double)sx * G.fxv_inv, S1 = (double)sy * G.fxv_inv, S2 = (double)sz * G.fxv_inv;
    // a cell total within a factor two of the int32 range of the momentum words, or too many particles for the tile's
    // packed count / energy words
    if (nreal >= 64u && (nreal >= MAX_CELL_COUNT || abs(sx) >= (1 << 30) || abs(sy) >= (1 << 30) || abs(sz) >= (1 << 30))) atomicAdd(G.nrange, 1ull);
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
        const double uw = (iw <= 1) ? -(double)G.wall_u : (double)G.wall_u;   // thermal about the wall velocity (U24)
        for (uint32_t j = 0; j < nv; ++j) {
          const Block4 o = philox_rk(cw.cid, j, G.t, TAG_WALL, G.rk);
          float g0, g1, g2;
          normals3(o, g0, g1, g2);
          const double a = (double)(G.sigma * g0) + uw, b = (double)(G.sigma * g1), c = (double)(G.sigma * g2);
          S0 += a; S1 += b; S2 += c; E += a * a + b * b + c * c;
        }
        Nc += nv;
      }
    }
    // 1 / N_c: float reciprocal refined by one Newton step in double (relative error < 1e-14; a double division costs twice as much)
    double inv = (double)__frcp_rn((float)Nc);
    inv = inv * (2.0 - (double)Nc * inv);
    cw.vx = (float)(S0 * inv); cw.vy = (float)(S1 * inv); cw.vz = (float)(S2 * inv);
    cw.nc = Nc;
    if (G.thermostat && Nc >= 2u) {
      const double W2 = E - (S0 * S0 + S1 * S1 + S2 * S2) * inv;   // sum |v - vcm|^2
      if (W2 > 0.0) cw.w2 = (float)W2;
    }
  }
  if (cw.nc == 0u) return;
  // ---- axis and thermostat draw ----
  const Block4 o = philox_rk(cw.cid, 0u, G.t, TAG_AXIS, G.rk);
  const float kappa = (cw.w2 > 0.0f) ? mbs_kappa(G, cw.cid, o, cw.nc, G.mass * cw.w2) : 1.0f;
  // axis: z = 2 u0 - 1, phi = 2 pi u1 (U11). cos / sin of phi - pi in [-pi, pi) with the hardware approximations (absolute
  // error ~4e-7 there, inside the 2e-5 parity budget of the velocities): cos phi = -cos(phi - pi), sin phi = -sin(phi - pi)
  const float zz = 2.0f * u01_co(o.a) - 1.0f;
  const float t2 = (1.0f - zz) * (1.0f + zz);
  const float rr = -t2 * rsqrtf(fmaxf(t2, 1e-30f));
  const float ph = 6.2831853071795865f * (u01_co(o.b) - 0.5f);
  float4* out = reinterpret_cast<float4*>(rec) + (size_t)(kbase + tid) * 2;
  out[0] = make_float4(cw.vx, cw.vy, cw.vz, kappa);
  out[1] = make_float4(rr * __cosf(ph), rr * __sinf(ph), zz, 0.0f);
}

}  // namespace mpc
