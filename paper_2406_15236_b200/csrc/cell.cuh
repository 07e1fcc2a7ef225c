// cell.cuh -- PROCESS_CELLS for a batch of cells: per cell v_cm, the SRD rotation axis, the
// thermostat factor kappa (Eqs. 5-7) and the virtual wall particles of wall-cut cells (U8).
// Used by k_cell (cell.cu) and by the sweep that finalises the previous step's cells itself (sweep.cu).
#pragma once
#include "internal.cuh"

namespace mpc {


// E_k / k_BT ~ Gamma(3(Nc-1)/2, 1) (Eq. 7; U6): minus the log of a product of floor(f/2)
// uniforms (the product is renormalised by exponent extraction so it never underflows: one log per cell instead
// of one per uniform), plus half a squared normal if f is odd.
__device__ __forceinline__ void renorm(float& p, int& ex) {   // p = m * 2^e with m in [0.5,1): keep m, bank e
  const int bits = __float_as_int(p);
  ex += (bits >> 23) - 126;
  p = __int_as_float((bits & 0x007fffff) | 0x3f000000);
}
// 2^24 * u01_oc(w): the power-of-two scale of every uniform is banked in the exponent instead (exact)
__device__ __forceinline__ float u24_oc(uint32_t w) { return (float)((w >> 8) + 1u); }

// -ln of the product of the first M uniforms of the cell's TAG_MBS stream (M = floor(f/2) unit exponentials)
__device__ __forceinline__ float mbs_exponentials(const Geo& G, uint32_t cid, uint32_t M) {
  if (M == 0u) return 0.0f;
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
  // p in [0.5, 1): __logf has an absolute error below 2^-21 there; the exponent part is added in double
  return -(float)((double)__logf(p) + (double)ex * 0.6931471805599453);
}


// kappa of Eq. (6) for a cell of nc >= 2 members with mw2 = sum m_i |v_i - v_cm|^2 > 0; o = the cell's TAG_AXIS block,
// whose words 2, 3 give the half squared normal when f = 3 (nc - 1) is odd (U6)
__device__ __forceinline__ float mbs_kappa(const Geo& G, uint32_t cid, const Block4& o, uint32_t nc, float mw2) {
  const uint32_t f = 3u * (nc - 1u);
  float ek = mbs_exponentials(G, cid, f >> 1);
  if (f & 1u) {
    // cos(2 pi u) = -cos(2 pi (u - 1/2)), argument in [-pi, pi): __cosf / __logf are accurate to ~4e-7 absolute there,
    // far below the statistical meaning of the draw and the 2e-5 parity budget
    const float cs = __cosf(6.2831853071795865f * (u01_co(o.d) - 0.5f));
    ek -= __logf(u01_oc(o.c)) * cs * cs;
  }
  const float x = __fdividef(2.0f * (G.kT * ek), mw2);
  return x * rsqrtf(fmaxf(x, 1e-37f));
}

// rec[key] = { vcm.x, vcm.y, vcm.z, kappa, n.x, n.y, n.z, - }
// grid = (mb0 * CTAs-per-brick, mb1, mb2): the brick coordinates come from blockIdx, no division.
// zero != 0: the sums of a cell are cleared once read, which saves the memset before the next step's sweep.
// The number of Philox blocks a cell needs for its thermostat draw grows with its occupancy (Poisson), and a warp runs
// as long as its fullest cell needs. Two phases: (A) thread t reads the sums of cell t (coalesced), reduces them to
// {v_cm, sum |v - v_cm|^2, N_c} and parks that in shared memory; the CT cells of the CTA are counting-sorted by their
// number of Philox blocks; (B) thread j finishes the j-th cell of the sorted order (draw, kappa, axis, one 32-byte
// record): every warp gets cells of nearly equal cost, and there is no barrier after the loop of variable length.
struct CellWork { float vx, vy, vz, w2; uint32_t cid, nc; };
template <int CT>
struct CellScratch { unsigned hist[32]; unsigned short order[CT]; CellWork work[CT]; };

// CT cells [lbase, lbase + CT) of brick (bx, by, bz), one per thread of the CTA (all CT threads must call)
template <int CT>
__device__ __forceinline__ void cell_batch(const Geo& G, uint32_t bx, uint32_t by, uint32_t bz, uint32_t lbase, u64* __restrict__ sums,
                                           float* __restrict__ rec, int zero, CellScratch<CT>& sh) {
  unsigned* hist = sh.hist;
  unsigned short* order = sh.order;
  CellWork* work = sh.work;
  const unsigned tid = threadIdx.x;
  if (tid < 32) hist[tid] = 0u;
  const int b0 = G.bs[0], b1 = G.bs[1], b2 = G.bs[2];
  const uint32_t local = lbase + tid;
  const bool valid = local < (1u << (b0 + b1 + b2));
  const uint32_t brick = (bz * (uint32_t)G.mb[1] + by) * (uint32_t)G.mb[0] + bx;
  const uint32_t kbase = (brick << (b0 + b1 + b2)) + lbase;
  // ---- phase A ----
  u64* s = sums + (size_t)(kbase + tid) * G.sw;
  u64 w0 = 0ull;
  if (valid) w0 = s[0];
  const uint32_t nreal = (uint32_t)(w0 & 0xffffull);
  CellWork cw = {0.f, 0.f, 0.f, 0.f, 0u, 0u};
  uint32_t M = 0u;
  if (valid && nreal != 0u) {
    const int ix = (int)((bx << b0) | (local & ((1u << b0) - 1u)));
    const int iy = (int)((by << b1) | ((local >> b0) & ((1u << b1) - 1u)));
    const int iz = (int)((bz << b2) | (local >> (b0 + b1)));
    cw.cid = canonical_id(G, ix, iy, iz);
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
      if (W2 > 0.0) { M = (3u * (Nc - 1u)) >> 1; cw.w2 = (float)W2; }
    }
  }
  // ---- counting sort of the CTA's cells by the number of Philox blocks of their draw (empty cells last) ----
  const unsigned bin = cw.nc ? min((M + 3u) >> 2, 30u) : 31u;
  __syncthreads();
  const unsigned rank = atomicAdd(&hist[bin], 1u);
  work[tid] = cw;
  __syncthreads();
  if (tid < 32) {
    const unsigned v = hist[tid];
    unsigned inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned t = __shfl_up_sync(0xffffffffu, inc, o);
      if (tid >= (unsigned)o) inc += t;
    }
    hist[tid] = inc - v;
  }
  __syncthreads();
  order[hist[bin] + rank] = (unsigned short)tid;
  __syncthreads();
  // ---- phase B ----
  const unsigned u = order[tid];
  const CellWork c = work[u];
  if (c.nc == 0u) return;
  const Block4 o = philox_rk(c.cid, 0u, G.t, TAG_AXIS, G.rk);
  const float kappa = (c.w2 > 0.0f) ? mbs_kappa(G, c.cid, o, c.nc, G.mass * c.w2) : 1.0f;
  const float zz = 2.0f * u01_co(o.a) - 1.0f;
  const float rr = sqrtf((1.0f - zz) * (1.0f + zz));
  float sp, cp;
  sincospif(2.0f * u01_co(o.b), &sp, &cp);
  float4* out = reinterpret_cast<float4*>(rec) + (size_t)(kbase + u) * 2;
  out[0] = make_float4(c.vx, c.vy, c.vz, kappa);
  out[1] = make_float4(rr * cp, rr * sp, zz, 0.0f);
}


}  // namespace mpc
