// observe.cu -- observables (the paper's Properties<FINALIZE>; profile binning PAPER.md:212) and the
// cell-sum test hook.
#include "internal.cuh"

namespace mpc {

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
// sums of m_i v_i, m_i |v_i|^2 and m_i in units of the fluid-particle mass (solutes: DESIGN.md U23)
__global__ void __launch_bounds__(256) k_obs_particles(Geo G, size_t n, const float* __restrict__ vx, const float* __restrict__ vy,
                                                       const float* __restrict__ vz, const uint32_t* __restrict__ id, double* __restrict__ part) {
  __shared__ double sh[8];
  double a = 0, b = 0, c = 0, e = 0, ms = 0;
  const bool solutes = G.solute_mass > 0.0f;
  const double mrs = (double)G.solute_mass / (double)G.mass;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const double p = vx[i], q = vy[i], r = vz[i];
    const double mr = (solutes && id[i] >= G.solute_id0) ? mrs : 1.0;
    a += mr * p; b += mr * q; c += mr * r; e += mr * (p * p + q * q + r * r); ms += mr;
  }
  a = block_sum(a, sh); b = block_sum(b, sh); c = block_sum(c, sh); e = block_sum(e, sh); ms = block_sum(ms, sh);
  if (threadIdx.x == 0) { double* o = part + (size_t)blockIdx.x * 8; o[0] = a; o[1] = b; o[2] = c; o[3] = e; o[7] = ms; }
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
// Layer-averaged velocity profile (the shear-profile binning of PAPER.md:212: few bins, all threads hit them). The
// particles are cell-ordered, so the lanes of a warp mostly fall into the same layer: the lanes of the leading lane's
// layer are summed with warp shuffles (fixed-point, so the sums do not depend on the order) and added with ONE shared
// atomic per warp and quantity; the remaining lanes repeat (usually no second round).
__global__ void __launch_bounds__(256) k_obs_profile(Geo G, size_t n, int nb, const float* __restrict__ rp,
                                                     const float* __restrict__ vf, u64* __restrict__ prof) {
  extern __shared__ u64 bins[];   // nb velocity sums (int64 at 2^28/u per unit), nb counts
  for (int b = threadIdx.x; b < 2 * nb; b += blockDim.x) bins[b] = 0ull;
  __syncthreads();
  const double fx = (double)G.fxv * 64.0;        // 2^28 / u: 2^32 particles at 8 u still fit in an int64
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  const size_t i0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  for (size_t base = i0 - (threadIdx.x & 31); base < n; base += stride) {   // whole warps iterate together
    const size_t i = base + (threadIdx.x & 31);
    int b = -1;
    long long q = 0;
    if (i < n) {
      b = max(0, min((int)floorf(rp[i] * G.inv_a), nb - 1));
      q = __double2ll_rn((double)vf[i] * fx);
    }
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
  for (int b = threadIdx.x; b < 2 * nb; b += blockDim.x) if (bins[b] != 0ull) atomicAdd(&prof[b], bins[b]);
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

// ---- slab subdomains: particles by owner ---------------------------------
// class of a particle of a slab subdomain: 0 = its layer floor(z / a) is one of this rank's own, 1 / 2 = it belongs to the
// neighbour below / above (the nearer one, periodically)
__device__ __forceinline__ int sub_class(const Geo& G, float z) {
  int l = __float2int_rd(z * G.inv_a);
  l = max(0, min(l, G.nzg - 1));
  const int z0 = G.zoff + (1 << G.bs[2]), nz = G.m[2] - (2 << G.bs[2]);      // own layers [z0, z0 + nz)
  int up = l - z0; up += (up < 0) ? G.nzg : 0;                               // layers above the slab's first layer, periodic
  if (up < nz) return 0;
  return (up - nz < G.nzg - up) ? 2 : 1;
}
// counts[0..2] += particles per class; then, with cursor[0..2] set to the first slot of every class, the second kernel
// writes the particles class by class (order inside a class: as it comes; the physics does not depend on it)
__global__ void __launch_bounds__(256) k_sub_count(Geo G, size_t n, const float* __restrict__ z, uint32_t* __restrict__ counts) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int cl = (i < n) ? sub_class(G, z[i]) : 3;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const unsigned m = __ballot_sync(0xffffffffu, cl == k);
    if (m && (threadIdx.x & 31) == (unsigned)(__ffs((int)m) - 1)) atomicAdd(counts + k, (uint32_t)__popc(m));
  }
}
struct Arrays7 { const uint32_t* src[7]; uint32_t* dst[7]; };
__global__ void __launch_bounds__(256) k_sub_split(Geo G, size_t n, Arrays7 a, uint32_t* __restrict__ cursor) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned lane = threadIdx.x & 31u;
  const int cl = (i < n) ? sub_class(G, __uint_as_float(a.src[2][i])) : 3;
  uint32_t slot = 0;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const unsigned m = __ballot_sync(0xffffffffu, cl == k);
    if (!m) continue;
    const int leader = __ffs((int)m) - 1;
    uint32_t base = 0;
    if ((int)lane == leader) base = atomicAdd(cursor + k, (uint32_t)__popc(m));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (cl == k) slot = base + (uint32_t)__popc(m & ((1u << lane) - 1u));
  }
  if (cl < 3) {
#pragma unroll
    for (int q = 0; q < 7; ++q) a.dst[q][slot] = a.src[q][i];
  }
}

}  // namespace mpc

using namespace mpc;

int sub_pack_impl(mpc_ctx* c, float* const out[6], unsigned* id_out, unsigned long long counts[3]) {
  const size_t n = c->n;
  counts[0] = counts[1] = counts[2] = 0;
  if (n == 0) return MPC_OK;
  uint32_t h[3] = {0, 0, 0};
  CU(cudaMemsetAsync(c->cursor, 0, 16, c->stream));
  k_sub_count<<<nblk(n, 256), 256, 0, c->stream>>>(c->G, n, reinterpret_cast<const float*>(c->A[2]), c->cursor);
  LAUNCH_CHECK("k_sub_count");
  CU(cudaMemcpyAsync(h, c->cursor, 12, cudaMemcpyDeviceToHost, c->stream));
  CU(cudaStreamSynchronize(c->stream));
  const uint32_t base[3] = {0u, h[0], h[0] + h[1]};
  CU(cudaMemcpyAsync(c->cursor, base, 12, cudaMemcpyHostToDevice, c->stream));
  Arrays7 a;
  for (int q = 0; q < 7; ++q) a.src[q] = c->A[q];
  for (int q = 0; q < 6; ++q) a.dst[q] = reinterpret_cast<uint32_t*>(out[q]);
  a.dst[6] = id_out;
  k_sub_split<<<nblk(n, 256), 256, 0, c->stream>>>(c->G, n, a, c->cursor);
  LAUNCH_CHECK("k_sub_split");
  CU(cudaStreamSynchronize(c->stream));      // `base` is read by the copy above
  for (int k = 0; k < 3; ++k) counts[k] = h[k];
  return MPC_OK;
}

int observables_impl(mpc_ctx* c, mpc_obs* out, float* profile_host, int n_profile) {
  memset(out, 0, sizeof(*out));
  const Geo& G = c->G;
  float** F = reinterpret_cast<float**>(c->A);
  const size_t n = c->n;
  double* part = c->obs;
  u64* prof = reinterpret_cast<u64*>(c->obs + (size_t)OBS_BLOCKS * 8);
  int pa = 2, fa = 0;
  for (int d = 0; d < 3; ++d) if (G.bc[d] != 0) pa = d;
  for (int d = 2; d >= 0; --d) if (G.g[d] != 0.0f) fa = d;
  const int nb = G.n[pa];
  if (profile_host && nb > MAX_PROFILE) return fail(c, MPC_EINVAL, "profile axis longer than 2048 layers");
  if (profile_host && n_profile != nb) return fail(c, MPC_EINVAL, "n_profile must equal the number of cell layers along the profile axis");
  {
    FamilyTimer ft(c, F_OBS);
    CU(cudaMemsetAsync(c->obs, 0, OBS_HOST_DOUBLES * 8, c->stream));
    if (n) {
      k_obs_particles<<<OBS_BLOCKS, 256, 0, c->stream>>>(G, n, F[3], F[4], F[5], c->A[6], part);
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
  unsigned long long nsing = 0, nrange = 0;
  CU(cudaMemcpyAsync(hbuf, c->obs, OBS_HOST_DOUBLES * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  if (c->have_cells && G.conserve_L) CU(cudaMemcpyAsync(&nsing, c->nsing, 8, cudaMemcpyDeviceToHost, c->stream));
  CU(cudaMemcpyAsync(&nrange, c->nrange, 8, cudaMemcpyDeviceToHost, c->stream));
  CU(cudaStreamSynchronize(c->stream));
  double P[3] = {0, 0, 0}, E = 0, num = 0, den = 0, mx = 0, Mr = 0;
  for (int b = 0; b < OBS_BLOCKS; ++b) {
    const double* o = hbuf + (size_t)b * 8;
    P[0] += o[0]; P[1] += o[1]; P[2] += o[2]; E += o[3]; num += o[4]; den += o[5]; Mr += o[7];
    if (o[6] > mx) mx = o[6];
  }
  const double m = G.mass;
  out->n = n; out->step = c->t;
  for (int d = 0; d < 3; ++d) out->P[d] = m * P[d];
  out->E_kin = 0.5 * m * E;
  out->kT_est = n > 1 ? m * (E - (P[0] * P[0] + P[1] * P[1] + P[2] * P[2]) / Mr) / (3.0 * (double)(n - 1)) : 0.0;
  out->kT_cell = (!G.generic && den > 0) ? num / den : 0.0;
  out->max_cell_count = (unsigned)mx;
  out->n_singular_cells = nsing;
  out->n_range_overflows = nrange;
  if (profile_host) {
    const long long* pr = reinterpret_cast<const long long*>(hbuf + (size_t)OBS_BLOCKS * 8);
    const double fxi = G.fxv_inv / 64.0;
    for (int b = 0; b < nb; ++b) profile_host[b] = pr[nb + b] > 0 ? (float)((double)pr[b] * fxi / (double)pr[nb + b]) : 0.0f;
  }
  if (nrange) return fail(c, MPC_ERANGE, "velocities outside the range of the fixed-point cell sums since the last mpc_set_state (PAPER.md:168): results invalid");
  return MPC_OK;
}

int get_cells_impl(mpc_ctx* c, unsigned* count, float* px, float* py, float* pz, float* e2, unsigned* key) {
  const Geo& G = c->G;   // G.s / G.t are still those of the last step
  k_export_cells<<<nblk(G.nkeys, 256), 256, 0, c->stream>>>(G, c->sums, count, px, py, pz, e2);
  LAUNCH_CHECK("k_export_cells");
  if (key && c->n) return launch_keys(c, key);
  return MPC_OK;
}
