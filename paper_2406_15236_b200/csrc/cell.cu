// cell.cu -- PROCESS_CELLS as a kernel of its own (see cell.cuh)
#include "cell.cuh"

namespace mpc {

// grid = (mb0 * CTAs-per-brick, mb1, mb2): the brick coordinates come from blockIdx, no division
constexpr int PF_CTAS = 1024;   // about the number of resident CTAs (148 SMs x 5..6) and a bit
template <int CT, bool SUB>
__global__ void __launch_bounds__(CT) k_cell(Geo G, int cpb_shift, int ct_shift, u64* __restrict__ sums, float* __restrict__ rec, int zero, uint32_t* __restrict__ counts, int handover) {
  // CTAs are dispatched in the order of their linear index L, and CTA L reads the CT cells from key L * CT on: pull the
  // sums of the CTA PF_CTAS further on into L2 now (every thread of this kernel loads once, computes for ~400
  // instructions, stores once: it is bound by the latency of that first load)
  if (threadIdx.x == 0 && G.bs[0] + G.bs[1] + G.bs[2] >= ct_shift) {   // bricks of at least CT cells: key of CTA L = L * CT
    const size_t L = blockIdx.x + (size_t)gridDim.x * (blockIdx.y + (size_t)gridDim.y * blockIdx.z) + PF_CTAS;
    if (L < (size_t)gridDim.x * gridDim.y * gridDim.z) {
      const uint32_t bytes = (uint32_t)(CT * G.sw * 8);
      asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(sums + L * (size_t)(CT * G.sw)), "r"(bytes));
    }
  }
  cell_batch<SUB>(G, blockIdx.x >> cpb_shift, blockIdx.y, blockIdx.z, (blockIdx.x & ((1u << cpb_shift) - 1u)) << ct_shift, sums, rec, zero, counts, handover);
}

}  // namespace mpc

using namespace mpc;

// (c, k) of the thermostat draw for N_c < MT_TABLE (reading U6), with the IEEE operations the kernels use
void fill_mt_table(float* host) {
  for (uint32_t nc = 0; nc < (uint32_t)MT_TABLE; ++nc) {
    host[2 * nc] = host[2 * nc + 1] = 0.0f;
    if (nc >= 2u) mt_shape_host(nc, host[2 * nc], host[2 * nc + 1]);
  }
}

int launch_cell(mpc_ctx* c, int zero, uint32_t* counts, bool handover) {
  if (c->G.sub) k_cell<256, true><<<c->cell_grid, 256, 0, c->stream>>>(c->G, c->cell_cpb_shift, 8, c->sums, c->rec, zero, counts, handover ? 1 : 0);
  else k_cell<256, false><<<c->cell_grid, 256, 0, c->stream>>>(c->G, c->cell_cpb_shift, 8, c->sums, c->rec, zero, counts, 0);
  LAUNCH_CHECK("k_cell");
  return MPC_OK;
}
