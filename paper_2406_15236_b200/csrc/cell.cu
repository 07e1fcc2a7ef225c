// cell.cu -- PROCESS_CELLS as a kernel of its own (see cell.cuh)
#include "cell.cuh"

namespace mpc {

// grid = (mb0 * CTAs-per-brick, mb1, mb2): the brick coordinates come from blockIdx, no division
template <int CT>
__global__ void __launch_bounds__(CT) k_cell(Geo G, int cpb_shift, int ct_shift, u64* __restrict__ sums, float* __restrict__ rec, int zero, uint32_t* __restrict__ counts) {
  cell_batch(G, blockIdx.x >> cpb_shift, blockIdx.y, blockIdx.z, (blockIdx.x & ((1u << cpb_shift) - 1u)) << ct_shift, sums, rec, zero, counts);
}

}  // namespace mpc

using namespace mpc;

// c = 1 / sqrt(9 d) of the thermostat draw for N_c < MT_TABLE (reading U6), with the IEEE operations the kernels use
void fill_mt_table(float* host) {
  host[0] = host[1] = 0.0f;
  for (uint32_t nc = 2; nc < (uint32_t)MT_TABLE; ++nc) host[nc] = mt_c_host(nc);
}

int launch_cell(mpc_ctx* c, int zero, uint32_t* counts) {
  k_cell<256><<<c->cell_grid, 256, 0, c->stream>>>(c->G, c->cell_cpb_shift, 8, c->sums, c->rec, zero, counts);
  LAUNCH_CHECK("k_cell");
  return MPC_OK;
}
