// cell.cu -- PROCESS_CELLS as a kernel of its own (see cell.cuh)
#include "cell.cuh"

namespace mpc {

// grid = (mb0 * CTAs-per-brick, mb1, mb2): the brick coordinates come from blockIdx, no division
template <int CT>
__global__ void __launch_bounds__(CT) k_cell(Geo G, int cpb_shift, int ct_shift, u64* __restrict__ sums, float* __restrict__ rec, int zero) {
  __shared__ CellScratch<CT> sh;
  cell_batch<CT>(G, blockIdx.x >> cpb_shift, blockIdx.y, blockIdx.z, (blockIdx.x & ((1u << cpb_shift) - 1u)) << ct_shift, sums, rec, zero, sh);
}

}  // namespace mpc

using namespace mpc;

int launch_cell(mpc_ctx* c, int zero) {
  k_cell<256><<<c->cell_grid, 256, 0, c->stream>>>(c->G, c->cell_cpb_shift, 8, c->sums, c->rec, zero);
  LAUNCH_CHECK("k_cell");
  return MPC_OK;
}
