// Block-id check (include/msa.h msa_check_block_ids; "block ids are validated only in a debug mode (they
// live on device)").  One small kernel over the block-table entries a plan refers to -- the PAGED virtual blocks of a
// forward plan, its write-back destinations, the copy units of an append plan -- never over entries the plan does not use,
// which may legitimately hold stale ids.  flag = smallest block-table index whose id is outside [0, num_blocks), else -1.
#include "msa_kernels.h"

namespace msa {

__global__ void __launch_bounds__(256) msa_check_ids_kernel(const CheckParams P)
{
    const int n_total = P.n_vblocks + P.n_vb_dst + P.n_units;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_total; i += gridDim.x * blockDim.x) {
        int bt_index = -1;
        if (i < P.n_vblocks) {
            const VBlock vb = P.vblocks[i];
            if (vb.paged && vb.nvalid > 0) bt_index = vb.src;
        } else if (i < P.n_vblocks + P.n_vb_dst) {
            bt_index = P.vb_dst[i - P.n_vblocks];                   // -1: this virtual block is not written back
        } else {
            bt_index = P.units[i - P.n_vblocks - P.n_vb_dst].bt_index;
        }
        if (bt_index < 0) continue;
        const int64_t id = P.block_table[bt_index];
        // the flag starts as 0xffffffff (-1): the unsigned minimum is the smallest offending index, or stays -1
        if (id < 0 || id >= P.num_blocks) atomicMin(reinterpret_cast<unsigned int *>(P.flag), static_cast<unsigned int>(bt_index));
    }
}

// reset: start the flag at -1 (a second launch that adds another set of entries to the same verdict passes false)
cudaError_t launch_check_ids(const CheckParams &p, bool reset, cudaStream_t stream)
{
    cudaError_t e = reset ? cudaMemsetAsync(p.flag, 0xff, sizeof(int32_t), stream) : cudaSuccess;
    if (e != cudaSuccess) return e;
    const int n_total = p.n_vblocks + p.n_vb_dst + p.n_units;
    if (n_total <= 0) return cudaSuccess;
    const int grid = (n_total + 255) / 256 < 592 ? (n_total + 255) / 256 : 592;
    msa_check_ids_kernel<<<grid, 256, 0, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace msa
