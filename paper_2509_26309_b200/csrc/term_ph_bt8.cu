// term_ph_bt8.cu -- instantiations of the fused Chebyshev-term kernel (term_ph.cuh) for tiles of 8 interleaved state(s).
#include "term_ph.cuh"

namespace tbpm_detail {
int launch_term_ph_bt8(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out)
{
    return ph::launch_bt<8>(p, num_sms, st, grid_out);
}
}  // namespace tbpm_detail
