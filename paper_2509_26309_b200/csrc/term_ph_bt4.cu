// term_ph_bt4.cu -- instantiations of the fused Chebyshev-term kernel (term_ph.cuh) for tiles of 4 interleaved state(s).
#include "term_ph.cuh"

namespace tbpm_detail {
int launch_term_ph_bt4(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out)
{
    return ph::launch_bt<4>(p, num_sms, st, grid_out);
}
}  // namespace tbpm_detail
