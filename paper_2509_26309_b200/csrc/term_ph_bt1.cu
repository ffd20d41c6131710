// term_ph_bt1.cu -- instantiations of the fused Chebyshev-term kernel (term_ph.cuh) for tiles of 1 interleaved state(s).
#include "term_ph.cuh"

namespace tbpm_detail {
int launch_term_ph_bt1(const TermParams &p, int num_sms, cudaStream_t st, int *grid_out)
{
    return ph::launch_bt<1>(p, num_sms, st, grid_out);
}
}  // namespace tbpm_detail
