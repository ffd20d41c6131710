// term_pair_bt2.cu -- instantiations of the two-terms-per-sweep kernel (term_pair.cuh) for tiles of 2 interleaved states.
#include "term_pair.cuh"

namespace tbpm_detail {
int launch_term_pair_bt2(const PairParams &q, int num_sms, cudaStream_t st, int *grid_out)
{
    return pair::launch_pair_bt<2>(q, num_sms, st, grid_out);
}
}  // namespace tbpm_detail
