// query4.cu -- placeholder until the 4pCF kernels land (S:8(a) A8, A9).
#include "internal.cuh"
void gr_4pcf(gramsci_graph *, int, uint64_t *, int64_t *, double *, double *)
{
    GR_FAIL(GRAMSCI_EINVAL, "4pcf: not implemented yet");
}
