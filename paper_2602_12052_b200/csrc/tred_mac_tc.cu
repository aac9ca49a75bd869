// Tensor-core variant of the spectrum product (step (b) of tred_conv.cu).  Placeholder
// until the tcgen05 kernel lands: reports "unsupported" so that tred_convolve uses the
// fp32 FMA kernel (mac_mode 2 then fails loudly).
#include "tred_common.cuh"

int tred_mac_tc(tred_ctx*, const float*, const float*, const float*, float*, int, int, cudaStream_t) {
  return TRED_EUNSUPPORTED;
}
