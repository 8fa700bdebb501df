// push2.cu -- second-order particles (b2 gather + Esirkepov deposit); see below.
#include "push_common.cuh"

int psc_push_order2(psc_ctx *c, cudaStream_t s) {
  (void)c;
  (void)s;
  return PSC_ERR_UNSUPPORTED;
}
