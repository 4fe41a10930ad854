// sps_exact.cu -- exact photometry path (Eq. 4).  [stub: filled in next]
#include "sps_internal.h"
struct ExactState { int dummy; };
sps_status sps_exact_setup(sps_table* t) { t->exact = nullptr; return SPS_OK; }
void sps_exact_teardown(sps_table* t) { (void)t; }
sps_status sps_exact_contract(sps_table*, int64_t, const int*, const int*, const float*, const float*, const float*, bool, cudaStream_t) {
  sps_set_error("exact path not built yet");
  return SPS_EUNSUPPORTED;
}
