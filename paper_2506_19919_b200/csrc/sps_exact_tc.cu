// sps_exact_tc.cu -- tcgen05 / TMA / TMEM kernels of the exact path.  [stub: filled in next]
#include "sps_exact.cuh"
sps_status sps_exact_tc_setup(sps_table* t) { t->exact->use_tc = false; t->exact->tc = nullptr; return SPS_OK; }
void sps_exact_tc_teardown(sps_table*) {}
sps_status sps_exact_tc_forward(sps_table*, int64_t, const int*, cudaStream_t) { sps_set_error("tcgen05 path not built"); return SPS_EUNSUPPORTED; }
sps_status sps_exact_tc_backward(sps_table*, int64_t, const int*, cudaStream_t) { sps_set_error("tcgen05 path not built"); return SPS_EUNSUPPORTED; }
