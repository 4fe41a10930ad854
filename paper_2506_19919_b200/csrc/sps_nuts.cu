// sps_nuts.cu -- NUTS engine (a13).  [stub: filled in next]
#include "sps_sampler.cuh"
sps_status nuts_run(sps_table*, const PriorDev&, const sps_hmc_config*, HmcProblem&, ChainState&, float*, cudaStream_t) {
  sps_set_error("NUTS not built yet");
  return SPS_EUNSUPPORTED;
}
