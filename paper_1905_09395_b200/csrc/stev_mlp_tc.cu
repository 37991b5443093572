// stev_mlp_tc.cu -- tensor-core (tcgen05 + TMEM) path of the standalone estimator forward pass (row a7).
#include "stev_host.h"

namespace stev {

int estimator_eval_tensor(const stev_estimator *, long long, const float *, float *, int, cudaStream_t) {
  set_error("stev_estimator_eval: tensor-core path not built yet");
  return STEV_EINVAL;
}

}  // namespace stev
