// ms_mlp_tc.cu -- placeholder until the tcgen05 kernel lands: no shape is covered yet.
#include "ms_mlp_tc.cuh"

int ms_tc_pack(const MsMlpShape &, int, const float *, MsTcWeights *out) {
  out->valid = false;
  return MS_OK;
}
void ms_tc_free(MsTcWeights *w) {
  if (w->image) cudaFree(w->image);
  w->image = nullptr;
  w->valid = false;
}
cudaError_t ms_mlp_tc(const MsTcWeights &, const MsMlpArgs &, cudaStream_t) { return cudaErrorNotSupported; }
