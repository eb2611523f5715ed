// ms_mlp_tc.cuh -- stage (d), bf16 tensor-core path (tcgen05 + TMEM, weights staged by bulk copy).
#pragma once
#include "ms_internal.cuh"

struct MsTcWeights {
  bool valid = false;          // the MLP shape is covered by the tensor kernels and the image is built
  void *image = nullptr;       // device: [N][bytes_per_prim] packed shared-memory image (bf16 + fp32 bias)
  size_t bytes_per_prim = 0;
  int k1_pad = 0;              // padded input width (multiple of 16)
  int n_out_pad = 0;           // padded head width (multiple of 16)
  int variant = -1;            // kernel instantiation
};

// Packs host fp32 weight values (bf16-representable matrices, fp32 biases) into the UMMA
// shared-memory image.  Leaves out->valid == false (and returns MS_OK) if the shape is not covered.
int ms_tc_pack(const MsMlpShape &shape, int n_prims, const float *weights, MsTcWeights *out);
void ms_tc_free(MsTcWeights *w);
cudaError_t ms_mlp_tc(const MsTcWeights &w, const MsMlpArgs &a, cudaStream_t s);
