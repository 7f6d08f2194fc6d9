// placeholder during bring-up
#include "common.cuh"
df_status ann_bf16_create(df_ann*, const float* const*, const float* const*) { return df_set_error(DF_ERR_UNSUPPORTED, "bf16 path not built yet"); }
void ann_bf16_destroy(df_ann*) {}
size_t ann_bf16_workspace(const df_ann*, long long) { return 0; }
df_status launch_ann_bf16(const df_ann*, const df_mech*, long long, long long, const float*, const float*, const float*, float*, float*, void*, size_t, cudaStream_t) { return df_set_error(DF_ERR_UNSUPPORTED, "bf16 path not built yet"); }
