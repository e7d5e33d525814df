// nif_fused_tc.cu -- placeholder until the tcgen05 fused encode+MLP kernel lands (next commit).
#include "nif_common.cuh"
int nif_tc_supported(const nif_net_desc*) { return 0; }
int nif_tc_pack_weights(nif_net*, cudaStream_t) { return NIF_ERR_UNSUPPORTED; }
int nif_launch_fused_tc(const nif_bvh*, const nif_net*, const nif_ray_batch*, const nif_query_out*,
                        NifQueryScratch*, const int32_t*, unsigned, cudaStream_t) { return NIF_ERR_UNSUPPORTED; }
