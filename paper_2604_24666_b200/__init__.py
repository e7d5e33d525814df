"""B200-native batched inference of the voxel-deformation-aware neural intersection query
(arxiv 2604.24666).  The product is libnif.so (CUDA, sm_100a; C ABI in include/nif.h); this
package is the thin binding over it.  See DESIGN.md."""
from .binding import (  # noqa: F401
    NIF_F16, NIF_F32, NIF_ENC_COMPOSE, NIF_ENC_CONCAT, NIF_N_OUT, NIF_OCCLUSION_ONLY, NIF_ENGINE_FFMA, NIF_TRAVERSE_ONLY, NIF_TRAVERSE_COHERENT, NIF_TRAVERSE_INCOHERENT, NIF_PROBE_SKIP_GATHER, NIF_DIST_LOG,
    Bvh, Net, NifError, Stage, alloc_outputs, lib,
    nif_build_deformed_bvh, nif_build_bvh_from_lattice, nif_bvh_workspace_bytes, nif_kernel_launch_count, nif_net_create,
    nif_query, nif_query_host, nif_query_host_compact, nif_net_uses_tensor_cores, nif_profile_enable, nif_profile_read, nif_probe_gather, nif_query_last_hit_count, nif_query_workspace_bytes,
    NIF_WALK_MISS, NIF_WALK_HIT, NIF_WALK_MAX_STEPS, alloc_walk_outputs, nif_query_multi, nif_query_multi_workspace_bytes, nif_query_poses, nif_query_poses_workspace_bytes, nif_query_static, NIF_STATIC_MAX_RAYS,
)
