"""`-m gpu`: nif_query / nif_query_multi only enqueue work (no sync, no allocation), so they can be captured
in a CUDA graph and replayed; the replay gives the same results as the direct call."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def H():
    import harness
    return harness


@pytest.fixture(scope="module")
def nif():
    import paper_2604_24666_b200 as nif
    return nif


def test_query_and_walk_replay_from_a_cuda_graph(H, nif):
    case = H.make_case(1, n_rays=40_000)
    n = len(case.origin)
    direct = H.run_gpu(case)
    out = nif.alloc_outputs(n, raw_logits=True)
    walk = nif.alloc_walk_outputs(n)
    ws = torch.empty(nif.nif_query_workspace_bytes(n) + 256, dtype=torch.uint8, device="cuda")
    ws = ws[(-ws.data_ptr()) % 256:][:nif.nif_query_workspace_bytes(n)]
    wsm = torch.empty(nif.nif_query_multi_workspace_bytes(n) + 256, dtype=torch.uint8, device="cuda")
    wsm = wsm[(-wsm.data_ptr()) % 256:][:nif.nif_query_multi_workspace_bytes(n)]
    nif.nif_query(case.bvh, case.net, case.origin_d, case.direction_d, out, workspace=ws)      # warm-up outside capture
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        nif.nif_query(case.bvh, case.net, case.origin_d, case.direction_d, out, workspace=ws)
    for v in out.values():
        v.zero_()
    g.replay(); torch.cuda.synchronize()
    for k in ("voxel_id", "t_in", "t_out", "occlusion", "dist_total", "normal", "material_logits", "raw_logits"):
        assert np.array_equal(out[k].cpu().numpy(), direct[k]), k
    # new rays through the same graph: inputs are read at replay time
    case.origin_d.copy_(torch.from_numpy(case.origin[::-1].copy()).cuda())
    case.direction_d.copy_(torch.from_numpy(case.direction[::-1].copy()).cuda())
    g.replay(); torch.cuda.synchronize()
    assert np.array_equal(out["voxel_id"].cpu().numpy(), direct["voxel_id"][::-1])
    assert np.array_equal(out["dist_total"].cpu().numpy(), direct["dist_total"][::-1])
    # the multi-voxel walk: 4 rounds = ~30 launches in one graph
    nif.nif_query_multi(case.bvh, case.net, case.origin_d, case.direction_d, out, walk, 4, workspace=wsm)
    torch.cuda.synchronize()
    ref = {k: v.clone() for k, v in {**out, **walk}.items()}
    g2 = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g2):
        nif.nif_query_multi(case.bvh, case.net, case.origin_d, case.direction_d, out, walk, 4, workspace=wsm)
    for v in list(out.values()) + list(walk.values()):
        v.zero_()
    g2.replay(); torch.cuda.synchronize()
    for k in ("status", "steps", "voxel_id", "occlusion", "dist_accum"):
        got = (walk[k] if k in walk else out[k])
        assert torch.equal(got, ref[k]), k
