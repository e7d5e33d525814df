"""`-m gpu`: nif_query / nif_query_multi / nif_query_poses only enqueue work (no sync, no allocation), so they can be captured
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


def test_query_poses_replays_from_a_cuda_graph(H, nif):
    """nif_query_poses copies nothing from host memory (pose descriptors travel as a kernel parameter), so it
    can be captured; a replay traces new rays against the captured poses, and it must keep doing so after the
    capturing call's stack frame is long gone (round 1 uploaded the descriptors from a stack array)."""
    import nif_inputs as I
    cfg = I.get_config(2)
    occ = I.occupancy(cfg)
    n_poses, n_per = 3, 20_000
    occ_d = torch.from_numpy(occ).cuda()
    poses = I.poses(cfg)[:n_poses]
    bvhs = [nif.nif_build_deformed_bvh(cfg.nv, occ_d, float(p[0]), float(p[1]), max_occupied=int(occ.sum())) for p in poses]
    rays = [I.rays(cfg, i, b.info()["lo"], b.info()["hi"], n=n_per) for i, b in enumerate(bvhs)]
    o = torch.from_numpy(np.concatenate([r[0] for r in rays])).cuda()
    d = torch.from_numpy(np.concatenate([r[1] for r in rays])).cuda()
    pid = torch.arange(n_poses, dtype=torch.int32, device="cuda").repeat_interleave(n_per)
    params = I.net_params(cfg, "varpres")
    net = H.make_net(params)
    n = n_poses * n_per
    out = nif.alloc_outputs(n, raw_logits=True)
    nb = nif.nif_query_poses_workspace_bytes(n)
    ws = torch.empty(nb + 256, dtype=torch.uint8, device="cuda")
    ws = ws[(-ws.data_ptr()) % 256:][:nb]
    nif.nif_query_poses(bvhs, net, o, d, pid, out, workspace=ws)
    torch.cuda.synchronize()
    direct = {k: v.clone() for k, v in out.items()}
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        nif.nif_query_poses(bvhs, net, o, d, pid, out, workspace=ws)

    def churn_the_stack(depth=50):          # overwrite whatever host stack the capturing call used
        junk = np.random.default_rng(depth).random(4096)
        return junk.sum() + (churn_the_stack(depth - 1) if depth else 0.0)
    churn_the_stack()
    for _ in range(2):
        for v in out.values():
            v.zero_()
        ws.zero_()
        g.replay(); torch.cuda.synchronize()
        for k in ("voxel_id", "t_in", "t_out", "occlusion", "dist_total", "normal", "material_logits", "raw_logits"):
            assert torch.equal(out[k], direct[k]), k
    # new rays (the poses' rays swapped round) through the same graph
    perm = torch.arange(n, device="cuda").flip(0)
    o.copy_(o[perm].clone()); d.copy_(d[perm].clone()); pid.copy_(pid[perm].clone())
    g.replay(); torch.cuda.synchronize()
    assert torch.equal(out["voxel_id"], direct["voxel_id"][perm])
    assert torch.equal(out["raw_logits"], direct["raw_logits"][perm])
