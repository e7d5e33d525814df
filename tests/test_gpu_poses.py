"""`-m gpu`: nif_query_poses (several poses of one object in one query, a pose id per ray; SURVEY 8(f) f2,
BASELINE.json:9) gives, ray for ray, what one nif_query per pose gives -- and with it the oracle's result."""
import numpy as np
import pytest
import torch

import nif_inputs as I

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def H():
    import harness
    return harness


@pytest.fixture(scope="module")
def P():
    import parity
    return parity


@pytest.fixture(scope="module")
def nif():
    import paper_2604_24666_b200 as nif
    return nif


def _batch(H, cfg_id, pose_indices, n_per_pose, seed=0):
    cases = [H.make_case(cfg_id, n_rays=n_per_pose, pose_index=pi, with_net=(k == 0)) for k, pi in enumerate(pose_indices)]
    for c in cases[1:]:
        c.net = cases[0].net
    o = np.concatenate([c.origin for c in cases]); d = np.concatenate([c.direction for c in cases])
    pid = np.concatenate([np.full(len(c.origin), k, np.int32) for k, c in enumerate(cases)])
    perm = np.random.default_rng(seed).permutation(len(o))          # poses interleaved at random
    return cases, np.ascontiguousarray(o[perm]), np.ascontiguousarray(d[perm]), np.ascontiguousarray(pid[perm]), perm


def _run_poses(nif, cases, o, d, pid, flags=0, hit_positions=False):
    n = len(o)
    out = nif.alloc_outputs(n, raw_logits=True, hit_positions=hit_positions)
    for v in out.values():
        v.fill_(float("nan") if v.dtype.is_floating_point else -7)
    nif.nif_query_poses([c.bvh for c in cases], cases[0].net, torch.from_numpy(o).cuda(), torch.from_numpy(d).cuda(),
                        torch.from_numpy(pid).cuda(), out, flags=flags)
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in out.items()}


@pytest.mark.parametrize("cfg_id,flags_name", [(2, "default"), (2, "ffma"), (3, "occlusion_only"), (2, "coherent"), (2, "incoherent")])
def test_batched_poses_equal_one_query_per_pose(oracle, H, P, nif, cfg_id, flags_name):
    flags = {"default": 0, "ffma": nif.NIF_ENGINE_FFMA, "occlusion_only": nif.NIF_OCCLUSION_ONLY,
             "coherent": nif.NIF_TRAVERSE_COHERENT, "incoherent": nif.NIF_TRAVERSE_INCOHERENT}[flags_name]
    pose_indices = [0, 3, 5, 6]
    cases, o, d, pid, perm = _batch(H, cfg_id, pose_indices, 12_000)
    hp = flags_name == "default"
    got = _run_poses(nif, cases, o, d, pid, flags=flags, hit_positions=hp)
    inv = np.argsort(perm)
    keys = ["voxel_id", "t_in", "t_out", "occlusion"]
    if not (flags & nif.NIF_OCCLUSION_ONLY):
        keys += ["distance", "dist_total", "normal", "albedo", "material_logits", "raw_logits"]
    if hp:
        keys += ["hit_position", "hit_position_rest"]
    off = 0
    for k, c in enumerate(cases):
        single = H.run_gpu(c, flags=flags, hit_positions=hp)
        m = len(c.origin)
        sel = inv[off:off + m]                      # positions of this pose's rays in the batched call
        off += m
        for key in keys:
            assert np.array_equal(got[key][sel], single[key], equal_nan=True), (k, key)
    # and against the oracle directly, on one pose's rays
    c = cases[2]
    sel = inv[2 * 12_000:3 * 12_000]              # all of this pose's rays: the argmax gate needs thousands of hits
    ref = H.OracleSide(oracle, c).query(occlusion_only=bool(flags & nif.NIF_OCCLUSION_ONLY))
    sub = {k: v[sel] for k, v in got.items()}
    P.assert_traversal(P.compare_traversal(sub, ref))
    oo = bool(flags & nif.NIF_OCCLUSION_ONLY)
    P.assert_network(P.compare_network(sub, ref, fp16=True, occlusion_only=oo), fp16=True, occlusion_only=oo)


def test_batched_lattice_poses(oracle, H, nif):
    cfg = I.get_config(1)
    occ = I.occupancy(cfg)
    occ_d = torch.from_numpy(occ).cuda()
    lats = [I.wavy_lattice(cfg.nv, seed=s) for s in (11, 12, 13)]
    bvhs = [nif.nif_build_bvh_from_lattice(cfg.nv, occ_d, torch.from_numpy(l).cuda(), max_occupied=int(occ.sum())) for l in lats]
    params = I.net_params(cfg, "varpres")
    net = H.make_net(params)
    cases = []
    for b in bvhs:
        info = b.info()
        o, d = I.rays(cfg, 0, info["lo"], info["hi"], n=15_000)
        cases.append(H.Case(cfg, np.zeros(2, np.float32), occ, params, b, net, o, d, torch.from_numpy(o).cuda(), torch.from_numpy(d).cuda()))
    o = np.concatenate([c.origin for c in cases]); d = np.concatenate([c.direction for c in cases])
    pid = np.concatenate([np.full(len(c.origin), k, np.int32) for k, c in enumerate(cases)])
    got = _run_poses(nif, cases, o, d, pid, hit_positions=True)
    off = 0
    for c in cases:
        single = H.run_gpu(c, hit_positions=True)
        m = len(c.origin)
        for key in ("voxel_id", "t_in", "occlusion", "dist_total", "normal", "hit_position_rest"):
            assert np.array_equal(got[key][off:off + m], single[key], equal_nan=True), key
        off += m


def test_query_poses_argument_validation(H, nif):
    a = H.make_case(0)
    b = H.make_case(1, n_rays=100, with_net=False)          # different grid size
    n = len(a.origin)
    out = nif.alloc_outputs(n)
    pid = torch.zeros(n, dtype=torch.int32, device="cuda")
    with pytest.raises(nif.NifError):
        nif.nif_query_poses([a.bvh, b.bvh], a.net, a.origin_d, a.direction_d, pid, out)
    with pytest.raises(nif.NifError):
        nif.nif_query_poses([], a.net, a.origin_d, a.direction_d, pid, out)
    nif.nif_query_poses([a.bvh], a.net, a.origin_d, a.direction_d, pid, out)      # one pose = nif_query
    torch.cuda.synchronize()
    single = H.run_gpu(a)
    assert np.array_equal(out["voxel_id"].cpu().numpy(), single["voxel_id"])
    assert np.array_equal(out["dist_total"].cpu().numpy(), single["dist_total"])


def test_full_size_config2_batched_equals_per_pose(oracle, H, P, nif):
    """BASELINE.json configs[2] at full size in the launch configuration bench.py times (one nif_query_poses
    over 8 x 2^20 rays): bit-identical, ray for ray, to one nif_query per pose; a seeded sample of one pose
    is recomputed by the oracle."""
    cfg = I.get_config(2)
    cases = [H.make_case(2, pose_index=pi, with_net=(pi == 0)) for pi in range(cfg.n_poses)]
    for c in cases[1:]:
        c.net = cases[0].net
    n = cfg.rays_per_pose
    o = torch.cat([c.origin_d for c in cases]); d = torch.cat([c.direction_d for c in cases])
    pid = torch.cat([torch.full((n,), k, dtype=torch.int32, device="cuda") for k in range(cfg.n_poses)])
    out = nif.alloc_outputs(n * cfg.n_poses)
    nif.nif_query_poses([c.bvh for c in cases], cases[0].net, o, d, pid, out)
    torch.cuda.synchronize()
    single = nif.alloc_outputs(n)
    for k, c in enumerate(cases):
        nif.nif_query(c.bvh, c.net, c.origin_d, c.direction_d, single)
        torch.cuda.synchronize()
        for key in ("voxel_id", "t_in", "t_out", "occlusion", "dist_total", "normal", "material_logits"):
            assert torch.equal(out[key][k * n:(k + 1) * n], single[key]), (k, key)
    k = 5
    rng = np.random.default_rng(2)
    hit = np.nonzero(out["voxel_id"][k * n:(k + 1) * n].cpu().numpy() >= 0)[0]
    idx = np.sort(rng.choice(hit, 8000, replace=False))      # the 99.9 % argmax gate needs thousands of hits
    ref = H.OracleSide(oracle, cases[k]).query(idx)
    got = {key: v[k * n:(k + 1) * n].cpu().numpy()[idx] for key, v in out.items()}
    P.assert_traversal(P.compare_traversal(got, ref))
    P.assert_network(P.compare_network(got, ref, fp16=True), fp16=True)
