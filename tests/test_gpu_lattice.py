"""`-m gpu` parity for deformations supplied as a corner lattice (nif_build_bvh_from_lattice; PAPER.md:39
"user-specified deformation"; R27): traversal over the user's lattice, map back with the
voxel-local trilinear inverse, network, heads, hit positions and the multi-voxel walk, against the
oracle's O7b path on the same lattice."""
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


def _lattice_case(H, nif, oracle, cfg_id, n_rays, lattice):
    """A harness Case whose BVH comes from `lattice`; rays aimed at that lattice's bounding box."""
    cfg = I.get_config(cfg_id)
    occ = I.occupancy(cfg)
    bvh = nif.nif_build_bvh_from_lattice(cfg.nv, torch.from_numpy(occ).cuda(), torch.from_numpy(lattice).cuda(),
                                         max_occupied=int(occ.sum()))
    info = bvh.info()
    o, d = I.rays(cfg, 0, info["lo"], info["hi"], n=n_rays)
    params = I.net_params(cfg, "varpres")
    case = H.Case(cfg, np.zeros(2, np.float32), occ, params, bvh, H.make_net(params), o, d,
                  torch.from_numpy(o).cuda(), torch.from_numpy(d).cuda())
    obvh = oracle.bvh_build(cfg.nv, occ, lattice)
    return case, obvh


def _oracle_query(oracle, case, obvh, lattice, idx=None, **kw):
    o = case.origin if idx is None else case.origin[idx]
    d = case.direction if idx is None else case.direction[idx]
    return oracle.query(case.cfg.nv, case.occ, lattice, obvh, case.pose, case.params, o, d, lattice_inverse=True, **kw)


@pytest.mark.parametrize("cfg_id,n_rays", [(0, None), (1, 30_000), (4, 12_000)])
def test_wavy_lattice_query(oracle, H, P, nif, cfg_id, n_rays):
    cfg = I.get_config(cfg_id)
    lattice = I.wavy_lattice(cfg.nv, seed=cfg_id)
    case, obvh = _lattice_case(H, nif, oracle, cfg_id, n_rays, lattice)
    assert torch.equal(case.bvh.lattice(), torch.from_numpy(lattice).cuda())
    fp16 = cfg.net.dtype == "f16"
    idx = None
    if cfg_id == 4:
        t = H.run_gpu(case, flags=nif.NIF_TRAVERSE_ONLY, raw_logits=False)
        hit = np.nonzero(t["voxel_id"] >= 0)[0]
        idx = np.unique(np.concatenate([hit[:: max(1, len(hit) // 800)], np.arange(0, len(case.origin), 173)]))
    ref = _oracle_query(oracle, case, obvh, lattice, idx, hit_positions=True)
    engines = [0, nif.NIF_ENGINE_FFMA] if fp16 else [0]
    for fl in engines:
        gpu = H.run_gpu(case, flags=fl, hit_positions=True)
        if idx is not None:
            gpu = H.subset(gpu, idx)
        P.assert_traversal(P.compare_traversal(gpu, ref))
        m = P.compare_network(gpu, ref, fp16=fp16)
        P.assert_network(m, fp16=fp16)
        assert m["n_hit"] > 300
        hit = ref["voxel_id"] >= 0
        tol = 1e-2 if fp16 else 1e-5
        ell = (ref["t_out"][hit] - ref["t_in"][hit]).astype(np.float64)
        e = np.abs(gpu["hit_position_rest"][hit].astype(np.float64) - ref["hit_position_rest"][hit]).max(1)
        assert (e <= 3 * (tol * ell + 1e-5 * ref["t_out"][hit]) + tol * 0.5 + 2e-5).all(), e.max()


def test_closed_form_lattice_fed_as_user_lattice(oracle, H, P, nif):
    """The same object posed two ways: closed form (nif_build_deformed_bvh) and its lattice handed over
    as a user lattice.  Traversal is identical; the rest points differ by the O(h^2) of R27 only."""
    cfg = I.get_config(1)
    pose = I.poses(cfg)[0]
    a = H.make_case(1, n_rays=30_000)
    lattice = oracle.deform_lattice(cfg.nv, float(pose[0]), float(pose[1]))
    assert torch.equal(a.bvh.lattice(), torch.from_numpy(lattice).cuda())         # GPU lattice == oracle lattice, bit for bit
    b, obvh = _lattice_case(H, nif, oracle, 1, 30_000, lattice)
    ga = H.run_gpu(a, hit_positions=True); gb = H.run_gpu(b, hit_positions=True)
    for k in ("voxel_id", "t_in", "t_out", "hit_position"):
        assert np.array_equal(ga[k], gb[k], equal_nan=True) or k == "hit_position", k
    hit = ga["voxel_id"] >= 0
    h = 2.0 / cfg.nv
    dev = np.abs(ga["hit_position_rest"][hit] - gb["hit_position_rest"][hit]).max()
    assert 0 < dev < 0.25 * h, dev / h            # measured 0.11 h (bend k = 0.8 on 64^3); a wrong voxel is >= 1 h off


def test_refit_lattice_and_walk(oracle, H, P, nif):
    import test_gpu_walk as W
    cfg = I.get_config(1)
    lat0 = I.wavy_lattice(cfg.nv, seed=7)
    lat1 = I.wavy_lattice(cfg.nv, seed=8)
    case, _ = _lattice_case(H, nif, oracle, 1, 20_000, lat0)
    case.bvh.refit_lattice(torch.from_numpy(lat1).cuda())
    fresh, obvh = _lattice_case(H, nif, oracle, 1, 20_000, lat1)
    assert torch.equal(case.bvh.lattice(), fresh.bvh.lattice())
    case.origin, case.direction, case.origin_d, case.direction_d = fresh.origin, fresh.direction, fresh.origin_d, fresh.direction_d
    g0 = H.run_gpu(case); g1 = H.run_gpu(fresh)
    for k in ("voxel_id", "t_in", "t_out", "occlusion", "dist_total"):
        assert np.array_equal(g0[k], g1[k]), k
    # multi-voxel walk on the lattice pose against the oracle's walk with the O7b inverse
    K = 5
    gpu = W.run_walk(nif, fresh, K)
    ref = oracle.query_multi(cfg.nv, fresh.occ, lat1, obvh, fresh.pose, fresh.params, fresh.origin, fresh.direction, K,
                             lattice_inverse=True)
    tid, tz = oracle.walk_trace(cfg.nv, fresh.occ, lat1, obvh, fresh.pose, fresh.params, fresh.origin, fresh.direction, K,
                                lattice_inverse=True)
    valid = tid >= 0
    rms = float(np.sqrt((tz[valid].astype(np.float64) ** 2).mean()))
    near = valid & (np.abs(tz) <= 5e-3 * rms)
    taken = np.arange(K)[None, :] < ref["steps"][:, None]
    clear = ~(near & taken).any(1)
    assert clear.mean() > 0.97
    for k in ("status", "steps", "voxel_id"):
        assert np.array_equal(gpu[k][clear], ref[k][clear]), k
    g = {k: v[clear] for k, v in gpu.items()}; r = {k: v[clear] for k, v in ref.items()}
    P.assert_traversal(P.compare_traversal(g, r))
    P.assert_network(P.compare_network(g, r, fp16=True), fp16=True)
    assert (r["steps"] > 1).sum() > 100
