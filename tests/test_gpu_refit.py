"""`-m gpu`: nif_bvh_refit (new pose, same voxel set, "For each
deformation pose, we build a simple BVH over the deformed voxels") gives bit-for-bit what a fresh
build with that pose gives, and the refitted BVH matches the oracle."""
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


def test_refit_equals_fresh_build_and_the_oracle(oracle, H, P, nif):
    cfg = I.get_config(2)
    poses = I.poses(cfg)
    case = H.make_case(2, n_rays=40_000, pose_index=0)
    for pi in (3, 6, 0):
        pose = poses[pi]
        case.bvh.refit(float(pose[0]), float(pose[1]))
        fresh = H.make_case(2, n_rays=40_000, pose_index=pi, with_net=False)
        assert torch.equal(case.bvh.lattice(), fresh.bvh.lattice())
        a, b = case.bvh.info(), fresh.bvh.info()
        for k in ("n_occupied", "n_nodes", "depth", "theta_max", "bend_k"):
            assert a[k] == b[k], k
        assert np.array_equal(a["lo"], b["lo"]) and np.array_equal(a["hi"], b["hi"])
        # same rays through both
        case.origin, case.direction = fresh.origin, fresh.direction
        case.origin_d, case.direction_d = fresh.origin_d, fresh.direction_d
        case.pose = fresh.pose
        g_refit = H.run_gpu(case)
        fresh.net = case.net
        g_fresh = H.run_gpu(fresh)
        for k in ("voxel_id", "t_in", "t_out", "occlusion", "dist_total", "normal", "material_logits"):
            assert np.array_equal(g_refit[k], g_fresh[k]), (pi, k)
        if pi == 6:
            ref = H.OracleSide(oracle, case).query(np.arange(0, 40_000, 8))
            sub = H.subset(g_refit, np.arange(0, 40_000, 8))
            P.assert_traversal(P.compare_traversal(sub, ref))
            P.assert_network(P.compare_network(sub, ref, fp16=True), fp16=True)


def test_refit_rejects_a_folding_pose_and_keeps_the_old_one(H, nif):
    case = H.make_case(0)
    before = H.run_gpu(case)
    with pytest.raises(nif.NifError) as e:
        case.bvh.refit(0.0, 2.0)                      # k*y >= 1 inside the sphere of radius 0.8
    assert e.value.status == -3
    after = H.run_gpu(case)
    for k in ("voxel_id", "t_in", "t_out", "occlusion"):
        assert np.array_equal(before[k], after[k]), k
