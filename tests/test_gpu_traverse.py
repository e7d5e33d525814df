"""`-m gpu` parity: steps (a0) build and (a1) traversal of the CUDA path against the oracle,
through the C ABI.  Ids and hit flags bit-exact, t within 1e-5 relative (BASELINE.json:5)."""
import math

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


def _trav(H, case, flags=0):
    import paper_2604_24666_b200 as nif
    return H.run_gpu(case, flags=nif.NIF_TRAVERSE_ONLY | flags, raw_logits=False)


LATTICE_CASES = [(0, 0), (1, 0), (4, 0), (5, 0)] + [(2, i) for i in range(8)]


@pytest.mark.parametrize("cfg_id,pose_index", LATTICE_CASES)
def test_deformed_lattice_matches_oracle(oracle, H, cfg_id, pose_index):
    # both sides produce the CORRECTLY ROUNDED fp32 value of the closed form (R28; oracle O2x:
    # binary128, here: fp64 with a double-double fallback near fp32 midpoints): not one entry may differ
    case = H.make_case(cfg_id, n_rays=16, pose_index=pose_index, with_net=False)
    got = case.bvh.lattice().cpu().numpy()
    want = oracle.deform_lattice(case.cfg.nv, float(case.pose[0]), float(case.pose[1]))
    assert int((got.view(np.int32) != want.view(np.int32)).sum()) == 0
    info = case.bvh.info()
    assert info["n_occupied"] == int(case.occ.sum())
    obvh = oracle.bvh_build(case.cfg.nv, case.occ, want)
    lo, hi = obvh.bounds()
    assert np.array_equal(lo, info["lo"]) and np.array_equal(hi, info["hi"])


@pytest.mark.parametrize("pose", [(3.0, -0.7), (-2.0, 0.9), (0.0, 0.0), (1e-3, 2e-6), (2.5, 0.0), (math.pi, 1.2)])
def test_deformed_lattice_exact_on_odd_poses(oracle, H, pose):
    # negative parameters, a non-power-of-two lattice (fp64-rounded rest coordinates), signed zeros
    cfg = I.scaled(I.get_config(0), nv=12)
    occ = np.zeros(12 ** 3, np.uint8); occ[:100] = 1        # low voxels only: no fold-over check for k*y
    case = H.make_case(0, n_rays=16, with_net=False, cfg=cfg, occ=occ, pose=list(pose))
    got = case.bvh.lattice().cpu().numpy()
    want = oracle.deform_lattice(12, float(np.float32(pose[0])), float(np.float32(pose[1])))
    assert np.array_equal(got.view(np.int32), want.view(np.int32))


def test_identity_pose_lattice_is_rest_lattice(H):
    cfg = I.get_config(0)
    case = H.make_case(0, n_rays=16, with_net=False, pose=[0.0, 0.0])
    nv = cfg.nv
    lat = case.bvh.lattice().cpu().numpy().reshape(nv + 1, nv + 1, nv + 1, 3)
    c = ((2.0 * np.arange(nv + 1) - nv) / nv).astype(np.float32)
    assert np.array_equal(lat[..., 0], np.broadcast_to(c[None, None, :], lat.shape[:3]))
    assert np.array_equal(lat[..., 1], np.broadcast_to(c[None, :, None], lat.shape[:3]))
    assert np.array_equal(lat[..., 2], np.broadcast_to(c[:, None, None], lat.shape[:3]))


def test_traversal_config0_all_rays_vs_brute_force_definition(oracle, H, P):
    case = H.make_case(0, with_net=False)
    gpu = _trav(H, case)
    lat = oracle.deform_lattice(case.cfg.nv, *map(float, case.pose))
    vid, ti, to = oracle.traverse_brute(case.cfg.nv, case.occ, lat, case.origin, case.direction)
    m = P.compare_traversal(gpu, {"voxel_id": vid, "t_in": ti, "t_out": to})
    P.assert_traversal(m)
    assert m["t_in_bit_mismatch"] == 0 and m["t_out_bit_mismatch"] == 0, m
    assert gpu["n_hit_counter"] == 0        # TRAVERSE_ONLY does not compact


@pytest.mark.parametrize("seed", range(4))
def test_traversal_random_grids_vs_brute_force(oracle, H, P, seed):
    rng = np.random.default_rng(200 + seed)
    nv = [8, 8, 6, 12][seed]                      # includes non-power-of-two lattices
    occ = I.random_occupancy(nv, float(rng.uniform(0.05, 0.6)), seed)
    pose = [float(rng.uniform(0, math.pi / 2)), float(rng.uniform(0, 0.9))]
    cfg = I.scaled(I.get_config(0), nv=nv)
    case = H.make_case(0, n_rays=16, with_net=False, cfg=cfg, occ=occ, pose=pose)
    lo, hi = case.bvh.info()["lo"], case.bvh.info()["hi"]
    n = 3000
    o1 = rng.standard_normal((n, 3)); o1 *= 3.0 / np.linalg.norm(o1, axis=1, keepdims=True)
    d1 = rng.uniform(lo, hi, (n, 3)) - o1
    o2 = rng.uniform(lo, hi, (n, 3)); d2 = rng.standard_normal((n, 3))
    o3 = rng.uniform(lo, hi, (333, 3)); d3 = np.eye(3)[rng.integers(0, 3, 333)] * rng.choice([-1, 1], (333, 1))
    o = np.concatenate([o1, o2, o3]); d = np.concatenate([d1, d2, d3])
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    case.origin = o.astype(np.float32); case.direction = d.astype(np.float32)
    case.origin_d = torch.from_numpy(case.origin).cuda(); case.direction_d = torch.from_numpy(case.direction).cuda()
    gpu = _trav(H, case)
    lat = oracle.deform_lattice(nv, *pose)
    vid, ti, to = oracle.traverse_brute(nv, occ, lat, case.origin, case.direction)
    m = P.compare_traversal(gpu, {"voxel_id": vid, "t_in": ti, "t_out": to})
    P.assert_traversal(m)
    assert m["t_in_bit_mismatch"] == 0 and m["t_out_bit_mismatch"] == 0, m
    assert m["n_hit"] > 500


def test_tie_lowest_id_and_face_plane_ray(oracle, H):
    # same construction as tests/test_oracle_traverse.py: the ray lies in a lattice plane
    nv = 4
    cfg = I.scaled(I.get_config(0), nv=nv)
    case = H.make_case(0, n_rays=16, with_net=False, cfg=cfg, occ=np.ones(nv ** 3, np.uint8), pose=[0.0, 0.0])
    case.origin = np.array([[-3.0, 0.0, 0.25]], np.float32); case.direction = np.array([[1.0, 0.0, 0.0]], np.float32)
    case.origin_d = torch.from_numpy(case.origin).cuda(); case.direction_d = torch.from_numpy(case.direction).cuda()
    gpu = _trav(H, case)
    assert gpu["voxel_id"][0] == 0 + nv * (1 + nv * 2) and gpu["t_in"][0] == 2.0 and gpu["t_out"][0] == 2.5


@pytest.mark.parametrize("n", [0, 1, 31, 129, 1000])
def test_ragged_and_empty_batches(oracle, H, P, n):
    case = H.make_case(0, n_rays=max(n, 1), with_net=False)
    case.origin = case.origin[:n]; case.direction = case.direction[:n]
    case.origin_d = case.origin_d[:n].contiguous(); case.direction_d = case.direction_d[:n].contiguous()
    gpu = _trav(H, case)
    if n == 0:
        assert gpu["voxel_id"].shape == (0,)
        return
    ref = H.OracleSide(oracle, case).query(traverse_only=True)
    P.assert_traversal(P.compare_traversal(gpu, ref))


def test_empty_grid_everything_misses(H):
    cfg = I.scaled(I.get_config(0), nv=8)
    case = H.make_case(0, n_rays=500, with_net=False, cfg=cfg, occ=np.zeros(512, np.uint8))
    assert case.bvh.info()["n_occupied"] == 0 and case.bvh.info()["n_nodes"] == 0
    gpu = _trav(H, case)
    assert (gpu["voxel_id"] == -1).all() and np.isinf(gpu["t_in"]).all() and np.isinf(gpu["t_out"]).all()


def test_single_voxel_and_full_grid(oracle, H, P):
    for occ in (np.eye(1, 64, 21, dtype=np.uint8)[0], np.ones(64, np.uint8)):
        cfg = I.scaled(I.get_config(0), nv=4)
        case = H.make_case(0, n_rays=2000, with_net=False, cfg=cfg, occ=occ, pose=[0.8, 0.5])
        gpu = _trav(H, case)
        lat = oracle.deform_lattice(4, 0.8, 0.5)
        vid, ti, to = oracle.traverse_brute(4, occ, lat, case.origin, case.direction)
        P.assert_traversal(P.compare_traversal(gpu, {"voxel_id": vid, "t_in": ti, "t_out": to}))


def test_fold_over_pose_is_rejected(H):
    import paper_2604_24666_b200 as nif
    cfg = I.scaled(I.get_config(0), nv=8)
    with pytest.raises(nif.NifError) as e:
        H.make_case(0, n_rays=16, with_net=False, cfg=cfg, occ=np.ones(512, np.uint8), pose=[0.0, 1.2])
    assert e.value.status == -3          # NIF_ERR_DEFORM_SINGULAR


def test_workspace_too_small_is_rejected(H):
    import paper_2604_24666_b200 as nif
    cfg = I.get_config(0)
    occ = torch.from_numpy(I.occupancy(cfg)).cuda()
    with pytest.raises(nif.NifError) as e:
        nif.nif_build_deformed_bvh(cfg.nv, occ, 1.0, 0.0, max_occupied=1)
    assert e.value.status == -4          # NIF_ERR_WORKSPACE


@pytest.mark.parametrize("cfg_id,n,pose_index", [(1, 40_000, 0), (2, 30_000, 0), (2, 30_000, 4), (3, 30_000, 2)])
def test_traversal_reduced_configs_all_rays(oracle, H, P, cfg_id, n, pose_index):
    # configs 1-3 at a size the oracle traverses completely in seconds (its own BVH, which
    # tests/test_oracle_traverse.py pins bit-exactly to the brute-force definition)
    case = H.make_case(cfg_id, n_rays=n, pose_index=pose_index, with_net=False)
    gpu = _trav(H, case)
    ref = H.OracleSide(oracle, case).query(traverse_only=True)
    m = P.compare_traversal(gpu, ref)
    P.assert_traversal(m)
    assert m["n_hit"] > 1000, m


@pytest.mark.parametrize("cfg_id,pose_index,n", [(1, 0, 60_000), (3, 2, 40_000), (0, 0, None)])
def test_both_traversal_kernels_agree_bit_for_bit(oracle, H, P, cfg_id, pose_index, n):
    # the per-thread kernel (coherent batches) and the persistent while-while kernel (incoherent
    # batches) implement the same definition; the device-side vote only picks the faster one
    import paper_2604_24666_b200 as nif
    case = H.make_case(cfg_id, n_rays=n, pose_index=pose_index, with_net=False)
    res = {}
    for name, fl in (("auto", 0), ("coherent", nif.NIF_TRAVERSE_COHERENT), ("incoherent", nif.NIF_TRAVERSE_INCOHERENT)):
        res[name] = H.run_gpu(case, flags=nif.NIF_TRAVERSE_ONLY | fl, raw_logits=False)
    for k in ("voxel_id", "t_in", "t_out"):
        a, b, c = (res[m][k].view(np.int32) for m in ("auto", "coherent", "incoherent"))
        assert np.array_equal(a, b) and np.array_equal(b, c), k
    side = H.OracleSide(oracle, case)
    idx = np.arange(0, len(case.origin), max(1, len(case.origin) // 4000))
    P.assert_traversal(P.compare_traversal(H.subset(res["incoherent"], idx), side.query(idx, traverse_only=True)))


def test_axis_parallel_rays_in_lattice_planes(oracle, H, P):
    """Degenerate rays for the node test (inverse direction +-inf, origin exactly on box planes): rays
    parallel to one or two axes whose origins lie exactly on lattice planes of an identity-pose grid,
    both signs of direction and of zero.  Ids and t must still equal the brute-force definition."""
    nv = 8
    rng = np.random.default_rng(5)
    occ = (rng.random(nv ** 3) < 0.6).astype(np.uint8)
    cfg = I.scaled(I.get_config(0), nv=nv)
    g = (2.0 * np.arange(nv + 1) - nv) / nv
    os_, ds_ = [], []
    for axis in range(3):
        for sign in (1.0, -1.0):
            for zero in (0.0, -0.0):
                for a in g:
                    for b in list(g[::2]) + [0.123, -0.456]:
                        o = np.zeros(3); d = np.full(3, zero)
                        o[axis] = -3.0 * sign; d[axis] = sign
                        o[(axis + 1) % 3] = a; o[(axis + 2) % 3] = b
                        os_.append(o.copy()); ds_.append(d.copy())
                        # parallel to one axis only: tilt within the plane of the second axis
                        d2 = d.copy(); d2[(axis + 2) % 3] = 0.25 * sign
                        d2 /= np.linalg.norm(d2)
                        os_.append(o.copy()); ds_.append(d2)
    o = np.array(os_, np.float32); d = np.array(ds_, np.float32)
    case = H.make_case(0, with_net=False, cfg=cfg, occ=occ, pose=[0.0, 0.0])
    case.origin, case.direction = o, d
    case.origin_d, case.direction_d = torch.from_numpy(o).cuda(), torch.from_numpy(d).cuda()
    lat = oracle.deform_lattice(nv, 0.0, 0.0)
    vid, ti, to = oracle.traverse_brute(nv, occ, lat, o, d)
    ref = {"voxel_id": vid, "t_in": ti, "t_out": to}
    for fl in (8, 16):                                   # NIF_TRAVERSE_COHERENT, NIF_TRAVERSE_INCOHERENT: both kernels
        gpu = _trav(H, case, flags=fl)
        m = P.compare_traversal(gpu, ref)
        P.assert_traversal(m)
        assert m["t_in_bit_mismatch"] == 0 and m["t_out_bit_mismatch"] == 0, m
    assert (vid >= 0).sum() > 1000


def _query_with_workspace(nif, case, o, d, flags):
    od, dd = torch.from_numpy(o).cuda(), torch.from_numpy(d).cuda()
    out = nif.alloc_outputs(len(o))
    for v in out.values():
        v.fill_(float("nan") if v.dtype.is_floating_point else -7)
    ws = nif.nif_query(case.bvh, None, od, dd, out, flags=nif.NIF_TRAVERSE_ONLY | flags)
    torch.cuda.synchronize()
    header = ws[:64].view(torch.int32).cpu().numpy()         # NifQueryScratch: n_hit (8 B), tile counter, pad[13]
    return {k: out[k].cpu().numpy() for k in ("voxel_id", "t_in", "t_out")}, int(header[3 + 5])   # pad[5] = image width


@pytest.mark.parametrize("width,height,expect", [
    (256, 128, 256),        # an image: walked in 8 x 4 pixel tiles per warp
    (1920, 1080, 1920),     # configs[1]'s frame
    (40, 36, 40),           # the smallest shapes that tile: width 40, one row of tiles high ...
    (64, 32, 64),
    (64, 4, None),          # a 16:1 strip (pixel steps vary 40-fold along the row): whatever is decided, same result
    (250, 120, 0),          # width not a multiple of 8: plain assignment
    (256, 126, 0),          # height not a multiple of 4
    (24, 64, 0),            # rows shorter than a warp
])
def test_image_shaped_batches_are_recognised_and_give_the_same_result(H, width, height, expect):
    """k_ray_coherence recognises a row-major image and k_traverse_simple then assigns 8 x 4 pixel tiles to warps.
    That is a re-assignment of rays to threads only: ids and t must be bit-equal to the persistent kernel's, which
    never looks at the width, on every ray -- recognised or not."""
    import paper_2604_24666_b200 as nif
    case = H.make_case(1, n_rays=16, with_net=False)
    info = case.bvh.info()
    o, d = I.camera_rays(width, height, 0.5 * (np.asarray(info["lo"]) + np.asarray(info["hi"])))
    auto, w_auto = _query_with_workspace(nif, case, o, d, 0)
    ref, w_ref = _query_with_workspace(nif, case, o, d, nif.NIF_TRAVERSE_INCOHERENT)
    assert expect is None or w_auto == expect, (w_auto, expect)
    for k in ("voxel_id", "t_in", "t_out"):
        assert np.array_equal(auto[k].view(np.int32), ref[k].view(np.int32)), k
    assert (auto["voxel_id"] >= 0).sum() > (0 if expect is None else min(200, width * height // 50))


def test_batches_that_are_not_images_are_left_alone(H):
    import paper_2604_24666_b200 as nif
    case = H.make_case(1, n_rays=16, with_net=False)
    info = case.bvh.info()
    o, d = I.camera_rays(256, 128, 0.5 * (np.asarray(info["lo"]) + np.asarray(info["hi"])))
    rng = np.random.default_rng(3)
    perm = rng.permutation(len(o))
    shuffled, w = _query_with_workspace(nif, case, o[perm], d[perm], nif.NIF_TRAVERSE_COHERENT)    # forced onto the simple kernel
    assert w == 0
    plain, w2 = _query_with_workspace(nif, case, o, d, 0)
    assert w2 == 256
    for k in ("voxel_id", "t_in", "t_out"):
        assert np.array_equal(shuffled[k].view(np.int32), plain[k][perm].view(np.int32)), k
    # a transposed image (column-major pixel order): consecutive rays are a pixel apart as well, rows are 128 long
    ot = o.reshape(128, 256, 3).transpose(1, 0, 2).reshape(-1, 3).copy(); dt = d.reshape(128, 256, 3).transpose(1, 0, 2).reshape(-1, 3).copy()
    tr, w3 = _query_with_workspace(nif, case, ot, dt, 0)
    assert w3 == 128
    back = {k: tr[k].reshape(256, 128).T.reshape(-1) for k in tr}
    for k in ("voxel_id", "t_in", "t_out"):
        assert np.array_equal(back[k].view(np.int32), plain[k].view(np.int32)), k
