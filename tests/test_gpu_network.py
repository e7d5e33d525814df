"""`-m gpu` parity: whole query (a1)-(a5) of the CUDA path against the oracle, through the C ABI.
Tolerances: tests/parity.py (from BASELINE.json:5)."""
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


def _engines(nif, case):
    """flag sets to exercise: default engine, and the FFMA cross-check for fp16 nets"""
    if case.params.shape.dtype == "f16":
        return [("default", 0), ("ffma", nif.NIF_ENGINE_FFMA)]
    return [("default", 0)]


@pytest.mark.parametrize("variant", ["uniform0.1", "varpres"])
def test_config0_fp32_all_rays(oracle, H, P, nif, variant):
    case = H.make_case(0, variant=variant)
    ref = H.OracleSide(oracle, case).query()
    gpu = H.run_gpu(case)
    P.assert_traversal(P.compare_traversal(gpu, ref))
    m = P.compare_network(gpu, ref, fp16=False)
    P.assert_network(m, fp16=False)
    assert gpu["n_hit_counter"] == m["n_hit"]


@pytest.mark.parametrize("variant", ["uniform0.1", "varpres"])
def test_config1_fp16_reduced_all_rays(oracle, H, P, nif, variant):
    case = H.make_case(1, n_rays=30_000, variant=variant)
    ref = H.OracleSide(oracle, case).query()
    for name, fl in _engines(nif, case):
        gpu = H.run_gpu(case, flags=fl)
        P.assert_traversal(P.compare_traversal(gpu, ref))
        m = P.compare_network(gpu, ref, fp16=True)
        P.assert_network(m, fp16=True)
        assert gpu["n_hit_counter"] == m["n_hit"] > 1000, (name, m)


def test_config4_shape_reduced(oracle, H, P, nif):
    # F = 4, W = 128, H = 4, T = 2^22 (table 512 MiB as fp16)
    case = H.make_case(4, n_rays=20_000)
    side = H.OracleSide(oracle, case)
    gpu_t = H.run_gpu(case, flags=nif.NIF_TRAVERSE_ONLY, raw_logits=False)
    hit = np.nonzero(gpu_t["voxel_id"] >= 0)[0]
    idx = np.sort(np.concatenate([hit[:: max(1, len(hit) // 1500)], np.arange(0, len(case.origin), 97)]))
    idx = np.unique(idx)
    ref = side.query(idx)
    for name, fl in _engines(nif, case):
        gpu = H.subset(H.run_gpu(case, flags=fl), idx)
        P.assert_traversal(P.compare_traversal(gpu, ref))
        P.assert_network(P.compare_network(gpu, ref, fp16=True), fp16=True)


def test_occlusion_only_flag(oracle, H, P, nif):
    case = H.make_case(3, n_rays=20_000, pose_index=1)
    ref = H.OracleSide(oracle, case).query(occlusion_only=True)
    for name, fl in _engines(nif, case):
        gpu = H.run_gpu(case, flags=fl | nif.NIF_OCCLUSION_ONLY)
        P.assert_traversal(P.compare_traversal(gpu, ref))
        P.assert_network(P.compare_network(gpu, ref, fp16=True, occlusion_only=True), fp16=True, occlusion_only=True)
        # untouched outputs keep the poison the harness wrote
        assert np.isnan(gpu["normal"]).all() and np.isnan(gpu["distance"]).all()


@pytest.mark.parametrize("n", [1, 7, 127, 129, 1000])
def test_ragged_hit_tiles(oracle, H, P, nif, n):
    # hit counts that do not fill a tile of the encode kernels
    case = H.make_case(0, n_rays=n)
    ref = H.OracleSide(oracle, case).query()
    gpu = H.run_gpu(case)
    P.assert_traversal(P.compare_traversal(gpu, ref))
    P.assert_network(P.compare_network(gpu, ref, fp16=False), fp16=False)


def test_all_miss_batch(H, nif):
    case = H.make_case(0, n_rays=300)
    case.direction_d = (-case.direction_d).contiguous()
    gpu = H.run_gpu(case)
    assert (gpu["voxel_id"] == -1).all() and gpu["n_hit_counter"] == 0
    for k in ("occlusion", "distance", "dist_total", "normal", "albedo", "material_logits", "raw_logits"):
        assert not gpu[k].any(), k


def test_host_buffer_entry_matches_device_entry(H, nif):
    # nif_query_host = same kernels behind pinned-host staging in chunks (ragged last chunk)
    case = H.make_case(1, n_rays=50_000)
    dev = H.run_gpu(case)
    n = len(case.origin)
    o = torch.from_numpy(case.origin).pin_memory(); d = torch.from_numpy(case.direction).pin_memory()
    out = nif.alloc_outputs(n, raw_logits=True, pinned_host=True)
    stage = nif.Stage(16_384)
    nif.nif_query_host(case.bvh, case.net, stage, o, d, out)
    for k, v in out.items():
        assert np.array_equal(v.numpy(), dev[k], equal_nan=True), k


FULL = [  # cfg, pose, sampled rays for traversal parity, sampled hit rays for network parity
    (1, 0, 1 << 15, 6000),
    (2, 5, 1 << 14, 5000),
    (3, 6, 1 << 14, 5000),
    (4, 0, 1 << 14, 3000),
]


@pytest.mark.parametrize("cfg_id,pose_index,n_trav,n_net", FULL)
def test_full_size_configs_sampled(oracle, H, P, nif, cfg_id, pose_index, n_trav, n_net):
    """BASELINE.json's full sizes in the launch configuration bench.py times; the oracle
    recomputes a seeded sample of the rays one by one (rays are independent)."""
    case = H.make_case(cfg_id, pose_index=pose_index)
    cfg = case.cfg
    n = len(case.origin)
    assert n == cfg.rays_per_pose
    flags = nif.NIF_OCCLUSION_ONLY if cfg.occlusion_only else 0
    gpu = H.run_gpu(case, flags=flags)
    side = H.OracleSide(oracle, case)
    rng = np.random.default_rng(cfg_id)
    idx_t = np.sort(rng.choice(n, n_trav, replace=False))
    ref_t = side.query(idx_t, traverse_only=True)
    mt = P.compare_traversal(H.subset(gpu, idx_t), ref_t)
    P.assert_traversal(mt)
    hit = np.nonzero(gpu["voxel_id"] >= 0)[0]
    assert gpu["n_hit_counter"] == len(hit) > 10_000
    idx_n = np.sort(rng.choice(hit, n_net, replace=False))
    ref_n = side.query(idx_n, occlusion_only=cfg.occlusion_only)
    mn = P.compare_network(H.subset(gpu, idx_n), ref_n, fp16=True, occlusion_only=cfg.occlusion_only)
    P.assert_network(mn, fp16=True, occlusion_only=cfg.occlusion_only)
    # properties that hold at any size
    h = gpu["voxel_id"] >= 0
    assert case.occ[gpu["voxel_id"][h]].all()
    assert (gpu["t_out"][h] >= gpu["t_in"][h]).all() and (gpu["t_in"][h] >= 0).all()
    assert ((gpu["occlusion"][h] > 0) & (gpu["occlusion"][h] < 1)).all() and not gpu["occlusion"][~h].any()
    if not cfg.occlusion_only:
        ell = gpu["t_out"][h] - gpu["t_in"][h]
        assert (gpu["distance"][h] >= 0).all() and (gpu["distance"][h] <= ell * (1 + 1e-6) + 1e-12).all()
        np.testing.assert_allclose(np.linalg.norm(gpu["normal"][h], axis=1), 1.0, atol=1e-5)
        assert not gpu["normal"][~h].any() and not gpu["material_logits"][~h].any()


SHAPES = [  # (pe_bands, levels, log2_T, feat, base_res, growth, hidden_layers, width)
    (2, 8, 14, 2, 8, 1.5, 1, 32),      # smallest tensor-core shape: L*F = 16, one hidden layer, W = 32
    (3, 4, 12, 4, 4, 2.0, 2, 32),      # F = 4, L*F = 16
    (1, 16, 15, 4, 8, 1.3, 3, 64),     # L*F = 64: one sample per K chunk
    (5, 4, 13, 2, 16, 1.7, 5, 128),    # L*F = 8, W = 128, deep
    (0, 16, 16, 2, 16, 1.38, 2, 64),   # no positional bands: S = 1, a single (padded) K chunk per endpoint pair
    (3, 2, 19, 3, 64, 2.0, 3, 64),     # the paper's own shape: two levels, F = 3 (stored padded to 4), B = 3
    (2, 8, 14, 3, 8, 1.5, 2, 32),      # F = 3, L*F(padded) = 32
]


@pytest.mark.parametrize("shape", SHAPES)
def test_tensor_core_kernel_shape_sweep(oracle, H, P, nif, shape):
    """Every template instantiation / chunking case of the fused kernel against the oracle."""
    b, L, t, f, base, growth, hl, w = shape
    net = I.NetShape(pe_bands=b, levels=L, log2_T=t, feat=f, base_res=base, growth=growth,
                     hidden_layers=hl, width=w, dtype="f16")
    cfg = I.scaled(I.get_config(1), net=net)
    case = H.make_case(1, n_rays=12_000, cfg=cfg)
    assert nif.nif_net_uses_tensor_cores(case.net)
    ref = H.OracleSide(oracle, case).query()
    for name, fl in _engines(nif, case):
        gpu = H.run_gpu(case, flags=fl)
        P.assert_traversal(P.compare_traversal(gpu, ref))
        m = P.compare_network(gpu, ref, fp16=True)
        P.assert_network(m, fp16=True)
        assert m["n_hit"] > 500, (name, m)


@pytest.mark.parametrize("variant", ["uniform0.1", "varpres"])
def test_paper_shape_config5(oracle, H, P, nif, variant):
    """32^3 voxels, two-level hash grid (base 64, feature dim 3), 3 PE bands."""
    case = H.make_case(5, n_rays=40_000, variant=variant)
    assert nif.nif_net_uses_tensor_cores(case.net)
    ref = H.OracleSide(oracle, case).query()
    for name, fl in _engines(nif, case):
        gpu = H.run_gpu(case, flags=fl)
        P.assert_traversal(P.compare_traversal(gpu, ref))
        m = P.compare_network(gpu, ref, fp16=True)
        P.assert_network(m, fp16=True)
        assert m["n_hit"] > 2000, (name, m)


def test_three_features_fp32(oracle, H, P, nif):
    net = I.NetShape(pe_bands=2, levels=3, log2_T=12, feat=3, base_res=4, growth=2.0,
                     hidden_layers=2, width=32, dtype="f32")
    case = H.make_case(0, cfg=I.scaled(I.get_config(0), net=net))
    ref = H.OracleSide(oracle, case).query()
    gpu = H.run_gpu(case)
    P.assert_traversal(P.compare_traversal(gpu, ref))
    P.assert_network(P.compare_network(gpu, ref, fp16=False), fp16=False)


def test_empty_batch_is_a_no_op(H, nif):
    case = H.make_case(0, n_rays=16)
    out = nif.alloc_outputs(0)
    nif.nif_query(case.bvh, case.net, case.origin_d[:0].contiguous(), case.direction_d[:0].contiguous(), out)
    torch.cuda.synchronize()
