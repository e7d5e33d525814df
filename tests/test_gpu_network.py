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


@pytest.mark.parametrize("occlusion_only", [False, True])
def test_compact_host_return_matches_device_entry(H, nif, occlusion_only):
    # nif_query_host_compact: dense ids/t, head rows only for the hit rays (row i <-> ray hit_ray[i]); chunked
    case = H.make_case(1, n_rays=50_000)
    flags = nif.NIF_OCCLUSION_ONLY if occlusion_only else 0
    dev = H.run_gpu(case, flags=flags, raw_logits=False)
    n = len(case.origin)
    o = torch.from_numpy(case.origin).pin_memory(); d = torch.from_numpy(case.direction).pin_memory()
    out = nif.alloc_outputs(n, pinned_host=True)
    for v in out.values():
        v.fill_(-7)
    hit_ray = torch.full((n,), -1, dtype=torch.int32).pin_memory()
    stage = nif.Stage(16_384)
    n_hit = nif.nif_query_host_compact(case.bvh, case.net, stage, o, d, out, hit_ray, flags=flags)
    hits = np.nonzero(dev["voxel_id"] >= 0)[0]
    assert n_hit == len(hits) > 1000
    for k in ("voxel_id", "t_in", "t_out"):
        assert np.array_equal(out[k].numpy(), dev[k]), k
    hr = hit_ray.numpy()[:n_hit]
    assert np.array_equal(np.sort(hr), hits)                      # every hit ray exactly once
    keys = ["occlusion"] if occlusion_only else ["occlusion", "distance", "dist_total", "normal", "albedo", "material_logits"]
    for k in keys:
        assert np.array_equal(out[k].numpy()[:n_hit], dev[k][hr]), k
        assert (out[k].numpy()[n_hit:] == -7).all(), k             # nothing written past the hit rows
    if occlusion_only:
        assert (out["normal"].numpy() == -7).all()


FULL = [  # cfg, pose, parameter variant
    (1, 0, "varpres"),
    (1, 0, "uniform0.1"),
    (2, 5, "varpres"),
    (3, 6, "varpres"),
    (4, 0, "varpres"),
]
ORACLE_BUDGET_S = 150.0          # per oracle pass over the hit rays, on the cores this box gives us
MIN_NET_RAYS = 1 << 17           # never fewer hit rays than this in the network comparison


@pytest.mark.parametrize("cfg_id,pose_index,variant", FULL)
def test_full_size_parity_protocol(oracle, H, P, nif, cfg_id, pose_index, variant):
    """SURVEY.md 8(c).4 at BASELINE.json's full sizes, in the launch configuration bench.py times:
    traversal parity on ALL rays (ids and hit flags exact, t bit-equal); network parity on ALL hit rays
    when the oracle gets through them within ORACLE_BUDGET_S on this box's cores, else on a seeded
    sample of at least 2^17 hit rays.  The oracle runs on every core (oracle/pool.py)."""
    import json, os, time
    from oracle.pool import OraclePool, n_cores
    case = H.make_case(cfg_id, pose_index=pose_index, variant=variant)
    cfg = case.cfg
    n = len(case.origin)
    assert n == cfg.rays_per_pose
    flags = nif.NIF_OCCLUSION_ONLY if cfg.occlusion_only else 0
    gpu = H.run_gpu(case, flags=flags)
    rec = {"cfg": cfg_id, "pose": pose_index, "variant": variant, "rays": n, "cores": n_cores()}
    # (a0) the deformed lattice is correctly rounded on both sides (R28): not one entry differs
    lat = oracle.deform_lattice(cfg.nv, float(case.pose[0]), float(case.pose[1]))
    lat_gpu = case.bvh.lattice().cpu().numpy()
    rec["lattice_entries"] = int(lat.size)
    rec["lattice_mismatch"] = int((lat.view(np.int32) != lat_gpu.view(np.int32)).sum())
    assert rec["lattice_mismatch"] == 0, rec
    with OraclePool(cfg.nv, case.occ, case.pose, lat, case.params) as pool:
        # (a1) every ray
        t0 = time.time()
        ref_t = pool.query(case.origin, case.direction, traverse_only=True)
        rec["oracle_traverse_s"] = time.time() - t0
        mt = P.compare_traversal(gpu, ref_t)
        rec["traversal"] = mt
        P.assert_traversal(mt)
        assert mt["t_in_bit_mismatch"] == 0 and mt["t_out_bit_mismatch"] == 0, mt
        hit = np.nonzero(ref_t["voxel_id"] >= 0)[0]
        assert gpu["n_hit_counter"] == len(hit) > 10_000
        # (a2)-(a5): all hit rays if the oracle is fast enough here, else a seeded sample
        probe = hit[:: max(1, len(hit) // 4096)][:4096]
        t0 = time.time()
        pool.query(case.origin[probe], case.direction[probe], occlusion_only=cfg.occlusion_only)
        rate = len(probe) / (time.time() - t0)
        rng = np.random.default_rng(cfg_id)
        n_net = len(hit) if len(hit) / rate <= ORACLE_BUDGET_S else max(MIN_NET_RAYS, int(rate * ORACLE_BUDGET_S))
        n_net = min(n_net, len(hit))
        idx = hit if n_net == len(hit) else np.sort(rng.choice(hit, n_net, replace=False))
        rec["hit_rays"] = int(len(hit)); rec["network_rays_compared"] = int(n_net)
        o, d = case.origin[idx], case.direction[idx]
        t0 = time.time()
        ref_n = pool.query(o, d, occlusion_only=cfg.occlusion_only)
        rec["oracle_network_s"] = time.time() - t0
        sub = H.subset(gpu, idx)
        mn = P.compare_network(sub, ref_n, fp16=True, occlusion_only=cfg.occlusion_only)
        rec["network_vs_fp32_oracle"] = mn
        hsel = ref_n["voxel_id"] >= 0
        cols = slice(0, 1) if cfg.occlusion_only else slice(0, 12)
        dz = np.abs(sub["raw_logits"][hsel][:, cols] - ref_n["raw_logits"][hsel][:, cols]) / mn["logit_rms"]
        zn = np.abs(ref_n["raw_logits"][hsel][:, cols]).max(axis=1) / mn["logit_rms"]
        rec["logit_err_over_rms_quantiles"] = {q: float(np.quantile(dz, float(q))) for q in ("0.5", "0.99", "0.9999", "0.999999")}
        rec["logit_err_rms_over_rms"] = float(np.sqrt((dz.astype(np.float64) ** 2).mean()))
        worst = np.argsort(dz.max(axis=1))[-5:]
        rec["worst_rays"] = [{"dz_over_rms": float(dz[i].max()), "ray_logit_inf_norm_over_rms": float(zn[i])} for i in worst]
        # the same rays against the oracle in the precision B:8 fixes for the fp16 networks (O9b: fp16
        # activations): what is left is fp32 summation order, so the argmax -- an integer decided by
        # floating point -- is compared in the same precision on both sides, with a 10x stricter gate
        ref_h = pool.query(o, d, occlusion_only=cfg.occlusion_only, act_f16=True)
        mh = P.compare_network(sub, ref_h, fp16=True, occlusion_only=cfg.occlusion_only)
        rec["network_vs_f16act_oracle"] = mh
        if os.path.isdir("gpurun_out"):
            with open("gpurun_out/parity_protocol.jsonl", "a") as f:
                f.write(json.dumps(rec) + "\n")
        P.assert_network(mn, fp16=True, occlusion_only=cfg.occlusion_only)
        # both sides round to fp16 here, so a value on a rounding boundary can go either way on EITHER side:
        # the logit gate is sqrt(2) x the one against the unrounded oracle
        P.assert_network(mh, fp16=True, occlusion_only=cfg.occlusion_only, logit_tol=7.5e-3)
        assert rec["logit_err_rms_over_rms"] <= 6e-4, rec       # four fp16 roundings ~ 5.6e-4 rms
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
