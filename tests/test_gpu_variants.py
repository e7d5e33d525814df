"""`-m gpu` parity of the variant outputs against the oracle, through the C ABI: the ReLU +
log-transformed distance head (NIF_DIST_LOG, R24) and the hit positions in
deformed and rest space.  Tolerances derive from tests/parity.py: an error dz in the
logit z1 is a relative error dz in (1 + D) for the log head, and an error of tol in the fraction u
moves the rest-space hit by at most tol x the rest segment."""
import numpy as np
import pytest

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
    return [0, nif.NIF_ENGINE_FFMA] if case.params.shape.dtype == "f16" else [0]


def _check_positions(gpu, ref, tol, d_bound):
    hit = ref["voxel_id"] >= 0
    assert not gpu["hit_position"][~hit].any() and not gpu["hit_position_rest"][~hit].any()
    e = np.abs(gpu["hit_position"][hit].astype(np.float64) - ref["hit_position"][hit]).max(1)
    assert (e <= d_bound + 1e-5).all(), (e / (d_bound + 1e-5)).max()
    er = np.abs(gpu["hit_position_rest"][hit].astype(np.float64) - ref["hit_position_rest"][hit]).max(1)
    assert (er <= 3 * d_bound + tol * 0.5 + 1e-5).all(), er.max()


@pytest.mark.parametrize("cfg_id,n_rays", [(0, None), (1, 30_000), (4, 12_000)])
def test_hit_positions_default_head(oracle, H, P, nif, cfg_id, n_rays):
    case = H.make_case(cfg_id, n_rays=n_rays)
    fp16 = case.params.shape.dtype == "f16"
    tol = 1e-2 if fp16 else 1e-5
    side = H.OracleSide(oracle, case)
    idx = None
    if cfg_id == 4:
        t = H.run_gpu(case, flags=nif.NIF_TRAVERSE_ONLY, raw_logits=False)
        hit = np.nonzero(t["voxel_id"] >= 0)[0]
        idx = np.unique(np.concatenate([hit[:: max(1, len(hit) // 1000)], np.arange(0, len(case.origin), 131)]))
    ref = side.query(idx, hit_positions=True)
    for fl in _engines(nif, case):
        gpu = H.run_gpu(case, flags=fl, hit_positions=True)
        if idx is not None:
            gpu = H.subset(gpu, idx)
        P.assert_traversal(P.compare_traversal(gpu, ref))
        P.assert_network(P.compare_network(gpu, ref, fp16=fp16), fp16=fp16)
        hit = ref["voxel_id"] >= 0
        ell = (ref["t_out"][hit] - ref["t_in"][hit]).astype(np.float64)
        _check_positions(gpu, ref, tol, tol * ell + 1e-5 * ref["t_out"][hit])
    # outputs not asked for stay untouched: same query without the position pointers gives the same heads
    plain = H.run_gpu(case)
    full = H.run_gpu(case, hit_positions=True)
    for k in ("voxel_id", "distance", "dist_total", "normal"):
        assert np.array_equal(plain[k], full[k]), k


@pytest.mark.parametrize("cfg_id,n_rays", [(0, None), (1, 30_000)])
def test_log_distance_head(oracle, H, P, nif, cfg_id, n_rays):
    case = H.make_case(cfg_id, n_rays=n_rays)
    fp16 = case.params.shape.dtype == "f16"
    tol = 1e-2 if fp16 else 1e-5
    ref = H.OracleSide(oracle, case).query(dist_log=True, hit_positions=True)
    hit = ref["voxel_id"] >= 0
    assert ((ref["raw_logits"][hit, 1] > 0.05).sum() > 100) and ((ref["raw_logits"][hit, 1] < -0.05).sum() > 100)
    for fl in _engines(nif, case):
        gpu = H.run_gpu(case, flags=fl | nif.NIF_DIST_LOG, hit_positions=True)
        P.assert_traversal(P.compare_traversal(gpu, ref))
        m = P.compare_network(gpu, ref, fp16=fp16, occlusion_only=True)      # occlusion + raw logits (all 12 below)
        P.assert_network(m, fp16=fp16, occlusion_only=True)
        zr = ref["raw_logits"][hit]; zg = gpu["raw_logits"][hit]
        rms = np.sqrt((zr.astype(np.float64) ** 2).mean())
        assert np.abs(zg - zr).max() <= (5e-3 if fp16 else 5e-5) * rms
        for k in ("albedo", "normal"):
            assert np.abs(gpu[k][hit] - ref[k][hit]).max() <= 2e-2
        D_ref = ref["dist_total"][hit].astype(np.float64); D_gpu = gpu["dist_total"][hit].astype(np.float64)
        d_bound = tol * (1.0 + D_ref)
        assert (np.abs(D_gpu - D_ref) <= d_bound).all(), (np.abs(D_gpu - D_ref) / d_bound).max()
        assert (D_gpu >= 0).all() and not gpu["dist_total"][~hit].any()
        np.testing.assert_allclose(gpu["distance"][hit], gpu["dist_total"][hit] - gpu["t_in"][hit], atol=1e-6)
        # where the oracle's logit is clearly negative the ReLU gives exactly 0 on both sides
        neg = zr[:, 1] < -(5e-3 if fp16 else 5e-5) * rms
        assert (D_gpu[neg] == 0).all()
        _check_positions(gpu, ref, tol, d_bound)


def test_query_host_carries_the_hit_positions(H, nif):
    import torch
    case = H.make_case(1, n_rays=50_000)
    dev = H.run_gpu(case, hit_positions=True)
    n = len(case.origin)
    out_h = nif.alloc_outputs(n, pinned_host=True, hit_positions=True)
    stage = nif.Stage(16_384)
    nif.nif_query_host(case.bvh, case.net, stage, torch.from_numpy(case.origin).pin_memory(),
                       torch.from_numpy(case.direction).pin_memory(), out_h)
    for k in ("voxel_id", "dist_total", "hit_position", "hit_position_rest"):
        assert np.array_equal(out_h[k].numpy(), dev[k]), k


@pytest.mark.parametrize("cfg_id,n_rays,tc", [(0, None, False), (1, 30_000, True), (4, 12_000, True)])
def test_concatenation_encoding(oracle, H, P, nif, cfg_id, n_rays, tc):
    """NIF_ENC_CONCAT (psi = [gamma(x), phi(x)], B:5 reading of the hybrid encoding; oracle O8b): config 0
    on the fp32 engine, the shapes of config 1 (L*F = 32) and config 4 (L*F = 64) on the tcgen05 kernel
    and on the FFMA cross-check."""
    from dataclasses import replace
    base = I.get_config(cfg_id)
    cfg = replace(base, net=replace(base.net, enc_mode="concat"))
    case = H.make_case(cfg_id, n_rays=n_rays, cfg=cfg)
    assert case.params.weights[0].shape[1] == 2 * (3 + 6 * base.net.pe_bands + base.net.levels * base.net.feat)
    assert nif.nif_net_uses_tensor_cores(case.net) == tc
    fp16 = base.net.dtype == "f16"
    side = H.OracleSide(oracle, case)
    idx = None
    if cfg_id == 4:
        t = H.run_gpu(case, flags=nif.NIF_TRAVERSE_ONLY, raw_logits=False)
        hit = np.nonzero(t["voxel_id"] >= 0)[0]
        idx = np.unique(np.concatenate([hit[:: max(1, len(hit) // 1000)], np.arange(0, len(case.origin), 131)]))
    ref = side.query(idx)
    for fl in _engines(nif, case):
        gpu = H.run_gpu(case, flags=fl)
        if idx is not None:
            gpu = H.subset(gpu, idx)
        P.assert_traversal(P.compare_traversal(gpu, ref))
        m = P.compare_network(gpu, ref, fp16=fp16)
        P.assert_network(m, fp16=fp16)
        assert m["n_hit"] > 500
