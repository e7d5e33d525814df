"""`-m gpu` parity of nif_query_multi (multi-voxel walk; R22/R23)
against the oracle's O11, through the C ABI.

The accept decision (occlusion >= 0.5) is a floating-point value deciding an integer outcome.  The
oracle's trace gives every voxel of a ray's sequence with its occlusion logit; a ray is CLEAR when
every decision the oracle took on it has |z0| above the logit tolerance of tests/parity.py -- the
CUDA path must then agree exactly on status, steps and voxel, and its outputs are compared element
by element.  On the remaining rays (a logit within rounding of the threshold) either decision is
correct: the CUDA result must be a VALID walk of the oracle's voxel sequence."""
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


def run_walk(nif, case, K, flags=0):
    n = len(case.origin)
    out = nif.alloc_outputs(n, raw_logits=True)
    walk = nif.alloc_walk_outputs(n)
    for v in list(out.values()) + list(walk.values()):
        v.fill_(float("nan") if v.dtype.is_floating_point else -7)
    nif.nif_query_multi(case.bvh, case.net, case.origin_d, case.direction_d, out, walk, K, flags=flags)
    torch.cuda.synchronize()
    res = {k: v.cpu().numpy() for k, v in out.items()}
    res.update({k: v.cpu().numpy() for k, v in walk.items()})
    return res


def check_walk(P, oracle, side, case, gpu, K, fp16, occlusion_only=False, idx=None, min_multi=10):
    c = case
    o = c.origin if idx is None else c.origin[idx]
    d = c.direction if idx is None else c.direction[idx]
    if idx is not None:
        gpu = {k: v[idx] for k, v in gpu.items()}
    ref = oracle.query_multi(c.cfg.nv, c.occ, side.lattice, side.bvh, c.pose, c.params, o, d, K,
                             occlusion_only=occlusion_only)
    tid, tz = oracle.walk_trace(c.cfg.nv, c.occ, side.lattice, side.bvh, c.pose, c.params, o, d, K)
    valid = tid >= 0
    rms = float(np.sqrt((tz[valid].astype(np.float64) ** 2).mean())) if valid.any() else 1.0
    margin = (5e-3 if fp16 else 5e-5) * rms
    near = valid & (np.abs(tz) <= margin)
    steps_ref = ref["steps"]
    taken = np.arange(K)[None, :] < steps_ref[:, None]               # decisions the oracle took
    clear = ~(near & taken).any(1)
    n = len(o)
    assert clear.mean() > 0.97, clear.mean()

    # ---- clear rays: exact agreement on the integers, tolerances on the rest
    for k in ("status", "steps", "voxel_id"):
        assert np.array_equal(gpu[k][clear], ref[k][clear]), (k, int((gpu[k][clear] != ref[k][clear]).sum()))
    g = {k: v[clear] for k, v in gpu.items()}
    r = {k: v[clear] for k, v in ref.items()}
    P.assert_traversal(P.compare_traversal(g, r))
    m = P.compare_network(g, r, fp16=fp16, occlusion_only=occlusion_only)
    P.assert_network(m, fp16=fp16, occlusion_only=occlusion_only)
    tol = 1e-2 if fp16 else 1e-5
    done = r["status"] != 0
    ell = (r["t_out"][done] - r["t_in"][done]).astype(np.float64)
    bound = tol * ell + 2e-5 * np.abs(r["dist_accum"][done]) + 1e-6
    assert (np.abs(g["dist_accum"][done].astype(np.float64) - r["dist_accum"][done]) <= bound).all()
    assert not g["dist_accum"][~done].any()
    multi = int((r["steps"] > 1).sum())
    assert multi >= min_multi, multi

    # ---- rays with a logit within rounding of the threshold: any consistent walk is valid
    for i in np.nonzero(~clear)[0]:
        s, st = int(gpu["steps"][i]), int(gpu["status"][i])
        n_vox = int(valid[i].sum())
        assert 0 <= s <= min(n_vox, K)
        assert (tz[i, :max(s - 1, 0)] < margin).all()                 # every voxel before the last was rejected
        if st == 1:
            assert gpu["voxel_id"][i] == tid[i, s - 1] and tz[i, s - 1] > -margin
        elif st == 2:
            assert s == K and gpu["voxel_id"][i] == tid[i, K - 1] and tz[i, K - 1] < margin
        else:
            assert s == n_vox < K or (s == n_vox == K and False), (s, n_vox)
            assert gpu["voxel_id"][i] == -1 and (tz[i, :s] < margin).all()
    return {"n": n, "clear": float(clear.mean()), "multi": multi, **m}


@pytest.mark.parametrize("variant", ["varpres", "uniform0.1"])
def test_walk_config0_fp32_all_rays(oracle, H, P, nif, variant):
    case = H.make_case(0, variant=variant)
    side = H.OracleSide(oracle, case)
    K = 8
    gpu = run_walk(nif, case, K)
    check_walk(P, oracle, side, case, gpu, K, fp16=False, min_multi=10 if variant == "varpres" else 0)


def test_walk_config1_fp16_reduced(oracle, H, P, nif):
    case = H.make_case(1, n_rays=30_000)
    side = H.OracleSide(oracle, case)
    K = 6
    for fl in (0, nif.NIF_ENGINE_FFMA):
        gpu = run_walk(nif, case, K, flags=fl)
        m = check_walk(P, oracle, side, case, gpu, K, fp16=True, min_multi=100)
        assert m["n_hit"] > 1000


def test_walk_config3_incoherent_occlusion_only(oracle, H, P, nif):
    case = H.make_case(3, n_rays=12_000, pose_index=2)
    side = H.OracleSide(oracle, case)
    K = 5
    gpu = run_walk(nif, case, K, flags=nif.NIF_OCCLUSION_ONLY)
    idx = np.arange(0, len(case.origin), 4)
    check_walk(P, oracle, side, case, gpu, K, fp16=True, occlusion_only=True, idx=idx, min_multi=50)


def test_walk_config4_shape_reduced(oracle, H, P, nif):
    case = H.make_case(4, n_rays=20_000)
    side = H.OracleSide(oracle, case)
    K = 4
    gpu = run_walk(nif, case, K)
    hit = np.nonzero(gpu["steps"] > 0)[0]
    idx = np.unique(np.concatenate([hit[:: max(1, len(hit) // 800)], np.arange(0, len(case.origin), 211)]))
    check_walk(P, oracle, side, case, gpu, K, fp16=True, idx=idx, min_multi=20)


def _net_with(H, case, kind):
    P = case.params
    if kind == "always_accept":          # every logit 0 on both sides -> occlusion exactly 0.5 -> accept
        P.weights = [np.zeros_like(w) for w in P.weights]
    else:                                # positive features and weights, z0 = -sum(a) < 0: never accept
        P.table = np.full_like(P.table, 0.5)
        P.weights = [np.full_like(w, 0.01) for w in P.weights]
        P.weights[-1][0, :] = -1.0
    if P.shape.dtype == "f16":           # both sides consume fp16-representable parameters (R20)
        P.table = P.table.astype(np.float16).astype(np.float32)
        P.weights = [w.astype(np.float16).astype(np.float32) for w in P.weights]
    case.net = H.make_net(P)
    return case


@pytest.mark.parametrize("cfg_id,n_rays", [(0, None), (1, 20_000), (2, 20_000)])
def test_all_zero_network_reduces_to_the_single_voxel_query(oracle, H, nif, cfg_id, n_rays):
    case = _net_with(H, H.make_case(cfg_id, n_rays=n_rays), "always_accept")
    single = H.run_gpu(case)
    gpu = run_walk(nif, case, 7)
    hit = single["voxel_id"] >= 0
    assert np.array_equal(gpu["voxel_id"], single["voxel_id"])
    assert np.array_equal(gpu["status"], hit.astype(np.int32)) and np.array_equal(gpu["steps"], hit.astype(np.int32))
    for k in ("t_in", "t_out", "occlusion", "distance", "dist_total", "normal", "albedo", "material_logits"):
        assert np.array_equal(gpu[k], single[k]), k
    # one segment: dist_accum = (0 + t_in) + t_k
    np.testing.assert_array_equal(gpu["dist_accum"][hit], (single["t_in"][hit] + single["distance"][hit]).astype(np.float32))


@pytest.mark.parametrize("cfg_id,n_rays,pose_index,K", [(0, None, 0, 10), (1, 6_000, 0, 24), (3, 3_000, 5, 24)])
def test_never_accepting_network_walks_the_oracles_voxel_sequence(oracle, H, nif, cfg_id, n_rays, pose_index, K):
    """Exercises the successor traversal alone, bit-exactly and many voxels deep: with a network that
    never accepts, steps = the number of occupied voxels the ray crosses (capped at K), status is MISS
    or MAX_STEPS, and the last voxel is the oracle's K-th."""
    case = _net_with(H, H.make_case(cfg_id, n_rays=n_rays, pose_index=pose_index), "never_accept")
    side = H.OracleSide(oracle, case)
    gpu = run_walk(nif, case, K)
    o, d = case.origin, case.direction
    n = len(o)
    at = np.full(n, -np.inf, np.float32); ai = np.full(n, -1, np.int32)
    count = np.zeros(n, np.int32); last = np.full(n, -1, np.int32)
    last_ti = np.full(n, np.inf, np.float32); acc = np.zeros(n, np.float32); prev = np.zeros(n, np.float32)
    for _ in range(K):
        v, ti, to = side.bvh.next_voxel(o, d, at, ai)
        live = v >= 0
        if not live.any():
            break
        count += live
        acc = np.where(live, acc + ((ti - prev) + (to - ti)), acc).astype(np.float32)
        prev = np.where(live, to, prev)
        last = np.where(live, v, last); last_ti = np.where(live, ti, last_ti)
        at = np.where(live, ti, at); ai = np.where(live, v, ai)
    assert np.array_equal(gpu["steps"], count)
    capped = count >= K
    assert capped.sum() > 0 and (~capped).sum() > 0
    assert (gpu["status"][capped] == 2).all() and (gpu["status"][~capped] == 0).all()
    assert np.array_equal(gpu["voxel_id"][capped], last[capped]) and (gpu["voxel_id"][~capped] == -1).all()
    assert np.array_equal(gpu["t_in"][capped].view(np.int32), last_ti[capped].view(np.int32))
    np.testing.assert_allclose(gpu["dist_accum"][capped], acc[capped], rtol=1e-6)
    assert not gpu["dist_accum"][~capped].any() and not gpu["occlusion"][~capped].any()


def test_walk_argument_validation(H, nif):
    case = H.make_case(0)
    n = len(case.origin)
    out = nif.alloc_outputs(n); walk = nif.alloc_walk_outputs(n)
    with pytest.raises(nif.NifError):
        nif.nif_query_multi(case.bvh, case.net, case.origin_d, case.direction_d, out, walk, 0)
    with pytest.raises(nif.NifError):
        nif.nif_query_multi(case.bvh, case.net, case.origin_d, case.direction_d, out, walk, 4, flags=nif.NIF_TRAVERSE_ONLY)
    with pytest.raises(nif.NifError):
        nif.nif_query_multi(case.bvh, case.net, case.origin_d, case.direction_d, out, walk, 4,
                            workspace=torch.empty(256, dtype=torch.uint8, device="cuda"))
    # empty batch
    e = torch.empty(0, 3, device="cuda")
    nif.nif_query_multi(case.bvh, case.net, e, e, nif.alloc_outputs(0), nif.alloc_walk_outputs(0), 4)
