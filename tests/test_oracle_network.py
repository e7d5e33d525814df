"""Pins for oracle steps O9 (MLP), O10 (heads) and the wiring of the whole query."""
import numpy as np
import torch

import nif_inputs as I


def test_mlp_equals_torch_fp64_linear_relu_chain(oracle):
    # library routine: torch.nn.functional.linear + relu in fp64 (R16: no bias, linear output)
    for cfg_id, variant in ((0, "uniform0.1"), (0, "varpres"), (1, "varpres")):
        cfg = I.get_config(cfg_id)
        P = I.net_params(cfg, variant)
        # tiny table stand-in is irrelevant here; only the weights are used
        x = np.random.default_rng(0).uniform(-1, 1, (64, cfg.net.d_in)).astype(np.float32)
        got = oracle.mlp(P, x)
        a = torch.from_numpy(x.astype(np.float64))
        for w in P.weights[:-1]:
            a = torch.relu(torch.nn.functional.linear(a, torch.from_numpy(w.astype(np.float64))))
        z = torch.nn.functional.linear(a, torch.from_numpy(P.weights[-1].astype(np.float64))).numpy()
        scale = np.abs(z).max()
        assert np.abs(got - z).max() <= 1e-5 * scale, (np.abs(got - z).max(), scale)


def test_decode_closed_forms_and_invariants(oracle):
    rng = np.random.default_rng(1)
    n = 1000
    z = rng.normal(0, 3, (n, 12)).astype(np.float32)
    t_in = rng.uniform(1, 3, n).astype(np.float32)
    t_out = t_in + rng.uniform(0, 0.2, n).astype(np.float32)
    o = oracle.decode(z, t_in, t_out)
    ell = (t_out - t_in).astype(np.float64)
    # heads (B:7): sigmoid / sigmoid x segment length / normalised / sigmoid / raw logits
    sig = lambda v: np.exp(-np.logaddexp(0, -v.astype(np.float64)))      # textbook stable sigmoid
    np.testing.assert_allclose(o["occlusion"], sig(z[:, 0]), atol=2e-7)
    np.testing.assert_allclose(o["albedo"], sig(z[:, 5:8]), atol=2e-7)
    np.testing.assert_allclose(o["distance"], sig(z[:, 1]) * ell, atol=1e-7)
    assert np.array_equal(o["material_logits"], z[:, 8:12])
    # invariants ("local hit distance t_i in [0, l_i]", P:61 with k = 0)
    assert (o["distance"] >= 0).all() and (o["distance"] <= (t_out - t_in) * (1 + 1e-6)).all()
    np.testing.assert_allclose(o["dist_total"], t_in + o["distance"], rtol=2e-7)
    np.testing.assert_allclose(np.linalg.norm(o["normal"], axis=1), 1.0, atol=1e-6)
    cos = (o["normal"] * z[:, 2:5]).sum(1) / np.linalg.norm(z[:, 2:5], axis=1)
    np.testing.assert_allclose(cos, 1.0, atol=1e-6)
    # special values: sigma(0) = 1/2; s -> 0 gives D = t_in, s -> 1 gives D = t_out
    z0 = np.zeros((3, 12), np.float32); z0[1, 1] = -200; z0[2, 1] = 200
    ti = np.array([2, 2, 2], np.float32); to = np.array([2.5, 2.5, 2.5], np.float32)
    o = oracle.decode(z0, ti, to)
    assert o["occlusion"][0] == 0.5 and o["distance"][0] == 0.25 and (o["albedo"][0] == 0.5).all()
    assert o["dist_total"][1] == 2.0 and o["dist_total"][2] == 2.5
    assert np.array_equal(o["normal"][0], [0, 0, 0])        # z = 0 -> rsqrt clamp, no NaN (R17)


def _setup(oracle, cfg_id, n, variant):
    cfg = I.get_config(cfg_id)
    occ = I.occupancy(cfg); pose = I.poses(cfg)[0]
    lat = oracle.deform_lattice(cfg.nv, *pose)
    bvh = oracle.bvh_build(cfg.nv, occ, lat)
    lo, hi = bvh.bounds()
    o, d = I.rays(cfg, 0, lo, hi, n=n)
    return cfg, occ, pose, lat, bvh, o, d, I.net_params(cfg, variant)


def test_query_is_the_composition_entry_then_exit(oracle):
    # wiring (B:7 "Both rest-space endpoints are encoded and concatenated", entry first):
    # traverse -> inverse-map -> normalise -> psi(entry) ++ psi(exit) -> MLP -> heads
    cfg, occ, pose, lat, bvh, o, d, P = _setup(oracle, 0, 600, "varpres")
    out = oracle.query(cfg.nv, occ, lat, bvh, pose, P, o, d)
    v, ti, to = bvh.traverse(o, d)
    assert np.array_equal(out["voxel_id"], v) and np.array_equal(out["t_in"], ti)
    hit = v >= 0
    rest = oracle.rest_endpoints(pose[0], pose[1], o, d, v, ti, to)[hit]
    xn = np.clip((rest + 1.0) * 0.5, 0.0, 1.0).astype(np.float32)
    feats = np.concatenate([oracle.encode(P, xn[:, 0]), oracle.encode(P, xn[:, 1])], axis=1)
    assert feats.shape[1] == cfg.net.d_in == 144
    z = oracle.mlp(P, feats)
    np.testing.assert_allclose(out["raw_logits"][hit], z, atol=1e-5 * np.abs(z).max())
    dec = oracle.decode(out["raw_logits"][hit], ti[hit], to[hit])
    for k in ("occlusion", "distance", "dist_total", "normal", "albedo", "material_logits"):
        np.testing.assert_allclose(out[k][hit], dec[k], atol=1e-6)
    # swapping the endpoints must change the result (the order is observable)
    z_swapped = oracle.mlp(P, np.concatenate([feats[:, 72:], feats[:, :72]], axis=1))
    assert np.abs(z_swapped - z).max() > 1e-3


def test_bvh_query_equals_brute_force_query(oracle):
    cfg, occ, pose, lat, bvh, o, d, P = _setup(oracle, 0, 300, "varpres")
    a = oracle.query(cfg.nv, occ, lat, bvh, pose, P, o, d)
    b = oracle.query(cfg.nv, occ, lat, None, pose, P, o, d)
    for k in a:
        assert np.array_equal(a[k], b[k]), k


def test_miss_rays_output_zero(oracle):
    cfg, occ, pose, lat, bvh, o, d, P = _setup(oracle, 0, 64, "varpres")
    d = -d                                              # shoot away from the object
    out = oracle.query(cfg.nv, occ, lat, bvh, pose, P, o, d)
    assert (out["voxel_id"] == -1).all() and np.isinf(out["t_in"]).all()
    for k in ("occlusion", "distance", "dist_total", "normal", "albedo", "material_logits", "raw_logits"):
        assert not out[k].any(), k


def test_occlusion_only_equals_the_occlusion_head(oracle):
    cfg, occ, pose, lat, bvh, o, d, P = _setup(oracle, 0, 300, "varpres")
    full = oracle.query(cfg.nv, occ, lat, bvh, pose, P, o, d)
    occ_only = oracle.query(cfg.nv, occ, lat, bvh, pose, P, o, d, occlusion_only=True)
    assert np.array_equal(full["occlusion"], occ_only["occlusion"])
    assert not occ_only["normal"].any()


def test_fp32_oracle_is_within_1e5_of_fp64_accumulation(oracle, oracle64):
    # bounds the oracle's own rounding: the north star fixes an fp32 oracle; the same source
    # compiled with double accumulation must agree to the fp32-config tolerance (1e-5).
    assert oracle.acc_bytes == 4 and oracle64.acc_bytes == 8
    for cfg_id, n in ((0, 1024), (1, 3000)):
        cfg, occ, pose, lat, bvh, o, d, P = _setup(oracle, cfg_id, n, "varpres")
        a = oracle.query(cfg.nv, occ, lat, bvh, pose, P, o, d)
        bvh64 = oracle64.bvh_build(cfg.nv, occ, lat)
        b = oracle64.query(cfg.nv, occ, lat, bvh64, pose, P, o, d)
        assert np.array_equal(a["voxel_id"], b["voxel_id"]) and np.array_equal(a["t_in"], b["t_in"])
        hit = a["voxel_id"] >= 0
        assert hit.sum() > 100
        zr = np.sqrt((b["raw_logits"][hit] ** 2).mean())
        assert np.abs(a["raw_logits"] - b["raw_logits"]).max() <= 1e-5 * zr
        for k in ("occlusion", "albedo", "normal"):
            assert np.abs(a[k] - b[k]).max() <= 1e-5, k


# ---- O9b: fp16 activations (B:8 "fp16 weights and activations, fp32 accumulate") -------------------
def test_round_f16_equals_numpy_float16_conversion(oracle):
    rng = np.random.default_rng(9)
    x = np.concatenate([
        rng.standard_normal(200_000).astype(np.float32) * 10.0 ** rng.uniform(-9, 5, 200_000).astype(np.float32),
        np.array([0.0, -0.0, 1.0, -1.0, 65504.0, 65519.99, 65520.0, 70000.0, -65520.0, 2.0 ** -14, 2.0 ** -24,
                  2.0 ** -25, 1.5 * 2.0 ** -25, 2.0 ** -26, np.inf, -np.inf, 1.0 + 2.0 ** -11, 1.0 + 3 * 2.0 ** -11,
                  1.0 + 2.0 ** -11 + 2.0 ** -20, 2049.0, 2051.0], np.float32),
        np.arange(0, 70000, 0.37, dtype=np.float32) * 2.0 ** -20])       # ties and subnormal halves
    with np.errstate(over="ignore"):
        want = x.astype(np.float16).astype(np.float32)
    got = oracle.round_f16(x)
    assert np.array_equal(got.view(np.int32), want.view(np.int32))


def test_act_f16_mode_rounds_where_the_precision_contract_says(oracle):
    # the rounded mode equals the plain MLP applied to an fp16-rounded input with every hidden activation
    # rounded: checked through a numpy float16 chain with fp64 accumulation (sums differ at 1e-6, not 1e-3)
    cfg, occ, pose, lat, bvh, o, d, P = _setup(oracle, 1, 400, "varpres")
    a = oracle.query(cfg.nv, occ, lat, bvh, pose, P, o, d)
    b = oracle.query(cfg.nv, occ, lat, bvh, pose, P, o, d, act_f16=True)
    hit = a["voxel_id"] >= 0
    assert hit.sum() > 30
    assert np.array_equal(a["voxel_id"], b["voxel_id"]) and np.array_equal(a["t_in"], b["t_in"])
    rest = oracle.rest_endpoints(float(pose[0]), float(pose[1]), o[hit], d[hit], a["voxel_id"][hit], a["t_in"][hit], a["t_out"][hit])
    xn = np.clip((rest + 1.0) * 0.5, 0.0, 1.0).astype(np.float32)
    feats = np.concatenate([oracle.encode(P, xn[:, 0]), oracle.encode(P, xn[:, 1])], axis=1)
    act = feats.astype(np.float16).astype(np.float64)
    for w in P.weights[:-1]:
        act = np.maximum(act @ w.astype(np.float64).T, 0.0).astype(np.float16).astype(np.float64)
    z = act @ P.weights[-1].astype(np.float64).T
    rms = np.sqrt((z ** 2).mean())
    # fp32 vs fp64 sums differ by ~1e-7: almost every logit agrees to 1e-5 rms; where a sum sits on an fp16
    # rounding boundary one hidden activation moves by one fp16 ulp, a logit error of ~1e-3 rms at most
    err = np.abs(b["raw_logits"][hit] - z) / rms
    assert np.median(err) <= 1e-6 and (err > 1e-5).mean() < 0.05 and err.max() <= 3e-3, (np.median(err), (err > 1e-5).mean(), err.max())
    # and the two modes differ by fp16 noise: well above fp32 rounding, well inside the logit gate
    diff = np.abs(a["raw_logits"][hit] - b["raw_logits"][hit]).max() / rms
    assert 1e-5 < diff < 5e-3, diff
