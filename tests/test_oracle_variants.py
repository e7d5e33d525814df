"""Pins for the oracle's variant outputs: O10b (ReLU + log-transformed distance head, PAPER.md:87,
DESIGN.md R24) and O12 (hit positions).  CPU only.  Each pin is an inverse
function, an invariant or a special case -- none re-evaluates the oracle's own expression."""
import numpy as np

import nif_inputs as I


def _setup(oracle, pose=None, n=600, variant="varpres"):
    cfg = I.get_config(0)
    occ = I.occupancy(cfg)
    pose = I.poses(cfg)[0] if pose is None else np.asarray(pose, np.float32)
    lat = oracle.deform_lattice(cfg.nv, float(pose[0]), float(pose[1]))
    bvh = oracle.bvh_build(cfg.nv, occ, lat)
    o, d = I.rays(cfg, 0, n=n)
    return cfg, occ, pose, lat, bvh, o, d, I.net_params(cfg, variant)


def test_log_distance_head_inverts_to_relu_of_the_logit(oracle):
    cfg, occ, pose, lat, bvh, o, d, P = _setup(oracle)
    a = oracle.query(cfg.nv, occ, lat, bvh, pose, P, o, d)
    b = oracle.query(cfg.nv, occ, lat, bvh, pose, P, o, d, dist_log=True)
    hit = a["voxel_id"] >= 0
    z1 = b["raw_logits"][hit, 1].astype(np.float64)
    assert (z1 > 0.05).sum() > 20 and (z1 < -0.05).sum() > 20
    # log(1 + D) = ReLU(z1): the network output is the log-transformed accumulated distance
    np.testing.assert_allclose(np.log1p(b["dist_total"][hit].astype(np.float64)), np.maximum(z1, 0), atol=3e-7, rtol=3e-7)
    assert (b["dist_total"][hit][z1 <= 0] == 0).all() and (b["dist_total"][hit] >= 0).all()
    np.testing.assert_allclose(b["distance"][hit], b["dist_total"][hit] - b["t_in"][hit], atol=5e-7)
    # monotone in the logit, and nothing else changes
    order = np.argsort(z1)
    assert (np.diff(b["dist_total"][hit][order]) >= 0).all()
    for k in ("voxel_id", "t_in", "t_out", "occlusion", "normal", "albedo", "material_logits", "raw_logits"):
        assert np.array_equal(a[k], b[k]), k
    assert not b["dist_total"][~hit].any() and not b["distance"][~hit].any()


def test_hit_position_lies_on_the_ray_at_the_accumulated_distance(oracle):
    cfg, occ, pose, lat, bvh, o, d, P = _setup(oracle)
    r = oracle.query(cfg.nv, occ, lat, bvh, pose, P, o, d, hit_positions=True)
    hit = r["voxel_id"] >= 0
    v = (r["hit_position"][hit] - o[hit]).astype(np.float64)
    dd = d[hit].astype(np.float64)
    np.testing.assert_allclose((v * dd).sum(1), r["dist_total"][hit], rtol=2e-6)      # projection on the ray
    assert np.abs(np.cross(v, dd)).max() < 2e-6                                      # no off-ray component
    assert not r["hit_position"][~hit].any() and not r["hit_position_rest"][~hit].any()


def test_identity_pose_rest_and_deformed_hit_positions_coincide(oracle):
    cfg, occ, pose, lat, bvh, o, d, P = _setup(oracle, pose=(0.0, 0.0))
    r = oracle.query(cfg.nv, occ, lat, bvh, pose, P, o, d, hit_positions=True)
    hit = r["voxel_id"] >= 0
    assert hit.sum() > 100
    np.testing.assert_allclose(r["hit_position_rest"][hit], r["hit_position"][hit], atol=2e-6)


def test_rest_hit_position_maps_forward_onto_the_deformed_one(oracle):
    # P:43 local linear approximation: the straight rest-space segment, pushed forward, deviates from
    # the straight deformed-space ray by O(h^2 x curvature) only; a wrong fraction, a swapped
    # endpoint or a wrong inverse is off by a voxel size.
    for pose in ((1.0, 0.0), (0.0, 0.8), (0.9, 0.6)):
        cfg, occ, pose, lat, bvh, o, d, P = _setup(oracle, pose=pose)
        r = oracle.query(cfg.nv, occ, lat, bvh, pose, P, o, d, hit_positions=True)
        hit = r["voxel_id"] >= 0
        h = 2.0 / cfg.nv
        fwd = oracle.forward_f64(float(pose[0]), float(pose[1]), r["hit_position_rest"][hit].astype(np.float64))
        dev = np.linalg.norm(fwd - r["hit_position"][hit], axis=1)
        assert dev.max() < 0.06 * h, (pose, dev.max() / h)
        ell = (r["t_out"] - r["t_in"])[hit]
        assert np.median(ell) > 0.2 * h                       # the segments are not degenerate


def test_rest_hit_position_fraction_special_cases(oracle):
    # all-zero network: sigmoid(0) = 1/2 -> the hit is the midpoint of the rest-space segment;
    # log head with z1 = 0: D = 0 -> distance = -t_in < 0 -> fraction clamps to 0 -> the entry point
    cfg, occ, pose, lat, bvh, o, d, P = _setup(oracle)
    P.weights = [np.zeros_like(w) for w in P.weights]
    r = oracle.query(cfg.nv, occ, lat, bvh, pose, P, o, d, hit_positions=True)
    hit = r["voxel_id"] >= 0
    ends = oracle.rest_endpoints(float(pose[0]), float(pose[1]), o, d, r["voxel_id"], r["t_in"], r["t_out"])
    ends = ends.reshape(-1, 2, 3)
    np.testing.assert_allclose(r["hit_position_rest"][hit], 0.5 * (ends[hit, 0] + ends[hit, 1]), atol=1e-6)
    r2 = oracle.query(cfg.nv, occ, lat, bvh, pose, P, o, d, dist_log=True, hit_positions=True)
    np.testing.assert_allclose(r2["hit_position_rest"][hit], ends[hit, 0], atol=1e-7)
    np.testing.assert_allclose(r2["hit_position"][hit], o[hit], atol=0)       # D = 0: the ray origin


def test_concatenation_encoding_layout_and_values(oracle):
    """O8b: psi(x) = [x, sin/cos bands, phi(x)].  gamma against numpy in fp64; the grid part against
    the composition encoding's sample-0 block (same phi, already pinned by test_oracle_encode.py)."""
    from dataclasses import replace
    cfg = I.get_config(0)
    shape_c = replace(cfg.net, enc_mode="concat")
    assert shape_c.d_in == 2 * (3 + 6 * cfg.net.pe_bands + cfg.net.levels * cfg.net.feat) == 70
    P = I.net_params(cfg, "varpres")
    Pc = I.net_params(replace(cfg, net=shape_c), "varpres")
    assert np.array_equal(P.table, Pc.table) and Pc.weights[0].shape == (cfg.net.width, 70)
    xn = np.random.default_rng(3).uniform(0, 1, (200, 3)).astype(np.float32)
    comp = oracle.encode(P, xn)
    cat = oracle.encode(Pc, xn)
    B, LF = cfg.net.pe_bands, cfg.net.levels * cfg.net.feat
    assert cat.shape == (200, 3 + 6 * B + LF)
    assert np.array_equal(cat[:, :3], xn)
    x64 = xn.astype(np.float64)
    for k in range(B):
        np.testing.assert_allclose(cat[:, 3 + 6 * k:6 + 6 * k], np.sin(2.0 ** k * x64), atol=2e-7)
        np.testing.assert_allclose(cat[:, 6 + 6 * k:9 + 6 * k], np.cos(2.0 ** k * x64), atol=2e-7)
    assert np.array_equal(cat[:, 3 + 6 * B:], comp[:, :LF])          # phi(x) = the s = 0 block of phi(gamma(x))


def test_concatenation_query_equals_mlp_of_the_concatenated_endpoint_encodings(oracle):
    from dataclasses import replace
    cfg = I.get_config(0)
    cfgc = replace(cfg, net=replace(cfg.net, enc_mode="concat"))
    occ = I.occupancy(cfg); pose = I.poses(cfg)[0]
    lat = oracle.deform_lattice(cfg.nv, *map(float, pose)); bvh = oracle.bvh_build(cfg.nv, occ, lat)
    o, d = I.rays(cfg, 0, n=300)
    Pc = I.net_params(cfgc, "varpres")
    r = oracle.query(cfg.nv, occ, lat, bvh, pose, Pc, o, d)
    hit = r["voxel_id"] >= 0
    ends = oracle.rest_endpoints(float(pose[0]), float(pose[1]), o, d, r["voxel_id"], r["t_in"], r["t_out"])[hit]
    xn = np.clip((ends + 1.0) * 0.5, 0.0, 1.0).astype(np.float32)
    feats = np.concatenate([oracle.encode(Pc, xn[:, 0]), oracle.encode(Pc, xn[:, 1])], axis=1)   # entry then exit (R15)
    z = oracle.mlp(Pc, feats)
    np.testing.assert_allclose(r["raw_logits"][hit], z, atol=2e-6, rtol=1e-5)
