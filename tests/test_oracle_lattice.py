"""Pins for O7b, the voxel-local trilinear inverse used when the deformation is given only as a
deformed corner lattice (R27).  CPU only."""
import numpy as np

import nif_inputs as I


def _trilinear(q, uvw):
    """textbook trilinear interpolation of 8 corners q[c], c = dx + 2 dy + 4 dz (fp64)"""
    u, v, w = uvw
    out = np.zeros(3)
    for c in range(8):
        b = (u if c & 1 else 1 - u) * (v if c & 2 else 1 - v) * (w if c & 4 else 1 - w)
        out += b * q[c]
    return out


def _corners(lat, nv, vid):
    ix, iy, iz = vid % nv, (vid // nv) % nv, vid // (nv * nv)
    np1 = nv + 1
    return np.array([lat[(ix + (c & 1)) + np1 * ((iy + ((c >> 1) & 1)) + np1 * (iz + (c >> 2)))] for c in range(8)],
                    dtype=np.float64), np.array([ix, iy, iz])


def test_solution_substituted_back_reproduces_the_point(oracle):
    # the defining equation T(u,v,w) = P, checked by substitution with an independent fp64 trilinear
    nv = 8
    rng = np.random.default_rng(0)
    for pose in ((1.0, 0.0), (0.0, 0.8), (1.3, 0.9)):
        lat = oracle.deform_lattice(nv, *pose)
        vids = rng.integers(0, nv ** 3, 200).astype(np.int32)
        uvw = rng.uniform(0, 1, (200, 3))
        P = np.array([_trilinear(_corners(lat, nv, int(v))[0], t) for v, t in zip(vids, uvw)], dtype=np.float32)
        rest = oracle.inverse_trilinear(lat, nv, vids, P)
        for i in range(200):
            q, cell = _corners(lat, nv, int(vids[i]))
            got_uvw = (rest[i].astype(np.float64) + 1.0) * nv / 2.0 - cell
            assert np.abs(_trilinear(q, got_uvw) - P[i]).max() < 2e-6
            assert np.abs(got_uvw - uvw[i]).max() < 2e-4


def test_affine_lattice_gives_the_exact_affine_inverse(oracle):
    # a lattice that is an affine image of the rest lattice: the trilinear interpolant IS that affine map
    nv = 6
    rng = np.random.default_rng(1)
    A = np.eye(3) + 0.3 * rng.standard_normal((3, 3)); b = rng.uniform(-0.2, 0.2, 3)
    g = (2.0 * np.arange(nv + 1) - nv) / nv
    z, y, x = np.meshgrid(g, g, g, indexing="ij")
    rest_lat = np.stack([x.ravel(), y.ravel(), z.ravel()], axis=1)
    lat = np.ascontiguousarray((rest_lat @ A.T + b).astype(np.float32))
    vids = rng.integers(0, nv ** 3, 300).astype(np.int32)
    cells = np.stack([vids % nv, (vids // nv) % nv, vids // (nv * nv)], axis=1)
    rest_true = (2.0 * (cells + rng.uniform(0, 1, (300, 3))) - nv) / nv
    P = (rest_true @ A.T + b).astype(np.float32)
    rest = oracle.inverse_trilinear(lat, nv, vids, P)
    np.testing.assert_allclose(rest, rest_true, atol=3e-6)
    # identity lattice: identity
    rest_id = oracle.inverse_trilinear(np.ascontiguousarray(rest_lat.astype(np.float32)), nv, vids, rest_true.astype(np.float32))
    np.testing.assert_allclose(rest_id, rest_true, atol=1e-6)


def test_local_inverse_approaches_the_closed_form_inverse_quadratically(oracle):
    # the field is approximately linear inside a voxel -- the voxel-local inverse of a twist+bend
    # lattice differs from the closed-form inverse by O(h^2): halving h must cut the error ~4x
    errs = []
    for nv in (8, 16, 32):
        pose = (0.9, 0.6)
        lat = oracle.deform_lattice(nv, *pose)
        rng = np.random.default_rng(2)
        vids = rng.integers(0, nv ** 3, 400).astype(np.int32)
        cells = np.stack([vids % nv, (vids // nv) % nv, vids // (nv * nv)], axis=1)
        rest_true = (2.0 * (cells + rng.uniform(0, 1, (400, 3))) - nv) / nv
        P = oracle.forward_f64(pose[0], pose[1], rest_true).astype(np.float32)
        rest = oracle.inverse_trilinear(lat, nv, vids, P)
        errs.append(np.abs(rest - rest_true).max())
    # absolute error: 0.05 voxel at nv = 8, then at least 2.5x smaller per halving of h (4x in the limit;
    # the maximum over a random sample is noisy)
    assert errs[0] < 0.05 * 0.25 and errs[1] < errs[0] / 2.5 and errs[2] < errs[1] / 2.5, errs


def test_query_with_lattice_inverse_stays_close_to_the_closed_form_query(oracle):
    cfg = I.get_config(0)
    occ = I.occupancy(cfg); pose = I.poses(cfg)[0]
    lat = oracle.deform_lattice(cfg.nv, *map(float, pose)); bvh = oracle.bvh_build(cfg.nv, occ, lat)
    o, d = I.rays(cfg, 0, n=400)
    P = I.net_params(cfg, "varpres")
    a = oracle.query(cfg.nv, occ, lat, bvh, pose, P, o, d, hit_positions=True)
    b = oracle.query(cfg.nv, occ, lat, bvh, pose, P, o, d, hit_positions=True, lattice_inverse=True)
    hit = a["voxel_id"] >= 0
    for k in ("voxel_id", "t_in", "t_out"):
        assert np.array_equal(a[k], b[k])
    h = 2.0 / cfg.nv
    assert np.abs(a["hit_position_rest"][hit] - b["hit_position_rest"][hit]).max() < 0.05 * h
    assert np.abs(a["hit_position_rest"][hit] - b["hit_position_rest"][hit]).max() > 0          # it is a different map
    # the network sees slightly different points: outputs move a little, not wildly
    assert np.abs(a["occlusion"][hit] - b["occlusion"][hit]).max() < 0.2
