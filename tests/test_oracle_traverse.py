"""Pins for oracle steps O3-O6 (ray / deformed-voxel intersection and the nearest-voxel query).

Closed forms and invariants only; the BVH is checked bit-exactly against the brute-force
definition (BASELINE.json:5 "BVH hits match brute force over all deformed voxels on tiny grids").
"""
import math

import numpy as np
import pytest

import nif_inputs as I


def _slab_f64(lo, hi, o, d):
    """Textbook slab test in fp64 for an axis-aligned cube (the closed form the identity pose
    must reduce to)."""
    with np.errstate(divide="ignore", invalid="ignore"):
        t0 = (lo - o) / d
        t1 = (hi - o) / d
    tn = np.max(np.minimum(t0, t1)); tf = np.min(np.maximum(t0, t1))
    return tn, tf


def _ulps(a, b):
    a = np.float32(a); b = np.float32(b)
    return abs(float(a) - float(b)) / float(np.spacing(max(abs(a), abs(b), np.float32(1e-30))))


def test_identity_pose_voxel_is_a_cube_slab_closed_form(oracle):
    # zero pose => each voxel is an axis-aligned cube => t_in/t_out equal the slab closed form
    nv = 8
    lat = oracle.deform_lattice(nv, 0.0, 0.0)
    rng = np.random.default_rng(0)
    h = 2.0 / nv
    n_hit = 0
    for _ in range(3000):
        vid = int(rng.integers(0, nv ** 3))
        ix, iy, iz = vid % nv, (vid // nv) % nv, vid // (nv * nv)
        lo = np.array([ix, iy, iz]) * h - 1.0
        o = rng.standard_normal(3); o = 3.0 * o / np.linalg.norm(o)
        tgt = lo + rng.uniform(-0.3, 1.3, 3) * h
        d = tgt - o; d /= np.linalg.norm(d)
        o32 = o.astype(np.float32); d32 = d.astype(np.float32)
        hit, ti, to = oracle.voxel_hit(lat, nv, vid, o32, d32)
        tn, tf = _slab_f64(lo, lo + h, o32.astype(np.float64), d32.astype(np.float64))
        margin = 1e-5                       # closed form decides hit/miss away from the silhouette
        if tn < tf - margin and tf > 0:
            assert hit
            n_hit += 1
            # |t| ~ 3, box at |x| <= 1: absolute error budget of a few ulp of t
            assert abs(ti - max(tn, 0.0)) <= 4 * np.spacing(np.float32(3.0)), (ti, tn)
            assert abs(to - tf) <= 4 * np.spacing(np.float32(4.0)), (to, tf)
        elif tn > tf + margin or tf < -margin:
            assert not hit
    assert n_hit > 300


def test_reversed_ray_swaps_entry_and_exit(oracle):
    # ray from o + T d along -d through one voxel: t_in' = T - t_out, t_out' = T - t_in
    nv = 8
    lat = oracle.deform_lattice(nv, 0.9, 0.7)
    rng = np.random.default_rng(1)
    n = 0
    for _ in range(2000):
        vid = int(rng.integers(0, nv ** 3))
        o = rng.standard_normal(3); o = 3.0 * o / np.linalg.norm(o)
        centre = lat.reshape(nv + 1, nv + 1, nv + 1, 3)[vid // 64, (vid // 8) % 8, vid % 8]
        d = centre + rng.uniform(0, 0.2, 3) - o; d /= np.linalg.norm(d)
        o32 = o.astype(np.float32); d32 = d.astype(np.float32)
        hit, ti, to = oracle.voxel_hit(lat, nv, vid, o32, d32)
        if not hit or to - ti < 1e-3:
            continue
        T = np.float32(8.0)
        o2 = (o32.astype(np.float64) + float(T) * d32.astype(np.float64)).astype(np.float32)
        hit2, ti2, to2 = oracle.voxel_hit(lat, nv, vid, o2, -d32)
        assert hit2
        assert abs(ti2 - (float(T) - to)) <= 1e-5 * 8 and abs(to2 - (float(T) - ti)) <= 1e-5 * 8
        n += 1
    assert n > 200


def test_origin_inside_voxel_gives_t_in_zero(oracle):
    # B:10 "origins uniform inside the deformed bounding box"; R11
    nv = 4
    lat = oracle.deform_lattice(nv, 0.5, 0.3)
    L = lat.reshape(nv + 1, nv + 1, nv + 1, 3)
    vid = 1 + nv * (2 + nv * 1)
    centre = L[1:3, 2:4, 1:3].reshape(-1, 3).mean(0)
    rng = np.random.default_rng(2)
    for _ in range(50):
        d = rng.standard_normal(3); d /= np.linalg.norm(d)
        hit, ti, to = oracle.voxel_hit(lat, nv, vid, centre, d)
        assert hit and ti == 0.0 and 0 < to < 1.0


def test_voxel_behind_origin_is_a_miss(oracle):
    nv = 4
    lat = oracle.deform_lattice(nv, 0.0, 0.0)
    hit, _, _ = oracle.voxel_hit(lat, nv, 0, [3.0, -0.75, -0.75], [1.0, 0.0, 0.0])
    assert not hit
    hit, ti, to = oracle.voxel_hit(lat, nv, 0, [3.0, -0.75, -0.75], [-1.0, 0.0, 0.0])
    assert hit and ti == 3.5 and to == 4.0


def test_tie_on_t_in_lowest_id_wins_and_edges_are_inclusive(oracle):
    # R9/R12: a ray lying in the plane shared by two voxel layers enters both at the same t;
    # the faces in that plane are parallel (det == 0 rejects) and the ray crosses the side
    # faces exactly on their shared edge (u or v == 0: inclusive).  Lowest id must win.
    nv = 4
    occ = np.ones(nv ** 3, np.uint8)
    lat = oracle.deform_lattice(nv, 0.0, 0.0)
    o = np.array([[-3.0, 0.0, 0.25]], np.float32)     # y = 0 is the lattice plane j = 2
    d = np.array([[1.0, 0.0, 0.0]], np.float32)
    vid, ti, to = oracle.traverse_brute(nv, occ, lat, o, d)
    lower = 0 + nv * (1 + nv * 2)                        # iy = 1 (below the plane), iz = 2
    upper = 0 + nv * (2 + nv * 2)
    h1, t1, _ = oracle.voxel_hit(lat, nv, lower, o[0], d[0])
    h2, t2, _ = oracle.voxel_hit(lat, nv, upper, o[0], d[0])
    assert h1 and h2 and t1 == t2 == 2.0
    assert vid[0] == lower and ti[0] == 2.0 and to[0] == 2.5
    bvh = oracle.bvh_build(nv, occ, lat)
    vb, tib, tob = bvh.traverse(o, d)
    assert vb[0] == lower and tib[0] == 2.0 and tob[0] == 2.5


def test_miss_convention(oracle):
    nv = 4
    occ = np.zeros(nv ** 3, np.uint8); occ[5] = 1
    lat = oracle.deform_lattice(nv, 0.2, 0.1)
    o = np.array([[0.0, 5.0, 0.0]], np.float32); d = np.array([[0.0, 1.0, 0.0]], np.float32)
    for fn in (lambda: oracle.traverse_brute(nv, occ, lat, o, d),
               lambda: oracle.bvh_build(nv, occ, lat).traverse(o, d)):
        vid, ti, to = fn()
        assert vid[0] == -1 and np.isinf(ti[0]) and np.isinf(to[0])


def test_bvh_equals_brute_force_config0(oracle):
    cfg = I.get_config(0)
    occ = I.occupancy(cfg); pose = I.poses(cfg)[0]
    lat = oracle.deform_lattice(cfg.nv, *pose)
    o, d = I.rays(cfg)
    vb, tib, tob = oracle.traverse_brute(cfg.nv, occ, lat, o, d)
    v, ti, to = oracle.bvh_build(cfg.nv, occ, lat).traverse(o, d)
    assert np.array_equal(v, vb) and np.array_equal(ti, tib) and np.array_equal(to, tob)
    assert (v >= 0).mean() > 0.9


@pytest.mark.parametrize("seed", range(6))
def test_bvh_equals_brute_force_random_grids(oracle, seed):
    rng = np.random.default_rng(100 + seed)
    nv = 8
    occ = I.random_occupancy(nv, fill=float(rng.uniform(0.05, 0.6)), seed=seed)
    th, k = float(rng.uniform(0, math.pi / 2)), float(rng.uniform(0, 0.9))
    lat = oracle.deform_lattice(nv, th, k)
    bvh = oracle.bvh_build(nv, occ, lat)
    lo, hi = bvh.bounds()
    n = 1500
    # outside-in rays, inside-out rays (origins in the box), axis-parallel rays
    o1 = 3.0 * rng.standard_normal((n, 3)); o1 /= np.linalg.norm(o1, axis=1, keepdims=True) / 3.0
    d1 = rng.uniform(lo, hi, (n, 3)) - o1
    o2 = rng.uniform(lo, hi, (n, 3)); d2 = rng.standard_normal((n, 3))
    o3 = rng.uniform(lo, hi, (300, 3)); d3 = np.eye(3)[rng.integers(0, 3, 300)] * rng.choice([-1, 1], (300, 1))
    o = np.concatenate([o1, o2, o3]); d = np.concatenate([d1, d2, d3])
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    o = o.astype(np.float32); d = d.astype(np.float32)
    vb, tib, tob = oracle.traverse_brute(nv, occ, lat, o, d)
    v, ti, to = bvh.traverse(o, d)
    assert np.array_equal(v, vb) and np.array_equal(ti, tib) and np.array_equal(to, tob)
    assert 0.05 < (v >= 0).mean()


@pytest.mark.parametrize("cfg_id,n", [(0, 4096), (1, 20000)])
def test_rest_images_of_entry_and_exit_lie_in_the_hit_voxels_rest_cell(oracle, cfg_id, n):
    # O5-O7 invariant: a wrong id or a wrong inverse is off by >= one voxel edge h; the local
    # linearisation keeps the mapped endpoints within a fraction of h.
    cfg = I.get_config(cfg_id)
    occ = I.occupancy(cfg); pose = I.poses(cfg)[0]
    lat = oracle.deform_lattice(cfg.nv, *pose)
    bvh = oracle.bvh_build(cfg.nv, occ, lat)
    lo, hi = bvh.bounds()
    o, d = I.rays(cfg, 0, lo, hi, n=n)
    v, ti, to = bvh.traverse(o, d)
    hit = v >= 0
    assert hit.sum() > 500
    rest = oracle.rest_endpoints(pose[0], pose[1], o, d, v, ti, to)[hit]      # [m, 2, 3]
    nv = cfg.nv; h = 2.0 / nv
    ids = v[hit]
    cell_lo = np.stack([ids % nv, (ids // nv) % nv, ids // (nv * nv)], -1) * h - 1.0
    below = (cell_lo[:, None, :] - rest).max()
    above = (rest - (cell_lo[:, None, :] + h)).max()
    assert max(below, above) <= 0.25 * h, (below / h, above / h)
    assert occ[ids].all()
