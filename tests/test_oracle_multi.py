"""Pins for O11, the multi-voxel walk of the oracle (R22).
CPU only.  Each pin is something the paper or the geometry fixes, not a re-run of the oracle's
own formula: brute force over all voxels, the per-voxel test enumerated independently, the
straight-line closed form of the segmented distance, the DDA sequence on the undeformed grid,
and networks built so that the walk's outcome is known in advance."""
import math

import numpy as np
import pytest

import nif_inputs as I


def _setup(oracle, nv=8, fill=0.5, seed=0, pose=(0.7, 0.5)):
    occ = I.random_occupancy(nv, fill, seed)
    lat = oracle.deform_lattice(nv, *pose)
    bvh = oracle.bvh_build(nv, occ, lat)
    cfg = I.scaled(I.get_config(0), nv=nv)
    o, d = I.rays(cfg, 0, n=200)
    return occ, lat, bvh, o, d


@pytest.mark.parametrize("seed", range(3))
def test_successor_bvh_equals_brute_force(oracle, seed):
    nv = [8, 6, 10][seed]
    occ, lat, bvh, o, d = _setup(oracle, nv=nv, fill=0.4 + 0.1 * seed, seed=seed)
    n = len(o)
    at = np.full(n, -np.inf, np.float32); ai = np.full(n, -1, np.int32)
    for _ in range(6):                                   # walk six voxels deep, both ways in lockstep
        vb, tib, tob = oracle.next_voxel_brute(nv, occ, lat, o, d, at, ai)
        vh, tih, toh = bvh.next_voxel(o, d, at, ai)
        assert np.array_equal(vb, vh)
        assert np.array_equal(tib.view(np.int32), tih.view(np.int32))
        assert np.array_equal(tob.view(np.int32), toh.view(np.int32))
        live = vb >= 0
        at = np.where(live, tib, at); ai = np.where(live, vb, ai)
    # the first successor of (-inf, -1) is the plain nearest-voxel query
    v0, t0, _ = oracle.traverse_brute(nv, occ, lat, o, d)
    v1, t1, _ = oracle.next_voxel_brute(nv, occ, lat, o, d, np.full(n, -np.inf, np.float32), np.full(n, -1, np.int32))
    assert np.array_equal(v0, v1) and np.array_equal(t0.view(np.int32), t1.view(np.int32))


def test_walk_enumerates_exactly_the_voxels_the_ray_hits_in_order(oracle):
    nv = 8
    occ, lat, bvh, o, d = _setup(oracle, nv=nv, fill=0.6, seed=3)
    ids = np.nonzero(occ)[0]
    for r in range(0, len(o), 7):
        # independent enumeration: the per-voxel test on every occupied voxel
        want = []
        for vid in ids:
            hit, ti, _ = oracle.voxel_hit(lat, nv, int(vid), o[r], d[r])
            if hit:
                want.append((np.float32(ti), int(vid)))
        want.sort()
        got = []
        at = np.array([-np.inf], np.float32); ai = np.array([-1], np.int32)
        while True:
            v, ti, _ = bvh.next_voxel(o[r:r + 1], d[r:r + 1], at, ai)
            if v[0] < 0:
                break
            got.append((np.float32(ti[0]), int(v[0])))
            at, ai = ti.copy(), v.copy()
        assert got == want


def test_identity_pose_axis_ray_visits_the_row_like_a_dda(oracle):
    # undeformed grid: a ray along +x through the middle of a row visits that row's occupied
    # voxels left to right, entering voxel i at x = -1 + i*h (closed form)
    nv = 8; h = 2.0 / nv
    occ = np.zeros(nv ** 3, np.uint8)
    iy, iz = 3, 5
    row = [0, 2, 3, 6]
    for ix in row:
        occ[ix + nv * (iy + nv * iz)] = 1
    lat = oracle.deform_lattice(nv, 0.0, 0.0)
    bvh = oracle.bvh_build(nv, occ, lat)
    o = np.array([[-3.0, -1 + (iy + 0.5) * h, -1 + (iz + 0.5) * h]], np.float32)
    d = np.array([[1.0, 0.0, 0.0]], np.float32)
    at = np.array([-np.inf], np.float32); ai = np.array([-1], np.int32)
    for ix in row:
        v, ti, to = bvh.next_voxel(o, d, at, ai)
        assert v[0] == ix + nv * (iy + nv * iz)
        assert abs(ti[0] - (2.0 + ix * h)) < 1e-6 and abs(to[0] - (2.0 + (ix + 1) * h)) < 1e-6
        at, ai = ti.copy(), v.copy()
    assert bvh.next_voxel(o, d, at, ai)[0][0] == -1


def _params(cfg, kind):
    P = I.net_params(cfg, "varpres")
    if kind == "always_accept":           # all weights zero -> every logit 0 -> occlusion = 0.5 >= 0.5
        P.weights = [np.zeros_like(w) for w in P.weights]
    elif kind == "never_accept":          # positive table and hidden weights -> positive activations; z0 = -sum
        P.table = np.full_like(P.table, 0.5)
        P.weights = [np.full_like(w, 0.01) for w in P.weights]
        P.weights[-1][0, :] = -1.0
    return P


def test_all_zero_network_accepts_the_first_voxel(oracle):
    cfg = I.get_config(0)
    occ = I.occupancy(cfg); pose = I.poses(cfg)[0]
    lat = oracle.deform_lattice(cfg.nv, *map(float, pose)); bvh = oracle.bvh_build(cfg.nv, occ, lat)
    o, d = I.rays(cfg, 0, n=300)
    P = _params(cfg, "always_accept")
    single = oracle.query(cfg.nv, occ, lat, bvh, pose, P, o, d)
    multi = oracle.query_multi(cfg.nv, occ, lat, bvh, pose, P, o, d, max_steps=8)
    hit = single["voxel_id"] >= 0
    assert np.array_equal(multi["voxel_id"], single["voxel_id"])
    assert np.array_equal(multi["status"], hit.astype(np.int32)) and np.array_equal(multi["steps"], hit.astype(np.int32))
    for k in ("t_in", "occlusion", "distance", "dist_total", "normal"):
        assert np.array_equal(multi[k][hit], single[k][hit]), k


def test_never_accepting_network_walks_every_voxel_and_reports_a_miss(oracle):
    cfg = I.scaled(I.get_config(0), nv=8)
    occ = I.random_occupancy(8, 0.5, 11); pose = (0.6, 0.4)
    lat = oracle.deform_lattice(8, *pose); bvh = oracle.bvh_build(8, occ, lat)
    o, d = I.rays(cfg, 0, n=120)
    P = _params(cfg, "never_accept")
    multi = oracle.query_multi(8, occ, lat, bvh, pose, P, o, d, max_steps=64)
    ids = np.nonzero(occ)[0]
    for r in range(len(o)):
        crossed = sum(oracle.voxel_hit(lat, 8, int(v), o[r], d[r])[0] for v in ids)
        assert multi["steps"][r] == crossed and multi["status"][r] == 0
    assert (multi["voxel_id"] == -1).all() and not multi["occlusion"].any() and np.isinf(multi["t_in"]).all()
    # with a step budget smaller than the crossing count the walk stops with status 2 on the budget-th voxel
    capped = oracle.query_multi(8, occ, lat, bvh, pose, P, o, d, max_steps=2)
    long = multi["steps"] > 2
    assert (capped["status"][long] == 2).all() and (capped["steps"][long] == 2).all()
    assert (capped["voxel_id"][long] >= 0).all()


def test_segmented_distance_sum_reduces_to_the_straight_line_parameter(oracle):
    # P:61 sums segment and gap lengths along one straight ray with a unit direction; with signed
    # gaps (R23) the sum telescopes to t_in,k + t_k (= dist_total of voxel k).  The oracle
    # accumulates it term by term: a dropped or doubled term breaks this equality.
    cfg = I.get_config(0)
    occ = I.occupancy(cfg); pose = I.poses(cfg)[0]
    lat = oracle.deform_lattice(cfg.nv, *map(float, pose)); bvh = oracle.bvh_build(cfg.nv, occ, lat)
    o, d = I.rays(cfg, 0, n=400)
    multi = oracle.query_multi(cfg.nv, occ, lat, bvh, pose, I.net_params(cfg, "varpres"), o, d, max_steps=16)
    acc = multi["status"] == 1
    assert acc.sum() > 50 and (multi["steps"][acc] > 1).sum() > 10      # some rays accept beyond the first voxel
    np.testing.assert_allclose(multi["dist_accum"][acc], multi["dist_total"][acc], rtol=3e-6, atol=3e-6)
    assert (multi["occlusion"][acc] >= 0.5).all()
    ell = multi["t_out"][acc] - multi["t_in"][acc]
    assert (multi["distance"][acc] >= 0).all() and (multi["distance"][acc] <= ell * (1 + 1e-6)).all()


def test_paper_norm_form_of_the_sum_on_non_overlapping_segments(oracle):
    # P:59 defines delta_i and l_i as NORMS of differences of entry/exit points.  On the undeformed
    # grid the segments of a row do not overlap, and the norm form, evaluated here in numpy from the
    # points, must equal the oracle's accumulated value.
    nv = 8; h = 2.0 / nv
    occ = np.zeros(nv ** 3, np.uint8)
    iy, iz = 2, 4
    row = [1, 2, 5, 7]
    for ix in row:
        occ[ix + nv * (iy + nv * iz)] = 1
    lat = oracle.deform_lattice(nv, 0.0, 0.0); bvh = oracle.bvh_build(nv, occ, lat)
    o = np.array([[-2.5, -1 + (iy + 0.4) * h, -1 + (iz + 0.6) * h]], np.float32)
    d = np.array([[1.0, 0.0, 0.0]], np.float32)
    cfg = I.scaled(I.get_config(0), nv=nv)
    P = _params(cfg, "never_accept")
    m = oracle.query_multi(nv, occ, lat, bvh, (0.0, 0.0), P, o, d, max_steps=3)     # stops on the 3rd voxel
    assert m["status"][0] == 2 and m["steps"][0] == 3
    pts = []                                                                      # (entry, exit) points, in order
    at = np.array([-np.inf], np.float32); ai = np.array([-1], np.int32)
    for _ in range(3):
        v, ti, to = bvh.next_voxel(o, d, at, ai)
        pts.append((o[0] + ti[0] * d[0], o[0] + to[0] * d[0]))
        at, ai = ti.copy(), v.copy()
    prev = o[0].astype(np.float64); total = 0.0
    for x0, x1 in pts:
        total += np.linalg.norm(x0 - prev) + np.linalg.norm(x1 - x0); prev = x1
    assert abs(m["dist_accum"][0] - total) < 1e-5


def test_trace_is_the_walk_without_stopping(oracle):
    # the trace lists the ray's voxel sequence with each voxel's occlusion logit; the walk must stop at
    # the first non-negative one (sigmoid(z) >= 0.5 <=> z >= 0), and the sequence must be the successor
    # chain (ids from next_voxel).
    cfg = I.get_config(0)
    occ = I.occupancy(cfg); pose = I.poses(cfg)[0]
    lat = oracle.deform_lattice(cfg.nv, *map(float, pose)); bvh = oracle.bvh_build(cfg.nv, occ, lat)
    o, d = I.rays(cfg, 0, n=300)
    P = I.net_params(cfg, "varpres")
    K = 12
    tid, tz = oracle.walk_trace(cfg.nv, occ, lat, bvh, pose, P, o, d, K)
    multi = oracle.query_multi(cfg.nv, occ, lat, bvh, pose, P, o, d, max_steps=K)
    at = np.full(len(o), -np.inf, np.float32); ai = np.full(len(o), -1, np.int32)
    for k in range(K):
        v, ti, _ = bvh.next_voxel(o, d, at, ai)
        assert np.array_equal(v, tid[:, k])
        live = v >= 0
        at = np.where(live, ti, at); ai = np.where(live, v, ai)
    clear = np.abs(tz) > 1e-6
    for r in range(len(o)):
        if not clear[r][tid[r] >= 0].all():
            continue
        acc = np.nonzero((tid[r] >= 0) & (tz[r] >= 0))[0]
        n_vox = int((tid[r] >= 0).sum())
        if len(acc):
            assert multi["status"][r] == 1 and multi["steps"][r] == acc[0] + 1 and multi["voxel_id"][r] == tid[r, acc[0]]
        elif n_vox < K:
            assert multi["status"][r] == 0 and multi["steps"][r] == n_vox and multi["voxel_id"][r] == -1
        else:
            assert multi["status"][r] == 2 and multi["steps"][r] == K and multi["voxel_id"][r] == tid[r, K - 1]


# ---- O11x: the literal exit-face walk of P:51 pins reading R22 (successor order) --------------------
def _successor_sequences(bvh, o, d, max_vox):
    n = len(o)
    seq = np.full((n, max_vox), -1, np.int32)
    tin = np.full((n, max_vox), np.nan, np.float32); tout = tin.copy()
    at = np.full(n, -np.inf, np.float32); ai = np.full(n, -1, np.int32)
    live = np.arange(n)
    for k in range(max_vox):
        vid, ti, to = bvh.next_voxel(o[live], d[live], at[live], ai[live])
        ok = vid >= 0
        seq[live[ok], k] = vid[ok]; tin[live[ok], k] = ti[ok]; tout[live[ok], k] = to[ok]
        at[live[ok]] = ti[ok]; ai[live[ok]] = vid[ok]
        live = live[ok]
        if len(live) == 0:
            break
    return seq, tin, tout


EXIT_FACE_CASES = [  # name, config, pose index, rays, lattice kind, minimum fraction of identical sequences
    ("cfg0 twist", 0, 0, 4096, "pose", 0.995),
    ("cfg1 bend (reduced frame)", 1, 0, 20_000, "pose", 0.999),
    ("cfg2 twist+bend, pose 5 (reduced)", 2, 5, 5_000, "pose", 0.995),
    ("wavy user lattice", 0, 0, 4096, "wavy", 0.999),
    ("cfg0 identity", 0, 0, 4096, "identity", 0.999),
]


@pytest.mark.parametrize("name,cfg_id,pose_index,n_rays,kind,min_same", EXIT_FACE_CASES)
def test_exit_face_walk_visits_the_successor_sequence(oracle, name, cfg_id, pose_index, n_rays, kind, min_same):
    """P:51 words the walk as "determine the face through which the ray exits, select the neighbouring voxel";
    the product (and O11) define it as the successor in (t_in, id) order over all occupied voxels (R22).
    On a conforming lattice the two visit the same occupied voxels in the same order, except where "the
    exit face" is not a well-defined notion:
      (i)  a warped (non-convex) voxel the ray crosses twice: the literal walk leaves it at its LAST crossing
           and never sees the voxels in the notch between the two crossings; the successor order lists them
           after it (their [t_in, t_out] lies inside the crossed-twice voxel's);
      (ii) a ray through a lattice edge or corner: the next cell is only touched (status 1: no progress).
    Every differing ray must be of kind (i) or (ii), and they must be rare."""
    cfg = I.get_config(cfg_id)
    occ = I.occupancy(cfg)
    pose = I.poses(cfg)[pose_index]
    if kind == "wavy":
        lat = I.wavy_lattice(cfg.nv, 3)
    elif kind == "identity":
        lat = oracle.deform_lattice(cfg.nv, 0.0, 0.0)
    else:
        lat = oracle.deform_lattice(cfg.nv, float(pose[0]), float(pose[1]))
    bvh = oracle.bvh_build(cfg.nv, occ, lat)
    lo, hi = bvh.bounds()
    o, d = I.rays(cfg, pose_index, lo, hi, n=n_rays)
    M = 3 * cfg.nv
    seq, status = oracle.exit_face_walk(cfg.nv, occ, lat, bvh, o, d, M)
    suc, tin, tout = _successor_sequences(bvh, o, d, M)
    hit = suc[:, 0] >= 0
    assert hit.sum() > 1000 and np.array_equal(seq[:, 0], suc[:, 0])          # same first voxel, same misses
    assert (status[~hit] == -1).all() and np.isin(status[hit], (0, 1)).all()  # never "no triangle", never truncated
    same = (seq == suc).all(axis=1)
    assert same[hit].mean() >= min_same, (name, same[hit].mean())
    n_notch = n_touch = 0
    for r in np.nonzero(hit & ~same)[0]:
        E = [int(v) for v in seq[r] if v >= 0]
        S = [(int(v), float(a), float(b)) for v, a, b in zip(suc[r], tin[r], tout[r]) if v >= 0]
        ids = [v for v, _, _ in S]
        pos = [ids.index(v) for v in E]                       # every voxel of the literal walk is in the successor list ...
        assert pos == sorted(pos), (name, r)                  # ... in the same order
        iv = {v: (a, b) for v, a, b in S}
        # a walk that stopped (ii) misses everything from the touched cell on (ties in t_in included)
        tol = 4e-6 * max(1.0, abs(iv[E[-1]][1]))              # a few fp32 ulps of t
        t_stop = np.inf if status[r] == 0 else iv[E[-1]][0] - tol
        skipped = [v for v in ids if v not in E and iv[v][0] < t_stop]
        for v in skipped:                                     # (i): nested inside a voxel the literal walk did visit
            a, b = iv[v]
            assert any(iv[e][0] <= a + tol and b <= iv[e][1] + tol for e in E), (name, r, v)
        if status[r] == 1:
            n_touch += 1
        else:
            assert skipped, (name, r)                         # status 0: the only difference is notch voxels
            n_notch += 1
    if kind == "identity":
        assert n_notch == 0                                   # cubes are convex
