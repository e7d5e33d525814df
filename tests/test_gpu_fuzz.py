"""`-m gpu`: randomised traversal parity against the brute-force definition (oracle O4-O6): random small grids,
occupancies and poses (twists up to +-3.5 rad, bends of either sign), four families of rays including the
degenerate ones -- axis-parallel directions with +-0 components and origins on (or one float away from) lattice
planes, and rays aimed exactly at deformed lattice corners (edge and corner ties).  Ids and t bit-exact, both
traversal kernels."""
import numpy as np
import pytest
import torch

import nif_inputs as I

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("seed", [1, 2])
def test_random_scenes_bit_exact(oracle, seed):
    import harness as H
    import paper_2604_24666_b200 as nif
    rng = np.random.default_rng(seed)
    done = 0
    for it in range(40):
        nv = int(rng.choice([2, 3, 4, 5, 7, 8, 11, 16]))
        occ = (rng.random(nv ** 3) < rng.uniform(0.05, 1.0)).astype(np.uint8)
        if not occ.any():
            occ[rng.integers(nv ** 3)] = 1
        theta = float(rng.choice([0.0, rng.uniform(-3.5, 3.5)]))
        k = float(rng.choice([0.0, rng.uniform(-0.9, 0.9)]))
        cfg = I.scaled(I.get_config(0), nv=nv)
        try:
            case = H.make_case(0, with_net=False, cfg=cfg, occ=occ, pose=[theta, k])
        except nif.NifError as e:                      # a bend that folds the grid over is rejected (R7)
            assert e.status == -3
            continue
        lat = oracle.deform_lattice(nv, theta, k)
        info = case.bvh.info()
        lo, hi = info["lo"].astype(np.float64), info["hi"].astype(np.float64)
        n = 2000
        kind = it % 4
        if kind == 0:                                  # from outside towards the box
            o = rng.standard_normal((n, 3)); o *= 3.0 / np.linalg.norm(o, axis=1, keepdims=True)
            d = rng.uniform(lo, hi, (n, 3)) - o
        elif kind == 1:                                # origins inside, random directions
            o = rng.uniform(lo, hi, (n, 3)); d = rng.standard_normal((n, 3))
        elif kind == 2:                                # axis-parallel, origins on / next to lattice planes, +-0 components
            g = (2.0 * np.arange(nv + 1) - nv) / nv
            o = rng.choice(g, (n, 3)) + rng.choice([0.0, 0.0, 1e-7, -1e-7], (n, 3))
            d = np.zeros((n, 3)); ax = rng.integers(0, 3, n); d[np.arange(n), ax] = rng.choice([-1.0, 1.0], n)
            o[np.arange(n), ax] -= 3.0 * d[np.arange(n), ax]
            d[d == 0] = rng.choice([0.0, -0.0], int((d == 0).sum()))
        else:                                          # through deformed lattice corners
            o = rng.standard_normal((n, 3)); o *= 3.0 / np.linalg.norm(o, axis=1, keepdims=True)
            d = lat[rng.integers(0, len(lat), n)].astype(np.float64) - o
        d = d / np.linalg.norm(d, axis=1, keepdims=True)
        o = np.ascontiguousarray(o, np.float32); d = np.ascontiguousarray(d, np.float32)
        case.origin, case.direction = o, d
        case.origin_d, case.direction_d = torch.from_numpy(o).cuda(), torch.from_numpy(d).cuda()
        vid, ti, to = oracle.traverse_brute(nv, occ, lat, o, d)
        hit = vid >= 0
        for fl in (nif.NIF_TRAVERSE_COHERENT, nif.NIF_TRAVERSE_INCOHERENT):
            g = H.run_gpu(case, flags=nif.NIF_TRAVERSE_ONLY | fl, raw_logits=False)
            assert np.array_equal(g["voxel_id"], vid), (it, nv, theta, k, kind, fl, int((g["voxel_id"] != vid).sum()))
            assert np.array_equal(g["t_in"][hit].view(np.int32), ti[hit].view(np.int32)), (it, kind, fl)
            assert np.array_equal(g["t_out"][hit].view(np.int32), to[hit].view(np.int32)), (it, kind, fl)
        done += 1
    assert done >= 30


def test_random_scenes_walk_successor_sequence(oracle):
    """The successor traversal of nif_query_multi on random grids and poses: with a network that never accepts,
    the number of voxels walked and the last voxel equal the oracle's successor chain."""
    import harness as H
    import paper_2604_24666_b200 as nif
    import test_gpu_walk as W
    rng = np.random.default_rng(3)
    done = 0
    for it in range(24):
        nv = int(rng.choice([3, 4, 6, 8, 12, 16]))
        occ = (rng.random(nv ** 3) < rng.uniform(0.2, 1.0)).astype(np.uint8)
        if not occ.any():
            occ[0] = 1
        theta = float(rng.uniform(-2.0, 2.0)); k = float(rng.uniform(-0.8, 0.8))
        cfg = I.scaled(I.get_config(0), nv=nv)
        try:
            case = H.make_case(0, cfg=cfg, occ=occ, pose=[theta, k], n_rays=1200)
        except nif.NifError as e:
            assert e.status == -3
            continue
        case = W._net_with(H, case, "never_accept")
        K = int(rng.choice([3, 8, 30]))
        gpu = W.run_walk(nif, case, K)
        lat = oracle.deform_lattice(nv, theta, k); bvh = oracle.bvh_build(nv, occ, lat)
        o, d = case.origin, case.direction
        n = len(o)
        at = np.full(n, -np.inf, np.float32); ai = np.full(n, -1, np.int32)
        count = np.zeros(n, np.int32); last = np.full(n, -1, np.int32)
        for _ in range(K):
            v, ti, _ = bvh.next_voxel(o, d, at, ai)
            live = v >= 0
            if not live.any():
                break
            count += live; last = np.where(live, v, last)
            at = np.where(live, ti, at); ai = np.where(live, v, ai)
        capped = count >= K
        assert np.array_equal(gpu["steps"], count), (it, nv, theta, k, K)
        assert np.array_equal(gpu["voxel_id"][capped], last[capped]) and (gpu["voxel_id"][~capped] == -1).all()
        done += 1
    assert done >= 16
