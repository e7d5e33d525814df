"""Pins for oracle step O8: composite encoding psi(x) = phi(gamma(x)) (Eq. 1)."""
import numpy as np
import torch

import nif_inputs as I
from conftest import read_golden


def test_hash_grid_toy_table_hand_computed(oracle):
    # BASELINE.json:5 "hash-grid indices match hand-computed values for a 2-level toy table"
    p = np.array([0.3, 0.6, 0.9], np.float32)
    rows = [r for r in read_golden("hash_toy.txt") if r[0] == "lookup"]
    assert len(rows) == 2
    for r in rows:
        N, log2_T = int(r[1]), int(r[2])
        want_idx = np.array(r[3:11], dtype=np.int64)
        want_w = np.array(r[11:19], dtype=np.float64)
        idx, w = oracle.level_lookup(N, log2_T, p)
        assert np.array_equal(idx.astype(np.int64), want_idx)
        np.testing.assert_allclose(w, want_w, atol=2e-7)


def test_hash_of_single_vertices_hand_computed(oracle):
    # hashed levels only: N = 2005 -> 2006^3 > T for every T used (2^12, 2^19, 2^22)
    N = 2005
    for r in [r for r in read_golden("hash_toy.txt") if r[0] == "vertex"]:
        i, j, k = int(r[1]), int(r[2]), int(r[3])
        for log2_T, want in zip((12, 19, 22), map(int, r[4:7])):
            if max(i, j, k) < N:                       # vertex is corner 000 of its own cell
                p = (np.array([i, j, k]) + 0.5) / N
                corner = 0
            else:                                      # top boundary: cell N-1, corner 111
                p = np.array([1.0, 1.0, 1.0])
                corner = 7
            idx, _ = oracle.level_lookup(N, log2_T, p.astype(np.float32))
            assert int(idx[corner]) == want, (i, j, k, log2_T)


def test_dense_switch_uses_64_bit_compare(oracle):
    # (N+1)^3 overflows 32 bits at the finest levels; those levels must be hashed, not dense
    idx, _ = oracle.level_lookup(2005, 19, np.array([0.999, 0.999, 0.999], np.float32))
    assert idx.max() < (1 << 19)
    # boundary: 58 -> 59^3 = 205379 <= 2^19 dense; 80 -> 81^3 = 531441 > 2^19 hashed
    idx, _ = oracle.level_lookup(58, 19, np.array([1.0, 1.0, 1.0], np.float32))
    assert int(idx[7]) == 59 ** 3 - 1
    idx, _ = oracle.level_lookup(80, 19, np.array([1.0, 1.0, 1.0], np.float32))
    assert int(idx[7]) == ((80 * 1) ^ ((80 * 2654435761) & 0xFFFFFFFF) ^ ((80 * 805459861) & 0xFFFFFFFF)) & ((1 << 19) - 1)


def test_weights_are_a_partition_of_unity_and_top_boundary(oracle):
    rng = np.random.default_rng(0)
    for _ in range(200):
        p = rng.uniform(0, 1, 3).astype(np.float32)
        _, w = oracle.level_lookup(int(rng.integers(2, 3000)), 19, p)
        assert abs(w.sum() - 1.0) < 1e-6 and (w >= 0).all()
    # p = 1 exactly: cell N-1 with w = 1 -> all weight on corner 111
    _, w = oracle.level_lookup(16, 19, np.array([1.0, 1.0, 1.0], np.float32))
    assert w[7] == 1.0 and w[:7].sum() == 0.0


def test_positional_samples_against_numpy(oracle):
    # gamma(x) = [x, {sin(2^k x), cos(2^k x)}] (Eq. 1, no factor pi), mapped (v+1)/2 (R3)
    rng = np.random.default_rng(1)
    B = 6
    for _ in range(50):
        x = rng.uniform(0, 1, 3).astype(np.float32)
        s = oracle.pe_samples(B, x)
        assert s.shape == (13, 3) and np.array_equal(s[0], x)
        x64 = x.astype(np.float64)
        for k in range(B):
            np.testing.assert_allclose(s[1 + 2 * k], (np.sin(2.0 ** k * x64) + 1) / 2, atol=3e-7)
            np.testing.assert_allclose(s[2 + 2 * k], (np.cos(2.0 ** k * x64) + 1) / 2, atol=3e-7)
    s = oracle.pe_samples(4, np.zeros(3, np.float32))       # SURVEY 8(c).3 "O8 PE"
    assert np.array_equal(s[0], [0, 0, 0])
    assert np.array_equal(s[1::2], np.full((4, 3), 0.5, np.float32))
    assert np.array_equal(s[2::2], np.full((4, 3), 1.0, np.float32))


def _params(shape, table):
    return I.NetParams(shape, shape.level_res(), table.astype(np.float32), [], "test")


def test_constant_table_gives_constant_features_and_flatten_order(oracle):
    # weights sum to 1 => a table that is constant per (level, feature) comes back unchanged;
    # using a different constant per (l, f) pins the flatten order out[(s*L + l)*F + f].
    shape = I.NetShape(pe_bands=3, levels=5, log2_T=10, feat=3, base_res=2, growth=1.7,
                       hidden_layers=1, width=8, dtype="f32")
    L, T, F = shape.levels, shape.table_entries, shape.feat
    table = np.zeros((L, T, F), np.float32)
    for l in range(L):
        for f in range(F):
            table[l, :, f] = (l + 1) + 0.125 * f
    xn = np.random.default_rng(2).uniform(0, 1, (20, 3)).astype(np.float32)
    out = oracle.encode(_params(shape, table), xn).reshape(20, shape.samples, L, F)
    want = (np.arange(L)[:, None] + 1) + 0.125 * np.arange(F)[None, :]
    np.testing.assert_allclose(out, np.broadcast_to(want, out.shape), rtol=1e-6)


def test_dense_levels_equal_torch_grid_sample_and_sample_order(oracle):
    # library routine: trilinear interpolation with align_corners=True on the (N+1)^3 volume.
    # The volume differs per level and the query differs per PE sample, so this also pins which
    # sample s feeds which output slot.
    shape = I.NetShape(pe_bands=2, levels=3, log2_T=12, feat=2, base_res=3, growth=1.6,
                       hidden_layers=1, width=8, dtype="f32")
    res = shape.level_res()
    assert all((int(n) + 1) ** 3 <= shape.table_entries for n in res)     # all dense
    rng = np.random.default_rng(3)
    table = rng.uniform(-1, 1, (shape.levels, shape.table_entries, shape.feat)).astype(np.float32)
    xn = rng.uniform(0, 1, (64, 3)).astype(np.float32)
    out = oracle.encode(_params(shape, table), xn).reshape(64, shape.samples, shape.levels, shape.feat)
    x64 = xn.astype(np.float64)
    samples = [x64]
    for k in range(shape.pe_bands):
        samples += [(np.sin(2.0 ** k * x64) + 1) / 2, (np.cos(2.0 ** k * x64) + 1) / 2]
    for l, N in enumerate(res):
        n1 = int(N) + 1
        vol = table[l, :n1 ** 3].reshape(n1, n1, n1, shape.feat)              # [k, j, i, f]
        vol_t = torch.from_numpy(vol.astype(np.float64)).permute(3, 0, 1, 2)[None]   # [1,F,D,H,W]
        for s, p in enumerate(samples):
            grid = torch.from_numpy(p * 2 - 1).reshape(1, -1, 1, 1, 3)         # (x,y,z) -> (W,H,D)
            ref = torch.nn.functional.grid_sample(vol_t, grid, mode="bilinear",
                                                  align_corners=True)[0, :, :, 0, 0].T.numpy()
            np.testing.assert_allclose(out[:, s, l, :], ref, atol=5e-6)


def test_affine_table_is_reproduced_exactly_on_a_dense_level(oracle):
    shape = I.NetShape(pe_bands=0, levels=1, log2_T=12, feat=1, base_res=7, growth=1.0,
                       hidden_layers=1, width=8, dtype="f32")
    N = 7; n1 = N + 1
    k, j, i = np.meshgrid(np.arange(n1), np.arange(n1), np.arange(n1), indexing="ij")
    vals = 0.5 + 0.25 * i / N - 0.75 * j / N + 0.125 * k / N
    table = np.zeros((1, shape.table_entries, 1), np.float32)
    table[0, :n1 ** 3, 0] = vals.reshape(-1)
    xn = np.random.default_rng(4).uniform(0, 1, (100, 3)).astype(np.float32)
    out = oracle.encode(_params(shape, table), xn)[:, 0]
    want = 0.5 + 0.25 * xn[:, 0] - 0.75 * xn[:, 1] + 0.125 * xn[:, 2]
    np.testing.assert_allclose(out, want, atol=3e-7)


def test_hashed_level_interpolates_the_hashed_entries(oracle):
    # brute force on a tiny hashed level: recompute from the golden-pinned lookup
    shape = I.NetShape(pe_bands=0, levels=1, log2_T=5, feat=2, base_res=4, growth=1.0,
                       hidden_layers=1, width=8, dtype="f32")
    rng = np.random.default_rng(5)
    table = rng.uniform(-1, 1, (1, 32, 2)).astype(np.float32)
    p = np.array([[0.3, 0.6, 0.9]], np.float32)
    out = oracle.encode(_params(shape, table), p)[0]
    idx = [28, 31, 13, 14, 23, 20, 6, 5]                       # tests/golden/hash_toy.txt
    w = [0.192, 0.048, 0.128, 0.032, 0.288, 0.072, 0.192, 0.048]
    want = sum(wi * table[0, ii].astype(np.float64) for wi, ii in zip(w, idx))
    np.testing.assert_allclose(out, want, atol=1e-6)
