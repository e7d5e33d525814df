"""`-m gpu`: nif_query_static -- the query with its scratch in the library's fixed device array, for callers that
cannot allocate (include/nif.h).  It launches the kernels nif_query launches, so the bar is the one the other
same-kernel comparisons in this suite use (host entry vs device entry, graph replay): bit-equal outputs.
Collected last on purpose (file name): the suite runs with `pytest -x`."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def H():
    import harness
    return harness


@pytest.fixture(scope="module")
def nif():
    import paper_2604_24666_b200 as nif
    return nif


def _poisoned_outputs(nif, n):
    out = nif.alloc_outputs(n, raw_logits=True)
    for v in out.values():
        v.fill_(float("nan") if v.dtype.is_floating_point else -7)     # everything must be written
    return out


def _existing_path(nif, case, sel, flags=0):
    o = case.origin_d[sel].contiguous(); d = case.direction_d[sel].contiguous()
    out = _poisoned_outputs(nif, o.shape[0])
    nif.nif_query(case.bvh, case.net, o, d, out, flags=flags)
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in out.items()}


def _static_path(nif, case, sel, flags=0, check_free_memory=False):
    o = case.origin_d[sel].contiguous(); d = case.direction_d[sel].contiguous()
    out = _poisoned_outputs(nif, o.shape[0])
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    nif.nif_query_static(case.bvh, case.net, o, d, out, flags=flags)
    torch.cuda.synchronize()
    if check_free_memory:                     # the driver's own count of free device memory did not move
        assert torch.cuda.mem_get_info()[0] == free0
    return {k: v.cpu().numpy() for k, v in out.items()}


def _assert_same(got, ref):
    assert (ref["voxel_id"] >= 0).sum() > 1000                 # the comparison is about hit rays
    for k, v in ref.items():
        assert np.array_equal(got[k], v, equal_nan=True), k


def test_two_calls_in_a_row_match_the_existing_path(H, nif):
    # tensor-core net (configs[1]); the second call is a DIFFERENT, smaller batch, so whatever the first call left
    # in the shared array (bin counters, hit list, counters) is stale for it
    case = H.make_case(1, n_rays=60_000)
    first, second = slice(0, 60_000), slice(7, 60_000, 2)
    ref1, ref2 = _existing_path(nif, case, first), _existing_path(nif, case, second)
    got1 = _static_path(nif, case, first)
    got2 = _static_path(nif, case, second, check_free_memory=True)
    _assert_same(got1, ref1)
    _assert_same(got2, ref2)
    # and once more with other flags on the same array: occlusion head only
    ref3 = _existing_path(nif, case, first, flags=nif.NIF_OCCLUSION_ONLY)
    got3 = _static_path(nif, case, first, flags=nif.NIF_OCCLUSION_ONLY, check_free_memory=True)
    for k in ("voxel_id", "t_in", "t_out", "occlusion"):
        assert np.array_equal(got3[k], ref3[k], equal_nan=True), k


def test_fp32_engine_and_traverse_only(H, nif):
    case = H.make_case(0)                                      # fp32 net: the FFMA kernel
    sel = slice(0, len(case.origin))
    ref = _existing_path(nif, case, sel)
    for _ in range(2):
        _assert_same(_static_path(nif, case, sel), ref)
    ref_t = _existing_path(nif, case, sel, flags=nif.NIF_TRAVERSE_ONLY)
    got_t = _static_path(nif, case, sel, flags=nif.NIF_TRAVERSE_ONLY)
    for k in ("voxel_id", "t_in", "t_out"):
        assert np.array_equal(got_t[k], ref_t[k]), k


def test_full_frame_fits_and_one_ray_more_than_the_limit_is_refused(H, nif):
    case = H.make_case(1)                                      # 1920 x 1080 = 2,073,600 rays <= NIF_STATIC_MAX_RAYS
    n = len(case.origin)
    assert n <= nif.NIF_STATIC_MAX_RAYS
    sel = slice(0, n)
    ref = _existing_path(nif, case, sel)
    for _ in range(2):
        _assert_same(_static_path(nif, case, sel, check_free_memory=True), ref)
    # beyond the limit: a clear error, nothing enqueued, outputs untouched
    m = nif.NIF_STATIC_MAX_RAYS + 1
    o = torch.zeros((m, 3), dtype=torch.float32, device="cuda"); d = torch.zeros((m, 3), dtype=torch.float32, device="cuda")
    d[:, 2] = 1.0
    out = nif.alloc_outputs(m)
    for v in out.values():
        v.fill_(-7)
    with pytest.raises(nif.NifError) as e:
        nif.nif_query_static(case.bvh, case.net, o, d, out)
    assert e.value.status == -7 and "NIF_STATIC_MAX_RAYS" in str(e.value)
    torch.cuda.synchronize()
    for k, v in out.items():
        assert bool((v == -7).all()), k
    # exactly the limit is served (traversal only: the rays are synthetic)
    out_t = nif.alloc_outputs(m - 1)
    nif.nif_query_static(case.bvh, case.net, o[:m - 1], d[:m - 1], out_t, flags=nif.NIF_TRAVERSE_ONLY)
    ws_out = nif.alloc_outputs(m - 1)
    nif.nif_query(case.bvh, case.net, o[:m - 1], d[:m - 1], ws_out, flags=nif.NIF_TRAVERSE_ONLY)
    torch.cuda.synchronize()
    for k in ("voxel_id", "t_in", "t_out"):
        assert torch.equal(out_t[k], ws_out[k]), k
