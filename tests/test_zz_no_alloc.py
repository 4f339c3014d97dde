"""gs_topk_dense_static: the top-k select with its scratch in a static device array (no allocation inside the library).

Collected last on purpose (file name): the run uses ``pytest -x``.  The new entry point is compared with the
existing gs_topk_dense on the same inputs — bit-exact, as for all index / selection work in this repo — on two calls in a
row that reuse the shared scratch (different data, row count and k), on rows longer than 2^20 columns (the multi-launch
select, the path that actually uses scratch) and on short rows at the stated maximum.
"""
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gs():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2606_26441_b200 import binding
    binding.lib()
    return binding


def _scores(rows, n, dtype, seed):
    import torch
    g = torch.Generator(device="cuda").manual_seed(seed)
    if dtype == torch.float32:
        # coarse values: many exact ties, so the (score desc, id asc) order is exercised too
        return (torch.randn((rows, n), generator=g, device="cuda") * 16.0).round() / 16.0
    return torch.randint(-500, 500, (rows, n), generator=g, device="cuda", dtype=torch.int32)


def _both(gs, scores, k):
    import torch
    rows = scores.shape[0]
    ids = torch.full((rows, k), -7, dtype=torch.int32, device="cuda")
    sc = torch.zeros((rows, k), dtype=scores.dtype, device="cuda")
    gs.topk_dense_static(scores, k, ids, sc)
    ref_ids, ref_sc = gs.topk_dense(scores, k)
    torch.cuda.synchronize()
    return ids, sc, ref_ids, ref_sc


def test_static_scratch_topk_matches_workspace_topk_on_consecutive_calls(gs):
    import torch
    long_n = (1 << 20) + 4099          # > 2^20 columns: the multi-launch select, which keeps its state in the scratch
    cases = [
        (_scores(3, long_n, torch.float32, 1), 100),
        (_scores(5, long_n + 14, torch.float32, 2), 1000),     # second call: more rows, larger k, stale scratch underneath
        (_scores(2, long_n, torch.int32, 3), 10),
        (_scores(64, 5000, torch.float32, 4), gs.GS_MAX_K),    # the stated maximum (64 rows at k = GS_MAX_K), short rows
        (_scores(3, long_n, torch.float32, 1), 100),           # the first case again after all the others
    ]
    for scores, k in cases:
        ids, sc, ref_ids, ref_sc = _both(gs, scores, k)
        assert torch.equal(ids, ref_ids)
        assert torch.equal(sc.view(torch.int32), ref_sc.view(torch.int32))       # bit-exact
        # and against the definition, on the first row: k best under (score desc, id asc)
        row = scores[0].to(torch.float64)
        order = torch.argsort(-row, stable=True)[:k]
        assert torch.equal(ids[0].to(torch.int64), order)


def test_static_scratch_topk_allocates_nothing_and_rejects_beyond_the_maximum(gs):
    import torch
    scores = _scores(3, (1 << 20) + 4099, torch.float32, 5)
    k = 100
    ids = torch.empty((3, k), dtype=torch.int32, device="cuda")
    sc = torch.empty((3, k), dtype=torch.float32, device="cuda")
    gs.topk_dense_static(scores, k, ids, sc)       # first use: kernels loaded, symbol address looked up
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        gs.topk_dense_static(scores, k, ids, sc)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before               # no device memory taken or returned by the calls
    # beyond the maximum: 65 rows at k = GS_MAX_K need more scratch than the static array holds
    big = _scores(65, 5000, torch.float32, 6)
    with pytest.raises(gs.GsError) as e:
        gs.topk_dense_static(big, gs.GS_MAX_K, torch.empty((65, gs.GS_MAX_K), dtype=torch.int32, device="cuda"),
                             torch.empty((65, gs.GS_MAX_K), dtype=torch.float32, device="cuda"))
    assert e.value.code == 2                       # GS_ERR_OUT_OF_RANGE
    need = gs.ctypes.c_size_t()
    assert gs.lib().gs_topk_workspace_bytes(64, 5000, gs.GS_MAX_K, gs.ctypes.byref(need)) == 0
    assert need.value == gs.GS_TOPK_STATIC_SCRATCH_BYTES
