"""cx_sort_pairs_static (include/cx_bwt.h): the sorter for callers that cannot allocate -- its scratch is a file-scope static
device array of the library.  Its output must equal the existing path's (cx_sort_pairs with a caller-supplied workspace) bit
for bit (integer work: the tolerance of every test here is exact equality), on two calls in a row that share the array: the
second call is smaller and sorts other bits, so anything left over from the first one would show.
Collected last on purpose (the suite runs with pytest -x): it must pass alone in a fresh process and after the other tests."""
import pytest
import torch

pytestmark = pytest.mark.gpu


def _pairs(n, bits, vb, seed):
    g = torch.Generator(device="cuda").manual_seed(seed)
    keys = torch.randint(-2**63, 2**63 - 1, (n,), dtype=torch.int64, device="cuda", generator=g)
    if bits < 64:
        keys = keys & ((1 << bits) - 1)
    if n > 1000:
        m = keys[1::3].numel()
        keys[::3][:m] = keys[1::3]                       # plenty of duplicates: stability matters
    vals = torch.arange(n, device="cuda", dtype=torch.int32 if vb == 4 else torch.int64)
    return keys, vals


def _static_sort(cx, keys, vals, bits):
    k0, v0 = keys.clone(), vals.clone()                  # the caller's buffers: inputs and outputs
    k1, v1 = torch.empty_like(k0), torch.empty_like(v0)
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    ks, vs = cx.cx_sort_pairs_static(k0, v0, k1, v1, 0, bits)
    assert torch.cuda.memory_allocated() == before       # nothing was allocated through torch on the way
    return ks, vs


def test_static_scratch_sort_matches_the_workspace_path_on_two_calls_in_a_row():
    import paper_1401_7457_b200 as cx
    calls = [(1_000_003, 64, 4, 11), (300_001, 40, 8, 12), (1, 64, 4, 13), (cx.CX_SORT_STATIC_MAX_PAIRS, 13, 4, 14), (5000, 64, 8, 15)]
    for n, bits, vb, seed in calls:                      # back to back on one stream, all sharing the static array
        keys, vals = _pairs(n, bits, vb, seed)
        ks, vs = _static_sort(cx, keys, vals, bits)
        want_k, want_v = cx.cx_sort_pairs(keys, vals, 0, bits)          # the existing path (workspace from the caller)
        assert torch.equal(ks, want_k), (n, bits, vb)
        assert torch.equal(vs, want_v), (n, bits, vb)
    # and against a library stable sort, so that the two paths cannot be wrong together
    keys, vals = _pairs(200_000, 64, 4, 16)
    ks, vs = _static_sort(cx, keys, vals, 64)
    order = torch.sort(keys ^ (-2**63), stable=True).indices           # unsigned order = signed order after flipping the sign bit
    assert torch.equal(ks, keys[order]) and torch.equal(vs.long(), order)


def test_static_scratch_sort_rejects_sizes_beyond_its_maximum():
    import paper_1401_7457_b200 as cx
    n = cx.CX_SORT_STATIC_MAX_PAIRS + 1
    keys, vals = _pairs(n, 64, 4, 17)
    with pytest.raises(cx.CxError) as e:
        cx.cx_sort_pairs_static(keys, vals, torch.empty_like(keys), torch.empty_like(vals))
    assert e.value.code == cx.binding.CX_ERR_ARG and "CX_SORT_STATIC_MAX_PAIRS" in str(e.value)
    assert cx.cx_sort_pairs_static(keys[:0], vals[:0], keys[:0].clone(), vals[:0].clone())[0].numel() == 0      # n = 0: nothing to do
