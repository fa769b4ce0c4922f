"""workloads/generate_torch.py must reproduce workloads/generate.py byte for byte (CPU tensors here; the
large-config GPU tests run the same code on the device)."""
import numpy as np
import pytest
import torch

from workloads import generate as gen
from workloads import generate_torch as gt


def test_counter_based_generator_matches_numpy():
    c = np.array([0, 1, 2, 12345, 2**40 + 7, 2**62], dtype=np.uint64)
    for seed, stream in [(gen.BASE_SEED, 0), (gen.BASE_SEED + 4, 21), (1, 5)]:
        want = gen.H(seed, stream, c)
        got = gt.H(seed, stream, torch.from_numpy(c.astype(np.int64))).numpy().view(np.uint64)
        assert np.array_equal(got, want)
    x = torch.from_numpy(gen.H(3, 3, np.arange(1000, dtype=np.uint64)).view(np.int64).copy())
    for m in (3, 201, 999_901, 3_300_000_000 - 99):
        assert np.array_equal(gt.umod(x, m).numpy().astype(np.uint64), x.numpy().view(np.uint64) % np.uint64(m))


@pytest.mark.parametrize("idx,scale", [(1, 0.003), (2, 0.0007), (3, 0.0004), (4, 0.000004)])
def test_read_recipes_match_numpy(idx, scale):
    want = gen.config(idx, scale)
    r = gt.ReadRecipe(idx, scale)
    assert r.n_reads == want.n_reads
    lens = r.lengths(0, r.n_reads)
    assert np.array_equal(np.diff(want.offsets.astype(np.int64)), lens.numpy())
    assert np.array_equal(r.reads_ascii(0, r.n_reads).numpy(), want.ascii)
    # chunked generation gives the same bytes
    a, b = r.n_reads // 3, r.n_reads // 3 + min(17, r.n_reads - r.n_reads // 3)
    assert np.array_equal(r.reads_ascii(a, b).numpy(), want.ascii[int(want.offsets[a]):int(want.offsets[b])])
