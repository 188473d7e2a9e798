"""lt_sort_keys_static (the entry point that allocates nothing: radix-sort scratch in a static device
array of the library) against the existing path lt_sort_keys, bit for bit (integer work), on two calls
in a row that share the scratch.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest
import torch

import parity as P
from paper_2306_06744_b200 import lt

pytestmark = pytest.mark.gpu

DIM, MAXL = 3, 9
BITS = DIM * MAXL + 5


def to_dev(k):
    return torch.from_numpy(np.ascontiguousarray(k, np.uint64).view(np.int64)).cuda()


def test_static_sort_matches_sort_keys_on_two_calls_in_a_row():
    rng = np.random.default_rng(2306)
    n1, n2 = lt.SORT_STATIC_MAX_KEYS, 100003        # the maximum, then a ragged size over stale scratch
    k1 = rng.integers(0, 1 << BITS, n1, dtype=np.uint64)
    k2 = rng.integers(0, 1 << BITS, n2, dtype=np.uint64)
    k2[: n2 // 3] = k2[n2 // 3: 2 * (n2 // 3)]      # duplicates
    want1 = lt.sort_keys(DIM, MAXL, to_dev(k1))     # the existing, allocating path
    want2 = lt.sort_keys(DIM, MAXL, to_dev(k2))
    d1, d2 = to_dev(k1), to_dev(k2)
    lt.sort_keys_static_(DIM, MAXL, d1)             # two calls back to back on one stream, no host wait between
    lt.sort_keys_static_(DIM, MAXL, d2)
    torch.cuda.synchronize()
    assert torch.equal(d1, want1) and torch.equal(d2, want2)
    assert np.array_equal(P.u64(d1), np.sort(k1)) and np.array_equal(P.u64(d2), np.sort(k2))
    # and once more over the scratch the second call left behind; the library must not have taken memory
    d3 = to_dev(k1)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    lt.sort_keys_static_(DIM, MAXL, d3)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before
    assert torch.equal(d3, want1)


@pytest.mark.parametrize("n", [0, 1, 2, 4097])
def test_static_sort_small_sizes(n):
    k = np.random.default_rng(n).integers(0, 1 << BITS, n, dtype=np.uint64)
    d = to_dev(k)
    lt.sort_keys_static_(DIM, MAXL, d)
    torch.cuda.synchronize()
    assert np.array_equal(P.u64(d), np.sort(k))


def test_static_sort_rejects_sizes_beyond_the_maximum():
    d = torch.zeros(lt.SORT_STATIC_MAX_KEYS + 1, dtype=torch.int64, device="cuda")
    d[0] = 5
    with pytest.raises(lt.LtError) as e:
        lt.sort_keys_static_(DIM, MAXL, d)
    assert e.value.status == lt.LT_ERR_CAPACITY and "capacity" in str(e.value)
    torch.cuda.synchronize()
    assert int(d[0]) == 5                            # nothing was launched
