"""vibe_permute_static -- the permutation (a3) for callers that cannot allocate device memory: its scratch is a static
device array inside libvibe.so (include/vibe.h).  Checked against the existing path (vibe_permute with a caller-provided
workspace) bit for bit -- indices and rows are integer / byte work -- on calls in a row that share the static array:
a large batch first (cooperative index kernel, grid-barrier counters in the array), then smaller ones that find the
large call's contents in it (single-cluster kernel), then an expert-parallel shard, then the large one again.

Collected last on purpose (file name): the suite runs with pytest -x.  Passes alone in a fresh process and after the
other tests (nothing here depends on what ran before; the array is cleared where it must be by every call)."""
import numpy as np
import pytest
import torch

from paper_2606_00735_b200 import binding as B
from paper_2606_00735_b200 import inputs as I

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required for -m gpu tests (no CPU fallback exists)")
    B.load()
    torch.cuda.set_device(0)


def _case(T, d, k, E, E_loc, align, seed):
    rng = np.random.default_rng(seed)
    X = torch.from_numpy(I.make_X(T, d, seed).view(np.int16)).cuda().view(torch.bfloat16)
    ids = np.argsort(rng.random((T, E)), axis=1)[:, :k].astype(np.int32)          # k distinct experts per token
    emap = None
    if E_loc < E:
        m = np.full(E, -1, np.int32)
        m[rng.permutation(E)[:E_loc]] = rng.permutation(E_loc).astype(np.int32)
        emap = torch.from_numpy(m).cuda()
    return X, torch.from_numpy(ids).cuda(), emap, E, E_loc, align


def _outputs(T, d, k, E_loc, align):
    # the same sentinel in both paths' outputs: whole-buffer equality then also says both wrote the same places
    Rcap = max(1, B.rows_cap(T, k, E_loc, align))
    return (torch.full((Rcap, d), -3.0, dtype=torch.bfloat16, device="cuda"),
            torch.full((E_loc + 1,), -7, dtype=torch.int32, device="cuda"),
            torch.full((Rcap,), -7, dtype=torch.int32, device="cuda"),
            torch.full((T * k,), -7, dtype=torch.int32, device="cuda"))


def test_permute_static_matches_permute_on_calls_in_a_row():
    cases = [_case(20000, 64, 8, 64, 64, 1, 1),        # A = 160 000: cooperative grid, barrier counters in the array
             _case(1500, 128, 4, 32, 32, 16, 2),       # A = 6000: one cluster; the array holds the large call's table
             _case(1500, 128, 4, 32, 32, 16, 3),       # the same shape again, other inputs
             _case(4096, 256, 8, 256, 32, 64, 4),      # expert-parallel shard (rows gathered by row), padded segments
             _case(20000, 64, 8, 64, 64, 1, 5)]        # the large shape after the small ones
    for X, ids, emap, E, E_loc, align in cases:
        T, d = X.shape
        k = ids.shape[1]
        ref = B.permute(X, ids, None, emap, E, E_loc, align, out=_outputs(T, d, k, E_loc, align))
        got = B.permute_static(X, ids, None, emap, E, E_loc, align, out=_outputs(T, d, k, E_loc, align))
        torch.cuda.synchronize()
        names = ("Xp", "offsets", "row_to_assign", "assign_to_row")
        for n, r, g in zip(names, ref, got):
            r = r.view(torch.int16) if r.dtype == torch.bfloat16 else r
            g = g.view(torch.int16) if g.dtype == torch.bfloat16 else g
            assert torch.equal(r, g), (n, T, k, E_loc)
        assert int(ref[1][-1]) > 0


def test_permute_static_rejects_sizes_beyond_the_static_array():
    # 1024 slots: 4 * 148 * 1024 bytes of slot totals do not fit the 304 KiB array (vibe_permute itself takes them)
    X, ids, emap, E, E_loc, align = _case(512, 64, 4, 2048, 1024, 1, 6)
    out = _outputs(512, 64, 4, E_loc, align)
    n0 = B.launch_count()
    with pytest.raises(B.VibeError, match="static array"):
        B.permute_static(X, ids, None, emap, E, E_loc, align, out=out)
    assert B.launch_count() == n0                      # nothing was launched
    torch.cuda.synchronize()
    assert int(out[1][0]) == -7                        # ... and nothing written
    B.permute(X, ids, None, emap, E, E_loc, align, out=out)
    torch.cuda.synchronize()
    assert int(out[1][0]) == 0
