"""axg_bfs_noalloc (include/axg.h): the BFS of PAPER.md:249-255 (Fig. 5; reading A-30) for callers that may not
allocate device memory -- its scratch is a fixed file-scope device array of the library, not allocator memory.

Checked against the EXISTING path (axg_build_graph + axg_bfs on a context): same adjacency list in, same levels out,
bit for bit (integers: the tolerance of the graph tests is zero), on two calls in a row that share the scratch array --
the second on a smaller graph and another root, so that anything the first call left behind would show.  Named test_zz_*
so that pytest collects it last: the suite runs with `pytest -x`."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

NONE = 0xFFFFFFFF


def _random_targets(rng, n):
    t = np.full(n, NONE, np.uint32)
    pick = np.flatnonzero(rng.uniform(size=n) < 0.85)
    j = rng.integers(0, n - 1, len(pick))
    t[pick] = np.where(j < pick, j, j + 1).astype(np.uint32)
    hub = rng.choice(n, min(3000, n // 4), replace=False)
    t[hub[hub != 7]] = 7                                    # one vertex with thousands of neighbours
    return t


def _existing_path(axg, n, targets, roots, seed):
    """the adjacency list and the BFS levels as the context-based calls give them"""
    pos = np.random.default_rng(seed).uniform(1, 63, (n, 3)).astype(np.float32)
    g = axg.Axg((64, 64, 64), 0.5, 1, 2.0, 0.25, 0.1, 3)
    g.set_capacity(1024, 2)
    g.place_neurons(pos, None)
    g.load_targets(targets)
    g.build_graph(False)
    va, ea = g.read_state("GRAPH_VA").copy(), g.read_state("GRAPH_EA").copy()
    levels = [g.bfs(r).copy() for r in roots]
    g.close()
    return va, ea, levels


def test_bfs_noalloc_equals_axg_bfs_on_two_calls_in_a_row():
    import torch
    from paper_1405_3331_b200 import axg
    axg.lib()
    rng = np.random.default_rng(2024)
    cases = [(150_000, (7, 12_345)), (4_097, (0,))]         # second graph smaller: stale scratch beyond it must not matter
    prepared = []
    for k, (n, roots) in enumerate(cases):
        t = _random_targets(rng, n)
        va, ea, want = _existing_path(axg, n, t, roots, seed=k)
        assert len(va) == n + 1 and len(ea) == va[-1] > n // 2
        # inputs and outputs are the CALLER's device memory (torch tensors here); the entry point allocates nothing
        d_va = torch.from_numpy(va.view(np.int32)).cuda()
        d_ea = torch.from_numpy(ea.view(np.int32)).cuda()
        d_lv = torch.full((n,), 12345, dtype=torch.int32, device="cuda")
        prepared.append((n, roots, want, d_va, d_ea, d_lv))
    torch.cuda.synchronize()
    stream = torch.cuda.current_stream().cuda_stream
    calls = 0
    for n, roots, want, d_va, d_ea, d_lv in prepared:       # back to back: no other library call in between
        for root, lv_want in zip(roots, want):
            axg.bfs_noalloc(d_va.data_ptr(), d_ea.data_ptr(), n, root, d_lv.data_ptr(), stream)
            got = d_lv.cpu().numpy()
            assert np.array_equal(got, lv_want), "root %d of %d vertices: %d levels differ" % (
                root, n, int((got != lv_want).sum()))
            assert got[root] == 0 and got.max() > 2
            calls += 1
    assert calls == 3
    # and once more on the first graph after the small one
    n, roots, want, d_va, d_ea, d_lv = prepared[0]
    axg.bfs_noalloc(d_va.data_ptr(), d_ea.data_ptr(), n, roots[1], d_lv.data_ptr(), stream)
    assert np.array_equal(d_lv.cpu().numpy(), want[1])


def test_bfs_noalloc_rejects_what_it_cannot_hold():
    import torch
    from paper_1405_3331_b200 import axg
    axg.lib()
    d = torch.zeros(8, dtype=torch.int32, device="cuda")
    with pytest.raises(axg.AxgError) as e:
        axg.bfs_noalloc(d.data_ptr(), d.data_ptr(), axg.BFS_NOALLOC_MAX_VERTICES + 1, 0, d.data_ptr())
    assert e.value.code == -1 and "AXG_BFS_NOALLOC_MAX_VERTICES" in str(e.value)
    with pytest.raises(axg.AxgError) as e:
        axg.bfs_noalloc(d.data_ptr(), d.data_ptr(), 4, 4, d.data_ptr())      # root out of range
    assert e.value.code == -1
    with pytest.raises(axg.AxgError):
        axg.bfs_noalloc(0, d.data_ptr(), 4, 0, d.data_ptr())                 # null pointer
