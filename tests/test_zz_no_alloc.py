"""qp_guide_tree_static against qp_guide_tree (GPU, through the C ABI).

Some users of libqp.so cannot allocate device memory where they call it: a plug-in whose host application owns the
device heap and passes in only inputs and outputs, a loop that must never block inside cudaMalloc / cudaFree, a job
with a fixed memory reservation on a shared GPU. qp_guide_tree needs a workspace from them; qp_guide_tree_static
keeps the merge loop's scratch in an array inside the library instead (up to 1024 sequences, about 4 MiB per GPU) and
allocates nothing. These tests check that it returns exactly what the workspace path returns -- merges, heights,
leaf counts, parents and tree distances are bit-equal, the bar of tests/test_gpu_tree.py -- on two calls in a row
that share the array (a large family first, then a small one over its left-overs, then the large one again), that
the calls leave the device's free memory where it was, and that a family beyond the limit is refused with its own
status before anything is launched.

This file sorts last on purpose: `pytest -x` stops at the first failure, so a failure here hides nothing else. It
does not depend on the tests before it (it also passes alone in a fresh process).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _symmetric(k, seed):
    rng = np.random.default_rng(seed)
    A = rng.random((k, k)).astype(np.float32)
    return np.ascontiguousarray(np.triu(A, 1) + np.triu(A, 1).T)


def _empty_tree(qp, torch, k, fill):
    """Output tensors for k sequences, made by the caller BEFORE the call (the static path creates none), pre-filled so
    that an element the kernels fail to write cannot pass by accident."""
    dev, i32 = torch.device("cuda:0"), torch.int32
    return qp.GuideTree(merge=torch.full((max(k - 1, 0), 2), fill, dtype=i32, device=dev),
                        height=torch.full((max(k - 1, 0),), float(fill), dtype=torch.float32, device=dev),
                        leaves=torch.full((2 * k - 1,), fill, dtype=i32, device=dev),
                        parent=torch.full((2 * k - 1,), fill, dtype=i32, device=dev),
                        treedist=torch.full((k, k), fill, dtype=i32, device=dev))


def _same(a, b):
    for name in ("merge", "height", "leaves", "parent", "treedist"):
        x, y = getattr(a, name).cpu().numpy(), getattr(b, name).cpu().numpy()
        assert np.array_equal(x, y), f"{name} differs between qp_guide_tree_static and qp_guide_tree"


def test_static_scratch_matches_workspace_path_on_calls_in_a_row():
    import torch
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    from paper_1512_07437_b200 import qp
    ks = [700, 37, 700, 1, 2, qp.GUIDE_TREE_STATIC_MAX_K]   # large, then small over its left-overs, then large again
    dists = [torch.from_numpy(_symmetric(k, 100 + n)).cuda() for n, k in enumerate(ks)]
    want = [qp.guide_tree(d) for d in dists]                  # existing path: caller-supplied workspace
    got = [_empty_tree(qp, torch, k, -7) for k in ks]
    qp.guide_tree_static(_empty_tree(qp, torch, 3, -7), dists[0][:3, :3].contiguous())   # per-device set-up call
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    reserved_before = torch.cuda.memory_reserved()
    for d, g in zip(dists, got):                              # back to back on one stream, sharing the one array
        qp.guide_tree_static(g, d)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before and torch.cuda.memory_reserved() == reserved_before, \
        "the no-allocation entry point changed the device's free memory"
    for w, g in zip(want, got):
        _same(g, w)
    # and a second round over the same array gives the same answers
    again = [_empty_tree(qp, torch, k, -9) for k in ks]
    for d, g in zip(reversed(dists), reversed(again)):
        qp.guide_tree_static(g, d)
    torch.cuda.synchronize()
    for w, g in zip(want, again):
        _same(g, w)


def test_static_scratch_without_tree_distances():
    import torch
    from paper_1512_07437_b200 import qp
    k = 129
    d = torch.from_numpy(_symmetric(k, 7)).cuda()
    want = qp.guide_tree(d, want_treedist=False)
    got = _empty_tree(qp, torch, k, -7)
    got.treedist = None
    qp.guide_tree_static(got, d)
    torch.cuda.synchronize()
    for name in ("merge", "height", "leaves", "parent"):
        assert np.array_equal(getattr(got, name).cpu().numpy(), getattr(want, name).cpu().numpy())


def test_static_scratch_refuses_families_beyond_its_limit():
    import torch
    from paper_1512_07437_b200 import qp
    k = qp.GUIDE_TREE_STATIC_MAX_K + 1
    d = torch.zeros((k, k), dtype=torch.float32, device="cuda:0")
    out = _empty_tree(qp, torch, k, -7)
    with pytest.raises(qp.QpError) as ei:
        qp.guide_tree_static(out, d)
    assert ei.value.code == qp.ERR["STATIC_LIMIT"] and "1024" in qp.status_string(ei.value.code)
    torch.cuda.synchronize()
    assert (out.leaves == -7).all() and (out.parent == -7).all(), "a refused call must not launch anything"
    # the ordinary path takes the same family
    t = qp.guide_tree(d)
    torch.cuda.synchronize()
    assert int(t.leaves[-1]) == k
