"""sph_cell_sort_static (include/sph.h): the cell-list radix sort with its scratch in a static device array, for
callers that must not allocate.  Checked bit for bit (integer work) against the existing path:
the cell-sorted order a context produces (sph_debug_cells: sort buffers from cudaMalloc), on two calls in a row that
share the scratch array, and against a host stable sort at the largest size it takes.

Collected last on purpose (pytest -x): a failure here hides no other test.
"""
import numpy as np
import pytest

from paper_2110_02621_b200 import inputs, sph

pytestmark = pytest.mark.gpu


def _bits(count):
    b = 1
    while (1 << b) < count:
        b += 1
    return b


def _sorted_blocks():
    """Existing path: cell ids (caller order) and the cell-sorted permutation of a context (fluid block, wall block)."""
    cfg = inputs.shuffled(inputs.box_sweep_3d(n=40), seed=17)
    g = sph.Sph(cfg)
    g.set_particles(cfg["pos"], cfg["vel"], cfg["rho"], cfg["tag"])
    cid, perm, _, _ = g.debug_cells()
    nf = int((cfg["tag"] >= 0).sum())
    blocks = []
    for ids, ref in ((np.flatnonzero(cfg["tag"] >= 0), perm[:nf]), (np.flatnonzero(cfg["tag"] < 0), perm[nf:])):
        blocks.append((ids.astype(np.int32), cid[ids].astype(np.int32), ref, cid[ref]))
    return blocks, _bits(g.num_cells())


def _run(keys, vals, key_bits):
    import torch
    dk = torch.from_numpy(keys).cuda()
    dv = torch.from_numpy(vals).cuda() if vals is not None else None
    ko, vo = torch.empty_like(dk), torch.empty_like(dk)
    sph.cell_sort_static(dk, dv, key_bits, ko, vo)
    torch.cuda.synchronize()
    return ko.cpu().numpy(), vo.cpu().numpy()


def test_static_sort_matches_context_path_on_two_calls_in_a_row():
    ((fid, fkey, fperm, fsorted), (wid, wkey, wperm, wsorted)), bits = _sorted_blocks()
    assert len(fid) > 50000 and len(wid) > 10000 and len(fid) <= sph.STATIC_SORT_MAX_KEYS
    # call 1: fluid block; call 2 (scratch still holds call 1's histograms and buffers): wall block; call 3: fluid again
    for ids, key, ref_perm, ref_keys in ((fid, fkey, fperm, fsorted), (wid, wkey, wperm, wsorted), (fid, fkey, fperm, fsorted)):
        ko, vo = _run(key, ids, bits)
        assert np.array_equal(ko, ref_keys)
        assert np.array_equal(vo, ref_perm)
    # values = NULL: the indices 0..n-1; every pass count 1..4 of the radix plan, so both ping-pong parities
    small = (fkey & 0xff).astype(np.int32)
    for kb, key in ((8, small), (bits, fkey), (18, fkey), (24, fkey), (32, fkey)):
        ko, vo = _run(key, None, kb)
        order = np.argsort(key, kind="stable")
        assert np.array_equal(vo, order.astype(np.int32)), kb
        assert np.array_equal(ko, key[order]), kb
        if key is fkey:
            assert np.array_equal(fid[vo], fperm), kb


def test_static_sort_largest_size_no_allocation_and_limit():
    import torch
    torch.cuda.set_device(0)
    n = sph.STATIC_SORT_MAX_KEYS
    rng = np.random.default_rng(5)
    for rep in range(2):   # two calls in a row at the largest size, different keys and key widths
        kb = (20, 27)[rep]
        key = rng.integers(0, 1 << kb, size=n - 777 * rep, dtype=np.int64).astype(np.int32)
        ko, vo = _run(key, None, kb)
        order = np.argsort(key, kind="stable")
        assert np.array_equal(vo, order.astype(np.int32))
        assert np.array_equal(ko, key[order])
    # a repeated call changes neither the driver's free memory nor torch's: nothing is allocated
    dk = torch.from_numpy(key).cuda()
    ko, vo = torch.empty_like(dk), torch.empty_like(dk)
    sph.cell_sort_static(dk, None, 27, ko, vo)
    torch.cuda.synchronize()
    free0, res0 = torch.cuda.mem_get_info()[0], torch.cuda.memory_reserved()
    sph.cell_sort_static(dk, None, 27, ko, vo)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0 and torch.cuda.memory_reserved() == res0
    # beyond the limit: refused with a clear error, nothing launched, outputs untouched
    big = torch.zeros(n + 1, dtype=torch.int32, device="cuda")
    out_k, out_v = torch.full_like(big, -7), torch.full_like(big, -7)
    with pytest.raises(sph.SphError, match="exceeds SPH_STATIC_SORT_MAX_KEYS"):
        sph.cell_sort_static(big, None, 20, out_k, out_v)
    torch.cuda.synchronize()
    assert int((out_k != -7).sum()) == 0 and int((out_v != -7).sum()) == 0
    with pytest.raises(sph.SphError, match="key_bits"):
        sph.cell_sort_static(dk, None, 33, ko, vo)
    # n = 0 is a no-op
    e = torch.empty(0, dtype=torch.int32, device="cuda")
    sph.cell_sort_static(e, None, 8, e.clone(), e.clone())
