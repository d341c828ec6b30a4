"""sq_edit_distance_hits_static: the entry point that allocates nothing (its scratch is a file-scope
__device__ array inside libsubquad.so).  Checked bit for bit -- all work is integer -- against the
existing paths: sq_edit_distance + a filter of its output, the workspace-scratch variant
sq_edit_distance_hits, and the oracle; on TWO calls in a row of different sizes (the static array
keeps the first call's contents).  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2602_17330_b200 import datagen as dg

pytestmark = pytest.mark.gpu


def _u32(t):
    return t.cpu().numpy().view(np.uint32)


def _u16(t):
    return t.cpu().numpy().view(np.uint16)


def test_static_scratch_hits_equal_the_existing_path_on_two_calls_in_a_row():
    from paper_2602_17330_b200 import binding
    rep = dg.config2(20_011, seed=51)
    sq = binding.SubQuad(0)
    max_len = int(rep.lengths.max())
    sq.set_workspace(sq.workspace_bytes(binding.OP_EDIT_DISTANCE, rep.n, int(rep.offsets[-1]), max_len) + (1 << 20))
    sq.pack(torch.from_numpy(rep.seqs).cuda(), torch.from_numpy(rep.offsets).cuda(), 20, max_len)
    rng = np.random.default_rng(52)
    fam_order = np.argsort(rep.family, kind="stable")
    # first call: 300,011 pairs, half of them inside families (many hits), ragged last tile;
    # second call: fewer pairs and another threshold (stale tile counts beyond its own must not matter)
    for n_pairs, max_d in ((300_011, 3), (70_001, 1), (2_049, 5)):
        q = rng.integers(0, rep.n - 1, n_pairs // 2)
        near = np.stack([fam_order[q], fam_order[q + 1]], 1)
        far = rng.integers(0, rep.n, (n_pairs - near.shape[0], 2))
        pl = np.concatenate([near, far]).astype(np.uint32)
        pl = pl[rng.permutation(n_pairs)]
        pt = torch.from_numpy(pl.view(np.int32)).cuda()
        # existing path: sq_edit_distance, then a filter of its output
        d_ref = _u16(sq.edit_distance(pt, n_pairs, max_d))[:n_pairs]
        keep = d_ref <= max_d
        want_p, want_d = pl[keep], d_ref[keep]
        assert 0 < want_p.shape[0] < n_pairs
        # ... which the oracle confirms
        assert np.array_equal(d_ref, oracle.edit_distance_pairs(rep.seqs, rep.offsets, pl, max_d))
        cap = want_p.shape[0] + 7
        for static in (True, False, True):
            dist = torch.full((n_pairs,), 0x5A5A, dtype=torch.int16, device="cuda")
            hp = torch.full((cap, 2), -1, dtype=torch.int32, device="cuda")
            hd = torch.full((cap,), -1, dtype=torch.int16, device="cuda")
            cnt = sq.edit_distance_hits(pt, n_pairs, max_d, dist, hp, hd, static=static)
            assert cnt == want_p.shape[0]
            assert np.array_equal(_u16(dist), d_ref)
            assert np.array_equal(_u32(hp)[:cnt], want_p)
            assert np.array_equal(_u16(hd)[:cnt], want_d)
            assert (_u32(hp)[cnt:] == 0xFFFFFFFF).all()            # nothing written past the hits
        # capacity protocol: the required count comes back, the first `capacity` hits are written
        small = torch.empty((10, 2), dtype=torch.int32, device="cuda")
        small_d = torch.empty(10, dtype=torch.int16, device="cuda")
        with pytest.raises(binding.SubQuadError) as ei:
            sq.edit_distance_hits(pt, n_pairs, max_d, dist, small, small_d, static=True)
        assert ei.value.code == binding.SQ_ERR_CAPACITY and ei.value.required == want_p.shape[0]
        assert np.array_equal(_u32(small), want_p[:10])
    sq.close()


def test_static_scratch_limits_and_edge_cases():
    from paper_2602_17330_b200 import binding
    rep = dg.from_list([[1, 2, 3, 4], [1, 2, 3, 5], [], [7] * 20])
    sq = binding.SubQuad(0)
    sq.set_workspace(sq.workspace_bytes(binding.OP_EDIT_DISTANCE, rep.n, int(rep.offsets[-1]), 20) + (1 << 16))
    sq.pack(torch.from_numpy(rep.seqs).cuda(), torch.from_numpy(rep.offsets).cuda(), 20, 20)
    pl = np.array([[0, 1], [0, 2], [2, 2], [0, 3], [9, 1]], np.uint32)       # the last index is out of range
    pt = torch.from_numpy(pl.view(np.int32)).cuda()
    dist = torch.empty(5, dtype=torch.int16, device="cuda")
    hp = torch.empty((5, 2), dtype=torch.int32, device="cuda")
    hd = torch.empty(5, dtype=torch.int16, device="cuda")
    cnt = sq.edit_distance_hits(pt, 5, 1, dist, hp, hd, static=True)
    assert _u16(dist).tolist() == [1, 2, 0, 2, 0xFFFF]                      # saturated at max_d + 1; 0xFFFF = bad index
    assert cnt == 2 and _u32(hp)[:2].tolist() == [[0, 1], [2, 2]] and _u16(hd)[:2].tolist() == [1, 0]
    assert sq.edit_distance_hits(pt, 0, 1, dist, hp, hd, static=True) == 0   # no pairs
    with pytest.raises(binding.SubQuadError) as ei:                          # beyond the static scratch
        sq.edit_distance_hits(pt, binding.SQ_HITS_STATIC_MAX_PAIRS + 1, 1, dist, hp, hd, static=True)
    assert ei.value.code == binding.SQ_ERR_UNSUPPORTED
    with pytest.raises(binding.SubQuadError) as ei:                          # a threshold is required
        sq.edit_distance_hits(pt, 5, -1, dist, hp, hd, static=True)
    assert ei.value.code == binding.SQ_ERR_INVALID_ARG
    sq.close()
