"""-m gpu: hit masking between iterations (reading R9) against the oracle: mask and masked index bit-exact,
the second iteration's hit lists as for any build (identical up to small oracle margins)."""
import numpy as np
import pytest

from oracle import mkfo
from workloads import datagen

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("which,scale", [(2, 0.05), (3, 0.01)])
def test_two_iterations_with_masking(which, scale):
    from gpu_helpers import gpu_two_iterations
    ev, prm = datagen.config(which, scale=scale)
    s, h = ev["seeds"], ev["hits"]
    nh = h["x"].shape[0]
    r1, mask, im, r2 = gpu_two_iterations(ev, prm, min_hits=8, max_chi2_ndf=5.0)
    # the mask from the kernel's own first iteration (same inputs to both sides)
    ref_mask = mkfo.mask_hits(nh, r1["hit_ids"], r1["nhits"], r1["chi2"], keep=r1["keep"], min_hits=8, max_chi2_ndf=5.0)
    assert np.array_equal(mask, ref_mask) and 0 < mask.sum() < nh
    # masked index bit-exact
    o = mkfo.Oracle(ev["geom"], prm)
    ref = o.build_hit_index(h, mask=ref_mask)
    assert np.array_equal(im["bin_off"], ref["bin_off"]) and np.array_equal(im["sorted_id"], ref["sorted_id"])
    assert np.array_equal(im["vmax"].view(np.uint32), ref["vmax"].view(np.uint32))
    # second iteration against the oracle on the same masked index
    rb = o.build_tracks(h, ref, s["par"], s["cov"], s["q"], s["event"], s["hits"], s["plan"])
    same = np.all(r2["hit_ids"] == rb["hit_ids"], axis=0)
    assert same.mean() >= 0.999 and np.all(rb["margin"][~same] < 1e-3), same.mean()
    own = (r2["hit_ids"][:, None, :] == s["hits"][None, :, :]).any(axis=1)          # the seed's own hits are read by id
    picked = r2["hit_ids"][(r2["hit_ids"] >= 0) & ~own]
    assert mask[picked].sum() == 0                              # nothing masked is picked up beyond the seed hits
    assert (r2["nhits"] < r1["nhits"]).mean() > 0.3             # the good tracks of iteration 1 lost their hits


def test_mask_rules_and_degenerate_inputs():
    import torch
    from gpu_helpers import strip_context
    ctx = strip_context()
    hit_ids = np.array([[0, 3, 6, 8], [1, -1, 7, 9], [2, 5, -2, 4]], np.int32)
    nhits = np.array([3, 2, 2, 3], np.int32)
    chi2 = np.array([1.0, 0.0, 0.0, 6.0], np.float32)
    for keep, mh, mc in ((None, 3, 5.0), (None, 3, 6.0), (np.array([0, 1, 1, 1], np.uint8), 3, 6.0), (None, 2, 5.0), (None, 0, 1e30)):
        m = torch.zeros(10, dtype=torch.uint8, device="cuda")
        ctx.mask_hits(torch.from_numpy(hit_ids).cuda(), torch.from_numpy(nhits).cuda(), torch.from_numpy(chi2).cuda(),
                      torch.from_numpy(keep).cuda() if keep is not None else None, mh, mc, m)
        assert m.cpu().numpy().tolist() == mkfo.mask_hits(10, hit_ids, nhits, chi2, keep=keep, min_hits=mh, max_chi2_ndf=mc).tolist()
    # no tracks: nothing happens
    m = torch.zeros(10, dtype=torch.uint8, device="cuda")
    e = torch.zeros((3, 0), dtype=torch.int32, device="cuda")
    ctx.mask_hits(e, torch.zeros(0, dtype=torch.int32, device="cuda"), torch.zeros(0, device="cuda"), None, 0, 1.0, m)
    assert int(m.sum()) == 0
    # everything masked: an empty index
    from paper_2002_06295_b200 import binding as B
    ev, prm = datagen.config(2, scale=0.01)
    c2 = B.Context(ev["geom"], prm)
    hits = B.hits_to_device(ev["hits"])
    nh = hits["x"].shape[0]
    idx, ws = B.alloc_hit_index(c2, hits["n_events"], nh)
    c2.build_hit_index(hits, idx, ws, mask=torch.ones(nh, dtype=torch.uint8, device="cuda"))
    torch.cuda.synchronize()
    assert int(idx["bin_off"].max()) == 0 and float(idx["vmax"].max()) == 0.0
    c2.close()
