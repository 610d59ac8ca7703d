"""-m gpu: strip clustering (reading R8) against the oracle, bit-exact in every output."""
import numpy as np
import pytest

from oracle import mkfo
from workloads import datagen

pytestmark = pytest.mark.gpu


def check(d, sp, capacity=None):
    from gpu_helpers import gpu_cluster_strips
    ref = mkfo.cluster_strips(d["module_off"], d["adc"], d["noise"], d["bad"], **sp)
    got = gpu_cluster_strips(d, sp, capacity)
    assert got["n_clusters"] == len(ref["module"])
    if capacity is not None and capacity < got["n_clusters"]:
        return ref                                    # incomplete by contract: only the count is defined
    k = len(got["module"])
    for key in ("module", "first", "last", "charge"):
        assert np.array_equal(got[key], ref[key][:k]), key
    assert np.array_equal(got["bary"].view(np.uint32), ref["bary"][:k].view(np.uint32))
    return ref


def test_strips_default_rules_bit_exact():
    # 3000 modules of 512 / 256 strips: ~1.4 M strips = 176 tiles of 8192, modules straddle tile boundaries, ragged tail
    d = datagen.make_strips(11, 3000)
    ref = check(d, datagen.default_strip_params())
    assert len(ref["module"]) > 3000


def test_strips_gap_rules_and_thresholds():
    d = datagen.make_strips(12, 700, strips_per_module=300, occupancy=0.05, bad_frac=0.05)     # 300: tiles unaligned to modules
    for kw in (dict(max_holes=1, max_bad=0), dict(max_holes=2, max_bad=2, min_charge=0), dict(max_holes=0, max_bad=0),
               dict(max_holes=15, max_bad=16), dict(clus_thr=8.0, seed_thr=4.0, chan_thr=1.0), dict(min_charge=200)):
        check(d, datagen.default_strip_params(**kw))


def test_strips_degenerate_inputs():
    sp = datagen.default_strip_params()
    d = datagen.make_strips(13, 64, strips_per_module=37)                 # tiny modules, length not a multiple of 8
    check(d, sp)
    # every strip passes: one cluster per module, walked across tiles (TILE = SC_TILE of csrc/mkf_strips.cu)
    TILE = 8192
    n = 3 * TILE + 5
    off = np.array([0, 9000, 9000, 20000, n], np.int32)                  # an empty module, modules longer than a tile
    full = dict(module_off=off, adc=np.full(n, 100, np.uint16), noise=np.full(n, 4, np.float32), bad=np.zeros(n, np.uint8))
    ref = check(full, sp)
    assert ref["module"].tolist() == [0, 2, 3] and ref["last"].tolist() == [8999, 10999, n - 20001]
    # alternating strips: the largest number of clusters a tile can hold (TILE / 2 starts per tile)
    alt = dict(full, adc=np.where(np.arange(n) % 2 == 0, 100, 0).astype(np.uint16))
    ref = check(alt, sp)
    assert len(ref["module"]) == (n + 1) // 2
    # all bad, all quiet
    check(dict(full, bad=np.ones(n, np.uint8)), sp)
    check(dict(full, adc=np.zeros(n, np.uint16)), sp)
    # one-strip modules over more than two tiles: every tile meets thousands of modules (the global module_of path)
    m1 = 2 * TILE + 77
    one = dict(module_off=np.arange(m1 + 1, dtype=np.int32), adc=np.full(m1, 100, np.uint16), noise=np.full(m1, 4, np.float32),
               bad=np.zeros(m1, np.uint8))
    assert len(check(one, sp, capacity=m1)["module"]) == m1
    # capacity smaller than the number found: the count is still exact (the records are then incomplete)
    check(alt, sp, capacity=100)
    # saturated counts: 16-bit ADC at full scale over a long cluster (sums beyond 32 bits)
    sat = dict(full, adc=np.full(n, 65535, np.uint16))
    check(sat, sp)


def test_strips_empty_and_host_entry():
    from gpu_helpers import gpu_cluster_strips, strip_context
    sp = datagen.default_strip_params()
    empty = dict(module_off=np.zeros(1, np.int32), adc=np.zeros(0, np.uint16), noise=np.zeros(0, np.float32), bad=np.zeros(0, np.uint8))
    assert gpu_cluster_strips(empty, sp)["n_clusters"] == 0
    d = datagen.make_strips(14, 500)
    ref = mkfo.cluster_strips(d["module_off"], d["adc"], d["noise"], d["bad"], **sp)
    got = strip_context().cluster_strips_host(d, sp, capacity=len(d["adc"]) // 2 + 1)
    assert got["n_clusters"] == len(ref["module"])
    for key in ("module", "first", "last", "charge"):
        assert np.array_equal(got[key], ref[key]), key
    assert np.array_equal(got["bary"].view(np.uint32), ref["bary"].view(np.uint32))
    assert got["h2d_bytes"] == 7 * len(d["adc"]) + 4 * len(d["module_off"]) and got["d2h_bytes"] == 4 + 20 * len(ref["module"])


def test_strips_argument_errors():
    import torch
    from gpu_helpers import strip_context
    from paper_2002_06295_b200 import binding as B
    ctx = strip_context()
    d = datagen.make_strips(15, 20)
    sd = B.strips_to_device(d)
    n = len(d["adc"])
    out = B.alloc_clusters(n // 2 + 1)
    ws = torch.empty(ctx.workspace_bytes(B.MKF_CALL_CLUSTER_STRIPS, 0, n, n // 2 + 1), dtype=torch.uint8, device="cuda")
    with pytest.raises(B.MkfError):                   # the gap must fit the 32-strip halo
        ctx.cluster_strips(sd, datagen.default_strip_params(max_holes=20, max_bad=20), out, ws)
    with pytest.raises(B.MkfError):                   # workspace too small
        ctx.cluster_strips(sd, datagen.default_strip_params(), out, ws[:64])
    with pytest.raises(B.MkfError):                   # adc not 16-byte aligned
        bad = dict(sd, adc=sd["adc"][1:], noise=sd["noise"][1:], bad=sd["bad"][1:],
                   module_off=torch.tensor([0, n - 1], dtype=torch.int32, device="cuda"))
        ctx.cluster_strips(bad, datagen.default_strip_params(), out, ws)
    ctx.cluster_strips(sd, datagen.default_strip_params(), out, ws)      # and the context still works afterwards
    torch.cuda.synchronize()
    ref = mkfo.cluster_strips(d["module_off"], d["adc"], d["noise"], d["bad"], **datagen.default_strip_params())
    assert int(out["n_clusters"].item()) == len(ref["module"])
