"""hea_pool_rank_static -- the allocation-free ranking entry point (static device scratch, include/hea.h) -- against the
existing path, hea_pool_select, which keeps the same scratch in cudaMalloc'ed buffers.  Integer output: bit-equal, the
bar of every index test here.  Several calls in a row with different sizes and data: the static array is shared and
keeps the previous call's contents, which must not leak into the next result.

Collected LAST on purpose (file name): the suite runs with `pytest -x`.  The test holds no state of other tests and
passes alone in a fresh process (the first call on a device resolves the scratch address) as well as after them."""
import ctypes as C

import numpy as np
import pytest
import torch

from test_gpu_parity import small

pytestmark = pytest.mark.gpu


def existing_path_order(h, occ, counts, stats, n_keep):
    """order_dev of hea_pool_select on copies (n_keep == C: nothing is regenerated, the call only ranks and permutes)."""
    o, c, s = occ.clone(), counts.clone(), stats.clone()
    order = h.pool_select(o, c, s, n_keep, seed=1, new_chain0=1 << 20)
    torch.cuda.synchronize()
    return order.cpu().numpy().copy()


def test_pool_rank_static_matches_pool_select_on_calls_in_a_row(hb):
    w = small("bcc", (6, 5, 4), [0.25] * 4, 3, target_seed=5, K=16, rng=(-0.15, 0.15))
    h = hb.Hea(*w.create_args())
    C1 = 700                                                   # three blocks of the ranking kernel and a ragged tail
    occ = h.init_random(C1, seed=w.seed)
    counts, _, _ = h.sro_full(occ, want_alpha=False, want_obj=False)
    stats, _ = h.mc_run(occ, counts, 10, w.K, w.seed)            # chains at different J, some of them equal
    counts[5] = counts[400]                                    # exact ties: the lower index ranks first
    counts[6] = counts[400]
    occ[5] = occ[400]
    occ[6] = occ[400]
    _, _, obj = h.sro_full(occ)
    J = obj.cpu().numpy()
    assert len(np.unique(J)) > 50 and J[5] == J[400] == J[6]

    # ---- call 1: every chain ranked
    order1 = torch.full((C1,), -1, dtype=torch.int32, device=h.device)
    h.pool_rank_static(counts, C1, order1)
    torch.cuda.synchronize()
    want1 = existing_path_order(h, occ, counts, stats, C1)
    np.testing.assert_array_equal(order1.cpu().numpy(), want1)
    np.testing.assert_array_equal(want1, np.argsort(J, kind="stable").astype(np.int32))
    assert list(want1).index(5) + 1 == list(want1).index(6) and list(want1).index(6) + 1 == list(want1).index(400)

    # ---- call 2, straight after: fewer chains, other data, n_keep < C (the scratch still holds call 1's 700 values)
    lo, C2, keep2 = 300, 150, 37
    occ2, counts2, stats2 = occ[lo:lo + C2].clone(), counts[lo:lo + C2].clone(), stats[lo:lo + C2].clone()
    order2 = torch.full((keep2 + 3,), -7, dtype=torch.int32, device=h.device)
    free_before = torch.cuda.mem_get_info()[0]
    h.pool_rank_static(counts2, keep2, order2)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before         # no device memory was taken by the call
    want2 = existing_path_order(h, occ2, counts2, stats2, keep2)
    got2 = order2.cpu().numpy()
    np.testing.assert_array_equal(got2[:keep2], want2)
    np.testing.assert_array_equal(got2[keep2:], -7)            # nothing written beyond n_keep
    np.testing.assert_array_equal(want2, np.argsort(J[lo:lo + C2], kind="stable")[:keep2].astype(np.int32))

    # ---- call 3: call 1 again -- the same answer after the smaller call
    order3 = torch.full((C1,), -1, dtype=torch.int32, device=h.device)
    h.pool_rank_static(counts, C1, order3)
    torch.cuda.synchronize()
    np.testing.assert_array_equal(order3.cpu().numpy(), want1)
    h.close()


def test_pool_rank_static_at_its_maximum_and_beyond(hb):
    w = small("fcc", (3, 3, 3), [0.5, 0.5], 1, target_seed=3, K=8)
    h = hb.Hea(*w.create_args())
    Cmax = hb.Hea.POOL_RANK_STATIC_MAX
    base = 512
    occ_b = h.init_random(base, seed=7)
    cnt_b, _, _ = h.sro_full(occ_b, want_alpha=False, want_obj=False)
    reps = Cmax // base
    occ, counts = occ_b.repeat(reps, 1).contiguous(), cnt_b.repeat(reps, 1, 1, 1).contiguous()    # many exact ties
    stats = h.new_stats(Cmax)
    order = torch.full((Cmax,), -1, dtype=torch.int32, device=h.device)
    for _ in range(2):                                         # two calls in a row at the full size of the scratch
        order.fill_(-1)
        h.pool_rank_static(counts, Cmax, order)
        torch.cuda.synchronize()
        got = order.cpu().numpy()
        np.testing.assert_array_equal(np.sort(got), np.arange(Cmax, dtype=np.int32))             # a permutation
    np.testing.assert_array_equal(got, existing_path_order(h, occ, counts, stats, Cmax))
    # one chain more than the scratch holds: refused before any launch, with the limit in the message
    L = hb.lib()
    p = C.c_void_p(counts.data_ptr())
    assert L.hea_pool_rank_static(h._h, p, Cmax + 1, 1, C.c_void_p(order.data_ptr()), None) == hb.HEA_EINVAL
    assert str(Cmax).encode() in L.hea_last_error() and b"HEA_POOL_RANK_STATIC_MAX" in L.hea_last_error()
    assert L.hea_pool_rank_static(h._h, p, 10, 11, C.c_void_p(order.data_ptr()), None) == hb.HEA_EINVAL
    assert L.hea_pool_rank_static(h._h, None, 10, 5, C.c_void_p(order.data_ptr()), None) == hb.HEA_EINVAL
    assert L.hea_pool_rank_static(h._h, None, 0, 0, None, None) == hb.HEA_OK                    # empty pool
    h.close()
