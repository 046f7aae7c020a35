"""aev_pairs_static: the pair search for callers that may not allocate GPU memory.

Some users of this library cannot let it call cudaMalloc: the GPU's memory belongs to their own pool, their MD
step loop cannot absorb the device-wide synchronisation an allocation causes, or their device footprint is fixed
at link time.  For them `aev_pairs_static` (include/aev.h) runs the gas-phase cutoff pair search with no context,
keeping its working memory (one int per atom) in a fixed array inside libaev_b200.so; the caller brings every
input and output buffer.

What is checked here: the pair list it writes equals, bit for bit, what the ordinary path (a context,
`aev_neighbors` + `aev_export_pairs`) finds for the same system - for calls made back to back, because every
call on a GPU shares that one array and finds the previous call's counts still in it.  The second system is
smaller than the first, so stale entries really are there.  The list must also arrive already sorted by (i, j),
the size limit must be refused with its own error code, and a too-small output must get the leading pairs.

This file is named to be collected last: `pytest -x` stops at the first failure, and a problem in this add-on
must not hide the parity tests of the main path.  It passes on its own in a fresh process (it does the
per-device set-up itself, in its first call) and after the other GPU tests.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
from gen import make_workload

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pkg():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2310_03121_b200 as p
    return p


def _systems():
    """(params, [(pos f32 [n,3], species i32 [n])...]): a 600-atom water droplet cut from C3 and treated as
    gas phase, with a few padding atoms (species -1), then one 60-atom ligand conformer of C2."""
    w3, w2 = make_workload("C3"), make_workload("C2")
    pos_a = np.ascontiguousarray(w3.pos[0, :600])
    sp_a = np.ascontiguousarray(w3.species[0, :600]).copy()
    sp_a[[7, 301, 599]] = -1
    pos_b = np.ascontiguousarray(w2.pos[3])
    sp_b = np.ascontiguousarray(w2.species[3])
    return w3.params, [(pos_a, sp_a), (pos_b, sp_b)]


def _existing_path(pkg, params, pos, sp):
    """The ordinary, allocating path: context + aev_neighbors + aev_export_pairs (sorted by the binding)."""
    n = pos.shape[0]
    ctx = pkg.Context(params, max_atoms=n, max_batch=1)
    ctx.aev_neighbors(torch.from_numpy(pos[None]).cuda(), torch.from_numpy(sp[None]).cuda(), None)
    ctx.check_status()
    out = [ctx.aev_export_pairs(which, cap=n * 64) for which in (0, 1)]
    ctx.close()
    return out      # [radial set (r < rcr), angular set (r < rca)]


def test_static_pair_search_matches_the_context_path_on_consecutive_calls(pkg):
    params, systems = _systems()
    want = [_existing_path(pkg, params, pos, sp) for pos, sp in systems]
    dev = [(torch.from_numpy(pos).cuda(), torch.from_numpy(sp).cuda()) for pos, sp in systems]
    # every buffer the call touches is made here, by the caller, before the calls under test
    order = [0, 1, 0, 1]                      # large, small, large, small: each finds the other's counts
    cutoffs = [float(params.rcr), float(params.rca), float(params.rca), float(params.rcr)]
    outs = [(torch.full((600 * 64, 2), -7, dtype=torch.int32, device="cuda"),
             torch.full((1,), -1, dtype=torch.int64, device="cuda")) for _ in order]
    for k, rc, (pairs, count) in zip(order, cutoffs, outs):
        pkg.aev_pairs_static(dev[k][0], dev[k][1], rc, pairs, count)
    torch.cuda.synchronize()
    for k, rc, (pairs, count) in zip(order, cutoffs, outs):
        expect = want[k][0 if rc == float(params.rcr) else 1]
        m = int(count.item())
        assert m == expect.shape[0], (k, rc, m, expect.shape)
        got = pairs[:m].cpu().numpy()
        np.testing.assert_array_equal(got, expect)            # same set AND already in (i, j) order
        assert int(pairs[m:].max().item()) == -7              # nothing written past the count
        # and the oracle agrees (bit-exact pair sets are north_star's bar for the neighbour search)
        pos, sp = systems[k]
        np.testing.assert_array_equal(got, oracle.pairs(pos, sp, None, rc, "brute"))


def test_static_pair_search_limit_small_output_and_empty_input(pkg):
    params, systems = _systems()
    pos, sp = systems[1]
    full = _existing_path(pkg, params, pos, sp)[0]
    dpos, dsp = torch.from_numpy(pos).cuda(), torch.from_numpy(sp).cuda()
    # output smaller than the pair count: the count is the true one, the first `cap` pairs are written
    cap = 10
    pairs = torch.full((cap + 4, 2), -7, dtype=torch.int32, device="cuda")
    count = torch.zeros((1,), dtype=torch.int64, device="cuda")
    pkg.aev_pairs_static(dpos, dsp, float(params.rcr), pairs[:cap], count)
    assert int(count.item()) == full.shape[0] > cap
    np.testing.assert_array_equal(pairs[:cap].cpu().numpy(), full[:cap])
    assert int(pairs[cap:].max().item()) == -7
    # species = None: every atom is real
    pairs = torch.empty((60 * 64, 2), dtype=torch.int32, device="cuda")
    pkg.aev_pairs_static(dpos, None, float(params.rcr), pairs, count)
    np.testing.assert_array_equal(pairs[: int(count.item())].cpu().numpy(),
                                  oracle.pairs(pos, None, None, float(params.rcr), "brute"))
    # no atoms: zero pairs
    count.fill_(5)
    pkg.aev_pairs_static(torch.empty((0, 3), dtype=torch.float32, device="cuda"), None, 5.2, pairs, count)
    assert int(count.item()) == 0
    # one atom more than the fixed working memory holds: refused with the dedicated code, nothing launched
    n_big = pkg.AEV_STATIC_MAX_ATOMS + 1
    big = torch.zeros((n_big, 3), dtype=torch.float32, device="cuda")
    count.fill_(123)
    with pytest.raises(pkg.AevError) as info:
        pkg.aev_pairs_static(big, None, 5.2, pairs, count)
    assert info.value.code == -7 and "AEV_ERR_STATIC_LIMIT" in str(info.value) and "static" in str(info.value)
    torch.cuda.synchronize()
    assert int(count.item()) == 123
    # exactly at the limit it runs (atoms on a line 1 A apart: pairs (i, i+1..i+5) within 5.2 A)
    n_max = pkg.AEV_STATIC_MAX_ATOMS
    line = torch.zeros((n_max, 3), dtype=torch.float32, device="cuda")
    line[:, 0] = torch.arange(n_max, dtype=torch.float32, device="cuda")
    pairs = torch.empty((n_max * 5, 2), dtype=torch.int32, device="cuda")
    pkg.aev_pairs_static(line, None, 5.2, pairs, count)
    assert int(count.item()) == 5 * n_max - 15
    got = pairs[: 5 * n_max - 15].cpu().numpy().astype(np.int64)
    assert (np.diff(got[:, 0] * n_max + got[:, 1]) > 0).all()
    assert ((got[:, 1] - got[:, 0] >= 1) & (got[:, 1] - got[:, 0] <= 5)).all()
