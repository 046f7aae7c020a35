"""GPU tests added in round 3: host-side bookkeeping around the replayed host-call graph, reproducibility of ensembles,
degenerate angular parameters, and the configurations round 2 left without a parity test (C4 in deterministic and
Verlet-skin contexts).  Tolerances as in tests/test_gpu_parity.py.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
from gen import make_c5_weights, make_workload
from gen.workloads import CELU_ALPHA

from test_gpu_parity import C5_FORCE_MAX_TOL, C5_FORCE_TOL, _check_forces

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pkg():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2310_03121_b200 as p
    return p


def test_host_graph_replay_on_a_skin_context_after_a_call_with_other_shapes(pkg):
    """A Verlet-skin context replays ani_energy_forces_host as a CUDA graph.  The "shapes changed, drop the Verlet lists"
    decision is host-side bookkeeping that is not part of the graph: when another entry point evaluates a different
    system in between (here the first 40 atoms of the same molecule, so the displacement check alone sees nothing
    move), the next replay must still rebuild its lists, and the context's geometry must be the replayed system's
    afterwards (aev_export_pairs reads it)."""
    w = make_workload("C2")
    nets = make_c5_weights(seed=3, arch={s: [384, 96, 64, 1] for s in range(4)})
    ctx = pkg.Context(w.params, max_atoms=60, skin=0.5)
    for s, (ws, bs) in nets.items():
        ctx.ani_mlp_load(s, ws, bs, CELU_ALPHA)
    pos, sp = np.ascontiguousarray(w.pos[:1]), np.ascontiguousarray(w.species[:1])
    pos40, sp40 = np.ascontiguousarray(pos[:, :40]), np.ascontiguousarray(sp[:, :40])
    want_e, want_f, _ = oracle.energy_forces(w.params, pos, sp, None, nets, CELU_ALPHA)
    want_e40, want_f40, _ = oracle.energy_forces(w.params, pos40, sp40, None, nets, CELU_ALPHA)
    want_pairs = oracle.pairs(pos[0], sp[0], None, float(w.params.rcr), "brute")

    def host_call(what):
        e, f = ctx.ani_energy_forces_host(pos, sp, None)
        assert abs(e[0] - want_e[0]) <= 1e-4 * max(1.0, abs(want_e[0])), what
        _check_forces(f.astype(np.float64), want_f, C5_FORCE_TOL, C5_FORCE_MAX_TOL, what=what)

    for k in range(3):                                    # eager, capture, replay
        host_call(("before", k))
    builds = ctx.neighbor_builds()
    e40, f40 = ctx.ani_energy_forces(torch.from_numpy(pos40).cuda(), torch.from_numpy(sp40).cuda(), None)
    ctx.check_status()
    assert abs(float(e40[0]) - want_e40[0]) <= 1e-4 * max(1.0, abs(want_e40[0]))
    _check_forces(f40.cpu().numpy().astype(np.float64), want_f40, C5_FORCE_TOL, C5_FORCE_MAX_TOL, what="40 atoms")
    assert ctx.neighbor_builds() == builds + 1
    host_call("replay after the 40-atom call")          # without the fix: lists of the 40-atom system, wrong forces
    assert ctx.neighbor_builds() == builds + 2
    np.testing.assert_array_equal(ctx.aev_export_pairs(0, cap=60 * 60), want_pairs)      # geometry of the replayed call
    host_call("replay again")
    assert ctx.neighbor_builds() == builds + 2           # nothing moved: the lists are reused
    ctx.close()
