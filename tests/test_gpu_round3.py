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


@pytest.mark.parametrize("zeta", [1.0, 1.5, 32.0])
@pytest.mark.parametrize("name", ["line3", "grid9"])
def test_collinear_triplets_where_the_angular_base_is_exactly_zero(pkg, name, zeta):
    """8 x 4 angular split (always the exp2(zeta log2 b) kernels) with angle shifts 0 and pi and cos_scale = 1: an
    exactly collinear triplet makes b = (1 + cos(theta - shf_z))/2 exactly 0.  The backward needs b^(zeta-1) there:
    1 for zeta = 1 (computed as ex2(0 * lg2(0)) it would be NaN), 0 otherwise."""
    import dataclasses
    from gen import ani2x_shaped_params
    from test_gpu_edge_cases import _collinear_systems
    from test_gpu_parity import AEV_TOL
    pos, sp = _collinear_systems()[name]
    p = dataclasses.replace(ani2x_shaped_params(1.0, num_species=4), zeta=np.float32(zeta),
                            shf_z=np.array([0.0, np.pi / 3, 2 * np.pi / 3, np.pi], dtype=np.float32))
    g = np.random.default_rng(6).standard_normal((1, len(sp), p.aev_length)).astype(np.float32)
    ctx = pkg.Context(p, max_atoms=len(sp))
    aev = ctx.aev_forward(torch.from_numpy(pos[None]).cuda(), torch.from_numpy(sp[None]).cuda(), None)
    f = ctx.aev_backward(torch.from_numpy(g).cuda())
    ctx.check_status()
    want_a = oracle.aev_forward(p, pos[None], sp[None], None)
    want_f = oracle.aev_backward(p, pos[None], sp[None], None, g)
    assert np.isfinite(f.cpu().numpy()).all()
    assert np.abs(aev.cpu().numpy() - want_a).max() <= AEV_TOL * np.abs(want_a).max()
    _check_forces(f.cpu().numpy(), want_f, what=(name, zeta))
    ctx.close()


@pytest.mark.parametrize("round_bf16", [True, False])
def test_kernel_choice_follows_the_documented_envelope(pkg, round_bf16):
    """include/aev.h (ani_mlp_load) states which shapes run on the tensor cores; ani_mlp_kernel must agree, for
    bf16-representable and for fp32 weights alike (hi + lo operands get two buffers, so the rule is the same)."""
    from gen import ani1x_style_params
    from test_gpu_fuzz import _in_tensor_core_envelope
    p = ani1x_style_params(num_species=1)
    L = p.aev_length
    cases = {(160, 128, 96): "tcgen05", (128, 160): "tcgen05", (160, 128): "tcgen05", (144, 128): "tcgen05",
             (144, 160): "fp32", (160, 160): "fp32", (96, 160, 160): "fp32", (176,): "fp32", (256, 192, 160): "fp32"}
    for hidden, want in cases.items():
        dims = [L] + list(hidden) + [1]
        assert _in_tensor_core_envelope(dims) == (want == "tcgen05"), hidden      # the restated rule itself
        nets = make_c5_weights(seed=11, arch={0: dims}, round_bf16=round_bf16)
        ctx = pkg.Context(p, max_atoms=8)
        ctx.ani_mlp_load(0, nets[0][0], nets[0][1], CELU_ALPHA)
        assert ctx.mlp_kernel() == want, (hidden, round_bf16)
        ctx.close()


@pytest.mark.parametrize("flags", [1, 1 | 2])
def test_deterministic_ensemble_forces_are_bit_identical(pkg, flags):
    """AEV_FLAG_DETERMINISTIC with an ensemble: the mean dE/dAEV is accumulated over the models in model order (one MLP
    launch per model), so ani_energy_forces returns bit-identical forces run to run - on the tensor-core kernel and
    (flag 2) on the fp32 kernel - and they still match the oracle."""
    from gen import make_ensemble_weights, make_water_box
    w = make_water_box(216, 18.64, 300, "det-ens")
    models = make_ensemble_weights(3)
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms, flags=flags)
    ctx.ani_mlp_set_ensemble(len(models))
    for m, nets in enumerate(models):
        for s, (ws, bs) in nets.items():
            ctx.ani_mlp_load_model(m, s, ws, bs, CELU_ALPHA)
    assert ctx.mlp_kernel() == ("fp32" if flags & 2 else "tcgen05")
    pos, sp = torch.from_numpy(w.pos).cuda(), torch.from_numpy(w.species).cuda()
    runs = []
    for _ in range(4):
        e, f = ctx.ani_energy_forces(pos, sp, w.box)
        runs.append((e.clone(), f.clone()))
    ctx.check_status()
    for e, f in runs[1:]:
        assert torch.equal(f, runs[0][1])
    we, wf, _ = oracle.energy_forces_ensemble(w.params, w.pos, w.species, w.box, models, CELU_ALPHA, use_cells=True)
    assert abs(float(runs[0][0][0]) - we[0]) <= 1e-4 * max(1.0, abs(we[0]))
    _check_forces(runs[0][1].cpu().numpy().astype(np.float64), wf, C5_FORCE_TOL, C5_FORCE_MAX_TOL, what=("det ens", flags))
    ctx.close()


def test_c4_in_a_deterministic_context(pkg):
    """The headline workload (23,559 atoms, cell list) under AEV_FLAG_DETERMINISTIC: k_rank's per-bin ordering and the
    fixed-point accumulator at full size; AEV and forces bit-identical over two runs and within the oracle tolerances."""
    from test_gpu_parity import AEV_TOL
    w = make_workload("C4")
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms, flags=pkg.AEV_FLAG_DETERMINISTIC)
    pos, sp, g = (torch.from_numpy(x).cuda() for x in (w.pos, w.species, w.grad_aev))
    a1 = ctx.aev_forward(pos, sp, w.box).clone()
    f1 = ctx.aev_backward(g).clone()
    a2 = ctx.aev_forward(pos, sp, w.box)
    f2 = ctx.aev_backward(g)
    ctx.check_status()
    assert torch.equal(a1, a2) and torch.equal(f1, f2)
    want_a = oracle.aev_forward(w.params, w.pos, w.species, w.box, use_cells=True)
    want_f = oracle.aev_backward(w.params, w.pos, w.species, w.box, w.grad_aev, use_cells=True)
    assert np.abs(a1.cpu().numpy() - want_a).max() <= AEV_TOL * np.abs(want_a).max()
    _check_forces(f1.cpu().numpy(), want_f, what="C4 deterministic")
    ctx.close()


def test_c4_with_a_verlet_skin(pkg):
    """C4 with skin = 0.5 over three frames of a random walk: the Verlet capacities (vcap_r) at full size; pair sets
    bit-exact against the oracle and forces within tolerance at every frame, lists reused at least once."""
    from gen import random_walk
    w = make_workload("C4")
    frames = random_walk(w, 3, 0.02, 11)
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms, skin=0.5)
    sp, g = torch.from_numpy(w.species).cuda(), torch.from_numpy(w.grad_aev).cuda()
    for t, fr in enumerate(frames):
        fr = np.ascontiguousarray(fr)
        ctx.aev_forward(torch.from_numpy(fr).cuda(), sp, w.box)
        f = ctx.aev_backward(g)
        ctx.check_status()
        got = ctx.aev_export_pairs(0, cap=w.n_atoms * 40)
        np.testing.assert_array_equal(got, oracle.pairs(fr[0], w.species[0], w.box, float(w.params.rcr), "cell"))
        if t in (0, 2):
            want_f = oracle.aev_backward(w.params, fr, w.species, w.box, w.grad_aev, use_cells=True)
            _check_forces(f.cpu().numpy(), want_f, what=("C4 skin", t))
    assert 1 <= ctx.neighbor_builds() < len(frames)
    ctx.close()


def test_ensemble_of_three_seven_species_models_on_the_tensor_cores(pkg):
    """Ensemble x L = 1008 together: three models per species of a seven-species set, so the
    mean dE/dAEV is built by vector REDs over 8 column chunks per model; tcgen05 kernel, oracle tolerances of C5."""
    from gen import ani1x_style_params, make_water_box
    from gen.workloads import C5_ARCH
    p7 = ani1x_style_params(num_species=7)
    w = make_water_box(216, 18.64, 303, "s7-ens")
    sp = np.random.default_rng(71).integers(0, 7, size=w.species.shape).astype(np.int32)
    arch = {s: [1008] + C5_ARCH[0 if s % 2 == 0 else 3][1:] for s in range(7)}
    models = [make_c5_weights(seed=20 + m, arch=arch, round_bf16=(m != 1)) for m in range(3)]
    ctx = pkg.Context(p7, max_atoms=w.n_atoms)
    ctx.ani_mlp_set_ensemble(3)
    for m, nets in enumerate(models):
        for s, (ws, bs) in nets.items():
            ctx.ani_mlp_load_model(m, s, ws, bs, CELU_ALPHA)
    assert ctx.mlp_kernel() == "tcgen05"
    e, f = ctx.ani_energy_forces(torch.from_numpy(w.pos).cuda(), torch.from_numpy(sp).cuda(), w.box)
    ctx.check_status()
    we, wf, _ = oracle.energy_forces_ensemble(p7, w.pos, sp, w.box, models, CELU_ALPHA, use_cells=True)
    assert abs(float(e[0]) - we[0]) <= 1e-4 * max(1.0, abs(we[0]))
    _check_forces(f.cpu().numpy().astype(np.float64), wf, C5_FORCE_TOL, C5_FORCE_MAX_TOL, what="S=7 ensemble of 3")
    ctx.close()


def test_deterministic_flag_on_the_unstaged_neighbour_scan(pkg):
    """A 1,200-atom gas-phase cluster is one cell whose candidates exceed the shared-memory stage, so k_nbr scans global
    memory with warp ballots.  Under AEV_FLAG_DETERMINISTIC that scan reads the cell in atom-index order (k_rank), so
    lists, AEV and forces are bit-identical run to run here too, and match the oracle."""
    from gen import make_water_box
    from test_gpu_parity import AEV_TOL
    wb = make_water_box(400, 24.0, 910, "cluster")
    pos, sp, g = (torch.from_numpy(x).cuda() for x in (wb.pos, wb.species, wb.grad_aev))
    ctx = pkg.Context(wb.params, max_atoms=wb.n_atoms, flags=pkg.AEV_FLAG_DETERMINISTIC)
    runs = []
    for _ in range(3):
        a = ctx.aev_forward(pos, sp, None).clone()
        runs.append((a, ctx.aev_backward(g).clone()))
    ctx.check_status()
    for a, f in runs[1:]:
        assert torch.equal(a, runs[0][0]) and torch.equal(f, runs[0][1])
    got = ctx.aev_export_pairs(0, cap=wb.n_atoms * 64)
    np.testing.assert_array_equal(got, oracle.pairs(wb.pos[0], wb.species[0], None, float(wb.params.rcr), "brute"))
    want_aev = oracle.aev_forward(wb.params, wb.pos, wb.species, None, use_cells=False)
    want_f = oracle.aev_backward(wb.params, wb.pos, wb.species, None, wb.grad_aev, use_cells=False)
    assert np.abs(runs[0][0].cpu().numpy() - want_aev).max() <= AEV_TOL * np.abs(want_aev).max()
    _check_forces(runs[0][1].cpu().numpy(), want_f, what="unstaged, deterministic")
    ctx.close()


@pytest.mark.parametrize("k_slabs", [2, 4])
def test_slabs_of_central_atoms_add_up_to_the_full_evaluation(pkg, k_slabs):
    """SURVEY 8(f) rank 4 (sharding over GPUs), testable on one GPU: C3 evaluated as K slabs of central atoms with
    aev_forward_range.  Each slab's AEV rows equal the oracle's rows, rows outside the slab are not written, each
    slab's partial forces equal the oracle's backward with the upstream gradient masked to the slab (forces are linear
    in the gradient rows), and the partial forces add up to the full forces."""
    from paper_2310_03121_b200.sharded import central_ranges
    from test_gpu_parity import AEV_TOL
    w = make_workload("C3")
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms)
    pos, sp, g = (torch.from_numpy(x).cuda() for x in (w.pos, w.species, w.grad_aev))
    want_a = oracle.aev_forward(w.params, w.pos, w.species, w.box, use_cells=True)
    want_f = oracle.aev_backward(w.params, w.pos, w.species, w.box, w.grad_aev, use_cells=True)
    scale = np.abs(want_a).max()
    total = np.zeros_like(want_f)
    ranges = central_ranges(w.n_atoms, k_slabs)
    assert ranges[0][0] == 0 and sum(c for _, c in ranges) == w.n_atoms
    for first, count in ranges:
        out = torch.full((1, w.n_atoms, ctx.length), -3.0, dtype=torch.float32, device="cuda")
        ctx.aev_forward_range(pos, sp, w.box, first, count, aev_out=out)
        f = ctx.aev_backward(g)
        ctx.check_status()
        a = out.cpu().numpy()[0]
        assert np.abs(a[first:first + count] - want_a[0, first:first + count]).max() <= AEV_TOL * scale
        assert (a[:first] == -3.0).all() and (a[first + count:] == -3.0).all()
        gm = np.zeros_like(w.grad_aev)
        gm[0, first:first + count] = w.grad_aev[0, first:first + count]
        want_p = oracle.aev_backward(w.params, w.pos, w.species, w.box, gm, use_cells=True)
        _check_forces(f.cpu().numpy(), want_p, what=("slab", k_slabs, first))
        total += f.cpu().numpy().astype(np.float64)
    _check_forces(total, want_f, what=("slabs summed", k_slabs))
    # the next plain call is a full evaluation again (the range does not stick)
    ctx.aev_forward(pos, sp, w.box)
    _check_forces(ctx.aev_backward(g).cpu().numpy(), want_f, what="full after slabs")
    with pytest.raises(pkg.AevError):
        ctx.aev_forward_range(pos, sp, w.box, w.n_atoms - 10, 11)
    ctx.close()
