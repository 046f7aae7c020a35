"""GPU parity for the SURVEY.md 8(f) rows built in round 2: ensembles of networks,
fp32 (non-bf16) weights and the 7-species AEV on the tensor-core MLP, the deterministic backward,
flags and deferred errors of the host entry points.  Tolerances as in tests/test_gpu_parity.py.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
from gen import ani1x_style_params, make_c5_weights, make_ensemble_weights, make_water_box, make_workload
from gen.workloads import C5_ARCH, CELU_ALPHA

from test_gpu_parity import C5_FORCE_MAX_TOL, C5_FORCE_TOL, _check_forces, _dev

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pkg():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2310_03121_b200 as p
    return p


def _load_ensemble(ctx, models):
    ctx.ani_mlp_set_ensemble(len(models))
    for m, nets in enumerate(models):
        for s, (ws, bs) in nets.items():
            ctx.ani_mlp_load_model(m, s, ws, bs, CELU_ALPHA)


def _energy_forces(ctx, w):
    pos, sp, _ = _dev(w)
    e, f = ctx.ani_energy_forces(pos, sp, w.box)
    ctx.check_status()
    return e.cpu().numpy(), f.cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("flags", [0, 2])
def test_ensemble_of_eight_on_c5(pkg, flags):
    """eight networks per species over one AEV; energy and forces are the
    mean over the models (one AEV forward, one AEV backward).  flags = 2 runs the fp32 CUDA-core kernel."""
    w = make_workload("C5")
    models = make_ensemble_weights(8)
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms, flags=flags)
    _load_ensemble(ctx, models)
    e, f = _energy_forces(ctx, w)
    we, wf, _ = oracle.energy_forces_ensemble(w.params, w.pos, w.species, w.box, models, CELU_ALPHA, use_cells=True)
    assert abs(e[0] - we[0]) <= 1e-4 * max(1.0, abs(we[0]))
    _check_forces(f, wf, C5_FORCE_TOL, C5_FORCE_MAX_TOL, what=("ens8", flags))
    # a second evaluation on the same context (the cleared mean-gradient buffer is rebuilt every call)
    e2, f2 = _energy_forces(ctx, w)
    assert abs(e2[0] - e[0]) <= 1e-6 * max(1.0, abs(e[0]))      # order inside a cell, RED order
    np.testing.assert_allclose(f2, f, rtol=0, atol=1e-5 * np.abs(f).max())
    ctx.close()


def test_ensemble_of_identical_models_equals_one_model(pkg):
    w = make_water_box(216, 18.64, 300, "ens-box")
    nets = make_c5_weights()
    c1 = pkg.Context(w.params, max_atoms=w.n_atoms)
    for s, (ws, bs) in nets.items():
        c1.ani_mlp_load(s, ws, bs, CELU_ALPHA)
    e1, f1 = _energy_forces(c1, w)
    c4 = pkg.Context(w.params, max_atoms=w.n_atoms)
    _load_ensemble(c4, [nets] * 4)
    e4, f4 = _energy_forces(c4, w)
    assert abs(e4[0] - e1[0]) <= 1e-6 * max(1.0, abs(e1[0]))
    np.testing.assert_allclose(f4, f1, rtol=0, atol=2e-5 * np.abs(f1).max())
    c1.close(); c4.close()


@pytest.mark.parametrize("n_models", [1, 3])
def test_fp32_weights_stay_on_the_tensor_cores(pkg, n_models):
    """Weights that are not bf16-representable (any trained network): hi + lo weight operands, three MMAs
    per K step; same tolerance as the bf16 model of C5."""
    w = make_workload("C5")
    models = make_ensemble_weights(n_models, round_bf16=False)
    assert any(np.any(x.view(np.uint32) & 0xFFFF) for x in models[0][0][0])
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms)
    ctx.aev_set_profiling(True)
    _load_ensemble(ctx, models)
    e, f = _energy_forces(ctx, w)
    we, wf, _ = oracle.energy_forces_ensemble(w.params, w.pos, w.species, w.box, models, CELU_ALPHA, use_cells=True)
    assert abs(e[0] - we[0]) <= 1e-4 * max(1.0, abs(we[0]))
    _check_forces(f, wf, C5_FORCE_TOL, C5_FORCE_MAX_TOL, what=("fp32 weights on tcgen05", n_models))
    assert ctx.mlp_kernel() == "tcgen05"
    ctx.close()


def test_fp32_flag_runs_the_cuda_core_kernel_within_fp32_tolerance(pkg):
    w = make_workload("C5")
    nets = make_c5_weights(round_bf16=False)
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms, flags=pkg.AEV_FLAG_MLP_FP32)
    for s, (ws, bs) in nets.items():
        ctx.ani_mlp_load(s, ws, bs, CELU_ALPHA)
    e, f = _energy_forces(ctx, w)
    we, wf, _ = oracle.energy_forces(w.params, w.pos, w.species, w.box, nets, CELU_ALPHA, use_cells=True)
    assert abs(e[0] - we[0]) <= 1e-4 * max(1.0, abs(we[0]))
    _check_forces(f, wf, what="fp32 kernel")
    assert ctx.mlp_kernel() == "fp32"
    ctx.close()


def test_seven_species_model_on_the_tensor_cores(pkg):
    """ANI-2x-shaped model (seven elements): L = 1008 through k_mlp_tc (16 K-stages of layer 0,
    8 column chunks of dE/dAEV through two alternating TMEM slots)."""
    p7 = ani1x_style_params(num_species=7)
    w = make_water_box(216, 18.64, 301, "s7-box")
    rng = np.random.default_rng(70)
    sp = rng.integers(0, 7, size=w.species.shape).astype(np.int32)
    arch = {s: [1008] + C5_ARCH[0 if s % 2 == 0 else 3][1:] for s in range(7)}
    nets = make_c5_weights(seed=5, arch=arch, round_bf16=(False))
    ctx = pkg.Context(p7, max_atoms=w.n_atoms)
    for s, (ws, bs) in nets.items():
        ctx.ani_mlp_load(s, ws, bs, CELU_ALPHA)
    e, f = ctx.ani_energy_forces(torch.from_numpy(w.pos).cuda(), torch.from_numpy(sp).cuda(), w.box)
    ctx.check_status()
    assert ctx.mlp_kernel() == "tcgen05"
    we, wf, _ = oracle.energy_forces(p7, w.pos, sp, w.box, nets, CELU_ALPHA, use_cells=True)
    assert abs(float(e[0]) - we[0]) <= 1e-4 * max(1.0, abs(we[0]))
    _check_forces(f.cpu().numpy().astype(np.float64), wf, C5_FORCE_TOL, C5_FORCE_MAX_TOL, what="S=7 model")
    ctx.close()


@pytest.mark.parametrize("name", ["C2", "C3"])
def test_deterministic_flag_gives_bit_identical_forces(pkg, name):
    """AEV_FLAG_DETERMINISTIC: neighbour contributions are accumulated in 64-bit fixed
    point, so forces are bit-identical run to run, and still match the oracle."""
    w = make_workload(name)
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms, max_batch=w.batch, flags=pkg.AEV_FLAG_DETERMINISTIC)
    pos, sp, g = _dev(w)
    runs = []
    for _ in range(3):
        a = ctx.aev_forward(pos, sp, w.box).clone()
        f = ctx.aev_backward(g).clone()
        runs.append((a, f))
    ctx.check_status()
    for a, f in runs[1:]:
        assert torch.equal(a, runs[0][0])
        assert torch.equal(f, runs[0][1])
    want = oracle.aev_backward(w.params, w.pos, w.species, w.box, w.grad_aev, use_cells=w.box is not None)
    _check_forces(runs[0][1].cpu().numpy(), want, what=("deterministic", name))
    ctx.close()


def test_host_entry_points_report_device_side_errors(pkg):
    """a capacity overflow must not come back as AEV_OK from the synchronous host calls."""
    w = make_workload("C1")
    ctx = pkg.Context(w.params, max_atoms=24, max_radial_nbrs=16, max_angular_nbrs=4)
    with pytest.raises(pkg.AevError) as e:
        ctx.aev_forward_backward_host(w.pos, w.species, None, w.grad_aev)
    assert e.value.code == -3
    ctx.close()
    # a species without a network: AEV_ERR_STATE from ani_energy_forces_host
    ctx = pkg.Context(w.params, max_atoms=24)
    ws, bs = make_c5_weights()[0]
    ctx.ani_mlp_load(0, ws, bs, CELU_ALPHA)
    with pytest.raises(pkg.AevError) as e:
        ctx.ani_energy_forces_host(w.pos, w.species, None)
    assert e.value.code == -4
    ctx.close()


# --------------------------------------------------------------------------- small and triclinic cells (8(f) rank 3)
def _check_cell(pkg, w, flags=0, lattice=None):
    from test_gpu_parity import AEV_TOL
    import contextlib
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms, flags=flags)
    pos, sp, g = _dev(w)
    ctx.aev_neighbors(pos, sp, w.box)
    ctx.check_status()
    scope = oracle.lattice(lattice) if lattice is not None else contextlib.nullcontext()
    obox = None if lattice is not None else w.box
    with scope:
        for which, rc in ((0, w.params.rcr), (1, w.params.rca)):
            got = ctx.aev_export_pairs(which, cap=w.n_atoms * 80)
            want = oracle.pairs(w.pos[0], w.species[0], obox, float(rc), "brute").astype(np.int32)
            np.testing.assert_array_equal(got, want)
        want_a = oracle.aev_forward(w.params, w.pos, w.species, obox)
        want_f = oracle.aev_backward(w.params, w.pos, w.species, obox, w.grad_aev)
    aev = ctx.aev_forward(pos, sp, w.box)
    f = ctx.aev_backward(g)
    ctx.check_status()
    assert np.abs(aev.cpu().numpy() - want_a).max() <= AEV_TOL * np.abs(want_a).max()
    _check_forces(f.cpu().numpy(), want_f, what=(w.name, flags))
    ctx.close()


@pytest.mark.parametrize("cell", [(12.0, 13.0, 14.5), (11.0, 24.0, 17.0)])
def test_orthorhombic_boxes_with_fewer_than_three_cells_per_edge(pkg, cell):
    """PAPER.md:223 (a 528-atom periodic ML cell): edges between 2*R_cr and 3 cells (10.4 .. 15.6 A) are searched as
    one cell with the minimum image per pair; (11, 24, 17) has one short and two long edges."""
    from gen import make_periodic_cell
    n = int(0.1 * cell[0] * cell[1] * cell[2])
    _check_cell(pkg, make_periodic_cell(n, cell, 45, name="small-box"))


@pytest.mark.parametrize("det", [0, 1])
def test_triclinic_cell(pkg, det):
    from gen import make_periodic_cell
    lat = [[14.0, 0.0, 0.0], [3.0, 13.0, 0.0], [-2.0, 4.0, 12.5]]
    w = make_periodic_cell(240, lat, 46, name="triclinic")
    _check_cell(pkg, w, flags=pkg.AEV_FLAG_TRICLINIC | det, lattice=w.box)


def test_triclinic_argument_checks(pkg):
    p = ani1x_style_params()
    ctx = pkg.Context(p, max_atoms=8, flags=pkg.AEV_FLAG_TRICLINIC)
    pos = torch.rand((1, 8, 3), device="cuda") * 5
    sp = torch.zeros((1, 8), dtype=torch.int32, device="cuda")
    with pytest.raises(pkg.AevError) as e:      # not reduced: |bx| > ax/2
        ctx.aev_forward(pos, sp, np.array([14, 0, 0, 9, 13, 0, 0, 0, 12], dtype=np.float32))
    assert e.value.code == -1
    with pytest.raises(pkg.AevError) as e:      # cz < 2 R_cr
        ctx.aev_forward(pos, sp, np.array([14, 0, 0, 3, 13, 0, 0, 0, 9], dtype=np.float32))
    assert e.value.code == -2
    ctx.close()


# --------------------------------------------------------------------------- ml_atoms of a mixed system (8(f) rank 2)
def test_ml_subset_gathers_positions_and_adds_forces(pkg):
    """a 60-atom ML region inside a 4,500-atom system; the ML forces are added onto the
    (MM) forces already in the array, every other entry stays bit-identical."""
    big = make_workload("C3")
    lig = make_workload("C2")
    rng = np.random.default_rng(9)
    n_all, n_ml = big.n_atoms, lig.n_atoms
    idx = np.sort(rng.choice(n_all, size=n_ml, replace=False)).astype(np.int32)
    idx = rng.permutation(idx).astype(np.int32)
    pos_all = big.pos[0].copy()
    pos_all[idx] = lig.pos[0]                       # conformer 0 of the ligand sits at the ML indices
    sp_ml = lig.species[0].copy()
    f_mm = rng.standard_normal((n_all, 3)).astype(np.float32)
    nets = make_c5_weights(seed=3, arch={s: [384, 96, 64, 1] for s in range(4)})
    ctx = pkg.Context(lig.params, max_atoms=n_ml)
    for s, (ws, bs) in nets.items():
        ctx.ani_mlp_load(s, ws, bs, CELU_ALPHA)
    f_all = torch.from_numpy(f_mm.copy()).cuda()
    e = ctx.ani_energy_forces_subset(torch.from_numpy(pos_all).cuda(), torch.from_numpy(idx).cuda(),
                                     torch.from_numpy(sp_ml).cuda(), f_all)
    ctx.check_status()
    we, wf, _ = oracle.energy_forces(lig.params, lig.pos[:1], lig.species[:1], None, nets, CELU_ALPHA)
    got = f_all.cpu().numpy()
    assert abs(float(e[0]) - we[0]) <= 1e-4 * max(1.0, abs(we[0]))
    rest = np.ones(n_all, dtype=bool)
    rest[idx] = False
    np.testing.assert_array_equal(got[rest], f_mm[rest])
    _check_forces((got[idx].astype(np.float64) - f_mm[idx])[None], wf, C5_FORCE_TOL, C5_FORCE_MAX_TOL, what="ml subset")
    ctx.close()


# --------------------------------------------------------------------------- Verlet-skin reuse (8(f) rank 2)
@pytest.mark.parametrize("kind", ["water-box", "gas-batch", "small-cell"])
def test_verlet_skin_random_walk_matches_a_rebuild_every_step(pkg, kind):
    """PAPER.md:199 (10,000 consecutive MD steps): with aev_params.skin the lists are rebuilt only when an atom has
    moved more than skin/2; the exact cutoffs are applied when the lists are read, so every frame of a 20-step
    random walk gives the pair sets (bit-exact), AEV and forces of a context that rebuilds every call, and of the
    oracle.  Half-way the whole system is shifted by box vectors (a wrap is not a displacement)."""
    from gen import make_periodic_cell, random_walk
    from test_gpu_parity import AEV_TOL
    if kind == "water-box":
        w = make_water_box(216, 18.64, 310, "skin-box")
    elif kind == "gas-batch":
        w0 = make_workload("C2")
        w = type(w0)("skin-gas", w0.pos[:8].copy(), w0.species[:8].copy(), None, w0.grad_aev[:8].copy(), w0.params)
    else:
        w = make_periodic_cell(180, (13.0, 13.5, 14.0), 47, name="skin-cell")
    frames = random_walk(w, 20, 0.04, 5)
    skin = 0.6
    cs = pkg.Context(w.params, max_atoms=w.n_atoms, max_batch=w.batch, skin=skin)
    cr = pkg.Context(w.params, max_atoms=w.n_atoms, max_batch=w.batch)
    sp = torch.from_numpy(w.species).cuda()
    g = torch.from_numpy(w.grad_aev).cuda()
    for t, fr in enumerate(frames):
        fr = fr.copy()
        if w.box is not None and t >= 10:
            fr[:, ::3] += (np.asarray(w.box[:3]) * np.array([1, -1, 1])).astype(np.float32)
        pos = torch.from_numpy(fr).cuda()
        a_s = cs.aev_forward(pos, sp, w.box)
        f_s = cs.aev_backward(g)
        a_r = cr.aev_forward(pos, sp, w.box)
        f_r = cr.aev_backward(g)
        cs.check_status(); cr.check_status()
        for which in (0, 1):
            np.testing.assert_array_equal(cs.aev_export_pairs(which, cap=w.batch * w.n_atoms * 64),
                                          cr.aev_export_pairs(which, cap=w.batch * w.n_atoms * 64))
        # (the two contexts round displacements differently - wrapped position + image shift vs raw difference -
        #  so they agree to fp32 rounding of the coordinates, inside north_star's bounds)
        assert float((a_s - a_r).abs().max()) <= AEV_TOL * float(a_r.abs().max())
        assert float((f_s - f_r).abs().max()) <= 5e-5 * float(f_r.abs().max())
        if t in (0, 9, 19):
            want_a = oracle.aev_forward(w.params, fr, w.species, w.box)
            want_f = oracle.aev_backward(w.params, fr, w.species, w.box, w.grad_aev)
            assert np.abs(a_s.cpu().numpy() - want_a).max() <= AEV_TOL * np.abs(want_a).max()
            _check_forces(f_s.cpu().numpy(), want_f, what=("skin", kind, t))
    builds = cs.neighbor_builds()
    print("SKIN %s: %d builds in %d calls" % (kind, builds, len(frames)))
    assert 2 <= builds <= 8
    cs.close(); cr.close()


def test_verlet_skin_inside_a_cuda_graph(pkg):
    """The rebuild decision is taken on the device: one captured evaluation replayed over a trajectory (positions
    updated in place) rebuilds when it must and matches the uncaptured context frame by frame."""
    from gen import random_walk
    w = make_water_box(216, 18.64, 311, "skin-graph")
    frames = random_walk(w, 12, 0.05, 6)
    cs = pkg.Context(w.params, max_atoms=w.n_atoms, skin=0.5)
    cr = pkg.Context(w.params, max_atoms=w.n_atoms)
    sp = torch.from_numpy(w.species).cuda()
    g = torch.from_numpy(w.grad_aev).cuda()
    pos = torch.from_numpy(w.pos).cuda()
    aev = torch.empty((1, w.n_atoms, cs.length), dtype=torch.float32, device="cuda")
    f = torch.empty((1, w.n_atoms, 3), dtype=torch.float32, device="cuda")

    def step():
        cs.aev_forward(pos, sp, w.box, aev_out=aev)
        cs.aev_backward(g, forces_out=f)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        step()
    torch.cuda.current_stream().wait_stream(side)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        step()
    b0 = cs.neighbor_builds()
    for fr in frames:
        pos.copy_(torch.from_numpy(fr).cuda())
        graph.replay()
        a_r = cr.aev_forward(pos, sp, w.box)
        f_r = cr.aev_backward(g)
        assert float((aev - a_r).abs().max()) <= 1e-5 * float(a_r.abs().max())
        assert float((f - f_r).abs().max()) <= 5e-5 * float(f_r.abs().max())
    cs.check_status()
    builds = cs.neighbor_builds() - b0
    assert 1 <= builds < len(frames)
    del graph
    cs.close(); cr.close()


# --------------------------------------------------------------------------- the other angular split (8 x 4), zeta = 14.1
@pytest.mark.parametrize("cos_scale", [1.0, 0.95])
def test_eight_by_four_angular_split_with_general_zeta(pkg, cos_scale):
    """8 angular radial shifts x 4 angle shifts, zeta = 14.1, 7 species (L = 1008): the templated lane mappings of
    k_aev / k_backward (16 accumulators as 8 x 2 packed pairs) and the exp2(zeta log2 b) power, gas phase and periodic."""
    from gen import ani2x_shaped_params
    from test_gpu_parity import AEV_TOL
    p = ani2x_shaped_params(cos_scale)
    assert p.aev_length == 1008 and len(p.shf_a) == 8 and len(p.shf_z) == 4
    rng = np.random.default_rng(78)
    for name in ("C2", "C3"):
        w = make_workload(name)
        pos = w.pos[:4] if name == "C2" else w.pos
        sp = rng.integers(0, 7, size=pos.shape[:2]).astype(np.int32)
        g = rng.standard_normal(pos.shape[:2] + (1008,)).astype(np.float32)
        ctx = pkg.Context(p, max_atoms=pos.shape[1], max_batch=pos.shape[0])
        aev = ctx.aev_forward(torch.from_numpy(pos).cuda(), torch.from_numpy(sp).cuda(), w.box)
        f = ctx.aev_backward(torch.from_numpy(g).cuda())
        ctx.check_status()
        want_a = oracle.aev_forward(p, pos, sp, w.box, use_cells=w.box is not None)
        want_f = oracle.aev_backward(p, pos, sp, w.box, g, use_cells=w.box is not None)
        assert np.abs(aev.cpu().numpy() - want_a).max() <= AEV_TOL * np.abs(want_a).max()
        _check_forces(f.cpu().numpy(), want_f, what=("8x4 split", name, cos_scale))
        ctx.close()


def test_wide_hidden_layers_run_the_cuda_core_kernel(pkg):
    """Hidden widths above the tensor-core envelope (256 / 192 / 160: more than 512 TMEM columns) with the 8 x 4 split and
    7 species: the fp32 CUDA-core kernel takes over (ani_mlp_kernel says so) within the fp32 force tolerance."""
    from gen import ani2x_shaped_params
    p = ani2x_shaped_params()
    w = make_water_box(125, 15.6, 302, "wide-box")
    rng = np.random.default_rng(71)
    sp = rng.integers(0, 7, size=w.species.shape).astype(np.int32)
    nets = make_c5_weights(seed=6, arch={s: [1008, 256, 192, 160, 1] for s in range(7)}, round_bf16=False)
    ctx = pkg.Context(p, max_atoms=w.n_atoms)
    for s, (ws, bs) in nets.items():
        ctx.ani_mlp_load(s, ws, bs, CELU_ALPHA)
    assert ctx.mlp_kernel() == "fp32"
    e, f = ctx.ani_energy_forces(torch.from_numpy(w.pos).cuda(), torch.from_numpy(sp).cuda(), w.box)
    ctx.check_status()
    we, wf, _ = oracle.energy_forces(p, w.pos, sp, w.box, nets, CELU_ALPHA)
    assert abs(float(e[0]) - we[0]) <= 1e-4 * max(1.0, abs(we[0]))
    _check_forces(f.cpu().numpy().astype(np.float64), wf, what="wide hidden layers")
    ctx.close()


def test_host_call_graph_survives_reallocation_and_other_calls(pkg):
    """ani_energy_forces_host replays a captured CUDA graph from the second call with one key on; a call that makes the
    context reallocate workspace (a periodic box after gas-phase calls), other shapes and a network reload in between
    must not leave a stale graph behind."""
    w = make_workload("C2")
    box_w = make_water_box(216, 18.64, 312, "graph-box")
    nets = make_c5_weights(seed=3, arch={s: [384, 96, 64, 1] for s in range(4)})
    ctx = pkg.Context(w.params, max_atoms=box_w.n_atoms)
    for s, (ws, bs) in nets.items():
        ctx.ani_mlp_load(s, ws, bs, CELU_ALPHA)
    pos, sp = np.ascontiguousarray(w.pos[:1]), np.ascontiguousarray(w.species[:1])
    want_e, want_f, _ = oracle.energy_forces(w.params, pos, sp, None, nets, CELU_ALPHA)

    def check(n_calls):
        for _ in range(n_calls):
            e, f = ctx.ani_energy_forces_host(pos, sp, None)
            assert abs(e[0] - want_e[0]) <= 1e-4 * max(1.0, abs(want_e[0]))
            _check_forces(f.astype(np.float64), want_f, C5_FORCE_TOL, C5_FORCE_MAX_TOL, what="host graph")
    check(4)                                                   # eager, capture, replay, replay
    eb, fb = ctx.ani_energy_forces_host(box_w.pos, box_w.species, box_w.box)      # other key; bin tables are allocated
    wbe, wbf, _ = oracle.energy_forces(box_w.params, box_w.pos, box_w.species, box_w.box, nets, CELU_ALPHA)
    _check_forces(fb.astype(np.float64), wbf, C5_FORCE_TOL, C5_FORCE_MAX_TOL, what="host call, box")
    check(4)
    pos2 = np.ascontiguousarray(w.pos[1:2])                    # same key, new positions: the replay reads the staging buffer
    e2, f2 = ctx.ani_energy_forces_host(pos2, sp, None)
    we2, wf2, _ = oracle.energy_forces(w.params, pos2, sp, None, nets, CELU_ALPHA)
    _check_forces(f2.astype(np.float64), wf2, C5_FORCE_TOL, C5_FORCE_MAX_TOL, what="host graph, new positions")
    nets2 = make_c5_weights(seed=4, arch={s: [384, 96, 64, 1] for s in range(4)})
    for s, (ws, bs) in nets2.items():
        ctx.ani_mlp_load(s, ws, bs, CELU_ALPHA)                # reload: the graph with the old networks is dropped
    want_e, want_f, _ = oracle.energy_forces(w.params, pos, sp, None, nets2, CELU_ALPHA)
    check(3)
    ctx.close()


@pytest.mark.parametrize("flags,skin", [(0, 0.0), (1, 0.0), (0, 0.5), (1, 0.5)])
def test_host_call_over_a_trajectory_in_every_mode(pkg, flags, skin):
    """ani_energy_forces_host (replayed CUDA graph from the second call on) over an 8-frame random walk, default /
    deterministic contexts with and without a Verlet skin (the rebuild decision is taken inside the replayed graph)."""
    from gen import random_walk
    w = make_water_box(216, 18.64, 320, "host-modes")
    nets = make_c5_weights()
    frames = random_walk(w, 8, 0.05, 9)
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms, flags=flags, skin=skin)
    for s, (ws, bs) in nets.items():
        ctx.ani_mlp_load(s, ws, bs, CELU_ALPHA)
    for t, fr in enumerate(frames):
        e, f = ctx.ani_energy_forces_host(np.ascontiguousarray(fr), w.species, w.box)
        if t in (0, 1, 2, 7):
            we, wf, _ = oracle.energy_forces(w.params, fr, w.species, w.box, nets, CELU_ALPHA, use_cells=True)
            assert abs(e[0] - we[0]) <= 1e-4 * max(1.0, abs(we[0]))
            _check_forces(f.astype(np.float64), wf, C5_FORCE_TOL, C5_FORCE_MAX_TOL, what=("host modes", flags, skin, t))
    if skin > 0:
        assert 1 <= ctx.neighbor_builds() < len(frames)
    ctx.close()
