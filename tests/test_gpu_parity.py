"""GPU parity tests: the CUDA path (through the C ABI) against the fp64 oracle on the same
seeded inputs (BASELINE.json:north_star tolerances, written out below).

  neighbour pair sets ........ bit-exact (sorted (i<j) arrays equal)
  AEV ........................ max-abs error <= 1e-5 * max|AEV|
  forces (fp32) .............. relative RMS error <= 1e-4, and every component within
                               FORCE_MAX_TOL * max|F| (an error confined to a few atoms cannot hide in the norm)
  C5 energy+forces ........... forces relative RMS <= 1e-3 (bf16-split GEMMs, fp32 accumulate)
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
from gen import ani1x_style_params, make_c5_weights, make_workload
from gen.workloads import CELU_ALPHA

pytestmark = pytest.mark.gpu

AEV_TOL = 1e-5       # max-abs relative to max|AEV|          (north_star)
FORCE_TOL = 1e-4     # relative RMS, fp32                     (north_star)
C5_FORCE_TOL = 1e-3  # relative RMS with bf16 GEMMs           (BASELINE.json:configs[4])
# per-component bound relative to max|F| (DESIGN.md section 6 lists the measured values: fp32 gives ~1e-6
# on C1-C4; the bound leaves a decade of headroom and is still 10x below what one wrong atom would produce)
FORCE_MAX_TOL = 2e-5
C5_FORCE_MAX_TOL = 2e-4


@pytest.fixture(scope="module")
def pkg():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2310_03121_b200 as p
    return p


def _dev(w):
    pos = torch.from_numpy(w.pos).cuda()
    sp = torch.from_numpy(w.species).cuda()
    g = torch.from_numpy(w.grad_aev).cuda()
    return pos, sp, g


def _rel_rms(a, b):
    return float(np.sqrt(((a - b) ** 2).sum() / (b ** 2).sum()))


def _check_forces(f, want, rms_tol=FORCE_TOL, max_tol=FORCE_MAX_TOL, what=""):
    """north_star's relative-RMS bound plus a per-component max-abs bound relative to max|F|."""
    f = np.asarray(f, dtype=np.float64)
    rms = _rel_rms(f, want)
    assert rms <= rms_tol, (what, "rel rms", rms)
    worst = float(np.abs(f - want).max() / np.abs(want).max())
    print("PARITY forces %s rel_rms %.3e max_abs_over_maxF %.3e" % (what, rms, worst))
    assert worst <= max_tol, (what, "max abs / max|F|", worst)
    return rms, worst


def _oracle_pairs(w, rc):
    uc = "cell" if (w.box is not None and w.n_atoms > 6000) else "brute"
    out = []
    for b in range(w.batch):
        p = oracle.pairs(w.pos[b], w.species[b], w.box, rc, uc)
        out.append(p.astype(np.int64) + b * w.n_atoms)
    return np.concatenate(out).astype(np.int32)


@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4"])
def test_pair_sets_bit_exact(pkg, name):
    w = make_workload(name)
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms, max_batch=w.batch)
    pos, sp, _ = _dev(w)
    ctx.aev_neighbors(pos, sp, w.box)
    ctx.check_status()
    for which, rc in ((0, w.params.rcr), (1, w.params.rca)):
        got = ctx.aev_export_pairs(which, cap=w.batch * w.n_atoms * 40)
        want = _oracle_pairs(w, float(rc))
        assert got.shape == want.shape, (name, which, got.shape, want.shape)
        np.testing.assert_array_equal(got, want)
    ctx.close()


@pytest.mark.parametrize("name,cos_scale", [("C1", 1.0), ("C1", 0.95), ("C2", 1.0), ("C2", 0.95),
                                            ("C3", 1.0), ("C3", 0.95), ("C4", 1.0)])
def test_aev_and_forces_match_oracle(pkg, name, cos_scale):
    w = make_workload(name, cos_scale)
    uc = w.box is not None
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms, max_batch=w.batch)
    pos, sp, g = _dev(w)
    aev = ctx.aev_forward(pos, sp, w.box)
    forces = ctx.aev_backward(g)
    ctx.check_status()
    aev = aev.cpu().numpy().astype(np.float64)
    forces = forces.cpu().numpy().astype(np.float64)
    want_aev = oracle.aev_forward(w.params, w.pos, w.species, w.box, use_cells=uc)
    want_f = oracle.aev_backward(w.params, w.pos, w.species, w.box, w.grad_aev, use_cells=uc)
    err = np.abs(aev - want_aev).max() / np.abs(want_aev).max()
    assert err <= AEV_TOL, (name, cos_scale, err)
    _check_forces(forces, want_f, what=(name, cos_scale))
    # zero net force per system (north_star), relative to the force scale
    net = np.abs(forces.sum(axis=1)).max()
    assert net <= 1e-3 * np.sqrt((forces ** 2).mean()) * np.sqrt(w.n_atoms), net
    ctx.close()


def test_run_to_run_stability_in_the_default_mode(pkg):
    """Default mode: the order inside a cell follows k_bin's atomics and forces are accumulated with fp32
    REDs, so two runs agree to rounding (bit-identical results: AEV_FLAG_DETERMINISTIC, tests/test_gpu_round2.py)."""
    w = make_workload("C3")
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms)
    pos, sp, g = _dev(w)
    a1 = ctx.aev_forward(pos, sp, w.box).clone()
    f1 = ctx.aev_backward(g).clone()
    a2 = ctx.aev_forward(pos, sp, w.box)
    f2 = ctx.aev_backward(g)
    ctx.check_status()
    assert float((a1 - a2).abs().max()) <= 1e-6 * float(a1.abs().max())
    assert float((f1 - f2).abs().max()) <= 1e-5 * float(f1.abs().max())
    ctx.close()


def test_atoms_outside_the_box_and_permutation(pkg):
    """Periodic images and atom order do not change the AEV (rows permute)."""
    w = make_workload("C3")
    rng = np.random.default_rng(7)
    shift = rng.integers(-2, 3, size=(w.n_atoms, 3)).astype(np.float32) * w.box[None, :]
    pos2 = (w.pos[0] + shift).astype(np.float32)
    perm = rng.permutation(w.n_atoms)
    pos2, sp2 = pos2[perm][None], w.species[0][perm][None]
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms)
    a1 = ctx.aev_forward(torch.from_numpy(w.pos).cuda(), torch.from_numpy(w.species).cuda(), w.box).cpu().numpy()
    a2 = ctx.aev_forward(torch.from_numpy(pos2).cuda(), torch.from_numpy(sp2).cuda(), w.box).cpu().numpy()
    ctx.check_status()
    # float32 image shifts of up to 2 box lengths perturb coordinates by ~1e-5 A
    assert np.abs(a2[0] - a1[0][perm]).max() <= 2e-3 * np.abs(a1).max()
    want = oracle.aev_forward(w.params, pos2, sp2, w.box, use_cells=True)
    assert np.abs(a2 - want).max() <= AEV_TOL * np.abs(want).max()
    ctx.close()


def test_padding_atoms_and_tiny_systems(pkg):
    p = ani1x_style_params()
    w = make_workload("C1")
    # two copies of C1, the second padded with 8 extra species -1 atoms placed on top of real ones
    n = w.n_atoms + 8
    pos = np.zeros((2, n, 3), dtype=np.float32)
    sp = -np.ones((2, n), dtype=np.int32)
    pos[0, :24], sp[0, :24] = w.pos[0], w.species[0]
    pos[1, 8:], sp[1, 8:] = w.pos[0], w.species[0]
    pos[1, :8] = w.pos[0, :8] + 0.3
    g = np.random.default_rng(0).standard_normal((2, n, p.aev_length)).astype(np.float32)
    ctx = pkg.Context(p, max_atoms=n, max_batch=2)
    aev = ctx.aev_forward(torch.from_numpy(pos).cuda(), torch.from_numpy(sp).cuda(), None)
    f = ctx.aev_backward(torch.from_numpy(g).cuda())
    ctx.check_status()
    aev, f = aev.cpu().numpy(), f.cpu().numpy()
    want = oracle.aev_forward(p, pos, sp, None)
    want_f = oracle.aev_backward(p, pos, sp, None, g)
    assert np.abs(aev - want).max() <= AEV_TOL * np.abs(want).max()
    _check_forces(f, want_f)
    assert np.all(aev[0, 24:] == 0) and np.all(aev[1, :8] == 0)
    assert np.all(f[0, 24:] == 0) and np.all(f[1, :8] == 0)
    # one atom, two atoms: empty / single-pair environments
    for m in (1, 2):
        pos1 = np.array([[[0, 0, 0], [1.0, 0, 0]][:m]], dtype=np.float32)
        sp1 = np.zeros((1, m), dtype=np.int32)
        a = ctx.aev_forward(torch.from_numpy(pos1).cuda(), torch.from_numpy(sp1).cuda(), None)
        ff = ctx.aev_backward(torch.ones_like(a))
        ctx.check_status()
        wa = oracle.aev_forward(p, pos1, sp1, None)
        wf = oracle.aev_backward(p, pos1, sp1, None, np.ones_like(wa, dtype=np.float32))
        assert np.abs(a.cpu().numpy() - wa).max() <= 1e-6
        assert np.abs(ff.cpu().numpy() - wf).max() <= 1e-5
    ctx.close()


def test_golden_one_water(pkg, golden):
    """The closed-form pin of SURVEY.md 8(c) (tests/golden/one_water_c100.txt) through the GPU path."""
    import math
    gold = golden("one_water_c100.txt")
    a = math.radians(52.26)
    pos = np.array([[[0, 0, 0], [0.9572 * math.sin(a), 0, 0.9572 * math.cos(a)],
                     [-0.9572 * math.sin(a), 0, 0.9572 * math.cos(a)]]], dtype=np.float32)
    sp = np.array([[3, 0, 0]], dtype=np.int32)
    p = ani1x_style_params()
    ctx = pkg.Context(p, max_atoms=3)
    aev = ctx.aev_forward(torch.from_numpy(pos).cuda(), torch.from_numpy(sp).cuda(), None)
    f = ctx.aev_backward(torch.ones_like(aev)).cpu().numpy()
    aev = aev.cpu().numpy()
    assert aev.sum() == pytest.approx(gold["energy_g1"][0], rel=2e-6)
    np.testing.assert_allclose(aev[0, 0, 64:72], gold["centreO_HH_row0"], rtol=2e-5, atol=1e-9)
    np.testing.assert_allclose(aev[0, 1, 64 + 3 * 32:64 + 3 * 32 + 8], gold["centreH1_HO_row0"], rtol=2e-5, atol=1e-9)
    for row, key in enumerate(("grad_O", "grad_H1", "grad_H2")):       # forces = -grad
        np.testing.assert_allclose(f[0, row], -np.array(gold[key]), rtol=2e-5, atol=2e-6)
    ctx.close()


def test_errors(pkg):
    p = ani1x_style_params()
    w = make_workload("C1")
    ctx = pkg.Context(p, max_atoms=64, max_batch=1)
    pos, sp, g = _dev(w)
    with pytest.raises(pkg.AevError) as e:          # backward before forward
        ctx.aev_backward(g)
    assert e.value.code == -4
    with pytest.raises(pkg.AevError) as e:          # box edge < 2*rcr
        ctx.aev_forward(pos, sp, np.array([9.0, 20.0, 20.0], dtype=np.float32))
    assert e.value.code == -2
    with pytest.raises(pkg.AevError) as e:          # more atoms than the context was sized for
        big = torch.zeros((1, 65, 3), device="cuda")
        ctx.aev_forward(big, torch.zeros((1, 65), dtype=torch.int32, device="cuda"), None)
    assert e.value.code == -1
    ctx.close()
    # capacity overflow is detected on the device and surfaced by aev_status
    ctx = pkg.Context(p, max_atoms=24, max_radial_nbrs=16, max_angular_nbrs=4)
    ctx.aev_forward(pos, sp, None)
    assert ctx.aev_status() == -3
    ctx.close()


def test_host_entry_point_matches_device_entry_point(pkg):
    w = make_workload("C2")
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms, max_batch=w.batch)
    pos, sp, g = _dev(w)
    a1 = ctx.aev_forward(pos, sp, None).cpu().numpy()
    f1 = ctx.aev_backward(g).cpu().numpy()
    a2, f2 = ctx.aev_forward_backward_host(w.pos, w.species, None, w.grad_aev)
    np.testing.assert_allclose(a1, a2, rtol=0, atol=1e-6 * np.abs(a1).max())   # order inside a cell
    np.testing.assert_allclose(f1, f2, rtol=0, atol=1e-5 * np.abs(f1).max())   # RED order
    ctx.close()


def test_c5_energy_and_forces(pkg):
    w = make_workload("C5")
    nets = make_c5_weights()
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms)
    for s, (ws, bs) in nets.items():
        ctx.ani_mlp_load(s, ws, bs, CELU_ALPHA)
    pos, sp, _ = _dev(w)
    e, f = ctx.ani_energy_forces(pos, sp, w.box)
    ctx.check_status()
    e, f = e.cpu().numpy(), f.cpu().numpy().astype(np.float64)
    we, wf, _ = oracle.energy_forces(w.params, w.pos, w.species, w.box, nets, CELU_ALPHA, use_cells=True)
    assert abs(e[0] - we[0]) <= 1e-4 * max(1.0, abs(we[0]))
    _check_forces(f, wf, C5_FORCE_TOL, C5_FORCE_MAX_TOL)
    e2, f2 = ctx.ani_energy_forces_host(w.pos, w.species, w.box)
    assert abs(e2[0] - e[0]) <= 1e-6 * max(1.0, abs(e[0]))      # order inside a cell, RED order
    np.testing.assert_allclose(f2, f, rtol=0, atol=1e-5 * np.abs(f).max())   # RED order
    ctx.close()


def test_weights_that_are_not_bf16_are_not_rounded(pkg):
    """Weights that are not bf16-representable must not be rounded: the tensor-core kernel takes them as
    hi + lo bf16 operands; a rounded model would miss the tolerance by two orders."""
    w = make_workload("C5")
    nets = make_c5_weights()
    rng = np.random.default_rng(7)
    nets = {s: ([(x * (1.0 + 2.0 ** -11 * rng.standard_normal(x.shape))).astype(np.float32) for x in ws], bs)
            for s, (ws, bs) in nets.items()}
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms)
    for s, (ws, bs) in nets.items():
        ctx.ani_mlp_load(s, ws, bs, CELU_ALPHA)
    pos, sp, _ = _dev(w)
    e, f = ctx.ani_energy_forces(pos, sp, w.box)
    ctx.check_status()
    e, f = e.cpu().numpy(), f.cpu().numpy().astype(np.float64)
    we, wf, _ = oracle.energy_forces(w.params, w.pos, w.species, w.box, nets, CELU_ALPHA, use_cells=True)
    assert abs(e[0] - we[0]) <= 1e-4 * max(1.0, abs(we[0]))
    _check_forces(f, wf, C5_FORCE_TOL, C5_FORCE_MAX_TOL, what="perturbed weights")
    ctx.close()


def test_mlp_tensor_core_path_other_depths(pkg):
    """One and two hidden layers, widths that are not powers of two (tcgen05 N = 160, 96, 48)."""
    w = make_workload("C5")
    nets = make_c5_weights(seed=3, arch={0: [384, 96, 48, 1], 3: [384, 160, 1]})
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms)
    for s, (ws, bs) in nets.items():
        ctx.ani_mlp_load(s, ws, bs, CELU_ALPHA)
    pos, sp, _ = _dev(w)
    e, f = ctx.ani_energy_forces(pos, sp, w.box)
    ctx.check_status()
    e, f = e.cpu().numpy(), f.cpu().numpy().astype(np.float64)
    we, wf, _ = oracle.energy_forces(w.params, w.pos, w.species, w.box, nets, CELU_ALPHA, use_cells=True)
    assert abs(e[0] - we[0]) <= 1e-4 * max(1.0, abs(we[0]))
    _check_forces(f, wf, C5_FORCE_TOL, C5_FORCE_MAX_TOL)
    ctx.close()


def test_large_gas_phase_cluster_uses_the_unstaged_scan(pkg):
    """1,200 atoms without a box: one cell whose 1,200 candidates exceed the shared-memory stage,
    so k_nbr takes its global-memory ballot path; pair sets stay bit-exact."""
    from gen import make_water_box
    wb = make_water_box(400, 24.0, 910, "cluster")
    pos, sp, g = _dev(wb)
    ctx = pkg.Context(wb.params, max_atoms=wb.n_atoms)
    aev = ctx.aev_forward(pos, sp, None)
    forces = ctx.aev_backward(g)
    ctx.check_status()
    for which, rc in ((0, wb.params.rcr), (1, wb.params.rca)):
        got = ctx.aev_export_pairs(which, cap=wb.n_atoms * 64)
        want = oracle.pairs(wb.pos[0], wb.species[0], None, float(rc), "brute").astype(np.int32)
        np.testing.assert_array_equal(got, want)
    want_aev = oracle.aev_forward(wb.params, wb.pos, wb.species, None, use_cells=False)
    want_f = oracle.aev_backward(wb.params, wb.pos, wb.species, None, wb.grad_aev, use_cells=False)
    a = aev.cpu().numpy().astype(np.float64)
    assert np.abs(a - want_aev).max() / np.abs(want_aev).max() <= AEV_TOL
    _check_forces(forces.cpu().numpy().astype(np.float64), want_f)
    ctx.close()


@pytest.mark.gpu
def test_seven_species_ani2x_shape(pkg):
    """S = 7 (ANI-2x-shaped AEV, L = 7*16 + 28*32 = 1008): the neighbour kernel's
    64-bit packed species fields and 28 species-pair blocks, gas phase and periodic."""
    p7 = ani1x_style_params(num_species=7)
    assert p7.aev_length == 1008
    rng = np.random.default_rng(77)
    for name in ("C1", "C3"):
        w = make_workload(name)
        sp = rng.integers(0, 7, size=w.species.shape).astype(np.int32)
        g = rng.standard_normal((w.batch, w.n_atoms, 1008)).astype(np.float32)
        ctx = pkg.Context(p7, max_atoms=w.n_atoms, max_batch=w.batch)
        pos_d, sp_d = torch.from_numpy(w.pos).cuda(), torch.from_numpy(sp).cuda()
        aev = ctx.aev_forward(pos_d, sp_d, w.box)
        f = ctx.aev_backward(torch.from_numpy(g).cuda())
        ctx.check_status()
        for which, rc in ((0, p7.rcr), (1, p7.rca)):
            got = ctx.aev_export_pairs(which, cap=w.n_atoms * 64)
            want = oracle.pairs(w.pos[0], sp[0], w.box, float(rc), "brute")
            np.testing.assert_array_equal(got, want.astype(np.int32))
        want_a = oracle.aev_forward(p7, w.pos, sp, w.box, use_cells=w.box is not None)
        want_f = oracle.aev_backward(p7, w.pos, sp, w.box, g, use_cells=w.box is not None)
        assert np.abs(aev.cpu().numpy() - want_a).max() <= AEV_TOL * np.abs(want_a).max()
        _check_forces(f.cpu().numpy().astype(np.float64), want_f)
        ctx.close()


@pytest.mark.gpu
def test_large_box_is_periodic_replication(pkg):
    """288,000 atoms: C3's box replicated 4x4x4 (L = 142 A, 27^3 cells x 4 species = 78,732 bins). Every atom
    of a replica has the environment of its original, so the first replica's rows must equal the 4,500-atom
    oracle result (coordinates shifted by up to 3 box lengths perturb fp32 positions by ~1e-5 A)."""
    w = make_workload("C3")
    L0 = np.asarray(w.box, dtype=np.float64)
    reps = 4
    shifts = np.array([[i, j, k] for i in range(reps) for j in range(reps) for k in range(reps)], dtype=np.float64)
    pos = (w.pos[0].astype(np.float64)[None] + (shifts * L0)[:, None, :]).reshape(1, -1, 3).astype(np.float32)
    sp = np.tile(w.species[0], reps ** 3)[None].astype(np.int32)
    box = (L0 * reps).astype(np.float32)
    n = pos.shape[1]
    ctx = pkg.Context(w.params, max_atoms=n)
    aev = ctx.aev_forward(torch.from_numpy(pos).cuda(), torch.from_numpy(sp).cuda(), box)
    g = torch.zeros_like(aev)
    g[0, :w.n_atoms] = torch.from_numpy(w.grad_aev[0]).cuda()
    f = ctx.aev_backward(g)
    ctx.check_status()
    counts = ctx.aev_export_counts(1, n).cpu().numpy().reshape(n, 2)
    a0 = aev[0, :w.n_atoms].cpu().numpy().astype(np.float64)
    want = oracle.aev_forward(w.params, w.pos, w.species, w.box, use_cells=True)[0]
    assert np.abs(a0 - want).max() <= 2e-3 * np.abs(want).max()
    # all 64 replicas have identical neighbour counts
    c = counts.reshape(reps ** 3, w.n_atoms, 2)
    assert np.all(c == c[0][None])
    # forces: upstream gradient only on the first replica's rows; total force is zero
    ff = f[0].cpu().numpy().astype(np.float64)
    assert np.abs(ff.sum(axis=0)).max() <= 1e-3 * np.abs(ff).max()
    ctx.close()


@pytest.mark.gpu
def test_wide_capacity_takes_the_ballot_path_of_the_staged_scan(pkg):
    """max_radial_nbrs = 256 does not fit the 8-bit packed slot fields: k_nbr compacts with ballots from the
    staged stencil instead; results must not change."""
    w = make_workload("C3")
    pos, sp, g = _dev(w)
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms, max_radial_nbrs=256)
    aev = ctx.aev_forward(pos, sp, w.box)
    f = ctx.aev_backward(g)
    ctx.check_status()
    for which, rc in ((0, w.params.rcr), (1, w.params.rca)):
        got = ctx.aev_export_pairs(which, cap=w.n_atoms * 40)
        np.testing.assert_array_equal(got, _oracle_pairs(w, float(rc)))
    want_a = oracle.aev_forward(w.params, w.pos, w.species, w.box, use_cells=True)
    want_f = oracle.aev_backward(w.params, w.pos, w.species, w.box, w.grad_aev, use_cells=True)
    assert np.abs(aev.cpu().numpy() - want_a).max() <= AEV_TOL * np.abs(want_a).max()
    _check_forces(f.cpu().numpy().astype(np.float64), want_f)
    ctx.close()


@pytest.mark.gpu
def test_cuda_graph_replay_with_new_positions(pkg):
    """One evaluation captured in a CUDA graph and replayed after the positions changed in place (the MD-loop
    calling pattern): no host-side state may be baked into the capture."""
    w = make_workload("C2")
    pos, sp, g = _dev(w)
    ctx = pkg.Context(w.params, max_atoms=w.n_atoms, max_batch=w.batch)
    aev = torch.empty_like(g)
    f = torch.empty((w.batch, w.n_atoms, 3), dtype=torch.float32, device="cuda")

    def step():
        ctx.aev_forward(pos, sp, w.box, aev_out=aev)
        ctx.aev_backward(g, forces_out=f)

    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        step()
    torch.cuda.current_stream().wait_stream(side)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        step()
    # conformers in reverse order, written into the captured buffers
    pos2 = np.ascontiguousarray(w.pos[::-1])
    pos.copy_(torch.from_numpy(pos2).cuda())
    for _ in range(3):
        graph.replay()
    torch.cuda.synchronize()
    ctx.check_status()
    want_a = oracle.aev_forward(w.params, pos2, w.species, None)
    want_f = oracle.aev_backward(w.params, pos2, w.species, None, w.grad_aev)
    assert np.abs(aev.cpu().numpy() - want_a).max() <= AEV_TOL * np.abs(want_a).max()
    _check_forces(f.cpu().numpy().astype(np.float64), want_f)
    del graph
    ctx.close()


@pytest.mark.gpu
@pytest.mark.parametrize("zeta", [8.0, 16.0, 14.1, 1.0, 3.5])
def test_other_zeta(pkg, zeta):
    """zeta != 32: powers of two take the run-time squaring-chain instantiations of k_aev / k_backward, any other
    value (14.1: the exponent the advisor recalls for published ANI-2x parameters) the exp2(zeta log2 b) ones."""
    import dataclasses
    w = make_workload("C2")
    p = dataclasses.replace(w.params, zeta=np.float32(zeta))
    pos, sp, g = _dev(w)
    ctx = pkg.Context(p, max_atoms=w.n_atoms, max_batch=w.batch)
    aev = ctx.aev_forward(pos, sp, w.box)
    f = ctx.aev_backward(g)
    ctx.check_status()
    want_a = oracle.aev_forward(p, w.pos, w.species, None)
    want_f = oracle.aev_backward(p, w.pos, w.species, None, w.grad_aev)
    assert np.abs(aev.cpu().numpy() - want_a).max() <= AEV_TOL * np.abs(want_a).max()
    _check_forces(f.cpu().numpy().astype(np.float64), want_f)
    ctx.close()
