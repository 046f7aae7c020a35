"""Seeded sweep over the parameter space of the library against the oracle: species counts 1..8, both angular splits,
several zeta, both cos_scale, gas phase / cell-list boxes / small cells / triclinic cells, batches, padding atoms,
default / deterministic / Verlet-skin contexts.  Pair sets bit-exact, AEV and forces at north_star's tolerances."""
import contextlib
import dataclasses

import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
from gen import ani1x_style_params, ani2x_shaped_params, make_periodic_cell

from test_gpu_parity import AEV_TOL, _check_forces

pytestmark = pytest.mark.gpu

CELLS = [None, None, (12.0, 13.0, 14.5), (17.0, 16.5, 18.0), (16.0, 22.0, 27.5),
         [[14.0, 0.0, 0.0], [3.0, 13.0, 0.0], [-2.0, 4.0, 12.5]]]


@pytest.mark.parametrize("seed", range(16))
def test_random_configuration(seed):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2310_03121_b200 as pkg
    rng = np.random.default_rng(1000 + seed)
    S = int(rng.integers(1, 9))
    base = ani2x_shaped_params(num_species=S) if seed % 3 == 2 else ani1x_style_params(num_species=S)
    p = dataclasses.replace(base, zeta=np.float32(rng.choice([1.0, 2.0, 14.1, 32.0])),
                            cos_scale=np.float32(rng.choice([1.0, 0.95])))
    cell = CELLS[seed % len(CELLS)]
    tri = cell is not None and np.ndim(cell) == 2
    vol = 14.0 ** 3 if cell is None else (np.prod(cell) if not tri else 14.0 * 13.0 * 12.5)
    n = int(rng.integers(1, max(2, int(0.09 * vol))))
    batch = int(rng.integers(1, 4))
    ws = [make_periodic_cell(n, cell, 5000 + 10 * seed + b, params=p) for b in range(batch)]
    pos = np.stack([w.pos[0] for w in ws])
    sp = np.stack([w.species[0] for w in ws])
    if n > 3:                                            # padding atoms (G12)
        sp[:, rng.integers(0, n, size=2)] = -1
    box = ws[0].box
    g = rng.standard_normal((batch, n, p.aev_length)).astype(np.float32)
    flags = (pkg.AEV_FLAG_TRICLINIC if tri else 0) | (pkg.AEV_FLAG_DETERMINISTIC if seed % 4 == 1 else 0)
    skin = 0.4 if (seed % 5 == 3 and (cell is None or min(np.ravel(cell)[[0, 4, 8]] if tri else cell) >= 2 * 5.6)) else 0.0
    ctx = pkg.Context(p, max_atoms=n, max_batch=batch, flags=flags, skin=skin)
    pos_d, sp_d = torch.from_numpy(pos).cuda(), torch.from_numpy(sp).cuda()
    scope = oracle.lattice(box) if tri else contextlib.nullcontext()
    obox = None if tri else box
    for rep in range(2 if skin > 0 else 1):              # second call: the reuse path of the skin mode
        aev = ctx.aev_forward(pos_d, sp_d, box)
        f = ctx.aev_backward(torch.from_numpy(g).cuda())
        ctx.check_status()
        with scope:
            for which, rc in ((0, p.rcr), (1, p.rca)):
                got = ctx.aev_export_pairs(which, cap=batch * n * 64 + 8)
                want = [oracle.pairs(pos[b], sp[b], obox, float(rc), "brute").astype(np.int64) + b * n for b in range(batch)]
                np.testing.assert_array_equal(got, np.concatenate(want).astype(np.int32).reshape(-1, 2))
            want_a = oracle.aev_forward(p, pos, sp, obox)
            want_f = oracle.aev_backward(p, pos, sp, obox, g)
        scale = max(np.abs(want_a).max(), 1e-30)
        assert np.abs(aev.cpu().numpy() - want_a).max() <= AEV_TOL * scale, (seed, S, n, batch, cell)
        assert not np.any(aev.cpu().numpy()[sp < 0])
        if np.abs(want_f).max() > 0:
            _check_forces(f.cpu().numpy(), want_f, what=("fuzz", seed, S, n, batch, float(p.zeta), skin, flags))
        else:
            assert not np.any(f.cpu().numpy())
    ctx.close()


def _in_tensor_core_envelope(dims):
    """include/aev.h, ani_mlp_load: 1-3 hidden layers, widths multiples of 16 in 16..160; every pair of consecutive hidden
    widths (a, b) with ceil(a/64)*b <= 384 and ceil(b/64)*a <= 384 (the operand of that layer, forward and transposed,
    fits one 48 KB shared-memory buffer; hi + lo operands use two); TMEM: the hidden widths sum to <= 512 columns and
    the backward accumulator of layer l fits behind z_1..z_l."""
    h = list(dims[1:-1])
    if not 1 <= len(h) <= 3 or any(x % 16 or not 16 <= x <= 160 for x in h) or sum(h) > 512:
        return False
    for a, b in zip(h[:-1], h[1:]):
        if -(-a // 64) * b > 384 or -(-b // 64) * a > 384:
            return False
    return all(sum(h[:l + 1]) + h[l] <= 512 for l in range(len(h) - 1))


@pytest.mark.parametrize("seed", range(8))
def test_random_network_shapes(seed):
    """Random per-species architectures inside the tensor-core envelope (1-3 hidden layers, widths 16..160), ensembles
    of 1-3 models, bf16-representable or fp32 weights, on a small periodic cell or a gas-phase cluster."""
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2310_03121_b200 as pkg
    from gen import make_c5_weights
    from gen.workloads import CELU_ALPHA
    from test_gpu_parity import C5_FORCE_MAX_TOL, C5_FORCE_TOL
    rng = np.random.default_rng(2000 + seed)
    S = int(rng.integers(1, 5))
    p = ani1x_style_params(num_species=S)
    cell = [None, (12.0, 13.0, 14.5), (17.0, 16.5, 18.0)][seed % 3]
    n = int(rng.integers(40, 220))
    w = make_periodic_cell(n, cell, 7000 + seed, params=p)
    L = p.aev_length
    arch = {}
    for s in range(S):
        nh = int(rng.integers(1, 4))
        arch[s] = [L] + [int(16 * rng.integers(1, 11)) for _ in range(nh)] + [1]
    n_models = int(rng.integers(1, 4))
    exact = bool(seed % 2)
    models = [make_c5_weights(seed=40 + seed + 10 * m, arch=arch, round_bf16=exact) for m in range(n_models)]
    ctx = pkg.Context(p, max_atoms=n)
    ctx.ani_mlp_set_ensemble(n_models)
    for m, nets in enumerate(models):
        for s, (ws, bs) in nets.items():
            ctx.ani_mlp_load_model(m, s, ws, bs, CELU_ALPHA)
    # which kernel runs is part of the contract: the rule ani_mlp_load documents in include/aev.h, restated
    want_kernel = "tcgen05" if all(_in_tensor_core_envelope(d) for d in arch.values()) else "fp32"
    assert ctx.mlp_kernel() == want_kernel, arch
    e, f = ctx.ani_energy_forces(torch.from_numpy(w.pos).cuda(), torch.from_numpy(w.species).cuda(), w.box)
    ctx.check_status()
    we, wf, _ = oracle.energy_forces_ensemble(p, w.pos, w.species, w.box, models, CELU_ALPHA)
    assert abs(float(e[0]) - we[0]) <= 1e-4 * max(1.0, abs(we[0])), (arch, n_models)
    _check_forces(f.cpu().numpy().astype(np.float64), wf, C5_FORCE_TOL, C5_FORCE_MAX_TOL, what=("net fuzz", seed, arch, n_models, exact))
    ctx.close()
