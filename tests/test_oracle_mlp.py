"""Pins for the oracle's per-species network (oracle_mlp)
and the full energy+forces chain -- CPU only.

Checks against things other than the oracle: the 1-layer special case is a dot
product; CELU values from its definition typed with math; the full chain against
torch-CPU fp64 (`torch.nn.functional.celu` + autograd, a library routine); finite
differences of the total energy; zero net force.
"""
import math

import numpy as np
import pytest

import oracle
from gen import ani1x_style_params, make_c1, make_c5_weights, make_ensemble_weights
from gen.workloads import C5_ARCH, CELU_ALPHA


def test_single_linear_layer_is_a_dot_product():
    rng = np.random.default_rng(0)
    x = rng.standard_normal((7, 13))
    w = rng.standard_normal((13, 1))
    b = rng.standard_normal(1)
    e, g = oracle.mlp(x, [w], [b], 0.1)
    np.testing.assert_allclose(e, x @ w[:, 0] + b[0], rtol=1e-14)
    np.testing.assert_allclose(g, np.broadcast_to(w[:, 0], (7, 13)), rtol=1e-15)


def test_celu_values_and_slope():
    # two layers 1 -> 1 -> 1 with identity weights: E = CELU_alpha(x)
    alpha = 0.1
    xs = np.array([-3.0, -0.25, -1e-3, 0.0, 1e-3, 0.7, 5.0]).reshape(-1, 1)
    one, zero = np.ones((1, 1)), np.zeros(1)
    e, g = oracle.mlp(xs, [one, one], [zero, zero], alpha)
    for x, ei, gi in zip(xs[:, 0], e, g[:, 0]):
        want = max(0.0, x) + min(0.0, alpha * (math.exp(x / alpha) - 1.0))
        assert ei == pytest.approx(want, rel=1e-14, abs=1e-18)
        dwant = 1.0 if x > 0 else math.exp(x / alpha)
        assert gi == pytest.approx(dwant, rel=1e-14)
    # slope by central differences
    h = 1e-6
    ep, _ = oracle.mlp(xs + h, [one, one], [zero, zero], alpha, want_grad=False)
    em, _ = oracle.mlp(xs - h, [one, one], [zero, zero], alpha, want_grad=False)
    keep = np.abs(xs[:, 0]) > 1e-5          # CELU' is continuous but kinked in 2nd order at 0
    np.testing.assert_allclose(((ep - em) / (2 * h))[keep], g[keep, 0], rtol=1e-7, atol=1e-9)


@pytest.mark.parametrize("builtin", [False, True])
@pytest.mark.parametrize("s", [0, 3])
def test_full_chain_against_torch(s, builtin):
    import torch
    nets = make_c5_weights()
    ws, bs = nets[s]
    assert [ws[0].shape[0]] + [w.shape[1] for w in ws] == C5_ARCH[s]
    rng = np.random.default_rng(3)
    x = np.abs(rng.standard_normal((11, 384))) * 0.3
    e, g = oracle.mlp(x, ws, bs, CELU_ALPHA)
    xt = torch.tensor(x, requires_grad=True)
    h = xt
    for l, (w, b) in enumerate(zip(ws, bs)):
        h = h @ torch.tensor(w.astype(np.float64)) + torch.tensor(b.astype(np.float64))
        if l < len(ws) - 1:
            if builtin:
                h = torch.nn.functional.celu(h, alpha=CELU_ALPHA)
            else:   # CELU written out from its definition; autograd differentiates it
                h = torch.where(h > 0, h, CELU_ALPHA * (torch.exp(torch.clamp(h, max=0.0) / CELU_ALPHA) - 1.0))
    h[:, 0].sum().backward()
    np.testing.assert_allclose(e, h[:, 0].detach().numpy(), rtol=1e-12, atol=1e-14)
    # torch's built-in celu backward carries a ~1e-8 relative error even in float64 (its
    # 1/alpha is not double precision); the written-out definition agrees to rounding
    tol = 1e-6 if builtin else 1e-11
    np.testing.assert_allclose(g, xt.grad.numpy(), rtol=tol, atol=tol * np.abs(g).max())


def test_weights_recipe():
    nets = make_c5_weights()
    for s, (ws, bs) in nets.items():
        for w in ws:
            # bf16-representable (G14): low 16 bits of the float32 pattern are zero
            assert np.all(w.view(np.uint32) & 0xFFFF == 0)
            # variance 1/fan_in (G13)
            assert w.std() == pytest.approx(w.shape[0] ** -0.5, rel=0.1)


def test_energy_forces_fd_and_net_force():
    w = make_c1()
    p = w.params
    rng = np.random.default_rng(5)
    arch = {s: [384, 24, 16, 1] for s in range(4)}
    nets = make_c5_weights(seed=7, arch=arch)
    e, f, aev = oracle.energy_forces(p, w.pos, w.species, None, nets, CELU_ALPHA)
    assert e.shape == (1,) and f.shape == (1, 24, 3)
    assert np.abs(f[0].sum(axis=0)).max() < 1e-12 * np.abs(f).max()
    coords = [(int(i), int(a)) for i, a in zip(rng.integers(0, 24, 10), rng.integers(0, 3, 10))]
    for (i, a) in coords:
        xp, xm = w.pos.copy(), w.pos.copy()
        xp[0, i, a] = np.float32(w.pos[0, i, a] + 1e-4)
        xm[0, i, a] = np.float32(w.pos[0, i, a] - 1e-4)
        step = float(xp[0, i, a]) - float(xm[0, i, a])
        ep = oracle.energy_forces(p, xp, w.species, None, nets, CELU_ALPHA)[0][0]
        em = oracle.energy_forces(p, xm, w.species, None, nets, CELU_ALPHA)[0][0]
        assert -(ep - em) / step == pytest.approx(f[0, i, a], rel=1e-5, abs=1e-5 * np.abs(f).max())
    # energy is the plain sum over atoms of the species network on that atom's AEV row
    tot = 0.0
    for i in range(24):
        s = int(w.species[0, i])
        tot += oracle.mlp(aev[0, i:i + 1], nets[s][0], nets[s][1], CELU_ALPHA, want_grad=False)[0][0]
    assert e[0] == pytest.approx(tot, rel=1e-13)


def test_ensemble_of_identical_networks_is_one_network_and_fd():
    """PAPER.md:193 (ensemble of eight models): the ensemble result is the mean over the models.
    Pins: eight copies of one network give that network's result; the mean energy of distinct
    networks has the ensemble forces as its negative gradient (central differences); zero net force."""
    w = make_c1()
    p = w.params
    arch = {s: [384, 24, 16, 1] for s in range(4)}
    one = make_c5_weights(seed=7, arch=arch)
    e1, f1, _ = oracle.energy_forces(p, w.pos, w.species, None, one, CELU_ALPHA)
    e8, f8, _ = oracle.energy_forces_ensemble(p, w.pos, w.species, None, [one] * 8, CELU_ALPHA)
    np.testing.assert_allclose(e8, e1, rtol=1e-14)
    np.testing.assert_allclose(f8, f1, rtol=1e-13, atol=1e-13 * np.abs(f1).max())
    models = make_ensemble_weights(3, arch=arch, round_bf16=False)
    e, f, _ = oracle.energy_forces_ensemble(p, w.pos, w.species, None, models, CELU_ALPHA)
    assert abs(e[0] - e1[0]) > 1e-6          # the models really differ
    assert np.abs(f[0].sum(axis=0)).max() < 1e-12 * np.abs(f).max()
    rng = np.random.default_rng(11)
    for i, a in zip(rng.integers(0, 24, 6), rng.integers(0, 3, 6)):
        xp, xm = w.pos.copy(), w.pos.copy()
        xp[0, i, a] = np.float32(w.pos[0, i, a] + 1e-4)
        xm[0, i, a] = np.float32(w.pos[0, i, a] - 1e-4)
        step = float(xp[0, i, a]) - float(xm[0, i, a])
        ep = oracle.energy_forces_ensemble(p, xp, w.species, None, models, CELU_ALPHA)[0][0]
        em = oracle.energy_forces_ensemble(p, xm, w.species, None, models, CELU_ALPHA)[0][0]
        assert -(ep - em) / step == pytest.approx(f[0, i, a], rel=1e-5, abs=1e-5 * np.abs(f).max())
