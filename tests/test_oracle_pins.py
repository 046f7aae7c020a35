"""Pins for the fp64 oracle (oracle/aev_oracle.c) -- CPU only.

Each test checks the oracle against something other than itself: closed-form values
fixed before the oracle existed (tests/golden/), expressions
evaluated here with `math` for the few terms a 2-/3-atom system has, invariances,
finite differences, and an independently written torch-CPU fp64 autograd definition.
"""
import math

import numpy as np
import pytest

import oracle
from gen import ani1x_style_params, make_c1, make_c3, make_water_box

from conftest import read_golden

P100 = ani1x_style_params(1.0)
P095 = ani1x_style_params(0.95)
# exact-decimal (float64) parameters: what the tests/golden fixtures were computed with
E100 = ani1x_style_params(1.0, dtype=np.float64)
E095 = ani1x_style_params(0.95, dtype=np.float64)
H, Cc, N, O = 0, 1, 2, 3


def _water():
    a = math.radians(52.26)
    return np.array([[0.0, 0.0, 0.0],
                     [+0.9572 * math.sin(a), 0.0, 0.9572 * math.cos(a)],
                     [-0.9572 * math.sin(a), 0.0, 0.9572 * math.cos(a)]], dtype=np.float32)


def _energy(p, pos, species, box, g, use_cells=False):
    return float((oracle.aev_forward(p, pos, species, box, use_cells) * g).sum())


def _fd_forces(p, pos, species, box, g, coords, h=1e-4, use_cells=False):
    """Central differences on float64-perturbed positions are impossible through the
    float32 API, so perturb in float32 and use the ACTUAL step taken."""
    out = []
    for (i, a) in coords:
        xp = pos.copy(); xm = pos.copy()
        xp[0, i, a] = np.float32(pos[0, i, a] + h)
        xm[0, i, a] = np.float32(pos[0, i, a] - h)
        step = float(xp[0, i, a]) - float(xm[0, i, a])
        out.append(-(_energy(p, xp, species, box, g, use_cells)
                     - _energy(p, xm, species, box, g, use_cells)) / step)
    return np.array(out)


# ----------------------------------------------------------------------------- closed forms
def test_two_atoms_closed_form():
    gold = read_golden("two_atoms.txt")
    pos = np.array([[[0, 0, 0], [1, 0, 0]]], dtype=np.float32)
    sp = np.array([[H, H]], dtype=np.int32)
    aev = oracle.aev_forward(E100, pos, sp, None)
    assert aev.shape == (1, 2, 384)
    np.testing.assert_allclose(aev[0, 0, :4], gold["aev0_radial_first4"], rtol=1e-11)
    g = np.ones_like(aev, dtype=np.float32)
    assert aev.sum() == pytest.approx(gold["energy_g1"][0], rel=1e-11)
    f = oracle.aev_backward(E100, pos, sp, None, g)
    dEdr = gold["dE_dr"][0]
    np.testing.assert_allclose(f[0, 1], [-dEdr, 0, 0], rtol=1e-10, atol=1e-15)
    np.testing.assert_allclose(f[0, 0], [+dEdr, 0, 0], rtol=1e-10, atol=1e-15)
    # float32 parameters (what every workload uses, G9) move the values by ~1e-7 relative
    aev = oracle.aev_forward(P100, pos, sp, None)
    np.testing.assert_allclose(aev[0, 0, :4], gold["aev0_radial_first4"], rtol=1e-6)
    # the same numbers from the formula, typed here with math (float32 shifts promoted)
    fc = 0.5 * math.cos(math.pi * 1.0 / float(np.float32(5.2))) + 0.5
    for m in range(16):
        want = 0.25 * math.exp(-16.0 * (1.0 - float(P100.shf_r[m])) ** 2) * fc
        assert aev[0, 0, m] == pytest.approx(want, rel=1e-13, abs=1e-300)
    assert np.all(aev[0, :, 16:] == 0.0)          # no C/N/O neighbours, no triplets
    np.testing.assert_array_equal(aev[0, 0], aev[0, 1])


def test_three_atoms_angular_block_and_slot_order():
    gold = read_golden("three_atoms.txt")
    pos = np.array([[[0, 0, 0], [1, 0, 0], [0, 1, 0]]], dtype=np.float32)
    sp = np.array([[O, H, H]], dtype=np.int32)
    for p in (E100, E095, P100, P095):
        exact = p.shf_r.dtype == np.float64
        aev = oracle.aev_forward(p, pos, sp, None)
        ang = aev[0, 0, 64:].reshape(10, 4, 8)
        np.testing.assert_allclose(ang[0, 0], gold["centreO_HH_row0"], rtol=2e-9 if exact else 5e-6)
        # only block p(H,H)=0 is populated for the centre O (one unordered triplet, G1/G4)
        assert np.all(ang[1:] == 0.0)
        # formula typed with math for every (a,z) of that block
        fc = 0.5 * math.cos(math.pi / float(p.rca)) + 0.5
        for a in range(4):
            for z in range(8):
                want = (2.0 * ((1 + math.cos(math.pi / 2 - float(p.shf_z[z]))) / 2) ** 32
                        * math.exp(-8.0 * (1.0 - float(p.shf_a[a])) ** 2) * fc * fc)
                assert ang[0, a, z] == pytest.approx(want, rel=1e-12)
        # centre H (atom 1): neighbours O (r=1) and H (r=sqrt2) -> block p(H,O)=3 only
        angH = aev[0, 1, 64:].reshape(10, 4, 8)
        nz = [b for b in range(10) if np.any(angH[b] != 0.0)]
        assert nz == [3]
        # radial: O sees two H at r=1 -> twice the two-atom value, in the H columns
        two = read_golden("two_atoms.txt")["aev0_radial_first4"]
        np.testing.assert_allclose(aev[0, 0, :4], 2 * np.array(two), rtol=1e-11 if exact else 1e-6)
        assert np.all(aev[0, 0, 16:64] == 0.0)
        # H(1) sees O at 1.0 (columns 48..63) and H at sqrt2 (columns 0..15)
        np.testing.assert_allclose(aev[0, 1, 48:52], two, rtol=1e-11 if exact else 1e-6)


@pytest.mark.parametrize("fname,p", [("one_water_c100.txt", P100), ("one_water_c095.txt", P095)])
def test_one_water_values_and_gradient(fname, p):
    gold = read_golden(fname)
    pos = _water()[None]
    sp = np.array([[O, H, H]], dtype=np.int32)
    aev = oracle.aev_forward(p, pos, sp, None)
    # the fixture was computed from the exact geometry; pos here is float32-rounded: ~1e-7
    assert aev.sum() == pytest.approx(gold["energy_g1"][0], rel=2e-6)
    ang = aev[0, :, 64:].reshape(3, 10, 4, 8)
    np.testing.assert_allclose(ang[0, 0, 0], gold["centreO_HH_row0"], rtol=2e-5)
    if "centreH1_HO_row0" in gold:
        np.testing.assert_allclose(ang[1, 3, 0], gold["centreH1_HO_row0"], rtol=2e-5, atol=1e-30)
    g = np.ones_like(aev, dtype=np.float32)
    grad = -oracle.aev_backward(p, pos, sp, None, g)[0]
    np.testing.assert_allclose(grad[0], gold["grad_O"], rtol=2e-5, atol=1e-9)
    # the fixture names the hydrogens only as a mirrored pair: x-components +-, same z
    gx = sorted([grad[1, 0], grad[2, 0]])
    np.testing.assert_allclose(gx, sorted([gold["grad_H1"][0], gold["grad_H2"][0]]), rtol=2e-5)
    np.testing.assert_allclose([grad[1, 2], grad[2, 2]], [gold["grad_H1"][2]] * 2, rtol=2e-5)
    np.testing.assert_allclose(grad[:, 1], 0.0, atol=1e-12)
    # and which hydrogen is which: finite differences decide
    fd = _fd_forces(p, pos, sp, None, g, [(1, 0), (2, 0)])
    np.testing.assert_allclose(-fd, grad[1:, 0], rtol=1e-5)


def test_radial_comb_sum():
    """sum_m exp(-eta(r-R_m)^2) ~ sqrt(pi/eta)/spacing inside the shift range
    (Poisson summation; ripple ~5e-4): catches a wrong eta, spacing or prefactor."""
    want = math.sqrt(math.pi / 16.0) / 0.27125
    for r in (2.0, 2.6, 3.3, 3.9):
        pos = np.array([[[0, 0, 0], [r, 0, 0]]], dtype=np.float32)
        aev = oracle.aev_forward(P100, pos, np.array([[Cc, N]], dtype=np.int32), None)
        fc = 0.5 * math.cos(math.pi * float(np.float32(r)) / float(np.float32(5.2))) + 0.5
        # atom 0 (C) sees N -> columns 32..47
        assert aev[0, 0, 32:48].sum() / (0.25 * fc) == pytest.approx(want, rel=2e-3)
        assert aev[0, 0, :32].sum() == 0.0 and aev[0, 0, 48:].sum() == 0.0


def test_cutoff_is_strict_and_smooth():
    sp = np.array([[H, H]], dtype=np.int32)
    inside = np.array([[[0, 0, 0], [5.1999, 0, 0]]], dtype=np.float32)
    outside = np.array([[[0, 0, 0], [5.2001, 0, 0]]], dtype=np.float32)
    a_in = oracle.aev_forward(P100, inside, sp, None)
    assert 0.0 < a_in[0, 0, 15] < 1e-9                 # f_c -> 0 at the cutoff
    assert np.all(oracle.aev_forward(P100, outside, sp, None) == 0.0)
    assert len(oracle.pairs(inside[0], None, None, 5.2)) == 1
    assert len(oracle.pairs(outside[0], None, None, 5.2)) == 0


# ----------------------------------------------------------------------------- neighbour search
def test_pairs_brute_vs_cell_vs_kdtree():
    from scipy.spatial import cKDTree
    w = make_c3()
    pos, box = w.pos[0], w.box
    for rc in (float(w.params.rcr), float(w.params.rca)):
        brute = oracle.pairs(pos, w.species[0], box, rc, "brute")
        cell = oracle.pairs(pos, w.species[0], box, rc, "cell")
        np.testing.assert_array_equal(brute, cell)
        # library routine on wrapped double copies of the same float32 positions
        b = box.astype(np.float64)
        p64 = pos.astype(np.float64)
        wrapped = p64 - b * np.floor(p64 / b)
        tree = cKDTree(wrapped, boxsize=b)
        kd = tree.query_pairs(float(np.float32(rc)) - 1e-9, output_type="ndarray")
        kd = np.sort(kd, axis=1)
        kd = kd[np.lexsort((kd[:, 1], kd[:, 0]))]
        np.testing.assert_array_equal(brute, kd.astype(np.int32))
    # statistics SURVEY.md section 8(d) recorded for this recipe: ~59.3 radial neighbours/atom
    assert 2 * len(oracle.pairs(pos, None, box, 5.2, "cell")) / 4500 == pytest.approx(59.3, abs=1.0)


def test_cell_list_on_a_non_cubic_box():
    """The cell-list path (the checker of C3/C4 and the timed CPU baseline) on an orthorhombic box
    whose edges give three DIFFERENT cell counts (16 x 22 x 27.5 A -> 3 x 4 x 5 cells at 5.2 A, 4 x 6 x 7
    at 3.5 A), atoms pushed outside [0, L): an x/y/z mix-up in the cell index or its decode fails here.
    Pinned against the O(N^2) loop, scipy's periodic cKDTree and, for the featurizer and its gradient,
    the brute-force result."""
    from scipy.spatial import cKDTree
    w = make_water_box(320, (16.0, 22.0, 27.5), 500, "ortho")
    box = w.box
    assert [int(np.floor(float(b) / 5.2)) for b in box] == [3, 4, 5]
    rng = np.random.default_rng(11)
    pos = (w.pos[0] + (rng.integers(-2, 3, size=w.pos[0].shape) * box)).astype(np.float32)
    for rc in (5.2, 3.5):
        brute = oracle.pairs(pos, w.species[0], box, rc, "brute")
        cell = oracle.pairs(pos, w.species[0], box, rc, "cell")
        np.testing.assert_array_equal(brute, cell)
        b = box.astype(np.float64)
        p64 = pos.astype(np.float64)
        wrapped = p64 - b * np.floor(p64 / b)
        wrapped = np.where(wrapped >= b, wrapped - b, wrapped)
        kd = cKDTree(wrapped, boxsize=b).query_pairs(float(np.float32(rc)) - 1e-6, output_type="ndarray")
        kd = np.sort(kd, axis=1)
        kd = kd[np.lexsort((kd[:, 1], kd[:, 0]))]
        # image shifts of up to two box lengths move float32 coordinates by ~1e-6 A: the generator's
        # 1e-4 A cutoff margin keeps the pair set unchanged
        np.testing.assert_array_equal(brute, kd.astype(np.int32))
    a_b = oracle.aev_forward(w.params, pos[None], w.species, box, use_cells=False)
    a_c = oracle.aev_forward(w.params, pos[None], w.species, box, use_cells=True)
    np.testing.assert_array_equal(a_b, a_c)
    f_b = oracle.aev_backward(w.params, pos[None], w.species, box, w.grad_aev, use_cells=False)
    f_c = oracle.aev_backward(w.params, pos[None], w.species, box, w.grad_aev, use_cells=True)
    np.testing.assert_allclose(f_b, f_c, rtol=0, atol=1e-12 * np.abs(f_b).max())   # OpenMP summation order
    assert np.abs(f_b.sum(axis=1)).max() < 1e-9 * np.abs(f_b).max() * w.n_atoms


def test_pairs_padding_and_images():
    w = make_c3()
    pos, box = w.pos[0].copy(), w.box
    ref = oracle.pairs(pos, None, box, 5.2, "brute")
    # shift individual atoms by whole box vectors: same pair set (G16)
    rng = np.random.default_rng(5)
    shifted = pos + (rng.integers(-2, 3, size=pos.shape) * box).astype(np.float32)
    np.testing.assert_array_equal(ref, oracle.pairs(shifted, None, box, 5.2, "cell"))
    # padding atoms (species < 0) are in no pair
    sp = w.species[0].copy()
    sp[::7] = -1
    got = oracle.pairs(pos, sp, box, 5.2, "cell")
    keep = (sp[ref[:, 0]] >= 0) & (sp[ref[:, 1]] >= 0)
    np.testing.assert_array_equal(ref[keep], got)


# ----------------------------------------------------------------------------- invariances
def _rotation(seed):
    q = np.random.default_rng(seed).standard_normal(4)
    q /= np.linalg.norm(q)
    w, x, y, z = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                     [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                     [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])


def test_invariance_translation_rotation_permutation():
    w = make_c1()
    p = w.params
    # exact float32 arithmetic would be needed for 1e-12; use dyadic translations and
    # compare at the level float32 re-rounding of rotated coordinates allows
    base = oracle.aev_forward(p, w.pos, w.species, None)
    moved = w.pos + np.array([8.0, -16.0, 4.0], dtype=np.float32)     # exact in float32 here? not quite
    a2 = oracle.aev_forward(p, moved, w.species, None)
    np.testing.assert_allclose(a2, base, atol=2e-5 * np.abs(base).max())
    R = _rotation(3)
    rot = (w.pos[0].astype(np.float64) @ R.T).astype(np.float32)[None]
    a3 = oracle.aev_forward(p, rot, w.species, None)
    np.testing.assert_allclose(a3, base, atol=2e-5 * np.abs(base).max())
    perm = np.random.default_rng(9).permutation(24)
    a4 = oracle.aev_forward(p, w.pos[:, perm], w.species[:, perm], None)
    np.testing.assert_allclose(a4[0], base[0, perm], rtol=1e-12, atol=1e-15)
    # forces rotate with the frame and permute with the atoms
    f = oracle.aev_backward(p, w.pos, w.species, None, w.grad_aev)
    f4 = oracle.aev_backward(p, w.pos[:, perm], w.species[:, perm], None, w.grad_aev[:, perm])
    np.testing.assert_allclose(f4[0], f[0, perm], rtol=1e-10, atol=1e-12)


def test_invariance_exact_translation_small_system():
    """A translation that IS exact in float32 (all coordinates multiples of 2^-10,
    shift a multiple of 2^-10): AEV must agree to fp64 rounding."""
    rng = np.random.default_rng(11)
    pos = (rng.integers(0, 4096, size=(1, 10, 3)) / 1024.0).astype(np.float32)
    sp = rng.integers(0, 4, size=(1, 10)).astype(np.int32)
    a = oracle.aev_forward(P100, pos, sp, None)
    b = oracle.aev_forward(P100, pos + np.float32(3.5), sp, None)
    np.testing.assert_allclose(a, b, rtol=1e-12, atol=1e-14)
    box = np.array([16.0, 16.0, 16.0], dtype=np.float32)
    c = oracle.aev_forward(P100, pos, sp, box)
    shift = (rng.integers(-1, 2, size=(1, 10, 3)) * 16.0).astype(np.float32)
    d = oracle.aev_forward(P100, pos + shift, sp, box)
    np.testing.assert_allclose(c, d, rtol=1e-12, atol=1e-14)


def test_zero_net_force_and_torque():
    w = make_c1()
    f = oracle.aev_backward(w.params, w.pos, w.species, None, w.grad_aev)[0]
    scale = np.abs(f).max()
    assert np.abs(f.sum(axis=0)).max() < 1e-12 * scale
    torque = np.cross(w.pos[0].astype(np.float64), f).sum(axis=0)
    assert np.abs(torque).max() < 1e-11 * scale
    w3 = make_c3()
    f3 = oracle.aev_backward(w3.params, w3.pos, w3.species, w3.box, w3.grad_aev, use_cells=True)[0]
    assert np.abs(f3.sum(axis=0)).max() < 1e-10 * np.abs(f3).max()
    # scales SURVEY.md section 8(c) recorded for C3 with g ~ N(0,1): force rms ~5.9
    assert np.sqrt((f3 ** 2).mean()) == pytest.approx(5.9, rel=0.15)


# ----------------------------------------------------------------------------- gradient
@pytest.mark.parametrize("cos_scale", [1.0, 0.95])
def test_finite_differences_c1(cos_scale):
    w = make_c1(cos_scale)
    f = oracle.aev_backward(w.params, w.pos, w.species, None, w.grad_aev)[0]
    coords = [(i, a) for i in range(24) for a in range(3)]
    fd = _fd_forces(w.params, w.pos, w.species, None, w.grad_aev, coords).reshape(24, 3)
    # BASELINE.json:north_star: step 1e-4 A, relative error < 1e-5
    assert np.abs(fd - f).max() / np.abs(f).max() < 1e-5
    assert np.sqrt(((fd - f) ** 2).sum() / (f ** 2).sum()) < 1e-5


def test_finite_differences_periodic_c3_sample():
    w = make_c3()
    f = oracle.aev_backward(w.params, w.pos, w.species, w.box, w.grad_aev, use_cells=True)[0]
    rng = np.random.default_rng(1)
    coords = [(int(i), int(a)) for i, a in zip(rng.integers(0, 4500, 6), rng.integers(0, 3, 6))]
    fd = _fd_forces(w.params, w.pos, w.species, w.box, w.grad_aev, coords, use_cells=True)
    got = np.array([f[i, a] for i, a in coords])
    assert np.abs(fd - got).max() / np.abs(f).max() < 1e-5


# ----------------------------------------------------------------------------- autograd cross-check
def _torch_aev(pos, species, p, box=None):
    """Independent dense-tensor restatement of north_star steps 1-4 (masks and einsum
    instead of neighbour loops).  Returns [n, L]."""
    import torch
    n, S = pos.shape[0], int(p.num_species)
    f64 = lambda a: torch.tensor(np.asarray(a, dtype=np.float32).astype(np.float64))  # noqa: E731
    shf_r, shf_a, shf_z = f64(p.shf_r), f64(p.shf_a), f64(p.shf_z)
    rcr, rca = float(np.float32(p.rcr)), float(np.float32(p.rca))
    eta_r, eta_a, zeta, c = (float(np.float32(v)) for v in (p.eta_r, p.eta_a, p.zeta, p.cos_scale))
    d = pos[None, :, :] - pos[:, None, :]
    if box is not None:
        b = f64(box)
        d = d - b * torch.round(d / b)
    eye = torch.eye(n, dtype=torch.bool)
    r = torch.sqrt((d * d).sum(-1) + eye.double())
    onehot = torch.nn.functional.one_hot(torch.tensor(species, dtype=torch.long), S).double()
    mr = ((r < rcr) & ~eye).double()
    rad = 0.25 * torch.exp(-eta_r * (r[..., None] - shf_r) ** 2) * (0.5 * torch.cos(math.pi * r / rcr) + 0.5)[..., None]
    radial = torch.einsum("ijm,ij,js->ism", rad, mr, onehot).reshape(n, -1)
    ma = (r < rca) & ~eye
    fca = (0.5 * torch.cos(math.pi * r / rca) + 0.5) * ma.double()
    u = d / r[..., None]
    cosr = torch.einsum("ijd,ikd->ijk", u, u)
    jk = torch.triu(torch.ones(n, n, dtype=torch.bool), diagonal=1)
    valid = ma[:, :, None] & ma[:, None, :] & jk[None]
    cosr = torch.where(valid, cosr, torch.zeros_like(cosr))
    theta = torch.acos(torch.clamp(c * cosr, -1.0, 1.0))
    ang = 2.0 ** (1.0 - zeta) * (1.0 + torch.cos(theta[..., None] - shf_z)) ** zeta        # ijkz
    rho = 0.5 * (r[:, :, None] + r[:, None, :])
    radA = torch.exp(-eta_a * (rho[..., None] - shf_a) ** 2)                                  # ijka
    wgt = fca[:, :, None] * fca[:, None, :] * valid.double()                                  # ijk
    blocks = []
    for s1 in range(S):
        for s2 in range(s1, S):
            sel = onehot[:, s1][:, None] * onehot[:, s2][None, :]
            if s1 != s2:
                sel = sel + sel.T
            blocks.append(torch.einsum("ijkz,ijka,ijk,jk->iaz", ang, radA, wgt, sel).reshape(n, -1))
    return torch.cat([radial] + blocks, dim=1)


@pytest.mark.parametrize("cos_scale,periodic", [(1.0, False), (0.95, False), (1.0, True)])
def test_against_torch_autograd(cos_scale, periodic):
    import torch
    p = ani1x_style_params(cos_scale)
    rng = np.random.default_rng(21)
    n = 9
    while True:
        pos = rng.uniform(0, 4.0, size=(n, 3)).astype(np.float32)
        dd = pos[:, None] - pos[None]
        if np.sqrt((dd ** 2).sum(-1))[np.triu_indices(n, 1)].min() > 0.8:
            break
    species = rng.integers(0, 4, size=n).astype(np.int32)
    box = np.array([10.5, 11.0, 12.5], dtype=np.float32) if periodic else None
    if periodic:
        pos[:, 0] += 8.0          # push atoms across the boundary
    g = rng.standard_normal((1, n, 384)).astype(np.float32)
    x = torch.tensor(pos.astype(np.float64), requires_grad=True)
    aev_t = _torch_aev(x, species, p, box)
    e = (aev_t * torch.tensor(g[0].astype(np.float64))).sum()
    e.backward()
    aev_o = oracle.aev_forward(p, pos[None], species[None], box)[0]
    np.testing.assert_allclose(aev_o, aev_t.detach().numpy(), rtol=1e-11, atol=1e-14)
    f_o = oracle.aev_backward(p, pos[None], species[None], box, g)[0]
    np.testing.assert_allclose(f_o, -x.grad.numpy(), rtol=1e-9, atol=1e-11)
    assert np.count_nonzero(aev_o[:, 64:]) > 500     # the angular part is exercised


def test_other_angular_split_and_general_zeta_against_torch_autograd():
    """8 angular radial shifts x 4 angle shifts, zeta = 14.1, 7 species (L = 1008): the slot order a*nZ + z, the block
    index and the pow() of the oracle with parameter counts other than the default, against the dense restatement."""
    import torch
    from gen import ani2x_shaped_params
    p = ani2x_shaped_params(0.95)
    rng = np.random.default_rng(22)
    n = 9
    while True:
        pos = rng.uniform(0, 4.0, size=(n, 3)).astype(np.float32)
        dd = pos[:, None] - pos[None]
        if np.sqrt((dd ** 2).sum(-1))[np.triu_indices(n, 1)].min() > 0.8:
            break
    species = rng.integers(0, 7, size=n).astype(np.int32)
    g = rng.standard_normal((1, n, 1008)).astype(np.float32)
    x = torch.tensor(pos.astype(np.float64), requires_grad=True)
    aev_t = _torch_aev(x, species, p, None)
    assert aev_t.shape == (n, 1008)
    (aev_t * torch.tensor(g[0].astype(np.float64))).sum().backward()
    aev_o = oracle.aev_forward(p, pos[None], species[None], None)[0]
    np.testing.assert_allclose(aev_o, aev_t.detach().numpy(), rtol=1e-11, atol=1e-14)
    f_o = oracle.aev_backward(p, pos[None], species[None], None, g)[0]
    np.testing.assert_allclose(f_o, -x.grad.numpy(), rtol=1e-9, atol=1e-11)
    assert np.count_nonzero(aev_o[:, 112:]) > 300


def test_cell_list_featurizer_equals_brute_force():
    w = make_c3()
    a = oracle.aev_forward(w.params, w.pos, w.species, w.box, use_cells=False)
    b = oracle.aev_forward(w.params, w.pos, w.species, w.box, use_cells=True)
    np.testing.assert_array_equal(a, b)
    # scales SURVEY.md section 8(c) recorded: max|AEV| ~2.8, 256 of 384 columns zero on water
    assert np.abs(a).max() == pytest.approx(2.8, rel=0.2)
    assert np.count_nonzero(np.abs(a[0]).sum(axis=0)) == 128


def test_batch_is_independent_conformers():
    w = make_c1()
    rng = np.random.default_rng(2)
    pos2 = np.concatenate([w.pos, w.pos + rng.normal(0, 0.3, w.pos.shape).astype(np.float32)])
    sp2 = np.concatenate([w.species, w.species])
    both = oracle.aev_forward(w.params, pos2, sp2, None)
    np.testing.assert_array_equal(both[0], oracle.aev_forward(w.params, pos2[:1], sp2[:1], None)[0])
    np.testing.assert_array_equal(both[1], oracle.aev_forward(w.params, pos2[1:], sp2[1:], None)[0])
    # padding atoms: rows are zero and they contribute to nobody (G12)
    sp_pad = w.species.copy()
    sp_pad[0, 20:] = -1
    a_pad = oracle.aev_forward(w.params, w.pos, sp_pad, None)
    a_cut = oracle.aev_forward(w.params, w.pos[:, :20], w.species[:, :20], None)
    np.testing.assert_array_equal(a_pad[0, :20], a_cut[0])
    assert np.all(a_pad[0, 20:] == 0.0)


# ----------------------------------------------------------------------------- the cone point (G2)
def _line3():
    pos = np.array([[[0.0, 0.0, 0.0], [1.3, 0.0, 0.0], [2.9, 0.0, 0.0]]], dtype=np.float32)
    return pos, np.array([[1, 3, 0]], dtype=np.int32)


def test_collinear_triplet_damped_angle_matches_autograd():
    """Exactly collinear j-i-k with c = 0.95: a regular point, so torch autograd of the independent
    restatement pins the oracle's value and gradient there (cos = -1 for the middle atom, +1 for the ends)."""
    import torch
    pos, sp = _line3()
    g = np.random.default_rng(6).standard_normal((1, 3, 384)).astype(np.float32)
    x = torch.tensor(pos[0].astype(np.float64), requires_grad=True)
    aev_t = _torch_aev(x, sp[0], P095)
    (aev_t * torch.tensor(g[0].astype(np.float64))).sum().backward()
    np.testing.assert_allclose(oracle.aev_forward(P095, pos, sp, None)[0], aev_t.detach().numpy(), rtol=1e-11, atol=1e-14)
    np.testing.assert_allclose(oracle.aev_backward(P095, pos, sp, None, g)[0], -x.grad.numpy(), rtol=1e-9, atol=1e-11)
    assert np.count_nonzero(aev_t.detach().numpy()[:, 64:]) > 0


def test_collinear_triplet_literal_angle_cone_point():
    """Exactly collinear j-i-k with c = 1 (the literal north_star formula): d(theta)/d(cos) is 0/0.
    Reading G2 defines the perpendicular part of the gradient as 0.  What the mathematics fixes:
    (a) by symmetry about the axis every force is along the line; (b) moving the atoms ALONG the line keeps
    theta at 0 or pi, so E is smooth in those coordinates and central differences pin the axial forces;
    (c) the value is the c -> 1 limit of the regular case."""
    pos, sp = _line3()
    g = np.random.default_rng(6).standard_normal((1, 3, 384)).astype(np.float32)
    f = oracle.aev_backward(P100, pos, sp, None, g)[0]
    assert np.all(np.isfinite(f))
    assert np.all(f[:, 1:] == 0.0)
    fd = _fd_forces(P100, pos, sp, None, g, [(0, 0), (1, 0), (2, 0)])
    np.testing.assert_allclose(f[:, 0], fd, rtol=1e-5, atol=1e-7)
    a1 = oracle.aev_forward(P100, pos, sp, None)
    a2 = oracle.aev_forward(ani1x_style_params(1.0 - 1e-7), pos, sp, None)
    # theta moves by sqrt(2e-7) = 4.5e-4 rad; zeta = 32 amplifies: a continuity check, not an identity
    np.testing.assert_allclose(a1, a2, rtol=0, atol=1e-2 * np.abs(a1).max())


# --------------------------------------------------------------------------- triclinic cells
TRI_LAT = np.array([[14.0, 0.0, 0.0], [3.0, 13.0, 0.0], [-2.0, 4.0, 12.5]])


def test_lattice_mode_with_a_diagonal_lattice_is_the_orthorhombic_minimum_image():
    """The triclinic image search (oracle.lattice) reduces to the already pinned L*rint(d/L) routine when the
    lattice is diagonal: same pair sets, AEV and forces."""
    from gen import make_periodic_cell
    w = make_periodic_cell(160, [12.0, 13.0, 14.5], 42)
    g = w.grad_aev
    a1 = oracle.aev_forward(w.params, w.pos, w.species, w.box)
    f1 = oracle.aev_backward(w.params, w.pos, w.species, w.box, g)
    p1 = oracle.pairs(w.pos[0], w.species[0], w.box, float(w.params.rcr))
    with oracle.lattice(np.diag(w.box)):
        a2 = oracle.aev_forward(w.params, w.pos, w.species, None)
        f2 = oracle.aev_backward(w.params, w.pos, w.species, None, g)
        p2 = oracle.pairs(w.pos[0], w.species[0], None, float(w.params.rcr))
    np.testing.assert_array_equal(p1, p2)
    np.testing.assert_allclose(a2, a1, rtol=0, atol=1e-13)
    np.testing.assert_allclose(f2, f1, rtol=0, atol=1e-11 * np.abs(f1).max())


def test_triclinic_cell_equals_its_explicit_replication():
    """A periodic triclinic cell is, by definition, the infinite lattice of its copies: the AEV rows and forces of
    the cell's atoms must equal those of the same atoms inside a NON-periodic cluster of 5x5x5 explicit copies
    (every neighbour within R_cr of a central-copy atom lies in that cluster).  This checks the image search
    against plain open-boundary arithmetic that does not use it."""
    from gen import make_periodic_cell
    w = make_periodic_cell(40, TRI_LAT, 43, min_dist=1.3)
    n = w.n_atoms
    lat = w.box.reshape(3, 3).astype(np.float64)
    g = w.grad_aev
    with oracle.lattice(w.box):
        a_p = oracle.aev_forward(w.params, w.pos, w.species, None)
        f_p = oracle.aev_backward(w.params, w.pos, w.species, None, g)
        pr = oracle.pairs(w.pos[0], w.species[0], None, float(w.params.rcr))
    # the cluster: wrap every atom into the cell first (copies of an atom far outside would leave the 5x5x5 block)
    frac = w.pos[0].astype(np.float64) @ np.linalg.inv(lat)
    base = (frac - np.floor(frac)) @ lat
    shifts = [np.array([i, j, k], dtype=np.float64) @ lat for i in range(-2, 3) for j in range(-2, 3) for k in range(-2, 3)]
    centre = len(shifts) // 2
    assert np.all(shifts[centre] == 0.0)
    big = np.concatenate([base + s for s in shifts]).astype(np.float64)
    big_sp = np.tile(w.species[0], len(shifts))
    # float32 inputs: use the replicated float64 positions rounded once, and the same rounded base inside the cell
    big32 = big.astype(np.float32)
    lo, hi = centre * n, (centre + 1) * n
    with oracle.lattice(w.box):
        a_p = oracle.aev_forward(w.params, big32[lo:hi][None], w.species, None)
        pr = oracle.pairs(big32[lo:hi], w.species[0], None, float(w.params.rcr))
    a_c = oracle.aev_forward(w.params, big32[None], big_sp[None], None)[:, lo:hi]
    # float32 rounding of the replicas' coordinates moves distances by ~1e-6 A: compare at that level
    np.testing.assert_allclose(a_p, a_c, rtol=0, atol=2e-5 * np.abs(a_c).max())
    # pair set: periodic pairs (i<j) <-> cluster pairs with one end in the central copy, folded back to (i, j mod n)
    pc = oracle.pairs(big32, big_sp, None, float(w.params.rcr))
    inc = (pc[:, 0] >= lo) & (pc[:, 0] < hi) | (pc[:, 1] >= lo) & (pc[:, 1] < hi)
    fold = np.sort(np.stack([pc[inc, 0] % n, pc[inc, 1] % n], axis=1), axis=1)
    fold = np.unique(fold[fold[:, 0] != fold[:, 1]], axis=0)
    np.testing.assert_array_equal(fold, pr)
    # forces: upstream gradient only on the central copy's rows; the force on a periodic atom is the sum over its copies
    gbig = np.zeros((1, len(big32), g.shape[2]), dtype=np.float32)
    gbig[0, lo:hi] = g[0]
    f_c = oracle.aev_backward(w.params, big32[None], big_sp[None], None, gbig)[0].reshape(len(shifts), n, 3).sum(axis=0)
    with oracle.lattice(w.box):
        f_p = oracle.aev_backward(w.params, big32[lo:hi][None], w.species, None, g)[0]
    np.testing.assert_allclose(f_p, f_c, rtol=0, atol=2e-4 * np.abs(f_c).max())


def test_triclinic_lattice_translation_invariance_and_finite_differences():
    from gen import make_periodic_cell
    w = make_periodic_cell(60, TRI_LAT, 44)
    lat = w.box.reshape(3, 3).astype(np.float64)
    g = w.grad_aev
    rng = np.random.default_rng(3)
    with oracle.lattice(w.box):
        a0 = oracle.aev_forward(w.params, w.pos, w.species, None)
        f0 = oracle.aev_backward(w.params, w.pos, w.species, None, g)
        moved = w.pos.copy()
        moved[0] += (rng.integers(-1, 2, size=(w.n_atoms, 3)).astype(np.float64) @ lat).astype(np.float32)
        a1 = oracle.aev_forward(w.params, moved, w.species, None)
        np.testing.assert_allclose(a1, a0, rtol=0, atol=3e-5 * np.abs(a0).max())     # float32 coordinates of the moved atoms
        assert np.abs(f0[0].sum(axis=0)).max() < 1e-10 * np.abs(f0).max() * w.n_atoms
        for i, c in zip(rng.integers(0, w.n_atoms, 5), rng.integers(0, 3, 5)):
            xp, xm = w.pos.copy(), w.pos.copy()
            xp[0, i, c] = np.float32(w.pos[0, i, c] + 1e-4)
            xm[0, i, c] = np.float32(w.pos[0, i, c] - 1e-4)
            step = float(xp[0, i, c]) - float(xm[0, i, c])
            ep = (oracle.aev_forward(w.params, xp, w.species, None) * g).sum()
            em = (oracle.aev_forward(w.params, xm, w.species, None) * g).sum()
            assert -(ep - em) / step == pytest.approx(f0[0, i, c], rel=2e-5, abs=2e-5 * np.abs(f0).max())
