"""GPU parity on the configurations round 1 left untested ("What's weak" 2a-2d):
orthorhombic boxes with three different cell counts, periodic batches, exactly collinear
triplets (the cone point of reading G2).  Same tolerances as tests/test_gpu_parity.py.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
from gen import ani1x_style_params, make_water_box

from test_gpu_parity import AEV_TOL, _check_forces

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pkg():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2310_03121_b200 as p
    return p


def _ortho_batch(cos_scale=1.0):
    """Three different 960-atom water boxes that share one 16 x 22 x 27.5 A cell (3 x 4 x 5 cells of >= 5.2 A),
    a third of the atoms moved by whole box vectors so that the wrap is exercised."""
    ws = [make_water_box(320, (16.0, 22.0, 27.5), 500 + k, "ortho%d" % k, cos_scale) for k in range(3)]
    rng = np.random.default_rng(12)
    pos = np.stack([w.pos[0] for w in ws])
    move = rng.random(pos.shape[:2]) < 0.33
    shift = rng.integers(-2, 3, size=pos.shape) * ws[0].box
    pos = np.where(move[..., None], pos + shift, pos).astype(np.float32)
    sp = np.stack([w.species[0] for w in ws])
    g = np.random.default_rng(13).standard_normal((3, pos.shape[1], ws[0].params.aev_length)).astype(np.float32)
    return ws[0].params, pos, sp, ws[0].box, g


@pytest.mark.parametrize("cos_scale", [1.0, 0.95])
def test_orthorhombic_box_three_cell_counts_periodic_batch(pkg, cos_scale):
    """PAPER.md:223 (orthorhombic periodic cells are a user workload): ncx != ncy != ncz through k_bin's cell
    index and k_nbr's stencil decode, with batch = 3 periodic systems in one call (bins indexed b*ncell+cell)."""
    p, pos, sp, box, g = _ortho_batch(cos_scale)
    batch, n = pos.shape[:2]
    ctx = pkg.Context(p, max_atoms=n, max_batch=batch)
    pos_d, sp_d = torch.from_numpy(pos).cuda(), torch.from_numpy(sp).cuda()
    ctx.aev_neighbors(pos_d, sp_d, box)
    ctx.check_status()
    for which, rc in ((0, p.rcr), (1, p.rca)):
        got = ctx.aev_export_pairs(which, cap=batch * n * 40)
        want = np.concatenate([oracle.pairs(pos[b], sp[b], box, float(rc), "brute").astype(np.int64) + b * n
                               for b in range(batch)]).astype(np.int32)
        np.testing.assert_array_equal(got, want)
    aev = ctx.aev_forward(pos_d, sp_d, box)
    f = ctx.aev_backward(torch.from_numpy(g).cuda())
    ctx.check_status()
    want_a = oracle.aev_forward(p, pos, sp, box, use_cells=False)
    want_f = oracle.aev_backward(p, pos, sp, box, g, use_cells=False)
    assert np.abs(aev.cpu().numpy() - want_a).max() <= AEV_TOL * np.abs(want_a).max()
    _check_forces(f.cpu().numpy(), want_f, what=("ortho batch 3", cos_scale))
    ctx.close()


def _collinear_systems():
    """Exactly collinear j-i-k triplets (the generators reject these; here they are the point).
    line3: three atoms on the x axis (centre atom sees cos = -1, end atoms see cos = +1);
    grid9: a 3 x 3 planar lattice, spacing 1.4 A (rows, columns and diagonals are collinear);
    no distance lies within 1e-4 A of a cutoff (1.4, 1.98, 2.8, 3.13, 3.96 A)."""
    line3 = np.array([[0.0, 0.0, 0.0], [1.3, 0.0, 0.0], [2.9, 0.0, 0.0]], dtype=np.float32)
    grid9 = np.array([[1.4 * i, 1.4 * j, 0.0] for i in range(3) for j in range(3)], dtype=np.float32)
    return {"line3": (line3, np.array([1, 3, 0], dtype=np.int32)),
            "grid9": (grid9, np.array([0, 1, 2, 3, 0, 1, 2, 3, 0], dtype=np.int32))}


@pytest.mark.parametrize("cos_scale", [1.0, 0.95])
@pytest.mark.parametrize("name", ["line3", "grid9"])
def test_exactly_collinear_triplets(pkg, name, cos_scale):
    """Reading G2: at sin(theta) = 0 and c = 1 the gradient direction is 0/0; both sides define the
    perpendicular part as 0 (oracle: 1 - c^2 cos^2 < 1e-12; GPU: < 1e-10 in fp32).  With c = 0.95 the
    point is regular.  Values and forces must agree with the oracle either way."""
    pos, sp = _collinear_systems()[name]
    p = ani1x_style_params(cos_scale)
    g = np.random.default_rng(5).standard_normal((1, len(sp), p.aev_length)).astype(np.float32)
    ctx = pkg.Context(p, max_atoms=len(sp))
    aev = ctx.aev_forward(torch.from_numpy(pos[None]).cuda(), torch.from_numpy(sp[None]).cuda(), None)
    f = ctx.aev_backward(torch.from_numpy(g).cuda())
    ctx.check_status()
    want_a = oracle.aev_forward(p, pos[None], sp[None], None)
    want_f = oracle.aev_backward(p, pos[None], sp[None], None, g)
    assert np.isfinite(f.cpu().numpy()).all()
    assert np.abs(aev.cpu().numpy() - want_a).max() <= AEV_TOL * np.abs(want_a).max()
    _check_forces(f.cpu().numpy(), want_f, what=(name, cos_scale))
    ctx.close()
