"""fp64 CPU oracle for the ANI-style AEV hot path -- TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` /
`--impl reference` legs may import this package.  The product path
(`paper_2310_03121_b200`) never does, and this package never imports it.

The arithmetic lives in `aev_oracle.c` (plain C99, double, explicit loops in the
order of BASELINE.json:north_star steps 1-4 as restated in SURVEY.md section 8(c));
this module is argument marshalling (ctypes) plus the species gather/scatter around
the per-species network (step 6).

Parity status: pinned by tests/test_oracle_*.py (closed forms in tests/golden/,
brute force vs cell list vs scipy cKDTree, invariances, zero net force/torque,
finite differences, torch-CPU fp64 autograd, MLP special cases).
"""
from __future__ import annotations

import ctypes as C
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

from .build import build as _build

_lib = None


class _Params(C.Structure):
    _fields_ = [
        ("num_species", C.c_int32),
        ("rcr", C.c_double), ("rca", C.c_double),
        ("eta_r", C.c_double),
        ("n_shf_r", C.c_int32), ("shf_r", C.POINTER(C.c_double)),
        ("eta_a", C.c_double), ("zeta", C.c_double),
        ("n_shf_a", C.c_int32), ("shf_a", C.POINTER(C.c_double)),
        ("n_shf_z", C.c_int32), ("shf_z", C.POINTER(C.c_double)),
        ("cos_scale", C.c_double),
    ]


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        f32p, i32p, f64p = C.POINTER(C.c_float), C.POINTER(C.c_int32), C.POINTER(C.c_double)
        L.oracle_max_threads.restype = C.c_int
        L.oracle_set_threads.argtypes = [C.c_int]
        for fn in (L.oracle_pairs_brute, L.oracle_pairs_cell):
            fn.restype = C.c_int64
            fn.argtypes = [f32p, i32p, f32p, C.c_int32, C.c_double, i32p, C.c_int64]
        L.oracle_aev_length.restype = C.c_int32
        L.oracle_aev_length.argtypes = [C.POINTER(_Params)]
        L.oracle_aev_forward.restype = C.c_int
        L.oracle_aev_forward.argtypes = [C.POINTER(_Params), f32p, i32p, f32p, C.c_int32, C.c_int32,
                                         C.c_int, f64p]
        L.oracle_aev_backward.restype = C.c_int
        L.oracle_aev_backward.argtypes = [C.POINTER(_Params), f32p, i32p, f32p, C.c_int32, C.c_int32,
                                          C.c_int, f32p, f64p]
        L.oracle_set_lattice.restype = C.c_int
        L.oracle_set_lattice.argtypes = [f64p]
        L.oracle_mlp.restype = C.c_int
        L.oracle_mlp.argtypes = [C.c_int32, f64p, C.c_int32, i32p, C.POINTER(f64p), C.POINTER(f64p),
                                 C.c_double, f64p, f64p]
        _lib = L
    return _lib


def max_threads() -> int:
    return int(lib().oracle_max_threads())


def set_threads(n: int) -> None:
    lib().oracle_set_threads(int(n))


def _ptr(a: Optional[np.ndarray], ctype):
    return None if a is None else a.ctypes.data_as(C.POINTER(ctype))


class _P:
    """Keeps the double copies of the float32 parameters alive next to the C struct."""

    def __init__(self, p):
        # G9: the generators emit float32 parameters and the oracle promotes those same
        # values to double.  A parameter set built in float64 (the closed-form pin tests,
        # whose fixtures were computed with exact parameters) is taken as given.
        def arr(a):
            a = np.asarray(a)
            if a.dtype != np.float64:
                a = a.astype(np.float32)
            return np.ascontiguousarray(a.astype(np.float64))

        def f(v):
            return float(v) if isinstance(v, (np.float64, float)) else float(np.float32(v))

        self.shf_r, self.shf_a, self.shf_z = arr(p.shf_r), arr(p.shf_a), arr(p.shf_z)
        self.c = _Params(int(p.num_species), f(p.rcr), f(p.rca), f(p.eta_r),
                         len(self.shf_r), _ptr(self.shf_r, C.c_double),
                         f(p.eta_a), f(p.zeta),
                         len(self.shf_a), _ptr(self.shf_a, C.c_double),
                         len(self.shf_z), _ptr(self.shf_z, C.c_double),
                         f(p.cos_scale))


class lattice:
    """Context manager: inside it every periodic displacement is the minimum image of the triclinic cell
    with rows a, b, c (`box` arguments are then ignored and the cell list is not available):

        with oracle.lattice(lat): aev = oracle.aev_forward(p, pos, species, None)
    """

    def __init__(self, lat):
        self.lat = np.ascontiguousarray(np.asarray(lat, dtype=np.float32).astype(np.float64).reshape(9))

    def __enter__(self):
        if lib().oracle_set_lattice(_ptr(self.lat, C.c_double)) != 0:
            raise ValueError("singular lattice")
        return self

    def __exit__(self, *exc):
        lib().oracle_set_lattice(None)
        return False


def aev_length(p) -> int:
    return int(lib().oracle_aev_length(C.byref(_P(p).c)))


def _prep(pos, species, box):
    pos = np.ascontiguousarray(pos, dtype=np.float32)
    if pos.ndim == 2:
        pos = pos[None]
    batch, n = pos.shape[0], pos.shape[1]
    species = np.ascontiguousarray(species, dtype=np.int32).reshape(batch, n)
    box = None if box is None else np.ascontiguousarray(box, dtype=np.float32).reshape(3)
    return pos, species, box, batch, n


def pairs(pos, species, box, rc: float, method: str = "brute") -> np.ndarray:
    """Sorted unique (i<j) pairs with r_ij < rc for ONE system."""
    pos = np.ascontiguousarray(pos, dtype=np.float32).reshape(-1, 3)
    n = pos.shape[0]
    species = None if species is None else np.ascontiguousarray(species, dtype=np.int32).reshape(n)
    box = None if box is None else np.ascontiguousarray(box, dtype=np.float32).reshape(3)
    fn = {"brute": lib().oracle_pairs_brute, "cell": lib().oracle_pairs_cell}[method]
    cap = max(64, 64 * n)
    while True:
        out = np.empty((cap, 2), dtype=np.int32)
        cnt = int(fn(_ptr(pos, C.c_float), _ptr(species, C.c_int32), _ptr(box, C.c_float),
                     n, float(np.float32(rc)), _ptr(out, C.c_int32), cap))
        if cnt < 0:
            raise ValueError("cell list needs a periodic box with >= 3 cells per edge")
        if cnt <= cap:
            return out[:cnt].copy()
        cap = cnt


def aev_forward(p, pos, species, box=None, use_cells: bool = False) -> np.ndarray:
    """AEV f64 [batch, n, L]."""
    pos, species, box, batch, n = _prep(pos, species, box)
    P = _P(p)
    L = int(lib().oracle_aev_length(C.byref(P.c)))
    out = np.empty((batch, n, L), dtype=np.float64)
    rc = lib().oracle_aev_forward(C.byref(P.c), _ptr(pos, C.c_float), _ptr(species, C.c_int32),
                                  _ptr(box, C.c_float), n, batch, int(use_cells), _ptr(out, C.c_double))
    if rc != 0:
        raise ValueError("oracle_aev_forward failed (box too small for the cell list?)")
    return out


def aev_backward(p, pos, species, box, grad_aev, use_cells: bool = False) -> np.ndarray:
    """forces f64 [batch, n, 3] = - sum g * dAEV/dx."""
    pos, species, box, batch, n = _prep(pos, species, box)
    P = _P(p)
    L = int(lib().oracle_aev_length(C.byref(P.c)))
    g = np.ascontiguousarray(grad_aev, dtype=np.float32).reshape(batch, n, L)
    out = np.empty((batch, n, 3), dtype=np.float64)
    rc = lib().oracle_aev_backward(C.byref(P.c), _ptr(pos, C.c_float), _ptr(species, C.c_int32),
                                   _ptr(box, C.c_float), n, batch, int(use_cells),
                                   _ptr(g, C.c_float), _ptr(out, C.c_double))
    if rc != 0:
        raise ValueError("oracle_aev_backward failed (box too small for the cell list?)")
    return out


def mlp(x: np.ndarray, weights: Sequence[np.ndarray], biases: Sequence[np.ndarray],
        alpha: float, want_grad: bool = True) -> Tuple[np.ndarray, Optional[np.ndarray]]:
    """One network on rows x [n_rows, dims0] -> (energy [n_rows], dE/dx [n_rows, dims0])
    (SURVEY 8(c) step 6).  weights[l] is [in][out]; promoted to double."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    n_rows = x.shape[0]
    Ws = [np.ascontiguousarray(w, dtype=np.float64) for w in weights]
    bs = [np.ascontiguousarray(b, dtype=np.float64) for b in biases]
    dims = np.array([Ws[0].shape[0]] + [w.shape[1] for w in Ws], dtype=np.int32)
    f64p = C.POINTER(C.c_double)
    Wp = (f64p * len(Ws))(*[_ptr(w, C.c_double) for w in Ws])
    bp = (f64p * len(bs))(*[_ptr(b, C.c_double) for b in bs])
    energy = np.empty(n_rows, dtype=np.float64)
    grad = np.empty_like(x) if want_grad else None
    rc = lib().oracle_mlp(n_rows, _ptr(x, C.c_double), len(Ws), _ptr(dims, C.c_int32), Wp, bp,
                          float(alpha), _ptr(energy, C.c_double), _ptr(grad, C.c_double))
    if rc != 0:
        raise ValueError("oracle_mlp: last layer must have one output")
    return energy, grad


def energy_forces(p, pos, species, box, nets: Dict[int, Tuple[List[np.ndarray], List[np.ndarray]]],
                  alpha: float, use_cells: bool = False):
    """E [batch] and forces [batch, n, 3] for E = sum_i NN_{s_i}(AEV_i) (G15): AEV forward,
    per-species networks on the rows of each species, dE/dAEV scattered back, AEV backward.
    The network's float64 dE/dAEV is handed to the backward as float64 (not rounded)."""
    pos, species, box, batch, n = _prep(pos, species, box)
    aev = aev_forward(p, pos, species, box, use_cells)
    L = aev.shape[2]
    flat = aev.reshape(-1, L)
    sp = species.reshape(-1)
    e_atom = np.zeros(flat.shape[0], dtype=np.float64)
    g = np.zeros_like(flat)
    for s in np.unique(sp[sp >= 0]):
        if int(s) not in nets:
            raise ValueError("no network for species %d" % s)
        rows = np.nonzero(sp == s)[0]
        e, gr = mlp(flat[rows], nets[int(s)][0], nets[int(s)][1], alpha)
        e_atom[rows] = e
        g[rows] = gr
    energy = e_atom.reshape(batch, n).sum(axis=1)
    forces = _backward_f64(p, pos, species, box, g.reshape(batch, n, L), use_cells)
    return energy, forces, aev


def energy_forces_ensemble(p, pos, species, box, models, alpha: float, use_cells: bool = False):
    """Ensemble of networks over one AEV ("an ensemble of eight models"): `models` is a
    list of `nets` dictionaries; the result is the plain mean over the models of `energy_forces`
    (energy and forces are both linear in the per-model outputs).  Written as the definition:
    one full evaluation per model, then the average."""
    es, fs = [], []
    aev = None
    for nets in models:
        e, f, aev = energy_forces(p, pos, species, box, nets, alpha, use_cells)
        es.append(e)
        fs.append(f)
    return sum(es) / len(models), sum(fs) / len(models), aev


def _backward_f64(p, pos, species, box, g64, use_cells):
    """aev_backward takes float32 g (the API's dtype).  For the full-model oracle the
    float64 g is split as hi(float32) + lo(float32); the backward is linear in g, so the
    two results add to the float64-g answer to ~1e-15 relative."""
    hi = g64.astype(np.float32)
    lo = (g64 - hi.astype(np.float64)).astype(np.float32)
    return (aev_backward(p, pos, species, box, hi, use_cells)
            + aev_backward(p, pos, species, box, lo, use_cells))
