"""Thin ctypes binding of libaev_b200.so (include/aev.h) -- argument marshalling only.

Every step of the path (neighbour search, AEV forward/backward, per-species MLPs) runs in
the CUDA kernels of `csrc/`; PyTorch is used here for device memory and streams only.
There is no CPU fallback: loading fails loudly if the library is missing, and every call
raises `AevError` on a non-zero return code.  This package never imports `oracle`.

The functions carry the names of the C ABI (PAPER.md:75 contract; BASELINE.json:north_star
entry points): aev_create, aev_neighbors, aev_forward, aev_backward, ani_mlp_load,
ani_energy_forces, aev_export_pairs, aev_status.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libaev_b200.so")

AEV_OK = 0
ERRORS = {
    -1: "AEV_ERR_INVALID_ARG", -2: "AEV_ERR_BOX_TOO_SMALL", -3: "AEV_ERR_CAPACITY",
    -4: "AEV_ERR_STATE", -5: "AEV_ERR_UNSUPPORTED", -6: "AEV_ERR_CUDA", -7: "AEV_ERR_STATIC_LIMIT",
}
AEV_STATIC_MAX_ATOMS = 4096      # include/aev.h

EXPORTS = [
    "aev_create", "aev_destroy", "aev_length", "aev_neighbors", "aev_forward", "aev_backward",
    "ani_mlp_load", "ani_mlp_set_ensemble", "ani_mlp_load_model", "ani_mlp_kernel", "ani_energy_forces", "ani_energy_forces_subset", "aev_forward_backward_host", "ani_energy_forces_host",
    "aev_export_pairs", "aev_export_counts", "aev_set_profiling", "aev_get_profile", "aev_status", "aev_launch_count", "aev_neighbor_builds", "aev_probe_fp32_tflops",
    "aev_error_string", "aev_pairs_static", "aev_forward_range",
]


class AevError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        msg = lib().aev_error_string(code).decode() if _lib is not None else ""
        super().__init__("%s failed: %s (%d) %s" % (where, ERRORS.get(code, "?"), code, msg))


class _Params(C.Structure):
    _fields_ = [
        ("num_species", C.c_int32),
        ("rcr", C.c_float), ("rca", C.c_float),
        ("eta_r", C.c_float), ("n_shf_r", C.c_int32), ("shf_r", C.POINTER(C.c_float)),
        ("eta_a", C.c_float), ("zeta", C.c_float),
        ("n_shf_a", C.c_int32), ("shf_a", C.POINTER(C.c_float)),
        ("n_shf_z", C.c_int32), ("shf_z", C.POINTER(C.c_float)),
        ("cos_scale", C.c_float),
        ("max_atoms", C.c_int32), ("max_batch", C.c_int32),
        ("max_radial_nbrs", C.c_int32), ("max_angular_nbrs", C.c_int32),
        ("device", C.c_int32),
        ("flags", C.c_uint32),
        ("skin", C.c_float),
    ]


AEV_FLAG_DETERMINISTIC, AEV_FLAG_MLP_FP32, AEV_FLAG_TRICLINIC = 1, 2, 4


_lib = None


def lib():
    """Loads the C-ABI library (building it with nvcc first if the .so is absent or stale
    and a compiler is present).  Raises if it cannot be had: there is no fallback."""
    global _lib
    if _lib is None:
        from .build import build, compiler_present
        if compiler_present():
            path = build()          # a failed compile raises: never fall back to a library built from older sources
        elif os.path.exists(LIB_PATH):
            path = LIB_PATH         # no nvcc on this machine: use the library that was shipped with the tree
        else:
            raise RuntimeError("libaev_b200.so is missing and there is no nvcc to build it (no fallback exists)")
        L = C.CDLL(path)
        vp, i32, i64, f32p, i32p = C.c_void_p, C.c_int32, C.c_int64, C.c_void_p, C.c_void_p
        L.aev_create.restype = C.c_int
        L.aev_create.argtypes = [C.POINTER(_Params), C.POINTER(vp)]
        L.aev_destroy.restype = C.c_int
        L.aev_destroy.argtypes = [vp]
        L.aev_length.restype = C.c_int
        L.aev_length.argtypes = [vp]
        L.aev_neighbors.restype = C.c_int
        L.aev_neighbors.argtypes = [vp, f32p, i32p, C.POINTER(C.c_float), i32, i32, vp]
        L.aev_forward.restype = C.c_int
        L.aev_forward.argtypes = [vp, f32p, i32p, C.POINTER(C.c_float), i32, i32, f32p, vp]
        L.aev_forward_range.restype = C.c_int
        L.aev_forward_range.argtypes = [vp, f32p, i32p, C.POINTER(C.c_float), i32, i32, i32, i32, f32p, vp]
        L.aev_backward.restype = C.c_int
        L.aev_backward.argtypes = [vp, f32p, f32p, vp]
        L.ani_mlp_load.restype = C.c_int
        L.ani_mlp_load.argtypes = [vp, i32, i32, C.POINTER(i32), C.POINTER(C.POINTER(C.c_float)),
                                   C.POINTER(C.POINTER(C.c_float)), C.c_float]
        L.ani_mlp_set_ensemble.restype = C.c_int
        L.ani_mlp_set_ensemble.argtypes = [vp, i32]
        L.ani_mlp_load_model.restype = C.c_int
        L.ani_mlp_load_model.argtypes = [vp, i32, i32, i32, C.POINTER(i32), C.POINTER(C.POINTER(C.c_float)),
                                         C.POINTER(C.POINTER(C.c_float)), C.c_float]
        L.ani_mlp_kernel.restype = C.c_int
        L.ani_mlp_kernel.argtypes = [vp]
        L.ani_energy_forces.restype = C.c_int
        L.ani_energy_forces.argtypes = [vp, f32p, i32p, C.POINTER(C.c_float), i32, i32, vp, f32p, vp]
        L.ani_energy_forces_subset.restype = C.c_int
        L.ani_energy_forces_subset.argtypes = [vp, f32p, i32p, i32p, C.POINTER(C.c_float), i32, vp, f32p, vp]
        L.aev_forward_backward_host.restype = C.c_int
        L.aev_forward_backward_host.argtypes = [vp, vp, vp, C.POINTER(C.c_float), i32, i32, vp, vp, vp]
        L.ani_energy_forces_host.restype = C.c_int
        L.ani_energy_forces_host.argtypes = [vp, vp, vp, C.POINTER(C.c_float), i32, i32, vp, vp]
        L.aev_export_pairs.restype = C.c_int
        L.aev_export_pairs.argtypes = [vp, i32, i32p, i64, C.POINTER(i64)]
        L.aev_export_counts.restype = C.c_int
        L.aev_export_counts.argtypes = [vp, i32p]
        L.aev_set_profiling.restype = C.c_int
        L.aev_set_profiling.argtypes = [vp, i32]
        L.aev_get_profile.restype = C.c_int
        L.aev_get_profile.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(i64)]
        L.aev_status.restype = C.c_int
        L.aev_status.argtypes = [vp]
        L.aev_neighbor_builds.restype = C.c_int
        L.aev_neighbor_builds.argtypes = [vp, C.POINTER(i64)]
        L.aev_launch_count.restype = i64
        L.aev_launch_count.argtypes = [vp]
        L.aev_probe_fp32_tflops.restype = C.c_int
        L.aev_probe_fp32_tflops.argtypes = [i32, C.POINTER(C.c_double)]
        L.aev_pairs_static.restype = C.c_int
        L.aev_pairs_static.argtypes = [f32p, i32p, i32, C.c_float, i32p, i64, vp, i32, vp]
        L.aev_error_string.restype = C.c_char_p
        L.aev_error_string.argtypes = [C.c_int]
        _lib = L
    return _lib


def _check(rc: int, where: str) -> None:
    if rc != AEV_OK:
        raise AevError(rc, where)


def _box(box):
    if box is None:
        return None, None
    arr = np.ascontiguousarray(np.asarray(box, dtype=np.float32).reshape(-1))      # 3 edges, or 9 with AEV_FLAG_TRICLINIC
    if arr.size not in (3, 9):
        raise ValueError("box must have 3 (orthorhombic) or 9 (triclinic lattice rows) entries")
    return arr, arr.ctypes.data_as(C.POINTER(C.c_float))


def _stream(stream) -> int:
    if stream is None:
        import torch
        return int(torch.cuda.current_stream().cuda_stream)
    return int(getattr(stream, "cuda_stream", stream))


def _dev_ptr(t, dtype, name):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError("%s must be a CUDA tensor" % name)
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError("%s must be contiguous %s" % (name, dtype))
    return t.data_ptr()


class Context:
    """Owns one `aev_ctx`.  `params` is any object with the fields of gen.AniParams."""

    def __init__(self, params, max_atoms: int, max_batch: int = 1, device: int = 0,
                 max_radial_nbrs: int = 0, max_angular_nbrs: int = 0, flags: int = 0, skin: float = 0.0):
        self._h = C.c_void_p()
        shf_r = np.ascontiguousarray(params.shf_r, dtype=np.float32)
        shf_a = np.ascontiguousarray(params.shf_a, dtype=np.float32)
        shf_z = np.ascontiguousarray(params.shf_z, dtype=np.float32)
        fp = lambda a: a.ctypes.data_as(C.POINTER(C.c_float))
        p = _Params(int(params.num_species), float(params.rcr), float(params.rca),
                    float(params.eta_r), len(shf_r), fp(shf_r),
                    float(params.eta_a), float(params.zeta), len(shf_a), fp(shf_a),
                    len(shf_z), fp(shf_z), float(params.cos_scale),
                    int(max_atoms), int(max_batch), int(max_radial_nbrs), int(max_angular_nbrs),
                    int(device), int(flags), float(skin))
        _check(lib().aev_create(C.byref(p), C.byref(self._h)), "aev_create")
        self.device = int(device)
        self.length = int(lib().aev_length(self._h))

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().aev_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- device-pointer calls (torch CUDA tensors in, asynchronous on the current stream)
    def aev_neighbors(self, pos, species, box=None, stream=None):
        import torch
        batch, n = pos.shape[0], pos.shape[1]
        keep, bp = _box(box)
        sp = None if species is None else _dev_ptr(species, torch.int32, "species")
        _check(lib().aev_neighbors(self._h, _dev_ptr(pos, torch.float32, "pos"), sp, bp, n, batch,
                                   _stream(stream)), "aev_neighbors")

    def aev_forward(self, pos, species, box=None, aev_out=None, stream=None):
        import torch
        batch, n = pos.shape[0], pos.shape[1]
        if aev_out is None:
            aev_out = torch.empty((batch, n, self.length), dtype=torch.float32, device=pos.device)
        keep, bp = _box(box)
        _check(lib().aev_forward(self._h, _dev_ptr(pos, torch.float32, "pos"),
                                 _dev_ptr(species, torch.int32, "species"), bp, n, batch,
                                 _dev_ptr(aev_out, torch.float32, "aev_out"), _stream(stream)),
               "aev_forward")
        return aev_out

    def aev_forward_range(self, pos, species, box, first: int, count: int, aev_out=None, stream=None):
        """aev_forward for the central atoms [first, first + count) (flat index) only; rows outside the slab are left
        as they are in `aev_out` (zeros if this call allocates it).  The next aev_backward returns the slab's partial
        forces on all atoms."""
        import torch
        batch, n = pos.shape[0], pos.shape[1]
        if aev_out is None:
            aev_out = torch.zeros((batch, n, self.length), dtype=torch.float32, device=pos.device)
        keep, bp = _box(box)
        _check(lib().aev_forward_range(self._h, _dev_ptr(pos, torch.float32, "pos"),
                                       _dev_ptr(species, torch.int32, "species"), bp, n, batch, int(first), int(count),
                                       _dev_ptr(aev_out, torch.float32, "aev_out"), _stream(stream)),
               "aev_forward_range")
        return aev_out

    def aev_backward(self, grad_aev, forces_out=None, stream=None):
        import torch
        if forces_out is None:
            forces_out = torch.empty(grad_aev.shape[:2] + (3,), dtype=torch.float32, device=grad_aev.device)
        _check(lib().aev_backward(self._h, _dev_ptr(grad_aev, torch.float32, "grad_aev"),
                                  _dev_ptr(forces_out, torch.float32, "forces_out"), _stream(stream)),
               "aev_backward")
        return forces_out

    @staticmethod
    def _net_args(weights, biases):
        ws = [np.ascontiguousarray(w, dtype=np.float32) for w in weights]
        bs = [np.ascontiguousarray(b, dtype=np.float32) for b in biases]
        dims = (C.c_int32 * (len(ws) + 1))(*([ws[0].shape[0]] + [w.shape[1] for w in ws]))
        fpp = C.POINTER(C.c_float)
        wp = (fpp * len(ws))(*[w.ctypes.data_as(fpp) for w in ws])
        bp = (fpp * len(bs))(*[b.ctypes.data_as(fpp) for b in bs])
        return ws, bs, dims, wp, bp

    def ani_mlp_load(self, species: int, weights: Sequence[np.ndarray], biases: Sequence[np.ndarray],
                     celu_alpha: float):
        ws, bs, dims, wp, bp = self._net_args(weights, biases)
        _check(lib().ani_mlp_load(self._h, int(species), len(ws), dims, wp, bp, float(celu_alpha)),
               "ani_mlp_load")

    def mlp_kernel(self) -> str:
        """'tcgen05' or 'fp32': the kernel ani_energy_forces runs for the loaded networks."""
        rc = int(lib().ani_mlp_kernel(self._h))
        _check(min(rc, 0), "ani_mlp_kernel")
        return "tcgen05" if rc == 1 else "fp32"

    def ani_mlp_set_ensemble(self, n_models: int):
        _check(lib().ani_mlp_set_ensemble(self._h, int(n_models)), "ani_mlp_set_ensemble")

    def ani_mlp_load_model(self, model: int, species: int, weights: Sequence[np.ndarray],
                           biases: Sequence[np.ndarray], celu_alpha: float):
        ws, bs, dims, wp, bp = self._net_args(weights, biases)
        _check(lib().ani_mlp_load_model(self._h, int(model), int(species), len(ws), dims, wp, bp,
                                        float(celu_alpha)), "ani_mlp_load_model")

    def ani_energy_forces(self, pos, species, box=None, energy_out=None, forces_out=None, stream=None):
        import torch
        batch, n = pos.shape[0], pos.shape[1]
        if energy_out is None:
            energy_out = torch.empty((batch,), dtype=torch.float64, device=pos.device)
        if forces_out is None:
            forces_out = torch.empty((batch, n, 3), dtype=torch.float32, device=pos.device)
        keep, bp = _box(box)
        _check(lib().ani_energy_forces(self._h, _dev_ptr(pos, torch.float32, "pos"),
                                       _dev_ptr(species, torch.int32, "species"), bp, n, batch,
                                       _dev_ptr(energy_out, torch.float64, "energy_out"),
                                       _dev_ptr(forces_out, torch.float32, "forces_out"),
                                       _stream(stream)), "ani_energy_forces")
        return energy_out, forces_out

    def ani_energy_forces_subset(self, pos_all, ml_index, species_ml, forces_all, box=None, energy_out=None,
                                 stream=None):
        """ML region of a mixed system: forces_all[ml_index] += F_ml (in place); returns the energy tensor."""
        import torch
        if energy_out is None:
            energy_out = torch.empty((1,), dtype=torch.float64, device=pos_all.device)
        keep, bp = _box(box)
        _check(lib().ani_energy_forces_subset(self._h, _dev_ptr(pos_all, torch.float32, "pos_all"),
                                              _dev_ptr(ml_index, torch.int32, "ml_index"),
                                              _dev_ptr(species_ml, torch.int32, "species_ml"), bp,
                                              int(ml_index.numel()),
                                              _dev_ptr(energy_out, torch.float64, "energy_out"),
                                              _dev_ptr(forces_all, torch.float32, "forces_all"),
                                              _stream(stream)), "ani_energy_forces_subset")
        return energy_out

    # -- host-buffer calls (numpy in / out; synchronous)
    def aev_forward_backward_host(self, pos: np.ndarray, species: np.ndarray, box, grad_aev: Optional[np.ndarray],
                                  aev_out: Optional[np.ndarray] = None, forces_out: Optional[np.ndarray] = None):
        batch, n = pos.shape[0], pos.shape[1]
        assert pos.dtype == np.float32 and pos.flags.c_contiguous
        assert species.dtype == np.int32 and species.flags.c_contiguous
        keep, bp = _box(box)
        if aev_out is None:
            aev_out = np.empty((batch, n, self.length), dtype=np.float32)
        gp = None
        if grad_aev is not None:
            assert grad_aev.dtype == np.float32 and grad_aev.flags.c_contiguous
            gp = grad_aev.ctypes.data
            if forces_out is None:
                forces_out = np.empty((batch, n, 3), dtype=np.float32)
        _check(lib().aev_forward_backward_host(self._h, pos.ctypes.data, species.ctypes.data, bp, n, batch,
                                               gp, aev_out.ctypes.data,
                                               None if forces_out is None else forces_out.ctypes.data),
               "aev_forward_backward_host")
        return aev_out, forces_out

    def ani_energy_forces_host(self, pos: np.ndarray, species: np.ndarray, box):
        batch, n = pos.shape[0], pos.shape[1]
        assert pos.dtype == np.float32 and pos.flags.c_contiguous
        assert species.dtype == np.int32 and species.flags.c_contiguous
        keep, bp = _box(box)
        energy = np.empty((batch,), dtype=np.float64)
        forces = np.empty((batch, n, 3), dtype=np.float32)
        _check(lib().ani_energy_forces_host(self._h, pos.ctypes.data, species.ctypes.data, bp, n, batch,
                                            energy.ctypes.data, forces.ctypes.data),
               "ani_energy_forces_host")
        return energy, forces

    # -- diagnostics
    def aev_export_pairs(self, which: int, cap: int):
        """Returns the (i<j) pairs of the last neighbour build as a sorted int32 [count,2] array."""
        import torch
        out = torch.empty((max(cap, 1), 2), dtype=torch.int32, device="cuda:%d" % self.device)
        cnt = C.c_int64(0)
        _check(lib().aev_export_pairs(self._h, int(which), out.data_ptr(), int(cap), C.byref(cnt)),
               "aev_export_pairs")
        if cnt.value > cap:
            return self.aev_export_pairs(which, int(cnt.value))
        arr = out[: cnt.value].cpu().numpy()
        order = np.lexsort((arr[:, 1], arr[:, 0]))
        return arr[order]

    def aev_export_counts(self, batch: int, n_atoms: int):
        """(angular, radial-only) neighbour counts per atom, int32 [batch, n_atoms, 2] on the device."""
        import torch
        out = torch.empty((batch, n_atoms, 2), dtype=torch.int32, device="cuda:%d" % self.device)
        _check(lib().aev_export_counts(self._h, out.data_ptr()), "aev_export_counts")
        return out

    def aev_set_profiling(self, enable: bool):
        _check(lib().aev_set_profiling(self._h, int(bool(enable))), "aev_set_profiling")

    def aev_get_profile(self):
        """{kernel: (total ms, launches)} since the last call (syncs)."""
        ms = (C.c_double * 6)()
        n = (C.c_int64 * 6)()
        _check(lib().aev_get_profile(self._h, ms, n), "aev_get_profile")
        names = ("bin", "fout", "aev", "backward", "nbr", "mlp")
        return {k: (float(ms[i]), int(n[i])) for i, k in enumerate(names)}

    def aev_status(self) -> int:
        return int(lib().aev_status(self._h))

    def check_status(self):
        _check(self.aev_status(), "aev_status")

    def neighbor_builds(self) -> int:
        out = C.c_int64(0)
        _check(lib().aev_neighbor_builds(self._h, C.byref(out)), "aev_neighbor_builds")
        return int(out.value)

    def launch_count(self) -> int:
        return int(lib().aev_launch_count(self._h))


def aev_pairs_static(pos, species, rc: float, pairs_out, count_out, stream=None) -> None:
    """Pair search of one non-periodic system without any device allocation (include/aev.h, aev_pairs_static).

    For callers that must not allocate on the GPU (the device belongs to their own pool, their step loop cannot
    take the synchronisation cudaMalloc brings, or their footprint is fixed at link time): no context, and the
    library's working memory is a fixed array inside the .so.  So this wrapper allocates nothing either - the
    caller brings every buffer: `pos` f32 [n, 3], `species` i32 [n] or None, `pairs_out` i32 [cap, 2],
    `count_out` i64 [1], all CUDA tensors on one device.  On return (asynchronously, on the current stream)
    `count_out[0]` pairs (i < j, r < rc) sit in `pairs_out`, sorted by (i, j).  n > AEV_STATIC_MAX_ATOMS raises
    AevError(AEV_ERR_STATIC_LIMIT).  One call per GPU at a time: all calls on a device share that array.
    """
    import torch
    n = int(pos.shape[0])
    if pos.dim() != 2 or pos.shape[1] != 3:
        raise TypeError("pos must be [n_atoms, 3]")
    sp = None if species is None else _dev_ptr(species, torch.int32, "species")
    cap = int(pairs_out.shape[0])
    _check(lib().aev_pairs_static(_dev_ptr(pos, torch.float32, "pos"), sp, n, float(rc),
                                  _dev_ptr(pairs_out, torch.int32, "pairs_out"), cap,
                                  _dev_ptr(count_out, torch.int64, "count_out"), int(pos.device.index or 0),
                                  _stream(stream)), "aev_pairs_static")


def probe_fp32_tflops(device: int = 0) -> float:
    out = C.c_double(0.0)
    _check(lib().aev_probe_fp32_tflops(int(device), C.byref(out)), "aev_probe_fp32_tflops")
    return float(out.value)
