"""Thin ctypes binding of include/nnp.h (argument marshalling only; every step runs in the CUDA kernels).

Names follow the header: create / compute / compute_host / status / destroy and the debug exports.
There is no CPU fallback: if libnnp_b200.so is missing or no sm_100 GPU is present this raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libnnp_b200.so")

NNP_OK = 0
NNP_FLAG_NO_GRAPH = 1
NNP_FLAG_NO_UMMA = 4
NNP_FLAG_NO_SMALL = 8
NNP_FLAG_NO_MID = 16
NNP_FLAG_NO_PDL = 32
NNP_FLAG_NO_CELLS = 64
NNP_FLAG_FORCE_CELLS = 128
NNP_FLAG_NO_FWD1 = 256
NNP_FLAG_NO_SWEEP_REVERSAL = 512
NNP_FLAG_NO_NBR_FUSION = 1024
NNP_FLAG_NO_ZERO_SKIP = 2048
NNP_FLAG_UMMA_PAIRS = 4096
NNP_FLAG_NO_TAIL_SPLIT = 8192
ERRORS = {
    -1: "NNP_ERR_INVALID_ARG",
    -2: "NNP_ERR_CUDA",
    -3: "NNP_ERR_UNSUPPORTED_ARCH",
    -4: "NNP_ERR_CAPACITY",
    -5: "NNP_ERR_NONFINITE",
    -6: "NNP_ERR_ALLOC",
    -7: "NNP_ERR_STATIC_LIMIT",
}

# every symbol include/nnp.h declares (tests check the library exports exactly these)
SYMBOLS = (
    "nnp_create", "nnp_compute", "nnp_compute_host", "nnp_status", "nnp_destroy", "nnp_error_string",
    "nnp_launches_per_compute", "nnp_set_profiling", "nnp_get_stage_times", "nnp_stage_name", "nnp_get_work",
    "nnp_debug_pairs", "nnp_debug_aev", "nnp_debug_atomic_energies", "nnp_debug_daev", "nnp_n_features",
    "nnp_get_stage_work", "nnp_get_stage_bytes", "nnp_create_from_file", "nnp_compute_fixed", "nnp_compute_async", "nnp_measure_peaks",
    "nnp_coupling_create", "nnp_coupling_compute", "nnp_coupling_compute_fixed", "nnp_coupling_destroy",
    "nnp_coupling_static_init", "nnp_coupling_compute_static",
)
FIXED_ONE = float(1 << 32)  # 64-bit fixed-point force format: round(F * 2^32)


class NNPError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {ERRORS.get(code, code)}")


class _Config(C.Structure):
    _fields_ = [
        ("n_species", C.c_int32),
        ("n_models", C.c_int32),
        ("rc_radial", C.c_float),
        ("rc_angular", C.c_float),
        ("eta_r", C.c_float),
        ("n_shf_r", C.c_int32),
        ("shf_r", C.POINTER(C.c_float)),
        ("eta_a", C.c_float),
        ("zeta", C.c_float),
        ("n_shf_a", C.c_int32),
        ("shf_a", C.POINTER(C.c_float)),
        ("n_shf_z", C.c_int32),
        ("shf_z", C.POINTER(C.c_float)),
        ("cos_scale", C.c_float),
        ("celu_alpha", C.c_float),
        ("n_layers", C.c_int32),
        ("layer_dims", C.POINTER(C.c_int32)),
        ("weights", C.POINTER(C.c_void_p)),
        ("biases", C.POINTER(C.c_void_p)),
        ("self_energy", C.POINTER(C.c_double)),
        ("energy_scale", C.c_double),
        ("length_scale", C.c_double),
        ("max_radial_neighbors", C.c_int32),
        ("max_angular_neighbors", C.c_int32),
        ("flags", C.c_int32),
    ]


_lib = None


def load_library():
    """dlopen libnnp_b200.so (built in-tree by paper_2201_08110_b200.build); raises if missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(
                f"{LIB_PATH} not built: run `python -m paper_2201_08110_b200.build` (there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        lib.nnp_create.restype = C.c_int
        lib.nnp_create.argtypes = [C.POINTER(C.c_void_p), C.POINTER(_Config), C.c_int32, C.c_void_p, C.c_int32,
                                   C.c_void_p]
        lib.nnp_compute.restype = C.c_int
        lib.nnp_compute.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32,
                                    C.c_void_p]
        lib.nnp_compute_host.restype = C.c_int
        lib.nnp_compute_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        lib.nnp_status.restype = C.c_int
        lib.nnp_status.argtypes = [C.c_void_p]
        lib.nnp_destroy.restype = None
        lib.nnp_destroy.argtypes = [C.c_void_p]
        lib.nnp_error_string.restype = C.c_char_p
        lib.nnp_error_string.argtypes = [C.c_int]
        lib.nnp_launches_per_compute.restype = C.c_int
        lib.nnp_launches_per_compute.argtypes = [C.c_void_p]
        lib.nnp_set_profiling.restype = C.c_int
        lib.nnp_set_profiling.argtypes = [C.c_void_p, C.c_int32]
        lib.nnp_get_stage_times.restype = C.c_int
        lib.nnp_get_stage_times.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.POINTER(C.c_int32)]
        lib.nnp_stage_name.restype = C.c_char_p
        lib.nnp_stage_name.argtypes = [C.c_void_p, C.c_int32]
        lib.nnp_get_work.restype = C.c_int
        lib.nnp_get_work.argtypes = [C.c_void_p, C.c_void_p, C.c_int32]
        lib.nnp_debug_pairs.restype = C.c_int
        lib.nnp_debug_pairs.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_int64), C.c_void_p, C.c_int64]
        for name in ("nnp_debug_aev", "nnp_debug_atomic_energies", "nnp_debug_daev"):
            getattr(lib, name).restype = C.c_int
            getattr(lib, name).argtypes = [C.c_void_p, C.c_void_p]
        lib.nnp_n_features.restype = C.c_int
        lib.nnp_n_features.argtypes = [C.c_void_p]
        lib.nnp_get_stage_work.restype = C.c_int
        lib.nnp_get_stage_work.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_int32)]
        lib.nnp_get_stage_bytes.restype = C.c_int
        lib.nnp_get_stage_bytes.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_double)]
        lib.nnp_create_from_file.restype = C.c_int
        lib.nnp_create_from_file.argtypes = [C.POINTER(C.c_void_p), C.c_char_p, C.c_int32, C.c_void_p, C.c_int32, C.c_void_p,
                                             C.c_int32, C.c_double, C.c_int32]
        lib.nnp_compute_fixed.restype = C.c_int
        lib.nnp_compute_fixed.argtypes = lib.nnp_compute.argtypes
        lib.nnp_compute_async.restype = C.c_int
        lib.nnp_compute_async.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32,
                                          C.c_int32, C.c_void_p, C.c_void_p]
        lib.nnp_measure_peaks.restype = C.c_int
        lib.nnp_measure_peaks.argtypes = [C.c_void_p, C.c_int32]
        lib.nnp_coupling_create.restype = C.c_int
        lib.nnp_coupling_create.argtypes = [C.POINTER(C.c_void_p), C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                            C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double,
                                            C.c_double, C.c_double]
        for name in ("nnp_coupling_compute", "nnp_coupling_compute_fixed"):
            getattr(lib, name).restype = C.c_int
            getattr(lib, name).argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p]
        lib.nnp_coupling_static_init.restype = C.c_int
        lib.nnp_coupling_static_init.argtypes = []
        lib.nnp_coupling_compute_static.restype = C.c_int
        lib.nnp_coupling_compute_static.argtypes = [C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32,
                                                    C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_double,
                                                    C.c_double, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_int32,
                                                    C.c_void_p]
        lib.nnp_coupling_destroy.restype = None
        lib.nnp_coupling_destroy.argtypes = [C.c_void_p]
        _lib = lib
    return _lib


def _check(rc: int, where: str):
    if rc != NNP_OK:
        raise NNPError(rc, where)


class NNP:
    """One nnp_handle: a fixed set of NNP atoms + one model."""

    def __init__(self, params, weights, biases, species, mol_offsets=None, self_energy=None, energy_scale=None,
                 length_scale: float = 1.0, max_radial_neighbors: int = 0, max_angular_neighbors: int = 0,
                 flags: int = 0):
        self.lib = load_library()
        S = int(params.n_species)
        M = len(weights)
        dims = np.ascontiguousarray(params.layer_dims, dtype=np.int32)
        L = dims.shape[1] - 1
        keep = []
        f32 = lambda v: np.ascontiguousarray(v, dtype=np.float32)
        shf_r, shf_a, shf_z = f32(params.shf_r), f32(params.shf_a), f32(params.shf_z)
        wptr = (C.c_void_p * (M * S * L))()
        bptr = (C.c_void_p * (M * S * L))()
        for m in range(M):
            for e in range(S):
                for l in range(L):
                    idx = (m * S + e) * L + l
                    w = f32(weights[m][e][l])
                    assert w.shape == (dims[e, l + 1], dims[e, l])
                    keep.append(w)
                    wptr[idx] = w.ctypes.data
                    if biases is not None:
                        b = f32(biases[m][e][l])
                        keep.append(b)
                        bptr[idx] = b.ctypes.data
        fp = lambda a: a.ctypes.data_as(C.POINTER(C.c_float))
        cfg = _Config()
        cfg.n_species, cfg.n_models = S, M
        cfg.rc_radial, cfg.rc_angular = float(params.rc_radial), float(params.rc_angular)
        cfg.eta_r, cfg.n_shf_r, cfg.shf_r = float(params.eta_r), shf_r.size, fp(shf_r)
        cfg.eta_a, cfg.zeta = float(params.eta_a), float(params.zeta)
        cfg.n_shf_a, cfg.shf_a, cfg.n_shf_z, cfg.shf_z = shf_a.size, fp(shf_a), shf_z.size, fp(shf_z)
        cfg.cos_scale, cfg.celu_alpha = float(params.cos_scale), float(params.celu_alpha)
        cfg.n_layers, cfg.layer_dims = L, dims.ctypes.data_as(C.POINTER(C.c_int32))
        cfg.weights = C.cast(wptr, C.POINTER(C.c_void_p))
        cfg.biases = C.cast(bptr, C.POINTER(C.c_void_p)) if biases is not None else None
        se = None
        if self_energy is not None:
            se = np.ascontiguousarray(self_energy, dtype=np.float64)
            cfg.self_energy = se.ctypes.data_as(C.POINTER(C.c_double))
        cfg.energy_scale = float(params.energy_scale if energy_scale is None else energy_scale)
        cfg.length_scale = float(length_scale)
        cfg.max_radial_neighbors, cfg.max_angular_neighbors, cfg.flags = max_radial_neighbors, max_angular_neighbors, flags
        spc = np.ascontiguousarray(species, dtype=np.int32)
        self.n_atoms = int(spc.size)
        off = None
        self.n_molecules = 1
        if mol_offsets is not None:
            off = np.ascontiguousarray(mol_offsets, dtype=np.int32)
            self.n_molecules = int(off.size - 1)
        self.n_models = M
        h = C.c_void_p()
        rc = self.lib.nnp_create(C.byref(h), C.byref(cfg), self.n_atoms, spc.ctypes.data if spc.size else None,
                                 self.n_molecules, off.ctypes.data if off is not None else None)
        _check(rc, "nnp_create")
        self.h = h
        self.n_features = int(self.lib.nnp_n_features(self.h))

    @classmethod
    def from_file(cls, path: str, atomic_numbers, mol_offsets=None, n_models_to_use: int = 0, length_scale: float = 1.0,
                  flags: int = 0):
        """nnp_create_from_file: a handle from a parameter file; atoms are named by atomic number."""
        self = cls.__new__(cls)
        self.lib = load_library()
        z = np.ascontiguousarray(atomic_numbers, dtype=np.int32)
        self.n_atoms = int(z.size)
        off = None
        self.n_molecules = 1
        if mol_offsets is not None:
            off = np.ascontiguousarray(mol_offsets, dtype=np.int32)
            self.n_molecules = int(off.size - 1)
        h = C.c_void_p()
        rc = self.lib.nnp_create_from_file(C.byref(h), os.fsencode(path), self.n_atoms, z.ctypes.data if z.size else None,
                                           self.n_molecules, off.ctypes.data if off is not None else None,
                                           int(n_models_to_use), float(length_scale), int(flags))
        _check(rc, "nnp_create_from_file")
        self.h = h
        self.n_features = int(self.lib.nnp_n_features(self.h))
        self.n_models = int(n_models_to_use) if n_models_to_use else read_parameter_file_header(path)["n_models"]
        return self

    # ---- the hot path
    def compute_fixed(self, d_pos: int, pos_stride: int, d_atom_index, d_energy: int, d_force_fixed, force_stride: int,
                      stream: int = 0):
        """nnp_compute_fixed: forces added as round(F * 2^32) into an int64 buffer with integer atomics."""
        _check(self.lib.nnp_compute_fixed(self.h, d_pos, pos_stride, d_atom_index, d_energy, d_force_fixed, force_stride,
                                          stream or None), "nnp_compute_fixed")

    def compute_async(self, d_pos: int, pos_stride: int, d_atom_index, d_energy: int, d_force, force_stride: int,
                      fixed: bool, wait_event=None, done_event=None):
        """nnp_compute_async: on the library's own stream, ordered by CUDA events (raw cudaEvent_t values)."""
        _check(self.lib.nnp_compute_async(self.h, d_pos, pos_stride, d_atom_index, d_energy, d_force, force_stride,
                                          1 if fixed else 0, wait_event, done_event), "nnp_compute_async")

    def compute(self, d_pos: int, pos_stride: int, d_atom_index, d_energy: int, d_force, force_stride: int,
                stream: int = 0):
        """nnp_compute with raw device addresses (ints)."""
        _check(self.lib.nnp_compute(self.h, d_pos, pos_stride, d_atom_index, d_energy, d_force, force_stride,
                                    stream or None), "nnp_compute")

    def compute_torch(self, pos, energy, force=None, atom_index=None, stream=None):
        """nnp_compute on torch CUDA tensors (device memory + stream plumbing only)."""
        import torch

        assert pos.is_cuda and pos.dtype == torch.float32 and pos.stride(-1) == 1
        assert energy.is_cuda and energy.dtype == torch.float64
        s = torch.cuda.current_stream().cuda_stream if stream is None else stream
        self.compute(pos.data_ptr(), int(pos.stride(0)), atom_index.data_ptr() if atom_index is not None else None,
                     energy.data_ptr(), force.data_ptr() if force is not None else None,
                     int(force.stride(0)) if force is not None else 3, s)

    def compute_host(self, pos_host: np.ndarray, stream: int = 0):
        """nnp_compute_host: host positions in, host (E f64[n_mol], F f32[N,3]) out."""
        pos = np.ascontiguousarray(pos_host, dtype=np.float32)
        E = np.empty(self.n_molecules, dtype=np.float64)
        F = np.empty((self.n_atoms, 3), dtype=np.float32)
        _check(self.lib.nnp_compute_host(self.h, pos.ctypes.data, E.ctypes.data, F.ctypes.data, stream or None),
               "nnp_compute_host")
        return E, F

    def compute_host_into(self, pos_ptr: int, e_ptr: int, f_ptr: int, stream: int = 0):
        _check(self.lib.nnp_compute_host(self.h, pos_ptr, e_ptr, f_ptr, stream or None), "nnp_compute_host")

    def status(self) -> int:
        return int(self.lib.nnp_status(self.h))

    def check(self):
        _check(self.status(), "nnp_status")

    # ---- measurement helpers
    @property
    def launches_per_compute(self) -> int:
        return int(self.lib.nnp_launches_per_compute(self.h))

    def set_profiling(self, on: bool):
        _check(self.lib.nnp_set_profiling(self.h, 1 if on else 0), "nnp_set_profiling")

    def stage_times(self):
        n = C.c_int32()
        _check(self.lib.nnp_get_stage_times(self.h, None, 0, C.byref(n)), "nnp_get_stage_times")
        ms = np.zeros(n.value, dtype=np.float32)
        _check(self.lib.nnp_get_stage_times(self.h, ms.ctypes.data, n.value, C.byref(n)), "nnp_get_stage_times")
        names = [self.lib.nnp_stage_name(self.h, k).decode() for k in range(n.value)]
        return dict(zip(names, ms.tolist()))

    def stage_work(self):
        """{stage name: (flops issued by a tensor-engine launch, its atom-tile width)}; (0, 0) for other stages."""
        n = C.c_int32()
        _check(self.lib.nnp_get_stage_times(self.h, None, 0, C.byref(n)), "nnp_get_stage_times")
        out = {}
        for k in range(n.value):
            fl, tile = C.c_double(), C.c_int32()
            _check(self.lib.nnp_get_stage_work(self.h, k, C.byref(fl), C.byref(tile)), "nnp_get_stage_work")
            out[self.lib.nnp_stage_name(self.h, k).decode()] = (fl.value, tile.value)
        return out

    def stage_bytes(self):
        """{stage name: algorithmic bytes of a tensor-engine launch (operands, outputs, epilogue reads, each once)}."""
        n = C.c_int32()
        _check(self.lib.nnp_get_stage_times(self.h, None, 0, C.byref(n)), "nnp_get_stage_times")
        out = {}
        for k in range(n.value):
            b = C.c_double()
            _check(self.lib.nnp_get_stage_bytes(self.h, k, C.byref(b)), "nnp_get_stage_bytes")
            out[self.lib.nnp_stage_name(self.h, k).decode()] = b.value
        return out

    def work(self):
        w = np.zeros(4, dtype=np.float64)
        _check(self.lib.nnp_get_work(self.h, w.ctypes.data, 4), "nnp_get_work")
        return {"weight_bytes": w[0], "mlp_flops": w[1], "aev_bytes": w[2], "layer1_weight_bytes": w[3]}

    # ---- debug / parity exports
    def debug_pairs(self, which: str = "radial") -> np.ndarray:
        w = 0 if which == "radial" else 1
        n = C.c_int64()
        _check(self.lib.nnp_debug_pairs(self.h, w, C.byref(n), None, 0), "nnp_debug_pairs")
        ij = np.empty((max(n.value, 1), 2), dtype=np.int32)
        _check(self.lib.nnp_debug_pairs(self.h, w, C.byref(n), ij.ctypes.data, n.value), "nnp_debug_pairs")
        return ij[: n.value]

    def debug_aev(self) -> np.ndarray:
        out = np.empty((self.n_atoms, self.n_features), dtype=np.float32)
        _check(self.lib.nnp_debug_aev(self.h, out.ctypes.data), "nnp_debug_aev")
        return out

    def debug_daev(self) -> np.ndarray:
        out = np.empty((self.n_atoms, self.n_features), dtype=np.float32)
        _check(self.lib.nnp_debug_daev(self.h, out.ctypes.data), "nnp_debug_daev")
        return out

    def debug_atomic_energies(self) -> np.ndarray:
        out = np.empty((self.n_models, self.n_atoms), dtype=np.float64)
        _check(self.lib.nnp_debug_atomic_energies(self.h, out.ctypes.data), "nnp_debug_atomic_energies")
        return out

    def destroy(self):
        if getattr(self, "h", None) is not None and self.h:
            self.lib.nnp_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def measure_peaks():
    """nnp_measure_peaks: dict of what the device sustains (FP32 FFMA, tcgen05 TF32, L2 reads, DRAM reads)."""
    lib = load_library()
    out = np.zeros(4, dtype=np.float64)
    _check(lib.nnp_measure_peaks(out.ctypes.data, 4), "nnp_measure_peaks")
    return {"fp32_ffma_tflops": float(out[0]), "tf32_tcgen05_tflops": float(out[1]), "l2_read_gbs": float(out[2]),
            "dram_read_gbs": float(out[3])}


COUPLING_STATIC_MAX_NNP = 128    # NNP_COUPLING_STATIC_MAX_NNP
COUPLING_STATIC_MAX_MM = 65536   # NNP_COUPLING_STATIC_MAX_MM


def coupling_static_init():
    """nnp_coupling_static_init: resolve the static scratch array's device address for the current device."""
    _check(load_library().nnp_coupling_static_init(), "nnp_coupling_static_init")


def coupling_compute_static(n_nnp: int, d_nnp_rows, d_q_nnp, d_sigma_nnp, d_eps_nnp, n_mm: int, d_mm_rows, d_q_mm,
                            d_sigma_mm, d_eps_mm, coulomb_const: float, cutoff: float, length_scale: float, d_pos: int,
                            pos_stride: int, d_energy, d_force, force_stride: int, stream: int = 0):
    """nnp_coupling_compute_static with raw device addresses (ints or None): Eq. 4 without any allocation."""
    _check(load_library().nnp_coupling_compute_static(
        int(n_nnp), d_nnp_rows, d_q_nnp, d_sigma_nnp, d_eps_nnp, int(n_mm), d_mm_rows, d_q_mm, d_sigma_mm, d_eps_mm,
        float(coulomb_const), float(cutoff), float(length_scale), d_pos, int(pos_stride), d_energy, d_force,
        int(force_stride), stream or None), "nnp_coupling_compute_static")


class Coupling:
    """One nnp_coupling handle: the NNP-MM coupling term of mechanical embedding (Eq. 4)."""

    def __init__(self, nnp_rows, q_nnp, sigma_nnp, eps_nnp, mm_rows, q_mm, sigma_mm, eps_mm, coulomb_const: float,
                 cutoff: float = 0.0, length_scale: float = 1.0):
        self.lib = load_library()
        i32 = lambda v: np.ascontiguousarray(v, dtype=np.int32)
        f32 = lambda v: np.ascontiguousarray(v, dtype=np.float32)
        a = [i32(nnp_rows), f32(q_nnp), f32(sigma_nnp), f32(eps_nnp), i32(mm_rows), f32(q_mm), f32(sigma_mm), f32(eps_mm)]
        self.n_nnp, self.n_mm = int(a[0].size), int(a[4].size)
        p = [x.ctypes.data if x.size else None for x in a]
        h = C.c_void_p()
        _check(self.lib.nnp_coupling_create(C.byref(h), self.n_nnp, p[0], p[1], p[2], p[3], self.n_mm, p[4], p[5], p[6],
                                            p[7], float(coulomb_const), float(cutoff), float(length_scale)),
               "nnp_coupling_create")
        self.h = h

    def compute(self, d_pos: int, pos_stride: int, d_energy, d_force, force_stride: int, stream: int = 0, fixed: bool = False):
        fn = self.lib.nnp_coupling_compute_fixed if fixed else self.lib.nnp_coupling_compute
        _check(fn(self.h, d_pos, pos_stride, d_energy, d_force, force_stride, stream or None), "nnp_coupling_compute")

    def destroy(self):
        if getattr(self, "h", None) is not None and self.h:
            self.lib.nnp_coupling_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


# ------------------------------------------------------------------------------------------------
# parameter files (format: csrc/params_file.cu).  Pure byte marshalling: nothing of the method is computed here.
PARAM_MAGIC = b"NNPB200P"


def write_parameter_file(path: str, params, weights, biases, atomic_numbers, self_energy=None, energy_scale=None):
    """Write an ANI-style parameter set (any species order: `atomic_numbers[s]` is the element of species s)."""
    S = int(params.n_species)
    M = len(weights)
    dims = np.ascontiguousarray(params.layer_dims, dtype="<i4")
    L = dims.shape[1] - 1
    z = np.ascontiguousarray(atomic_numbers, dtype="<i4")
    assert z.size == S
    se = np.zeros(S, "<f8") if self_energy is None else np.ascontiguousarray(self_energy, dtype="<f8")
    f4 = lambda v: np.ascontiguousarray(v, dtype="<f4")
    with open(path, "wb") as f:
        f.write(PARAM_MAGIC)
        f.write(np.array([1, S, M, L], "<i4").tobytes())
        f.write(f4([params.rc_radial, params.rc_angular, params.eta_r, params.eta_a, params.zeta, params.cos_scale,
                    params.celu_alpha]).tobytes())
        f.write(np.array([params.shf_r.size, params.shf_a.size, params.shf_z.size], "<i4").tobytes())
        f.write(np.array([params.energy_scale if energy_scale is None else energy_scale], "<f8").tobytes())
        f.write(z.tobytes())
        for v in (params.shf_r, params.shf_a, params.shf_z):
            f.write(f4(v).tobytes())
        f.write(dims.tobytes())
        f.write(se.tobytes())
        for m in range(M):
            for e in range(S):
                for l in range(L):
                    w = f4(weights[m][e][l])
                    assert w.shape == (dims[e, l + 1], dims[e, l])
                    f.write(w.tobytes())
                    b = np.zeros(dims[e, l + 1], "<f4") if biases is None else f4(biases[m][e][l])
                    f.write(b.tobytes())


def read_parameter_file_header(path: str):
    with open(path, "rb") as f:
        assert f.read(8) == PARAM_MAGIC
        version, S, M, L = np.frombuffer(f.read(16), "<i4")
    return {"version": int(version), "n_species": int(S), "n_models": int(M), "n_layers": int(L)}
