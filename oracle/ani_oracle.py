"""ctypes wrapper around oracle/ani_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
import this.  It imports nothing from the CUDA package; inputs are plain numpy arrays
(the same seeded arrays the CUDA path receives).  float32 inputs are widened to float64
here, bit-exactly, before the C code sees them (SURVEY.md 8(c) "Inputs").
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ani_oracle.c")
_LIB = os.path.join(_HERE, "libani_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (float64, no FMA contraction, OpenMP over centre atoms)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC",
               _SRC, "-o", tmp, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


class _Params(C.Structure):
    _fields_ = [
        ("n_species", C.c_int),
        ("n_models", C.c_int),
        ("rc_r", C.c_double),
        ("rc_a", C.c_double),
        ("eta_r", C.c_double),
        ("n_shf_r", C.c_int),
        ("shf_r", C.POINTER(C.c_double)),
        ("eta_a", C.c_double),
        ("zeta", C.c_double),
        ("n_shf_a", C.c_int),
        ("shf_a", C.POINTER(C.c_double)),
        ("n_shf_z", C.c_int),
        ("shf_z", C.POINTER(C.c_double)),
        ("cos_scale", C.c_double),
        ("celu_alpha", C.c_double),
        ("n_layers", C.c_int),
        ("layer_dims", C.POINTER(C.c_int)),
        ("weights", C.POINTER(C.c_void_p)),
        ("biases", C.POINTER(C.c_void_p)),
        ("self_energy", C.POINTER(C.c_double)),
        ("energy_scale", C.c_double),
    ]


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        lib.ani_n_features.restype = C.c_int
        lib.ani_oracle_threads.restype = C.c_int
        lib.ani_pairs.restype = C.c_long
        lib.ani_energy_forces.restype = C.c_int
        lib.ani_aev.restype = None
        lib.ani_mlp.restype = None
        _lib = lib
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int))


class AniOracle:
    """float64 oracle for one parameter set + ensemble weights.

    params: any object with the attribute names of workloads.AniParams (values are widened).
    weights/biases: nested lists [m][e][l] of f32 arrays [out][in] / [out]; biases may be None.
    """

    def __init__(self, params, weights, biases=None, self_energy=None, energy_scale=None):
        self.lib = _load()
        self.n_species = int(params.n_species)
        self.n_models = len(weights)
        dims = np.ascontiguousarray(params.layer_dims, dtype=np.int32)
        self.n_layers = dims.shape[1] - 1
        self._keep = []
        f64 = lambda v: np.ascontiguousarray(np.asarray(v, dtype=np.float32).astype(np.float64))
        shf_r, shf_a, shf_z = f64(params.shf_r), f64(params.shf_a), f64(params.shf_z)
        nw = self.n_models * self.n_species * self.n_layers
        wptr = (C.c_void_p * nw)()
        bptr = (C.c_void_p * nw)()
        for m in range(self.n_models):
            for e in range(self.n_species):
                for l in range(self.n_layers):
                    idx = (m * self.n_species + e) * self.n_layers + l
                    w = np.ascontiguousarray(weights[m][e][l], dtype=np.float32)
                    assert w.shape == (dims[e, l + 1], dims[e, l]), (w.shape, dims[e])
                    self._keep.append(w)
                    wptr[idx] = w.ctypes.data
                    if biases is not None:
                        b = np.ascontiguousarray(biases[m][e][l], dtype=np.float32)
                        assert b.shape == (dims[e, l + 1],)
                        self._keep.append(b)
                        bptr[idx] = b.ctypes.data
                    else:
                        bptr[idx] = None
        se = None
        if self_energy is not None:
            se = np.ascontiguousarray(self_energy, dtype=np.float64)
        self._keep += [dims, shf_r, shf_a, shf_z, wptr, bptr, se]
        wf = lambda v: float(np.float64(np.float32(v)))
        p = _Params()
        p.n_species, p.n_models = self.n_species, self.n_models
        p.rc_r, p.rc_a = wf(params.rc_radial), wf(params.rc_angular)
        p.eta_r, p.n_shf_r, p.shf_r = wf(params.eta_r), shf_r.size, _dp(shf_r)
        p.eta_a, p.zeta = wf(params.eta_a), wf(params.zeta)
        p.n_shf_a, p.shf_a, p.n_shf_z, p.shf_z = shf_a.size, _dp(shf_a), shf_z.size, _dp(shf_z)
        p.cos_scale, p.celu_alpha = wf(params.cos_scale), wf(params.celu_alpha)
        p.n_layers, p.layer_dims = self.n_layers, _ip(dims)
        p.weights = C.cast(wptr, C.POINTER(C.c_void_p))
        p.biases = C.cast(bptr, C.POINTER(C.c_void_p))
        p.self_energy = _dp(se) if se is not None else None
        p.energy_scale = float(params.energy_scale if energy_scale is None else energy_scale)
        self.p = p
        self.rc_r, self.rc_a = p.rc_r, p.rc_a
        self.n_features = int(self.lib.ani_n_features(C.byref(p)))

    @property
    def threads(self) -> int:
        return int(self.lib.ani_oracle_threads())

    @staticmethod
    def _prep(pos, species, mol_offsets):
        pos = np.asarray(pos)
        assert pos.ndim == 2 and pos.shape[1] == 3
        pos64 = np.ascontiguousarray(pos.astype(np.float64))  # exact widening for f32 input
        spc = np.ascontiguousarray(species, dtype=np.int32)
        n = pos64.shape[0]
        off = np.array([0, n], np.int32) if mol_offsets is None else np.ascontiguousarray(mol_offsets, dtype=np.int32)
        return pos64, spc, off, n

    def pairs(self, pos, which: str = "radial", mol_offsets=None) -> np.ndarray:
        """O2: sorted array of (i,j), i<j, with D2 <= Rc^2, same molecule."""
        pos64, _, off, n = self._prep(pos, np.zeros(len(pos), np.int32), mol_offsets)
        rc = self.rc_r if which == "radial" else self.rc_a
        cnt = self.lib.ani_pairs(n, _dp(pos64), off.size - 1, _ip(off), C.c_double(rc), None, C.c_long(0))
        ij = np.empty((max(cnt, 1), 2), dtype=np.int32)
        self.lib.ani_pairs(n, _dp(pos64), off.size - 1, _ip(off), C.c_double(rc), _ip(ij), C.c_long(cnt))
        return ij[:cnt]

    def aev(self, pos, species, mol_offsets=None) -> np.ndarray:
        """O3+O4: f64[N][n_features]."""
        pos64, spc, off, n = self._prep(pos, species, mol_offsets)
        G = np.empty((n, self.n_features), dtype=np.float64)
        self.lib.ani_aev(C.byref(self.p), n, _dp(pos64), _ip(spc), off.size - 1, _ip(off), _dp(G))
        return G

    def mlp(self, G, species):
        """O5: (e f64[M][n] in model units, dG f64[n][nf] = (1/M) sum_m de^(m)/dG)."""
        G = np.ascontiguousarray(G, dtype=np.float64)
        spc = np.ascontiguousarray(species, dtype=np.int32)
        n = G.shape[0]
        e = np.empty((self.n_models, n), dtype=np.float64)
        dG = np.empty_like(G)
        self.lib.ani_mlp(C.byref(self.p), n, _ip(spc), _dp(G), _dp(e), _dp(dG))
        return e, dG

    def energy_forces(self, pos, species, mol_offsets=None, want_intermediates: bool = False):
        """O1-O7.  Returns dict(E f64[n_mol], F f64[N][3] [, G, e_atom f64[M][N], dG])."""
        pos64, spc, off, n = self._prep(pos, species, mol_offsets)
        E = np.empty(off.size - 1, dtype=np.float64)
        F = np.empty((n, 3), dtype=np.float64)
        out = {"E": E, "F": F}
        G = e = dG = None
        if want_intermediates:
            G = np.empty((n, self.n_features), dtype=np.float64)
            e = np.empty((self.n_models, n), dtype=np.float64)
            dG = np.empty((n, self.n_features), dtype=np.float64)
            out.update(G=G, e_atom=e, dG=dG)
        rc = self.lib.ani_energy_forces(
            C.byref(self.p), n, _dp(pos64), _ip(spc), off.size - 1, _ip(off), _dp(E), _dp(F),
            _dp(G) if G is not None else None, _dp(e) if e is not None else None,
            _dp(dG) if dG is not None else None)
        if rc != 0:
            raise ValueError("oracle: bad species or molecule offsets")
        return out

    def energy(self, pos, species, mol_offsets=None) -> np.ndarray:
        """Energy only (used by the finite-difference pin; accepts f64 positions as they are)."""
        pos64, spc, off, n = self._prep(pos, species, mol_offsets)
        E = np.empty(off.size - 1, dtype=np.float64)
        rc = self.lib.ani_energy_forces(C.byref(self.p), n, _dp(pos64), _ip(spc), off.size - 1, _ip(off), _dp(E),
                                        None, None, None, None)
        if rc != 0:
            raise ValueError("oracle: bad species or molecule offsets")
        return E
