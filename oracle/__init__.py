"""TEST INFRASTRUCTURE — ctypes access to the fp64 CPU oracle (oracle/tdpd_oracle.c).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  The product (paper_1611_06163_b200) never does, and fails loudly without its CUDA
library.  Nothing here is shared with the CUDA path.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tdpd_oracle.c")
_LIB = os.path.join(_HERE, "libtdpd_oracle.so")
T, S = 4, 10


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=gnu11", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


class Params(C.Structure):
    _fields_ = [("n_types", C.c_int32), ("n_species", C.c_int32), ("box", C.c_double * 3),
                ("r_c", C.c_double), ("r_cc", C.c_double), ("dt", C.c_double), ("kBT", C.c_double),
                ("rho", C.c_double), ("a", C.c_double * (T * T)), ("gamma", C.c_double * (T * T)),
                ("s_R", C.c_double * (T * T)), ("kappa", C.c_double * (S * T * T)), ("s_c", C.c_double * S),
                ("m_s", C.c_double * S), ("body_force", C.c_double * 3), ("body_mode", C.c_int32),
                ("seed", C.c_uint64), ("exclude_same_cell_membrane_pairs", C.c_int32),
                ("source", C.c_double * (S * T)), ("decay", C.c_double * (S * T))]


class RbcParams(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("p", "x0", "m", "gamma_T", "gamma_C", "k_g", "k_l", "k_v", "k_b",
                                          "theta0", "VR_over_AR32")]


def make_params(p: dict) -> Params:
    """Workload parameter dict (fp32 values) -> oracle struct (the same values, widened to fp64)."""
    P = Params()
    P.n_types, P.n_species = int(p["n_types"]), int(p["n_species"])
    for k in ("r_c", "r_cc", "dt", "kBT", "rho"):
        setattr(P, k, float(np.float32(p[k])))
    for k, n in (("box", 3), ("a", T * T), ("gamma", T * T), ("s_R", T * T), ("kappa", S * T * T), ("s_c", S),
                 ("m_s", S), ("body_force", 3)):
        arr = np.asarray(p[k], dtype=np.float32).astype(np.float64).ravel()
        assert arr.size == n, k
        getattr(P, k)[:] = arr.tolist()
    for k in ("source", "decay"):
        if k in p:
            arr = np.asarray(p[k], dtype=np.float32).astype(np.float64).ravel()
            assert arr.size == S * T, k
            getattr(P, k)[:] = arr.tolist()
    P.body_mode = int(p["body_mode"])
    P.seed = int(p["seed"])
    P.exclude_same_cell_membrane_pairs = int(p["exclude_same_cell_membrane_pairs"])
    return P


def make_rbc_params(rp: dict) -> RbcParams:
    R = RbcParams()
    for k, _ in RbcParams._fields_:
        setattr(R, k, float(np.float32(rp[k])))
    return R


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        vp, i32, i64, u32, u64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_uint32, C.c_uint64, C.c_double
        P = C.POINTER
        L.orc_create.restype = vp
        L.orc_create.argtypes = [P(Params)]
        L.orc_load_particles.argtypes = [vp, i64, vp, vp, vp, vp]
        L.orc_add_rbc_mesh.restype = i32
        L.orc_add_rbc_mesh.argtypes = [vp, i32, vp, vp, vp, i32, vp, P(RbcParams), i32]
        L.orc_set_params.argtypes = [vp, P(Params)]
        L.orc_set_brute.argtypes = [vp, i32]
        L.orc_set_lagged_area_volume.argtypes = [vp, i32]
        L.orc_n.restype = i64
        L.orc_n.argtypes = [vp]
        L.orc_step_count.restype = i64
        L.orc_step_count.argtypes = [vp]
        L.orc_set_state.argtypes = [vp, vp, vp, vp]
        L.orc_get_state.argtypes = [vp, vp, vp, vp, vp, vp, vp]
        L.orc_compute_forces.argtypes = [vp, i64]
        L.orc_step.argtypes = [vp, i32]
        L.orc_get_census_totals.argtypes = [vp, vp]
        L.orc_get_rbc_stats.argtypes = [vp, vp, vp, vp, vp]
        L.orc_rbc_topology.restype = i32
        L.orc_rbc_topology.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp]
        L.orc_destroy.argtypes = [vp]
        L.orc_philox4x32_10.argtypes = [vp, vp, vp]
        L.orc_gauss4.argtypes = [i64, i64, i64, u32, u64, vp]
        L.orc_pair_terms.restype = i32
        L.orc_pair_terms.argtypes = [P(Params), i64, i64, i32, i32, vp, vp, vp, vp, i64, vp, vp]
        L.orc_bond_terms.argtypes = [dbl, dbl, P(RbcParams), dbl, dbl, vp, vp, vp, vp, vp, vp]
        L.orc_dihedral_terms.restype = dbl
        L.orc_dihedral_terms.argtypes = [dbl, dbl, vp, vp, vp, vp, vp]
        L.orc_bin_fp32.argtypes = [vp, C.c_float, i64, vp, vp, vp]
        L.orc_neighbor_census.argtypes = [vp, vp, vp, vp, vp, vp]
        L.orc_philox_batch.argtypes = [i64, vp, vp, vp]
        L.orc_gauss_batch.argtypes = [i64, vp, vp, i64, u32, u64, vp]
        L.orc_pair_forces_subset.argtypes = [vp, i64, i64, vp, vp, vp]
        L.orc_num_threads.restype = i32
        L.orc_set_threads.argtypes = [i32]
        _lib = L
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float32)


class Oracle:
    """One simulation.  Mirrors the C-ABI of the product (load / add mesh / step / get_state)."""

    def __init__(self, params: dict, brute: bool = False):
        self.L = lib()
        self.p = params
        self.ns = int(params["n_species"])
        self._P = make_params(params)
        self.h = C.c_void_p(self.L.orc_create(C.byref(self._P)))
        self.n_rbc = 0
        self._rbc_nv = []
        self._rbc_ntri = []
        if brute:
            self.L.orc_set_brute(self.h, 1)

    @classmethod
    def from_workload(cls, w, brute: bool = False) -> "Oracle":
        o = cls(w.params, brute=brute)
        o.load_particles(w.pos, w.vel, w.type, w.conc)
        for r in w.rbcs:
            o.add_rbc_mesh(r["verts"], r["vel"], r["conc"], r["tris"], w.rbc_params)
        return o

    def __del__(self):
        try:
            self.L.orc_destroy(self.h)
        except Exception:
            pass

    @property
    def n(self) -> int:
        return int(self.L.orc_n(self.h))

    @property
    def step_count(self) -> int:
        return int(self.L.orc_step_count(self.h))

    def set_params(self, params: dict):
        self.p = params
        self._P = make_params(params)
        self.L.orc_set_params(self.h, C.byref(self._P))

    def load_particles(self, pos, vel, type_, conc):
        if len(pos) == 0:
            return
        pos, vel, conc = _f32(pos), _f32(vel), _f32(conc)
        conc = None if conc is None else np.ascontiguousarray(conc.reshape(len(pos), -1)[:, :self.ns])
        ty = None if type_ is None else np.ascontiguousarray(type_, dtype=np.int32)
        self.L.orc_load_particles(self.h, len(pos), _ptr(pos), _ptr(vel), _ptr(ty), _ptr(conc))

    def add_rbc_mesh(self, verts, vel, conc, tris, rp: dict, mtype: int = 2) -> int:
        verts, vel, conc = _f32(verts), _f32(vel), _f32(conc)
        conc = None if conc is None else np.ascontiguousarray(conc.reshape(len(verts), -1)[:, :self.ns])
        tris = np.ascontiguousarray(tris, dtype=np.int32)
        R = make_rbc_params(rp)
        k = self.L.orc_add_rbc_mesh(self.h, len(verts), _ptr(verts), _ptr(vel), _ptr(conc), len(tris), _ptr(tris),
                                    C.byref(R), mtype)
        if k < 0:
            raise ValueError("mesh is not a closed, consistently oriented manifold")
        self.n_rbc += 1
        self._rbc_nv.append(len(verts))
        self._rbc_ntri.append(len(tris))
        return k

    def set_lagged_area_volume(self, on: bool):
        """PAPER.md:156 variant: K-Apply with the previous step's area / volume."""
        self.L.orc_set_lagged_area_volume(self.h, int(on))

    def compute_forces(self, step: int):
        self.L.orc_compute_forces(self.h, step)

    def step(self, n: int = 1):
        self.L.orc_step(self.h, n)

    def set_state(self, x=None, v=None, C_=None):
        f = lambda a: None if a is None else np.ascontiguousarray(a, dtype=np.float64)
        x, v, C_ = f(x), f(v), f(C_)
        self.L.orc_set_state(self.h, _ptr(x), _ptr(v), _ptr(C_))

    def get_state(self, forces: bool = True) -> dict:
        n, ns = self.n, self.ns
        out = dict(pos=np.empty((n, 3)), vel=np.empty((n, 3)), conc=np.empty((n, ns)))
        if forces:
            out.update(force_pair=np.empty((n, 3)), force_bonded=np.empty((n, 3)), flux=np.empty((n, ns)))
        self.L.orc_get_state(self.h, _ptr(out["pos"]), _ptr(out["vel"]), _ptr(out["conc"]),
                             _ptr(out.get("force_pair")), _ptr(out.get("force_bonded")), _ptr(out.get("flux")))
        if forces:
            out["force"] = out["force_pair"] + out["force_bonded"]
        out["step"] = self.step_count
        return out

    def pair_forces_subset(self, step: int, ids):
        ids = np.ascontiguousarray(ids, dtype=np.int64)
        F, Q = np.zeros((len(ids), 3)), np.zeros((len(ids), self.ns))
        self.L.orc_pair_forces_subset(self.h, step, len(ids), _ptr(ids), _ptr(F), _ptr(Q))
        return F, Q

    def census_totals(self) -> dict:
        t = np.zeros(3, np.int64)
        self.L.orc_get_census_totals(self.h, _ptr(t))
        return dict(n_cand=int(t[0]), n_cc=int(t[1]), n_c=int(t[2]))

    def rbc_stats(self) -> dict:
        m = self.n_rbc
        out = {k: np.zeros(m) for k in ("area", "volume", "A0", "V0")}
        self.L.orc_get_rbc_stats(self.h, _ptr(out["area"]), _ptr(out["volume"]), _ptr(out["A0"]), _ptr(out["V0"]))
        return out

    def rbc_topology(self, m: int) -> dict:
        nb = C.c_int32(0)
        self.L.orc_rbc_topology(self.h, m, C.byref(nb), None, None, None, None, None)
        nb = nb.value
        out = dict(bond=np.zeros((nb, 2), np.int32), dih=np.zeros((nb, 4), np.int32), h0=np.zeros(nb), kp=np.zeros(nb),
                   A0t=np.zeros(self._rbc_ntri[m]))
        nbr = C.c_int32(0)
        self.L.orc_rbc_topology(self.h, m, C.byref(nbr), _ptr(out["bond"]), _ptr(out["dih"]), _ptr(out["h0"]),
                                _ptr(out["kp"]), _ptr(out["A0t"]))
        return out

    def neighbor_census(self) -> dict:
        n = self.n
        out = dict(n_rc=np.zeros(n, np.int32), n_rcc=np.zeros(n, np.int32), xor_rc=np.zeros(n, np.uint32),
                   xor_rcc=np.zeros(n, np.uint32), margin=np.zeros(n))
        self.L.orc_neighbor_census(self.h, _ptr(out["n_rc"]), _ptr(out["n_rcc"]), _ptr(out["xor_rc"]),
                                   _ptr(out["xor_rcc"]), _ptr(out["margin"]))
        return out


# ---- stand-alone term functions (used by the pins) -------------------------------------------------

def philox4x32_10(ctr, key) -> np.ndarray:
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32)
    key = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros(4, np.uint32)
    lib().orc_philox4x32_10(_ptr(ctr), _ptr(key), _ptr(out))
    return out


def philox_batch(ctr, key) -> np.ndarray:
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    key = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros_like(ctr)
    lib().orc_philox_batch(len(ctr), _ptr(ctr), _ptr(key), _ptr(out))
    return out


def gauss_batch(id_i, id_j, step: int, tag: int, seed: int) -> np.ndarray:
    id_i = np.ascontiguousarray(id_i, dtype=np.int64)
    id_j = np.ascontiguousarray(id_j, dtype=np.int64)
    g = np.zeros((len(id_i), 4))
    lib().orc_gauss_batch(len(id_i), _ptr(id_i), _ptr(id_j), step, tag, seed, _ptr(g))
    return g


def gauss4(id_i: int, id_j: int, step: int, tag: int, seed: int) -> np.ndarray:
    g = np.zeros(4)
    lib().orc_gauss4(id_i, id_j, step, tag, seed, _ptr(g))
    return g


def pair_terms(params: dict, id_i, id_j, ti, tj, d, dv, Ci, Cj, step):
    P = make_params(params)
    d, dv = np.ascontiguousarray(d, np.float64), np.ascontiguousarray(dv, np.float64)
    Ci, Cj = np.ascontiguousarray(Ci, np.float64), np.ascontiguousarray(Cj, np.float64)
    F, Q = np.zeros(3), np.zeros(S)
    kind = lib().orc_pair_terms(C.byref(P), id_i, id_j, ti, tj, _ptr(d), _ptr(dv), _ptr(Ci), _ptr(Cj), step,
                                _ptr(F), _ptr(Q))
    return kind, F, Q[:int(params["n_species"])]


def bond_terms(kBT, dt, rp: dict, h0, kp, d, dv, N):
    R = make_rbc_params(rp)
    d, dv, N = (np.ascontiguousarray(a, np.float64) for a in (d, dv, N))
    Fc, Fd, Fr = np.zeros(3), np.zeros(3), np.zeros(3)
    lib().orc_bond_terms(kBT, dt, C.byref(R), h0, kp, _ptr(d), _ptr(dv), _ptr(N), _ptr(Fc), _ptr(Fd), _ptr(Fr))
    return Fc, Fd, Fr


def dihedral_terms(k_b, theta0, r1, r2, r3, r4):
    r = [np.ascontiguousarray(a, np.float64) for a in (r1, r2, r3, r4)]
    F = np.zeros(12)
    th = lib().orc_dihedral_terms(k_b, theta0, _ptr(r[0]), _ptr(r[1]), _ptr(r[2]), _ptr(r[3]), _ptr(F))
    return th, F.reshape(4, 3)


def bin_fp32(box, r_cc, pos):
    box = np.ascontiguousarray(box, np.float32)
    pos = np.ascontiguousarray(pos, np.float32)
    cells = np.zeros((len(pos), 3), np.int32)
    nc = np.zeros(3, np.int32)
    lib().orc_bin_fp32(_ptr(box), C.c_float(float(np.float32(r_cc))), len(pos), _ptr(pos), _ptr(cells), _ptr(nc))
    return cells, nc


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_threads(n: int):
    lib().orc_set_threads(int(n))
