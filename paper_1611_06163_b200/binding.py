"""Thin ctypes binding of libtdpd.so (include/tdpd.h).  Argument marshalling only: every step of the path runs in
the library's CUDA kernels.  PyTorch supplies the workspace (device memory) and the two CUDA streams.

There is no CPU fallback: importing works without a GPU (so the symbol table can be checked), but creating a
simulation without the built library or without a CUDA device raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtdpd.so")
MAX_TYPES, MAX_SPECIES, N_TIMERS = 4, 10, 7
TIMER_NAMES = ("integrate", "sort", "reorder", "pair", "membrane", "closing_kick", "nlist")
OK, EINVAL, ESTATE, ENOMEM, ECUDA, EUNSTABLE = 0, -1, -2, -3, -4, -5

# every symbol include/tdpd.h declares
SYMBOLS = (
    "tdpd_create", "tdpd_load_particles", "tdpd_add_rbc_mesh", "tdpd_workspace_bytes", "tdpd_set_workspace",
    "tdpd_set_params", "tdpd_set_state", "tdpd_step", "tdpd_sync", "tdpd_get_state", "tdpd_get_forces_split",
    "tdpd_num_particles", "tdpd_num_rbc", "tdpd_get_rbc_stats", "tdpd_get_rbc_topology", "tdpd_debug_get_binning",
    "tdpd_debug_neighbor_census", "tdpd_debug_pair_census", "tdpd_debug_set_run_meta", "tdpd_debug_rng", "tdpd_debug_box_muller", "tdpd_host_grid", "tdpd_set_timing", "tdpd_get_timing", "tdpd_measure_peaks", "tdpd_launch_count",
    "tdpd_set_tuning", "tdpd_set_neighbor_list", "tdpd_set_membrane_variant", "tdpd_get_neighbor_list_stats", "tdpd_set_graph", "tdpd_last_error", "tdpd_destroy",
    "tdpd_noalloc_init", "tdpd_sort_cells_noalloc", "tdpd_noalloc_last_error",
)


class TdpdError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libtdpd error {code}: {msg}")
        self.code = code


class Params(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_types", C.c_int32), ("n_species", C.c_int32),
                ("box", C.c_float * 3), ("r_c", C.c_float), ("r_cc", C.c_float), ("dt", C.c_float),
                ("kBT", C.c_float), ("rho", C.c_float),
                ("a", C.c_float * (MAX_TYPES * MAX_TYPES)), ("gamma", C.c_float * (MAX_TYPES * MAX_TYPES)),
                ("s_R", C.c_float * (MAX_TYPES * MAX_TYPES)),
                ("kappa", C.c_float * (MAX_SPECIES * MAX_TYPES * MAX_TYPES)),
                ("s_c", C.c_float * MAX_SPECIES), ("m_s", C.c_float * MAX_SPECIES),
                ("body_force", C.c_float * 3), ("body_mode", C.c_int32), ("seed", C.c_uint64),
                ("exclude_same_cell_membrane_pairs", C.c_int32), ("reserved", C.c_int32),
                ("source", C.c_float * (MAX_SPECIES * MAX_TYPES)), ("decay", C.c_float * (MAX_SPECIES * MAX_TYPES))]


class RbcParams(C.Structure):
    _fields_ = [(k, C.c_float) for k in ("p", "x0", "m", "gamma_T", "gamma_C", "k_g", "k_l", "k_v", "k_b", "theta0",
                                         "VR_over_AR32")]


class Peaks(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("fp32_fma_tflops", "fp32_fma2_tflops", "l2_read_gbs", "hbm_read_gbs")] \
        + [("n_sm", C.c_int32), ("reserved", C.c_int32)]


def measure_peaks(device: int = 0) -> dict:
    """Measured FP32 / L2 / HBM peaks of the device (tdpd_measure_peaks): the roofline denominators of bench.py."""
    L = load_library()
    pk = Peaks()
    rc = L.tdpd_measure_peaks(int(device), C.byref(pk))
    if rc != OK:
        raise TdpdError(rc, "tdpd_measure_peaks failed")
    return {k: getattr(pk, k) for k, _ in Peaks._fields_ if k != "reserved"}


NOALLOC_MAX_N = 262144  # TDPD_NOALLOC_MAX_N


def noalloc_init() -> None:
    """tdpd_noalloc_init: looks up the fixed sort scratch on the current CUDA device (call before a stream capture)."""
    L = load_library()
    rc = L.tdpd_noalloc_init()
    if rc != OK:
        raise TdpdError(rc, L.tdpd_noalloc_last_error().decode())


def sort_cells_noalloc(d_keys: int, d_vals: int, n: int, key_bits: int, d_keys_out: int, d_vals_out: int,
                       stream: int = 0) -> None:
    """tdpd_sort_cells_noalloc: stable radix sort of n (key, value) pairs given as DEVICE addresses (ints; d_vals = 0
    for the values 0 .. n-1), scratch in a fixed device array of the library, no allocation; enqueues on `stream`."""
    L = load_library()
    rc = L.tdpd_sort_cells_noalloc(C.c_void_p(d_keys), C.c_void_p(d_vals or None), int(n), int(key_bits),
                                   C.c_void_p(d_keys_out), C.c_void_p(d_vals_out), C.c_void_p(stream or None))
    if rc != OK:
        raise TdpdError(rc, L.tdpd_noalloc_last_error().decode())


def make_params(p: dict) -> Params:
    P = Params()
    P.struct_size = C.sizeof(Params)
    P.n_types, P.n_species = int(p["n_types"]), int(p["n_species"])
    for k in ("r_c", "r_cc", "dt", "kBT", "rho"):
        setattr(P, k, float(np.float32(p[k])))
    for k, n in (("box", 3), ("a", 16), ("gamma", 16), ("s_R", 16), ("kappa", MAX_SPECIES * 16), ("s_c", MAX_SPECIES), ("m_s", MAX_SPECIES),
                 ("body_force", 3)):
        arr = np.asarray(p[k], dtype=np.float32).ravel()
        if arr.size != n:
            raise ValueError(f"parameter {k}: expected {n} values, got {arr.size}")
        getattr(P, k)[:] = arr.tolist()
    for k in ("source", "decay"):   # optional: Q^S (zero when absent)
        if k in p:
            arr = np.asarray(p[k], dtype=np.float32).ravel()
            if arr.size != MAX_SPECIES * MAX_TYPES:
                raise ValueError(f"parameter {k}: expected {MAX_SPECIES * MAX_TYPES} values, got {arr.size}")
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


def load_library() -> C.CDLL:
    """Loads libtdpd.so (built in-tree by paper_1611_06163_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_1611_06163_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i32, i64, u32, sz = C.c_void_p, C.c_int32, C.c_int64, C.c_uint32, C.c_size_t
    P = C.POINTER
    L.tdpd_create.argtypes = [P(Params), C.c_int, vp, vp, P(vp)]
    L.tdpd_load_particles.argtypes = [vp, i64, vp, vp, vp, vp]
    L.tdpd_add_rbc_mesh.argtypes = [vp, i32, vp, vp, vp, i32, vp, P(RbcParams), i32, P(i32)]
    L.tdpd_workspace_bytes.argtypes = [vp, P(sz)]
    L.tdpd_set_workspace.argtypes = [vp, vp, sz]
    L.tdpd_set_params.argtypes = [vp, P(Params)]
    L.tdpd_set_state.argtypes = [vp, vp, vp, vp]
    L.tdpd_step.argtypes = [vp, i32]
    L.tdpd_sync.argtypes = [vp]
    L.tdpd_get_state.argtypes = [vp, vp, vp, vp, vp, vp, P(i64)]
    L.tdpd_get_forces_split.argtypes = [vp, vp, vp]
    L.tdpd_num_particles.argtypes = [vp]
    L.tdpd_num_particles.restype = i64
    L.tdpd_num_rbc.argtypes = [vp]
    L.tdpd_num_rbc.restype = i32
    L.tdpd_get_rbc_stats.argtypes = [vp, vp, vp, vp, vp]
    L.tdpd_get_rbc_topology.argtypes = [vp, i32, P(i32), vp, vp, vp, vp, vp]
    L.tdpd_debug_get_binning.argtypes = [vp, vp, vp, vp, vp]
    L.tdpd_debug_neighbor_census.argtypes = [vp, vp, vp, vp, vp]
    L.tdpd_debug_pair_census.argtypes = [vp, vp, vp, vp, vp]
    L.tdpd_debug_set_run_meta.argtypes = [vp, u32, u32]
    L.tdpd_debug_rng.argtypes = [vp, i64, vp, vp, i64, u32, vp, vp]
    L.tdpd_debug_box_muller.argtypes = [vp, i64, vp, vp]
    L.tdpd_host_grid.argtypes = [P(Params), vp, P(u32), vp, vp, vp, vp]
    L.tdpd_set_timing.argtypes = [vp, i32]
    L.tdpd_get_timing.argtypes = [vp, vp, vp]
    L.tdpd_measure_peaks.argtypes = [C.c_int, P(Peaks)]
    L.tdpd_launch_count.argtypes = [vp]
    L.tdpd_launch_count.restype = i64
    L.tdpd_set_tuning.argtypes = [vp, i32, i32, i32]
    L.tdpd_set_neighbor_list.argtypes = [vp, C.c_float, i32]
    L.tdpd_get_neighbor_list_stats.argtypes = [vp, P(i64), P(i64), P(i32), P(i32)]
    L.tdpd_set_membrane_variant.argtypes = [vp, i32]
    L.tdpd_set_graph.argtypes = [vp, i32]
    L.tdpd_last_error.argtypes = [vp]
    L.tdpd_last_error.restype = C.c_char_p
    L.tdpd_destroy.argtypes = [vp]
    L.tdpd_noalloc_init.argtypes = []
    L.tdpd_sort_cells_noalloc.argtypes = [vp, vp, i64, i32, vp, vp, vp]
    L.tdpd_noalloc_last_error.argtypes = []
    L.tdpd_noalloc_last_error.restype = C.c_char_p
    for name in SYMBOLS:
        getattr(L, name)  # AttributeError if the library does not export a declared symbol
    _lib = L
    return L


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float32)


def host_grid(params: dict) -> dict:
    """Static grid tables of the pair kernel (host-only; needs the built library, not a GPU)."""
    L = load_library()
    Pm = make_params(params)
    nc = np.zeros(3, np.int32)
    nr = C.c_uint32(0)
    rc = L.tdpd_host_grid(C.byref(Pm), _ptr(nc), C.byref(nr), None, None, None, None)
    if rc != OK:
        raise TdpdError(rc, "tdpd_host_grid: bad parameters")
    ncells = int(nc.prod())
    o = dict(ncell=nc, cell_rank=np.zeros(ncells, np.uint32), seg_off=np.zeros(ncells + 1, np.uint32),
             seg_first=np.zeros(nr.value, np.uint32), seg_meta=np.zeros(nr.value, np.uint32))
    L.tdpd_host_grid(C.byref(Pm), _ptr(nc), C.byref(nr), _ptr(o["cell_rank"]), _ptr(o["seg_off"]), _ptr(o["seg_first"]),
                     _ptr(o["seg_meta"]))
    return o


class Simulation:
    """One tDPD + RBC simulation on one GPU.  Methods mirror the C ABI one to one."""

    def __init__(self, params: dict, device: int = 0, pair_threads: int = 0, list_cap: int = 0,
                 pair_split: int = 0, skin: float = 0.0, nlist_cap: int = 0,
                 single_stream: bool = False):
        import torch

        self.L = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1611_06163_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self.torch = torch
        self.device = int(device)
        self.p = params
        self.ns = int(params["n_species"])
        self._P = make_params(params)
        with torch.cuda.device(self.device):
            self.stream_pair = torch.cuda.Stream(device=self.device)
            # membrane kernel on its own, higher-priority stream (single_stream: on the pair stream, to measure the overlap)
            self.stream_bonded = self.stream_pair if single_stream else torch.cuda.Stream(device=self.device, priority=-1)
        h = C.c_void_p()
        rc = self.L.tdpd_create(C.byref(self._P), self.device, C.c_void_p(self.stream_pair.cuda_stream),
                                C.c_void_p(self.stream_bonded.cuda_stream), C.byref(h))
        if rc != OK:
            raise TdpdError(rc, "tdpd_create failed (bad parameters or no CUDA device)")
        self.h = h
        self.workspace = None
        self._ntri = []
        if pair_threads or list_cap or pair_split:
            self._ck(self.L.tdpd_set_tuning(self.h, pair_threads, list_cap, pair_split))
        if skin or nlist_cap:
            self._ck(self.L.tdpd_set_neighbor_list(self.h, float(skin), int(nlist_cap)))

    def _ck(self, rc):
        if rc != OK:
            raise TdpdError(rc, self.L.tdpd_last_error(self.h).decode())

    @classmethod
    def from_workload(cls, w, device: int = 0, **kw) -> "Simulation":
        s = cls(w.params, device=device, **kw)
        s.load_particles(w.pos, w.vel, w.type, w.conc)
        for r in w.rbcs:
            s.add_rbc_mesh(r["verts"], r["vel"], r["conc"], r["tris"], w.rbc_params)
        s.finalize()
        return s

    def close(self):
        if getattr(self, "h", None):
            self.L.tdpd_destroy(self.h)
            self.h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def n(self) -> int:
        return int(self.L.tdpd_num_particles(self.h))

    @property
    def n_rbc(self) -> int:
        return int(self.L.tdpd_num_rbc(self.h))

    def load_particles(self, pos, vel=None, type_=None, conc=None):
        pos, vel, conc = _f32(pos), _f32(vel), _f32(conc)
        n = 0 if pos is None else len(pos)
        if n == 0:
            return
        if conc is not None:
            conc = np.ascontiguousarray(conc.reshape(n, -1)[:, :self.ns])
        ty = None if type_ is None else np.ascontiguousarray(type_, dtype=np.int32)
        self._ck(self.L.tdpd_load_particles(self.h, n, _ptr(pos), _ptr(vel), _ptr(ty), _ptr(conc)))

    def add_rbc_mesh(self, verts, vel, conc, tris, rp: dict, mtype: int = 2) -> int:
        verts, vel, conc = _f32(verts), _f32(vel), _f32(conc)
        if conc is not None:
            conc = np.ascontiguousarray(conc.reshape(len(verts), -1)[:, :self.ns])
        tris = np.ascontiguousarray(tris, dtype=np.int32)
        R = make_rbc_params(rp)
        k = C.c_int32(-1)
        self._ck(self.L.tdpd_add_rbc_mesh(self.h, len(verts), _ptr(verts), _ptr(vel), _ptr(conc), len(tris),
                                          _ptr(tris), C.byref(R), mtype, C.byref(k)))
        self._ntri.append(len(tris))
        return int(k.value)

    def finalize(self):
        """Allocates the workspace through torch and uploads the system."""
        nbytes = C.c_size_t(0)
        self._ck(self.L.tdpd_workspace_bytes(self.h, C.byref(nbytes)))
        self.workspace = self.torch.empty(int(nbytes.value) + 256, dtype=self.torch.uint8,
                                          device=f"cuda:{self.device}")
        base = (self.workspace.data_ptr() + 255) & ~255
        self._ck(self.L.tdpd_set_workspace(self.h, C.c_void_p(base), nbytes))

    def set_params(self, params: dict):
        self.p = params
        self._P = make_params(params)
        self._ck(self.L.tdpd_set_params(self.h, C.byref(self._P)))

    def set_state(self, pos=None, vel=None, conc=None):
        pos, vel, conc = _f32(pos), _f32(vel), _f32(conc)
        self._ck(self.L.tdpd_set_state(self.h, _ptr(pos), _ptr(vel), _ptr(conc)))

    def step(self, n: int = 1):
        self._ck(self.L.tdpd_step(self.h, int(n)))

    def sync(self):
        self._ck(self.L.tdpd_sync(self.h))

    def get_state(self, forces: bool = True, out: dict | None = None) -> dict:
        n, ns = self.n, self.ns
        o = out if out is not None else {}
        for k, w in (("pos", 3), ("vel", 3), ("conc", ns)) + ((("force", 3), ("flux", ns)) if forces else ()):
            if k not in o:
                o[k] = np.empty((n, w), np.float32)
        st = C.c_int64(0)
        self._ck(self.L.tdpd_get_state(self.h, _ptr(o["pos"]), _ptr(o["vel"]), _ptr(o["conc"]), _ptr(o.get("force")),
                                       _ptr(o.get("flux")), C.byref(st)))
        o["step"] = int(st.value)
        return o

    def get_forces_split(self):
        fp, fb = np.empty((self.n, 3), np.float32), np.empty((self.n, 3), np.float32)
        self._ck(self.L.tdpd_get_forces_split(self.h, _ptr(fp), _ptr(fb)))
        return fp, fb

    def rbc_stats(self) -> dict:
        m = self.n_rbc
        o = {k: np.zeros(m) for k in ("area", "volume", "A0", "V0")}
        self._ck(self.L.tdpd_get_rbc_stats(self.h, _ptr(o["area"]), _ptr(o["volume"]), _ptr(o["A0"]), _ptr(o["V0"])))
        return o

    def rbc_topology(self, m: int) -> dict:
        nb = C.c_int32(0)
        self._ck(self.L.tdpd_get_rbc_topology(self.h, m, C.byref(nb), None, None, None, None, None))
        nb = nb.value
        o = dict(bond=np.zeros((nb, 2), np.int32), dih=np.zeros((nb, 4), np.int32), h0=np.zeros(nb, np.float32),
                 kp=np.zeros(nb, np.float32), A0t=np.zeros(self._ntri[m], np.float32))
        self._ck(self.L.tdpd_get_rbc_topology(self.h, m, None, _ptr(o["bond"]), _ptr(o["dih"]), _ptr(o["h0"]),
                                              _ptr(o["kp"]), _ptr(o["A0t"])))
        return o

    def debug_binning(self) -> dict:
        nc = np.zeros(3, np.int32)
        self._ck(self.L.tdpd_debug_get_binning(self.h, None, _ptr(nc), None, None))
        o = dict(cell_xyz=np.zeros((self.n, 3), np.int32), ncell=nc, cell_count=np.zeros(int(nc.prod()), np.int32),
                 sorted_id=np.zeros(self.n, np.int32))
        self._ck(self.L.tdpd_debug_get_binning(self.h, _ptr(o["cell_xyz"]), _ptr(nc), _ptr(o["cell_count"]),
                                               _ptr(o["sorted_id"])))
        return o

    def debug_neighbor_census(self) -> dict:
        n = self.n
        o = dict(n_rc=np.zeros(n, np.int32), n_rcc=np.zeros(n, np.int32), xor_rc=np.zeros(n, np.uint32),
                 xor_rcc=np.zeros(n, np.uint32))
        self._ck(self.L.tdpd_debug_neighbor_census(self.h, _ptr(o["n_rc"]), _ptr(o["n_rcc"]), _ptr(o["xor_rc"]),
                                                   _ptr(o["xor_rcc"])))
        return o

    def debug_pair_census(self) -> dict:
        n = self.n
        o = dict(n_front=np.zeros(n, np.int32), n_ring=np.zeros(n, np.int32), xor_front=np.zeros(n, np.uint32),
                 xor_ring=np.zeros(n, np.uint32))
        self._ck(self.L.tdpd_debug_pair_census(self.h, _ptr(o["n_front"]), _ptr(o["n_ring"]), _ptr(o["xor_front"]),
                                               _ptr(o["xor_ring"])))
        return o

    def debug_set_run_meta(self, run_index: int, meta: int):
        self._ck(self.L.tdpd_debug_set_run_meta(self.h, int(run_index), int(meta)))

    def debug_rng(self, id_i, id_j, step: int, tag: int):
        id_i = np.ascontiguousarray(id_i, np.int64)
        id_j = np.ascontiguousarray(id_j, np.int64)
        w = np.zeros((len(id_i), 4), np.uint32)
        g = np.zeros((len(id_i), 4), np.float32)
        self._ck(self.L.tdpd_debug_rng(self.h, len(id_i), _ptr(id_i), _ptr(id_j), step, tag, _ptr(w), _ptr(g)))
        return w, g

    def neighbor_list_stats(self) -> dict:
        a, b, c, d = C.c_int64(0), C.c_int64(0), C.c_int32(0), C.c_int32(0)
        self._ck(self.L.tdpd_get_neighbor_list_stats(self.h, C.byref(a), C.byref(b), C.byref(c), C.byref(d)))
        return dict(rebuilds=int(a.value), evaluations=int(b.value), list_cap=int(c.value), max_entries=int(d.value))

    def debug_box_muller(self, words):
        words = np.ascontiguousarray(words, np.uint32).reshape(-1, 2)
        g = np.zeros((len(words), 2), np.float32)
        self._ck(self.L.tdpd_debug_box_muller(self.h, len(words), _ptr(words), _ptr(g)))
        return g

    def set_membrane_variant(self, previous_step_area_volume: bool):
        self._ck(self.L.tdpd_set_membrane_variant(self.h, int(previous_step_area_volume)))

    def set_graph(self, on: bool):
        self._ck(self.L.tdpd_set_graph(self.h, int(on)))

    def set_timing(self, on: bool):
        self._ck(self.L.tdpd_set_timing(self.h, int(on)))

    def get_timing(self) -> dict:
        cnt = np.zeros(N_TIMERS, np.int64)
        ms = np.zeros(N_TIMERS, np.float64)
        self._ck(self.L.tdpd_get_timing(self.h, _ptr(cnt), _ptr(ms)))
        return {k: dict(launches=int(cnt[i]), ms=float(ms[i])) for i, k in enumerate(TIMER_NAMES)}

    @property
    def launch_count(self) -> int:
        return int(self.L.tdpd_launch_count(self.h))
