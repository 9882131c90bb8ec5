"""Seeded synthetic inputs for the five BASELINE.json configs (and reduced copies for tests).

INPUTS ONLY: positions, velocities, types, concentrations, membrane vertices/triangles and the
parameter values.  None of the method's arithmetic lives here.
Everything is generated in fp64, rounded ONCE to fp32, and the same fp32 arrays are handed to
the CUDA library and to the oracle.

Recipe = SURVEY.md §8(d): base seed 20161118, config c uses seed base+c; positions uniform in
[0,L); velocities N(0,kBT) minus the mean; config 1 C~U[0,1]; config 2 C = 1 for x<L/2 else 0;
configs 3-5 Evans-Fung RBC meshes (tdpd_workloads.mesh), solvent inside a cell -> type 1, C0=1,
outside -> type 0, C0=0, membrane -> type 2, C0=1; second species (configs 4-5) outer 1, inner 0,
membrane 0.  Parameter values = SURVEY P-table (the paper prints none for the
membrane; PAPER.md:102-128 defers to its ref [10]).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from . import mesh as _mesh

BASE_SEED = 20161118
MAX_TYPES = 4
MAX_SPECIES = 10

BODY_OFF, BODY_UNIFORM, BODY_DOUBLE_POISEUILLE_Z = 0, 1, 2

# closed-form area / volume of the Evans-Fung surface at D0 = 7.82 (re-derived by
# quadrature in tests/test_workloads.py)
A_R = 134.0932
V_R = 94.0984


def _f32(x):
    return np.asarray(x, dtype=np.float64).astype(np.float32)


def fluid_params(box, rho, n_species=1, a=None, gamma=4.5, kBT=1.0, s_R=0.5, kappa=10.0, kappa_m=1.0,
                 s_c=2.0, m_s=0.01, r_c=1.0, r_cc=1.58, dt=0.01, body=0.0, body_mode=BODY_OFF, seed=1,
                 n_types=1, source=0.0, decay=0.0):
    """Parameter dict mirroring `tdpd_params` (include/tdpd.h).  Types: 0 outer solvent, 1 inner
    solvent, 2 membrane: kappa_00 = kappa_11 = kappa, kappa_01 = 0,
    kappa_x2 = kappa_m."""
    if a is None:
        a = 75.0 * kBT / rho
    T, S = MAX_TYPES, MAX_SPECIES
    A = np.zeros((T, T)); G = np.zeros((T, T)); SR = np.zeros((T, T)); K = np.zeros((S, T, T))
    A[:n_types, :n_types] = a
    G[:n_types, :n_types] = gamma
    SR[:n_types, :n_types] = s_R
    for s in range(n_species):
        K[s, :n_types, :n_types] = kappa
        if n_types >= 2:
            K[s, 0, 1] = K[s, 1, 0] = 0.0
        if n_types >= 3:
            K[s, 2, :n_types] = kappa_m
            K[s, :n_types, 2] = kappa_m
    SRC = np.zeros((S, T)); DEC = np.zeros((S, T))     # Q^S: the same rate for every species, per type if a sequence
    SRC[:n_species, :n_types] = np.asarray(source, dtype=np.float64)
    DEC[:n_species, :n_types] = np.asarray(decay, dtype=np.float64)
    sc = np.zeros(S); ms = np.zeros(S)
    sc[:n_species] = s_c
    ms[:n_species] = m_s
    return dict(
        n_types=int(n_types), n_species=int(n_species), box=_f32(box), r_c=np.float32(r_c),
        r_cc=np.float32(r_cc), dt=np.float32(dt), kBT=np.float32(kBT), rho=np.float32(rho),
        a=_f32(A), gamma=_f32(G), s_R=_f32(SR), kappa=_f32(K), s_c=_f32(sc), m_s=_f32(ms),
        body_force=_f32([body, 0.0, 0.0]), body_mode=int(body_mode), seed=int(seed),
        exclude_same_cell_membrane_pairs=1, source=_f32(SRC), decay=_f32(DEC),
    )


def rbc_params(kBT=1.0):
    """SURVEY P-table (proposed constants; inputs to both sides)."""
    nv = 642
    theta0 = float(np.arccos((np.sqrt(3.0) * (nv - 2) - 5.0 * np.pi) / (np.sqrt(3.0) * (nv - 2) - 3.0 * np.pi)))
    return dict(
        p=np.float32(0.00845), x0=np.float32(2.2), m=np.float32(2.0),
        gamma_T=np.float32(3.0), gamma_C=np.float32(2.0),
        k_g=np.float32(20000.0), k_l=np.float32(400.0), k_v=np.float32(20000.0),
        k_b=np.float32(2.4e-19 / (1.380649e-23 * 296.15)),  # 58.70 kBT
        theta0=np.float32(theta0), VR_over_AR32=np.float32(V_R / A_R ** 1.5),
    )


@dataclass
class Workload:
    name: str
    params: dict
    pos: np.ndarray      # [n,3] f32 solvent
    vel: np.ndarray      # [n,3] f32
    type: np.ndarray     # [n]   i32
    conc: np.ndarray     # [n,S] f32
    rbcs: list = field(default_factory=list)   # dicts: verts, vel, conc (f32), tris (i32)
    rbc_params: dict | None = None
    steps: int = 100

    @property
    def n_solvent(self) -> int:
        return int(self.pos.shape[0])

    @property
    def n_total(self) -> int:
        return self.n_solvent + sum(int(r["verts"].shape[0]) for r in self.rbcs)

    def all_particles(self):
        """(pos, vel, type, conc, rbc_id) over all ids in load order (solvent, then each mesh)."""
        S = self.params["n_species"]
        pos = [self.pos]; vel = [self.vel]; typ = [self.type]; conc = [self.conc[:, :S]]
        rid = [np.zeros(self.n_solvent, np.int32)]
        for k, r in enumerate(self.rbcs):
            nv = r["verts"].shape[0]
            pos.append(r["verts"]); vel.append(r["vel"]); conc.append(r["conc"][:, :S])
            typ.append(np.full(nv, 2, np.int32)); rid.append(np.full(nv, k + 1, np.int32))
        return (np.concatenate(pos), np.concatenate(vel), np.concatenate(typ),
                np.concatenate(conc), np.concatenate(rid))


def _positions(rng, n, box):
    box = np.asarray(box, dtype=np.float64)
    p = (rng.random((n, 3)) * box).astype(np.float32)
    top = np.nextafter(box.astype(np.float32), np.float32(0.0))
    return np.minimum(p, top)


def _velocities(rng, n, kBT):
    return rng.standard_normal((n, 3)) * np.sqrt(kBT)


def make_fluid(name, box, rho, seed, conc="uniform", steps=100, **kw) -> Workload:
    """Pure tDPD fluid (BASELINE configs 1-2; PAPER.md:218-222 benchmark family)."""
    box = np.asarray(box, dtype=np.float64)
    n = int(round(rho * box.prod()))
    rng = np.random.Generator(np.random.PCG64(seed))
    params = fluid_params(box, rho, seed=seed, n_types=1, **kw)
    S = params["n_species"]
    pos = _positions(rng, n, box)
    vel = _velocities(rng, n, float(params["kBT"]))
    vel -= vel.mean(axis=0)
    c = np.zeros((n, S))
    if conc == "uniform":
        c[:] = rng.random((n, S))
    elif conc == "step":
        c[:] = (pos[:, :1] < 0.5 * box[0]).astype(np.float64)
    elif conc == "zero":
        pass
    else:
        raise ValueError(conc)
    return Workload(name, params, pos, vel.astype(np.float32), np.zeros(n, np.int32),
                    c.astype(np.float32), steps=steps)


def make_suspension(name, box, rho, seed, centers, rotations, n_species=1, body=0.02,
                    body_mode=BODY_DOUBLE_POISEUILLE_Z, steps=100, mesh_level=3, **kw) -> Workload:
    """Solvent + explicit RBC membranes (BASELINE configs 3-5; PAPER.md:224-237 family)."""
    from scipy.spatial import cKDTree

    box = np.asarray(box, dtype=np.float64)
    n = int(round(rho * box.prod()))
    rng = np.random.Generator(np.random.PCG64(seed))
    params = fluid_params(box, rho, n_species=n_species, seed=seed, n_types=3, body=body,
                          body_mode=body_mode, **kw)
    kBT = float(params["kBT"])
    S = n_species
    pos = _positions(rng, n, box)
    vel = _velocities(rng, n, kBT)
    centers = np.asarray(centers, dtype=np.float64).reshape(-1, 3)
    M = centers.shape[0]
    mverts, tris = _mesh.rbc_mesh(mesh_level)
    nv = mverts.shape[0]
    mvel = _velocities(rng, M * nv, kBT).reshape(M, nv, 3)
    allv = np.concatenate([vel, mvel.reshape(-1, 3)])
    mean = allv.mean(axis=0)
    vel -= mean
    mvel -= mean

    typ = np.zeros(n, np.int32)
    if M:
        tree = cKDTree(pos.astype(np.float64))
        rad = 0.5 * _mesh.D0_RBC + 0.05
        for k in range(M):
            idx = np.asarray(tree.query_ball_point(centers[k], rad), dtype=np.int64)
            if idx.size == 0:
                continue
            local = (pos[idx].astype(np.float64) - centers[k]) @ rotations[k]  # R^T (p - c)
            typ[idx[_mesh.evans_fung_inside(local)]] = 1
    c = np.zeros((n, S))
    c[:, 0] = (typ == 1)
    if S >= 2:
        c[:, 1] = (typ == 0)
    rbcs = []
    for k in range(M):
        v = centers[k] + mverts @ rotations[k].T
        v = np.mod(v, box)
        mc = np.zeros((nv, S)); mc[:, 0] = 1.0
        v32 = np.minimum(v.astype(np.float32), np.nextafter(box.astype(np.float32), np.float32(0)))
        rbcs.append(dict(verts=v32, vel=mvel[k].astype(np.float32), conc=mc.astype(np.float32),
                         tris=tris.copy()))
    return Workload(name, params, pos, vel.astype(np.float32), typ, c.astype(np.float32),
                    rbcs=rbcs, rbc_params=rbc_params(kBT), steps=steps)


def lattice_centers(box, grid, rng=None, jitter=0.0):
    box = np.asarray(box, dtype=np.float64)
    g = np.asarray(grid)
    sp = box / g
    ii = np.stack(np.meshgrid(*[np.arange(k) for k in g], indexing="ij"), axis=-1).reshape(-1, 3)
    c = (ii + 0.5) * sp
    if jitter and rng is not None:
        c = c + rng.uniform(-jitter, jitter, size=c.shape)
    return c


def config(c: int, **over) -> Workload:
    """BASELINE.json configs 1..5 at full size."""
    seed = BASE_SEED + c
    if c == 1:
        return make_fluid("config1", (10, 10, 10), 4.0, seed, conc="uniform", steps=100, **over)
    if c == 2:
        return make_fluid("config2", (32, 32, 32), 4.0, seed, conc="step", steps=1000, **over)
    if c == 3:
        return make_suspension("config3", (40, 20, 20), 3.0, seed, [(20.0, 10.0, 10.0)],
                               np.eye(3)[None], n_species=1, steps=1000, **over)
    rng = np.random.Generator(np.random.PCG64(seed + 1000))
    if c == 4:
        box = (64, 64, 64)
        ctr = lattice_centers(box, (5, 5, 4))
        return make_suspension("config4", box, 3.0, seed, ctr, _mesh.random_rotations(rng, len(ctr)),
                               n_species=2, steps=500, **over)
    if c == 5:
        box = (128, 128, 128)
        ctr = lattice_centers(box, (10, 10, 10), rng, jitter=2.0)
        return make_suspension("config5", box, 3.0, seed, ctr, _mesh.random_rotations(rng, len(ctr)),
                               n_species=2, steps=200, **over)
    raise ValueError(f"no config {c}")


def small_suspension(seed=7, box=(20, 20, 12), n_rbc=1, n_species=1, **over) -> Workload:
    """Reduced copy of config 3/4 for tests the oracle finishes in seconds."""
    rng = np.random.Generator(np.random.PCG64(seed + 1000))
    box = np.asarray(box, dtype=np.float64)
    if n_rbc == 1:
        ctr = [box * 0.5]
        rot = np.eye(3)[None]
    else:
        ctr = lattice_centers(box, (n_rbc, 1, 1))
        rot = _mesh.random_rotations(rng, n_rbc)
    return make_suspension(f"small_susp{n_rbc}", box, 3.0, seed, ctr, rot, n_species=n_species, **over)
