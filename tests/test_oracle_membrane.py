"""Pins for the oracle's membrane terms (Eq 13-19): forces are minus the gradient of the paper's
potentials (central differences of energies written HERE from the printed equations), rigid-body invariance,
rest state, the fluctuation-dissipation covariance of Eq 15/16 and the wiring of the Philox rows."""
import numpy as np
import pytest

import tdpd_workloads as W


# ---- the paper's potentials, written out from the text (not from the oracle) -----------------------------------
def U_wlc(h, hm, kBT, p):                       # Eq 13
    x = h / hm
    return kBT * hm / (4 * p) * (3 * x ** 2 - 2 * x ** 3) / (1 - x)


def U_pow(h, kp, m):                            # Eq 14
    return kp / ((m - 1) * h ** (m - 1)) if m != 1 else -kp * np.log(h)


def tri_geom(r, tris):
    a, b, c = r[tris[:, 0]], r[tris[:, 1]], r[tris[:, 2]]
    n = np.cross(b - a, c - a)
    return 0.5 * np.linalg.norm(n, axis=1), np.einsum("ij,ij->i", a, np.cross(b, c)) / 6.0


def dihedral_angles(r, dih):
    r1, r2, r3, r4 = (r[dih[:, k]] for k in range(4))
    n1 = np.cross(r2 - r1, r3 - r1)              # triangle (v1,v2,v3)
    n2 = np.cross(r3 - r4, r2 - r4)              # triangle (v4,v3,v2)
    n1 /= np.linalg.norm(n1, axis=1, keepdims=True)
    n2 /= np.linalg.norm(n2, axis=1, keepdims=True)
    e = r3 - r2
    e /= np.linalg.norm(e, axis=1, keepdims=True)
    return np.arctan2(np.einsum("ij,ij->i", np.cross(n1, n2), e), np.einsum("ij,ij->i", n1, n2))


def total_energy(r, tris, topo, stats, rp, kBT, terms):
    U = 0.0
    if "bond" in terms:
        h = np.linalg.norm(r[topo["bond"][:, 0]] - r[topo["bond"][:, 1]], axis=1)
        U += (U_wlc(h, rp["x0"] * topo["h0"], kBT, rp["p"]) + U_pow(h, topo["kp"], rp["m"])).sum()
    At, Vt = tri_geom(r, tris)
    if "area" in terms:                          # Eq 17
        U += rp["k_g"] * (At.sum() - stats["A0"]) ** 2 / (2 * stats["A0"])
        U += (rp["k_l"] * (At - topo["A0t"]) ** 2 / (2 * topo["A0t"])).sum()
    if "volume" in terms:                        # Eq 18
        U += rp["k_v"] * (Vt.sum() - stats["V0"]) ** 2 / (2 * stats["V0"])
    if "bend" in terms:                          # Eq 19
        U += (rp["k_b"] * (1 - np.cos(dihedral_angles(r, topo["dih"]) - rp["theta0"]))).sum()
    return U


def membrane_only(orc, rp_over, level=2, box=(30.0, 30.0, 30.0), seed=3, shift=None):
    verts, tris = W.rbc_mesh(level)
    rp = {k: float(v) for k, v in W.rbc_params().items()}
    rp.update(rp_over)
    p = W.fluid_params(box, 3.0, n_types=3, seed=seed)
    o = orc.Oracle(p)
    c = np.asarray(box) / 2 if shift is None else np.asarray(shift)
    v32 = np.mod(verts + c, box).astype(np.float32)
    o.add_rbc_mesh(v32, np.zeros_like(v32), np.ones((len(v32), 1), np.float32), tris, rp)
    rp32 = {k: float(np.float32(v)) for k, v in rp.items()}
    return o, v32.astype(np.float64), tris, rp32


@pytest.mark.parametrize("terms", [("bond",), ("area",), ("volume",), ("bend",), ("bond", "area", "volume", "bend")])
def test_conservative_forces_are_minus_grad_U(orc, terms):
    off = dict(gamma_T=0.0, gamma_C=0.0)
    if "area" not in terms:
        off.update(k_g=0.0, k_l=0.0)
    if "volume" not in terms:
        off.update(k_v=0.0)
    if "bend" not in terms:
        off.update(k_b=0.0)
    if "bond" not in terms:
        off.update(p=1e30)                       # WLC prefactor kBT/p -> 0, and k_p follows
    o, x0, tris, rp = membrane_only(orc, off)
    topo, stats = o.rbc_topology(0), {k: v[0] for k, v in o.rbc_stats().items()}
    rng = np.random.Generator(np.random.PCG64(9))
    x = x0 + 0.03 * rng.standard_normal(x0.shape)
    o.set_state(x=x)
    o.compute_forces(0)
    F = o.get_state()["force_bonded"]
    kBT = 1.0
    h = 1e-5
    G = np.zeros_like(x)
    for i in range(x.shape[0]):
        for a in range(3):
            xp, xm = x.copy(), x.copy()
            xp[i, a] += h; xm[i, a] -= h
            G[i, a] = (total_energy(xp, tris, topo, stats, rp, kBT, terms)
                       - total_energy(xm, tris, topo, stats, rp, kBT, terms)) / (2 * h)
    scale = np.abs(F).max()
    assert scale > 1e-3
    assert np.abs(F + G).max() < 2e-6 * scale
    # internal forces: no net force, no net torque
    assert np.abs(F.sum(0)).max() < 1e-10 * np.abs(F).sum()
    assert np.abs(np.cross(x, F).sum(0)).max() < 1e-9 * np.abs(np.cross(x, F)).sum()


def test_rest_state_and_derived_parameters(orc):
    o, x0, tris, rp = membrane_only(orc, dict(gamma_T=0.0, gamma_C=0.0, k_b=0.0))
    topo, stats = o.rbc_topology(0), {k: v[0] for k, v in o.rbc_stats().items()}
    h = np.linalg.norm(x0[topo["bond"][:, 0]] - x0[topo["bond"][:, 1]], axis=1)
    assert np.allclose(topo["h0"], h, rtol=1e-12)                  # R11: rest length = initial length
    At, Vt = tri_geom(x0, tris)
    assert np.allclose(topo["A0t"], At, rtol=1e-12)
    assert stats["A0"] == pytest.approx(At.sum(), rel=1e-12)       # PAPER.md:122 "summing the area of each triangle"
    assert stats["V0"] == pytest.approx(At.sum() ** 1.5 * rp["VR_over_AR32"], rel=1e-12)
    o.compute_forces(0)
    s = o.get_state()
    # bonds are force-free at h0 (k_p from the force balance), local area term vanishes; global area/volume
    # terms remain only through (A-A0) = 0 and (V-V0) != 0
    o2, *_ = membrane_only(orc, dict(gamma_T=0.0, gamma_C=0.0, k_b=0.0, k_v=0.0))
    o2.compute_forces(0)
    assert np.abs(o2.get_state()["force_bonded"]).max() < 1e-9
    st = o.rbc_stats()
    assert st["area"][0] == pytest.approx(At.sum(), rel=1e-12) and st["volume"][0] == pytest.approx(Vt.sum(), rel=1e-12)
    # WLC derivative identity used by SURVEY O5: (6x-9x^2+4x^3)/(4(1-x)^2) = 1/(4(1-x)^2) - 1/4 + x
    x = np.linspace(0.05, 0.9, 18)
    assert np.allclose((6 * x - 9 * x ** 2 + 4 * x ** 3) / (4 * (1 - x) ** 2), 1 / (4 * (1 - x) ** 2) - 0.25 + x)


def test_dihedral_sign_convention_and_mesh_statistics(orc):
    """theta > 0 on a convex body; RBC mesh statistics of SURVEY §8(c) (min/mean/max -0.179/0.0849/0.319)."""
    o, x0, tris, rp = membrane_only(orc, {}, level=3)
    dih = o.rbc_topology(0)["dih"]
    assert dih.shape == (1920, 4)
    th = np.array([orc.dihedral_terms(1.0, 0.0, *x0[d])[0] for d in dih])
    assert th.min() == pytest.approx(-0.179, abs=2e-3) and th.max() == pytest.approx(0.319, abs=2e-3)
    assert th.mean() == pytest.approx(0.0849, abs=5e-4)
    assert np.allclose(th, dihedral_angles(x0, dih), atol=1e-12)
    sph, st = W.icosphere(2)
    p = W.fluid_params((30, 30, 30), 3.0, n_types=3)
    o2 = orc.Oracle(p)
    o2.add_rbc_mesh((sph * 3 + 15).astype(np.float32), None, None, st, W.rbc_params())
    d2 = o2.rbc_topology(0)["dih"]
    xs = (sph * 3 + 15).astype(np.float32).astype(np.float64)
    assert all(orc.dihedral_terms(1.0, 0.0, *xs[d])[0] > 0 for d in d2)
    # each dihedral = the two triangles sharing edge (v2,v3), both listed CCW
    tset = set(map(tuple, np.concatenate([st, st[:, [1, 2, 0]], st[:, [2, 0, 1]]]).tolist()))
    assert all((d[0], d[1], d[2]) in tset and (d[3], d[2], d[1]) in tset for d in d2.tolist())


def test_membrane_across_periodic_boundary(orc):
    """Unwrapping relative to vertex 0: a cell straddling the box corner feels the same forces."""
    off = dict(gamma_T=0.0, gamma_C=0.0)
    o1, x1, tris, _ = membrane_only(orc, off, shift=(15.0, 15.0, 15.0))
    o2, x2, _, _ = membrane_only(orc, off, shift=(0.5, 29.75, 0.25))
    rng = np.random.Generator(np.random.PCG64(2))
    dx = 0.02 * rng.standard_normal(x1.shape)
    box = np.array([30.0, 30.0, 30.0])
    o1.set_state(x=np.mod(x1 + dx, box)); o2.set_state(x=np.mod(x2 + dx, box))
    o1.compute_forces(0); o2.compute_forces(0)
    f1, f2 = o1.get_state()["force_bonded"], o2.get_state()["force_bonded"]
    assert np.abs(f1 - f2).max() < 2e-3 * np.abs(f1).max()    # fp32 rounding of the two initial placements differs
    st1, st2 = o1.rbc_stats(), o2.rbc_stats()
    assert st2["volume"][0] == pytest.approx(st1["volume"][0], rel=1e-5)


def test_bond_dissipative_and_random_terms(orc):
    rp = {k: float(v) for k, v in W.rbc_params().items()}
    rng = np.random.Generator(np.random.PCG64(4))
    d = np.array([0.3, -0.2, 0.35]); dv = np.array([0.5, 1.0, -2.0])
    e = d / np.linalg.norm(d)
    Fc, Fd, Fr = orc.bond_terms(1.0, 0.01, rp, 0.5, 1.0, d, dv, np.zeros(9))
    gT, gC = float(np.float32(3.0)), float(np.float32(2.0))
    assert np.allclose(Fd, -gT * dv - gC * (dv @ e) * e, rtol=1e-12)              # Eq 15
    assert np.all(Fr == 0)
    assert np.allclose(np.cross(Fc, e), 0, atol=1e-12)                            # central force
    # Eq 15/16 fluctuation-dissipation: Cov[F^R] = (2 kBT/dt) (gT I + gC e e^T)
    n = 400_000   # SURVEY §8(c) "Bond random force": >= 4e5 draws
    Ns = rng.standard_normal((n, 9))
    fr = np.array([orc.bond_terms(1.0, 0.01, rp, 0.5, 1.0, d, dv, N)[2] for N in Ns])
    cov = fr.T @ fr / n
    target = 2 * 1.0 / 0.01 * (gT * np.eye(3) + gC * np.outer(e, e))
    assert np.abs(fr.mean(0)).max() < 0.02 * np.sqrt(target.max())
    assert np.abs(cov - target).max() < 0.02 * target.max()
    # exact linear-algebra restatement of Eq 16 for one draw
    N = Ns[0].reshape(3, 3)
    NS = 0.5 * (N + N.T); tr = np.trace(N)
    M = np.sqrt(2 * gT) * (NS - tr / 3 * np.eye(3)) + np.sqrt(3 * gC - gT) / 3 * tr * np.eye(3)
    assert np.allclose(fr[0], np.sqrt(2 * 1.0 / 0.01) * M @ e, rtol=1e-12)


def test_bond_random_force_wiring_on_a_tetrahedron(orc):
    """Full path on the smallest closed mesh: rows of N come from Philox tags 1,2,3 of (min id, max id, step);
    force on the higher id is the negative; solvent ids come first."""
    verts = np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], np.float64) * 0.4 + 5.0
    tris = np.array([[0, 1, 2], [0, 3, 1], [0, 2, 3], [1, 3, 2]], np.int32)
    a, b, c = verts[tris[:, 0]], verts[tris[:, 1]], verts[tris[:, 2]]
    if np.einsum("ij,ij->i", np.cross(b - a, c - a), a + b + c - 15.0).min() < 0:
        tris = tris[:, [0, 2, 1]]
    rp = {k: float(v) for k, v in W.rbc_params().items()}
    rp.update(k_g=0.0, k_l=0.0, k_v=0.0, k_b=0.0, p=1e30)
    p = W.fluid_params((10, 10, 10), 3.0, n_types=3, seed=77)
    o = orc.Oracle(p)
    o.load_particles(np.array([[1, 1, 1], [2, 2, 2], [3, 3, 3]], np.float32), np.zeros((3, 3), np.float32),
                     np.zeros(3, np.int32), np.zeros((3, 1), np.float32))
    o.add_rbc_mesh(verts.astype(np.float32), np.zeros((4, 3), np.float32), None, tris, rp)
    o.compute_forces(6)
    F = o.get_state()["force_bonded"]
    assert np.all(F[:3] == 0)
    topo = o.rbc_topology(0)
    assert len(topo["bond"]) == 6
    x = verts.astype(np.float32).astype(np.float64)
    expect = np.zeros((4, 3))
    rp32 = {k: float(np.float32(v)) for k, v in rp.items()}
    for (i, j) in topo["bond"]:
        N = np.array([orc.gauss4(3 + i, 3 + j, 6, 1 + row, 77)[:3] for row in range(3)])
        NS = 0.5 * (N + N.T); tr = np.trace(N)
        M = (np.sqrt(2 * rp32["gamma_T"]) * (NS - tr / 3 * np.eye(3))
             + np.sqrt(3 * rp32["gamma_C"] - rp32["gamma_T"]) / 3 * tr * np.eye(3))
        e = (x[i] - x[j]) / np.linalg.norm(x[i] - x[j])
        f = np.sqrt(2 * 1.0 / float(np.float32(0.01))) * M @ e
        expect[i] += f; expect[j] -= f
    assert np.allclose(F[3:], expect, rtol=1e-10, atol=1e-10)


def test_open_or_misoriented_mesh_is_rejected(orc):
    verts, tris = W.icosphere(1)
    p = W.fluid_params((10, 10, 10), 3.0, n_types=3)
    o = orc.Oracle(p)
    with pytest.raises(ValueError):
        o.add_rbc_mesh((verts + 5).astype(np.float32), None, None, tris[:-1], W.rbc_params())
    bad = tris.copy(); bad[0] = bad[0, [0, 2, 1]]
    with pytest.raises(ValueError):
        o.add_rbc_mesh((verts + 5).astype(np.float32), None, None, bad, W.rbc_params())


def test_previous_step_area_volume_variant(orc):
    """SURVEY §8(f) row 3 / PAPER.md:156: K-Apply with the totals of the previous step.  The global area and volume terms
    of Eq 17-18 are linear in (A - A0) / A0 and (V - V0) / V0, so the variant's bonded force differs from the sequential
    one by exactly  -k_g (A_prev - A) / A0 * dA/dr  -  k_v (V_prev - V) / V0 * dV/dr,  with the gradients taken here by
    central differences of the numpy area / volume of this file.  The first evaluation, and one after set_state, use
    their own totals."""
    o, r0, tris, rp = membrane_only(orc, dict(gamma_T=0.0, gamma_C=0.0), level=2, seed=5)   # no random bond force
    ref, _, _, _ = membrane_only(orc, dict(gamma_T=0.0, gamma_C=0.0), level=2, seed=5)
    o.set_lagged_area_volume(True)
    # first evaluation: identical to the sequential variant
    o.compute_forces(0); ref.compute_forces(0)
    assert np.array_equal(o.get_state()["force_bonded"], ref.get_state()["force_bonded"])
    # kick the membrane so that area and volume change, step both once
    rng = np.random.Generator(np.random.PCG64(2))
    v = 2.0 * rng.standard_normal(r0.shape)
    o.set_state(None, v, None); ref.set_state(None, v, None)
    o.compute_forces(0); ref.compute_forces(0)
    A_prev, V_prev = o.rbc_stats()["area"][0], o.rbc_stats()["volume"][0]
    o.step(1); ref.step(1)
    so, sr = o.get_state(), ref.get_state()
    assert np.allclose(so["pos"], sr["pos"], rtol=0, atol=1e-15)        # same positions after one drift (same F^0)
    st = o.rbc_stats()
    A, V, A0, V0 = st["area"][0], st["volume"][0], st["A0"][0], st["V0"][0]
    assert abs(A - A_prev) > 1e-4 * A0                                  # the totals did change
    r = so["pos"]
    r = r - 30.0 * np.round((r - r[0]) / 30.0)

    def grad(fun):
        g = np.zeros_like(r)
        h = 1e-6
        for i in range(len(r)):
            for a in range(3):
                rp_ = r.copy(); rm_ = r.copy()
                rp_[i, a] += h; rm_[i, a] -= h
                g[i, a] = (fun(rp_) - fun(rm_)) / (2 * h)
        return g

    gA = grad(lambda x: tri_geom(x, tris)[0].sum())
    gV = grad(lambda x: tri_geom(x, tris)[1].sum())
    expect = -rp["k_g"] * (A_prev - A) / A0 * gA - rp["k_v"] * (V_prev - V) / V0 * gV
    diff = so["force_bonded"] - sr["force_bonded"]
    assert np.abs(diff).max() > 1e-3
    assert np.allclose(diff, expect, rtol=0, atol=2e-6 * np.abs(expect).max() + 1e-7)
    # a replaced state voids the lagged totals: the evaluation that follows is the sequential one again
    x = so["pos"]
    o.set_state(x, so["vel"], None); ref.set_state(x, so["vel"], None)
    o.compute_forces(1); ref.compute_forces(1)
    assert np.array_equal(o.get_state()["force_bonded"], ref.get_state()["force_bonded"])
