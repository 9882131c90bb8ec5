"""Pins for the input generators (tdpd_workloads): mesh topology and geometry fixed by the recipe
(SURVEY §8(c) "Mesh" pin; BASELINE config 3: 642 vertices / 1920 bonds / 1280 triangles)."""
import numpy as np
import pytest

import tdpd_workloads as W


def test_rbc_mesh_topology():
    v, t = W.rbc_mesh(3)
    assert v.shape == (642, 3) and t.shape == (1280, 3)
    e = np.concatenate([t[:, [0, 1]], t[:, [1, 2]], t[:, [2, 0]]])
    und = np.unique(np.sort(e, axis=1), axis=0)
    assert len(und) == 1920
    assert 642 - 1920 + 1280 == 2                       # Euler characteristic of a sphere
    deg = np.bincount(und.ravel(), minlength=642)
    assert (deg == 5).sum() == 12 and (deg == 6).sum() == 630
    # closed + consistently oriented: every directed edge appears once and its reverse once
    d = set(map(tuple, e.tolist()))
    assert len(d) == 3840 and all((b, a) in d for a, b in d)


def test_rbc_mesh_geometry_matches_recipe_numbers():
    v, t = W.rbc_mesh(3)
    a, b, c = v[t[:, 0]], v[t[:, 1]], v[t[:, 2]]
    area = 0.5 * np.linalg.norm(np.cross(b - a, c - a), axis=1).sum()
    vol = np.einsum("ij,ij->i", a, np.cross(b, c)).sum() / 6.0
    assert vol > 0                                       # CCW from outside
    assert area == pytest.approx(133.2538, abs=2e-4)     # SURVEY §8(c) mesh pin
    assert vol == pytest.approx(93.2872, abs=2e-4)
    assert np.abs(v[:, 0]).max() == pytest.approx(W.D0_RBC / 2, rel=1e-12)
    # thickness at the centre (2 D0 a0) and maximum thickness of the biconcave profile
    assert 2 * W.D0_RBC * 0.0518 == pytest.approx(0.810, abs=1e-3)
    assert 2 * np.abs(v[:, 2]).max() == pytest.approx(2.566, abs=5e-3)


def test_evans_fung_closed_form_area_volume():
    """A^R, V^R used for V0/A0^{3/2} = surface of revolution z(r) by quadrature."""
    from scipy.integrate import quad
    d0 = W.D0_RBC
    a0, a1, a2 = 0.0518, 2.0026, -4.491

    def z(r):
        t = r * r / d0 ** 2
        return d0 * np.sqrt(max(1 - 4 * t, 0.0)) * (a0 + a1 * t + a2 * t * t)

    # parametrise r = (d0/2) sin(phi) to remove the square-root singularity at the rim
    def zphi(phi):
        s = np.sin(phi) ** 2 / 4.0
        return d0 * np.cos(phi) * (a0 + a1 * s + a2 * s * s)

    def dz(phi, h=1e-6):
        return (zphi(phi + h) - zphi(phi - h)) / (2 * h)

    R = d0 / 2
    area = 2 * quad(lambda p: 2 * np.pi * R * np.sin(p) * np.hypot(R * np.cos(p), dz(p)), 0, np.pi / 2, limit=200)[0]
    vol = 2 * quad(lambda r: 2 * np.pi * r * z(r), 0, R, limit=200)[0]
    from tdpd_workloads.configs import A_R, V_R
    assert area == pytest.approx(A_R, rel=2e-5)
    assert vol == pytest.approx(V_R, rel=2e-5)


def test_inside_test_agrees_with_mesh():
    v, _ = W.rbc_mesh(3)
    assert not W.evans_fung_inside(v * 1.02).any()
    assert W.evans_fung_inside(v * 0.9).all()


@pytest.mark.parametrize("c,n_solv,n_tot,S", [(1, 4000, 4000, 1), (3, 48000, 48642, 1)])
def test_config_sizes(c, n_solv, n_tot, S):
    w = W.config(c)
    assert w.n_solvent == n_solv and w.n_total == n_tot and w.params["n_species"] == S
    assert w.pos.dtype == np.float32 and (w.pos >= 0).all() and (w.pos < w.params["box"]).all()
    vel_all = w.all_particles()[1]
    assert np.abs(vel_all.astype(np.float64).sum(0)).max() < 1e-2      # zero total momentum
    w2 = W.config(c)
    assert np.array_equal(w.pos, w2.pos) and np.array_equal(w.vel, w2.vel)   # seeded


def test_config3_typing():
    w = W.config(3)
    inner = (w.type == 1)
    assert 200 < inner.sum() < 330            # ~ rho * V_rbc = 3 * 93.3
    assert np.array_equal(w.conc[:, 0], inner.astype(np.float32))
    assert len(w.rbcs) == 1 and (w.rbcs[0]["conc"][:, 0] == 1).all()


def test_rotations_are_orthonormal():
    rng = np.random.Generator(np.random.PCG64(1))
    R = W.random_rotations(rng, 50)
    assert np.allclose(R @ R.transpose(0, 2, 1), np.eye(3), atol=1e-12)
    assert np.allclose(np.linalg.det(R), 1.0)
