"""Pins for the oracle's non-bonded pair terms (Eq 2-10), neighbour search and conservation laws."""
import os

import numpy as np
import pytest

import tdpd_workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))


def golden(name):
    out = {}
    for line in open(os.path.join(HERE, "golden", name)):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        out[k] = float(v)
    return out


def test_two_particle_closed_form(orc):
    """Values of tests/golden/pair_two_particle.txt (hand arithmetic on Eq 3-6, 8)."""
    g = golden("pair_two_particle.txt")
    p = W.fluid_params((10, 10, 10), 4.0, a=18.75, m_s=0.0, seed=3)
    d, dv = [0.5, 0, 0], [1.0, 0, 0]
    xi = orc.gauss4(0, 1, 0, 0, 3)[0]
    kind, F, Q = orc.pair_terms(p, 0, 1, 0, 0, d, dv, [0.75], [0.25], 0)
    assert kind == 2
    assert F[0] == pytest.approx(g["F_C"] + g["F_D"] + g["F_R_per_xi"] * xi, rel=1e-6)
    assert F[1] == 0 and F[2] == 0
    assert Q[0] == pytest.approx(g["Q_D_per_dC"] * 0.5, rel=1e-6)
    # separate the three terms by switching coefficients off
    p0 = W.fluid_params((10, 10, 10), 4.0, a=18.75, gamma=0.0, m_s=0.0)
    assert orc.pair_terms(p0, 0, 1, 0, 0, d, dv, [0], [0], 0)[1][0] == pytest.approx(g["F_C"], rel=1e-7)
    p1 = W.fluid_params((10, 10, 10), 4.0, a=0.0, kBT=0.0, m_s=0.0)
    assert orc.pair_terms(p1, 0, 1, 0, 0, d, dv, [0], [0], 0)[1][0] == pytest.approx(g["F_D"], rel=1e-7)
    # antisymmetry F_ji = -F_ij, Q_ji = -Q_ij (also with the random flux on: zeta_ij = -zeta_ji)
    pr = W.fluid_params((10, 10, 10), 4.0, a=18.75, m_s=0.05, seed=3)
    k1, F1, Q1 = orc.pair_terms(pr, 5, 9, 0, 0, [0.3, -0.2, 0.4], [1, 2, 3], [0.7], [0.2], 4)
    k2, F2, Q2 = orc.pair_terms(pr, 9, 5, 0, 0, [-0.3, 0.2, -0.4], [-1, -2, -3], [0.2], [0.7], 4)
    assert k1 == k2 == 2 and np.allclose(F1, -F2, rtol=0, atol=1e-13) and np.allclose(Q1, -Q2, rtol=0, atol=1e-13)


def test_random_flux_term_eq9_eq10(orc):
    """Q^R = m_s sqrt(kappa rho (Ci+Cj)) (1-r/r_cc)^{s_c/2} zeta / sqrt(dt) (Eq 9-10), isolated via dC = 0."""
    p = W.fluid_params((10, 10, 10), 4.0, m_s=0.02, kappa=10.0, seed=8)
    r = 1.2
    zeta = orc.gauss4(2, 7, 1, 0, 8)[1]
    kind, F, Q = orc.pair_terms(p, 2, 7, 0, 0, [0, r, 0], [0, 0, 0], [0.3], [0.3], 1)
    rcc = float(np.float32(1.58)); ms = float(np.float32(0.02))
    expect = ms * np.sqrt(10.0 * 4.0 * 0.6) * (1 - r / rcc) ** 1.0 * zeta / np.sqrt(float(np.float32(0.01)))
    assert kind == 1 and np.all(F == 0)
    assert Q[0] == pytest.approx(expect, rel=1e-9)
    # clamp of C_i + C_j at zero, and cutoffs
    assert orc.pair_terms(p, 2, 7, 0, 0, [0, r, 0], [0, 0, 0], [-0.5], [0.2], 1)[2][0] == pytest.approx(
        -10.0 * (1 - r / rcc) ** 2 * (-0.7), rel=1e-9)
    assert orc.pair_terms(p, 2, 7, 0, 0, [0, 1.59, 0], [0, 0, 0], [1], [0], 1)[0] == 0
    assert orc.pair_terms(p, 2, 7, 0, 0, [0, 0.999, 0], [0, 0, 0], [1], [0], 1)[0] == 2
    assert orc.pair_terms(p, 2, 7, 0, 0, [0, 1.001, 0], [0, 0, 0], [1], [0], 1)[0] == 1


def _numpy_pair_census(pos, box, rc, rcc):
    d = pos[:, None, :] - pos[None, :, :]
    d -= box * np.round(d / box)
    r = np.sqrt((d ** 2).sum(-1))
    np.fill_diagonal(r, 1e9)
    return int((r < rcc).sum()), int((r < rc).sum())


@pytest.mark.parametrize("L", [(5.0, 5.0, 5.0), (6.5, 5.0, 8.0), (8.0, 8.0, 8.0)])
def test_cell_list_equals_brute_force(orc, L):
    """O(N^2) search == cell list (identical pair sets; sums equal to rounding) incl. pairs across all faces,
    and both equal an independent numpy count of pairs inside the cutoffs."""
    w = W.make_fluid("t", L, 4.0, seed=11, conc="uniform")
    a = orc.Oracle.from_workload(w, brute=True)
    b = orc.Oracle.from_workload(w, brute=False)
    a.compute_forces(2); b.compute_forces(2)
    sa, sb = a.get_state(), b.get_state()
    ca, cb = a.census_totals(), b.census_totals()
    assert ca["n_cc"] == cb["n_cc"] and ca["n_c"] == cb["n_c"]
    ncc, nc = _numpy_pair_census(w.pos.astype(np.float64), np.asarray(L), float(np.float32(1.0)), float(np.float32(1.58)))
    assert (ca["n_cc"], ca["n_c"]) == (ncc, nc)
    scale = np.abs(sa["force"]).max()
    assert np.abs(sa["force"] - sb["force"]).max() < 1e-11 * scale
    assert np.abs(sa["flux"] - sb["flux"]).max() < 1e-11 * np.abs(sa["flux"]).max()
    # cells never miss a periodic image: particles within r_cc of every face exist in this box
    assert (w.pos.min(0) < 0.5).all() and (w.pos.max(0) > np.asarray(L) - 0.5).all()


def test_force_sum_matches_independent_numpy_evaluation(orc):
    """Whole-system force/flux sum re-evaluated in numpy from Eq 3-8 with the oracle's Gaussians as inputs."""
    w = W.make_fluid("t", (5, 5, 5), 4.0, seed=21, conc="uniform", m_s=0.0)
    o = orc.Oracle.from_workload(w)
    o.compute_forces(0)
    s = o.get_state()
    p = w.params
    x, v, C = w.pos.astype(np.float64), w.vel.astype(np.float64), w.conc.astype(np.float64)[:, 0]
    n = len(x)
    box = p["box"].astype(np.float64)
    d = x[:, None] - x[None]
    d -= box * np.round(d / box)
    r = np.sqrt((d ** 2).sum(-1)); np.fill_diagonal(r, 1e9)
    e = d / r[..., None]
    ii, jj = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    xi = orc.gauss_batch(ii.ravel(), jj.ravel(), 0, 0, p["seed"])[:, 0].reshape(n, n)
    rc, rcc, dt = float(p["r_c"]), float(p["r_cc"]), float(p["dt"])
    a, gam = float(p["a"][0, 0]), float(p["gamma"][0, 0])
    wc = np.clip(1 - r / rc, 0, None)
    edv = (e * (v[:, None] - v[None])).sum(-1)
    f = a * wc - gam * wc * edv + np.sqrt(2 * gam) * np.sqrt(wc) * xi / np.sqrt(dt)      # s = 1/2: w_R^2 = w_c
    F = ((f * (r < rc))[..., None] * e).sum(1)
    Q = (-10.0 * np.clip(1 - r / rcc, 0, None) ** 2 * (C[:, None] - C[None])).sum(1)
    assert np.abs(F - s["force"]).max() < 1e-9 * np.abs(F).max()
    assert np.abs(Q - s["flux"][:, 0]).max() < 1e-9 * np.abs(Q).max()


def test_momentum_and_concentration_sums_vanish(orc):
    w = W.config(1)
    o = orc.Oracle.from_workload(w)
    o.compute_forces(0)
    s = o.get_state()
    assert np.abs(s["force"].sum(0)).max() < 1e-12 * np.abs(s["force"]).sum()
    assert abs(s["flux"].sum()) < 1e-12 * np.abs(s["flux"]).sum()
    c = o.census_totals()
    n = w.n_total
    assert c["n_cc"] / n == pytest.approx(4 * np.pi / 3 * 1.58 ** 3 * 4, rel=0.02)      # 16.52 rho
    assert c["n_c"] / n == pytest.approx(4 * np.pi / 3 * 4, rel=0.03)                   # 4.19 rho


def test_subset_forces_equal_full_sum(orc):
    w = W.make_fluid("t", (6, 6, 6), 4.0, seed=5, conc="uniform")
    o = orc.Oracle.from_workload(w)
    o.compute_forces(3)
    s = o.get_state()
    ids = np.array([0, 17, 400, 863])
    F, Q = o.pair_forces_subset(3, ids)
    assert np.abs(F - s["force_pair"][ids]).max() < 1e-11 * np.abs(F).max()
    assert np.abs(Q - s["flux"][ids]).max() < 1e-11 * np.abs(Q).max()


def test_type_pair_coefficients_and_membrane_exclusion(orc):
    """kappa_01 = 0 blocks inner<->outer flux (R15); same-membrane vertex pairs are skipped (R16)."""
    p = W.fluid_params((10, 10, 10), 3.0, n_types=3, m_s=0.0)
    k, F, Q = orc.pair_terms(p, 0, 1, 0, 1, [0.5, 0, 0], [0, 0, 0], [1.0], [0.0], 0)
    assert k == 2 and Q[0] == 0.0
    k, F, Q = orc.pair_terms(p, 0, 1, 0, 2, [0.5, 0, 0], [0, 0, 0], [1.0], [0.0], 0)
    assert Q[0] == pytest.approx(-1.0 * (1 - 0.5 / float(np.float32(1.58))) ** 2, rel=1e-9)
    w = W.small_suspension(box=(20, 20, 12))
    w.pos, w.vel, w.type, w.conc = w.pos[:0], w.vel[:0], w.type[:0], w.conc[:0]      # membrane only
    o = orc.Oracle.from_workload(w)
    o.compute_forces(0)
    s = o.get_state()
    assert np.all(s["force_pair"] == 0) and np.all(s["flux"] == 0)
    assert o.census_totals()["n_cc"] == 0
