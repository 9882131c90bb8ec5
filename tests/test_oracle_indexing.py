"""Pins for the two oracle functions the bit-exact "cell and neighbour indexing" claim rests on (SURVEY §8(c) O11,
"Neighbour search" pin): orc_bin_fp32 against a numpy float32 restatement of the binning rule
(DESIGN.md R-bin) and orc_neighbor_census against a brute-force numpy loop, plus the Gaussian wiring of the species
(DESIGN.md R-RNG) and the general exponents of Eq 5 / Eq 8 in orc_pair_terms."""
import numpy as np
import pytest

import tdpd_workloads as W


def _bin_numpy(box, r_cut, pos):
    """R-bin written out with numpy float32 scalars: n_a = floor(L_a / r_cut) in double from the fp32 values,
    inv_a = float32(n_a / L_a), wrap once, c_a = min(n_a - 1, floor(float32(x) * inv_a)) with ONE rounded multiply."""
    box32 = np.asarray(box, np.float32)
    n = np.floor(box32.astype(np.float64) / np.float64(np.float32(r_cut))).astype(np.int64)
    inv = (n.astype(np.float64) / box32.astype(np.float64)).astype(np.float32)
    x = np.asarray(pos, np.float32).copy()
    for a in range(3):
        hi = x[:, a] >= box32[a]
        x[hi, a] = x[hi, a] - box32[a]
        lo = x[:, a] < np.float32(0)
        x[lo, a] = x[lo, a] + box32[a]
    t = x * inv[None, :]                      # float32 * float32 -> float32, one rounding
    assert t.dtype == np.float32
    c = np.floor(t).astype(np.int64)
    c = np.minimum(np.maximum(c, 0), n[None, :] - 1)
    return c.astype(np.int32), n.astype(np.int32)


@pytest.mark.parametrize("box,rcut", [((10, 10, 10), 1.58), ((40, 20, 20), 1.58), ((128, 128, 128), 1.58),
                                      ((13, 11, 8), 1.2), ((7.3, 9.1, 5.5), 1.0)])
def test_bin_fp32_matches_numpy_float32_rule(orc, box, rcut):
    rng = np.random.Generator(np.random.PCG64(12))
    box32 = np.asarray(box, np.float32)
    pos = (rng.random((20000, 3)) * box32).astype(np.float32)
    # the wrap cases: x = L, x just below L, x < 0, x = 0, x on cell boundaries (k / inv rounded both ways)
    top = np.nextafter(box32, np.float32(0))
    special = [box32, top, -np.float32(1e-3) * np.ones(3, np.float32), np.zeros(3, np.float32),
               box32 + np.float32(0.25), np.float32(-0.5) * np.ones(3, np.float32)]
    n = np.floor(box32.astype(np.float64) / np.float64(np.float32(rcut))).astype(int)
    edge = (box32.astype(np.float64) / n)
    for k in range(1, 4):
        b = (k * edge).astype(np.float32)
        special += [b, np.nextafter(b, np.float32(0)), np.nextafter(b, np.float32(1e9))]
    pos = np.concatenate([pos, np.asarray(special, np.float32)])
    cells, nc = orc.bin_fp32(box, rcut, pos)
    ref, nref = _bin_numpy(box, rcut, pos)
    assert np.array_equal(nc, nref)
    assert np.array_equal(cells, ref)
    assert cells.min() >= 0 and np.all(cells.max(axis=0) <= nc - 1)


def _census_numpy(pos, ids_rbc, box, rc, rcc, excl):
    n = len(pos)
    n_rc = np.zeros(n, np.int32); n_rcc = np.zeros(n, np.int32)
    x_rc = np.zeros(n, np.uint32); x_rcc = np.zeros(n, np.uint32)
    box = np.asarray(box, np.float64)
    for i in range(n):
        d = pos[i] - pos
        d -= box * np.floor(d / box + 0.5)
        r = np.sqrt((d * d).sum(1))
        ok = np.ones(n, bool)
        ok[i] = False
        if excl:
            ok &= ~((ids_rbc == ids_rbc[i]) & (ids_rbc[i] > 0))
        ok &= (d * d).sum(1) >= 1e-12
        ja = np.flatnonzero(ok & (r < rc)); jb = np.flatnonzero(ok & (r < rcc))
        n_rc[i], n_rcc[i] = len(ja), len(jb)
        x_rc[i] = np.bitwise_xor.reduce(ja.astype(np.uint32)) if len(ja) else 0
        x_rcc[i] = np.bitwise_xor.reduce(jb.astype(np.uint32)) if len(jb) else 0
    return n_rc, n_rcc, x_rc, x_rcc


@pytest.mark.parametrize("box,rc,rcc", [((5, 5, 5), 1.0, 1.58), ((8, 6, 7), 1.0, 1.58), ((6, 6, 6), 1.5, 1.2),
                                        ((7, 7, 7), 1.7, 0.8)])   # last: r_c > 2 r_cc
def test_neighbor_census_matches_brute_force_numpy(orc, box, rc, rcc):
    w = W.make_fluid("t", box, 3.0, seed=5, r_c=rc, r_cc=rcc)
    o = orc.Oracle.from_workload(w)
    c = o.neighbor_census()
    pos = w.pos.astype(np.float64)
    n_rc, n_rcc, x_rc, x_rcc = _census_numpy(pos, np.zeros(len(pos), np.int32), box, float(np.float32(rc)),
                                             float(np.float32(rcc)), True)
    assert np.array_equal(c["n_rc"], n_rc) and np.array_equal(c["n_rcc"], n_rcc)
    assert np.array_equal(c["xor_rc"], x_rc) and np.array_equal(c["xor_rcc"], x_rcc)
    # margin = distance of the closest pair to either cutoff
    d = pos[:, None, :] - pos[None, :, :]
    d -= np.asarray(box, np.float64) * np.floor(d / np.asarray(box, np.float64) + 0.5)
    r = np.sqrt((d ** 2).sum(-1)); np.fill_diagonal(r, 1e9)
    mg = np.minimum(np.abs(r - float(np.float32(rc))), np.abs(r - float(np.float32(rcc))))
    near = r < 2 * max(rc, rcc)
    assert np.allclose(c["margin"], np.where(near, mg, 1e30).min(axis=1), rtol=0, atol=1e-12)


def test_neighbor_census_excludes_same_membrane_pairs_only(orc):
    w = W.small_suspension(seed=2, box=(18, 18, 8), n_rbc=1)
    o = orc.Oracle.from_workload(w)
    c = o.neighbor_census()
    pos, vel, typ, conc, rid = w.all_particles()
    rc, rcc = float(w.params["r_c"]), float(w.params["r_cc"])
    n_rc, n_rcc, x_rc, x_rcc = _census_numpy(pos.astype(np.float64), rid, w.params["box"], rc, rcc, True)
    assert np.array_equal(c["n_rc"], n_rc) and np.array_equal(c["n_rcc"], n_rcc)
    assert np.array_equal(c["xor_rc"], x_rc) and np.array_equal(c["xor_rcc"], x_rcc)
    # and the exclusion matters: without it the membrane vertices would see their bonded neighbours
    n2 = _census_numpy(pos.astype(np.float64), rid, w.params["box"], rc, rcc, False)[1]
    mem = rid > 0
    assert np.all(n2[mem] > n_rcc[mem]) and np.array_equal(n2[~mem], n_rcc[~mem])


def test_species_gaussian_wiring(orc):
    """DESIGN.md R-RNG: tag 0 -> (xi, zeta_0, zeta_1, -); species 2 + 4q .. 5 + 4q <- the four Gaussians of tag 4 + q."""
    S = 10
    p = W.fluid_params((10, 10, 10), 4.0, n_species=S, m_s=0.03, kappa=7.0, seed=77)
    i, j, step, r = 11, 4, 9, 0.9
    Ci = np.full(S, 0.4); Cj = np.full(S, 0.4)          # dC = 0: only the random flux is left
    kind, F, Q = orc.pair_terms(p, i, j, 0, 0, [0, 0, r], [0, 0, 0], Ci, Cj, step)
    g0 = orc.gauss4(i, j, step, 0, 77)
    g4 = orc.gauss4(i, j, step, 4, 77)
    g5 = orc.gauss4(i, j, step, 5, 77)
    zeta = [g0[1], g0[2], g4[0], g4[1], g4[2], g4[3], g5[0], g5[1], g5[2], g5[3]]
    rcc, ms, dt = float(np.float32(1.58)), float(np.float32(0.03)), float(np.float32(0.01))
    amp = -ms * np.sqrt(7.0 * 4.0 * 0.8) * (1 - r / rcc) / np.sqrt(dt)     # sgn = -1: id_i > id_j
    assert kind == 2
    assert np.allclose(Q, amp * np.asarray(zeta), rtol=1e-10, atol=0)
    assert len(set(np.round(zeta, 12))) == S                               # ten different Gaussians
    # xi of the force is g0[0]
    p2 = W.fluid_params((10, 10, 10), 4.0, a=0.0, gamma=4.5, m_s=0.0, seed=77)
    F2 = orc.pair_terms(p2, i, j, 0, 0, [0, 0, r], [0, 0, 0], [0], [0], step)[1]
    assert F2[2] == pytest.approx(3.0 * np.sqrt(1 - r) * g0[0] / np.sqrt(dt), rel=1e-10)


@pytest.mark.parametrize("s_R,s_c", [(0.41, 1.5), (1.0, 3.0), (0.25, 1.0)])
def test_general_exponents_closed_form(orc, s_R, s_c):
    """omega_R = (1 - r/r_c)^s_R, omega_D = omega_R^2 (Eq 5-6, R3); omega_DC = (1 - r/r_cc)^s_c, omega_RC = omega_DC^(1/2)
    (Eq 8-10, R4) written out with ** for exponents other than 1/2 and 2."""
    gam, kap, a, ms, rho, kBT = 4.5, 6.0, 18.75, 0.04, 4.0, 1.0
    p = W.fluid_params((10, 10, 10), rho, a=a, gamma=gam, s_R=s_R, s_c=s_c, kappa=kap, m_s=ms, seed=5)
    d = np.array([0.3, -0.4, 0.5]); dv = np.array([0.7, 0.1, -0.9])
    r = np.linalg.norm(d); e = d / r
    Ci, Cj = [0.9], [0.35]
    kind, F, Q = orc.pair_terms(p, 3, 8, 0, 0, d, dv, Ci, Cj, 2)
    g = orc.gauss4(3, 8, 2, 0, 5)
    f32 = lambda v: float(np.float32(v))
    rc, rcc, dt = f32(1.0), f32(1.58), f32(0.01)
    wc = 1 - r / rc
    wR = wc ** f32(s_R)
    f = f32(a) * wc - f32(gam) * wR ** 2 * e.dot(dv) + np.sqrt(2 * kBT * f32(gam)) * wR * g[0] / np.sqrt(dt)
    assert kind == 2 and np.allclose(F, f * e, rtol=1e-11, atol=0)
    w = 1 - r / rcc
    q = -f32(kap) * w ** f32(s_c) * (Ci[0] - Cj[0]) + f32(ms) * np.sqrt(f32(kap) * rho * (Ci[0] + Cj[0])) \
        * w ** (0.5 * f32(s_c)) * g[1] / np.sqrt(dt)
    assert Q[0] == pytest.approx(q, rel=1e-11)
