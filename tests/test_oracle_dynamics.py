"""Pins for the oracle's time stepping: conservation over a run, equilibrium temperature (Eq 6), diffusion of a
concentration step against Eq 11-12, integrator order / reversibility, and the RBC at rest (BASELINE north_star)."""
import numpy as np
import pytest

import tdpd_workloads as W


def kinetic_T(v):
    v = v - v.mean(0)
    return (v ** 2).sum() / (3 * len(v) - 3)


def test_conservation_over_a_run_with_body_force(orc):
    """Momentum changes by exactly dt * sum g_i per step (double Poiseuille: zero net input up to the z-split),
    total concentration is constant (Eq 7 without Q^S; antisymmetric Eq 8-9)."""
    w = W.make_fluid("t", (6, 6, 6), 4.0, seed=31, conc="uniform", body=0.3, body_mode=W.BODY_UNIFORM)
    o = orc.Oracle.from_workload(w)
    s0 = o.get_state(forces=False)
    o.step(20)
    s1 = o.get_state(forces=False)
    n, dt = w.n_total, float(np.float32(0.01))
    dP = s1["vel"].sum(0) - s0["vel"].sum(0)
    assert dP[0] == pytest.approx(20 * dt * n * float(np.float32(0.3)), rel=1e-9)
    assert abs(dP[1]) < 1e-9 and abs(dP[2]) < 1e-9
    assert s1["conc"].sum() == pytest.approx(s0["conc"].sum(), rel=1e-13)
    assert s1["step"] == 20
    # double Poiseuille: +f below Lz/2, -f above, evaluated at the force-evaluation positions
    w2 = W.make_fluid("t", (6, 6, 6), 4.0, seed=31, conc="zero", body=0.3, body_mode=W.BODY_DOUBLE_POISEUILLE_Z,
                      a=0.0, gamma=0.0, kBT=0.0)
    w2.vel[:] = 0
    o2 = orc.Oracle.from_workload(w2)
    o2.step(1)
    v = o2.get_state(forces=False)["vel"]
    up = w2.pos[:, 2] < 3.0
    assert np.allclose(v[up, 0], dt * float(np.float32(0.3)), rtol=1e-12)
    assert np.allclose(v[~up, 0], -dt * float(np.float32(0.3)), rtol=1e-12)


def test_step_batching_is_irrelevant(orc):
    w = W.make_fluid("t", (5, 5, 5), 4.0, seed=32, conc="uniform")
    a, b = orc.Oracle.from_workload(w), orc.Oracle.from_workload(w)
    a.step(6)
    for _ in range(6):
        b.step(1)
    sa, sb = a.get_state(), b.get_state()
    for k in ("pos", "vel", "conc", "force", "flux"):
        assert np.array_equal(sa[k], sb[k])


def test_velocity_verlet_order_and_reversibility(orc):
    """gamma = sigma = kappa = 0: H = KE + sum a r_c/2 (1-r/r_c)^2 has error ~ dt^2; reversing v retraces the path."""
    def run(dt, nsteps):
        w = W.make_fluid("t", (5, 5, 5), 4.0, seed=33, conc="uniform", gamma=0.0, kappa=0.0, m_s=0.0, dt=dt)
        w.vel *= 0.3
        o = orc.Oracle.from_workload(w)
        return w, o

    def energy(w, s):
        x, v = s["pos"], s["vel"]
        box = w.params["box"].astype(np.float64)
        d = x[:, None] - x[None]; d -= box * np.round(d / box)
        r = np.sqrt((d ** 2).sum(-1)); np.fill_diagonal(r, 9.0)
        a = float(w.params["a"][0, 0])
        return 0.5 * (v ** 2).sum() + 0.5 * (0.5 * a * np.clip(1 - r, 0, None) ** 2).sum()

    errs = []
    for dt, n in ((0.01, 10), (0.005, 20)):
        w, o = run(dt, n)
        e0 = energy(w, o.get_state(forces=False))
        dev = 0.0
        for _ in range(n):
            o.step(1)
            dev = max(dev, abs(energy(w, o.get_state(forces=False)) - e0))
        errs.append(dev)
    assert 3.0 < errs[0] / errs[1] < 5.5                       # second order: halving dt quarters the error
    w, o = run(0.01, 0)
    s0 = o.get_state(forces=False)
    o.step(15)
    s = o.get_state(forces=False)
    o.set_state(v=-s["vel"])
    o.step(15)
    s2 = o.get_state(forces=False)
    d = s2["pos"] - s0["pos"]; d -= 5.0 * np.round(d / 5.0)
    assert np.abs(d).max() < 1e-10 and np.abs(s2["vel"] + s0["vel"]).max() < 1e-10


def test_equilibrium_temperature_matches_kBT(orc):
    """Fluctuation-dissipation theorem, Eq 6: <kBT> within 1 % of 1.0 (config-1 parameters; time average after
    the initial potential-energy release has been thermostatted away)."""
    w = W.config(1)
    o = orc.Oracle.from_workload(w)
    o.step(150)
    T = []
    for _ in range(70):
        o.step(5)
        T.append(kinetic_T(o.get_state(forces=False)["vel"]))
    assert np.mean(T) == pytest.approx(1.0, abs=0.01)


def test_concentration_step_relaxes_with_tdpd_diffusivity(orc):
    """Periodic square wave C(x,0) = [x < L/2]: mode k decays as exp(-D k^2 t), D = D^F + D^zeta with
    D^F = (2 pi kappa rho / 3) int r^4 w_DC g dr (Eq 12) and D^zeta = 3 kBT / (4 pi gamma rho int r^2 w_D g dr)
    (Eq 11), both evaluated with the run's own measured g(r)."""
    L = (32.0, 6.32, 6.32)
    w = W.make_fluid("t", L, 4.0, seed=41, conc="step", m_s=0.0)
    o = orc.Oracle.from_workload(w)
    o.step(60)                                               # let the fluid structure (g(r)) equilibrate
    k1 = 2 * np.pi / L[0]
    ts, amp = [], []
    for it in range(30):
        s = o.get_state(forces=False)
        amp.append(2 * np.mean(s["conc"][:, 0] * np.sin(k1 * s["pos"][:, 0])))
        ts.append(o.step_count * 0.01)
        o.step(4)
    rate = -np.polyfit(ts, np.log(amp), 1)[0]
    D_meas = rate / k1 ** 2
    # measured g(r)
    x = o.get_state(forces=False)["pos"]
    box = np.asarray(L)
    edges = np.linspace(0, 1.58, 80)
    hist = np.zeros(len(edges) - 1)
    for i0 in range(0, len(x), 512):
        d = x[i0:i0 + 512, None] - x[None]
        d -= box * np.round(d / box)
        r = np.sqrt((d ** 2).sum(-1)).ravel()
        hist += np.histogram(r[r > 1e-9], edges)[0]
    rm = 0.5 * (edges[1:] + edges[:-1]); dr = edges[1] - edges[0]
    rho = len(x) / box.prod()
    g = hist / (len(x) * rho * 4 * np.pi * rm ** 2 * dr)
    kappa, gamma, kBT, rcc = 10.0, 4.5, 1.0, 1.58
    DF = 2 * np.pi * kappa * rho / 3 * np.sum(rm ** 4 * (1 - rm / rcc) ** 2 * g) * dr
    wD = np.clip(1 - rm, 0, None)                            # w_D = w_R^2 = 1 - r/r_c at s = 1/2
    Dz = 3 * kBT / (4 * np.pi * gamma * rho * np.sum(rm ** 2 * wD * g) * dr)
    # g = 1 closed forms quoted in SURVEY §8(c): D^F = 2 pi kappa rho r_cc^5 / 315, D^zeta = 9 kBT / (pi gamma rho r_c^3)
    assert 2 * np.pi * kappa * 4 * rcc ** 5 / 315 == pytest.approx(7.856, abs=2e-3)
    assert DF == pytest.approx(7.856, rel=0.06) and Dz == pytest.approx(0.159, rel=0.25)
    assert D_meas == pytest.approx(DF + Dz, rel=0.06)
    assert amp[0] == pytest.approx(2 / np.pi * np.exp(-(DF + Dz) * k1 ** 2 * 0.6), rel=0.08)


def test_rbc_at_rest_holds_area_and_volume(orc):
    """BASELINE: "An RBC at rest holds its area and volume within 0.5 % of target" (reduced box, f = 0)."""
    w = W.small_suspension(box=(17, 17, 9), body=0.0, body_mode=W.BODY_OFF)
    o = orc.Oracle.from_workload(w)
    o.step(100)
    dev_a, dev_v = [], []
    for _ in range(10):
        o.step(10)
        st = o.rbc_stats()
        dev_a.append(st["area"][0] / st["A0"][0] - 1)
        dev_v.append(st["volume"][0] / st["V0"][0] - 1)
    assert np.abs(dev_a).max() < 0.005 and np.abs(dev_v).max() < 0.005
    s = o.get_state(forces=False)
    assert np.isfinite(s["pos"]).all()
    assert kinetic_T(s["vel"][-642:]) == pytest.approx(1.0, abs=0.15)     # membrane thermalised by Eq 15/16


def test_trajectory_sensitivity_of_the_oracle_itself(orc):
    """DESIGN.md reading R-traj (why "positions after 100 steps within 1e-3 r_c" is a statement about N): two runs of the
    ORACLE on config 1 whose initial positions differ by one fp32 rounding (|dx0| <= 3e-7) drift apart exponentially,
    the maximum over the particles growing by more than 2x per 25 steps.  The GPU-vs-oracle difference grows at the
    same rate from the fp32 round-off of the forces, so its maximum depends on the number of particles."""
    w = W.config(1)
    a = orc.Oracle.from_workload(w)
    b = orc.Oracle.from_workload(w)
    s0 = a.get_state(forces=False)
    rng = np.random.Generator(np.random.PCG64(9))
    x = s0["pos"] * (1.0 + (rng.random(s0["pos"].shape) - 0.5) * 2.0 ** -23)     # within half an fp32 ulp
    b.set_state(x, None, None)
    box = np.asarray(w.params["box"], np.float64)
    gaps = [np.abs(x - s0["pos"]).max()]
    for _ in range(4):
        a.step(25); b.step(25)
        d = a.get_state(forces=False)["pos"] - b.get_state(forces=False)["pos"]
        d -= box * np.round(d / box)
        gaps.append(np.abs(d).max())
    print("[sensitivity] max |dx| at steps 0, 25, 50, 75, 100:", ["%.2e" % g for g in gaps])
    assert gaps[0] < 1e-6                              # half an fp32 ulp of a coordinate below 10
    assert gaps[4] > 100 * gaps[0]                     # two orders of magnitude in one time unit (measured: ~800x)
    assert gaps[4] > 2.0 * gaps[2] > 2.0 * gaps[0]     # and still growing between steps 50 and 100


def test_source_term_first_order_kinetics(orc):
    """Q^S of Eq 7 (reading R-QS): Q^S_i = source - decay C_i by species and type.  With a
    uniform concentration the Fickian flux vanishes (m_s = 0: no random flux), so every particle follows
    dC/dt = q - k C:  C(t) = q/k + (C_0 - q/k) exp(-k t), whatever the particles do."""
    q, k, C0 = 0.3, 0.8, 1.5
    w = W.make_fluid("t", (6, 6, 6), 3.0, seed=4, m_s=0.0, source=q, decay=k)
    w.conc[:] = C0
    o = orc.Oracle.from_workload(w)
    o.step(100)
    C = o.get_state(forces=False)["conc"][:, 0]
    exact = q / k + (C0 - q / k) * np.exp(-k * 1.0)
    assert np.ptp(C) < 1e-12                                   # uniform stays uniform
    assert C.mean() == pytest.approx(exact, rel=3e-3)          # Q is evaluated with the half-step C (R21): first order in dt
    # halving the time step halves the error
    e = []
    for dt, n in ((0.02, 50), (0.01, 100)):
        w2 = W.make_fluid("t", (6, 6, 6), 3.0, seed=4, m_s=0.0, source=q, decay=k, dt=dt)
        w2.conc[:] = C0
        o2 = orc.Oracle.from_workload(w2)
        o2.step(n)
        e.append(abs(o2.get_state(forces=False)["conc"][:, 0].mean() - exact))
    assert 1.7 < e[0] / e[1] < 2.4
    # by type: only type-1 particles decay; and the flux reported at a force evaluation contains Q^S
    p = W.fluid_params((6, 6, 6), 3.0, n_types=2, m_s=0.0, kappa=0.0, decay=[0.0, 2.0], seed=4)
    o3 = orc.Oracle(p)
    pos = np.array([[1, 1, 1], [4, 4, 4]], np.float32)
    o3.load_particles(pos, np.zeros((2, 3), np.float32), np.array([0, 1], np.int32), np.array([[0.5], [0.5]], np.float32))
    o3.compute_forces(0)
    assert np.allclose(o3.get_state()["flux"][:, 0], [0.0, -1.0], atol=1e-7)
