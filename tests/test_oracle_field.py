"""Pins for the oracle's local field terms, torque and Dormand-Prince stepper (CPU only)."""
import numpy as np
import pytest

from oracle import field as fld
from oracle import sim as osim
from oracle import RefSim, MM_DEMAG, MM_EXCH, MM_ANIS, MM_ZEEMAN, MM_ALL
from synth import Params, random_unit_vectors

GAMMA = 1.7595e11


def _rand_m(seed, shape):
    return random_unit_vectors(seed, int(np.prod(shape))).astype(np.float64).reshape((3,) + tuple(shape))


# ------------------------------------------------------------------ exchange
def test_exchange_field_vanishes_for_uniform_m():
    rng = np.random.default_rng(0)
    regions = rng.integers(0, 5, size=(3, 6, 7))
    S = rng.uniform(0.5, 1.0, size=15)
    p = Params.uniform(5, Msat=rng.uniform(5e5, 1e6, 5), Aex=rng.uniform(1e-11, 2e-11, 5), exch_scale=S)
    L = fld.exchange_table(p.Aex, p.Msat, p.exch_scale)
    m = np.zeros((3, 3, 6, 7)); m[0], m[1], m[2] = 0.6, 0.0, 0.8
    for pbc in ((0, 0, 0), (1, 1, 1)):
        assert np.abs(fld.b_exchange(m, regions, L, (1e-9, 2e-9, 3e-9), pbc)).max() == 0.0


def test_exchange_spiral_energy_matches_the_papers_closed_form():
    # N = 1024 cells of 1 nm with PBC, m rotating k times in the yz-plane;
    # exact energy (Eq. 7) = vol * A * (2 pi k / (N c))^2.  Eq. 6 + Eq. 8 give instead
    # (2A/c^2)(1 - cos theta) per unit volume, theta = 2 pi k / N.
    N, c, A, Ms = 1024, 1e-9, 10e-12, 1e6
    sim = RefSim((N, 1, 1), (c, c, c), (1, 0, 0))
    sim.set_params(Params.uniform(1, Msat=Ms, Aex=A))
    vol = N * c ** 3
    i = np.arange(N)
    for k in (1, 8, 32, 100):
        phase = i * k * 2 * np.pi / N
        m = np.zeros((3, 1, 1, N)); m[1, 0, 0] = np.sin(phase); m[2, 0, 0] = np.cos(phase)
        B = fld.b_exchange(m, sim.regions, sim.L, sim.cell, sim.pbc)
        E = (-0.5 * Ms * (m * B).sum()) * c ** 3                       # Eq. 8
        theta = 2 * np.pi * k / N
        exact = vol * A * (2 * np.pi * k / (N * c)) ** 2               # L723
        assert np.isclose(E / exact, 2 * (1 - np.cos(theta)) / theta ** 2, rtol=1e-10)
        if k <= 8:
            assert np.isclose(E, exact, rtol=theta ** 2 / 10)           # small-angle limit (Fig. 5)


def test_exchange_neumann_boundary_and_axis_spacing():
    # 3 cells along y with a linear tilt: the middle cell sees +d and -d (field 0), the edge cells see
    # one neighbour only; prefactor 2A/(Ms dy^2)
    A, Ms, dy = 1.3e-11, 8e5, 2e-9
    sim = RefSim((1, 3, 1), (5e-9, dy, 7e-9))
    sim.set_params(Params.uniform(1, Msat=Ms, Aex=A))
    m = np.zeros((3, 1, 3, 1)); m[0] = 1.0; m[1, 0, :, 0] = (-0.01, 0.0, 0.01)
    B = fld.b_exchange(m, sim.regions, sim.L, sim.cell, sim.pbc)
    assert np.isclose(B[1, 0, 0, 0], 2 * A / Ms * 0.01 / dy ** 2, rtol=1e-12)
    assert abs(B[1, 0, 1, 0]) < 1e-12 and np.isclose(B[1, 0, 2, 0], -B[1, 0, 0, 0], rtol=1e-12)


def test_interregion_exchange_is_the_harmonic_mean_with_scale():
    # Eq. 9 (L208): 2 S (2 q1 q2)/(q1+q2), q = Aex/Msat; equal materials reduce to Eq. 6
    A = np.array([1.0e-11, 2.0e-11]); M = np.array([5e5, 8e5])
    L = fld.exchange_table(A, M, np.array([1.0, 0.25, 1.0]))
    q = A / M
    assert np.isclose(L[0, 0], q[0]) and np.isclose(L[1, 1], q[1])
    assert np.isclose(L[0, 1], 0.25 * 2 * q[0] * q[1] / (q[0] + q[1])) and L[0, 1] == L[1, 0]
    assert np.isclose(fld.exchange_table(A[[0, 0]], M[[0, 0]], None)[0, 1], q[0])
    assert fld.exchange_table(np.array([1e-11, 0.0]), np.array([8e5, 0.0]), None)[0, 1] == 0.0   # vacuum


# ------------------------------------------------------------------ anisotropy
def _params_anis(rng, n):
    p = Params.uniform(n, Msat=rng.uniform(5e5, 1e6, n), Ku1=rng.uniform(-5e5, 5e5, n), Ku2=rng.uniform(-2e5, 2e5, n),
                       Kc1=rng.uniform(-5e4, 5e4, n), Kc2=rng.uniform(-5e4, 5e4, n), Kc3=rng.uniform(-5e4, 5e4, n))
    p.anisU = rng.normal(size=(n, 3))
    c1 = rng.normal(size=(n, 3)); c1 /= np.linalg.norm(c1, axis=1, keepdims=True)
    t = rng.normal(size=(n, 3)); c2 = t - (t * c1).sum(1, keepdims=True) * c1
    p.anisC1, p.anisC2 = c1 * 3.0, c2           # not normalised on purpose
    return p


def _energy_density_eq19_eq22(m, regions, p):
    """Eq. 19 (L274) and Eq. 22 (L288, garbled; reading SURVEY.md 8(c) #6) written independently."""
    u = p.anisU / np.linalg.norm(p.anisU, axis=1, keepdims=True)
    c1 = p.anisC1 / np.linalg.norm(p.anisC1, axis=1, keepdims=True)
    c2 = p.anisC2 / np.linalg.norm(p.anisC2, axis=1, keepdims=True)
    c3 = np.cross(c1, c2)
    dot = lambda v: np.einsum("zyxc,czyx->zyx", v[regions], m)
    um, a1, a2, a3 = dot(u), dot(c1), dot(c2), dot(c3)
    e = -p.Ku1[regions] * um ** 2 - p.Ku2[regions] * um ** 4
    e += p.Kc1[regions] * (a1 ** 2 * a2 ** 2 + a1 ** 2 * a3 ** 2 + a2 ** 2 * a3 ** 2)
    e += p.Kc2[regions] * (a1 ** 2 * a2 ** 2 * a3 ** 2)
    e += p.Kc3[regions] * (a1 ** 4 * a2 ** 4 + a1 ** 4 * a3 ** 4 + a2 ** 4 * a3 ** 4)
    return e


def test_anisotropy_energy_identities_eq20_eq23():
    rng = np.random.default_rng(5)
    shape = (2, 3, 4)
    regions = rng.integers(0, 3, size=shape)
    p = _params_anis(rng, 3)
    m = _rand_m(9, shape)
    M = p.Msat[regions][None] * m
    e = (-0.5 * (M * fld.b_anis_uniaxial(m, regions, p, only=1)).sum(0)
         - 0.25 * (M * fld.b_anis_uniaxial(m, regions, p, only=2)).sum(0)
         - (1 / 4) * (M * fld.b_anis_cubic(m, regions, p, only=1)).sum(0)
         - (1 / 6) * (M * fld.b_anis_cubic(m, regions, p, only=2)).sum(0)
         - (1 / 8) * (M * fld.b_anis_cubic(m, regions, p, only=3)).sum(0))
    assert np.allclose(e, _energy_density_eq19_eq22(m, regions, p), rtol=1e-11, atol=1e-6)


def test_anisotropy_field_is_minus_dE_dM():
    rng = np.random.default_rng(6)
    shape = (1, 2, 3)
    regions = rng.integers(0, 2, size=shape)
    p = _params_anis(rng, 2)
    m = _rand_m(10, shape) * 0.9            # off the unit sphere on purpose: B = -dE/dM holds for any m
    B = fld.b_anis_uniaxial(m, regions, p) + fld.b_anis_cubic(m, regions, p)
    h = 1e-6
    for c in range(3):
        mp = m.copy(); mp[c] += h
        mm = m.copy(); mm[c] -= h
        dE = (_energy_density_eq19_eq22(mp, regions, p) - _energy_density_eq19_eq22(mm, regions, p)) / (2 * h)
        assert np.allclose(B[c], -dE / p.Msat[regions], rtol=1e-6, atol=1e-9)


def test_fig7_uniaxial_energy_versus_angle():
    # L746-L763: Msat 1e6, u = x, m in the xy-plane: E = -Ku1 cos^2(theta) - Ku2 cos^4(theta)
    p = Params.uniform(1, Msat=1000e3, Ku1=1e6, Ku2=-3e5, anisU=(1, 0, 0))
    regions = np.zeros((1, 1, 1), dtype=int)
    for deg in (0, 30, 77, 135, 260):
        th = np.deg2rad(deg)
        m = np.array([np.cos(th), np.sin(th), 0.0]).reshape(3, 1, 1, 1)
        M = 1000e3 * m
        e = -0.5 * (M * fld.b_anis_uniaxial(m, regions, p, only=1)).sum() - 0.25 * (M * fld.b_anis_uniaxial(m, regions, p, only=2)).sum()
        assert np.isclose(e, -1e6 * np.cos(th) ** 2 + 3e5 * np.cos(th) ** 4, rtol=1e-12, atol=1e-6)


# ------------------------------------------------------------------ torque and time stepping
def _macrospin(alpha=0.0, B=(0, 0, 0.1), m0=(1, 0, 0)):
    sim = RefSim((1, 1, 1), (1e-9, 1e-9, 1e-9))
    sim.set_params(Params.uniform(1, Msat=1 / fld.MU0, Aex=10e-12, alpha=alpha, B_ext=B))
    sim.set_terms(MM_EXCH | MM_ANIS | MM_ZEEMAN)         # EnableDemag = false (L611)
    sim.set_m(np.array(m0, dtype=float).reshape(3, 1, 1, 1))
    return sim


def test_fig3_larmor_precession():
    # Fig. 3 (L97): m_x = cos(gamma_LL * 0.1 T * t); frequency gamma B / 2 pi = 2.8003 GHz
    sim = _macrospin()
    sim.set_solver(max_err=1e-7)
    for t in (0.1e-9, 0.35e-9, 1.0e-9):
        sim.run(t - sim.t)
        mx, my, mz = sim.m[:, 0, 0, 0]
        assert abs(mx - np.cos(GAMMA * 0.1 * t)) < 2e-6 and abs(mz) < 1e-12
        assert abs(my - np.sin(GAMMA * 0.1 * t)) < 2e-6          # sense fixed by the sign reading #5
    assert np.isclose(GAMMA * 0.1 / (2 * np.pi), 2.8003e9, rtol=1e-4)


def test_damping_moves_m_towards_the_field_and_lowers_the_energy():
    sim = _macrospin(alpha=0.3, m0=(1, 0, 0.2))
    sim.set_solver(max_err=1e-6)
    e0, mz0 = sim.energy(), sim.m[2, 0, 0, 0]
    sim.run(0.2e-9)
    assert sim.m[2, 0, 0, 0] > mz0 and sim.energy() < e0


def test_fig10_fifth_order_convergence_over_one_period():
    # L840-L865: m = (1,0,1)/sqrt2, B = 0.1 T z, one period 2 pi/(B gamma); error ~ dt^5
    period = 2 * np.pi / (0.1 * GAMMA)
    errs = []
    for n in (20, 40, 80):
        sim = _macrospin(m0=(1, 0, 1))
        sim.set_solver(fix_dt=period / n)
        for _ in range(n):
            sim.step()
        errs.append(np.linalg.norm(sim.m[:, 0, 0, 0] - np.array([1, 0, 1]) / np.sqrt(2)))
    assert 26 < errs[0] / errs[1] < 60 and 26 < errs[1] / errs[2] < 42    # 2^5 = 32 asymptotically
    assert errs[2] < 1e-7


def test_fig11_end_error_scales_with_maxerr():
    period = 2 * np.pi / (0.1 * GAMMA)
    errs = []
    for tol in (1e-4, 1e-5, 1e-6):
        sim = _macrospin(m0=(1, 0, 1))
        sim.set_solver(max_err=tol, dt_init=1e-13)
        sim.run(period)
        assert abs(sim.t - period) < 1e-24
        errs.append(np.linalg.norm(sim.m[:, 0, 0, 0] - np.array([1, 0, 1]) / np.sqrt(2)))
    assert 3 < errs[0] / errs[1] < 30 and 3 < errs[1] / errs[2] < 30


def test_dormand_prince_tableau_conditions():
    A, c, b5, b4 = osim.DP_A, np.array(osim.DP_C), np.array(osim.DP_B5), np.array(osim.DP_B4)
    for i in range(7):
        assert abs(sum(A[i]) - c[i]) < 1e-15
    assert tuple(A[6]) == tuple(b5[:6])                      # FSAL: stage 7 is evaluated at y_{n+1}
    for q in range(5):                                        # quadrature conditions up to order 5 / 4
        assert abs((b5 * c ** q).sum() - 1 / (q + 1)) < 1e-15
    for q in range(4):
        assert abs((b4 * c ** q).sum() - 1 / (q + 1)) < 1e-15
    Am = np.zeros((7, 7))
    for i in range(7):
        Am[i, :len(A[i])] = A[i]
    assert abs(b5 @ Am @ c - 1 / 6) < 1e-15 and abs(b4 @ Am @ c - 1 / 6) < 1e-15
    assert abs(b5 @ Am @ Am @ c - 1 / 24) < 1e-15 and abs(b5 @ Am @ Am @ Am @ c - 1 / 120) < 1e-15
    assert abs(sum(osim.DP_E)) < 1e-15


def test_bogacki_shampine_tableau_conditions_and_third_order_convergence():
    # RK23 (L366): 3rd-order solution, 2nd-order embedded estimate, FSAL; Fig. 10 shows its 3rd-order slope
    A, b3, b2 = osim.BS_A, np.array(osim.BS_B3), np.array(osim.BS_B2)
    c = np.array([sum(r) for r in A])
    assert np.allclose(c, [0, 1 / 2, 3 / 4, 1]) and tuple(A[3]) == tuple(b3[:3])      # FSAL
    for q in range(3):
        assert abs((b3 * c ** q).sum() - 1 / (q + 1)) < 1e-15
    for q in range(2):
        assert abs((b2 * c ** q).sum() - 1 / (q + 1)) < 1e-15
    Am = np.zeros((4, 4))
    for i in range(4):
        Am[i, :len(A[i])] = A[i]
    assert abs(b3 @ Am @ c - 1 / 6) < 1e-15 and abs(b2 @ Am @ c - 1 / 6) > 1e-3    # order 3 vs only order 2
    assert abs(sum(osim.BS_E)) < 1e-15
    period = 2 * np.pi / (0.1 * GAMMA)
    errs = []
    for n in (40, 80, 160):
        sim = _macrospin(m0=(1, 0, 1))
        sim.set_solver_kind("rk23")
        sim.set_solver(fix_dt=period / n)
        for _ in range(n):
            sim.step()
        errs.append(np.linalg.norm(sim.m[:, 0, 0, 0] - np.array([1, 0, 1]) / np.sqrt(2)))
    assert 6.5 < errs[0] / errs[1] < 10 and 7 < errs[1] / errs[2] < 9.5          # 2^3 = 8 asymptotically
    # adaptive: lands on time, error scales with MaxErr (Fig. 11), three evaluations per step
    sim = _macrospin(m0=(1, 0, 1))
    sim.set_solver_kind("rk23")
    sim.set_solver(max_err=1e-6, dt_init=1e-13)
    sim.run(period)
    assert abs(sim.t - period) < 1e-24
    assert np.linalg.norm(sim.m[:, 0, 0, 0] - np.array([1, 0, 1]) / np.sqrt(2)) < 1e-3
    assert sim.n_eval == 1 + 3 * (sim.n_steps + sim.n_rejected)


def test_no_precession_torque_only_lowers_the_energy():
    # relax() "disables the precession term" (L388): m then moves straight towards B_eff
    sim = _macrospin(alpha=0.5, m0=(1, 0, 0.2))
    sim.precession = False
    sim.set_solver(max_err=1e-6)
    e0 = sim.energy()
    sim.run(0.05e-9)
    mx, my, mz = sim.m[:, 0, 0, 0]
    assert abs(my) < 1e-12 and mz > 0.2 and sim.energy() < e0      # stays in the x-z plane: no precession


def _small_film(alpha, seed=21, grid=(12, 6, 1), fix_dt=0.0):
    sim = RefSim(grid, (4e-9, 4e-9, 3e-9))
    sim.set_params(Params.uniform(1, Msat=8e5, Aex=1.3e-11, alpha=alpha))
    sim.set_m(_rand_m(seed, sim.shape))
    sim.set_solver(fix_dt=fix_dt)
    return sim


def test_norm_conserved_and_energy_monotone_with_damping():
    sim = _small_film(alpha=0.5)
    e = [sim.energy()]
    for _ in range(40):
        info = sim.step()
        if info["accepted"]:
            e.append(sim.energy())
        assert np.abs(np.sqrt((sim.m ** 2).sum(0)) - 1).max() < 1e-14
    e = np.array(e)
    assert len(e) > 10 and np.all(np.diff(e) < 0)


def test_energy_conserved_without_damping():
    sim = _small_film(alpha=0.0)
    sim.set_solver(max_err=1e-7)
    e0 = sim.energy()
    sim.run(5e-12)
    assert abs(sim.energy() - e0) < 1e-6 * abs(e0)


def test_run_lands_on_time_and_fsal_slope_is_consistent():
    sim = _small_film(alpha=0.1)
    sim.run(1e-12); sim.run(0.5e-12)
    assert abs(sim.t - 1.5e-12) < 1e-27
    k1 = sim.k1.copy()
    assert np.allclose(k1, sim.torque(sim.m), rtol=0, atol=1e-3 * np.abs(k1).max() * 1e-9)
    # fixed step: exact count, always accepted
    sim = _small_film(alpha=0.1, fix_dt=1e-13)
    sim.run(1e-12)
    assert sim.n_steps == 10 and sim.n_rejected == 0 and abs(sim.t - 1e-12) < 1e-27


def test_term_mask_sums():
    sim = _small_film(alpha=0.1, grid=(6, 5, 2))
    sim.p.Ku1[:] = 1e5; sim.p.B_ext = np.array([0.01, -0.02, 0.03])
    parts = sum(sim.b_eff(t) for t in (MM_DEMAG, MM_EXCH, MM_ANIS, MM_ZEEMAN))
    assert np.allclose(parts, sim.b_eff(MM_ALL), rtol=1e-13, atol=1e-15)


def test_relax_reaches_a_torque_free_state_of_lower_energy():
    # relax() (L388-L392): the procedure's sampling details are readings (unpinned), its outcome is not:
    # an equilibrium - lower energy, residual torque far below the paper's 1e-4..1e-7 T, nothing moves after
    sim = RefSim((32, 8, 1), (4e-9, 4e-9, 3e-9), demag_method="fft")
    sim.set_params(Params.uniform(1, Msat=8e5, Aex=1.3e-11, alpha=0.5))
    m0 = np.zeros((3, 1, 8, 32)); m0[0] = 1.0; m0[1] = 0.1
    sim.set_m(m0)
    e0 = sim.energy()
    sim.relax()
    assert sim.energy() < e0 and sim.max_torque() < 1e-7
    assert (sim.solver, sim.precession, sim.max_err, sim.fix_dt) == ("rk45", True, 1e-5, 0.0)
    assert abs(np.sqrt((sim.m ** 2).sum(axis=0)) - 1).max() < 1e-12
    before = sim.avg_m().copy()
    sim.run(0.1e-9)                                   # full LLG with precession: an equilibrium stays put
    assert np.abs(sim.avg_m() - before).max() < 1e-6


def test_heun_second_order_convergence_and_adaptive_rule():
    # RK12 (L367): 2nd-order solution, 1st-order (Euler) embedded estimate; Fig. 10 shows its 2nd-order slope
    assert abs(sum(osim.HEUN_B2) - 1) < 1e-15 and abs(sum(osim.HEUN_E)) < 1e-15
    assert abs(osim.HEUN_B2[1] * osim.HEUN_A[1][0] - 0.5) < 1e-15                  # order-2 condition b2 c2 = 1/2
    period = 2 * np.pi / (0.1 * GAMMA)
    errs = []
    for n in (100, 200, 400):
        sim = _macrospin(m0=(1, 0, 1))
        sim.set_solver_kind("rk12")
        sim.set_solver(fix_dt=period / n)
        for _ in range(n):
            sim.step()
        errs.append(np.linalg.norm(sim.m[:, 0, 0, 0] - np.array([1, 0, 1]) / np.sqrt(2)))
    assert 3.8 < errs[0] / errs[1] < 4.2 and 3.9 < errs[1] / errs[2] < 4.1       # 2^2
    sim = _macrospin(m0=(1, 0, 1))
    sim.set_solver_kind("rk12")
    sim.set_solver(max_err=1e-6, dt_init=1e-13)
    sim.run(period)
    assert abs(sim.t - period) < 1e-24 and sim.n_eval == 2 * sim.n_steps + sim.n_rejected   # no FSAL; k1 survives a rejection


def test_thermal_field_amplitude_and_langevin_equilibrium():
    # Eq. 24 (L303-L308). (i) the field of one step has zero mean and the standard deviation of the formula,
    # is reproducible from (seed, step) and changes with the step; (ii) an ensemble of uncoupled macrospins
    # in a field B reaches the Boltzmann distribution: <m_z> = coth(xi) - 1/xi, <m_z^2> = 1 - 2 <m_z>/xi,
    # xi = Msat V B / kT - which fixes the amplitude (twice the variance would give <m_z> = 0.60, not 0.79).
    n, Ms, B, T, c, dt = 64, 1e6, 0.02, 300.0, 10e-9, 2e-12
    sim = RefSim((n, n, 1), (c, c, c))
    sim.set_params(Params.uniform(1, Msat=Ms, Aex=0.0, alpha=1.0, B_ext=(0, 0, B)))
    sim.set_terms(MM_ZEEMAN)
    m = np.zeros((3, 1, n, n)); m[2] = 1.0
    sim.set_m(m)
    sim.set_solver_kind("rk12")
    sim.set_temperature(T, seed=7)
    with pytest.raises(AssertionError):
        sim.step()                                    # adaptive step + thermal field is refused (L310)
    sim.set_solver(fix_dt=dt)
    b0 = sim.b_thermal(dt)
    amp = np.sqrt(2 * fld.MU0 * 1.0 * 1.380649e-23 * T / (fld.MU0 * Ms * GAMMA * c ** 3 * dt))
    assert abs(b0.mean()) < 0.03 * amp and abs(b0.std() / amp - 1) < 0.02
    assert np.array_equal(b0, sim.b_thermal(dt))
    acc1, acc2 = [], []
    for i in range(4000):
        sim.step()
        if i == 0:
            assert not np.array_equal(b0, sim.b_thermal(dt))
        if i > 1500 and i % 10 == 0:
            acc1.append(sim.avg_m()[2]); acc2.append((sim.m[2] ** 2).mean())
    xi = Ms * c ** 3 * B / (1.380649e-23 * T)
    L = 1 / np.tanh(xi) - 1 / xi
    assert abs(np.mean(acc1) - L) < 0.01 and abs(np.mean(acc2) - (1 - 2 * L / xi)) < 0.012
    assert abs(np.sqrt((sim.m ** 2).sum(axis=0)) - 1).max() < 1e-12


def test_sp3_vortex_transition_from_the_stored_oracle_energies():
    # Standard problem 3 (L414-L428): the oracle's relaxed twisted-flower and vortex energies (stored by
    # tests/golden/make_sp3_oracle.py, which calls only oracle/ - 25 minutes of relax() in fp64) must cross
    # at the edge length the paper prints, L = 8.47 (L426, tests/golden/sp3_transitions.txt). This pins
    # relax(), the energies and the 3D field terms of the oracle to a number printed in the paper.
    import os
    g = os.path.join(os.path.dirname(__file__), "golden")
    e = {}
    for line in open(os.path.join(g, "sp3_oracle_energies.txt")):
        if not line.startswith("#"):
            L, kind, val = line.split()[:3]
            e[(float(L), kind)] = float(val)
    paper = {l.split()[0]: float(l.split()[1]) for l in open(os.path.join(g, "sp3_transitions.txt"))
             if l.strip() and not l.startswith("#")}
    d0 = e[(8.44, "twisted")] - e[(8.44, "vortex")]
    d1 = e[(8.50, "twisted")] - e[(8.50, "vortex")]
    assert d0 < 0 < d1
    assert abs(8.44 + 0.06 * d0 / (d0 - d1) - paper["twisted_flower_to_vortex"]) < 0.01


def test_slonczewski_torque_closed_form_for_a_macrospin():
    # Eq. 28-30 (L336-L347) with Lambda = 1 (eps = P/2), eps' = 0, no field: the polar angle to m_P obeys
    # d theta/dt = -gamma beta eps/(1+alpha^2) sin theta, i.e. tan(theta/2) = tan(theta0/2) exp(-gamma beta eps t/(1+alpha^2)),
    # and the azimuth turns at the constant rate -alpha gamma beta eps/(1+alpha^2) (the +alpha eps m x m_P term:
    # m x z = (m_y, -m_x, 0) turns m clockwise about m_P).
    Ms, d, jz, P, alpha = 8e5, 2e-9, 4e11, 0.6, 0.05
    sim = RefSim((1, 1, 1), (5e-9, 5e-9, d))
    sim.set_params(Params.uniform(1, Msat=Ms, Aex=0.0, alpha=alpha))
    sim.set_terms(MM_ZEEMAN)                             # no field at all
    th0 = 2.0
    sim.set_m(np.array([np.sin(th0), 0.0, np.cos(th0)]).reshape(3, 1, 1, 1))
    sim.set_slonczewski(jz, P, lam=1.0, eps_prime=0.0, mp=(0, 0, 1))
    sim.set_solver(max_err=1e-8)
    beta = jz * fld.HBAR / (Ms * fld.E_CHARGE * d)       # tesla
    rate = GAMMA * beta * (P / 2) / (1 + alpha ** 2)
    t = 1.5 / rate
    sim.run(t)
    mx, my, mz = sim.m[:, 0, 0, 0]
    th = 2 * np.arctan(np.tan(th0 / 2) * np.exp(-rate * t))
    assert abs(np.arccos(mz) - th) < 1e-6
    assert abs(np.arctan2(my, mx) + alpha * rate * t) < 1e-6
    # angle dependence of eps (Eq. 30) and the eps' term: torque components against the printed expression
    lam, epsp = 1.7, 0.3
    m = np.array([0.36, -0.48, 0.8]).reshape(3, 1, 1, 1)
    mp = np.array([0.0, 0.6, 0.8])
    tq = fld.slonczewski_torque_over_gamma(m, np.array([[[Ms]]]), np.array([[[alpha]]]), jz, P, lam, epsp, mp, d)[:, 0, 0, 0]
    mm_, c = m[:, 0, 0, 0], float(m[:, 0, 0, 0] @ mp)
    eps = P * lam ** 2 / ((lam ** 2 + 1) + (lam ** 2 - 1) * c)
    want = beta * ((eps - alpha * epsp) * np.cross(mm_, np.cross(mp, mm_)) - (epsp - alpha * eps) * np.cross(mm_, mp)) / (1 + alpha ** 2)
    assert np.allclose(tq, want, rtol=1e-13) and abs(tq @ mm_) < 1e-15
    # sign: reversing the current reverses the torque (switching in both directions, Fig. 9)
    assert np.allclose(fld.slonczewski_torque_over_gamma(m, np.array([[[Ms]]]), np.array([[[alpha]]]), -jz, P, lam, epsp, mp, d)[:, 0, 0, 0], -tq)


def test_zhang_li_torque_advects_a_spiral():
    # Eq. 26 (L327-L331, reading #19). With xi = alpha the torque is -(gamma u . grad) m: any texture is carried
    # along with velocity gamma u. For the spiral m = (cos kx, sin kx, 0) on a periodic chain the central
    # difference gives exactly m(x, t) = (cos(kx - w t), sin(kx - w t), 0), w = gamma u sin(k dx)/dx.
    n, dx, Ms, alpha, j = 32, 4e-9, 8e5, 0.1, 2e12
    sim = RefSim((n, 1, 1), (dx, dx, dx), pbc=(1, 0, 0))
    sim.set_params(Params.uniform(1, Msat=Ms, Aex=0.0, alpha=alpha))
    sim.set_terms(MM_ZEEMAN)                             # no field at all
    k = 2 * np.pi * 2 / (n * dx)
    x = np.arange(n) * dx
    m0 = np.zeros((3, 1, 1, n)); m0[0, 0, 0] = np.cos(k * x); m0[1, 0, 0] = np.sin(k * x)
    sim.set_m(m0)
    sim.set_zhang_li((j, 0, 0), xi=alpha)
    sim.set_solver(max_err=1e-8)
    u = fld.MU_BOHR * fld.MU0 / (2 * fld.E_CHARGE * GAMMA * fld.MU0 * Ms * (1 + alpha ** 2)) * j      # T m
    assert abs(GAMMA * u - fld.MU_BOHR * j / (2 * fld.E_CHARGE * Ms * (1 + alpha ** 2))) < 1e-9 * GAMMA * u   # a velocity, m/s
    w = GAMMA * u * np.sin(k * dx) / dx
    t = 1.0 / w
    sim.run(t)
    assert np.abs(sim.m[0, 0, 0] - np.cos(k * x - w * t)).max() < 1e-6
    assert np.abs(sim.m[1, 0, 0] - np.sin(k * x - w * t)).max() < 1e-6 and np.abs(sim.m[2]).max() < 1e-12
    # xi != alpha: the field-like term tilts the spiral out of the plane at the printed rate
    sim.set_m(m0); sim.set_zhang_li((j, 0, 0), xi=0.4)
    tq = sim.torque(sim.m) / GAMMA
    u4 = u * (1 + alpha ** 2) / (1 + 0.4 ** 2)
    assert np.allclose(tq[2, 0, 0], (0.4 - alpha) / (1 + alpha ** 2) * u4 * np.sin(k * dx) / dx, rtol=1e-12)
    # open boundary: the end cells see a one-sided half difference (own m stands in for the missing neighbour)
    sim2 = RefSim((n, 1, 1), (dx, dx, dx))
    sim2.set_params(Params.uniform(1, Msat=Ms, Aex=0.0, alpha=alpha)); sim2.set_terms(MM_ZEEMAN)
    sim2.set_m(m0); sim2.set_zhang_li((j, 0, 0), xi=alpha)
    t2 = sim2.torque(sim2.m) / GAMMA
    want0 = -u * (m0[:, 0, 0, 1] - m0[:, 0, 0, 0]) / (2 * dx)
    want0 = want0 - (want0 @ m0[:, 0, 0, 0]) * m0[:, 0, 0, 0]        # m x (m x D) = -(D - (m.D) m)
    assert np.allclose(t2[:, 0, 0, 0], want0, rtol=1e-10, atol=1e-18)


def test_zhang_li_next_to_vacuum_is_an_open_end():
    # A shape inside the box ends where Msat = 0 (L53): for the current-driven gradient (u . grad) m a vacuum
    # neighbour must count as a missing neighbour, exactly like the end of the box (L196). Pin: a chain whose right
    # half is vacuum carries, cell by cell, the torque of the chain that simply ends there; and a vacuum cell in the
    # middle of a uniform spiral does not act as a neighbour with m = 0 (which would give a gradient of m / 2 dx).
    n, dx, Ms, alpha, j = 12, 4e-9, 8e5, 0.1, 2e12
    k = 2 * np.pi / (20 * dx)
    x = np.arange(n) * dx
    m0 = np.zeros((3, 1, 1, n)); m0[0, 0, 0] = np.cos(k * x); m0[1, 0, 0] = np.sin(k * x)
    regions = np.zeros((1, 1, n), dtype=np.uint8); regions[..., n // 2:] = 1
    p2 = Params.uniform(2, Msat=[Ms, 0.0], Aex=0.0, alpha=alpha)
    full = RefSim((n, 1, 1), (dx, dx, dx)); full.set_params(p2); full.set_regions(regions); full.set_terms(MM_ZEEMAN)
    full.set_m(m0); full.set_zhang_li((j, 0, 0), xi=0.3)
    half = RefSim((n // 2, 1, 1), (dx, dx, dx)); half.set_params(Params.uniform(1, Msat=Ms, Aex=0.0, alpha=alpha))
    half.set_terms(MM_ZEEMAN); half.set_m(m0[..., :n // 2].copy()); half.set_zhang_li((j, 0, 0), xi=0.3)
    tf, th = full.torque(full.m), half.torque(half.m)
    assert np.abs(th).max() > 0 and np.array_equal(tf[..., :n // 2], th) and np.all(tf[..., n // 2:] == 0)
    # the wrong rule (vacuum neighbour read as m = 0) would make the interface torque about 1 / (k dx) times larger
    inner = np.abs(tf[:, 0, 0, 2]).max()
    assert np.abs(tf[:, 0, 0, n // 2 - 1]).max() < 1.01 * inner


# ------------------------------------------------------------------ pins added in round 2 ("What's weak" #1)
def test_energy_conserved_without_damping_on_a_3d_box_with_unequal_cell_edges():
    # alpha = 0: the torque is gamma m x B_eff with B_eff = -dE/dM, so E is a constant of the motion - but only
    # if the convolution kernel is the symmetric one, K_ij(-R) = K_ij(R) with K_xz, K_yz odd in z as well as
    # in x resp. y. A wrong z-mirror sign of an off-diagonal component breaks the symmetry
    # of the pair energy and the energy drifts (about 5e-4 relative here instead of 1e-8). Cell edges 4 x 3 x 2 nm
    # also make every axis of the exchange stencil use its own spacing.
    sim = RefSim((6, 5, 4), (4e-9, 3e-9, 2e-9))
    sim.set_params(Params.uniform(1, Msat=8e5, Aex=1.3e-11, alpha=0.0))
    sim.set_m(_rand_m(33, sim.shape))
    sim.set_solver(max_err=1e-7)
    e0 = sim.energy()
    sim.run(5e-12)
    assert abs(sim.energy() - e0) < 2e-7 * abs(e0)


def test_off_diagonal_kernel_signs_follow_the_point_dipole():
    # Far from the source cell N_ij -> -(V / 4 pi) (3 R_i R_j - R^2 d_ij) / R^5 (Fig. 4), so
    # K_xz = -N_xz has the sign of +x z, K_yz of +y z, K_xy of +x y in every octant of the displacement grid.
    grid, cell = (10, 9, 8), (4e-9, 3e-9, 2e-9)
    from oracle import demag_tensor as dt
    K, (oz, oy, ox) = dt.kernel_displacements(grid, cell, (0, 0, 0))
    V = cell[0] * cell[1] * cell[2]
    for (dx_, dy_, dz_) in ((7, 6, 7), (-7, 6, 7), (7, -6, 7), (7, 6, -7), (-7, -6, -7), (9, 0, -7), (-9, 0, 7), (0, 8, -7), (0, -8, -7)):
        R = np.array([dx_ * cell[0], dy_ * cell[1], dz_ * cell[2]])
        r = np.linalg.norm(R)
        dip = lambda i, j: (V / (4 * np.pi)) * (3 * R[i] * R[j]) / r ** 5       # K_ij = -N_ij, i != j
        for key, (i, j) in (("xy", (0, 1)), ("xz", (0, 2)), ("yz", (1, 2))):
            got = K[key][oz + dz_, oy + dy_, ox + dx_]
            want = dip(i, j)
            if want == 0:
                assert abs(got) < 1e-12
            else:
                assert np.isclose(got, want, rtol=0.05), (key, dx_, dy_, dz_, got, want)


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_exchange_spacing_of_every_axis(axis):
    # Eq. 6 (L187): the neighbour along axis i enters with 2 A / (Msat Delta_i^2); three different cell edges,
    # a 3-cell chain with a linear tilt along one axis at a time (Neumann ends, L196)
    A, Ms, cell = 1.3e-11, 8e5, (5e-9, 2e-9, 7e-9)
    grid = [1, 1, 1]; grid[axis] = 3
    sim = RefSim(tuple(grid), cell)
    sim.set_params(Params.uniform(1, Msat=Ms, Aex=A))
    m = np.zeros((3,) + sim.shape); m[0] = 1.0
    tilt = np.array([-0.01, 0.0, 0.01]).reshape([3 if a == 2 - axis else 1 for a in range(3)])
    m[1] = tilt
    B = fld.b_exchange(m, sim.regions, sim.L, sim.cell, sim.pbc)[1].ravel()
    d = cell[axis]
    assert np.isclose(B[0], 2 * A / Ms * 0.01 / d ** 2, rtol=1e-12)
    assert abs(B[1]) < 1e-12 and np.isclose(B[2], -B[0], rtol=1e-12)


def test_zeeman_energy_is_minus_M_dot_B_times_volume():
    # B_ext enters B_eff undivided (L108), so its energy density is -M . B_ext (no factor 1/2: the field does
    # not depend on m). (i) one cell, closed form; (ii) a macrospin with uniaxial anisotropy precessing in a
    # tilted field at alpha = 0 trades Zeeman against anisotropy energy: the sum is conserved only with the
    # right relative prefactor (Eq. 20: -Ku1 (u.m)^2 against -Msat m.B).
    Ms, c = 8e5, 3e-9
    sim = RefSim((1, 1, 1), (c, 2 * c, 3 * c))
    sim.set_params(Params.uniform(1, Msat=Ms, Aex=0.0, alpha=0.0, B_ext=(0.03, -0.02, 0.05)))
    m = np.array([0.36, 0.48, 0.8]).reshape(3, 1, 1, 1)
    sim.set_m(m)
    want = -Ms * (0.36 * 0.03 - 0.48 * 0.02 + 0.8 * 0.05) * (c * 2 * c * 3 * c)
    assert np.isclose(sim.energy(terms=MM_ZEEMAN), want, rtol=1e-13)
    sim = RefSim((1, 1, 1), (c, c, c))
    sim.set_params(Params.uniform(1, Msat=Ms, Aex=0.0, alpha=0.0, Ku1=4e4, anisU=(0, 0, 1), B_ext=(0.08, 0.0, 0.03)))
    sim.set_terms(MM_ANIS | MM_ZEEMAN)
    sim.set_m(np.array([0.0, 0.6, 0.8]).reshape(3, 1, 1, 1))
    sim.set_solver(max_err=1e-8)
    e0 = sim.energy(terms=MM_ANIS | MM_ZEEMAN)
    ez0 = sim.energy(terms=MM_ZEEMAN)
    swing = 0.0
    for _ in range(12):
        sim.run(0.02e-9)
        swing = max(swing, abs(sim.energy(terms=MM_ZEEMAN) - ez0))
        assert abs(sim.energy(terms=MM_ANIS | MM_ZEEMAN) - e0) < 1e-6 * abs(e0)
    assert swing > 0.5 * abs(e0)                         # energy really is traded between the two terms


# ------------------------------------------------------------------ Dzyaloshinskii-Moriya exchange (Eq. 10-17)
def _dmi_sim(grid, cell, pbc, D, A=16e-12, Ms=1100e3, Ku1=0.0, alpha=0.5):
    sim = RefSim(grid, cell, pbc)
    sim.set_params(Params.uniform(1, Msat=Ms, Aex=A, alpha=alpha, Ku1=Ku1, anisU=(0, 0, 1)))
    sim.set_dmi(D)
    sim.set_terms(MM_EXCH | MM_ANIS)                       # no demag: closed forms below
    return sim


def test_dmi_energy_density_eq16_equals_eq17_and_field_is_minus_dE_dM():
    # periodic box (no boundary terms): (i) -1/2 M . B_DM (Eq. 17) equals D [m_z div m - (m . grad) m_z] (Eq. 16)
    # cell by cell when both use the central differences of L246; (ii) the total exchange + DM field is
    # -dE/dM of the summed energy (finite differences on single cells)
    D, A, Ms = 1.3e-3, 16e-12, 1100e3
    cell = (2e-9, 3e-9, 1e-9)
    sim = _dmi_sim((8, 6, 1), cell, (1, 1, 0), D, A, Ms)
    m = _rand_m(71, sim.shape)
    sim.set_m(m)
    Bdm = sim.b_exch(sim.m) - fld.b_exchange(sim.m, sim.regions, sim.L, sim.cell, sim.pbc)
    dx = lambda f: (np.roll(f, -1, axis=2) - np.roll(f, 1, axis=2)) / (2 * cell[0])
    dy = lambda f: (np.roll(f, -1, axis=1) - np.roll(f, 1, axis=1)) / (2 * cell[1])
    mx, my, mz = sim.m
    eq16 = D * (mz * (dx(mx) + dy(my)) - (mx * dx(mz) + my * dy(mz)))
    eq17 = -0.5 * Ms * (sim.m * Bdm).sum(axis=0)
    assert np.allclose(eq16, eq17, rtol=1e-12, atol=1e-9 * np.abs(eq16).max())
    V = cell[0] * cell[1] * cell[2]
    B = sim.b_exch(sim.m)
    h = 1e-6
    for (c, iy, ix) in ((0, 2, 3), (1, 0, 7), (2, 5, 0)):
        mp = sim.m.copy(); mp[c, 0, iy, ix] += h
        mn = sim.m.copy(); mn[c, 0, iy, ix] -= h
        dE = (sim.energy(mp, MM_EXCH) - sim.energy(mn, MM_EXCH)) / (2 * h)
        assert np.isclose(B[c, 0, iy, ix], -dE / (Ms * V), rtol=1e-6)


def test_dmi_cycloid_energy_and_chirality():
    # Neel cycloid m = (s sin kx, 0, cos kx) on a periodic chain: Eq. 16 gives the energy density s D k' with
    # k' = sin(k dx)/dx the central-difference wave number; D > 0 favours s = -1 (m turns from +z towards -x)
    n, dx_, D, A, Ms = 64, 1e-9, 2e-3, 16e-12, 1100e3
    sim = _dmi_sim((n, 1, 1), (dx_, dx_, dx_), (1, 0, 0), D, A, Ms)
    k = 2 * np.pi * 3 / (n * dx_)
    x = np.arange(n) * dx_
    for s_ in (+1, -1):
        m = np.zeros((3, 1, 1, n)); m[0, 0, 0] = s_ * np.sin(k * x); m[2, 0, 0] = np.cos(k * x)
        sim.set_m(m)
        e_ex = (2 * A / dx_ ** 2) * (1 - np.cos(k * dx_))                       # Eq. 6 + 8 (spiral identity)
        want = (e_ex + s_ * D * np.sin(k * dx_) / dx_) * n * dx_ ** 3
        assert np.isclose(sim.energy(terms=MM_EXCH), want, rtol=1e-12)


def test_dmi_boundary_conditions_tilt_the_edge_magnetisation():
    # Eq. 11-13 with the exchange field under the same boundary conditions (L248): for m = (sin th, 0, cos th)
    # the energy density is A th'^2 + K sin^2 th + D th', so th'' = sin th cos th / xi^2 (xi^2 = A/K), first
    # integral th' = -sin th / xi, and the boundary condition th' = -D/2A fixes the edge tilt
    #     sin th_edge = D / (2 sqrt(A K)),   tan(th/2) = tan(th_edge/2) exp(-x/xi)  from the left edge,
    # with the opposite sign of m_x at the right edge. A chain of 0.25 nm cells, xi = 5.66 nm, relaxed.
    n, dx_, D, A, K, Ms = 240, 0.25e-9, 1e-3, 16e-12, 0.5e6, 1100e3
    sim = _dmi_sim((n, 1, 1), (dx_, 1e-9, 1e-9), (0, 0, 0), D, A, Ms, Ku1=K)
    m = np.zeros((3, 1, 1, n)); m[2] = 1.0
    sim.set_m(m)
    sim.relax()
    assert sim.max_torque() < 1e-5
    xi = np.sqrt(A / K)
    th_e = np.arcsin(D / (2 * np.sqrt(A * K)))
    x = (np.arange(n) + 0.5) * dx_                                             # cell centres from the left edge
    th = 2 * np.arctan(np.tan(th_e / 2) * np.exp(-x / xi))
    mx = sim.m[0, 0, 0]
    assert abs(np.sin(th_e) - 0.17678) < 1e-5
    assert np.abs(mx[:n // 2] - np.sin(th[:n // 2])).max() < 0.01 * np.sin(th_e)
    assert np.abs(mx[::-1][:n // 2] + np.sin(th[:n // 2])).max() < 0.01 * np.sin(th_e)
    assert np.abs(sim.m[1]).max() < 1e-9


def test_dmi_off_reduces_to_plain_exchange_and_vacuum_is_a_boundary():
    # D = 0: the boundary conditions vanish and Eq. 6 is recovered exactly; a vacuum neighbour (Msat = 0) is a
    # missing neighbour (geometry, L53): the cell next to it sees the same virtual neighbour as at the box edge
    rng = np.random.default_rng(3)
    sim = RefSim((7, 5, 2), (2e-9, 3e-9, 1e-9))
    p = Params.uniform(2, Msat=np.array([1100e3, 0.0]), Aex=16e-12, alpha=0.5)
    sim.set_params(p)
    reg = np.zeros(sim.shape, dtype=np.int64); reg[:, :, 5:] = 1              # columns x >= 5 are empty
    sim.set_regions(reg)
    sim.set_m(_rand_m(5, sim.shape))
    B0 = fld.b_exchange(sim.m, sim.regions, sim.L, sim.cell, sim.pbc)
    Bz = fld.b_exchange_dmi(sim.m, sim.regions, sim.L, sim.cell, sim.pbc, p.Msat, p.Aex, np.zeros(2))
    assert np.allclose(Bz, B0, rtol=0, atol=1e-12 * np.abs(B0).max())
    # the same film cut out of a 5-column box: identical field in the magnetic cells when D != 0
    sim.set_dmi(1.5e-3)
    small = RefSim((5, 5, 2), (2e-9, 3e-9, 1e-9))
    small.set_params(Params.uniform(1, Msat=1100e3, Aex=16e-12, alpha=0.5))
    small.set_m(sim.m[:, :, :, :5]); small.set_dmi(1.5e-3)
    assert np.allclose(sim.b_exch(sim.m)[:, :, :, :5], small.b_exch(small.m), rtol=1e-13)
    assert np.abs(sim.b_exch(sim.m)[:, :, :, 5:]).max() == 0.0
