"""RefSim: the oracle's call sequence (mirrors mm_create / mm_set_* / mm_b_eff / mm_step_rk45 /
mm_run of include/mm.h, but shares no code with it).  fp64, numpy.  Test infrastructure.

Time stepping: Dormand-Prince 5(4), 7 stages with FSAL ("RK45, the Dormand-Prince method",
PAPER.md L365), error eps = dt * max_cells ||tau_high - tau_low||_2 (L372), MaxErr 1e-5 and
headroom 0.8 (L372-L374); the controller details are the readings of SURVEY.md 8(c) #7-#10.
"""
import numpy as np
from . import demag_tensor as dt
from . import field as fld

MM_DEMAG, MM_EXCH, MM_ANIS, MM_ZEEMAN, MM_ALL = 1, 2, 4, 8, 15

# Dormand-Prince tableau (textbook); tests pin row sums, order and convergence
DP_C = (0.0, 1 / 5, 3 / 10, 4 / 5, 8 / 9, 1.0, 1.0)
DP_A = (
    (),
    (1 / 5,),
    (3 / 40, 9 / 40),
    (44 / 45, -56 / 15, 32 / 9),
    (19372 / 6561, -25360 / 2187, 64448 / 6561, -212 / 729),
    (9017 / 3168, -355 / 33, 46732 / 5247, 49 / 176, -5103 / 18656),
    (35 / 384, 0.0, 500 / 1113, 125 / 192, -2187 / 6784, 11 / 84),
)
DP_B5 = (35 / 384, 0.0, 500 / 1113, 125 / 192, -2187 / 6784, 11 / 84, 0.0)
DP_B4 = (5179 / 57600, 0.0, 7571 / 16695, 393 / 640, -92097 / 339200, 187 / 2100, 1 / 40)
DP_E = tuple(b5 - b4 for b5, b4 in zip(DP_B5, DP_B4))

# Bogacki-Shampine 3(2), 4 stages with FSAL ("RK32, the Bogacki-Shampine method, 3-th order convergence
# and a 2nd order error estimate"; the paper prints no tableau: textbook coefficients)
BS_A = ((), (1 / 2,), (0.0, 3 / 4), (2 / 9, 1 / 3, 4 / 9))
BS_B3 = (2 / 9, 1 / 3, 4 / 9, 0.0)
BS_B2 = (7 / 24, 1 / 4, 1 / 3, 1 / 8)
BS_E = tuple(b3 - b2 for b3, b2 in zip(BS_B3, BS_B2))

# Heun 2(1), 2 stages, no FSAL ("RK12, Heun's method, 2nd order convergence and a 1st order error estimate
# ... used for finite temperature simulations"): result m0 + h (k1 + k2) / 2
HEUN_A = ((), (1.0,))
HEUN_B2 = (1 / 2, 1 / 2)
HEUN_E = (1 / 2 - 1.0, 1 / 2)            # b(2nd) - b(1st, Euler)

# solver -> (a rows, error weights, exponent of the step-size rule = 1 / order of the solution,
#            weights of the result if the last stage input is not the result (no FSAL))
SOLVERS = {"rk45": (DP_A, DP_E, 1 / 5, None), "rk23": (BS_A, BS_E, 1 / 3, None),
           "rk12": (HEUN_A, HEUN_E, 1 / 2, HEUN_B2)}

K_BOLTZMANN = 1.380649e-23               # J/K

DIRECT_SUM_MAX_CELLS = 2048


def _normalise(v):
    n = np.sqrt((v * v).sum(axis=0, keepdims=True))
    return np.where(n > 0, v / np.where(n > 0, n, 1.0), 0.0)


class RefSim:
    def __init__(self, grid, cell, pbc=(0, 0, 0), demag_method=None):
        self.grid = tuple(int(g) for g in grid)
        self.cell = tuple(float(c) for c in cell)
        self.pbc = tuple(int(p) for p in pbc)
        nx, ny, nz = self.grid
        self.shape = (nz, ny, nx)
        self.ncells = nx * ny * nz
        self.regions = np.zeros(self.shape, dtype=np.int64)
        self.p = None
        self.m = None
        self.t = 0.0
        self.max_err, self.headroom, self.fix_dt = 1e-5, 0.8, 0.0
        self.dt, self.dt_min, self.dt_max = 1e-14, 1e-18, 1e-9
        self.k1 = None
        self.n_eval = self.n_steps = self.n_rejected = 0
        self.demag_method = demag_method or ("direct" if self.ncells <= DIRECT_SUM_MAX_CELLS else "fft")
        self._K = None
        self._Kp = None
        self.terms = MM_ALL
        self.solver = "rk45"
        self.precession = True
        self.temp, self.seed = 0.0, 0
        self.stt = None
        self.zl = None
        self.Dind = None

    def set_dmi(self, D):
        """Interfacial Dzyaloshinskii-Moriya strength D [J/m^2] (Eq. 10): a scalar or one value per
        region. Part of the exchange term (the paper's E_exch(DM), Eq. 16-17): MM_EXCH selects both."""
        D = np.atleast_1d(np.asarray(D, dtype=np.float64))
        self.Dind = None if not np.any(D) else (np.full(self.p.nregions, D[0]) if D.size == 1 else D.copy())
        self.k1 = None

    def b_exch(self, m):
        if self.Dind is None:
            return fld.b_exchange(m, self.regions, self.L, self.cell, self.pbc)
        return fld.b_exchange_dmi(m, self.regions, self.L, self.cell, self.pbc, self.p.Msat, self.p.Aex, self.Dind)

    def set_slonczewski(self, jz, pol, lam=1.0, eps_prime=0.0, mp=(0, 0, 1)):
        """Spin-transfer torque of Eq. 28-30 (L336-L347): current density j_z [A/m^2] through the layer
        thickness d = Nz dz, polarisation P, Slonczewski Lambda, secondary term eps', fixed layer m_P."""
        self.stt = None if jz == 0 else (float(jz), float(pol), float(lam), float(eps_prime), tuple(mp))
        self.k1 = None

    def set_zhang_li(self, j, xi):
        """Zhang-Li torque of Eq. 26 (L327-L331): current density vector j [A/m^2], non-adiabaticity xi."""
        self.zl = None if not np.any(np.asarray(j)) else (tuple(float(x) for x in j), float(xi))
        self.k1 = None

    def set_temperature(self, temp, seed=0):
        """Thermal field of Eq. 24 (L303-L310) at `temp` kelvin; eta comes from the counter-based
        generator synth.rng (seed, component stream, step * N + cell). Needs a fixed step and the
        Heun solver (L310)."""
        self.temp, self.seed = float(temp), int(seed)
        self.k1 = None

    def b_thermal(self, h):
        """Eq. 24: eta * sqrt(2 mu0 alpha kB T / (Bsat gamma dV dt)); one eta per cell, component, step."""
        from synth import rng
        n = self.ncells
        idx = np.uint64(self.n_steps + self.n_rejected) * np.uint64(n) + np.arange(n, dtype=np.uint64)
        eta = np.empty((3, n))
        for c in range(3):
            u1 = rng.uniform01(self.seed, c, idx)
            u2 = rng.uniform01(self.seed, 3 + c, idx)
            eta[c] = np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * np.pi * u2)       # Box-Muller
        Bsat = fld.MU0 * self.p.Msat[self.regions]
        alpha = self.p.alpha[self.regions]
        dV = self.cell[0] * self.cell[1] * self.cell[2]
        with np.errstate(divide="ignore", invalid="ignore"):
            amp = np.sqrt(2.0 * fld.MU0 * alpha * K_BOLTZMANN * self.temp / (Bsat * self.p.gamma_LL * dV * h))
        amp = np.where(Bsat > 0, amp, 0.0)
        return eta.reshape((3,) + self.shape) * amp[None]

    def set_solver_kind(self, name):
        """"rk45" (default), "rk23" (L366) or "rk12" (Heun, L367). Invalidates the FSAL slope."""
        assert name in SOLVERS
        self.solver = name
        self.k1 = None

    # ---- setup
    def set_terms(self, mask):
        """Which B_eff terms drive the dynamics (the paper's EnableDemag = false, L611)."""
        self.terms = int(mask)
        self.k1 = None

    def set_regions(self, regions):
        self.regions = np.asarray(regions).reshape(self.shape).astype(np.int64)
        self.k1 = None

    def set_params(self, p):
        self.p = p
        self.L = fld.exchange_table(p.Aex, p.Msat, p.exch_scale)
        self.k1 = None

    def set_solver(self, max_err=1e-5, headroom=0.8, fix_dt=0.0, dt_init=1e-14, dt_min=1e-18, dt_max=1e-9):
        self.max_err, self.headroom, self.fix_dt = max_err, headroom, fix_dt
        self.dt, self.dt_min, self.dt_max = (fix_dt if fix_dt > 0 else dt_init), dt_min, dt_max

    def set_m(self, m):
        self.m = _normalise(np.asarray(m, dtype=np.float64).reshape((3,) + self.shape))
        if self.p is not None:                      # vacuum cells (Msat = 0) carry no magnetisation (#12)
            self.m = self.m * (self.p.Msat[self.regions] > 0)[None]
        self.k1 = None

    def kernel(self):
        if self._K is None:
            self._K = dt.kernel_displacements(self.grid, self.cell, self.pbc)
        return self._K

    # ---- field (L108-L113)
    def b_demag(self, m):
        K, origin = self.kernel()
        M = (fld.MU0 * self.p.Msat)[self.regions][None] * m
        if self.demag_method == "direct":
            return fld.b_demag_direct(M, K, origin, self.pbc)
        if self._Kp is None:                      # kernel spectrum: computed once per box
            self._Kp = fld.kernel_spectrum(K, origin, fld.padded_shape(self.shape, self.pbc))
        return fld.b_demag_fft(M, K, origin, self.pbc, self._Kp)

    def b_eff(self, term_mask=MM_ALL, m=None):
        m = self.m if m is None else m
        B = np.zeros_like(m)
        if term_mask & MM_DEMAG:
            B += self.b_demag(m)
        if term_mask & MM_EXCH:
            B += self.b_exch(m)
        if term_mask & MM_ANIS:
            B += fld.b_anis_uniaxial(m, self.regions, self.p) + fld.b_anis_cubic(m, self.regions, self.p)
        if term_mask & MM_ZEEMAN:
            B += np.asarray(self.p.B_ext, dtype=np.float64)[:, None, None, None]
        return B

    def torque(self, m, b_extra=0.0):
        """dm/dt [1/s] (Eq. 1-2); b_extra: an additional field term (the thermal field of the step)."""
        self.n_eval += 1
        alpha = self.p.alpha[self.regions]
        tq = fld.ll_torque_over_gamma(m, self.b_eff(self.terms, m) + b_extra, alpha, self.precession)
        if self.stt is not None:
            jz, pol, lam, epsp, mp = self.stt
            tq = tq + fld.slonczewski_torque_over_gamma(m, self.p.Msat[self.regions], alpha, jz, pol, lam, epsp, mp,
                                                        self.grid[2] * self.cell[2])
        if self.zl is not None:
            tq = tq + fld.zhang_li_torque_over_gamma(m, self.p.Msat[self.regions], alpha, self.zl[0], self.zl[1], self.cell,
                                                     self.pbc, self.p.gamma_LL)
        return self.p.gamma_LL * tq

    # ---- energies (Eq. 4, 8, 20, 23; Zeeman -M.B_ext), joules
    def energy(self, m=None, terms=MM_ALL):
        m = self.m if m is None else m
        Ms = self.p.Msat[self.regions][None]
        M = Ms * m
        e = 0.0
        if terms & MM_DEMAG:
            e += -0.5 * (M * self.b_demag(m)).sum()                                            # Eq. 4
        if terms & MM_EXCH:
            e += -0.5 * (M * self.b_exch(m)).sum()                                             # Eq. 8 (+ Eq. 17)
        if terms & MM_ANIS:
            e += -0.5 * (M * fld.b_anis_uniaxial(m, self.regions, self.p, only=1)).sum()       # Eq. 20
            e += -0.25 * (M * fld.b_anis_uniaxial(m, self.regions, self.p, only=2)).sum()
            e += -(1 / 4) * (M * fld.b_anis_cubic(m, self.regions, self.p, only=1)).sum()      # Eq. 23
            e += -(1 / 6) * (M * fld.b_anis_cubic(m, self.regions, self.p, only=2)).sum()
            e += -(1 / 8) * (M * fld.b_anis_cubic(m, self.regions, self.p, only=3)).sum()
        if terms & MM_ZEEMAN:
            e += -(M * np.asarray(self.p.B_ext)[:, None, None, None]).sum()
        return e * self.cell[0] * self.cell[1] * self.cell[2]

    # ---- one attempted Runge-Kutta step of the selected embedded pair
    def step(self, dt_force=None):
        A, E, expo, B = SOLVERS[self.solver]
        ns = len(A)
        h = self.dt if dt_force is None else dt_force
        bth = 0.0
        if self.temp > 0:
            assert self.fix_dt > 0 and self.solver == "rk12", "thermal field: fixed step and Heun only (L310)"
            bth = self.b_thermal(h)                    # constant during the step, new after it (L308)
            self.k1 = None                             # no torque continuity between steps
        if self.k1 is None:
            self.k1 = self.torque(self.m, bth)
        m0 = self.m
        k = [self.k1]
        y = None
        for i in range(1, ns):
            y = _normalise(m0 + h * sum(a * kj for a, kj in zip(A[i], k)))       # every stage input
            k.append(self.torque(y, bth))                                         # is renormalised (#9)
        err_vec = sum(e * kj for e, kj in zip(E, k))
        err = h * np.sqrt((err_vec * err_vec).sum(axis=0)).max()
        fixed = self.fix_dt > 0
        accepted = fixed or (err <= self.max_err)
        if accepted:
            if B is None:
                self.m, self.k1 = y, k[ns - 1]   # last stage input = the high-order result; FSAL
            else:
                self.m, self.k1 = _normalise(m0 + h * sum(b * kj for b, kj in zip(B, k))), None
            self.t += h
            self.n_steps += 1
        else:
            self.n_rejected += 1
        if not fixed:
            fac = 2.0 if err == 0 else min(2.0, max(0.5, (self.max_err / err) ** expo))
            self.dt = min(self.dt_max, max(self.dt_min, h * self.headroom * fac))
        return dict(t=self.t, dt_taken=h, dt_next=self.dt, err=err, accepted=accepted)

    def run(self, duration):
        """Advance t by exactly `duration` (last step clipped; controller's dt restored, #10)."""
        t_end = self.t + duration
        while t_end - self.t > 1e-12 * max(duration, 1e-30):
            remaining = t_end - self.t
            if self.dt >= remaining:
                keep = self.dt
                info = self.step(dt_force=remaining)
                if info["accepted"]:
                    self.dt = keep
                    self.t = t_end
            else:
                self.step()

    def max_torque(self):
        """max over cells of |tau| / gamma_LL [T] (what relax() monitors near equilibrium)."""
        tq = self.torque(self.m) / self.p.gamma_LL
        return float(np.sqrt((tq * tq).sum(axis=0)).max())

    def relax(self, max_batches=20000):
        """relax() as the paper describes it (L388-L392): precession term off, RK23, adaptive step.
        Advance while the total energy keeps falling; then monitor the maximum torque instead and
        advance while it keeps falling; each time it stops falling decrease MaxErr, until MaxErr = 1e-9.
        Readings (the paper gives no numbers; #15): quantities are sampled every 3 steps,
        MaxErr is divided by sqrt(2) each time. Solver settings are restored afterwards."""
        saved = (self.solver, self.precession, self.max_err, self.fix_dt)
        self.set_solver_kind("rk23")
        self.precession, self.fix_dt = False, 0.0
        n = 3

        def advance():
            for _ in range(n):
                self.step()

        batches = 0
        advance(); e0 = self.energy(terms=self.terms)
        advance(); e1 = self.energy(terms=self.terms)
        while e1 < e0 and batches < max_batches:
            advance(); e0, e1 = e1, self.energy(terms=self.terms); batches += 1
        t0 = self.max_torque()
        while batches < max_batches:
            advance(); t1 = self.max_torque(); batches += 1
            if t1 < t0:
                t0 = t1
                continue
            if self.max_err <= 1e-9:
                break
            self.max_err = max(self.max_err / np.sqrt(2.0), 1e-9)
            t0 = t1
        self.solver, self.precession, self.max_err, self.fix_dt = saved
        self.k1 = None
        return batches

    def avg_m(self):
        return self.m.reshape(3, -1).mean(axis=1)
