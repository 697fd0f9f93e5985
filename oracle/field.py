"""Effective-field terms, torque and energies, fp64, written out from the paper's definitions.
Test infrastructure.  Arrays are [component][z][y][x]; `Lnnn` = PAPER.md line.
"""
import os

import numpy as np
from scipy import fft as _fft          # same pocketfft routine as numpy.fft, with a `workers` argument

MU0 = 4e-7 * np.pi
FFT_WORKERS = int(os.environ.get("ORACLE_FFT_WORKERS", "0")) or (os.cpu_count() or 1)   # threads of the library FFT
COMPS = (("xx", "xy", "xz"), ("xy", "yy", "yz"), ("xz", "yz", "zz"))


# ---------------------------------------------------------------- demag (Eq. 3)
def b_demag_direct(M, K, origin, pbc):
    """B_i(r) = sum_r' sum_j K_ij(r - r') M_j(r'), the double sum written out (O(N^2)).

    M = mu0 Msat m in tesla, [3][z][y][x]. K, origin from demag_tensor.kernel_displacements.
    """
    _, nz, ny, nx = M.shape
    oz, oy, ox = origin
    B = np.zeros_like(M)
    zs = np.arange(nz)[:, None, None]; ys = np.arange(ny)[None, :, None]; xs = np.arange(nx)[None, None, :]
    for z in range(nz):
        iz = np.mod(z - zs, nz) if pbc[2] else (z - zs + oz)
        for y in range(ny):
            iy = np.mod(y - ys, ny) if pbc[1] else (y - ys + oy)
            for x in range(nx):
                ix = np.mod(x - xs, nx) if pbc[0] else (x - xs + ox)
                for i in range(3):
                    acc = 0.0
                    for j in range(3):
                        acc += (K[COMPS[i][j]][iz, iy, ix] * M[j]).sum()
                    B[i, z, y, x] = acc
    return B


def padded_shape(shape, pbc):
    """FFT lengths (z, y, x): open axes zero-padded to 2N (any length >= 2N-1 gives the identical
    linear convolution); periodic axes not padded (L509); 1 stays 1."""
    n = tuple(shape)
    return tuple(n[a] if pbc[2 - a] else (2 * n[a] if n[a] > 1 else 1) for a in range(3))


def kernel_spectrum(K, origin, P):
    """rfftn of every kernel component laid out on the padded, wrapped displacement grid."""
    Kp = {}
    for k, arr in K.items():
        buf = np.zeros(P)
        idx = []
        for a in range(3):
            d = np.arange(arr.shape[a]) - origin[a]          # displacement of every stored entry
            idx.append(np.mod(d, P[a]))
        buf[np.ix_(*idx)] = arr
        Kp[k] = _fft.rfftn(buf, workers=FFT_WORKERS)
    return Kp


def b_demag_fft(M, K, origin, pbc, Kp=None):
    """The same sum through the convolution theorem (L123) with the library's fp64 FFT (scipy.fft = pocketfft,
    threaded over the host cores; a library primitive, no blocking or reordering of the method here).
    `Kp` may carry the kernel spectrum computed once by kernel_spectrum()."""
    _, nz, ny, nx = M.shape
    P = padded_shape((nz, ny, nx), pbc)
    if Kp is None:
        Kp = kernel_spectrum(K, origin, P)
    Mf = [_fft.rfftn(M[j], s=P, axes=(0, 1, 2), workers=FFT_WORKERS) for j in range(3)]
    B = np.empty_like(M)
    for i in range(3):
        acc = sum(Kp[COMPS[i][j]] * Mf[j] for j in range(3))
        B[i] = _fft.irfftn(acc, s=P, axes=(0, 1, 2), workers=FFT_WORKERS)[:nz, :ny, :nx]
    return B


# ---------------------------------------------------------------- exchange (Eq. 6, 9)
def exchange_table(Aex, Msat, scale):
    """L[a, b] = S_ab * 2 (A_a/M_a)(A_b/M_b) / (A_a/M_a + A_b/M_b)  (Eq. 9), in T m^2.

    `scale` is None (S = 1) or lower-triangular S[i(i+1)/2 + j], i >= j.  Msat = 0 -> A/M := 0.
    """
    n = len(Msat)
    q = np.where(Msat > 0, Aex / np.where(Msat > 0, Msat, 1.0), 0.0)
    L = np.zeros((n, n))
    for a in range(n):
        for b in range(n):
            s = q[a] + q[b]
            h = 2.0 * q[a] * q[b] / s if s > 0 else 0.0
            i, j = max(a, b), min(a, b)
            S = 1.0 if scale is None else scale[i * (i + 1) // 2 + j]
            L[a, b] = S * h
    return L


def b_exchange(m, regions, L, cell, pbc):
    """B_exch = sum over the 6 nearest neighbours of (2 / D_i^2) L[r, r_i] (m_i - m)  (Eq. 6).

    A missing neighbour at an open boundary contributes 0 (own value used, L196);
    periodic axes wrap (L173).
    """
    B = np.zeros_like(m)
    for axis, d in ((3, cell[0]), (2, cell[1]), (1, cell[2])):       # array axes x, y, z
        n = m.shape[axis]
        periodic = pbc[3 - axis] > 0
        if n == 1 and not periodic:
            continue
        for shift in (+1, -1):
            mi = np.roll(m, -shift, axis=axis)                        # neighbour at +shift
            ri = np.roll(regions, -shift, axis=axis - 1)
            w = (2.0 / (d * d)) * L[regions, ri]
            if not periodic:                                          # cut the wrap-around link
                sl = [slice(None)] * 3
                sl[axis - 1] = (n - 1) if shift == +1 else 0
                w[tuple(sl)] = 0.0
            B += w[None] * (mi - m)
    return B


# ---------------------------------------------------------------- Dzyaloshinskii-Moriya exchange (Eq. 10-17)
def _neighbour_with_bc(m, live, axis, shift, d, periodic, bc):
    """m of the neighbour cell at +shift along array axis `axis` (1 = z, 2 = y, 3 = x of [c][z][y][x]).

    Where the neighbour is missing - outside an open box, or a cell without magnetisation (Msat = 0: geometry,
    L53) - "its magnetization is replaced by m + dm/di|_dV Delta_i n" (L246) with the boundary derivatives of
    Eq. 11-15 (bc = D / 2A of the central cell):
        x boundary:  d(m_x, m_y, m_z)/dx = (-bc m_z, 0, bc m_x)      (Eq. 11, 13, 14)
        y boundary:  d(m_x, m_y, m_z)/dy = (0, -bc m_z, bc m_y)      (Eq. 12, 13, 14)
        z boundary:  0                                                (Eq. 15)
    and n = shift the outward direction.  Returns (neighbour m, mask of cells whose neighbour is real)."""
    n = m.shape[axis]
    mi = np.roll(m, -shift, axis=axis)
    real = np.roll(live, -shift, axis=axis - 1).copy()
    if not periodic:
        sl = [slice(None)] * 3
        sl[axis - 1] = (n - 1) if shift == +1 else 0
        real[tuple(sl)] = False
    if axis == 3:
        dm = np.stack([-bc * m[2], np.zeros_like(bc), bc * m[0]])
    elif axis == 2:
        dm = np.stack([np.zeros_like(bc), -bc * m[2], bc * m[1]])
    else:
        dm = np.zeros_like(m)
    virtual = m + shift * d * dm
    return np.where(real[None], mi, virtual), real


def b_exchange_dmi(m, regions, L, cell, pbc, Msat, Aex, Dind):
    """Heisenberg exchange (Eq. 6) plus the interfacial Dzyaloshinskii-Moriya field of Eq. 10,
        B_DM = (2D / Msat) ( dm_z/dx, dm_z/dy, -dm_x/dx - dm_y/dy ),
    with central differences (m_{i+1} - m_{i-1}) / (2 Delta_i) (L246) and the boundary conditions of Eq. 11-15,
    which "in case of nonzero D ... are simultaneously applied to the Heisenberg exchange field" (L248).
    Msat, Aex, Dind: per-region tables; D and D/2A are those of the central cell's region (#20)."""
    Ms = Msat[regions]
    live = Ms > 0
    with np.errstate(divide="ignore", invalid="ignore"):
        bc = np.where(live & (Aex[regions] > 0), Dind[regions] / (2.0 * Aex[regions]), 0.0)
        cD = np.where(live, 2.0 * Dind[regions] / Ms, 0.0)
    B = np.zeros_like(m)
    for axis, d in ((3, cell[0]), (2, cell[1]), (1, cell[2])):
        n = m.shape[axis]
        periodic = pbc[3 - axis] > 0
        if n == 1 and not periodic:
            continue
        nb = {}
        for shift in (+1, -1):
            mi, real = _neighbour_with_bc(m, live, axis, shift, d, periodic, bc)
            ri = np.where(real, np.roll(regions, -shift, axis=axis - 1), regions)     # virtual neighbour: own material
            B += ((2.0 / (d * d)) * L[regions, ri])[None] * (mi - m)                    # Eq. 6 / Eq. 9
            nb[shift] = mi
        diff = (nb[+1] - nb[-1]) / (2.0 * d)                                            # central difference (L246)
        if axis == 3:      # d/dx
            B[0] += cD * diff[2]
            B[2] -= cD * diff[0]
        elif axis == 2:    # d/dy
            B[1] += cD * diff[2]
            B[2] -= cD * diff[1]
    return B * live[None]


# ---------------------------------------------------------------- anisotropy (Eq. 18, 21)
def _unit(v):
    nrm = np.sqrt((v * v).sum(axis=-1, keepdims=True))
    return np.where(nrm > 0, v / np.where(nrm > 0, nrm, 1.0), 0.0)


def _inv_msat(Msat):
    return np.where(Msat > 0, 1.0 / np.where(Msat > 0, Msat, 1.0), 0.0)


def b_anis_uniaxial(m, regions, p, only=None):
    """Eq. 18 (L269) with B_sat read as Msat [A/m]."""
    u = _unit(p.anisU)[regions]                                       # [z][y][x][3]
    um = sum(u[..., c] * m[c] for c in range(3))
    im = _inv_msat(p.Msat)[regions]
    k1 = p.Ku1[regions] if only in (None, 1) else 0.0
    k2 = p.Ku2[regions] if only in (None, 2) else 0.0
    mag = 2.0 * k1 * im * um + 4.0 * k2 * im * um ** 3
    return np.stack([mag * u[..., c] for c in range(3)])


def b_anis_cubic(m, regions, p, only=None):
    """Eq. 21 (L284-L286), c3 = c1 x c2."""
    c1 = _unit(p.anisC1); c2 = _unit(p.anisC2); c3 = np.cross(c1, c2)
    c = [c1[regions], c2[regions], c3[regions]]
    a = [sum(ci[..., k] * m[k] for k in range(3)) for ci in c]
    im = _inv_msat(p.Msat)[regions]
    K1 = p.Kc1[regions] if only in (None, 1) else 0.0
    K2 = p.Kc2[regions] if only in (None, 2) else 0.0
    K3 = p.Kc3[regions] if only in (None, 3) else 0.0
    B = np.zeros_like(m)
    for i in range(3):
        j, k = (i + 1) % 3, (i + 2) % 3
        coef = (-2.0 * K1 * im * (a[j] ** 2 + a[k] ** 2) * a[i]
                - 2.0 * K2 * im * (a[j] ** 2 * a[k] ** 2) * a[i]
                - 4.0 * K3 * im * (a[j] ** 4 + a[k] ** 4) * a[i] ** 3)
        for comp in range(3):
            B[comp] += coef * c[i][..., comp]
    return B


# ---------------------------------------------------------------- torque (Eq. 2)
def cross(a, b):
    return np.stack([a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0]])


def ll_torque_over_gamma(m, B, alpha_cell, precession=True):
    """tau / gamma_LL = -1/(1+alpha^2) [ m x B + alpha m x (m x B) ]  (Eq. 2 with the sign of
    SURVEY.md 8(c) #5: damping must move m towards B).  precession=False drops the m x B term
    ("disables the precession term", relax())."""
    mxB = cross(m, B)
    damp = alpha_cell[None] * cross(m, mxB)
    return -((mxB if precession else 0.0) + damp) / (1.0 + alpha_cell[None] ** 2)


HBAR = 1.054571817e-34       # J s
E_CHARGE = 1.602176634e-19   # C


def slonczewski_torque_over_gamma(m, Msat_cell, alpha_cell, jz, pol, lam, eps_prime, mp, thickness):
    """Eq. 28-30 (L336-L347), divided by gamma_LL [T]:
       tau_SL = beta (eps - alpha eps')/(1+alpha^2) m x (m_P x m) - beta (eps' - alpha eps)/(1+alpha^2) m x m_P,
       beta = j_z hbar / (Msat e d),  eps = P Lambda^2 / ((Lambda^2 + 1) + (Lambda^2 - 1) m.m_P).
    As printed beta is a field (tesla) while Eq. 1 wants 1/s: the torque is gamma_LL times this (#18)."""
    mp = np.asarray(mp, dtype=float)
    mp = mp / np.linalg.norm(mp)
    mpv = mp[:, None, None, None] * np.ones_like(m)
    with np.errstate(divide="ignore", invalid="ignore"):
        beta = np.where(Msat_cell > 0, jz * HBAR / (Msat_cell * E_CHARGE * thickness), 0.0)[None]
    l2 = lam * lam
    eps = pol * l2 / ((l2 + 1.0) + (l2 - 1.0) * (m * mpv).sum(axis=0, keepdims=True))
    a = alpha_cell[None]
    den = 1.0 + a * a
    return beta * ((eps - a * eps_prime) / den * cross(m, cross(mpv, m)) - (eps_prime - a * eps) / den * cross(m, mpv))


MU_BOHR = 9.2740100783e-24   # J/T


def zhang_li_torque_over_gamma(m, Msat_cell, alpha_cell, j, xi, cell, pbc, gamma):
    """Zhang-Li spin-transfer torque, Eq. 26 (L327-L331), divided by gamma_LL [T]:
       tau_ZL = 1/(1+alpha^2) [ (1 + xi alpha) m x (m x (u.grad) m) + (xi - alpha) m x (u.grad) m ],
       u = mu_B mu0 / (2 e gamma_LL Bsat (1 + xi^2)) j      [T m].
    PAPER.md prints the two terms identically (garbled); the double cross product in the first term is the
    reading of DESIGN.md #19. (u.grad) m by central differences; a missing neighbour - beyond an open boundary, or
    a vacuum cell (Msat = 0), which is how a shape inside the box ends (L53) - is replaced by the cell's own m
    (as for the exchange stencil, L196); periodic axes wrap."""
    j = np.asarray(j, dtype=float)
    D = np.zeros_like(m)
    with np.errstate(divide="ignore", invalid="ignore"):
        pref = np.where(Msat_cell > 0, MU_BOHR * MU0 / (2.0 * E_CHARGE * gamma * (MU0 * Msat_cell) * (1.0 + xi * xi)), 0.0)
    for axis_m, (ja, d, per) in enumerate(zip(j[::-1], cell[::-1], pbc[::-1])):      # array axes are z, y, x
        if ja == 0 or m.shape[1 + axis_m] == 1:
            continue
        ax = 1 + axis_m
        if per:
            up, dn = np.roll(m, -1, axis=ax), np.roll(m, 1, axis=ax)
        else:
            up, dn = m.copy(), m.copy()
            sl_hi = [slice(None)] * 4; sl_lo = [slice(None)] * 4
            sl_hi[ax] = slice(1, None); sl_lo[ax] = slice(None, -1)
            up[tuple(sl_lo)] = m[tuple(sl_hi)]        # neighbour at +1 (the last cell keeps its own m)
            dn[tuple(sl_hi)] = m[tuple(sl_lo)]        # neighbour at -1 (the first cell keeps its own m)
        # the same shifts of Msat tell which neighbours are vacuum
        if per:
            ms_up, ms_dn = np.roll(Msat_cell, -1, axis=ax - 1), np.roll(Msat_cell, 1, axis=ax - 1)
        else:
            ms_up, ms_dn = Msat_cell.copy(), Msat_cell.copy()
            ms_up[tuple(sl_lo[1:])] = Msat_cell[tuple(sl_hi[1:])]
            ms_dn[tuple(sl_hi[1:])] = Msat_cell[tuple(sl_lo[1:])]
        up = np.where(ms_up[None] > 0, up, m)
        dn = np.where(ms_dn[None] > 0, dn, m)
        D += (pref * ja)[None] * (up - dn) / (2.0 * d)
    a = alpha_cell[None]
    mxD = cross(m, D)
    return ((1.0 + xi * a) * cross(m, mxD) + (xi - a) * mxD) / (1.0 + a * a)
