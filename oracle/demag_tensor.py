"""Demagnetising tensor between two identical, uniformly magnetised cuboid cells, averaged
over the destination cell ("constant magnetization in each finite difference
cell ... average the resulting B_demag over the cell volumes"), fp64.  Test infrastructure.

N_ij(R) is defined by  <H_i>_dest = - N_ij(R) M_j  for a source cell at the origin and a
destination cell displaced by R;  K_ij = -N_ij  (paper's tables list N = H/M, L127).

Two evaluations of the same definition:
  * near (|R| < R_SWITCH largest cell edges): the closed form of the six-fold integral
    (27-point second difference of the auxiliary functions f and g);
  * far: the point-dipole tensor T_ij(r) = (3 r_i r_j - r^2 d_ij) / (4 pi r^5) integrated over
    source and destination cell by a tensor-product Gauss-Legendre rule.  The closed form
    cancels catastrophically at long range in fp64, the quadrature is
    exact to rounding there.  tests/test_oracle_demag.py checks that the two agree in the
    overlap band.
"""
import numpy as np

R_SWITCH = 12.0      # in units of the largest cell edge
R_FAR2 = 48.0        # beyond this a 2-point rule per axis is exact to ~1e-7 * (48)^-4


def _term(pref, fn, a, b):
    """pref * fn(a / b); a term whose prefactor is zero, or whose argument is 0/0, is dropped
    (its limit is 0, SURVEY.md Appendix A evaluation rules)."""
    out = np.zeros_like(pref)
    ok = (pref != 0) & (a != 0)
    out[ok] = pref[ok] * fn(a[ok] / b[ok])
    return out


def newell_f(x, y, z):
    """Auxiliary function f; even in x, y, z."""
    x, y, z = np.broadcast_arrays(np.abs(x), np.abs(y), np.abs(z))
    x2 = x * x; y2 = y * y; z2 = z * z
    R = np.sqrt(x2 + y2 + z2)
    f = _term(0.5 * y * (z2 - x2), np.arcsinh, y, np.sqrt(x2 + z2))
    f += _term(0.5 * z * (y2 - x2), np.arcsinh, z, np.sqrt(x2 + y2))
    f -= _term(x * y * z, np.arctan, y * z, x * R)
    f += (1.0 / 6.0) * (2.0 * x2 - y2 - z2) * R
    return f


def newell_g(x, y, z):
    """Auxiliary function g; odd in x, odd in y, even in z."""
    sgn = np.sign(x) * np.sign(y)
    x, y, z = np.broadcast_arrays(np.abs(x), np.abs(y), np.abs(z))
    x2 = x * x; y2 = y * y; z2 = z * z
    R = np.sqrt(x2 + y2 + z2)
    g = _term(x * y * z, np.arcsinh, z, np.sqrt(x2 + y2))
    g += _term((y / 6.0) * (3.0 * z2 - y2), np.arcsinh, x, np.sqrt(y2 + z2))
    g += _term((x / 6.0) * (3.0 * z2 - x2), np.arcsinh, y, np.sqrt(x2 + z2))
    g -= _term(z * z2 / 6.0, np.arctan, x * y, z * R)
    g -= _term(z * y2 / 2.0, np.arctan, x * z, y * R)
    g -= _term(z * x2 / 2.0, np.arctan, y * z, x * R)
    g -= x * y * R / 3.0
    return sgn * g


def _second_difference(F, X, Y, Z, dx, dy, dz):
    """D[F] = sum_{a,b,c in {-1,0,1}} w_a w_b w_c F(X + a dx, Y + b dy, Z + c dz), w = (-1, 2, -1)."""
    w = (-1.0, 2.0, -1.0)
    acc = np.zeros(np.broadcast(X, Y, Z).shape)
    for a in (-1, 0, 1):
        for b in (-1, 0, 1):
            for c in (-1, 0, 1):
                acc = acc + (w[a + 1] * w[b + 1] * w[c + 1]) * F(X + a * dx, Y + b * dy, Z + c * dz)
    return acc


def tensor_analytic(X, Y, Z, cell):
    """Closed form. Returns dict with keys xx, yy, zz, xy, xz, yz (arrays like X)."""
    dx, dy, dz = cell
    X, Y, Z = np.broadcast_arrays(np.asarray(X, float), np.asarray(Y, float), np.asarray(Z, float))
    c = 1.0 / (4.0 * np.pi * dx * dy * dz)
    return dict(
        xx=c * _second_difference(newell_f, X, Y, Z, dx, dy, dz),
        yy=c * _second_difference(newell_f, Y, X, Z, dy, dx, dz),
        zz=c * _second_difference(newell_f, Z, Y, X, dz, dy, dx),
        xy=c * _second_difference(newell_g, X, Y, Z, dx, dy, dz),
        xz=c * _second_difference(newell_g, X, Z, Y, dx, dz, dy),
        yz=c * _second_difference(newell_g, Y, Z, X, dy, dz, dx),
    )


def _difference_rule(d, npts):
    """Nodes/weights of s = u - u' for u, u' on an npts Gauss-Legendre rule over [-d/2, d/2].

    Equal to the tensor-product rule over (u, u'); duplicates of s are merged.
    """
    xi, wi = np.polynomial.legendre.leggauss(npts)
    u = 0.5 * d * xi
    w = 0.5 * d * wi
    s = (u[:, None] - u[None, :]).ravel()
    ws = (w[:, None] * w[None, :]).ravel()
    key = np.round(s / d * 1e12).astype(np.int64)
    uniq, inv = np.unique(key, return_inverse=True)
    s_out = np.zeros(len(uniq)); w_out = np.zeros(len(uniq))
    np.add.at(w_out, inv, ws)
    s_out[inv] = s
    return s_out, w_out


def tensor_quadrature(X, Y, Z, cell, npts=3):
    """N_ij = -(1/V) int_cell int_cell' T_ij(R + u - u') d3u' d3u by Gauss-Legendre."""
    dx, dy, dz = cell
    X, Y, Z = np.broadcast_arrays(np.asarray(X, float), np.asarray(Y, float), np.asarray(Z, float))
    sx, wx = _difference_rule(dx, npts)
    sy, wy = _difference_rule(dy, npts)
    sz, wz = _difference_rule(dz, npts)
    out = {k: np.zeros(X.shape) for k in ("xx", "yy", "zz", "xy", "xz", "yz")}
    for a, wa in zip(sx, wx):
        for b, wb in zip(sy, wy):
            for c, wc in zip(sz, wz):
                x = X + a; y = Y + b; z = Z + c
                r2 = x * x + y * y + z * z
                w = (wa * wb * wc) / (4.0 * np.pi * r2 * r2 * np.sqrt(r2))
                out["xx"] += w * (3.0 * x * x - r2)
                out["yy"] += w * (3.0 * y * y - r2)
                out["zz"] += w * (3.0 * z * z - r2)
                out["xy"] += w * (3.0 * x * y)
                out["xz"] += w * (3.0 * x * z)
                out["yz"] += w * (3.0 * y * z)
    V = dx * dy * dz
    for k in out:
        out[k] *= -1.0 / V
    return out


def tensor(X, Y, Z, cell):
    """N_ij at displacements (X, Y, Z) [metres]: closed form near, quadrature far."""
    X, Y, Z = np.broadcast_arrays(np.asarray(X, float), np.asarray(Y, float), np.asarray(Z, float))
    dmax = max(cell)
    rr = np.sqrt(X * X + Y * Y + Z * Z) / dmax
    out = {k: np.zeros(X.shape) for k in ("xx", "yy", "zz", "xy", "xz", "yz")}
    zones = ((rr < R_SWITCH, None), ((rr >= R_SWITCH) & (rr < R_FAR2), 3), (rr >= R_FAR2, 2))
    for mask, npts in zones:
        if not mask.any():
            continue
        if npts is None:
            part = tensor_analytic(X[mask], Y[mask], Z[mask], cell)
        else:
            part = tensor_quadrature(X[mask], Y[mask], Z[mask], cell, npts)
        for k in out:
            out[k][mask] = part[k]
    return out


def kernel_displacements(grid, cell, pbc):
    """K_ij = -N_ij on the displacement grid of a simulation box (Eq. 3).

    Open axis: displacements -(N-1)..(N-1), array length 2N-1, index d + N - 1.
    Periodic axis with `P` repeats (SetPBC, L175-L177; reading SURVEY.md 8(c) #2): every
    displacement D with |D| <= N*P - 1 is summed into D mod N, array length N, index D mod N.
    Returns (K, origin) with K[comp] of shape (Lz, Ly, Lx) and origin = index of D = 0 per
    axis (z, y, x).
    """
    N = (grid[0], grid[1], grid[2])
    axes = []
    for a in range(3):
        if pbc[a] > 0:
            D = np.arange(-(N[a] * pbc[a] - 1), N[a] * pbc[a])
            axes.append((D, np.mod(D, N[a]), N[a], 0))
        else:
            D = np.arange(-(N[a] - 1), N[a])
            axes.append((D, D + N[a] - 1, 2 * N[a] - 1, N[a] - 1))
    (Dx, ix, Lx, ox), (Dy, iy, Ly, oy), (Dz, iz, Lz, oz) = axes
    # evaluate on the non-negative octant only and mirror with the parity of each component
    ax = np.arange(0, np.abs(Dx).max() + 1); ay = np.arange(0, np.abs(Dy).max() + 1)
    az = np.arange(0, np.abs(Dz).max() + 1)
    T = tensor(ax[None, None, :] * cell[0], ay[None, :, None] * cell[1], az[:, None, None] * cell[2], cell)
    parity = dict(xx=(0, 0, 0), yy=(0, 0, 0), zz=(0, 0, 0), xy=(1, 1, 0), xz=(1, 0, 1), yz=(0, 1, 1))
    K = {}
    for k, (px, py, pz) in parity.items():
        full = T[k][np.abs(Dz)[:, None, None], np.abs(Dy)[None, :, None], np.abs(Dx)[None, None, :]]
        sg = (np.where(Dx < 0, -1.0, 1.0) if px else np.ones(len(Dx)))[None, None, :] \
            * (np.where(Dy < 0, -1.0, 1.0) if py else np.ones(len(Dy)))[None, :, None] \
            * (np.where(Dz < 0, -1.0, 1.0) if pz else np.ones(len(Dz)))[:, None, None]
        acc = np.zeros((Lz, Ly, Lx))
        np.add.at(acc, (iz[:, None, None], iy[None, :, None], ix[None, None, :]), -(sg * full))
        K[k] = acc
    return K, (oz, oy, ox)
