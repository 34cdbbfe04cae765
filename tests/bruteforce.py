"""Independent numpy restatements used to PIN the oracle (never imported by oracle/ or by the
CUDA path).  Everything here is the plain definition written out a second time, vectorised:

* ray endpoints from the O0 convention,
* one system-matrix entry = length of (segment S->D) ∩ (voxel box), by slab clipping,
* smoothed isotropic TV value and its exact gradient,
* a dense-matrix FBS iteration.
"""
import numpy as np


def ray_endpoints(g):
    """S: (na,3); D: (na,nv,nu,3)."""
    t = np.asarray(g.angles)
    c, s = np.cos(t), np.sin(t)
    S = np.stack([g.sad * c, g.sad * s, np.zeros_like(t)], axis=-1)
    # a shifted panel (half-fan): every pixel centre moves by (off_u, off_v) in the detector plane
    uu = np.linspace(-(g.nu - 1) / 2.0, (g.nu - 1) / 2.0, g.nu) * g.du + getattr(g, "off_u", 0.0)
    vv = np.linspace(-(g.nv - 1) / 2.0, (g.nv - 1) / 2.0, g.nv) * g.dv + getattr(g, "off_v", 0.0)
    D = np.empty((len(t), g.nv, g.nu, 3))
    D[..., 0] = (-(g.sdd - g.sad) * c)[:, None, None] + uu[None, None, :] * (-s)[:, None, None]
    D[..., 1] = (-(g.sdd - g.sad) * s)[:, None, None] + uu[None, None, :] * c[:, None, None]
    D[..., 2] = vv[None, :, None]
    return S, D


def clip_lengths(S, D, lo, hi):
    """Length of segment S[r]->D[r] inside box [lo[b],hi[b]) for all (r,b): shape (R,B)."""
    S = S[:, None, :]
    d = (D[:, None, :] - S)
    L = np.sqrt((d ** 2).sum(-1))
    lo = lo[None, :, :]
    hi = hi[None, :, :]
    with np.errstate(divide="ignore", invalid="ignore"):
        a0 = (lo - S) / d
        a1 = (hi - S) / d
    amin_a = np.minimum(a0, a1)
    amax_a = np.maximum(a0, a1)
    par = (d == 0.0)
    inside = (S >= lo) & (S < hi)
    amin_a = np.where(par, np.where(inside, -np.inf, np.inf), amin_a)
    amax_a = np.where(par, np.where(inside, np.inf, -np.inf), amax_a)
    amin = np.maximum(amin_a.max(-1), 0.0)
    amax = np.minimum(amax_a.min(-1), 1.0)
    return np.maximum(amax - amin, 0.0) * L


def voxel_boxes(g):
    i, j, k = np.meshgrid(np.arange(g.nx), np.arange(g.ny), np.arange(g.nz), indexing="ij")
    # order boxes like the volume layout f[k][j][i]
    i = i.transpose(2, 1, 0).ravel()
    j = j.transpose(2, 1, 0).ravel()
    k = k.transpose(2, 1, 0).ravel()
    lo = np.stack([(i - g.nx / 2.0) * g.hx, (j - g.ny / 2.0) * g.hy, (k - g.nz / 2.0) * g.hz], -1)
    hi = lo + np.array([g.hx, g.hy, g.hz])
    return lo, hi


def dense_matrix(g):
    """(n_rays, n_vox) matrix of chord lengths, rows ordered [theta][iv][iu], columns [k][j][i]."""
    S, D = ray_endpoints(g)
    lo, hi = voxel_boxes(g)
    rows = []
    for ia in range(g.n_angles):
        Dr = D[ia].reshape(-1, 3)
        Sr = np.repeat(S[ia][None], Dr.shape[0], 0)
        rows.append(clip_lengths(Sr, Dr, lo, hi))
    return np.concatenate(rows, 0)


def box_chords(g):
    """P applied to the all-ones volume = length of each ray inside the volume's bounding box (pin I1)."""
    S, D = ray_endpoints(g)
    ext = np.array([g.nx * g.hx, g.ny * g.hy, g.nz * g.hz])
    lo = (-ext / 2.0)[None]
    hi = (ext / 2.0)[None]
    out = np.empty(g.proj_shape)
    for ia in range(g.n_angles):
        Dr = D[ia].reshape(-1, 3)
        Sr = np.repeat(S[ia][None], Dr.shape[0], 0)
        out[ia] = clip_lengths(Sr, Dr, lo, hi)[:, 0].reshape(g.nv, g.nu)
    return out


# ---------------------------------------------------------------- TV (independent) -----
def _diffs(f, g):
    dx = np.zeros_like(f); dy = np.zeros_like(f); dz = np.zeros_like(f)
    dx[:, :, :-1] = (f[:, :, 1:] - f[:, :, :-1]) / g.hx
    dy[:, :-1, :] = (f[:, 1:, :] - f[:, :-1, :]) / g.hy
    dz[:-1, :, :] = (f[1:, :, :] - f[:-1, :, :]) / g.hz
    return dx, dy, dz


def tv_value(f, g, eps):
    dx, dy, dz = _diffs(f, g)
    return np.sqrt(dx * dx + dy * dy + dz * dz + eps * eps).sum()   # keeps the input precision (longdouble for FD checks)


def tv_grad(f, g, eps):
    dx, dy, dz = _diffs(f, g)
    n = np.sqrt(dx * dx + dy * dy + dz * dz + eps * eps)
    px, py, pz = dx / n / g.hx, dy / n / g.hy, dz / n / g.hz
    out = -(px + py + pz)
    out[:, :, 1:] += px[:, :, :-1]
    out[:, 1:, :] += py[:, :-1, :]
    out[1:, :, :] += pz[:-1, :, :]
    return out


def dense_fbs(A, g, Y, f0, n_outer, n_inner, step, mu, eps, omega=1.0, u0_mode="g", clamp=True):
    """Algorithm A1 with explicit matrix algebra; returns the list of iterates."""
    f = f0.ravel().copy()
    y = Y.ravel()
    beta = mu / step
    c = 2.0 * step * g.n_vox / (g.n_angles * g.n_pix)
    dt = omega / (beta + 4.0 * (1 / g.hx ** 2 + 1 / g.hy ** 2 + 1 / g.hz ** 2) / eps)
    its = []
    for _ in range(n_outer):
        gv = f - c * (A.T @ (A @ f - y))
        u = (gv if u0_mode == "g" else f).copy()
        for _ in range(n_inner):
            u = u - dt * (beta * (u - gv) + tv_grad(u.reshape(g.vol_shape), g, eps).ravel())
        f = np.maximum(u, 0.0) if clamp else u
        its.append(f.reshape(g.vol_shape).copy())
    return its


def eq2_backproject(g, r):
    """Eq. 2 a second time, from similar triangles instead of 3-D distances, with the
    interpolation done by a library routine (scipy.ndimage.map_coordinates, order 1, zero beyond the grid):
    voxel centre x; t = depth of x along the central ray, s = lateral offset; u* = SDD s/t, v* = SDD z/t;
    L/l = SDD/t  =>  L^3/(L0 l^2) = (SDD/t)^2 (l/t)."""
    from scipy.ndimage import map_coordinates
    xs = (np.arange(g.nx) - (g.nx - 1) / 2.0) * g.hx
    ys = (np.arange(g.ny) - (g.ny - 1) / 2.0) * g.hy
    zs = (np.arange(g.nz) - (g.nz - 1) / 2.0) * g.hz
    Z, Y, X = np.meshgrid(zs, ys, xs, indexing="ij")
    out = np.zeros(g.vol_shape)
    for ia, th in enumerate(np.asarray(g.angles)):
        c, s = np.cos(th), np.sin(th)
        t = g.sad - (X * c + Y * s)
        lat = -X * s + Y * c
        pu = (g.sdd * lat / t - getattr(g, "off_u", 0.0)) / g.du + (g.nu - 1) / 2.0
        pv = (g.sdd * Z / t - getattr(g, "off_v", 0.0)) / g.dv + (g.nv - 1) / 2.0
        val = map_coordinates(np.asarray(r[ia], dtype=np.float64), [pv.ravel(), pu.ravel()], order=1,
                              mode="grid-constant", cval=0.0).reshape(g.vol_shape)
        w = (g.sdd / t) ** 2 * np.sqrt(t * t + lat * lat + Z * Z) / t
        out += w * val
    return out


# ------------------------------------------------ NEXT-3: FAS V-cycle with explicit matrices -----
def _axis_restrict(n_fine):
    """(n_fine/2, n_fine): mean of the two children."""
    R = np.zeros((n_fine // 2, n_fine))
    for I in range(n_fine // 2):
        R[I, 2 * I] = 0.5
        R[I, 2 * I + 1] = 0.5
    return R


def _axis_prolong(n_coarse):
    """(2 n_coarse, n_coarse): fine 2I = 3/4 c[I] + 1/4 c[I-1], fine 2I+1 = 3/4 c[I] + 1/4 c[I+1], indices clamped."""
    P = np.zeros((2 * n_coarse, n_coarse))
    for I in range(n_coarse):
        P[2 * I, I] += 0.75
        P[2 * I, max(I - 1, 0)] += 0.25
        P[2 * I + 1, I] += 0.75
        P[2 * I + 1, min(I + 1, n_coarse - 1)] += 0.25
    return P


def transfer_matrices(g_fine, g_coarse):
    """Dense restriction (n_c x n_f) and prolongation (n_f x n_c) between two levels, volumes flattened [k][j][i];
    an axis that keeps its size gets the identity."""
    def ax(nf, nc):
        return (np.eye(nf), np.eye(nf)) if nf == nc else (_axis_restrict(nf), _axis_prolong(nc))
    Rx, Px = ax(g_fine.nx, g_coarse.nx)
    Ry, Py = ax(g_fine.ny, g_coarse.ny)
    Rz, Pz = ax(g_fine.nz, g_coarse.nz)
    return np.kron(Rz, np.kron(Ry, Rx)), np.kron(Pz, np.kron(Py, Px))


def dense_vcycle(levels, f0, n_cycles, nu_pre, nu_post, nu_coarse, n_inner, step, mu, eps, omega=1.0):
    """Brandt's full approximation scheme around Algorithm A1, written with explicit matrices.
    levels[l] = dict(g=geometry, A=dense system matrix, Y=data); level 0 is the finest.  Objective per level
    F(f) = TV_eps(f) + mu' |A f - y|^2 with mu' = mu N_vox/(N_theta N_pix); smoother = A1 with the extra gradient term -tau."""
    beta = mu / step
    T = [transfer_matrices(levels[l]["g"], levels[l + 1]["g"]) for l in range(len(levels) - 1)]

    def grad(l, f):
        g, A, y = levels[l]["g"], levels[l]["A"], levels[l]["Y"].ravel()
        mu_p = mu * g.n_vox / (g.n_angles * g.n_pix)
        return tv_grad(f.reshape(g.vol_shape), g, eps).ravel() + 2.0 * mu_p * (A.T @ (A @ f - y))

    def smooth(l, f, tau, n):
        g, A, y = levels[l]["g"], levels[l]["A"], levels[l]["Y"].ravel()
        c = 2.0 * step * g.n_vox / (g.n_angles * g.n_pix)
        dt = omega / (beta + 4.0 * (1 / g.hx ** 2 + 1 / g.hy ** 2 + 1 / g.hz ** 2) / eps)
        for _ in range(n):
            gv = f - c * (A.T @ (A @ f - y)) + tau / beta
            u = gv.copy()
            for _ in range(n_inner):
                u = u - dt * (beta * (u - gv) + tv_grad(u.reshape(g.vol_shape), g, eps).ravel())
            f = np.maximum(u, 0.0)
        return f

    def V(l, f, tau):
        if l == len(levels) - 1:
            return smooth(l, f, tau, nu_coarse)
        f = smooth(l, f, tau, nu_pre)
        R, P = T[l]
        fH0 = R @ f
        tauH = grad(l + 1, fH0) - R @ (grad(l, f) - tau)
        fH = V(l + 1, fH0, tauH)
        f = np.maximum(f + P @ (fH - fH0), 0.0)
        return smooth(l, f, tau, nu_post)

    f = f0.ravel().astype(np.float64).copy()
    for _ in range(n_cycles):
        f = V(0, f, np.zeros_like(f))
    return f.reshape(levels[0]["g"].vol_shape)


# ------------------------------------------------ NEXT-4: FDK backprojection a second time -----
def fdk_backproject(g, q, scale):
    """scale * sum_theta SAD^2/U^2 q(u*,v*), the interpolation done by scipy.ndimage.map_coordinates (order 1, zero beyond
    the grid), coordinates from similar triangles."""
    from scipy.ndimage import map_coordinates
    xs = (np.arange(g.nx) - (g.nx - 1) / 2.0) * g.hx
    ys = (np.arange(g.ny) - (g.ny - 1) / 2.0) * g.hy
    zs = (np.arange(g.nz) - (g.nz - 1) / 2.0) * g.hz
    Z, Y, X = np.meshgrid(zs, ys, xs, indexing="ij")
    out = np.zeros(g.vol_shape)
    for ia, th in enumerate(np.asarray(g.angles)):
        c, s = np.cos(th), np.sin(th)
        U = g.sad - (X * c + Y * s)
        pu = (g.sdd * (-X * s + Y * c) / U - getattr(g, "off_u", 0.0)) / g.du + (g.nu - 1) / 2.0
        pv = (g.sdd * Z / U - getattr(g, "off_v", 0.0)) / g.dv + (g.nv - 1) / 2.0
        val = map_coordinates(np.asarray(q[ia], dtype=np.float64), [pv.ravel(), pu.ravel()], order=1,
                              mode="grid-constant", cval=0.0).reshape(g.vol_shape)
        out += (g.sad / U) ** 2 * val
    return scale * out
