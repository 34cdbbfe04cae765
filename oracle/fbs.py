"""Oracle: discrete energy (O3), outer forward-backward splitting loop (O5) and the
coarse-to-fine multigrid cascade with its transfer operators (O6), in plain numpy fp64 on top
of the C primitives.  TEST INFRASTRUCTURE — see oracle/__init__.py.

Follows Algorithm A1 of the paper step by step:
  1. g = f - (mu V / beta) dE2/df
  2. f = argmin E1 + (beta/2) E3            (n_inner gradient-descent steps)
  3. f = 0 where f < 0
Readings of what the paper leaves open (Q-numbers) are listed in DESIGN.md "Readings".
"""
from __future__ import annotations

import math
from dataclasses import replace
from typing import List, Optional, Sequence

import numpy as np


def _prims():
    import oracle as o   # the C-backed primitives
    return o


# ----------------------------------------------------------------------------------------
# O3: discrete energy  (PAPER.md:65-69 with V = N_vox dV, A = N_pix du dv)
#   E_eps(f) = (1/N_vox) sum n_ijk + mu (1/(N_theta N_pix)) sum (P f - Y)^2
# ----------------------------------------------------------------------------------------
def energy(g, f, Y, mu: float, eps: float, Pf: Optional[np.ndarray] = None) -> dict:
    o = _prims()
    if Pf is None:
        Pf = o.forward(g, f)
    data = float(np.sum((Pf - Y) ** 2)) / (g.n_angles * g.n_pix)
    tv_eps = o.tv_value(g, f, eps) / g.n_vox
    tv_0 = o.tv_value(g, f, 0.0) / g.n_vox
    return {"E_eps": tv_eps + mu * data, "E_0": tv_0 + mu * data, "E1_eps": tv_eps, "E1_0": tv_0, "E2": data}


# ----------------------------------------------------------------------------------------
# O5: one level of Algorithm A1 with fixed iteration counts (Q10)
#   c = 2 s N_vox / (N_theta N_pix),  s = step = mu/beta   (P:87 with eq. 2's factor 2; Q9)
# ----------------------------------------------------------------------------------------
def fbs_level(g, Y, f0, n_outer: int, n_inner: int, step: float, mu: float, eps: float,
              omega: float = 1.0, u0_mode: str = "g", clamp: bool = True,
              trace: Optional[list] = None, backprojector: str = "exact",
              rel_tol: float = 0.0, iters_done: Optional[list] = None, tau: Optional[np.ndarray] = None) -> np.ndarray:
    """tau (NEXT-3, FAS coarse problems): a linear term -<tau, f> added to the smooth part of the level's objective
    N_vox E = TV_eps(f) + mu' ||P f - Y||^2, mu' = mu N_vox / (N_theta N_pix); it joins the gradient of step 1:
    g = f - (1/beta) (2 mu' P^T (P f - Y) - tau) = f - c P^T (P f - Y) + tau / beta.  tau = None is Algorithm A1 as printed.
    rel_tol > 0: "Repeat ... until convergence" read as: stop after the first iteration whose update
    satisfies ||f_new - f_old||_2 <= rel_tol ||f_new||_2 (NEXT-2; n_outer is then the maximum count);
    the number of iterations run is appended to iters_done.
    backprojector = "exact": dE2/df through the matrix transpose (the hot path);
    "eq2": through the paper's eq. 2: dE2/df(x) = (2/(N_theta A)) (B r)(x), so step 1 reads
    g = f - (mu V/beta) dE2/df = f - c (dV/(du dv)) (B r) with the same c."""
    o = _prims()
    f = np.array(f0, dtype=np.float64, copy=True)
    beta = mu / step
    c = 2.0 * step * g.n_vox / (g.n_angles * g.n_pix)
    done = 0
    for _ in range(n_outer):
        f_old = f
        r = o.forward(g, f) - Y                      # P f - Y
        if backprojector == "exact":
            G = o.backproject(g, r)                  # P^T (P f - Y)
        else:
            G = (g.hx * g.hy * g.hz / (g.du * g.dv)) * o.backproject_eq2(g, r)   # eq. 2
        gv = f - c * G                               # step 1
        if tau is not None:
            gv = gv + tau / beta                     # FAS right-hand side (Q21)
        u0 = gv if u0_mode == "g" else f             # Q7: start of the inner descent
        u = o.tv_prox(g, gv, u0, beta, eps, omega, n_inner)   # step 2
        f = np.maximum(u, 0.0) if clamp else u       # step 3             (Q18)
        if trace is not None:
            trace.append(energy(g, f, Y, mu, eps))
        done += 1
        if rel_tol > 0.0 and np.sqrt(np.sum((f - f_old) ** 2)) <= rel_tol * np.sqrt(np.sum(f ** 2)):
            break
    if iters_done is not None:
        iters_done.append(done)
    return f


# ----------------------------------------------------------------------------------------
# O6: multigrid cascade ("multi-grid method", no details given: Q11)
# ----------------------------------------------------------------------------------------
def coarsen_axes(g) -> tuple:
    """Axes (x,y,z) coarsened by 2 at the next level: those with spacing <= sqrt(2) min(h)."""
    h = (g.hx, g.hy, g.hz)
    m = min(h)
    return tuple(ha <= math.sqrt(2.0) * m * (1.0 + 1e-9) for ha in h)


def coarsen_geometry(g, bin_detector: bool = True):
    """Next-coarser level: halve the dims / double the spacing on coarsen_axes; bin the detector
    2x2 (pitch doubles) iff both x and y were coarsened.  Returns (geometry, axes, binned).
    bin_detector = False (NEXT-3, Q20): the coarse levels keep the detector, and the data, at full resolution."""
    ax = coarsen_axes(g)
    n = [g.nx, g.ny, g.nz]
    h = [g.hx, g.hy, g.hz]
    for a in range(3):
        if ax[a]:
            if n[a] % 2:
                raise ValueError("odd dimension on an axis that must coarsen")
            n[a] //= 2
            h[a] *= 2.0
    binned = bool(ax[0] and ax[1]) and bin_detector
    nu, nv, du, dv = g.nu, g.nv, g.du, g.dv
    if binned:
        if nu % 2 or nv % 2:
            raise ValueError("odd detector dimension on a level that bins the detector")
        nu, nv, du, dv = nu // 2, nv // 2, du * 2.0, dv * 2.0
    gc = replace(g, nu=nu, nv=nv, du=du, dv=dv, nx=n[0], ny=n[1], nz=n[2], hx=h[0], hy=h[1], hz=h[2])
    return gc, ax, binned


def level_geometries(g, n_levels: int, bin_detector: bool = True):
    """[level 0 (finest), ..., level n_levels-1 (coarsest)] with the transfer descriptors."""
    geoms, axes, binned = [g], [], []
    for _ in range(n_levels - 1):
        gc, ax, b = coarsen_geometry(geoms[-1], bin_detector)
        geoms.append(gc)
        axes.append(ax)
        binned.append(b)
    return geoms, axes, binned


def bin2x2(Y: np.ndarray) -> np.ndarray:
    """Mean of each 2x2 block of detector pixels, per angle."""
    na, nv, nu = Y.shape
    return Y.reshape(na, nv // 2, 2, nu // 2, 2).mean(axis=(2, 4))


def restrict_volume(f: np.ndarray, axes) -> np.ndarray:
    """Mean over the 2 children along every coarsened axis (used only to bring a caller's f0 down)."""
    out = f
    for a, arr_axis in zip(range(3), (2, 1, 0)):          # x is the last array axis
        if axes[a]:
            sh = list(out.shape)
            sh[arr_axis] //= 2
            sh.insert(arr_axis + 1, 2)
            out = out.reshape(sh).mean(axis=arr_axis + 1)
    return out


def _prolong_axis(c: np.ndarray, arr_axis: int) -> np.ndarray:
    """Cell-centred linear interpolation along one array axis:
    fine[2I] = 3/4 c[I] + 1/4 c[I-1],  fine[2I+1] = 3/4 c[I] + 1/4 c[I+1], indices clamped."""
    c = np.moveaxis(c, arr_axis, 0)
    n = c.shape[0]
    lo = np.concatenate([c[:1], c[:-1]], axis=0)          # c[I-1], clamped
    hi = np.concatenate([c[1:], c[-1:]], axis=0)          # c[I+1], clamped
    out = np.empty((2 * n,) + c.shape[1:], dtype=c.dtype)
    out[0::2] = 0.75 * c + 0.25 * lo
    out[1::2] = 0.75 * c + 0.25 * hi
    return np.moveaxis(out, 0, arr_axis)


def prolong(c: np.ndarray, axes) -> np.ndarray:
    """Coarse volume -> next finer level (cell-centred trilinear over the coarsened axes, x then y then z)."""
    out = c
    for a, arr_axis in zip(range(3), (2, 1, 0)):
        if axes[a]:
            out = _prolong_axis(out, arr_axis)
    return np.ascontiguousarray(out)


def fbs_reconstruct(g, Y, f0, n_levels: int, n_outer: Sequence[int], n_inner: int, step: float,
                    mu: float, eps: float, omega: float = 1.0, u0_mode: str = "g",
                    clamp: bool = True, trace: Optional[list] = None, backprojector: str = "exact",
                    rel_tol: float = 0.0, iters_done: Optional[list] = None, bin_detector: bool = True) -> np.ndarray:
    """O6: run O5 at the coarsest level from f0 (zeros if None; a caller's fine-grid f0 is
    restricted down), prolong to the next level, repeat; n_outer is listed coarsest first.
    n_levels = 1 is exactly O5."""
    assert len(n_outer) == n_levels
    geoms, axes, binned = level_geometries(g, n_levels, bin_detector)
    Ys = [np.asarray(Y, dtype=np.float64)]
    for b in binned:
        Ys.append(bin2x2(Ys[-1]) if b else Ys[-1])
    if f0 is None:
        f = np.zeros(geoms[-1].vol_shape)
    else:
        f = np.asarray(f0, dtype=np.float64)
        for ax in axes:
            f = restrict_volume(f, ax)
    for n, lev in enumerate(range(n_levels - 1, -1, -1)):
        f = fbs_level(geoms[lev], Ys[lev], f, n_outer[n], n_inner, step, mu, eps, omega,
                      u0_mode=u0_mode, clamp=clamp, trace=trace, backprojector=backprojector,
                      rel_tol=rel_tol, iters_done=iters_done)
        if lev > 0:
            f = prolong(f, axes[lev - 1])
    return f


# ----------------------------------------------------------------------------------------
# NEXT-3: FAS V-cycles ("multi-grid method", ref. 20 = Brandt; no details given: reading Q21)
#
# Every level l has the same kind of objective, scaled by its voxel count:
#   F_l(f) = N_vox,l E_eps,l(f) = TV_eps,l(f) + mu'_l ||P_l f - Y_l||^2,  mu'_l = mu N_vox,l / (N_theta N_pix,l),
# whose gradient  grad F_l(f) = grad TV_eps,l(f) + 2 mu'_l P_l^T (P_l f - Y_l)  is a discretisation of the
# level-independent functional derivative V dE/df (P:65-69 normalise E1 by V and E2 by A), so gradients can be moved
# between levels by plain averaging.  Brandt's full approximation scheme for the nonlinear problem:
#   V(l, f, tau):   f <- nu_pre iterations of A1 on  F_l(f) - <tau, f>                      (pre-smoothing)
#                   if l is not the coarsest level:
#                       f_H0  = R f                     (R = mean of the children, restrict_volume)
#                       tau_H = grad F_{l+1}(f_H0) - R (grad F_l(f) - tau)                 (residual restriction)
#                       f_H   = V(l+1, f_H0, tau_H)
#                       f <- max(f + Prolong(f_H - f_H0), 0)                                (correction, kept feasible: P:91)
#                       f <- nu_post iterations of A1 on  F_l(f) - <tau, f>                 (post-smoothing)
#   at the coarsest level the smoother runs nu_coarse iterations instead.
# The finest level has tau = 0.  The linear term enters A1 through step 1 (fbs_level(tau=...)).
# ----------------------------------------------------------------------------------------
def grad_objective(g, f, Y, mu: float, eps: float) -> np.ndarray:
    """grad F_l(f) = grad TV_eps(f) + 2 mu' P^T (P f - Y),  mu' = mu N_vox / (N_theta N_pix)   (N_vox times the gradient of O3)."""
    o = _prims()
    mu_p = mu * g.n_vox / (g.n_angles * g.n_pix)
    return o.tv_grad(g, f, eps) + 2.0 * mu_p * o.backproject(g, o.forward(g, f) - Y)


def fbs_vcycle(g, Y, f0, n_levels: int, n_cycles: int, nu_pre: int, nu_post: int, nu_coarse: int, n_inner: int,
               step: float, mu: float, eps: float, omega: float = 1.0, bin_detector: bool = True,
               trace: Optional[list] = None) -> np.ndarray:
    """n_cycles FAS V-cycles on the finest level, starting from f0 (zeros if None).  n_levels = 1 is plain A1 with
    n_cycles * nu_coarse iterations.  trace (optional) receives energy(f) after every cycle."""
    geoms, axes, binned = level_geometries(g, n_levels, bin_detector)
    Ys = [np.asarray(Y, dtype=np.float64)]
    for b in binned:
        Ys.append(bin2x2(Ys[-1]) if b else Ys[-1])

    def smooth(l, f, tau, n):
        return fbs_level(geoms[l], Ys[l], f, n, n_inner, step, mu, eps, omega, tau=tau)

    def V(l, f, tau):
        if l == n_levels - 1:
            return smooth(l, f, tau, nu_coarse)
        f = smooth(l, f, tau, nu_pre)
        D = grad_objective(geoms[l], f, Ys[l], mu, eps)
        if tau is not None:
            D = D - tau
        fH0 = restrict_volume(f, axes[l])
        tauH = grad_objective(geoms[l + 1], fH0, Ys[l + 1], mu, eps) - restrict_volume(D, axes[l])
        fH = V(l + 1, fH0, tauH)
        f = np.maximum(f + prolong(fH - fH0, axes[l]), 0.0)
        return smooth(l, f, tau, nu_post)

    f = np.zeros(g.vol_shape) if f0 is None else np.array(f0, dtype=np.float64, copy=True)
    for _ in range(n_cycles):
        f = V(0, f, None)
        if trace is not None:
            trace.append(energy(g, f, Ys[0], mu, eps))
    return f


def lambda_max(g, iters: int = 30, seed: int = 0) -> float:
    """Largest eigenvalue of P^T P by power iteration from a seeded positive start (Q8)."""
    o = _prims()
    x = np.random.default_rng(seed).random(g.vol_shape) + 0.5
    x /= np.linalg.norm(x)
    lam = 0.0
    for _ in range(iters):
        y = o.backproject(g, o.forward(g, x))
        lam = float(np.linalg.norm(y))
        x = y / lam
    return lam
