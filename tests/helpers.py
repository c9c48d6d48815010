"""Test-side machinery that is independent of the oracle's arithmetic: high-order
quadrature on triangles/edges, exact monomial integrals, a brute-force evaluation of the
weak form (eq. (3)) with a numpy LLF flux written in the x-y frame, and
small mesh builders.  Nothing here is imported by the product or by oracle/."""
from __future__ import annotations

from math import factorial

import numpy as np
from numpy.polynomial.legendre import leggauss

G = 9.81


# ----------------------------------------------------------------------- quadrature
def tri_rule_bary(n: int = 12):
    """Collapsed (Duffy) Gauss rule on the unit-area-normalised triangle: returns
    barycentrics lam[nq,3] and weights summing to 1; exact to degree 2n-2."""
    x, w = leggauss(n)
    u, wu = 0.5 * (x + 1.0), 0.5 * w
    U, V = np.meshgrid(u, u, indexing="ij")
    WU, WV = np.meshgrid(wu, wu, indexing="ij")
    l1 = U.ravel()
    l2 = (V * (1.0 - U)).ravel()
    wt = (WU * WV * (1.0 - U)).ravel() * 2.0
    lam = np.stack([1.0 - l1 - l2, l1, l2], axis=1)
    return lam, wt


def monomial_integral_bary(a: int, b: int, c: int, area: float = 1.0) -> float:
    """Exact: int_T lam0^a lam1^b lam2^c = 2 A a! b! c! / (a+b+c+2)!"""
    return 2.0 * area * factorial(a) * factorial(b) * factorial(c) / factorial(a + b + c + 2)


def gauss_edge(n: int = 8):
    x, w = leggauss(n)
    return 0.5 * (x + 1.0), 0.5 * w  # s in [0,1], weights sum 1


# ----------------------------------------------------------------------- tiny meshes
def two_element_mesh():
    from workloads.mesh import make_mesh
    xy = np.array([[0.0, 0.0], [900.0, 100.0], [1000.0, 1100.0], [-50.0, 800.0]])
    tri = np.array([[0, 1, 2], [0, 2, 3]], dtype=np.int32)
    return make_mesh(xy, tri)


def small_mesh(nq=2, L=1000.0, jitter=0.25, seed=7, permute=True, ocean=False):
    from workloads.mesh import rect_mesh
    rng = np.random.default_rng(seed)
    pred = (lambda xm, ym: xm > L - 1e-6 * L) if ocean else None
    return rect_mesh(nq, nq, L, L, diag="random", jitter=jitter, permute=permute, rng=rng, ocean_pred=pred)


# ----------------------------------------------------------------------- oracle-basis utilities
def eval_basis(O, lam, ndof=6):
    """phi[nq, ndof] via the oracle's (separately pinned) basis (it evaluates all ten modes up to p = 3)."""
    return np.array([O.basis(*l)[0] for l in lam])[:, :ndof]


def l2_project(O, mesh, fn, p):
    """Modal coefficients [ndof, n_elem] of the L2 projection of fn(x, y) (vectorised)
    onto the Dubiner basis, by high-order quadrature; M_k from the closed form."""
    ndof = (p + 1) * (p + 2) // 2
    lam, wt = tri_rule_bary(10)
    phi = eval_basis(O, lam, 10)[:, :ndof]
    Mref = np.array([2.0, 1.0, 1.0 / 3.0, 2.0 / 3.0, 2.0 / 9.0, 2.0 / 15.0, 0.5, 1.0 / 6.0, 0.1, 1.0 / 14.0])[:ndof]
    xy, tri = mesh.xy, mesh.tri
    out = np.zeros((ndof, tri.shape[0]))
    for e, t in enumerate(tri):
        P = lam @ xy[t]
        f = fn(P[:, 0], P[:, 1])
        out[:, e] = (2.0 * wt * f) @ phi / Mref      # reference area 2
    return out


# ----------------------------------------------------------------------- brute force weak form
def phys_flux(z, qx, qy, h, h0):
    H = np.maximum(z + h, h0)
    P = 0.5 * G * ((z + h) ** 2 - h ** 2)
    return (np.stack([qx, qx * qx / H + P, qx * qy / H]),     # x-flux of (zeta, Qx, Qy)
            np.stack([qy, qx * qy / H, qy * qy / H + P]))     # y-flux


def llf_xy(wp, wm, h, n, h0):
    """Local Lax-Friedrichs normal flux written in the x-y frame (independent of the
    oracle's rotated-frame code): 1/2 (F(w+)+F(w-)).n - 1/2 lam (w- - w+)."""
    Fxp, Fyp = phys_flux(*wp, h, h0)
    Fxm, Fym = phys_flux(*wm, h, h0)
    Hp, Hm = np.maximum(wp[0] + h, h0), np.maximum(wm[0] + h, h0)
    unp = (wp[1] * n[0] + wp[2] * n[1]) / Hp
    unm = (wm[1] * n[0] + wm[2] * n[1]) / Hm
    lam = np.maximum(np.abs(unp) + np.sqrt(G * Hp), np.abs(unm) + np.sqrt(G * Hm))
    return 0.5 * ((Fxp + Fxm) * n[0] + (Fyp + Fym) * n[1]) - 0.5 * lam * (np.stack(wm) - np.stack(wp))


def brute_force_rhs(O, mesh, bathy, p, ze, qx, qy, *, h0=1e-3, cf=0.0, fcor=0.0, zeta_b=0.0, nq_tri=12, nq_edge=10):
    """d/dt of the modal coefficients from eq. (3) with the volume sign of eq. (6) and a
    DENSE mass-matrix solve, all integrals by high-order quadrature.  Returns [3, ndof, n_elem]."""
    ndof = (p + 1) * (p + 2) // 2
    lam, wt = tri_rule_bary(nq_tri)
    B = np.array([O.basis(*l) for l in lam])      # [nq, 3(phi,d1,d2), 6]
    phi, d1, d2 = B[:, 0, :ndof], B[:, 1, :ndof], B[:, 2, :ndof]
    s_e, w_e = gauss_edge(nq_edge)
    xy, tri = mesh.xy, mesh.tri
    W = np.stack([ze, qx, qy])                    # [3, ndof, ne]
    out = np.zeros((3, ndof, tri.shape[0]))
    for e, t in enumerate(tri):
        X = xy[t]
        d1v, d2v = X[1] - X[0], X[2] - X[0]
        A = 0.5 * (d1v[0] * d2v[1] - d2v[0] * d1v[1])
        # grad lambda_1, lambda_2 ; xi_i = 2 lam_i - 1
        gl1 = np.array([d2v[1], -d2v[0]]) / (2 * A)
        gl2 = np.array([-d1v[1], d1v[0]]) / (2 * A)
        gphix = d1 * (2 * gl1[0]) + d2 * (2 * gl2[0])
        gphiy = d1 * (2 * gl1[1]) + d2 * (2 * gl2[1])
        hv = bathy[t]
        hq = lam @ hv
        gh = hv[0] * (-(gl1 + gl2)) + hv[1] * gl1 + hv[2] * gl2
        wq = [phi @ W[c, :, e] for c in range(3)]
        Fx, Fy = phys_flux(*wq, hq, h0)
        H = np.maximum(wq[0] + hq, h0)
        tau = cf * np.sqrt(wq[1] ** 2 + wq[2] ** 2) / H ** 2
        S = np.stack([np.zeros_like(hq),
                      G * wq[0] * gh[0] - tau * wq[1] + fcor * wq[2],
                      G * wq[0] * gh[1] - tau * wq[2] - fcor * wq[1]])
        R = np.zeros((3, ndof))
        for c in range(3):
            R[c] = A * ((wt * Fx[c]) @ gphix + (wt * Fy[c]) @ gphiy + (wt * S[c]) @ phi)
        # edges
        for l in range(3):
            a, b = (l + 1) % 3, (l + 2) % 3
            d = mesh.elem_edge[e, l]
            ep, em = mesh.edge_elem[d]
            other = em if ep == e else ep
            ev = X[b] - X[a]
            Ln = np.hypot(*ev)
            n = np.array([ev[1], -ev[0]]) / Ln
            pts = X[a][None, :] + s_e[:, None] * ev[None, :]
            lam_own = np.zeros((len(s_e), 3)); lam_own[:, a] = 1 - s_e; lam_own[:, b] = s_e
            ph_own = eval_basis(O, lam_own, 10)[:, :ndof]
            wp = [ph_own @ W[c, :, e] for c in range(3)]
            hq_e = lam_own @ hv
            bc = mesh.edge_bc[d]
            if bc == 0:
                Xo = xy[tri[other]]
                # barycentrics of the same physical points in the neighbour
                T = np.array([[Xo[1][0] - Xo[0][0], Xo[2][0] - Xo[0][0]], [Xo[1][1] - Xo[0][1], Xo[2][1] - Xo[0][1]]])
                l12 = np.linalg.solve(T, (pts - Xo[0]).T).T
                lam_o = np.stack([1 - l12.sum(1), l12[:, 0], l12[:, 1]], 1)
                ph_o = eval_basis(O, lam_o, 10)[:, :ndof]
                wm = [ph_o @ W[c, :, other] for c in range(3)]
            elif bc == 1:
                qn = wp[1] * n[0] + wp[2] * n[1]
                wm = [wp[0], wp[1] - 2 * qn * n[0], wp[2] - 2 * qn * n[1]]
            else:
                wm = [np.full_like(wp[0], zeta_b), wp[1], wp[2]]
            Fh = llf_xy(wp, wm, hq_e, n, h0)
            for c in range(3):
                R[c] -= Ln * ((w_e * Fh[c]) @ ph_own)
        Mass = A * (phi * wt[:, None]).T @ phi       # dense
        for c in range(3):
            out[c, :, e] = np.linalg.solve(Mass, R[c])
    return out
