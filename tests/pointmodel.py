"""Plain point (non-interval) evaluation of the paper's equations, for the pins.

Written directly from PAPER.md Appendix A in the paper's notation, in double (numpy) or in
mpmath when `mp` is passed.  It is test support: it never calls the oracle or the CUDA path.
It is itself pinned by the identity test (f = 0 at the generated truth with the exact Phi,
tests/test_eventgen.py), which fixes every sign and convention in (A.3)-(A.7).
"""
from __future__ import annotations

import numpy as np


def _lib(mp):
    if mp is None:
        return np.sin, np.cos, np.arctan2, np.sqrt
    return mp.sin, mp.cos, mp.atan2, mp.sqrt


def axial_quantities(xc, yc, x0, y0, sphi, cphi, T, x_ref=0.0, y_ref=0.0, z_ref=0.0, mp=None):
    """(A.4d,e), (A.7a,d,e,f), (1d): returns xA, yA, RAx^2, cAx, sAx, phiAx - phi0 (principal value)."""
    sin, cos, atan2, sqrt = _lib(mp)
    xA = x0 + z_ref * sphi * T                       # (A.4d)
    yA = y0 - z_ref * cphi * T                       # (A.4e)
    Q = (xA - xc) ** 2 + (yA - yc) ** 2              # (A.7a) squared
    cA = -(xc - xA) * sphi + (yc - yA) * cphi        # (A.7d)
    sA = -(xc - xA) * cphi - (yc - yA) * sphi        # (A.7e)
    phi0 = atan2(x_ref - xc, yc - y_ref)             # (1d)
    phiA = atan2(xA - xc, yc - yA)                   # (A.7f)
    dphi = phiA - phi0
    pi = np.pi if mp is None else mp.pi
    if mp is None:
        dphi = np.where(dphi > pi, dphi - 2 * pi, np.where(dphi <= -pi, dphi + 2 * pi, dphi))
    else:
        if dphi > pi:
            dphi -= 2 * pi
        elif dphi <= -pi:
            dphi += 2 * pi
    return xA, yA, Q, cA, sA, dphi


def phi_series(order, xc, yc, R, z0, lam, d, Q, cA, sA, dphi, T, z_ref=0.0, mp=None):
    """e = Phi - Phi_Ax from (A.8a-d) truncated at `order` (1 or 2)."""
    sin, cos, atan2, sqrt = _lib(mp)
    RA = sqrt(Q)
    zA = z0 - z_ref + lam * R * dphi                                  # (A.8d)
    sinA, cosA = sA / RA, cA / RA                                     # (A.7d,e,g)
    P1 = -(zA * sinA + lam * d * cosA) / RA                           # (A.8b)
    e = P1 * T
    if order >= 2:
        cos2A = cosA * cosA - sinA * sinA
        sin2A = 2 * sinA * cosA
        P2 = (lam * R * zA - lam * zA * (R - 2 * d) * cos2A
              + (zA ** 2 + d * (RA + lam ** 2 * (R + RA - d))) * sin2A) / (2 * Q)   # (A.8c)
        e = e + P2 * T * T
    return e


def residual_given_e(e, xc, yc, R, z0, lam, d, Q, cA, sA, dphi, T, z_ref=0.0, mp=None):
    """f = RAx^2 - (R + d_Ax)^2 of (A.5a,b) with Phi = Phi_Ax + e.  Returns (f, d_Ax, u_d)."""
    sin, cos, atan2, sqrt = _lib(mp)
    RA = sqrt(Q)
    sinP = (sA * cos(e) + cA * sin(e)) / RA                           # sin(Phi_Ax + e)
    cosP = (cA * cos(e) - sA * sin(e)) / RA
    u = sqrt(1 + 2 * lam * sinP * T + lam ** 2 * T ** 2 + cosP ** 2 * T ** 2)   # (A.3a)
    dl = d / u
    s_perp = R * (dphi + e)                                           # (A.3b): rho s = Phi + phi_s - phi0
    z = z0 + lam * s_perp - z_ref - dl * cosP * T                     # (A.4c)
    ct = -lam * dl * sA + z * cA                                      # (A.7b)
    rad = (R + dl) ** 2 - 2 * ct * T - (z * T) ** 2 - (lam * dl * T) ** 2   # radicand of (A.5b)
    f = Q - rad                                                       # (A.5a)
    dAx = sqrt(rad) - R if mp is not None or np.all(rad >= 0) else np.sqrt(np.maximum(rad, 0)) - R
    return f, dAx, u


def residual_point(params, wire, d_signed, order=2, x_ref=0.0, y_ref=0.0, z_ref=0.0, mp=None):
    """wire = (x0, y0, sin phi_s, cos phi_s, tan tau); params = (xc, yc, R, z0, lambda)."""
    xc, yc, R, z0, lam = params
    x0, y0, sphi, cphi, T = wire
    xA, yA, Q, cA, sA, dphi = axial_quantities(xc, yc, x0, y0, sphi, cphi, T, x_ref, y_ref, z_ref, mp)
    e = phi_series(order, xc, yc, R, z0, lam, d_signed, Q, cA, sA, dphi, T, z_ref, mp)
    f, dAx, u = residual_given_e(e, xc, yc, R, z0, lam, d_signed, Q, cA, sA, dphi, T, z_ref, mp)
    return f, Q, e
