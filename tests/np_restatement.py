"""Independently STRUCTURED restatement of the scheme for tiny grids (pin P11).

Whole-array NumPy slicing on ghost-padded arrays (np.pad mode 'wrap' / 'edge'), no pencils, no
gather loops -- the opposite structure from oracle/mhd_oracle.cpp.  Used only by
tests/test_oracle_pins.py to catch index-offset, halo-width and boundary-rule slips; it is not an
oracle and nothing else imports it.  Equations: PAPER.md:76 (6), 97-124 (11)-(17), 126, 147-158
(20)-(22).  Arrays are (nz, ny, nx); axis number a (0 = x) is numpy axis 2 - a.
"""
import numpy as np


def _vl(a, b):
    ab = a * b
    with np.errstate(divide="ignore", invalid="ignore"):
        r = 2.0 * ab / (a + b)
    return np.where(ab > 0, r, 0.0)


def _pad(a, w, bc):
    return np.pad(a, w, mode="wrap" if bc == 0 else "edge")


def _sh(a, k, ax):
    """a shifted so that result[i] = a[i + k] along numpy axis ax (valid away from the array ends)."""
    return np.roll(a, -k, ax)


def _flux(u, b, gamma):
    rho, m1, m2, m3, E = u
    v = m1 / rho
    b2 = b[0] ** 2 + b[1] ** 2 + b[2] ** 2
    p = (gamma - 1) * (E - 0.5 * (m1 * m1 + m2 * m2 + m3 * m3) / rho - 0.5 * b2)
    ps = p + 0.5 * b2
    F = [m1, m1 * v + ps - b[0] ** 2, m2 * v - b[1] * b[0], m3 * v - b[2] * b[0],
         (E + ps) * v - b[0] * (b[0] * m1 + b[1] * m2 + b[2] * m3) / rho]
    c = np.abs(v) + np.sqrt(np.abs(gamma * p + b2) / rho)
    return F, c


def fluid(f, gamma, bc, d, dt):
    W = 5
    t1, t2 = (d + 1) % 3, (d + 2) % 3
    ad, a1, a2 = 2 - d, 2 - t1, 2 - t2
    P = [_pad(a, W, bc) for a in f]
    u = [P[0], P[1 + d], P[1 + t1], P[1 + t2], P[4]]
    b = [0.5 * (P[5 + d] + _sh(P[5 + d], 1, ad)), 0.5 * (P[5 + t1] + _sh(P[5 + t1], 1, a1)),
         0.5 * (P[5 + t2] + _sh(P[5 + t2], 1, a2))]
    F, c = _flux(u, b, gamma)
    R = [c * u[k] + F[k] for k in range(5)]
    G = [c * u[k] - F[k] for k in range(5)]
    phi = [0.5 * (R[k] - _sh(G[k], 1, ad)) for k in range(5)]            # face +1/2
    u1 = [u[k] - (phi[k] - _sh(phi[k], -1, ad)) * (dt * 0.5) for k in range(5)]
    F, c = _flux(u1, b, gamma)
    R = [c * u1[k] + F[k] for k in range(5)]
    G = [c * u1[k] - F[k] for k in range(5)]
    out = []
    for k in range(5):
        r, g = R[k], G[k]
        rp = r + _vl(0.5 * (r - _sh(r, -1, ad)), 0.5 * (_sh(r, 1, ad) - r))
        g1, g2 = _sh(g, 1, ad), _sh(g, 2, ad)
        lp = g1 + _vl(0.5 * (g1 - g2), 0.5 * (g - g1))
        ph = 0.5 * (rp - lp)
        out.append(u[k] - (ph - _sh(ph, -1, ad)) * dt)
    core = (slice(W, -W),) * 3
    res = [a.copy() for a in f]
    for k, idx in enumerate([0, 1 + d, 1 + t1, 1 + t2, 4]):
        res[idx] = np.ascontiguousarray(out[k][core])
    return res


def badvect(f, gamma, bc, d, t, dt):
    W = 6
    ad, at = 2 - d, 2 - t
    rho, md, bt, bd = (_pad(f[i], W, bc) for i in (0, 1 + d, 5 + t, 5 + d))
    vt = (_sh(md, -1, at) + md) / (_sh(rho, -1, at) + rho)
    vg = 0.25 * ((_sh(vt, -1, ad) + _sh(vt, 1, ad)) + 2.0 * vt)
    vh = 0.5 * (vg + _sh(vg, 1, ad))                                   # face +1/2
    w = vg * bt
    f1 = np.where(vh > 0, w, _sh(w, 1, ad))
    b1 = bt - (f1 - _sh(f1, -1, ad)) * (dt * 0.5)
    w = vg * b1
    wm, wp, wpp = _sh(w, -1, ad), _sh(w, 1, ad), _sh(w, 2, ad)
    fr = w + _vl(0.5 * (w - wm), 0.5 * (wp - w))
    fl = wp + _vl(0.5 * (wp - wpp), 0.5 * (w - wp))
    fl2 = np.where(vh > 0, fr, fl) * dt                                # at (n+1/2, tau-1/2)
    fm = _sh(fl2, -1, ad)                                              # at (n-1/2, tau-1/2)
    bt_new = bt - (fl2 - fm)
    bd_new = bd + (_sh(fm, 1, at) - fm)
    core = (slice(W, -W),) * 3
    res = [a.copy() for a in f]
    res[5 + t] = np.ascontiguousarray(bt_new[core])
    res[5 + d] = np.ascontiguousarray(bd_new[core])
    return res


def sweep(f, gamma, bc, d, reverse, dt):
    t1, t2 = (d + 1) % 3, (d + 2) % 3
    if not reverse:
        f = fluid(f, gamma, bc, d, dt)
        f = badvect(f, gamma, bc, d, t1, dt)
        f = badvect(f, gamma, bc, d, t2, dt)
    else:
        f = badvect(f, gamma, bc, d, t2, dt)
        f = badvect(f, gamma, bc, d, t1, dt)
        f = fluid(f, gamma, bc, d, dt)
    return f


def step(f, gamma, bc, s, dt):
    order = [(0, 1, 2), (2, 0, 1), (1, 2, 0)][s % 3]
    for d in order:
        f = sweep(f, gamma, bc, d, False, dt)
    for d in reversed(order):
        f = sweep(f, gamma, bc, d, True, dt)
    return f


def cmax(f, gamma, bc):
    P = [_pad(a, 1, bc) for a in f]
    bx = 0.5 * (P[5] + _sh(P[5], 1, 2))
    by = 0.5 * (P[6] + _sh(P[6], 1, 1))
    bz = 0.5 * (P[7] + _sh(P[7], 1, 0))
    rho = P[0]
    b2 = bx * bx + by * by + bz * bz
    p = (gamma - 1) * (P[4] - 0.5 * (P[1] ** 2 + P[2] ** 2 + P[3] ** 2) / rho - 0.5 * b2)
    c = np.maximum(np.maximum(np.abs(P[1] / rho), np.abs(P[2] / rho)), np.abs(P[3] / rho)) + np.sqrt(
        np.abs(gamma * p + b2) / rho)
    return c[1:-1, 1:-1, 1:-1].max()
