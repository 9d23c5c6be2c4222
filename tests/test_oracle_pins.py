"""Pins of the oracle (oracle/mhd_oracle.cpp) to things OTHER than itself  (-m "not gpu").

The paper prints no numerical field values (figures only), so the pins are what the paper and the
mathematics fix: conservation (flux form), div B (constrained transport), second
order in space and time measured on linear MHD eigenmodes against their closed-form
solution, the exact Riemann solution for B = 0, symmetries, exact special cases, and a brute-force
comparison with an independently structured NumPy restatement on tiny grids.
"""
import math

import numpy as np
import pytest

import oracle
from paper_0908_4362_b200 import inputs
from tests import np_restatement as npr

P, O = inputs.PERIODIC, inputs.OUTFLOW


def c64(fields):
    return [np.array(f, dtype=np.float64, order="C", copy=True) for f in fields]   # never aliased


def divb(f, bc=P):
    """discrete div B in grid units (SURVEY.md pin P2); last cell of an outflow axis excluded by caller"""
    sp = lambda a, ax: inputs._shift_plus(a, ax, bc)
    return (sp(f[5], 2) - f[5]) + (sp(f[6], 1) - f[6]) + (sp(f[7], 0) - f[7])


def ksum(a):
    return math.fsum(a.ravel().tolist())


# ---------------------------------------------------------------------------------------------
# P1 / P2: conservation and div B
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("case", ["ot64", "turb3d"])
def test_conservation_and_divb_periodic(case):
    if case == "ot64":
        f, meta = inputs.orszag_tang(64)
        nsteps = 30
    else:
        f, meta = inputs.turbulence(24, 20, 16)
        nsteps = 6
    f = c64(f)
    assert np.abs(divb(f)).max() <= 1e-13 * max(np.abs(f[5]).max(), np.abs(f[6]).max(), np.abs(f[7]).max()) * 64
    s0 = [ksum(a) for a in f]
    a0 = [ksum(np.abs(a)) for a in f]
    oracle.run(f, meta["gamma"], meta["bc"], 0, nsteps, 0.8)
    s1 = [ksum(a) for a in f]
    for name, x0, x1, sc in zip(inputs.FIELD_NAMES, s0, s1, a0):
        if sc > 0:
            assert abs(x1 - x0) <= 1e-13 * sc, (name, x0, x1)
        else:
            assert x1 == 0.0, name
    bmax = max(np.abs(f[5]).max(), np.abs(f[6]).max(), np.abs(f[7]).max())
    assert np.abs(divb(f)).max() <= 1e-12 * bmax
    assert f[0].min() > 0


def test_divb_outflow_interior():
    f, meta = inputs.turbulence(16, 12, 10)
    f = c64(f)
    oracle.run(f, meta["gamma"], O, 0, 4, 0.8)
    dv = divb(f, O)[:-1, :-1, :-1]      # the +face of the last cell is the clamped copy (reading R9)
    assert np.abs(dv).max() <= 1e-12 * np.abs(f[5]).max()


# ---------------------------------------------------------------------------------------------
# P3: linear MHD eigenmodes along x -- closed-form solution, second-order convergence
# ---------------------------------------------------------------------------------------------
V0 = 0.3   # background flow along x: keeps v_x away from 0, where |v_x| in the freezing speed
           # puts a kink into the right/left-going split and the measured order of
           # compressive modes drops to ~1.5 ("What the pins found")


def _eigenmode(kind, n, eps, phase_shift=0.0):
    """Right-going plane-wave eigenmode of linearised ideal MHD about rho=1, p=1, B=(1,1,0.5), v=(V0,0,0).

    Linearising eqs (1)-(4) PAPER.md:51-62 for f(x - c t):  dvx = c e, dp = gamma p e, drho = rho e,
    dB_perp = B_perp c^2 e / (c^2 - ca^2), dv_perp = -bx dB_perp / (rho c); c solves
    (c^2 - a^2)(c^2 - ca^2) = c^2 ct^2 (fast/slow); Alfven: c = ca, dB_perp orthogonal to B_perp.
    Returns (fields for the given phase shift, pattern speed V0 + c, gamma).
    """
    gamma = 5.0 / 3.0
    rho0, p0, bx, by, bz = 1.0, 1.0, 1.0, 1.0, 0.5
    a2, ca2, ct2 = gamma * p0 / rho0, bx * bx / rho0, (by * by + bz * bz) / rho0
    s = a2 + ca2 + ct2
    disc = math.sqrt(s * s - 4 * a2 * ca2)
    xc = np.arange(n) + 0.5
    e = eps * np.sin(2 * math.pi * (xc - phase_shift) / n)
    if kind == "alfven":
        c = math.sqrt(ca2)
        nb = math.hypot(by, bz)
        dby, dbz = e * (-bz / nb), e * (by / nb)
        drho, dvx, dp = 0 * e, V0 + 0 * e, 0 * e
    else:
        c2 = 0.5 * (s + disc) if kind == "fast" else 0.5 * (s - disc)
        c = math.sqrt(c2)
        drho, dvx, dp = rho0 * e, V0 + c * e, gamma * p0 * e
        dby, dbz = by * c2 * e / (c2 - ca2), bz * c2 * e / (c2 - ca2)
    dvy, dvz = -bx * dby / (rho0 * c), -bx * dbz / (rho0 * c)
    shape = (1, 1, n)
    rho = (rho0 + drho).reshape(shape)
    vx, vy, vz = dvx.reshape(shape), dvy.reshape(shape), dvz.reshape(shape)
    p = (p0 + dp).reshape(shape)
    Bx = np.full(shape, bx)
    By, Bz = (by + dby).reshape(shape), (bz + dbz).reshape(shape)   # transverse faces sit at the x centre
    E = inputs.total_energy(rho, vx, vy, vz, p, Bx, By, Bz, gamma, P)
    return c64([rho, rho * vx, rho * vy, rho * vz, E, Bx, By, Bz]), V0 + c, gamma


@pytest.mark.parametrize("kind", ["alfven", "fast", "slow"])
def test_eigenmode_second_order_convergence(kind):
    eps = 1e-6
    errs = []
    sizes = [32, 64, 128, 256]
    for n in sizes:
        f, c, gamma = _eigenmode(kind, n, eps)
        cm = oracle.cmax(f, gamma, P)
        t_end = n / c                                  # one period in grid units
        nsteps = math.ceil(t_end / (2 * 0.8 / cm))
        dt = t_end / (2 * nsteps)
        for s in range(nsteps):
            oracle.step_fixed(f, gamma, P, s, dt)
        ref, _, _ = _eigenmode(kind, n, eps, phase_shift=c * t_end)
        err = sum(np.abs(a - b).mean() for a, b in zip(f, ref)) / eps
        errs.append(err)
    orders = [math.log2(errs[i] / errs[i + 1]) for i in range(len(errs) - 1)]
    # a dropped or mis-signed flux term gives a wrong wave speed: O(1) error and no convergence
    assert errs[-1] < 8e-3, (errs, orders)
    assert all(o > 1.7 for o in orders), (errs, orders)
    assert orders[-1] > 1.9, (errs, orders)


def test_eigenmode_travels_at_wave_speed_not_half_period():
    """After HALF a period the fast mode must match the half-shifted profile and NOT the initial one."""
    n, eps = 128, 1e-6
    f, c, gamma = _eigenmode("fast", n, eps)
    cm = oracle.cmax(f, gamma, P)
    t_end = 0.5 * n / c
    nsteps = math.ceil(t_end / (2 * 0.8 / cm))
    for s in range(nsteps):
        oracle.step_fixed(f, gamma, P, s, t_end / (2 * nsteps))
    moved, _, _ = _eigenmode("fast", n, eps, phase_shift=c * t_end)
    still, _, _ = _eigenmode("fast", n, eps)
    e_moved = sum(np.abs(a - b).mean() for a, b in zip(f, moved)) / eps
    e_still = sum(np.abs(a - b).mean() for a, b in zip(f, still)) / eps
    assert e_moved < 0.03 and e_still > 1.0, (e_moved, e_still)


# ---------------------------------------------------------------------------------------------
# B = 0: exact Riemann solution of the Euler equations (Sod tube), textbook closed form
# ---------------------------------------------------------------------------------------------
def _sod_exact(x, t, gamma=1.4, left=(1.0, 0.0, 1.0), right=(0.125, 0.0, 0.1), x0=0.5):
    rl, ul, pl = left
    rr, ur, pr = right
    g = gamma
    al, ar = math.sqrt(g * pl / rl), math.sqrt(g * pr / rr)

    def fk(p, rk, pk, ak):
        if p > pk:   # shock
            A, B = 2 / ((g + 1) * rk), (g - 1) / (g + 1) * pk
            return (p - pk) * math.sqrt(A / (p + B))
        return 2 * ak / (g - 1) * ((p / pk) ** ((g - 1) / (2 * g)) - 1)

    lo, hi = 1e-8, 10.0
    for _ in range(200):   # bisection on f(p) = fL + fR + (uR - uL)
        mid = 0.5 * (lo + hi)
        if fk(mid, rl, pl, al) + fk(mid, rr, pr, ar) + (ur - ul) > 0:
            hi = mid
        else:
            lo = mid
    ps = 0.5 * (lo + hi)
    us = 0.5 * (ul + ur) + 0.5 * (fk(ps, rr, pr, ar) - fk(ps, rl, pl, al))
    # left rarefaction, right shock (Sod)
    rsl = rl * (ps / pl) ** (1 / g)
    asl = al * (ps / pl) ** ((g - 1) / (2 * g))
    rsr = rr * ((ps / pr + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * ps / pr + 1))
    S = ur + ar * math.sqrt((g + 1) / (2 * g) * ps / pr + (g - 1) / (2 * g))
    xi = (x - x0) / t
    rho = np.empty_like(x)
    head, tail = ul - al, us - asl
    for i, s in enumerate(xi):
        if s < head:
            rho[i] = rl
        elif s < tail:
            rho[i] = rl * (2 / (g + 1) + (g - 1) / ((g + 1) * al) * (ul - s)) ** (2 / (g - 1))
        elif s < us:
            rho[i] = rsl
        elif s < S:
            rho[i] = rsr
        else:
            rho[i] = rr
    return rho


def test_sod_tube_against_exact_riemann_solution():
    gamma, t_phys = 1.4, 0.2
    errs = []
    for n in (100, 200, 400):
        x = (np.arange(n) + 0.5) / n
        shape = (1, 1, n)
        rho = np.where(x < 0.5, 1.0, 0.125).reshape(shape)
        p = np.where(x < 0.5, 1.0, 0.1).reshape(shape)
        z = np.zeros(shape)
        f = c64([rho, z, z, z, p / (gamma - 1), z, z, z])
        t, s = 0.0, 0
        t_end = t_phys * n
        while t < t_end - 1e-12:
            dt = min(0.8 / oracle.cmax(f, gamma, O), 0.5 * (t_end - t))
            oracle.step_fixed(f, gamma, O, s, dt)
            t += 2 * dt
            s += 1
        for b in f[5:]:
            assert not b.any()                       # B stays bitwise zero (pin P9)
        exact = _sod_exact(x, t_phys, gamma)
        errs.append(np.abs(f[0].ravel() - exact).mean())
    assert errs[0] < 1.2e-2 and errs[2] < 4e-3, errs
    assert errs[1] < 0.75 * errs[0] and errs[2] < 0.75 * errs[1], errs     # converging (first order at shocks)


# ---------------------------------------------------------------------------------------------
# P4: Orszag-Tang 180-degree rotation symmetry
# ---------------------------------------------------------------------------------------------
def test_orszag_tang_rotation_symmetry():
    n = 64
    f, meta = inputs.orszag_tang(n)
    f = c64(f)
    oracle.run(f, meta["gamma"], meta["bc"], 0, 30, 0.8)
    rot = lambda a: a[:, ::-1, ::-1]
    scale = np.abs(f[4]).max()
    assert np.abs(rot(f[0]) - f[0]).max() <= 1e-10 * scale
    assert np.abs(rot(f[4]) - f[4]).max() <= 1e-10 * scale
    assert np.abs(rot(f[1]) + f[1]).max() <= 1e-10 * scale
    assert np.abs(rot(f[2]) + f[2]).max() <= 1e-10 * scale
    # faces: Bx[i,j] at (i-1/2, j) maps to ((n-i) mod n, n-1-j)
    bx, by = f[5][0], f[6][0]
    i = np.arange(n)
    bxr = bx[np.ix_(n - 1 - i, (n - i) % n)]          # [j', i'] = [n-1-j, (n-i)%n]
    byr = by[np.ix_((n - i) % n, n - 1 - i)]
    assert np.abs(bxr + bx).max() <= 1e-10
    assert np.abs(byr + by).max() <= 1e-10
    assert np.abs(bx).max() > 0.1


# ---------------------------------------------------------------------------------------------
# P5 / P6 / P7: exact special cases
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", [P, O])
def test_uniform_state_is_a_bitwise_fixed_point(bc):
    shape = (5, 6, 7)
    vals = [1.3, 0.4, -0.7, 0.2, 3.1, 0.6, -0.3, 0.9]
    f = [np.full(shape, v) for v in vals]
    g = [a.copy() for a in f]
    for s in range(3):
        oracle.step_fixed(g, 5.0 / 3.0, bc, s, 0.37)
    for a, b in zip(f, g):
        assert np.array_equal(a, b)


def test_1d_data_replicated_in_3d_is_bitwise_1d():
    f1, meta = inputs.brio_wu(64)
    f1 = c64(f1)
    f3 = c64([np.broadcast_to(a, (4, 4, 64)) for a in f1])
    for s in range(4):
        oracle.step_fixed(f1, meta["gamma"], meta["bc"], s, 0.2)
        oracle.step_fixed(f3, meta["gamma"], meta["bc"], s, 0.2)
    for a, b in zip(f1, f3):
        assert np.array_equal(np.broadcast_to(a, b.shape), b)


def _cyclic(f):
    """x->y->z->x: new field(y=a, z=b, x=c) = old field(x=a, y=b, z=c); vector components follow."""
    tr = lambda a: np.ascontiguousarray(a.transpose(1, 2, 0))    # new[z,y,x] = old[k=y', ...]
    # old array index order (z,y,x); new axes: new_x = old_z, new_y = old_x, new_z = old_y
    # new[z',y',x'] = old[z=x', y=z', x=y']  -> transpose(1,2,0) of old gives axes (y,x,z) -> indices [z'=y, y'=x, x'=z]
    rho, mx, my, mz, E, bx, by, bz = f
    return [tr(rho), tr(mz), tr(mx), tr(my), tr(E), tr(bz), tr(bx), tr(by)]


@pytest.mark.parametrize("bc", [P, O])
def test_cyclic_permutation_equivariance_bitwise(bc):
    f, meta = inputs.turbulence(12, 10, 8)
    f = c64(f)
    g = _cyclic(f)                      # axes rotated: old x-direction is the new y-direction
    for s in range(3):
        oracle.step_fixed(f, meta["gamma"], bc, s, 0.11)
        # old order (x,y,z) at s=0 is (y,z,x) in the new frame = the table row for s+2
        oracle.step_fixed(g, meta["gamma"], bc, s + 2, 0.11)
    for a, b in zip(_cyclic(f), g):
        assert np.array_equal(a, b)


def test_thread_count_does_not_change_bits():
    f, meta = inputs.turbulence(16, 12, 10)
    a, b = c64(f), c64(f)
    n0 = oracle.num_threads()
    try:
        oracle.set_num_threads(1)
        oracle.run(a, meta["gamma"], meta["bc"], 0, 2, 0.8)
        oracle.set_num_threads(max(2, n0))
        oracle.run(b, meta["gamma"], meta["bc"], 0, 2, 0.8)
    finally:
        oracle.set_num_threads(n0)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)


# ---------------------------------------------------------------------------------------------
# P8: Brio-Wu invariants and qualitative wave structure
# ---------------------------------------------------------------------------------------------
def _run_to(f, meta, t_end_grid, cfl=0.8):
    t, s = 0.0, 0
    while t < t_end_grid - 1e-12:
        dt = min(cfl / oracle.cmax(f, meta["gamma"], meta["bc"]), 0.5 * (t_end_grid - t))
        oracle.step_fixed(f, meta["gamma"], meta["bc"], s, dt)
        t += 2 * dt
        s += 1
    return s


def test_brio_wu_invariants_and_structure():
    n = 512
    f, meta = inputs.brio_wu(n)
    f = c64(f)
    nsteps = _run_to(f, meta, 0.1 * n)
    assert 100 < nsteps < 200
    rho, mx, my, mz, E, bx, by, bz = [a.ravel() for a in f]
    assert np.all(bx == 0.75) and not mz.any() and not bz.any()
    b2 = bx ** 2 + (0.5 * (by + by)) ** 2
    p = (meta["gamma"] - 1) * (E - 0.5 * (mx ** 2 + my ** 2) / rho - 0.5 * b2)
    assert rho.min() > 0 and p.min() > 0
    # undisturbed end states
    assert abs(rho[5] - 1.0) < 1e-12 and abs(rho[-5] - 0.125) < 1e-12
    assert abs(by[5] - 1.0) < 1e-12 and abs(by[-5] + 1.0) < 1e-12
    # By goes from +1 to -1; fluid is pushed to the right in the middle (vx > 0), v_y < 0
    assert by[n // 4] > 0 > by[3 * n // 4]
    assert (mx / rho).max() > 0.5 and (my / rho).min() < -1.0
    # density: left rarefaction fan (monotone decreasing), and somewhere a dip below the right state
    # (right-going fast rarefaction), and an intermediate plateau between 0.6 and 0.75
    x = (np.arange(n) + 0.5) / n
    fan = rho[(x > 0.33) & (x < 0.42)]
    assert np.all(np.diff(fan) < 0)
    assert rho.min() < 0.125 - 1e-3
    plateau = rho[(x > 0.50) & (x < 0.54)]
    assert 0.6 < plateau.mean() < 0.75


# ---------------------------------------------------------------------------------------------
# P10: the scalar B advection scheme with constant velocity on linear data is exact
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("d,t", [(0, 1), (0, 2), (1, 2), (1, 0), (2, 0), (2, 1)])
@pytest.mark.parametrize("v", [0.7, -0.45])
def test_badvect_constant_velocity_linear_data_exact(d, t, v):
    n = [9, 10, 11]
    shape = (n[2], n[1], n[0])
    slope, dt = 0.25, 0.6
    idx = np.arange(n[d], dtype=np.float64)
    bshape = [1, 1, 1]
    bshape[2 - d] = n[d]
    lin = np.broadcast_to((slope * idx).reshape(bshape), shape)
    f = [np.ones(shape), np.zeros(shape), np.zeros(shape), np.zeros(shape), np.full(shape, 10.0),
         np.zeros(shape), np.zeros(shape), np.zeros(shape)]
    f[1 + d] = np.full(shape, v)
    f[5 + t] = lin.copy()
    f[5 + d] = np.full(shape, 0.3)
    f = c64(f)
    oracle.badvect(f, 5.0 / 3.0, P, d, t, dt)
    sl = [slice(None)] * 3
    sl[2 - d] = slice(3, n[d] - 3)          # away from the wrap-around jump of the linear profile
    got = f[5 + t][tuple(sl)]
    want = (lin - v * dt * slope)[tuple(sl)]
    assert np.abs(got - want).max() < 1e-14
    assert np.abs(f[5 + d][tuple(sl)] - 0.3).max() < 1e-15     # same flux on every row: no constraint change
    s = 3 - d - t
    assert np.array_equal(f[5 + s], np.zeros(shape))


# ---------------------------------------------------------------------------------------------
# P10b: along an axis of extent 1 Algorithm 2 collapses (reading R10): B_t comes back bit for bit and B_d changes by the
# difference of the first-order edge fluxes f = (vt B_t) dt of the rows tau+1 and tau.  Hand-derivable from
# eqs (20)-(22): every index along d maps to the only cell, so vg = vt, both upwind candidates coincide and the limited
# differences vanish.  (The CUDA path has a closed-form kernel for this case; this pins the oracle's side of it.)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", [P, O])
@pytest.mark.parametrize("d", [0, 1, 2])
def test_badvect_along_an_extent_one_axis_is_the_constraint_term_alone(d, bc):
    rng = np.random.default_rng(5 + d)
    n = [6, 5, 7]
    n[d] = 1
    shape = (n[2], n[1], n[0])
    f = c64([1.0 + 0.3 * rng.random(shape)] + [rng.standard_normal(shape) * 0.4 for _ in range(3)] + [10.0 + rng.random(shape)] +
            [rng.standard_normal(shape) * 0.5 for _ in range(3)])
    dt = 0.37
    for t in ((d + 1) % 3, (d + 2) % 3):
        g = [a.copy() for a in f]
        oracle.badvect(g, 5.0 / 3.0, bc, d, t, dt)
        ax = 2 - t                                           # numpy axis of direction t
        def shift(a, k):                                     # a[tau + k] with the boundary rule
            if bc == P:
                return np.roll(a, -k, axis=ax)
            idx = np.clip(np.arange(a.shape[ax]) + k, 0, a.shape[ax] - 1)
            return np.take(a, idx, axis=ax)
        rho, md, bt = f[0], f[1 + d], f[5 + t]
        flux = lambda k: (((shift(md, k - 1) + shift(md, k)) / (shift(rho, k - 1) + shift(rho, k))) * shift(bt, k)) * dt
        # row tau+1 uses the MAPPED cells tau and tau+1 (at a clamped last row both are the last cell)
        f_here = flux(0)
        if bc == P:
            f_next = flux(1)
        else:
            f_next = (((md + shift(md, 1)) / (rho + shift(rho, 1))) * shift(bt, 1)) * dt
        assert np.array_equal(g[5 + t], f[5 + t])            # advected into itself, bit for bit
        want = f[5 + d] + (f_next - f_here)
        assert np.abs(g[5 + d] - want).max() <= 4e-16 * max(1.0, np.abs(want).max())
        for k in range(5):
            assert np.array_equal(g[k], f[k])


# ---------------------------------------------------------------------------------------------
# P11: brute force on tiny grids against the independently structured NumPy restatement
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape", [(4, 1, 1), (1, 5, 1), (1, 1, 4), (4, 4, 1), (4, 3, 2), (7, 5, 6), (2, 2, 2)])
@pytest.mark.parametrize("bc", [P, O])
def test_tiny_grids_against_numpy_restatement(shape, bc):
    nx, ny, nz = shape
    rng = np.random.default_rng(nx * 100 + ny * 10 + nz + bc)
    sh = (nz, ny, nx)
    rho = 1.0 + 0.3 * rng.random(sh)
    v = [0.5 * rng.standard_normal(sh) for _ in range(3)]
    B = [0.5 * rng.standard_normal(sh) for _ in range(3)]
    E = 2.5 + rng.random(sh) + 0.5 * rho * sum(x * x for x in v) + sum(x * x for x in B)
    f0 = c64([rho, rho * v[0], rho * v[1], rho * v[2], E] + B)
    gamma, dt = 5.0 / 3.0, 0.13
    assert abs(oracle.cmax(f0, gamma, bc) - npr.cmax(f0, gamma, bc)) < 1e-14
    for d in range(3):
        a = [x.copy() for x in f0]
        oracle.fluid(a, gamma, bc, d, dt)
        b = npr.fluid(f0, gamma, bc, d, dt)
        for x, y in zip(a, b):
            assert np.abs(x - y).max() < 1e-13
        for t in range(3):
            if t == d:
                continue
            a = [x.copy() for x in f0]
            oracle.badvect(a, gamma, bc, d, t, dt)
            b = npr.badvect(f0, gamma, bc, d, t, dt)
            for x, y in zip(a, b):
                assert np.abs(x - y).max() < 1e-13
    for s in range(3):
        a = [x.copy() for x in f0]
        oracle.step_fixed(a, gamma, bc, s, dt)
        b = npr.step(f0, gamma, bc, s, dt)
        for x, y in zip(a, b):
            assert np.abs(x - y).max() < 1e-12


# ---------------------------------------------------------------------------------------------
# P12: fp32 instantiation sanity (same magnitudes as PAPER.md:567-583)
# ---------------------------------------------------------------------------------------------
def test_fp32_oracle_tracks_fp64_oracle():
    f, meta = inputs.brio_wu(512)
    a = inputs.to_precision(f, np.float64)
    b = inputs.to_precision(f, np.float32)
    for s in range(40):
        dt = 0.8 / oracle.cmax(a, meta["gamma"], meta["bc"])
        oracle.step_fixed(a, meta["gamma"], meta["bc"], s, dt)
        oracle.step_fixed(b, meta["gamma"], meta["bc"], s, dt)
    for x, y in zip(a, b):
        assert np.abs(x - y).max() < 2e-5      # paper: <= 1e-6-ish for Brio-Wu at t = 0.08


def test_cmax_surfaces_nan():
    f, meta = inputs.turbulence(8, 8, 8)
    f = c64(f)
    f[0][3, 3, 3] = np.nan
    assert math.isnan(oracle.cmax(f, meta["gamma"], meta["bc"]))


# ---------------------------------------------------------------------------------------------
# c_max of eq (18), against hand-computed values.  Every state below is built from numbers
# chosen so that the expected c is a short decimal worked out on paper (the arithmetic is written in the
# comments, the expected values are literals): c = max(|vx|,|vy|,|vz|) + sqrt(|gamma p + B^2| / rho) with B the
# cell-centred average of the two faces (reading R4) and p = (gamma-1)(E - rho v^2/2 - B^2/2).
# ---------------------------------------------------------------------------------------------
def _const_state(shape, rho, v, E, B):
    nz, ny, nx = shape
    full = lambda x: np.full((nz, ny, nx), float(x))
    return [full(rho), full(rho * v[0]), full(rho * v[1]), full(rho * v[2]), full(E), full(B[0]), full(B[1]), full(B[2])]


@pytest.mark.parametrize("bc", [P, O])
@pytest.mark.parametrize("perm", [(0, 1, 2), (1, 2, 0), (2, 0, 1)])
def test_cmax_uniform_state_hand_computed(bc, perm):
    # rho = 4, gamma = 5/3, v = (0.3, -0.7, 0.2) (permuted), B = (1, 2, 2) (permuted): B^2 = 9, v^2 = 0.62.
    # p = 4.2  ->  gamma p = 7,  gamma p + B^2 = 16,  /rho = 4,  sqrt = 2;  max|v| = 0.7  ->  c = 2.7
    # E = p/(gamma-1) + rho v^2/2 + B^2/2 = 6.3 + 1.24 + 4.5 = 12.04
    v0, B0 = (0.3, -0.7, 0.2), (1.0, 2.0, 2.0)
    v = [v0[perm[i]] for i in range(3)]
    B = [B0[perm[i]] for i in range(3)]
    f = _const_state((3, 4, 5), 4.0, v, 12.04, B)
    assert abs(oracle.cmax(f, 5.0 / 3.0, bc) - 2.7) < 1e-14
    # the largest |v| must come from whichever component holds it: dropping a component from the max would give
    # 0.3 + 2 = 2.3 for one of the three permutations


@pytest.mark.parametrize("comp", [1, 2, 3])
def test_cmax_picks_the_one_cell_and_the_one_velocity_component(comp):
    # background at rest: rho = 1, gamma = 2, B = 0, E = 2  ->  p = 2, c = sqrt(4) = 2.
    # one cell moves with v = -3 along `comp` only: E = 2 + rho v^2/2 = 6.5 keeps p = 2  ->  c = 3 + 2 = 5
    f = _const_state((4, 3, 6), 1.0, (0, 0, 0), 2.0, (0, 0, 0))
    assert abs(oracle.cmax(f, 2.0, P) - 2.0) < 1e-15
    f[comp][2, 1, 4] = -3.0
    f[4][2, 1, 4] = 6.5
    assert abs(oracle.cmax(f, 2.0, P) - 5.0) < 1e-15
    assert abs(oracle.cmax(f, 2.0, O) - 5.0) < 1e-15


def test_cmax_uses_the_cell_centred_average_of_the_two_faces():
    # gamma = 3, rho = 1, v = 0:  c^2 = 3 p + B^2 = 3 * 2 (E - B^2/2) + B^2 = 6 E - 2 B^2  (gamma = 2 would hide B in c).
    # E = 3; the component along the axis alternates 2, 0 from face to face, so every cell-centred value is 1:
    #   centre (B = 1): c^2 = 18 - 2 = 16, c = 4.   A face value instead of the average gives B = 2: c^2 = 10, or B = 0: 18.
    pattern = [2, 0, 2, 0, 2, 0, 2, 0]
    for axis in range(3):                       # Bx on x-faces, By on y-faces, Bz on z-faces
        shape = [1, 1, 1]
        shape[2 - axis] = 8
        f = _const_state(tuple(shape), 1.0, (0, 0, 0), 3.0, (0, 0, 0))
        f[5 + axis].ravel()[:] = pattern
        assert abs(oracle.cmax(f, 3.0, P) - 4.0) < 1e-15
    # By varies along y only; averaging it along x instead (a transposed operand) would see equal neighbours,
    # B = 2 or 0, and return sqrt 18
    k = _const_state((1, 8, 2), 1.0, (0, 0, 0), 3.0, (0, 0, 0))
    k[6][0, :, :] = np.array(pattern)[:, None]
    assert abs(oracle.cmax(k, 3.0, P) - 4.0) < 1e-15


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_cmax_last_cell_follows_the_boundary_rule(axis):
    # gamma = 3, rho = 1, v = 0, E = 9:  c^2 = 6 E - 2 B_c^2 = 54 - 2 B_c^2  (see the test above).
    # Faces along `axis`: B = 5, 4, 3, 1.  Centres of cells 0..2: 4.5, 3.5, 2  ->  c^2 = 13.5, 29.5, 46.
    # Last cell (reading R9): periodic wraps to face 0: (1 + 5)/2 = 3 -> c^2 = 36, so the maximum is 46 (cell 2);
    #                         outflow clamps to its own face: (1 + 1)/2 = 1 -> c^2 = 52, the maximum.
    shape = [1, 1, 1]
    shape[2 - axis] = 4
    f = _const_state(tuple(shape), 1.0, (0, 0, 0), 9.0, (0, 0, 0))
    f[5 + axis].ravel()[:] = [5, 4, 3, 1]
    assert abs(oracle.cmax(f, 3.0, P) - math.sqrt(46.0)) < 1e-14
    assert abs(oracle.cmax(f, 3.0, O) - math.sqrt(52.0)) < 1e-14


def test_cmax_negative_pressure_takes_the_absolute_value():
    # reading R3: c = |v| + sqrt(|gamma p + B^2| / rho).  rho = 2, gamma = 2, v = 0, B = 0, E = -4: p = -4,
    # gamma p + B^2 = -8, |.|/rho = 4, c = 2 (never NaN for rho > 0)
    f = _const_state((2, 2, 2), 2.0, (0, 0, 0), -4.0, (0, 0, 0))
    assert abs(oracle.cmax(f, 2.0, P) - 2.0) < 1e-15


def test_oracle_regression_fixture():
    """tests/golden/oracle_tiny_state.txt (written by tests/golden/make_golden.py from the oracle alone) is reproduced
    bit for bit: the oracle's arithmetic has not changed unnoticed"""
    import os
    from tests.golden import make_golden
    want = {}
    with open(os.path.join(os.path.dirname(make_golden.__file__), "oracle_tiny_state.txt")) as fh:
        for line in fh:
            if line.startswith("#"):
                continue
            tok = line.split()
            want[(int(tok[0]), int(tok[1]))] = np.array([float.fromhex(t) for t in tok[2:]])
    assert len(want) == 16
    for bc in (0, 1):
        for i, a in enumerate(make_golden.tiny_state(bc)):
            assert np.array_equal(a.ravel(), want[(bc, i)]), (bc, i)


def test_second_workload_set_generators():
    """initial data of the paper's E4 / E6: uniform B (div B = 0
    exactly), v = 0, p jump 10 / 0.1 at r = 0.1, and the oracle keeps the 2-D run 2-D"""
    from paper_0908_4362_b200 import inputs
    f, meta = inputs.blast2d(64)
    g = meta["gamma"]
    p = (g - 1.0) * (f[4] - 0.5 * (f[5] ** 2 + f[6] ** 2 + f[7] ** 2))
    assert abs(p.max() - 10.0) < 1e-12 and abs(p.min() - 0.1) < 1e-12
    assert abs((p > 1).mean() - np.pi * 0.01) < 2e-3            # disc of radius 0.1 in the unit square
    assert np.all(f[5] == f[5].flat[0]) and np.all(f[6] == f[5].flat[0]) and not f[7].any()
    st = [a.copy() for a in f]
    oracle.step_fixed(st, g, meta["bc"], 0, 0.05)
    assert not st[3].any() and not st[7].any() and np.abs(st[0] - 1).max() > 1e-3
    f3, m3 = inputs.blast3d(24, paper_field=True)
    assert np.allclose(f3[5] ** 2 + f3[6] ** 2 + f3[7] ** 2, 1.0)
    p3 = (m3["gamma"] - 1.0) * (f3[4] - 0.5)
    assert abs(p3.max() - 10.0) < 1e-12 and abs(p3.min() - 0.1) < 1e-12


# ---- visualisation stage (oracle/viz.py; include/mhd.h is the definition, the paper prints none) --------------------
def _viz_fields(shape, seed):
    from tests.parity_utils import random_state
    return random_state(*shape, seed=seed)


def test_viz_value_pressure_recovers_the_pressure_the_state_was_built_from():
    from oracle import viz
    from paper_0908_4362_b200 import inputs
    f, meta = inputs.blast2d(64)
    p = viz.value(f, viz.PRESSURE, meta["gamma"], meta["bc"])
    assert abs(float(p.max()) - 10.0) < 1e-5 and abs(float(p.min()) - 0.1) < 1e-5
    f3, m3 = inputs.turbulence(16, 12, 8)                    # p = 1 everywhere by construction
    p3 = viz.value(f3, viz.PRESSURE, m3["gamma"], m3["bc"])
    assert np.abs(p3 - 1.0).max() < 2e-5
    assert viz.value(f3, 0, m3["gamma"], m3["bc"]).dtype == np.float32


def test_viz_unit_byte_and_curve_closed_forms():
    from oracle import viz
    v = np.array([-1.0, 0.0, 0.25, 0.5, 1.0, 7.0, np.nan], dtype=np.float32)
    t = viz.unit(v, 0.0, 1.0)
    assert list(t) == [0.0, 0.0, 0.25, 0.5, 1.0, 1.0, 0.0]
    assert list(viz.byte(t)) == [0, 0, 64, 128, 255, 255, 0]          # trunc(t*255 + 0.5)
    nx = 8
    f = [np.zeros((1, 1, nx)) for _ in range(8)]
    f[0][0, 0, :] = np.linspace(2.0, 4.0, nx)
    xy = viz.curve(f, 0, 1.4, 0, 0, 0, 2.0, 4.0)
    assert xy.shape == (nx, 2)
    assert np.allclose(xy[:, 0], -1 + (2 * np.arange(nx) + 1) / nx, atol=1e-7)      # cell centres of [-1, 1]
    assert np.allclose(xy[:, 1], np.linspace(-1.0, 1.0, nx), atol=1e-6)
    assert viz.value_range(f, 0, 1.4, 0) == (2.0, 4.0)


def test_viz_slice_is_a_table_lookup_and_volume_follows_the_compositing_closed_form():
    from oracle import viz
    lut = np.zeros((256, 4), dtype=np.uint8)
    lut[:, 0] = np.arange(256)
    lut[:, 1] = 255 - np.arange(256)
    lut[:, 2] = 7
    lut[:, 3] = 51                                                        # a = 0.2 per sample
    f = _viz_fields((12, 9, 30), 4)
    g = 5.0 / 3.0
    lo, hi = viz.value_range(f, 0, g, 0)
    img = viz.slice_rgba(f, 0, g, 0, 3, lo, hi, lut)
    t = (np.asarray(f[0][3], np.float64) - lo) / (hi - lo)
    assert img.shape == (9, 12, 4) and img.dtype == np.uint8
    assert np.abs(img[..., 0].astype(int) - np.rint(t * 255)).max() <= 1     # red channel = byte(t), up to fp32 rounding
    assert np.all(img[..., 0].astype(int) + img[..., 1] == 255) and np.all(img[..., 2] == 7)
    assert img[..., 0].max() == 255 and img[..., 0].min() == 0
    # volume: constant colour and opacity a per sample -> A_n = 1 - (1-a)^n, C = A * colour, cut at the first A >= 0.99
    const = [np.ones((30, 9, 12)) for _ in range(8)]
    lut2 = np.zeros((256, 4), dtype=np.uint8)
    lut2[:] = (255, 128, 0, 51)
    out = viz.volume_rgba(const, 0, g, 0, 0.0, 2.0, lut2, 1.0)
    n_stop = int(np.ceil(np.log(0.01) / np.log(0.8)))                      # 21 samples reach A >= 0.99
    A = 1 - 0.8 ** n_stop
    assert n_stop == 21 and np.all(out[..., 3] == int(A * 255 + 0.5))
    assert np.all(out[..., 0] == int(A * 255 + 0.5)) and np.all(out[..., 2] == 0)
    assert np.all(np.abs(out[..., 1].astype(int) - int(A * 128 / 255 * 255 + 0.5)) <= 1)
    out_thin = viz.volume_rgba(const, 0, g, 0, 0.0, 2.0, lut2, 0.01)       # never terminates early: all 30 samples
    a = 51 / 255 * 0.01
    assert np.all(np.abs(out_thin[..., 3].astype(int) - int((1 - (1 - a) ** 30) * 255 + 0.5)) <= 1)
    # opaque first sample hides everything behind it
    lut3 = lut.copy(); lut3[:, 3] = 255
    front = viz.volume_rgba(f, 0, g, 0, lo, hi, lut3, 1.0)
    assert np.array_equal(front[..., :3], viz.slice_rgba(f, 0, g, 0, 0, lo, hi, lut3)[..., :3]) and np.all(front[..., 3] == 255)


# ---------------------------------------------------------------------------------------------------------------
# The one discontinuous decision of the scheme: the upwind switch of eq (21), PAPER.md:152 --
#     (v B)_{i+1/2} = (v B)_i  if  v_{i+1/2} > 0,     (v B)_{i+1}  if  v_{i+1/2} <= 0
# so at an EXACT tie v_{i+1/2} = 0 the flux comes from cell i+1.  Random data never hit the tie; mirror-symmetric data
# (the blast waves c3, E4, E6) do.  Worked example, every number dyadic until the one limiter quotient:
#   16 cells along d, periodic, rho = 1, B_t = 1, dt = 1/2, velocity along d
#     v  = 0 0 0 0 | 1 1 1 1 | -1 -1 -1 -1 | 0 0 0 0          (cells 0..15: a converging flow)
#   eq (20)  vg_p = (v_{p-1} + 2 v_p + v_{p+1}) / 4:
#     vg = 0 0 0 1/4 3/4 1 1 1/2 | -1/2 -1 -1 -3/4 -1/4 0 0 0   (cells 0..15)
#   eq (22)  v_{7+1/2} = (vg_7 + vg_8)/2 = (1/2 - 1/2)/2 = 0 exactly, with vg_7 = -vg_8 != 0: THE TIE.
#   eq (21), first-order fluxes f1 = vg B at faces 6.5, 7.5, 8.5:  1 (from cell 6),  vg_8 B_8 = -1/2 (tie: from cell 8,
#     the "<= 0" arm; the "> 0" arm would give vg_7 B_7 = +1/2),  -1 (from cell 9)
#   eq (16) half step  B' = B - (f1_{p+1/2} - f1_{p-1/2}) dt/2:   B'_6 = 1, B'_7 = 1 + 3/8 = 11/8, B'_8 = 1 + 1/8 = 9/8,
#     B'_9 = 1, B'_5 = B'_10 = 15/16
#   w = vg B':  w_5 = 15/16, w_6 = 1, w_7 = 11/16, w_8 = -9/16, w_9 = -1, w_10 = -15/16
#   second-order fluxes (eqs (11)-(15) with the van Leer limiter 2ab/(a+b), zero when a b <= 0):
#     face 6.5 (v > 0):  w_6 + vl((w_6 - w_5)/2, (w_7 - w_6)/2) = 1 + vl(1/32, -5/32) = 1
#     face 8.5 (v < 0):  w_9 + vl((w_9 - w_10)/2, (w_8 - w_9)/2) = -1 + vl(-1/32, 7/32) = -1
#     face 7.5 (tie, the arm of cell 8):  w_8 + vl((w_8 - w_9)/2, (w_7 - w_8)/2) = -9/16 + vl(7/32, 5/8)
#                                         = -9/16 + 2 (7/32)(5/8) / (27/32) = -9/16 + 35/108 = -103/432
#   eq (17)  B_7 = 1 - (-103/432 - 1)/2 = 1399/864,   B_8 = 1 - (-1 + 103/432)/2 = 1193/864.
# With the tie sent to cell 7 instead ("v >= 0") the mirror image comes out: B_7 = 1193/864, B_8 = 1399/864.
# ---------------------------------------------------------------------------------------------------------------
TIE_V = [0, 0, 0, 0, 1, 1, 1, 1, -1, -1, -1, -1, 0, 0, 0, 0]
TIE_B7, TIE_B8 = 1399.0 / 864.0, 1193.0 / 864.0


def tie_state(d, t, shape3, dtype=np.float64, offset=0):
    """the worked example laid along axis d (0 = x) of a grid of extents shape3 = (nx, ny, nz), uniform across the
    pencils, the 16 cells starting at `offset` along d (zeros around them)"""
    nx, ny, nz = shape3
    sh = (nz, ny, nx)
    nd = shape3[d]
    v = np.zeros(nd)
    v[offset:offset + 16] = TIE_V
    bshape = [1, 1, 1]
    bshape[2 - d] = nd
    f = [np.ones(sh)] + [np.zeros(sh) for _ in range(3)] + [np.full(sh, 4.0)] + [np.zeros(sh) for _ in range(3)]
    f[1 + d] = f[1 + d] + v.reshape(bshape)
    f[5 + t] = f[5 + t] + 1.0
    return [np.ascontiguousarray(a, dtype=dtype) for a in f]


@pytest.mark.parametrize("d,t", [(0, 1), (0, 2), (1, 2), (1, 0), (2, 0), (2, 1)])
@pytest.mark.parametrize("dtype,tol", [(np.float64, 1e-15), (np.float32, 3e-7)])
def test_upwind_tie_takes_the_cell_on_the_right(d, t, dtype, tol):
    shape3 = [1, 1, 1]
    shape3[d] = 16
    f = tie_state(d, t, shape3, dtype)
    oracle.badvect(f, 5.0 / 3.0, P, d, t, 0.5)
    b = f[5 + t].astype(np.float64).ravel()
    assert abs(b[7] - TIE_B7) <= tol * TIE_B7, (b[7], TIE_B7)
    assert abs(b[8] - TIE_B8) <= tol * TIE_B8, (b[8], TIE_B8)
    assert b[7] > b[8] + 0.2                                  # the asymmetry IS the rule: "<= 0" sends the tie to cell i+1
    assert abs(b.sum() - 16.0) <= 16 * tol                   # flux form: B_t is conserved along the pencil
    for c in range(5, 8):                                    # nothing else moves
        if c != 5 + t:
            assert not f[c].any()
    assert np.array_equal(f[0], np.ones_like(f[0])) and np.array_equal(f[4], np.full_like(f[4], 4.0))
