"""Seeded, synthetic initial states for the MHD update (the five BASELINE.json configs + test states).

This module holds NONE of the method's arithmetic (no fluxes, limiters, sweeps, CFL): it only
builds initial data, and it is the one module that serves both the CUDA path's callers and the
oracle's callers (tests, bench.py).  It imports neither of them.

Every generator returns ``(fields, meta)``:
  fields : list of 8 float64 arrays of shape (nz, ny, nx) (x fastest) in the order
           rho, m_x, m_y, m_z, E, Bx, By, Bz.  B is staggered as in eq (19) PAPER.md:136-141:
           Bx[k,j,i] sits on the face (i-1/2, j, k), etc.
  meta   : dict(gamma=..., bc=0 periodic | 1 outflow, name=..., box=physical box length per axis)

Cell centres sit at x_i = x_min + (i + 1/2)/n, faces at x_min + i/n.
The scheme itself works in grid units (cells of unit width): velocities and B keep
their physical values and t_phys = t_grid / n for a unit box.
Initial total energy (paper silent, reading R18): E = p/(gamma-1) + rho |v|^2/2 + |B_c|^2/2
with B_c the average of the two faces of the cell, the same interpolation the scheme uses.

``xp`` may be ``numpy`` (default) or ``torch`` (with ``xp_kw={"device": "cuda"}``) for the
Fourier-mode state, so bench.py can build the 512^3 state in seconds on the device; the formula is
the same either way.  ``box=((k0,k1),(j0,j1),(i0,i1))`` evaluates only a sub-box of global indices.
"""
from __future__ import annotations

import math

import numpy as np

PERIODIC, OUTFLOW = 0, 1
FIELD_NAMES = ("rho", "mx", "my", "mz", "E", "Bx", "By", "Bz")


# ----------------------------------------------------------------------------------------------
# helpers
# ----------------------------------------------------------------------------------------------
def _shift_plus(a, axis, bc, xp=np):
    """a at index+1 along axis, index mapped by wrap (periodic) or clamp (outflow)."""
    if bc == PERIODIC:
        return xp.roll(a, -1, axis)
    n = a.shape[axis]
    idx = [slice(None)] * a.ndim
    idx[axis] = slice(1, n)
    last = [slice(None)] * a.ndim
    last[axis] = slice(n - 1, n)
    cat = xp.concatenate if xp is np else xp.cat
    return cat([a[tuple(idx)], a[tuple(last)]], axis)


def total_energy(rho, vx, vy, vz, p, bx, by, bz, gamma, bc, xp=np):
    """E = p/(gamma-1) + rho v^2/2 + B_c^2/2 with B_c the face average (axes: 2 = x, 1 = y, 0 = z)."""
    bcx = 0.5 * (bx + _shift_plus(bx, 2, bc, xp))
    bcy = 0.5 * (by + _shift_plus(by, 1, bc, xp))
    bcz = 0.5 * (bz + _shift_plus(bz, 0, bc, xp))
    return p / (gamma - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz) + 0.5 * (bcx * bcx + bcy * bcy + bcz * bcz)


def to_precision(fields, dtype):
    """Round a float64 state to the run precision (identical input for oracle and GPU)."""
    return [np.array(f, dtype=dtype, order="C", copy=True) for f in fields]   # fresh, never aliased


class SplitMix64:
    """Counter-based splitmix64 -> uniform(0,1) and Box-Muller normals; explicit so any language agrees."""

    def __init__(self, seed: int):
        self.s = seed & 0xFFFFFFFFFFFFFFFF

    def next_u64(self) -> int:
        self.s = (self.s + 0x9E3779B97F4A7C15) & 0xFFFFFFFFFFFFFFFF
        z = self.s
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & 0xFFFFFFFFFFFFFFFF
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & 0xFFFFFFFFFFFFFFFF
        return z ^ (z >> 31)

    def uniform(self) -> float:
        return ((self.next_u64() >> 11) + 0.5) / 9007199254740992.0   # (0,1), 53 bits

    def normal(self) -> float:
        u1, u2 = self.uniform(), self.uniform()
        return math.sqrt(-2.0 * math.log(u1)) * math.cos(2.0 * math.pi * u2)


# ----------------------------------------------------------------------------------------------
# config 1: Brio-Wu shock tube (BASELINE.json configs[0]; PAPER.md:347-383 for gamma, B, rho, p)
# ----------------------------------------------------------------------------------------------
def brio_wu(nx=512, ny=1, nz=1):
    gamma = 2.0
    x = (np.arange(nx) + 0.5) / nx
    left = (x < 0.5)[None, None, :] & np.ones((nz, ny, 1), bool)
    rho = np.where(left, 1.0, 0.125)
    p = np.where(left, 1.0, 0.1)
    z = np.zeros((nz, ny, nx))
    bx = np.full((nz, ny, nx), 0.75)
    by = np.where(left, 1.0, -1.0)          # By lives at y-faces; it depends on x only
    E = total_energy(rho, z, z, z, p, bx, by, z, gamma, OUTFLOW)
    return [rho, z.copy(), z.copy(), z.copy(), E, bx, by, z.copy()], dict(
        gamma=gamma, bc=OUTFLOW, name="brio_wu", box=(1.0, 1.0, 1.0))


# ----------------------------------------------------------------------------------------------
# config 2: Orszag-Tang vortex (BASELINE.json configs[1]; PAPER.md:433-465 for rho, p, B, gamma)
# ----------------------------------------------------------------------------------------------
def orszag_tang(n=256, nz=1):
    gamma = 5.0 / 3.0
    xc = (np.arange(n) + 0.5) / n
    xf = np.arange(n) / n
    shape = (nz, n, n)
    X = np.broadcast_to(xc[None, None, :], shape)
    Y = np.broadcast_to(xc[None, :, None], shape)
    rho = np.full(shape, 25.0 / (36.0 * math.pi))
    p = np.full(shape, 5.0 / (12.0 * math.pi))
    vx = -np.sin(2 * math.pi * Y)
    vy = np.sin(2 * math.pi * X)
    vz = np.zeros(shape)
    b0 = 1.0 / math.sqrt(4.0 * math.pi)
    # Bx on x-faces depends on y (cell centre) only; By on y-faces depends on x (cell centre) only
    bx = np.broadcast_to((-b0 * np.sin(2 * math.pi * xc))[None, :, None], shape).copy()
    by = np.broadcast_to((b0 * np.sin(4 * math.pi * xc))[None, None, :], shape).copy()
    del xf
    bz = np.zeros(shape)
    E = total_energy(rho, vx, vy, vz, p, bx, by, bz, gamma, PERIODIC)
    return [rho, rho * vx, rho * vy, rho * vz, E, bx, by, bz], dict(
        gamma=gamma, bc=PERIODIC, name="orszag_tang", box=(1.0, 1.0, 1.0))


# ----------------------------------------------------------------------------------------------
# config 3: 3-D blast wave (BASELINE.json configs[2]; PAPER.md:539-559 for rho, p, r, gamma)
# ----------------------------------------------------------------------------------------------
def blast3d(n=256, xp=np, xp_kw=None, paper_field=False, centre=(0.0, 0.0, 0.0)):
    """paper_field=True: the paper's own experiment E6, B = (1,1,1)/sqrt(3) instead of
    BASELINE.json's (1,1,0)/sqrt(2); same rho, p, radius.
    centre = (x, y, z) of the high-pressure sphere (default: the origin, as BASELINE.json configs[2] has it; an
    off-grid centre removes the mirror symmetry of the discrete data, R15)"""
    xp_kw = xp_kw or {}
    gamma = 5.0 / 3.0
    c = (xp.arange(n, dtype=xp.float64, **xp_kw) + 0.5) / n - 0.5
    r2 = (c[None, None, :] - centre[0]) ** 2 + (c[None, :, None] - centre[1]) ** 2 + (c[:, None, None] - centre[2]) ** 2
    shape = (n, n, n)
    one = xp.ones(shape, dtype=xp.float64, **xp_kw)
    p = xp.where(r2 < 0.1 * 0.1, 10.0 * one, 0.1 * one)
    rho = one
    z = xp.zeros(shape, dtype=xp.float64, **xp_kw)
    if paper_field:
        b = 1.0 / math.sqrt(3.0)
        bx, by, bz = b * one, b * one, b * one
    else:
        b = 1.0 / math.sqrt(2.0)
        bx, by, bz = b * one, b * one, z * 1.0
    E = p / (gamma - 1.0) + 0.5 * (bx * bx + by * by + bz * bz)       # v = 0, uniform B
    return [rho, z, z * 1.0, z * 1.0, E, bx, by, bz], dict(
        gamma=gamma, bc=PERIODIC, name="blast3d_paper" if paper_field else "blast3d", box=(1.0, 1.0, 1.0))


# ----------------------------------------------------------------------------------------------
# the paper's experiment E4: 2-D blast wave: rho = 1, p = 10 inside r < 0.1 of the centre of the
# unit square, 0.1 outside, B = (1/sqrt 2, 1/sqrt 2, 0), gamma = 5/3, v = 0; periodic.  Initial data only
# (SURVEY.md 8(f) rank 3); the stray "p = 5/(12 pi)" of eq (48) is a garble from the Orszag-Tang block (R19).
# ----------------------------------------------------------------------------------------------
def blast2d(n=512, nz=1):
    gamma = 5.0 / 3.0
    c = (np.arange(n, dtype=np.float64) + 0.5) / n - 0.5
    r2 = c[None, None, :] ** 2 + c[None, :, None] ** 2 + np.zeros((nz, 1, 1))
    one = np.ones((nz, n, n))
    p = np.where(r2 < 0.1 * 0.1, 10.0 * one, 0.1 * one)
    z = np.zeros((nz, n, n))
    b = 1.0 / math.sqrt(2.0)
    bx, by = b * one, b * one
    E = p / (gamma - 1.0) + 0.5 * (bx * bx + by * by)
    return [one.copy(), z, z.copy(), z.copy(), E, bx, by, z.copy()], dict(
        gamma=gamma, bc=PERIODIC, name="blast2d", box=(1.0, 1.0, 1.0 / n))


# ----------------------------------------------------------------------------------------------
# configs 4/5: turbulence-like periodic state from seeded random Fourier modes
# ----------------------------------------------------------------------------------------------
def fourier_modes(seed=4362, nmodes=32, kmax=8):
    """Draw the shared wavevector set and per-component amplitudes/phases (DESIGN.md input recipe).

    32 integer wavevectors uniform in [-kmax,kmax]^3, rejected unless 0 < |k| <= kmax; amplitudes
    ~ N(0, 0.1), phases ~ U[0, 2 pi), independent for each of the 7 scalar components
    (density perturbation f, v_x, v_y, v_z, A_x, A_y, A_z)."""
    rng = SplitMix64(seed)
    ks = []
    while len(ks) < nmodes:
        k = tuple(int(rng.uniform() * (2 * kmax + 1)) - kmax for _ in range(3))
        k2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2]
        if 0 < k2 <= kmax * kmax:
            ks.append(k)
    comps = {}
    for name in ("f", "vx", "vy", "vz", "ax", "ay", "az"):
        amp = [0.1 * rng.normal() for _ in range(nmodes)]
        ph = [2.0 * math.pi * rng.uniform() for _ in range(nmodes)]
        comps[name] = (amp, ph)
    return ks, comps


def _mode_sum(xp, xp_kw, ks, amp, ph, n, ranges, offsets, scale_by_invk=False):
    """sum_m a_m cos(2 pi (kx x + ky y + kz z) + phi_m) at x = (i + ox)/nx etc. on index ranges."""
    nx, ny, nz = n
    (k0, k1), (j0, j1), (i0, i1) = ranges
    ox, oy, oz = offsets
    xi = (xp.arange(i0, i1, dtype=xp.float64, **xp_kw) + ox) / nx
    yj = (xp.arange(j0, j1, dtype=xp.float64, **xp_kw) + oy) / ny
    zk = (xp.arange(k0, k1, dtype=xp.float64, **xp_kw) + oz) / nz
    out = xp.zeros((k1 - k0, j1 - j0, i1 - i0), dtype=xp.float64, **xp_kw)
    two_pi = 2.0 * math.pi
    for (kx, ky, kz), a, p in zip(ks, amp, ph):
        if scale_by_invk:
            a = a / (two_pi * math.sqrt(kx * kx + ky * ky + kz * kz))
        axy = (two_pi * kx) * xi[None, :] + ((two_pi * ky) * yj[:, None] + p)
        cxy, sxy = xp.cos(axy), xp.sin(axy)
        az = (two_pi * kz) * zk
        cz, sz = a * xp.cos(az), a * xp.sin(az)
        out += cz[:, None, None] * cxy[None, :, :]
        out -= sz[:, None, None] * sxy[None, :, :]
    return out


def turbulence(nx=64, ny=None, nz=None, seed=4362, xp=np, xp_kw=None, box=None, nmodes=32, kmax=8):
    """rho = 1 + 0.1 f, p = 1, v and B = curl A from seeded Fourier modes; periodic; gamma = 5/3.

    Reading of BASELINE.json's "amplitudes ~ N(0, 0.1)" for B (DESIGN.md input recipe): the
    B-mode amplitudes are ~ N(0, 0.1), i.e. the physical A-mode amplitude is a_m / (2 pi |k_m|).
    A sits on cell edges, B is its discrete curl on faces, so the discrete div B is zero to rounding.
    """
    xp_kw = xp_kw or {}
    ny = nx if ny is None else ny
    nz = nx if nz is None else nz
    n = (nx, ny, nz)
    gamma = 5.0 / 3.0
    ks, comps = fourier_modes(seed, nmodes, kmax)
    if box is None:
        box = ((0, nz), (0, ny), (0, nx))
    (k0, k1), (j0, j1), (i0, i1) = box

    def ms(name, ranges, offs, invk=False):
        return _mode_sum(xp, xp_kw, ks, comps[name][0], comps[name][1], n, ranges, offs, invk)

    cc = (0.5, 0.5, 0.5)
    rho = 1.0 + 0.1 * ms("f", box, cc)
    vx, vy, vz = ms("vx", box, cc), ms("vy", box, cc), ms("vz", box, cc)
    p = 1.0
    # vector potential on edges, one extra index on the high side (and for the E average, B needs
    # one extra face on the high side too, so A gets two)
    kk, jj, ii = (k0, k1 + 2), (j0, j1 + 2), (i0, i1 + 2)
    ax = ms("ax", (kk, jj, ii), (0.5, 0.0, 0.0), True)   # A_x at (x_c, y_f, z_f)
    ay = ms("ay", (kk, jj, ii), (0.0, 0.5, 0.0), True)   # A_y at (x_f, y_c, z_f)
    az = ms("az", (kk, jj, ii), (0.0, 0.0, 0.5), True)   # A_z at (x_f, y_f, z_c)
    # discrete curl.  On the cubic grids of the configs this is the physical curl on the unit box
    # (d/dx -> n * difference); on a non-cubic test grid the same n = nx multiplies every difference so
    # that the GRID-UNIT divergence the scheme preserves (unit-width cells) is zero.
    bx = nx * ((az[:-1, 1:, :-1] - az[:-1, :-1, :-1]) - (ay[1:, :-1, :-1] - ay[:-1, :-1, :-1]))
    by = nx * ((ax[1:, :-1, :-1] - ax[:-1, :-1, :-1]) - (az[:-1, :-1, 1:] - az[:-1, :-1, :-1]))
    bz = nx * ((ay[:-1, :-1, 1:] - ay[:-1, :-1, :-1]) - (ax[:-1, 1:, :-1] - ax[:-1, :-1, :-1]))
    del ax, ay, az
    # b* have one extra face on the high side of every axis
    bcx = 0.5 * (bx[:-1, :-1, :-1] + bx[:-1, :-1, 1:])
    bcy = 0.5 * (by[:-1, :-1, :-1] + by[:-1, 1:, :-1])
    bcz = 0.5 * (bz[:-1, :-1, :-1] + bz[1:, :-1, :-1])
    E = p / (gamma - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz) + 0.5 * (bcx * bcx + bcy * bcy + bcz * bcz)
    del bcx, bcy, bcz
    core = (slice(0, k1 - k0), slice(0, j1 - j0), slice(0, i1 - i0))
    contig = (lambda a: np.ascontiguousarray(a)) if xp is np else (lambda a: a.contiguous())
    fields = [rho, rho * vx, rho * vy, rho * vz, E, contig(bx[core]), contig(by[core]), contig(bz[core])]
    return fields, dict(gamma=gamma, bc=PERIODIC, name="turbulence", box=(1.0, 1.0, 1.0))


CONFIGS = {
    # name: (generator kwargs, precision(s), steps)  -- BASELINE.json "configs", in order
    "c1_brio_wu_512": dict(gen="brio_wu", kw=dict(nx=512), dtypes=("f64",), t_end=0.1, cfl=0.8),
    "c2_orszag_tang_256": dict(gen="orszag_tang", kw=dict(n=256), dtypes=("f32", "f64"), steps=500, cfl=0.8),
    "c3_blast_256": dict(gen="blast3d", kw=dict(n=256), dtypes=("f32",), steps=200, cfl=0.8),
    "c4_turb_512_f32": dict(gen="turbulence", kw=dict(nx=512), dtypes=("f32",), steps=100, cfl=0.8),
    "c5_turb_512_f64": dict(gen="turbulence", kw=dict(nx=512), dtypes=("f64",), steps=50, cfl=0.8),
}


def make(gen: str, **kw):
    return {"brio_wu": brio_wu, "orszag_tang": orszag_tang, "blast3d": blast3d, "blast2d": blast2d, "turbulence": turbulence}[gen](**kw)
