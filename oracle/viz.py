"""oracle.viz -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Plain NumPy restatement of the headless visualisation stage (section 8; SURVEY.md 8(f)
rank 4) exactly as include/mhd.h fixes it: the paper gives no formulas for its vertex-buffer, transfer-function and
volume-rendering mappings, so mhd.h is the definition and this file follows it operation by operation in fp32
(every NumPy float32 operation is one IEEE rounding, like the single CUDA intrinsics on the other side).
**Parity unpinned by the paper** for this stage; the pins in tests/test_oracle_pins.py are closed forms and
hand-computable cases.  Shares no code with the CUDA path.

Fields: list of eight arrays of shape (nz, ny, nx), any float dtype; ``field`` 0..7 or 8 (gas pressure).
"""
from __future__ import annotations

import numpy as np

F = np.float32
PRESSURE = 8


def _next(a, axis, bc):
    """a at index + 1 along axis, mapped by the boundary rule (0 periodic: wrap, 1 outflow: clamp)"""
    if bc == 0:
        return np.roll(a, -1, axis=axis)
    idx = np.minimum(np.arange(a.shape[axis]) + 1, a.shape[axis] - 1)
    return np.take(a, idx, axis=axis)


def value(fields, field, gamma, bc):
    """the selected value of every cell as fp32 (mhd.h: 'value v')"""
    f = [np.asarray(a).astype(F) for a in fields]
    if field < 8:
        return f[field]
    rho, mx, my, mz, E, Bx, By, Bz = f
    half = F(0.5)
    bx = half * (Bx + _next(Bx, 2, bc))
    by = half * (By + _next(By, 1, bc))
    bz = half * (Bz + _next(Bz, 0, bc))
    m2 = (mx * mx + my * my) + mz * mz
    b2 = (bx * bx + by * by) + bz * bz
    ke = (half * m2) / rho
    return (F(gamma) - F(1.0)) * ((E - ke) - half * b2)


def unit(v, vmin, vmax):
    """t = min(max((v - vmin) * inv, 0), 1), NaN -> 0"""
    inv = F(1.0 / (float(vmax) - float(vmin)))
    with np.errstate(invalid="ignore"):
        t = (v - F(vmin)) * inv
        t = np.where(t > 0, np.where(t < 1, t, F(1.0)), F(0.0)).astype(F)
    return t


def byte(t):
    return (t * F(255.0) + F(0.5)).astype(np.int32)          # truncation


def value_range(fields, field, gamma, bc):
    v = value(fields, field, gamma, bc)
    v = v[np.isfinite(v)]                                     # NaN and +-Inf cells are skipped (mhd.h: finite values)
    return float(v.min()), float(v.max())


def curve(fields, field, gamma, bc, j, k, vmin, vmax):
    """(nx, 2) float32: x = -1 + (2 i + 1) * fp32(1/nx), y = -1 + 2 t"""
    v = value(fields, field, gamma, bc)[k, j, :]
    nx = v.shape[0]
    invn = F(1.0 / nx)
    x = F(-1.0) + (2 * np.arange(nx) + 1).astype(F) * invn
    y = F(-1.0) + F(2.0) * unit(v, vmin, vmax)
    return np.stack([x, y], axis=1).astype(F)


def slice_rgba(fields, field, gamma, bc, k, vmin, vmax, lut):
    """(ny, nx, 4) uint8: lut[byte(t)] for the plane k; lut: (256, 4) uint8"""
    v = value(fields, field, gamma, bc)[k]
    return np.asarray(lut, dtype=np.uint8)[byte(unit(v, vmin, vmax))]


def volume_rgba(fields, field, gamma, bc, vmin, vmax, lut, opacity):
    """(ny, nx, 4) uint8: front-to-back compositing along +z with early termination at A >= 0.99"""
    lut = np.asarray(lut, dtype=np.uint8)
    v = value(fields, field, gamma, bc)
    nz, ny, nx = v.shape
    inv255 = F(1.0) / F(255.0)
    C = np.zeros((ny, nx, 3), dtype=F)
    A = np.zeros((ny, nx), dtype=F)
    live = np.ones((ny, nx), dtype=bool)
    for k in range(nz):
        s = lut[byte(unit(v[k], vmin, vmax))]
        a = (s[..., 3].astype(F) * inv255) * F(opacity)
        a = np.where(a < 1, a, F(1.0)).astype(F)
        w = (F(1.0) - A) * a
        Cn = C + w[..., None] * (s[..., :3].astype(F) * inv255)
        An = A + w
        C = np.where(live[..., None], Cn, C).astype(F)
        A = np.where(live, An, A).astype(F)
        live = live & (A < F(0.99))
    out = np.empty((ny, nx, 4), dtype=np.uint8)
    one = F(1.0)
    out[..., :3] = byte(np.where(C < one, C, one).astype(F))
    out[..., 3] = byte(np.where(A < one, A, one).astype(F))
    return out
