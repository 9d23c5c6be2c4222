"""Error measures shared by the GPU parity tests ("Tolerances")."""
import numpy as np

GROUPS = {"rho": [0], "m": [1, 2, 3], "E": [4], "B": [5, 6, 7]}


def max_rel(got, ref):
    """per field group: max|got - ref| / max|ref|  (reading R15 of BASELINE.json's 'max relative error')"""
    out = {}
    for name, idx in GROUPS.items():
        scale = max(float(np.abs(ref[i]).max()) for i in idx)
        err = max(float(np.abs(np.asarray(got[i], np.float64) - np.asarray(ref[i], np.float64)).max()) for i in idx)
        out[name] = err / scale if scale > 0 else err
    return out


def l1_rel(got, ref):
    """per field group: sum|got - ref| / sum|ref|"""
    out = {}
    for name, idx in GROUPS.items():
        scale = sum(float(np.abs(ref[i]).sum()) for i in idx)
        err = sum(float(np.abs(np.asarray(got[i], np.float64) - np.asarray(ref[i], np.float64)).sum()) for i in idx)
        out[name] = err / scale if scale > 0 else err
    return out


def worst(d):
    return max(d.values())


# ---------------------------------------------------------------------------------------------------------------
# fp32 per-step gate (reading R15).  north_star: 1e-5 max relative error after one step.  The scheme has ONE
# discontinuous decision, the upwind switch of eq (21): where the smoothed face velocities of two
# neighbouring faces cancel EXACTLY (vg_n = -vg_{n+1} != 0, so vh = 0 in exact arithmetic) the edge flux jumps by
# |vg| |B_n + B_{n+1}| dt depending on the sign rounding leaves in vh.  Mirror-symmetric data with piecewise constant
# initial values (the blast waves: config c3, E4, E6) produce such exact ties on their symmetry planes, and there every
# fp32 evaluation order -- the oracle's own included -- lands up to ~1e-3 from the fp64 result in a few dozen cells.
# At those cells "the" fp32 answer does not exist, so the yardstick is the oracle's own sensitivity on the same block:
# oracle<float>, oracle<double> from inputs perturbed by +-6e-8 relative (half an fp32 ulp), TIE_WITNESSES times, and
# oracle<float> from such inputs, TIE_WITNESSES / 2 times.
# A block passes when it meets the plain 1e-5 everywhere, or when
#   every cell above 1e-5 lies within TIE_RADIUS cells (per axis) of a cell where some WITNESS is above 1e-5 too -- the
#     excuse is by LOCATION: a cell the witnesses do not point at must meet the plain 1e-5, so a seam, halo or
#     ghost-thread bug of a few dozen cells by 1e-3 somewhere else in a blast-wave block fails (count printed, must be 0),
#   max error        <= 1e-5 + 1.5 x (largest deviation any witness shows from oracle<double>), and <= TIE_CEILING,
#   cells above 1e-5 <= 2 x (largest such count among the witnesses) + 16,
#   mean error       <= 1e-6
# (measured on c3, 256^3, 6 steps: ratio of maxima <= 1.32, ratio of counts <= 1.76, mean <= 5e-7; an IEEE-division,
# no-FMA build of the kernels gives the same figures, so none of it is MUFU or contraction).
# Why a radius: a tie flips the flux of ONE edge; which of the 1 + TIE_WITNESSES evaluations flips at a given edge is
# a coin toss per edge, and the cells that see the flip are that edge's two cells and, through the operators that
# follow in the same step, their neighbours at a much smaller amplitude (tests/test_parity_gate.py: an fp32 evaluation
# that is none of the witnesses is covered at radius 3 by two witnesses already, and at radius 2 never).
# ---------------------------------------------------------------------------------------------------------------
TIE_WITNESSES = 8
TIE_RADIUS = 3
TIE_CEILING = 5e-3


def fp32_step_gate(got, before, gamma, bc, k, dt, core=None, scale=None, tol=1e-5, tag=""):
    """got: GPU fp32 result (arrays, any float dtype); before: the fp32 pre-step state as float64 arrays.
    core: index tuple selecting the cells to compare (default all).  Returns per-group max relative error."""
    import oracle
    core = core if core is not None else (slice(None),) * 3
    ref = [np.array(a, dtype=np.float64, order="C", copy=True) for a in before]
    oracle.step_fixed(ref, gamma, bc, k, dt)
    got = [np.asarray(a, dtype=np.float64) for a in got]
    if scale is None:
        scale = {g: max(float(np.abs(ref[i]).max()) for i in idx) for g, idx in GROUPS.items()}
    out, wit, hot = {}, None, None
    for g, idx in GROUPS.items():
        e = np.stack([np.abs(got[i][core] - ref[i][core]) for i in idx]) / scale[g]
        out[g] = float(e.max())
        if out[g] <= tol:
            continue
        if wit is None:
            b32 = [np.array(a, dtype=np.float32, order="C", copy=True) for a in before]
            oracle.step_fixed(b32, gamma, bc, k, dt)
            wit = [[a.astype(np.float64) for a in b32]]
            prng = np.random.default_rng(7 + 1000 * k)
            for w in range(TIE_WITNESSES + TIE_WITNESSES // 2):
                bp = [np.ascontiguousarray(a * (1.0 + 6e-8 * prng.choice([-1.0, 1.0], size=a.shape))) for a in before]
                if w >= TIE_WITNESSES:                           # oracle<float> from the moved inputs as well
                    bp = [np.array(a, dtype=np.float32, order="C") for a in bp]
                oracle.step_fixed(bp, gamma, bc, k, dt)
                wit.append([np.asarray(a, dtype=np.float64) for a in bp])
        ws = [np.stack([np.abs(w[i][core] - ref[i][core]) for i in idx]) / scale[g] for w in wit]
        wmax = max(float(w.max()) for w in ws)
        wcount = max(int((w > tol).sum()) for w in ws)
        n_bad = int((e > tol).sum())
        # where the witnesses are sensitive, on the WHOLE block (a tie just outside the core reaches into it), in ANY of
        # the eight fields (the flipped edge flux of B reaches m and E through the fluid operators that follow in the
        # same step, at a hundredth of the amplitude), widened by TIE_RADIUS cells per axis
        if hot is None:
            hot = np.zeros(ref[0].shape, dtype=bool)
            for w in wit:
                for g2, idx2 in GROUPS.items():
                    for i in idx2:
                        hot |= np.abs(w[i] - ref[i]) > tol * scale[g2]
        from scipy import ndimage
        unexcused = {}
        for r in range(TIE_RADIUS + 2):
            near = hot if r == 0 else ndimage.binary_dilation(hot, structure=np.ones((3, 3, 3), bool), iterations=r)
            unexcused[r] = int(((e > tol).any(axis=0) & ~near[core]).sum())
        print(f"fp32 tie gate {tag} step {k} {g}: max {out[g]:.2e} in {n_bad} cells; witnesses max {wmax:.2e} in <= {wcount} cells; "
              f"vs oracle<float> {float(np.stack([np.abs(got[i][core] - wit[0][i][core]) for i in idx]).max()) / scale[g]:.2e}; "
              f"cells above tol farther than r from every witness-sensitive cell, r: count = {unexcused}")
        assert unexcused[TIE_RADIUS] == 0, (tag, k, g, unexcused)
        assert out[g] <= tol + 1.5 * wmax and out[g] <= TIE_CEILING, (tag, k, g, out[g], wmax)
        assert n_bad <= 2 * wcount + 16, (tag, k, g, n_bad, wcount)
        assert float(e.mean()) <= 1e-6, (tag, k, g, float(e.mean()))
    return out


def random_state(nx, ny, nz, seed, positive_v=False):
    """smooth-ish random state with a few sharp features (exercises both limiter branches)"""
    rng = np.random.default_rng(seed)
    sh = (nz, ny, nx)
    z, y, x = np.meshgrid(np.arange(nz) / max(nz, 1), np.arange(ny) / max(ny, 1), np.arange(nx) / max(nx, 1), indexing="ij")

    def smooth():
        a = np.zeros(sh)
        for _ in range(4):
            k = rng.integers(0, 3, 3)
            ph = rng.random(3) * 2 * np.pi
            a += rng.standard_normal() * np.cos(2 * np.pi * (k[0] * x + k[1] * y + k[2] * z) + ph.sum())
        return a + 0.05 * rng.standard_normal(sh)

    rho = 1.0 + 0.2 * np.tanh(smooth()) + 0.5 * (smooth() > 0.8)
    v = [0.4 * smooth() + (0.3 if positive_v else 0.0) for _ in range(3)]
    B = [0.5 * smooth() + 0.3 for _ in range(3)]
    p = 0.6 + 0.3 * np.tanh(smooth()) + 2.0 * (smooth() > 1.0)
    E = p / (2.0 / 3.0) + 0.5 * rho * sum(a * a for a in v) + 0.5 * sum(a * a for a in B) + 0.3
    return [np.ascontiguousarray(a, dtype=np.float64) for a in [rho, rho * v[0], rho * v[1], rho * v[2], E] + B]
