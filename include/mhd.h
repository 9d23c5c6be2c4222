/* mhd.h -- C ABI of libmhd.so: the per-timestep update of the 3-D ideal-MHD conserved state by the
 * second-order relaxing-TVD scheme of arxiv/paper_0908_4362 (section 3, lines 47-172),
 * hand-written for NVIDIA B200 (sm_100a).  The calls follow the paper's program flow
 * (PAPER.md:233-243): initial u on cells and B on faces in; loop { c_max -> dt; six L_i; t += 2 dt };
 * state out.
 *
 * Conventions
 *   - Plain C.  No exception crosses this boundary and the library never calls exit().  Every call
 *     that returns int returns MHD_OK (0) or a negative mhd_status; the message of the last failure
 *     of a context is available from mhd_last_error().
 *   - Grid units: cells have unit width; dt, t and all speeds are in cells per unit
 *     time.  For a unit box of n cells t_physical = t_grid / n.
 *   - State: eight fields in the order rho, m_x, m_y, m_z, E, Bx, By, Bz, each a
 *     dense array of N = nx*ny*nz elements of the context's precision, x fastest:
 *         idx = i + nx*(j + ny*k).
 *     u = (rho, m, E) is cell centred; B is face centred (eq (19)):
 *     Bx[i,j,k] = B_x at (i-1/2,j,k), By[i,j,k] = B_y at (i,j-1/2,k), Bz[i,j,k] = B_z at (i,j,k-1/2).
 *   - Boundary rule (the paper is silent; reading R9): every read of an operator's input at
 *     an out-of-range index is mapped by wrap (MHD_BC_PERIODIC) or clamp (MHD_BC_OUTFLOW), the same
 *     rule on all three axes.
 *   - One step = one c_max reduction + one double sweep of six L_i operators with the rotation of
 *     eqs (23)-(25), advancing t by 2 dt.
 *   - Ownership: the context owns (or, after mhd_bind, borrows) all device memory.  set/get copy; the
 *     caller keeps every pointer it passes and none needs to outlive the call.
 *   - Pointers are HOST pointers unless the argument says otherwise ("where" = MHD_DEVICE).
 *   - All work is enqueued on the context's CUDA stream; calls marked "synchronises" wait for it.
 *   - Not thread safe per context; distinct contexts are independent.
 */
#ifndef MHD_H_
#define MHD_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mhd_ctx mhd_ctx; /* opaque, owned by the library */

enum mhd_precision { MHD_F32 = 0, MHD_F64 = 1 };
enum mhd_bc { MHD_BC_PERIODIC = 0, MHD_BC_OUTFLOW = 1 };
enum mhd_where { MHD_HOST = 0, MHD_DEVICE = 1 };
enum mhd_status {
  MHD_OK = 0,
  MHD_EINVAL = -1,     /* bad argument: extent < 1, gamma <= 1, unknown enum, NULL pointer, cfl <= 0, n < 0 */
  MHD_ENOMEM = -2,     /* allocation failed, or mhd_bind workspace too small / misaligned */
  MHD_ECUDA = -3,      /* a CUDA call failed (message in mhd_last_error) */
  MHD_ENONFINITE = -4, /* the c_max reduction saw NaN/Inf or c_max <= 0 (state is poisoned) */
  MHD_ENOSTATE = -5    /* stepping or reading before mhd_set_state */
};
enum mhd_operator { MHD_OP_FLUID = 0, MHD_OP_BPAIR = 1, MHD_OP_SWEEP_FORWARD = 2, MHD_OP_SWEEP_REVERSE = 3, MHD_OP_MIDDLE_PAIR = 4 };

/* Bytes of device memory a context of this shape needs (two copies of the 8 fields for out-of-place
 * operators plus a small scalar block).  Returns 0 on invalid arguments. */
size_t mhd_workspace_bytes(int nx, int ny, int nz, int precision);

/* Create a context for an nx*ny*nz grid (any extents >= 1; an extent of 1 makes that axis
 * degenerate, e.g. 512x1x1 for 1-D runs).  gamma > 1 is the adiabatic index of
 * P = (gamma-1)(E - rho v^2/2 - B^2/2).  No device memory is touched until the first
 * call that needs it (mhd_bind or mhd_set_state).  *out receives the context.
 * Every size and both boundary rules give the same results to rounding; the specialised kernels
 * want nx to be a multiple of 16 bytes (4 floats / 2 doubles), rows of at most 2048 (fp32) / 1024 (fp64) cells and fewer
 * than 2^31 cells, otherwise slower generic kernels run. */
int mhd_create(int nx, int ny, int nz, double gamma, int precision, int bc, mhd_ctx** out);

/* Optional.  Use caller-owned DEVICE memory (at least mhd_workspace_bytes, 256-byte aligned) and/or a
 * caller-owned CUDA stream (a cudaStream_t passed as void*; NULL = the default stream) instead of
 * the library's own cudaMalloc / own stream.  Must precede mhd_set_state.  The memory is borrowed
 * until mhd_destroy.  device_workspace == NULL keeps library-owned memory and only sets the stream. */
int mhd_bind(mhd_ctx* ctx, void* device_workspace, size_t bytes, void* cuda_stream);

/* Free the context and everything it owns.  Synchronises.  NULL is allowed. */
int mhd_destroy(mhd_ctx* ctx);

/* Copy a full state IN.  fields[0..7] point to N elements each of the context's precision, in host
 * (where = MHD_HOST, pageable or pinned) or device (MHD_DEVICE) memory.  Resets the time
 * accumulated by the context to 0 but not the step index.  Synchronises for host sources.  Device sources are
 * copied on the context's stream without waiting for any other stream: the caller orders the producer of the data
 * before this call (e.g. a device synchronise, or by binding the producer's stream with mhd_bind). */
int mhd_set_state(mhd_ctx* ctx, const void* const fields[8], int where);

/* Copy the current state OUT into fields[0..7] (N elements each).  Synchronises. */
int mhd_get_state(mhd_ctx* ctx, void* const fields[8], int where);

/* c_max of eq (18) (B interpolated to cell centres) and dt = cfl / c_max, in grid
 * units.  Writes dt to *dt_out and, if cmax_out != NULL, c_max to *cmax_out.  Synchronises.
 * MHD_ENONFINITE if c_max is NaN, Inf or <= 0. */
int mhd_cfl_dt(mhd_ctx* ctx, double cfl, double* dt_out, double* cmax_out);

/* n steps (n >= 0), each: c_max reduction, dt = cfl / c_max kept on the device, six L_i with that
 * dt, step index += 1, t += 2 dt.  If t_advanced != NULL the call synchronises,
 * writes the time advanced by THIS call and reports MHD_ENONFINITE if any reduction was poisoned;
 * if it is NULL nothing is read back and the call returns as soon as the work is enqueued. */
int mhd_step(mhd_ctx* ctx, int n, double cfl, double* t_advanced);

/* n steps with the caller's dt (> 0, grid units) instead of the CFL value; no reduction is run.
 * Used for parity tests and for clipping the last step to a target time.  Does not synchronise. */
int mhd_step_fixed(mhd_ctx* ctx, int n, double dt);

/* The flow loop of PAPER.md:233-243 up to a target time, with the stop test on the device: repeat
 * { c_max; dt = min(cfl / c_max, (t_end - t) / 2); six L_i; t += 2 dt } until t = t_end (reading R14: the last
 * step is shortened to land on t_end, and t is then set to t_end exactly) or max_steps steps were taken.
 * t and t_end are times since mhd_set_state, in grid units.  dt, t and the clipping never leave the GPU
 * between steps (the paper reads dt back every step); the host enqueues batches of steps sized
 * from the last dt and reads (t, steps) back once per batch, so the call synchronises a few times.
 * *steps_done (may be NULL) = steps that advanced time, *t_reached (may be NULL) = t afterwards; the step
 * index advances by *steps_done.  MHD_EINVAL for cfl <= 0, max_steps < 0 or a NaN t_end; MHD_ENOSTATE before
 * mhd_set_state; MHD_ENONFINITE if a reduction was poisoned (the state is then whatever the last batch left). */
int mhd_run_until(mhd_ctx* ctx, double t_end, double cfl, long long max_steps, long long* steps_done,
                  double* t_reached);

/* One operator of the step, for per-operator parity tests: op = MHD_OP_FLUID (fluid_d, Algorithm 1,
 * PAPER.md:273-285), MHD_OP_BPAIR (B_{t1->d} then B_{t2->d}, or t2 then t1 if reverse != 0;
 * Algorithm 2), MHD_OP_SWEEP_FORWARD / MHD_OP_SWEEP_REVERSE (L_d, PAPER.md:162,
 * 317; `reverse` is ignored), MHD_OP_MIDDLE_PAIR (forward L_d followed by reverse L_d, the third and fourth
 * operator of every step, eqs (23)-(25) PAPER.md:164-170; `reverse` is ignored).  d = 0, 1, 2 for x, y, z.
 * Does not synchronise. */
int mhd_apply(mhd_ctx* ctx, int op, int d, int reverse, double dt);

/* Step index s selects the sweep order (x,y,z), (z,x,y), (y,z,x) for s mod 3 = 0, 1, 2. */
int mhd_get_step_index(mhd_ctx* ctx, long long* s);
int mhd_set_step_index(mhd_ctx* ctx, long long s);

/* Total time advanced since the last mhd_set_state (grid units).  Synchronises. */
int mhd_get_time(mhd_ctx* ctx, double* t);

/* Not on the timed path.  sums[0..7] = sum over cells of each field (double accumulation);
 * *max_abs_divb = max |(Bx[i+1]-Bx[i]) + (By[j+1]-By[j]) + (Bz[k+1]-Bz[k])| over cells, +1 mapped by
 * the boundary rule (cells on the high side of an outflow axis are skipped).  Either pointer may be
 * NULL.  Synchronises. */
int mhd_diagnostics(mhd_ctx* ctx, double sums[8], double* max_abs_divb);

/* ---- Headless visualisation stage (section 8) --------------------
 * The paper renders the state where it lives: a vertex buffer for 1-D runs, a pixel buffer with a transfer function
 * for 2-D runs, a volume renderer for 3-D runs, through OpenGL.  Here the same buffers are plain DEVICE memory owned
 * by the caller (no graphics API).  The paper gives no formulas, so the mappings are fixed here; all arithmetic is
 * IEEE fp32, one rounding per operation, in the order written:
 *   value v   field 0..7: the stored field converted to fp32; MHD_VIZ_PRESSURE (8): with every input converted to
 *             fp32 first, p = (gamma-1) * ((E - (0.5*((mx*mx + my*my) + mz*mz)) / rho) - 0.5*((bx*bx + by*by) + bz*bz)),
 *             b = 0.5*(face + next face), next face mapped by the boundary rule
 *   unit   t = min(max((v - vmin) * inv, 0), 1), inv = fp32(1 / (vmax - vmin)), NaN -> 0;  byte(t) = trunc(t*255 + 0.5)
 * None of these calls synchronises except mhd_viz_range.  MHD_EINVAL: field out of range, NULL pointer,
 * vmax <= vmin, index out of range, opacity <= 0; MHD_ENOSTATE before mhd_set_state. */
enum { MHD_VIZ_PRESSURE = 8 };

/* Smallest and largest finite v over all cells (what a caller passes as vmin, vmax).  Synchronises.
 * MHD_ENONFINITE if no cell is finite. */
int mhd_viz_range(mhd_ctx* ctx, int field, double* vmin, double* vmax);

/* 1-D (vertex buffer): for the row (j, k), xy_device[2*i] = -1 + (2*i + 1) * fp32(1/nx), xy_device[2*i+1] = -1 + 2*t;
 * xy_device: 2*nx floats of device memory. */
int mhd_viz_curve(mhd_ctx* ctx, int field, int j, int k, double vmin, double vmax, float* xy_device);

/* 2-D (pixel buffer): for the plane k, pixel (i, j) = lut[byte(t)]; lut_rgba_device: 256 RGBA8 entries,
 * rgba_device: nx*ny RGBA8 pixels, x fastest, both device memory. */
int mhd_viz_slice(mhd_ctx* ctx, int field, int k, double vmin, double vmax, const unsigned char* lut_rgba_device,
                  unsigned char* rgba_device);

/* 3-D (volume rendering, orthographic rays along +z, front to back): per pixel (i, j), starting from C = 0, A = 0,
 * for k = 0 .. nz-1: s = lut[byte(t)], a = min((s.a * fp32(1/255)) * opacity, 1), w = (1 - A) * a,
 * C.c += w * (s.c * fp32(1/255)) for c = r, g, b, A += w, stop after the sample that makes A >= 0.99.
 * Pixel = (byte(min(C.r,1)), byte(min(C.g,1)), byte(min(C.b,1)), byte(min(A,1))).  rgba_device: nx*ny RGBA8 pixels. */
int mhd_viz_volume(mhd_ctx* ctx, int field, double vmin, double vmax, const unsigned char* lut_rgba_device,
                   double opacity, unsigned char* rgba_device);

/* Tuning knobs, all optional; none changes what is computed beyond rounding order inside the stated tolerances.
 *   "graph"   -1 auto (default: grids of <= 2^22 cells) | 0 | 1: replay whole steps of mhd_step / mhd_run_until
 *             as CUDA graphs (small grids are bound by launch latency)
 *   "fuse"    sweeps along y, z on periodic grids: 0 (default) two kernels per L_d | 1 reverse L_d (B pair + fluid) and the
 *             middle pair of a step (B pair + B pair + fluid) run as one kernel each | 2 the middle pair fuses its two B
 *             pairs only.  Measured slower than the two-kernel path on B200, hence not the default.
 *   "cmax_reuse" 1 (default) mhd_cfl_dt returns the cached c_max while the state is unchanged | 0 always reduces
 *   "path"    0 auto (default) | 1 generic marching kernels only (any extents, both BCs)
 *   "segment" cells per block along the sweep for the marching kernels (-1 auto, 0 = whole pencil); the fused sweeps
 *             of "fuse" 1 / 2 raise a value below 16 to 16 (or to the whole pencil where that is shorter)
 *   "block"   threads per block of the generic kernels (multiple of 32 in [32, 256])
 *   "brows"   B pair along y, z in fp32 on 256-column tiles: 2 (default) two rows per thread where the extent along the other
 *             transverse axis is even | 1 one row per thread
 *   "tmap"    fluid_y / fluid_z ring kernel in fp32 on whole 256-column tiles: 0 (default) 1-D bulk copies | 1 the nine row
 *             copies of a stage as tensor-map TMA copies (same bits, measured no faster: DESIGN.md section 12)
 *   "xpack"   x kernels: 1 two rows per thread in packed f32x2 arithmetic (fp32, even ny) | 2 one row per thread (default)
 *             | 3 packed fluid_x only
 *   "xfuse"   reverse L_x in one kernel: 0 off | 1 fp32 only (default) | 2 always | 3 fp32, packed
 * Unknown keys and out-of-range values return MHD_EINVAL. */
int mhd_set_option(mhd_ctx* ctx, const char* key, long long value);

/* c_max of eq (18) WITHOUT a context and WITHOUT any allocation, for callers that cannot call
 * cudaMalloc: code that lives inside a host program which owns all device memory through its own pool and forbids
 * allocations behind its back, loops that cannot afford cudaMalloc's device-wide synchronisation, processes already at
 * their memory limit.  (Every other compute call needs a context, whose workspace is cudaMalloc'ed by the library or by
 * whoever passes it to mhd_bind.)  The call issues no cudaMalloc / cudaFree / cudaMallocAsync, creates no stream or event
 * and makes no host allocation of its own: it enqueues one 256-byte memset and one kernel on `cuda_stream` and returns.
 *   fields_device[0..7]  DEVICE pointers, same order, layout and precision rules as mhd_set_state; only read
 *   nx, ny, nz, gamma, precision, bc   as in mhd_create
 *   cuda_stream          a cudaStream_t passed as void* (NULL = the default stream)
 *   cmax_device          DEVICE pointer to one double: receives c_max (fp32 states: the float maximum, widened).
 *                        Written as the reduction produced it: there is no counterpart of mhd_cfl_dt's
 *                        MHD_ENONFINITE here, so test it for finite and > 0 before forming dt = cfl / c_max.
 *   errbuf, errbuf_len   optional HOST buffer for the message of a failure (may be NULL / 0)
 * Does not synchronise: the result is there once work enqueued on `cuda_stream` up to this call has finished.
 * The kernel's scratch (per-block partial maxima and a block counter) is a fixed 262400-byte array inside the library
 * image; every GPU on which libmhd.so's kernels are loaded holds it until the process exits.  Consequences:
 *   - LIMIT: nx*ny*nz <= 2^27 = 134217728 cells (512^3).  Larger grids are refused with MHD_EINVAL and a message;
 *     nothing is launched.
 *   - All calls on one GPU share that array, from any thread, stream or context.  Two calls whose kernels can be in
 *     flight at the same time on one GPU race on it and both results are garbage: keep such calls on one stream, or
 *     order them yourself.  Calls on different GPUs are independent.
 *   - The FIRST call on each device (with that device current) also looks up the array's device address
 *     (cudaGetSymbolAddress, which loads the library's kernels onto the device if nothing has yet).  Make that first
 *     call during start-up, outside any stream capture.
 * The result equals mhd_cfl_dt's c_max of a context holding the same state (same per-cell arithmetic; a maximum does
 * not depend on the order it is taken in).  MHD_EINVAL: NULL pointer, extent < 1, gamma <= 1, unknown enum, too many
 * cells; MHD_ECUDA: a CUDA call failed. */
int mhd_cmax_noalloc(const void* const fields_device[8], int nx, int ny, int nz, double gamma, int precision, int bc,
                     void* cuda_stream, double* cmax_device, char* errbuf, size_t errbuf_len);

/* Number of kernels this context has launched since creation (bench.py's gpu_launches claim). */
long long mhd_launch_count(const mhd_ctx* ctx);

/* Message of the most recent failure on this context ("" if none); valid until the next call on it.
 * For ctx == NULL returns the message of the last failed mhd_create on this thread. */
const char* mhd_last_error(const mhd_ctx* ctx);

/* Library version string, e.g. "mhd-b200 0.1 (sm_100a)". */
const char* mhd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MHD_H_ */
