// mhd_api.cu -- the C ABI of include/mhd.h: context, SoA device buffers, operator sequencing.
// PRODUCT code (CUDA path).  No CPU fallback: every step of the hot path runs in the kernels of
// this directory; if CUDA is unavailable every compute call returns MHD_ECUDA.
#include "../../include/mhd.h"

#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <type_traits>

#include "mhd_generic.cuh"
#include "mhd_yz2.cuh"
#include "mhd_bring.cuh"
#include "mhd_x2.cuh"
#include "mhd_lrev.cuh"
#include "mhd_viz.cuh"

using namespace mhd;

// One whole step (dt kernel + the operator launches of a double sweep) captured as a CUDA graph.  A step leaves
// every ping-pong pointer where it found it (each field is swapped an even number of times), so a graph captured
// at step index s can be replayed at every later step with the same index mod 3, the same pointer assignment,
// the same cfl and the same state of the reduction flags.  For grids of a few thousand to a few million cells
// a step is bound by launch latency (13 launches of a few microseconds each); replaying it as one graph removes
// most of that.
struct StepGraph {
  cudaGraphExec_t exec;
  double cfl;
  void* cur[8];
  long long launches;       // kernel launches inside the graph
  bool acc_valid, fin_valid, acc_dirty;   // flags after the step
};

struct mhd_ctx {
  int n[3];
  double gamma;
  int precision, bc;
  size_t esize;            // bytes per element
  size_t N;                // cells
  size_t field_bytes;      // N*esize rounded up to 256
  // device memory
  void* ws;                // workspace base
  size_t ws_bytes;
  bool owns_ws;
  void* cur[8];            // current state, field order rho,mx,my,mz,E,Bx,By,Bz
  void* alt[8];            // scratch copy (out-of-place operators ping-pong field by field)
  Scalars* sc;             // device scalar block
  double* diag;            // device: 8 sums + divb bits
  cudaStream_t stream;
  bool owns_stream;
  bool stream_set;
  bool has_state;
  bool acc_valid;          // the device accumulator cmax_bits holds c_max of the CURRENT state (fused reduction)
  bool fin_valid;          // sc->cmax holds c_max of the current state
  bool acc_dirty;          // the accumulator may be non-zero (must be zeroed before a new reduction starts)
  long long step_index;
  long long launches;
  // options
  int opt_segment, opt_block, opt_path, opt_xpack, opt_xfuse, opt_brows, opt_tmap;
  // tensor maps of the field buffers (option tmap): one per buffer, box 256 x 1 x 1
  const void* tmap_ptr[16];
  CUtensorMap tmap[16];
  int n_tmap;
  const void* smem_set[48];   // kernels whose dynamic shared-memory limit has been raised on this context's device
  int n_smem_set;
  int opt_fuse;            // fused reverse L_y / L_z and fused middle pair (mhd_lrev.cuh): 0 off, 1 on, 2 middle pair fuses the two B pairs only
  int opt_cmax_reuse;      // 1: mhd_cfl_dt returns the cached c_max when the state has not changed; 0: always reduce
  int opt_graph;           // -1 auto (small grids), 0 never, 1 always: replay whole steps as CUDA graphs
  StepGraph graphs[64];    // one per (step index mod 3, reduction flags, clip)
  int sm_count;
  char err[512];
};

static thread_local char g_create_err[256] = "";

static void drop_graphs(mhd_ctx* c) {
  for (StepGraph& g : c->graphs) {
    if (g.exec) cudaGraphExecDestroy(g.exec);
    g.exec = nullptr;
  }
}

static int fail(mhd_ctx* c, int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  if (c) vsnprintf(c->err, sizeof(c->err), fmt, ap);
  else vsnprintf(g_create_err, sizeof(g_create_err), fmt, ap);
  va_end(ap);
  return code;
}

#define CUDA_TRY(c, expr)                                                                       \
  do {                                                                                          \
    cudaError_t e_ = (expr);                                                                    \
    if (e_ != cudaSuccess) return fail((c), MHD_ECUDA, "%s failed: %s", #expr, cudaGetErrorString(e_)); \
  } while (0)

static size_t round256(size_t x) { return (x + 255) & ~(size_t)255; }
static const size_t kScalarBlock = 1024;   // Scalars + diagnostics scratch

static bool shape_ok(int nx, int ny, int nz, int precision) {
  if (nx < 1 || ny < 1 || nz < 1) return false;
  if (precision != MHD_F32 && precision != MHD_F64) return false;
  if ((double)nx * ny * nz > 4.0e9) return false;
  return true;
}

extern "C" size_t mhd_workspace_bytes(int nx, int ny, int nz, int precision) {
  if (!shape_ok(nx, ny, nz, precision)) return 0;
  const size_t es = precision == MHD_F32 ? 4 : 8;
  const size_t fb = round256((size_t)nx * ny * nz * es);
  return 16 * fb + kScalarBlock;
}

extern "C" const char* mhd_version(void) { return "mhd-b200 0.1 (sm_100a)"; }

extern "C" const char* mhd_last_error(const mhd_ctx* c) { return c ? c->err : g_create_err; }

extern "C" long long mhd_launch_count(const mhd_ctx* c) { return c ? c->launches : 0; }

extern "C" int mhd_create(int nx, int ny, int nz, double gamma, int precision, int bc, mhd_ctx** out) {
  if (!out) return fail(nullptr, MHD_EINVAL, "mhd_create: out is NULL");
  *out = nullptr;
  if (!shape_ok(nx, ny, nz, precision)) return fail(nullptr, MHD_EINVAL, "mhd_create: bad extents or precision");
  if (!(gamma > 1.0)) return fail(nullptr, MHD_EINVAL, "mhd_create: gamma must be > 1");
  if (bc != MHD_BC_PERIODIC && bc != MHD_BC_OUTFLOW) return fail(nullptr, MHD_EINVAL, "mhd_create: unknown bc");
  mhd_ctx* c = new (std::nothrow) mhd_ctx();
  if (!c) return fail(nullptr, MHD_ENOMEM, "mhd_create: out of host memory");
  memset(c, 0, sizeof(*c));
  c->n[0] = nx; c->n[1] = ny; c->n[2] = nz;
  c->gamma = gamma; c->precision = precision; c->bc = bc;
  c->esize = precision == MHD_F32 ? 4 : 8;
  c->N = (size_t)nx * ny * nz;
  c->field_bytes = round256(c->N * c->esize);
  c->opt_segment = -1;   // auto
  c->opt_block = 128;
  c->opt_path = 0;
  c->opt_xpack = 2;
  c->opt_xfuse = 1;
  c->opt_brows = 2;
  c->opt_tmap = 0;
  c->n_tmap = 0;
  c->opt_graph = -1;
  c->opt_cmax_reuse = 1;
  c->opt_fuse = 0;
  c->sm_count = 148;
  *out = c;
  return MHD_OK;
}

static int carve(mhd_ctx* c) {
  char* base = (char*)c->ws;
  for (int f = 0; f < 8; ++f) {
    c->cur[f] = base + (size_t)f * c->field_bytes;
    c->alt[f] = base + (size_t)(8 + f) * c->field_bytes;
  }
  c->sc = (Scalars*)(base + 16 * c->field_bytes);
  c->diag = (double*)(base + 16 * c->field_bytes + 256);
  c->n_tmap = 0;                       // tensor maps are keyed by buffer address: a new workspace invalidates them
  CUDA_TRY(c, cudaMemsetAsync(c->sc, 0, kScalarBlock, c->stream));
  return MHD_OK;
}

static int ensure_ready(mhd_ctx* c) {
  if (!c->stream_set) {
    CUDA_TRY(c, cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking));
    c->owns_stream = true;
    c->stream_set = true;
  }
  if (!c->ws) {
    c->ws_bytes = mhd_workspace_bytes(c->n[0], c->n[1], c->n[2], c->precision);
    cudaError_t e = cudaMalloc(&c->ws, c->ws_bytes);
    if (e != cudaSuccess) {
      c->ws = nullptr;
      return fail(c, e == cudaErrorMemoryAllocation ? MHD_ENOMEM : MHD_ECUDA, "cudaMalloc(%zu) failed: %s", c->ws_bytes,
                  cudaGetErrorString(e));
    }
    c->owns_ws = true;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) == cudaSuccess &&
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
      c->sm_count = sms;
    return carve(c);
  }
  return MHD_OK;
}

extern "C" int mhd_bind(mhd_ctx* c, void* device_workspace, size_t bytes, void* cuda_stream) {
  if (!c) return MHD_EINVAL;
  if (c->has_state || c->ws) return fail(c, MHD_EINVAL, "mhd_bind: must precede mhd_set_state");
  c->stream = (cudaStream_t)cuda_stream;
  c->owns_stream = false;
  c->stream_set = true;
  if (device_workspace) {
    const size_t need = mhd_workspace_bytes(c->n[0], c->n[1], c->n[2], c->precision);
    if (bytes < need) return fail(c, MHD_ENOMEM, "mhd_bind: workspace of %zu bytes < %zu needed", bytes, need);
    if (((size_t)device_workspace & 255) != 0) return fail(c, MHD_ENOMEM, "mhd_bind: workspace not 256-byte aligned");
    c->ws = device_workspace;
    c->ws_bytes = bytes;
    c->owns_ws = false;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) == cudaSuccess &&
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
      c->sm_count = sms;
    return carve(c);
  }
  return MHD_OK;
}

extern "C" int mhd_destroy(mhd_ctx* c) {
  if (!c) return MHD_OK;
  if (c->stream_set) cudaStreamSynchronize(c->stream);
  drop_graphs(c);
  if (c->owns_ws && c->ws) cudaFree(c->ws);
  if (c->owns_stream && c->stream_set) cudaStreamDestroy(c->stream);
  delete c;
  return MHD_OK;
}

extern "C" int mhd_set_state(mhd_ctx* c, const void* const fields[8], int where) {
  if (!c) return MHD_EINVAL;
  if (!fields || (where != MHD_HOST && where != MHD_DEVICE)) return fail(c, MHD_EINVAL, "mhd_set_state: bad argument");
  for (int f = 0; f < 8; ++f)
    if (!fields[f]) return fail(c, MHD_EINVAL, "mhd_set_state: fields[%d] is NULL", f);
  int rc = ensure_ready(c);
  if (rc) return rc;
  const cudaMemcpyKind kind = where == MHD_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
  for (int f = 0; f < 8; ++f) CUDA_TRY(c, cudaMemcpyAsync(c->cur[f], fields[f], c->N * c->esize, kind, c->stream));
  CUDA_TRY(c, cudaMemsetAsync(c->sc, 0, sizeof(Scalars), c->stream));
  // the caller's pointers need not outlive the call (mhd.h): wait for the copies, device sources included
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  c->has_state = true;
  c->acc_valid = c->fin_valid = false;
  return MHD_OK;
}

static int check_poison(mhd_ctx* c, const Scalars& h) {
  if (h.nonfinite) return fail(c, MHD_ENONFINITE, "c_max reduction saw a non-finite or non-positive value (c_max = %g)", h.cmax);
  return MHD_OK;
}

extern "C" int mhd_get_state(mhd_ctx* c, void* const fields[8], int where) {
  if (!c) return MHD_EINVAL;
  if (!fields || (where != MHD_HOST && where != MHD_DEVICE)) return fail(c, MHD_EINVAL, "mhd_get_state: bad argument");
  for (int f = 0; f < 8; ++f)
    if (!fields[f]) return fail(c, MHD_EINVAL, "mhd_get_state: fields[%d] is NULL", f);
  if (!c->has_state) return fail(c, MHD_ENOSTATE, "mhd_get_state: no state set");
  const cudaMemcpyKind kind = where == MHD_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
  for (int f = 0; f < 8; ++f) CUDA_TRY(c, cudaMemcpyAsync(fields[f], c->cur[f], c->N * c->esize, kind, c->stream));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  return MHD_OK;
}

// ---------------------------------------------------------------------------------------------
// operator launches
// ---------------------------------------------------------------------------------------------
template <class real>
static SweepGeom<real> make_geom(const mhd_ctx* c, int d) {
  const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
  const long long stride[3] = {1, c->n[0], (long long)c->n[0] * c->n[1]};
  SweepGeom<real> g;
  g.nd = c->n[d]; g.na = c->n[t1]; g.nb = c->n[t2];
  g.sd = stride[d]; g.sa = stride[t1]; g.sb = stride[t2];
  g.bc = c->bc;
  g.gamma = (real)c->gamma;
  // consecutive threads should walk the transverse axis with the smaller stride (x when d != x)
  g.a_fast = (g.sa < g.sb || g.nb == 1) && g.na > 1 ? 1 : (g.nb > 1 ? 0 : 1);
  // segment length: whole pencils when that already fills the machine, else split
  int seg = c->opt_segment;
  if (seg < 0) {
    const long long pencils = (long long)g.na * g.nb;
    const long long want = (long long)c->sm_count * 2048;      // resident-thread capacity
    seg = g.nd;
    while (seg > 8 && pencils * ((g.nd + seg - 1) / seg) < want) seg = (seg + 1) / 2;
  }
  if (seg == 0 || seg > g.nd) seg = g.nd;
  g.seg = seg;
  g.nseg = (g.nd + seg - 1) / seg;
  return g;
}

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) once per kernel and context (the attribute is per device; a context
// lives on one device), not on every launch
static int want_smem(mhd_ctx* c, const void* kernel, size_t bytes) {
  for (int i = 0; i < c->n_smem_set; ++i)
    if (c->smem_set[i] == kernel) return MHD_OK;
  CUDA_TRY(c, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
  if (c->n_smem_set < (int)(sizeof(c->smem_set) / sizeof(c->smem_set[0]))) c->smem_set[c->n_smem_set++] = kernel;
  return MHD_OK;
}

static void swap_fields(mhd_ctx* c, const int* f, int n) {
  for (int i = 0; i < n; ++i) { void* t = c->cur[f[i]]; c->cur[f[i]] = c->alt[f[i]]; c->alt[f[i]] = t; }
}
static const int kBFields[3] = {5, 6, 7};

// ---- ring marches for sweeps along y and z (mhd_yz2.cuh, mhd_bring.cuh) ------------------------
// tile width in columns: fp32 256 (128 threads, two pencils each) or 128, fp64 128; the last tile of a row may be narrower
// (rows must be a multiple of 16 bytes for the bulk copies), so the width that wastes fewer lanes is taken
static int yz_tile(const mhd_ctx* c) {
  const int nx = c->n[0], ch = c->precision == MHD_F32 ? 4 : 2;
  if (nx % ch != 0) return 0;
  if (c->precision != MHD_F32) return 128;
  const double e256 = (double)nx / (((nx + 255) / 256) * 256), e128 = (double)nx / (((nx + 127) / 128) * 128);
  return e256 + 0.02 >= e128 ? 256 : 128;
}

static bool yz_ok(const mhd_ctx* c, int d) {
  return c->opt_path == 0 && d != 0 && c->n[d] >= 8 && yz_tile(c) != 0 && c->N < ((size_t)1 << 31);
}

// Segment length along the sweep for a march kernel whose blocks cover `pencil_blocks` tiles of the transverse
// plane: more segments fill the last wave of blocks but every segment re-marches `halo` warm-up cells.
// Picks the number of segments that minimises  waves * (segment + halo)  for `slots` co-resident blocks.
static int pick_segment(int nd, long long pencil_blocks, long long slots, int halo) {
  int best_seg = nd;
  double best = 1e300;
  for (int nseg = 1; nseg <= 64 && nd / nseg >= 8; ++nseg) {
    const int seg = ((nd + nseg - 1) / nseg + 3) & ~3;              // multiple of 4 (the marches are unrolled by 4)
    const long long blocks = pencil_blocks * ((nd + seg - 1) / seg);
    const double cost = (double)((blocks + slots - 1) / slots) * (seg + halo);
    if (cost < best * 0.999) { best = cost; best_seg = seg; }
  }
  return best_seg;
}

template <class real>
static YZArgs<real> make_yz(mhd_ctx* c, int d, int tile, int blocks_per_sm, int halo) {
  const int o = 3 - d;                        // the other transverse axis (x is always one of them)
  const int stride[3] = {1, c->n[0], c->n[0] * c->n[1]};
  YZArgs<real> A;
  memset(&A, 0, sizeof(A));
  A.nx = c->n[0]; A.nd = c->n[d]; A.no = c->n[o];
  A.sd = stride[d]; A.so = stride[o];
  A.bc = c->bc;
  A.x_is_t1 = (d == 2) ? 1 : 0;               // z: (t1,t2) = (x,y);  y: (t1,t2) = (z,x)
  A.gamma = (real)c->gamma;
  A.dt = &c->sc->dt;
  int seg = c->opt_segment;
  if (seg < 0) seg = pick_segment(A.nd, (long long)((A.nx + tile - 1) / tile) * A.no, (long long)c->sm_count * blocks_per_sm, halo);
  if (seg == 0 || seg > A.nd) seg = A.nd;
  A.seg = seg;
  return A;
}

// 3-D tensor map (x, y, z) of one field buffer with a box of `tile` x 1 x 1 elements, cached per buffer.  The driver's
// encoder is looked up at run time (the library links the static runtime only).
static int get_tmap(mhd_ctx* c, const void* ptr, int tile, CUtensorMap* out) {
  for (int i = 0; i < c->n_tmap; ++i)
    if (c->tmap_ptr[i] == ptr) { *out = c->tmap[i]; return MHD_OK; }
  typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static encode_fn enc = nullptr;
  if (!enc) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    CUDA_TRY(c, cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q));
    if (!fn || q != cudaDriverEntryPointSuccess) return fail(c, MHD_ECUDA, "cuTensorMapEncodeTiled is not available");
    enc = (encode_fn)fn;
  }
  const cuuint64_t dims[3] = {(cuuint64_t)c->n[0], (cuuint64_t)c->n[1], (cuuint64_t)c->n[2]};
  const cuuint64_t strides[2] = {(cuuint64_t)c->n[0] * c->esize, (cuuint64_t)c->n[0] * c->n[1] * c->esize};
  const cuuint32_t box[3] = {(cuuint32_t)tile, 1, 1}, estr[3] = {1, 1, 1};
  alignas(64) CUtensorMap m;
  const CUresult r = enc(&m, c->precision == MHD_F32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void*>(ptr),
                         dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(c, MHD_ECUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
  if (c->n_tmap < 16) { c->tmap_ptr[c->n_tmap] = ptr; c->tmap[c->n_tmap] = m; c->n_tmap++; }
  *out = m;
  return MHD_OK;
}

template <class real>
static int launch_fluid_yz(mhd_ctx* c, int d, bool want_cmax) {
  constexpr bool f32 = std::is_same<real, float>::value;
  using T = typename std::conditional<f32, f2, real>::type;
  const int t1 = (d + 1) % 3, t2 = (d + 2) % 3, o = 3 - d;
  const int P = yz_tile(c);
  YZArgs<real> A = make_yz<real>(c, d, P, MHD_YZ2_MINB * ((f32 && P == 128) ? 2 : 1), 6);
  const int role[5] = {0, 1 + d, 1 + t1, 1 + t2, 4};
  for (int k = 0; k < 5; ++k) { A.u[k] = (const real*)c->cur[role[k]]; A.uo[k] = (real*)c->alt[role[k]]; }
  A.bd = (const real*)c->cur[5 + d]; A.bx = (const real*)c->cur[5]; A.bo = (const real*)c->cur[5 + o];
  A.cmax_bits = want_cmax ? &c->sc->cmax_bits : nullptr;
  for (int k = 0; k < 5; ++k) A.src[k] = (const char*)A.u[k] - (const char*)A.u[0];
  A.src[5] = (const char*)A.bd - (const char*)A.u[0];
  A.src[6] = (const char*)A.bo - (const char*)A.u[0];
  A.src[7] = (const char*)A.bx - (const char*)A.u[0];
  const dim3 grid((A.nx + P - 1) / P, A.no, (A.nd + A.seg - 1) / A.seg);
  void (*k)(const YZArgs<real>) = nullptr;
  size_t smem = 0;
  constexpr int DR = MHD_YZ2_STAGES;
  const bool xt1 = A.x_is_t1 != 0;
  const bool rag = A.nx % P != 0;
#define MHD_FYZ_PICK(TX_, RAG_)                                                                                          \
  do {                                                                                                                   \
    smem = FluidRing<real, TX_>::smem_bytes(DR);                                                                         \
    k = want_cmax ? (xt1 ? fluid_yz_ring_kernel<real, T, TX_, DR, true, true, RAG_> : fluid_yz_ring_kernel<real, T, TX_, DR, false, true, RAG_>) \
                  : (xt1 ? fluid_yz_ring_kernel<real, T, TX_, DR, true, false, RAG_> : fluid_yz_ring_kernel<real, T, TX_, DR, false, false, RAG_>); \
  } while (0)
  if (P == 256) {
    if constexpr (f32) { if (rag) MHD_FYZ_PICK(256, true); else MHD_FYZ_PICK(256, false); }
  } else {
    if (rag) MHD_FYZ_PICK(128, true); else MHD_FYZ_PICK(128, false);
  }
#undef MHD_FYZ_PICK
  if constexpr (f32) {
    if (c->opt_tmap && P == 256 && !rag) {      // option tmap: the nine row copies of a stage as tensor-map TMA (UTMALDG)
      alignas(64) FluidMaps M;
      int rcm;
      for (int q = 0; q < 5; ++q) if ((rcm = get_tmap(c, A.u[q], 256, &M.m[q]))) return rcm;
      if ((rcm = get_tmap(c, A.bd, 256, &M.m[5])) || (rcm = get_tmap(c, A.bo, 256, &M.m[6])) || (rcm = get_tmap(c, A.bx, 256, &M.m[7]))) return rcm;
      void (*kt)(const YZArgs<real>, const FluidMaps) =
          want_cmax ? (xt1 ? fluid_yz_ring_tm_kernel<real, T, 256, DR, true, true> : fluid_yz_ring_tm_kernel<real, T, 256, DR, false, true>)
                    : (xt1 ? fluid_yz_ring_tm_kernel<real, T, 256, DR, true, false> : fluid_yz_ring_tm_kernel<real, T, 256, DR, false, false>);
      const size_t smem_t = FluidRing<real, 256, true>::smem_bytes(DR);
      if ((rcm = want_smem(c, (const void*)kt, smem_t))) return rcm;
      kt<<<grid, 256 / PackOf<T>::L, smem_t, c->stream>>>(A, M);
      c->launches++;
      CUDA_TRY(c, cudaGetLastError());
      swap_fields(c, role, 5);
      return MHD_OK;
    }
  }
  int rc = want_smem(c, (const void*)k, smem);
  if (rc) return rc;
  k<<<grid, P / PackOf<T>::L, smem, c->stream>>>(A);
  c->launches++;
  CUDA_TRY(c, cudaGetLastError());
  swap_fields(c, role, 5);
  return MHD_OK;
}

template <class real>
static int launch_bpair_yz(mhd_ctx* c, int d, int t2_first) {
  constexpr bool f32 = std::is_same<real, float>::value;
  using T = typename std::conditional<f32, f2, real>::type;
  const int o = 3 - d;
  const int W = yz_tile(c);
  // brows = 2: two rows o, o+1 per thread (bpair_ring2_kernel): fp32, even extent along o
  const bool two = f32 && c->opt_brows == 2 && c->n[o] % 2 == 0;
  YZArgs<real> A = make_yz<real>(c, d, W, two ? 2 : MHD_BRING_MINB, 8);
  if (two) {                                   // a block covers two rows: half as many pencil blocks
    int seg = c->opt_segment;
    if (seg < 0) seg = pick_segment(A.nd, (long long)((A.nx + W - 1) / W) * (A.no / 2), (long long)c->sm_count * (W == 256 ? 2 : 4), 8);
    if (seg == 0 || seg > A.nd) seg = A.nd;
    A.seg = seg;
  }
  A.u[0] = (const real*)c->cur[0]; A.u[1] = (const real*)c->cur[1 + d];
  A.bd = (const real*)c->cur[5 + d]; A.bx = (const real*)c->cur[5]; A.bo = (const real*)c->cur[5 + o];
  A.bdo = (real*)c->alt[5 + d]; A.bxo = (real*)c->alt[5]; A.boo = (real*)c->alt[5 + o];
  A.t2_first = t2_first;
  A.src[0] = 0;
  A.src[1] = (const char*)A.u[1] - (const char*)A.u[0];
  A.src[5] = (const char*)A.bd - (const char*)A.u[0];
  A.src[6] = (const char*)A.bo - (const char*)A.u[0];
  A.src[7] = (const char*)A.bx - (const char*)A.u[0];
  const dim3 grid((A.nx + W - 1) / W, two ? A.no / 2 : A.no, (A.nd + A.seg - 1) / A.seg);
  constexpr int D = MHD_BRING_STAGES;
  void (*k)(const YZArgs<real>) = nullptr;
  size_t smem = 0;
  const bool rag = A.nx % W != 0;
  if (two) {
    if constexpr (f32) {
      if (W == 256) { k = rag ? bpair_ring2_kernel<256, MHD_BRING2_STAGES, true> : bpair_ring2_kernel<256, MHD_BRING2_STAGES, false>; smem = BRowRing2<real, 256>::smem_bytes(MHD_BRING2_STAGES); }
      else          { k = rag ? bpair_ring2_kernel<128, MHD_BRING2_STAGES, true> : bpair_ring2_kernel<128, MHD_BRING2_STAGES, false>; smem = BRowRing2<real, 128>::smem_bytes(MHD_BRING2_STAGES); }
    }
  } else if (W == 256) {
    if constexpr (f32) { k = rag ? bpair_ring_kernel<real, T, 256, D, true> : bpair_ring_kernel<real, T, 256, D, false>; smem = BRowRing<real, 256>::smem_bytes(D); }
  } else { k = rag ? bpair_ring_kernel<real, T, 128, D, true> : bpair_ring_kernel<real, T, 128, D, false>; smem = BRowRing<real, 128>::smem_bytes(D); }
  int rc = want_smem(c, (const void*)k, smem);
  if (rc) return rc;
  k<<<grid, W / PackOf<T>::L, smem, c->stream>>>(A);
  c->launches++;
  CUDA_TRY(c, cudaGetLastError());
  swap_fields(c, kBFields, 3);
  return MHD_OK;
}

// ---- sweeps along x and the fused reverse L_x (mhd_x2.cuh) ------------------------------------------------------
// kind: 0 fluid_x, 1 B pair, 2 reverse L_x in one pass (B pair then fluid)
template <class real>
static bool x2_ok(const mhd_ctx* c, int kind) {
  constexpr bool f32 = std::is_same<real, float>::value;
  const int V = VecOf<real>::V;
  // outflow: one row per thread with 4 clamped ghost cells on either side of the row (mhd_x2.cuh ghost_fix); the fused
  // reverse L_x does not exist there (its fluid stage would read the B pair's ghost values instead of the clamped outputs)
  const bool out = c->bc != MHD_BC_PERIODIC;
  if (out && (kind == 2 || c->n[0] < 8)) return false;
  if (c->opt_path != 0 || c->n[0] % V != 0 || c->n[0] / V + (out ? 2 * (4 / V) : 0) > X2Block<real>::NT_MAX ||
      c->n[2] > 65535 || c->N >= ((size_t)1 << 31))
    return false;
  // xfuse: 0 never | 1 fp32 only (default; in fp64 the fused kernel is slower than the pair) | 2 always | 3 fp32, packed
  if (kind == 2) return c->opt_xfuse == 2 || ((c->opt_xfuse == 1 || c->opt_xfuse == 3) && f32);
  return true;
}

template <class real>
static int launch_x2(mhd_ctx* c, int kind, int t2_first, bool want_cmax) {
  constexpr bool f32 = std::is_same<real, float>::value;
  using T2 = typename std::conditional<f32, f2, real>::type;
  // xpack: 1 two rows per thread in packed f2 arithmetic (fp32, even ny) | 2 one row per thread (default) | 3 packed fluid_x only
  // measured at 512^3 fp32: fluid_x one row per thread at six blocks per SM 1.21 ms, packed (two rows per thread,
  // three blocks per SM) 1.23; B pair one row per thread 0.89 ms, packed 1.14: the x kernels want occupancy
  const bool out = c->bc != MHD_BC_PERIODIC;
  const bool pack = !out && f32 && c->n[1] % 2 == 0 && c->n[0] / VecOf<real>::V <= X2Block<real>::NT && (c->opt_xpack == 1 || (c->opt_xpack == 3 && kind == 0) || (kind == 2 && c->opt_xfuse == 3));
  const int V = VecOf<real>::V, L = pack ? 2 : 1;
  XArgs<real> A;
  memset(&A, 0, sizeof(A));
  A.nx = c->n[0]; A.ny = c->n[1]; A.nz = c->n[2];
  A.ghost = out ? 4 / V : 0;
  A.tpr = A.nx / V + 2 * A.ghost;
  A.tpr_shift = -1;
  for (int b = 0; b < 11; ++b) if ((1 << b) == A.tpr) A.tpr_shift = b;
  // block size: the smallest of NT, 2 NT, 4 NT threads that holds a whole row (packed variants: NT only)
  constexpr int NT0 = X2Block<real>::NT;
  const int NT = A.tpr <= NT0 ? NT0 : (A.tpr <= 2 * NT0 ? 2 * NT0 : 4 * NT0);
  A.one = (real)1;
  A.rpb = NT / A.tpr;
  const int gpp = A.ny / L;                          // row groups per plane
  if (A.rpb > gpp) A.rpb = gpp;
  A.gamma = (real)c->gamma;
  A.dt = &c->sc->dt;
  const int block = A.tpr * A.rpb;
  const dim3 grid((unsigned)((gpp + A.rpb - 1) / A.rpb), (unsigned)A.nz);
  for (int k = 0; k < 5; ++k) { A.u[k] = (const real*)c->cur[k]; A.uo[k] = (real*)c->alt[k]; }
  A.bx = (const real*)c->cur[5]; A.by = (const real*)c->cur[6]; A.bz = (const real*)c->cur[7];
  A.bxo = (real*)c->alt[5]; A.byo = (real*)c->alt[6]; A.bzo = (real*)c->alt[7];
  A.t2_first = t2_first;
  A.cmax_bits = want_cmax ? &c->sc->cmax_bits : nullptr;
  void (*k)(const XArgs<real>) = nullptr;
  const size_t slots = kind == 1 ? 24 : 35;
  if (pack) {
    if constexpr (f32) k = kind == 0 ? fluid_x2_kernel<real, T2> : (kind == 1 ? bpair_x2_kernel<real, T2> : lrev_x2_kernel<real, T2>);
  } else if (out) {
    if (NT == NT0) k = kind == 0 ? fluid_x2_kernel<real, real, NT0, true> : bpair_x2_kernel<real, real, NT0, true>;
    else if (NT == 2 * NT0) k = kind == 0 ? fluid_x2_kernel<real, real, 2 * NT0, true> : bpair_x2_kernel<real, real, 2 * NT0, true>;
    else if constexpr (4 * NT0 <= X2Block<real>::NT_MAX) k = kind == 0 ? fluid_x2_kernel<real, real, 4 * NT0, true> : bpair_x2_kernel<real, real, 4 * NT0, true>;
  } else if (NT == NT0) {
    k = kind == 0 ? fluid_x2_kernel<real, real> : (kind == 1 ? bpair_x2_kernel<real, real> : lrev_x2_kernel<real, real>);
  } else if (NT == 2 * NT0) {
    k = kind == 0 ? fluid_x2_kernel<real, real, 2 * NT0> : (kind == 1 ? bpair_x2_kernel<real, real, 2 * NT0> : lrev_x2_kernel<real, real, 2 * NT0>);
  } else {
    if constexpr (4 * NT0 <= X2Block<real>::NT_MAX)
      k = kind == 0 ? fluid_x2_kernel<real, real, 4 * NT0> : (kind == 1 ? bpair_x2_kernel<real, real, 4 * NT0> : lrev_x2_kernel<real, real, 4 * NT0>);
  }
  if (!k) return fail(c, MHD_EINVAL, "launch_x2: no kernel for %d threads per row", A.tpr);
  const size_t smem = slots * NT * (pack ? 2 : 1) * sizeof(real);
  int rc = want_smem(c, (const void*)k, 35 * (size_t)NT * (pack ? 2 : 1) * sizeof(real));
  if (rc) return rc;
  k<<<grid, block, smem, c->stream>>>(A);
  c->launches++;
  CUDA_TRY(c, cudaGetLastError());
  static const int kUFields[5] = {0, 1, 2, 3, 4};
  if (kind != 1) swap_fields(c, kUFields, 5);
  if (kind != 0) swap_fields(c, kBFields, 3);
  return MHD_OK;
}

// ---- fused reverse L_d and fused middle pair for d = y, z (mhd_lrev.cuh) ---------------------------------------------
// np: number of B passes (1: reverse L_d; 2: forward B pair + reverse B pair), fl: followed by the fluid update
static bool lrev_ok(const mhd_ctx* c, int d) {
  const int tile = c->precision == MHD_F32 ? 128 : 64;
  return c->opt_fuse && c->opt_path == 0 && d != 0 && c->bc == MHD_BC_PERIODIC && c->n[d] >= 32 && c->n[0] % tile == 0 &&
         c->N < ((size_t)1 << 31);
}

template <class real>
static int launch_lrev(mhd_ctx* c, int d, int np, bool fl, bool want_cmax) {
  constexpr bool f32 = std::is_same<real, float>::value;
  using T = typename std::conditional<f32, f2, real>::type;
  constexpr int TXB = f32 ? 128 : 64;
  const int t1 = (d + 1) % 3, t2 = (d + 2) % 3, o = 3 - d;
  const int stride[3] = {1, c->n[0], c->n[0] * c->n[1]};
  LRevArgs<real> A;
  memset(&A, 0, sizeof(A));
  const int role[5] = {0, 1 + d, 1 + t1, 1 + t2, 4};
  for (int k = 0; k < 5; ++k) { A.u[k] = (const real*)c->cur[role[k]]; A.uo[k] = (real*)c->alt[role[k]]; }
  A.bd = (const real*)c->cur[5 + d]; A.bx = (const real*)c->cur[5]; A.bo = (const real*)c->cur[5 + o];
  A.bdo = (real*)c->alt[5 + d]; A.bxo = (real*)c->alt[5]; A.boo = (real*)c->alt[5 + o];
  A.dt = &c->sc->dt;
  A.cmax_bits = want_cmax ? &c->sc->cmax_bits : nullptr;
  A.nx = c->n[0]; A.nd = c->n[d]; A.no = c->n[o];
  A.sd = stride[d]; A.so = stride[o];
  A.x_is_t1 = (d == 2) ? 1 : 0;
  A.t2_first[0] = np == 2 ? 0 : 1;            // middle pair: the forward operator's B pair comes first
  A.t2_first[1] = 1;
  A.gamma = (real)c->gamma;
  const int minb = (np == 2 && fl) ? 2 : 3;
  const int halo = 8 * np + (fl ? 7 : 0);
  A.seg = c->opt_segment;
  if (A.seg < 0) A.seg = pick_segment(A.nd, ((long long)A.nx / TXB) * A.no, (long long)c->sm_count * minb, halo);
  if (A.seg == 0 || A.seg > A.nd) A.seg = A.nd;
  if (A.seg < 16) A.seg = A.nd < 16 ? A.nd : 16;
  const dim3 grid(A.nx / TXB, A.no, (A.nd + A.seg - 1) / A.seg);
  void (*k)(const LRevArgs<real>) = nullptr;
  size_t smem = 0;
  const bool xt1 = A.x_is_t1 != 0;
#define MHD_LREV_PICK(NP_, FL_)                                                                                        \
  do {                                                                                                                 \
    smem = LRevLayout<real, TXB, NP_, FL_>::smem_bytes();                                                              \
    k = want_cmax ? (xt1 ? lrev_ring_kernel<real, T, TXB, NP_, FL_, true, true> : lrev_ring_kernel<real, T, TXB, NP_, FL_, false, true>) \
                  : (xt1 ? lrev_ring_kernel<real, T, TXB, NP_, FL_, true, false> : lrev_ring_kernel<real, T, TXB, NP_, FL_, false, false>); \
  } while (0)
  if (np == 1) MHD_LREV_PICK(1, true);
  else if (fl) MHD_LREV_PICK(2, true);
  else { smem = LRevLayout<real, TXB, 2, false>::smem_bytes(); k = lrev_ring_kernel<real, T, TXB, 2, false, false, false>; }
#undef MHD_LREV_PICK
  const int nthr = (np + (fl ? 1 : 0)) * (TXB / PackOf<T>::L);
  int rc = want_smem(c, (const void*)k, smem);
  if (rc) return rc;
  k<<<grid, nthr, smem, c->stream>>>(A);
  c->launches++;
  CUDA_TRY(c, cudaGetLastError());
  swap_fields(c, kBFields, 3);
  if (fl) swap_fields(c, role, 5);
  return MHD_OK;
}

// want_cmax: this is the last operator of a step; fuse the c_max reduction of the NEXT step into it.
// *fused reports whether the kernel that ran could do so.
template <class real>
static int launch_fluid(mhd_ctx* c, int d, bool want_cmax = false, bool* fused = nullptr) {
  const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
  if (fused) *fused = false;
  if (c->n[d] == 1) return MHD_OK;   // both face fluxes of the only cell are identical: exact no-op (R10)
  if (yz_ok(c, d)) { if (fused) *fused = want_cmax; return launch_fluid_yz<real>(c, d, want_cmax); }
  if (d == 0 && x2_ok<real>(c, 0)) { if (fused) *fused = want_cmax; return launch_x2<real>(c, 0, 0, want_cmax); }
  FluidArgs<real> A;
  const int role[5] = {0, 1 + d, 1 + t1, 1 + t2, 4};
  for (int k = 0; k < 5; ++k) { A.u[k] = (const real*)c->cur[role[k]]; A.uo[k] = (real*)c->alt[role[k]]; }
  A.bd = (const real*)c->cur[5 + d]; A.bt1 = (const real*)c->cur[5 + t1]; A.bt2 = (const real*)c->cur[5 + t2];
  A.dt = &c->sc->dt;
  A.g = make_geom<real>(c, d);
  const long long threads = (long long)A.g.na * A.g.nb * A.g.nseg;
  const int block = c->opt_block;
  const unsigned grid = (unsigned)((threads + block - 1) / block);
  fluid_march_kernel<real><<<grid, block, 0, c->stream>>>(A);
  c->launches++;
  CUDA_TRY(c, cudaGetLastError());
  for (int k = 0; k < 5; ++k) { void* t = c->cur[role[k]]; c->cur[role[k]] = c->alt[role[k]]; c->alt[role[k]] = t; }
  return MHD_OK;
}

template <class real>
static int launch_bpair(mhd_ctx* c, int d, int t2_first) {
  const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
  if (yz_ok(c, d)) return launch_bpair_yz<real>(c, d, t2_first);
  if (d == 0 && x2_ok<real>(c, 1)) return launch_x2<real>(c, 1, t2_first, false);
  BPairArgs<real> A;
  A.rho = (const real*)c->cur[0]; A.md = (const real*)c->cur[1 + d];
  A.bd = (const real*)c->cur[5 + d]; A.bt1 = (const real*)c->cur[5 + t1]; A.bt2 = (const real*)c->cur[5 + t2];
  A.bdo = (real*)c->alt[5 + d]; A.bt1o = (real*)c->alt[5 + t1]; A.bt2o = (real*)c->alt[5 + t2];
  A.dt = &c->sc->dt;
  A.t2_first = t2_first;
  A.g = make_geom<real>(c, d);
  if (c->n[d] == 1 && c->opt_path == 0) {      // extent 1 along the sweep: only the constraint term acts (bpair_flat_kernel)
    A.g.seg = 1; A.g.nseg = 1;
    const long long cells = (long long)A.g.na * A.g.nb;
    bpair_flat_kernel<real><<<(unsigned)((cells + 255) / 256), 256, 0, c->stream>>>(A);
    c->launches++;
    CUDA_TRY(c, cudaGetLastError());
    void* t = c->cur[5 + d]; c->cur[5 + d] = c->alt[5 + d]; c->alt[5 + d] = t;
    return MHD_OK;
  }
  const long long threads = (long long)A.g.na * A.g.nb * A.g.nseg;
  const int block = c->opt_block;
  const unsigned grid = (unsigned)((threads + block - 1) / block);
  bpair_march_kernel<real><<<grid, block, 0, c->stream>>>(A);
  c->launches++;
  CUDA_TRY(c, cudaGetLastError());
  for (int f = 5; f < 8; ++f) { void* t = c->cur[f]; c->cur[f] = c->alt[f]; c->alt[f] = t; }
  return MHD_OK;
}

template <class real>
static int launch_cfl(mhd_ctx* c) {
  CflArgs<real> A;
  for (int f = 0; f < 8; ++f) A.f[f] = (const real*)c->cur[f];
  A.nx = c->n[0]; A.ny = c->n[1]; A.nz = c->n[2]; A.bc = c->bc;
  A.gamma = (real)c->gamma;
  A.cmax_bits = &c->sc->cmax_bits;
  const int block = 256;
  long long want = ((long long)c->N + block - 1) / block;
  const long long cap = (long long)c->sm_count * 8;
  const unsigned grid = (unsigned)(want < cap ? want : cap);
  cfl_kernel<real><<<grid, block, 0, c->stream>>>(A);
  c->launches++;
  CUDA_TRY(c, cudaGetLastError());
  return MHD_OK;
}

#define BY_PRECISION(c, CALL32, CALL64) ((c)->precision == MHD_F32 ? (CALL32) : (CALL64))

static int arm_accumulator(mhd_ctx* c) {
  if (c->acc_dirty) {
    CUDA_TRY(c, cudaMemsetAsync(&c->sc->cmax_bits, 0, sizeof(unsigned long long), c->stream));
    c->acc_dirty = false;
  }
  return MHD_OK;
}

static int sweep(mhd_ctx* c, int d, bool reverse, bool want_cmax = false, bool* fused = nullptr) {
  int rc;
  c->acc_valid = c->fin_valid = false;          // the state changes
  if (!reverse) {
    if ((rc = BY_PRECISION(c, launch_fluid<float>(c, d), launch_fluid<double>(c, d)))) return rc;
    return BY_PRECISION(c, launch_bpair<float>(c, d, 0), launch_bpair<double>(c, d, 0));
  }
  if (d == 0 && c->n[0] > 1 && BY_PRECISION(c, x2_ok<float>(c, 2), x2_ok<double>(c, 2))) {   // B pair + fluid in one pass
    if (fused) *fused = want_cmax;
    return BY_PRECISION(c, launch_x2<float>(c, 2, 1, want_cmax), launch_x2<double>(c, 2, 1, want_cmax));
  }
  if (c->n[d] > 1 && lrev_ok(c, d)) {                            // reverse L_y / L_z: B pair + fluid in one pass (mhd_lrev.cuh)
    if (fused) *fused = want_cmax;
    return BY_PRECISION(c, launch_lrev<float>(c, d, 1, true, want_cmax), launch_lrev<double>(c, d, 1, true, want_cmax));
  }
  if ((rc = BY_PRECISION(c, launch_bpair<float>(c, d, 1), launch_bpair<double>(c, d, 1)))) return rc;
  return BY_PRECISION(c, launch_fluid<float>(c, d, want_cmax, fused), launch_fluid<double>(c, d, want_cmax, fused));
}

// The middle pair of a step: forward L_d followed by reverse L_d (eqs (23)-(25) PAPER.md:164-170: every step's third and
// fourth operator share a direction) = fluid_d, B pair, B pair (t2 first), fluid_d.  For d = y, z the last three run as ONE
// kernel (fuse = 2: the two B pairs only).
static int middle_pair(mhd_ctx* c, int d, bool want_cmax = false, bool* fused = nullptr) {
  int rc;
  if (c->n[d] > 1 && lrev_ok(c, d)) {
    c->acc_valid = c->fin_valid = false;
    if ((rc = BY_PRECISION(c, launch_fluid<float>(c, d), launch_fluid<double>(c, d)))) return rc;
    if (c->opt_fuse == 2) {
      if ((rc = BY_PRECISION(c, launch_lrev<float>(c, d, 2, false, false), launch_lrev<double>(c, d, 2, false, false)))) return rc;
      return BY_PRECISION(c, launch_fluid<float>(c, d, want_cmax, fused), launch_fluid<double>(c, d, want_cmax, fused));
    }
    if (fused) *fused = want_cmax;
    return BY_PRECISION(c, launch_lrev<float>(c, d, 2, true, want_cmax), launch_lrev<double>(c, d, 2, true, want_cmax));
  }
  if ((rc = sweep(c, d, false))) return rc;
  return sweep(c, d, true, want_cmax, fused);
}

// one double sweep, eqs (23)-(25) PAPER.md:164-170
static int double_sweep(mhd_ctx* c) {
  static const int order[3][3] = {{0, 1, 2}, {2, 0, 1}, {1, 2, 0}};
  const int* o = order[((c->step_index % 3) + 3) % 3];
  int rc;
  bool fused = false;
  if ((rc = arm_accumulator(c))) return rc;
  for (int i = 0; i < 2; ++i) if ((rc = sweep(c, o[i], false))) return rc;
  if ((rc = middle_pair(c, o[2]))) return rc;
  // the last operator of the step (fluid of the reverse L along o[0]) also reduces c_max of the new
  // state, so the next step needs no separate pass over the 8 fields
  for (int i = 1; i >= 0; --i) if ((rc = sweep(c, o[i], true, i == 0, &fused))) return rc;
  c->acc_valid = fused;
  if (fused) c->acc_dirty = true;
  c->step_index++;
  return MHD_OK;
}

static int read_scalars(mhd_ctx* c, Scalars* h) {
  CUDA_TRY(c, cudaMemcpyAsync(h, c->sc, sizeof(Scalars), cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  return MHD_OK;
}

// make sc->cmax / sc->dt current: run the reduction only if no fused one is pending
static int refresh_dt(mhd_ctx* c, double cfl, int advance, int clip = 0) {
  int reuse = 0;
  if (c->fin_valid && (c->opt_cmax_reuse || advance)) reuse = 1;
  else if (!c->acc_valid) {
    int rc = arm_accumulator(c);
    if (rc) return rc;
    if ((rc = BY_PRECISION(c, launch_cfl<float>(c), launch_cfl<double>(c)))) return rc;
    c->acc_dirty = true;
  }
  dt_from_cmax_kernel<<<1, 1, 0, c->stream>>>(c->sc, cfl, advance, reuse, clip);
  c->launches++;
  CUDA_TRY(c, cudaGetLastError());
  if (!reuse) c->acc_dirty = false;            // finalising re-arms the accumulator
  c->acc_valid = false;
  c->fin_valid = true;
  return MHD_OK;
}

static bool graphs_wanted(const mhd_ctx* c) {
  // stream capture is not permitted on the legacy default stream (mhd_bind with a NULL stream) nor on the
  // per-thread default stream: launch the kernels directly there
  if (c->stream == nullptr || c->stream == cudaStreamLegacy || c->stream == cudaStreamPerThread) return false;
  if (c->opt_graph >= 0) return c->opt_graph != 0;
  return c->N <= ((size_t)1 << 22);
}

// one step: c_max -> dt (kept on the device) -> six L_i, directly or as a replayed CUDA graph
static int step_once(mhd_ctx* c, double cfl, int clip) {
  int rc;
  if (!graphs_wanted(c)) {
    if ((rc = refresh_dt(c, cfl, 1, clip))) return rc;
    return double_sweep(c);
  }
  const int key = (int)(((c->step_index % 3) + 3) % 3) | (c->acc_valid ? 4 : 0) | (c->fin_valid ? 8 : 0) |
                  (c->acc_dirty ? 16 : 0) | (clip ? 32 : 0);
  StepGraph& g = c->graphs[key];
  bool hit = g.exec != nullptr && g.cfl == cfl;
  for (int f = 0; hit && f < 8; ++f) hit = g.cur[f] == c->cur[f];
  if (!hit) {
    if (g.exec) { cudaGraphExecDestroy(g.exec); g.exec = nullptr; }
    const long long step0 = c->step_index, launches0 = c->launches;
    void* cur0[8];
    memcpy(cur0, c->cur, sizeof(cur0));
    CUDA_TRY(c, cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
    rc = refresh_dt(c, cfl, 1, clip);
    if (!rc) rc = double_sweep(c);
    cudaGraph_t graph = nullptr;
    const cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
    if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
    if (e != cudaSuccess) return fail(c, MHD_ECUDA, "cudaStreamEndCapture failed: %s", cudaGetErrorString(e));
    const cudaError_t e2 = cudaGraphInstantiate(&g.exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e2 != cudaSuccess) { g.exec = nullptr; return fail(c, MHD_ECUDA, "cudaGraphInstantiate failed: %s", cudaGetErrorString(e2)); }
    for (int f = 0; f < 8; ++f)
      if (c->cur[f] != cur0[f]) {          // cannot happen (even number of swaps per field); never replay such a graph
        cudaGraphExecDestroy(g.exec); g.exec = nullptr;
        return fail(c, MHD_ECUDA, "internal: a step did not restore the ping-pong pointers");
      }
    g.cfl = cfl;
    memcpy(g.cur, cur0, sizeof(cur0));
    g.launches = c->launches - launches0;
    g.acc_valid = c->acc_valid; g.fin_valid = c->fin_valid; g.acc_dirty = c->acc_dirty;
    c->step_index = step0; c->launches = launches0;   // the capture recorded the work; the launch below does it
  }
  CUDA_TRY(c, cudaGraphLaunch(g.exec, c->stream));
  c->acc_valid = g.acc_valid; c->fin_valid = g.fin_valid; c->acc_dirty = g.acc_dirty;
  c->launches += g.launches;
  c->step_index++;
  return MHD_OK;
}

extern "C" int mhd_cfl_dt(mhd_ctx* c, double cfl, double* dt_out, double* cmax_out) {
  if (!c) return MHD_EINVAL;
  if (!(cfl > 0.0) || !dt_out) return fail(c, MHD_EINVAL, "mhd_cfl_dt: bad argument");
  if (!c->has_state) return fail(c, MHD_ENOSTATE, "mhd_cfl_dt: no state set");
  int rc = refresh_dt(c, cfl, 0);
  if (rc) return rc;
  Scalars h;
  if ((rc = read_scalars(c, &h))) return rc;
  *dt_out = h.dt;
  if (cmax_out) *cmax_out = h.cmax;
  return check_poison(c, h);
}

extern "C" int mhd_step(mhd_ctx* c, int n, double cfl, double* t_advanced) {
  if (!c) return MHD_EINVAL;
  if (n < 0 || !(cfl > 0.0)) return fail(c, MHD_EINVAL, "mhd_step: bad argument");
  if (!c->has_state) return fail(c, MHD_ENOSTATE, "mhd_step: no state set");
  int rc;
  reset_call_kernel<<<1, 1, 0, c->stream>>>(c->sc);
  c->launches++;
  for (int it = 0; it < n; ++it)
    if ((rc = step_once(c, cfl, 0))) return rc;
  CUDA_TRY(c, cudaGetLastError());
  if (t_advanced) {
    Scalars h;
    if ((rc = read_scalars(c, &h))) return rc;
    *t_advanced = h.t_call;
    return check_poison(c, h);
  }
  return MHD_OK;
}

// The flow loop of PAPER.md:233-243 with the stop test on the device.  The paper reads
// dt back to the host every step; here dt, t and the clipping of the last step stay in the
// scalar block, the host enqueues batches of steps sized from the last dt so that a batch cannot pass t_end
// unless dt grows by more than 10 % inside it (steps enqueued past t_end run with dt = 0 and change nothing),
// and reads (t, steps) back once per batch.
extern "C" int mhd_run_until(mhd_ctx* c, double t_end, double cfl, long long max_steps, long long* steps_done,
                             double* t_reached) {
  if (!c) return MHD_EINVAL;
  if (!(cfl > 0.0) || max_steps < 0 || !(t_end == t_end)) return fail(c, MHD_EINVAL, "mhd_run_until: bad argument");
  if (!c->has_state) return fail(c, MHD_ENOSTATE, "mhd_run_until: no state set");
  int rc;
  Scalars h;
  begin_run_kernel<<<1, 1, 0, c->stream>>>(c->sc, t_end);
  c->launches++;
  if ((rc = refresh_dt(c, cfl, 0))) return rc;          // first dt estimate (the first step reuses this c_max)
  if ((rc = read_scalars(c, &h))) return rc;
  if ((rc = check_poison(c, h))) return rc;
  const long long step0 = c->step_index;
  long long done = 0;
  double dt_est = h.dt;
  while (h.t_total < t_end && done < max_steps) {
    const double est = (t_end - h.t_total) / (2.0 * dt_est);
    long long batch = est < 4.0e9 ? (long long)(0.9 * est) : 4000000000ll;
    if (batch < 1) batch = 1;
    if (batch > 512) batch = 512;
    if (batch > max_steps - done) batch = max_steps - done;
    for (long long it = 0; it < batch; ++it)
      if ((rc = step_once(c, cfl, 1))) return rc;
    if ((rc = read_scalars(c, &h))) return rc;
    c->step_index = step0 + h.steps_real;               // steps enqueued past t_end did nothing: do not count them
    if ((rc = check_poison(c, h))) return rc;
    done = h.steps_real;
    dt_est = h.dt_last > 0.0 ? h.dt_last : dt_est;
  }
  if (steps_done) *steps_done = done;
  if (t_reached) *t_reached = h.t_total;
  return MHD_OK;
}

extern "C" int mhd_step_fixed(mhd_ctx* c, int n, double dt) {
  if (!c) return MHD_EINVAL;
  if (n < 0 || !(dt > 0.0)) return fail(c, MHD_EINVAL, "mhd_step_fixed: bad argument");
  if (!c->has_state) return fail(c, MHD_ENOSTATE, "mhd_step_fixed: no state set");
  set_dt_kernel<<<1, 1, 0, c->stream>>>(c->sc, dt, n);
  c->launches++;
  int rc;
  for (int it = 0; it < n; ++it)
    if ((rc = double_sweep(c))) return rc;
  CUDA_TRY(c, cudaGetLastError());
  return MHD_OK;
}

extern "C" int mhd_apply(mhd_ctx* c, int op, int d, int reverse, double dt) {
  if (!c) return MHD_EINVAL;
  if (d < 0 || d > 2 || !(dt > 0.0)) return fail(c, MHD_EINVAL, "mhd_apply: bad argument");
  if (!c->has_state) return fail(c, MHD_ENOSTATE, "mhd_apply: no state set");
  set_dt_kernel<<<1, 1, 0, c->stream>>>(c->sc, dt, 0);
  c->launches++;
  c->acc_valid = c->fin_valid = false;
  switch (op) {
    case MHD_OP_FLUID: return BY_PRECISION(c, launch_fluid<float>(c, d), launch_fluid<double>(c, d));
    case MHD_OP_BPAIR:
      return BY_PRECISION(c, launch_bpair<float>(c, d, reverse ? 1 : 0), launch_bpair<double>(c, d, reverse ? 1 : 0));
    case MHD_OP_SWEEP_FORWARD: return sweep(c, d, false);
    case MHD_OP_SWEEP_REVERSE: return sweep(c, d, true);
    case MHD_OP_MIDDLE_PAIR: return middle_pair(c, d);
    default: return fail(c, MHD_EINVAL, "mhd_apply: unknown operator %d", op);
  }
}

extern "C" int mhd_get_step_index(mhd_ctx* c, long long* s) {
  if (!c || !s) return MHD_EINVAL;
  *s = c->step_index;
  return MHD_OK;
}

extern "C" int mhd_set_step_index(mhd_ctx* c, long long s) {
  if (!c) return MHD_EINVAL;
  c->step_index = s;
  return MHD_OK;
}

extern "C" int mhd_get_time(mhd_ctx* c, double* t) {
  if (!c || !t) return MHD_EINVAL;
  if (!c->has_state) return fail(c, MHD_ENOSTATE, "mhd_get_time: no state set");
  Scalars h;
  int rc = read_scalars(c, &h);
  if (rc) return rc;
  *t = h.t_total;
  return MHD_OK;
}

extern "C" int mhd_diagnostics(mhd_ctx* c, double sums[8], double* max_abs_divb) {
  if (!c) return MHD_EINVAL;
  if (!c->has_state) return fail(c, MHD_ENOSTATE, "mhd_diagnostics: no state set");
  CUDA_TRY(c, cudaMemsetAsync(c->diag, 0, 9 * sizeof(double), c->stream));
  const int block = 256;
  long long want = ((long long)c->N + block - 1) / block;
  const long long cap = (long long)c->sm_count * 8;
  const unsigned grid = (unsigned)(want < cap ? want : cap);
  if (c->precision == MHD_F32) {
    CflArgs<float> A;
    for (int f = 0; f < 8; ++f) A.f[f] = (const float*)c->cur[f];
    A.nx = c->n[0]; A.ny = c->n[1]; A.nz = c->n[2]; A.bc = c->bc; A.gamma = (float)c->gamma; A.cmax_bits = nullptr;
    diag_kernel<float><<<grid, block, 0, c->stream>>>(A, c->diag, (unsigned long long*)(c->diag + 8));
  } else {
    CflArgs<double> A;
    for (int f = 0; f < 8; ++f) A.f[f] = (const double*)c->cur[f];
    A.nx = c->n[0]; A.ny = c->n[1]; A.nz = c->n[2]; A.bc = c->bc; A.gamma = c->gamma; A.cmax_bits = nullptr;
    diag_kernel<double><<<grid, block, 0, c->stream>>>(A, c->diag, (unsigned long long*)(c->diag + 8));
  }
  c->launches++;
  CUDA_TRY(c, cudaGetLastError());
  double h[9];
  CUDA_TRY(c, cudaMemcpyAsync(h, c->diag, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  if (sums) memcpy(sums, h, 8 * sizeof(double));
  if (max_abs_divb) *max_abs_divb = h[8];   // the bit pattern of a non-negative double IS that double
  return MHD_OK;
}

// ---------------------------------------------------------------------------------------------
// headless visualisation stage (section 8; mhd_viz.cuh)
// ---------------------------------------------------------------------------------------------
template <class real>
static VizArgs<real> make_viz(const mhd_ctx* c, int field, double vmin, double vmax) {
  VizArgs<real> A;
  for (int f = 0; f < 8; ++f) A.f[f] = (const real*)c->cur[f];
  A.nx = c->n[0]; A.ny = c->n[1]; A.nz = c->n[2]; A.bc = c->bc;
  A.field = field;
  A.gamma = (float)c->gamma;
  A.vmin = (float)vmin;
  A.inv = (float)(1.0 / (vmax - vmin));
  return A;
}

static int viz_check(mhd_ctx* c, int field, const char* who) {
  if (field < 0 || field > MHD_VIZ_PRESSURE) return fail(c, MHD_EINVAL, "%s: field must be 0..8", who);
  if (!c->has_state) return fail(c, MHD_ENOSTATE, "%s: no state set", who);
  return MHD_OK;
}

static unsigned viz_grid(const mhd_ctx* c, long long items) {
  const long long want = (items + 255) / 256, cap = (long long)c->sm_count * 8;
  return (unsigned)(want < cap ? (want > 0 ? want : 1) : cap);
}

extern "C" int mhd_viz_range(mhd_ctx* c, int field, double* vmin, double* vmax) {
  if (!c) return MHD_EINVAL;
  if (!vmin || !vmax) return fail(c, MHD_EINVAL, "mhd_viz_range: NULL output");
  int rc = viz_check(c, field, "mhd_viz_range");
  if (rc) return rc;
  unsigned int* lohi = (unsigned int*)(c->diag + 16);          // scratch inside the scalar block
  const unsigned int init[2] = {0xffffffffu, 0u};
  CUDA_TRY(c, cudaMemcpyAsync(lohi, init, sizeof(init), cudaMemcpyHostToDevice, c->stream));
  const unsigned grid = viz_grid(c, (long long)c->N);
  if (c->precision == MHD_F32) viz_range_kernel<float><<<grid, 256, 0, c->stream>>>(make_viz<float>(c, field, 0.0, 1.0), lohi);
  else viz_range_kernel<double><<<grid, 256, 0, c->stream>>>(make_viz<double>(c, field, 0.0, 1.0), lohi);
  c->launches++;
  CUDA_TRY(c, cudaGetLastError());
  unsigned int h[2];
  CUDA_TRY(c, cudaMemcpyAsync(h, lohi, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  if (h[0] > h[1]) return fail(c, MHD_ENONFINITE, "mhd_viz_range: no finite value");
  auto unkey = [](unsigned int k) { unsigned int b = (k & 0x80000000u) ? (k & 0x7fffffffu) : ~k; float v; memcpy(&v, &b, 4); return (double)v; };
  *vmin = unkey(h[0]);
  *vmax = unkey(h[1]);
  return MHD_OK;
}

extern "C" int mhd_viz_curve(mhd_ctx* c, int field, int j, int k, double vmin, double vmax, float* xy_device) {
  if (!c) return MHD_EINVAL;
  int rc = viz_check(c, field, "mhd_viz_curve");
  if (rc) return rc;
  if (!xy_device || !(vmax > vmin) || j < 0 || j >= c->n[1] || k < 0 || k >= c->n[2]) return fail(c, MHD_EINVAL, "mhd_viz_curve: bad argument");
  const float invn = (float)(1.0 / c->n[0]);
  const unsigned grid = (unsigned)((c->n[0] + 255) / 256);
  if (c->precision == MHD_F32) viz_curve_kernel<float><<<grid, 256, 0, c->stream>>>(make_viz<float>(c, field, vmin, vmax), j, k, invn, (float2*)xy_device);
  else viz_curve_kernel<double><<<grid, 256, 0, c->stream>>>(make_viz<double>(c, field, vmin, vmax), j, k, invn, (float2*)xy_device);
  c->launches++;
  CUDA_TRY(c, cudaGetLastError());
  return MHD_OK;
}

extern "C" int mhd_viz_slice(mhd_ctx* c, int field, int k, double vmin, double vmax, const unsigned char* lut_rgba_device,
                             unsigned char* rgba_device) {
  if (!c) return MHD_EINVAL;
  int rc = viz_check(c, field, "mhd_viz_slice");
  if (rc) return rc;
  if (!lut_rgba_device || !rgba_device || !(vmax > vmin) || k < 0 || k >= c->n[2]) return fail(c, MHD_EINVAL, "mhd_viz_slice: bad argument");
  const unsigned grid = viz_grid(c, (long long)c->n[0] * c->n[1]);
  if (c->precision == MHD_F32) viz_slice_kernel<float><<<grid, 256, 0, c->stream>>>(make_viz<float>(c, field, vmin, vmax), k, (const uchar4*)lut_rgba_device, (uchar4*)rgba_device);
  else viz_slice_kernel<double><<<grid, 256, 0, c->stream>>>(make_viz<double>(c, field, vmin, vmax), k, (const uchar4*)lut_rgba_device, (uchar4*)rgba_device);
  c->launches++;
  CUDA_TRY(c, cudaGetLastError());
  return MHD_OK;
}

extern "C" int mhd_viz_volume(mhd_ctx* c, int field, double vmin, double vmax, const unsigned char* lut_rgba_device,
                              double opacity, unsigned char* rgba_device) {
  if (!c) return MHD_EINVAL;
  int rc = viz_check(c, field, "mhd_viz_volume");
  if (rc) return rc;
  if (!lut_rgba_device || !rgba_device || !(vmax > vmin) || !(opacity > 0.0)) return fail(c, MHD_EINVAL, "mhd_viz_volume: bad argument");
  const unsigned grid = viz_grid(c, (long long)c->n[0] * c->n[1]);
  if (c->precision == MHD_F32) viz_volume_kernel<float><<<grid, 256, 0, c->stream>>>(make_viz<float>(c, field, vmin, vmax), (const uchar4*)lut_rgba_device, (float)opacity, (uchar4*)rgba_device);
  else viz_volume_kernel<double><<<grid, 256, 0, c->stream>>>(make_viz<double>(c, field, vmin, vmax), (const uchar4*)lut_rgba_device, (float)opacity, (uchar4*)rgba_device);
  c->launches++;
  CUDA_TRY(c, cudaGetLastError());
  return MHD_OK;
}

extern "C" int mhd_set_option(mhd_ctx* c, const char* key, long long value) {
  if (!c || !key) return MHD_EINVAL;
  drop_graphs(c);                                       // captured steps bake in the kernel choice
  if (!strcmp(key, "segment")) { if (value < -1) return fail(c, MHD_EINVAL, "segment < -1"); c->opt_segment = (int)value; return MHD_OK; }
  if (!strcmp(key, "block")) {
    if (value < 32 || value > 256 || (value & 31)) return fail(c, MHD_EINVAL, "block must be a multiple of 32 in [32,256]");
    c->opt_block = (int)value; return MHD_OK;
  }
  if (!strcmp(key, "xpack")) { if (value < 1 || value > 3) return fail(c, MHD_EINVAL, "xpack must be 1, 2 or 3"); c->opt_xpack = (int)value; return MHD_OK; }
  if (!strcmp(key, "brows")) { if (value < 1 || value > 2) return fail(c, MHD_EINVAL, "brows must be 1 or 2"); c->opt_brows = (int)value; return MHD_OK; }
  if (!strcmp(key, "tmap")) { if (value < 0 || value > 1) return fail(c, MHD_EINVAL, "tmap must be 0 or 1"); c->opt_tmap = (int)value; return MHD_OK; }
  if (!strcmp(key, "xfuse")) { if (value < 0 || value > 3) return fail(c, MHD_EINVAL, "xfuse must be 0, 1 (fp32 only), 2 (always) or 3 (fp32, packed)"); c->opt_xfuse = (int)value; return MHD_OK; }
  if (!strcmp(key, "fuse")) { if (value < 0 || value > 2) return fail(c, MHD_EINVAL, "fuse must be 0, 1 or 2"); c->opt_fuse = (int)value; return MHD_OK; }
  if (!strcmp(key, "cmax_reuse")) { if (value < 0 || value > 1) return fail(c, MHD_EINVAL, "cmax_reuse must be 0 or 1"); c->opt_cmax_reuse = (int)value; return MHD_OK; }
  if (!strcmp(key, "graph")) { if (value < -1 || value > 1) return fail(c, MHD_EINVAL, "graph must be -1 (auto), 0 or 1"); c->opt_graph = (int)value; return MHD_OK; }
  if (!strcmp(key, "path")) { if (value < 0 || value > 1) return fail(c, MHD_EINVAL, "path must be 0 or 1"); c->opt_path = (int)value; return MHD_OK; }
  return fail(c, MHD_EINVAL, "unknown option '%s'", key);
}
