// mhd_noalloc.cu -- mhd_cmax_noalloc: the c_max reduction of eq (18) for callers that must not
// allocate.  PRODUCT code (CUDA path); shares nothing with oracle/.
//
// Who this is for.  Every other compute call of libmhd.so works on a context whose workspace comes from cudaMalloc
// (or from memory the caller cudaMalloc'ed and handed to mhd_bind), and the reduction kernel of mhd_cfl_dt keeps its
// accumulator in that workspace.  Some callers cannot do either: code running inside a framework that owns all of the
// device memory and forbids driver allocations behind its back (a caching allocator with a fixed pool, a solver plugged
// into someone else's time loop), a real-time loop in which cudaMalloc's implicit device-wide synchronisation is not
// acceptable, or a process that is already at its memory limit when it wants one more c_max.  They have the eight fields
// on the device and room for one double; this entry point needs nothing more.
//
// How.  The kernel is a variant of cfl_kernel (mhd_generic.cuh): the same per-cell arithmetic (cfl_speed), but the
// partial maxima go to a scratch array that is part of the library image instead of to allocated memory: a file-scope
// `static __device__` array below, 256 KB + 256 B, which every GPU that loads libmhd.so holds from module load until the
// process exits, whether or not this entry point is ever called.  That fixed size is what bounds the grid: one partial
// per block of 4096 cells, 32768 partials, hence at most 2^27 cells (512^3).
//
// The array's NAME is only usable as an address in device code.  In host code it names a host-side shadow of the
// symbol: handing `g_scratch` itself to a kernel passes a host address that the GPU either faults on or, on systems
// where the GPU can reach host memory, silently reads and writes instead of the real array.  So the device address is
// looked up once per device with cudaGetSymbolAddress while that device is current (scratch_of_current_device), kept in
// a table indexed by device ordinal, and THAT pointer is what the kernel receives.
#include "../../include/mhd.h"

#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "mhd_device.cuh"

using namespace mhd;

static constexpr int kThreads = 256;
static constexpr int kCellsPerThread = 16;
static constexpr long long kCellsPerBlock = (long long)kThreads * kCellsPerThread;   // 4096
static constexpr int kMaxPartials = 32768;                                           // one per block
static constexpr long long kMaxCells = kCellsPerBlock * kMaxPartials;                // 2^27 = 512^3
static constexpr size_t kHeaderBytes = 256;                                          // ticket counter, padded
static constexpr size_t kScratchBytes = kHeaderBytes + sizeof(unsigned long long) * kMaxPartials;
static constexpr int kMaxDevices = 64;

// The scratch.  Layout: [0, 4) ticket counter (blocks that have published their partial; must be 0 when a launch
// starts), [256, 256 + 8 * kMaxPartials) one partial maximum per block, as the bit pattern of a non-negative double.
static __device__ __align__(256) unsigned char g_scratch[kScratchBytes];

namespace {

// Device address of g_scratch on each device, filled on first use (never the host-side symbol, see the file header).
std::atomic<void*> g_scratch_addr[kMaxDevices];
std::mutex g_setup_mutex;

struct CmaxArgs {
  const void* f[8];
  int nx, ny, nz, bc;
  double gamma;
  long long N;
  unsigned char* scratch;   // device address of g_scratch, from cudaGetSymbolAddress
  double* out;              // caller's device double
};

// One block per 4096 consecutive cells; threads stride by the block width so that every load is coalesced.  Each block
// publishes its maximum into its own slot of the scratch, then takes a ticket; the block that draws the last ticket
// knows every slot is written, folds them, writes the caller's output and puts the counter back to zero.
// c >= 0 and non-negative IEEE doubles order like unsigned integers, so the maximum is taken on bit patterns, exactly
// as cfl_kernel does.
template <class real>
__global__ void __launch_bounds__(kThreads) cmax_noalloc_kernel(const CmaxArgs A) {
  const real* const rho = (const real*)A.f[0];
  const real* const mx = (const real*)A.f[1];
  const real* const my = (const real*)A.f[2];
  const real* const mz = (const real*)A.f[3];
  const real* const en = (const real*)A.f[4];
  const real* const bxf = (const real*)A.f[5];
  const real* const byf = (const real*)A.f[6];
  const real* const bzf = (const real*)A.f[7];
  const long long sy = A.nx, sz = (long long)A.nx * A.ny;
  const real gamma = (real)A.gamma;
  unsigned int* const ticket = reinterpret_cast<unsigned int*>(A.scratch);
  unsigned long long* const partial = reinterpret_cast<unsigned long long*>(A.scratch + kHeaderBytes);

  const long long base = (long long)blockIdx.x * kCellsPerBlock;
  unsigned long long best = 0ull;
#pragma unroll 4
  for (int r = 0; r < kCellsPerThread; ++r) {
    const long long idx = base + (long long)r * kThreads + threadIdx.x;
    if (idx < A.N) {
      const int i = (int)(idx % A.nx);
      const int j = (int)((idx / A.nx) % A.ny);
      const int k = (int)(idx / sz);
      // B at the cell centre: mean of the two faces of the cell (eq (19)), the far face mapped by
      // the boundary rule
      const long long ip = map_index(i + 1, A.nx, A.bc) + j * sy + k * sz;
      const long long jp = i + map_index(j + 1, A.ny, A.bc) * sy + k * sz;
      const long long kp = i + j * sy + map_index(k + 1, A.nz, A.bc) * sz;
      const real bx = real(0.5) * (bxf[idx] + bxf[ip]);
      const real by = real(0.5) * (byf[idx] + byf[jp]);
      const real bz = real(0.5) * (bzf[idx] + bzf[kp]);
      const unsigned long long bits = speed_bits(cfl_speed(rho[idx], mx[idx], my[idx], mz[idx], en[idx], bx, by, bz, gamma));
      best = bits > best ? bits : best;
    }
  }
  best = warp_max_u64(best);
  __shared__ unsigned long long sm[kThreads / 32];
  __shared__ bool is_last;
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = best;
  __syncthreads();
  if (threadIdx.x < 32) {
    best = threadIdx.x < kThreads / 32 ? sm[threadIdx.x] : 0ull;
    best = warp_max_u64(best);
    if (threadIdx.x == 0) {
      partial[blockIdx.x] = best;
      __threadfence();                                   // the slot is visible before the ticket is
      is_last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
  }
  __syncthreads();
  if (!is_last) return;
  __threadfence();                                       // the other blocks' slots, published before their tickets
  best = 0ull;
  for (unsigned b = threadIdx.x; b < gridDim.x; b += kThreads) {
    const unsigned long long v = __ldcg(partial + b);
    best = v > best ? v : best;
  }
  best = warp_max_u64(best);
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = best;
  __syncthreads();
  if (threadIdx.x < 32) {
    best = threadIdx.x < kThreads / 32 ? sm[threadIdx.x] : 0ull;
    best = warp_max_u64(best);
    if (threadIdx.x == 0) {
      *A.out = __longlong_as_double((long long)best);
      *ticket = 0u;                                      // leave the counter as the next launch needs it
    }
  }
}

int fail(char* errbuf, size_t errlen, int code, const char* fmt, ...) {
  if (errbuf && errlen) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(errbuf, errlen, fmt, ap);
    va_end(ap);
  }
  return code;
}

// Set-up, once per device: the device address of g_scratch on the CURRENT device.  cudaGetSymbolAddress loads the
// library's module on that device if nothing has yet (that is where the 256 KB are claimed); it is not cudaMalloc.
cudaError_t scratch_of_current_device(unsigned char** out, int* device) {
  cudaError_t e = cudaGetDevice(device);
  if (e != cudaSuccess) return e;
  if (*device < 0 || *device >= kMaxDevices) return cudaErrorInvalidDevice;
  void* p = g_scratch_addr[*device].load(std::memory_order_acquire);
  if (!p) {
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    p = g_scratch_addr[*device].load(std::memory_order_relaxed);
    if (!p) {
      e = cudaGetSymbolAddress(&p, g_scratch);
      if (e != cudaSuccess) return e;
      if (!p) return cudaErrorInvalidSymbol;
      g_scratch_addr[*device].store(p, std::memory_order_release);
    }
  }
  *out = static_cast<unsigned char*>(p);
  return cudaSuccess;
}

}  // namespace

extern "C" int mhd_cmax_noalloc(const void* const fields_device[8], int nx, int ny, int nz, double gamma, int precision,
                                int bc, void* cuda_stream, double* cmax_device, char* errbuf, size_t errbuf_len) {
  if (errbuf && errbuf_len) errbuf[0] = '\0';
  if (!fields_device || !cmax_device) return fail(errbuf, errbuf_len, MHD_EINVAL, "mhd_cmax_noalloc: NULL pointer");
  for (int f = 0; f < 8; ++f)
    if (!fields_device[f]) return fail(errbuf, errbuf_len, MHD_EINVAL, "mhd_cmax_noalloc: fields_device[%d] is NULL", f);
  if (nx < 1 || ny < 1 || nz < 1) return fail(errbuf, errbuf_len, MHD_EINVAL, "mhd_cmax_noalloc: extents must be >= 1");
  if (precision != MHD_F32 && precision != MHD_F64) return fail(errbuf, errbuf_len, MHD_EINVAL, "mhd_cmax_noalloc: unknown precision");
  if (bc != MHD_BC_PERIODIC && bc != MHD_BC_OUTFLOW) return fail(errbuf, errbuf_len, MHD_EINVAL, "mhd_cmax_noalloc: unknown bc");
  if (!(gamma > 1.0)) return fail(errbuf, errbuf_len, MHD_EINVAL, "mhd_cmax_noalloc: gamma must be > 1");
  const double cells = (double)nx * (double)ny * (double)nz;
  if (cells > (double)kMaxCells)
    return fail(errbuf, errbuf_len, MHD_EINVAL,
                "mhd_cmax_noalloc: %d x %d x %d = %.0f cells is more than the %lld cells (512^3) the fixed %zu-byte scratch "
                "holds partial maxima for; use mhd_cfl_dt on a context",
                nx, ny, nz, cells, kMaxCells, kScratchBytes);

  unsigned char* scratch = nullptr;
  int device = -1;
  cudaError_t e = scratch_of_current_device(&scratch, &device);
  if (e != cudaSuccess)
    return fail(errbuf, errbuf_len, MHD_ECUDA, "mhd_cmax_noalloc: looking up the scratch on device %d failed: %s", device,
                cudaGetErrorString(e));

  cudaStream_t stream = (cudaStream_t)cuda_stream;
  // The array keeps whatever the last call left.  The partial slots need no clearing (every slot that is read was
  // written by this launch first); the ticket counter must start at zero, and a launch that never finished (a fault,
  // a device reset of another context) could have left it anywhere, so it is cleared on every call, in stream order.
  e = cudaMemsetAsync(scratch, 0, kHeaderBytes, stream);
  if (e != cudaSuccess)
    return fail(errbuf, errbuf_len, MHD_ECUDA, "mhd_cmax_noalloc: clearing the ticket counter failed: %s", cudaGetErrorString(e));

  CmaxArgs A;
  for (int f = 0; f < 8; ++f) A.f[f] = fields_device[f];
  A.nx = nx; A.ny = ny; A.nz = nz; A.bc = bc;
  A.gamma = gamma;
  A.N = (long long)nx * ny * nz;
  A.scratch = scratch;
  A.out = cmax_device;
  const unsigned grid = (unsigned)((A.N + kCellsPerBlock - 1) / kCellsPerBlock);   // <= kMaxPartials
  if (precision == MHD_F32) cmax_noalloc_kernel<float><<<grid, kThreads, 0, stream>>>(A);
  else cmax_noalloc_kernel<double><<<grid, kThreads, 0, stream>>>(A);
  e = cudaGetLastError();
  if (e != cudaSuccess)
    return fail(errbuf, errbuf_len, MHD_ECUDA, "mhd_cmax_noalloc: kernel launch failed: %s", cudaGetErrorString(e));
  return MHD_OK;
}
