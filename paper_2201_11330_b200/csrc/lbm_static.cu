// lbm_static.cu — lbm_diagnostics_static (include/lbm.h): the Monitor / PostProcessing reduction (P:295-304,
// P:404-427; Eq. 8-9) for callers that may not allocate device memory.
//
// The handle-based path (lbm_moments with diagnostics != NULL) reduces in two passes and keeps the per-block
// records of the first pass in an array that lbm_create took from cudaMalloc.  Some users of this library cannot go
// that way.  Their process has handed every byte of the device to a pool of its own (torch's caching allocator, a
// solver that sizes its arrays to the card), so a cudaMalloc made behind that pool's back fails or steals the room
// the next time step needs.  Or they sit in a time loop whose other streams must not be stalled by the device-wide
// synchronisation cudaMalloc / cudaFree imply.  Or they only hold a pointer to somebody else's populations (a
// checkpoint, another code's arrays) and have no handle, whose creation allocates.  For them the same reduction is
// offered here with its records in a fixed array that is part of the library image.  Nothing in this file calls
// cudaMalloc, cudaFree or a library routine that allocates.
//
// The price, stated once: the array below (2 MiB) is resident on every GPU that loads this library's code, from load
// to process exit, whether or not this entry point is ever called; grids beyond LBM_STATIC_MAX_CELLS are refused;
// and all calls on one device share the array (see "Sharing" at the entry point).
#include <cmath>
#include <mutex>
#include <string>

#include "../../include/lbm.h"
#include "lbm_kernels.cuh"

namespace lbm {
void set_last_error(const std::string& msg);  // lbm_abi.cu: the message lbm_last_error() returns on this thread
}

using namespace lbm;

namespace {

constexpr int kThreads = 256;
constexpr int kCellsPerThread = 16;
// A block always covers the same 4096 consecutive cells, whatever the device: the records, and therefore the
// rounding of the five sums, do not depend on the number of SMs (same bits on every GPU and on every call).
constexpr long long kCellsPerBlock = (long long)kThreads * kCellsPerThread;
constexpr long long kMaxCells = LBM_STATIC_MAX_CELLS;
constexpr int kMaxBlocks = (int)(kMaxCells / kCellsPerBlock);  // 32768 records of 8 doubles = 2 MiB
static_assert(kMaxCells % kCellsPerBlock == 0, "LBM_STATIC_MAX_CELLS must be a whole number of blocks");

// The scratch: one record of kDiag doubles per block of the first pass.  In HOST code this name is only a stand-in
// for the symbol — it is not a device address, and a kernel handed `g_block_records` from host code would fault (or,
// on a system where the GPU can reach host memory, quietly work on the wrong bytes).  Host code therefore asks the
// runtime for the address once per device (records_on_current_device) and passes that pointer to the kernels.
static __device__ __align__(256) double g_block_records[(size_t)kMaxBlocks * kDiag];

constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
double* g_records_addr[kMaxDevices];  // device address of g_block_records on device d, nullptr = not looked up yet

int fail(int code, const std::string& msg) {
  set_last_error(msg);
  return code;
}
int cuda_fail(cudaError_t e, const char* what) {
  set_last_error(std::string(what) + ": " + cudaGetErrorString(e));
  return LBM_ECUDA;
}

// Set-up, once per device, with that device current: the device address of the static array.
int records_on_current_device(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return cuda_fail(e, "lbm_diagnostics_static: cudaGetDevice");
  if (dev < 0 || dev >= kMaxDevices) return fail(LBM_EUNSUPPORTED, "lbm_diagnostics_static: device ordinal beyond 63");
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  if (!g_records_addr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_block_records);
    if (e != cudaSuccess) return cuda_fail(e, "lbm_diagnostics_static: cudaGetSymbolAddress(g_block_records)");
    if (!p) return fail(LBM_ECUDA, "lbm_diagnostics_static: cudaGetSymbolAddress returned a null address");
    g_records_addr[dev] = (double*)p;
  }
  *out = g_records_addr[dev];
  return LBM_OK;
}

// First pass: the variant of moments_kernel that needs no handle.  Reads the canonical populations f[a*n + i]
// (include/lbm.h "Conventions"), evaluates rho and u per cell with the same moments<> the step and moments kernels
// use (Eq. 8-9 with the F/2 shift of D:R7), accumulates the 8 diagnostics exactly as moments_kernel does and leaves
// one record per block in `records` (= g_block_records, address supplied by the host).
template <int Q, int EQ>
__global__ void __launch_bounds__(kThreads) diagnostics_static_kernel(const double* __restrict__ f, long long n, double Fx, double Fy, double Fz,
                                                                    double* __restrict__ records) {
  Params p;  // moments<> reads p.F only
  p.F[0] = Fx;
  p.F[1] = Fy;
  p.F[2] = Fz;
  double acc[kDiag] = {0, 0, 0, 0, 0, 0, INFINITY, 0};
  const long long first = (long long)blockIdx.x * kCellsPerBlock + threadIdx.x;
#pragma unroll 2
  for (int k = 0; k < kCellsPerThread; ++k) {
    const long long i = first + (long long)k * kThreads;  // consecutive threads, consecutive cells: every stream unit-stride
    if (i >= n) break;
    double v[Q];
    static_for<0, Q>([&](auto A) {
      constexpr int a = decltype(A)::value;
      v[a] = __ldg(f + (long long)a * n + i);
    });
    double rho, ux, uy, uz;
    moments<Q, EQ, true>(v, p, rho, ux, uy, uz);
    const double usq = ux * ux + uy * uy + uz * uz;
    if (isfinite(rho) && isfinite(usq)) {
      const double rw = (EQ == EQ_STANDARD) ? rho : 1.0;
      acc[0] += rho;
      acc[1] += rw * ux;
      acc[2] += rw * uy;
      acc[3] += rw * uz;
      acc[4] += 0.5 * rw * usq;
      acc[5] = fmax(acc[5], sqrt(usq));
      acc[6] = fmin(acc[6], rho);
    } else {
      acc[7] += 1.0;
    }
  }
  block_reduce_diag(acc, records + (long long)blockIdx.x * kDiag);
}

template <int Q>
void launch_first_pass(int eq, int nblocks, cudaStream_t st, const double* f, long long n, const double* F, double* records) {
  if (eq == EQ_STANDARD) diagnostics_static_kernel<Q, EQ_STANDARD><<<nblocks, kThreads, 0, st>>>(f, n, F[0], F[1], F[2], records);
  else diagnostics_static_kernel<Q, EQ_INCOMP><<<nblocks, kThreads, 0, st>>>(f, n, F[0], F[1], F[2], records);
}

}  // namespace

// Contract: include/lbm.h.  Summary of what matters to a caller that cannot allocate:
//   * no cudaMalloc / cudaFree / cudaMallocAsync / cudaHostAlloc and no allocating library call, on any path;
//   * the first call on a device looks up the address of the static array (cudaGetSymbolAddress) — make that first
//     call during start-up, before any stream capture is begun;
//   * the array keeps whatever the previous call left in it.  Nothing in it has to start at zero: with nblocks =
//     ceil(ncells / 4096), pass 1 overwrites records 0 .. nblocks-1 in full and pass 2 reads exactly those, so
//     records of an earlier, larger call are never looked at and no clearing pass is needed;
//   * Sharing: two calls whose kernels may run at the same time on one device (different streams, different host
//     threads without ordering between their streams) race on the array and both results are garbage.  Calls on one
//     stream, or ordered by events, are fine.  Different devices have different copies and do not interact.
extern "C" int lbm_diagnostics_static(const double* f, int64_t ncells, int lattice, const double* force, double* diagnostics, void* stream) {
  const int Q = lattice & 0xFF;
  if (Q != LBM_D2Q9 && Q != LBM_D3Q19 && Q != LBM_D3Q27)
    return fail(LBM_EINVAL, "lbm_diagnostics_static: lattice must be LBM_D2Q9, LBM_D3Q19 or LBM_D3Q27");
  if ((lattice & ~(0xFF | LBM_EQ_INCOMP)) != 0)
    return fail(LBM_EINVAL, "lbm_diagnostics_static: only the velocity set and LBM_EQ_INCOMP may be set in `lattice` "
                            "(f is always fp64 in the canonical layout f[a*ncells + i])");
  if (ncells < 1) return fail(LBM_EINVAL, "lbm_diagnostics_static: ncells must be >= 1");
  if (ncells > kMaxCells)
    return fail(LBM_EINVAL, "lbm_diagnostics_static: ncells = " + std::to_string((long long)ncells) + " exceeds LBM_STATIC_MAX_CELLS = " +
                                std::to_string(kMaxCells) + " (the static scratch array holds one record per 4096 cells and cannot grow; "
                                "use lbm_moments on a handle for larger grids)");
  if (!f || !diagnostics) return fail(LBM_EINVAL, "lbm_diagnostics_static: f and diagnostics must be device pointers, not NULL");
  double F[3] = {0.0, 0.0, 0.0};
  if (force) {
    F[0] = force[0];
    F[1] = force[1];
    F[2] = force[2];
  }
  double* records = nullptr;
  {
    const int rc = records_on_current_device(&records);
    if (rc) return rc;
  }
  const cudaStream_t st = (cudaStream_t)stream;
  const int eq = (lattice & LBM_EQ_INCOMP) ? EQ_INCOMP : EQ_STANDARD;
  const int nblocks = (int)((ncells + kCellsPerBlock - 1) / kCellsPerBlock);
  const long long n = (long long)ncells;
  if (Q == 9) launch_first_pass<9>(eq, nblocks, st, f, n, F, records);
  else if (Q == 19) launch_first_pass<19>(eq, nblocks, st, f, n, F, records);
  else launch_first_pass<27>(eq, nblocks, st, f, n, F, records);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(e, "lbm_diagnostics_static: first pass");
  // second pass: one block folds the nblocks records in index order and writes the caller's 8 doubles
  reduce_final_kernel<><<<1, 256, 0, st>>>(records, nblocks, diagnostics);
  e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(e, "lbm_diagnostics_static: final pass");
  return LBM_OK;
}
