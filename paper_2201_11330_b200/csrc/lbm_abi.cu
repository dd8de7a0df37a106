// lbm_abi.cu — the C ABI declared in include/lbm.h: handle, argument checks, kernel dispatch.
// No torch types, no exceptions across the boundary, no CPU path.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <unistd.h>

#include <cuda.h>  // types of the stream memory operations only; entry points come from cudaGetDriverEntryPoint

#include "../../include/lbm.h"
#include "lbm_launch.cuh"

using namespace lbm;

namespace {

thread_local std::string g_err;

int fail(int code, const std::string& msg) {
  g_err = msg;
  return code;
}
int cuda_fail(cudaError_t e, const char* what) {
  g_err = std::string(what) + ": " + cudaGetErrorString(e);
  return LBM_ECUDA;
}
#define CUDA_TRY(expr)                                 \
  do {                                                 \
    cudaError_t e__ = (expr);                          \
    if (e__ != cudaSuccess) return cuda_fail(e__, #expr); \
  } while (0)

constexpr int kReduceBlocks = 148 * 8;  // one wave of 256-thread blocks on 148 SMs
constexpr size_t kGuard = 64u << 10;    // bytes of guard zone before and after every device array of a handle
constexpr int kGuardByte = 0xFF;        // all-ones: a NaN as fp64 / fp32, so that an out-of-bounds READ that is used shows up too
constexpr int kMaxOwned = 24;
constexpr int kMaxChunks = 16;          // z-chunks of the host entry points (copy of chunk k+1 overlaps the kernel of chunk k)
constexpr size_t kChunkBytes = 64u << 20;  // ... each at least this many bytes of rho, u (smaller grids: one chunk)

}  // namespace

namespace lbm {
// for the library's other translation units (lbm_static.cu): leave a message for lbm_last_error() on this thread
void set_last_error(const std::string& msg) { g_err = msg; }
}  // namespace lbm

struct lbm_handle_s {
  int nx, ny, nz, Q, eq, scheme, f32;
  int soa;            // LBM_LAYOUT_SOA: plain structure of arrays instead of the row-interleaved layout
  long long N;
  double tau;
  Params p;
  bool walls, forced;
  int wall_model;     // LBM_WALL_HALFWAY / LBM_WALL_NODAL (lbm_set_geometry)
  bool has_geo;       // the BC_GEO kernels are in use (a solid mask and/or the nodal model was set)
  uint8_t* geo;       // N, device: 1 = solid node
  uint8_t* active;    // N, device: node takes part in collision and propagation (D:R16)
  uint32_t* links;    // N, device: per-cell link mask read by the BC_GEO kernels
  bool stepped;       // at least one step since the populations were last set (lbm_boundary_force)
  cudaStream_t stream;
  void* buf[2];       // A/B: both used, buf[cur] holds S^-1 f;  AA: buf[0] only
  int cur;
  int phase;          // AA: 0 = natural layout, 1 = after an even step
  long long time, launches;
  double* partials;   // kReduceBlocks * 8
  double* diag_dev;   // 8
  double* diag_pinned;  // 8, host
  void* scratch;
  size_t scratch_bytes;
  // debug aids (lbm_debug_arm / lbm_debug_check): every device array is allocated with a guard zone on both sides
  struct { void* p; size_t bytes; bool floating; } owned[kMaxOwned];
  int n_owned;
  unsigned long long* guard_bad;     // device counter of guard bytes that lost their pattern
  cudaStream_t copy_stream;          // host entry points: the copies run here, the kernels on `stream` (created on first use)
  cudaEvent_t chunk_ev[kMaxChunks];  // chunk k has landed (init) / has been computed (moments)
  cudaEvent_t fence_ev;              // orders the two streams at the start and at the end of a host call
  // z-slab of a decomposed box (D:R21)
  bool slab;
  int z0, nz_global, nz_local;
  uint32_t* flags;        // device, 2 counters: steps finished by the lower / by the upper neighbour (they write, we wait)
  uint32_t sync_count;    // steps this slab has finished since it was created (never reset)
  int device_sync;
  bool shares_stream;  // a connected neighbour of this process runs on this handle's stream (legal only host-ordered)
  void* peer_lo[2];       // lower / upper neighbour's population buffers as seen from this process
  void* peer_hi[2];
  long long peer_lo_N, peer_hi_N;
  long long peer_lo_off, peer_hi_off;
  uint32_t* peer_lo_flag;  // the counter we write in the lower neighbour (its "upper" one) / in the upper neighbour
  uint32_t* peer_hi_flag;
  void* ipc_opened[6];
  int n_ipc_opened;
  int l2_bytes;       // L2 cache size of the device (0 = unknown)
  int persistent;     // lbm_step may take all steps of a call in one cooperative launch (small grids; lbm_set_persistent)
  int two_step;       // lbm_step takes steps in pairs through stream_collide_ab2: 0 never, 1 where it pays (default), 2 wherever it exists
  int bx, by;         // block shape of the fused kernel (lbm_set_block), 0,0 = default_block()
  int fbx;            // row width (power of two <= 256) of the row-wise sweeps off the per-step path
  size_t elem() const { return f32 ? 4 : 8; }
  size_t buf_bytes() const { return (size_t)N * Q * elem(); }
};

namespace {

// Q dispatch: the per-lattice launchers live in lbm_inst.cu (one object per lattice and part).
#define LBM_Q_CALL_RET(h, ret, fn, ...)                 \
  do {                                                  \
    if ((h)->Q == 19) ret = fn<19>(__VA_ARGS__);        \
    else if ((h)->Q == 27) ret = fn<27>(__VA_ARGS__);   \
    else ret = fn<9>(__VA_ARGS__);                      \
  } while (0)
#define LBM_Q_CALL(h, fn, ...)                 \
  do {                                         \
    if ((h)->Q == 19) fn<19>(__VA_ARGS__);     \
    else if ((h)->Q == 27) fn<27>(__VA_ARGS__); \
    else fn<9>(__VA_ARGS__);                   \
  } while (0)

Ctx make_ctx(const lbm_handle_s* h);

// blocks of the row-wise sweeps (for_each_cell): 256/fbx rows per block, at most one wave
int flat_grid(const lbm_handle_s* h) {
  const long long rows = (long long)h->ny * h->nz, by = 256 / h->fbx;
  const long long b = (rows + by - 1) / by;
  return (int)(b < kReduceBlocks ? b : kReduceBlocks);
}

// Default block of the fused kernels, by measurement: rows of 256 threads for the kernels that
// keep three or four 256-thread blocks per SM (D3Q19 / D2Q9 A/B without forcing or mask); 128 threads where the
// register count allows only two of them (D3Q27, forcing, every in-place AA kernel: 512^3 D3Q19 AA 21 778 -> 22 025,
// cavity AA 20 553 -> 21 332 MLUPS) and for the link-mask kernels, whose face / wall cells make single warps run
// long: a block holds its registers until its last warp retires, smaller blocks hold fewer.
void default_block(const lbm_handle_s* h, int& bx, int& by) {
  const bool small = h->scheme == LBM_SCHEME_AA || h->Q == 27 || h->forced || h->has_geo;
  const int threads = small ? 128 : 256;
  bx = 32;
  while (bx < h->nx && bx < threads) bx *= 2;
  by = threads / bx;
  while (by > 1 && (h->ny + by - 1) / by > 65535) by /= 2;
}

Ctx make_ctx(const lbm_handle_s* h) {
  Ctx c;
  int bx = h->bx, by = h->by;
  if (bx == 0) default_block(h, bx, by);
  c.eq = h->eq ? EQ_INCOMP : EQ_STANDARD;
  c.bc = h->has_geo ? BC_GEO : (h->walls ? BC_WALLS : BC_PERIODIC);
  c.forced = h->forced;
  c.f32 = h->f32;
  c.block = dim3(bx, by, 1);
  c.grid = dim3((h->nx + bx - 1) / bx, (h->ny + by - 1) / by, h->p.z_hi - h->p.z_lo);
  c.flat_grid = flat_grid(h);
  c.fbx = h->fbx;
  c.stream = h->stream;
  c.p = h->p;
  return c;
}

// canonical-state read mode of the current storage state
int read_mode(const lbm_handle_s* h) {
  if (h->scheme == LBM_SCHEME_AB) return MODE_PULL;
  return h->phase ? MODE_PULL_SWAP : MODE_NATURAL;
}

// Stream memory operation "wait until *addr >= value" (cyclic 32-bit compare), resolved once at run time so that
// the library has no link-time dependency on libcuda.
typedef CUresult (*wait_value32_fn)(CUstream, CUdeviceptr, cuuint32_t, unsigned int);
wait_value32_fn wait_value32() {
  static wait_value32_fn fn = [] {
    void* f = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuStreamWaitValue32", &f, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) f = nullptr;
    cudaGetLastError();
    return (wait_value32_fn)f;
  }();
  return fn;
}

// "this slab has finished `count` steps", written into the neighbours' counters after everything the step
// kernel stored (their halo planes included) is visible system-wide
__global__ void slab_signal_kernel(uint32_t* lo, uint32_t* hi, uint32_t count) {
  __threadfence_system();
  if (lo) *(volatile uint32_t*)lo = count;
  if (hi) *(volatile uint32_t*)hi = count;
}

// One step of a z-slab: wait for both neighbours' previous step, run the fused kernel (which also fills the
// neighbours' halo planes of the buffer it writes), tell the neighbours.
// Make the stream wait until both neighbours have finished as many steps as this slab has: their stores into
// this slab's halo planes are then complete, and they no longer read what the next step overwrites.
int slab_wait_neighbours(lbm_handle_s* h) {
  if (!h->slab || !h->device_sync) return LBM_OK;
  wait_value32_fn wait = wait_value32();
  if (!wait) return fail(LBM_ECUDA, "cuStreamWaitValue32 is not available on this driver");
  for (int side = 0; side < 2; ++side) {
    if (!(side ? h->peer_hi[0] : h->peer_lo[0])) continue;
    CUresult r = wait((CUstream)h->stream, (CUdeviceptr)(h->flags + side), h->sync_count, CU_STREAM_WAIT_VALUE_GEQ);
    if (r != CUDA_SUCCESS) return fail(LBM_ECUDA, "cuStreamWaitValue32 failed");
  }
  return LBM_OK;
}

int launch_step_slab(lbm_handle_s* h, Ctx& c) {
  const int dst = h->cur ^ 1;
  {
    int rc = slab_wait_neighbours(h);
    if (rc) return rc;
  }
  c.p.push_lo = h->peer_lo[dst];
  c.p.push_hi = h->peer_hi[dst];
  LBM_Q_CALL(h, launch_step_ab_slab, c, h->buf[h->cur], h->buf[dst]);
  h->cur = dst;
  ++h->launches;
  ++h->sync_count;
  if (h->device_sync && (h->peer_lo_flag || h->peer_hi_flag)) {
    slab_signal_kernel<<<1, 1, 0, h->stream>>>(h->peer_lo_flag, h->peer_hi_flag, h->sync_count);
    ++h->launches;
  }
  return LBM_OK;
}

void launch_step(lbm_handle_s* h, const Ctx& c) {
  if (h->scheme == LBM_SCHEME_AB) {
    LBM_Q_CALL(h, launch_step_ab, c, h->buf[h->cur], h->buf[h->cur ^ 1]);
    h->cur ^= 1;
  } else {
    if (h->phase == 0) LBM_Q_CALL(h, launch_step_aa_even, c, h->buf[0]);
    else LBM_Q_CALL(h, launch_step_aa_odd, c, h->buf[0]);
    h->phase ^= 1;
  }
  ++h->launches;
}

// canonical fp64 array `in` -> storage buffer `dst_idx` in the layout the scheme wants at an even phase
void do_import(lbm_handle_s* h, const double* in, int dst_idx) {
  const Ctx c = make_ctx(h);
  LBM_Q_CALL(h, launch_import, c, h->scheme == LBM_SCHEME_AB ? MODE_PULL : MODE_NATURAL, in, h->buf[dst_idx]);
  ++h->launches;
}

// Device arrays of a handle: `bytes` usable bytes between two guard zones filled with kGuardByte (lbm_debug_check counts
// the guard bytes that changed: an out-of-bounds store of the library's kernels that lands within 64 KB of an array).
// floating: holds populations / moments (what lbm_debug_arm may poison with NaNs).
cudaError_t gmalloc(lbm_handle_s* h, void** out, size_t bytes, bool floating) {
  *out = nullptr;
  if (h->n_owned >= kMaxOwned) return cudaErrorMemoryAllocation;
  char* raw = nullptr;
  cudaError_t e = cudaMalloc((void**)&raw, bytes + 2 * kGuard);
  if (e != cudaSuccess) return e;
  e = cudaMemsetAsync(raw, kGuardByte, kGuard, h->stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(raw + kGuard + bytes, kGuardByte, kGuard, h->stream);
  if (e != cudaSuccess) { cudaFree(raw); return e; }
  *out = raw + kGuard;
  h->owned[h->n_owned].p = *out;
  h->owned[h->n_owned].bytes = bytes;
  h->owned[h->n_owned].floating = floating;
  ++h->n_owned;
  return cudaSuccess;
}
void gfree(lbm_handle_s* h, void* p) {
  if (!p) return;
  for (int k = 0; k < h->n_owned; ++k)
    if (h->owned[k].p == p) {
      h->owned[k] = h->owned[h->n_owned - 1];
      --h->n_owned;
      break;
    }
  cudaFree((char*)p - kGuard);
}

__global__ void guard_count_kernel(const unsigned char* __restrict__ g, size_t n, unsigned long long* bad) {
  unsigned long long c = 0;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) c += g[i] != kGuardByte;
  if (c) atomicAdd(bad, c);
}

int ensure_scratch(lbm_handle_s* h, size_t bytes) {
  if (h->scratch_bytes >= bytes) return LBM_OK;
  if (h->scratch) {
    cudaStreamSynchronize(h->stream);
    gfree(h, h->scratch);
    h->scratch = nullptr;
    h->scratch_bytes = 0;
  }
  cudaError_t e = gmalloc(h, &h->scratch, bytes, true);
  if (e != cudaSuccess) {
    cudaGetLastError();
    return fail(LBM_ENOMEM, "out of device memory for the scratch buffer");
  }
  h->scratch_bytes = bytes;
  return LBM_OK;
}

int check_launch(const char* what) {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(e, what);
  return LBM_OK;
}

// rows r = y + ny*z of the planes this handle updates, and the blocks of a row-wise sweep over `nrows` of them
int rows_begin(const lbm_handle_s* h) { return h->ny * h->p.z_lo; }
int rows_end(const lbm_handle_s* h) { return h->ny * h->p.z_hi; }
int grid_for_rows(const lbm_handle_s* h, long long nrows) {
  const long long by = 256 / h->fbx, b = (nrows + by - 1) / by;
  return (int)(b < 1 ? 1 : b < kReduceBlocks ? b : kReduceBlocks);
}

// storage buffer and mode an initialisation writes (always an even phase); connected slabs must agree on the buffer
int init_target(lbm_handle_s* h) {
  if (h->slab || h->scheme != LBM_SCHEME_AB) h->cur = 0;
  return h->scheme == LBM_SCHEME_AB ? MODE_PULL : MODE_NATURAL;
}

void finish_init(lbm_handle_s* h) {
  h->phase = 0;
  h->time = 0;
  h->stepped = false;
}

// InitPDF on rows [r0, r1): ONE kernel, feq straight into the storage buffer (init_equilibrium_kernel)
void launch_init_rows(lbm_handle_s* h, const Ctx& c, int mode, const double* rho, const double* u, int r0, int r1) {
  LBM_Q_CALL(h, launch_init, c, mode, rho, u, h->buf[h->cur], r0, r1, grid_for_rows(h, r1 - r0));
  ++h->launches;
}

int do_init(lbm_handle_s* h, const double* rho, const double* u) {
  const int mode = init_target(h);
  const Ctx c = make_ctx(h);
  launch_init_rows(h, c, mode, rho, u, rows_begin(h), rows_end(h));
  finish_init(h);
  return check_launch("init_equilibrium");
}

// diagnostics: reduce the `nblocks` block partials, copy the 8 doubles to the host, synchronise
int finish_diagnostics(lbm_handle_s* h, int nblocks, double* diagnostics) {
  reduce_final_kernel<><<<1, 256, 0, h->stream>>>(h->partials, nblocks, h->diag_dev);
  ++h->launches;
  int rc = check_launch("moments");
  if (rc) return rc;
  CUDA_TRY(cudaMemcpyAsync(h->diag_pinned, h->diag_dev, kDiag * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  std::memcpy(diagnostics, h->diag_pinned, kDiag * sizeof(double));
  return LBM_OK;
}

int do_moments(lbm_handle_s* h, double* rho, double* u, double* diagnostics) {
  {
    int rc = slab_wait_neighbours(h);  // the pull reads the halo planes
    if (rc) return rc;
  }
  const Ctx c = make_ctx(h);
  const int grid = grid_for_rows(h, rows_end(h) - rows_begin(h));
  LBM_Q_CALL(h, launch_moments, c, read_mode(h), h->buf[h->cur], rho, u, diagnostics ? h->partials : nullptr, rows_begin(h), rows_end(h), grid);
  ++h->launches;
  if (diagnostics) return finish_diagnostics(h, grid, diagnostics);
  return check_launch("moments");
}

// ---- host entry points: z-chunked so that the PCIe copies overlap the kernels ----------------------------------
// Device staging for the 4N doubles of rho, u: the idle A/B buffer (Q*elem >= 32 B per cell for every lattice), else —
// in-place scheme, or a z-slab, whose idle buffer's halo planes belong to the neighbours' next step — the scratch buffer.
int host_staging(lbm_handle_s* h, double** out) {
  if (h->scheme == LBM_SCHEME_AB && !h->slab) {
    *out = (double*)h->buf[h->cur ^ 1];
    return LBM_OK;
  }
  int rc = ensure_scratch(h, (size_t)h->N * 4 * sizeof(double));
  if (rc) return rc;
  *out = (double*)h->scratch;
  return LBM_OK;
}

int ensure_copy_stream(lbm_handle_s* h) {
  if (h->copy_stream) return LBM_OK;
  CUDA_TRY(cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking));
  for (int k = 0; k < kMaxChunks; ++k) CUDA_TRY(cudaEventCreateWithFlags(&h->chunk_ev[k], cudaEventDisableTiming));
  CUDA_TRY(cudaEventCreateWithFlags(&h->fence_ev, cudaEventDisableTiming));
  return LBM_OK;
}

// plane ranges [zc[k], zc[k+1]) of the updated planes, k < n
int plane_chunks(const lbm_handle_s* h, int* zc) {
  const int planes = h->p.z_hi - h->p.z_lo;
  const size_t plane_bytes = (size_t)h->nx * h->ny * 4 * sizeof(double);
  long long n = (long long)(plane_bytes * planes / kChunkBytes);
  n = n < 1 ? 1 : n > kMaxChunks ? kMaxChunks : n;
  if (n > planes) n = planes;
  for (int k = 0; k <= n; ++k) zc[k] = h->p.z_lo + (int)((long long)planes * k / n);
  return (int)n;
}

// one chunk of rho / u between host and device staging (planes [z0, z1) of each component)
int copy_chunk(lbm_handle_s* h, double* dev_rho, double* dev_u, double* host_rho, double* host_u, int z0, int z1, bool to_device) {
  const size_t off = (size_t)h->nx * h->ny * z0, n = (size_t)h->nx * h->ny * (z1 - z0) * sizeof(double);
  const cudaMemcpyKind kind = to_device ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToHost;
  if (host_rho) {
    if (to_device) CUDA_TRY(cudaMemcpyAsync(dev_rho + off, host_rho + off, n, kind, h->copy_stream));
    else CUDA_TRY(cudaMemcpyAsync(host_rho + off, dev_rho + off, n, kind, h->copy_stream));
  }
  if (host_u) {
    for (int d = 0; d < 3; ++d) {
      const size_t o = (size_t)h->N * d + off;
      if (to_device) CUDA_TRY(cudaMemcpyAsync(dev_u + o, host_u + o, n, kind, h->copy_stream));
      else CUDA_TRY(cudaMemcpyAsync(host_u + o, dev_u + o, n, kind, h->copy_stream));
    }
  }
  return LBM_OK;
}

void free_geometry(lbm_handle_s* h) {
  gfree(h, h->geo);
  gfree(h, h->active);
  gfree(h, h->links);
  h->geo = h->active = nullptr;
  h->links = nullptr;
  h->has_geo = false;
  h->wall_model = LBM_WALL_HALFWAY;
  h->p.links = nullptr;
  h->p.nodal = 0;
}

int alloc_geometry(lbm_handle_s* h) {
  if (h->geo) return LBM_OK;
  cudaError_t e = gmalloc(h, (void**)&h->geo, (size_t)h->N, false);
  if (e == cudaSuccess) e = gmalloc(h, (void**)&h->active, (size_t)h->N, false);
  if (e == cudaSuccess) e = gmalloc(h, (void**)&h->links, (size_t)h->N * sizeof(uint32_t), false);
  if (e != cudaSuccess) {
    cudaGetLastError();
    free_geometry(h);
    return fail(LBM_ENOMEM, "lbm_set_geometry: out of device memory for the geometry arrays");
  }
  return LBM_OK;
}

// geo_dev: device pointer to N bytes (must not alias h->geo or h->active), or NULL (all fluid)
int do_set_geometry(lbm_handle_s* h, const uint8_t* geo_dev, int wall_model) {
  if (wall_model != LBM_WALL_HALFWAY && wall_model != LBM_WALL_NODAL)
    return fail(LBM_EINVAL, "lbm_set_geometry: wall_model must be LBM_WALL_HALFWAY or LBM_WALL_NODAL");
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  if (!geo_dev && wall_model == LBM_WALL_HALFWAY && !h->p.any_sym) {  // back to the analytic box
    free_geometry(h);
    return LBM_OK;
  }
  {
    int rc = alloc_geometry(h);
    if (rc) return rc;
  }
  h->wall_model = wall_model;
  h->has_geo = true;
  h->p.links = h->links;
  h->p.nodal = wall_model == LBM_WALL_NODAL;
  const Ctx c = make_ctx(h);
  // the kernels read the caller's mask directly (no runtime memcpy on a pointer the library does not own)
  LBM_Q_CALL(h, launch_geometry, c, geo_dev, h->geo, h->active, h->links, h->p.nodal);
  h->launches += 2;
  h->stepped = false;
  int rc = check_launch("lbm_set_geometry");
  if (rc) return rc;
  // the caller's mask has been read when the call returns (it may be a temporary)
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  return LBM_OK;
}

}  // namespace

// =========================================================================================
extern "C" {

const char* lbm_last_error(void) { return g_err.c_str(); }

int lbm_lattice(int lattice, int32_t* e, double* t) {
  const int Q = lattice & 0xff;
  if (!e || !t) return fail(LBM_EINVAL, "lbm_lattice: NULL output");
  auto fill = [&](auto L, int q) {
    using Lt = decltype(L);
    for (int a = 0; a < q; ++a) {
      int s = 0;
      for (int d = 0; d < 3; ++d) {
        e[3 * a + d] = Lt::e[a][d];
        s += e[3 * a + d] * e[3 * a + d];
      }
      t[a] = s == 0 ? Lt::w0 : s == 1 ? Lt::w1 : s == 2 ? Lt::w2 : Lt::w3;
    }
  };
  if (Q == 9) fill(Lattice<9>{}, 9);
  else if (Q == 19) fill(Lattice<19>{}, 19);
  else if (Q == 27) fill(Lattice<27>{}, 27);
  else return fail(LBM_EINVAL, "lbm_lattice: lattice must be LBM_D2Q9, LBM_D3Q19 or LBM_D3Q27");
  return LBM_OK;
}

// slab: nz = nz_local + 2 planes are allocated (halo below and above), z0 / nz_global place the slab in the box
static lbm_handle create_impl(int nx, int ny, int nz, int lattice, double tau, const lbm_bc_t* bc, bool slab, int z0, int nz_global) {
  const int Q = lattice & 0xff;
  if (Q != 9 && Q != 19 && Q != 27) { fail(LBM_EINVAL, "lbm_create: lattice must be LBM_D2Q9, LBM_D3Q19 or LBM_D3Q27"); return nullptr; }
  if (nx < 1 || ny < 1 || nz < 1) { fail(LBM_EINVAL, "lbm_create: nx, ny, nz must be >= 1"); return nullptr; }
  if ((long long)nx * ny * nz >= (1LL << 31)) { fail(LBM_EUNSUPPORTED, "lbm_create: nx*ny*nz must be < 2^31 (cell indices are 32-bit)"); return nullptr; }
  if (nz > 65535 || ny > 65535) { fail(LBM_EINVAL, "lbm_create: ny or nz exceeds the launch grid limits"); return nullptr; }
  if (!(tau > 0.5) || !std::isfinite(tau)) { fail(LBM_EINVAL, "lbm_create: tau must be finite and > 0.5"); return nullptr; }
  int scheme = lattice & (3 << 12);
  const bool scheme_auto = scheme == LBM_SCHEME_AUTO;
  if (scheme_auto) scheme = LBM_SCHEME_AB;  // revisited below once the faces are known
  if (scheme != LBM_SCHEME_AB && scheme != LBM_SCHEME_AA) { fail(LBM_EINVAL, "lbm_create: unknown storage scheme"); return nullptr; }
  if (lattice & ~(0xff | LBM_EQ_INCOMP | (3 << 12) | LBM_STORE_F32 | LBM_LAYOUT_SOA)) { fail(LBM_EINVAL, "lbm_create: unknown bits in lattice"); return nullptr; }

  lbm_handle_s* h = new (std::nothrow) lbm_handle_s();
  if (!h) { fail(LBM_ENOMEM, "lbm_create: out of host memory"); return nullptr; }
  std::memset(h, 0, sizeof(*h));
  h->nx = nx; h->ny = ny; h->nz = nz; h->Q = Q;
  h->eq = (lattice & LBM_EQ_INCOMP) ? 1 : 0;
  h->scheme = scheme;
  h->f32 = (lattice & LBM_STORE_F32) ? 1 : 0;
  h->N = (long long)nx * ny * nz;
  h->tau = tau;
  h->soa = (lattice & LBM_LAYOUT_SOA) ? 1 : 0;
  // In-plane storage offsets x + y*rs are 32-bit in the kernels.  Row-interleaved: rs = Q*nx, so the bound is
  // Q*nx*ny < 2^31; a plane beyond it (a 16384^2 D2Q9 grid) is stored as a plain structure of arrays, whose in-plane
  // bound nx*ny < 2^31 holds for every grid accepted above.  The layout is internal: results are identical bit for bit.
  if (!h->soa && (long long)Q * nx * ny >= (1LL << 31)) h->soa = 1;
  Params& p = h->p;
  p.nx = nx; p.ny = ny; p.nz = nz; p.N = h->N;
  if (h->soa) { p.ds = h->N; p.rs = nx; p.zs = (long long)nx * ny; }
  else { p.ds = nx; p.rs = Q * nx; p.zs = (long long)Q * nx * ny; }
  p.omega = 1.0 / tau;
  if (bc) {
    for (int k = 0; k < 6; ++k) {
      const int kind = bc->face_kind[k];
      if (kind != LBM_FACE_PERIODIC && kind != LBM_FACE_BOUNCE && kind != LBM_FACE_MOVING && kind != LBM_FACE_PRESSURE && kind != LBM_FACE_SYMMETRY) {
        delete h; fail(LBM_EINVAL, "lbm_create: unknown face kind"); return nullptr;
      }
      p.wall[k] = kind != LBM_FACE_PERIODIC;
      p.kind[k] = kind;
      p.open[k] = kind == LBM_FACE_MOVING || kind == LBM_FACE_PRESSURE;
      p.sym[k] = kind == LBM_FACE_SYMMETRY;
      p.any_sym |= p.sym[k];
      for (int d = 0; d < 3; ++d) {
        p.face_u[k][d] = kind == LBM_FACE_MOVING ? bc->face_u[k][d] : 0.0;
        if (!std::isfinite(p.face_u[k][d])) { delete h; fail(LBM_EINVAL, "lbm_create: non-finite wall velocity"); return nullptr; }
      }
      p.any_open |= p.open[k];
    }
    for (int d = 0; d < 3; ++d) {
      if (p.wall[2 * d] != p.wall[2 * d + 1]) { delete h; fail(LBM_EINVAL, "lbm_create: periodic must be set on both faces of an axis"); return nullptr; }
      p.F[d] = bc->force[d];
      if (!std::isfinite(p.F[d])) { delete h; fail(LBM_EINVAL, "lbm_create: non-finite force"); return nullptr; }
    }
    h->stream = (cudaStream_t)bc->stream;
  }
  // LBM_SCHEME_AUTO: two buffers (faster on every grid that streams from HBM) — except where ONE
  // buffer fits the L2 and two do not: there the in-place scheme runs out of the L2 and the two-buffer one does not
  // (1024^2 D2Q9, 75 MB per buffer: 61.1 vs 43.1 GLUPS; 80^3 D3Q19, 78 MB: 23.9 vs 19.2; at 104 MB +4 %, at 42 MB +-0).
  if (scheme_auto && !slab && !p.any_sym) {
    int dev = 0, l2 = 0;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev) == cudaSuccess && l2 > 0) {
      const double one = (double)h->N * Q * (h->f32 ? 4 : 8);
      if (one > 0.4 * l2 && one <= 0.8 * l2) scheme = h->scheme = LBM_SCHEME_AA;
    }
    cudaGetLastError();
  }
  if (p.any_sym && scheme == LBM_SCHEME_AA) {
    delete h; fail(LBM_EUNSUPPORTED, "lbm_create: LBM_FACE_SYMMETRY needs LBM_SCHEME_AB"); return nullptr;
  }
  p.z_lo = 0;
  p.z_hi = nz;
  p.zg_off = 0;
  p.nz_glob = nz;
  for (int k = 0; k < 6; ++k) p.face_rho[k] = 1.0;
  if (slab) {
    h->slab = true;
    h->z0 = z0; h->nz_global = nz_global; h->nz_local = nz - 2;
    h->device_sync = 1;
    p.slab = 1;
    p.z_lo = 1;
    p.z_hi = nz - 1;
    // the z faces of the box act only on the slab that owns them; elsewhere the cut is an ordinary interior plane
    const bool owns_lo = z0 == 0, owns_hi = z0 + h->nz_local == nz_global;
    if (!owns_lo) { p.wall[4] = 0; p.open[4] = 0; p.sym[4] = 0; p.kind[4] = LBM_FACE_PERIODIC; }
    if (!owns_hi) { p.wall[5] = 0; p.open[5] = 0; p.sym[5] = 0; p.kind[5] = LBM_FACE_PERIODIC; }
    p.any_open = 0;
    for (int k = 0; k < 6; ++k) p.any_open |= p.open[k];
    p.zg_off = z0 - 1;
    p.nz_glob = nz_global;
  }
  // (walls: the coordinate-test kernels are needed if ANY face of this handle is a wall)
  h->walls = p.wall[0] || p.wall[1] || p.wall[2] || p.wall[3] || p.wall[4] || p.wall[5];
  h->forced = p.F[0] != 0.0 || p.F[1] != 0.0 || p.F[2] != 0.0;
  // default block: as long along x as the row allows (coalesced, vector-friendly), 256 threads
  int bx = 32;
  while (bx < nx && bx < 256) bx *= 2;
  h->bx = h->by = 0;  // default_block() at launch time (it depends on the geometry)
  h->persistent = 1;
  h->two_step = 1;
  {
    int dev = 0, l2 = 0;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev) == cudaSuccess) h->l2_bytes = l2;
    cudaGetLastError();
  }
  h->fbx = bx;

  const int nbuf = scheme == LBM_SCHEME_AB ? 2 : 1;
  cudaError_t e = cudaSuccess;
  for (int b = 0; b < nbuf && e == cudaSuccess; ++b) e = gmalloc(h, &h->buf[b], h->buf_bytes(), true);
  if (e == cudaSuccess) e = gmalloc(h, (void**)&h->partials, (size_t)kMaxChunks * kReduceBlocks * kDiag * sizeof(double), true);
  if (e == cudaSuccess) e = gmalloc(h, (void**)&h->diag_dev, kDiag * sizeof(double), true);
  if (e == cudaSuccess) e = cudaMalloc((void**)&h->guard_bad, sizeof(unsigned long long));
  if (e == cudaSuccess) e = cudaMallocHost((void**)&h->diag_pinned, kDiag * sizeof(double));
  if (e == cudaSuccess && slab) {
    e = gmalloc(h, (void**)&h->flags, 2 * sizeof(uint32_t), false);
    if (e == cudaSuccess) e = cudaMemset(h->flags, 0, 2 * sizeof(uint32_t));
  }
  if (e != cudaSuccess) {
    const bool oom = (e == cudaErrorMemoryAllocation);
    std::string msg = std::string("lbm_create: ") + cudaGetErrorString(e);
    cudaGetLastError();
    lbm_destroy(h);
    fail(oom ? LBM_ENOMEM : LBM_ECUDA, msg);
    return nullptr;
  }
  if (p.any_sym) {  // D:R25: mirror links are resolved through the link mask: build it for the empty geometry
    if (do_set_geometry(h, nullptr, LBM_WALL_HALFWAY) != LBM_OK) {
      const std::string msg = g_err;
      lbm_destroy(h);
      g_err = msg;
      return nullptr;
    }
  }
  return h;
}

lbm_handle lbm_create(int nx, int ny, int nz, int lattice, double tau, const lbm_bc_t* bc) {
  return create_impl(nx, ny, nz, lattice, tau, bc, false, 0, nz);
}

lbm_handle lbm_create_slab(int nx, int ny, int nz_local, int z0, int nz_global, int lattice, double tau, const lbm_bc_t* bc) {
  if (nz_local < 1 || z0 < 0 || nz_global < 1 || (long long)z0 + nz_local > nz_global) {
    fail(LBM_EINVAL, "lbm_create_slab: need nz_local >= 1, z0 >= 0 and z0 + nz_local <= nz_global");
    return nullptr;
  }
  int scheme = lattice & (3 << 12);
  if (scheme == LBM_SCHEME_AA) { fail(LBM_EUNSUPPORTED, "lbm_create_slab: z-slabs need LBM_SCHEME_AB"); return nullptr; }
  if (nz_local > 65533) { fail(LBM_EINVAL, "lbm_create_slab: nz_local exceeds the launch grid limits"); return nullptr; }
  return create_impl(nx, ny, nz_local + 2, lattice, tau, bc, true, z0, nz_global);
}

int lbm_slab_export(lbm_handle h, lbm_slab_peer_t* out) {
  if (!h || !out) return fail(LBM_EINVAL, "lbm_slab_export: NULL argument");
  if (!h->slab) return fail(LBM_EINVAL, "lbm_slab_export: not a slab handle (lbm_create_slab)");
  std::memset(out, 0, sizeof(*out));
  out->buf[0] = (uint64_t)h->buf[0];
  out->buf[1] = (uint64_t)h->buf[1];
  out->flags = (uint64_t)h->flags;
  out->plane_stride = h->N;
  out->nz_local = h->nz_local;
  out->Q = h->Q;
  out->elem_bytes = (int32_t)h->elem();
  out->layout_soa = h->soa;
  out->stream = (uint64_t)h->stream;
  int dev = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  out->device = dev;
  out->pid = (int64_t)getpid();
  static_assert(sizeof(cudaIpcMemHandle_t) == 64, "lbm_slab_peer_t reserves 64 bytes per IPC handle");
  cudaIpcMemHandle_t ih;
  void* ptrs[3] = {h->buf[0], h->buf[1], (void*)h->flags};
  uint8_t* dsts[3] = {out->ipc_buf[0], out->ipc_buf[1], out->ipc_flags};
  for (int k = 0; k < 3; ++k) {
    // without IPC support the descriptor still serves slabs of the same process
    // (the handle names the whole allocation, guard zone included: map_peer adds kGuard to what it opens)
    if (cudaIpcGetMemHandle(&ih, (char*)ptrs[k] - kGuard) == cudaSuccess) std::memcpy(dsts[k], &ih, sizeof(ih));
    else cudaGetLastError();
  }
  return LBM_OK;
}

namespace {
// Address of a neighbour's allocation as this process / device may use it.
int map_peer(lbm_handle_s* h, const lbm_slab_peer_t* d, uint64_t addr, const uint8_t* ipc, void** out) {
  if (d->pid == (int64_t)getpid()) {
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (d->device != dev) {
      int can = 0;
      CUDA_TRY(cudaDeviceCanAccessPeer(&can, dev, d->device));
      if (!can) return fail(LBM_EUNSUPPORTED, "lbm_slab_connect: no peer access between the two devices");
      cudaError_t e = cudaDeviceEnablePeerAccess(d->device, 0);
      if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled) return cuda_fail(e, "cudaDeviceEnablePeerAccess");
      cudaGetLastError();
    }
    *out = (void*)addr;
    return LBM_OK;
  }
  cudaIpcMemHandle_t ih;
  std::memcpy(&ih, ipc, sizeof(ih));
  void* ptr = nullptr;
  cudaError_t e = cudaIpcOpenMemHandle(&ptr, ih, cudaIpcMemLazyEnablePeerAccess);
  if (e != cudaSuccess) return cuda_fail(e, "cudaIpcOpenMemHandle");
  if (h->n_ipc_opened < 6) h->ipc_opened[h->n_ipc_opened++] = ptr;
  *out = (char*)ptr + kGuard;
  return LBM_OK;
}

void close_peers(lbm_handle_s* h) {
  for (int k = 0; k < h->n_ipc_opened; ++k) cudaIpcCloseMemHandle(h->ipc_opened[k]);
  h->n_ipc_opened = 0;
  h->peer_lo[0] = h->peer_lo[1] = h->peer_hi[0] = h->peer_hi[1] = nullptr;
  h->peer_lo_flag = h->peer_hi_flag = nullptr;
  h->shares_stream = false;
  cudaGetLastError();
}
}  // namespace

int lbm_slab_connect(lbm_handle h, const lbm_slab_peer_t* lower, const lbm_slab_peer_t* upper) {
  if (!h) return fail(LBM_EINVAL, "lbm_slab_connect: NULL handle");
  if (!h->slab) return fail(LBM_EINVAL, "lbm_slab_connect: not a slab handle (lbm_create_slab)");
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  close_peers(h);
  const long long plane = (long long)h->nx * h->ny;
  bool shares = false;
  for (int side = 0; side < 2; ++side) {
    const lbm_slab_peer_t* d = side ? upper : lower;
    if (!d) continue;
    if (d->plane_stride != plane * (d->nz_local + 2) || d->nz_local < 1)
      { close_peers(h); return fail(LBM_EINVAL, "lbm_slab_connect: neighbour descriptor does not match this slab's nx, ny"); }
    // the halo stores write the neighbour's buffer in THIS slab's lattice, element type and layout
    if (d->Q != h->Q || d->elem_bytes != (int32_t)h->elem() || d->layout_soa != h->soa)
      { close_peers(h); return fail(LBM_EINVAL, "lbm_slab_connect: neighbour has another lattice, storage type or layout"); }
    // two different slabs of one process on ONE stream.  With device-side ordering the second step of one waits (in the
    // stream) for the first step of the other, which is queued behind that wait: refused.  Host-ordered
    // (lbm_slab_set_sync(h, 0) before this call) the stream itself orders the steps issued slab by slab: allowed.
    if (d->pid == (int64_t)getpid() && d->buf[0] != (uint64_t)h->buf[0] && d->stream == (uint64_t)h->stream) {
      int dev = 0;
      cudaGetDevice(&dev);
      if (d->device == dev) {
        if (h->device_sync) {
          close_peers(h);
          return fail(LBM_EINVAL, "lbm_slab_connect: connected slabs of one process need a stream each (lbm_bc_t.stream) under device-side "
                                  "ordering; for host-ordered stepping on a shared stream call lbm_slab_set_sync(h, 0) before lbm_slab_connect");
        }
        shares = true;
      }
    }
    void* b[2] = {nullptr, nullptr};
    void* fl = nullptr;
    int rc = map_peer(h, d, d->buf[0], d->ipc_buf[0], &b[0]);
    if (!rc) rc = map_peer(h, d, d->buf[1], d->ipc_buf[1], &b[1]);
    if (!rc) rc = map_peer(h, d, d->flags, d->ipc_flags, &fl);
    if (rc) { close_peers(h); return rc; }
    if (side == 0) {  // lower neighbour: we fill its UPPER halo plane and write its "upper neighbour" counter
      h->peer_lo[0] = b[0]; h->peer_lo[1] = b[1];
      // the neighbour stores in the same layout: its direction stride and the offset of its upper halo plane
      h->peer_lo_N = h->soa ? d->plane_stride : h->p.ds;
      h->peer_lo_off = h->p.zs * (d->nz_local + 1);
      h->peer_lo_flag = (uint32_t*)fl + 1;
    } else {          // upper neighbour: its LOWER halo plane, its "lower neighbour" counter
      h->peer_hi[0] = b[0]; h->peer_hi[1] = b[1];
      h->peer_hi_N = h->soa ? d->plane_stride : h->p.ds;
      h->peer_hi_off = 0;
      h->peer_hi_flag = (uint32_t*)fl;
    }
  }
  h->p.push_lo_N = h->peer_lo_N; h->p.push_lo_off = h->peer_lo_off;
  h->p.push_hi_N = h->peer_hi_N; h->p.push_hi_off = h->peer_hi_off;
  h->shares_stream = shares;
  return LBM_OK;
}

int lbm_slab_set_sync(lbm_handle h, int device_sync) {
  if (!h || !h->slab) return fail(LBM_EINVAL, "lbm_slab_set_sync: not a slab handle");
  if (device_sync && h->shares_stream)
    return fail(LBM_EINVAL, "lbm_slab_set_sync: this slab is connected to a slab on the same stream; device-side ordering would deadlock there");
  h->device_sync = device_sync ? 1 : 0;
  return LBM_OK;
}

void lbm_destroy(lbm_handle h) {
  if (!h) return;
  cudaStreamSynchronize(h->stream);
  if (h->slab) close_peers(h);
  gfree(h, h->flags);
  for (int b = 0; b < 2; ++b) gfree(h, h->buf[b]);
  gfree(h, h->partials);
  gfree(h, h->diag_dev);
  if (h->guard_bad) cudaFree(h->guard_bad);
  if (h->diag_pinned) cudaFreeHost(h->diag_pinned);
  gfree(h, h->scratch);
  if (h->copy_stream) {
    cudaStreamSynchronize(h->copy_stream);
    for (int k = 0; k < kMaxChunks; ++k) cudaEventDestroy(h->chunk_ev[k]);
    cudaEventDestroy(h->fence_ev);
    cudaStreamDestroy(h->copy_stream);
  }
  for (int k = 0; k < 6; ++k)
    gfree(h, (void*)h->p.face_prof[k]);
  free_geometry(h);
  cudaGetLastError();
  delete h;
}

// cells of face `face` of the WHOLE box (a slab handle takes the profile of the whole face)
static long long face_cells(const lbm_handle_s* h, int face) {
  const long long nzg = h->slab ? h->nz_global : h->nz;
  return face < 2 ? (long long)h->ny * nzg : face < 4 ? (long long)h->nx * nzg : (long long)h->nx * h->ny;
}

static int set_face_velocity_impl(lbm_handle h, int face, const double* u, cudaMemcpyKind kind, const char* who) {
  if (!h) return fail(LBM_EINVAL, std::string(who) + ": NULL handle");
  if (face < 0 || face > 5) return fail(LBM_EINVAL, std::string(who) + ": face must be 0..5");
  // the kind the caller gave the face of the box (a slab that does not own a z face still accepts its profile)
  const bool owns = !(h->slab && face >= 4 && h->p.kind[face] == LBM_FACE_PERIODIC);
  if (owns && h->p.kind[face] != LBM_FACE_MOVING) return fail(LBM_EINVAL, std::string(who) + ": the face is not LBM_FACE_MOVING");
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  if (!u) {
    gfree(h, (void*)h->p.face_prof[face]);
    h->p.face_prof[face] = nullptr;
    return LBM_OK;
  }
  const size_t bytes = (size_t)face_cells(h, face) * 3 * sizeof(double);
  double* dst = (double*)h->p.face_prof[face];
  if (!dst) {
    if (gmalloc(h, (void**)&dst, bytes, false) != cudaSuccess) {
      cudaGetLastError();
      return fail(LBM_ENOMEM, std::string(who) + ": out of device memory for the face profile");
    }
    h->p.face_prof[face] = dst;
  }
  CUDA_TRY(cudaMemcpyAsync(dst, u, bytes, kind, h->stream));
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  return LBM_OK;
}

int lbm_set_face_velocity(lbm_handle h, int face, const double* u) {
  return set_face_velocity_impl(h, face, u, cudaMemcpyDeviceToDevice, "lbm_set_face_velocity");
}

int lbm_set_face_velocity_host(lbm_handle h, int face, const double* u_host) {
  return set_face_velocity_impl(h, face, u_host, cudaMemcpyHostToDevice, "lbm_set_face_velocity_host");
}

int lbm_set_face_density(lbm_handle h, const double* rho6) {
  if (!h || !rho6) return fail(LBM_EINVAL, "lbm_set_face_density: NULL argument");
  for (int k = 0; k < 6; ++k)
    if (!std::isfinite(rho6[k])) return fail(LBM_EINVAL, "lbm_set_face_density: non-finite density");
  for (int k = 0; k < 6; ++k) h->p.face_rho[k] = rho6[k];  // read by the kernels launched from now on
  return LBM_OK;
}

int lbm_set_geometry(lbm_handle h, const uint8_t* geo, int wall_model) {
  if (!h) return fail(LBM_EINVAL, "lbm_set_geometry: NULL handle");
  return do_set_geometry(h, geo, wall_model);
}

// bytes of the mask the caller passes: N, or on a z-slab two more planes (two halo planes per side, include/lbm.h)
static size_t geo_input_bytes(const lbm_handle_s* h) {
  return (size_t)h->N + (h->slab ? 2 * (size_t)h->nx * h->ny : 0);
}

int lbm_set_geometry_host(lbm_handle h, const uint8_t* geo_host, int wall_model) {
  if (!h) return fail(LBM_EINVAL, "lbm_set_geometry_host: NULL handle");
  if (!geo_host) return do_set_geometry(h, nullptr, wall_model);
  if (wall_model != LBM_WALL_HALFWAY && wall_model != LBM_WALL_NODAL)
    return fail(LBM_EINVAL, "lbm_set_geometry: wall_model must be LBM_WALL_HALFWAY or LBM_WALL_NODAL");
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  {
    int rc = alloc_geometry(h);
    if (rc) return rc;
  }
  // stage the host mask in the tail of the link-mask array (4N bytes, rebuilt last by do_set_geometry); a slab's
  // mask is two planes longer than N and goes to the scratch buffer instead
  uint8_t* stage = nullptr;
  if (h->slab) {
    int rc = ensure_scratch(h, geo_input_bytes(h));
    if (rc) return rc;
    stage = (uint8_t*)h->scratch;
  } else {
    stage = (uint8_t*)h->links + (size_t)h->N * 3;
  }
  CUDA_TRY(cudaMemcpyAsync(stage, geo_host, geo_input_bytes(h), cudaMemcpyHostToDevice, h->stream));
  return do_set_geometry(h, stage, wall_model);
}

int lbm_boundary_force(lbm_handle h, double* F) {
  if (!h || !F) return fail(LBM_EINVAL, "lbm_boundary_force: NULL argument");
  if (!h->has_geo) return fail(LBM_EINVAL, "lbm_boundary_force: no geometry set (lbm_set_geometry)");
  if (!h->stepped) return fail(LBM_EINVAL, "lbm_boundary_force: defined only after at least one lbm_step since the populations were set");
  const Ctx c = make_ctx(h);
  LBM_Q_CALL(h, launch_boundary_force, c, read_mode(h), h->buf[h->cur], h->geo, h->partials);
  reduce_final_kernel<><<<1, 256, 0, h->stream>>>(h->partials, c.flat_grid, h->diag_dev);
  h->launches += 2;
  int rc = check_launch("lbm_boundary_force");
  if (rc) return rc;
  CUDA_TRY(cudaMemcpyAsync(h->diag_pinned, h->diag_dev, kDiag * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  for (int d = 0; d < 3; ++d) F[d] = h->diag_pinned[d];
  return LBM_OK;
}

int lbm_init_equilibrium(lbm_handle h, const double* rho, const double* u) {
  if (!h) return fail(LBM_EINVAL, "lbm_init_equilibrium: NULL handle");
  return do_init(h, rho, u);
}

int lbm_init_equilibrium_host(lbm_handle h, const double* rho_host, const double* u_host) {
  if (!h) return fail(LBM_EINVAL, "lbm_init_equilibrium_host: NULL handle");
  if (!rho_host && !u_host) return do_init(h, nullptr, nullptr);
  const int mode = init_target(h);  // fixes h->cur: the staging below is the OTHER buffer
  double* stage = nullptr;
  int rc = host_staging(h, &stage);
  if (!rc) rc = ensure_copy_stream(h);
  if (rc) return rc;
  double* d_rho = rho_host ? stage : nullptr;
  double* d_u = u_host ? stage + h->N : nullptr;
  const Ctx c = make_ctx(h);
  int zc[kMaxChunks + 1];
  const int n = plane_chunks(h, zc);
  // the copies may start once everything queued on the handle's stream has left the staging buffer
  CUDA_TRY(cudaEventRecord(h->fence_ev, h->stream));
  CUDA_TRY(cudaStreamWaitEvent(h->copy_stream, h->fence_ev, 0));
  for (int k = 0; k < n; ++k) {
    // the kernel of a chunk reads rho, u of its own cells only (it pushes f_a towards the upstream slot), so chunk k
    // is initialised while chunk k+1 is still on the bus
    rc = copy_chunk(h, d_rho, d_u, const_cast<double*>(rho_host), const_cast<double*>(u_host), zc[k], zc[k + 1], true);
    if (rc) return rc;
    CUDA_TRY(cudaEventRecord(h->chunk_ev[k], h->copy_stream));
    CUDA_TRY(cudaStreamWaitEvent(h->stream, h->chunk_ev[k], 0));
    launch_init_rows(h, c, mode, d_rho, d_u, h->ny * zc[k], h->ny * zc[k + 1]);
  }
  finish_init(h);
  rc = check_launch("init_equilibrium_host");
  // The copies run on a stream the caller cannot see, so the caller cannot know when the host arrays may be reused:
  // wait here until the last chunk has left the host (the copy stream is in order, so that covers every chunk).  Only
  // the copies are waited for; the initialisation kernels of the last chunks may still be running on return.
  CUDA_TRY(cudaEventSynchronize(h->chunk_ev[n - 1]));
  return rc;
}

int lbm_step(lbm_handle h, int nsteps) {
  if (!h) return fail(LBM_EINVAL, "lbm_step: NULL handle");
  if (nsteps < 0) return fail(LBM_EINVAL, "lbm_step: nsteps must be >= 0");
  if (nsteps == 0) return LBM_OK;
  Ctx c = make_ctx(h);
  // Small grids (both buffers fit the L2): all steps of this call in ONE cooperative launch of the persistent kernel;
  // otherwise pairs of steps where stream_collide_ab2 applies (below), and one launch per step for everything else.
  if (h->persistent && h->scheme == LBM_SCHEME_AB && !h->slab && nsteps >= 2 && h->l2_bytes > 0 &&
      2.0 * (double)h->buf_bytes() <= 0.8 * h->l2_bytes) {
    bool ok = false;
    LBM_Q_CALL_RET(h, ok, launch_step_ab_persistent, c, h->buf[h->cur], h->buf[h->cur ^ 1], nsteps);
    if (ok) {
      h->cur ^= (nsteps & 1);
      h->time += nsteps;
      ++h->launches;
      h->stepped = true;
      return check_launch("lbm_step");
    }
  }
  if (h->persistent && h->scheme == LBM_SCHEME_AA && nsteps >= 2 && h->l2_bytes > 0 &&
      (double)h->buf_bytes() <= 0.8 * h->l2_bytes) {
    bool ok = false;
    LBM_Q_CALL_RET(h, ok, launch_step_aa_persistent, c, h->buf[0], nsteps, h->phase);
    if (ok) {
      h->phase ^= (nsteps & 1);
      h->time += nsteps;
      ++h->launches;
      h->stepped = true;
      return check_launch("lbm_step");
    }
  }
  // A/B, periodic D3Q19 in fp64: steps in pairs, two per pass through HBM (stream_collide_ab2); bit-identical to two
  // single steps, so a trailing odd step — or every step, where that kernel does not apply — takes the one-step kernel
  bool pairs = h->two_step && h->scheme == LBM_SCHEME_AB && !h->slab;
  for (int s = 0; s < nsteps;) {
    if (pairs && s + 2 <= nsteps) {
      bool ok = false;
      LBM_Q_CALL_RET(h, ok, launch_step_ab2, c, h->buf[h->cur], h->buf[h->cur ^ 1], h->two_step == 2);
      if (ok) {
        h->cur ^= 1;
        ++h->launches;
        h->time += 2;
        s += 2;
        continue;
      }
      pairs = false;
    }
    if (h->slab) {
      int rc = launch_step_slab(h, c);
      if (rc) return rc;
    } else {
      launch_step(h, c);
    }
    ++h->time;
    ++s;
  }
  h->stepped = true;
  return check_launch("lbm_step");
}

int lbm_moments(lbm_handle h, double* rho, double* u, double* diagnostics) {
  if (!h) return fail(LBM_EINVAL, "lbm_moments: NULL handle");
  if (!rho && !u && !diagnostics) return LBM_OK;
  return do_moments(h, rho, u, diagnostics);
}

int lbm_moments_host(lbm_handle h, double* rho_host, double* u_host, double* diagnostics) {
  if (!h) return fail(LBM_EINVAL, "lbm_moments_host: NULL handle");
  if (!rho_host && !u_host && !diagnostics) return LBM_OK;
  if (!rho_host && !u_host) return do_moments(h, nullptr, nullptr, diagnostics);
  double* stage = nullptr;
  int rc = host_staging(h, &stage);
  if (!rc) rc = ensure_copy_stream(h);
  if (!rc) rc = slab_wait_neighbours(h);  // the pull reads the halo planes
  if (rc) return rc;
  double* d_rho = rho_host ? stage : nullptr;
  double* d_u = u_host ? stage + h->N : nullptr;
  const Ctx c = make_ctx(h);
  int zc[kMaxChunks + 1];
  const int n = plane_chunks(h, zc);
  int nblocks = 0;
  for (int k = 0; k < n; ++k) {
    // chunk k goes to the host while chunk k+1 is being computed; every chunk keeps its own block partials
    const int r0 = h->ny * zc[k], r1 = h->ny * zc[k + 1], grid = grid_for_rows(h, r1 - r0);
    LBM_Q_CALL(h, launch_moments, c, read_mode(h), h->buf[h->cur], d_rho, d_u, diagnostics ? h->partials + (size_t)nblocks * kDiag : nullptr, r0, r1, grid);
    ++h->launches;
    nblocks += grid;
    CUDA_TRY(cudaEventRecord(h->chunk_ev[k], h->stream));
    CUDA_TRY(cudaStreamWaitEvent(h->copy_stream, h->chunk_ev[k], 0));
    rc = copy_chunk(h, d_rho, d_u, rho_host, u_host, zc[k], zc[k + 1], false);
    if (rc) return rc;
  }
  rc = check_launch("moments_host");
  if (rc) return rc;
  // whatever the handle's stream runs next (a step overwrites the staging buffer) comes after the copies
  CUDA_TRY(cudaEventRecord(h->fence_ev, h->copy_stream));
  CUDA_TRY(cudaStreamWaitEvent(h->stream, h->fence_ev, 0));
  if (diagnostics) return finish_diagnostics(h, nblocks, diagnostics);  // synchronises the stream, hence the copies
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  return LBM_OK;
}

int lbm_get_populations(lbm_handle h, double* f) {
  if (!h || !f) return fail(LBM_EINVAL, "lbm_get_populations: NULL argument");
  {
    int rc = slab_wait_neighbours(h);
    if (rc) return rc;
  }
  const Ctx c = make_ctx(h);
  LBM_Q_CALL(h, launch_export, c, read_mode(h), h->buf[h->cur], f);
  ++h->launches;
  return check_launch("lbm_get_populations");
}

int lbm_set_populations(lbm_handle h, const double* f) {
  if (!h || !f) return fail(LBM_EINVAL, "lbm_set_populations: NULL argument");
  if (h->scheme != LBM_SCHEME_AB || h->slab) h->cur = 0;
  do_import(h, f, h->cur);
  h->phase = 0;
  h->stepped = false;
  return check_launch("lbm_set_populations");
}

int lbm_debug_arm(lbm_handle h, int poison) {
  if (!h) return fail(LBM_EINVAL, "lbm_debug_arm: NULL handle");
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  for (int k = 0; k < h->n_owned; ++k) {
    char* p = (char*)h->owned[k].p;
    CUDA_TRY(cudaMemsetAsync(p - kGuard, kGuardByte, kGuard, h->stream));
    CUDA_TRY(cudaMemsetAsync(p + h->owned[k].bytes, kGuardByte, kGuard, h->stream));
    // all-ones bytes are a NaN as fp64 and as fp32: whatever is computed from a slot nobody wrote shows up as a
    // non-finite cell (diagnostics[7]) and in every comparison
    if (poison && h->owned[k].floating) CUDA_TRY(cudaMemsetAsync(p, 0xFF, h->owned[k].bytes, h->stream));
  }
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  if (poison) h->stepped = false;
  return LBM_OK;
}

int64_t lbm_debug_check(lbm_handle h) {
  if (!h) return fail(LBM_EINVAL, "lbm_debug_check: NULL handle");
  if (cudaMemsetAsync(h->guard_bad, 0, sizeof(unsigned long long), h->stream) != cudaSuccess) return cuda_fail(cudaGetLastError(), "lbm_debug_check");
  for (int k = 0; k < h->n_owned; ++k) {
    const unsigned char* p = (const unsigned char*)h->owned[k].p;
    guard_count_kernel<<<8, 256, 0, h->stream>>>(p - kGuard, kGuard, h->guard_bad);
    guard_count_kernel<<<8, 256, 0, h->stream>>>(p + h->owned[k].bytes, kGuard, h->guard_bad);
  }
  unsigned long long bad = 0;
  cudaError_t e = cudaMemcpyAsync(&bad, h->guard_bad, sizeof(bad), cudaMemcpyDeviceToHost, h->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
  if (e != cudaSuccess) return cuda_fail(e, "lbm_debug_check");
  return (int64_t)bad;
}

int64_t lbm_time(lbm_handle h) { return h ? h->time : -1; }
int64_t lbm_launch_count(lbm_handle h) { return h ? h->launches : -1; }

int lbm_set_persistent(lbm_handle h, int on) {
  if (!h) return fail(LBM_EINVAL, "lbm_set_persistent: NULL handle");
  h->persistent = on ? 1 : 0;
  return LBM_OK;
}

int lbm_set_two_step(lbm_handle h, int on) {
  if (!h) return fail(LBM_EINVAL, "lbm_set_two_step: NULL handle");
  if (on < 0 || on > 2) return fail(LBM_EINVAL, "lbm_set_two_step: on must be 0, 1 or 2");
  h->two_step = on;
  return LBM_OK;
}

int lbm_set_block(lbm_handle h, int bx, int by) {
  if (!h) return fail(LBM_EINVAL, "lbm_set_block: NULL handle");
  if (bx == 0 && by == 0) {
    h->bx = h->by = 0;
    return LBM_OK;
  }
  if (bx < 1 || by < 1 || bx * by > 256 || (bx * by) % 32 != 0)
    return fail(LBM_EINVAL, "lbm_set_block: bx*by must be a multiple of 32 and <= 256");
  if ((h->ny + by - 1) / by > 65535) return fail(LBM_EINVAL, "lbm_set_block: grid.y would exceed 65535");
  h->bx = bx;
  h->by = by;
  return LBM_OK;
}

}  // extern "C"
