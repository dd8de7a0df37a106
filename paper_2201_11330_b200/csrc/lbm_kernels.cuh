// lbm_kernels.cuh — hand-written sm_100a kernels of the fused stream-collide hot path.
//
// P:n = PAPER.md line n; D:Rk = DESIGN.md §2 reading k; S:§8 = SURVEY.md hot-path table.
// Everything here is HBM-bound (S:§8d: 2*Q*8 B per lattice update, ~1 flop/B): no tensor cores.
// The one-step-per-pass kernels (stream_collide_ab, _ab_f32x2, _aa_*, the persistent kernels) use no shared-memory
// staging: one thread owns one cell (two in _ab_f32x2), the Q populations live in registers, every per-direction stream is
// unit-stride in x (rows f[z][y][a][x]: the Q rows of one grid row are adjacent).
// stream_collide_ab2 — the default for D3Q19 / D3Q27 fp64 boxes without a mask — takes TWO steps per pass: step t runs on
// a tile extended by one cell and stays in shared memory, step t+1 runs from there.
#pragma once
#include <type_traits>
#include <cstdint>
#include <cuda_runtime.h>
#include <cooperative_groups.h>

namespace lbm {

// ---------------------------------------------------------------------------------------
// Compile-time lattice tables (D:R4).  Hand-written; the oracle generates its own.
template <int Q>
struct Lattice;

// D2Q9 exactly as printed in the paper (Eq. 3-4), embedded with e_z = 0.
template <>
struct Lattice<9> {
  static constexpr int e[9][3] = {{-1, -1, 0}, {-1, 0, 0}, {-1, 1, 0}, {0, -1, 0}, {0, 0, 0},
                                  {0, 1, 0},   {1, -1, 0}, {1, 0, 0},  {1, 1, 0}};
  static constexpr double w0 = 4.0 / 9.0, w1 = 1.0 / 9.0, w2 = 1.0 / 36.0, w3 = 0.0;
};

template <>
struct Lattice<19> {
  static constexpr int e[19][3] = {
      {-1, -1, 0}, {-1, 0, -1}, {-1, 0, 0}, {-1, 0, 1}, {-1, 1, 0},                         //  0.. 4
      {0, -1, -1}, {0, -1, 0},  {0, -1, 1}, {0, 0, -1}, {0, 0, 0},                          //  5.. 9
      {0, 0, 1},   {0, 1, -1},  {0, 1, 0},  {0, 1, 1},                                      // 10..13
      {1, -1, 0},  {1, 0, -1},  {1, 0, 0},  {1, 0, 1},  {1, 1, 0}};                         // 14..18
  static constexpr double w0 = 1.0 / 3.0, w1 = 1.0 / 18.0, w2 = 1.0 / 36.0, w3 = 0.0;
};

template <>
struct Lattice<27> {
  static constexpr int e[27][3] = {
      {-1, -1, -1}, {-1, -1, 0}, {-1, -1, 1}, {-1, 0, -1}, {-1, 0, 0}, {-1, 0, 1}, {-1, 1, -1}, {-1, 1, 0}, {-1, 1, 1},
      {0, -1, -1},  {0, -1, 0},  {0, -1, 1},  {0, 0, -1},  {0, 0, 0},  {0, 0, 1},  {0, 1, -1},  {0, 1, 0},  {0, 1, 1},
      {1, -1, -1},  {1, -1, 0},  {1, -1, 1},  {1, 0, -1},  {1, 0, 0},  {1, 0, 1},  {1, 1, -1},  {1, 1, 0},  {1, 1, 1}};
  static constexpr double w0 = 8.0 / 27.0, w1 = 2.0 / 27.0, w2 = 1.0 / 54.0, w3 = 1.0 / 216.0;
};

template <int Q, int A>
struct Dir {
  static constexpr int ex = Lattice<Q>::e[A][0], ey = Lattice<Q>::e[A][1], ez = Lattice<Q>::e[A][2];
  static constexpr int s = ex * ex + ey * ey + ez * ez;
  static constexpr double t = (s == 0) ? Lattice<Q>::w0 : (s == 1) ? Lattice<Q>::w1 : (s == 2) ? Lattice<Q>::w2 : Lattice<Q>::w3;
  static constexpr int opp = Q - 1 - A;
};

template <int I>
struct IC {
  static constexpr int value = I;
};
template <int I, int N, typename F>
__device__ __forceinline__ void static_for(F&& f) {
  if constexpr (I < N) {
    f(IC<I>{});
    static_for<I + 1, N>(f);
  }
}

// Resident 256-thread blocks per SM the fused kernels are compiled for (register cap 80 / 128).
// Measured on B200: the A/B D3Q19 kernels fit 80 registers without spilling and need the third block;
// the fp32-storage A/B kernel keeps its populations packed (collide_shifted) and fits 64 registers, which
// buys the fourth block its half-size loads need; the forced and in-place variants and D3Q27 spill below 128.
template <int Q, bool FORCE, bool INPLACE, int STBYTES = 8>
constexpr int kMinBlocks = (Q == 9) ? (FORCE || INPLACE ? 3 : 4) : (Q == 27 && STBYTES == 4 && !INPLACE) ? 3 : (Q == 19 && STBYTES == 4 && !INPLACE) ? (FORCE ? 3 : 4) : (Q == 19 && !FORCE && !INPLACE) ? 3 : 2;

// ---------------------------------------------------------------------------------------
// How a cell finds out that a link has no upstream node (template parameter BC):
//   BC_PERIODIC  never                                           (no test at all)
//   BC_WALLS     coordinate tests against the non-periodic faces (0 B/cell)
//   BC_GEO       one 32-bit link mask per cell, built once by build_links_kernel from the
//                solid mask `geo` and the faces           (4 B/cell read per step);
//                also every handle with a SYMMETRY face (D:R25)
enum { BC_PERIODIC = 0, BC_WALLS = 1, BC_GEO = 2 };

struct Params {
  int nx, ny, nz;
  long long N;          // cells = component stride of the arrays at the interface (rho, u, canonical f)
  // Storage layout of the population buffers: element (x, y, z, a) sits at
  //   a*ds + x + y*rs + z*zs.
  // Row-interleaved (default): ds = nx, rs = Q*nx, zs = Q*nx*ny, i.e. f[z][y][a][x] — the Q rows a block streams
  // lie next to each other in memory instead of N elements apart (measured +1.8 % D3Q19, +3 % D3Q27 at 512^3).
  // Plain structure of arrays (LBM_LAYOUT_SOA): ds = N, rs = nx, zs = nx*ny, i.e. f[a][z][y][x].
  long long ds, zs;
  int rs;
  double omega;         // 1/tau (D:R1)
  double F[3];          // body force (D:R7)
  int wall[6];          // face is non-periodic (BOUNCE, MOVING or PRESSURE), order x-,x+,y-,y+,z-,z+
  int kind[6];          // FACE_PERIODIC / FACE_BOUNCE / FACE_MOVING / FACE_PRESSURE
  int open[6];          // face is MOVING or PRESSURE: a wall link through it changes the bounced value (D:R6, D:R22)
  double face_u[6][3];  // wall velocity of MOVING faces (uniform part)
  // D:R22: optional per-cell wall velocity of a MOVING face (velocity inlet), u[c*n + j], j over the two in-face
  // coordinates (lower axis fastest; z is the GLOBAL plane index), n = cells of the face; NULL = uniform face_u
  const double* face_prof[6];
  double face_rho[6];   // D:R22: density prescribed on PRESSURE faces (anti-bounce-back)
  int any_open;
  int sym[6];           // face is SYMMETRY (D:R25); such handles always run the BC_GEO kernels (link mask)
  int any_sym;
  int zg_off, nz_glob;  // global plane index of local plane z = z + zg_off; planes of the whole box (slabs: D:R21)
  // BC_GEO only (D:R16): bit a (a != rest) of links[i]: link a of node i has no active source node — i - e_a is
  // solid, or lies beyond a non-periodic face; through SYMMETRY faces only (D:R25) the source is the mirror image
  // and the bit says whether THAT node is inactive.  Bit `rest`: node i itself is inactive.
  const uint32_t* links;
  int nodal;            // D:R3/R17: the paper's modified nodal bounce-back (Eq. 10) instead of halfway
  // Planes [z_lo, z_hi) are the ones this handle updates and the z faces of the box lie at z_lo and z_hi-1.
  // Whole box: 0, nz.  z-slab of a decomposed box (D:R21): 1, nz-1 — planes 0 and nz-1 are halo
  // planes that hold the neighbouring slab's values; wall[4] / wall[5] are set only on the slab that owns the face.
  int z_lo, z_hi;
  int slab;
  // slab only, A/B scheme: where the fused kernel ALSO stores the populations the neighbouring slab will pull
  // across the cut (the paper's PassF, done by peer stores instead of a host-staged MPI exchange):
  // direction plane a of the lower / upper neighbour's destination buffer starts at push_lo + a*push_lo_N;
  // push_lo_off / push_hi_off = in-plane offset of that neighbour's receiving halo plane.  NULL = nothing to push.
  void* push_lo;
  void* push_hi;
  long long push_lo_N, push_hi_N;      // the neighbours' direction strides ds
  long long push_lo_off, push_hi_off;  // offset of their receiving halo plane (plane index * zs)
};

enum { EQ_STANDARD = 0, EQ_INCOMP = 1 };
enum { FACE_PERIODIC = 0, FACE_BOUNCE = 1, FACE_MOVING = 2, FACE_PRESSURE = 3, FACE_SYMMETRY = 4 };

// Position of a cell relative to the non-periodic faces, and (BC_GEO) its link mask.
template <int BC>
struct CellFlags {
  bool lo[3], hi[3];  // cell is in the first / last plane of an axis whose face there is a wall
  uint32_t m;
  __device__ __forceinline__ CellFlags(const Params& p, int x, int y, int z, int ic) {
    if constexpr (BC != BC_PERIODIC) {
      lo[0] = (x == 0) & (p.wall[0] != 0);
      hi[0] = (x == p.nx - 1) & (p.wall[1] != 0);
      lo[1] = (y == 0) & (p.wall[2] != 0);
      hi[1] = (y == p.ny - 1) & (p.wall[3] != 0);
      lo[2] = (z == p.z_lo) & (p.wall[4] != 0);
      hi[2] = (z == p.z_hi - 1) & (p.wall[5] != 0);
    } else {
      lo[0] = lo[1] = lo[2] = hi[0] = hi[1] = hi[2] = false;
    }
    if constexpr (BC == BC_GEO) m = __ldg(p.links + ic);
    else m = 0u;
  }
  // true if the node x + s*e_A lies outside the box (s = +1: downstream, s = -1: upstream)
  template <int Q, int A, int S>
  __device__ __forceinline__ bool leaves_box() const {
    if constexpr (BC == BC_PERIODIC) return false;
    constexpr int dx = S * Dir<Q, A>::ex, dy = S * Dir<Q, A>::ey, dz = S * Dir<Q, A>::ez;
    // bitwise OR on purpose: a short-circuit || makes ptxas branch around the loads it guards
    bool out = false;
    if constexpr (dx == -1) out = out | lo[0];
    if constexpr (dx == 1) out = out | hi[0];
    if constexpr (dy == -1) out = out | lo[1];
    if constexpr (dy == 1) out = out | hi[1];
    if constexpr (dz == -1) out = out | lo[2];
    if constexpr (dz == 1) out = out | hi[2];
    return out;
  }
  // true if there is no active node at x + s*e_A (beyond a wall face, or — BC_GEO — solid)
  template <int Q, int A, int S>
  __device__ __forceinline__ bool leaves() const {
    if constexpr (Dir<Q, A>::s == 0) return false;
    if constexpr (BC == BC_GEO) {
      constexpr int bit = (S == -1) ? A : Dir<Q, A>::opp;  // x + e_A = x - e_opp(A)
      return (m >> bit) & 1u;
    } else {
      return leaves_box<Q, A, S>();
    }
  }
  template <int Q>
  __device__ __forceinline__ bool active() const {
    if constexpr (BC == BC_GEO) return !((m >> ((Q - 1) / 2)) & 1u);
    return true;
  }
};

// Neighbour offsets of one cell with periodic wrap by conditional add (no %).  Two index spaces:
//   storage  at<>() / ic   offset of the node inside a population buffer, direction excluded (add a*ds): x + y*rs as
//                          32 bits, the plane part z*zs as 64 bits (thread-invariant in the step kernels, where z =
//                          blockIdx.z: it lives in uniform registers together with the direction base);
//   cells    cat<>() / cell the node's linear index x + nx*(y + ny*z) in the arrays at the interface (link mask, geo,
//                          rho, u, canonical f): 32 bits (lbm_create refuses N >= 2^31).
struct Neigh {
  int ox[3], oy[3];   // index 0: coordinate-1, 1: same, 2: coordinate+1
  long long oz[3];
  int cy[3], cz[3];
  long long ic;
  int cell;
  __device__ __forceinline__ Neigh(const Params& p, int x, int y, int z) {
    const int xm = (x == 0) ? p.nx - 1 : x - 1, xp = (x == p.nx - 1) ? 0 : x + 1;
    const int ym = (y == 0) ? p.ny - 1 : y - 1, yp = (y == p.ny - 1) ? 0 : y + 1;
    const int zm = (z == 0) ? p.nz - 1 : z - 1, zp = (z == p.nz - 1) ? 0 : z + 1;
    ox[0] = xm; ox[1] = x; ox[2] = xp;
    oy[0] = ym * p.rs; oy[1] = y * p.rs; oy[2] = yp * p.rs;
    oz[0] = zm * p.zs; oz[1] = z * p.zs; oz[2] = zp * p.zs;
    const int sy = p.nx, sz = p.nx * p.ny;
    cy[0] = ym * sy; cy[1] = y * sy; cy[2] = yp * sy;
    cz[0] = zm * sz; cz[1] = z * sz; cz[2] = zp * sz;
    ic = ox[1] + oy[1] + oz[1];
    cell = ox[1] + cy[1] + cz[1];
  }
  // storage offset of x + s*e_A (wrapped)
  template <int Q, int A, int S>
  __device__ __forceinline__ long long at() const {
    return (ox[1 + S * Dir<Q, A>::ex] + oy[1 + S * Dir<Q, A>::ey]) + oz[1 + S * Dir<Q, A>::ez];
  }
  // cell index of x + s*e_A (wrapped)
  template <int Q, int A, int S>
  __device__ __forceinline__ int cat() const {
    return ox[1 + S * Dir<Q, A>::ex] + cy[1 + S * Dir<Q, A>::ey] + cz[1 + S * Dir<Q, A>::ez];
  }
};

// Index of the lattice vector (ex,ey,ez) in Lattice<Q> (compile time), -1 if the set has no such vector.
template <int Q>
__host__ __device__ constexpr int dir_index(int ex, int ey, int ez) {
  for (int a = 0; a < Q; ++a)
    if (Lattice<Q>::e[a][0] == ex && Lattice<Q>::e[a][1] == ey && Lattice<Q>::e[a][2] == ez) return a;
  return -1;
}

// SYMMETRY faces (D:R25; "the left and right boundaries are symmetric"): a mirror plane half a link beyond
// the last node.  If the node x + S*e_A lies beyond SYMMETRY faces ONLY, the link connects x with the mirror image:
// the node whose coordinates along the crossed axes are those of x, and the population there has the direction
// e_A with those components negated.  Returns false for every other link (inside the box, or through a face of
// another kind: MOVING > BOUNCE > PRESSURE decide those, D:R22).  idx / cidx = storage offset / cell index of that node.
template <int BC>
__device__ __forceinline__ bool touches_sym(const Params& p, const CellFlags<BC>& c) {
  if constexpr (BC == BC_PERIODIC) return false;
  if (!p.any_sym) return false;
  return (c.lo[0] && p.sym[0]) || (c.hi[0] && p.sym[1]) || (c.lo[1] && p.sym[2]) || (c.hi[1] && p.sym[3]) ||
         (c.lo[2] && p.sym[4]) || (c.hi[2] && p.sym[5]);
}

template <int Q, int A, int S, int BC>
__device__ __forceinline__ bool mirror_link(const Params& p, const CellFlags<BC>& c, const Neigh& nb, int& dir, long long& idx, int& cidx) {
  using D = Dir<Q, A>;
  constexpr int dx = S * D::ex, dy = S * D::ey, dz = S * D::ez;
  const bool cx = (dx == -1) ? c.lo[0] : (dx == 1) ? c.hi[0] : false;
  const bool cy = (dy == -1) ? c.lo[1] : (dy == 1) ? c.hi[1] : false;
  const bool cz = (dz == -1) ? c.lo[2] : (dz == 1) ? c.hi[2] : false;
  const bool sx = cx && p.sym[dx == 1 ? 1 : 0], sy = cy && p.sym[dy == 1 ? 3 : 2], sz = cz && p.sym[dz == 1 ? 5 : 4];
  if ((cx && !sx) || (cy && !sy) || (cz && !sz) || !(sx || sy || sz)) return false;
  const int mx = sx ? nb.ox[1] : nb.ox[1 + dx];
  idx = (mx + (sy ? nb.oy[1] : nb.oy[1 + dy])) + (sz ? nb.oz[1] : nb.oz[1 + dz]);  // storage offset of the mirror image
  cidx = mx + (sy ? nb.cy[1] : nb.cy[1 + dy]) + (sz ? nb.cz[1] : nb.cz[1 + dz]);   // its cell index
  constexpr int t1 = dir_index<Q>(-D::ex, D::ey, D::ez), t2 = dir_index<Q>(D::ex, -D::ey, D::ez), t3 = dir_index<Q>(-D::ex, -D::ey, D::ez),
                t4 = dir_index<Q>(D::ex, D::ey, -D::ez), t5 = dir_index<Q>(-D::ex, D::ey, -D::ez), t6 = dir_index<Q>(D::ex, -D::ey, -D::ez),
                t7 = dir_index<Q>(-D::ex, -D::ey, -D::ez);
  dir = sz ? (sy ? (sx ? t7 : t6) : (sx ? t5 : t4)) : (sy ? (sx ? t3 : t2) : (sx ? t1 : A));
  return true;
}

// Base of component A of an array whose components are `N` elements apart (64-bit, thread-invariant): the direction
// rows of a population buffer (N = p.ds) or the components of rho / u / canonical f (N = p.N).
template <int A, typename T>
__device__ __forceinline__ T* plane(T* buf, long long N) {
  return buf + (long long)A * N;
}

// The population streams of the A/B step kernel: every value is read once and written once per step, nothing is
// re-used.  Loads take the non-coherent path (ld.global.nc), stores are plain: every other cache policy measured the
// same or slower (profiles/cache_policy_r01d.txt).
#define LBM_LD_STREAM(q) __ldg(q)
#define LBM_ST_STREAM(q, v) (*(q) = (v))

// ---------------------------------------------------------------------------------------
// Storage element access.  fp64: the value itself.  fp32 storage (S:§8f NEXT-1): f - t_a is
// kept as float, arithmetic stays fp64.
template <typename ST, int Q, int A>
__device__ __forceinline__ double ld_pop(const ST* __restrict__ p, long long i) {
  if constexpr (sizeof(ST) == 8) return __ldg(p + i);
  else return (double)__ldg(p + i) + Dir<Q, A>::t;
}
// same through a plain (coherent) load: the in-place kernels read the buffer they write
template <typename ST, int Q, int A>
__device__ __forceinline__ double ld_pop_rw(const ST* p, long long i) {
  if constexpr (sizeof(ST) == 8) return p[i];
  else return (double)p[i] + Dir<Q, A>::t;
}
template <typename ST, int Q, int A>
__device__ __forceinline__ void st_pop(ST* __restrict__ p, long long i, double v) {
  if constexpr (sizeof(ST) == 8) p[i] = v;
  else p[i] = (float)(v - Dir<Q, A>::t);
}

// ---------------------------------------------------------------------------------------
// Moments (Eq. 8-9; D:R5, D:R7): rho = sum f; u = (sum e f + F/2)/rho  [Eq. 5: /rho0 = 1]
// Sums over +- pairs first (s_a = f_a + f_abar feeds rho, d_a = f_a - f_abar feeds the momentum): 39 instead of 49 additions
// for D3Q19 and dependency chains of depth 5 instead of 19 — the kernels that keep few warps per SM (stream_collide_ab2)
// are bound by exactly that latency.
template <int Q, int EQ, bool FORCE>
__device__ __forceinline__ void moments(const double (&f)[Q], const Params& p, double& rho, double& ux, double& uy, double& uz) {
  constexpr int H = (Q - 1) / 2;  // pairs (a, Q-1-a), a < H; the rest direction is H
  double sp[H], dp[H];
  static_for<0, H>([&](auto A) {
    constexpr int a = decltype(A)::value;
    sp[a] = f[a] + f[Q - 1 - a];
    dp[a] = f[a] - f[Q - 1 - a];
  });
  // balanced sums over compile-time index lists
  double r = f[H], mx = 0.0, my = 0.0, mz = 0.0;
  double r2 = 0.0, mx2 = 0.0, my2 = 0.0, mz2 = 0.0;  // two accumulators per sum halve the chains once more
  static_for<0, H>([&](auto A) {
    constexpr int a = decltype(A)::value;
    using D = Dir<Q, a>;
    if constexpr (a % 2 == 0) {
      r += sp[a];
      if constexpr (D::ex == 1) mx += dp[a];
      if constexpr (D::ex == -1) mx -= dp[a];
      if constexpr (D::ey == 1) my += dp[a];
      if constexpr (D::ey == -1) my -= dp[a];
      if constexpr (D::ez == 1) mz += dp[a];
      if constexpr (D::ez == -1) mz -= dp[a];
    } else {
      r2 += sp[a];
      if constexpr (D::ex == 1) mx2 += dp[a];
      if constexpr (D::ex == -1) mx2 -= dp[a];
      if constexpr (D::ey == 1) my2 += dp[a];
      if constexpr (D::ey == -1) my2 -= dp[a];
      if constexpr (D::ez == 1) mz2 += dp[a];
      if constexpr (D::ez == -1) mz2 -= dp[a];
    }
  });
  r += r2; mx += mx2; my += my2; mz += mz2;
  if constexpr (FORCE) {
    mx += 0.5 * p.F[0];
    my += 0.5 * p.F[1];
    mz += 0.5 * p.F[2];
  }
  rho = r;
  if constexpr (EQ == EQ_STANDARD) {
    const double inv = 1.0 / r;
    ux = mx * inv; uy = my * inv; uz = mz * inv;
  } else {
    ux = mx; uy = my; uz = mz;
  }
}

template <int Q, int A>
__device__ __forceinline__ double edot(double vx, double vy, double vz) {
  using D = Dir<Q, A>;
  double r = 0.0;
  if constexpr (D::ex == 1) r += vx;
  if constexpr (D::ex == -1) r -= vx;
  if constexpr (D::ey == 1) r += vy;
  if constexpr (D::ey == -1) r -= vy;
  if constexpr (D::ez == 1) r += vz;
  if constexpr (D::ez == -1) r -= vz;
  return r;
}

// Equilibrium: Eq. 2  feq = t rho (1 + 3 e.u + 4.5 (e.u)^2 - 1.5 u.u)
//              Eq. 5  feq = t (rho + rho0 (3 e.u + 4.5 (e.u)^2 - 1.5 u.u)), rho0 = 1, rho = p/c_s^2
template <int Q, int EQ>
__device__ __forceinline__ void equilibrium(double (&feq)[Q], double rho, double ux, double uy, double uz) {
  const double usq15 = 1.5 * (ux * ux + uy * uy + uz * uz);
  const double A = (EQ == EQ_STANDARD) ? rho : 1.0;
  const double base = (EQ == EQ_STANDARD) ? rho * (1.0 - usq15) : rho - usq15;
  static_for<0, (Q + 1) / 2>([&](auto AA) {
    constexpr int a = decltype(AA)::value;
    using D = Dir<Q, a>;
    if constexpr (a == D::opp) {
      feq[a] = D::t * base;
    } else {
      const double eu = edot<Q, a>(ux, uy, uz);
      const double s = D::t * fma(4.5 * A * eu, eu, base);
      const double d = (3.0 * D::t) * (A * eu);
      feq[a] = s + d;
      feq[D::opp] = s - d;
    }
  });
}

// Faces that change the value a wall link bounces back (D:R6 Ladd moving wall; D:R22 velocity inlet and pressure
// outlet).  Both rules are folded in on the collide side, while rho and u of time t are live: the slot an outgoing
// wall link b of cell x would have streamed into is read by nobody but x's own bounce-back along a = opp(b) one
// step later, so the cell stores there what that bounce-back must return:
//   MOVING   f_a(x,t+1) = f*_b(x,t) + 6 t_a rho_w (e_a.u_w) = f*_b - 6 t_b rho_w (e_b.u_w),  u_w uniform or per cell
//   PRESSURE f_a(x,t+1) = -f*_b(x,t) + 2 feq+_b(rho_face, u(x,t)),  feq+ = the part of Eq. 2 / Eq. 5 even in e
// Precedence when x + e_b lies beyond several non-periodic faces: MOVING (highest face index) > BOUNCE > PRESSURE
// (highest face index).  `touches_open` keeps the per-direction tests off every cell not next to such a face.
template <int BC>
__device__ __forceinline__ bool touches_open(const Params& p, const CellFlags<BC>& c) {
  if constexpr (BC == BC_PERIODIC) return false;
  if (!p.any_open) return false;
  return (c.lo[0] && p.open[0]) || (c.hi[0] && p.open[1]) || (c.lo[1] && p.open[2]) || (c.hi[1] && p.open[3]) ||
         (c.lo[2] && p.open[4]) || (c.hi[2] && p.open[5]);
}

struct CellState {  // what the open faces need from the collision of this cell
  double rw;              // rho(x,t) under Eq. 2, rho0 = 1 under Eq. 5
  double ux, uy, uz, usq15;
  int ic, z;              // in-plane index and (local) plane of the cell
  // Fast path: the cell touches exactly ONE non-periodic face (every face cell except edges and corners), so every
  // link that leaves the box leaves through it.  With the inlet / outlet on the x faces there is one such cell per
  // row, i.e. one lane of one warp in every block runs this code while the rest of the block waits for it: it has
  // to be short (512x128x128 D3Q27 with inlet + outlet: 673 -> ... us per step once the per-direction face
  // classification was taken off this path).
  int face;               // that face, or -1: classify every direction (edges, corners)
  int kind;               // its kind (FACE_MOVING or FACE_PRESSURE)
  double wx, wy, wz, rf;  // its wall velocity at this cell / its density
};

// Wall velocity of MOVING face `face` at the cell with in-plane index ic in local plane z: the uniform face_u or the
// cell's entry of the per-cell profile (D:R22).
__device__ __forceinline__ void wall_velocity(const Params& p, int face, int ic, int z, double& wx, double& wy, double& wz) {
  wx = p.face_u[face][0]; wy = p.face_u[face][1]; wz = p.face_u[face][2];
  const double* prof = p.face_prof[face];
  if (prof) {
    // in-face index of the cell from its in-plane index: the face fixes one coordinate
    const int axis = face >> 1, side = face & 1;
    const int zg = z + p.zg_off;
    long long j, n;
    if (axis == 0) {        // j = y + ny*zg
      const int xf = side ? p.nx - 1 : 0;
      j = (ic - xf) / p.nx + (long long)p.ny * p.zg_off;
      n = (long long)p.ny * p.nz_glob;
    } else if (axis == 1) { // j = x + nx*zg
      const int yf = side ? p.ny - 1 : 0;
      j = (long long)(ic - p.nx * yf - p.nx * p.ny * z) + (long long)p.nx * zg;
      n = (long long)p.nx * p.nz_glob;
    } else {                // j = x + nx*y
      j = ic - p.nx * p.ny * z;
      n = (long long)p.nx * p.ny;
    }
    wx = __ldg(prof + j); wy = __ldg(prof + n + j); wz = __ldg(prof + 2 * n + j);
  }
}

// Fill the single-face part of the cell state (call once per cell that touches an open face).
template <int BC>
__device__ __forceinline__ void classify_open_cell(CellState& s, const Params& p, const CellFlags<BC>& c) {
  s.face = -1;
  s.kind = 0;
  s.wx = s.wy = s.wz = 0.0;
  s.rf = 1.0;
  const int nwall = (int)c.lo[0] + (int)c.hi[0] + (int)c.lo[1] + (int)c.hi[1] + (int)c.lo[2] + (int)c.hi[2];
  if (nwall == 1) {
    const int k = c.lo[0] ? 0 : c.hi[0] ? 1 : c.lo[1] ? 2 : c.hi[1] ? 3 : c.lo[2] ? 4 : 5;
    s.face = k;
    s.kind = p.kind[k];  // MOVING or PRESSURE: the caller checked touches_open and this is the only face
    if (s.kind == FACE_MOVING) wall_velocity(p, k, s.ic, s.z, s.wx, s.wy, s.wz);
    else s.rf = p.face_rho[k];
  }
}

// v = post-collision value of outgoing direction B (in the stored variable: f*, or f* - t_B if SHIFTED);
// returns what the slot must hold.
template <int Q, int EQ, int BC, int B, bool SHIFTED>
__device__ __forceinline__ double open_link(double v, const Params& p, const CellFlags<BC>& c, const CellState& s) {
  using D = Dir<Q, B>;
  if constexpr (BC == BC_PERIODIC || D::s == 0) {
    return v;
  } else {
    auto moving = [&](double wx, double wy, double wz) { return v - (6.0 * D::t) * s.rw * edot<Q, B>(wx, wy, wz); };
    auto pressure = [&](double rf) {
      const double eu = edot<Q, B>(s.ux, s.uy, s.uz);
      const double poly = fma(4.5 * eu, eu, -s.usq15);
      // Eq. 2: t rf (1 + poly);  Eq. 5: t (rf + rho0 poly);  SHIFTED: minus t_B for the stored variable
      double even = (EQ == EQ_STANDARD) ? fma(rf, poly, rf) : rf + poly;
      if constexpr (SHIFTED) even -= 1.0;
      return fma(2.0 * D::t, even, -v);
    };
    if (s.face >= 0) {  // one face only: the link leaves through it or not at all
      const bool leaves = (D::ex == -1 && s.face == 0) || (D::ex == 1 && s.face == 1) || (D::ey == -1 && s.face == 2) ||
                          (D::ey == 1 && s.face == 3) || (D::ez == -1 && s.face == 4) || (D::ez == 1 && s.face == 5);
      if (!leaves) return v;
      return s.kind == FACE_MOVING ? moving(s.wx, s.wy, s.wz) : pressure(s.rf);
    }
    int mface = -1, pface = -1;
    bool bounce = false;
    auto crossed = [&](int face) {
      const int k = p.kind[face];
      if (k == FACE_MOVING) mface = face;
      else if (k == FACE_PRESSURE) pface = face;
      else if (k == FACE_BOUNCE) bounce = true;  // a SYMMETRY face crossed together with another kind: the other decides
    };
    // x, then y, then z: the highest face index crossed wins within a kind
    if constexpr (D::ex != 0) {
      if (D::ex == 1 ? c.hi[0] : c.lo[0]) crossed(D::ex == 1 ? 1 : 0);
    }
    if constexpr (D::ey != 0) {
      if (D::ey == 1 ? c.hi[1] : c.lo[1]) crossed(D::ey == 1 ? 3 : 2);
    }
    if constexpr (D::ez != 0) {
      if (D::ez == 1 ? c.hi[2] : c.lo[2]) crossed(D::ez == 1 ? 5 : 4);
    }
    if (mface >= 0) {
      double wx, wy, wz;
      wall_velocity(p, mface, s.ic, s.z, wx, wy, wz);
      return moving(wx, wy, wz);
    }
    if (pface >= 0 && !bounce) return pressure(p.face_rho[pface]);
    return v;
  }
}

// BGK relaxation, Eq. 6: f* = f - omega (f - feq), plus Guo's source (D:R7)
//   S_a = (1 - omega/2) t_a [3 (e_a - u) + 9 (e_a.u) e_a] . F
// and, on cells touching a MOVING face, the Ladd term folded into the outgoing wall links
// (D:R6): the value kept for an outgoing link b is f*_b - 6 t_b rho_w (e_b . u_w), which the
// bounce-back read f_bbar(x, t+1) = stored_b(x) turns into f*_b + 6 t_bbar rho_w (e_bbar . u_w).
// f is replaced by the post-collision populations.
template <int Q, int EQ, int BC, bool FORCE>
__device__ __forceinline__ void collide(double (&f)[Q], const Params& p, const CellFlags<BC>& c, int ic, int z) {
  double rho, ux, uy, uz;
  moments<Q, EQ, FORCE>(f, p, rho, ux, uy, uz);
  const double om = p.omega, om1 = 1.0 - p.omega;
  const double usq15 = 1.5 * (ux * ux + uy * uy + uz * uz);
  const double A = (EQ == EQ_STANDARD) ? rho : 1.0;
  const double base = (EQ == EQ_STANDARD) ? rho * (1.0 - usq15) : rho - usq15;
  double k = 0.0, uF3 = 0.0;
  if constexpr (FORCE) {
    k = 1.0 - 0.5 * om;
    uF3 = 3.0 * (ux * p.F[0] + uy * p.F[1] + uz * p.F[2]);
  }
  static_for<0, (Q + 1) / 2>([&](auto AA) {
    constexpr int a = decltype(AA)::value;
    using D = Dir<Q, a>;
    if constexpr (a == D::opp) {
      double g = (om * D::t) * base;
      if constexpr (FORCE) g -= (k * D::t) * uF3;
      f[a] = fma(om1, f[a], g);
    } else {
      // omega t_a (base + 4.5 A (e.u)^2) and 3 omega t_a A (e.u) with the factors that depend on the speed class only
      // (three values of t_a) folded once per cell: 7 instead of 10 fp64 operations per +- pair
      const double eu = edot<Q, a>(ux, uy, uz);
      const double w = om * D::t;
      double s = fma(((4.5 * w) * A) * eu, eu, w * base);
      double d = ((3.0 * w) * A) * eu;
      if constexpr (FORCE) {
        const double eF = edot<Q, a>(p.F[0], p.F[1], p.F[2]);
        s = fma(k * D::t, fma(9.0 * eu, eF, -uF3), s);
        d = fma(3.0 * k * D::t, eF, d);
      }
      f[a] = fma(om1, f[a], s + d);
      f[D::opp] = fma(om1, f[D::opp], s - d);
    }
  });
  if constexpr (BC != BC_PERIODIC) {
    if (touches_open<BC>(p, c)) {
      // rho and u of time t are recomputed from f*: the collision conserves mass and changes sum e f by exactly F
      // (Guo), so u = (sum e f* - F/2)/rho.  Nothing of the collision stays live across it for these few cells.
      double r = 0.0, mx = 0.0, my = 0.0, mz = 0.0;
      static_for<0, Q>([&](auto BB) {
        constexpr int b = decltype(BB)::value;
        using D = Dir<Q, b>;
        r += f[b];
        if constexpr (D::ex == 1) mx += f[b];
        if constexpr (D::ex == -1) mx -= f[b];
        if constexpr (D::ey == 1) my += f[b];
        if constexpr (D::ey == -1) my -= f[b];
        if constexpr (D::ez == 1) mz += f[b];
        if constexpr (D::ez == -1) mz -= f[b];
      });
      if constexpr (FORCE) {
        mx -= 0.5 * p.F[0];
        my -= 0.5 * p.F[1];
        mz -= 0.5 * p.F[2];
      }
      CellState st;
      st.rw = (EQ == EQ_STANDARD) ? r : 1.0;
      const double inv = (EQ == EQ_STANDARD) ? 1.0 / r : 1.0;
      st.ux = mx * inv; st.uy = my * inv; st.uz = mz * inv;
      st.usq15 = 1.5 * (st.ux * st.ux + st.uy * st.uy + st.uz * st.uz);
      st.ic = ic; st.z = z;
      classify_open_cell<BC>(st, p, c);
      static_for<0, Q>([&](auto BB) {
        constexpr int b = decltype(BB)::value;
        f[b] = open_link<Q, EQ, BC, b, false>(f[b], p, c, st);
      });
    }
  }
}

// The same collision for the fp32-storage variant, written in the stored variable g_a = f_a - t_a (S:§8f NEXT-1):
//   rho = 1 + sum g,  sum e f = sum e g  (sum t = 1, sum t e = 0),
//   g*_a = (1 - omega) g_a + omega t_a [ (rho - 1) + A (3 e.u + 4.5 (e.u)^2 - 1.5 u.u) ]  (+ source, Ladd term)
// so the populations stay packed as floats in registers until they are used, no t_a is added or subtracted and
// the small deviations are not rounded against O(t_a).  `store(IC<a>, g*_a)` writes one result.
template <int Q, int EQ, int BC, bool FORCE, typename StoreF>
__device__ __forceinline__ void collide_shifted(const float (&g)[Q], const Params& p, const CellFlags<BC>& c, int ic, int z, StoreF&& store) {
  double dr = 0.0, mx = 0.0, my = 0.0, mz = 0.0;
  static_for<0, Q>([&](auto AA) {
    constexpr int a = decltype(AA)::value;
    using D = Dir<Q, a>;
    const double v = (double)g[a];
    dr += v;
    if constexpr (D::ex == 1) mx += v;
    if constexpr (D::ex == -1) mx -= v;
    if constexpr (D::ey == 1) my += v;
    if constexpr (D::ey == -1) my -= v;
    if constexpr (D::ez == 1) mz += v;
    if constexpr (D::ez == -1) mz -= v;
  });
  if constexpr (FORCE) {
    mx += 0.5 * p.F[0];
    my += 0.5 * p.F[1];
    mz += 0.5 * p.F[2];
  }
  const double rho = 1.0 + dr;
  double ux = mx, uy = my, uz = mz;
  if constexpr (EQ == EQ_STANDARD) {
    const double inv = 1.0 / rho;
    ux *= inv; uy *= inv; uz *= inv;
  }
  const double om = p.omega, om1 = 1.0 - p.omega;
  const double usq15 = 1.5 * (ux * ux + uy * uy + uz * uz);
  const double A = (EQ == EQ_STANDARD) ? rho : 1.0;
  const double base = dr - A * usq15;  // feq_a - t_a = t_a (base + A (3 e.u + 4.5 (e.u)^2))
  double k = 0.0, uF3 = 0.0;
  if constexpr (FORCE) {
    k = 1.0 - 0.5 * om;
    uF3 = 3.0 * (ux * p.F[0] + uy * p.F[1] + uz * p.F[2]);
  }
  // open faces (D:R6, D:R22): what an outgoing wall link keeps in its slot; identity on every other cell.  The cells
  // next to such a face take their own copy of the relaxation loop, so that every other cell runs it without a test per
  // direction (ncu, 256^3 cavity with fp32 storage: 624 -> instructions per cell as in the periodic kernel, and the hot
  // path fits the instruction cache again).
  auto relax = [&](auto OPEN, const CellState& st) {
    auto open = [&](auto BB, double v) -> double {
      constexpr int b = decltype(BB)::value;
      if constexpr (decltype(OPEN)::value != 0 && BC != BC_PERIODIC && Dir<Q, b>::s > 0) return open_link<Q, EQ, BC, b, true>(v, p, c, st);
      else return v;
    };
    static_for<0, (Q + 1) / 2>([&](auto AA) {
      constexpr int a = decltype(AA)::value;
      using D = Dir<Q, a>;
      if constexpr (a == D::opp) {
        double gq = (om * D::t) * base;
        if constexpr (FORCE) gq -= (k * D::t) * uF3;
        store(IC<a>{}, fma(om1, (double)g[a], gq));
      } else {
        const double eu = edot<Q, a>(ux, uy, uz);
        const double w = om * D::t;  // per speed class, as in collide
        double s = fma(((4.5 * w) * A) * eu, eu, w * base);
        double d = ((3.0 * w) * A) * eu;
        if constexpr (FORCE) {
          const double eF = edot<Q, a>(p.F[0], p.F[1], p.F[2]);
          s = fma(k * D::t, fma(9.0 * eu, eF, -uF3), s);
          d = fma(3.0 * k * D::t, eF, d);
        }
        store(IC<a>{}, open(IC<a>{}, fma(om1, (double)g[a], s + d)));
        store(IC<D::opp>{}, open(IC<D::opp>{}, fma(om1, (double)g[D::opp], s - d)));
      }
    });
  };
  CellState st{A, ux, uy, uz, usq15, ic, z, -1, 0, 0.0, 0.0, 0.0, 1.0};
  if constexpr (BC != BC_PERIODIC) {
    if (touches_open<BC>(p, c)) {
      classify_open_cell<BC>(st, p, c);
      relax(IC<1>{}, st);
      return;
    }
  }
  relax(IC<0>{}, st);
}

// D:R24: true if the outgoing link B of this cell (node x + e_B) is resolved by an open face — it crosses a MOVING
// face, or a PRESSURE face and no BOUNCE face.  Such a link is no wall link: Eq. 10 leaves it alone.
template <int Q, int B, int BC>
__device__ __forceinline__ bool open_resolved(const Params& p, const CellFlags<BC>& c) {
  using D = Dir<Q, B>;
  bool moving = false, pressure = false, bounce = false;
  auto crossed = [&](int face) {
    const int k = p.kind[face];
    moving = moving | (k == FACE_MOVING);
    pressure = pressure | (k == FACE_PRESSURE);
    bounce = bounce | (k == FACE_BOUNCE);
  };
  if constexpr (D::ex != 0) {
    if (D::ex == 1 ? c.hi[0] : c.lo[0]) crossed(D::ex == 1 ? 1 : 0);
  }
  if constexpr (D::ey != 0) {
    if (D::ey == 1 ? c.hi[1] : c.lo[1]) crossed(D::ey == 1 ? 3 : 2);
  }
  if constexpr (D::ez != 0) {
    if (D::ez == 1 ? c.hi[2] : c.lo[2]) crossed(D::ez == 1 ? 5 : 4);
  }
  return moving | (pressure & !bounce);
}

// Eq. 10 of the paper's modified nodal bounce-back (D:R17), applied to the populations a
// wall node has just gathered: a direction a nothing streamed in along (link bit a set) takes the
// value that arrived along its opposite, f_a = f_abar, if abar did arrive from an active node (bit
// abar clear).  When neither end of the link is active the halfway value already in f[a] stays; so does the value of
// a link through an open face (D:R24: MOVING / PRESSURE faces keep their own rule next to nodal walls).
template <int Q, int BC, typename T>
__device__ __forceinline__ void nodal_replicate(T (&f)[Q], const Params& p, const CellFlags<BC>& c) {
  if constexpr (BC == BC_GEO) {
    if (p.nodal && (c.m != 0u)) {
      // D:R24: cells next to an open face must tell wall links from open links; with exactly one non-periodic face
      // at the cell (the usual case, one lane per row for x faces: keep it short) every link that leaves the box is open
      const bool open_cell = touches_open<BC>(p, c);
      const bool single = ((int)c.lo[0] + (int)c.hi[0] + (int)c.lo[1] + (int)c.hi[1] + (int)c.lo[2] + (int)c.hi[2]) == 1;
      static_for<0, Q>([&](auto A) {
        constexpr int a = decltype(A)::value;
        constexpr int o = Dir<Q, a>::opp;
        if constexpr (a != o) {
          // each +- pair is touched at most once: the condition excludes its mirror image
          if (((c.m >> a) & 1u) && !((c.m >> o) & 1u)) {
            // link a arrives from x - e_a = x + e_o: open-resolved links are not wall links
            bool open = false;
            if (open_cell) open = single ? c.template leaves_box<Q, a, -1>() : open_resolved<Q, o, BC>(p, c);
            if (!open) f[a] = f[o];
          }
        }
      });
    }
  }
}

// Gather of the Q populations of one cell.  link(IC<a>) is the address f_a comes from when the link has an
// upstream node, wall(IC<a>) the one it comes from otherwise (both always point into the buffer: the upstream
// index is wrapped even across a wall face).  BC_WALLS selects the address (flags cost no memory access);
// BC_GEO issues every regular load at once, WITHOUT waiting for the link mask, and re-reads only the wall links
// afterwards: with address selection all Q loads would queue behind the mask load and the latency to cover
// would double.  A regular load of a wall link reads a slot nobody writes; the value is discarded.  The price
// is Q wasted loads on an inactive node, which is right for the paper's workloads (an obstacle in a channel:
// a fraction of a percent of the nodes are solid).  Returns false for an inactive node.
struct NoMirror {};  // gather() without SYMMETRY faces (the in-place kernels: lbm_create refuses the combination)

template <int Q, int BC, bool PREFETCH_FACES = false, typename T, typename LinkF, typename WallF, typename LoadF, typename MirrorF = NoMirror>
__device__ __forceinline__ bool gather(T (&f)[Q], const CellFlags<BC>& c, LinkF&& link, WallF&& wall, LoadF&& load, MirrorF&& mirror = NoMirror{}, bool at_mirror = false,
                                       const Params* pp = nullptr /* PREFETCH_FACES only */) {
  if constexpr (BC == BC_GEO && PREFETCH_FACES) {
    // Cells in a first / last plane of a non-periodic face know their box-face wall links from the coordinates: they
    // prefetch those slots now (no destination register, no hazard), so that the re-read below — which has to wait for
    // the link mask — finds them in L1 instead of making a second trip to DRAM.  With an inlet / outlet on the x faces
    // that cell is ONE lane of a warp the rest of its block waits for (ncu, sphere case: 37 % of the divergent-lane
    // stall samples sat on that second trip).
    if (c.lo[0] | c.hi[0] | c.lo[1] | c.hi[1] | c.lo[2] | c.hi[2]) {
      static_for<0, Q>([&](auto A) {
        constexpr int a = decltype(A)::value;
        if constexpr (Dir<Q, a>::s > 0) {
          // (links through SYMMETRY faces are no wall links: their value comes from the mirror image, below)
          using D = Dir<Q, a>;
          bool w = false;
          if constexpr (D::ex == 1) w = w | (c.lo[0] & !pp->sym[0]);
          if constexpr (D::ex == -1) w = w | (c.hi[0] & !pp->sym[1]);
          if constexpr (D::ey == 1) w = w | (c.lo[1] & !pp->sym[2]);
          if constexpr (D::ey == -1) w = w | (c.hi[1] & !pp->sym[3]);
          if constexpr (D::ez == 1) w = w | (c.lo[2] & !pp->sym[4]);
          if constexpr (D::ez == -1) w = w | (c.hi[2] & !pp->sym[5]);
          if (w) asm volatile("prefetch.global.L1 [%0];" ::"l"(wall(A)));
        }
      });
    }
  }
  static_for<0, Q>([&](auto A) {
    constexpr int a = decltype(A)::value;
    auto q = link(A);
    if constexpr (BC == BC_WALLS) {
      if (c.template leaves<Q, a, -1>()) q = wall(A);  // a select, not a branch
    }
    f[a] = load(A, q);
  });
  if constexpr (BC == BC_GEO) {
    if (!c.template active<Q>()) return false;
    if (c.m != 0u) {
      static_for<0, Q>([&](auto A) {
        constexpr int a = decltype(A)::value;
        if constexpr (Dir<Q, a>::s > 0) {
          if (c.template leaves<Q, a, -1>()) f[a] = load(A, wall(A));
        }
      });
    }
    // D:R25: links through SYMMETRY faces come from the mirror image (mirror(A) = its address, or NULL for every
    // other link); the link bit says whether that node is active.  Only cells next to such a face get here.
    if constexpr (!std::is_same<std::decay_t<MirrorF>, NoMirror>::value) {
      if (at_mirror) {
        static_for<0, Q>([&](auto A) {
          constexpr int a = decltype(A)::value;
          if constexpr (Dir<Q, a>::s > 0) {
            auto q = mirror(A);
            if (q && !c.template leaves<Q, a, -1>()) f[a] = load(A, q);
          }
        });
      }
    }
  }
  return true;
}

// ---------------------------------------------------------------------------------------
// A/B scheme ("stream on read").  The buffer holds the post-collision populations aligned at their
// own cell, B = S^-1 f, S the slot permutation of one propagation (Eq. 7 with wall links, Eq. 10):
// f_a(x) = B_a(x - e_a)  inside,  = B_abar(x)  at a wall link.  One step = pull (gives the canonical
// pre-collision f of this time level), collide, store aligned at the own cell into the other buffer.
// SLAB (D:R21): the handle is one z-slab of a decomposed box.  Cells of the first / last updated plane store the
// populations that cross the cut a second time, straight into the neighbouring slab's halo plane (peer memory over
// NVLink, or the same device): e_z = -1 directions from plane z_lo, e_z = +1 directions from plane z_hi-1.  The
// neighbour then pulls them like any other upstream value.  Compute and exchange are one kernel; the ordering
// between slabs is stream-level (lbm_abi.cu: wait on the neighbours' step counters, launch, signal).
template <int Q, int A, typename ST>
__device__ __forceinline__ void push_one(const Params& p, int z, int ixy /* x + y*rs */, ST v) {
  if constexpr (Dir<Q, A>::ez == -1) {
    if (z == p.z_lo && p.push_lo) ((ST*)p.push_lo + (long long)A * p.push_lo_N)[p.push_lo_off + ixy] = v;
  }
  if constexpr (Dir<Q, A>::ez == 1) {
    if (z == p.z_hi - 1 && p.push_hi) ((ST*)p.push_hi + (long long)A * p.push_hi_N)[p.push_hi_off + ixy] = v;
  }
}

// SYM (D:R25): the box has SYMMETRY faces (always BC_GEO).  A separate instantiation: the mirror fix-up costs the
// link-mask kernels registers even where it never runs (sphere case 15.4 -> 15.0 GLUPS when it was compiled in).
// One cell of the A/B step.  COHERENT: the loads go through L2 (ld.global.cg) instead of the non-coherent path — needed
// by the persistent kernel below, whose source buffer was written by other SMs earlier in the SAME launch.
template <int Q, int EQ, int BC, bool FORCE, typename ST, bool SLAB, bool SYM, bool COHERENT>
__device__ __forceinline__ void ab_cell(const ST* src, ST* dst, const Params& p, int x, int y, int z) {
  const Neigh nb(p, x, y, z);
  const CellFlags<BC> c(p, x, y, z, nb.cell);
  auto link = [&](auto A) { return plane<decltype(A)::value>(src, p.ds) + nb.template at<Q, decltype(A)::value, -1>(); };
  auto wall = [&](auto A) { return plane<Dir<Q, decltype(A)::value>::opp>(src, p.ds) + nb.ic; };  // t_a == t_abar: same shift
  // D:R25: through SYMMETRY faces f_a comes from the mirror image (same speed class: same fp32 shift)
  auto mirror = [&](auto A) -> const ST* {
    int dir, cidx;
    long long idx;
    if (!mirror_link<Q, decltype(A)::value, -1, BC>(p, c, nb, dir, idx, cidx)) return nullptr;
    return src + dir * p.ds + idx;
  };
  const bool at_mirror = SYM ? touches_sym<BC>(p, c) : false;
  auto pull = [&](auto& f) {
    auto load = [](auto, const ST* q) {
      if constexpr (COHERENT) return __ldcg(q);
      else return LBM_LD_STREAM(q);
    };
    // (no prefetch in the SYM instantiation: measured slower there, 609 -> 625 us on the sphere case)
    if constexpr (SYM) return gather<Q, BC>(f, c, link, wall, load, mirror, at_mirror);
    else return gather<Q, BC, true>(f, c, link, wall, load, NoMirror{}, false, &p);
  };
  if constexpr (sizeof(ST) == 4) {
    float g[Q];  // packed: stays fp32 in registers until used (collide_shifted)
    if (!pull(g)) return;
    nodal_replicate<Q, BC>(g, p, c);
    collide_shifted<Q, EQ, BC, FORCE>(g, p, c, nb.cell, z, [&](auto A, double v) {
      constexpr int a = decltype(A)::value;
      const float s = (float)v;
      LBM_ST_STREAM(plane<a>(dst, p.ds) + nb.ic, s);
      if constexpr (SLAB) push_one<Q, a, ST>(p, z, nb.ox[1] + nb.oy[1], s);
    });
  } else {
    double f[Q];
    if (!pull(f)) return;
    nodal_replicate<Q, BC>(f, p, c);
    collide<Q, EQ, BC, FORCE>(f, p, c, nb.cell, z);
    static_for<0, Q>([&](auto A) {
      constexpr int a = decltype(A)::value;
      LBM_ST_STREAM(plane<a>(dst, p.ds) + nb.ic, f[a]);  // ST = double in this branch
      if constexpr (SLAB) push_one<Q, a, ST>(p, z, nb.ox[1] + nb.oy[1], f[a]);
    });
  }
}

template <int Q, int EQ, int BC, bool FORCE, typename ST, bool SLAB = false, bool SYM = false>
__global__ void __launch_bounds__(256, kMinBlocks<Q, FORCE, false, sizeof(ST)>) stream_collide_ab(const ST* __restrict__ src, ST* __restrict__ dst, const __grid_constant__ Params p) {
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  const int y = blockIdx.y * blockDim.y + threadIdx.y;
  int z = blockIdx.z;
  if constexpr (SLAB) z += p.z_lo;
  if (x >= p.nx || y >= p.ny) return;
  ab_cell<Q, EQ, BC, FORCE, ST, SLAB, SYM, false>(src, dst, p, x, y, z);
}

// fp32 storage, two cells per thread (S:§8f NEXT-1).  With half the bytes per cell the one-cell kernel above is bound by
// instruction issue and by POWER, not by DRAM: ncu (512^3 D3Q19) shows 576 instructions per cell, 165 of them integer
// address arithmetic; under the 1 kW cap of a sustained run the SM clock falls to ~1.6 GHz and the kernel to 0.91 of
// the copy bandwidth although one launch at full clock is DRAM-bound.  Here a thread owns the x-adjacent cells
// (x, x+1), x even, of a row that is uniform per block (the block is bx x 1, y = blockIdx.y, z = blockIdx.z): the Q
// row bases are block-invariant (uniform datapath), the e_x = 0 streams are read and ALL streams are written as aligned
// 8-byte vectors, and the address arithmetic — byte addresses as integers, one 64-bit add per access — is paid once
// per pair: 400 instructions per cell.  Same arithmetic per cell as ab_cell (collide_shifted): bit-identical results.
// A/B, D3Q19 / D2Q9, BC_PERIODIC / BC_WALLS, even nx; everything else (link mask, z-slabs, odd nx, and D3Q27, whose
// pair needs 168 registers) stays with the one-cell kernel.
// Measured, 512^3 D3Q19 sustained: 39.1 -> 42.0-42.3 GLUPS (0.98 of the copy bandwidth); one launch at full clock
// (ncu) 3.01 ms = 44.6 GLUPS = 1.036, DRAM-bound — in the sustained run the power cap (sw_power_cap, ~1.65 GHz) is the
// limit, i.e. energy per cell.  Tried and not kept: four cells per thread with 16-byte vectors and shuffles for the
// shifted streams (306 instructions per cell, but 168 registers = 12 warps per SM and ptxas serialises the loads
// through a few registers: 21-30 GLUPS); the collision in +- pair sums / differences (6 fp64 operations fewer per
// cell, more spills: 41.0 vs 42.0 GLUPS).
constexpr int kF32x2Threads = 128;  // D3Q19: 5 blocks per SM = 96 registers (44 B of spills; 128 registers, no spills: the same MLUPS)
template <int Q, int EQ, int BC, bool FORCE>
__global__ void __launch_bounds__(kF32x2Threads, 5) stream_collide_ab_f32x2(const float* __restrict__ src, float* __restrict__ dst, const __grid_constant__ Params p) {
  static_assert(BC != BC_GEO, "the link-mask kernels keep one cell per thread");
  typedef unsigned long long addr_t;
  const int x = 2 * (blockIdx.x * blockDim.x + threadIdx.x);
  const int y = blockIdx.y, z = blockIdx.z;
  if (x >= p.nx) return;
  // the thread's x in row 0 of each of the three z-planes + a block-uniform in-plane offset (direction row + y row;
  // periodic wrap by conditional add as in Neigh)
  const int ym = (y == 0) ? p.ny - 1 : y - 1, yp = (y == p.ny - 1) ? 0 : y + 1;
  const int zm = (z == 0) ? p.nz - 1 : z - 1, zp = (z == p.nz - 1) ? 0 : z + 1;
  const long long oyb[3] = {4LL * ym * p.rs, 4LL * y * p.rs, 4LL * yp * p.rs};
  const addr_t xb = (addr_t)__cvta_generic_to_global(src) + 4ull * x;
  const addr_t P[3] = {xb + 4ull * (zm * p.zs), xb + 4ull * (z * p.zs), xb + 4ull * (zp * p.zs)};
  const long long dsb = 4LL * p.ds;
  const long long dm = (x == 0) ? 4LL * (p.nx - 1) : -4LL;  // cell 0's x - 1, in bytes relative to x
  const long long dp = (x + 2 == p.nx) ? -4LL * x : 8LL;    // cell 1's x + 1
  const int cell0 = x + p.nx * (y + p.ny * z);
  const CellFlags<BC> c0(p, x, y, z, cell0), c1(p, x + 1, y, z, cell0 + 1);
  float g0[Q], g1[Q];
  static_for<0, Q>([&](auto A) {
    constexpr int a = decltype(A)::value;
    using D = Dir<Q, a>;
    constexpr int o = D::opp;
    // pair base in the row of the upstream node (x - e_a), and in the wall slot's row (own row, opposite direction;
    // t_a == t_abar: same shift)
    const addr_t up = P[1 - D::ez] + (addr_t)(a * dsb + oyb[1 - D::ey]);
    if constexpr (D::ex == 0) {
      addr_t q = up;
      if constexpr (BC == BC_WALLS && D::s > 0) {
        if (c0.template leaves<Q, a, -1>()) q = P[1] + (addr_t)(o * dsb + oyb[1]);  // depends on y, z only: the same for both cells
      }
      asm("ld.global.nc.v2.f32 {%0, %1}, [%2];" : "=f"(g0[a]), "=f"(g1[a]) : "l"(q));
    } else {
      // e_x = +1 pulls from (x-1, x), e_x = -1 from (x+1, x+2)
      addr_t q0 = up + (addr_t)(D::ex == 1 ? dm : 4LL);
      addr_t q1 = up + (addr_t)(D::ex == 1 ? 0LL : dp);
      if constexpr (BC == BC_WALLS) {
        const addr_t wl = P[1] + (addr_t)(o * dsb + oyb[1]);
        if (c0.template leaves<Q, a, -1>()) q0 = wl;
        if (c1.template leaves<Q, a, -1>()) q1 = wl + 4;
      }
      asm("ld.global.nc.f32 %0, [%1];" : "=f"(g0[a]) : "l"(q0));
      asm("ld.global.nc.f32 %0, [%1];" : "=f"(g1[a]) : "l"(q1));
    }
  });
  const addr_t O = (addr_t)__cvta_generic_to_global(dst) + 4ull * (z * p.zs + x) + (addr_t)oyb[1];
  // cell 0 in place (its results wait in g0 for their partners), then cell 1, stored as pairs
  collide_shifted<Q, EQ, BC, FORCE>(g0, p, c0, cell0, z, [&](auto A, double v) { g0[decltype(A)::value] = (float)v; });
  collide_shifted<Q, EQ, BC, FORCE>(g1, p, c1, cell0 + 1, z, [&](auto A, double v) {
    constexpr int a = decltype(A)::value;
    asm volatile("st.global.v2.f32 [%0], {%1, %2};" ::"l"(O + (addr_t)(a * dsb)), "f"(g0[a]), "f"((float)v) : "memory");
  });
}

// ---------------------------------------------------------------------------------------
// Two time steps per pass through HBM (A/B scheme, fp64, BC_PERIODIC / BC_WALLS).  The one-step kernel above sits at the ceiling of
// its access pattern (every population read once and written once per step: 0.999 x algorithmic DRAM bytes at 1.05 x the
// device-copy bandwidth), so more lattice updates per second means fewer bytes per update.  A block owns a TX x TY
// column of the box and marches along z.  Per plane it runs
//   stage 1  the ordinary step t -> t+1 (pull from `src`, collide) on the tile EXTENDED by one cell on every side in
//            x and y, and keeps the result in shared memory instead of storing it;
//   stage 2  step t+1 -> t+2 on the tile itself, one plane behind, pulling from the three planes of stage-1 results in
//            shared memory, and stores to `dst`.
// What stage 2 pulls from plane q-1 are the e_z = +1 populations only, from plane q the e_z = 0 ones and from plane q+1
// the e_z = -1 ones, so a plane's stage-1 result is kept per class for exactly as long as it is needed: the e_z = -1
// class for the rest of the iteration that made it, e_z = 0 for one more iteration (2 slots), e_z = +1 for two more
// (3 slots) — 38 population planes of the extended tile for D3Q19 instead of 3 x 19 — when a second barrier follows
// stage 2; one slot more per class (57 planes) lets ONE barrier per plane do (Ab2Tile).  HBM traffic per TWO steps: one read
// of the extended tile (the rim is shared with the neighbouring blocks through the L2) and one write of the tile,
// against two reads and two writes; the price is (TX+2)(TY+2)/(TX TY) collisions in stage 1 and the block barriers.
// Same arithmetic per cell as ab_cell (collide): bit-identical to two launches of stream_collide_ab.
// Measured (lbm_inst.cu picks the variant): D3Q19 32 x 8 tiles, one barrier, register prefetch, one block per SM:
// 512^3 22.5 -> 33.6 GLUPS in one launch, 31.4 sustained; D3Q27 16 x 8, two barriers, two blocks: 400^3 15.8 -> 21.0.
template <int Q, int EZ>
__host__ __device__ constexpr int ez_class_size() {
  int n = 0;
  for (int a = 0; a < Q; ++a) n += (Lattice<Q>::e[a][2] == EZ);
  return n;
}
template <int Q, int A>
__host__ __device__ constexpr int ez_class_index() {  // position of direction A among the directions with the same e_z
  int n = 0;
  for (int a = 0; a < A; ++a) n += (Lattice<Q>::e[a][2] == Lattice<Q>::e[A][2]);
  return n;
}

// ONEBAR: one more slot per class (2 / 3 / 4), so that stage 1 of the next plane never writes a slot stage 2 of this plane
// still reads and ONE block barrier per plane is enough.  PREFETCH: the stage-1 loads of the next plane are issued
// before stage 2 of this one, so that their latency is covered by it (Q more register pairs).
template <int Q, int TX, int TY, bool ONEBAR, bool WALLS = false>
struct Ab2Tile {
  static constexpr int EX = TX + 2, EY = TY + 2, CELLS = EX * EY;  // stage-1 tile
  static constexpr int THREADS = ((CELLS + 31) / 32) * 32;
  static constexpr int NM = ez_class_size<Q, -1>(), N0 = ez_class_size<Q, 0>(), NP = ez_class_size<Q, 1>();
  // Slots per class.  With one barrier per plane (between stage 1 and stage 2) a warp may run stage 1 of iteration k+1
  // while another still runs stage 2 of iteration k, so slot (k+1) mod S must differ from every slot stage 2(k) reads:
  // e_z = -1: k, and with walls k-1 (a wall link's own-plane value);  e_z = 0: k-1;  e_z = +1: k-2, with walls k-1.
  // With two barriers per plane (the second after stage 2) stage 1 of iteration k only has to spare what stage 2 of the
  // SAME iteration reads: 1 / 2 / 3 slots, with walls 2 / 2 / 3.
  static constexpr int SM_ = ONEBAR ? (WALLS ? 3 : 2) : (WALLS ? 2 : 1), S0 = ONEBAR ? 3 : 2, SP = ONEBAR ? 4 : 3;
  // shared memory, in doubles: [SM_][NM][CELLS] | [S0][N0][CELLS] | [SP][NP][CELLS]
  static constexpr int OFF0 = SM_ * NM * CELLS, OFFP = OFF0 + S0 * N0 * CELLS, DOUBLES = OFFP + SP * NP * CELLS;
  static constexpr size_t SMEM_BYTES = (size_t)DOUBLES * sizeof(double);
};

// BC_WALLS (halfway bounce-back, Ladd lid, inlet / outlet through collide's open_link): cells of the extended tile that lie
// beyond a wall face are no nodes and are skipped; stage 1 pulls with the wall-slot select of the one-step kernel; stage 2
// takes a wall link from the OWN cell's opposite direction in plane q — the e_z = +1 / 0 / -1 class of the previous
// iteration (the e_z = -1 class lives one iteration longer for that: three slots instead of two).
template <int Q, int EQ, int BC, bool FORCE, int TX, int TY, int MINB, bool ONEBAR, bool PREFETCH>
__global__ void __launch_bounds__(Ab2Tile<Q, TX, TY, ONEBAR, BC == BC_WALLS && ONEBAR>::THREADS, MINB)
    stream_collide_ab2(const double* __restrict__ src, double* __restrict__ dst, int zchunk, const __grid_constant__ Params p) {
  static_assert(BC == BC_PERIODIC || BC == BC_WALLS, "no link mask");
  // ZGHOST (BC_WALLS with two barriers per plane; the launcher admits it for boxes whose x and y faces are periodic): the
  // z walls act through GHOST planes.  When stage 1 has plane 0, every cell also puts its outgoing e_z = -1 values where
  // stage 2 of plane 0 will look for the e_z = +1 populations of plane -1 (f_a(x) = f*_abar(x): Eq. 10's rule), and
  // in the iteration of the missing plane nz the e_z = +1 values of plane nz-1 go where its e_z = -1 populations are
  // expected; stage 2 then runs the periodic code on the periodic slot set, with no select and no extra slot.
  constexpr bool ZGHOST = (BC == BC_WALLS) && !ONEBAR;
  using T = Ab2Tile<Q, TX, TY, ONEBAR, BC == BC_WALLS && ONEBAR>;
  extern __shared__ double sm[];
  const int t = threadIdx.x;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
  const int zs = blockIdx.z * zchunk, ze = min(zs + zchunk, p.nz);  // stage-2 planes [zs, ze)
  // stage 1: thread t owns cell (xe, ye) of the extended tile = node (x0-1+xe, y0-1+ye), wrapped periodically
  bool s1 = t < T::CELLS;
  const int ye = t / T::EX, xe = t - ye * T::EX;
  int gx = x0 - 1 + xe, gy = y0 - 1 + ye;
  if constexpr (BC == BC_WALLS) {  // beyond a wall face: no node (faces of an axis are periodic or walls in pairs)
    s1 = s1 & !(((gx < 0) | (gx >= p.nx)) & (p.wall[0] != 0)) & !(((gy < 0) | (gy >= p.ny)) & (p.wall[2] != 0));
  }
  gx = (gx < 0) ? gx + p.nx : (gx >= p.nx) ? gx - p.nx : gx;
  gy = (gy < 0) ? gy + p.ny : (gy >= p.ny) ? gy - p.ny : gy;
  const int ox[3] = {(gx == 0) ? p.nx - 1 : gx - 1, gx, (gx == p.nx - 1) ? 0 : gx + 1};
  const int oy[3] = {((gy == 0) ? p.ny - 1 : gy - 1) * p.rs, gy * p.rs, ((gy == p.ny - 1) ? 0 : gy + 1) * p.rs};
  const int c1xy = gx + p.nx * gy;
  // stage 2: thread t < TX*TY owns node (x0+xi, y0+yi) = cell t2 of the extended tile
  const int yi = t / TX, xi = t - yi * TX;
  const bool s2 = (t < TX * TY) & (x0 + xi < p.nx) & (y0 + yi < p.ny);  // (ragged grids: the last tiles hang over the box)
  const int t2 = (yi + 1) * T::EX + xi + 1;
  const int o2 = (x0 + xi) + (y0 + yi) * p.rs;
  const int c2xy = (x0 + xi) + p.nx * (y0 + yi);
  // plane pz of stage 1 exists unless it lies beyond a z wall (block-uniform)
  auto plane_exists = [&](int pz) { return BC == BC_PERIODIC || !((pz < 0 || pz >= p.nz) && p.wall[4] != 0); };
  auto wrap_z = [&](int pz) { return (pz < 0) ? pz + p.nz : (pz >= p.nz) ? pz - p.nz : pz; };
  // BC_WALLS: only the tiles on an x / y wall and the planes on a z wall hold wall links; everything else takes the
  // periodic code (no flag tests, no second address, no select: block-uniform branches), which is what the step costs
  // in this latency-bound kernel (512^3, z walls: 28.7 against 31.2 GLUPS periodic when every cell ran the selects).
  // (the extended tile reaches one cell beyond the tile: it must not contain the last node either)
  const bool tile_walls = (BC == BC_WALLS) && ((((x0 == 0) | (x0 + TX >= p.nx - 1)) & (p.wall[0] != 0)) | (((y0 == 0) | (y0 + TY >= p.ny - 1)) & (p.wall[2] != 0)));
  auto plane_walls = [&](int z) { return (BC == BC_WALLS) && (tile_walls | (((z == 0) | (z == p.nz - 1)) & (p.wall[4] != 0))); };
  auto pull_plane_as = [&](auto W, double (&f)[Q], int z) {
    const int zm = (z == 0) ? p.nz - 1 : z - 1, zp = (z == p.nz - 1) ? 0 : z + 1;
    const long long oz[3] = {zm * p.zs, z * p.zs, zp * p.zs};
    const CellFlags<decltype(W)::value ? BC_WALLS : BC_PERIODIC> c(p, gx, gy, z, 0);
    static_for<0, Q>([&](auto A) {
      constexpr int a = decltype(A)::value;
      using D = Dir<Q, a>;
      const double* q = plane<a>(src, p.ds) + ((ox[1 - D::ex] + oy[1 - D::ey]) + oz[1 - D::ez]);
      if constexpr (decltype(W)::value != 0 && D::s > 0) {
        if (c.template leaves<Q, a, -1>()) q = plane<D::opp>(src, p.ds) + ((ox[1] + oy[1]) + oz[1]);  // a select, not a branch
      }
      f[a] = LBM_LD_STREAM(q);
    });
  };
  auto pull_plane = [&](double (&f)[Q], int pz) {  // the Q populations that stream into the thread's stage-1 cell in plane pz
    const int z = wrap_z(pz);
    if (plane_walls(z)) pull_plane_as(IC<1>{}, f, z);
    else pull_plane_as(IC<0>{}, f, z);
  };
  double fn[PREFETCH ? Q : 1];
  if constexpr (PREFETCH) {
    if (s1 && plane_exists(zs - 1)) pull_plane(fn, zs - 1);
  }
  for (int k = 0, pz = zs - 1; pz <= ze; ++pz, ++k) {
    const int km = k % T::SM_, k0 = k % T::S0, kp = k % T::SP;
    if (s1) {
      if (plane_exists(pz)) {
        const int z = wrap_z(pz);
        double f[Q];
        if constexpr (PREFETCH) {
          static_for<0, Q>([&](auto A) { f[decltype(A)::value] = fn[decltype(A)::value]; });
        } else {
          pull_plane(f, pz);
        }
        const CellFlags<BC> c(p, gx, gy, z, 0);
        collide<Q, EQ, BC, FORCE>(f, p, c, c1xy + p.nx * p.ny * z, z);
        static_for<0, Q>([&](auto A) {
          constexpr int a = decltype(A)::value;
          constexpr int j = ez_class_index<Q, a>();
          if constexpr (Dir<Q, a>::ez == -1) sm[(km * T::NM + j) * T::CELLS + t] = f[a];
          else if constexpr (Dir<Q, a>::ez == 0) sm[T::OFF0 + (k0 * T::N0 + j) * T::CELLS + t] = f[a];
          else sm[T::OFFP + (kp * T::NP + j) * T::CELLS + t] = f[a];
        });
        if constexpr (ZGHOST) {
          if (z == 0 && p.wall[4] != 0) {  // ghost plane -1: its e_z = +1 class lives in the slot of the previous iteration
            static_for<0, Q>([&](auto A) {
              constexpr int a = decltype(A)::value;
              using D = Dir<Q, a>;
              if constexpr (D::ez == 1) {
                // the reader is the cell itself, one plane up the link: it pulls direction a from the cell at -e_a (x, y)
                const bool in = (xe - D::ex >= 0) & (xe - D::ex < T::EX) & (ye - D::ey >= 0) & (ye - D::ey < T::EY);
                if (in) sm[T::OFFP + (((k + T::SP - 1) % T::SP) * T::NP + ez_class_index<Q, a>()) * T::CELLS + t - D::ey * T::EX - D::ex] = f[D::opp];
              }
            });
          }
        }
      } else if constexpr (ZGHOST) {
        if (pz == p.nz) {  // ghost plane nz: its e_z = -1 class, from the e_z = +1 values this thread stored for plane nz-1
          static_for<0, Q>([&](auto A) {
            constexpr int a = decltype(A)::value;
            using D = Dir<Q, a>;
            if constexpr (D::ez == -1) {
              const bool in = (xe - D::ex >= 0) & (xe - D::ex < T::EX) & (ye - D::ey >= 0) & (ye - D::ey < T::EY);
              const double v = sm[T::OFFP + (((k + T::SP - 1) % T::SP) * T::NP + ez_class_index<Q, D::opp>()) * T::CELLS + t];
              if (in) sm[(km * T::NM + ez_class_index<Q, a>()) * T::CELLS + t - D::ey * T::EX - D::ex] = v;
            }
          });
        }
      }
      // the next plane's loads go out AFTER this plane's collision and shared-memory stores (measured: issued before
      // the collision, 512^3 falls from 33.6 to 24.4 GLUPS) and have the barrier and stage 2 to arrive
      if constexpr (PREFETCH) {
        if (pz < ze && plane_exists(pz + 1)) pull_plane(fn, pz + 1);
      }
    }
    __syncthreads();
    if (s2 && k >= 2) {
      // plane q = pz - 1: e_z = -1 populations of plane q+1 (this iteration), e_z = 0 of plane q (previous iteration),
      // e_z = +1 of plane q-1 (the one before)
      const int q = pz - 1;
      const double* sn = sm + (km * T::NM) * T::CELLS + t2;
      const double* s0 = sm + T::OFF0 + (((k + T::S0 - 1) % T::S0) * T::N0) * T::CELLS + t2;
      const double* sp = sm + T::OFFP + (((k + T::SP - 2) % T::SP) * T::NP) * T::CELLS + t2;
      // the own plane's classes, for wall links: e_z = -1 and e_z = +1 of plane q were stored in the previous iteration
      const double* snq = sm + (((k + T::SM_ - 1) % T::SM_) * T::NM) * T::CELLS + t2;
      const double* spq = sm + T::OFFP + (((k + T::SP - 1) % T::SP) * T::NP) * T::CELLS + t2;
      const CellFlags<BC> c(p, x0 + xi, y0 + yi, q, 0);
      double f[Q];
      auto gather2 = [&](auto W) {
        static_for<0, Q>([&](auto A) {
          constexpr int a = decltype(A)::value;
          using D = Dir<Q, a>;
          constexpr int j = ez_class_index<Q, a>();
          constexpr int d = j * T::CELLS - D::ey * T::EX - D::ex;  // class row + the upstream cell inside the extended tile
          const double* r = (D::ez == -1) ? sn + d : (D::ez == 0) ? s0 + d : sp + d;
          if constexpr (decltype(W)::value != 0 && D::s > 0) {
            constexpr int jo = ez_class_index<Q, D::opp>() * T::CELLS;  // f_a = f*_abar of the own cell (Eq. 10's rule)
            if (c.template leaves<Q, a, -1>()) r = (D::ez == -1) ? spq + jo : (D::ez == 0) ? s0 + jo : snq + jo;
          }
          f[a] = *r;
        });
      };
      if (!ZGHOST && plane_walls(q)) gather2(IC<1>{});
      else gather2(IC<0>{});
      collide<Q, EQ, BC, FORCE>(f, p, c, c2xy + p.nx * p.ny * q, q);
      double* out = dst + (o2 + q * p.zs);
      static_for<0, Q>([&](auto A) {
        constexpr int a = decltype(A)::value;
        LBM_ST_STREAM(plane<a>(out, p.ds), f[a]);
      });
    }
    if constexpr (!ONEBAR) __syncthreads();
  }
}

// Small grids (both buffers resident in the L2: 32^3, 64^3, the paper's 512 x 128 channel) are bound by the launch
// rate of one kernel per step (4-5 us), and CUDA-graph replay is slower still.  This persistent kernel takes all the steps of one lbm_step call in ONE cooperative
// launch: every thread keeps its cell, the two buffers swap roles each step, a grid-wide barrier separates the steps
// (stores fenced before it, loads through L2 after it), and the populations never leave the L2.  Compiled for two
// blocks per SM (128 registers: no spills): a grid that fits at all is far from filling the device.
template <int Q, int EQ, int BC, bool FORCE, typename ST, bool SYM = false>
__global__ void __launch_bounds__(256, 2) stream_collide_ab_persistent(ST* b0, ST* b1, int nsteps, const __grid_constant__ Params p) {
  cooperative_groups::grid_group grid = cooperative_groups::this_grid();
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  const int y0 = blockIdx.y * blockDim.y + threadIdx.y, ystep = gridDim.y * blockDim.y;
  for (int s = 0; s < nsteps; ++s) {
    const ST* src = (s & 1) ? b1 : b0;
    ST* dst = (s & 1) ? b0 : b1;
    if (x < p.nx) {
      // the launcher gives the grid as many layers of blocks along z (then y) as fit the device at once; a block takes
      // every gridDim.z-th plane and every gridDim.y-th group of rows
      for (int z = blockIdx.z; z < p.nz; z += gridDim.z)
        for (int y = y0; y < p.ny; y += ystep) ab_cell<Q, EQ, BC, FORCE, ST, false, SYM, true>(src, dst, p, x, y, z);
    }
    if (s + 1 < nsteps) grid.sync();
  }
}

// AA pattern (one buffer, in place).  Even phase: slot (x,a) holds f_a(x); read local, collide,
// write f*_a(x) into slot (x, abar) — every access aligned.  Odd phase: f_a(x) = slot(x - e_a, abar)
// (wall link: slot(x, a)); collide; write f*_a(x) into slot (x + e_a, a) (wall link: slot(x, abar)),
// after which the buffer is in natural layout again.  Each thread reads and writes exactly its
// own set of Q slots (the odd phase writes f*_a where it read f_abar), so there is no
// inter-thread hazard in either phase.
// COHERENT: loads through L2 (ld.global.cg) for the persistent kernel, as in ab_cell.
template <bool COHERENT, typename ST, int Q, int A>
__device__ __forceinline__ double ld_pop_aa(const ST* q) {
  if constexpr (COHERENT) {
    if constexpr (sizeof(ST) == 8) return __ldcg(q);
    else return (double)__ldcg(q) + Dir<Q, A>::t;
  } else {
    return ld_pop_rw<ST, Q, A>(q, 0);
  }
}

template <int Q, int EQ, int BC, bool FORCE, typename ST, bool COHERENT>
__device__ __forceinline__ void aa_even_cell(ST* buf, const Params& p, int x, int y, int z) {
  const int cell = x + p.nx * (y + p.ny * z);
  const long long ic = (x + y * p.rs) + z * p.zs;  // storage offset (Neigh::ic)
  const CellFlags<BC> c(p, x, y, z, cell);
  double f[Q];
  static_for<0, Q>([&](auto A) {
    constexpr int a = decltype(A)::value;
    f[a] = ld_pop_aa<COHERENT, ST, Q, a>(plane<a>(buf, p.ds) + ic);
  });
  if (!c.template active<Q>()) return;  // after the loads: they do not wait for the link mask (see gather)
  nodal_replicate<Q, BC>(f, p, c);
  collide<Q, EQ, BC, FORCE>(f, p, c, cell, z);
  static_for<0, Q>([&](auto A) {
    constexpr int a = decltype(A)::value;
    st_pop<ST, Q, a>(plane<Dir<Q, a>::opp>(buf, p.ds), ic, f[a]);
  });
}

template <int Q, int EQ, int BC, bool FORCE, typename ST, bool COHERENT>
__device__ __forceinline__ void aa_odd_cell(ST* buf, const Params& p, int x, int y, int z) {
  const Neigh nb(p, x, y, z);
  const CellFlags<BC> c(p, x, y, z, nb.cell);
  double f[Q];
  // f_a(x) comes from the slot that f*_abar(x) goes to (link x <-> x - e_a traversed both ways)
  auto link = [&](auto A) { return (const ST*)plane<Dir<Q, decltype(A)::value>::opp>(buf, p.ds) + nb.template at<Q, decltype(A)::value, -1>(); };
  auto wall = [&](auto A) { return (const ST*)plane<decltype(A)::value>(buf, p.ds) + nb.ic; };
  if (!gather<Q, BC>(f, c, link, wall, [](auto A, const ST* q) { return ld_pop_aa<COHERENT, ST, Q, decltype(A)::value>(q); })) return;
  nodal_replicate<Q, BC>(f, p, c);
  collide<Q, EQ, BC, FORCE>(f, p, c, nb.cell, z);
  static_for<0, Q>([&](auto A) {
    constexpr int a = decltype(A)::value;
    constexpr int o = Dir<Q, a>::opp;
    ST* q = plane<a>(buf, p.ds) + nb.template at<Q, a, 1>();
    if constexpr (BC != BC_PERIODIC) {
      if (c.template leaves<Q, a, 1>()) q = plane<o>(buf, p.ds) + nb.ic;
    }
    st_pop<ST, Q, a>(q, 0, f[a]);
  });
}

template <int Q, int EQ, int BC, bool FORCE, typename ST>
__global__ void __launch_bounds__(256, kMinBlocks<Q, FORCE, true>) stream_collide_aa_even(ST* buf, const __grid_constant__ Params p) {
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  const int y = blockIdx.y * blockDim.y + threadIdx.y;
  const int z = blockIdx.z;
  if (x >= p.nx || y >= p.ny) return;
  aa_even_cell<Q, EQ, BC, FORCE, ST, false>(buf, p, x, y, z);
}

template <int Q, int EQ, int BC, bool FORCE, typename ST>
__global__ void __launch_bounds__(256, kMinBlocks<Q, FORCE, true>) stream_collide_aa_odd(ST* buf, const __grid_constant__ Params p) {
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  const int y = blockIdx.y * blockDim.y + threadIdx.y;
  const int z = blockIdx.z;
  if (x >= p.nx || y >= p.ny) return;
  aa_odd_cell<Q, EQ, BC, FORCE, ST, false>(buf, p, x, y, z);
}

// Odd phase, one grid row per block (y = blockIdx.y, z = blockIdx.z; BC_PERIODIC / BC_WALLS).  The odd phase touches Q
// DIFFERENT slots per cell and touches each of them twice (f_a is read where f*_abar is written: the link x <-> x - e_a
// traversed both ways); in aa_odd_cell ptxas keeps or rebuilds Q 64-bit addresses across the collision (124-128
// registers, D3Q27 spills up to 360 B, two blocks per SM).  Here everything but x is block-uniform: the row base of
// every slot (direction row + y row + z plane, wall rows included for the y / z faces) lives in the uniform datapath, a
// thread holds x-1, x, x+1 and its two x-face flags, and a slot address is one 64-bit add that is simply repeated
// for the store.
template <int Q, bool FORCE>
constexpr int kAaRowMinBlocks = (Q == 27) ? 2 : (Q == 19) ? (FORCE ? 2 : 3) : (FORCE ? 3 : 4);

template <int Q, int EQ, int BC, bool FORCE, typename ST>
__global__ void __launch_bounds__(256, kAaRowMinBlocks<Q, FORCE>) stream_collide_aa_odd_row(ST* buf, const __grid_constant__ Params p) {
  static_assert(BC != BC_GEO, "the link-mask kernels keep aa_odd_cell");
  typedef unsigned long long addr_t;
  constexpr long long E = sizeof(ST);
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  const int y = blockIdx.y, z = blockIdx.z;
  if (x >= p.nx) return;
  const int ym = (y == 0) ? p.ny - 1 : y - 1, yp = (y == p.ny - 1) ? 0 : y + 1;
  const int zm = (z == 0) ? p.nz - 1 : z - 1, zp = (z == p.nz - 1) ? 0 : z + 1;
  // block-uniform byte offsets of the three y rows and the three z planes; per thread: the byte address of x-1, x, x+1
  // in row 0 of plane 0 of direction 0
  long long oy[3] = {E * ym * p.rs, E * y * p.rs, E * yp * p.rs};
  long long oz[3] = {E * zm * p.zs, E * z * p.zs, E * zp * p.zs};
  const long long dsb = E * p.ds;
  const addr_t b0 = (addr_t)__cvta_generic_to_global(buf);
  addr_t X[3] = {b0 + E * ((x == 0) ? p.nx - 1 : x - 1), b0 + E * x, b0 + E * ((x == p.nx - 1) ? 0 : x + 1)};
  const int cell = x + p.nx * (y + p.ny * z);
  const CellFlags<BC> c(p, x, y, z, cell);
  // slot(a): where f_a(x) is read and f*_abar(x) is written — slot (x - e_a, abar), or (x, a) at a wall link
  auto slot = [&](auto A) -> addr_t {
    constexpr int a = decltype(A)::value;
    using D = Dir<Q, a>;
    const long long row = D::opp * dsb + oy[1 - D::ey] + oz[1 - D::ez];  // block-uniform
    addr_t q = X[1 - D::ex] + (addr_t)row;
    if constexpr (BC == BC_WALLS && D::s > 0) {
      bool w = false;
      if constexpr (D::ey == 1) w = w | c.lo[1];
      if constexpr (D::ey == -1) w = w | c.hi[1];
      if constexpr (D::ez == 1) w = w | c.lo[2];
      if constexpr (D::ez == -1) w = w | c.hi[2];
      if constexpr (D::ex == 1) w = w | c.lo[0];
      if constexpr (D::ex == -1) w = w | c.hi[0];
      if (w) q = X[1] + (addr_t)(a * dsb + oy[1] + oz[1]);
    }
    return q;
  };
  double f[Q];
  static_for<0, Q>([&](auto A) {
    constexpr int a = decltype(A)::value;
    f[a] = ld_pop_rw<ST, Q, a>((const ST*)slot(A), 0);
  });
  // the store addresses are rebuilt after the collision (two adds each) instead of Q of them staying live across it
  asm volatile("" : "+l"(X[0]), "+l"(X[1]), "+l"(X[2]));
  asm volatile("" : "+l"(oy[0]), "+l"(oy[1]), "+l"(oy[2]), "+l"(oz[0]), "+l"(oz[1]), "+l"(oz[2]));
  collide<Q, EQ, BC, FORCE>(f, p, c, cell, z);
  static_for<0, Q>([&](auto A) {
    constexpr int a = decltype(A)::value;
    constexpr int o = Dir<Q, a>::opp;
    st_pop<ST, Q, o>((ST*)slot(A), 0, f[o]);
  });
}

// The in-place scheme in one cooperative launch per lbm_step call, for grids whose ONE buffer fits the L2 (where
// LBM_SCHEME_AUTO picks this scheme): phases alternate from `phase` on, a grid-wide barrier after each step.
template <int Q, int EQ, int BC, bool FORCE, typename ST>
__global__ void __launch_bounds__(256, 2) stream_collide_aa_persistent(ST* buf, int nsteps, int phase, const __grid_constant__ Params p) {
  cooperative_groups::grid_group grid = cooperative_groups::this_grid();
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  const int y0 = blockIdx.y * blockDim.y + threadIdx.y, ystep = gridDim.y * blockDim.y;
  for (int s = 0; s < nsteps; ++s, phase ^= 1) {
    if (x < p.nx) {
      for (int z = blockIdx.z; z < p.nz; z += gridDim.z)
        for (int y = y0; y < p.ny; y += ystep) {
          if (phase == 0) aa_even_cell<Q, EQ, BC, FORCE, ST, true>(buf, p, x, y, z);
          else aa_odd_cell<Q, EQ, BC, FORCE, ST, true>(buf, p, x, y, z);
        }
    }
    if (s + 1 < nsteps) grid.sync();
  }
}

// ---------------------------------------------------------------------------------------
// Canonical state access (D:R15).  MODE selects how slot contents map to f_a(x):
//   NATURAL   : f_a(x) = slot(x, a)                                   (AA, even phase)
//   PULL      : f_a(x) = slot(x - e_a, a),   wall link: slot(x, abar)   (A/B)
//   PULL_SWAP : f_a(x) = slot(x - e_a, abar), wall link: slot(x, a)      (AA, odd phase)
// followed by Eq. 10 on wall nodes under the nodal model.
enum { MODE_NATURAL = 0, MODE_PULL = 1, MODE_PULL_SWAP = 2 };

template <int Q, int BC, int MODE, typename ST>
__device__ __forceinline__ void load_canonical(double (&f)[Q], const ST* buf, const Params& p, const Neigh& nb, const CellFlags<BC>& c) {
  static_for<0, Q>([&](auto A) {
    constexpr int a = decltype(A)::value;
    constexpr int o = Dir<Q, a>::opp;
    const ST* q;
    if constexpr (MODE == MODE_NATURAL) {
      q = plane<a>(buf, p.ds) + nb.ic;
    } else {
      constexpr int q_in = (MODE == MODE_PULL) ? a : o, q_wall = (MODE == MODE_PULL) ? o : a;
      q = plane<q_in>(buf, p.ds) + nb.template at<Q, a, -1>();
      if constexpr (BC != BC_PERIODIC) {
        if (c.template leaves<Q, a, -1>()) q = plane<q_wall>(buf, p.ds) + nb.ic;
      }
    }
    f[a] = ld_pop_rw<ST, Q, a>(q, 0);
  });
  if constexpr (BC == BC_GEO && MODE == MODE_PULL) {
    if (touches_sym<BC>(p, c)) {  // D:R25: links through SYMMETRY faces read the mirror image
      static_for<0, Q>([&](auto A) {
        constexpr int a = decltype(A)::value;
        if constexpr (Dir<Q, a>::s > 0) {
          int dir, cidx;
          long long idx;
          if (mirror_link<Q, a, -1, BC>(p, c, nb, dir, idx, cidx) && !c.template leaves<Q, a, -1>())
            f[a] = ld_pop_rw<ST, Q, a>(buf + dir * p.ds, idx);
        }
      });
    }
  }
  nodal_replicate<Q, BC>(f, p, c);
}

// Row-wise grid-stride loop of the sweeps off the per-step path: a 256-thread block is bx x (256/bx)
// with bx a power of two covering the row (or 256); rows (y,z) are dealt to the blocks round-robin.
// One 32-bit division per row, none per cell; x stays the coalesced direction.
// The rows are those of the updated planes [z_lo, z_hi), or of every plane (the halo planes of a slab too).
template <typename F>
__device__ __forceinline__ void for_each_cell_in_rows(const Params& p, int bx, int r0, int rows, F&& body) {
  const int tx = threadIdx.x & (bx - 1), ty = threadIdx.x / bx, by = blockDim.x / bx;
  for (int r = r0 + blockIdx.x * by + ty; r < rows; r += gridDim.x * by) {
    const int z = r / p.ny, y = r - z * p.ny;
    for (int x = tx; x < p.nx; x += bx) body(x, y, z, x + p.nx * r);
  }
}
template <typename F>
__device__ __forceinline__ void for_each_cell(const Params& p, int bx, F&& body, bool with_halo = false) {
  for_each_cell_in_rows(p, bx, with_halo ? 0 : p.ny * p.z_lo, with_halo ? p.ny * p.nz : p.ny * p.z_hi, body);
}

// lbm_get_populations: canonical f[a*N+i] (always fp64) out of the storage buffer; inactive nodes report 0.
template <int Q, int BC, int MODE, typename ST>
__global__ void __launch_bounds__(256, 2) export_canonical(const ST* buf, double* __restrict__ out, int bx, const __grid_constant__ Params p) {
  for_each_cell(p, bx, [&](int x, int y, int z, int i) {
    const Neigh nb(p, x, y, z);
    const CellFlags<BC> c(p, x, y, z, i);
    double f[Q];
    if (c.template active<Q>()) {
      load_canonical<Q, BC, MODE, ST>(f, buf, p, nb, c);
    } else {
      static_for<0, Q>([&](auto A) { f[decltype(A)::value] = 0.0; });
    }
    static_for<0, Q>([&](auto A) {
      constexpr int a = decltype(A)::value;
      plane<a>(out, p.N)[i] = f[a];
    });
  });
}

// lbm_set_populations / init: canonical f[a*N+i] (fp64) into the storage buffer.
//   NATURAL: slot(x,a) = f_a(x).   PULL (A/B): slot(y,a) = f_a(y + e_a) if y + e_a is an active node, else f_abar(y).
template <int Q, int BC, int MODE, typename ST>
__global__ void __launch_bounds__(256) import_canonical(const double* __restrict__ in, ST* __restrict__ buf, int bx, const __grid_constant__ Params p) {
  static_assert(MODE != MODE_PULL_SWAP, "imports always land in an even phase");
  for_each_cell(p, bx, [&](int x, int y, int z, int i) {
    const Neigh nb(p, x, y, z);
    const CellFlags<BC> c(p, x, y, z, i);
    if (!c.template active<Q>()) return;
    static_for<0, Q>([&](auto A) {
      constexpr int a = decltype(A)::value;
      constexpr int o = Dir<Q, a>::opp;
      const double* q = plane<a>(in, p.N) + i;
      if constexpr (MODE != MODE_NATURAL) {
        q = plane<a>(in, p.N) + nb.template cat<Q, a, 1>();
        if constexpr (BC != BC_PERIODIC) {
          if (c.template leaves<Q, a, 1>()) q = plane<o>(in, p.N) + i;
        }
        if constexpr (BC == BC_GEO && Dir<Q, a>::s > 0) {
          // D:R25: a slot whose link leaves through SYMMETRY faces is read by the mirror image, as direction `dir`
          int dir, cidx;
          long long idx;
          if (p.any_sym && mirror_link<Q, a, 1, BC>(p, c, nb, dir, idx, cidx) && !c.template leaves<Q, a, 1>())
            q = in + (long long)dir * p.N + cidx;
        }
        // slab: the halo planes are filled here too (the canonical arrays of a slab carry the neighbour's
        // planes); a slot whose downstream node would lie beyond a halo plane is never read: leave it.
        if constexpr (Dir<Q, a>::ez != 0) {
          const int zd = z + Dir<Q, a>::ez;
          if (p.slab && (zd < 0 || zd >= p.nz) && !c.template leaves<Q, a, 1>()) return;
        }
      }
      st_pop<ST, Q, a>(plane<a>(buf, p.ds), nb.ic, __ldg(q));
    });
  }, p.slab != 0);
}

// InitPDF: f_a(x, 0) = feq_a(rho(x), u(x)), written straight into the storage buffer in the layout the
// scheme wants at an even phase (S:§8c-S: "f^eq evaluated at the downstream cell") — one pass, 32 B read + Q stored
// elements per cell, instead of a canonical array that is written, read back and written again.
//   NATURAL (AA):  slot(x, a) = f_a(x).
//   PULL (A/B):    B = S^-1 f as a PUSH from the cell that owns the value: f_a(x) goes where the pull of x will look for
//                  it — slot(x - e_a, a) if the link has an active upstream node, the wall slot(x, abar) otherwise, the
//                  mirror image's slot through SYMMETRY faces (D:R25).  Every slot the first step reads is written by
//                  exactly one cell (S is a bijection on the slots); shifted stores stay unit-stride in x.
// Eq. 10 at t = 0 (D:R17) needs nothing here: the pull replicates f_abar into the wall links of a nodal wall node
// every time it gathers, so what their wall slots hold is never used.  A z-slab pushes from its own planes only: the
// slots of its halo planes that the first step reads are exactly the ones its first / last plane push into.
// Rows [r0, r1) of the grid (r = y + ny*z): the host entry point initialises z-chunks as their rho, u arrive.
template <int Q, int EQ, int BC, int MODE, typename ST>
__global__ void __launch_bounds__(256, 2) init_equilibrium_kernel(const double* __restrict__ rho, const double* __restrict__ u, ST* __restrict__ buf, int bx,
                                                               int r0, int r1, const __grid_constant__ Params p) {
  static_assert(MODE != MODE_PULL_SWAP, "initialisation always lands in an even phase");
  for_each_cell_in_rows(p, bx, r0, r1, [&](int x, int y, int z, int i) {
    const Neigh nb(p, x, y, z);
    const CellFlags<BC> c(p, x, y, z, i);
    if (!c.template active<Q>()) return;
    const double r = rho ? rho[i] : 1.0;
    const double ux = u ? u[i] : 0.0, uy = u ? plane<1>(u, p.N)[i] : 0.0, uz = u ? plane<2>(u, p.N)[i] : 0.0;
    double feq[Q];
    equilibrium<Q, EQ>(feq, r, ux, uy, uz);
    const bool at_mirror = (BC == BC_GEO) ? touches_sym<BC>(p, c) : false;
    static_for<0, Q>([&](auto A) {
      constexpr int a = decltype(A)::value;
      constexpr int o = Dir<Q, a>::opp;
      ST* q = plane<a>(buf, p.ds) + nb.ic;
      if constexpr (MODE == MODE_PULL && Dir<Q, a>::s > 0) {
        q = plane<a>(buf, p.ds) + nb.template at<Q, a, -1>();
        if constexpr (BC != BC_PERIODIC) {
          if (c.template leaves<Q, a, -1>()) q = plane<o>(buf, p.ds) + nb.ic;
        }
        if constexpr (BC == BC_GEO) {
          if (at_mirror) {
            int dir, cidx;
            long long idx;
            if (mirror_link<Q, a, -1, BC>(p, c, nb, dir, idx, cidx) && !c.template leaves<Q, a, -1>()) q = buf + dir * p.ds + idx;
          }
        }
      }
      st_pop<ST, Q, a>(q, 0, feq[a]);
    });
  });
}

// ---------------------------------------------------------------------------------------
// SetGeometry (D:R16).  classify: a node is active if it is fluid (geo = 0) or — nodal
// model — a solid node with at least one fluid node among its lattice neighbours (the wall nodes
// Eq. 10 and the collision act on).  links: the per-cell mask the BC_GEO kernels read.
template <int Q>
__global__ void __launch_bounds__(256) classify_nodes_kernel(const uint8_t* __restrict__ geo_in, uint8_t* __restrict__ geo, uint8_t* __restrict__ active,
                                                             int nodal, int bx, const __grid_constant__ Params p) {
  // geo_in: the caller's mask (any device-readable memory; NULL = no solid nodes); geo: the library's 0/1 copy.
  // z-slab (D:R21): geo_in carries TWO halo planes per side (nz + 2 planes, plane 1 + z of the handle's plane z), so
  // that the halo nodes — whose wall-node status the own planes' links depend on — see all their neighbours.
  const int pl = p.nx * p.ny;
  const int zin = p.slab ? 1 : 0;
  for_each_cell(p, bx, [&](int x, int y, int z, int i) {
    const bool solid = geo_in ? geo_in[i + zin * pl] != 0 : false;
    bool a = !solid;
    if (solid && nodal) {
      const Neigh nb(p, x, y, z);
      const CellFlags<BC_WALLS> c(p, x, y, z, i);
      static_for<0, Q>([&](auto A) {
        constexpr int b = decltype(A)::value;
        using D = Dir<Q, b>;
        if constexpr (D::s > 0) {
          if (!c.template leaves_box<Q, b, 1>()) {
            // slab: no wrap along z inside the handle — the neighbouring planes are in geo_in as they are
            const int j = p.slab ? nb.ox[1 + D::ex] + nb.cy[1 + D::ey] + (z + D::ez + zin) * pl : nb.template cat<Q, b, 1>();
            a = a | (geo_in[j] == 0);
          }
        }
      });
    }
    geo[i] = solid ? 1 : 0;
    active[i] = a ? 1 : 0;
  }, p.slab != 0);
}

template <int Q>
__global__ void __launch_bounds__(256) build_links_kernel(const uint8_t* __restrict__ active, uint32_t* __restrict__ links, int bx,
                                                          const __grid_constant__ Params p) {
  for_each_cell(p, bx, [&](int x, int y, int z, int i) {
    const Neigh nb(p, x, y, z);
    const CellFlags<BC_WALLS> c(p, x, y, z, i);
    uint32_t m = active[i] ? 0u : (1u << ((Q - 1) / 2));
    static_for<0, Q>([&](auto A) {
      constexpr int a = decltype(A)::value;
      if constexpr (Dir<Q, a>::s > 0) {
        bool none;
        int dir, cidx;
        long long idx;
        if (p.any_sym && mirror_link<Q, a, -1, BC_WALLS>(p, c, nb, dir, idx, cidx)) {
          none = active[cidx] == 0;  // D:R25: the source is the mirror image
        } else {
          none = c.template leaves_box<Q, a, -1>();
          if (!none) none = active[nb.template cat<Q, a, -1>()] == 0;
        }
        m |= none ? (1u << a) : 0u;
      }
    });
    links[i] = m;
  }, p.slab != 0);  // slab: the halo planes too (import_canonical fills their slots); bits of links that point
                   // beyond a halo plane are meaningless and never used
}

// ---------------------------------------------------------------------------------------
// PostProcessing + Monitor: rho, u fields and the 8 diagnostics.
// Per-thread accumulation over a grid-stride loop, warp shuffles, one partial per block,
// then a single-block final pass in fixed order (deterministic, no floating-point atomics).
constexpr int kDiag = 8;

__device__ __forceinline__ void diag_combine(double (&a)[kDiag], const double (&b)[kDiag]) {
  a[0] += b[0]; a[1] += b[1]; a[2] += b[2]; a[3] += b[3]; a[4] += b[4];
  a[5] = fmax(a[5], b[5]);
  a[6] = fmin(a[6], b[6]);
  a[7] += b[7];
}

__device__ __forceinline__ void block_reduce_diag(double (&acc)[kDiag], double* __restrict__ out) {
  __shared__ double sh[32][kDiag];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = (blockDim.x + 31) >> 5;
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    double o[kDiag];
#pragma unroll
    for (int k = 0; k < kDiag; ++k) o[k] = __shfl_down_sync(0xffffffffu, acc[k], off);
    diag_combine(acc, o);
  }
  if (lane == 0) {
#pragma unroll
    for (int k = 0; k < kDiag; ++k) sh[warp][k] = acc[k];
  }
  __syncthreads();
  if (warp == 0) {
    double v[kDiag] = {0, 0, 0, 0, 0, 0, INFINITY, 0};
    if (lane < nwarp) {
#pragma unroll
      for (int k = 0; k < kDiag; ++k) v[k] = sh[lane][k];
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
      double o[kDiag];
#pragma unroll
      for (int k = 0; k < kDiag; ++k) o[k] = __shfl_down_sync(0xffffffffu, v[k], off);
      diag_combine(v, o);
    }
    if (lane == 0) {
#pragma unroll
      for (int k = 0; k < kDiag; ++k) out[k] = v[k];
    }
  }
}

// The F/2 shift of D:R7 is always applied (adding 0.5*0 is exact), so there is no FORCE variant here.
template <int Q, int EQ, int BC, int MODE, typename ST>
__global__ void __launch_bounds__(256, 2) moments_kernel(const ST* buf, double* __restrict__ rho_out, double* __restrict__ u_out,
                                                      double* __restrict__ partials, int bx, int r0, int r1, const __grid_constant__ Params p) {
  // rows [r0, r1) of the grid (r = y + ny*z): lbm_moments_host sweeps z-chunks so that their copies to the host overlap
  double acc[kDiag] = {0, 0, 0, 0, 0, 0, INFINITY, 0};
  for_each_cell_in_rows(p, bx, r0, r1, [&](int x, int y, int z, int i) {
    const Neigh nb(p, x, y, z);
    const CellFlags<BC> c(p, x, y, z, i);
    if (!c.template active<Q>()) {  // Monitor runs over the fluid nodes; inactive nodes report 0
      if (rho_out) rho_out[i] = 0.0;
      if (u_out) {
        u_out[i] = 0.0;
        plane<1>(u_out, p.N)[i] = 0.0;
        plane<2>(u_out, p.N)[i] = 0.0;
      }
      return;
    }
    double f[Q];
    load_canonical<Q, BC, MODE, ST>(f, buf, p, nb, c);
    double rho, ux, uy, uz;
    moments<Q, EQ, true>(f, p, rho, ux, uy, uz);
    if (rho_out) rho_out[i] = rho;
    if (u_out) {
      u_out[i] = ux;
      plane<1>(u_out, p.N)[i] = uy;
      plane<2>(u_out, p.N)[i] = uz;
    }
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
  });
  if (partials) block_reduce_diag(acc, partials + (long long)blockIdx.x * kDiag);
}

// (a template only so that the definition may live in this header, which several units include)
template <int K = kDiag>
__global__ void __launch_bounds__(256) reduce_final_kernel(const double* __restrict__ partials, int nblocks, double* __restrict__ out) {
  double acc[kDiag] = {0, 0, 0, 0, 0, 0, INFINITY, 0};
  for (int b = threadIdx.x; b < nblocks; b += blockDim.x) {
    double v[kDiag];
#pragma unroll
    for (int k = 0; k < kDiag; ++k) v[k] = partials[(long long)b * kDiag + k];
    diag_combine(acc, v);
  }
  block_reduce_diag(acc, out);
}

// Momentum-exchange force on the solid nodes of `geo` (Eq. 13) for the step just taken:
//   F = sum over fluid nodes x (geo = 0), sum over a with x + e_a a solid node of geo (inside the box):
//       [ f*_a(x, t) + f_abar(x, t + dt) ] e_a
// f_abar(x, t+dt) is the canonical state; the post-collision f*_a(x, t) is still in the storage:
//   A/B                : slot(x, a) of the current buffer
//   AA after even step : slot(x, abar)
//   AA after odd step  : slot(x + e_a, a) if x + e_a is active (a nodal wall node), else slot(x, abar)
// partials[b*8 + 0..2] receive the block sums (slots 3..7 stay neutral).
template <int Q, int MODE, typename ST>
__global__ void __launch_bounds__(256, 2) boundary_force_kernel(const ST* buf, const uint8_t* __restrict__ geo, double* __restrict__ partials, int bx,
                                                             const __grid_constant__ Params p) {
  double acc[kDiag] = {0, 0, 0, 0, 0, 0, INFINITY, 0};
  for_each_cell(p, bx, [&](int x, int y, int z, int i) {
    if (geo[i] != 0) return;
    const Neigh nb(p, x, y, z);
    const CellFlags<BC_GEO> c(p, x, y, z, i);
    uint32_t solid = 0u;  // bit a: x + e_a is a solid node of geo
    static_for<0, Q>([&](auto A) {
      constexpr int a = decltype(A)::value;
      if constexpr (Dir<Q, a>::s > 0) {
        if (!c.template leaves_box<Q, a, 1>()) solid |= (geo[nb.template cat<Q, a, 1>()] != 0) ? (1u << a) : 0u;
      }
    });
    if (solid == 0u) return;
    double f[Q];
    load_canonical<Q, BC_GEO, MODE, ST>(f, buf, p, nb, c);
    static_for<0, Q>([&](auto A) {
      constexpr int a = decltype(A)::value;
      constexpr int o = Dir<Q, a>::opp;
      using D = Dir<Q, a>;
      if constexpr (D::s > 0) {
        if ((solid >> a) & 1u) {
          double post;
          if constexpr (MODE == MODE_PULL) {
            post = ld_pop_rw<ST, Q, a>(plane<a>(buf, p.ds), nb.ic);
          } else if constexpr (MODE == MODE_PULL_SWAP) {
            post = ld_pop_rw<ST, Q, a>(plane<o>(buf, p.ds), nb.ic);
          } else {
            if (c.template leaves<Q, a, 1>()) post = ld_pop_rw<ST, Q, a>(plane<o>(buf, p.ds), nb.ic);
            else post = ld_pop_rw<ST, Q, a>(plane<a>(buf, p.ds), nb.template at<Q, a, 1>());
          }
          const double term = post + f[o];
          if constexpr (D::ex != 0) acc[0] += D::ex * term;
          if constexpr (D::ey != 0) acc[1] += D::ey * term;
          if constexpr (D::ez != 0) acc[2] += D::ez * term;
        }
      }
    });
  });
  block_reduce_diag(acc, partials + (long long)blockIdx.x * kDiag);
}

}  // namespace lbm
