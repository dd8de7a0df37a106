// lbm_launch.cuh — host-side launch interface between the C ABI (lbm_abi.cu) and the kernel
// instantiation units (lbm_inst.cu compiled once per lattice and part, in parallel).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "lbm_kernels.cuh"

namespace lbm {

// Everything a launcher needs to pick the compile-time variant and the launch shape.
struct Ctx {
  int eq;        // EQ_STANDARD / EQ_INCOMP
  int bc;        // BC_PERIODIC / BC_WALLS / BC_GEO
  int forced;    // body force != 0
  int f32;       // populations stored as float
  dim3 grid, block;  // fused stream-collide kernels
  int flat_grid, fbx;  // row-wise sweeps off the per-step path (for_each_cell)
  cudaStream_t stream;
  Params p;
};

// One explicit specialisation of each per lattice Q in {9, 19, 27} (lbm_inst.cu).
template <int Q> void launch_step_ab(const Ctx& c, const void* src, void* dst);
template <int Q> void launch_step_ab_slab(const Ctx& c, const void* src, void* dst);
template <int Q> void launch_step_ab_sym(const Ctx& c, const void* src, void* dst);
template <int Q> void launch_step_ab_slab_sym(const Ctx& c, const void* src, void* dst);
// all nsteps in one cooperative launch (b0 = current buffer); false = the grid does not fit the device at once
template <int Q> bool launch_step_ab_persistent(const Ctx& c, void* b0, void* b1, int nsteps);
template <int Q> bool launch_step_aa_persistent(const Ctx& c, void* buf, int nsteps, int phase);
// TWO steps in one pass through HBM (stream_collide_ab2); false = this handle has no such kernel, or — unless `always` —
// the grid gives it too few blocks to pay (use two single steps)
template <int Q> bool launch_step_ab2(const Ctx& c, const void* src, void* dst, bool always);
template <int Q> void launch_step_aa_even(const Ctx& c, void* buf);
template <int Q> void launch_step_aa_odd(const Ctx& c, void* buf);
template <int Q> void launch_export(const Ctx& c, int mode, const void* buf, double* out);
template <int Q> void launch_import(const Ctx& c, int mode, const double* in, void* buf);
// rows [r0, r1) of the grid (r = y + ny*z) on `grid` blocks: the host entry points work through z-chunks
template <int Q> void launch_init(const Ctx& c, int mode, const double* rho, const double* u, void* buf, int r0, int r1, int grid);
template <int Q> void launch_moments(const Ctx& c, int mode, const void* buf, double* rho, double* u, double* partials, int r0, int r1, int grid);
template <int Q> void launch_geometry(const Ctx& c, const uint8_t* geo_in, uint8_t* geo, uint8_t* active, uint32_t* links, int nodal);
template <int Q> void launch_boundary_force(const Ctx& c, int mode, const void* buf, const uint8_t* geo, double* partials);

}  // namespace lbm
