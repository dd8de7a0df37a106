// lbm_inst.cu — kernel instantiations.  Compiled once per (LBM_Q, LBM_PART) by build.py, in parallel:
//   LBM_Q    9 | 19 | 27
//   LBM_PART 0 A/B step   1 AA even step   2 AA odd step   3 export/import/init/geometry   4 moments/force
//            5 A/B step of a z-slab (fused halo push)   6 A/B step with SYMMETRY faces (link mask + mirror links)
//            7 A/B step of a z-slab with SYMMETRY faces   8 persistent A/B kernel (all steps of a call in one launch)
//            9 persistent in-place AA kernel   10 A/B, two steps per pass (stream_collide_ab2)
// Each unit defines the launch_* specialisations of lbm_launch.cuh for its lattice.
#include <atomic>

#include "lbm_launch.cuh"

#ifndef LBM_Q
#error "compile with -DLBM_Q=9|19|27 -DLBM_PART=0..10"
#endif

namespace lbm {
namespace {

// Runtime flags -> compile-time variant: f(IC<EQ>, IC<BC>, IC<FORCE>, storage type tag).
template <typename F>
void dispatch_storage(const Ctx& c, F&& f) {
  if (c.f32) f(float{});
  else f(double{});
}
template <typename F>
void dispatch_bc(const Ctx& c, F&& f) {
  switch (c.bc) {
    case BC_PERIODIC: f(IC<BC_PERIODIC>{}); break;
    case BC_WALLS: f(IC<BC_WALLS>{}); break;
    default: f(IC<BC_GEO>{}); break;
  }
}
template <typename F>
void dispatch_eq(const Ctx& c, F&& f) {
  if (c.eq) f(IC<EQ_INCOMP>{});
  else f(IC<EQ_STANDARD>{});
}
template <typename F>
void dispatch_force(const Ctx& c, F&& f) {
  if (c.forced) f(IC<1>{});
  else f(IC<0>{});
}
template <typename F>
void dispatch_step(const Ctx& c, F&& f) {
  dispatch_eq(c, [&](auto eq) {
    dispatch_bc(c, [&](auto bc) {
      dispatch_force(c, [&](auto force) { dispatch_storage(c, [&](auto st) { f(eq, bc, force, st); }); });
    });
  });
}
template <typename F>
void dispatch_mode(int mode, F&& f) {
  switch (mode) {
    case MODE_NATURAL: f(IC<MODE_NATURAL>{}); break;
    case MODE_PULL: f(IC<MODE_PULL>{}); break;
    default: f(IC<MODE_PULL_SWAP>{}); break;
  }
}

}  // namespace

constexpr int Q_ = LBM_Q;

#if LBM_PART == 8 || LBM_PART == 9
namespace {
// cooperative launch of one instantiation with as many layers of blocks along z (then along y) as can be resident at
// once (the kernel strides over the rest); false = not even one layer fits, or no cooperative launch: use the per-step kernels
template <typename K>
bool launch_cooperative(K kernel, const Ctx& c, void** args, bool allow_stride) {
  int per_sm = 0, dev = 0, sms = 0, coop = 0;
  const int threads = c.block.x * c.block.y * c.block.z;
  if (cudaGetDevice(&dev) != cudaSuccess) return false;
  cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (!coop || cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, 0) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  const long long capacity = (long long)per_sm * sms;
  dim3 grid = c.grid;
  if ((long long)grid.x > capacity) return false;
  if ((long long)grid.x * grid.y * grid.z > capacity) {
    if (!allow_stride) return false;
    const long long zl = capacity / ((long long)grid.x * grid.y);
    if (zl >= 1) {
      grid.z = (unsigned)zl;
    } else {
      grid.z = 1;
      grid.y = (unsigned)(capacity / grid.x);
    }
  }
  if (cudaLaunchCooperativeKernel((const void*)kernel, grid, c.block, args, 0, c.stream) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  return true;
}
}  // namespace
#endif

#if LBM_PART == 0
template <>
void launch_step_ab<Q_>(const Ctx& c, const void* src, void* dst) {
  if (c.p.any_sym) return launch_step_ab_sym<Q_>(c, src, dst);  // part 6
  if constexpr (Q_ != 27) if (c.f32 && c.bc != BC_GEO && c.p.nx % 2 == 0 && !c.p.slab) {
    // fp32 storage: two cells per thread, one row per block (stream_collide_ab_f32x2)
    int bx = 32;
    while (bx < kF32x2Threads && 2 * bx < c.p.nx) bx *= 2;
    const dim3 block(bx, 1, 1), grid((c.p.nx / 2 + bx - 1) / bx, c.p.ny, c.p.nz);
    dispatch_eq(c, [&](auto eq) {
      dispatch_force(c, [&](auto force) {
        if (c.bc == BC_WALLS)
          stream_collide_ab_f32x2<Q_, decltype(eq)::value, BC_WALLS, decltype(force)::value != 0><<<grid, block, 0, c.stream>>>((const float*)src, (float*)dst, c.p);
        else
          stream_collide_ab_f32x2<Q_, decltype(eq)::value, BC_PERIODIC, decltype(force)::value != 0><<<grid, block, 0, c.stream>>>((const float*)src, (float*)dst, c.p);
      });
    });
    return;
  }
  dispatch_step(c, [&](auto eq, auto bc, auto force, auto st) {
    using ST = decltype(st);
    stream_collide_ab<Q_, decltype(eq)::value, decltype(bc)::value, decltype(force)::value != 0, ST>
        <<<c.grid, c.block, 0, c.stream>>>((const ST*)src, (ST*)dst, c.p);
  });
}
#elif LBM_PART == 6
template <>
void launch_step_ab_sym<Q_>(const Ctx& c, const void* src, void* dst) {
  // D:R25: handles with SYMMETRY faces always carry the link mask (BC_GEO)
  dispatch_eq(c, [&](auto eq) {
    dispatch_force(c, [&](auto force) {
      dispatch_storage(c, [&](auto st) {
        using ST = decltype(st);
        stream_collide_ab<Q_, decltype(eq)::value, BC_GEO, decltype(force)::value != 0, ST, false, true>
            <<<c.grid, c.block, 0, c.stream>>>((const ST*)src, (ST*)dst, c.p);
      });
    });
  });
}
#elif LBM_PART == 8
namespace {
template <typename K>
bool launch_persistent(K kernel, const Ctx& c, void* b0, void* b1, int nsteps) {
  Params p = c.p;
  void* args[] = {&b0, &b1, &nsteps, &p};
  // With inlet / outlet on the x faces single lanes run long ("One lane per row"): a grid that has to
  // stride then waits for them at every barrier (512^2 D2Q9 channel-cylinder x0.95, 128x32x32 sphere case x0.81), so
  // such grids must be resident in one pass; without open faces striding pays (64^3 cavity x1.14, 48^3 D3Q27 channel x1.23).
  return launch_cooperative(kernel, c, args, !(c.p.open[0] || c.p.open[1]));
}
}  // namespace

template <>
bool launch_step_ab_persistent<Q_>(const Ctx& c, void* b0, void* b1, int nsteps) {
  // fp64 storage only: grids this small have no use for the fp32-storage variant, and it would double the build
  if (c.f32) return false;
  bool ok = false;
  dispatch_eq(c, [&](auto eq) {
    dispatch_force(c, [&](auto force) {
      if (c.p.any_sym) {
        ok = launch_persistent(stream_collide_ab_persistent<Q_, decltype(eq)::value, BC_GEO, decltype(force)::value != 0, double, true>, c, b0, b1, nsteps);
      } else {
        dispatch_bc(c, [&](auto bc) {
          ok = launch_persistent(stream_collide_ab_persistent<Q_, decltype(eq)::value, decltype(bc)::value, decltype(force)::value != 0, double, false>, c, b0, b1, nsteps);
        });
      }
    });
  });
  return ok;
}
#elif LBM_PART == 9
template <>
bool launch_step_aa_persistent<Q_>(const Ctx& c, void* buf, int nsteps, int phase) {
  if (c.f32) return false;  // fp64 storage only, as above
  bool ok = false;
  dispatch_eq(c, [&](auto eq) {
    dispatch_bc(c, [&](auto bc) {
      dispatch_force(c, [&](auto force) {
        Params p = c.p;
        void* args[] = {&buf, &nsteps, &phase, &p};
        // in place: only grids resident in one pass (striding is neutral at best: 1200 x 1100 D2Q9 x0.92, 80^3 x0.99)
        ok = launch_cooperative(stream_collide_aa_persistent<Q_, decltype(eq)::value, decltype(bc)::value, decltype(force)::value != 0, double>, c, args, false);
      });
    });
  });
  return ok;
}
#elif LBM_PART == 5
template <>
void launch_step_ab_slab<Q_>(const Ctx& c, const void* src, void* dst) {
  if (c.p.any_sym) return launch_step_ab_slab_sym<Q_>(c, src, dst);  // part 7
  dispatch_step(c, [&](auto eq, auto bc, auto force, auto st) {
    using ST = decltype(st);
    stream_collide_ab<Q_, decltype(eq)::value, decltype(bc)::value, decltype(force)::value != 0, ST, true>
        <<<c.grid, c.block, 0, c.stream>>>((const ST*)src, (ST*)dst, c.p);
  });
}
#elif LBM_PART == 7
template <>
void launch_step_ab_slab_sym<Q_>(const Ctx& c, const void* src, void* dst) {
  dispatch_eq(c, [&](auto eq) {
    dispatch_force(c, [&](auto force) {
      dispatch_storage(c, [&](auto st) {
        using ST = decltype(st);
        stream_collide_ab<Q_, decltype(eq)::value, BC_GEO, decltype(force)::value != 0, ST, true, true>
            <<<c.grid, c.block, 0, c.stream>>>((const ST*)src, (ST*)dst, c.p);
      });
    });
  });
}
#elif LBM_PART == 10
namespace {
// tile, blocks per SM, barrier scheme and prefetch of stream_collide_ab2 per lattice (measured; comment in launch_step_ab2)
template <int Q, int BCV>
struct Ab2Pick {
  static constexpr int TX = (Q == 19) ? 32 : 16, TY = 8, MINB = (Q == 19) ? 1 : 2;
  static constexpr bool ONEBAR = (Q == 19), PREFETCH = (Q == 19);
  using T = Ab2Tile<Q, TX, TY, ONEBAR, (BCV == BC_WALLS) && ONEBAR>;
};
}  // namespace

template <>
bool launch_step_ab2<Q_>(const Ctx& c, const void* src, void* dst, bool always) {
  // fp64 storage, no link mask, whole box.  D3Q19: 32 x 8 tiles, one block of 352 threads per SM, one barrier per plane,
  // register prefetch of the next plane (512^3 periodic: 22.5 -> 33.6 GLUPS in one launch; z walls + forcing 22.5 -> 26.7).
  // D3Q27 keeps 27 populations of three planes: 16 x 8 tiles, two blocks of 192 threads per SM, two barriers per plane
  // (fewer shared-memory slots), no prefetch (400^3 periodic: 15.8 -> 21.0 GLUPS, with forcing 18.7).  Walls through the
  // stage-2 select and the extra slots ate that gain (15.2-16.3 against 15.5, six tile shapes), so D3Q27 takes walls
  // only as ghost planes in z (x, y periodic: 512^3 channel with forcing 15.7 -> 17.1 GLUPS).  D2Q9 has no z to march along.
  if constexpr (Q_ == 9) {
    return false;
  } else {
    constexpr int TX = Ab2Pick<Q_, 0>::TX, TY = Ab2Pick<Q_, 0>::TY;
    // D3Q27 with walls: z walls only (x and y periodic), which the two-barrier kernel resolves through ghost planes
    const bool q27_ok = c.bc == BC_PERIODIC || (c.bc == BC_WALLS && !c.p.wall[0] && !c.p.wall[1] && !c.p.wall[2] && !c.p.wall[3]);
    if (c.bc == BC_GEO || (Q_ == 27 && !q27_ok) || c.f32 || c.p.slab || c.p.nx < TX || c.p.ny < TY || c.p.nz < 4) return false;
    bool ok = true;
    dispatch_eq(c, [&](auto eq) {
      dispatch_force(c, [&](auto force) {
        dispatch_bc(c, [&](auto bc) {
          if constexpr (decltype(bc)::value == BC_GEO) {
            ok = false;
          } else {
            using P = Ab2Pick<Q_, decltype(bc)::value>;
            using T = typename P::T;
            auto kernel = stream_collide_ab2<Q_, decltype(eq)::value, decltype(bc)::value, decltype(force)::value != 0, P::TX, P::TY, P::MINB, P::ONEBAR, P::PREFETCH>;
            // per device: blocks of this instantiation resident at once (0 = not asked yet, or to be asked again).  Atomic:
            // handles driven from several host threads share it (they would all store the same value).
            static std::atomic<int> resident_on[64];
            int dev = 0;
            if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) {
              cudaGetLastError();
              ok = false;
              return;
            }
            if (resident_on[dev].load(std::memory_order_relaxed) == 0) {
              int sms = 0, per_sm = 0;
              if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)T::SMEM_BYTES) != cudaSuccess ||
                  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
                  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, T::THREADS, T::SMEM_BYTES) != cudaSuccess || per_sm < 1) {
                cudaGetLastError();
                resident_on[dev].store(-1, std::memory_order_relaxed);
              } else {
                resident_on[dev].store(per_sm * sms, std::memory_order_relaxed);
              }
            }
            const int resident = resident_on[dev].load(std::memory_order_relaxed);
            if (resident < 0) {
              ok = false;
              return;
            }
            // z-chunks.  Every chunk runs stage 1 on two planes more than it stores (stage 1 is about 55 % of a plane's
            // work: a chunk of zc planes costs zc + 1.1), and the last wave of blocks leaves SMs idle unless the block count
            // is close to a multiple of what the device holds: take the chunk count that loses least to both.
            const long long tiles = (long long)((c.p.nx + TX - 1) / TX) * ((c.p.ny + TY - 1) / TY);
            int zchunk = c.p.nz;
            double best = 0.0;
            for (int n = 1; n <= 64 && n * 8 <= c.p.nz; ++n) {
              const int zc = (c.p.nz + n - 1) / n;
              const long long blocks = tiles * ((c.p.nz + zc - 1) / zc);
              const double waves = (double)blocks / resident;
              // (+ 0.25 wave: blocks do not all take the same time, so a nearly full last wave still costs)
              const double eff = waves / ((double)((blocks + resident - 1) / resident) + 0.25) * zc / (zc + 1.1);
              if (eff > best * 1.002) {  // (ties go to fewer, longer chunks)
                best = eff;
                zchunk = zc;
              }
            }
            const dim3 grid((c.p.nx + TX - 1) / TX, (c.p.ny + TY - 1) / TY, (c.p.nz + zchunk - 1) / zchunk);
            // Too few blocks: the only wave or two leave SMs idle and ragged tiles waste lanes.  Measured, one-step /
            // two-step GLUPS: 72^3 (135 blocks) 18.1 / 19.2 at best, 80^3 (300 blocks of 8 planes) 18.8 / 22.7, 88^3 19.6 / 24.7,
            // 96^3 20.5 / 28.6, 128^3 21.8 / 29.1.  Below 1.4 waves the one-step kernel takes the steps.
            if (!always && 10LL * grid.x * grid.y * grid.z < 14LL * resident) {
              ok = false;
              return;
            }
            kernel<<<grid, T::THREADS, T::SMEM_BYTES, c.stream>>>((const double*)src, (double*)dst, zchunk, c.p);
            // A launch that was refused (after cudaDeviceReset or in a new context the opt-in shared-memory size above is
            // gone while the cache still says "ready") must not count as two steps taken: report "not launched" so that
            // lbm_step leaves cur / time alone and takes the steps with the one-step kernel, and ask again next time.
            if (cudaPeekAtLastError() != cudaSuccess) {
              cudaGetLastError();
              resident_on[dev].store(0, std::memory_order_relaxed);
              ok = false;
              return;
            }
          }
        });
      });
    });
    return ok;
  }
}
#elif LBM_PART == 1
template <>
void launch_step_aa_even<Q_>(const Ctx& c, void* buf) {
  dispatch_step(c, [&](auto eq, auto bc, auto force, auto st) {
    using ST = decltype(st);
    stream_collide_aa_even<Q_, decltype(eq)::value, decltype(bc)::value, decltype(force)::value != 0, ST>
        <<<c.grid, c.block, 0, c.stream>>>((ST*)buf, c.p);
  });
}
#elif LBM_PART == 2
template <>
void launch_step_aa_odd<Q_>(const Ctx& c, void* buf) {
  if (c.bc != BC_GEO) {
    // one grid row per block (stream_collide_aa_odd_row): the row bases of all Q slots are block-uniform
    int bx = 32;
    while (bx < 256 && bx < c.p.nx) bx *= 2;
    const dim3 block(bx, 1, 1), grid((c.p.nx + bx - 1) / bx, c.p.ny, c.p.nz);
    dispatch_eq(c, [&](auto eq) {
      dispatch_force(c, [&](auto force) {
        dispatch_storage(c, [&](auto st) {
          using ST = decltype(st);
          if (c.bc == BC_WALLS)
            stream_collide_aa_odd_row<Q_, decltype(eq)::value, BC_WALLS, decltype(force)::value != 0, ST><<<grid, block, 0, c.stream>>>((ST*)buf, c.p);
          else
            stream_collide_aa_odd_row<Q_, decltype(eq)::value, BC_PERIODIC, decltype(force)::value != 0, ST><<<grid, block, 0, c.stream>>>((ST*)buf, c.p);
        });
      });
    });
    return;
  }
  dispatch_eq(c, [&](auto eq) {
    dispatch_force(c, [&](auto force) {
      dispatch_storage(c, [&](auto st) {
        using ST = decltype(st);
        stream_collide_aa_odd<Q_, decltype(eq)::value, BC_GEO, decltype(force)::value != 0, ST><<<c.grid, c.block, 0, c.stream>>>((ST*)buf, c.p);
      });
    });
  });
}
#elif LBM_PART == 3
template <>
void launch_export<Q_>(const Ctx& c, int mode, const void* buf, double* out) {
  dispatch_mode(mode, [&](auto m) {
    dispatch_bc(c, [&](auto bc) {
      dispatch_storage(c, [&](auto st) {
        using ST = decltype(st);
        export_canonical<Q_, decltype(bc)::value, decltype(m)::value, ST><<<c.flat_grid, 256, 0, c.stream>>>((const ST*)buf, out, c.fbx, c.p);
      });
    });
  });
}
template <>
void launch_import<Q_>(const Ctx& c, int mode, const double* in, void* buf) {
  dispatch_bc(c, [&](auto bc) {
    dispatch_storage(c, [&](auto st) {
      using ST = decltype(st);
      if (mode == MODE_PULL)
        import_canonical<Q_, decltype(bc)::value, MODE_PULL, ST><<<c.flat_grid, 256, 0, c.stream>>>(in, (ST*)buf, c.fbx, c.p);
      else
        import_canonical<Q_, decltype(bc)::value, MODE_NATURAL, ST><<<c.flat_grid, 256, 0, c.stream>>>(in, (ST*)buf, c.fbx, c.p);
    });
  });
}
template <>
void launch_init<Q_>(const Ctx& c, int mode, const double* rho, const double* u, void* buf, int r0, int r1, int grid) {
  dispatch_eq(c, [&](auto eq) {
    dispatch_bc(c, [&](auto bc) {
      dispatch_storage(c, [&](auto st) {
        using ST = decltype(st);
        if (mode == MODE_PULL)
          init_equilibrium_kernel<Q_, decltype(eq)::value, decltype(bc)::value, MODE_PULL, ST><<<grid, 256, 0, c.stream>>>(rho, u, (ST*)buf, c.fbx, r0, r1, c.p);
        else
          init_equilibrium_kernel<Q_, decltype(eq)::value, decltype(bc)::value, MODE_NATURAL, ST><<<grid, 256, 0, c.stream>>>(rho, u, (ST*)buf, c.fbx, r0, r1, c.p);
      });
    });
  });
}
template <>
void launch_geometry<Q_>(const Ctx& c, const uint8_t* geo_in, uint8_t* geo, uint8_t* active, uint32_t* links, int nodal) {
  classify_nodes_kernel<Q_><<<c.flat_grid, 256, 0, c.stream>>>(geo_in, geo, active, nodal, c.fbx, c.p);
  build_links_kernel<Q_><<<c.flat_grid, 256, 0, c.stream>>>(active, links, c.fbx, c.p);
}
#elif LBM_PART == 4
template <>
void launch_moments<Q_>(const Ctx& c, int mode, const void* buf, double* rho, double* u, double* partials, int r0, int r1, int grid) {
  dispatch_mode(mode, [&](auto m) {
    dispatch_eq(c, [&](auto eq) {
      dispatch_bc(c, [&](auto bc) {
        dispatch_storage(c, [&](auto st) {
          using ST = decltype(st);
          moments_kernel<Q_, decltype(eq)::value, decltype(bc)::value, decltype(m)::value, ST>
              <<<grid, 256, 0, c.stream>>>((const ST*)buf, rho, u, partials, c.fbx, r0, r1, c.p);
        });
      });
    });
  });
}
template <>
void launch_boundary_force<Q_>(const Ctx& c, int mode, const void* buf, const uint8_t* geo, double* partials) {
  dispatch_mode(mode, [&](auto m) {
    dispatch_storage(c, [&](auto st) {
      using ST = decltype(st);
      boundary_force_kernel<Q_, decltype(m)::value, ST><<<c.flat_grid, 256, 0, c.stream>>>((const ST*)buf, geo, partials, c.fbx, c.p);
    });
  });
}
#else
#error "LBM_PART must be 0..10"
#endif

}  // namespace lbm
