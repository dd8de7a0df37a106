/* include/lbm.h — C ABI of the B200-native lattice-Boltzmann hot path.
 *
 * The operation: the per-time-step fused streaming + BGK collision update of the
 * D3Q19 / D3Q27 (and D2Q9) populations of IMEXLBM (arXiv 2201.11330) on an nx*ny*nz box, fp64.
 * "P:n" = line n of the paper text; "D:Rk" = reading k in DESIGN.md §2.
 *
 *   collision    f*_a = f_a - omega (f_a - feq_a)                 P:61-63, Eq. 6
 *   propagation  f_a(x, t) = f*_a(x - e_a, t - 1)                 P:65-69, Eq. 7
 *   moments      rho = sum_a f_a (= p/c_s^2), u = sum_a e_a f_a / rho      P:71-78, Eq. 8-9
 *   equilibrium  Eq. 2 or the incompressible Eq. 5 (code form P:375)
 *   walls        f_a = f_abar, abar = Q-1-a                        P:84-88 Eq. 10
 *
 * Conventions
 *   - c_s^2 = 1/3, dx = dt = 1.  Linear cell index i = x + nx*(y + ny*z),
 *     N = nx*ny*nz.  Field layouts (structure of arrays, x fastest):
 *       rho[i]   (N doubles)      u[c*N + i], c = 0,1,2  (3N doubles)      f[a*N + i]  (Q*N doubles)
 *   - Velocity numbering (D:R4): lexicographic over (e_x, e_y, e_z), each -1,0,+1, e_x
 *     outermost; D3Q19 omits the 8 corner vectors.  opposite(a) = Q-1-a, rest = (Q-1)/2.
 *     lbm_lattice() returns the table.
 *   - `tau` is the lattice relaxation time with omega = 1/tau and nu = (tau - 1/2)/3
 *     (D:R1: tau = tau_paper/dt + 1/2 of P:61-63).
 *   - "Populations" at this interface are always the canonical state (D:R15): the
 *     pre-collision f(x, t) after `Propagation`, whatever the library stores internally.
 *   - Pointers are DEVICE pointers (cudaMalloc'ed / torch CUDA tensors, 8-byte aligned) owned
 *     by the caller unless a parameter says "host"; the *_host entry points take HOST
 *     pointers (pinned memory recommended) and do the host<->device copies themselves on the
 *     handle's stream.  The library owns the population buffers from lbm_create to lbm_destroy.
 *   - Everything is enqueued on the handle's CUDA stream and is asynchronous unless stated.
 *   - Errors: functions return 0 on success or a negative LBM_E* code; lbm_create returns
 *     NULL.  lbm_last_error() gives the message of the calling thread's last failure.  No
 *     exception or abort crosses this boundary; a failed call leaves the state unchanged.
 *   - A handle is not thread-safe; use one thread per handle at a time.
 */
#ifndef LBM_B200_H
#define LBM_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lbm_handle_s* lbm_handle; /* opaque, owned by the library */

/* `lattice` argument of lbm_create: velocity set | equilibrium | storage scheme | storage type */
enum {
  LBM_D2Q9 = 9,             /* low byte: number of velocities.  D2Q9 exactly as printed in      */
  LBM_D3Q19 = 19,           /* Eq. 3-4, e_z = 0: every z-plane is an independent 2-D     */
  LBM_D3Q27 = 27,           /* domain (use nz = 1 for one)                                      */
  LBM_EQ_STANDARD = 0,      /* Eq. 2, weakly compressible (default)                            */
  LBM_EQ_INCOMP = 1 << 8,   /* Eq. 5, incompressible model with rho0 = 1               */
  LBM_SCHEME_AUTO = 0,      /* LBM_SCHEME_AB, except LBM_SCHEME_AA where one buffer fits the L2 and two do not */
  LBM_SCHEME_AB = 1 << 12,  /* two buffers, pull ("stream on read")                            */
  LBM_SCHEME_AA = 2 << 12,  /* one buffer, in-place AA pattern.  Measured cost against LBM_SCHEME_AB on one B200 (one step
                               per pass, MLUPS, AA / AB): 512^3 D3Q19 periodic 22 470 / 22 520; 256^3 D3Q19 cavity
                               22 420 / 22 560; 512^3 D3Q27 channel with forcing 14 760 / 15 900; with a solid mask the
                               odd phase keeps Q addresses live (124-128 registers) and runs at 0.75-0.9 of AB.  AB also
                               takes two steps per pass for D3Q19 fp64 (lbm_set_two_step: 31 400), AA does not.         */
  LBM_STORE_F64 = 0,        /* populations stored as fp64 (default)                            */
  LBM_STORE_F32 = 1 << 16,  /* populations stored as fp32 (f - t_a), arithmetic in fp64        */
  LBM_LAYOUT_ROWS = 0,      /* internal buffers f[z][y][a][x]: the Q rows of a grid row adjacent (default, faster);
                               a grid with Q*nx*ny >= 2^31 (e.g. D2Q9 16384^2) is stored as LBM_LAYOUT_SOA instead,
                               because in-plane offsets are 32-bit — same results bit for bit                    */
  LBM_LAYOUT_SOA = 1 << 20  /* internal buffers f[a][z][y][x] (for measurements; also accepted on z-slab handles,
                               all connected slabs must then use it)                                            */
};

enum { LBM_FACE_PERIODIC = 0, LBM_FACE_BOUNCE = 1, LBM_FACE_MOVING = 2, LBM_FACE_PRESSURE = 3, LBM_FACE_SYMMETRY = 4 };

/* Wall model of lbm_set_geometry (D:R3, D:R16, D:R17). */
enum {
  LBM_WALL_HALFWAY = 0, /* link-wise bounce-back, wall half a link beyond the last fluid node (default) */
  LBM_WALL_NODAL = 1    /* the paper's modified nodal bounce-back (Eq. 10): wall ON the nodes  */
};

enum {
  LBM_OK = 0,
  LBM_EINVAL = -1,      /* invalid argument                                                     */
  LBM_ENOMEM = -2,      /* out of device memory                                                 */
  LBM_ECUDA = -3,       /* CUDA runtime error (message in lbm_last_error)                       */
  LBM_EUNSUPPORTED = -4 /* valid but unsupported combination                                    */
};

/* Boundary description (D:R3, D:R6, D:R7).  Faces in the order x-, x+, y-, y+, z-, z+.
 * LBM_FACE_PERIODIC must be set on both faces of an axis or on neither.  BOUNCE = halfway
 * bounce-back wall at rest, half a cell outside the first/last node.  MOVING = the same wall
 * moving with face_u (Ladd): a wall link a gains 6 t_a rho_w (e_a . u_w); at edges a MOVING face
 * takes precedence over BOUNCE, and among MOVING faces the highest face index wins.
 * Open boundaries (D:R22; the paper names a parabolic inlet and an outflow, without formulae):
 *   inlet  = MOVING with a per-cell wall velocity (lbm_set_face_velocity): velocity bounce-back;
 *   outlet = PRESSURE: anti-bounce-back at a prescribed density rho_f (lbm_set_face_density, default 1):
 *            f_a(x,t+1) = -f*_abar(x,t) + 2 feq+_a(rho_f, u(x,t)), feq+ = the part of Eq. 2 / Eq. 5 even in e_a
 *            (Eq. 2: t_a rho_f (1 + 4.5 (e_a.u)^2 - 1.5 u.u); Eq. 5: t_a (rho_f + rho0 (4.5 (e_a.u)^2 - 1.5 u.u))).
 *   A link that leaves through several non-periodic faces: MOVING > BOUNCE > PRESSURE (highest index within a kind).
 * SYMMETRY (D:R25; "the left and right boundaries are symmetric"): a mirror plane half a link beyond the last
 *   node (specular reflection, free slip).  A link that leaves through SYMMETRY faces only connects the node with the
 *   mirror image: f_a(x,t+1) = f*_a'(x', t), x' = x - e_a on the axes not crossed, a' = e_a with the crossed components
 *   negated; if x' is not an active node the link is a wall link.  Together with a face of another kind, that kind
 *   decides.  Handles with a SYMMETRY face always use the link mask of lbm_set_geometry (+4 B per node and step) and
 *   need LBM_SCHEME_AB (LBM_EUNSUPPORTED otherwise).
 * Under LBM_WALL_NODAL (D:R24) the MOVING / PRESSURE / SYMMETRY faces keep these link-wise rules; Eq. 10 acts on the
 *   wall links only (BOUNCE faces and solid nodes). */
typedef struct {
  int32_t face_kind[6];
  double face_u[6][3]; /* read only where face_kind == LBM_FACE_MOVING                          */
  double force[3];     /* uniform body-force density F (Guo forcing); all zero = no forcing     */
  void* stream;        /* cudaStream_t to run on (NULL = legacy default stream); caller-owned   */
} lbm_bc_t;

/* Create a solver on the current CUDA device.  nx >= 1, 1 <= ny, nz <= 65535, nx*ny*nz < 2^31 (LBM_EUNSUPPORTED
 * beyond: cell indices are 32-bit); tau > 0.5; bc may be NULL
 * (all periodic, no force, default stream).  Allocates the population buffers (Q*N doubles,
 * twice for LBM_SCHEME_AB).  Populations are undefined until lbm_init_equilibrium or
 * lbm_set_populations.  Returns NULL on failure. */
lbm_handle lbm_create(int nx, int ny, int nz, int lattice, double tau, const lbm_bc_t* bc);

/* Free all device memory of the handle (synchronises its stream).  NULL is a no-op. */
void lbm_destroy(lbm_handle h);

/* SetGeometry (`geo` P:210) and the wall model.  geo: N bytes (DEVICE pointer), non-zero =
 * solid node, or NULL = no solid nodes.  Call before lbm_init_equilibrium / lbm_set_populations.
 *   Active nodes (D:R16): HALFWAY: the fluid nodes (geo = 0).  NODAL: also every solid node with
 *   a fluid node among its lattice neighbours (the wall nodes, which collide "like in the fluid
 *   bulk"); with geo = NULL the first / last planes of BOUNCE faces are the wall nodes.
 *   Only active nodes are updated; inactive nodes report 0 in every output and are excluded
 *   from the diagnostics.  A link whose upstream node x - e_a is not active (solid, or beyond a
 *   non-periodic face) is resolved as
 *     HALFWAY: f_a(x, t+1) = f*_abar(x, t)                  (+ the Ladd term through a MOVING face)
 *     NODAL  : f_a(x, t+1) = f_abar(x, t+1) (Eq. 10: the value that has just arrived along abar)
 *              if x + e_a is active, else f*_abar(x, t) (D:R17: links inside the wall)
 * One 32-bit link mask per node is built here and read by the step kernel (+4 B per node and
 * step); (NULL, LBM_WALL_HALFWAY) returns to the mask-free analytic box.  Synchronises the stream. */
int lbm_set_geometry(lbm_handle h, const uint8_t* geo, int wall_model);
/* Same with a HOST pointer to the N mask bytes. */
int lbm_set_geometry_host(lbm_handle h, const uint8_t* geo_host, int wall_model);

/* D:R22.  Per-cell wall velocity of MOVING face `face` (0..5 = x-,x+,y-,y+,z-,z+): u[c*n + j], c = 0,1,2, n = cells
 * of the face, j runs over the two in-face coordinates with the lower axis fastest (x- / x+: j = y + ny*z; y- / y+:
 * j = x + nx*z; z- / z+: j = x + nx*y).  DEVICE pointer; the library keeps its own copy.  NULL restores the uniform
 * face_u of lbm_create.  On a z-slab handle the profile is that of the WHOLE box face (z = global plane index).
 * LBM_EINVAL if the face is not LBM_FACE_MOVING.  Synchronises the stream. */
int lbm_set_face_velocity(lbm_handle h, int face, const double* u);
/* Same with a HOST pointer. */
int lbm_set_face_velocity_host(lbm_handle h, int face, const double* u_host);

/* D:R22.  Density prescribed on the LBM_FACE_PRESSURE faces: rho6 = HOST pointer to 6 doubles in face order (entries
 * of other faces are ignored).  Default 1.  Takes effect from the next lbm_step. */
int lbm_set_face_density(lbm_handle h, const double* rho6);

/* Momentum-exchange force on the solid nodes of geo (Eq. 13) for the last step taken:
 *   F = sum over fluid nodes x, over a with x + e_a a solid node of geo (inside the box):
 *       [ f*_a(x, t) + f_abar(x, t + 1) ] e_a
 * F: HOST pointer to 3 doubles.  Box-face walls are not part of the body.  Needs a geometry and
 * at least one lbm_step since the populations were last set (else LBM_EINVAL).  Synchronises. */
int lbm_boundary_force(lbm_handle h, double* F);

/* P:82, P:276-278 (InitPDF): f_a(x, 0) = feq_a(rho(x), u(x)); resets the step counter.
 * rho: N doubles or NULL (= 1 everywhere); u: 3N doubles or NULL (= 0).  Device pointers.
 * Under LBM_WALL_NODAL the wall nodes then satisfy Eq. 10 (D:R17). */
int lbm_init_equilibrium(lbm_handle h, const double* rho, const double* u);
/* Same with HOST pointers (pinned memory recommended).  The fields are copied in z-chunks on an internal copy stream
 * and chunk k is initialised on the handle's stream while chunk k+1 is still on the bus.  The call returns when the
 * host arrays have been read in full — they may be freed, reused or overwritten at once (the copy stream is not
 * visible to the caller, so nothing else could tell) — while the initialisation kernels of the last chunks may still
 * be running on the handle's stream.  On a z-slab handle only the own planes of the arrays are read. */
int lbm_init_equilibrium_host(lbm_handle h, const double* rho_host, const double* u_host);

/* Advance nsteps >= 0 time steps: per step and cell, pull-stream (Eq. 7) with wall links
 * (Eq. 10, D:R6), moments (Eq. 8-9), equilibrium (Eq. 2 / 5), BGK relaxation (Eq. 6), forcing
 * (D:R7) and store, all fused: nothing but the populations (and the 4-byte link mask of a geometry) touches HBM.
 * How many kernel launches that takes depends on the handle, and the results are the same bit for bit in every regime:
 *   - persistent: a grid small enough to be resident on the device at once, with its buffers in the L2, takes all
 *     nsteps in ONE cooperative launch (lbm_set_persistent);
 *   - pairs: D3Q19 / D3Q27 fp64 boxes under LBM_SCHEME_AB without a solid mask take TWO steps per launch, each
 *     population read from HBM once and written once per two steps; an odd nsteps ends with one single step
 *     (lbm_set_two_step lists the exact conditions);
 *   - singles: everything else — fp32 storage, LBM_SCHEME_AA, solid masks, SYMMETRY faces, z-slabs, D2Q9 on large
 *     grids — takes one launch per step.
 * lbm_launch_count tells which regime ran.  Asynchronous. */
int lbm_step(lbm_handle h, int nsteps);

/* P:295-304 (PostProcessing, Monitor): moments of the current canonical state.
 * rho: N doubles or NULL; u: 3N doubles or NULL (device).  diagnostics: HOST pointer to 8
 * doubles or NULL: { sum rho, sum rho u_x, sum rho u_y, sum rho u_z, 1/2 sum rho |u|^2,
 * max |u|, min rho, number of cells with non-finite rho or u }; non-finite cells are excluded
 * from the sums; under LBM_EQ_INCOMP "rho u" means rho0 u (D:R5); with forcing u includes the
 * F/2 shift (D:R7).  Synchronises the stream only if diagnostics != NULL. */
int lbm_moments(lbm_handle h, double* rho, double* u, double* diagnostics);
/* Same with HOST output pointers for the fields (either may be NULL); always synchronises.  The moments are
 * computed in z-chunks and chunk k travels to the host while chunk k+1 is computed.  The fields are staged in the idle
 * A/B buffer (in a scratch allocation for LBM_SCHEME_AA and on z-slab handles, whose idle buffer's halo planes belong
 * to the neighbours' next step); on a z-slab handle only the own planes of the host arrays are written. */
int lbm_moments_host(lbm_handle h, double* rho_host, double* u_host, double* diagnostics);

/* The 8 diagnostics of lbm_moments (P:295-304 PostProcessing, P:404-427 Monitor; Eq. 8-9) WITHOUT a handle
 * and WITHOUT allocating anything — for callers that must not call cudaMalloc:
 *   - a process whose device memory is owned outright by a pool of its own (torch's caching allocator, a solver that
 *     sizes its arrays to the card): an allocation made behind the pool's back fails, or takes the room the next
 *     time step needs;
 *   - a monitor inside a running time loop: cudaMalloc / cudaFree synchronise the whole device and would stall the
 *     other streams of the loop;
 *   - code that only holds a pointer to populations somebody else owns (a checkpoint, another solver's arrays) and
 *     has no handle — lbm_create allocates.
 * lbm_moments keeps the per-block records of its two-pass reduction in memory lbm_create allocated; this entry point
 * runs the same reduction (same per-cell arithmetic, same non-finite rule, same 8 outputs) with the records in a
 * fixed 2 MiB `static __device__` array inside the library.  It calls no cudaMalloc, cudaFree or allocating routine.
 *   f           DEVICE, Q*ncells doubles, canonical populations f[a*ncells + i] (what lbm_get_populations returns;
 *               no solid mask: every cell counts), read only, caller-owned;
 *   ncells      1 <= ncells <= LBM_STATIC_MAX_CELLS (2^27 = 512^3), else LBM_EINVAL — the array holds one record
 *               per 4096 cells and cannot grow; larger grids go through lbm_moments on a handle;
 *   lattice     LBM_D2Q9 / LBM_D3Q19 / LBM_D3Q27, optionally | LBM_EQ_INCOMP; any other bit: LBM_EINVAL;
 *   force       HOST pointer to the 3 doubles of the body force F (u includes the F/2 shift, D:R7) or NULL = 0;
 *   diagnostics DEVICE, 8 doubles, written by the call (same order and meaning as lbm_moments), caller-owned;
 *   stream      cudaStream_t the two kernels are enqueued on (NULL = legacy default stream).  Asynchronous.
 * The cost of the fixed array: its 2 MiB stay resident on every GPU that loads this library, until the process exits.
 * First call on a device: looks up the array's device address (cudaGetSymbolAddress; once per device, cached) — make
 *   that first call at start-up, before any stream capture is begun.  After cudaDeviceReset the cached address is stale.
 * Sharing: every call on a device uses the same array, and the array keeps the previous call's records.  That needs
 *   no clearing (pass 1 overwrites every record pass 2 reads), but two calls that can overlap on the GPU — different
 *   streams with no event between them — race and both results are wrong.  Keep the calls of one device on one stream
 *   or order them.  Block records always cover the same 4096 cells, so the result does not depend on the SM count. */
enum { LBM_STATIC_MAX_CELLS = 1 << 27 };
int lbm_diagnostics_static(const double* f, int64_t ncells, int lattice, const double* force, double* diagnostics, void* stream);

/* Canonical populations f[a*N+i] (Q*N doubles, device): export / import.  Not on the hot path
 * (tests, checkpointing).  lbm_set_populations does not change the step counter. */
int lbm_get_populations(lbm_handle h, double* f);
int lbm_set_populations(lbm_handle h, const double* f);

/* Lattice tables in the library's order (HOST pointers): e[3*Q] as e[a*3 + d], t[Q].  `lattice`
 * is LBM_D2Q9, LBM_D3Q19 or LBM_D3Q27 (other bits ignored). */
int lbm_lattice(int lattice, int32_t* e, double* t);

/* Number of time steps taken since the last lbm_init_equilibrium (or -1 for a NULL handle). */
int64_t lbm_time(lbm_handle h);

/* Number of kernels this handle has launched so far (bookkeeping for benchmarks). */
int64_t lbm_launch_count(lbm_handle h);

/* Debug aids that work on the production kernels at any grid size (stand-ins for compute-sanitizer's memcheck /
 * initcheck, which is not available on every pool).  Every device array a handle owns is allocated between two 64 KB
 * guard zones filled with all-ones bytes (a NaN as fp64 and as fp32: a load that strays into a guard zone and is USED
 * poisons the result like an uninitialised slot does).
 *   lbm_debug_arm    rewrites the guard patterns and, poison != 0, fills every population / moment / scratch array of
 *                    the handle with all-ones bytes (a NaN as fp64 and as fp32) — call it before lbm_init_equilibrium /
 *                    lbm_set_populations: whatever the kernels then compute from a slot nobody wrote is NaN and shows up
 *                    in diagnostics[7] and in every comparison (geometry, face profiles, slab counters are left alone).
 *   lbm_debug_check  synchronises and returns the number of guard bytes that no longer hold the pattern: 0 = no store
 *                    of the library's kernels landed within 64 KB outside an array; negative = LBM_E* error.
 * Both synchronise the stream; neither costs anything between the two calls. */
int lbm_debug_arm(lbm_handle h, int poison);
int64_t lbm_debug_check(lbm_handle h);

/* Small grids (every block of the step kernel resident on the device at once, e.g. 32^3 or the paper's 512 x 128
 * channel) are bound by the launch rate of one kernel per step; for them lbm_step(h, n) takes all n steps in ONE
 * cooperative launch of a persistent kernel (a grid-wide barrier separates the steps; same arithmetic per cell, same
 * results bit for bit).  on = 0 switches that off (the grid is then stepped like a larger one: in pairs where
 * lbm_set_two_step applies, else one launch per step); default on. */
int lbm_set_persistent(lbm_handle h, int on);

/* Two time steps per pass through HBM (Eq. 7 applied twice; the same collision, Eq. 6, in between).  For a
 * whole box (no z-slab) of populations stored as fp64 under LBM_SCHEME_AB, without a solid mask (lbm_set_geometry) and
 * without SYMMETRY faces — D3Q19 with periodic, BOUNCE, MOVING and PRESSURE faces; D3Q27 with periodic x and y faces
 * (any z faces of those kinds) — lbm_step(h, n) takes the steps in pairs: one kernel runs step t on a tile extended by one cell, keeps the result in shared memory and
 * runs step t+1 from there, so that every population is read from HBM once and written once per TWO steps.  Same
 * arithmetic per cell, same results bit for bit as single steps; an odd n ends with one single step.  on = 1 (default):
 * where it pays — grids that give the kernel at least 1.4 waves of blocks (from about 80^3 up); on = 2: wherever the
 * kernel exists (tests); on = 0: never (one pass per step, as for every other variant).  Grids small enough for the
 * persistent kernel (lbm_set_persistent) keep using that one. */
int lbm_set_two_step(lbm_handle h, int on);

/* Tuning knob for measurements: CUDA block shape (threads along x, along y) of the
 * stream-collide kernel; 0,0 restores the default.  bx*by must be <= 256 and a multiple of 32.
 * The kernels with a fixed thread-to-cell mapping keep their own shape: two steps per pass (lbm_set_two_step), the
 * in-place odd phase without a mask (one grid row per block), fp32 storage with two cells per thread. */
int lbm_set_block(lbm_handle h, int bx, int by);

/* ---------------------------------------------------------------------------------------------
 * z-slab decomposition over several GPUs (Cartesian blocks, one process per device;
 * the populations that cross a cut are exchanged once per step, `PassF`).
 * D:R21.  The box nx*ny*nz_global is cut into slabs of whole z-planes; one handle per slab, one
 * slab per GPU (several slabs on one device also work).  A slab handle is a box of
 *     nz_local + 2  planes: plane 0 and plane nz_local+1 are HALO planes that stand for the last
 *     plane of the slab below and the first plane of the slab above,
 * so every array at this interface (rho, u, f, outputs) has N = nx*ny*(nz_local+2) cells per
 * component, plane index 1 + (z_global - z0).  Inputs (lbm_init_equilibrium, lbm_set_populations)
 * must carry the neighbouring slabs' values in the halo planes (periodic wrap included; ignored
 * beyond a non-periodic z face); outputs are written on the nz_local own planes only and the
 * diagnostics cover only them (sum / max / min them over the slabs).
 * Per step the fused kernel also stores the 5 (D3Q19) / 9 (D3Q27) / 0 (D2Q9) populations per cell of
 * its first and last plane that cross the cut directly into the neighbouring slab's halo plane (peer
 * memory: NVLink between GPUs); there is no separate exchange pass and no host staging.  Ordering between
 * slabs is on the device: step t of a slab starts when both neighbours have finished step t-1 (a 32-bit step
 * counter per side in the slab's own memory, written by the neighbour, waited for by the stream).
 * Geometry on a slab: lbm_set_geometry takes the mask with TWO halo planes per side — nx*ny*(nz_local+4) bytes, plane
 * index 2 + (z_global - z0), periodic wrap included, ignored beyond a non-periodic z face — because under
 * LBM_WALL_NODAL the wall-node status of a halo node depends on the plane beyond it (D:R16).  lbm_boundary_force
 * returns the part of Eq. 13 carried by the fluid nodes of the own planes: sum it over the slabs.
 * Restrictions: LBM_SCHEME_AB only; every slab must be advanced by the same number of steps; under device-side
 * ordering connected slabs of one process need a stream each (lbm_slab_connect returns LBM_EINVAL otherwise: on a shared
 * stream the second step of one slab would wait for a step of the other that is queued behind it) — host-ordered slabs
 * (lbm_slab_set_sync(h, 0) BEFORE lbm_slab_connect) may share a stream, the NULL stream included, as long as the
 * caller issues the steps one per slab in turn; lbm_init_equilibrium(_host) /
 * lbm_set_populations / lbm_set_geometry need all connected slabs idle (they rewrite halo planes the neighbours
 * store into); lbm_moments(_host) / lbm_get_populations may be called between unsynchronised steps (they wait for
 * the neighbours' last step on the device and touch no memory a neighbour writes).  SYMMETRY faces are supported. */

/* What a neighbour needs to know about a slab.  Plain data: pass it to another process as bytes. */
typedef struct {
  uint64_t buf[2];        /* device addresses of the two population buffers (valid in the owner process) */
  uint64_t flags;         /* device address of the two step counters {written by lower, by upper neighbour} */
  int64_t plane_stride;   /* cells of the handle = nx*ny*(nz_local+2) (checked by lbm_slab_connect)             */
  int32_t nz_local;
  int32_t device;         /* CUDA device ordinal of the owner                                           */
  int64_t pid;            /* owner process                                                              */
  int32_t Q;              /* lattice, bytes per stored population (8 / 4) and internal layout (1 = LBM_LAYOUT_SOA):  */
  int32_t elem_bytes;     /*   lbm_slab_connect refuses a neighbour that differs in any of them (LBM_EINVAL)    */
  int32_t layout_soa;
  int32_t reserved;
  uint64_t stream;        /* the owner's cudaStream_t (compared only within one process)                */
  uint8_t ipc_buf[2][64]; /* cudaIpcMemHandle_t of buf[0], buf[1]                                        */
  uint8_t ipc_flags[64];  /* cudaIpcMemHandle_t of flags                                                 */
} lbm_slab_peer_t;

/* Create the slab that owns global planes z0 .. z0+nz_local-1 of an nx*ny*nz_global box.  bc describes the
 * WHOLE box: its z- / z+ faces act on the slab that owns plane 0 / nz_global-1.  lattice: as lbm_create,
 * LBM_SCHEME_AA is refused (LBM_EUNSUPPORTED). */
lbm_handle lbm_create_slab(int nx, int ny, int nz_local, int z0, int nz_global, int lattice, double tau, const lbm_bc_t* bc);

/* Fill *out with this slab's addresses and IPC handles. */
int lbm_slab_export(lbm_handle h, lbm_slab_peer_t* out);

/* Connect the slab to its lower (z0-1) and upper (z0+nz_local) neighbours; NULL = none (a non-periodic z
 * face, or nothing to exchange).  A periodic box of one slab connects to itself.  Descriptors of the same
 * process are used as plain addresses (peer access between devices is enabled if needed); descriptors of
 * another process are opened through their IPC handles.  Call on every slab before the first lbm_step. */
int lbm_slab_connect(lbm_handle h, const lbm_slab_peer_t* lower, const lbm_slab_peer_t* upper);

/* 1 = (default) device-side ordering by step counters; 0 = none: the caller synchronises all slabs between
 * steps (lbm_step(h,1); stream sync; barrier) — for debugging and for several processes on ONE device; slabs of one
 * process that share one stream need no synchronisation at all, only one step per slab in turn.  May be called before
 * or after lbm_slab_connect; switching back to 1 on a slab that is connected to a slab on its own stream is refused
 * (LBM_EINVAL). */
int lbm_slab_set_sync(lbm_handle h, int device_sync);

/* Message of the calling thread's last failed call ("" if none).  Static storage. */
const char* lbm_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* LBM_B200_H */
