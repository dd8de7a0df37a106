/* include/lbm.h — C ABI of the B200-native lattice-Boltzmann hot path.
 *
 * The operation: the per-time-step fused streaming + BGK collision update of the
 * D3Q19 / D3Q27 populations of IMEXLBM (arXiv 2201.11330) on an nx*ny*nz box, fp64.
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
  LBM_D3Q19 = 19,           /* low byte: number of velocities                                  */
  LBM_D3Q27 = 27,
  LBM_EQ_STANDARD = 0,      /* Eq. 2, weakly compressible (default)                            */
  LBM_EQ_INCOMP = 1 << 8,   /* Eq. 5, incompressible model with rho0 = 1               */
  LBM_SCHEME_AUTO = 0,      /* = LBM_SCHEME_AB                                                 */
  LBM_SCHEME_AB = 1 << 12,  /* two buffers, pull ("stream on read")                            */
  LBM_SCHEME_AA = 2 << 12,  /* one buffer, in-place AA pattern                                 */
  LBM_STORE_F64 = 0,        /* populations stored as fp64 (default)                            */
  LBM_STORE_F32 = 1 << 16   /* populations stored as fp32 (f - t_a), arithmetic in fp64        */
};

enum { LBM_FACE_PERIODIC = 0, LBM_FACE_BOUNCE = 1, LBM_FACE_MOVING = 2 };

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
 * takes precedence over BOUNCE, and among MOVING faces the highest face index wins. */
typedef struct {
  int32_t face_kind[6];
  double face_u[6][3]; /* read only where face_kind == LBM_FACE_MOVING                          */
  double force[3];     /* uniform body-force density F (Guo forcing); all zero = no forcing     */
  void* stream;        /* cudaStream_t to run on (NULL = legacy default stream); caller-owned   */
} lbm_bc_t;

/* Create a solver on the current CUDA device.  nx >= 1, 1 <= ny, nz <= 65535; tau > 0.5; bc may be NULL
 * (all periodic, no force, default stream).  Allocates the population buffers (Q*N doubles,
 * twice for LBM_SCHEME_AB).  Populations are undefined until lbm_init_equilibrium or
 * lbm_set_populations.  Returns NULL on failure. */
lbm_handle lbm_create(int nx, int ny, int nz, int lattice, double tau, const lbm_bc_t* bc);

/* Free all device memory of the handle (synchronises its stream).  NULL is a no-op. */
void lbm_destroy(lbm_handle h);

/* P:82, P:276-278 (InitPDF): f_a(x, 0) = feq_a(rho(x), u(x)); resets the step counter.
 * rho: N doubles or NULL (= 1 everywhere); u: 3N doubles or NULL (= 0).  Device pointers. */
int lbm_init_equilibrium(lbm_handle h, const double* rho, const double* u);
/* Same with HOST pointers; the fields are copied to the device on the handle's stream. */
int lbm_init_equilibrium_host(lbm_handle h, const double* rho_host, const double* u_host);

/* Advance nsteps >= 0 time steps: per step and cell, pull-stream (Eq. 7) with wall links
 * (Eq. 10, D:R6), moments (Eq. 8-9), equilibrium (Eq. 2 / 5), BGK relaxation (Eq. 6), forcing
 * (D:R7) and store, in ONE kernel launch per step.  Asynchronous. */
int lbm_step(lbm_handle h, int nsteps);

/* P:295-304 (PostProcessing, Monitor): moments of the current canonical state.
 * rho: N doubles or NULL; u: 3N doubles or NULL (device).  diagnostics: HOST pointer to 8
 * doubles or NULL: { sum rho, sum rho u_x, sum rho u_y, sum rho u_z, 1/2 sum rho |u|^2,
 * max |u|, min rho, number of cells with non-finite rho or u }; non-finite cells are excluded
 * from the sums; under LBM_EQ_INCOMP "rho u" means rho0 u (D:R5); with forcing u includes the
 * F/2 shift (D:R7).  Synchronises the stream only if diagnostics != NULL. */
int lbm_moments(lbm_handle h, double* rho, double* u, double* diagnostics);
/* Same with HOST output pointers for the fields (either may be NULL); always synchronises. */
int lbm_moments_host(lbm_handle h, double* rho_host, double* u_host, double* diagnostics);

/* Canonical populations f[a*N+i] (Q*N doubles, device): export / import.  Not on the hot path
 * (tests, checkpointing).  lbm_set_populations does not change the step counter. */
int lbm_get_populations(lbm_handle h, double* f);
int lbm_set_populations(lbm_handle h, const double* f);

/* Lattice tables in the library's order (HOST pointers): e[3*Q] as e[a*3 + d], t[Q].  `lattice`
 * is LBM_D3Q19 or LBM_D3Q27 (other bits ignored). */
int lbm_lattice(int lattice, int32_t* e, double* t);

/* Number of time steps taken since the last lbm_init_equilibrium (or -1 for a NULL handle). */
int64_t lbm_time(lbm_handle h);

/* Number of kernels this handle has launched so far (bookkeeping for benchmarks). */
int64_t lbm_launch_count(lbm_handle h);

/* Tuning knob for measurements: CUDA block shape (threads along x, along y) of the
 * stream-collide kernel; 0,0 restores the default.  bx*by must be <= 256 and a multiple of 32. */
int lbm_set_block(lbm_handle h, int bx, int by);

/* Message of the calling thread's last failed call ("" if none).  Static storage. */
const char* lbm_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* LBM_B200_H */
