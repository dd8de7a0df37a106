// oracle/lbm_oracle.cpp
//
// TEST INFRASTRUCTURE — NOT THE PRODUCT.  This is the plain, slow, CPU oracle of
// the lattice-Boltzmann hot path of IMEXLBM (arXiv 2201.11330).  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// build, load or call it.  It shares no code, header, table or constant with the
// CUDA path under paper_2201_11330_b200/csrc/ and includes nothing from it.
//
// It follows the paper step by step, un-fused, in the paper's own order
// (section 3.1): Collision -> BoundaryCondition -> Propagation ->
// PostProcessing, on the paper's two arrays `f` and `fb` (Table 3)
// in the paper's array-of-structures indexing f(id*nq+iq).
// "P:n" below = /root/reference/PAPER.md line n.  "D:Rk" = reading Rk in DESIGN.md
// (points where the paper is silent and BASELINE.json fixes the behaviour).
//
// Pin status (tests/test_oracle_pins.py, run with -m "not gpu"):
//   lattice tables ............ pinned: Eq. 3-4 as printed (tests/golden), isotropy identities
//   equilibrium Eq. 2 / Eq. 5 . pinned: moment identities, fixed point, P:375 constants
//   collision + propagation ... pinned: conservation, Taylor-Green decay rate, shear-wave decay
//   halfway bounce-back ....... pinned: Poiseuille parabola + BGK slip constant (closed form)
//   moving wall (Ladd) ........ pinned: planar Couette exact linear profile, cavity mass
//   Guo forcing ............... pinned: momentum gain F*N per step, Poiseuille
//   indexing .................. pinned: independent brute-force gather on 4^3 (long double)
//   moments + diagnostics[8] .. pinned: fields by closed forms (Couette, Poiseuille); all eight diagnostics against a
//                               direct NumPy evaluation of their definition (random f, solid mask, both wall models,
//                               F/2 shift, Eq. 5 weighting), NaN / Inf cells counted and left out of the sums
//   D3Q27 ..................... pinned only through the same invariants and closed forms;
//                               no D3Q27-specific printed value exists in the paper.
//   D2Q9 ...................... pinned: the table is Eq. 3-4 as printed; dynamics by 2-D isotropy, brute-force
//                               gather, exact 2-D Taylor-Green decay, Poiseuille closed form (tests/test_oracle_d2q9_pins.py)
//   solid mask `geo` .......... pinned: brute-force gather with a mask; staircase channel built from
//                               the mask equals the face-built channel bit for bit
//   nodal bounce-back (Eq. 10)  pinned: second-order convergence of the channel profile (the
//                               paper's own claim), wall position, mirror symmetry
//   momentum exchange (Eq. 13)  pinned: exact momentum balance of the fluid region per step;
//                               steady drag = total body force
//   open faces (D:R22) ........ pinned: brute-force gather over every face mix, pressure-driven Poiseuille closed
//                               form, inlet flux (tests/test_oracle_open_pins.py)
//   symmetry faces (D:R25), open faces next to nodal walls (D:R24)
//                               pinned: equality with the mirror-extended domain (one plane, two planes, an edge,
//                               a body cut by the plane, both wall models), free slip, half channel = full channel
//                               closed form, brute-force gather over every rule at once
//                               (tests/test_oracle_symmetry_pins.py)
//
// Floating point: IEEE double throughout ("double precision"); compile with
// -ffp-contract=off so that no FMA contraction happens.  Reductions for the
// diagnostics are accumulated in long double.

#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

struct Lattice {
  int Q = 0;
  int e[27][3];
  double t[27];
};

// Velocity set and weights.  P:49-53: the paper prints only D2Q9 (Eq. 3-4); its
// columns run lexicographically over (e_x, e_y), each component -1 -> 0 -> +1, e_x
// outermost, which gives the stated property opposite(alpha) = m-1-alpha.
// D:R4: the 3-D sets extend the same rule to (e_x, e_y, e_z); D3Q19 is that list
// without the 8 corner vectors.  Weights by squared speed (Qian et al., refs [11],
// [12] cited at P:43).  Q = 9 is the printed D2Q9 itself (e_z = 0).
bool make_lattice(int Q, Lattice& L) {
  if (Q != 9 && Q != 19 && Q != 27) return false;
  L.Q = Q;
  int q = 0;
  for (int ex = -1; ex <= 1; ++ex)
    for (int ey = -1; ey <= 1; ++ey)
      for (int ez = -1; ez <= 1; ++ez) {
        const int s = ex * ex + ey * ey + ez * ez;
        if (Q == 9 && ez != 0) continue;
        if (Q == 19 && s == 3) continue;
        double w = 0.0;
        if (Q == 9) w = (s == 0) ? 4.0 / 9.0 : (s == 1) ? 1.0 / 9.0 : 1.0 / 36.0;
        if (Q == 19) w = (s == 0) ? 1.0 / 3.0 : (s == 1) ? 1.0 / 18.0 : 1.0 / 36.0;
        if (Q == 27)
          w = (s == 0) ? 8.0 / 27.0 : (s == 1) ? 2.0 / 27.0 : (s == 2) ? 1.0 / 54.0 : 1.0 / 216.0;
        L.e[q][0] = ex;
        L.e[q][1] = ey;
        L.e[q][2] = ez;
        L.t[q] = w;
        ++q;
      }
  return q == Q;
}

enum { EQ_STANDARD = 0, EQ_INCOMP = 1 };              // Eq. 2 | Eq. 5
enum { FACE_PERIODIC = 0, FACE_BOUNCE = 1, FACE_MOVING = 2, FACE_PRESSURE = 3, FACE_SYMMETRY = 4 };
// D:R22 (open boundaries; the paper names a parabolic inlet and an outflow, with no formulae):
//   inlet  = FACE_MOVING with a per-cell wall velocity profile (velocity bounce-back, Ladd),
//   outlet = FACE_PRESSURE: anti-bounce-back at the prescribed density face_rho.
// D:R25 ("the left and right boundaries are symmetric", no formula): FACE_SYMMETRY = a mirror plane half a
//   link beyond the last node (specular reflection, free slip).
// D:R3 / D:R16.  HALFWAY: the wall lies half a link beyond the last fluid node (BASELINE.json
// configs).  NODAL: the paper's "modified nodal bounce back" (Eq. 10): wall nodes lie on
// the wall, receive f_alpha = f_abar for the directions no node streams into them, and collide.
enum { WALL_HALFWAY = 0, WALL_NODAL = 1 };

struct Oracle {
  int nx, ny, nz;
  int64_t N;
  Lattice L;
  int eq;            // EQ_STANDARD or EQ_INCOMP
  double omega;      // P:61-63 Eq. 6: 1/(tau/dt + 1/2); D:R1: API tau = tau_paper/dt + 1/2
  double rho0;       // constant density of the incompressible model, 1
  int face_kind[6];  // x-, x+, y-, y+, z-, z+
  double face_u[6][3];
  double face_rho[6];                      // density prescribed on FACE_PRESSURE faces (D:R22)
  std::vector<double> face_profile[6];     // optional per-cell wall velocity of a MOVING face: [c*n + j] (D:R22)
  double F[3];       // uniform body force density (D:R7, Guo forcing; not in the paper)
  std::vector<double> f;      // P:208 `f`:  pre-collision populations, AoS f[id*Q+iq]
  std::vector<double> fb;     // P:208 `fb`: "backup" = post-collision populations
  std::vector<double> rho_w;  // density seen by the collision sweep, kept for the wall term (D:R6)
  std::vector<double> u_w;    // velocity seen by the collision sweep, [i*3+d], kept for the pressure faces (D:R22)
  std::vector<uint8_t> geo;     // P:210 `geo`: 1 = solid node, 0 = fluid node (all fluid by default)
  std::vector<uint8_t> active;  // node takes part in collision and propagation (D:R16)
  int wall_model = WALL_HALFWAY;
  int64_t steps_done = 0;

  int64_t cell(int x, int y, int z) const { return (int64_t)x + (int64_t)nx * ((int64_t)y + (int64_t)ny * z); }
};

// Eq. 2 with c_s^2 = 1/3  (P:375-376 prints the constants 3, 4.5, 1.5):
//   feq = t rho [1 + 3 e.u + 4.5 (e.u)^2 - 1.5 u.u]
// Eq. 5 (code form P:375): feq = t [ p/c_s^2 + rho0 (3 e.u + 4.5 (e.u)^2 - 1.5 u.u) ],
//   where `rho` below stands for p/c_s^2 = sum_alpha f_alpha (Eq. 8).
inline double feq_value(const Oracle& o, int iq, double rho, const double u[3]) {
  double edu = 0.0, udu = 0.0;
  for (int d = 0; d < 3; ++d) {
    edu += o.L.e[iq][d] * u[d];
    udu += u[d] * u[d];
  }
  if (o.eq == EQ_STANDARD) return o.L.t[iq] * rho * (1.0 + 3.0 * edu + 4.5 * edu * edu - 1.5 * udu);
  return o.L.t[iq] * (rho + o.rho0 * (3.0 * edu + 4.5 * edu * edu - 1.5 * udu));
}

// Moments, Eq. 8-9:  rho = sum f (= p/c_s^2),  u = (1/rho) sum e f.
// D:R5: under Eq. 5 the divisor is the constant rho0 (the code multiplies the velocity
// terms by rho0).  D:R7: with a body force the velocity carries the half-force
// shift, u = (sum e f + F/2)/rho (Guo et al.).
inline void moments_of(const Oracle& o, const double* fc, double& rho, double u[3]) {
  rho = 0.0;
  double m[3] = {0.0, 0.0, 0.0};
  for (int iq = 0; iq < o.L.Q; ++iq) {
    rho += fc[iq];
    for (int d = 0; d < 3; ++d) m[d] += o.L.e[iq][d] * fc[iq];
  }
  const double div = (o.eq == EQ_STANDARD) ? rho : o.rho0;
  for (int d = 0; d < 3; ++d) u[d] = (m[d] + 0.5 * o.F[d]) / div;
}

// Node x + s*e_iq with periodic wrap; false if it lies outside the box through a non-periodic face of any kind
// (used where only nodes of the box count: node classification, D:R16, and the body force, Eq. 13).
inline bool neighbour(const Oracle& o, int x, int y, int z, int iq, int sgn, int out[3]) {
  const int c[3] = {x, y, z}, n[3] = {o.nx, o.ny, o.nz};
  bool inside = true;
  for (int d = 0; d < 3; ++d) {
    out[d] = c[d] + sgn * o.L.e[iq][d];
    if (out[d] < 0 || out[d] >= n[d]) {
      const int face = 2 * d + (out[d] < 0 ? 0 : 1);
      if (o.face_kind[face] == FACE_PERIODIC) out[d] = ((out[d] % n[d]) + n[d]) % n[d];
      else inside = false;
    }
  }
  return inside;
}

// Wall velocity of MOVING face `face` as seen by cell (x,y,z): the uniform face_u, or the cell's entry of the
// per-cell profile (D:R22), indexed by the two in-face coordinates of the cell, lower axis fastest.
inline void wall_velocity(const Oracle& o, int face, int x, int y, int z, double uw[3]) {
  if (o.face_profile[face].empty()) {
    for (int d = 0; d < 3; ++d) uw[d] = o.face_u[face][d];
    return;
  }
  const int axis = face / 2;
  int64_t j, n;
  if (axis == 0) { j = y + (int64_t)o.ny * z; n = (int64_t)o.ny * o.nz; }
  else if (axis == 1) { j = x + (int64_t)o.nx * z; n = (int64_t)o.nx * o.nz; }
  else { j = x + (int64_t)o.nx * y; n = (int64_t)o.nx * o.ny; }
  for (int d = 0; d < 3; ++d) uw[d] = o.face_profile[face][(size_t)d * n + j];
}

// Where the population that arrives at node (x,y,z) along iq comes from (sgn = -1), or where the one that leaves
// along iq goes to (sgn = +1).  D:R6 / D:R22 / D:R24 / D:R25.  The node (x,y,z) + sgn*e_iq is wrapped on periodic
// axes; if it lies beyond non-periodic faces the kinds of ALL faces crossed decide, in this order:
//   any MOVING   -> LINK_MOVING   (face = the highest-index MOVING face crossed):   velocity bounce-back (Ladd)
//   any BOUNCE   -> LINK_WALL:     a wall link (halfway bounce-back, or unknown of Eq. 10 under the nodal model)
//   any PRESSURE -> LINK_PRESSURE (face = the highest-index PRESSURE face crossed): anti-bounce-back
//   else (only SYMMETRY faces)     -> LINK_NODE at the mirror image: the coordinates along the crossed axes stay
//                                    those of (x,y,z), `dir` = e_iq with those components negated.
// LINK_NODE says nothing about the node being active: the caller checks, and treats an inactive one as LINK_WALL.
enum { LINK_NODE = 0, LINK_WALL = 1, LINK_MOVING = 2, LINK_PRESSURE = 3 };
struct Link {
  int kind;
  int node[3];
  int dir;   // direction index the population has at `node` (LINK_NODE)
  int face;  // LINK_MOVING / LINK_PRESSURE
};

inline int direction_index(const Lattice& L, const int e[3]) {
  for (int iq = 0; iq < L.Q; ++iq)
    if (L.e[iq][0] == e[0] && L.e[iq][1] == e[1] && L.e[iq][2] == e[2]) return iq;
  return -1;
}

inline Link resolve(const Oracle& o, int x, int y, int z, int iq, int sgn) {
  const int c[3] = {x, y, z}, n[3] = {o.nx, o.ny, o.nz};
  Link L;
  L.kind = LINK_NODE;
  L.dir = iq;
  L.face = -1;
  bool inside = true;
  for (int d = 0; d < 3; ++d) {
    L.node[d] = c[d] + sgn * o.L.e[iq][d];
    inside = inside && L.node[d] >= 0 && L.node[d] < n[d];
  }
  if (inside) return L;  // the bulk of the nodes
  int mf = -1, pf = -1, e2[3];
  bool bounce = false, sym = false;
  for (int d = 0; d < 3; ++d) {
    e2[d] = o.L.e[iq][d];
    if (L.node[d] < 0 || L.node[d] >= n[d]) {
      const int face = 2 * d + (L.node[d] < 0 ? 0 : 1);
      switch (o.face_kind[face]) {
        case FACE_PERIODIC: L.node[d] = ((L.node[d] % n[d]) + n[d]) % n[d]; break;
        case FACE_MOVING: if (face > mf) mf = face; break;
        case FACE_BOUNCE: bounce = true; break;
        case FACE_PRESSURE: if (face > pf) pf = face; break;
        default:  // FACE_SYMMETRY: mirror image
          sym = true;
          L.node[d] = c[d];
          e2[d] = -e2[d];
          break;
      }
    }
  }
  if (mf >= 0) { L.kind = LINK_MOVING; L.face = mf; }
  else if (bounce) L.kind = LINK_WALL;
  else if (pf >= 0) { L.kind = LINK_PRESSURE; L.face = pf; }
  else if (sym) L.dir = direction_index(o.L, e2);
  return L;
}

inline bool link_has_active_node(const Oracle& o, const Link& L) {
  return L.kind == LINK_NODE && o.active[o.cell(L.node[0], L.node[1], L.node[2])];
}

// D:R16.  HALFWAY: the active nodes are the fluid nodes (geo = 0).  NODAL: also every solid node
// with at least one fluid node among its lattice neighbours — these are the wall nodes on which
// "a collision operation is then applied ... like in the fluid bulk"; deeper solid nodes
// take no part.
void classify_nodes(Oracle& o) {
  for (int z = 0; z < o.nz; ++z)
    for (int y = 0; y < o.ny; ++y)
      for (int x = 0; x < o.nx; ++x) {
        const int64_t i = o.cell(x, y, z);
        uint8_t a = o.geo[i] == 0;
        if (!a && o.wall_model == WALL_NODAL) {
          for (int iq = 0; iq < o.L.Q && !a; ++iq) {
            int s[3];
            if (neighbour(o, x, y, z, iq, +1, s) && o.geo[o.cell(s[0], s[1], s[2])] == 0) a = 1;
          }
        }
        o.active[i] = a;
      }
}

// Eq. 10 on the wall nodes of the NODAL model: a direction alpha that no active node
// streams into the node ("unknown") takes the value of its opposite, f_alpha = f_abar, when abar
// itself arrived from an active node.  D:R17: if both ends of the link are inactive (an edge or
// corner of the wall) the pair keeps what `keep` holds for it (propagation passes the node's own
// post-collision fb_abar, i.e. plain bounce-back; init/set pass nothing and leave f untouched).
void replicate_nodal(Oracle& o, int x, int y, int z, const double* keep /* fb of this node or NULL */) {
  const int Q = o.L.Q;
  const int64_t i = o.cell(x, y, z);
  for (int iq = 0; iq < Q; ++iq) {
    const Link up = resolve(o, x, y, z, iq, -1);
    // D:R24: a link through an open face (MOVING / PRESSURE) is no wall link: its value is the face's rule
    if (up.kind == LINK_MOVING || up.kind == LINK_PRESSURE || link_has_active_node(o, up)) continue;
    if (link_has_active_node(o, resolve(o, x, y, z, iq, +1))) o.f[i * Q + iq] = o.f[i * Q + (Q - 1 - iq)];
    else if (keep) o.f[i * Q + iq] = keep[Q - 1 - iq];
  }
}

void make_state_consistent(Oracle& o) {
  if (o.wall_model != WALL_NODAL) return;
  for (int z = 0; z < o.nz; ++z)
    for (int y = 0; y < o.ny; ++y)
      for (int x = 0; x < o.nx; ++x)
        if (o.active[o.cell(x, y, z)]) replicate_nodal(o, x, y, z, nullptr);
}

// InitPDF: f(x, 0) = feq(rho0(x), u0(x)).  D:R17: under the NODAL model the state
// is then made consistent with Eq. 10 on the wall nodes.
void init_pdf(Oracle& o, const double* rho, const double* u /* SoA u[c*N+i] */) {
#pragma omp parallel for schedule(static) if (o.N >= 16384)  // tiny grids: a thread team costs more than the sweep
  for (int64_t i = 0; i < o.N; ++i) {
    const double r = rho ? rho[i] : 1.0;
    double uu[3] = {0.0, 0.0, 0.0};
    if (u)
      for (int d = 0; d < 3; ++d) uu[d] = u[(int64_t)d * o.N + i];
    for (int iq = 0; iq < o.L.Q; ++iq) o.f[i * o.L.Q + iq] = feq_value(o, iq, r, uu);
  }
  make_state_consistent(o);
  o.steps_done = 0;
}

// Sweep 1 — Collision (Eq. 6; listing P:357-382):  f -> fb.
//   fb = f - omega (f - feq)                                       [Eq. 6]
//      + (1 - omega/2) t [3 (e - u) + 9 (e.u) e] . F              [D:R7, only when F != 0]
void collision(Oracle& o) {
  const int Q = o.L.Q;
  const bool forced = (o.F[0] != 0.0 || o.F[1] != 0.0 || o.F[2] != 0.0);
#pragma omp parallel for schedule(static) if (o.N >= 16384)  // tiny grids: a thread team costs more than the sweep
  for (int64_t i = 0; i < o.N; ++i) {
    if (!o.active[i]) continue;  // the loop runs over `fluid_id` (here: the active nodes, D:R16)
    const double* fc = &o.f[i * Q];
    double rho, u[3];
    moments_of(o, fc, rho, u);
    o.rho_w[i] = (o.eq == EQ_STANDARD) ? rho : o.rho0;
    for (int d = 0; d < 3; ++d) o.u_w[i * 3 + d] = u[d];
    for (int iq = 0; iq < Q; ++iq) {
      const double feq = feq_value(o, iq, rho, u);
      double out = fc[iq] - o.omega * (fc[iq] - feq);
      if (forced) {
        double edu = 0.0;
        for (int d = 0; d < 3; ++d) edu += o.L.e[iq][d] * u[d];
        double s = 0.0;
        for (int d = 0; d < 3; ++d) s += (3.0 * (o.L.e[iq][d] - u[d]) + 9.0 * edu * o.L.e[iq][d]) * o.F[d];
        out += (1.0 - 0.5 * o.omega) * o.L.t[iq] * s;
      }
      o.fb[i * Q + iq] = out;
    }
  }
}

// Sweep 2 — BoundaryCondition, pre-propagation.  On a single domain there
// is no halo to exchange (P:395-397 is the MPI part); the wall links are resolved in
// the propagation sweep below from fb of the same cell, which is the equivalent
// pre-propagation form of Eq. 10 for a wall half-way between nodes (D:R3).
void boundary_condition(Oracle&) {}

// Sweep 3 — Propagation (Eq. 7):  f_alpha(x, t) = fb_alpha(x - e_alpha, t - 1), for every
// active node x.  If x - e_alpha is not an active node (it is a solid node of `geo`, or lies
// outside the box through a non-periodic face) nothing streams in along alpha:
//   HALFWAY (D:R3):  f_alpha(x) = fb_opp(alpha)(x)                  [Eq. 10; opp = Q-1-alpha, P:49]
//                               + 6 t_alpha rho_w (e_alpha . u_w)   [D:R6, Ladd; only through a MOVING face]
//   NODAL: f_alpha(x) = f_opp(alpha)(x), the value that has just arrived at the wall
//                    node from the fluid side (Eq. 10 applied after propagation); D:R17 for
//                    links with no active node at either end.
// D:R6 tie-break: when the upstream node lies beyond several non-periodic faces, a MOVING
// face takes precedence over BOUNCE faces; among several MOVING faces the highest face
// index (z+ > z- > y+ > y- > x+ > x-) is used.
void propagation(Oracle& o) {
  const int Q = o.L.Q;
#pragma omp parallel for schedule(static) if (o.N >= 16384)  // tiny grids: a thread team costs more than the sweep
  for (int z = 0; z < o.nz; ++z)
    for (int y = 0; y < o.ny; ++y)
      for (int x = 0; x < o.nx; ++x) {
        const int64_t i = o.cell(x, y, z);
        if (!o.active[i]) continue;
        for (int iq = 0; iq < Q; ++iq) {
          const Link L = resolve(o, x, y, z, iq, -1);
          if (link_has_active_node(o, L)) {
            // Eq. 7; through a SYMMETRY face (D:R25) the mirror image: direction L.dir of the mirrored node
            o.f[i * Q + iq] = o.fb[o.cell(L.node[0], L.node[1], L.node[2]) * Q + L.dir];
          } else if (L.kind == LINK_MOVING) {
            double uw[3], eduw = 0.0;
            wall_velocity(o, L.face, x, y, z, uw);
            for (int d = 0; d < 3; ++d) eduw += o.L.e[iq][d] * uw[d];
            o.f[i * Q + iq] = o.fb[i * Q + (Q - 1 - iq)] + 6.0 * o.L.t[iq] * o.rho_w[i] * eduw;
          } else if (L.kind == LINK_PRESSURE) {
            // D:R22 anti-bounce-back: f_a = -f*_abar + 2 feq+_a(rho_face, u(x,t)), feq+ = the part of the
            // equilibrium that is even in e (Eq. 2: t rho (1 + 4.5 (e.u)^2 - 1.5 u.u); Eq. 5: t (rho + rho0 (...)))
            const double* uu = &o.u_w[i * 3];
            double edu = 0.0, udu = 0.0;
            for (int d = 0; d < 3; ++d) {
              edu += o.L.e[iq][d] * uu[d];
              udu += uu[d] * uu[d];
            }
            const double rf = o.face_rho[L.face];
            const double even = (o.eq == EQ_STANDARD) ? o.L.t[iq] * rf * (1.0 + 4.5 * edu * edu - 1.5 * udu)
                                                      : o.L.t[iq] * (rf + o.rho0 * (4.5 * edu * edu - 1.5 * udu));
            o.f[i * Q + iq] = -o.fb[i * Q + (Q - 1 - iq)] + 2.0 * even;
          } else if (o.wall_model == WALL_HALFWAY) {
            o.f[i * Q + iq] = o.fb[i * Q + (Q - 1 - iq)];  // Eq. 10 for a wall half-way between nodes (D:R3)
          }
        }
        if (o.wall_model == WALL_NODAL) replicate_nodal(o, x, y, z, &o.fb[i * Q]);
      }
}

// Momentum-exchange force on the solid nodes of `geo` (Eq. 13), for the step that
// has just been taken (fb = post-collision populations f* of time t, f = populations after
// propagation):
//   F = sum over fluid nodes x next to the body, sum over outgoing directions alpha
//       (x + e_alpha is a solid node of geo):  [ f*_alpha(x, t) + f_abar(x, t + dt) ] e_alpha
// "Fluid node" = geo 0.  Box-face walls are not part of the body.  Defined after >= 1 step.
void boundary_force(const Oracle& o, double F[3]) {
  const int Q = o.L.Q;
  long double acc[3] = {0, 0, 0};
  for (int z = 0; z < o.nz; ++z)
    for (int y = 0; y < o.ny; ++y)
      for (int x = 0; x < o.nx; ++x) {
        const int64_t i = o.cell(x, y, z);
        if (o.geo[i] != 0 || !o.active[i]) continue;
        for (int iq = 0; iq < Q; ++iq) {
          int d3[3];
          if (!neighbour(o, x, y, z, iq, +1, d3)) continue;
          if (o.geo[o.cell(d3[0], d3[1], d3[2])] == 0) continue;
          const double term = o.fb[i * Q + iq] + o.f[i * Q + (Q - 1 - iq)];
          for (int d = 0; d < 3; ++d) acc[d] += (long double)term * o.L.e[iq][d];
        }
      }
  for (int d = 0; d < 3; ++d) F[d] = (double)acc[d];
}

// Sweep 4 — PostProcessing (Eq. 8-9) and Monitor, on
// demand.  diagnostics[8] = { sum rho, sum rho u_x, sum rho u_y, sum rho u_z,
// 1/2 sum rho |u|^2, max |u|, min rho, number of cells with a non-finite rho or u }.
// Sums run over the active nodes (D:R16).  Under Eq. 5 "rho u" and "rho |u|^2" use rho0 (D:R5).  D:R13: 3-component magnitude,
// all cells (the listing's 2-D magnitude and idn=1 start are typos of the extraction).
void post_processing(const Oracle& o, double* rho_out, double* u_out, double* diag) {
  long double s_rho = 0, s_m[3] = {0, 0, 0}, s_e = 0;
  double umax = 0.0, rmin = INFINITY;
  int64_t bad = 0;
  for (int64_t i = 0; i < o.N; ++i) {
    double rho, u[3];
    if (!o.active[i]) {  // Monitor runs over the fluid nodes only; inactive nodes report 0
      if (rho_out) rho_out[i] = 0.0;
      if (u_out)
        for (int d = 0; d < 3; ++d) u_out[(int64_t)d * o.N + i] = 0.0;
      continue;
    }
    moments_of(o, &o.f[i * o.L.Q], rho, u);
    if (rho_out) rho_out[i] = rho;
    if (u_out)
      for (int d = 0; d < 3; ++d) u_out[(int64_t)d * o.N + i] = u[d];
    if (!diag) continue;
    const double usq = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
    if (!std::isfinite(rho) || !std::isfinite(usq)) {
      ++bad;
      continue;
    }
    const double rw = (o.eq == EQ_STANDARD) ? rho : o.rho0;
    s_rho += rho;
    for (int d = 0; d < 3; ++d) s_m[d] += (long double)rw * u[d];
    s_e += 0.5L * rw * usq;
    umax = std::fmax(umax, std::sqrt(usq));
    rmin = std::fmin(rmin, rho);
  }
  if (diag) {
    diag[0] = (double)s_rho;
    diag[1] = (double)s_m[0];
    diag[2] = (double)s_m[1];
    diag[3] = (double)s_m[2];
    diag[4] = (double)s_e;
    diag[5] = umax;
    diag[6] = rmin;
    diag[7] = (double)bad;
  }
}

}  // namespace

// ---- tiny C ABI so that tests can drive the oracle through ctypes ------------------
// All pointers are HOST pointers.  Field layouts at this interface are the canonical
// ones of include/lbm.h (rho[i], u[c*N+i], f[alpha*N+i], i = x + nx*(y + ny*z)); the
// AoS <-> SoA transposition happens here and nowhere else.
extern "C" {

void* orc_create(int nx, int ny, int nz, int Q, int eq, double tau, const int* face_kind,
                 const double* face_u /*6x3 or NULL*/, const double* force /*3 or NULL*/) {
  if (nx < 1 || ny < 1 || nz < 1 || !(tau > 0.5)) return nullptr;
  Oracle* o = new Oracle();
  if (!make_lattice(Q, o->L)) {
    delete o;
    return nullptr;
  }
  o->nx = nx;
  o->ny = ny;
  o->nz = nz;
  o->N = (int64_t)nx * ny * nz;
  o->eq = eq;
  o->omega = 1.0 / tau;  // D:R1
  o->rho0 = 1.0;
  for (int k = 0; k < 6; ++k) {
    o->face_kind[k] = face_kind ? face_kind[k] : FACE_PERIODIC;
    for (int d = 0; d < 3; ++d) o->face_u[k][d] = face_u ? face_u[3 * k + d] : 0.0;
    o->face_rho[k] = 1.0;
  }
  for (int d = 0; d < 3; ++d) o->F[d] = force ? force[d] : 0.0;
  o->f.assign((size_t)o->N * Q, 0.0);
  o->fb.assign((size_t)o->N * Q, 0.0);
  o->rho_w.assign((size_t)o->N, 1.0);
  o->u_w.assign((size_t)o->N * 3, 0.0);
  o->geo.assign((size_t)o->N, 0);
  o->active.assign((size_t)o->N, 1);
  return o;
}

void orc_destroy(void* h) { delete static_cast<Oracle*>(h); }

// SetGeometry: geo[i] != 0 marks a solid node (NULL = all fluid); wall_model is
// WALL_HALFWAY (0) or WALL_NODAL (1).  Re-classifies the nodes; call before init / set_f.
int orc_set_geometry(void* h, const uint8_t* geo, int wall_model) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (wall_model != WALL_HALFWAY && wall_model != WALL_NODAL) return -1;
  o.wall_model = wall_model;
  for (int64_t i = 0; i < o.N; ++i) o.geo[i] = (geo && geo[i]) ? 1 : 0;
  classify_nodes(o);
  return 0;
}

// D:R22.  Density of the FACE_PRESSURE faces (6 values; entries of other faces are ignored).
void orc_set_face_rho(void* h, const double* rho6) {
  Oracle& o = *static_cast<Oracle*>(h);
  for (int k = 0; k < 6; ++k) o.face_rho[k] = rho6[k];
}

// D:R22.  Per-cell wall velocity of MOVING face `face`: u[c*n + j], n = cells of the face, j over the two
// in-face coordinates (lower axis fastest); NULL restores the uniform face_u.
int orc_set_face_velocity(void* h, int face, const double* u) {
  Oracle& o = *static_cast<Oracle*>(h);
  if (face < 0 || face > 5) return -1;
  const int axis = face / 2;
  const int64_t n = axis == 0 ? (int64_t)o.ny * o.nz : axis == 1 ? (int64_t)o.nx * o.nz : (int64_t)o.nx * o.ny;
  if (u) o.face_profile[face].assign(u, u + 3 * n);
  else o.face_profile[face].clear();
  return 0;
}

void orc_get_active(void* h, uint8_t* out) {
  const Oracle& o = *static_cast<Oracle*>(h);
  for (int64_t i = 0; i < o.N; ++i) out[i] = o.active[i];
}

void orc_boundary_force(void* h, double* F) { boundary_force(*static_cast<Oracle*>(h), F); }

// Lattice tables in the oracle's order: e_out[3*Q] (e[iq*3+d], the paper's e(iq*dim+ind),
// P:373) and t_out[Q].
int orc_lattice(int Q, int* e_out, double* t_out) {
  Lattice L;
  if (!make_lattice(Q, L)) return -1;
  for (int q = 0; q < Q; ++q) {
    for (int d = 0; d < 3; ++d) e_out[3 * q + d] = L.e[q][d];
    t_out[q] = L.t[q];
  }
  return 0;
}

// Single-cell equilibrium for table-level tests: feq_out[Q].
int orc_feq(int Q, int eq, double rho, const double* u, double* feq_out) {
  Oracle o;
  if (!make_lattice(Q, o.L)) return -1;
  o.eq = eq;
  o.rho0 = 1.0;
  for (int q = 0; q < Q; ++q) feq_out[q] = feq_value(o, q, rho, u);
  return 0;
}

void orc_init_equilibrium(void* h, const double* rho, const double* u) { init_pdf(*static_cast<Oracle*>(h), rho, u); }

void orc_collision(void* h) { collision(*static_cast<Oracle*>(h)); }
void orc_boundary_condition(void* h) { boundary_condition(*static_cast<Oracle*>(h)); }
void orc_propagation(void* h) { propagation(*static_cast<Oracle*>(h)); }

// The time loop of P:112-114.
void orc_step(void* h, int nsteps) {
  Oracle& o = *static_cast<Oracle*>(h);
  for (int s = 0; s < nsteps; ++s) {
    collision(o);
    boundary_condition(o);
    propagation(o);
    ++o.steps_done;
  }
}

void orc_moments(void* h, double* rho, double* u, double* diag) { post_processing(*static_cast<Oracle*>(h), rho, u, diag); }

static void export_soa(const Oracle& o, const std::vector<double>& a, double* out) {
  for (int iq = 0; iq < o.L.Q; ++iq)
    for (int64_t i = 0; i < o.N; ++i) out[(int64_t)iq * o.N + i] = o.active[i] ? a[i * o.L.Q + iq] : 0.0;  // inactive nodes report 0
}

void orc_get_f(void* h, double* out) { export_soa(*static_cast<Oracle*>(h), static_cast<Oracle*>(h)->f, out); }
void orc_get_fb(void* h, double* out) { export_soa(*static_cast<Oracle*>(h), static_cast<Oracle*>(h)->fb, out); }

void orc_set_f(void* h, const double* in) {
  Oracle& o = *static_cast<Oracle*>(h);
  for (int iq = 0; iq < o.L.Q; ++iq)
    for (int64_t i = 0; i < o.N; ++i) o.f[i * o.L.Q + iq] = in[(int64_t)iq * o.N + i];
  make_state_consistent(o);  // D:R17
}

// Populations of selected cells only: out[k*Q + iq] for cell index cells[k].
void orc_get_f_cells(void* h, const int64_t* cells, int64_t ncells, double* out) {
  const Oracle& o = *static_cast<Oracle*>(h);
  for (int64_t k = 0; k < ncells; ++k)
    for (int iq = 0; iq < o.L.Q; ++iq) out[k * o.L.Q + iq] = o.f[cells[k] * o.L.Q + iq];
}

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
