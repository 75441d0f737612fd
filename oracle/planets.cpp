// planets.cpp -- SURVEY.md 8(f) NEXT-2: live planets (section 3.8).
// CPU oracle, TEST INFRASTRUCTURE (see fargo_oracle.h).
//
// * N point masses around a fixed central mass, advanced once per update over h = dt (the CFL time step) with the
//   fifth-order Cash-Karp Runge-Kutta method, Eq. 109 with the Butcher tableau of Tab. 3.
// * The force of the gas on each planet is evaluated once per update, by direct summation over all cells
//   (mode 1) or after removing the axisymmetric part of the density (mode 2), and used to update the
//   planetary velocities.
// * The potential of cell 5 is that of the star and of the planets where they are at the beginning of the update.
//
// Reading G33 (the paper gives the integrator and the two force modes, nothing else):
//   - y = positions and velocities in the frame rotating at the constant rate Omega_f about Z, Cartesian components;
//     f(t, y) = gravity of the star (at the origin, GM = gm_star; no indirect term: the paper describes none) and of
//     the other planets (unsoftened) + Coriolis and centrifugal accelerations (2 Om v_y + Om^2 x, -2 Om v_x + Om^2 y, 0),
//     so that no transcendental function is evaluated anywhere;
//   - gas -> planet acceleration: G sum_cells dm (x_c - x_p) / (|x_c - x_p|^2 + eps_p^2)^(3/2), dm = rho V (mode 1) or
//     (rho - <rho>_ring) V (mode 2), the same softening as the planet's potential so that it is minus the gradient
//     of the potential the gas feels; cell centre and volume as in the potential and Tab. 5; active cells only,
//     summed with i fastest, then j, then k;
//   - order inside one update: cell 5 (potential, planets at t^n) -> cell 6 (dt) -> cell 5a: kick v_p += dt a_gas(rho^n),
//     then the Cash-Karp step over dt (Fig. 2 is an image; 5a needs dt, so it runs right after cell 6).
// PARITY PINS: tests/test_oracle_planets.py.
#include "oracle_impl.hpp"

// Tab. 3: a_ij (rows 2..6), the fifth-order weights b_i (last row)
static const double CK_A[6][5] = {
    {0.0, 0.0, 0.0, 0.0, 0.0},
    {1.0 / 5.0, 0.0, 0.0, 0.0, 0.0},
    {3.0 / 40.0, 9.0 / 40.0, 0.0, 0.0, 0.0},
    {3.0 / 10.0, -9.0 / 10.0, 6.0 / 5.0, 0.0, 0.0},
    {-11.0 / 54.0, 5.0 / 2.0, -70.0 / 27.0, 35.0 / 27.0, 0.0},
    {1631.0 / 55296.0, 175.0 / 512.0, 575.0 / 13824.0, 44275.0 / 110592.0, 253.0 / 4096.0}};
static const double CK_B[6] = {37.0 / 378.0, 0.0, 250.0 / 621.0, 125.0 / 594.0, 0.0, 512.0 / 1771.0};

// f(y) of Eq. 108 for n planets; y = [x y z vx vy vz] per planet
static void planet_rhs(const oracle_ctx& c, const double* y, double* f) {
  const int n = c.npl;
  const double om = c.p.omega_frame, gms = c.p.gm_star;
  for (int p = 0; p < n; ++p) {
    const double* s = y + 6 * p;
    const double r2 = (s[0] * s[0] + s[1] * s[1]) + s[2] * s[2];
    const double ir3 = 1.0 / (r2 * std::sqrt(r2));
    double ax = -(gms * ir3) * s[0], ay = -(gms * ir3) * s[1], az = -(gms * ir3) * s[2];
    for (int q = 0; q < n; ++q) {
      if (q == p) continue;
      const double* o = y + 6 * q;
      const double dx = s[0] - o[0], dy = s[1] - o[1], dz = s[2] - o[2];
      const double d2 = (dx * dx + dy * dy) + dz * dz;
      const double w = c.pl_gm[q] / (d2 * std::sqrt(d2));
      ax = ax - w * dx; ay = ay - w * dy; az = az - w * dz;
    }
    ax = ax + ((2.0 * om) * s[4] + (om * om) * s[0]);
    ay = ay + ((om * om) * s[1] - (2.0 * om) * s[3]);
    double* o = f + 6 * p;
    o[0] = s[3]; o[1] = s[4]; o[2] = s[5]; o[3] = ax; o[4] = ay; o[5] = az;
  }
}

// One Cash-Karp step of size h (Eq. 109)
void orc_planets_rk5(oracle_ctx& c, double h) {
  const int m = 6 * c.npl;
  if (m == 0) return;
  double y[6 * ORC_MAX_PLANETS], yt[6 * ORC_MAX_PLANETS], k[6][6 * ORC_MAX_PLANETS];
  for (int p = 0; p < c.npl; ++p)
    for (int d = 0; d < 3; ++d) { y[6 * p + d] = c.pl_x[p][d]; y[6 * p + 3 + d] = c.pl_v[p][d]; }
  for (int i = 0; i < 6; ++i) {
    for (int q = 0; q < m; ++q) {
      double acc = 0.0;
      for (int j = 0; j < i; ++j) acc = acc + CK_A[i][j] * k[j][q];
      yt[q] = y[q] + h * acc;
    }
    planet_rhs(c, yt, k[i]);
  }
  for (int q = 0; q < m; ++q) {
    double acc = 0.0;
    for (int i = 0; i < 6; ++i) acc = acc + CK_B[i] * k[i][q];
    y[q] = y[q] + h * acc;
  }
  for (int p = 0; p < c.npl; ++p)
    for (int d = 0; d < 3; ++d) { c.pl_x[p][d] = y[6 * p + d]; c.pl_v[p][d] = y[6 * p + 3 + d]; }
}

// Acceleration of planet p due to the gas, per unit G: sum dm (x_c - x_p) / (d^2 + eps^2)^(3/2)
void orc_gas_force(const oracle_ctx& c, int p, double F[3]) {
  const double xp = c.pl_x[p][0], yp = c.pl_x[p][1], zp = c.pl_x[p][2];
  const double eps2 = c.pl_eps[p] * c.pl_eps[p];
  double Fx = 0.0, Fy = 0.0, Fz = 0.0;
  for (int k = c.k0(); k < c.k1(); ++k)
    for (int j = c.j0(); j < c.j1(); ++j) {
      double R, z;
      if (c.geometry == ORC_SPHERICAL) { R = c.yc[j] * c.sin_zc[k]; z = c.yc[j] * c.cos_zc[k]; }
      else { R = c.yc[j]; z = c.zc[k]; }
      const double vol = c.Vj[j] * c.syk[k];
      double mean = 0.0;
      if (c.force_mode == 2) {   // the axisymmetric part: the mean of the ring
        for (int i = c.i0(); i < c.i1(); ++i) mean = mean + c.rho[c.id(i, j, k)];
        mean = mean / (double)c.nx;
      }
      const double ddz = z - zp;
      for (int i = c.i0(); i < c.i1(); ++i) {
        const double x = R * c.cos_xc[i], y = R * c.sin_xc[i];
        const double ddx = x - xp, ddy = y - yp;
        const double d2 = ((ddx * ddx + ddy * ddy) + ddz * ddz) + eps2;
        const double w = ((c.rho[c.id(i, j, k)] - mean) * vol) / (d2 * std::sqrt(d2));
        Fx = Fx + w * ddx; Fy = Fy + w * ddy; Fz = Fz + w * ddz;
      }
    }
  F[0] = Fx; F[1] = Fy; F[2] = Fz;
}

// cell 5a: kick by the gas force of this update, then the Cash-Karp step over dt
void orc_planets_update(oracle_ctx& c) {
  if (c.npl == 0) return;
  if (c.force_mode != 0) {
    double F[ORC_MAX_PLANETS][3];
    for (int p = 0; p < c.npl; ++p) orc_gas_force(c, p, F[p]);   // all forces from the same positions
    for (int p = 0; p < c.npl; ++p)
      for (int d = 0; d < 3; ++d) {
        c.pl_f[p][d] = c.pl_gconst * F[p][d];
        c.pl_v[p][d] = c.pl_v[p][d] + c.dt * c.pl_f[p][d];
      }
  }
  orc_planets_rk5(c, c.dt);
}

extern "C" int oracle_set_planets(oracle_ctx* c, int n, const double* gm, const double* eps, const double* pos,
                                  const double* vel, int force_mode, double gconst) {
  if (!c || n < 0 || n > ORC_MAX_PLANETS || force_mode < 0 || force_mode > 2) return -1;
  if (n > 0 && (c->geometry == ORC_CARTESIAN || !c->hasx || !gm || !eps || !pos || !vel)) return -1;
  c->npl = n; c->force_mode = force_mode; c->pl_gconst = gconst;
  for (int p = 0; p < n; ++p) {
    c->pl_gm[p] = gm[p]; c->pl_eps[p] = eps[p];
    for (int d = 0; d < 3; ++d) { c->pl_x[p][d] = pos[3 * p + d]; c->pl_v[p][d] = vel[3 * p + d]; c->pl_f[p][d] = 0.0; }
  }
  if (n > 0) c->has_pot = true;
  return 0;
}

extern "C" int oracle_get_planets(oracle_ctx* c, double* pos, double* vel, double* gas_acc) {
  if (!c) return -1;
  for (int p = 0; p < c->npl; ++p)
    for (int d = 0; d < 3; ++d) {
      if (pos) pos[3 * p + d] = c->pl_x[p][d];
      if (vel) vel[3 * p + d] = c->pl_v[p][d];
      if (gas_acc) gas_acc[3 * p + d] = c->pl_f[p][d];
    }
  return c->npl;
}

// Test hooks: one Cash-Karp step of size h on the planets as they stand; the gas acceleration (per unit G) on planet p
extern "C" int oracle_planets_rk5(oracle_ctx* c, double h) { if (!c) return -1; orc_planets_rk5(*c, h); return 0; }
extern "C" int oracle_gas_force(oracle_ctx* c, int p, double* F) {
  if (!c || p < 0 || p >= c->npl || !F) return -1;
  orc_gas_force(*c, p, F);
  return 0;
}

// ---- cell 5b: change of the frame's rotation rate, Eq. 44 --------------------------------------------
// v_phi^c = v_phi^b - (Omega_f' - Omega_f) r sin(theta), the geometric factor taken at the centre of the face that
// carries v_phi, i.e. R_x(j, k) of Tab. 5.  Live planets are carried into the new frame the same way
// (v' = v - dOmega z^ x x), the fixed-orbit planet keeps its azimuth (its phase is re-based).  The paper does not say
// how Omega_f' is chosen (reading G33): the caller supplies it between updates.
extern "C" int oracle_set_omega_frame(oracle_ctx* c, double omega_new) {
  if (!c || c->midstep) return -1;
  if (c->geometry == ORC_CARTESIAN) return -1;   // no rotation; constant in the shearing sheet
  const double dom = omega_new - c->p.omega_frame;
  for (int k = 0; k < c->TZ; ++k)
    for (int j = 0; j < c->TY; ++j) {
      const double corr = dom * c->Rx(j, k);
      for (int i = 0; i < c->TX; ++i) c->vx[c->id(i, j, k)] = c->vx[c->id(i, j, k)] - corr;
    }
  for (int p = 0; p < c->npl; ++p) {
    const double x = c->pl_x[p][0], y = c->pl_x[p][1];
    c->pl_v[p][0] = c->pl_v[p][0] + dom * y;
    c->pl_v[p][1] = c->pl_v[p][1] - dom * x;
  }
  // fixed-orbit planet: same azimuth now, new drift rate afterwards
  const double phip = c->p.planet_phi0 + (c->p.planet_omega - c->p.omega_frame) * c->t;
  c->p.planet_phi0 = phip - (c->p.planet_omega - omega_new) * c->t;
  c->p.omega_frame = omega_new;
  return 0;
}

// ---- diagnostics: sum reductions over the whole mesh ("mass or angular momentum ... sum") -------------------
// out[0] = mass sum rho V; out[1..3] = the X, Y, Z momenta of Tab. 2 (X = angular momentum on curvilinear
// meshes), each cell carrying the mean of its left and right momenta (Eqs. 49-50); out[4] = internal energy sum e V
// (adiabatic; 0 otherwise).  Active cells, i fastest; the ghost fill of cell 2 is applied first (the upper-face
// velocities of the last active row and plane live in the ghosts; the next update starts with the same fill).
extern "C" int oracle_diagnostics(oracle_ctx* c, double* out) {
  if (!c || !out || c->midstep) return -1;
  oracle_ctx& o = *c;
  orc_bc_fill(o, o.rho, o.e, o.vx, o.vy, o.vz);
  orc_momenta(o);
  double m = 0.0, px = 0.0, py = 0.0, pz = 0.0, en = 0.0;
  for (int k = o.k0(); k < o.k1(); ++k)
    for (int j = o.j0(); j < o.j1(); ++j) {
      const double vol = o.Vj[j] * o.syk[k];
      for (int i = o.i0(); i < o.i1(); ++i) {
        const size_t l = o.id(i, j, k);
        m = m + o.rho[l] * vol;
        if (o.hasx) px = px + (0.5 * (o.pxm[l] + o.pxp[l])) * vol;
        if (o.hasy) py = py + (0.5 * (o.pym[l] + o.pyp[l])) * vol;
        if (o.hasz) pz = pz + (0.5 * (o.pzm[l] + o.pzp[l])) * vol;
        if (o.eos == ORC_ADIABATIC) en = en + o.e[l] * vol;
      }
    }
  out[0] = m; out[1] = px; out[2] = py; out[3] = pz; out[4] = en;
  return 0;
}
