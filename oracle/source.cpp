// source.cpp -- the operator-split source step, box 7 of Fig. 2: sub-steps 7a, 7b, 7c, 7d.
// CPU oracle, TEST INFRASTRUCTURE (see fargo_oracle.h).  Every loop covers the whole allocated
// array and computes wherever its stencil is in bounds; elsewhere the input is passed through.
// Only active cells are meaningful afterwards (the ghost fill of cell 9 overwrites the rest).
#include "oracle_impl.hpp"

static inline double pressure(const oracle_ctx& c, size_t l) {   // cell 4: Eq. 6 or Eq. 7
  return c.eos == ORC_ADIABATIC ? (c.p.gamma - 1.0) * c.e[l] : (c.e[l] * c.e[l]) * c.rho[l];
}

// ---- 7a: pressure gradient, potential gradient, centrifugal terms (Eqs. 27, 32-38, 53) ----------
// All three components read the state at the beginning of the sub-step (reading G18).
void orc_source_a(oracle_ctx& c) {
  const double dt = c.dt, om = c.p.omega_frame;
  const bool curv = c.geometry != ORC_CARTESIAN, sph = c.geometry == ORC_SPHERICAL;
#pragma omp parallel for collapse(2) schedule(static)   // OpenMP build only (liboracle_omp.so): cell-independent body
  for (int k = 0; k < c.TZ; ++k)
    for (int j = 0; j < c.TY; ++j)
      for (int i = 0; i < c.TX; ++i) {
        const size_t l = c.id(i, j, k);
        const bool ipok = c.xwrap || i + 1 < c.TX;
        const int ip = c.xw(i + 1);
        double vxb = c.vx[l], vyb = c.vy[l], vzb = c.vz[l];
        if (c.hasx && (c.xwrap || i >= 1)) {   // Eq. 53: density at the face = arithmetic mean
          const size_t lm = c.id(c.xw(i - 1), j, k);
          const double il = c.invLX(j, k);
          const double wf = (2.0 * il) / (c.rho[l] + c.rho[lm]);
          double acc = wf * (pressure(c, l) - pressure(c, lm));
          if (c.has_pot) acc = std::fma(c.phi[l] - c.phi[lm], il, acc);
          vxb = std::fma(-dt, acc, c.vx[l]);
        }
        if (c.hasy && j >= 1 && (!curv || ipok) && (!(sph && c.hasz) || k + 1 < c.TZ)) {
          const size_t lm = c.id(i, j - 1, k);
          const double il = c.invDY[j];
          const double wf = (2.0 * il) / (c.rho[l] + c.rho[lm]);
          double acc = wf * (pressure(c, l) - pressure(c, lm));
          if (c.has_pot) acc = std::fma(c.phi[l] - c.phi[lm], il, acc);
          vyb = std::fma(-dt, acc, c.vy[l]);
          if (curv) {   // Eq. 38: average the velocities, add the frame term, then square (G27)
            const double vphi = std::fma(0.25, ((c.vx[l] + c.vx[c.id(ip, j, k)]) + c.vx[lm]) + c.vx[c.id(ip, j - 1, k)],
                                         om * (c.ye[j] * c.Rxk[k]));
            double G = vphi * vphi;
            if (sph && c.hasz) {   // Eq. 36: + v_theta^2
              const double vth = 0.25 * (((c.vz[l] + c.vz[c.id(i, j, k + 1)]) + c.vz[lm]) + c.vz[c.id(i, j - 1, k + 1)]);
              G = std::fma(vth, vth, G);
            }
            vyb = std::fma(dt, G * c.inv_ye[j], vyb);
          }
          if (c.shear) {   // Eq. 29: + 2 Omega_f v_x - 4 A Omega_f y at the Y face; v_x averaged as in Eq. 38 (G32)
            const double vxa = 0.25 * (((c.vx[l] + c.vx[c.id(ip, j, k)]) + c.vx[lm]) + c.vx[c.id(ip, j - 1, k)]);
            vyb = std::fma(dt, std::fma(2.0 * om, vxa, -(((4.0 * c.p.oort_a) * om) * c.ye[j])), vyb);
          }
        }
        if (c.hasz && k >= 1 && (!sph || ipok)) {
          const size_t lm = c.id(i, j, k - 1);
          const double il = c.invDZ(j, k);
          const double wf = (2.0 * il) / (c.rho[l] + c.rho[lm]);
          double acc = wf * (pressure(c, l) - pressure(c, lm));
          if (c.has_pot) acc = std::fma(c.phi[l] - c.phi[lm], il, acc);
          vzb = std::fma(-dt, acc, c.vz[l]);
          if (sph) {   // Eq. 37: (v_phi^t)^2 cot(theta) / r at the theta face
            const double vphi = std::fma(0.25, ((c.vx[l] + c.vx[c.id(ip, j, k)]) + c.vx[lm]) + c.vx[c.id(ip, j, k - 1)],
                                         om * (c.yc[j] * c.sin_ze[k]));
            vzb = std::fma(dt, ((vphi * vphi) * c.cot_ze[k]) * c.inv_yc[j], vzb);
          }
        }
        c.vxb[l] = vxb; c.vyb[l] = vyb; c.vzb[l] = vzb;
      }
}

// ---- 7b: von Neumann-Richtmyer artificial viscosity, component-wise (readings G8, G19) ----
void orc_source_b(oracle_ctx& c) {
  const double dt = c.dt, cq2 = c.p.cvnr2;
  const size_t n = c.ncell();
  vec qx(n, 0.0), qy(n, 0.0), qz(n, 0.0), dvx(n, 0.0), dvy(n, 0.0), dvz(n, 0.0);
#pragma omp parallel for collapse(2) schedule(static)   // OpenMP build only (liboracle_omp.so): cell-independent body
  for (int k = 0; k < c.TZ; ++k)
    for (int j = 0; j < c.TY; ++j)
      for (int i = 0; i < c.TX; ++i) {
        const size_t l = c.id(i, j, k);
        if (c.hasx && (c.xwrap || i + 1 < c.TX)) {
          const double d = c.vxb[c.id(c.xw(i + 1), j, k)] - c.vxb[l];
          dvx[l] = d; qx[l] = d < 0.0 ? (cq2 * c.rho[l]) * (d * d) : 0.0;
        }
        if (c.hasy && j + 1 < c.TY) {
          const double d = c.vyb[c.id(i, j + 1, k)] - c.vyb[l];
          dvy[l] = d; qy[l] = d < 0.0 ? (cq2 * c.rho[l]) * (d * d) : 0.0;
        }
        if (c.hasz && k + 1 < c.TZ) {
          const double d = c.vzb[c.id(i, j, k + 1)] - c.vzb[l];
          dvz[l] = d; qz[l] = d < 0.0 ? (cq2 * c.rho[l]) * (d * d) : 0.0;
        }
      }
#pragma omp parallel for collapse(2) schedule(static)   // OpenMP build only (liboracle_omp.so): cell-independent body
  for (int k = 0; k < c.TZ; ++k)
    for (int j = 0; j < c.TY; ++j)
      for (int i = 0; i < c.TX; ++i) {
        const size_t l = c.id(i, j, k);
        double vxc = c.vxb[l], vyc = c.vyb[l], vzc = c.vzb[l];
        if (c.hasx && (c.xwrap || i >= 1)) {
          const size_t lm = c.id(c.xw(i - 1), j, k);
          const double wf = (2.0 * c.invLX(j, k)) / (c.rho[l] + c.rho[lm]);
          vxc = std::fma(-dt, wf * (qx[l] - qx[lm]), c.vxb[l]);
        }
        if (c.hasy && j >= 1) {
          const size_t lm = c.id(i, j - 1, k);
          const double wf = (2.0 * c.invDY[j]) / (c.rho[l] + c.rho[lm]);
          vyc = std::fma(-dt, wf * (qy[l] - qy[lm]), c.vyb[l]);
        }
        if (c.hasz && k >= 1) {
          const size_t lm = c.id(i, j, k - 1);
          const double wf = (2.0 * c.invDZ(j, k)) / (c.rho[l] + c.rho[lm]);
          vzc = std::fma(-dt, wf * (qz[l] - qz[lm]), c.vzb[l]);
        }
        c.vxc[l] = vxc; c.vyc[l] = vyc; c.vzc[l] = vzc;
        double ec = c.e[l];
        if (c.eos == ORC_ADIABATIC) {   // heating -q_d dv_d / Delta_d, same dv as in q (G19)
          double h = (qx[l] * dvx[l]) * c.invLX(j, k);
          h = std::fma(qy[l] * dvy[l], c.invLY[j], h);
          h = std::fma(qz[l] * dvz[l], c.invLZ(j, k), h);
          ec = std::fma(-dt, h, c.e[l]);
        }
        c.ec[l] = ec;
      }
}

// ---- 7c: compression work, time-centred form valid for gamma-law gases (G19) --------
void orc_source_c(oracle_ctx& c) {
  const double hd = (0.5 * c.dt) * (c.p.gamma - 1.0);
#pragma omp parallel for collapse(2) schedule(static)   // OpenMP build only (liboracle_omp.so): cell-independent body
  for (int k = 0; k < c.TZ; ++k)
    for (int j = 0; j < c.TY; ++j)
      for (int i = 0; i < c.TX; ++i) {
        const size_t l = c.id(i, j, k);
        double ed = c.ec[l];
        const bool ok = (!c.hasx || c.xwrap || i + 1 < c.TX) && (!c.hasy || j + 1 < c.TY) && (!c.hasz || k + 1 < c.TZ);
        if (c.eos == ORC_ADIABATIC && ok) {
          double tx = 0.0, ty = 0.0, tz = 0.0;
          if (c.hasx) tx = (c.vxc[c.id(c.xw(i + 1), j, k)] - c.vxc[l]) * c.Sx(j, k);
          if (c.hasy) ty = std::fma(c.vyc[c.id(i, j + 1, k)], c.Sy(j + 1, k), -(c.vyc[l] * c.Sy(j, k)));
          if (c.hasz) tz = std::fma(c.vzc[c.id(i, j, k + 1)], c.Sz(j, k + 1), -(c.vzc[l] * c.Sz(j, k)));
          const double D = c.invV(j, k) * ((tx + ty) + tz);
          const double a = hd * D;
          ed = (c.ec[l] * (1.0 - a)) / (1.0 + a);
        }
        c.ed[l] = ed;
      }
}
