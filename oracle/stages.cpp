// stages.cpp -- boundary fill (cells 2, 9), ring mean velocity (cell 3), potential (cell 5),
// time step (cell 6).  CPU oracle, TEST INFRASTRUCTURE (see fargo_oracle.h).
#include <algorithm>

#include "oracle_impl.hpp"

// ---- O1 / O7: ghost fill (kinds named at P:865, 877, 921, 948; formulas = reading G22) ----
// `normal` = the field is the velocity component normal to the boundary (stored on faces).
static void fill_dir(oracle_ctx& c, vec& a, int dir, bool normal) {
  const int N = dir == 0 ? c.nx : dir == 1 ? c.ny : c.nz;
  const int ng = dir == 0 ? c.ngx : dir == 1 ? c.ngy : c.ngz;
  if (ng == 0) return;
  const int m0 = ng, m1 = ng + N;
  const int P = dir == 0 ? c.TY : c.TX;                  // extents of the two other directions
  const int Q = dir == 2 ? c.TY : c.TZ;
#pragma omp parallel for collapse(2) schedule(static)   // OpenMP build only (liboracle_omp.so): lines are independent
  for (int q = 0; q < Q; ++q)
    for (int p = 0; p < P; ++p) {
      auto A = [&](int m) -> double& {
        return dir == 0 ? a[c.id(m, p, q)] : dir == 1 ? a[c.id(p, m, q)] : a[c.id(p, q, m)];
      };
      const int lo = c.bc[dir][0], hi = c.bc[dir][1];
      for (int g = 0; g < ng; ++g) {
        if (lo == ORC_PERIODIC) A(m0 - 1 - g) = A(m1 - 1 - g);
        else if (lo == ORC_OUTFLOW) A(m0 - 1 - g) = A(m0);
        else if (!normal) A(m0 - 1 - g) = A(m0 + g);
        if (hi == ORC_PERIODIC) A(m1 + g) = A(m0 + g);
        else if (hi == ORC_OUTFLOW) A(m1 + g) = A(m1 - 1);
        else if (!normal) A(m1 + g) = A(m1 - 1 - g);
      }
      if (normal && lo == ORC_REFLECTING) {   // wall face at rest, antisymmetric about it
        A(m0) = 0.0;
        for (int g = 1; g <= ng; ++g) A(m0 - g) = -A(m0 + g);
      }
      if (normal && hi == ORC_REFLECTING) {
        A(m1) = 0.0;
        for (int g = 1; g <= ng - 1; ++g) A(m1 + g) = -A(m1 - g);
      }
    }
}

void orc_bc_fill(oracle_ctx& c, vec& rho, vec& e, vec& vx, vec& vy, vec& vz) {
  for (int dir = 0; dir < 3; ++dir) {   // X, then Y, then Z so that edges and corners are filled
    fill_dir(c, rho, dir, false);
    fill_dir(c, e, dir, false);
    fill_dir(c, vx, dir, dir == 0);
    fill_dir(c, vy, dir, dir == 1);
    fill_dir(c, vz, dir, dir == 2);
  }
}

// ---- O2: v0_jk = (max_i v + min_i v)/2 per ring, ghost rings included (Eq. 72) ----------
void orc_vmean(oracle_ctx& c) {
#pragma omp parallel for collapse(2) schedule(static)   // OpenMP build only: rings are independent
  for (int k = 0; k < c.TZ; ++k)
    for (int j = 0; j < c.TY; ++j) {
      double v0 = 0.0;
      if (c.p.fargo_on) {
        double lo = c.vx[c.id(c.i0(), j, k)], hi = lo;
        for (int i = c.i0(); i < c.i1(); ++i) {
          const double v = c.vx[c.id(i, j, k)];
          lo = std::min(lo, v); hi = std::max(hi, v);
        }
        v0 = 0.5 * (hi + lo);
      }
      c.v0[c.rid(j, k)] = v0;
    }
}

// ---- O4: potential of the star and of a planet on a fixed circular orbit in the midplane --------
// Phi = -GM/|x| - G m_p / sqrt(|x - x_p|^2 + eps^2)   (reading G12: the paper prints no formula)
void orc_potential(oracle_ctx& c) {
  if (!c.has_pot) return;
  const double phip = c.p.planet_phi0 + (c.p.planet_omega - c.p.omega_frame) * c.t;
  const double xp = c.p.planet_r * std::cos(phip), yp = c.p.planet_r * std::sin(phip);
  const double eps2 = c.p.planet_eps * c.p.planet_eps;
#pragma omp parallel for collapse(2) schedule(static)   // OpenMP build only: cell-independent body
  for (int k = 0; k < c.TZ; ++k)
    for (int j = 0; j < c.TY; ++j) {
      double R, z, r;
      if (c.geometry == ORC_SPHERICAL) { R = c.yc[j] * c.sin_zc[k]; z = c.yc[j] * c.cos_zc[k]; r = c.yc[j]; }
      else { R = c.yc[j]; z = c.zc[k]; r = std::sqrt(R * R + z * z); }
      for (int i = 0; i < c.TX; ++i) {
        const double x = R * c.cos_xc[i], y = R * c.sin_xc[i];
        double phi = -(c.p.gm_star / r);
        if (c.npl > 0) {   // live planets (NEXT-2, reading G33): where they are at the beginning of the update
          for (int p = 0; p < c.npl; ++p) {
            const double ddx = x - c.pl_x[p][0], ddy = y - c.pl_x[p][1], ddz = z - c.pl_x[p][2];
            const double d2 = ((ddx * ddx + ddy * ddy) + ddz * ddz) + c.pl_eps[p] * c.pl_eps[p];
            phi = phi - c.pl_gm[p] / std::sqrt(d2);
          }
        } else if (c.p.planet_mass != 0.0) {
          const double ddx = x - xp, ddy = y - yp;
          const double d2 = ((ddx * ddx + ddy * ddy) + z * z) + eps2;
          phi = phi - c.p.planet_mass / std::sqrt(d2);
        }
        c.phi[c.id(i, j, k)] = phi;
      }
    }
}

// ---- O5: time step (Eq. 59; shear limit Eq. 73) ------------------------------
// Inverse form: I_n = 1/dt_n, "dt_i = min_j dt_ij" = max over directions of the rates.
// sqrt is monotone, so the max over cells is taken on the sum of squares and rooted once.
double orc_compute_dt(oracle_ctx& c, bool* clipped) {
  *clipped = false;
  const double gg1 = c.p.gamma * (c.p.gamma - 1.0);
  const double c3 = 4.0 * c.p.cvnr2;   // dt_3 = Delta/(4 C_q^2 |dv|)  (reading G8)
  const double c4 = 4.0 * c.p.nu;      // dt_4 = Delta^2/(4 nu)
  double M2 = 0.0;
#pragma omp parallel for collapse(2) schedule(static) reduction(max : M2)   // OpenMP build only: max is exact in any order
  for (int k = c.k0(); k < c.k1(); ++k)
    for (int j = c.j0(); j < c.j1(); ++j) {
      const double ilx = c.invLX(j, k), ily = c.invLY[j], ilz = c.invLZ(j, k);
      double ilmax = 0.0;
      if (c.hasx) ilmax = std::max(ilmax, ilx);
      if (c.hasy) ilmax = std::max(ilmax, ily);
      if (c.hasz) ilmax = std::max(ilmax, ilz);
      const double v0 = c.v0[c.rid(j, k)];
      for (int i = c.i0(); i < c.i1(); ++i) {
        const size_t l = c.id(i, j, k);
        double cs2 = (c.eos == ORC_ADIABATIC) ? (gg1 * c.e[l]) / c.rho[l] : c.e[l] * c.e[l];
        if (c.mhd && !c.mhd_passive) cs2 = cs2 + orc_mhd_alfven2(c, i, j, k);   // item 1: C_w^2 = C_s^2 + v_A^2
        const double I1sq = cs2 * (ilmax * ilmax);
        double I2 = 0.0, I3 = 0.0;
        if (c.hasx) {
          const double a = c.vx[l], b = c.vx[c.id(c.xw(i + 1), j, k)];
          I2 = std::max(I2, std::fabs(std::fma(0.5, a + b, -v0)) * ilx);
          I3 = std::max(I3, std::fabs(b - a) * ilx);
        }
        if (c.hasy) {
          const double a = c.vy[l], b = c.vy[c.id(i, j + 1, k)];
          I2 = std::max(I2, std::fabs(0.5 * (a + b)) * ily);
          I3 = std::max(I3, std::fabs(b - a) * ily);
        }
        if (c.hasz) {
          const double a = c.vz[l], b = c.vz[c.id(i, j, k + 1)];
          I2 = std::max(I2, std::fabs(0.5 * (a + b)) * ilz);
          I3 = std::max(I3, std::fabs(b - a) * ilz);
        }
        I3 = c3 * I3;
        const double I4 = c4 * (ilmax * ilmax);
        double Isq = std::fma(I4, I4, std::fma(I3, I3, std::fma(I2, I2, I1sq)));
        if (c.mhd && c.eta != 0.0) {   // item 5: dt_5 = Delta^2 / (4 eta)
          const double I5 = (4.0 * c.eta) * (ilmax * ilmax);
          Isq = std::fma(I5, I5, Isq);
        }
        M2 = std::max(M2, Isq);
      }
    }
  double dt = 1.0 / std::sqrt(M2);
  if (c.p.fargo_on) {   // Eq. 73 with V_X = v0_jk, C_0 = shear_c0 (reading G10)
    double s = 0.0;
#pragma omp parallel for collapse(2) schedule(static) reduction(max : s)
    for (int k = c.k0(); k < c.k1(); ++k)
      for (int j = c.j0(); j < c.j1() - 1; ++j)
        s = std::max(s, std::fabs(c.v0[c.rid(j, k)] * c.invLX(j, k) - c.v0[c.rid(j + 1, k)] * c.invLX(j + 1, k)));
    if (s > 0.0) dt = std::min(dt, c.p.shear_c0 / s);
  }
  dt = c.p.cfl * dt;
  if (c.p.dt_fixed > 0.0) dt = c.p.dt_fixed;
  if (c.p.t_stop > 0.0 && c.t + dt >= c.p.t_stop) { dt = c.p.t_stop - c.t; *clipped = true; }
  return dt;
}
