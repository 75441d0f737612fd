// viscosity3d.cpp -- sub-step 7d on 3-D meshes in the three geometries: viscous stress tensor (App. B,
// Eqs. B1, B2, B3) and its force on the velocities (Eqs. B4, B5, B6).
// SURVEY.md 8(f) NEXT-1.  CPU oracle, TEST INFRASTRUCTURE (see fargo_oracle.h).
//
// Axes (Tab. 1): X = x | phi | phi,  Y = y | r | r,  Z = z | z | theta (colatitude).
// Centring: diagonal components at cell centres; t_xy at the middle of the Z-directed edge with the
// lowest x and y, i.e. at (i-1/2, j-1/2, k); t_xz at (i-1/2, j, k-1/2); t_yz at (i, j-1/2, k-1/2).
// Velocities sit on the lower faces (reading G1), so every derivative below is a centred two-point difference.
// Readings: G24 (u_r = v_r; the force is divided by the face-mean density, also in B4; density at an
// edge = mean of the four cells around it) and, new here, G31: a quantity needed where it is not stored (v_r at a
// centre, tau_phi_phi on a radial face, ...) is the arithmetic mean of its two nearest stored values; metric
// factors r, sin(theta), cot(theta) are taken at the position of the term (centre or edge tables).
// PARITY PINS: tests/test_oracle_viscosity3d.py (exact decay of a discrete shear wave and of a compressive wave,
// vanishing stress of uniform translations and rigid rotations about any axis at second order, constant-shear
// tensor components, agreement with the pinned 2-D cylindrical routine).
#include "oracle_impl.hpp"

namespace {

struct Metric {   // per-position inverse lengths, written out for one geometry at a time
  int geo;
  const oracle_ctx& c;
  double invdx;
  explicit Metric(const oracle_ctx& cc) : geo(cc.geometry), c(cc), invdx(1.0 / cc.dx) {}
  // 1 / (length of an X step) at: cell centre | radial face (j-1/2, k) | polar face (j, k-1/2)
  double ix_c(int j, int k) const { return c.invLX(j, k); }
  double ix_je(int j, int k) const {
    return geo == ORC_CARTESIAN ? invdx : (c.inv_ye[j] * invdx) * c.invRxk[k];
  }
  double ix_ke(int j, int k) const {
    if (geo == ORC_CARTESIAN) return invdx;
    if (geo == ORC_CYLINDRICAL) return c.inv_yc[j] * invdx;
    return (c.inv_yc[j] * invdx) * c.inv_sin_ze[k];
  }
  // 1 / (length of a Z step) between centres k-1 and k at the radial face j-1/2
  double iz_je(int j, int k) const { return geo == ORC_SPHERICAL ? c.invdzc[k] * c.inv_ye[j] : c.invdzc[k]; }
};

}  // namespace

bool orc_visc3d_on(const oracle_ctx& c) { return c.p.nu > 0.0 && c.hasx && c.hasy && c.hasz; }

void orc_source_d3(oracle_ctx& c) {
  const Metric M(c);
  const int geo = c.geometry;
  const bool cyl = geo == ORC_CYLINDRICAL, sph = geo == ORC_SPHERICAL, curv = cyl || sph;
  const double dt = c.dt, nu = c.p.nu, two3 = 2.0 / 3.0;
  const size_t n = c.ncell();
  vec txx(n, 0.0), tyy(n, 0.0), tzz(n, 0.0), txy(n, 0.0), txz(n, 0.0), tyz(n, 0.0);
  const vec &vx = c.vxc, &vy = c.vyc, &vz = c.vzc, &rho = c.rho;

  // ---- stress tensor (B1 | B2 | B3) ----------------------------------------------------------------------
#pragma omp parallel for collapse(2) schedule(static)   // OpenMP build only (liboracle_omp.so): cell-independent body
  for (int k = 0; k < c.TZ; ++k)
    for (int j = 0; j < c.TY; ++j)
      for (int i = 0; i < c.TX; ++i) {
        const bool xp = c.xwrap || i + 1 < c.TX, xm = c.xwrap || i >= 1;
        const size_t l = c.id(i, j, k);
        const size_t lip = xp ? c.id(c.xw(i + 1), j, k) : l, lim = xm ? c.id(c.xw(i - 1), j, k) : l;
        if (xp && j + 1 < c.TY && k + 1 < c.TZ) {   // diagonal components, cell centre
          const size_t ljp = c.id(i, j + 1, k), lkp = c.id(i, j, k + 1);
          const double div = c.invV(j, k) * ((((vx[lip] - vx[l]) * c.Sx(j, k)) +
                                              (vy[ljp] * c.Sy(j + 1, k) - vy[l] * c.Sy(j, k))) +
                                             (vz[lkp] * c.Sz(j, k + 1) - vz[l] * c.Sz(j, k)));
          const double mrn = -(rho[l] * nu);
          const double vyc = 0.5 * (vy[l] + vy[ljp]), vzc = 0.5 * (vz[l] + vz[lkp]);   // G31
          double ex = (vx[lip] - vx[l]) * M.ix_c(j, k);          // d_x v_x | (1/r) d_phi v_phi | (1/(r sin)) d_phi v_phi
          if (curv) ex = ex + vyc * c.inv_yc[j];                 // + v_r / r                       (B2, B3)
          if (sph) ex = ex + (vzc * c.cot_zc[k]) * c.inv_yc[j];  // + v_theta cot(theta) / r        (B3)
          const double ey = (vy[ljp] - vy[l]) * c.invLY[j];      // d_y v_y | d_r v_r
          double ez = (vz[lkp] - vz[l]) * c.invLZ(j, k);         // d_z v_z | (1/r) d_theta v_theta
          if (sph) ez = ez + vyc * c.inv_yc[j];                  // + v_r / r                       (B3)
          txx[l] = mrn * (2.0 * ex - two3 * div);
          tyy[l] = mrn * (2.0 * ey - two3 * div);
          tzz[l] = mrn * (2.0 * ez - two3 * div);
        }
        if (xm && j >= 1) {   // t_xy = t_phi_r at (i-1/2, j-1/2, k)
          const size_t ljm = c.id(i, j - 1, k), limjm = c.id(c.xw(i - 1), j - 1, k);
          const double rhob = 0.25 * (((rho[l] + rho[lim]) + rho[ljm]) + rho[limjm]);
          double a = (vx[l] - vx[ljm]) * c.invDY[j];                              // d_y v_x | d_r v_phi
          if (curv) a = a - (0.5 * (vx[l] + vx[ljm])) * c.inv_ye[j];              // - v_phi / r
          txy[l] = -(rhob * nu) * (a + (vy[l] - vy[lim]) * M.ix_je(j, k));        // + d_x v_y | (1/r[sin]) d_phi v_r
        }
        if (xm && k >= 1) {   // t_xz = t_phi_z | t_phi_theta at (i-1/2, j, k-1/2)
          const size_t lkm = c.id(i, j, k - 1), limkm = c.id(c.xw(i - 1), j, k - 1);
          const double rhob = 0.25 * (((rho[l] + rho[lim]) + rho[lkm]) + rho[limkm]);
          double a;
          if (sph) a = ((vx[l] * c.invRxk[k] - vx[lkm] * c.invRxk[k - 1]) * c.sin_ze[k]) * c.invDZ(j, k);   // (sin/r) d_theta (v_phi / sin)
          else a = (vx[l] - vx[lkm]) * c.invDZ(j, k);                                                     // d_z v_x
          txz[l] = -(rhob * nu) * (a + (vz[l] - vz[lim]) * M.ix_ke(j, k));        // + d_x v_z | (1/(r sin)) d_phi v_theta
        }
        if (j >= 1 && k >= 1) {   // t_yz = t_r_z | t_r_theta at (i, j-1/2, k-1/2)
          const size_t ljm = c.id(i, j - 1, k), lkm = c.id(i, j, k - 1), ljmkm = c.id(i, j - 1, k - 1);
          const double rhob = 0.25 * (((rho[l] + rho[ljm]) + rho[lkm]) + rho[ljmkm]);
          double a = (vz[l] - vz[ljm]) * c.invDY[j];                              // d_y v_z | d_r v_theta
          if (sph) a = a - (0.5 * (vz[l] + vz[ljm])) * c.inv_ye[j];               // - v_theta / r          (B3)
          tyz[l] = -(rhob * nu) * (a + (vy[l] - vy[lkm]) * M.iz_je(j, k));        // + d_z v_y | (1/r) d_theta v_r
        }
      }

  // ---- force (B4 | B5 | B6), each divided by the face-mean density (G24) -----------------------------------
  c.vxd = c.vxc; c.vyd = c.vyc; c.vzd = c.vzc;   // pass-through where the stencil does not fit
#pragma omp parallel for collapse(2) schedule(static)   // OpenMP build only (liboracle_omp.so): cell-independent body
  for (int k = 1; k < c.TZ - 1; ++k)
    for (int j = 1; j < c.TY - 1; ++j)
      for (int i = 0; i < c.TX; ++i) {
        if (!c.xwrap && (i < 1 || i + 1 >= c.TX)) continue;
        const size_t l = c.id(i, j, k), lip = c.id(c.xw(i + 1), j, k), lim = c.id(c.xw(i - 1), j, k);
        const size_t ljp = c.id(i, j + 1, k), ljm = c.id(i, j - 1, k), lkp = c.id(i, j, k + 1), lkm = c.id(i, j, k - 1);
        const double y0 = c.ye[j], y1 = c.ye[j + 1];
        {   // X component, at (i-1/2, j, k)
          double a, s;
          if (curv) a = (((y1 * y1) * txy[ljp] - (y0 * y0) * txy[l]) * (c.inv_yc[j] * c.inv_yc[j])) * c.invLY[j];   // (1/r^2) d_r (r^2 t_phi_r)
          else a = (txy[ljp] - txy[l]) * c.invLY[j];                                                               // d_y t_xy
          const double b = (txx[l] - txx[lim]) * M.ix_c(j, k);                     // d_x t_xx | (1/r[sin]) d_phi t_phi_phi
          const double cc = (txz[lkp] - txz[l]) * c.invLZ(j, k);                  // d_z t_xz | (1/r) d_theta t_phi_theta
          s = (a + b) + cc;
          if (sph) {
            s = s + (0.5 * (txy[l] + txy[ljp])) * c.inv_yc[j];                               // + t_r_phi / r
            s = s + ((2.0 * (0.5 * (txz[l] + txz[lkp]))) * c.cot_zc[k]) * c.inv_yc[j];       // + 2 t_theta_phi cot / r
          }
          c.vxd[l] = vx[l] - dt * ((2.0 / (rho[l] + rho[lim])) * s);
        }
        {   // Y component, at (i, j-1/2, k)
          double a, cc, s;
          const double b = (txy[lip] - txy[l]) * M.ix_je(j, k);                    // d_x t_xy | (1/r[sin]) d_phi t_r_phi
          if (!curv) {
            a = (tyy[l] - tyy[ljm]) * c.invDY[j];                                  // d_y t_yy
            cc = (tyz[lkp] - tyz[l]) * c.invdz[k];                                 // d_z t_yz
            s = (a + b) + cc;
          } else if (cyl) {
            a = ((c.yc[j] * tyy[l] - c.yc[j - 1] * tyy[ljm]) * c.inv_ye[j]) * c.invDY[j];   // (1/r) d_r (r t_rr)
            cc = (tyz[lkp] - tyz[l]) * c.invdz[k];                                          // d_z t_rz
            s = ((a + b) - (0.5 * (txx[l] + txx[ljm])) * c.inv_ye[j]) + cc;                 // - t_phi_phi / r
          } else {
            a = ((((c.yc[j] * c.yc[j]) * tyy[l] - (c.yc[j - 1] * c.yc[j - 1]) * tyy[ljm])) * (c.inv_ye[j] * c.inv_ye[j])) * c.invDY[j];   // (1/r^2) d_r (r^2 t_rr)
            cc = ((tyz[lkp] * c.sin_ze[k + 1] - tyz[l] * c.sin_ze[k]) * c.invdz[k]) * (c.inv_ye[j] * c.invRxk[k]);   // (1/(r sin)) d_theta (t_r_theta sin)
            s = ((a + cc) + b) - ((0.5 * (tzz[l] + tzz[ljm])) + (0.5 * (txx[l] + txx[ljm]))) * c.inv_ye[j];          // - (t_theta_theta + t_phi_phi) / r
          }
          c.vyd[l] = vy[l] - dt * ((2.0 / (rho[l] + rho[ljm])) * s);
        }
        {   // Z component, at (i, j, k-1/2)
          double a, cc, s;
          const double b = (txz[lip] - txz[l]) * M.ix_ke(j, k);                    // d_x t_xz | (1/r) d_phi t_phi_z | (1/(r sin)) d_phi t_theta_phi
          if (!curv) {
            a = (tyz[ljp] - tyz[l]) * c.invLY[j];                                  // d_y t_yz
            cc = (tzz[l] - tzz[lkm]) * c.invdzc[k];                                // d_z t_zz
            s = (a + b) + cc;
          } else if (cyl) {
            a = ((y1 * tyz[ljp] - y0 * tyz[l]) * c.inv_yc[j]) * c.invLY[j];        // (1/r) d_r (r t_rz)
            cc = (tzz[l] - tzz[lkm]) * c.invdzc[k];                                // d_z t_zz
            s = (a + b) + cc;
          } else {
            a = ((((y1 * y1) * y1) * tyz[ljp] - ((y0 * y0) * y0) * tyz[l]) * ((c.inv_yc[j] * c.inv_yc[j]) * c.inv_yc[j])) * c.invLY[j];   // (1/r^3) d_r (r^3 t_r_theta)
            cc = ((tzz[l] * c.sin_zc[k] - tzz[lkm] * c.sin_zc[k - 1]) * c.invdzc[k]) * (c.inv_yc[j] * c.inv_sin_ze[k]);   // (1/(r sin)) d_theta (t_theta_theta sin)
            s = ((a + cc) + b) - ((0.5 * (txx[l] + txx[lkm])) * c.cot_ze[k]) * c.inv_yc[j];                              // - t_phi_phi cot / r
          }
          c.vzd[l] = vz[l] - dt * ((2.0 / (rho[l] + rho[lkm])) * s);
        }
      }
}
