// viscosity.cpp -- sub-step 7d: viscous stress tensor and force (App. B), 2-D cylindrical
// (phi, r) form needed by config 3: Eqs. B2 and B5.  Centring: diagonal
// terms at cell centres, tau_phi_r at the cell corner with the lowest phi and r.  Readings G24.
// CPU oracle, TEST INFRASTRUCTURE (see fargo_oracle.h).
#include "oracle_impl.hpp"

void orc_source_d(oracle_ctx& c) {
  if (orc_visc3d_on(c)) { orc_source_d3(c); return; }   // 3-D meshes, all geometries: viscosity3d.cpp
  c.vxd = c.vxc; c.vyd = c.vyc; c.vzd = c.vzc;
  const bool on = c.p.nu > 0.0 && c.geometry == ORC_CYLINDRICAL && c.hasx && c.hasy && !c.hasz && c.xwrap;
  if (!on) return;   // other geometries: SURVEY.md 8(f) NEXT-1
  const double dt = c.dt, nu = c.p.nu, two3 = 2.0 / 3.0, invdx = 1.0 / c.dx;
  const size_t n = c.ncell();
  vec tpp(n, 0.0), trr(n, 0.0), tpr(n, 0.0);
  const int k = 0;
  const vec &vx = c.vxc, &vy = c.vyc, &rho = c.rho;
#pragma omp parallel for schedule(static)   // OpenMP build only: cell-independent body
  for (int j = 0; j < c.TY; ++j)
    for (int i = 0; i < c.TX; ++i) {
      const size_t l = c.id(i, j, k), lip = c.id(c.xw(i + 1), j, k), lim = c.id(c.xw(i - 1), j, k);
      const double il = c.invLX(j, k);
      if (j + 1 < c.TY) {
        const size_t ljp = c.id(i, j + 1, k);
        const double div = c.invV(j, k) * ((vx[lip] - vx[l]) * c.Sx(j, k) + (vy[ljp] * c.Sy(j + 1, k) - vy[l] * c.Sy(j, k)));
        const double mrn = -(rho[l] * nu);
        tpp[l] = mrn * (2.0 * ((vx[lip] - vx[l]) * il + (0.5 * (vy[l] + vy[ljp])) * c.inv_yc[j]) - two3 * div);
        trr[l] = mrn * (2.0 * ((vy[ljp] - vy[l]) * c.invLY[j]) - two3 * div);
      }
      if (j >= 1) {
        const size_t ljm = c.id(i, j - 1, k), limjm = c.id(c.xw(i - 1), j - 1, k);
        const double rhob = 0.25 * (((rho[l] + rho[lim]) + rho[ljm]) + rho[limjm]);
        const double ilf = c.inv_ye[j] * invdx;   // 1/(r_f dphi)
        tpr[l] = -(rhob * nu) * (((vx[l] - vx[ljm]) * c.invDY[j] - (0.5 * (vx[l] + vx[ljm])) * c.inv_ye[j])
                                 + (vy[l] - vy[lim]) * ilf);
      }
    }
#pragma omp parallel for schedule(static)   // OpenMP build only: cell-independent body
  for (int j = 1; j < c.TY - 1; ++j)
    for (int i = 0; i < c.TX; ++i) {
      const size_t l = c.id(i, j, k), lip = c.id(c.xw(i + 1), j, k), lim = c.id(c.xw(i - 1), j, k);
      const size_t ljp = c.id(i, j + 1, k), ljm = c.id(i, j - 1, k);
      const double il = c.invLX(j, k), ilf = c.inv_ye[j] * invdx;
      const double y0 = c.ye[j], y1 = c.ye[j + 1];
      {   // B5, azimuthal: (1/r^2) d_r(r^2 tau_phi_r) + (1/r) d_phi tau_phi_phi
        const double a = (((y1 * y1) * tpr[ljp] - (y0 * y0) * tpr[l]) * (c.inv_yc[j] * c.inv_yc[j])) * c.invLY[j];
        const double b = (tpp[l] - tpp[lim]) * il;
        c.vxd[l] = vx[l] - dt * ((2.0 / (rho[l] + rho[lim])) * (a + b));
      }
      if (j >= 2) {   // B5, radial: (1/r) d_r(r tau_rr) + (1/r) d_phi tau_r_phi - tau_phi_phi / r
        const double a = ((c.yc[j] * trr[l] - c.yc[j - 1] * trr[ljm]) * c.inv_ye[j]) * c.invDY[j];
        const double b = (tpr[lip] - tpr[l]) * ilf;
        const double d = (0.5 * (tpp[l] + tpp[ljm])) * c.inv_ye[j];
        c.vyd[l] = vy[l] - dt * ((2.0 / (rho[l] + rho[ljm])) * ((a + b) - d));
      }
    }
}
