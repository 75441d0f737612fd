// tables.cpp -- see tables.h.  Surfaces of the lower faces and the inverse volume factor as products of
// a j-coefficient and a k-coefficient (Eqs. A1-A4): S_x = sxj*sxk, S_y = syj*syk, S_z = szj*szk,
// 1/V = invVj/syk.  Per geometry (Tab. 5), with (y0,y1) = radial edges, (z0,z1) = vertical/polar edges:
//   Cartesian    sxj = dy          syj = 1        szj = dx dy              invVj = 1/dy
//                sxk = dz          syk = dx dz    szk = 1
//   cylindrical  sxj = dr          syj = r0 dphi  szj = dphi (r1^2-r0^2)/2 invVj = 2/((r1^2-r0^2) dphi)
//                sxk = dz          syk = dz       szk = 1
//   spherical    sxj = (r1^2-r0^2)/2  syj = r0^2 dphi  szj = dphi (r1^2-r0^2)/2  invVj = 3/((r1^3-r0^3) dphi)
//                sxk = dtheta      syk = cos(t0)-cos(t1)   szk = sin(t0)
#include "tables.h"

#include <cmath>

namespace fg {

std::vector<double> ghosted_edges(const double* edges, int n, int ng, double lo, double hi) {
  std::vector<double> e((size_t)n + 2 * ng + 1);
  const double h = (hi - lo) / (double)n;
  for (int j = 0; j <= n; ++j) e[ng + j] = edges ? edges[j] : lo + (double)j * h;
  const double first = e[ng], last = e[ng + n];
  const double wlo = e[ng + 1] - first, whi = last - e[ng + n - 1];
  for (int g = 1; g <= ng; ++g) {
    e[ng - g] = first - (double)g * wlo;
    e[ng + n + g] = last + (double)g * whi;
  }
  return e;
}

static std::vector<double> reciprocal(const std::vector<double>& a) {
  std::vector<double> r(a.size());
  for (size_t n = 0; n < a.size(); ++n) r[n] = 1.0 / a[n];
  return r;
}

void build_tables(HostTables& t, int geometry, int TX, int TY, int TZ, int ngx, double xmin, double dx,
                  const std::vector<double>& ye, const std::vector<double>& ze) {
  const bool cart = geometry == 0, cyl = geometry == 1, sph = geometry == 2;
  t.ye = ye;
  t.ze = ze;

  // radial (j) tables
  t.yc.resize(TY); t.LY.resize(TY);
  for (int j = 0; j < TY; ++j) {
    t.yc[j] = 0.5 * (ye[j] + ye[j + 1]);
    t.LY[j] = ye[j + 1] - ye[j];
  }
  std::vector<double> DY(TY);
  for (int j = 0; j < TY; ++j) DY[j] = j ? t.yc[j] - t.yc[j - 1] : t.LY[0];   // centre-to-centre (reading G5)
  t.inv_ye = reciprocal(ye);
  t.inv_yc = reciprocal(t.yc);
  t.invLY = reciprocal(t.LY);
  t.invDY = reciprocal(DY);
  t.sxj.resize(TY); t.szj.resize(TY); t.invVj.resize(TY); t.Rxj.resize(TY); t.Rzj.resize(TY); t.LXj.resize(TY);
  t.syj.resize(TY + 1);
  for (int j = 0; j < TY; ++j) {
    const double y0 = ye[j], y1 = ye[j + 1];
    const double dsq = y1 * y1 - y0 * y0;
    if (cart) {
      t.sxj[j] = y1 - y0;
      t.szj[j] = dx * (y1 - y0);
      t.invVj[j] = 1.0 / (y1 - y0);
    } else if (cyl) {
      t.sxj[j] = y1 - y0;
      t.szj[j] = (0.5 * dx) * dsq;
      t.invVj[j] = 2.0 / (dsq * dx);
    } else {
      t.sxj[j] = 0.5 * dsq;
      t.szj[j] = (0.5 * dx) * dsq;
      t.invVj[j] = 3.0 / ((y1 * y1 * y1 - y0 * y0 * y0) * dx);
    }
    t.Rxj[j] = cart ? 1.0 : t.yc[j];   // R_x = 1 | r | r sin(theta) splits as Rxj * Rxk
    t.Rzj[j] = sph ? t.yc[j] : 1.0;    // R_z = 1 | 1 | r
    t.LXj[j] = dx * t.Rxj[j];
  }
  for (int j = 0; j <= TY; ++j) t.syj[j] = cart ? 1.0 : cyl ? ye[j] * dx : (ye[j] * ye[j]) * dx;
  t.invRxj = reciprocal(t.Rxj);
  t.invRzj = reciprocal(t.Rzj);
  t.invLXj = reciprocal(t.LXj);

  // vertical / polar (k) tables
  std::vector<double> cos_ze(TZ + 1);
  t.sin_ze.resize(TZ + 1); t.cot_ze.resize(TZ + 1); t.szk.resize(TZ + 1);
  t.inv_sin_ze.resize(TZ + 1); t.cot_zc.resize(TZ);
  for (int k = 0; k <= TZ; ++k) {
    t.sin_ze[k] = std::sin(ze[k]);
    cos_ze[k] = std::cos(ze[k]);
    t.cot_ze[k] = cos_ze[k] / t.sin_ze[k];
    t.inv_sin_ze[k] = 1.0 / t.sin_ze[k];
    t.szk[k] = sph ? t.sin_ze[k] : 1.0;
  }
  t.zc.resize(TZ); t.dz.resize(TZ); t.sin_zc.resize(TZ); t.cos_zc.resize(TZ);
  t.sxk.resize(TZ); t.syk.resize(TZ); t.Rxk.resize(TZ);
  for (int k = 0; k < TZ; ++k) {
    t.zc[k] = 0.5 * (ze[k] + ze[k + 1]);
    t.dz[k] = ze[k + 1] - ze[k];
    t.sin_zc[k] = std::sin(t.zc[k]);
    t.cos_zc[k] = std::cos(t.zc[k]);
    t.cot_zc[k] = t.cos_zc[k] / t.sin_zc[k];
    t.sxk[k] = ze[k + 1] - ze[k];
    t.syk[k] = cart ? dx * (ze[k + 1] - ze[k]) : cyl ? ze[k + 1] - ze[k] : cos_ze[k] - cos_ze[k + 1];
    t.Rxk[k] = sph ? t.sin_zc[k] : 1.0;
  }
  std::vector<double> dzc(TZ);
  for (int k = 0; k < TZ; ++k) dzc[k] = k ? t.zc[k] - t.zc[k - 1] : t.dz[0];
  t.invdz = reciprocal(t.dz);
  t.invdzc = reciprocal(dzc);
  t.inv_syk = reciprocal(t.syk);
  t.invRxk = reciprocal(t.Rxk);

  // azimuth of the cell centres (potential only)
  t.cos_xc.resize(TX); t.sin_xc.resize(TX);
  for (int i = 0; i < TX; ++i) {
    const double x = xmin + ((double)(i - ngx) + 0.5) * dx;
    t.cos_xc[i] = std::cos(x);
    t.sin_xc[i] = std::sin(x);
  }
}

}  // namespace fg
