// geometry.cpp -- mesh and the 1-D geometric coefficient tables of Tab. 5.
// CPU oracle, TEST INFRASTRUCTURE (see fargo_oracle.h).
#include "oracle_impl.hpp"

// Ghost-inclusive edges: active edges as given; ghost edges continue the mesh outward with the
// width of the adjacent active cell (the paper does not say).
static vec extend_edges(const double* act, int n, int ng, double lo, double hi) {
  vec a(n + 1);
  for (int j = 0; j <= n; ++j) a[j] = act ? act[j] : lo + (double)j * ((hi - lo) / (double)n);
  vec e(n + 2 * ng + 1);
  for (int j = 0; j <= n; ++j) e[ng + j] = a[j];
  const double w0 = a[1] - a[0], w1 = a[n] - a[n - 1];
  for (int g = 1; g <= ng; ++g) {
    e[ng - g] = a[0] - (double)g * w0;
    e[ng + n + g] = a[n] + (double)g * w1;
  }
  return e;
}

void orc_build_tables(oracle_ctx& c, const oracle_mesh& m) {
  const int TY = c.TY, TZ = c.TZ, TX = c.TX;
  const double dx = c.dx;
  c.ye = extend_edges(m.yedges, c.ny, c.ngy, m.ymin, m.ymax);
  c.ze = extend_edges(m.zedges, c.nz, c.ngz, m.zmin, m.zmax);

  // ---- j tables ------------------------------------------------------------------------------
  c.yc.resize(TY); c.inv_yc.resize(TY); c.inv_ye.resize(TY + 1);
  c.LY.resize(TY); c.invLY.resize(TY); c.DY.resize(TY); c.invDY.resize(TY);
  c.sxj.resize(TY); c.syj.resize(TY + 1); c.szj.resize(TY); c.invVj.resize(TY); c.Vj.resize(TY);
  c.Rxj.resize(TY); c.invRxj.resize(TY); c.LXj.resize(TY); c.invLXj.resize(TY);
  c.Rzj.resize(TY); c.invRzj.resize(TY);
  for (int j = 0; j <= TY; ++j) c.inv_ye[j] = 1.0 / c.ye[j];
  for (int j = 0; j < TY; ++j) {
    const double y0 = c.ye[j], y1 = c.ye[j + 1];
    c.yc[j] = 0.5 * (y0 + y1);
    c.inv_yc[j] = 1.0 / c.yc[j];
    c.LY[j] = y1 - y0;
    c.invLY[j] = 1.0 / c.LY[j];
  }
  for (int j = 0; j < TY; ++j) {
    c.DY[j] = (j == 0) ? c.LY[0] : c.yc[j] - c.yc[j - 1];
    c.invDY[j] = 1.0 / c.DY[j];
  }
  for (int j = 0; j < TY; ++j) {
    const double y0 = c.ye[j], y1 = c.ye[j + 1];
    switch (c.geometry) {
      case ORC_CARTESIAN:
        c.sxj[j] = y1 - y0;
        c.szj[j] = dx * (y1 - y0);
        c.invVj[j] = 1.0 / (y1 - y0);
        c.Rxj[j] = 1.0; c.Rzj[j] = 1.0;
        break;
      case ORC_CYLINDRICAL:
        c.sxj[j] = y1 - y0;
        c.szj[j] = (0.5 * dx) * (y1 * y1 - y0 * y0);
        c.invVj[j] = 2.0 / ((y1 * y1 - y0 * y0) * dx);
        c.Rxj[j] = c.yc[j]; c.Rzj[j] = 1.0;
        break;
      default:  // spherical
        c.sxj[j] = 0.5 * (y1 * y1 - y0 * y0);
        c.szj[j] = (0.5 * dx) * (y1 * y1 - y0 * y0);
        c.invVj[j] = 3.0 / ((y1 * y1 * y1 - y0 * y0 * y0) * dx);
        c.Rxj[j] = c.yc[j]; c.Rzj[j] = c.yc[j];
        break;
    }
    c.Vj[j] = 1.0 / c.invVj[j];
    c.invRxj[j] = 1.0 / c.Rxj[j];
    c.invRzj[j] = 1.0 / c.Rzj[j];
    c.LXj[j] = dx * c.Rxj[j];
    c.invLXj[j] = 1.0 / c.LXj[j];
  }
  for (int j = 0; j <= TY; ++j) {  // lower-face coefficient s_y^j needs the edge value
    const double y0 = c.ye[j];
    c.syj[j] = (c.geometry == ORC_CARTESIAN) ? 1.0 : (c.geometry == ORC_CYLINDRICAL) ? y0 * dx : (y0 * y0) * dx;
  }

  // ---- k tables ------------------------------------------------------------------------------
  c.zc.resize(TZ); c.dz.resize(TZ); c.invdz.resize(TZ); c.dzc.resize(TZ); c.invdzc.resize(TZ);
  c.sxk.resize(TZ); c.syk.resize(TZ); c.inv_syk.resize(TZ); c.szk.resize(TZ + 1);
  c.Rxk.resize(TZ); c.invRxk.resize(TZ);
  c.sin_zc.resize(TZ); c.cos_zc.resize(TZ); c.sin_ze.resize(TZ + 1); c.cos_ze.resize(TZ + 1); c.cot_ze.resize(TZ + 1);
  c.cot_zc.resize(TZ); c.inv_sin_ze.resize(TZ + 1);
  for (int k = 0; k <= TZ; ++k) {
    c.sin_ze[k] = std::sin(c.ze[k]);
    c.cos_ze[k] = std::cos(c.ze[k]);
    c.cot_ze[k] = c.cos_ze[k] / c.sin_ze[k];
    c.inv_sin_ze[k] = 1.0 / c.sin_ze[k];
    c.szk[k] = (c.geometry == ORC_SPHERICAL) ? c.sin_ze[k] : 1.0;
  }
  for (int k = 0; k < TZ; ++k) {
    const double z0 = c.ze[k], z1 = c.ze[k + 1];
    c.zc[k] = 0.5 * (z0 + z1);
    c.dz[k] = z1 - z0;
    c.invdz[k] = 1.0 / c.dz[k];
    c.sin_zc[k] = std::sin(c.zc[k]);
    c.cos_zc[k] = std::cos(c.zc[k]);
    c.cot_zc[k] = c.cos_zc[k] / c.sin_zc[k];
    c.sxk[k] = z1 - z0;
    switch (c.geometry) {
      case ORC_CARTESIAN: c.syk[k] = dx * (z1 - z0); c.Rxk[k] = 1.0; break;
      case ORC_CYLINDRICAL: c.syk[k] = z1 - z0; c.Rxk[k] = 1.0; break;
      default: c.syk[k] = c.cos_ze[k] - c.cos_ze[k + 1]; c.Rxk[k] = c.sin_zc[k]; break;
    }
    c.inv_syk[k] = 1.0 / c.syk[k];
    c.invRxk[k] = 1.0 / c.Rxk[k];
  }
  for (int k = 0; k < TZ; ++k) {
    c.dzc[k] = (k == 0) ? c.dz[0] : c.zc[k] - c.zc[k - 1];
    c.invdzc[k] = 1.0 / c.dzc[k];
  }

  // ---- azimuth of cell centres (potential only) ------------------------------------------------
  c.cos_xc.resize(TX); c.sin_xc.resize(TX);
  for (int i = 0; i < TX; ++i) {
    const double x = c.xmin + ((double)(i - c.ngx) + 0.5) * dx;
    c.cos_xc[i] = std::cos(x);
    c.sin_xc[i] = std::sin(x);
  }
}
