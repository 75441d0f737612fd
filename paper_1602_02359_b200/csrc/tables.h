// tables.h -- host-side 1-D geometric coefficient tables (Tab. 5; Eqs. A1-A4),
// lengths, and the trigonometric tables.  Built once per context in fp64 with libm and uploaded; the
// kernels never evaluate a transcendental.  Product code.
#pragma once
#include <vector>

namespace fg {

struct HostTables {
  // ghost-inclusive; "j" tables have TY entries (TY+1 where they live on edges), "k" tables TZ (TZ+1)
  std::vector<double> ye, yc, inv_ye, inv_yc, LY, invLY, invDY;
  std::vector<double> sxj, syj, szj, invVj, Rxj, invRxj, LXj, invLXj, Rzj, invRzj;
  std::vector<double> ze, zc, dz, invdz, invdzc, sxk, syk, inv_syk, szk, Rxk, invRxk;
  std::vector<double> sin_zc, cos_zc, sin_ze, cot_ze, cos_xc, sin_xc;
  std::vector<double> cot_zc, inv_sin_ze;   // cos/sin at polar centres, 1/sin at polar edges (3-D viscous stress)
};

// edges: n+1 active edges or nullptr (uniform lo + j*(hi-lo)/n); ng ghost layers continue the mesh with
// the width of the adjacent active cell.
std::vector<double> ghosted_edges(const double* edges, int n, int ng, double lo, double hi);

void build_tables(HostTables& t, int geometry, int TX, int TY, int TZ, int ngx, double xmin, double dx,
                  const std::vector<double>& ye, const std::vector<double>& ze);

}  // namespace fg
