// k_visc3d.cu -- sub-step 7d on 3-D meshes in the three geometries: viscous stress tensor
// (App. B, Eqs. B1 | B2 | B3) and its force on the velocities (Eqs. B4 | B5 | B6).
// Axes (Tab. 1): X = x | phi | phi, Y = y | r | r, Z = z | z | theta.  Centring: diagonal components at
// cell centres, t_xy at (i-1/2, j-1/2, k), t_xz at (i-1/2, j, k-1/2), t_yz at (i, j-1/2, k-1/2).  Readings G24
// (face-mean density divides the force, four-cell mean density at an edge) and G31 (two-point means, metric
// factors at the position of the term): DESIGN.md section 2.
// Two kernels, one thread per cell over the whole allocated array: the six components (read rho, v: 4 reals;
// write 6), then the force (read rho, v, 6 components; write 3).  Product code: shares nothing with oracle/.
#include "kernels.h"

namespace fg {

template <typename T, int GEO>
struct VMetric {   // inverse lengths of an X step and of a Z step at the staggered positions
  const Dev<T>& d;
  __device__ __forceinline__ T ix_c(int j, int k) const { return d.invLX(j, k); }
  __device__ __forceinline__ T ix_je(int j, int k) const {   // at the radial face (j-1/2, k)
    return GEO == GEO_CART ? d.invdx : (d.inv_ye[j] * d.invdx) * d.invRxk[k];
  }
  __device__ __forceinline__ T ix_ke(int j, int k) const {   // at the polar face (j, k-1/2)
    if (GEO == GEO_CART) return d.invdx;
    if (GEO == GEO_CYL) return d.inv_yc[j] * d.invdx;
    return (d.inv_yc[j] * d.invdx) * d.inv_sin_ze[k];
  }
  __device__ __forceinline__ T iz_je(int j, int k) const {   // between centres k-1 and k at the radial face j-1/2
    return GEO == GEO_SPH ? d.invdzc[k] * d.inv_ye[j] : d.invdzc[k];
  }
};

template <typename T, int GEO>
__global__ void __launch_bounds__(128) k_visc3d_tensor(const Dev<T> d, const T* __restrict__ rho, const T* __restrict__ vx,
                                                       const T* __restrict__ vy, const T* __restrict__ vz,
                                                       T* __restrict__ txx, T* __restrict__ tyy, T* __restrict__ tzz,
                                                       T* __restrict__ txy, T* __restrict__ txz, T* __restrict__ tyz) {
  constexpr bool CURV = GEO != GEO_CART, SPH = GEO == GEO_SPH;
  if (d.ctl->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
  if (i >= d.TX) return;
  const VMetric<T, GEO> M{d};
  const T nu = d.nu, two3 = T(2) / T(3);
  const bool xp = d.xwrap || i + 1 < d.TX, xm = d.xwrap || i >= 1;
  const long long l = d.id(i, j, k);
  const long long lip = xp ? d.id(d.xw(i + 1), j, k) : l, lim = xm ? d.id(d.xw(i - 1), j, k) : l;
  T oxx = T(0), oyy = T(0), ozz = T(0), oxy = T(0), oxz = T(0), oyz = T(0);
  if (xp && j + 1 < d.TY && k + 1 < d.TZ) {   // diagonal components, cell centre
    const long long ljp = l + d.pitch, lkp = l + d.plane;
    const T div = d.invV(j, k) * ((((vx[lip] - vx[l]) * d.Sx(j, k)) + (vy[ljp] * d.Sy(j + 1, k) - vy[l] * d.Sy(j, k))) +
                                  (vz[lkp] * d.Sz(j, k + 1) - vz[l] * d.Sz(j, k)));
    const T mrn = -(rho[l] * nu);
    const T vyc = T(0.5) * (vy[l] + vy[ljp]), vzc = T(0.5) * (vz[l] + vz[lkp]);
    T ex = (vx[lip] - vx[l]) * M.ix_c(j, k);
    if (CURV) ex = ex + vyc * d.inv_yc[j];                  // + v_r / r                 (B2, B3)
    if (SPH) ex = ex + (vzc * d.cot_zc[k]) * d.inv_yc[j];   // + v_theta cot(theta) / r  (B3)
    const T ey = (vy[ljp] - vy[l]) * d.invLY[j];
    T ez = (vz[lkp] - vz[l]) * d.invLZ(j, k);
    if (SPH) ez = ez + vyc * d.inv_yc[j];                   // + v_r / r                 (B3)
    oxx = mrn * (T(2) * ex - two3 * div);
    oyy = mrn * (T(2) * ey - two3 * div);
    ozz = mrn * (T(2) * ez - two3 * div);
  }
  if (xm && j >= 1) {   // t_xy = t_phi_r
    const long long ljm = l - d.pitch, limjm = lim - d.pitch;
    const T rhob = T(0.25) * (((rho[l] + rho[lim]) + rho[ljm]) + rho[limjm]);
    T a = (vx[l] - vx[ljm]) * d.invDY[j];
    if (CURV) a = a - (T(0.5) * (vx[l] + vx[ljm])) * d.inv_ye[j];   // - v_phi / r
    oxy = -(rhob * nu) * (a + (vy[l] - vy[lim]) * M.ix_je(j, k));
  }
  if (xm && k >= 1) {   // t_xz = t_phi_z | t_phi_theta
    const long long lkm = l - d.plane, limkm = lim - d.plane;
    const T rhob = T(0.25) * (((rho[l] + rho[lim]) + rho[lkm]) + rho[limkm]);
    T a;
    if (SPH) a = ((vx[l] * d.invRxk[k] - vx[lkm] * d.invRxk[k - 1]) * d.sin_ze[k]) * d.invDZ(j, k);   // (sin/r) d_theta (v_phi/sin)
    else a = (vx[l] - vx[lkm]) * d.invDZ(j, k);
    oxz = -(rhob * nu) * (a + (vz[l] - vz[lim]) * M.ix_ke(j, k));
  }
  if (j >= 1 && k >= 1) {   // t_yz = t_r_z | t_r_theta
    const long long ljm = l - d.pitch, lkm = l - d.plane, ljmkm = ljm - d.plane;
    const T rhob = T(0.25) * (((rho[l] + rho[ljm]) + rho[lkm]) + rho[ljmkm]);
    T a = (vz[l] - vz[ljm]) * d.invDY[j];
    if (SPH) a = a - (T(0.5) * (vz[l] + vz[ljm])) * d.inv_ye[j];    // - v_theta / r
    oyz = -(rhob * nu) * (a + (vy[l] - vy[lkm]) * M.iz_je(j, k));
  }
  txx[l] = oxx; tyy[l] = oyy; tzz[l] = ozz; txy[l] = oxy; txz[l] = oxz; tyz[l] = oyz;
}

template <typename T, int GEO>
__global__ void __launch_bounds__(128) k_visc3d_force(const Dev<T> d, const T* __restrict__ rho, const T* __restrict__ vx,
                                                      const T* __restrict__ vy, const T* __restrict__ vz,
                                                      const T* __restrict__ txx, const T* __restrict__ tyy,
                                                      const T* __restrict__ tzz, const T* __restrict__ txy,
                                                      const T* __restrict__ txz, const T* __restrict__ tyz,
                                                      T* __restrict__ vxd, T* __restrict__ vyd, T* __restrict__ vzd) {
  constexpr bool CURV = GEO != GEO_CART, CYL = GEO == GEO_CYL, SPH = GEO == GEO_SPH;
  if (d.ctl->done) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
  if (i >= d.TX) return;
  const VMetric<T, GEO> M{d};
  const T dt = (T)d.ctl->dt;
  const long long l = d.id(i, j, k);
  T ox = vx[l], oy = vy[l], oz = vz[l];   // pass-through where the stencil does not fit
  const bool fits = k >= 1 && k + 1 < d.TZ && j >= 1 && j + 1 < d.TY && (d.xwrap || (i >= 1 && i + 1 < d.TX));
  if (fits) {
    const long long lip = d.id(d.xw(i + 1), j, k), lim = d.id(d.xw(i - 1), j, k);
    const long long ljp = l + d.pitch, ljm = l - d.pitch, lkp = l + d.plane, lkm = l - d.plane;
    const T y0 = d.ye[j], y1 = d.ye[j + 1];
    {   // X component, at (i-1/2, j, k)
      T a;
      if (CURV) a = (((y1 * y1) * txy[ljp] - (y0 * y0) * txy[l]) * (d.inv_yc[j] * d.inv_yc[j])) * d.invLY[j];
      else a = (txy[ljp] - txy[l]) * d.invLY[j];
      const T b = (txx[l] - txx[lim]) * M.ix_c(j, k);
      const T cc = (txz[lkp] - txz[l]) * d.invLZ(j, k);
      T s = (a + b) + cc;
      if (SPH) {
        s = s + (T(0.5) * (txy[l] + txy[ljp])) * d.inv_yc[j];                              // + t_r_phi / r
        s = s + ((T(2) * (T(0.5) * (txz[l] + txz[lkp]))) * d.cot_zc[k]) * d.inv_yc[j];     // + 2 t_theta_phi cot / r
      }
      ox = vx[l] - dt * (rdiv(T(2), rho[l] + rho[lim]) * s);
    }
    {   // Y component, at (i, j-1/2, k)
      T a, cc, s;
      const T b = (txy[lip] - txy[l]) * M.ix_je(j, k);
      if (!CURV) {
        a = (tyy[l] - tyy[ljm]) * d.invDY[j];
        cc = (tyz[lkp] - tyz[l]) * d.invdz[k];
        s = (a + b) + cc;
      } else if (CYL) {
        a = ((d.yc[j] * tyy[l] - d.yc[j - 1] * tyy[ljm]) * d.inv_ye[j]) * d.invDY[j];
        cc = (tyz[lkp] - tyz[l]) * d.invdz[k];
        s = ((a + b) - (T(0.5) * (txx[l] + txx[ljm])) * d.inv_ye[j]) + cc;                 // - t_phi_phi / r
      } else {
        a = ((((d.yc[j] * d.yc[j]) * tyy[l] - (d.yc[j - 1] * d.yc[j - 1]) * tyy[ljm])) * (d.inv_ye[j] * d.inv_ye[j])) * d.invDY[j];
        cc = ((tyz[lkp] * d.sin_ze[k + 1] - tyz[l] * d.sin_ze[k]) * d.invdz[k]) * (d.inv_ye[j] * d.invRxk[k]);
        s = ((a + cc) + b) - ((T(0.5) * (tzz[l] + tzz[ljm])) + (T(0.5) * (txx[l] + txx[ljm]))) * d.inv_ye[j];
      }
      oy = vy[l] - dt * (rdiv(T(2), rho[l] + rho[ljm]) * s);
    }
    {   // Z component, at (i, j, k-1/2)
      T a, cc, s;
      const T b = (txz[lip] - txz[l]) * M.ix_ke(j, k);
      if (!CURV) {
        a = (tyz[ljp] - tyz[l]) * d.invLY[j];
        cc = (tzz[l] - tzz[lkm]) * d.invdzc[k];
        s = (a + b) + cc;
      } else if (CYL) {
        a = ((y1 * tyz[ljp] - y0 * tyz[l]) * d.inv_yc[j]) * d.invLY[j];
        cc = (tzz[l] - tzz[lkm]) * d.invdzc[k];
        s = (a + b) + cc;
      } else {
        a = ((((y1 * y1) * y1) * tyz[ljp] - ((y0 * y0) * y0) * tyz[l]) * ((d.inv_yc[j] * d.inv_yc[j]) * d.inv_yc[j])) * d.invLY[j];
        cc = ((tzz[l] * d.sin_zc[k] - tzz[lkm] * d.sin_zc[k - 1]) * d.invdzc[k]) * (d.inv_yc[j] * d.inv_sin_ze[k]);
        s = ((a + cc) + b) - ((T(0.5) * (txx[l] + txx[lkm])) * d.cot_ze[k]) * d.inv_yc[j];
      }
      oz = vz[l] - dt * (rdiv(T(2), rho[l] + rho[lkm]) * s);
    }
  }
  vxd[l] = ox; vyd[l] = oy; vzd[l] = oz;
}

// ---- 7d as ONE pass (wrapped X): (rho, v_c) -> v_d on ACTIVE cells, the stress tensor never stored --------------
// 56 B per cell instead of 184 B.  The ghost fill of cell 9 follows 7d and overwrites every ghost of v, so only active
// cells are produced; their stencils reach one ghost layer, where v_c is what 7a-7c computed there (the unfused
// kernels run over the whole allocated array for that reason).
//   X : a warp owns 32 consecutive cells of a row; values at i-1 / i+1 cross lanes by shuffle; lanes 0 and 31 are
//       recomputed halo (30 cells stored per warp).
//   Z : the thread marches along Z with the rows j-1, j, j+1 of (rho, v) of the current and the leading plane in
//       registers; t_xz, t_yz of the leading plane and the diagonal of the previous plane are carried.
//   Y : the components at j-1 (diagonal) and j+1 (t_xy, t_yz) are recomputed from the neighbour rows (the warps of a
//       block are consecutive rows, so L1/L2 serve them): 7 component evaluations per cell instead of 4.
// Every component and force expression is the one of k_visc3d_tensor / k_visc3d_force (same operands, same order),
// so the result is bit-identical to the two-kernel sequence on active cells.
constexpr int V3W = 4;     // warps (consecutive rows) per block
constexpr int V3IN = 30;   // cells stored per warp
constexpr int V3_PF = 2;   // planes ahead that are prefetched into L1

template <typename T> __device__ __forceinline__ T v_up1(T v) { return __shfl_up_sync(0xffffffffu, v, 1); }
template <typename T> __device__ __forceinline__ T v_dn1(T v) { return __shfl_down_sync(0xffffffffu, v, 1); }

template <typename T> struct Rows3 { T m, c, p; };   // rows j-1, j, j+1 of one array at one plane

template <typename T, int GEO>
__global__ void __launch_bounds__(32 * V3W) k_visc3d_fused(const Dev<T> d, const T* __restrict__ rho, const T* __restrict__ vx,
                                                           const T* __restrict__ vy, const T* __restrict__ vz,
                                                           T* __restrict__ vxd, T* __restrict__ vyd, T* __restrict__ vzd,
                                                           const int CH) {
  constexpr bool CURV = GEO != GEO_CART, CYL = GEO == GEO_CYL, SPH = GEO == GEO_SPH;
  if (d.ctl->done) return;
  const int lane = threadIdx.x;
  const int j = d.ngy + blockIdx.y * V3W + threadIdx.y;
  if (j >= d.ngy + d.ny) return;   // whole warps leave together
  const int m0 = d.ngz + blockIdx.z * CH;
  const int m1 = (m0 + CH < d.ngz + d.nz) ? m0 + CH : d.ngz + d.nz;   // planes this thread writes: [m0, m1)
  const int iu = blockIdx.x * V3IN - 1 + lane;   // un-wrapped cell index
  int i = iu % d.nx; if (i < 0) i += d.nx;
  const bool store = lane >= 1 && lane <= 30 && iu < d.nx;
  const VMetric<T, GEO> M{d};
  const T nu = d.nu, two3 = T(2) / T(3), dt = (T)d.ctl->dt;
  const long long P = d.plane, R = d.pitch;
  const long long base = d.id(i, j, 0);

  auto pf = [](const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); };
  auto load3 = [&](const T* __restrict__ a, const long long l) { Rows3<T> r; r.m = a[l - R]; r.c = a[l]; r.p = a[l + R]; return r; };
  // diagonal components at the centre of (row jj, plane kk): u0, u1 = vx at i, i+1; w0, w1 = vy at jj, jj+1; z0, z1 = vz at kk, kk+1
  auto diag = [&](const int jj, const int kk, const T rh, const T u0, const T u1, const T w0, const T w1, const T z0, const T z1,
                  T& oxx, T& oyy, T& ozz) {
    const T div = d.invV(jj, kk) * ((((u1 - u0) * d.Sx(jj, kk)) + (w1 * d.Sy(jj + 1, kk) - w0 * d.Sy(jj, kk))) +
                                    (z1 * d.Sz(jj, kk + 1) - z0 * d.Sz(jj, kk)));
    const T mrn = -(rh * nu);
    const T vyc = T(0.5) * (w0 + w1), vzc = T(0.5) * (z0 + z1);
    T ex = (u1 - u0) * M.ix_c(jj, kk);
    if (CURV) ex = ex + vyc * d.inv_yc[jj];
    if (SPH) ex = ex + (vzc * d.cot_zc[kk]) * d.inv_yc[jj];
    const T ey = (w1 - w0) * d.invLY[jj];
    T ez = (z1 - z0) * d.invLZ(jj, kk);
    if (SPH) ez = ez + vyc * d.inv_yc[jj];
    oxx = mrn * (T(2) * ex - two3 * div);
    oyy = mrn * (T(2) * ey - two3 * div);
    ozz = mrn * (T(2) * ez - two3 * div);
  };
  // t_xy at (i-1/2, jj-1/2, kk): r.. = rho at (i,jj) (i-1,jj) (i,jj-1) (i-1,jj-1); u = vx at jj, jj-1; w = vy(jj) at i, i-1
  auto f_txy = [&](const int jj, const int kk, const T r00, const T r10, const T r01, const T r11, const T u, const T um,
                   const T w, const T wm) {
    const T rhob = T(0.25) * (((r00 + r10) + r01) + r11);
    T a = (u - um) * d.invDY[jj];
    if (CURV) a = a - (T(0.5) * (u + um)) * d.inv_ye[jj];
    return -(rhob * nu) * (a + (w - wm) * M.ix_je(jj, kk));
  };
  // t_xz at (i-1/2, jj, kk-1/2): rho at (i,kk) (i-1,kk) (i,kk-1) (i-1,kk-1); u = vx at kk, kk-1; z = vz(kk) at i, i-1
  auto f_txz = [&](const int jj, const int kk, const T r00, const T r10, const T r01, const T r11, const T u, const T um,
                   const T z, const T zm) {
    const T rhob = T(0.25) * (((r00 + r10) + r01) + r11);
    T a;
    if (SPH) a = ((u * d.invRxk[kk] - um * d.invRxk[kk - 1]) * d.sin_ze[kk]) * d.invDZ(jj, kk);
    else a = (u - um) * d.invDZ(jj, kk);
    return -(rhob * nu) * (a + (z - zm) * M.ix_ke(jj, kk));
  };
  // t_yz at (i, jj-1/2, kk-1/2): rho at (jj,kk) (jj-1,kk) (jj,kk-1) (jj-1,kk-1); z = vz(kk) at jj, jj-1; w = vy(jj) at kk, kk-1
  auto f_tyz = [&](const int jj, const int kk, const T r00, const T r10, const T r01, const T r11, const T z, const T zm,
                   const T w, const T wm) {
    const T rhob = T(0.25) * (((r00 + r10) + r01) + r11);
    T a = (z - zm) * d.invDY[jj];
    if (SPH) a = a - (T(0.5) * (z + zm)) * d.inv_ye[jj];
    return -(rhob * nu) * (a + (w - wm) * M.iz_je(jj, kk));
  };

  // current plane c = n - 1 (rows j-1, j, j+1) and what is carried from earlier planes
  Rows3<T> rc = load3(rho, base + (long long)(m0 - 1) * P), uc = load3(vx, base + (long long)(m0 - 1) * P);
  Rows3<T> wc = load3(vy, base + (long long)(m0 - 1) * P), zc = load3(vz, base + (long long)(m0 - 1) * P);
  T txz_c = T(0), tyz_c = T(0), tyzp_c = T(0), tzz_b = T(0), txx_b = T(0), rho_b = T(1);   // rho_b: rho(i, j, c-1)
  const T y0 = d.ye[j], y1 = d.ye[j + 1];

#pragma unroll 1
  for (int n = m0; n <= m1; ++n) {
    const long long ln = base + (long long)n * P;
    if (n + V3_PF <= m1) {   // rows of a later plane into L1 (the block's other warps prefetch the rows between)
      const long long lq = ln + (long long)V3_PF * P;
      pf(rho + lq); pf(vx + lq); pf(vy + lq); pf(vz + lq);
      if (threadIdx.y == 0) { pf(rho + lq - R); pf(vx + lq - R); pf(vy + lq - R); pf(vz + lq - R); }
      if (threadIdx.y == V3W - 1) { pf(rho + lq + R); pf(vx + lq + R); pf(vy + lq + R); pf(vz + lq + R); }
    }
    const Rows3<T> rn = load3(rho, ln), un = load3(vx, ln), wn = load3(vy, ln), zn = load3(vz, ln);
    const int c = n - 1;
    // ---- leading plane n: t_xz(j, n), t_yz(j, n), t_yz(j+1, n) ----
    const T txz_n = f_txz(j, n, rn.c, v_up1(rn.c), rc.c, v_up1(rc.c), un.c, uc.c, zn.c, v_up1(zn.c));
    const T tyz_n = f_tyz(j, n, rn.c, rn.m, rc.c, rc.m, zn.c, zn.m, wn.c, wc.c);
    const T tyzp_n = f_tyz(j + 1, n, rn.p, rn.c, rc.p, rc.c, zn.p, zn.c, wn.p, wc.p);
    // ---- current plane c: diagonal at j and j-1, t_xy at j and j+1 ----
    T txx, tyy, tzz, txx_m, tyy_m, tzz_m;
    diag(j, c, rc.c, uc.c, v_dn1(uc.c), wc.c, wc.p, zc.c, zn.c, txx, tyy, tzz);
    diag(j - 1, c, rc.m, uc.m, v_dn1(uc.m), wc.m, wc.c, zc.m, zn.m, txx_m, tyy_m, tzz_m);
    const T rcl = v_up1(rc.c);
    const T txy = f_txy(j, c, rc.c, rcl, rc.m, v_up1(rc.m), uc.c, uc.m, wc.c, v_up1(wc.c));
    const T txy_p = f_txy(j + 1, c, rc.p, v_up1(rc.p), rc.c, rcl, uc.p, uc.c, wc.p, v_up1(wc.p));
    // ---- force on the three lower faces of cell (i, j, c): Eqs. B4 | B5 | B6 ----
    T ox, oy, oz;
    {   // X component, at (i-1/2, j, c)
      T a;
      if (CURV) a = (((y1 * y1) * txy_p - (y0 * y0) * txy) * (d.inv_yc[j] * d.inv_yc[j])) * d.invLY[j];
      else a = (txy_p - txy) * d.invLY[j];
      const T b = (txx - v_up1(txx)) * M.ix_c(j, c);
      const T cc = (txz_n - txz_c) * d.invLZ(j, c);
      T s = (a + b) + cc;
      if (SPH) {
        s = s + (T(0.5) * (txy + txy_p)) * d.inv_yc[j];
        s = s + ((T(2) * (T(0.5) * (txz_c + txz_n))) * d.cot_zc[c]) * d.inv_yc[j];
      }
      ox = uc.c - dt * (rdiv(T(2), rc.c + rcl) * s);
    }
    {   // Y component, at (i, j-1/2, c)
      T a, cc, s;
      const T b = (v_dn1(txy) - txy) * M.ix_je(j, c);
      if (!CURV) {
        a = (tyy - tyy_m) * d.invDY[j];
        cc = (tyz_n - tyz_c) * d.invdz[c];
        s = (a + b) + cc;
      } else if (CYL) {
        a = ((d.yc[j] * tyy - d.yc[j - 1] * tyy_m) * d.inv_ye[j]) * d.invDY[j];
        cc = (tyz_n - tyz_c) * d.invdz[c];
        s = ((a + b) - (T(0.5) * (txx + txx_m)) * d.inv_ye[j]) + cc;
      } else {
        a = ((((d.yc[j] * d.yc[j]) * tyy - (d.yc[j - 1] * d.yc[j - 1]) * tyy_m)) * (d.inv_ye[j] * d.inv_ye[j])) * d.invDY[j];
        cc = ((tyz_n * d.sin_ze[c + 1] - tyz_c * d.sin_ze[c]) * d.invdz[c]) * (d.inv_ye[j] * d.invRxk[c]);
        s = ((a + cc) + b) - ((T(0.5) * (tzz + tzz_m)) + (T(0.5) * (txx + txx_m))) * d.inv_ye[j];
      }
      oy = wc.c - dt * (rdiv(T(2), rc.c + rc.m) * s);
    }
    {   // Z component, at (i, j, c-1/2)
      T a, cc, s;
      const T b = (v_dn1(txz_c) - txz_c) * M.ix_ke(j, c);
      if (!CURV) {
        a = (tyzp_c - tyz_c) * d.invLY[j];
        cc = (tzz - tzz_b) * d.invdzc[c];
        s = (a + b) + cc;
      } else if (CYL) {
        a = ((y1 * tyzp_c - y0 * tyz_c) * d.inv_yc[j]) * d.invLY[j];
        cc = (tzz - tzz_b) * d.invdzc[c];
        s = (a + b) + cc;
      } else {
        a = ((((y1 * y1) * y1) * tyzp_c - ((y0 * y0) * y0) * tyz_c) * ((d.inv_yc[j] * d.inv_yc[j]) * d.inv_yc[j])) * d.invLY[j];
        cc = ((tzz * d.sin_zc[c] - tzz_b * d.sin_zc[c - 1]) * d.invdzc[c]) * (d.inv_yc[j] * d.inv_sin_ze[c]);
        s = ((a + cc) + b) - ((T(0.5) * (txx + txx_b)) * d.cot_ze[c]) * d.inv_yc[j];
      }
      oz = zc.c - dt * (rdiv(T(2), rc.c + rho_b) * s);
    }
    const bool st = store && c >= m0;
    const long long lc = base + (long long)c * P;
    st_if(vxd + lc, ox, st);
    st_if(vyd + lc, oy, st);
    st_if(vzd + lc, oz, st);
    // ---- shift the Z window ----
    rho_b = rc.c;
    rc = rn; uc = un; wc = wn; zc = zn;
    txz_c = txz_n; tyz_c = tyz_n; tyzp_c = tyzp_n; tzz_b = tzz; txx_b = txx;
  }
}

template <typename T, int GEO>
static int launch_v3(const Dev<T>& d, const T* rho, const T* vx, const T* vy, const T* vz, T* const* t, T* vxd, T* vyd,
                     T* vzd, cudaStream_t s) {
  dim3 b(128), g((d.TX + 127) / 128, d.TY, d.TZ);
  k_visc3d_tensor<T, GEO><<<g, b, 0, s>>>(d, rho, vx, vy, vz, t[0], t[1], t[2], t[3], t[4], t[5]);
  k_visc3d_force<T, GEO><<<g, b, 0, s>>>(d, rho, vx, vy, vz, t[0], t[1], t[2], t[3], t[4], t[5], vxd, vyd, vzd);
  return 2;
}

// cell 7d on a 3-D mesh: (rho, vc) -> vd, with the six stress components in t[0..5] = xx yy zz xy xz yz
template <typename T>
int launch_source_d3(const Dev<T>& d, const T* rho, const T* vxc, const T* vyc, const T* vzc, T* const* t, T* vxd, T* vyd,
                     T* vzd, cudaStream_t s) {
  switch (d.geometry) {
    case GEO_CART: return launch_v3<T, GEO_CART>(d, rho, vxc, vyc, vzc, t, vxd, vyd, vzd, s);
    case GEO_CYL: return launch_v3<T, GEO_CYL>(d, rho, vxc, vyc, vzc, t, vxd, vyd, vzd, s);
    default: return launch_v3<T, GEO_SPH>(d, rho, vxc, vyc, vzc, t, vxd, vyd, vzd, s);
  }
}

template <typename T, int GEO>
static int launch_v3f(const Dev<T>& d, const T* rho, const T* vx, const T* vy, const T* vz, T* vxd, T* vyd, T* vzd,
                      cudaStream_t s) {
  // chunk the march so that the grid fills the machine a few times over; each chunk re-reads 2 planes
  const int ntile = (d.nx + V3IN - 1) / V3IN, nrow = (d.ny + V3W - 1) / V3W;
  static int slots = 0;   // per instantiation
  if (!slots) slots = resident_slots(k_visc3d_fused<T, GEO>, 32 * V3W, 0);
  const int CH = pick_chunk_len((long long)ntile * nrow, d.nz, 4, slots, 16);
  dim3 b(32, V3W), g(ntile, nrow, (d.nz + CH - 1) / CH);
  k_visc3d_fused<T, GEO><<<g, b, 0, s>>>(d, rho, vx, vy, vz, vxd, vyd, vzd, CH);
  return 1;
}

// cell 7d on a 3-D mesh with a wrapped X axis in one pass, active cells only (the stress tensor is never stored)
template <typename T>
bool source_d3_fused_ok(const Dev<T>& d) { return d.hasx && d.hasy && d.hasz && d.xwrap; }

template <typename T>
int launch_source_d3_fused(const Dev<T>& d, const T* rho, const T* vxc, const T* vyc, const T* vzc, T* vxd, T* vyd,
                           T* vzd, cudaStream_t s) {
  switch (d.geometry) {
    case GEO_CART: return launch_v3f<T, GEO_CART>(d, rho, vxc, vyc, vzc, vxd, vyd, vzd, s);
    case GEO_CYL: return launch_v3f<T, GEO_CYL>(d, rho, vxc, vyc, vzc, vxd, vyd, vzd, s);
    default: return launch_v3f<T, GEO_SPH>(d, rho, vxc, vyc, vzc, vxd, vyd, vzd, s);
  }
}

#define INSTF(T)                                                                                                  \
  template bool source_d3_fused_ok<T>(const Dev<T>&);                                                             \
  template int launch_source_d3_fused<T>(const Dev<T>&, const T*, const T*, const T*, const T*, T*, T*, T*, cudaStream_t);
INSTF(double)
INSTF(float)
#undef INSTF

template int launch_source_d3<double>(const Dev<double>&, const double*, const double*, const double*, const double*,
                                      double* const*, double*, double*, double*, cudaStream_t);
template int launch_source_d3<float>(const Dev<float>&, const float*, const float*, const float*, const float*,
                                     float* const*, float*, float*, float*, cudaStream_t);

}  // namespace fg
