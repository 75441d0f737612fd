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

template int launch_source_d3<double>(const Dev<double>&, const double*, const double*, const double*, const double*,
                                      double* const*, double*, double*, double*, cudaStream_t);
template int launch_source_d3<float>(const Dev<float>&, const float*, const float*, const float*, const float*,
                                     float* const*, float*, float*, float*, cudaStream_t);

}  // namespace fg
