// k_planets.cu -- SURVEY.md 8(f) NEXT-2: live planets (section 3.8; reading G33).
//   k_potential_live : cell 5 with the planets where they are at the beginning of the update (device state)
//   k_planet_force   : the force of the gas on every planet, direct summation over the active cells or with the
//                      axisymmetric part of the density removed first: one warp per ring, lanes along the
//                      ring, warp-shuffle and block reduction into one partial per block (fixed shape: reproducible)
//   k_planets_update : sums the partials, kicks the velocities by dt a_gas and takes one fifth-order Cash-Karp step
//                      over dt (Eq. 109, Tab. 3) in the rotating frame -- one thread, fp64; the planets
//                      never visit the host, so fargo_step(n) stays free of host synchronisation
// Product code: shares nothing with oracle/.
#include "kernels.h"

namespace fg {

constexpr int PFW = 8;   // warps (rings) per block of the force kernel

int planets_blocks(int ny, int nz) { return (ny * nz + PFW - 1) / PFW; }

// One block per row (j, k): what depends on the row only (R, z, the star's term with its division) is formed once per
// thread, the planets' constants once per planet, and the thread walks the row.
template <typename T>
__global__ void __launch_bounds__(128) k_potential_live(const Dev<T> d, T* __restrict__ phi, const T gm_star,
                                                        const PlanetsDev* __restrict__ pl, const int npl) {
  const int j = blockIdx.x, k = blockIdx.y;
  T R, z, r;
  if (d.geometry == GEO_SPH) { R = d.yc[j] * d.sin_zc[k]; z = d.yc[j] * d.cos_zc[k]; r = d.yc[j]; }
  else { R = d.yc[j]; z = d.zc[k]; r = rsqrt_ieee(R * R + z * z); }
  const T star = -(gm_star / r);
  T* __restrict__ row = phi + d.id(0, j, k);
  if (npl == 1) {   // the common case: the planet's constants in registers
    const T xp = (T)pl->x[0][0], yp = (T)pl->x[0][1], ddz = z - (T)pl->x[0][2];
    const T eps2 = (T)(pl->eps[0] * pl->eps[0]), gm = (T)pl->gm[0];
    for (int i = threadIdx.x; i < d.TX; i += 128) {
      const T ddx = R * d.cos_xc[i] - xp, ddy = R * d.sin_xc[i] - yp;
      const T d2 = ((ddx * ddx + ddy * ddy) + ddz * ddz) + eps2;
      row[i] = star - rdiv(gm, rsqrt_ieee(d2));
    }
    return;
  }
  for (int i = threadIdx.x; i < d.TX; i += 128) {
    const T x = R * d.cos_xc[i], y = R * d.sin_xc[i];
    T p = star;
    for (int q = 0; q < npl; ++q) {
      const T ddx = x - (T)pl->x[q][0], ddy = y - (T)pl->x[q][1], ddz = z - (T)pl->x[q][2];
      const T d2 = ((ddx * ddx + ddy * ddy) + ddz * ddz) + (T)(pl->eps[q] * pl->eps[q]);
      p = p - rdiv((T)pl->gm[q], rsqrt_ieee(d2));
    }
    row[i] = p;
  }
}

template <typename T>
int launch_potential_live(const Dev<T>& d, T* phi, T gm_star, const PlanetsDev* pl, int npl, cudaStream_t s) {
  k_potential_live<T><<<dim3(d.TY, d.TZ), 128, 0, s>>>(d, phi, gm_star, pl, npl);
  return 1;
}

template <typename T> __device__ __forceinline__ T warp_sum(T v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = v + __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// sum over the active cells of dm (x_c - x_p) / (|x_c - x_p|^2 + eps_p^2)^(3/2), per planet: part[block][planet][3]
template <typename T>
__global__ void __launch_bounds__(32 * PFW) k_planet_force(const Dev<T> d, const T* __restrict__ rho,
                                                           const PlanetsDev* __restrict__ pl, const int npl, const int mode,
                                                           double* __restrict__ part) {
  __shared__ double sh[PFW][MAXPL][3];
  const int lane = threadIdx.x, w = threadIdx.y;
  const int row = blockIdx.x * PFW + w;
  const bool live = row < d.ny * d.nz && !d.ctl->done;
  const int j = d.ngy + (live ? row % d.ny : 0), k = d.ngz + (live ? row / d.ny : 0);
  T R, z;
  if (d.geometry == GEO_SPH) { R = d.yc[j] * d.sin_zc[k]; z = d.yc[j] * d.cos_zc[k]; }
  else { R = d.yc[j]; z = d.zc[k]; }
  const T vol = d.Vj[j] * d.syk[k];
  const T* __restrict__ ring = rho + d.id(d.ngx, j, k);
  T mean = T(0);
  if (mode == 2) {   // the axisymmetric part: the mean of the ring
    T sm = T(0);
    if (live) for (int i = lane; i < d.nx; i += 32) sm = sm + ring[i];
    mean = rdiv(warp_sum(sm), (T)d.nx);
  }
  for (int p = 0; p < npl; ++p) {
    const T xp = (T)pl->x[p][0], yp = (T)pl->x[p][1], zp = (T)pl->x[p][2];
    const T eps2 = (T)(pl->eps[p] * pl->eps[p]);
    const T ddz = z - zp;
    T Fx = T(0), Fy = T(0), Fz = T(0);
    if (live)
      for (int i = lane; i < d.nx; i += 32) {   // (unrolling by 4 was measured: 0.44 -> 0.58 ms)
        const T x = R * d.cos_xc[d.ngx + i], y = R * d.sin_xc[d.ngx + i];
        const T ddx = x - xp, ddy = y - yp;
        const T d2 = ((ddx * ddx + ddy * ddy) + ddz * ddz) + eps2;
        const T wgt = rdiv((ring[i] - mean) * vol, d2 * rsqrt_ieee(d2));
        Fx = Fx + wgt * ddx; Fy = Fy + wgt * ddy; Fz = Fz + wgt * ddz;
      }
    Fx = warp_sum(Fx); Fy = warp_sum(Fy); Fz = warp_sum(Fz);
    if (lane == 0) { sh[w][p][0] = (double)Fx; sh[w][p][1] = (double)Fy; sh[w][p][2] = (double)Fz; }
  }
  __syncthreads();
  const int t = w * 32 + lane;
  if (t < npl * 3) {
    const int p = t / 3, c = t % 3;
    double s = 0.0;
    for (int q = 0; q < PFW; ++q) s = s + sh[q][p][c];
    part[((size_t)blockIdx.x * MAXPL + p) * 3 + c] = s;
  }
}

// Tab. 3: a_ij of stages 2..6 and the fifth-order weights b_i
__constant__ double c_cka[6][5] = {
    {0.0, 0.0, 0.0, 0.0, 0.0},
    {1.0 / 5.0, 0.0, 0.0, 0.0, 0.0},
    {3.0 / 40.0, 9.0 / 40.0, 0.0, 0.0, 0.0},
    {3.0 / 10.0, -9.0 / 10.0, 6.0 / 5.0, 0.0, 0.0},
    {-11.0 / 54.0, 5.0 / 2.0, -70.0 / 27.0, 35.0 / 27.0, 0.0},
    {1631.0 / 55296.0, 175.0 / 512.0, 575.0 / 13824.0, 44275.0 / 110592.0, 253.0 / 4096.0}};
__constant__ double c_ckb[6] = {37.0 / 378.0, 0.0, 250.0 / 621.0, 125.0 / 594.0, 0.0, 512.0 / 1771.0};

// f(t, y) of Eq. 108 in the frame rotating at om about Z: star at the origin, the other planets, Coriolis and
// centrifugal accelerations (reading G33); y = [x y z vx vy vz] per planet
__device__ void planet_rhs(const int n, const double gms, const double om, const double* gm, const double* y, double* f) {
  for (int p = 0; p < n; ++p) {
    const double* s = y + 6 * p;
    const double r2 = (s[0] * s[0] + s[1] * s[1]) + s[2] * s[2];
    const double ir3 = 1.0 / (r2 * sqrt(r2));
    double ax = -(gms * ir3) * s[0], ay = -(gms * ir3) * s[1], az = -(gms * ir3) * s[2];
    for (int q = 0; q < n; ++q) {
      if (q == p) continue;
      const double* o = y + 6 * q;
      const double dx = s[0] - o[0], dy = s[1] - o[1], dz = s[2] - o[2];
      const double d2 = (dx * dx + dy * dy) + dz * dz;
      const double w = gm[q] / (d2 * sqrt(d2));
      ax = ax - w * dx; ay = ay - w * dy; az = az - w * dz;
    }
    ax = ax + ((2.0 * om) * s[4] + (om * om) * s[0]);
    ay = ay + ((om * om) * s[1] - (2.0 * om) * s[3]);
    double* o = f + 6 * p;
    o[0] = s[3]; o[1] = s[4]; o[2] = s[5]; o[3] = ax; o[4] = ay; o[5] = az;
  }
}

__global__ void __launch_bounds__(256) k_planets_update(Ctl* __restrict__ ctl, PlanetsDev* __restrict__ pl, const int npl,
                                                        const int mode, const double* __restrict__ part, const int nblk,
                                                        const double gms, const double om) {
  if (ctl->done) return;
  __shared__ double red[256];
  __shared__ double F[MAXPL * 3];
  const int t = threadIdx.x;
  if (mode != 0) {
    for (int q = 0; q < npl * 3; ++q) {   // fixed-shape tree: the sum does not depend on the launch
      const int p = q / 3, c = q % 3;
      double s = 0.0;
      for (int b = t; b < nblk; b += 256) s = s + part[((size_t)b * MAXPL + p) * 3 + c];
      red[t] = s;
      __syncthreads();
      for (int o = 128; o > 0; o >>= 1) {
        if (t < o) red[t] = red[t] + red[t + o];
        __syncthreads();
      }
      if (t == 0) F[q] = red[0];
      __syncthreads();
    }
  }
  if (t != 0) return;
  const double h = ctl->dt;
  double y[6 * MAXPL], yt[6 * MAXPL], k[6][6 * MAXPL];
  for (int p = 0; p < npl; ++p)
    for (int c = 0; c < 3; ++c) {
      double v = pl->v[p][c];
      if (mode != 0) {   // the gas force is evaluated once per update and used to update the velocities
        const double a = pl->gconst * F[3 * p + c];
        pl->f[p][c] = a;
        v = v + h * a;
      }
      y[6 * p + c] = pl->x[p][c]; y[6 * p + 3 + c] = v;
    }
  const int m = 6 * npl;
  for (int i = 0; i < 6; ++i) {   // Eq. 109
    for (int q = 0; q < m; ++q) {
      double acc = 0.0;
      for (int jj = 0; jj < i; ++jj) acc = acc + c_cka[i][jj] * k[jj][q];
      yt[q] = y[q] + h * acc;
    }
    planet_rhs(npl, gms, om, pl->gm, yt, k[i]);
  }
  for (int q = 0; q < m; ++q) {
    double acc = 0.0;
    for (int i = 0; i < 6; ++i) acc = acc + c_ckb[i] * k[i][q];
    y[q] = y[q] + h * acc;
  }
  for (int p = 0; p < npl; ++p)
    for (int c = 0; c < 3; ++c) { pl->x[p][c] = y[6 * p + c]; pl->v[p][c] = y[6 * p + 3 + c]; }
}

template <typename T>
int launch_planets_update(const Dev<T>& d, const T* rho, PlanetsDev* pl, int npl, int mode, double* part, double gm_star,
                          double omega, cudaStream_t s) {
  const int nblk = planets_blocks(d.ny, d.nz);
  int n = 0;
  if (mode != 0) {
    k_planet_force<T><<<nblk, dim3(32, PFW), 0, s>>>(d, rho, pl, npl, mode, part);
    ++n;
  }
  k_planets_update<<<1, 256, 0, s>>>(d.ctl, pl, npl, mode, part, nblk, gm_star, omega);
  return n + 1;
}

// ---- cell 5b: the frame's rotation rate changes by dom between two updates, Eq. 44 --------------------
// v_phi -= dom R_x(j, k) on every cell of the allocated array (R_x = r | r sin(theta) at the centre of the phi face,
// P:312); block (0, 0) also carries the live planets into the new frame: v' = v - dom z^ x x.
template <typename T>
__global__ void __launch_bounds__(128) k_frame_change(const Dev<T> d, T* __restrict__ vx, const T dom, PlanetsDev* __restrict__ pl,
                                                      const int npl, const double dom64) {
  const int j = blockIdx.x, k = blockIdx.y;
  const T corr = dom * d.Rx(j, k);
  T* __restrict__ row = vx + d.id(0, j, k);
  for (int i = threadIdx.x; i < d.TX; i += 128) row[i] = row[i] - corr;
  if (j == 0 && k == 0 && (int)threadIdx.x < npl) {
    const int p = threadIdx.x;
    const double x = pl->x[p][0], y = pl->x[p][1];
    pl->v[p][0] = pl->v[p][0] + dom64 * y;
    pl->v[p][1] = pl->v[p][1] - dom64 * x;
  }
}

template <typename T>
int launch_frame_change(const Dev<T>& d, T* vx, double dom, PlanetsDev* pl, int npl, cudaStream_t s) {
  k_frame_change<T><<<dim3(d.TY, d.TZ), 128, 0, s>>>(d, vx, (T)dom, pl, npl, dom);
  return 1;
}

// ---- diagnostics: sum reductions over the active cells ("the mass or angular momentum") -------------------
// part[block][5] = mass, X / Y / Z momentum of Tab. 2 (mean of the cell's left and right momenta, formed as cell 12a
// forms them), internal energy (adiabatic).  One warp per ring, warp-shuffle sums, one partial per block of 8 rings;
// the host adds the partials in block order (fixed shape: reproducible).
template <typename T>
__global__ void __launch_bounds__(32 * PFW) k_diagnostics(const Dev<T> d, const State<T> st, double* __restrict__ part) {
  __shared__ double sh[PFW][5];
  const int lane = threadIdx.x, w = threadIdx.y;
  const int row = blockIdx.x * PFW + w;
  const bool live = row < d.ny * d.nz;
  const int j = d.ngy + (live ? row % d.ny : 0), k = d.ngz + (live ? row / d.ny : 0);
  const T vol = d.Vj[j] * d.syk[k];
  const T rx = d.Rx(j, k), rx2om = d.xmom_off(j, rx), rz = d.Rzj[j];
  T m = T(0), px = T(0), py = T(0), pz = T(0), en = T(0);
  if (live)
    for (int ia = lane; ia < d.nx; ia += 32) {
      const int i = d.ngx + ia;
      const long long l = d.id(i, j, k);
      const T r0 = st.rho[l];
      m = m + r0 * vol;
      if (d.hasx) {
        const T v = st.vx[l];
        const T vp = (d.xwrap || i + 1 < d.TX) ? st.vx[d.id(d.xw(i + 1), j, k)] : v;
        px = px + (T(0.5) * (r0 * rfma(rx, v, rx2om) + r0 * rfma(rx, vp, rx2om))) * vol;
      }
      if (d.hasy) {
        const T v = st.vy[l];
        const T vp = j + 1 < d.TY ? st.vy[l + d.pitch] : v;
        py = py + (T(0.5) * (r0 * v + r0 * vp)) * vol;
      }
      if (d.hasz) {
        const T v = st.vz[l];
        const T vp = k + 1 < d.TZ ? st.vz[l + d.plane] : v;
        pz = pz + (T(0.5) * (r0 * (rz * v) + r0 * (rz * vp))) * vol;
      }
      if (d.eos == EOS_ADI) en = en + st.e[l] * vol;
    }
  m = warp_sum(m); px = warp_sum(px); py = warp_sum(py); pz = warp_sum(pz); en = warp_sum(en);
  if (lane == 0) { sh[w][0] = (double)m; sh[w][1] = (double)px; sh[w][2] = (double)py; sh[w][3] = (double)pz; sh[w][4] = (double)en; }
  __syncthreads();
  const int t = w * 32 + lane;
  if (t < 5) {
    double s = 0.0;
    for (int q = 0; q < PFW; ++q) s = s + sh[q][t];
    part[(size_t)blockIdx.x * 5 + t] = s;
  }
}

template <typename T>
int launch_diagnostics(const Dev<T>& d, const State<T>& st, double* part, cudaStream_t s) {
  k_diagnostics<T><<<planets_blocks(d.ny, d.nz), dim3(32, PFW), 0, s>>>(d, st, part);
  return 1;
}

#define INST(T)                                                                                               \
  template int launch_potential_live<T>(const Dev<T>&, T*, T, const PlanetsDev*, int, cudaStream_t);          \
  template int launch_frame_change<T>(const Dev<T>&, T*, double, PlanetsDev*, int, cudaStream_t);             \
  template int launch_diagnostics<T>(const Dev<T>&, const State<T>&, double*, cudaStream_t);                  \
  template int launch_planets_update<T>(const Dev<T>&, const T*, PlanetsDev*, int, int, double*, double, double, cudaStream_t);
INST(double)
INST(float)
#undef INST

}  // namespace fg
