// k_dt.cu -- ring mean velocity (Fig. 2 cell 3, Eq. 72), potential (cell 5, reading G12), CFL time
// step (cell 6, Eq. 59) with the FARGO shear limit (Eq. 73), and the clock.
// The time step is reduced wholly on the device (warp shuffles -> one atomic max per block -> a
// one-block finishing kernel): the paper finishes it on the CPU and names that its one bottleneck.
#include "kernels.h"

namespace fg {

// ---- cell 3: v0_jk = (max_i vx + min_i vx)/2, one warp per ring, ghost rings included --------------
template <typename T>
__global__ void k_vmean(const Dev<T> d, const T* __restrict__ vx, T* __restrict__ v0) {
  if (d.ctl->done) return;
  const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  const int nring = d.TY * d.TZ;
  if (warp >= nring) return;
  const int j = warp % d.TY, k = warp / d.TY;
  const T* row = vx + d.id(d.ngx, j, k);
  T lo = row[0], hi = lo;
  for (int i = lane; i < d.nx; i += 32) {
    const T v = row[i];
    lo = rmin(lo, v); hi = rmax(hi, v);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    lo = rmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
    hi = rmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
  }
  if (lane == 0) v0[warp] = T(0.5) * (hi + lo);
}

template <typename T>
int launch_vmean(const Dev<T>& d, const T* vx, T* v0, cudaStream_t s) {
  const int nring = d.TY * d.TZ;
  k_vmean<T><<<(nring + 7) / 8, 256, 0, s>>>(d, vx, v0);
  return 1;
}

// ---- cell 5: Phi = -GM/|x| - G m_p / sqrt(|x - x_p|^2 + eps^2) at cell centres ----------------------
// Trigonometry comes from host tables only (no device transcendental).
template <typename T>
__global__ void k_potential(const Dev<T> d, T* __restrict__ phi, const T gm_star, const T gm_planet, T xp,
                            T yp, const T eps2, const T* __restrict__ ppos) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
  if (i >= d.TX) return;
  if (ppos) { xp = ppos[0]; yp = ppos[1]; }   // the planet moves in the frame: (x_p, y_p) of this update, device resident
  T R, z, r;
  if (d.geometry == GEO_SPH) { R = d.yc[j] * d.sin_zc[k]; z = d.yc[j] * d.cos_zc[k]; r = d.yc[j]; }
  else { R = d.yc[j]; z = d.zc[k]; r = rsqrt_ieee(R * R + z * z); }
  const T x = R * d.cos_xc[i], y = R * d.sin_xc[i];
  T p = -(gm_star / r);
  if (gm_planet != T(0)) {
    const T ddx = x - xp, ddy = y - yp;
    const T d2 = ((ddx * ddx + ddy * ddy) + z * z) + eps2;
    p = p - gm_planet / rsqrt_ieee(d2);
  }
  phi[d.id(i, j, k)] = p;
}

template <typename T>
int launch_potential(const Dev<T>& d, T* phi, T gm_star, T gm_planet, T xp, T yp, T eps2, const T* ppos, cudaStream_t s) {
  dim3 b(128), g((d.TX + 127) / 128, d.TY, d.TZ);
  k_potential<T><<<g, b, 0, s>>>(d, phi, gm_star, gm_planet, xp, yp, eps2, ppos);
  return 1;
}

// ---- cell 6 ---------------------------------------------------------------------------------------------
// Per active cell: sum over the processes of Eq. 59 of the squared inverse time steps, each inverse
// time step being the max over the directions present ("dt_i = min_j dt_ij").  max is exact,
// so the block/grid reduction order does not matter: dt is bit-reproducible.
template <typename T>
__global__ void __launch_bounds__(256) k_dt_cells(const Dev<T> d, const State<T> st, const T* __restrict__ v0, const MhdDt<T> M) {
  if (d.ctl->done) return;
  const int nrow = d.ny * d.nz;
  T m2 = T(0);
  for (int row = blockIdx.x; row < nrow; row += gridDim.x) {
    const int j = d.ngy + row % d.ny, k = d.ngz + row / d.ny;
    const T ilx = d.invLX(j, k), ily = d.invLY[j], ilz = d.invLZ(j, k);
    T ilmax = T(0);
    if (d.hasx) ilmax = rmax(ilmax, ilx);
    if (d.hasy) ilmax = rmax(ilmax, ily);
    if (d.hasz) ilmax = rmax(ilmax, ilz);
    const T il2 = ilmax * ilmax;
    const T I4 = d.c4 * il2;
    const T vm = v0 ? v0[d.rid(j, k)] : T(0);
    for (int ia = threadIdx.x; ia < d.nx; ia += blockDim.x) {
      const int i = d.ngx + ia;
      const long long l = d.id(i, j, k);
      T cs2 = (d.eos == EOS_ADI) ? rdiv(d.gg1 * st.e[l], st.rho[l]) : st.e[l] * st.e[l];
      if (M.bx && !M.passive) {   // item 1 of Eq. 59: C_w^2 = C_s^2 + v_A^2, B at the zone centre
        const T cx = T(0.5) * (M.bx[l] + M.bx[d.id(d.xw(i + 1), j, k)]);
        const T cy = T(0.5) * (M.by[l] + M.by[l + d.pitch]);
        const T cz = T(0.5) * (M.bz[l] + M.bz[l + d.plane]);
        cs2 = cs2 + rdiv(rfma(cz, cz, rfma(cy, cy, rfma(cx, cx, T(0)))), M.mu0 * st.rho[l]);
      }
      const T I1sq = cs2 * il2;
      T I2 = T(0), I3 = T(0);
      if (d.hasx) {
        const T a = st.vx[l], b = st.vx[d.id(d.xw(i + 1), j, k)];
        I2 = rmax(I2, rabs(rfma(T(0.5), a + b, -vm)) * ilx);
        I3 = rmax(I3, rabs(b - a) * ilx);
      }
      if (d.hasy) {
        const T a = st.vy[l], b = st.vy[l + d.pitch];
        I2 = rmax(I2, rabs(T(0.5) * (a + b)) * ily);
        I3 = rmax(I3, rabs(b - a) * ily);
      }
      if (d.hasz) {
        const T a = st.vz[l], b = st.vz[l + d.plane];
        I2 = rmax(I2, rabs(T(0.5) * (a + b)) * ilz);
        I3 = rmax(I3, rabs(b - a) * ilz);
      }
      I3 = d.c3 * I3;
      T Isq = rfma(I4, I4, rfma(I3, I3, rfma(I2, I2, I1sq)));
      if (M.bx && M.eta4 != T(0)) { const T I5 = M.eta4 * il2; Isq = rfma(I5, I5, Isq); }   // item 5: dt_5 = Delta^2 / (4 eta)
      m2 = rmax(m2, Isq);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m2 = rmax(m2, __shfl_xor_sync(0xffffffffu, m2, o));
  __shared__ T sm[8];
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = m2;
  __syncthreads();
  if (threadIdx.x < 32) {
    m2 = threadIdx.x < (blockDim.x >> 5) ? sm[threadIdx.x] : T(0);
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) m2 = rmax(m2, __shfl_xor_sync(0xffffffffu, m2, o));
    if (threadIdx.x == 0) atomicMax(&d.ctl->m2bits, to_bits(m2));   // non-negative: bit order = value order
  }
}

// ---- cell 6, 3-D meshes with a wrapped X axis and an even nx: two cells per lane ----------------------------
// A warp owns a ring (j,k) and walks it 64 cells at a time with 16-byte loads; the upper X face of the pair is
// the next lane's first cell (lane 31 reads it).  Same expressions, in the same order, as k_dt_cells; the
// reduction is a max, so the result is bit-equal whatever the order.
template <typename T> struct DPair;
template <> struct DPair<double> { using type = double2; };
template <> struct DPair<float> { using type = float2; };

// MHD = true: C_w^2 = C_s^2 + v_A^2 with B averaged to the zone centre and the resistive item 5, as in k_dt_cells.
template <typename T, bool ADI, bool MHD>
__global__ void __launch_bounds__(256) k_dt_cells2(const Dev<T> d, const State<T> st, const T* __restrict__ v0, const MhdDt<T> M) {
  if (d.ctl->done) return;
  using P2 = typename DPair<T>::type;
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const int nrow = d.ny * d.nz, nwarp = gridDim.x * (blockDim.x >> 5);
  const int nx = d.nx;
  T m2 = T(0);
  for (int row = blockIdx.x * (blockDim.x >> 5) + wib; row < nrow; row += nwarp) {
    const int j = d.ngy + row % d.ny, k = d.ngz + row / d.ny;
    const T ilx = d.invLX(j, k), ily = d.invLY[j], ilz = d.invLZ(j, k);
    const T ilmax = rmax(rmax(rmax(T(0), ilx), ily), ilz);
    const T il2 = ilmax * ilmax;
    const T I4 = d.c4 * il2;
    const T vm = v0 ? v0[d.rid(j, k)] : T(0);
    const long long base = d.id(0, j, k);
    for (int i0 = 0; i0 < nx; i0 += 64) {
      const int i = i0 + 2 * lane;
      const bool live = i < nx;
      const long long l = base + (live ? i : 0);
      const P2 r = *reinterpret_cast<const P2*>(st.rho + l);
      const P2 e = *reinterpret_cast<const P2*>(st.e + l);
      const P2 ax = *reinterpret_cast<const P2*>(st.vx + l);
      const P2 ay = *reinterpret_cast<const P2*>(st.vy + l);
      const P2 by = *reinterpret_cast<const P2*>(st.vy + l + d.pitch);
      const P2 az = *reinterpret_cast<const P2*>(st.vz + l);
      const P2 bz = *reinterpret_cast<const P2*>(st.vz + l + d.plane);
      T nxt = __shfl_down_sync(0xffffffffu, ax.x, 1);
      const bool edge = lane == 31 || i + 2 >= nx;
      const int ip = i + 2 >= nx ? i + 2 - nx : i + 2;
      if (edge) nxt = st.vx[base + (live ? ip : 0)];
      P2 fx = {T(0), T(0)}, fy0 = fx, fy1 = fx, fz0 = fx, fz1 = fx;
      T fxn = T(0);
      const bool alfven = MHD && !M.passive;
      if (alfven) {
        fx = *reinterpret_cast<const P2*>(M.bx + l);
        fy0 = *reinterpret_cast<const P2*>(M.by + l);
        fy1 = *reinterpret_cast<const P2*>(M.by + l + d.pitch);
        fz0 = *reinterpret_cast<const P2*>(M.bz + l);
        fz1 = *reinterpret_cast<const P2*>(M.bz + l + d.plane);
        fxn = __shfl_down_sync(0xffffffffu, fx.x, 1);
        if (edge) fxn = M.bx[base + (live ? ip : 0)];
      }
#pragma unroll
      for (int c = 0; c < 2; ++c) {
        const T rho = c ? r.y : r.x, en = c ? e.y : e.x;
        T cs2 = ADI ? rdiv(d.gg1 * en, rho) : en * en;
        if (alfven) {
          const T cx = T(0.5) * ((c ? fx.y : fx.x) + (c ? fxn : fx.y));
          const T cy = T(0.5) * ((c ? fy0.y : fy0.x) + (c ? fy1.y : fy1.x));
          const T cz = T(0.5) * ((c ? fz0.y : fz0.x) + (c ? fz1.y : fz1.x));
          cs2 = cs2 + rdiv(rfma(cz, cz, rfma(cy, cy, rfma(cx, cx, T(0)))), M.mu0 * rho);
        }
        const T I1sq = cs2 * il2;
        T I2 = T(0), I3 = T(0);
        {
          const T a = c ? ax.y : ax.x, b = c ? nxt : ax.y;
          I2 = rmax(I2, rabs(rfma(T(0.5), a + b, -vm)) * ilx);
          I3 = rmax(I3, rabs(b - a) * ilx);
        }
        {
          const T a = c ? ay.y : ay.x, b = c ? by.y : by.x;
          I2 = rmax(I2, rabs(T(0.5) * (a + b)) * ily);
          I3 = rmax(I3, rabs(b - a) * ily);
        }
        {
          const T a = c ? az.y : az.x, b = c ? bz.y : bz.x;
          I2 = rmax(I2, rabs(T(0.5) * (a + b)) * ilz);
          I3 = rmax(I3, rabs(b - a) * ilz);
        }
        I3 = d.c3 * I3;
        T Isq = rfma(I4, I4, rfma(I3, I3, rfma(I2, I2, I1sq)));
        if (MHD && M.eta4 != T(0)) { const T I5 = M.eta4 * il2; Isq = rfma(I5, I5, Isq); }
        if (live) m2 = rmax(m2, Isq);
      }
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m2 = rmax(m2, __shfl_xor_sync(0xffffffffu, m2, o));
  __shared__ T sm[8];
  if (lane == 0) sm[wib] = m2;
  __syncthreads();
  if (threadIdx.x < 32) {
    m2 = threadIdx.x < (blockDim.x >> 5) ? sm[threadIdx.x] : T(0);
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) m2 = rmax(m2, __shfl_xor_sync(0xffffffffu, m2, o));
    if (threadIdx.x == 0) atomicMax(&d.ctl->m2bits, to_bits(m2));
  }
}

// One block: shear limit over the active rings (Eq. 73 with V_X = v0_jk), Courant factor, overrides.
template <typename T>
__global__ void __launch_bounds__(1024) k_dt_finish(const Dev<T> d, const T* __restrict__ v0) {
  Ctl* c = d.ctl;
  if (c->done) return;
  T s = T(0);
  if (d.fargo) {
    // pairs of radially neighbouring rings, both active; a slab also owns the pair across its upper (external) face,
    // unless that face is the periodic seam of the undivided mesh (rings ny-1 and 0 are no pair there either)
    const int nyp = d.ny - 1 + ((d.bc[1][1] == BC_EXTERNAL && !d.seam_above) ? 1 : 0);
    const int n = nyp > 0 ? nyp * d.nz : 0;
    for (int r = threadIdx.x; r < n; r += blockDim.x) {
      const int j = d.ngy + r % nyp, k = d.ngz + r / nyp;
      s = rmax(s, rabs(v0[d.rid(j, k)] * d.invLX(j, k) - v0[d.rid(j + 1, k)] * d.invLX(j + 1, k)));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s = rmax(s, __shfl_xor_sync(0xffffffffu, s, o));
  }
  __shared__ T sm[32];
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) s = rmax(s, sm[w]);
    const T M2 = from_bits<T>(c->m2bits);
    T dt = T(1) / rsqrt_ieee(M2);
    if (d.fargo && s > T(0)) dt = rmin(dt, d.shear_c0 / s);
    dt = d.cfl * dt;
    double dtd = (double)dt;
    if (d.dt_fixed > 0.0) dtd = (double)(T)d.dt_fixed;
    int clipped = 0;
    if (d.t_stop > 0.0 && c->t + dtd >= d.t_stop) { dtd = (double)(T)(d.t_stop - c->t); clipped = 1; }
    c->dt = dtd;
    c->clipped = clipped;
    c->m2bits = 0ull;
  }
}

template <typename T>
int launch_dt(const Dev<T>& d, const State<T>& st, const T* v0, cudaStream_t s, int mode, const MhdDt<T>* mhd) {
  MhdDt<T> M{nullptr, nullptr, nullptr, T(1), T(0), 0};
  if (mhd) M = *mhd;
  const int nrow = d.ny * d.nz;
  const int grid = nrow < 148 * 8 ? nrow : 148 * 8;
  if (mode == DT_FINISH) {   // the per-cell max was accumulated by k_newvel_dt at the end of the previous update
    k_dt_finish<T><<<1, 1024, 0, s>>>(d, v0);
    return 1;
  }
  if (d.hasx && d.hasy && d.hasz && d.xwrap && d.nx % 2 == 0) {
    const int g2 = nrow < 148 * 8 * 8 ? (nrow + 7) / 8 : 148 * 8;
    if (M.bx) {
      if (d.eos == EOS_ADI) k_dt_cells2<T, true, true><<<g2, 256, 0, s>>>(d, st, v0, M);
      else k_dt_cells2<T, false, true><<<g2, 256, 0, s>>>(d, st, v0, M);
    } else if (d.eos == EOS_ADI) k_dt_cells2<T, true, false><<<g2, 256, 0, s>>>(d, st, v0, M);
    else k_dt_cells2<T, false, false><<<g2, 256, 0, s>>>(d, st, v0, M);
  } else {
    k_dt_cells<T><<<grid, 256, 0, s>>>(d, st, v0, M);
  }
  if (mode == DT_CELLS) return 1;
  k_dt_finish<T><<<1, 1024, 0, s>>>(d, v0);
  return 2;
}

// The clock: t <- t + dt (or exactly t_stop on a clipped step); afterwards every kernel is a no-op.
__global__ void k_advance(Ctl* c, const double t_stop) {
  if (c->done) return;
  c->t = c->clipped ? t_stop : c->t + c->dt;
  c->nsteps += 1;
  if (t_stop > 0.0 && c->t >= t_stop) c->done = 1;
}
// Slab decomposition (NEXT-3): ctl->dt now holds the minimum over the slabs of their local time steps (all-reduced in
// place by the caller).  Each slab clipped its own dt to t_stop; the minimum is the right step (a clipped value is
// never below an unclipped one that ends before t_stop), only the `clipped` flag has to be taken again.
__global__ void k_dt_sync(Ctl* c, const double t_stop, const int single) {
  if (c->done) return;
  const double rest = single ? (double)(float)(t_stop - c->t) : t_stop - c->t;
  c->clipped = (t_stop > 0.0 && (c->t + c->dt >= t_stop || c->dt == rest)) ? 1 : 0;
}
// Sub-domains on one device: dt <- min(dt, *other), the all-reduce (min) of P:407 done pairwise by the caller
__global__ void k_dt_min(Ctl* c, const double* __restrict__ other) {
  if (c->done) return;
  const double o = *other;
  if (o < c->dt) c->dt = o;
}
int launch_dt_min(Ctl* ctl, const double* other, cudaStream_t s) {
  k_dt_min<<<1, 1, 0, s>>>(ctl, other);
  return 1;
}
int launch_dt_sync(Ctl* ctl, double t_stop, bool single, cudaStream_t s) {
  k_dt_sync<<<1, 1, 0, s>>>(ctl, t_stop, single ? 1 : 0);
  return 1;
}
int launch_advance(Ctl* ctl, double t_stop, cudaStream_t s) {
  k_advance<<<1, 1, 0, s>>>(ctl, t_stop);
  return 1;
}

__global__ void k_selftest_div(const double* __restrict__ a, const double* __restrict__ b, double* __restrict__ out,
                               const long long n) {
  for (long long m = blockIdx.x * (long long)blockDim.x + threadIdx.x; m < n; m += (long long)gridDim.x * blockDim.x)
    out[m] = b ? rdiv(a[m], b[m]) : rdiv6(a[m]);
}
int launch_selftest_div(const double* a, const double* b, double* out, long long n, cudaStream_t s) {
  k_selftest_div<<<148 * 8, 256, 0, s>>>(a, b, out, n);
  return 1;
}

#define INST(T)                                                                              \
  template int launch_vmean<T>(const Dev<T>&, const T*, T*, cudaStream_t);                   \
  template int launch_potential<T>(const Dev<T>&, T*, T, T, T, T, T, const T*, cudaStream_t);          \
  template int launch_dt<T>(const Dev<T>&, const State<T>&, const T*, cudaStream_t, int, const MhdDt<T>*);
INST(double)
INST(float)
#undef INST

}  // namespace fg
