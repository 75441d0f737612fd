// k_transport.cu -- the transport step, box 12 of Fig. 2:
//   12a left/right momenta with the quantities of Tab. 2 (Eqs. 49-50; Tab. 2)
//   12b van Leer slopes and upwind star values at half time step (Eq. 48)
//   12c conservative update per direction (Eqs. 41-43, 45-47 P:292-326) with consistent transport:
//       q = Q/rho is reconstructed, the flux of Q is the mass flux times q*
//   12d new velocities (Eq. 51 P:355 + Tab. 2 inverted, reading G28)
//
// One sweep = ONE kernel: divide-by-rho, slope, star value, flux and update of rho and of every
// transported quantity are fused, so each field is read once and written once per direction
// (the paper runs ~4 kernels per field per direction).  A thread block owns a tile of
// BM cells along the sweep axis (2 halo cells per side, recomputed) by BX cells along X; cell values,
// slopes and fluxes are exchanged between neighbouring threads through shared memory.
#include "kernels.h"

namespace fg {

constexpr int QB = 4;   // quantities processed together (shared memory = 3 * QB * tile * sizeof(T))

template <int DIR> struct Tile;
template <> struct Tile<0> { static constexpr int BX = 1, BM = 256; };
template <> struct Tile<1> { static constexpr int BX = 16, BM = 32; };
template <> struct Tile<2> { static constexpr int BX = 16, BM = 32; };

// van Leer slope per unit length; zero unless both one-sided differences have the same sign (reading G4)
template <typename T>
__device__ __forceinline__ T vl_slope(const T fm, const T f0, const T fp, const T invd0, const T invdp) {
  const T dm = (f0 - fm) * invd0;
  const T dp = (fp - f0) * invdp;
  const T pr = dm * dp;
  const bool flat = pr <= T(0);
  const T den = flat ? T(1) : dm + dp;   // keeps the division on its fast path when the slope is dropped
  const T a = (T(2) * pr) / den;
  return flat ? T(0) : a;
}

template <typename T, int DIR>
__global__ void __launch_bounds__(Tile<DIR>::BX * Tile<DIR>::BM)
k_sweep(const Dev<T> d, const SweepArgs<T> A) {
  constexpr int BX = Tile<DIR>::BX, BM = Tile<DIR>::BM, NT = BX * BM, INNER = BM - 4;
  if (d.ctl->done) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* const sf = reinterpret_cast<T*>(smem_raw);   // [QB][NT] cell values q
  T* const sa = sf + QB * NT;                     // [QB][NT] slopes
  T* const sF = sa + QB * NT;                     // [QB][NT] fluxes through the lower face

  const int tx = DIR == 0 ? 0 : threadIdx.x;
  const int tm = DIR == 0 ? threadIdx.x : threadIdx.y;
  const int sidx = tm * BX + tx;
  const int T_line = DIR == 0 ? d.TX : DIR == 1 ? d.TY : d.TZ;
  const bool wrap = DIR == 0 && d.xwrap;

  // position of this thread's cell: m along the sweep axis (wrapped in a periodic X), line (i | j, k)
  const int m_unwrapped = (DIR == 0 ? blockIdx.x : blockIdx.y) * INNER - 2 + tm;
  int m = m_unwrapped;
  if (wrap) { m %= d.nx; if (m < 0) m += d.nx; }
  int i, j, k;
  if (DIR == 0) { i = m; j = blockIdx.y; k = blockIdx.z; }
  else if (DIR == 1) { i = blockIdx.x * BX + tx; j = m; k = blockIdx.z; }
  else { i = blockIdx.x * BX + tx; j = blockIdx.z; k = m; }
  const bool valid = (m >= 0 && m < T_line) && (i < d.TX);
  // cells this thread writes: the tile's interior, once (the last X tile may run past the row)
  const bool inner = valid && tm >= 2 && tm < BM - 2 && m_unwrapped < T_line;
  const bool upd = inner && (wrap || (m >= 2 && m < T_line - 2));   // cells the sweep updates; others pass through

  const T dt = (T)d.ctl->dt;
  long long l = 0;
  T w = T(0), r0 = T(1), ir = T(1), Sm = T(0), dtiv = T(0), invd0 = T(0), invdp = T(0), hup = T(0), hdn = T(0);
  if (valid) {
    l = d.id(i, j, k);
    T len0, lenm;
    if (DIR == 0) {
      len0 = lenm = d.LX(j, k);
      invd0 = invdp = d.invLX(j, k);
      Sm = d.Sx(j, k);
      w = A.st.vx[l];
      if (A.v0) w = w - A.v0[d.rid(j, k)];   // residual velocity under orbital advection
    } else if (DIR == 1) {
      const int jm = j > 0 ? j - 1 : 0, jp = j + 1 < d.TY ? j + 1 : j;
      len0 = d.LY[j]; lenm = d.LY[jm];
      invd0 = d.invDY[j]; invdp = d.invDY[jp];
      Sm = d.Sy(j, k);
      w = A.st.vy[l];
    } else {
      const int km = k > 0 ? k - 1 : 0, kp = k + 1 < d.TZ ? k + 1 : k;
      len0 = d.LZ(j, k); lenm = d.LZ(j, km);
      invd0 = d.invDZ(j, k); invdp = d.invDZ(j, kp);
      Sm = d.Sz(j, k);
      w = A.st.vz[l];
    }
    dtiv = dt * d.invV(j, k);
    const T wdt = w * dt;
    hup = (lenm - wdt) * T(0.5);   // Eq. 48, upwind cell m-1
    hdn = (len0 + wdt) * T(0.5);   // Eq. 48, upwind cell m
    r0 = A.srho[l];
    ir = T(1) / r0;
  }
  const bool up = w >= T(0);   // reading G3: ties go to the first branch

  // momenta of Tab. 2 from the state (12a), only on the first pass
  T mom[7] = {T(0), T(0), T(0), T(0), T(0), T(0), T(0)};
  if (A.first && valid) {
    const T rx = d.Rx(j, k), rx2om = (rx * rx) * d.om_eff, rz = d.Rzj[j];
    mom[0] = d.eos == EOS_ADI ? A.st.e[l] : T(0);
    if (d.hasx) {
      const T v = A.st.vx[l];
      const bool ipok = d.xwrap || i + 1 < d.TX;
      const T vp = ipok ? A.st.vx[d.id(d.xw(i + 1), j, k)] : v;
      mom[1] = r0 * (rx * v + rx2om);
      mom[2] = r0 * (rx * vp + rx2om);
    }
    if (d.hasy) {
      const T v = A.st.vy[l];
      const T vp = j + 1 < d.TY ? A.st.vy[l + d.pitch] : v;
      mom[3] = r0 * v;
      mom[4] = r0 * vp;
    }
    if (d.hasz) {
      const T v = A.st.vz[l];
      const T vp = k + 1 < d.TZ ? A.st.vz[l + d.plane] : v;
      mom[5] = r0 * (rz * v);
      mom[6] = r0 * (rz * vp);
    }
  }

  // ---- density first: its mass flux F = w rho* S multiplies every other star value ----------------
  T Fr0;   // mass flux through this cell's lower face
  {
    sf[sidx] = r0;
    __syncthreads();
    T a = T(0);
    if (tm >= 1 && tm < BM - 1) a = vl_slope(sf[sidx - BX], r0, sf[sidx + BX], invd0, invdp);
    sa[sidx] = a;
    __syncthreads();
    T rs = r0;
    if (tm >= 1) rs = up ? sf[sidx - BX] + sa[sidx - BX] * hup : r0 - a * hdn;
    Fr0 = (w * rs) * Sm;
    sF[sidx] = Fr0;
    __syncthreads();
    if (inner) {
      T* out = A.drho;
      out[l] = upd ? r0 - dtiv * (sF[sidx + BX] - Fr0) : r0;
    }
  }

  // ---- the other quantities, QB at a time -------------------------------------------------------------
#pragma unroll
  for (int b0 = 0; b0 < 8; b0 += QB) {   // compile-time batch offsets: the pointer lists stay in the parameter bank
    if (b0 >= A.nq) break;
    T Q[QB], f[QB], a[QB], FQ[QB];
#pragma unroll
    for (int u = 0; u < QB; ++u) {
      Q[u] = T(0);
      if (b0 + u < A.nq && valid) {
        const int sl = A.slot[b0 + u];
        if (A.first) {
          // select from the small per-thread momentum set without dynamic register indexing
          T v = mom[0];
#pragma unroll
          for (int s = 1; s < 7; ++s) v = (sl == s) ? mom[s] : v;
          Q[u] = v;
        } else {
          Q[u] = A.sq[b0 + u][l];
        }
      }
      f[u] = Q[u] * ir;
    }
    __syncthreads();   // previous batch has finished reading sf / sa / sF
#pragma unroll
    for (int u = 0; u < QB; ++u) sf[u * NT + sidx] = f[u];
    __syncthreads();
#pragma unroll
    for (int u = 0; u < QB; ++u) {
      a[u] = T(0);
      if (tm >= 1 && tm < BM - 1) a[u] = vl_slope(sf[u * NT + sidx - BX], f[u], sf[u * NT + sidx + BX], invd0, invdp);
      sa[u * NT + sidx] = a[u];
    }
    __syncthreads();
#pragma unroll
    for (int u = 0; u < QB; ++u) {
      T fs = f[u];
      if (tm >= 1) fs = up ? sf[u * NT + sidx - BX] + sa[u * NT + sidx - BX] * hup : f[u] - a[u] * hdn;
      FQ[u] = Fr0 * fs;
      sF[u * NT + sidx] = FQ[u];
    }
    __syncthreads();
    if (inner) {
#pragma unroll
      for (int u = 0; u < QB; ++u) {
        if (b0 + u < A.nq) {
          T* out = A.dq[b0 + u];
          out[l] = upd ? Q[u] - dtiv * (sF[u * NT + sidx + BX] - FQ[u]) : Q[u];
        }
      }
    }
  }
}

template <typename T, int DIR>
static size_t sweep_smem() { return (size_t)3 * QB * Tile<DIR>::BX * Tile<DIR>::BM * sizeof(T); }

// Opt in to more than 48 KB of dynamic shared memory; called once per context, outside graph capture.
template <typename T>
void sweep_setup() {
  cudaFuncSetAttribute(k_sweep<T, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sweep_smem<T, 0>());
  cudaFuncSetAttribute(k_sweep<T, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sweep_smem<T, 1>());
  cudaFuncSetAttribute(k_sweep<T, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sweep_smem<T, 2>());
  cudaGetLastError();
}
template void sweep_setup<double>();
template void sweep_setup<float>();

template <typename T, int DIR>
static int launch_sweep_dir(const Dev<T>& d, const SweepArgs<T>& a, cudaStream_t s) {
  constexpr int BX = Tile<DIR>::BX, BM = Tile<DIR>::BM, INNER = BM - 4;
  dim3 b, g;
  if (DIR == 0) { b = dim3(BM); g = dim3((d.TX + INNER - 1) / INNER, d.TY, d.TZ); }
  else if (DIR == 1) { b = dim3(BX, BM); g = dim3((d.TX + BX - 1) / BX, (d.TY + INNER - 1) / INNER, d.TZ); }
  else { b = dim3(BX, BM); g = dim3((d.TX + BX - 1) / BX, (d.TZ + INNER - 1) / INNER, d.TY); }
  k_sweep<T, DIR><<<g, b, sweep_smem<T, DIR>(), s>>>(d, a);
  return 1;
}

template <typename T>
int launch_sweep(const Dev<T>& d, const SweepArgs<T>& a, int dir, cudaStream_t s) {
  if (dir == 0) return launch_sweep_dir<T, 0>(d, a, s);
  if (dir == 1) return launch_sweep_dir<T, 1>(d, a, s);
  return launch_sweep_dir<T, 2>(d, a, s);
}

// ---- 12d: new velocities from the transported left/right momenta (Eq. 51), active cells ----------------
template <typename T>
__global__ void __launch_bounds__(128) k_newvel(const Dev<T> d, const T* __restrict__ rho, const QSet<T> S,
                                                const State<T> st) {
  if (d.ctl->done) return;
  const int ia = blockIdx.x * blockDim.x + threadIdx.x;
  if (ia >= d.nx) return;
  const int i = d.ngx + ia, j = d.ngy + blockIdx.y, k = d.ngz + blockIdx.z;
  const long long l = d.id(i, j, k);
  const T r0 = rho[l];
  if (d.hasx) {
    const T rx = d.Rx(j, k), rx2om = (rx * rx) * d.om_eff, irx = d.invRx(j, k);
    const long long lm = d.id(d.xw(i - 1), j, k);
    st.vx[l] = ((S.q[2][lm] + S.q[1][l]) / (rho[lm] + r0) - rx2om) * irx;
  }
  if (d.hasy) {
    const long long lm = l - d.pitch;
    st.vy[l] = (S.q[4][lm] + S.q[3][l]) / (rho[lm] + r0);
  }
  if (d.hasz) {
    const long long lm = l - d.plane;
    st.vz[l] = ((S.q[6][lm] + S.q[5][l]) / (rho[lm] + r0)) * d.invRzj[j];
  }
}

template <typename T>
int launch_newvel(const Dev<T>& d, const T* rho, const QSet<T>& set, const State<T>& st, cudaStream_t s) {
  dim3 b(128), g((d.nx + 127) / 128, d.ny, d.nz);
  k_newvel<T><<<g, b, 0, s>>>(d, rho, set, st);
  return 1;
}

#define INST(T)                                                                                    \
  template int launch_sweep<T>(const Dev<T>&, const SweepArgs<T>&, int, cudaStream_t);             \
  template int launch_newvel<T>(const Dev<T>&, const T*, const QSet<T>&, const State<T>&, cudaStream_t);
INST(double)
INST(float)
#undef INST

}  // namespace fg
