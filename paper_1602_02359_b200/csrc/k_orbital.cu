// k_orbital.cu -- the FARGO orbital-advection step (section 3.5.1).  For each ring (j,k) the
// uniform part v0_jk of the azimuthal velocity (Eq. 72) displaces the ring by s = v0 dt / LX cells, split
// (Eqs. 65-68) into N = nearest integer (Eq. 66; reading G11: floor(s + 1/2)) and xi = s - N, |xi| <= 1/2.
// The fractional part is advected conservatively (Eq. 70) with the Piecewise Parabolic Advection star
// values on rho and q = Q/rho (reading G17); the integer part is a circular permutation
// (Eq. 69), done here for free by shifting the STORE index of the same kernel (aligned loads,
// shifted but still contiguous stores) instead of a separate pass over the data.
#include "kernels.h"

namespace fg {

constexpr int OBM = 256;         // threads = cells per tile along the ring, 3 halo cells per side
constexpr int OIN = OBM - 6;

// PPA star value on the upper face (i+1/2) of this thread's cell; tm = position in the tile.
// Shared arrays (OBM each): s_f cell values, s_dm monotonised differences, s_fu un-limited right interface
// values, s_fl / s_fr limited interface values.  Valid for tm in [2, OBM-4].
template <typename T>
__device__ __forceinline__ T ppa_star_upper(const T f, const int tm, const bool fwd, const T x, const T x1x,
                                            T* s_f, T* s_dm, T* s_fu, T* s_fl, T* s_fr) {
  s_f[tm] = f;
  __syncthreads();
  T a = T(0), b = T(0), dm = T(0);
  if (tm >= 1 && tm < OBM - 1) {
    const T fm = s_f[tm - 1], fp = s_f[tm + 1];
    a = f - fm; b = fp - f;
    const T dd = T(0.5) * (fp - fm);
    if (!(a * b <= T(0))) {
      const T mm = rmin(rmin(T(2) * rabs(a), T(2) * rabs(b)), rabs(dd));
      dm = dd < T(0) ? -mm : mm;
    }
  }
  s_dm[tm] = dm;
  __syncthreads();
  T fr = f;
  if (tm < OBM - 1) fr = (f + T(0.5) * (s_f[tm + 1] - f)) - rdiv(s_dm[tm + 1] - dm, T(6));   // Eq. 71
  s_fu[tm] = fr;
  __syncthreads();
  T fl = tm >= 1 ? s_fu[tm - 1] : f;
  if (a * b <= T(0)) { fl = f; fr = f; }   // the three mutually exclusive tests of P:484
  else {
    const T D = fr - fl;
    const T C = f - T(0.5) * (fl + fr);
    const T DC = D * C, D26 = rdiv(D * D, T(6));
    if (DC > D26) fl = T(3) * f - T(2) * fr;
    else if (-D26 > DC) fr = T(3) * f - T(2) * fl;
  }
  s_fl[tm] = fl; s_fr[tm] = fr;
  __syncthreads();
  // upwind cell of face i+1/2 (formula at P:470; reading G15: x = |xi| in both branches)
  const int u = fwd ? tm : (tm + 1 < OBM ? tm + 1 : tm);
  const T fu = s_f[u], flu = s_fl[u], fru = s_fr[u];
  const T edge = fwd ? fru : flu;
  return (edge + x * (fu - edge)) + x1x * ((T(2) * fu - fru) - flu);
}

template <typename T>
__global__ void __launch_bounds__(OBM) k_orbital(const Dev<T> d, const SweepArgs<T> A, T* __restrict__ nshift_out) {
  if (d.ctl->done) return;
  __shared__ T s_f[OBM], s_dm[OBM], s_fu[OBM], s_fl[OBM], s_fr[OBM], s_F[OBM];
  const int tm = threadIdx.x, j = blockIdx.y, k = blockIdx.z, n = d.nx;
  const int iu = blockIdx.x * OIN - 3 + tm;   // un-wrapped cell index
  int i = iu % n; if (i < 0) i += n;
  const bool inner = tm >= 3 && tm < OBM - 3 && iu < n;

  // ring quantities (uniform over the block)
  const T dt = (T)d.ctl->dt;
  const T s = (A.v0[d.rid(j, k)] * dt) * d.invLX(j, k);
  const T N = floor(s + T(0.5));
  const T xi = s - N;
  const T g = (d.LX(j, k) * d.Sx(j, k)) * d.invV(j, k);
  const bool fwd = xi >= T(0);
  const T x = rabs(xi), x1x = x * (T(1) - x);
  const long long Nl = (long long)N;
  const int sh = (int)(((Nl % n) + n) % n);
  if (nshift_out && blockIdx.x == 0 && tm == 0) nshift_out[d.rid(j, k)] = N;
  int io = i + sh; if (io >= n) io -= n;
  const long long row = d.id(0, j, k);
  const long long l = row + i, lo = row + io;

  const T r0 = A.srho[l];
  const T ir = rdiv(T(1), r0);
  const T rs = ppa_star_upper(r0, tm, fwd, x, x1x, s_f, s_dm, s_fu, s_fl, s_fr);
  const T Fr = xi * rs;   // mass through face i+1/2 per unit of (LX Sx)
  s_F[tm] = Fr;
  __syncthreads();
  if (inner) A.drho[lo] = r0 - g * (Fr - s_F[tm - 1]);

#pragma unroll
  for (int q = 0; q < 7; ++q) {
    if (q >= A.nq) break;
    const T Q = A.sq[q][l];
    const T fs = ppa_star_upper(Q * ir, tm, fwd, x, x1x, s_f, s_dm, s_fu, s_fl, s_fr);
    const T FQ = Fr * fs;
    s_F[tm] = FQ;
    __syncthreads();
    if (inner) A.dq[q][lo] = Q - g * (FQ - s_F[tm - 1]);
  }
}

template <typename T>
int launch_orbital(const Dev<T>& d, const SweepArgs<T>& a, T* nshift_out, cudaStream_t s) {
  dim3 b(OBM), g((d.nx + OIN - 1) / OIN, d.TY, d.TZ);
  k_orbital<T><<<g, b, 0, s>>>(d, a, nshift_out);
  return 1;
}

template int launch_orbital<double>(const Dev<double>&, const SweepArgs<double>&, double*, cudaStream_t);
template int launch_orbital<float>(const Dev<float>&, const SweepArgs<float>&, float*, cudaStream_t);

}  // namespace fg
