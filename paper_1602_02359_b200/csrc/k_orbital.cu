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
  if (tm < OBM - 1) fr = rfma(T(0.5), s_f[tm + 1] - f, f) - rdiv(s_dm[tm + 1] - dm, T(6));   // Eq. 71
  s_fu[tm] = fr;
  __syncthreads();
  T fl = tm >= 1 ? s_fu[tm - 1] : f;
  if (a * b <= T(0)) { fl = f; fr = f; }   // the three mutually exclusive tests of P:484
  else {
    const T D = fr - fl;
    const T C = rfma(T(-0.5), fl + fr, f);
    const T DC = D * C, D26 = rdiv(D * D, T(6));
    if (DC > D26) fl = rfma(T(3), f, -(T(2) * fr));
    else if (-D26 > DC) fr = rfma(T(3), f, -(T(2) * fl));
  }
  s_fl[tm] = fl; s_fr[tm] = fr;
  __syncthreads();
  // upwind cell of face i+1/2 (formula at P:470; reading G15: x = |xi| in both branches)
  const int u = fwd ? tm : (tm + 1 < OBM ? tm + 1 : tm);
  const T fu = s_f[u], flu = s_fl[u], fru = s_fr[u];
  const T edge = fwd ? fru : flu;
  return rfma(x1x, rfma(T(2), fu, -fru) - flu, rfma(x, fu - edge, edge));
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
  if (inner) A.drho[lo] = rfma(-g, Fr - s_F[tm - 1], r0);

#pragma unroll
  for (int q = 0; q < 7; ++q) {
    if (q >= A.nq) break;
    const T Q = A.sq[q][l];
    const T fs = ppa_star_upper(Q * ir, tm, fwd, x, x1x, s_f, s_dm, s_fu, s_fl, s_fr);
    const T FQ = Fr * fs;
    s_F[tm] = FQ;
    __syncthreads();
    if (inner) A.dq[q][lo] = rfma(-g, FQ - s_F[tm - 1], Q);
  }
}

// ---- two cells per lane, no shared memory, no barriers -----------------------------------------------------
// A warp owns 64 consecutive cells of one ring: lane L holds tile positions t = 2L, 2L+1 as one 16-byte
// vector per array.  The PPA chain (difference -> monotonised slope -> interface value -> limiter -> star
// value -> flux difference) needs 3 cells to the left and 3 to the right of a stored cell (the upwind cell of
// its upper face may be the next one); positions 4 .. 59 are stored (56 per warp), lanes 0, 1, 30 and 31
// are recomputed halo.  Per quantity five values cross
// lanes by shuffle (two more when xi < 0); the quantities are independent, so their chains interleave.
// Every expression is the one of k_orbital above: results are bit-identical.  Needs an even nx.
constexpr int O2W = 4;          // warps (rings) per block
constexpr int O2IN = 56;        // cells stored per warp

template <typename T> struct OPair;
template <> struct OPair<double> { using type = double2; };
template <> struct OPair<float> { using type = float2; };

template <typename T> __device__ __forceinline__ T o_up1(T v) { return __shfl_up_sync(0xffffffffu, v, 1); }
template <typename T> __device__ __forceinline__ T o_dn1(T v) { return __shfl_down_sync(0xffffffffu, v, 1); }

template <typename T>
__device__ __forceinline__ T ppa_mono(const T fm, const T f, const T fp, bool& flat) {
  const T a = f - fm, b = fp - f;
  const T dd = T(0.5) * (fp - fm);
  flat = a * b <= T(0);
  const T mm = rmin(rmin(T(2) * rabs(a), T(2) * rabs(b)), rabs(dd));
  // sign(dd) mm with one LOP3 on the high word (mm >= 0); where dd is a zero mm is a zero too and only the sign of
  // that zero can differ from the select's, which no later value depends on
  const T dm = copysign(mm, dd);
  return flat ? T(0) : dm;
}

template <typename T>
__device__ __forceinline__ void ppa_limit(const T f, const bool flat, T& fl, T& fr) {   // the three tests of P:484
  const T D = fr - fl;
  const T C = rfma(T(-0.5), fl + fr, f);
  const T DC = D * C, D26 = rdiv6(D * D);
  const T fl2 = rfma(T(3), f, -(T(2) * fr)), fr2 = rfma(T(3), f, -(T(2) * fl));
  const bool c1 = DC > D26, c2 = -D26 > DC;
  const T ol = flat ? f : (c1 ? fl2 : fl);
  const T orr = flat ? f : (c1 ? fr : (c2 ? fr2 : fr));
  fl = ol; fr = orr;
}

// star values on the upper faces of the lane's two cells (reading G15: x = |xi| in both branches).  FWD (xi >= 0:
// the upwind cell of a face is the cell itself, otherwise the next one) is uniform over a ring, hence over the warp:
// the kernel branches on it ONCE around its whole body, so each copy is a single basic block without the eight
// selects (sixteen SEL instructions) per pair that a run-time choice costs, and the xi >= 0 copy drops two shuffles.
template <typename T, bool FWD>
__device__ __forceinline__ void ppa_pair(const T fA, const T fB, const T x, const T x1x, T& sA, T& sB) {
  const T fm = o_up1(fB);        // position t-1
  const T fn = o_dn1(fA);        // position t+2
  bool flatA, flatB;
  const T dmA = ppa_mono(fm, fA, fB, flatA), dmB = ppa_mono(fA, fB, fn, flatB);
  const T dmn = o_dn1(dmA);
  const T fuA = rfma(T(0.5), fB - fA, fA) - rdiv6(dmB - dmA);   // Eq. 71, un-limited
  const T fuB = rfma(T(0.5), fn - fB, fB) - rdiv6(dmn - dmB);
  T flA = o_up1(fuB), frA = fuA, flB = fuA, frB = fuB;
  ppa_limit(fA, flatA, flA, frA);
  ppa_limit(fB, flatB, flB, frB);
  if (FWD) {
    sA = rfma(x1x, rfma(T(2), fA, -frA) - flA, rfma(x, fA - frA, frA));
    sB = rfma(x1x, rfma(T(2), fB, -frB) - flB, rfma(x, fB - frB, frB));
  } else {
    const T fln = o_dn1(flA), frn = o_dn1(frA);
    sA = rfma(x1x, rfma(T(2), fB, -frB) - flB, rfma(x, fB - flB, flB));
    sB = rfma(x1x, rfma(T(2), fn, -frn) - fln, rfma(x, fn - fln, fln));
  }
}

template <typename T, int NQ, bool FWD>
__device__ __forceinline__ void orbital2_body(const SweepArgs<T>& A, const typename OPair<T>::type r2,
                                              const typename OPair<T>::type (&Q2)[NQ], const T xi, const T x, const T x1x,
                                              const T g, const long long row, const int io, const int io1,
                                              const bool stA, const bool stB, const bool vec) {
  const T irA = rdiv(T(1), r2.x), irB = rdiv(T(1), r2.y);
  T sA, sB;
  ppa_pair<T, FWD>(r2.x, r2.y, x, x1x, sA, sB);
  const T FrA = xi * sA, FrB = xi * sB;   // mass through the upper face per unit of (LX Sx)
  {
    const T Fm = o_up1(FrB);
    const T oA = rfma(-g, FrA - Fm, r2.x), oB = rfma(-g, FrB - FrA, r2.y);
    st2_if(A.drho + row + io, oA, oB, vec && stB);
    st_if(A.drho + row + io, oA, stA && !(vec && stB));
    st_if(A.drho + row + io1, oB, stB && !vec);
  }
#pragma unroll
  for (int q = 0; q < NQ; ++q) {
    ppa_pair<T, FWD>(Q2[q].x * irA, Q2[q].y * irB, x, x1x, sA, sB);
    const T FA = FrA * sA, FB = FrB * sB;
    const T Fm = o_up1(FB);
    const T oA = rfma(-g, FA - Fm, Q2[q].x), oB = rfma(-g, FB - FA, Q2[q].y);
    st2_if(A.dq[q] + row + io, oA, oB, vec && stB);
    st_if(A.dq[q] + row + io, oA, stA && !(vec && stB));
    st_if(A.dq[q] + row + io1, oB, stB && !vec);
  }
}

template <typename T, int NQ>
__global__ void __launch_bounds__(32 * O2W) k_orbital2(const Dev<T> d, const SweepArgs<T> A, T* __restrict__ nshift_out) {
  if (d.ctl->done) return;
  using P2 = typename OPair<T>::type;
  const int lane = threadIdx.x;
  const int n = d.nx, ntile = (n + O2IN - 1) / O2IN;
  const int tile = blockIdx.x % ntile;   // 1-D grid: tiles of a ring are neighbours in launch order
  const int ring = (blockIdx.x / ntile) * O2W + threadIdx.y;
  if (ring >= d.TY * d.TZ) return;   // whole warps leave together
  const int j = ring % d.TY, k = ring / d.TY;
  const int iu = tile * O2IN - 4 + 2 * lane;   // un-wrapped index of the lane's first cell (even)
  int i = iu % n; if (i < 0) i += n;

  const T dt = (T)d.ctl->dt;
  const T s = (A.v0[ring] * dt) * d.invLX(j, k);
  const T N = floor(s + T(0.5));
  const T xi = s - N;
  const T g = (d.LX(j, k) * d.Sx(j, k)) * d.invV(j, k);
  const bool fwd = xi >= T(0);
  const T x = rabs(xi), x1x = x * (T(1) - x);
  const long long Nl = (long long)N;
  const int sh = (int)(((Nl % n) + n) % n);
  if (nshift_out && tile == 0 && lane == 0) nshift_out[ring] = N;
  int io = i + sh; if (io >= n) io -= n;
  int io1 = io + 1; if (io1 >= n) io1 -= n;
  const long long row = d.id(0, j, k);
  const long long l = row + i;
  const bool stA = lane >= 2 && lane <= 29 && iu < n, stB = stA && iu + 1 < n;
  const bool vec = (sh & 1) == 0;   // even shift: the pair stays 16-byte aligned

  // loads, all up front
  const P2 r2 = *reinterpret_cast<const P2*>(A.srho + l);
  P2 Q2[NQ];
#pragma unroll
  for (int q = 0; q < NQ; ++q) Q2[q] = *reinterpret_cast<const P2*>(A.sq[q] + l);

  // a vote result is uniform by construction: ptxas then emits no WARPSYNC region around the shuffles of either copy
  if (__all_sync(0xffffffffu, fwd)) orbital2_body<T, NQ, true>(A, r2, Q2, xi, x, x1x, g, row, io, io1, stA, stB, vec);
  else orbital2_body<T, NQ, false>(A, r2, Q2, xi, x, x1x, g, row, io, io1, stA, stB, vec);
}

template <typename T, int NQ>
static int launch_orbital2(const Dev<T>& d, const SweepArgs<T>& a, T* nshift_out, cudaStream_t s) {
  dim3 b(32, O2W), g((unsigned)(((d.nx + O2IN - 1) / O2IN) * ((d.TY * d.TZ + O2W - 1) / O2W)));
  k_orbital2<T, NQ><<<g, b, 0, s>>>(d, a, nshift_out);
  return 1;
}

template <typename T>
int launch_orbital(const Dev<T>& d, const SweepArgs<T>& a, T* nshift_out, cudaStream_t s) {
  if (d.nx % 2 == 0) {
    switch (a.nq) {
      case 2: return launch_orbital2<T, 2>(d, a, nshift_out, s);
      case 3: return launch_orbital2<T, 3>(d, a, nshift_out, s);
      case 4: return launch_orbital2<T, 4>(d, a, nshift_out, s);
      case 5: return launch_orbital2<T, 5>(d, a, nshift_out, s);
      case 6: return launch_orbital2<T, 6>(d, a, nshift_out, s);
      case 7: return launch_orbital2<T, 7>(d, a, nshift_out, s);
      default: break;
    }
  }
  dim3 b(OBM), g((d.nx + OIN - 1) / OIN, d.TY, d.TZ);
  k_orbital<T><<<g, b, 0, s>>>(d, a, nshift_out);
  return 1;
}

template int launch_orbital<double>(const Dev<double>&, const SweepArgs<double>&, double*, cudaStream_t);
template int launch_orbital<float>(const Dev<float>&, const SweepArgs<float>&, float*, cudaStream_t);

}  // namespace fg
