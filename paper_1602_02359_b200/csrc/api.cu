// api.cu -- the C ABI of include/fargo.h: context, workspace carving, field I/O and the step scheduler
// that enqueues the fixed kernel sequence of one update (Fig. 2, caption P:198) on one CUDA stream,
// with the time step and the clock resident on the device.  With use_graph the sequence of one update
// is captured once into a CUDA graph and replayed (small meshes are launch-bound).
// Product code: nothing here includes, links or calls anything under oracle/.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <string>
#include <vector>

#include "../../include/fargo.h"
#include "kernels.h"
#include "tables.h"

namespace fg {

template <typename T> void sweep_setup();   // k_transport.cu: opt-in shared memory sizes

static thread_local std::string g_init_error;

struct CtxBase {
  virtual ~CtxBase() {}
  std::string err;
  int precision = 64;
  virtual int set_fields(const void*, const void*, const void*, const void*, const void*) = 0;
  virtual int get_fields(void*, void*, void*, void*, void*) = 0;
  virtual int step(int n) = 0;
  virtual int step_until(int stage) = 0;
  virtual int get_time(double*, double*, long long*) = 0;
  virtual int get_array(const char*, void*) = 0;
  virtual void dims(int*, int*, int*, int*, int*, int*) const = 0;
  virtual int update_phase(int) = 0;
  virtual int halo(int, int, int, int, void*) = 0;
  virtual size_t halo_bytes(int, int) const = 0;
  virtual void* dt_ptr() = 0;
  virtual int dt_min_with(const void*) = 0;
  virtual int set_planets(int, const double*, const double*, const double*, const double*, int, double) = 0;
  virtual int get_planets(double*, double*, double*) = 0;
  virtual int set_omega_frame(double) = 0;
  virtual int diagnostics(double*) = 0;
  virtual int diagnostics_noalloc(double*) = 0;
  virtual int set_bfield(const void*, const void*, const void*, double, double, int) = 0;
  virtual int get_bfield(void*, void*, void*) = 0;
  virtual int profile(int enable) = 0;
  virtual int profile_report(char* buf, size_t len) = 0;
  long long launches = 0;
};

static inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Layout {   // sizes shared by fargo_workspace_bytes and fargo_init
  int nx, ny, nz, ngx, ngy, ngz, TX, TY, TZ;
  long long pitch, plane, narr;
  bool xwrap, hasx, hasy, hasz, has_pot, visc, visc3d, fargo, adi, mhd;
  int n3d;             // number of 3-D arrays
  size_t table_elems;  // total 1-D table elements (each table padded to 32 elements)
  size_t bytes(size_t es) const {
    size_t b = 256;                                              // Ctl
    b += align_up(sizeof(PlanetsDev), 256);                      // live planets (NEXT-2)
    b += 256;                                                    // position of the fixed-orbit planet when it moves in the frame
    b += align_up((size_t)planets_blocks(ny, nz) * MAXPL * 3 * sizeof(double), 256);   // their force partials
    b += align_up(table_elems * es, 256);                        // tables
    b += 2 * align_up((size_t)TY * TZ * es, 256);                // v0, nshift
    b += (size_t)n3d * align_up((size_t)narr * es, 256);
    return b;
  }
};

static bool make_layout(Layout& L, const fargo_mesh* m, int geometry, int eos, const fargo_params* p, std::string& err) {
  if (!m || !p) { err = "null mesh or params"; return false; }
  if (m->nx < 1 || m->ny < 1 || m->nz < 1) { err = "mesh extents must be >= 1"; return false; }
  if (geometry < 0 || geometry > 3) { err = "unknown geometry"; return false; }
  if (eos < 0 || eos > 1) { err = "unknown equation of state"; return false; }
  if (p->precision != 64 && p->precision != 32) { err = "precision must be 64 or 32"; return false; }
  for (int dd = 0; dd < 3; ++dd)
    for (int s = 0; s < 2; ++s)
      if (m->bc[dd][s] < 0 || m->bc[dd][s] > 3) { err = "unknown boundary kind"; return false; }
  for (int s = 0; s < 2; ++s)
    if (m->bc[0][s] == FARGO_EXTERNAL || (m->bc[1][s] == FARGO_EXTERNAL && m->ny < 3) || (m->bc[2][s] == FARGO_EXTERNAL && m->nz < 3)) {
      err = "FARGO_EXTERNAL is for the Y and Z faces of a sub-domain of at least 3 layers (X is never cut, P:728)"; return false;
    }
  if (!(m->xmax > m->xmin)) { err = "xmax must exceed xmin"; return false; }
  L.nx = m->nx; L.ny = m->ny; L.nz = m->nz;
  L.hasx = m->nx > 1; L.hasy = m->ny > 1; L.hasz = m->nz > 1;
  if (!L.hasx && !L.hasy && !L.hasz) { err = "at least one direction must have more than one cell"; return false; }
  L.xwrap = m->bc[0][0] == FARGO_PERIODIC;
  if (p->fargo_on && !(L.xwrap && L.hasx)) { err = "orbital advection needs a periodic X axis (P:728)"; return false; }
  const int ng = 3;
  L.ngx = (L.hasx && !L.xwrap) ? ng : 0;
  L.ngy = L.hasy ? ng : 0;
  L.ngz = L.hasz ? ng : 0;
  L.TX = L.nx + 2 * L.ngx; L.TY = L.ny + 2 * L.ngy; L.TZ = L.nz + 2 * L.ngz;
  L.pitch = (long long)align_up((size_t)L.TX, 16);
  L.plane = L.pitch * L.TY;
  L.narr = L.plane * L.TZ;
  if (geometry == FARGO_SHEARING_SHEET && !(L.hasx && L.xwrap && L.hasy)) {
    err = "the shearing sheet needs nx > 1 with a periodic X axis and ny > 1 (Tab. 1)"; return false;
  }
  const bool cartesian_metric = geometry == FARGO_CARTESIAN || geometry == FARGO_SHEARING_SHEET;
  L.has_pot = !cartesian_metric && (p->gm_star != 0.0 || p->planet_mass != 0.0);
  L.visc3d = p->nu > 0.0 && L.hasx && L.hasy && L.hasz;                                    // Eqs. B1-B6, any geometry
  L.visc = L.visc3d || (p->nu > 0.0 && geometry == FARGO_CYLINDRICAL && L.hasx && L.hasy && !L.hasz && L.xwrap);
  L.fargo = p->fargo_on != 0;
  L.adi = eos == FARGO_ADIABATIC;
  L.mhd = p->mhd != 0;
  if (L.mhd && !(L.hasx && L.hasy && L.hasz)) {
    err = "MHD: 3-D meshes (1.5-D and 2.5-D problems run on thin 3-D meshes)"; return false;
  }
  if (L.mhd && geometry == FARGO_SPHERICAL && p->fargo_on) {
    err = "MHD: the orbital advection of B (cell 11) is built for Cartesian and cylindrical meshes (DESIGN.md G38)"; return false;
  }
  for (int dd = 1; dd < 3 && L.mhd; ++dd)
    for (int s = 0; s < 2; ++s)
      if (m->bc[dd][s] == FARGO_EXTERNAL) { err = "MHD is not available on sub-domains"; return false; }
  L.n3d = 5 + (L.has_pot ? 1 : 0) + 16 + 4 + (L.mhd ? 13 : 0);   // state, Phi, two transport sets, the source step's output, MHD
  const size_t pad = 32;
  auto t1 = [&](int n) { return align_up((size_t)n, pad); };
  L.table_elems = 7 * t1(L.TY + 1) + 11 * t1(L.TY + 1) + 10 * t1(L.TZ + 1) + 6 * t1(L.TZ + 1) + 2 * t1(L.TX);
  return true;
}

template <typename T>
struct Sim : CtxBase {
  Layout L;
  Dev<T> d;
  State<T> st;
  T *phi = nullptr, *v0 = nullptr, *nshift = nullptr;
  T* ppos = nullptr;          // device: (x_p, y_p) of the fixed-orbit planet when it moves in the frame
  double* hclock = nullptr;   // pinned host: the clock read back for the planet's azimuth
  T* hppos = nullptr;         // pinned host: (x_p, y_p) formed by the host node with libm
  PlanetsDev* pl = nullptr;   // live planets (NEXT-2): device state, force partials, host copy of the constants
  double* pl_part = nullptr;
  int npl = 0, pl_mode = 0;
  T* pool[16];
  T* alt[4];            // e, vx, vy, vz written by the fused source step (the state stays intact while it is read)
  T *bfield[3] = {nullptr, nullptr, nullptr}, *emf[3], *bstar[6], *vxres = nullptr;   // MHD (NEXT-4): B on faces, EMFs and star values on edges
  bool mhd_on = false;  // fargo_set_bfield was called
  int mhd_passive = 0;
  double mu0 = 1.0, eta = 0.0;
  int next_phase = 0;   // slab mode: the phase fargo_update_phase expects next
  State<T> s2m;         // slab mode: where e and v are after the source step (phase 2 -> phases 3, 4)
  bool fuse_source = false;
  bool fuse_visc = false;   // 7d in one pass (k_visc3d_fused)
  bool fuse_dt = false;   // Eq. 51 and the next update's per-cell CFL rate in one kernel (k_newvel_dt)
  bool dt_ready = false;  // ctl->m2bits holds the running max for the coming update
  Ctl* ctl = nullptr;
  fargo_params prm;
  int geometry, eos;
  cudaStream_t stream = nullptr;
  cudaGraphExec_t gexec = nullptr;
  cudaGraphExec_t gphase[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};   // sub-domains: one captured graph per phase
  int gphase_launches[5] = {0, 0, 0, 0, 0};
  void drop_graphs() {
    if (gexec) { cudaGraphExecDestroy(gexec); gexec = nullptr; }
    for (auto& g : gphase) if (g) { cudaGraphExecDestroy(g); g = nullptr; }
  }
  int launches_per_step = 0;
  bool midstep = false, have_fields = false, pot_static = true, pot_valid = false;
  std::map<std::string, T*> dbg;
  // per-kernel CUDA-event timing (fargo_profile): one event pair per launcher call, on the context's stream
  struct Span { const char* name; cudaEvent_t a, b; int nk; };
  bool prof = false;
  std::vector<Span> spans;
  // transport plan
  int npass = 0, pass_kind[4];   // 0,1,2 = sweep direction, 3 = orbital
  int nq = 0, slots[8];

  ~Sim() override {
    cudaStreamSynchronize(stream);   // nothing of this context may still be running when the caller frees the workspace
    drop_graphs();
    if (hclock) cudaFreeHost(hclock);
    for (auto& sp : spans) { cudaEventDestroy(sp.a); cudaEventDestroy(sp.b); }
  }

  // run one launcher, bracketed by events when profiling
  template <typename F> int timed(const char* name, F&& f) {
    if (!prof) return f();
    Span sp{name, nullptr, nullptr, 0};
    cudaEventCreate(&sp.a); cudaEventCreate(&sp.b);
    cudaEventRecord(sp.a, stream);
    sp.nk = f();
    cudaEventRecord(sp.b, stream);
    spans.push_back(sp);
    return sp.nk;
  }

  int profile(int enable) override {
    for (auto& sp : spans) { cudaEventDestroy(sp.a); cudaEventDestroy(sp.b); }
    spans.clear();
    prof = enable != 0;
    return FARGO_OK;
  }

  int profile_report(char* buf, size_t len) override {
    if (!buf || len == 0) { err = "null buffer"; return FARGO_EINVAL; }
    if (!ck(cudaStreamSynchronize(stream), "profile sync")) return FARGO_ECUDA;
    std::map<std::string, std::pair<long long, double>> acc;   // name -> (kernel launches, total ms)
    std::vector<std::string> order;
    for (auto& sp : spans) {
      float ms = 0.f;
      if (!ck(cudaEventElapsedTime(&ms, sp.a, sp.b), "cudaEventElapsedTime")) return FARGO_ECUDA;
      if (!acc.count(sp.name)) order.push_back(sp.name);
      acc[sp.name].first += sp.nk;
      acc[sp.name].second += ms;
    }
    std::string out;
    char line[160];
    for (auto& nm : order) {
      snprintf(line, sizeof line, "%s %lld %.6f\n", nm.c_str(), acc[nm].first, acc[nm].second);
      out += line;
    }
    if (out.size() + 1 > len) { err = "profile buffer too small"; return FARGO_EINVAL; }
    memcpy(buf, out.c_str(), out.size() + 1);
    return FARGO_OK;
  }

  bool ck(cudaError_t e, const char* what) {
    if (e == cudaSuccess) return true;
    char buf[256];
    snprintf(buf, sizeof buf, "%s: %s", what, cudaGetErrorString(e));
    err = buf;
    return false;
  }

  T* set_arr(int s, int slot /* -1 = rho, 0 = e, 1..6 momenta */) { return pool[s * 8 + 1 + slot]; }

  int init(const fargo_mesh* m, int geo_in, int eos_, const fargo_params* p) {
    // the sheet is the Cartesian mesh (Tab. 5 unchanged) with Tab. 2's X momentum and Eq. 29 switched on (G32)
    const bool sheet = geo_in == FARGO_SHEARING_SHEET;
    const int geo = sheet ? FARGO_CARTESIAN : geo_in;
    geometry = geo_in; eos = eos_; prm = *p;
    stream = (cudaStream_t)p->cuda_stream;
    int ndev = 0;
    if (!ck(cudaGetDeviceCount(&ndev), "cudaGetDeviceCount") || ndev < 1) {
      if (err.empty()) err = "no CUDA device";
      return FARGO_ECUDA;
    }
    const size_t need = L.bytes(sizeof(T));
    if (!p->workspace || p->workspace_bytes < need) { err = "workspace missing or too small"; return FARGO_ENOMEM; }
    if (((uintptr_t)p->workspace) % 256) { err = "workspace must be 256-byte aligned"; return FARGO_EINVAL; }
    cudaPointerAttributes at;
    if (!ck(cudaPointerGetAttributes(&at, p->workspace), "cudaPointerGetAttributes(workspace)")) return FARGO_ECUDA;
    if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged) {
      err = "workspace is not device memory";
      return FARGO_EINVAL;
    }

    // ---- host tables (fp64, libm) ----
    const double dx = (m->xmax - m->xmin) / (double)m->nx;
    // a slab's cut faces (FARGO_EXTERNAL) come with the neighbour's true edges: 3 before the active ones when the lower
    // face is cut, 3 after them when the upper one is (a continuation by the last cell's width would differ from the
    // undivided mesh, in rounding on a uniform mesh and altogether on a non-uniform one)
    const int elo = m->bc[1][0] == FARGO_EXTERNAL ? 3 : 0, ehi = m->bc[1][1] == FARGO_EXTERNAL ? 3 : 0;
    if ((elo || ehi) && !m->yedges) { err = "a slab needs its yedges, with the neighbours' edges beyond the cut faces"; return FARGO_EINVAL; }
    std::vector<double> ye = ghosted_edges(m->yedges ? m->yedges + elo : nullptr, L.ny, L.ngy, m->ymin, m->ymax);
    for (int g = 0; g < elo; ++g) ye[g] = m->yedges[g];
    for (int g = 0; g < ehi; ++g) ye[L.ngy + L.ny + 1 + g] = m->yedges[elo + L.ny + 1 + g];
    const int zlo = m->bc[2][0] == FARGO_EXTERNAL ? 3 : 0, zhi = m->bc[2][1] == FARGO_EXTERNAL ? 3 : 0;
    if ((zlo || zhi) && !m->zedges) { err = "a sub-domain cut in Z needs its zedges, with the neighbours' edges beyond the cut faces"; return FARGO_EINVAL; }
    std::vector<double> ze = ghosted_edges(m->zedges ? m->zedges + zlo : nullptr, L.nz, L.ngz, m->zmin, m->zmax);
    for (int g = 0; g < zlo; ++g) ze[g] = m->zedges[g];
    for (int g = 0; g < zhi; ++g) ze[L.ngz + L.nz + 1 + g] = m->zedges[zlo + L.nz + 1 + g];
    for (size_t n = 1; n < ye.size(); ++n) if (!(ye[n] > ye[n - 1])) { err = "yedges must increase"; return FARGO_EINVAL; }
    for (size_t n = 1; n < ze.size(); ++n) if (!(ze[n] > ze[n - 1])) { err = "zedges must increase"; return FARGO_EINVAL; }
    HostTables ht;
    build_tables(ht, geo, L.TX, L.TY, L.TZ, L.ngx, m->xmin, dx, ye, ze);

    // ---- carve the workspace ----
    unsigned char* base = (unsigned char*)p->workspace;
    size_t off = 0;
    ctl = (Ctl*)base; off += 256;
    pl = (PlanetsDev*)(base + off); off += align_up(sizeof(PlanetsDev), 256);
    ppos = (T*)(base + off); off += 256;
    pl_part = (double*)(base + off); off += align_up((size_t)planets_blocks(L.ny, L.nz) * MAXPL * 3 * sizeof(double), 256);
    T* tab = (T*)(base + off);
    std::vector<T> htab(L.table_elems, T(0));
    size_t tpos = 0;
    auto put = [&](const std::vector<double>& v) -> const T* {
      const T* dev = tab + tpos;
      for (size_t n = 0; n < v.size(); ++n) htab[tpos + n] = (T)v[n];
      tpos += align_up(v.size(), 32);
      return dev;
    };
    memset(&d, 0, sizeof d);
    d.ye = put(ht.ye); d.yc = put(ht.yc); d.inv_ye = put(ht.inv_ye); d.inv_yc = put(ht.inv_yc);
    d.LY = put(ht.LY); d.invLY = put(ht.invLY); d.invDY = put(ht.invDY);
    d.sxj = put(ht.sxj); d.syj = put(ht.syj); d.szj = put(ht.szj); d.invVj = put(ht.invVj);
    d.Rxj = put(ht.Rxj); d.invRxj = put(ht.invRxj); d.LXj = put(ht.LXj); d.invLXj = put(ht.invLXj);
    d.Rzj = put(ht.Rzj); d.invRzj = put(ht.invRzj);
    d.zc = put(ht.zc); d.dz = put(ht.dz); d.invdz = put(ht.invdz); d.invdzc = put(ht.invdzc);
    d.sxk = put(ht.sxk); d.syk = put(ht.syk); d.inv_syk = put(ht.inv_syk); d.szk = put(ht.szk);
    d.Rxk = put(ht.Rxk); d.invRxk = put(ht.invRxk);
    d.sin_zc = put(ht.sin_zc); d.cos_zc = put(ht.cos_zc); d.sin_ze = put(ht.sin_ze); d.cot_ze = put(ht.cot_ze);
    d.cos_xc = put(ht.cos_xc); d.sin_xc = put(ht.sin_xc);
    d.cot_zc = put(ht.cot_zc); d.inv_sin_ze = put(ht.inv_sin_ze);
    {
      std::vector<double> Vj(ht.invVj.size());
      for (size_t n = 0; n < Vj.size(); ++n) Vj[n] = 1.0 / ht.invVj[n];
      d.Vj = put(Vj);
    }
    if (tpos > L.table_elems) { err = "internal: table area overflow"; return FARGO_EINVAL; }
    off += align_up(L.table_elems * sizeof(T), 256);
    const size_t ringb = align_up((size_t)L.TY * L.TZ * sizeof(T), 256);
    v0 = (T*)(base + off); off += ringb;
    nshift = (T*)(base + off); off += ringb;
    const size_t arrb = align_up((size_t)L.narr * sizeof(T), 256);
    auto arr = [&]() { T* a = (T*)(base + off); off += arrb; return a; };
    st.rho = arr(); st.e = arr(); st.vx = arr(); st.vy = arr(); st.vz = arr();
    if (L.has_pot) phi = arr();
    for (int n = 0; n < 16; ++n) pool[n] = arr();
    for (int n = 0; n < 4; ++n) alt[n] = arr();
    if (L.mhd) {
      for (int n = 0; n < 3; ++n) bfield[n] = arr();
      for (int n = 0; n < 3; ++n) emf[n] = arr();
      for (int n = 0; n < 6; ++n) bstar[n] = arr();
      vxres = arr();   // v_X - v0: what cell 8 sees under orbital advection
    }
    if (off > p->workspace_bytes) { err = "internal: workspace overflow"; return FARGO_ENOMEM; }

    if (!ck(cudaMemsetAsync(base, 0, off, stream), "cudaMemsetAsync(workspace)")) return FARGO_ECUDA;
    if (!ck(cudaMemcpyAsync(tab, htab.data(), L.table_elems * sizeof(T), cudaMemcpyHostToDevice, stream),
            "upload tables")) return FARGO_ECUDA;
    if (!ck(cudaStreamSynchronize(stream), "init sync")) return FARGO_ECUDA;

    // ---- device descriptor ----
    d.nx = L.nx; d.ny = L.ny; d.nz = L.nz; d.ngx = L.ngx; d.ngy = L.ngy; d.ngz = L.ngz;
    d.TX = L.TX; d.TY = L.TY; d.TZ = L.TZ; d.pitch = L.pitch; d.plane = L.plane; d.narr = L.narr;
    d.geometry = geo; d.eos = eos_;
    d.xwrap = L.xwrap; d.hasx = L.hasx; d.hasy = L.hasy; d.hasz = L.hasz;
    d.fargo = L.fargo; d.has_pot = L.has_pot; d.visc = L.visc;
    for (int a = 0; a < 3; ++a) for (int s = 0; s < 2; ++s) d.bc[a][s] = m->bc[a][s];
    d.dx = (T)dx; d.invdx = (T)(1.0 / dx);
    d.gamma = (T)p->gamma; d.gm1 = (T)(p->gamma - 1.0); d.gg1 = (T)(p->gamma * (p->gamma - 1.0));
    d.cfl = (T)p->cfl; d.cvnr2 = (T)p->cvnr2; d.nu = (T)p->nu;
    d.omega = (T)p->omega_frame; d.om_eff = geo == FARGO_CARTESIAN ? T(0) : (T)p->omega_frame;
    d.shear = sheet ? 1 : 0;
    d.two_om = sheet ? (T)(2.0 * p->omega_frame) : T(0);
    d.four_a_om = sheet ? (T)((4.0 * p->oort_a) * p->omega_frame) : T(0);
    d.shear_c0 = (T)p->shear_c0;
    d.c3 = (T)(4.0 * p->cvnr2); d.c4 = (T)(4.0 * p->nu);
    d.t_stop = p->t_stop; d.dt_fixed = p->dt_fixed;
    d.ctl = ctl;
    pot_static = !(L.has_pot && p->planet_mass != 0.0 && p->planet_omega != p->omega_frame);
    d.seam_above = (p->kernel_plan & FARGO_PLAN_SEAM_ABOVE) ? 1 : 0;
    if (L.has_pot && p->planet_mass != 0.0) {   // the planet may move in the frame (now, or after fargo_set_omega_frame)
      if (!ck(cudaHostAlloc((void**)&hclock, 64, cudaHostAllocDefault), "cudaHostAlloc(planet clock)")) return FARGO_ENOMEM;
      hppos = (T*)(hclock + 2);
    }

    // ---- transport plan: X, Y, Z sweeps (reading G14), then orbital advection ----
    npass = 0;
    if (L.hasx) pass_kind[npass++] = 0;
    if (L.hasy) pass_kind[npass++] = 1;
    if (L.hasz) pass_kind[npass++] = 2;
    if (L.fargo) pass_kind[npass++] = 3;
    nq = 0;
    if (L.adi) slots[nq++] = 0;
    if (L.hasx) { slots[nq++] = 1; slots[nq++] = 2; }
    if (L.hasy) { slots[nq++] = 3; slots[nq++] = 4; }
    if (L.hasz) { slots[nq++] = 5; slots[nq++] = 6; }
    sweep_setup<T>();
    // with viscosity the fused pass must be followed by the fused 7d (it then also produces the ghost layer 7d reads)
    fuse_visc = L.visc3d && source_d3_fused_ok<T>(d) && !(p->kernel_plan & FARGO_PLAN_UNFUSED_VISC);
    fuse_source = source_fused_ok<T>(d) && !(p->kernel_plan & FARGO_PLAN_UNFUSED_SOURCE) && (!L.visc || fuse_visc);
    fuse_dt = newvel_dt_ok<T>(d) && !(p->kernel_plan & FARGO_PLAN_UNFUSED_DT);
    return FARGO_OK;
  }

  // ---- field I/O --------------------------------------------------------------------------------------
  static bool on_device(const void* p) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
  }

  int set_fields(const void* rho, const void* e, const void* vx, const void* vy, const void* vz) override {
    if (!rho || !e || !vx) { err = "rho, e and vx are required"; return FARGO_EINVAL; }
    if ((L.hasy && !vy) || (L.hasz && !vz)) { err = "vy / vz required when that direction is present"; return FARGO_EINVAL; }
    const size_t nact = (size_t)L.nx * L.ny * L.nz;
    // ghost-inclusive arrays start from zero, as every intermediate does
    unsigned char* a0 = (unsigned char*)st.rho;
    unsigned char* a1 = (unsigned char*)alt[3] + align_up((size_t)L.narr * sizeof(T), 256);
    if (!ck(cudaMemsetAsync(a0, 0, (size_t)(a1 - a0), stream), "cudaMemsetAsync(fields)")) return FARGO_ECUDA;
    if (!ck(cudaMemsetAsync(ctl, 0, sizeof(Ctl), stream), "cudaMemsetAsync(ctl)")) return FARGO_ECUDA;
    const void* src[5] = {rho, e, vx, L.hasy ? vy : nullptr, L.hasz ? vz : nullptr};
    T* dst[5] = {st.rho, st.e, st.vx, st.vy, st.vz};
    T* staging = pool[15];   // dead between updates
    for (int f = 0; f < 5; ++f) {
      if (!src[f]) continue;
      const T* dev = (const T*)src[f];
      if (!on_device(src[f])) {
        if (!ck(cudaMemcpyAsync(staging, src[f], nact * sizeof(T), cudaMemcpyHostToDevice, stream), "H2D field"))
          return FARGO_ECUDA;
        dev = staging;
      }
      launches += launch_scatter<T>(d, dev, dst[f], stream);
    }
    if (!ck(cudaMemsetAsync(staging, 0, (size_t)L.narr * sizeof(T), stream), "cudaMemsetAsync(staging)")) return FARGO_ECUDA;
    pot_valid = false;
    dt_ready = false;
    if (!ck(cudaGetLastError(), "set_fields launch")) return FARGO_ECUDA;
    if (!ck(cudaStreamSynchronize(stream), "set_fields sync")) return FARGO_ECUDA;
    have_fields = true; midstep = false; next_phase = 0;
    return FARGO_OK;
  }

  int get_fields(void* rho, void* e, void* vx, void* vy, void* vz) override {
    if (!have_fields) { err = "no fields set"; return FARGO_ESTATE; }
    if (midstep) { err = "context is mid-step (fargo_step_until)"; return FARGO_ESTATE; }
    const size_t nact = (size_t)L.nx * L.ny * L.nz;
    void* dstp[5] = {rho, e, vx, L.hasy ? vy : nullptr, L.hasz ? vz : nullptr};
    const T* srcp[5] = {st.rho, st.e, st.vx, st.vy, st.vz};
    int nstage = 0;
    for (int f = 0; f < 5; ++f) {
      if (!dstp[f]) continue;
      if (on_device(dstp[f])) {
        launches += launch_gather<T>(d, srcp[f], (T*)dstp[f], stream);
      } else {
        T* staging = pool[8 + (nstage++ % 8)];   // set B is dead between updates
        launches += launch_gather<T>(d, srcp[f], staging, stream);
        if (!ck(cudaMemcpyAsync(dstp[f], staging, nact * sizeof(T), cudaMemcpyDeviceToHost, stream), "D2H field"))
          return FARGO_ECUDA;
      }
    }
    if (!ck(cudaGetLastError(), "get_fields launch")) return FARGO_ECUDA;
    if (!ck(cudaStreamSynchronize(stream), "get_fields sync")) return FARGO_ECUDA;
    return FARGO_OK;
  }

  int get_time(double* t, double* last_dt, long long* ns) override {
    Ctl h;
    if (!ck(cudaMemcpyAsync(&h, ctl, sizeof h, cudaMemcpyDeviceToHost, stream), "read clock")) return FARGO_ECUDA;
    if (!ck(cudaStreamSynchronize(stream), "clock sync")) return FARGO_ECUDA;
    if (t) *t = h.t;
    if (last_dt) *last_dt = h.dt;
    if (ns) *ns = h.nsteps;
    return FARGO_OK;
  }

  // ---- slab decomposition in Y (NEXT-3; section 4.1) ------------------------------------------------------
  bool is_slab() const {
    return d.bc[1][0] == BC_EXTERNAL || d.bc[1][1] == BC_EXTERNAL || d.bc[2][0] == BC_EXTERNAL || d.bc[2][1] == BC_EXTERNAL;
  }

  int update_phase(int phase) override {
    if (!have_fields) { err = "no fields set"; return FARGO_ESTATE; }
    if (midstep) { err = "context is mid-step (fargo_step_until)"; return FARGO_ESTATE; }
    if (phase < 0 || phase > 4) { err = "phase must be 0 .. 4"; return FARGO_EINVAL; }
    if (phase != next_phase) { err = "phases run in the order 0, 1, 2, 3, 4"; return FARGO_ESTATE; }
    if (npl > 0) { err = "live planets are not supported on slabs (the gas force is a sum over the whole mesh)"; return FARGO_EINVAL; }
    // the kernels of a phase are a fixed sequence too: captured once per phase and replayed (the halo copies and the
    // all-reduce of dt between the phases stay with the caller)
    if (prm.use_graph && stream != nullptr && !prof) {
      if (phase == 1 && L.has_pot && !pot_valid && npl == 0 && pot_static) { launches += potential(0.0); pot_valid = true; }
      if (!gphase[phase]) {
        cudaGraph_t g = nullptr;
        if (!ck(cudaStreamBeginCapture(stream, cudaStreamCaptureModeThreadLocal), "begin capture")) return FARGO_ECUDA;
        gphase_launches[phase] = enqueue_update(-1, true, phase);
        if (!ck(cudaStreamEndCapture(stream, &g), "end capture")) return FARGO_ECUDA;
        if (!ck(cudaGraphInstantiate(&gphase[phase], g, 0), "graph instantiate")) { cudaGraphDestroy(g); return FARGO_ECUDA; }
        cudaGraphDestroy(g);
      }
      if (!ck(cudaGraphLaunch(gphase[phase], stream), "graph launch")) return FARGO_ECUDA;
      launches += gphase_launches[phase];
    } else {
      launches += enqueue_update(-1, false, phase);
    }
    next_phase = (phase + 1) % 5;
    if (!ck(cudaGetLastError(), "phase launch")) return FARGO_ECUDA;
    return FARGO_OK;
  }

  // bytes of one halo message: 3 layers (rows for dir = 1, planes for dir = 2) over the full allocated extent, per field
  size_t halo_bytes(int which, int dir) const override {
    const size_t layer = dir == 1 ? (size_t)L.pitch * L.TZ : (size_t)L.plane;
    return (size_t)(which == 0 ? 5 : 4) * 3 * layer * sizeof(T);
  }

  // which: 0 = the state (rho, e, vx, vy, vz), 1 = (e, vx, vy, vz) after the source step.  dir: 1 = Y, 2 = Z.
  // side: 0 = lower face, 1 = upper.  pack: the 3 active layers next to that face -> buf; unpack: buf -> the 3 ghost
  // layers beyond it.  Device-to-device copies on the context's stream (3 rows of a plane, and 3 planes, are contiguous).
  int halo(int which, int dir, int side, int pack, void* buf) override {
    if (!buf || which < 0 || which > 1 || side < 0 || side > 1 || dir < 1 || dir > 2) { err = "bad halo argument"; return FARGO_EINVAL; }
    if ((dir == 1 && !L.hasy) || (dir == 2 && !L.hasz)) { err = "no such direction"; return FARGO_EINVAL; }
    if (which == 1 && next_phase != 3 && next_phase != 4) { err = "the source-step halos exist between phases 2 and 4"; return FARGO_ESTATE; }
    const State<T>& a = which == 0 ? st : s2m;
    T* f[5] = {a.rho, a.e, a.vx, a.vy, a.vz};
    const int first = which == 0 ? 0 : 1;
    const int ng = dir == 1 ? L.ngy : L.ngz, na = dir == 1 ? L.ny : L.nz;
    const int m = pack ? (side == 0 ? ng : ng + na - 3) : (side == 0 ? 0 : ng + na);
    unsigned char* b = (unsigned char*)buf;
    const size_t per_field = halo_bytes(0, dir) / 5;
    for (int q = first; q < 5; ++q) {
      if (!f[q]) continue;
      unsigned char* msg = b + (size_t)(q - first) * per_field;
      cudaError_t e;
      if (dir == 1) {
        const size_t row3 = 3 * (size_t)L.pitch * sizeof(T);
        unsigned char* field = (unsigned char*)(f[q] + (size_t)m * L.pitch);
        e = pack ? cudaMemcpy2DAsync(msg, row3, field, (size_t)L.plane * sizeof(T), row3, L.TZ, cudaMemcpyDeviceToDevice, stream)
                 : cudaMemcpy2DAsync(field, (size_t)L.plane * sizeof(T), msg, row3, row3, L.TZ, cudaMemcpyDeviceToDevice, stream);
      } else {
        unsigned char* field = (unsigned char*)(f[q] + (size_t)m * L.plane);
        e = pack ? cudaMemcpyAsync(msg, field, per_field, cudaMemcpyDeviceToDevice, stream)
                 : cudaMemcpyAsync(field, msg, per_field, cudaMemcpyDeviceToDevice, stream);
      }
      if (!ck(e, "halo copy")) return FARGO_ECUDA;
    }
    return FARGO_OK;
  }

  void* dt_ptr() override { return &ctl->dt; }
  int dt_min_with(const void* other) override {
    if (!other) { err = "null pointer"; return FARGO_EINVAL; }
    launches += launch_dt_min(ctl, (const double*)other, stream);
    if (!ck(cudaGetLastError(), "dt_min launch")) return FARGO_ECUDA;
    return FARGO_OK;
  }

  // ---- live planets (NEXT-2) ---------------------------------------------------------------------------
  int set_planets(int n, const double* gm, const double* eps, const double* pos, const double* vel, int mode, double gconst) override {
    if (n < 0 || n > MAXPL || mode < 0 || mode > 2) { err = "planet count or force mode out of range"; return FARGO_EINVAL; }
    if (n > 0 && (!gm || !eps || !pos || !vel)) { err = "null planet array"; return FARGO_EINVAL; }
    if (n > 0 && (d.geometry == GEO_CART || !L.hasx)) { err = "live planets need a cylindrical or spherical mesh"; return FARGO_EINVAL; }
    if (n > 0 && !L.has_pot) { err = "the context was created without a potential (gm_star = 0 and planet_mass = 0)"; return FARGO_ESTATE; }
    if (midstep) { err = "context is mid-step"; return FARGO_ESTATE; }
    PlanetsDev h;
    memset(&h, 0, sizeof h);
    h.n = n; h.mode = mode; h.gconst = gconst;
    for (int p = 0; p < n; ++p) {
      h.gm[p] = gm[p]; h.eps[p] = eps[p];
      for (int c = 0; c < 3; ++c) { h.x[p][c] = pos[3 * p + c]; h.v[p][c] = vel[3 * p + c]; }
    }
    if (!ck(cudaMemcpyAsync(pl, &h, sizeof h, cudaMemcpyHostToDevice, stream), "upload planets")) return FARGO_ECUDA;
    if (!ck(cudaStreamSynchronize(stream), "set_planets sync")) return FARGO_ECUDA;
    if ((n > 0) != (npl > 0) || n != npl || mode != pl_mode) {   // the kernel sequence changes: capture it again
      drop_graphs();
    }
    npl = n; pl_mode = mode;
    pot_valid = false;
    return FARGO_OK;
  }

  // cell 5b, Eq. 44: the frame rotates at omega_new from the next update on
  int set_omega_frame(double omega_new) override {
    if (d.geometry == GEO_CART) { err = "the frame rate is fixed on Cartesian meshes (P:214) and in the shearing sheet (P:101)"; return FARGO_EINVAL; }
    if (!have_fields) { err = "no fields set"; return FARGO_ESTATE; }
    if (midstep) { err = "context is mid-step"; return FARGO_ESTATE; }
    double t = 0.0;
    const int rc = get_time(&t, nullptr, nullptr);   // synchronises the stream
    if (rc != FARGO_OK) return rc;
    launches += launch_frame_change<T>(d, st.vx, omega_new - prm.omega_frame, pl, npl, stream);
    // fixed-orbit planet: same azimuth now, new drift rate afterwards
    const double phip = prm.planet_phi0 + (prm.planet_omega - prm.omega_frame) * t;
    prm.planet_phi0 = phip - (prm.planet_omega - omega_new) * t;
    prm.omega_frame = omega_new;
    d.omega = (T)omega_new; d.om_eff = (T)omega_new;
    pot_static = !(L.has_pot && prm.planet_mass != 0.0 && prm.planet_omega != prm.omega_frame);
    pot_valid = false;
    drop_graphs();   // Omega_f is a kernel argument: capture again
    if (!ck(cudaGetLastError(), "frame change launch")) return FARGO_ECUDA;
    return FARGO_OK;
  }

  // sum reductions over the mesh: mass, Tab. 2 momenta, internal energy; applies the ghost fill of cell 2
  int diagnostics(double* out) override {
    if (!out) { err = "null argument"; return FARGO_EINVAL; }
    if (!have_fields) { err = "no fields set"; return FARGO_ESTATE; }
    if (midstep) { err = "context is mid-step"; return FARGO_ESTATE; }
    launches += launch_bc<T>(d, st, field_mask(true, true), stream);
    launches += launch_diagnostics<T>(d, st, pl_part, stream);
    const int nblk = planets_blocks(L.ny, L.nz);
    std::vector<double> h((size_t)nblk * 5);
    if (!ck(cudaMemcpyAsync(h.data(), pl_part, h.size() * sizeof(double), cudaMemcpyDeviceToHost, stream), "D2H partial sums")) return FARGO_ECUDA;
    if (!ck(cudaStreamSynchronize(stream), "diagnostics sync")) return FARGO_ECUDA;
    for (int c = 0; c < 5; ++c) {
      double s = 0.0;
      for (int b = 0; b < nblk; ++b) s = s + h[(size_t)b * 5 + c];
      out[c] = s;
    }
    return FARGO_OK;
  }

  // the same without any allocation: partials in the static device array of k_noalloc.cu, sums added on the device
  // into out_device[5]; asynchronous on the context's stream
  int diagnostics_noalloc(double* out_device) override {
    if (!out_device) { err = "null argument"; return FARGO_EINVAL; }
    if (!have_fields) { err = "no fields set"; return FARGO_ESTATE; }
    if (midstep) { err = "context is mid-step"; return FARGO_ESTATE; }
    cudaPointerAttributes at;
    if (!ck(cudaPointerGetAttributes(&at, out_device), "cudaPointerGetAttributes(out_device)")) return FARGO_ECUDA;
    if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged) { err = "out_device is not device memory"; return FARGO_EINVAL; }
    if ((long long)L.ny * L.nz > diagnostics_noalloc_max_rings()) {   // before anything is launched
      std::string e;
      launch_diagnostics_noalloc<T>(d, st, out_device, stream, e);
      err = e;
      return FARGO_EINVAL;
    }
    launches += launch_bc<T>(d, st, field_mask(true, true), stream);
    std::string e;
    const int n = launch_diagnostics_noalloc<T>(d, st, out_device, stream, e);
    if (n < 0) { err = e; return n == -1 ? FARGO_EINVAL : FARGO_ECUDA; }
    launches += n;
    if (!ck(cudaGetLastError(), "diagnostics_noalloc launch")) return FARGO_ECUDA;
    return FARGO_OK;
  }

  // ---- MHD (NEXT-4) ----------------------------------------------------------------------------------
  int set_bfield(const void* bx, const void* by, const void* bz, double mu0_, double eta_, int passive) override {
    if (!L.mhd) { err = "the context was created without fargo_params.mhd"; return FARGO_ESTATE; }
    if (!bx || !by || !bz || !(mu0_ > 0.0) || eta_ < 0.0) { err = "bx, by, bz, mu0 > 0 and eta >= 0 are required"; return FARGO_EINVAL; }
    if (eta_ != 0.0 && d.geometry != GEO_CART) { err = "the resistive term is built for the Cartesian metric only"; return FARGO_EINVAL; }
    if (midstep) { err = "context is mid-step"; return FARGO_ESTATE; }
    const size_t nact = (size_t)L.nx * L.ny * L.nz;
    const size_t arrb = align_up((size_t)L.narr * sizeof(T), 256);
    if (!ck(cudaMemsetAsync(bfield[0], 0, 13 * arrb, stream), "cudaMemsetAsync(B)")) return FARGO_ECUDA;
    const void* src[3] = {bx, by, bz};
    T* staging = pool[15];   // dead between updates
    for (int f = 0; f < 3; ++f) {
      const T* dev = (const T*)src[f];
      if (!on_device(src[f])) {
        if (!ck(cudaMemcpyAsync(staging, src[f], nact * sizeof(T), cudaMemcpyHostToDevice, stream), "H2D field")) return FARGO_ECUDA;
        dev = staging;
      }
      launches += launch_scatter<T>(d, dev, bfield[f], stream);
    }
    if (!ck(cudaMemsetAsync(staging, 0, (size_t)L.narr * sizeof(T), stream), "cudaMemsetAsync(staging)")) return FARGO_ECUDA;
    launches += launch_bc_b<T>(d, bfield[0], bfield[1], bfield[2], stream);
    if (!ck(cudaGetLastError(), "set_bfield launch")) return FARGO_ECUDA;
    if (!ck(cudaStreamSynchronize(stream), "set_bfield sync")) return FARGO_ECUDA;
    const bool changed = !mhd_on || passive != mhd_passive || mu0_ != mu0 || eta_ != eta;
    mhd_on = true; mhd_passive = passive ? 1 : 0; mu0 = mu0_; eta = eta_;
    dt_ready = false;
    if (changed) drop_graphs();   // the kernel sequence and its arguments change
    return FARGO_OK;
  }

  int get_bfield(void* bx, void* by, void* bz) override {
    if (!mhd_on) { err = "no magnetic field set"; return FARGO_ESTATE; }
    if (midstep) { err = "context is mid-step"; return FARGO_ESTATE; }
    const size_t nact = (size_t)L.nx * L.ny * L.nz;
    void* dstp[3] = {bx, by, bz};
    for (int f = 0; f < 3; ++f) {
      if (!dstp[f]) continue;
      if (on_device(dstp[f])) { launches += launch_gather<T>(d, bfield[f], (T*)dstp[f], stream); continue; }
      T* staging = pool[8 + f];   // set B is dead between updates
      launches += launch_gather<T>(d, bfield[f], staging, stream);
      if (!ck(cudaMemcpyAsync(dstp[f], staging, nact * sizeof(T), cudaMemcpyDeviceToHost, stream), "D2H field")) return FARGO_ECUDA;
    }
    if (!ck(cudaGetLastError(), "get_bfield launch")) return FARGO_ECUDA;
    if (!ck(cudaStreamSynchronize(stream), "get_bfield sync")) return FARGO_ECUDA;
    return FARGO_OK;
  }

  int get_planets(double* pos, double* vel, double* gas_acc) override {
    PlanetsDev h;
    if (!ck(cudaMemcpyAsync(&h, pl, sizeof h, cudaMemcpyDeviceToHost, stream), "download planets")) return FARGO_ECUDA;
    if (!ck(cudaStreamSynchronize(stream), "get_planets sync")) return FARGO_ECUDA;
    for (int p = 0; p < npl; ++p)
      for (int c = 0; c < 3; ++c) {
        if (pos) pos[3 * p + c] = h.x[p][c];
        if (vel) vel[3 * p + c] = h.v[p][c];
        if (gas_acc) gas_acc[3 * p + c] = h.f[p][c];
      }
    return npl;
  }

  // ---- one update --------------------------------------------------------------------------------------
  int field_mask(bool with_rho, bool with_e) const {
    int mk = F_VX;
    if (with_rho) mk |= F_RHO;
    if (with_e) mk |= F_E;
    if (L.hasy) mk |= F_VY;
    if (L.hasz) mk |= F_VZ;
    return mk;
  }

  int potential(double t) {
    const double phip = prm.planet_phi0 + (prm.planet_omega - prm.omega_frame) * t;
    const double xp = prm.planet_r * std::cos(phip), yp = prm.planet_r * std::sin(phip);
    const double eps2 = prm.planet_eps * prm.planet_eps;
    return launch_potential<T>(d, phi, (T)prm.gm_star, (T)prm.planet_mass, (T)xp, (T)yp, (T)eps2, nullptr, stream);
  }

  // The fixed-orbit planet moves in the frame (planet_omega != omega_frame): its azimuth needs the clock, which lives
  // on the device, and its cosine and sine come from the host's libm (no device transcendental).
  // Everything is enqueued -- clock to pinned memory, a host node that forms (x_p, y_p), back to the device, the
  // kernel -- so fargo_step neither waits for the stream nor leaves its captured graph.
  static void CUDART_CB planet_host_node(void* self) {
    Sim* s = (Sim*)self;
    const double phip = s->prm.planet_phi0 + (s->prm.planet_omega - s->prm.omega_frame) * s->hclock[0];
    s->hppos[0] = (T)(s->prm.planet_r * std::cos(phip));
    s->hppos[1] = (T)(s->prm.planet_r * std::sin(phip));
  }
  int potential_moving() {
    const double eps2 = prm.planet_eps * prm.planet_eps;
    if (!ck(cudaMemcpyAsync(hclock, &ctl->t, sizeof(double), cudaMemcpyDeviceToHost, stream), "clock to host node")) return 0;
    if (!ck(cudaLaunchHostFunc(stream, planet_host_node, this), "planet host node")) return 0;
    if (!ck(cudaMemcpyAsync(ppos, hppos, 2 * sizeof(T), cudaMemcpyHostToDevice, stream), "planet position to device")) return 0;
    return launch_potential<T>(d, phi, (T)prm.gm_star, (T)prm.planet_mass, T(0), T(0), (T)eps2, ppos, stream);
  }

  // Enqueue the kernels of one update up to and including `until` (-1 = all).  Returns the launch count.
  // `phase` (domain decomposition, NEXT-3): -1 = the whole update; 0 = cell 2 (ghost fill of the faces that are not cut);
  // 1 = cells 3-6 (v0, potential, local dt); 2 = the dt fix-up after the all-reduce and the source step; 3 = cell 9;
  // 4 = the transport step.  The caller exchanges the Y halos before the fill (phases 0, 3) and the Z halos after it.
  int enqueue_update(int until, bool capturing, int phase = -1) {
    int n = 0;
    const T* v0p = L.fargo ? v0 : nullptr;
    State<T> s2 = st;   // the state the transport step reads: e and v after the source step
    if (phase == 4) { s2 = s2m; goto cell12; }
    if (phase == 3) { s2 = s2m; goto cell9; }
    if (phase == 2) { n += launch_dt_sync(ctl, prm.t_stop, sizeof(T) == 4, stream); goto cell7; }
    if (phase == 1) goto cell3;
    dbg.clear();
    dbg["rho"] = st.rho; dbg["e"] = st.e; dbg["vx"] = st.vx; dbg["vy"] = st.vy; dbg["vz"] = st.vz;
    dbg["phi"] = phi; dbg["v0"] = v0;
    if (L.mhd) { dbg["bx"] = bfield[0]; dbg["by"] = bfield[1]; dbg["bz"] = bfield[2]; dbg["emfx"] = emf[0]; dbg["emfy"] = emf[1]; dbg["emfz"] = emf[2]; }
    n += timed("bc", [&] { return launch_bc<T>(d, st, field_mask(true, true), stream); });                        // cell 2
    if (mhd_on) n += timed("bc_b", [&] { return launch_bc_b<T>(d, bfield[0], bfield[1], bfield[2], stream); });
    if (until == FARGO_ST_BC1 || phase == 0) return n;
  cell3:
    if (L.fargo) n += timed("vmean", [&] { return launch_vmean<T>(d, st.vx, v0, stream); });                         // cell 3
    if (until == FARGO_ST_VMEAN) return n;
    if (npl > 0) {                                                                    // cell 5, live planets (on the device)
      n += timed("potential", [&] { return launch_potential_live<T>(d, phi, (T)prm.gm_star, pl, npl, stream); });
    } else if (L.has_pot && !pot_static) {                                           // cell 5, planet moving in the frame
      n += timed("potential", [&] { return potential_moving(); });
    } else if (L.has_pot && !pot_valid) {                                            // cell 5, static in the frame
      n += timed("potential", [&] { return potential(0.0); });
      pot_valid = true;
    }
    if (until == FARGO_ST_POT) return n;
    {                                                                                // cell 6
      const int mode = (fuse_dt && !mhd_on && dt_ready) ? DT_FINISH : DT_BOTH;
      const MhdDt<T> M{bfield[0], bfield[1], bfield[2], (T)mu0, (T)(4.0 * eta), mhd_passive};
      n += timed("dt", [&] { return launch_dt<T>(d, st, v0p, stream, mode, mhd_on ? &M : nullptr); });
      dt_ready = false;   // k_dt_finish consumed and cleared the running max
    }
    if (until == FARGO_ST_DT) return n;
    if (npl > 0)                                                                      // cell 5a (reading G33)
      n += timed("planets", [&] { return launch_planets_update<T>(d, st.rho, pl, npl, pl_mode, pl_part, prm.gm_star, prm.omega_frame, stream); });
    if (phase == 1) return n;
  cell7:
    if (fuse_source && !mhd_on && (until < 0 || until == FARGO_ST_SRC_C || until == FARGO_ST_SRC_D)) {
      // cells 7a-7c in one pass; it reads neighbours of the state, so its output goes to arrays of its own
      if (L.adi) s2.e = alt[0];
      s2.vx = alt[1]; s2.vy = alt[2]; s2.vz = alt[3];
      n += timed("source", [&] { return launch_source_fused<T>(d, st, phi, s2, stream); });
      // fargo_step_until: the pass is observable at the last stage it contains (active cells; with viscosity one layer more)
      dbg["vxc"] = s2.vx; dbg["vyc"] = s2.vy; dbg["vzc"] = s2.vz; dbg["ed"] = L.adi ? alt[0] : nullptr;
      dbg["vx"] = dbg["vy"] = dbg["vz"] = nullptr;
      if (until == FARGO_ST_SRC_C || (until == FARGO_ST_SRC_D && !L.visc3d)) return n;
      if (L.visc3d) {   // cell 7d in one pass: reads v_c from the fused pass's arrays, writes the (dead) state velocities
        n += timed("source_d", [&] { return launch_source_d3_fused<T>(d, st.rho, s2.vx, s2.vy, s2.vz, st.vx, st.vy, st.vz, stream); });
        s2.vx = st.vx; s2.vy = st.vy; s2.vz = st.vz;
        dbg["vxd"] = st.vx; dbg["vyd"] = st.vy; dbg["vzd"] = st.vz;
        if (until == FARGO_ST_SRC_D) return n;
      }
    } else {
    // source step: intermediates live in transport set B (idle until the second pass)
      T *vxb = set_arr(1, 0), *vyb = set_arr(1, 1), *vzb = set_arr(1, 2), *ec = set_arr(1, 3);
      n += timed("source_a", [&] { return launch_source_a<T>(d, st, phi, vxb, vyb, vzb, stream); });                      // cell 7a
      if (mhd_on && !mhd_passive)   // ... and the gradient of the magnetic pressure of the transverse components
        n += timed("mhd_pressure", [&] { return launch_mhd_pressure<T>(d, st.rho, bfield[0], bfield[1], bfield[2], vxb, vyb, vzb, mu0, stream); });
      dbg["vxb"] = vxb; dbg["vyb"] = vyb; dbg["vzb"] = vzb;
      if (until == FARGO_ST_SRC_A) return n;
      T *vxc = st.vx, *vyc = st.vy, *vzc = st.vz;   // the state's velocities are dead after 7a (reading G18)
      if (L.visc) { vxc = set_arr(1, 4); vyc = set_arr(1, 5); }
      if (L.visc3d) vzc = set_arr(1, 6);
      // adiabatic: 7b and 7c run as ONE kernel (e_c is never stored); compared with the oracle at stage SRC_C
      if (L.adi) n += timed("source_bc", [&] { return launch_source_bc<T>(d, st, vxb, vyb, vzb, vxc, vyc, vzc, st.e, stream); });
      else n += timed("source_b", [&] { return launch_source_b<T>(d, st, vxb, vyb, vzb, vxc, vyc, vzc, ec, stream); });   // cell 7b
      dbg["vxc"] = vxc; dbg["vyc"] = vyc; dbg["vzc"] = vzc; dbg["ec"] = nullptr;
      dbg["vx"] = dbg["vy"] = dbg["vz"] = nullptr;
      dbg["ed"] = st.e;
      if (until == FARGO_ST_SRC_B || until == FARGO_ST_SRC_C) return n;
      if (L.visc3d) {                                                                  // cell 7d, 3-D (Eqs. B1-B6)
        if (until < 0 && fuse_visc) {   // one pass, the tensor is never stored
          n += timed("source_d", [&] { return launch_source_d3_fused<T>(d, st.rho, vxc, vyc, vzc, st.vx, st.vy, st.vz, stream); });
        } else {
          T* tens[6] = {set_arr(0, -1), set_arr(0, 0), set_arr(0, 1), set_arr(0, 2), set_arr(0, 3), set_arr(0, 4)};
          n += timed("source_d", [&] { return launch_source_d3<T>(d, st.rho, vxc, vyc, vzc, tens, st.vx, st.vy, st.vz, stream); });
        }
      } else if (L.visc) {                                                             // cell 7d, 2-D cylindrical
        n += timed("source_d", [&] { return launch_source_d<T>(d, st.rho, vxc, vyc, set_arr(0, 0), set_arr(0, 1), set_arr(0, 2), st.vx, st.vy, stream); });
      }
      dbg["vxd"] = st.vx; dbg["vyd"] = st.vy; dbg["vzd"] = st.vz;
      dbg["vx"] = st.vx; dbg["vy"] = st.vy; dbg["vz"] = st.vz;
      if (until == FARGO_ST_SRC_D) return n;
    }
    if (phase == 2) { s2m = s2; return n; }
    if (mhd_on) {   // cells 8 and 10 (reading G34): the star values reach two zones out, so the ghosts of (e, v) are filled
                    // before cell 8 as well as after it (8d changes the velocities)
      n += timed("bc", [&] { return launch_bc<T>(d, s2, field_mask(false, L.adi), stream); });
      T* vx8 = s2.vx;   // with orbital advection cell 8 sees the residual velocity (reading G37)
      if (L.fargo) { n += timed("mhd_resid", [&] { return launch_mhd_resid<T>(d, s2.vx, v0, vxres, stream); }); vx8 = vxres; }
      n += timed("mhd_emf", [&] { return launch_mhd_emf<T>(d, st.rho, vx8, s2.vy, s2.vz, bfield[0], bfield[1], bfield[2], emf, bstar, mu0, eta, stream); });
      if (!mhd_passive) n += timed("mhd_tension", [&] { return launch_mhd_tension<T>(d, st.rho, bfield, bstar, s2.vx, s2.vy, s2.vz, mu0, stream); });
      n += timed("mhd_ct", [&] { return launch_mhd_ct<T>(d, emf, bfield[0], bfield[1], bfield[2], stream); });
      if (L.fargo)   // cell 11: orbital advection of B (the arc integrals reuse the arrays of eps_Z and eps_Y)
        n += timed("mhd_orbital", [&] { return launch_mhd_orbital<T>(d, v0, bfield[0], bfield[1], bfield[2], emf[2], emf[1], stream); });
    }
  cell9:
    n += timed("bc", [&] { return launch_bc<T>(d, s2, field_mask(false, L.adi), stream); });                      // cell 9
    if (until == FARGO_ST_BC2 || until == FARGO_ST_MOM || phase == 3) return n;
  cell12:
    // transport: pass p reads set (p-1)%2 (the state on the first pass) and writes set p%2; the last pass
    // writes rho and e straight back into the state arrays, so one update leaves every array where it
    // started and the same captured graph serves every update.
    if (!L.hasx) {   // no X sweep to fuse 12a into: store the momenta once, in the set the first pass reads
      QSet<T> S;
      S.rho = nullptr;
      for (int q = 0; q < 7; ++q) S.q[q] = set_arr(1, q);
      n += timed("momenta", [&] { return launch_momenta<T>(d, st, S, stream); });
    }
    for (int p = 0; p < npass; ++p) {
      const bool first = p == 0, last = p == npass - 1;
      const int ds = p % 2, ss = 1 - ds;
      SweepArgs<T> a;
      memset(&a, 0, sizeof a);
      a.st = s2;
      a.first = (first && L.hasx) ? 1 : 0;   // 12a fused into the X sweep
      a.v0 = (pass_kind[p] == 0 || pass_kind[p] == 3) ? v0p : nullptr;
      a.nq = nq;
      const bool to_state = last && !first;
      a.srho = first ? st.rho : set_arr(ss, -1);
      a.drho = to_state ? st.rho : set_arr(ds, -1);
      for (int q = 0; q < nq; ++q) {
        a.slot[q] = slots[q];
        if (first) a.sq[q] = L.hasx ? nullptr : (slots[q] == 0 ? st.e : set_arr(1, slots[q]));
        else a.sq[q] = set_arr(ss, slots[q]);
        a.dq[q] = (to_state && slots[q] == 0) ? st.e : set_arr(ds, slots[q]);
      }
      static const char* pnames[4] = {"sweep_x", "sweep_y", "sweep_z", "orbital"};
      if (pass_kind[p] == 3) n += timed(pnames[3], [&] { return launch_orbital<T>(d, a, nshift, stream); });
      else n += timed(pnames[pass_kind[p]], [&] { return launch_sweep<T>(d, a, pass_kind[p], stream); });
      static const char* names[7] = {"te", "pxm", "pxp", "pym", "pyp", "pzm", "pzp"};
      dbg["trho"] = a.drho;
      for (int q = 0; q < nq; ++q) dbg[names[slots[q]]] = a.dq[q];
      if (last && first) {   // single pass: bring rho and e home
        n += launch_copy<T>(d, set_arr(ds, -1), st.rho, stream);
        if (L.adi) n += launch_copy<T>(d, set_arr(ds, 0), st.e, stream);
      }
      const int stage_of[4] = {FARGO_ST_SWEEP_X, FARGO_ST_SWEEP_Y, FARGO_ST_SWEEP_Z, FARGO_ST_ORB_SHIFT};
      if (until == stage_of[pass_kind[p]]) return n;
      if (pass_kind[p] == 3 && until == FARGO_ST_ORB_FRAC) return n;
    }
    if (until >= FARGO_ST_SWEEP_X && until < FARGO_ST_NEWVEL) return n;   // stage absent in this setup
    const int ls = (npass - 1) % 2;
    QSet<T> S;
    S.rho = st.rho;
    for (int q = 0; q < 7; ++q) S.q[q] = set_arr(ls, q);
    if (fuse_dt && !mhd_on) {                                                        // cell 12d (+ cell 6 of the next update)
      n += timed("newvel_dt", [&] { return launch_newvel_dt<T>(d, st.rho, st.e, S, st, stream); });
      dt_ready = true;
    } else {
      n += timed("newvel", [&] { return launch_newvel<T>(d, st.rho, S, st, stream); });
    }
    n += timed("advance", [&] { return launch_advance(ctl, prm.t_stop, stream); });
    return n;
  }

  int step(int nsteps) override {
    if (!have_fields) { err = "no fields set"; return FARGO_ESTATE; }
    if (midstep) { err = "context is mid-step (fargo_step_until)"; return FARGO_ESTATE; }
    if (nsteps < 0) { err = "negative step count"; return FARGO_EINVAL; }
    if (is_slab() && nsteps > 0) { err = "a slab advances through fargo_update_phase (its Y halos come from its neighbours)"; return FARGO_ESTATE; }
    if (next_phase != 0) { err = "an update is in progress (fargo_update_phase)"; return FARGO_ESTATE; }
    if (nsteps == 0) return FARGO_OK;
    // the legacy default stream cannot be captured: plain launches there
    const bool graph_ok = prm.use_graph && stream != nullptr && !prof;
    int s = 0;
    if (graph_ok && fuse_dt && !mhd_on && !dt_ready) {
      // the captured sequence relies on the previous update's k_newvel_dt for the per-cell CFL rate: the first
      // update after fargo_set_fields gets it from the dt pass, after the ghost fill it reads through
      launches += launch_bc<T>(d, st, field_mask(true, true), stream);
      launches += launch_dt<T>(d, st, nullptr, stream, DT_CELLS);
      dt_ready = true;
    }
    if (graph_ok) {
      // the static potential stays out of the graph: written once after every fargo_set_fields (which clears it),
      // also when the graph already exists
      if (L.has_pot && !pot_valid && npl == 0 && pot_static) { launches += potential(0.0); pot_valid = true; }
      if (!gexec) {
        cudaGraph_t g = nullptr;
        if (!ck(cudaStreamBeginCapture(stream, cudaStreamCaptureModeThreadLocal), "begin capture")) return FARGO_ECUDA;
        launches_per_step = enqueue_update(-1, true);
        if (!ck(cudaStreamEndCapture(stream, &g), "end capture")) return FARGO_ECUDA;
        if (!ck(cudaGraphInstantiate(&gexec, g, 0), "graph instantiate")) { cudaGraphDestroy(g); return FARGO_ECUDA; }
        cudaGraphDestroy(g);
      }
      for (; s < nsteps; ++s)
        if (!ck(cudaGraphLaunch(gexec, stream), "graph launch")) return FARGO_ECUDA;
      launches += (long long)launches_per_step * nsteps;
    } else {
      for (; s < nsteps; ++s) launches += enqueue_update(-1, false);
    }
    if (!ck(cudaGetLastError(), "step launch")) return FARGO_ECUDA;
    return FARGO_OK;
  }

  int step_until(int stage) override {
    if (!have_fields) { err = "no fields set"; return FARGO_ESTATE; }
    if (midstep) { err = "context is mid-step"; return FARGO_ESTATE; }
    if (stage < 0 || stage >= FARGO_ST_COUNT) { err = "unknown stage"; return FARGO_EINVAL; }
    launches += enqueue_update(stage == FARGO_ST_NEWVEL ? -1 : stage, false);
    midstep = stage != FARGO_ST_NEWVEL;
    if (!ck(cudaGetLastError(), "step_until launch")) return FARGO_ECUDA;
    if (!ck(cudaStreamSynchronize(stream), "step_until sync")) return FARGO_ECUDA;
    return FARGO_OK;
  }

  void dims(int* tx, int* ty, int* tz, int* ngx, int* ngy, int* ngz) const override {
    if (tx) *tx = L.TX; if (ty) *ty = L.TY; if (tz) *tz = L.TZ;
    if (ngx) *ngx = L.ngx; if (ngy) *ngy = L.ngy; if (ngz) *ngz = L.ngz;
  }

  int get_array(const char* name, void* out) override {
    if (!name || !out) { err = "null argument"; return FARGO_EINVAL; }
    if (dbg.empty()) {
      dbg["rho"] = st.rho; dbg["e"] = st.e; dbg["vx"] = st.vx; dbg["vy"] = st.vy; dbg["vz"] = st.vz;
      dbg["phi"] = phi; dbg["v0"] = v0;
    }
    if (L.mhd) { dbg["bx"] = bfield[0]; dbg["by"] = bfield[1]; dbg["bz"] = bfield[2]; dbg["emfx"] = emf[0]; dbg["emfy"] = emf[1]; dbg["emfz"] = emf[2]; }
    dbg["nshift"] = nshift;
    auto it = dbg.find(name);
    if (it == dbg.end() || !it->second) { err = std::string("array not available at this stage: ") + name; return FARGO_EINVAL; }
    if (!ck(cudaStreamSynchronize(stream), "get_array sync")) return FARGO_ECUDA;
    const std::string nm(name);
    if (nm == "v0" || nm == "nshift") {
      if (!ck(cudaMemcpy(out, it->second, (size_t)L.TY * L.TZ * sizeof(T), cudaMemcpyDeviceToHost), "D2H ring array"))
        return FARGO_ECUDA;
      return FARGO_OK;
    }
    const size_t n = (size_t)L.TX * L.TY * L.TZ;
    T* tmp = nullptr;
    if (!ck(cudaMalloc(&tmp, n * sizeof(T)), "cudaMalloc(debug)")) return FARGO_ENOMEM;
    launches += launch_unpad<T>(d, it->second, tmp, stream);
    bool ok = ck(cudaMemcpyAsync(out, tmp, n * sizeof(T), cudaMemcpyDeviceToHost, stream), "D2H array") &&
              ck(cudaStreamSynchronize(stream), "get_array sync");
    cudaFree(tmp);
    return ok ? FARGO_OK : FARGO_ECUDA;
  }
};

}  // namespace fg

// ---- C ABI ---------------------------------------------------------------------------------------------
struct fargo_ctx { fg::CtxBase* impl; };

extern "C" {

size_t fargo_workspace_bytes(const fargo_mesh* mesh, int geometry, int eos, const fargo_params* p) {
  fg::Layout L;
  std::string err;
  if (!fg::make_layout(L, mesh, geometry, eos, p, err)) return 0;
  return L.bytes(p->precision == 32 ? sizeof(float) : sizeof(double));
}

int fargo_init(fargo_ctx** out, const fargo_mesh* mesh, int geometry, int eos, const fargo_params* p) {
  if (!out) { fg::g_init_error = "null output pointer"; return FARGO_EINVAL; }
  *out = nullptr;
  fg::Layout L;
  if (!fg::make_layout(L, mesh, geometry, eos, p, fg::g_init_error)) return FARGO_EINVAL;
  int rc;
  fg::CtxBase* impl;
  if (p->precision == 32) {
    auto* s = new fg::Sim<float>(); s->L = L; s->precision = 32; rc = s->init(mesh, geometry, eos, p); impl = s;
  } else {
    auto* s = new fg::Sim<double>(); s->L = L; s->precision = 64; rc = s->init(mesh, geometry, eos, p); impl = s;
  }
  if (rc != FARGO_OK) { fg::g_init_error = impl->err; delete impl; return rc; }
  *out = new fargo_ctx{impl};
  return FARGO_OK;
}

int fargo_destroy(fargo_ctx* c) {
  if (!c) return FARGO_EINVAL;
  delete c->impl;
  delete c;
  return FARGO_OK;
}

int fargo_set_fields(fargo_ctx* c, const void* rho, const void* e, const void* vx, const void* vy, const void* vz) {
  return c ? c->impl->set_fields(rho, e, vx, vy, vz) : FARGO_EINVAL;
}
int fargo_get_fields(fargo_ctx* c, void* rho, void* e, void* vx, void* vy, void* vz) {
  return c ? c->impl->get_fields(rho, e, vx, vy, vz) : FARGO_EINVAL;
}
int fargo_step(fargo_ctx* c, int n) { return c ? c->impl->step(n) : FARGO_EINVAL; }
int fargo_get_time(fargo_ctx* c, double* t, double* last_dt, long long* nsteps) {
  return c ? c->impl->get_time(t, last_dt, nsteps) : FARGO_EINVAL;
}
long long fargo_kernel_launches(const fargo_ctx* c) { return c ? c->impl->launches : 0; }
int fargo_set_planets(fargo_ctx* c, int n, const double* gm, const double* eps, const double* pos, const double* vel,
                      int force_mode, double gconst) {
  return c ? c->impl->set_planets(n, gm, eps, pos, vel, force_mode, gconst) : FARGO_EINVAL;
}
int fargo_get_planets(fargo_ctx* c, double* pos, double* vel, double* gas_acc) {
  return c ? c->impl->get_planets(pos, vel, gas_acc) : FARGO_EINVAL;
}
int fargo_set_omega_frame(fargo_ctx* c, double omega_new) { return c ? c->impl->set_omega_frame(omega_new) : FARGO_EINVAL; }
int fargo_diagnostics(fargo_ctx* c, double* out) { return c ? c->impl->diagnostics(out) : FARGO_EINVAL; }
int fargo_diagnostics_noalloc(fargo_ctx* c, double* out_device) { return c ? c->impl->diagnostics_noalloc(out_device) : FARGO_EINVAL; }
int fargo_set_bfield(fargo_ctx* c, const void* bx, const void* by, const void* bz, double mu0, double eta, int passive) {
  return c ? c->impl->set_bfield(bx, by, bz, mu0, eta, passive) : FARGO_EINVAL;
}
int fargo_get_bfield(fargo_ctx* c, void* bx, void* by, void* bz) { return c ? c->impl->get_bfield(bx, by, bz) : FARGO_EINVAL; }
int fargo_update_phase(fargo_ctx* c, int phase) { return c ? c->impl->update_phase(phase) : FARGO_EINVAL; }
size_t fargo_halo_bytes(const fargo_ctx* c, int which, int dir) { return c ? c->impl->halo_bytes(which, dir) : 0; }
int fargo_halo(fargo_ctx* c, int which, int dir, int side, int pack, void* device_buffer) {
  return c ? c->impl->halo(which, dir, side, pack, device_buffer) : FARGO_EINVAL;
}
void* fargo_dt_device_ptr(fargo_ctx* c) { return c ? c->impl->dt_ptr() : nullptr; }
int fargo_dt_min_with(fargo_ctx* c, const void* other_dt_device_ptr) { return c ? c->impl->dt_min_with(other_dt_device_ptr) : FARGO_EINVAL; }
int fargo_step_until(fargo_ctx* c, int stage) { return c ? c->impl->step_until(stage) : FARGO_EINVAL; }
int fargo_dims(const fargo_ctx* c, int* tx, int* ty, int* tz, int* ngx, int* ngy, int* ngz) {
  if (!c) return FARGO_EINVAL;
  c->impl->dims(tx, ty, tz, ngx, ngy, ngz);
  return FARGO_OK;
}
int fargo_get_array(fargo_ctx* c, const char* name, void* out) { return c ? c->impl->get_array(name, out) : FARGO_EINVAL; }
int fargo_profile(fargo_ctx* c, int enable) { return c ? c->impl->profile(enable) : FARGO_EINVAL; }
int fargo_profile_report(fargo_ctx* c, char* buf, size_t len) { return c ? c->impl->profile_report(buf, len) : FARGO_EINVAL; }
int fargo_selftest_div(const double* a, const double* b, double* out, long long n, void* cuda_stream) {
  if (!a || !out || n < 0) return FARGO_EINVAL;
  if (n == 0) return FARGO_OK;
  fg::launch_selftest_div(a, b, out, n, (cudaStream_t)cuda_stream);
  if (cudaGetLastError() != cudaSuccess) return FARGO_ECUDA;
  return cudaStreamSynchronize((cudaStream_t)cuda_stream) == cudaSuccess ? FARGO_OK : FARGO_ECUDA;
}
const char* fargo_last_error(const fargo_ctx* c) { return c ? c->impl->err.c_str() : fg::g_init_error.c_str(); }

}  // extern "C"
