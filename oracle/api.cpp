// api.cpp -- C interface and the driver of one full update (Fig. 2 caption).
// CPU oracle, TEST INFRASTRUCTURE (see fargo_oracle.h).
#include <map>

#include "oracle_impl.hpp"

extern "C" int oracle_init(oracle_ctx** out, const oracle_mesh* m, int geometry, int eos, const oracle_params* p) {
  if (!out || !m || !p) return -1;
  if (m->nx < 1 || m->ny < 1 || m->nz < 1) return -1;
  if (geometry < 0 || geometry > 3 || eos < 0 || eos > 1) return -1;
  oracle_ctx* c = new oracle_ctx();
  c->nx = m->nx; c->ny = m->ny; c->nz = m->nz;
  c->ng = m->nghost > 0 ? m->nghost : 3;
  c->shear = geometry == ORC_SHEARING_SHEET;
  if (c->shear) geometry = ORC_CARTESIAN;   // same metric; Tab. 2 and Eq. 29 are the differences (G32)
  c->geometry = geometry; c->eos = eos; c->p = *p;
  for (int d = 0; d < 3; ++d) for (int s = 0; s < 2; ++s) c->bc[d][s] = m->bc[d][s];
  c->hasx = m->nx > 1; c->hasy = m->ny > 1; c->hasz = m->nz > 1;
  // X: no ghosts when periodic, index algebra wraps; ghosted otherwise (reading G20)
  c->xwrap = (m->bc[0][0] == ORC_PERIODIC);
  c->ngx = (c->hasx && !c->xwrap) ? c->ng : 0;
  c->ngy = c->hasy ? c->ng : 0;
  c->ngz = c->hasz ? c->ng : 0;
  c->TX = c->nx + 2 * c->ngx; c->TY = c->ny + 2 * c->ngy; c->TZ = c->nz + 2 * c->ngz;
  c->xmin = m->xmin; c->dx = (m->xmax - m->xmin) / (double)m->nx;
  if (p->fargo_on && !c->xwrap) { delete c; return -1; }  // rings must be whole and periodic
  if (c->shear && !(c->hasx && c->xwrap && c->hasy)) { delete c; return -1; }  // sheet: X along the flow, periodic; Y along the shear (Tab. 1)
  c->has_pot = (geometry != ORC_CARTESIAN) && (p->gm_star != 0.0 || p->planet_mass != 0.0);
  orc_build_tables(*c, *m);
  const size_t n = c->ncell();
  for (vec* f : {&c->rho, &c->e, &c->vx, &c->vy, &c->vz, &c->phi, &c->vxb, &c->vyb, &c->vzb, &c->vxc, &c->vyc,
                 &c->vzc, &c->ec, &c->ed, &c->vxd, &c->vyd, &c->vzd, &c->pxm, &c->pxp, &c->pym, &c->pyp, &c->pzm, &c->pzp})
    f->assign(n, 0.0);
  c->v0.assign((size_t)c->TY * c->TZ, 0.0);
  c->nshift.assign((size_t)c->TY * c->TZ, 0.0);
  c->xi.assign((size_t)c->TY * c->TZ, 0.0);
  c->t = 0.0; c->dt = 0.0; c->nsteps = 0; c->midstep = false;
  *out = c;
  return 0;
}

extern "C" int oracle_destroy(oracle_ctx* c) { delete c; return 0; }

static void scatter(oracle_ctx* c, vec& dst, const double* src) {
  if (!src) return;
  for (int k = 0; k < c->nz; ++k)
    for (int j = 0; j < c->ny; ++j)
      for (int i = 0; i < c->nx; ++i)
        dst[c->id(i + c->ngx, j + c->ngy, k + c->ngz)] = src[(size_t)i + (size_t)c->nx * (j + (size_t)c->ny * k)];
}
static void gather(oracle_ctx* c, const vec& src, double* dst) {
  if (!dst) return;
  for (int k = 0; k < c->nz; ++k)
    for (int j = 0; j < c->ny; ++j)
      for (int i = 0; i < c->nx; ++i)
        dst[(size_t)i + (size_t)c->nx * (j + (size_t)c->ny * k)] = src[c->id(i + c->ngx, j + c->ngy, k + c->ngz)];
}

extern "C" int oracle_set_fields(oracle_ctx* c, const double* rho, const double* e, const double* vx,
                                 const double* vy, const double* vz) {
  if (!c || !rho || !e || !vx) return -1;
  for (vec* f : {&c->rho, &c->e, &c->vx, &c->vy, &c->vz}) f->assign(c->ncell(), 0.0);
  scatter(c, c->rho, rho); scatter(c, c->e, e); scatter(c, c->vx, vx);
  if (c->hasy) scatter(c, c->vy, vy);
  if (c->hasz) scatter(c, c->vz, vz);
  c->t = 0.0; c->dt = 0.0; c->nsteps = 0; c->midstep = false;
  return 0;
}

// NEXT-4: switch the MHD substeps on and load the face-centred field (active cells, like the velocities; a component of
// an absent direction is uniform along it).  Cartesian meshes and the shearing sheet, with or without orbital advection.
extern "C" int oracle_set_bfield(oracle_ctx* c, const double* bx, const double* by, const double* bz, double mu0,
                                 double eta, int passive) {
  if (!c || !bx || !by || !bz || !(mu0 > 0.0) || eta < 0.0) return -1;
  if (c->geometry != ORC_CARTESIAN && eta != 0.0) return -1;   // the resistive term is built for the Cartesian metric only
  if (c->geometry == ORC_SPHERICAL && c->p.fargo_on) return -1;  // cell 11 is built for Cartesian and cylindrical meshes (G38)
  for (vec* f : {&c->bx, &c->by, &c->bz, &c->emfx, &c->emfy, &c->emfz, &c->bstar[0][0], &c->bstar[0][1], &c->bstar[1][0],
                 &c->bstar[1][1], &c->bstar[2][0], &c->bstar[2][1]})
    f->assign(c->ncell(), 0.0);
  scatter(c, c->bx, bx); scatter(c, c->by, by); scatter(c, c->bz, bz);
  c->mhd = true; c->mhd_passive = passive != 0; c->mu0 = mu0; c->eta = eta;
  orc_mhd_bc_fill(*c);
  return 0;
}
extern "C" int oracle_get_bfield(oracle_ctx* c, double* bx, double* by, double* bz) {
  if (!c || !c->mhd) return -1;
  gather(c, c->bx, bx); gather(c, c->by, by); gather(c, c->bz, bz);
  return 0;
}
// max over the active cells of |div B| (the ghost fill of cell 2 is applied first: the upper boundary faces)
extern "C" double oracle_max_divb(oracle_ctx* c) {
  if (!c || !c->mhd) return -1.0;
  orc_mhd_bc_fill(*c);
  double m = 0.0;
  for (int k = c->k0(); k < c->k1(); ++k)
    for (int j = c->j0(); j < c->j1(); ++j)
      for (int i = c->i0(); i < c->i1(); ++i) m = std::max(m, std::fabs(orc_mhd_divb(*c, i, j, k)));
  return m;
}

extern "C" int oracle_get_fields(oracle_ctx* c, double* rho, double* e, double* vx, double* vy, double* vz) {
  if (!c) return -1;
  gather(c, c->rho, rho); gather(c, c->e, e); gather(c, c->vx, vx); gather(c, c->vy, vy); gather(c, c->vz, vz);
  return 0;
}

extern "C" int oracle_get_time(oracle_ctx* c, double* t, double* last_dt, long long* nsteps) {
  if (!c) return -1;
  if (t) *t = c->t;
  if (last_dt) *last_dt = c->dt;
  if (nsteps) *nsteps = c->nsteps;
  return 0;
}

// One full update, boxes in the numerical order of Fig. 2 (reading G29).  `until` stops after a stage.
static void full_update(oracle_ctx* c, int until) {
  oracle_ctx& o = *c;
  if (o.p.t_stop > 0.0 && o.t >= o.p.t_stop) return;  // reading G21: nothing happens after t_stop
  bool clipped = false;
  orc_bc_fill(o, o.rho, o.e, o.vx, o.vy, o.vz);                                                       // cell 2
  if (o.mhd) orc_mhd_bc_fill(o);
  if (until == ORC_ST_BC1) return;
  orc_vmean(o);                                                 if (until == ORC_ST_VMEAN) return;    // cell 3
  orc_potential(o);                                             if (until == ORC_ST_POT) return;      // cells 4-5
  o.dt = orc_compute_dt(o, &clipped);                           if (until == ORC_ST_DT) return;       // cell 6
  orc_planets_update(o);                                                                              // cell 5a (G33)
  orc_source_a(o);                                                                                    // cell 7a
  if (o.mhd) { orc_mhd_source_a(o); orc_mhd_source_curv(o); }
  if (until == ORC_ST_SRC_A) return;
  orc_source_b(o);                                              if (until == ORC_ST_SRC_B) return;    // cell 7b
  orc_source_c(o);                                              if (until == ORC_ST_SRC_C) return;    // cell 7c
  orc_source_d(o);                                              if (until == ORC_ST_SRC_D) return;    // cell 7d
  // the source step leaves its result in (rho, ed, vxd, vyd, vzd); make it the state
  o.e = o.ed; o.vx = o.vxd; o.vy = o.vyd; o.vz = o.vzd;
  if (o.mhd) {   // cells 8 and 10 (reading G34): the star values reach two zones out, so the ghosts of the velocities
                 // are filled before cell 8 as well as after it (8d changes the velocities); B is transported here
    orc_bc_fill(o, o.rho, o.e, o.vx, o.vy, o.vz);
    orc_mhd_emf(o);                                                                                   // cells 8a-8c
    orc_mhd_lorentz(o);                                                                               // cell 8d
    orc_mhd_ct(o);                                                                                    // cell 10
    orc_mhd_orbital(o);                                                                               // cell 11
  }
  orc_bc_fill(o, o.rho, o.e, o.vx, o.vy, o.vz);                 if (until == ORC_ST_BC2) return;      // cell 9
  orc_momenta(o);                                               if (until == ORC_ST_MOM) return;      // cell 12a
  orc_sweep(o, 0);                                              if (until == ORC_ST_SWEEP_X) return;  // cells 12b-c
  orc_sweep(o, 1);                                              if (until == ORC_ST_SWEEP_Y) return;
  orc_sweep(o, 2);                                              if (until == ORC_ST_SWEEP_Z) return;
  orc_orbital_frac(o);                                          if (until == ORC_ST_ORB_FRAC) return;
  orc_orbital_shift(o);                                         if (until == ORC_ST_ORB_SHIFT) return;
  orc_newvel(o);                                                                                      // cell 12d
  o.t = clipped ? o.p.t_stop : o.t + o.dt;
  o.nsteps += 1;
}

extern "C" int oracle_step(oracle_ctx* c, int n) {
  if (!c || c->midstep) return -1;
  for (int s = 0; s < n; ++s) full_update(c, -1);
  return 0;
}

extern "C" int oracle_step_until(oracle_ctx* c, int stage) {
  if (!c || c->midstep) return -1;
  full_update(c, stage);
  c->midstep = (stage != ORC_ST_NEWVEL);
  return 0;
}

// Run ONE stage on the arrays as they stand (mid-step or not), with the current dt.  For tests that
// pin a single box of Fig. 2, and for per-kernel parity.  ORC_ST_BC2 first makes the source-step
// result the state, as the full update does.
extern "C" int oracle_run_stage(oracle_ctx* c, int stage) {
  if (!c) return -1;
  oracle_ctx& o = *c;
  bool clipped = false;
  switch (stage) {
    case ORC_ST_BC1: orc_bc_fill(o, o.rho, o.e, o.vx, o.vy, o.vz); break;
    case ORC_ST_VMEAN: orc_vmean(o); break;
    case ORC_ST_POT: orc_potential(o); break;
    case ORC_ST_DT: o.dt = orc_compute_dt(o, &clipped); break;
    case ORC_ST_SRC_A: orc_source_a(o); break;
    case ORC_ST_SRC_B: orc_source_b(o); break;
    case ORC_ST_SRC_C: orc_source_c(o); break;
    case ORC_ST_SRC_D: orc_source_d(o); break;
    case ORC_ST_BC2:
      o.e = o.ed; o.vx = o.vxd; o.vy = o.vyd; o.vz = o.vzd;
      orc_bc_fill(o, o.rho, o.e, o.vx, o.vy, o.vz);
      break;
    case ORC_ST_MOM: orc_momenta(o); break;
    case ORC_ST_SWEEP_X: orc_sweep(o, 0); break;
    case ORC_ST_SWEEP_Y: orc_sweep(o, 1); break;
    case ORC_ST_SWEEP_Z: orc_sweep(o, 2); break;
    case ORC_ST_ORB_FRAC: orc_orbital_frac(o); break;
    case ORC_ST_ORB_SHIFT: orc_orbital_shift(o); break;
    case ORC_ST_NEWVEL: orc_newvel(o); break;
    default: return -1;
  }
  c->midstep = true;
  return 0;
}
// The same for the MHD substeps: 0 = ghost fill of B (cell 2), 1 = star values and EMFs (cells 8a-8c), 2 = tension (8d),
// 3 = constrained transport (10), 4 = orbital advection of B (11; needs v0 of cell 3 and the current dt).
extern "C" int oracle_run_mhd_stage(oracle_ctx* c, int which) {
  if (!c || !c->mhd) return -1;
  switch (which) {
    case 0: orc_mhd_bc_fill(*c); break;
    case 1: orc_mhd_emf(*c); break;
    case 2: orc_mhd_lorentz(*c); break;
    case 3: orc_mhd_ct(*c); break;
    case 4: orc_mhd_orbital(*c); break;
    default: return -1;
  }
  return 0;
}
extern "C" int oracle_set_dt(oracle_ctx* c, double dt) { if (!c) return -1; c->dt = dt; return 0; }

static vec* find_array(oracle_ctx* c, const char* name) {
  const std::map<std::string, vec*> m = {
      {"rho", &c->rho}, {"e", &c->e}, {"vx", &c->vx}, {"vy", &c->vy}, {"vz", &c->vz}, {"phi", &c->phi},
      {"vxb", &c->vxb}, {"vyb", &c->vyb}, {"vzb", &c->vzb}, {"vxc", &c->vxc}, {"vyc", &c->vyc}, {"vzc", &c->vzc},
      {"ec", &c->ec}, {"ed", &c->ed}, {"vxd", &c->vxd}, {"vyd", &c->vyd}, {"vzd", &c->vzd}, {"pxm", &c->pxm}, {"pxp", &c->pxp},
      {"pym", &c->pym}, {"pyp", &c->pyp}, {"pzm", &c->pzm}, {"pzp", &c->pzp}, {"v0", &c->v0},
      {"nshift", &c->nshift}, {"xi", &c->xi},
      {"bx", &c->bx}, {"by", &c->by}, {"bz", &c->bz}, {"emfx", &c->emfx}, {"emfy", &c->emfy}, {"emfz", &c->emfz}};
  auto it = m.find(name ? name : "");
  return it == m.end() ? nullptr : it->second;
}

extern "C" int oracle_get_array(oracle_ctx* c, const char* name, double* out) {
  vec* a = c ? find_array(c, name) : nullptr;
  if (!a || !out) return -1;
  std::memcpy(out, a->data(), a->size() * sizeof(double));
  return 0;
}
extern "C" int oracle_set_array(oracle_ctx* c, const char* name, const double* in) {
  vec* a = c ? find_array(c, name) : nullptr;
  if (!a || !in) return -1;
  std::memcpy(a->data(), in, a->size() * sizeof(double));
  return 0;
}
extern "C" int oracle_dims(oracle_ctx* c, int* tx, int* ty, int* tz, int* ngx, int* ngy, int* ngz) {
  if (!c) return -1;
  *tx = c->TX; *ty = c->TY; *tz = c->TZ; *ngx = c->ngx; *ngy = c->ngy; *ngz = c->ngz;
  return 0;
}
extern "C" int oracle_geometry(oracle_ctx* c, int j, int k, double* sx, double* sy, double* sz, double* invv,
                               double* lx, double* ly, double* lz) {
  if (!c || j < 0 || j >= c->TY || k < 0 || k >= c->TZ) return -1;
  *sx = c->Sx(j, k); *sy = c->Sy(j, k); *sz = c->Sz(j, k); *invv = c->invV(j, k);
  *lx = c->LX(j, k); *ly = c->LY[j]; *lz = c->LZ(j, k);
  return 0;
}
