// TEST INFRASTRUCTURE ONLY (see vh_oracle.hpp).  C interface of the serial CPU oracle for ctypes
// (oracle/vh_oracle.py).  Nothing under paper_1608_06577_b200/ links or loads this.
#include "vh_oracle.hpp"
#include <chrono>
#include <cstring>

using Sol = vho::Solver<double>;
using SolF = vho::Solver<float>;      // the same algorithm in single precision: comparator of the FP32 build

extern "C" {

int vho_params_size() { return (int)sizeof(vho::Params); }

// one Solver per event of the batch (ev: double precision; evf: single precision, created by vho_create_f32 - then ev is empty)
struct vho_handle { vho::Params P; std::vector<Sol*> ev; std::vector<SolF*> evf; };

vho_handle* vho_create(const vho::Params* P) {
  if (!P || P->nx < 1 || P->ny < 1 || P->nz < 1 || P->n_batch < 1) return nullptr;
  vho_handle* h = new vho_handle;
  h->P = *P;
  for (int b = 0; b < P->n_batch; ++b) h->ev.push_back(new Sol(*P));
  return h;
}
vho_handle* vho_create_f32(const vho::Params* P) {
  if (!P || P->nx < 1 || P->ny < 1 || P->nz < 1 || P->n_batch < 1) return nullptr;
  vho_handle* h = new vho_handle;
  h->P = *P;
  for (int b = 0; b < P->n_batch; ++b) h->evf.push_back(new SolF(*P));
  return h;
}
void vho_destroy(vho_handle* h) { if (!h) return; for (Sol* s : h->ev) delete s; for (SolF* s : h->evf) delete s; delete h; }

}  // extern "C"

// the calls both precisions support, written once over the vector of solvers
template <class S> static void set_initial_t(const vho::Params& P, std::vector<S*>& ev, const double* e, const double* u4, const double* pi10, const double* Pi) {
  size_t np = (size_t)P.nx * P.ny * P.nz, nb = ev.size();
  std::vector<double> ub(4 * np), pb(10 * np);
  for (size_t b = 0; b < nb; ++b) {
    for (int m = 0; m < 4; ++m) std::memcpy(&ub[m * np], u4 + (m * nb + b) * np, np * sizeof(double));
    if (pi10) for (int n = 0; n < 10; ++n) std::memcpy(&pb[n * np], pi10 + (n * nb + b) * np, np * sizeof(double));
    ev[b]->set_initial(e + b * np, ub.data(), pi10 ? pb.data() : nullptr, Pi ? Pi + b * np : nullptr);
  }
}
template <class S> static void set_uprev_t(const vho::Params& P, std::vector<S*>& ev, const double* up4) {
  size_t np = (size_t)P.nx * P.ny * P.nz, nb = ev.size();
  std::vector<double> ub(4 * np);
  for (size_t b = 0; b < nb; ++b) {
    for (int m = 0; m < 4; ++m) std::memcpy(&ub[m * np], up4 + (m * nb + b) * np, np * sizeof(double));
    ev[b]->set_uprev(ub.data());
  }
}
template <class S> static void get_fields_t(const vho::Params& P, std::vector<S*>& ev, double* q15, double* e, double* p, double* u4, double* up4) {
  size_t np = (size_t)P.nx * P.ny * P.nz, nb = ev.size();
  std::vector<double> qb(15 * np), ub(4 * np), upb(4 * np);
  for (size_t b = 0; b < nb; ++b) {
    ev[b]->get_fields(q15 ? qb.data() : nullptr, e ? e + b * np : nullptr, p ? p + b * np : nullptr,
                      u4 ? ub.data() : nullptr, up4 ? upb.data() : nullptr);
    if (q15) for (int n = 0; n < 15; ++n) std::memcpy(q15 + (n * nb + b) * np, &qb[n * np], np * sizeof(double));
    if (u4) for (int m = 0; m < 4; ++m) std::memcpy(u4 + (m * nb + b) * np, &ub[m * np], np * sizeof(double));
    if (up4) for (int m = 0; m < 4; ++m) std::memcpy(up4 + (m * nb + b) * np, &upb[m * np], np * sizeof(double));
  }
}
template <class S> static void get_status_t(std::vector<S*>& ev, double* tau, long long* n_steps, long long* n_fail, long long* n_nonfinite, double* min_reg) {
  long long f = 0, nf = 0; double mr = 1.0;
  for (S* s : ev) { f += s->n_fail; nf += s->n_nonfinite; if (s->min_reg_factor < mr) mr = s->min_reg_factor; }
  if (tau) *tau = ev[0]->tau;
  if (n_steps) *n_steps = ev[0]->n_steps;
  if (n_fail) *n_fail = f;
  if (n_nonfinite) *n_nonfinite = nf;
  if (min_reg) *min_reg = mr;
}

extern "C" {
// arrays: physical cells only, x fastest, then y, eta, batch; component-major SoA per array (u4: [4][batch][cells]); always double
int vho_set_initial(vho_handle* h, const double* e, const double* u4, const double* pi10, const double* Pi) {
  if (h->evf.empty()) set_initial_t(h->P, h->ev, e, u4, pi10, Pi); else set_initial_t(h->P, h->evf, e, u4, pi10, Pi);
  return 0;
}
int vho_set_uprev(vho_handle* h, const double* up4) {
  if (h->evf.empty()) set_uprev_t(h->P, h->ev, up4); else set_uprev_t(h->P, h->evf, up4);
  return 0;
}
int vho_step(vho_handle* h, int n) {
  for (int it = 0; it < n; ++it) { for (Sol* s : h->ev) s->step(); for (SolF* s : h->evf) s->step(); }
  return 0;
}
int vho_get_fields(vho_handle* h, double* q15, double* e, double* p, double* u4, double* up4) {
  if (h->evf.empty()) get_fields_t(h->P, h->ev, q15, e, p, u4, up4); else get_fields_t(h->P, h->evf, q15, e, p, u4, up4);
  return 0;
}
int vho_get_status(vho_handle* h, double* tau, long long* n_steps, long long* n_fail, long long* n_nonfinite, double* min_reg) {
  if (h->evf.empty()) get_status_t(h->ev, tau, n_steps, n_fail, n_nonfinite, min_reg); else get_status_t(h->evf, tau, n_steps, n_fail, n_nonfinite, min_reg);
  return 0;
}

// maxima over all events of Solver::diagnostics (double instantiation only)
void vho_diagnostics(vho_handle* h, double* out10) {
  for (int i = 0; i < 10; ++i) out10[i] = 0.0;
  for (Sol* s : h->ev) { double o[10]; s->diagnostics(o); for (int i = 0; i < 10; ++i) if (o[i] > out10[i]) out10[i] = o[i]; }
}
// per-cell maps of the ten diagnostics: maps[m * np + c], np = all physical cells of all events
void vho_diagnostic_maps(vho_handle* h, double* maps) {
  const vho::Params& P = h->ev[0]->P;
  const size_t ne = (size_t)P.nx * P.ny * P.nz, np = ne * h->ev.size();
  for (size_t b = 0; b < h->ev.size(); ++b) h->ev[b]->diagnostic_maps(maps, np, b * ne);
}
void vho_last_failure(vho_handle* h, int ev, double* out4) { for (int i = 0; i < 4; ++i) out4[i] = h->ev[ev]->last_fail[i]; }

// ---- raw access to the padded arrays of one event, for unit pins.  which: 0 q 1 qS 2 Q 3 u 4 up 5 uS 6 e 7 p
double* vho_raw(vho_handle* h, int ev, int which, int comp) {
  Sol* s = h->ev[ev];
  switch (which) {
    case 0: return s->q[comp].data();  case 1: return s->qS[comp].data(); case 2: return s->Q[comp].data();
    case 3: return s->u[comp].data();  case 4: return s->up[comp].data(); case 5: return s->uS[comp].data();
    case 6: return s->e.data();        case 7: return s->p.data();
  }
  return nullptr;
}
void vho_set_tau(vho_handle* h, double tau) { for (Sol* s : h->ev) s->tau = tau; }
// J = S + G of Eq. 55 at padded cell (i,j,k) from the current (q,e,p,u,up) at time tau
void vho_sources_at(vho_handle* h, int ev, int i, int j, int k, double tau, double* J15) {
  Sol* s = h->ev[ev];
  s->sources(s->q, s->e, s->p, s->u, s->up, s->idx(i, j, k), tau, J15);
}
// numerical flux H (Eq. 61) of the current q at the interface between padded cells c and c+1 along r, seen from cell (i,j,k)
void vho_flux_at(vho_handle* h, int ev, int i, int j, int k, int r, int upper, double tau, double* H15) {
  Sol* s = h->ev[ev];
  const size_t stride[3] = {1, (size_t)s->NX, (size_t)s->NX * s->NY};
  const double dr[3] = {s->P.dx, s->P.dy, s->P.dz};
  double I[15][5], eI[5];
  size_t c0 = s->idx(i, j, k);
  for (int d = 0; d < 5; ++d) { size_t sn = c0 + d * stride[r] - 2 * stride[r]; for (int n = 0; n < 15; ++n) I[n][d] = s->q[n][sn]; eI[d] = s->e[sn]; }
  s->flux(I, eI, upper ? 2 : 1, r, dr[r], tau, false, H15);
}
void vho_regulation_map(vho_handle* h, double* out) {
  const vho::Params& P = h->ev[0]->P;
  const size_t ne = (size_t)P.nx * P.ny * P.nz;
  for (size_t b = 0; b < h->ev.size(); ++b) h->ev[b]->regulation_map(out + b * ne);
}
void vho_post(vho_handle* h, int ev, double tau) { Sol* s = h->ev[ev]; s->post(s->q, s->u, tau, s->u); }
// post() of q with the current u as the starting velocity of the reduced mode's fixed point (copied first: post overwrites u)
void vho_post_guess(vho_handle* h, int ev, double tau) {
  Sol* s = h->ev[ev];
  std::vector<double> g[4] = {s->u[0], s->u[1], s->u[2], s->u[3]};
  s->post(s->q, s->u, tau, g);
}
void vho_ghost(vho_handle* h, int ev) { Sol* s = h->ev[ev]; s->ghost(s->q, s->e, s->p, s->u); }

// ---- scalar pieces
double vho_minmod3(double x, double y, double z) { return vho::minmod3(x, y, z); }
void vho_eos(const vho::Params* P, double e, double* out3) { auto t = vho::eos<double>(*P, e); t.T = vho::temperature<double>(*P, e); out3[0] = t.p; out3[1] = t.cs2; out3[2] = t.T; }
void vho_transport(const vho::Params* P, double e, double* out5) {
  auto t = vho::eos<double>(*P, e); t.T = vho::temperature<double>(*P, e); auto c = vho::transport<double>(*P, e, t);
  out5[0] = c.inv_tau_pi; out5[1] = c.eta_over_tau_pi; out5[2] = c.inv_tau_Pi; out5[3] = c.zeta_over_tau_Pi; out5[4] = c.lambda_Pipi_over_tau_Pi;
}
double vho_invert(const vho::Params* P, double E, double M2, double Pi, double guess, int* iters, int* failed) {
  return vho::invert_energy<double>(*P, E, M2, Pi, guess, iters, failed);
}
int vho_vorticity_sign() { return vho::kVorticitySign; }

// wall-clock seconds for n steps (bench.py cpu_baseline leg)
double vho_time_steps(vho_handle* h, int n) {
  auto t0 = std::chrono::steady_clock::now();
  vho_step(h, n);
  return std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
}
}
