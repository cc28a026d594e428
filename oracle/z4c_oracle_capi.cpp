// z4c_oracle_capi.cpp -- TEST INFRASTRUCTURE (the oracle's own C interface).
//
// extern "C" entry points over the templated oracle, as double (the oracle) and
// as __float128 (referee: same source, 113-bit significand, inputs/outputs
// converted from/to double at the interface). Built by oracle/build.py with
//   g++ -O2 -std=c++17 -fopenmp -ffp-contract=off -fno-fast-math -shared -fPIC
// (the paper's flags: PAPER.md:206).
// This library is NOT the product's C ABI (that is include/sacra.h) and shares
// no code with it.
#include <cstring>
#include <vector>
#include <omp.h>
#include "z4c_grid.hpp"
#include "z4c_amr.hpp"
#include "z4c_boundary.hpp"
#include "z4c_subcycle.hpp"

using namespace z4c_oracle;

extern "C" {
struct orc_patch { int32_t nx, ny, nz, ng; int64_t pitch_x, field_stride, patch_offset; double dx, dt; };
struct orc_params { double kappa1, kappa2, eta, shift_coef, ko_sigma; int32_t lapse_uses_khat; };
}

static Patch to_patch(const orc_patch& q) {
  Patch p; p.nx = q.nx; p.ny = q.ny; p.nz = q.nz; p.pitch = q.pitch_x; p.fstride = q.field_stride;
  p.offset = q.patch_offset; p.dx = q.dx; p.dt = q.dt; return p;
}
template <class T> static Params<T> to_params(const orc_params& q) {
  Params<T> P; P.kappa1 = T(q.kappa1); P.kappa2 = T(q.kappa2); P.eta = T(q.eta);
  P.shift_coef = T(q.shift_coef); P.ko_sigma = T(q.ko_sigma); P.lapse_uses_khat = q.lapse_uses_khat;
  return P;
}

// ---- operation count (for the roofline's algorithmic flops) ----------------------------
// The same templated source instantiated with a scalar that counts its own +, -, *, / (unary minus is free).
struct Cnt {
  double v;
  static long add, mul, div;
  Cnt() : v(0) {}
  Cnt(double x) : v(x) {}
  Cnt(int x) : v(x) {}
  Cnt(long x) : v((double)x) {}
  friend Cnt operator+(Cnt a, Cnt b) { ++add; return Cnt(a.v + b.v); }
  friend Cnt operator-(Cnt a, Cnt b) { ++add; return Cnt(a.v - b.v); }
  friend Cnt operator*(Cnt a, Cnt b) { ++mul; return Cnt(a.v * b.v); }
  friend Cnt operator/(Cnt a, Cnt b) { ++div; return Cnt(a.v / b.v); }
  friend Cnt operator-(Cnt a) { return Cnt(-a.v); }
  friend bool operator>=(Cnt a, Cnt b) { return a.v >= b.v; }
  Cnt& operator+=(Cnt b) { ++add; v += b.v; return *this; }
  Cnt& operator-=(Cnt b) { ++add; v -= b.v; return *this; }
};
long Cnt::add = 0; long Cnt::mul = 0; long Cnt::div = 0;

extern "C" {

int orc_num_threads(void) { return omp_get_max_threads(); }
void orc_set_threads(int n) { omp_set_num_threads(n); }

// ---- double ---------------------------------------------------------------
void orc_fill_ghosts(const orc_patch* ps, int np, double* u) {
  for (int q = 0; q < np; ++q) fill_ghosts<double>(to_patch(ps[q]), u);
}
void orc_fill_ghosts_bc(const orc_patch* ps, int np, const int32_t* mode, double* u) {
  const int m[3] = {mode[0], mode[1], mode[2]};
  for (int q = 0; q < np; ++q) fill_ghosts_bc<double>(to_patch(ps[q]), m, u);
}
void orc_z4c_rhs(const orc_patch* ps, int np, const orc_params* prm, const double* u, double* rhs) {
  auto P = to_params<double>(*prm);
  for (int q = 0; q < np; ++q) rhs_patch<double>(to_patch(ps[q]), P, u, rhs);
}
// stage in 1..4; kbuf: scratch state of the same size
void orc_rk4_substep(const orc_patch* ps, int np, const orc_params* prm, int stage, const double* u_n,
                     const double* u_in, double* u_out, double* acc, double* kbuf) {
  auto P = to_params<double>(*prm);
  for (int q = 0; q < np; ++q) rk4_substep<double>(to_patch(ps[q]), P, stage, u_n, u_in, u_out, acc, kbuf);
}
// work: 4 states back to back, each nstate doubles: stage A, stage B, acc (returns S), k scratch
void orc_rk4_step(const orc_patch* ps, int np, const orc_params* prm, double* u, double* work, int64_t nstate) {
  auto P = to_params<double>(*prm);
  std::vector<Patch> v; for (int q = 0; q < np; ++q) v.push_back(to_patch(ps[q]));
  rk4_step<double>(v.data(), np, P, u, work, work + nstate, work + 2 * nstate, work + 3 * nstate);
}

// f-1: constraints on all active cells (con: state-shaped, fields 0..3), their norms (Eq. 22), and the point-wise
// form with caller-supplied derivatives (analytic-derivative pins)
void orc_constraints(const orc_patch* ps, int np, const double* u, double* con) {
  for (int q = 0; q < np; ++q) constraints_patch<double>(to_patch(ps[q]), u, con);
}
void orc_constraint_norms(const orc_patch* ps, int np, const double* con, double* norms) {
  std::vector<Patch> v; for (int q = 0; q < np; ++q) v.push_back(to_patch(ps[q]));
  constraint_norms<double>(v.data(), np, con, norms);
}
void orc_constraints_point(const double* u, const double* d1, const double* d2, double* out) {
  static thread_local Derivs<double> D;
  std::memcpy(D.d1, d1, sizeof(D.d1)); std::memcpy(D.d2, d2, sizeof(D.d2));
  constraints_point<double>(u, D, out);
}

// f-3: spatial inter-level operators (2:1, cell-centred): restriction child -> parent, prolongation of the child's ghosts
void orc_restrict(const orc_patch* parent, const orc_patch* child, const int32_t* org, double* u_parent,
                  const double* u_child) {
  const int o[3] = {org[0], org[1], org[2]};
  restrict_patch<double>(to_patch(*parent), to_patch(*child), o, u_parent, u_child);
}
void orc_prolong_ghosts(const orc_patch* parent, const orc_patch* child, const int32_t* org, const double* u_parent,
                        double* u_child) {
  const int o[3] = {org[0], org[1], org[2]};
  prolong_ghosts<double>(to_patch(*parent), to_patch(*child), o, u_parent, u_child);
}

// single-point algebra with caller-supplied derivatives (for analytic-derivative pins)
// d1: [25][3], d2: [25][6] (xx xy xz yy yz zz), adv: [25], ko: [25]
void orc_rhs_point(const orc_params* prm, const double* u, const double* d1, const double* d2,
                   const double* adv, const double* ko, double* out) {
  auto P = to_params<double>(*prm);
  Derivs<double> D;
  std::memcpy(D.d1, d1, sizeof(D.d1)); std::memcpy(D.d2, d2, sizeof(D.d2));
  std::memcpy(D.adv, adv, sizeof(D.adv)); std::memcpy(D.ko, ko, sizeof(D.ko));
  z4c_rhs_point<double>(u, D, P, out);
}

// per-point derivative bundle of one field at one active cell (stencil pins)
// out: d1[3], d2[6], adv, ko  (11 doubles)
void orc_derivs_field(const orc_patch* p_, const double* u, int field, int i, int j, int k,
                      double sigma, double* out) {
  Patch p = to_patch(*p_);
  const double* f[NF];
  for (int n = 0; n < NF; ++n) f[n] = u + p.offset + (long)n * p.fstride;
  Derivs<double> D;
  derivs_at<double>(f, cell(p, i + NG, j + NG, k + NG), sy_of(p), sz_of(p), p.dx, sigma, D);
  for (int a = 0; a < 3; ++a) out[a] = D.d1[field][a];
  for (int a = 0; a < 6; ++a) out[3 + a] = D.d2[field][a];
  out[9] = D.adv[field]; out[10] = D.ko[field];
}

// ---- operation count: entry point (Cnt is defined above) ----------------------------------------------------
// counts[0..2] = adds, muls, divs of the point-wise algebra (items 7-10) at one point;
// counts[3..5] = the same for the oracle's derivative bundle of ONE field (3 D1, 6 D2, upwind, KO)
void orc_count_ops(long* counts) {
  Params<Cnt> P; P.kappa1 = Cnt(0.02); P.kappa2 = Cnt(0.1); P.eta = Cnt(2.0); P.shift_coef = Cnt(0.75);
  P.ko_sigma = Cnt(0.1); P.lapse_uses_khat = 1;
  Cnt u[NF], out[NF];
  for (int n = 0; n < NF; ++n) u[n] = Cnt(0.01 * (n + 1));
  u[F_W] = Cnt(0.9); u[F_ALP] = Cnt(0.8); u[F_G] = Cnt(1.1); u[F_G + 3] = Cnt(1.2); u[F_G + 5] = Cnt(0.95);
  static Derivs<Cnt> D;
  for (int n = 0; n < NF; ++n) {
    for (int a = 0; a < 3; ++a) D.d1[n][a] = Cnt(0.003 * (n + a));
    for (int a = 0; a < 6; ++a) D.d2[n][a] = Cnt(0.002 * (n - a));
    D.adv[n] = Cnt(0.001 * n); D.ko[n] = Cnt(-0.001 * n);
  }
  Cnt::add = Cnt::mul = Cnt::div = 0;
  z4c_rhs_point<Cnt>(u, D, P, out);
  counts[0] = Cnt::add; counts[1] = Cnt::mul; counts[2] = Cnt::div;
  // derivative bundle: a 7^3 neighbourhood of 25 fields
  const int n = 7; const long sy = n, sz = n * n, fs = n * n * n;
  std::vector<Cnt> buf(NF * fs);
  for (size_t i = 0; i < buf.size(); ++i) buf[i] = Cnt(1e-3 * (double)(i % 97));
  const Cnt* f[NF];
  for (int q = 0; q < NF; ++q) f[q] = buf.data() + q * fs;
  Cnt::add = Cnt::mul = Cnt::div = 0;
  derivs_at<Cnt>(f, 3 * sz + 3 * sy + 3, sy, sz, Cnt(0.1), Cnt(0.1), D);
  counts[3] = Cnt::add / NF; counts[4] = Cnt::mul / NF; counts[5] = Cnt::div / NF;
}

// ---- physical boundaries: per-face ghost fill, Sommerfeld shell, RK4 step with boundaries ----------
struct orc_boundary { double origin[3]; int32_t face[6]; };
static Boundary to_boundary(const orc_boundary& q) {
  Boundary b;
  for (int a = 0; a < 3; ++a) b.origin[a] = q.origin[a];
  for (int a = 0; a < 6; ++a) b.face[a] = q.face[a];
  return b;
}
void orc_fill_ghosts_faces(const orc_patch* ps, const orc_boundary* bs, int np, double* u) {
  for (int q = 0; q < np; ++q) { Boundary b = to_boundary(bs[q]); fill_ghosts_faces<double>(to_patch(ps[q]), b.face, u); }
}
void orc_sommerfeld_rhs(const orc_patch* ps, const orc_boundary* bs, int np, const double* u, double* rhs) {
  for (int q = 0; q < np; ++q) sommerfeld_rhs_patch<double>(to_patch(ps[q]), to_boundary(bs[q]), u, rhs);
}
// first derivative along x of a 1-D array of n samples at index i using indices lo..hi only (stencil pins)
double orc_d1_bounded(const double* u, int i, int lo, int hi, double h) {
  return d1_bounded<double>([&](int q) { return u[i + q]; }, i, lo, hi, 1.0 / (12.0 * h));
}
void orc_rk4_substep_bc(const orc_patch* ps, const orc_boundary* bs, int np, const orc_params* prm, int stage,
                        const double* u_n, const double* u_in, double* u_out, double* acc, double* kbuf) {
  auto P = to_params<double>(*prm);
  for (int q = 0; q < np; ++q)
    rk4_substep_bc<double>(to_patch(ps[q]), P, to_boundary(bs[q]), stage, u_n, u_in, u_out, acc, kbuf);
}
void orc_rk4_step_bc(const orc_patch* ps, const orc_boundary* bs, int np, const orc_params* prm, double* u,
                     double* work, int64_t nstate) {
  auto P = to_params<double>(*prm);
  std::vector<Patch> v; std::vector<Boundary> b;
  for (int q = 0; q < np; ++q) { v.push_back(to_patch(ps[q])); b.push_back(to_boundary(bs[q])); }
  rk4_step_bc<double>(v.data(), b.data(), np, P, u, work, work + nstate, work + 2 * nstate, work + 3 * nstate);
}

// ---- subcycling: time weights, linear combination of parent levels, one Berger-Oliger step ---------
void orc_time_weights(int n, double theta, double* w) { time_weights<double>(n, theta, w); }
void orc_lincomb(const orc_patch* p, int n, const double* u0, const double* u1, const double* u2, const double* w,
                 double* out) {
  const double* u[3] = {u0, u1, u2};
  lincomb_patch<double>(to_patch(*p), n, u, w, out);
}
void orc_subcycle_step(const orc_patch* parent, const orc_patch* child, const int32_t* org, const orc_params* prm,
                       const orc_boundary* bnd, double* u_parent, double* u_parent_prev, int have_prev, double* u_child,
                       int64_t n_parent, int64_t n_child) {
  const int o[3] = {org[0], org[1], org[2]};
  subcycle_step<double>(to_patch(*parent), to_patch(*child), o, to_params<double>(*prm), to_boundary(*bnd), u_parent,
                        u_parent_prev, have_prev != 0, u_child, n_parent, n_child);
}

// one step of the coarsest level of a hierarchy of nlevels nested levels (level l + 1 inside level l); arrays of nlevels
// entries; nsteps is updated
void orc_hierarchy_step(const orc_patch* patches, const int32_t* orgs /* 3 per level */, int nlevels, const orc_params* prm,
                        const orc_boundary* bnd0, double* const* u, double* const* prev, const int64_t* ndoubles,
                        int64_t* nsteps) {
  std::vector<Level<double>> L(nlevels);
  for (int l = 0; l < nlevels; ++l) {
    L[l].p = to_patch(patches[l]);
    for (int a = 0; a < 3; ++a) L[l].org[a] = orgs[3 * l + a];
    L[l].u = u[l]; L[l].prev = prev[l]; L[l].n = ndoubles[l]; L[l].nsteps = nsteps[l];
  }
  hierarchy_advance<double>(L, 0, to_params<double>(*prm), to_boundary(*bnd0), 0);
  for (int l = 0; l < nlevels; ++l) nsteps[l] = L[l].nsteps;
}

// ---- __float128 referee ------------------------------------------------------
typedef __float128 Q;
void orc_z4c_rhs_q(const orc_patch* ps, int np, const orc_params* prm, const double* u, double* rhs,
                   int64_t nstate) {
  auto P = to_params<Q>(*prm);
  std::vector<Q> uq(nstate), rq(nstate, Q(0));
  for (int64_t i = 0; i < nstate; ++i) uq[i] = Q(u[i]);
  for (int q = 0; q < np; ++q) rhs_patch<Q>(to_patch(ps[q]), P, uq.data(), rq.data());
  for (int64_t i = 0; i < nstate; ++i) rhs[i] = (double)rq[i];
}
void orc_rk4_step_q(const orc_patch* ps, int np, const orc_params* prm, double* u, double* S,
                    int64_t nstate) {
  auto P = to_params<Q>(*prm);
  std::vector<Patch> v; for (int q = 0; q < np; ++q) v.push_back(to_patch(ps[q]));
  std::vector<Q> uq(nstate), w(4 * nstate, Q(0));
  for (int64_t i = 0; i < nstate; ++i) uq[i] = Q(u[i]);
  rk4_step<Q>(v.data(), np, P, uq.data(), w.data(), w.data() + nstate, w.data() + 2 * nstate,
              w.data() + 3 * nstate);
  for (int64_t i = 0; i < nstate; ++i) { u[i] = (double)uq[i]; S[i] = (double)w[2 * nstate + i]; }
}

}  // extern "C"
