// oracle_capi.cpp -- extern "C" entry points of the CPU oracle (TEST INFRASTRUCTURE, see gst_oracle.hpp).
// Built by oracle/build.py into oracle/liboracle.so and loaded by oracle/oracle.py (ctypes).
// State arrays cross this boundary as double; `prec` selects the arithmetic type the literal
// formulas are evaluated in between entry and exit: 0 = double, 1 = long double, 2 = __float128.
#include "gst_oracle.hpp"

#include <algorithm>
#include <thread>

using namespace orc;

namespace {

template <class R>
int track_range(const Element* el, size_t n_el, const Beam* beam, double* const* a, uint8_t* lost, size_t lo, size_t hi,
                int64_t n_turns, int split, int n_slices, int depth, double gamma0, double C) {
  for (size_t j = lo; j < hi; ++j) {
    if (lost[j]) continue;
    Particle<R> p;
    p.z = Orbit<R>{R(a[0][j]), R(a[1][j]), R(a[2][j]), R(a[3][j]), R(a[4][j]), R(a[5][j])};
    p.S = Vec3<R>{R(a[6][j]), R(a[7][j]), R(a[8][j])};
    Reference<R> ref;
    ref.set(R(gamma0) * R(beam->mass_eV), R(beam->mass_eV));
    bool alive = true;
    for (int64_t t = 0; alive && t < n_turns; ++t)            // turn loop, element loop
      for (size_t e = 0; alive && e < n_el; ++e)
        alive = track_element(p, el[e], ref, beam->G, split, n_slices, depth, C);
    if (!alive) lost[j] = 1;
    a[0][j] = m::val(p.z.X); a[1][j] = m::val(p.z.Px); a[2][j] = m::val(p.z.Y); a[3][j] = m::val(p.z.Py);
    a[4][j] = m::val(p.z.T); a[5][j] = m::val(p.z.Pt);
    a[6][j] = m::val(p.S.x); a[7][j] = m::val(p.S.y); a[8][j] = m::val(p.S.s);
  }
  return 0;
}

// the reference particle alone: gamma_o after n_turns (A13)
template <class R> double reference_after(const Element* el, size_t n_el, const Beam* beam, int64_t n_turns, double gamma0) {
  Reference<R> ref;
  ref.set(R(gamma0) * R(beam->mass_eV), R(beam->mass_eV));
  for (int64_t t = 0; t < n_turns; ++t)
    for (size_t e = 0; e < n_el; ++e)
      if (el[e].type == RFCAV) {
        Reference<R> nref;
        nref.set(ref.E0 + R(el[e].volt_eV) * m::sin(R(el[e].phi_s)), ref.mass);
        ref = nref;
      }
  return m::val(ref.gamma0);
}

int validate(const Element* el, size_t n_el, int split, int n_slices, int depth) {
  if (n_slices < 1 || depth < -1 || depth > 12 || split < 0 || split > 5) return 1;   // depth 0, -1: PWC (section 4.1)
  for (size_t e = 0; e < n_el; ++e) {
    int t = el[e].type;
    if (t < 0 || t > RBEND) return 1;
    if (t == SBEND || t == QUAD || t == MULTIPOLE || t == SOLENOID || t == RBEND) {
      if (el[e].slice_mult < 1 || el[e].L == 0) return 1;   // L < 0 allowed here: inverse flow, used by the reversibility pins
      long N = (long)n_slices * el[e].slice_mult;
      if (depth >= 1 && N % (1L << (depth - 1)) != 0) return 1;   // A4
      if (t == SBEND && (el[e].h == 0 || el[e].k0 == 0)) return 1;
      if (t == QUAD && el[e].kn[0] == 0) return 1;
      if ((t == SOLENOID || t == RBEND) && el[e].k0 == 0) return 1;
    }
  }
  return 0;
}

}  // namespace

extern "C" {

// Track n particles (SoA double arrays, updated in place) for n_turns.  lost[] is in/out.
// *gamma0 is the reference gamma at entry and is updated to its value after n_turns.
// Returns 0 on success, 1 on invalid arguments.
int orc_track(const Element* el, size_t n_el, const Beam* beam, double* x, double* px, double* y, double* py, double* t,
              double* pt, double* sx, double* sy, double* ss, uint8_t* lost, size_t n, int64_t n_turns, int split,
              int n_slices, int depth, int prec, int nthreads, double* gamma0) {
  if (validate(el, n_el, split, n_slices, depth)) return 1;
  double* a[9] = {x, px, y, py, t, pt, sx, sy, ss};
  double C = ring_circumference(el, n_el);
  if (nthreads < 1) nthreads = 1;
  nthreads = (int)std::min<size_t>((size_t)nthreads, std::max<size_t>(n, 1));
  std::vector<std::thread> pool;
  double g0 = *gamma0;
  for (int w = 0; w < nthreads; ++w) {
    size_t lo = n * w / nthreads, hi = n * (w + 1) / nthreads;
    pool.emplace_back([=]() {
      if (prec == 0) track_range<double>(el, n_el, beam, a, lost, lo, hi, n_turns, split, n_slices, depth, g0, C);
      else if (prec == 1) track_range<long double>(el, n_el, beam, a, lost, lo, hi, n_turns, split, n_slices, depth, g0, C);
      else track_range<__float128>(el, n_el, beam, a, lost, lo, hi, n_turns, split, n_slices, depth, g0, C);
    });
  }
  for (auto& th : pool) th.join();
  if (prec == 0) *gamma0 = reference_after<double>(el, n_el, beam, n_turns, g0);
  else if (prec == 1) *gamma0 = reference_after<long double>(el, n_el, beam, n_turns, g0);
  else *gamma0 = reference_after<__float128>(el, n_el, beam, n_turns, g0);
  return 0;
}

// One pass through el[0..n_el) starting from z0, with the 6x6 Jacobian d z_f / d z_0 (row-major)
// by forward-mode dual numbers through the same templated code.  Returns 0 ok, 1 invalid, 2 lost.
int orc_jacobian(const Element* el, size_t n_el, const Beam* beam, const double* z0, int split, int n_slices,
                 double circumference, double* J, double* zf) {
  if (validate(el, n_el, split, n_slices, 1)) return 1;
  typedef Dual<6> D;
  Particle<D> p;
  D* zz[6] = {&p.z.X, &p.z.Px, &p.z.Y, &p.z.Py, &p.z.T, &p.z.Pt};
  for (int i = 0; i < 6; ++i) { *zz[i] = D(z0[i]); zz[i]->d[i] = 1.0; }
  p.S = Vec3<D>{D(0.0), D(1.0), D(0.0)};
  Reference<D> ref;
  ref.set(D(beam->gamma0) * D(beam->mass_eV), D(beam->mass_eV));
  for (size_t e = 0; e < n_el; ++e)
    if (!track_element(p, el[e], ref, beam->G, split, n_slices, 1, circumference)) return 2;
  for (int i = 0; i < 6; ++i) {
    zf[i] = zz[i]->v;
    for (int k = 0; k < 6; ++k) J[6 * i + k] = zz[i]->d[k];
  }
  return 0;
}

// The spin scheme alone on caller-supplied edge vectors Om[3*(N+1)] (x,y,s interleaved).
int orc_romberg(const double* Om, int N, double ds, int depth, int prec, double* q_out) {
  if (N < 1 || depth < 1 || N % (1 << (depth - 1)) != 0) return 1;
  if (prec == 0) {
    std::vector<Vec3<double>> v(N + 1);
    for (int i = 0; i <= N; ++i) v[i] = Vec3<double>{Om[3 * i], Om[3 * i + 1], Om[3 * i + 2]};
    Quat<double> q = romberg_quaternion(v, N, ds, depth);
    q_out[0] = q.w; q_out[1] = q.x; q_out[2] = q.y; q_out[3] = q.s;
  } else {
    std::vector<Vec3<__float128>> v(N + 1);
    for (int i = 0; i <= N; ++i) v[i] = Vec3<__float128>{Om[3 * i], Om[3 * i + 1], Om[3 * i + 2]};
    Quat<__float128> q = romberg_quaternion(v, N, (__float128)ds, depth);
    q_out[0] = (double)q.w; q_out[1] = (double)q.x; q_out[2] = (double)q.y; q_out[3] = (double)q.s;
  }
  return 0;
}

// Omega of (6b) at one phase-space point of one element (for the pins on a9).
int orc_omega(const Element* e, const Beam* beam, const double* z, double* Om_out) {
  Reference<long double> ref;
  ref.set((long double)beam->gamma0 * beam->mass_eV, (long double)beam->mass_eV);
  Orbit<long double> o{z[0], z[1], z[2], z[3], z[4], z[5]};
  Vec3<long double> Om;
  if (!omega_tbmt(o, (long double)e->h, element_field(*e, o), beam->G, ref, Om)) return 2;
  Om_out[0] = (double)Om.x; Om_out[1] = (double)Om.y; Om_out[2] = (double)Om.s;
  return 0;
}

// A18: P = (1/N_alive) sum S_j ; out = {Px, Py, Ps, |P|}; returns number lost through *n_lost.
void orc_polarization(const double* sx, const double* sy, const double* ss, const uint8_t* lost, size_t n, double* out,
                      int64_t* n_lost) {
  long double a = 0, b = 0, c = 0;
  int64_t alive = 0;
  for (size_t j = 0; j < n; ++j) {
    if (lost && lost[j]) continue;
    a += sx[j]; b += sy[j]; c += ss[j]; ++alive;
  }
  if (alive) { a /= alive; b /= alive; c /= alive; }
  out[0] = (double)a; out[1] = (double)b; out[2] = (double)c; out[3] = (double)sqrtl(a * a + b * b + c * c);
  if (n_lost) *n_lost = (int64_t)n - alive;
}

// A19: geometric rms emittance sqrt(<u~^2><p~^2> - <u~ p~>^2), mean-subtracted, per plane.
void orc_emittance(const double* x, const double* px, const double* y, const double* py, const uint8_t* lost, size_t n,
                   double* out_exy) {
  const double* u[2] = {x, y};
  const double* p[2] = {px, py};
  for (int k = 0; k < 2; ++k) {
    long double mu = 0, mp = 0;
    int64_t alive = 0;
    for (size_t j = 0; j < n; ++j) { if (lost && lost[j]) continue; mu += u[k][j]; mp += p[k][j]; ++alive; }
    if (!alive) { out_exy[k] = 0; continue; }
    mu /= alive; mp /= alive;
    long double suu = 0, spp = 0, sup = 0;
    for (size_t j = 0; j < n; ++j) {
      if (lost && lost[j]) continue;
      long double du = u[k][j] - mu, dp = p[k][j] - mp;
      suu += du * du; spp += dp * dp; sup += du * dp;
    }
    suu /= alive; spp /= alive; sup /= alive;
    long double e2 = suu * spp - sup * sup;
    out_exy[k] = (double)sqrtl(e2 > 0 ? e2 : 0);
  }
}

}  // extern "C"
