// gst_oracle.hpp -- CPU ORACLE for spin-orbit tracking (arXiv:1501.03450, GPUSPINTRACK).
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may build, link or call anything in oracle/.
// It shares no code, header, table or helper with the CUDA path in paper_1501_03450_b200/csrc.
//
// It follows the paper's algorithm step by step, in the paper's order and notation, with the
// formulas typed as printed ("P:nnn" = /root/reference/PAPER.md line nnn).  There is no blocking,
// fusion, hoisting or algebraic rearrangement: every slice re-evaluates every square root,
// every trigonometric function and every arcsine, and all slice-edge precession vectors of an
// element are stored in a std::vector before the quaternion products are formed.
//
// Everything is templated on the scalar type R so that the SAME literal formulas can be run
//   * in double           (the fp64 CPU baseline that bench.py times),
//   * in long double      (x87 80-bit; the default parity reference -- the literal forms (10a),
//                          (29b), (25e) cancel O(1) terms, which in double costs ~1e-11 of the
//                          bunch scale per slice; DESIGN.md "Readings" R1),
//   * in __float128       (ground truth for the cancellation checks),
//   * in Dual<6>          (forward-mode derivatives -> Jacobians for symplecticity / optics pins).
//
// Parity status: every function here is pinned by tests/test_oracle_*.py.  The RF cavity with ramp
// (A12/A13) is a READING -- its formulas are not in the paper -- pinned by its linearised kick and the
// one-turn longitudinal map at two energies, the re-referencing element by element, the adiabatic
// invariants (transverse and longitudinal) and the Froissart-Stora crossing of a partial-snake
// resonance (tests/test_oracle_rf_reductions.py); the config-4 polarization curve of a real lattice
// has no closed form and is GPU-vs-oracle only.
#pragma once
#include <cmath>
#include <cstdint>
#include <vector>
#include <quadmath.h>

namespace orc {

// ----------------------------------------------------------------------------------------------
// element table entry (the oracle's own definition; field meaning identical to DESIGN.md §2)
// ----------------------------------------------------------------------------------------------
enum ElemType { DRIFT = 0, SBEND = 1, QUAD = 2, MULTIPOLE = 3, THINMULT = 4, RFCAV = 5, SNAKE = 6, MARKER = 7,
                FRINGE = 8,     // thin-fringe spin kick (41) P:557-563, SURVEY 8(f) f3
                SOLENOID = 9,   // solenoid with thin-pancake fringes (32)-(36), (40) P:420-464, f4
                RBEND = 10 };   // rectangular bend (11)-(19) P:161-261 with the fringe spin kick (42) P:567, f3
enum Split { SPLIT_DRIFT_KICK = 0, SPLIT_BEND_KICK = 1, SPLIT_MATRIX_KICK = 2,
             // the same splits with every second-order slice map (27) replaced by the fourth-order symmetric
             // composition of three of them ("more sophisticated symmetric compositions", "higher-order
             // versions of (27)", refs [62, 45, 23]); reading R5
             SPLIT_DRIFT_KICK_4 = 3, SPLIT_BEND_KICK_4 = 4, SPLIT_MATRIX_KICK_4 = 5 };

struct Element {
  int32_t type;
  int32_t slice_mult;   // slices = n_slices * slice_mult for thick magnets ("4 n_b")
  double L;             // length [m]
  double h;             // curvature of the local frame, 1/rho_c [1/m]
  double k0;            // b_1/(B rho)_o = eta*h [1/m] (9)
  double kn[4], ks[4];  // (b_m, a_m)/(B rho)_o for m = 2..5 in the convention of (28); thin: times L
  double volt_eV, harmonic, phi_s, sign;  // cavity (A12)
  double snake_mu, snake_phi;             // snake rotation angle, axis angle from s-hat in the x-s plane (A14)
};
struct Beam { double G, mass_eV, gamma0; };

// ----------------------------------------------------------------------------------------------
// scalar-type plumbing: double, long double, __float128, Dual<N>
// ----------------------------------------------------------------------------------------------
namespace m {
inline double sqrt(double x) { return std::sqrt(x); }
inline double sin(double x) { return std::sin(x); }
inline double cos(double x) { return std::cos(x); }
inline double tan(double x) { return std::tan(x); }
inline double asin(double x) { return std::asin(x); }
inline double sinh(double x) { return std::sinh(x); }
inline double cosh(double x) { return std::cosh(x); }
inline long double sqrt(long double x) { return sqrtl(x); }
inline long double sin(long double x) { return sinl(x); }
inline long double cos(long double x) { return cosl(x); }
inline long double tan(long double x) { return tanl(x); }
inline long double asin(long double x) { return asinl(x); }
inline long double sinh(long double x) { return sinhl(x); }
inline long double cosh(long double x) { return coshl(x); }
inline __float128 sqrt(__float128 x) { return sqrtq(x); }
inline __float128 sin(__float128 x) { return sinq(x); }
inline __float128 cos(__float128 x) { return cosq(x); }
inline __float128 tan(__float128 x) { return tanq(x); }
inline __float128 asin(__float128 x) { return asinq(x); }
inline __float128 sinh(__float128 x) { return sinhq(x); }
inline __float128 cosh(__float128 x) { return coshq(x); }
inline double pi_of(double) { return 3.14159265358979323846; }
inline long double pi_of(long double) { return 3.14159265358979323846264338327950288L; }
inline __float128 pi_of(__float128) { return __float128(4) * atanq(__float128(1)); }
inline double val(double x) { return x; }
inline double val(long double x) { return (double)x; }
inline double val(__float128 x) { return (double)x; }
}  // namespace m

// forward-mode dual number with N derivative slots
template <int N>
struct Dual {
  double v;
  double d[N];
  Dual() : v(0) { for (int i = 0; i < N; ++i) d[i] = 0; }
  Dual(double x) : v(x) { for (int i = 0; i < N; ++i) d[i] = 0; }
  Dual(int x) : v(x) { for (int i = 0; i < N; ++i) d[i] = 0; }
};
template <int N> Dual<N> chain(const Dual<N>& a, double f, double df) {
  Dual<N> r; r.v = f; for (int i = 0; i < N; ++i) r.d[i] = df * a.d[i]; return r;
}
template <int N> Dual<N> operator+(const Dual<N>& a, const Dual<N>& b) { Dual<N> r; r.v = a.v + b.v; for (int i = 0; i < N; ++i) r.d[i] = a.d[i] + b.d[i]; return r; }
template <int N> Dual<N> operator-(const Dual<N>& a, const Dual<N>& b) { Dual<N> r; r.v = a.v - b.v; for (int i = 0; i < N; ++i) r.d[i] = a.d[i] - b.d[i]; return r; }
template <int N> Dual<N> operator-(const Dual<N>& a) { Dual<N> r; r.v = -a.v; for (int i = 0; i < N; ++i) r.d[i] = -a.d[i]; return r; }
template <int N> Dual<N> operator*(const Dual<N>& a, const Dual<N>& b) { Dual<N> r; r.v = a.v * b.v; for (int i = 0; i < N; ++i) r.d[i] = a.d[i] * b.v + a.v * b.d[i]; return r; }
template <int N> Dual<N> operator/(const Dual<N>& a, const Dual<N>& b) { Dual<N> r; r.v = a.v / b.v; for (int i = 0; i < N; ++i) r.d[i] = (a.d[i] - r.v * b.d[i]) / b.v; return r; }
template <int N> Dual<N>& operator+=(Dual<N>& a, const Dual<N>& b) { a = a + b; return a; }
template <int N> Dual<N>& operator-=(Dual<N>& a, const Dual<N>& b) { a = a - b; return a; }
template <int N> bool operator<=(const Dual<N>& a, const Dual<N>& b) { return a.v <= b.v; }
template <int N> bool operator>=(const Dual<N>& a, const Dual<N>& b) { return a.v >= b.v; }
template <int N> bool operator<(const Dual<N>& a, const Dual<N>& b) { return a.v < b.v; }
template <int N> bool operator>(const Dual<N>& a, const Dual<N>& b) { return a.v > b.v; }
template <int N> bool operator==(const Dual<N>& a, const Dual<N>& b) { return a.v == b.v; }
namespace m {
template <int N> Dual<N> sqrt(const Dual<N>& a) { double f = std::sqrt(a.v); return chain(a, f, 0.5 / f); }
template <int N> Dual<N> sin(const Dual<N>& a) { return chain(a, std::sin(a.v), std::cos(a.v)); }
template <int N> Dual<N> cos(const Dual<N>& a) { return chain(a, std::cos(a.v), -std::sin(a.v)); }
template <int N> Dual<N> tan(const Dual<N>& a) { double t = std::tan(a.v); return chain(a, t, 1.0 + t * t); }
template <int N> Dual<N> asin(const Dual<N>& a) { return chain(a, std::asin(a.v), 1.0 / std::sqrt(1.0 - a.v * a.v)); }
template <int N> Dual<N> sinh(const Dual<N>& a) { return chain(a, std::sinh(a.v), std::cosh(a.v)); }
template <int N> Dual<N> cosh(const Dual<N>& a) { return chain(a, std::cosh(a.v), std::sinh(a.v)); }
template <int N> double val(const Dual<N>& a) { return a.v; }
template <int N> Dual<N> pi_of(const Dual<N>&) { return Dual<N>(3.14159265358979323846); }
}  // namespace m

// ----------------------------------------------------------------------------------------------
// state
// ----------------------------------------------------------------------------------------------
template <class R> struct Orbit { R X, Px, Y, Py, T, Pt; };   // (1) P:55, MAD canonical coordinates
template <class R> struct Vec3 { R x, y, s; };                 // components along (x-hat, y-hat, s-hat)
template <class R> struct Quat { R w, x, y, s; };              // scalar part w, vector part (x, y, s)

// reference particle: p_o = m gamma_o beta_o c.  Changes only at a ramping cavity (A13).
template <class R> struct Reference {
  R E0;      // reference total energy [eV]
  R mass;    // [eV]
  R gamma0, beta0, p0c;
  void set(R E, R mc2) {
    E0 = E; mass = mc2;
    gamma0 = E0 / mass;
    p0c = m::sqrt(E0 * E0 - mass * mass);
    beta0 = p0c / E0;
  }
};

// ----------------------------------------------------------------------------------------------
// orbit maps.  Every map returns false when a square-root argument or a denominator leaves its
// domain (A15: the particle is flagged lost).
// ----------------------------------------------------------------------------------------------

// (5) P:92   P_s^2 = 1 + 2 Pt/beta_o + Pt^2 - Px^2 - Py^2
template <class R> R Ps2(const Orbit<R>& z, const Reference<R>& ref) {
  return R(1) + R(2) * z.Pt / ref.beta0 + z.Pt * z.Pt - z.Px * z.Px - z.Py * z.Py;
}
// (22) P:289  P^2 = 1 + 2 Pt/beta_o + Pt^2
template <class R> R Ptot2(const Orbit<R>& z, const Reference<R>& ref) {
  return R(1) + R(2) * z.Pt / ref.beta0 + z.Pt * z.Pt;
}

// exact drift: flow of H_drift = -P_s + Pt/beta_o, (29b) P:371.  Hamilton's equations give
//   X' = Px/Ps, Y' = Py/Ps, T' = dH/dPt = -(1/beta_o + Pt)/Ps + 1/beta_o, momenta constant.
template <class R> bool drift(Orbit<R>& z, R L, const Reference<R>& ref) {
  R ps2 = Ps2(z, ref);
  if (ps2 <= R(0)) return false;
  R Ps = m::sqrt(ps2);
  z.X = z.X + L * z.Px / Ps;
  z.Y = z.Y + L * z.Py / Ps;
  z.T = z.T + L * (R(1) / ref.beta0 - (R(1) / ref.beta0 + z.Pt) / Ps);
  return true;
}

// exact sector bend, (8)-(10) P:127-151, over arc length s; eta = k0/h (9).
template <class R> bool sbend_exact(Orbit<R>& z, R s, R h, R k0, const Reference<R>& ref) {
  R eta = k0 / h;                                                                 // (9)
  R Pa2 = R(1) + R(2) * z.Pt / ref.beta0 + z.Pt * z.Pt - z.Py * z.Py;             // (8)
  if (Pa2 <= R(0)) return false;
  R Pa = m::sqrt(Pa2);
  R a2 = Pa2 - z.Px * z.Px;
  if (a2 <= R(0)) return false;
  R root_i = m::sqrt(a2);
  R c = m::cos(h * s), sn = m::sin(h * s);
  R bracket = root_i - eta * (R(1) + h * z.X);
  R Pxf = z.Px * c + bracket * sn;                                                // (10b)
  R dPxds = h * (-z.Px * sn + bracket * c);                                       // d/ds of (10b)
  R f2 = Pa2 - Pxf * Pxf;
  if (f2 <= R(0)) return false;
  R Xf = (R(1) / h) * ((R(1) / eta) * (m::sqrt(f2) - dPxds / h) - R(1));          // (10a)
  R dasin = m::asin(z.Px / Pa) - m::asin(Pxf / Pa);
  R Yf = z.Y + z.Py * s / eta + z.Py * dasin / (eta * h);                         // (10c)
  R Tf = z.T - z.Pt * s / eta - (R(1) / ref.beta0 + z.Pt) * dasin / (eta * h)
         + (R(1) - R(1) / eta) * s / ref.beta0;                                   // (10e)
  z.X = Xf; z.Px = Pxf; z.Y = Yf; z.T = Tf;                                       // (10d),(10f): Py, Pt constant
  return true;
}

// TEAPOT curved drift: flow of H_D (30b) over arc length s, (31) P:397-412, with the reading
// A5: + s/beta_o added to (31e) so that T stays a deviation consistent with (3)/(10e).
template <class R> bool curved_drift(Orbit<R>& z, R s, R h, const Reference<R>& ref) {
  R ps2 = Ps2(z, ref);
  if (ps2 <= R(0)) return false;
  R Ps = m::sqrt(ps2);
  R phi = h * s;
  R tn = m::tan(phi), cs = m::cos(phi), sn = m::sin(phi);
  R den = R(1) - (z.Px / Ps) * tn;
  if (den <= R(0)) return false;
  R rho_X = R(1) / h + z.X;
  R Xf = rho_X * (R(1) / cs) / den - R(1) / h;                                    // (31a)
  R Pxf = z.Px * cs + Ps * sn;                                                    // (31b)
  R Yf = z.Y + (z.Py / Ps) * rho_X * tn / den;                                    // (31c)
  R Tf = z.T - ((R(1) / ref.beta0 + z.Pt) / Ps) * rho_X * tn / den + s / ref.beta0;  // (31e) + A5
  z.X = Xf; z.Px = Pxf; z.Y = Yf; z.T = Tf;
  return true;
}
// kick of H_K (30c) with the sector-bend potential (7): -dH_K/dX = -eta h (1 + hX) = -k0 (1 + hX)
template <class R> void bend_kick(Orbit<R>& z, R s, R h, R k0) { z.Px = z.Px - s * k0 * (R(1) + h * z.X); }

// quadrupole linear part: flow of H_qL (21b) over s for a FOCUSING (k1 > 0) quad, (22)-(24) P:288-319
template <class R> bool quad_linear_focusing(Orbit<R>& z, R s, R k1, const Reference<R>& ref) {
  R p2 = Ptot2(z, ref);
  if (p2 <= R(0)) return false;
  R P = m::sqrt(p2);                                                              // (22)
  R kap = m::sqrt(k1 / P);                                                        // (23)
  R ks = kap * s;
  R C = m::cos(ks), S = m::sin(ks), Ch = m::cosh(ks), Sh = m::sinh(ks);
  R Xi = z.X, Pxi = z.Px, Yi = z.Y, Pyi = z.Py;
  R Xf = Xi * C + s * (Pxi / P) * (S / ks);                                       // (24a)
  R Pxf = Pxi * C - kap * P * Xi * S;                                             // (24b)
  R Yf = Yi * Ch + s * (Pyi / P) * (Sh / ks);                                     // (24c)
  R Pyf = Pyi * Ch + kap * P * Yi * Sh;                                           // (24d)
  R S2 = m::sin(R(2) * ks), Sh2 = m::sinh(R(2) * ks);
  R curly = (s / R(4)) * ((Pxi * Pxi + Pyi * Pyi) / (P * P) + kap * kap * (Xi * Xi - Yi * Yi))
          + (s / R(4)) * ((Pxi / P) * (Pxi / P) - (kap * Xi) * (kap * Xi)) * (S2 / (R(2) * ks))
          + (s / R(4)) * ((Pyi / P) * (Pyi / P) + (kap * Yi) * (kap * Yi)) * (Sh2 / (R(2) * ks))
          - (ks / R(2)) * (Xi * (Pxi / P) * (S * S / ks) - Yi * (Pyi / P) * (Sh * Sh / ks));
  R Tf = z.T - (R(1) / P) * (R(1) / ref.beta0 + z.Pt) * curly;                    // (24e)
  z.X = Xf; z.Px = Pxf; z.Y = Yf; z.Py = Pyf; z.T = Tf;
  return true;
}
// A11 / P:321: a defocusing quad is the focusing one seen after a 90 degree rotation about s:
// (X, Y) -> (Y, -X), so that k1 (X^2 - Y^2) = |k1| (X'^2 - Y'^2).
template <class R> bool quad_linear(Orbit<R>& z, R s, R k1, const Reference<R>& ref) {
  if (k1 > R(0)) return quad_linear_focusing(z, s, k1, ref);
  Orbit<R> r;
  r.X = z.Y; r.Px = z.Py; r.Y = -z.X; r.Py = -z.Px; r.T = z.T; r.Pt = z.Pt;
  if (!quad_linear_focusing(r, s, -k1, ref)) return false;
  z.X = -r.Y; z.Px = -r.Py; z.Y = r.X; z.Py = r.Px; z.T = r.T;
  return true;
}
// quadrupole nonlinear part: flow of H_qNL (21c), (25) P:325-346
template <class R> bool quad_nonlinear(Orbit<R>& z, R s, const Reference<R>& ref) {
  R p2 = Ptot2(z, ref);
  R ps2 = Ps2(z, ref);                                                            // (26)
  if (ps2 <= R(0) || p2 <= R(0)) return false;
  R P = m::sqrt(p2), Ps = m::sqrt(ps2);
  R Pxi = z.Px, Pyi = z.Py;
  z.X = z.X + s * Pxi * (R(1) / Ps - R(1) / P);                                   // (25a)
  z.Y = z.Y + s * Pyi * (R(1) / Ps - R(1) / P);                                   // (25c)
  z.T = z.T - s * (R(1) / ref.beta0 + z.Pt) * (R(1) / Ps - (R(1) / P) * (Pxi * Pxi + Pyi * Pyi) / (R(2) * P * P))
        + s / ref.beta0;                                                          // (25e)
  return true;
}

// transverse field of a straight multipole in units of (B rho)_o, from (28) P:362 (A22):
//   B_y + i B_x = sum_m (b_m + i a_m) (X + iY)^(m-1),   m = 2..5  <->  kn[m-2], ks[m-2]
template <class R> void multipole_field(const R& X, const R& Y, const double* kn, const double* ks, R& bx, R& by) {
  R re = R(1), im = R(0);   // (X + iY)^(m-1), starting at m = 1
  bx = R(0); by = R(0);
  for (int mm = 2; mm <= 5; ++mm) {
    R nre = re * X - im * Y, nim = re * Y + im * X;
    re = nre; im = nim;
    R b = R(kn[mm - 2]), a = R(ks[mm - 2]);
    by = by + (b * re - a * im);
    bx = bx + (b * im + a * re);
  }
}
// kick of H_m over s: dPx = -s dH_m/dX = -s B_y, dPy = -s dH_m/dY = +s B_x   (28),(29a)
template <class R> void multipole_kick(Orbit<R>& z, R s, const double* kn, const double* ks) {
  R bx, by;
  multipole_field(z.X, z.Y, kn, ks, bx, by);
  z.Px = z.Px - s * by;
  z.Py = z.Py + s * bx;
}

// ----------------------------------------------------------------------------------------------
// spin
// ----------------------------------------------------------------------------------------------

// (6b) P:108.  b = B/(B rho)_o (A8); u-hat = (Px, Py, Ps)/P; gamma = gamma_o (1 + beta_o Pt) from (2).
// `lengthwise` = true  -> Omega of (6b) [1/m] for frame curvature h;
// `lengthwise` = false -> thin-lens limit L*Omega with b the integrated field (A10) (then h = 0).
template <class R> bool omega_tbmt(const Orbit<R>& z, R h, const Vec3<R>& b, double G, const Reference<R>& ref, Vec3<R>& Om) {
  R ps2 = Ps2(z, ref);
  R p2 = Ptot2(z, ref);
  if (ps2 <= R(0)) return false;
  R Ps = m::sqrt(ps2), P = m::sqrt(p2);
  R gamma = ref.gamma0 * (R(1) + ref.beta0 * z.Pt);
  Vec3<R> u = {z.Px / P, z.Py / P, Ps / P};
  R udotb = u.x * b.x + u.y * b.y + u.s * b.s;
  R a1 = R(1) + R(G) * gamma, a2 = R(G) * (gamma - R(1));
  R pre = -(R(1) + h * z.X) / Ps;
  Om.x = pre * (a1 * b.x - a2 * udotb * u.x);
  Om.y = pre * (a1 * b.y - a2 * udotb * u.y) + h;
  Om.s = pre * (a1 * b.s - a2 * udotb * u.s);
  return true;
}

template <class R> Quat<R> quat_mul(const Quat<R>& a, const Quat<R>& b) {   // Hamilton product a (x) b
  Quat<R> r;
  r.w = a.w * b.w - a.x * b.x - a.y * b.y - a.s * b.s;
  r.x = a.w * b.x + a.x * b.w + a.y * b.s - a.s * b.y;
  r.y = a.w * b.y - a.x * b.s + a.y * b.w + a.s * b.x;
  r.s = a.w * b.s + a.x * b.y - a.y * b.x + a.s * b.w;
  return r;
}
// A6: rotation by angle |w| about w  ->  q = (cos(|w|/2), sin(|w|/2) w/|w|)
template <class R> Quat<R> quat_from_rotvec(const Vec3<R>& w) {
  R th2 = w.x * w.x + w.y * w.y + w.s * w.s;
  if (th2 == R(0)) return Quat<R>{R(1), R(0), R(0), R(0)};
  R th = m::sqrt(th2);
  R c = m::cos(th / R(2)), sn = m::sin(th / R(2));
  return Quat<R>{c, sn * w.x / th, sn * w.y / th, sn * w.s / th};
}
// S' = q S q*  (A6)
template <class R> Vec3<R> quat_rotate(const Quat<R>& q, const Vec3<R>& S) {
  Quat<R> p = {R(0), S.x, S.y, S.s};
  Quat<R> qc = {q.w, -q.x, -q.y, -q.s};
  Quat<R> r = quat_mul(quat_mul(q, p), qc);
  return Vec3<R>{r.x, r.y, r.s};
}

// trapezoid-weighted edge products at d step sizes + Romberg table (39b); A2, A4, A6, A7.
// Om[0..N] are the slice-edge precession vectors, ds the slice length.  Returns the normalised
// Romberg limit Q_{d-1,d-1}.
template <class R> Quat<R> romberg_quaternion(const std::vector<Vec3<R>>& Om, int N, R ds, int d) {
  std::vector<std::vector<Quat<R>>> Q(d, std::vector<Quat<R>>(d));
  for (int k = 0; k < d; ++k) {                       // Q_{0,k} = Q(h/2^k), k = 0 coarsest (38)
    int stride = 1 << (d - 1 - k);
    R step = R(stride) * ds;
    Quat<R> acc = {R(1), R(0), R(0), R(0)};
    for (int i = 0; i <= N; i += stride) {
      R wgt = (i == 0 || i == N) ? R(1) / R(2) : R(1);   // half step at first and last edge
      Vec3<R> w = {wgt * step * Om[i].x, wgt * step * Om[i].y, wgt * step * Om[i].s};
      acc = quat_mul(quat_from_rotvec(w), acc);          // later rotations on the left (37b)
    }
    Q[0][k] = acc;
  }
  R four = R(1);
  for (int j = 0; j + 1 < d; ++j) {                   // (39b)
    four = four * R(4);                                // 4^(j+1)
    for (int k = j + 1; k < d; ++k) {
      Q[j + 1][k].w = (four * Q[j][k].w - Q[j][k - 1].w) / (four - R(1));
      Q[j + 1][k].x = (four * Q[j][k].x - Q[j][k - 1].x) / (four - R(1));
      Q[j + 1][k].y = (four * Q[j][k].y - Q[j][k - 1].y) / (four - R(1));
      Q[j + 1][k].s = (four * Q[j][k].s - Q[j][k - 1].s) / (four - R(1));
    }
  }
  Quat<R> q = Q[d - 1][d - 1];
  R n = m::sqrt(q.w * q.w + q.x * q.x + q.y * q.y + q.s * q.s);   // "We normalise ... at the end of each element" P:546
  return Quat<R>{q.w / n, q.x / n, q.y / n, q.s / n};
}

// ----------------------------------------------------------------------------------------------
// one element (orbit through the element recording Omega at every slice edge, then spin)
// ----------------------------------------------------------------------------------------------
template <class R> struct Particle { Orbit<R> z; Vec3<R> S; };

template <class R> Vec3<R> element_field(const Element& e, const Orbit<R>& z) {
  if (e.type == SBEND) return Vec3<R>{R(0), R(e.k0), R(0)};
  R bx, by;
  multipole_field(z.X, z.Y, e.kn, e.ks, bx, by);
  return Vec3<R>{bx, by, R(0)};
}

// ---- rectangular bend (section 3.2).  e.k0 = b_1/(B rho)_o = 1/rho_b (12); e.kn[0], e.kn[1] = phi_entr, phi_exit ----
// body (13) P:170-186 over the length s along the magnet axis; coordinates internal to the magnet (Cartesian)
template <class R> bool rbend_body(Orbit<R>& z, R s, R k0, const Reference<R>& ref) {
  R Pa2 = R(1) + R(2) * z.Pt / ref.beta0 + z.Pt * z.Pt - z.Py * z.Py;             // (8)
  if (Pa2 <= R(0)) return false;
  R Pa = m::sqrt(Pa2);
  R Pxf = z.Px - s * k0;                                                          // (13b)
  R a2 = Pa2 - z.Px * z.Px, f2 = Pa2 - Pxf * Pxf;
  if (a2 <= R(0) || f2 <= R(0)) return false;
  R dasin = m::asin(z.Px / Pa) - m::asin(Pxf / Pa);
  z.X = z.X + (m::sqrt(f2) - m::sqrt(a2)) / k0;                                   // (13a)
  z.Y = z.Y + z.Py * dasin / k0;                                                  // (13c)
  z.T = z.T - (R(1) / ref.beta0 + z.Pt) * dasin / k0;                             // (13e): no +s/beta_o, see (19)
  z.Px = Pxf;
  return true;
}
// thin-fringe orbit map (15) P:204-224, sign = +1 entrance, -1 exit; "P_c" of (15e) read as P_s (A1)
template <class R> bool rbend_fringe(Orbit<R>& z, R sign, R k0, const Reference<R>& ref) {
  R ps2 = Ps2(z, ref);
  if (ps2 <= R(0)) return false;
  R Ps = m::sqrt(ps2);
  R xp = z.Px / Ps, yp = z.Py / Ps, b = sign * k0;
  R d = R(1) + yp * yp;
  R arg = R(1) + b * xp * yp / d * R(2) * z.Y;
  if (arg <= R(0)) return false;
  R Yf = R(2) * z.Y / (R(1) + m::sqrt(arg));                                      // (15c)
  z.X = z.X + b / (R(2) * Ps) * ((R(1) + xp * xp) / d - R(2) * xp * xp * yp * yp / (d * d)) * Yf * Yf;   // (15a)
  z.Py = z.Py - b * xp / d * Yf;                                                  // (15d)
  z.T = z.T - b * (R(1) / ref.beta0 + z.Pt) * xp / (R(2) * ps2) * (R(1) - yp * yp) / (d * d) * Yf * Yf;   // (15e)
  z.Y = Yf;
  return true;
}
// dynamic rotation by phi about y-hat (16)(17) P:228-248 ("P_z" of (17c) read as P_s, A1; the sign of (17e)
// is the one Hamilton's equations of (16) give, dT/dphi = dH/dPt = -X (1/beta_o + Pt)/P_s, as in (31e): A5),
// and the passive rotation of the spin components into the new frame
template <class R> bool rbend_rotate(Particle<R>& p, R phi, const Reference<R>& ref) {
  Orbit<R>& z = p.z;
  R ps2 = Ps2(z, ref);
  if (ps2 <= R(0)) return false;
  R Ps = m::sqrt(ps2);
  R c = m::cos(phi), sn = m::sin(phi), t = sn / c;
  R den = R(1) - z.Px / Ps * t;
  if (den <= R(0)) return false;
  R q = z.X * t / den;
  z.Y = z.Y + z.Py / Ps * q;                                                      // (17c)
  z.T = z.T - (R(1) / ref.beta0 + z.Pt) / Ps * q;                                 // (17e), sign per A5
  z.X = z.X / (c * den);                                                          // (17a)
  z.Px = z.Px * c + Ps * sn;                                                      // (17b)
  R Sx = p.S.x * c + p.S.s * sn, Ss = -p.S.x * sn + p.S.s * c;                    // same rotation as (Px, Ps)
  p.S.x = Sx; p.S.s = Ss;
  return true;
}
// fringe spin kick of a rectangular bend (42) P:567 = (41) with m = 1 plus the x-hat term; DESIGN.md reading
// R10: the printed x-hat term lacks a length -- T-BMT in the fringe's longitudinal field gives
// (+-b_1/(B rho)_o) G(gamma-1) P_x Y x-hat.
template <class R> Vec3<R> rbend_fringe_rotvec(const Orbit<R>& z, R sign, R k0, double G, const Reference<R>& ref) {
  R gamma = ref.gamma0 * (R(1) + ref.beta0 * z.Pt);
  R b = sign * k0;
  return Vec3<R>{b * R(G) * (gamma - R(1)) * z.Px * z.Y, R(0), -b * R(1.0 + G) * z.Y};
}

// ---- solenoid (section 3.7).  e.k0 holds b_0/(B rho)_o, so eta = e.k0/2 (35); (e/p_o) A = eta (-Y, X) (32) ----
// kinetic transverse momenta (36): canonical minus `frac` times the vector potential
template <class R> Orbit<R> solenoid_kinetic(const Orbit<R>& z, R eta, R frac) {
  Orbit<R> k = z;
  k.Px = z.Px + frac * eta * z.Y;
  k.Py = z.Py - frac * eta * z.X;
  return k;
}
// exact flow of H_sol (33) over s: z <- R2 R1 z on (X, Px, Y, Py), T by (34c); kappa = eta / Ps^i
template <class R> bool solenoid_body(Orbit<R>& z, R s, R eta, const Reference<R>& ref) {
  R ps2 = Ps2(solenoid_kinetic(z, eta, R(1)), ref);                  // the square root of (33)
  if (ps2 <= R(0)) return false;
  R Ps = m::sqrt(ps2);
  R kap = eta / Ps;
  R c = m::cos(kap * s), sn = m::sin(kap * s);
  R X1 = c * z.X + sn / eta * z.Px, Px1 = -eta * sn * z.X + c * z.Px;   // (34a)
  R Y1 = c * z.Y + sn / eta * z.Py, Py1 = -eta * sn * z.Y + c * z.Py;
  z.X = c * X1 + sn * Y1;    z.Px = c * Px1 + sn * Py1;                 // (34b)
  z.Y = -sn * X1 + c * Y1;   z.Py = -sn * Px1 + c * Py1;
  z.T = z.T - (R(1) / ref.beta0 + z.Pt) * s / Ps + s / ref.beta0;       // (34c)
  return true;
}
// Omega (6b) in the body: B/(B rho)_o = (0, 0, 2 eta), u-hat from the KINETIC momentum (36)
template <class R> bool solenoid_omega(const Orbit<R>& z, R eta, double G, const Reference<R>& ref, Vec3<R>& Om) {
  return omega_tbmt(solenoid_kinetic(z, eta, R(1)), R(0), Vec3<R>{R(0), R(0), R(2) * eta}, G, ref, Om);
}
// thin-pancake fringe spin kick (40) P:553: sign = +1 entrance, -1 exit; kinetic momentum and Ps with A/2
template <class R> bool solenoid_fringe_rotvec(const Orbit<R>& z, R eta, R sign, double G, const Reference<R>& ref, Vec3<R>& w) {
  Orbit<R> k = solenoid_kinetic(z, eta, R(1) / R(2));
  R ps2 = Ps2(k, ref);
  if (ps2 <= R(0)) return false;
  R Ps = m::sqrt(ps2), P2 = Ptot2(z, ref);
  R gamma = ref.gamma0 * (R(1) + ref.beta0 * z.Pt);
  R a1 = R(1) + R(G) * gamma, a2 = R(G) * (gamma - R(1));
  R proj = (z.X * k.Px + z.Y * k.Py) / P2;
  R pre = sign * eta / Ps;
  w.x = pre * (a1 * z.X - a2 * proj * k.Px);
  w.y = pre * (a1 * z.Y - a2 * proj * k.Py);
  w.s = pre * (-a2 * proj * Ps);
  return true;
}

// one second-order orbital slice of a thick magnet of the given type with the given split (A16)
template <class R> bool orbit_slice2(Orbit<R>& z, const Element& e, R ds, int split, const Reference<R>& ref) {
  if (e.type == SBEND) {
    if (split == SPLIT_DRIFT_KICK) {                                 // TEAPOT (30),(31), composed as (27)
      if (!curved_drift(z, ds / R(2), R(e.h), ref)) return false;
      bend_kick(z, ds, R(e.h), R(e.k0));
      return curved_drift(z, ds / R(2), R(e.h), ref);
    }
    return sbend_exact(z, ds, R(e.h), R(e.k0), ref);                 // bend-kick and matrix-kick: (10)
  }
  if (e.type == QUAD && split == SPLIT_MATRIX_KICK) {                // (27)
    if (!quad_linear(z, ds / R(2), R(e.kn[0]), ref)) return false;
    if (!quad_nonlinear(z, ds, ref)) return false;
    return quad_linear(z, ds / R(2), R(e.kn[0]), ref);
  }
  // drift-kick (29), composed as (27): quads outside matrix-kick, thick multipoles always
  if (!drift(z, ds / R(2), ref)) return false;
  multipole_kick(z, ds, e.kn, e.ks);
  return drift(z, ds / R(2), ref);
}

// is the slice map of this element exact under this split?  (an exact flow needs no composition)
inline bool slice_is_exact(const Element& e, int base_split) { return e.type == SBEND && base_split != SPLIT_DRIFT_KICK; }

// one orbital slice: second order (27), or the fourth-order symmetric composition
//   S4(ds) = S2(x1 ds) S2(x0 ds) S2(x1 ds),  x1 = 1/(2 - 2^(1/3)),  x0 = 1 - 2 x1 = -2^(1/3) x1
// (the triple-jump composition of refs [62, 23]: x0 + 2 x1 = 1 keeps the length, x0^3 + 2 x1^3 = 0 cancels
// the third-order error term of the symmetric S2).  The middle step runs backwards (x0 < 0).
template <class R> bool orbit_slice(Orbit<R>& z, const Element& e, R ds, int split, const Reference<R>& ref) {
  const int base = split % 3;
  if (split < 3 || slice_is_exact(e, base)) return orbit_slice2(z, e, ds, base, ref);
  R cbrt2 = R(1.2599210498948732);                                    // 2^(1/3), polished by Newton to the precision of R
  for (int it = 0; it < 3; ++it) cbrt2 = cbrt2 - (cbrt2 * cbrt2 * cbrt2 - R(2)) / (R(3) * cbrt2 * cbrt2);
  const R x1 = R(1) / (R(2) - cbrt2);
  const R x0 = R(1) - R(2) * x1;
  if (!orbit_slice2(z, e, x1 * ds, base, ref)) return false;
  if (!orbit_slice2(z, e, x0 * ds, base, ref)) return false;
  return orbit_slice2(z, e, x1 * ds, base, ref);
}

// Piece-wise constant spin precession (37) P:470-482 with Omega taken in the MIDDLE of each slice; the two
// orderings the paper names in the caption of Fig. 14:
//   PWC_HALF_SLICE (depth  0)  "DKDSDKD": half a slice map, spin rotation R(ds Omega), half a slice map --
//                              for any split (the half map is the split's own second-/fourth-order map over ds/2)
//   PWC_DKSKD      (depth -1)  "DKSKD": half drift, half kick, spin rotation, half kick, half drift -- for the
//                              elements integrated by a drift-kick map (29) or (30)(31); others as PWC_HALF_SLICE
// The spin is rotated slice by slice, later rotations on the left (37b).  DESIGN.md reading R7.
enum { PWC_HALF_SLICE = 0, PWC_DKSKD = -1 };

template <class R> bool track_thick_pwc(Particle<R>& p, const Element& e, const Reference<R>& ref, double G,
                                        int split, int N, R ds, int kind) {
  const int base = split % 3;
  const bool drift_kick_map = (e.type == SBEND) ? (base == SPLIT_DRIFT_KICK)
                                                : !(e.type == QUAD && base == SPLIT_MATRIX_KICK);
  for (int i = 0; i < N; ++i) {
    Vec3<R> Om;
    if (kind == PWC_DKSKD && drift_kick_map) {
      const R h2 = ds / R(2);
      if (e.type == SBEND) {
        if (!curved_drift(p.z, h2, R(e.h), ref)) return false;
        bend_kick(p.z, h2, R(e.h), R(e.k0));
      } else {
        if (!drift(p.z, h2, ref)) return false;
        multipole_kick(p.z, h2, e.kn, e.ks);
      }
      if (!omega_tbmt(p.z, R(e.h), element_field(e, p.z), G, ref, Om)) return false;
      p.S = quat_rotate(quat_from_rotvec(Vec3<R>{ds * Om.x, ds * Om.y, ds * Om.s}), p.S);
      if (e.type == SBEND) {
        bend_kick(p.z, h2, R(e.h), R(e.k0));
        if (!curved_drift(p.z, h2, R(e.h), ref)) return false;
      } else {
        multipole_kick(p.z, h2, e.kn, e.ks);
        if (!drift(p.z, h2, ref)) return false;
      }
    } else {
      if (!orbit_slice(p.z, e, ds / R(2), split, ref)) return false;
      if (!omega_tbmt(p.z, R(e.h), element_field(e, p.z), G, ref, Om)) return false;
      p.S = quat_rotate(quat_from_rotvec(Vec3<R>{ds * Om.x, ds * Om.y, ds * Om.s}), p.S);
      if (!orbit_slice(p.z, e, ds / R(2), split, ref)) return false;
    }
  }
  return true;
}

// returns false if the particle is lost inside this element (A15): p is then restored to its
// value at the element entrance.
template <class R> bool track_element(Particle<R>& p, const Element& e, Reference<R>& ref, double G,
                                      int split, int n_slices, int depth, double circumference) {
  Particle<R> entrance = p;
  bool ok = true;
  switch (e.type) {
    case MARKER: break;
    case FRINGE: {
      // (41) P:561: thin fringe of a 2m-pole, lowest order: rotation about s-hat by
      //   omega = -(+-)(1+G) [b_m r^m sin(m phi) + a_m r^m cos(m phi)]/(m (B rho)_o),  (X+iY)^m = r^m e^(i m phi),
      // + on entering (e.sign = +1), - on leaving (e.sign = -1).  m = 1 is the dipole term b_1 = k0;
      // kn[m-2], ks[m-2] hold m = 2..5 in the convention of (28).  The orbit is not touched (reading R8).
      R re = p.z.X, im = p.z.Y;                                      // (X + iY)^m, m = 1
      R psi = R(e.k0) * im;
      for (int m = 2; m <= 5; ++m) {
        R nre = re * p.z.X - im * p.z.Y, nim = re * p.z.Y + im * p.z.X;
        re = nre; im = nim;
        psi = psi + (R(e.kn[m - 2]) * im + R(e.ks[m - 2]) * re) / R(m);
      }
      R om = -R(e.sign) * R(1.0 + G) * psi;
      p.S = quat_rotate(quat_from_rotvec(Vec3<R>{R(0), R(0), om}), p.S);
      break;
    }
    case DRIFT: ok = drift(p.z, R(e.L), ref); break;                 // one exact step, no field, no spin (A17)
    case SBEND: case QUAD: case MULTIPOLE: {
      int N = n_slices * e.slice_mult;
      R ds = R(e.L) / R(N);
      if (depth <= 0) {                                              // comparison integrators of section 4.1
        ok = track_thick_pwc(p, e, ref, G, split, N, ds, depth);
        break;
      }
      std::vector<Vec3<R>> Om(N + 1);
      ok = omega_tbmt(p.z, R(e.h), element_field(e, p.z), G, ref, Om[0]);
      for (int i = 1; ok && i <= N; ++i) {
        ok = orbit_slice(p.z, e, ds, split, ref);
        if (ok) ok = omega_tbmt(p.z, R(e.h), element_field(e, p.z), G, ref, Om[i]);
      }
      if (ok) p.S = quat_rotate(romberg_quaternion(Om, N, ds, depth), p.S);
      break;
    }
    case RBEND: {
      // rotate into the magnet frame by phi_entr, entrance fringe (spin kick (42), orbit map (15)),
      // body (13) in N slices with the edge scheme (Cartesian frame: h = 0 in (6b)), exit fringe, offset (18),
      // rotate out by -phi_exit, and T_o of (19) so that T stays a deviation.
      const R k0 = R(e.k0), phi_in = R(e.kn[0]), phi_out = R(e.kn[1]);
      int N = n_slices * e.slice_mult;
      R ds = R(e.L) / R(N);
      const Vec3<R> bfield = {R(0), k0, R(0)};
      ok = rbend_rotate(p, phi_in, ref);
      if (!ok) break;
      p.S = quat_rotate(quat_from_rotvec(rbend_fringe_rotvec(p.z, R(1), k0, G, ref)), p.S);
      ok = rbend_fringe(p.z, R(1), k0, ref);
      if (!ok) break;
      if (depth <= 0) {
        for (int i = 0; ok && i < N; ++i) {
          Vec3<R> Om;
          ok = rbend_body(p.z, ds / R(2), k0, ref) && omega_tbmt(p.z, R(0), bfield, G, ref, Om);
          if (!ok) break;
          p.S = quat_rotate(quat_from_rotvec(Vec3<R>{ds * Om.x, ds * Om.y, ds * Om.s}), p.S);
          ok = rbend_body(p.z, ds / R(2), k0, ref);
        }
      } else {
        std::vector<Vec3<R>> Om(N + 1);
        ok = omega_tbmt(p.z, R(0), bfield, G, ref, Om[0]);
        for (int i = 1; ok && i <= N; ++i) ok = rbend_body(p.z, ds, k0, ref) && omega_tbmt(p.z, R(0), bfield, G, ref, Om[i]);
        if (ok) p.S = quat_rotate(romberg_quaternion(Om, N, ds, depth), p.S);
      }
      if (!ok) break;
      ok = rbend_fringe(p.z, R(-1), k0, ref);
      if (!ok) break;
      p.S = quat_rotate(quat_from_rotvec(rbend_fringe_rotvec(p.z, R(-1), k0, G, ref)), p.S);
      p.z.X = p.z.X - (m::cos(phi_out) - m::cos(phi_in)) / k0;                  // (18): L/(sin - sin) = rho_b
      ok = rbend_rotate(p, -phi_out, ref);
      p.z.T = p.z.T + (phi_in - phi_out) / (k0 * ref.beta0);                     // (19): T - T_o, L_arc = rho_b (phi_entr - phi_exit)
      break;
    }
    case SOLENOID: {   // entrance fringe kick (40), body (34) in N exact slices with the edge scheme (38)(39), exit kick
      const R eta = R(e.k0) / R(2);
      int N = n_slices * e.slice_mult;
      R ds = R(e.L) / R(N);
      Vec3<R> w;
      ok = solenoid_fringe_rotvec(p.z, eta, R(1), G, ref, w);                 // entrance: +
      if (!ok) break;
      p.S = quat_rotate(quat_from_rotvec(w), p.S);
      if (depth <= 0) {                                              // mid-slice PWC (37): half map, rotation, half map
        for (int i = 0; ok && i < N; ++i) {
          Vec3<R> Om;
          ok = solenoid_body(p.z, ds / R(2), eta, ref) && solenoid_omega(p.z, eta, G, ref, Om);
          if (!ok) break;
          p.S = quat_rotate(quat_from_rotvec(Vec3<R>{ds * Om.x, ds * Om.y, ds * Om.s}), p.S);
          ok = solenoid_body(p.z, ds / R(2), eta, ref);
        }
      } else {
        std::vector<Vec3<R>> Om(N + 1);
        ok = solenoid_omega(p.z, eta, G, ref, Om[0]);
        for (int i = 1; ok && i <= N; ++i) ok = solenoid_body(p.z, ds, eta, ref) && solenoid_omega(p.z, eta, G, ref, Om[i]);
        if (ok) p.S = quat_rotate(romberg_quaternion(Om, N, ds, depth), p.S);
      }
      if (!ok) break;
      ok = solenoid_fringe_rotvec(p.z, eta, R(-1), G, ref, w);                // exit: -
      if (ok) p.S = quat_rotate(quat_from_rotvec(w), p.S);
      break;
    }
    case THINMULT: {                                                 // A10: half kick, spin, half kick
      multipole_kick(p.z, R(1) / R(2), e.kn, e.ks);
      Vec3<R> w;
      ok = omega_tbmt(p.z, R(0), element_field(e, p.z), G, ref, w);
      if (ok) {
        p.S = quat_rotate(quat_from_rotvec(w), p.S);
        multipole_kick(p.z, R(1) / R(2), e.kn, e.ks);
      }
      break;
    }
    case RFCAV: {                                                    // A12, A13 (not in the paper)
      R two_pi = R(2) * m::pi_of(R(0));
      R krf = two_pi * R(e.harmonic) * ref.beta0 / R(circumference);
      R E = ref.E0 + ref.p0c * p.z.Pt;                                // particle energy from (2)
      E = E + R(e.volt_eV) * m::sin(R(e.phi_s) + R(e.sign) * krf * p.z.T);
      R dEs = R(e.volt_eV) * m::sin(R(e.phi_s));                      // synchronous gain per passage
      Reference<R> nref;
      nref.set(ref.E0 + dEs, ref.mass);
      R scale = ref.p0c / nref.p0c;
      p.z.Px = p.z.Px * scale;
      p.z.Py = p.z.Py * scale;
      p.z.Pt = (E - nref.E0) / nref.p0c;
      ref = nref;
      break;                                                          // spin: identity (A12)
    }
    case SNAKE: {                                                    // A14
      R half = R(e.snake_mu) / R(2);
      R sn = m::sin(half);
      Quat<R> q = {m::cos(half), sn * m::sin(R(e.snake_phi)), R(0), sn * m::cos(R(e.snake_phi))};
      p.S = quat_rotate(q, p.S);
      break;
    }
    default: ok = false;
  }
  if (!ok) p = entrance;
  return ok;
}

inline double ring_circumference(const Element* el, size_t n) {
  double C = 0;
  for (size_t i = 0; i < n; ++i)     // design path length: L, except the arc rho_b (phi_entr - phi_exit) of a rectangular bend (19)
    C += el[i].type == RBEND ? (el[i].kn[0] - el[i].kn[1]) / el[i].k0 : el[i].L;
  return C;
}

}  // namespace orc
