// track_kernel.cuh -- T1: the persistent turn-loop spin-orbit tracking kernel (sm_100a, fp64).
//
// One thread per particle.  The nine state doubles are loaded once, live in registers for
// all turns and all elements, and are stored once.  The slice-edge precession vectors are never
// stored: each edge's Omega is folded on the fly into DEPTH running quaternion products (one per
// Romberg level), which replaces the paper's global-memory Omega arrays and its separate orbit /
// spin / update kernels.  The element table lives in shared memory.
//
// The orbit maps are algebraically equal to the paper's formulas (10), (24), (25), (29), (31) but
// are written in cancellation-free form: the literal forms subtract O(1)
// quantities to get O(1e-3) results, which costs ~1e-11 of the bunch scale per slice in fp64.
#pragma once
#include <cstdint>

namespace gst {

enum : int { K_DRIFT = 0, K_SBEND = 1, K_QUAD = 2, K_MULT = 3, K_THIN = 4, K_RF = 5, K_SNAKE = 6, K_MARKER = 7 };
enum : int { SPLIT_DK = 0, SPLIT_BK = 1, SPLIT_MK = 2 };

// Unique-element record, derived on the host for one value of n_slices (a0).
struct __align__(16) DevElem {
  int type;
  int N;          // slices of this element (thick), else 1
  int order;      // highest multipole order present (2..5), 0 if none
  int pad;
  double L;       // length
  double ds;      // L / N
  double h, k0;
  // sector bend, exact map over ds
  double cm;      // 1 - cos(h ds) = 2 sin^2(h ds/2)
  double sn;      // sin(h ds)
  double ck;      // (1 - cos(h ds))/k0
  double sk;      // sin(h ds)/k0
  double ome;     // 1 - eta
  double inv_eta; // h/k0
  double inv_h;   // 1/h
  // sector bend, TEAPOT half drift over ds/2 (phi = h ds/2)
  double hc, hs, ht;   // cos phi, sin phi, tan phi
  double hcm;          // 1 - cos phi
  double r_secm1;      // rho (sec phi - 1)
  double r_tan;        // rho tan phi
  double r_tanmphi;    // rho (tan phi - phi)
  double hsec;         // sec phi
  double kn[4], ks[4]; // multipole strengths (28); thin: integrated
  // cavity
  double volt, krf_over_beta, phi_s, sign, dEs;
  // snake quaternion (w, x, y, s)
  double qw, qx, qy, qs;
};

struct TrackArgs {
  double* p[9];
  uint8_t* lost;
  const DevElem* tab;      // unique elements (global memory)
  const uint16_t* seq;     // element sequence, indices into tab
  int n_unique;
  int n_seq;
  int use_smem_seq;
  long long n;
  long long n_turns;
  double E0, mass, G;
};

struct Quat { double w, x, y, s; };

// reference-particle and per-particle constants that change only when Pt or E0 changes
struct Ref {
  double E0, mass, p0c, beta0, gamma0, ibeta0, ibg2;  // ibg2 = 1/(beta0 gamma0)^2 = 1/beta0^2 - 1
};
struct PCon {
  double e0;    // P^2 - 1 = 2 Pt/beta0 + Pt^2                      (22)
  double P, iP; // total momentum / p0 and its reciprocal
  double a1;    // 1 + G gamma                                       (6b)
  double a2p;   // G (gamma - 1) / P^2
  double tA;    // 2 Pt/(beta0 gamma0)^2 + Pt^2/beta0   (time-of-flight numerator, see drift())
  double tq;    // 1/beta0 - (1/beta0 + Pt)/P, cancellation-free
  double ibpt;  // 1/beta0 + Pt
};

__device__ __forceinline__ void ref_set(Ref& r, double E0, double mass) {
  r.E0 = E0; r.mass = mass;
  r.gamma0 = E0 / mass;
  r.p0c = sqrt((E0 - mass) * (E0 + mass));
  r.beta0 = r.p0c / E0;
  r.ibeta0 = E0 / r.p0c;
  r.ibg2 = (mass / r.p0c) * (mass / r.p0c);
}

__device__ __forceinline__ void pcon_set(PCon& c, double Pt, const Ref& r, double G) {
  c.e0 = Pt * fma(2.0, r.ibeta0, Pt);
  c.P = sqrt(1.0 + c.e0);
  c.iP = 1.0 / c.P;
  double gamma = r.gamma0 * fma(r.beta0, Pt, 1.0);
  c.a1 = fma(G, gamma, 1.0);
  c.a2p = G * (gamma - 1.0) * c.iP * c.iP;
  c.tA = Pt * fma(2.0, r.ibg2, Pt * r.ibeta0);
  c.ibpt = r.ibeta0 + Pt;
  // (P-1)/beta0 - Pt = [tA - Pt (P-1)]/(P+1),  P-1 = e0/(P+1)
  double ip1 = 1.0 / (c.P + 1.0);
  c.tq = (c.tA - Pt * c.e0 * ip1) * ip1 * c.iP;
}

// ---------------------------------------------------------------------------------------------
// quaternions (a10, a11)
// ---------------------------------------------------------------------------------------------
// q = (cos(th/2), sin(th/2) w/th) for rotation vector w: both factors are even in th, so for
// th^2/4 <= 0.5 they are polynomials in th^2 -- no sqrt, no division, no sincos ("low-order
// polynomials", here taken to full double precision).
__device__ __forceinline__ Quat quat_from_rotvec(double wx, double wy, double ws) {
  double t2 = fma(wx, wx, fma(wy, wy, ws * ws));
  double u = 0.25 * t2;   // (th/2)^2
  Quat q;
  if (u <= 0.5) {
    // cos x = sum (-u)^k/(2k)!,  sin x / x = sum (-u)^k/(2k+1)!,  k = 0..9  (remainder < 4e-20)
    double c = -1.0 / 6402373705728000.0;        // 1/18!
    double s = -1.0 / 121645100408832000.0;      // 1/19!
    c = fma(c, u, 1.0 / 20922789888000.0);       // 16!
    s = fma(s, u, 1.0 / 355687428096000.0);      // 17!
    c = fma(c, u, -1.0 / 87178291200.0);         // 14!
    s = fma(s, u, -1.0 / 1307674368000.0);       // 15!
    c = fma(c, u, 1.0 / 479001600.0);            // 12!
    s = fma(s, u, 1.0 / 6227020800.0);           // 13!
    c = fma(c, u, -1.0 / 3628800.0);             // 10!
    s = fma(s, u, -1.0 / 39916800.0);            // 11!
    c = fma(c, u, 1.0 / 40320.0);                // 8!
    s = fma(s, u, 1.0 / 362880.0);               // 9!
    c = fma(c, u, -1.0 / 720.0);                 // 6!
    s = fma(s, u, -1.0 / 5040.0);                // 7!
    c = fma(c, u, 1.0 / 24.0);
    s = fma(s, u, 1.0 / 120.0);
    c = fma(c, u, -0.5);
    s = fma(s, u, -1.0 / 6.0);
    c = fma(c, u, 1.0);
    s = fma(s, u, 1.0);
    s *= 0.5;                                    // sin(th/2)/th = (1/2) sin(x)/x
    q.w = c; q.x = s * wx; q.y = s * wy; q.s = s * ws;
  } else {
    double th = sqrt(t2), sn, cs;
    sincos(0.5 * th, &sn, &cs);
    double f = sn / th;
    q.w = cs; q.x = f * wx; q.y = f * wy; q.s = f * ws;
  }
  return q;
}
// a (x) b
__device__ __forceinline__ Quat quat_mul(const Quat& a, const Quat& b) {
  Quat r;
  r.w = fma(a.w, b.w, -fma(a.x, b.x, fma(a.y, b.y, a.s * b.s)));
  r.x = fma(a.w, b.x, fma(a.x, b.w, fma(a.y, b.s, -a.s * b.y)));
  r.y = fma(a.w, b.y, fma(a.y, b.w, fma(a.s, b.x, -a.x * b.s)));
  r.s = fma(a.w, b.s, fma(a.s, b.w, fma(a.x, b.y, -a.y * b.x)));
  return r;
}
// same axis, twice the angle
__device__ __forceinline__ Quat quat_double(const Quat& q) {
  double c2 = 2.0 * q.w;
  return Quat{fma(c2, q.w, -1.0), c2 * q.x, c2 * q.y, c2 * q.s};
}
// S <- q S q*  for unit q:  S + 2 w (v x S) + 2 v x (v x S)
__device__ __forceinline__ void quat_rotate(const Quat& q, double& Sx, double& Sy, double& Ss) {
  double tx = 2.0 * fma(q.y, Ss, -q.s * Sy);
  double ty = 2.0 * fma(q.s, Sx, -q.x * Ss);
  double ts = 2.0 * fma(q.x, Sy, -q.y * Sx);
  Sx += fma(q.w, tx, fma(q.y, ts, -q.s * ty));
  Sy += fma(q.w, ty, fma(q.s, tx, -q.x * ts));
  Ss += fma(q.w, ts, fma(q.x, ty, -q.y * tx));
}

// Running products of the DEPTH trapezoid levels.  Level l has stride 2^l (l = 0 is the
// finest); edge i belongs to it when 2^l | i.  The rotation for weight 2^l is obtained from the
// finest one by angle doubling instead of a new sincos.
template <int DEPTH> struct SpinAcc {
  Quat Q[DEPTH];
  __device__ __forceinline__ void reset() {
#pragma unroll
    for (int l = 0; l < DEPTH; ++l) Q[l] = Quat{1.0, 0.0, 0.0, 0.0};
  }
  // (wx,wy,ws) = weight * ds * Omega_i with weight 1/2 at the two ends of the element
  __device__ __forceinline__ void edge(int i, double wx, double wy, double ws) {
    Quat q = quat_from_rotvec(wx, wy, ws);
    Q[0] = quat_mul(q, Q[0]);
#pragma unroll
    for (int l = 1; l < DEPTH; ++l) {
      if ((i & ((1 << l) - 1)) == 0) {
        q = quat_double(q);
        Q[l] = quat_mul(q, Q[l]);
      }
    }
  }
  // Romberg limit (39b) P:542 of the level products, normalised, applied to S (a11)
  __device__ __forceinline__ void finish(double& Sx, double& Sy, double& Ss) {
    // Q[l] holds step h*2^l, i.e. column entry k = DEPTH-1-l of (38).  Run the table in place.
    double f = 1.0;
#pragma unroll
    for (int j = 1; j < DEPTH; ++j) {
      f *= 4.0;
      const double c1 = f / (f - 1.0), c2 = 1.0 / (f - 1.0);
#pragma unroll
      for (int l = 0; l + j < DEPTH; ++l) {        // finer entry Q[l], coarser Q[l+1]
        Q[l].w = fma(c1, Q[l].w, -c2 * Q[l + 1].w);
        Q[l].x = fma(c1, Q[l].x, -c2 * Q[l + 1].x);
        Q[l].y = fma(c1, Q[l].y, -c2 * Q[l + 1].y);
        Q[l].s = fma(c1, Q[l].s, -c2 * Q[l + 1].s);
      }
    }
    Quat q = Q[0];
    double n2 = fma(q.w, q.w, fma(q.x, q.x, fma(q.y, q.y, q.s * q.s)));
    double rn = rsqrt(n2);
    q.w *= rn; q.x *= rn; q.y *= rn; q.s *= rn;
    quat_rotate(q, Sx, Sy, Ss);
  }
};

// ---------------------------------------------------------------------------------------------
// particle state in registers
// ---------------------------------------------------------------------------------------------
struct State {
  double X, Px, Y, Py, T, Pt, Sx, Sy, Ss;
};

// a3: exact drift (29b).  T' = 1/beta0 - (1/beta0+Pt)/Ps is evaluated as
// [(Ps-1)/beta0 - Pt]/Ps with Ps-1 = (Ps^2-1)/(Ps+1) and the O(Pt) terms combined analytically.
__device__ __forceinline__ bool drift(State& z, double L, const PCon& c, const Ref& r) {
  double pt2 = fma(z.Px, z.Px, z.Py * z.Py);
  double ps2m1 = c.e0 - pt2;
  double ps2 = 1.0 + ps2m1;
  if (!(ps2 > 0.0)) return false;
  double Ps = sqrt(ps2);
  double rr = 1.0 / (Ps * (Ps + 1.0));
  double iPs = rr * (Ps + 1.0), iPs1 = rr * Ps;
  double LiPs = L * iPs;
  z.X = fma(LiPs, z.Px, z.X);
  z.Y = fma(LiPs, z.Py, z.Y);
  double num = (c.tA - pt2 * r.ibeta0 - z.Pt * ps2m1 * iPs1) * iPs1;
  z.T = fma(LiPs, num, z.T);
  return true;
}

// multipole field (28): By + i Bx = sum_m (kn_m + i ks_m)(X+iY)^(m-1), Horner from the top order
__device__ __forceinline__ void mult_field(const DevElem& e, double X, double Y, double& bx, double& by) {
  int m = e.order;
  double re = e.kn[m - 2], im = e.ks[m - 2];
  for (--m; m >= 2; --m) {
    double nre = fma(re, X, -im * Y) + e.kn[m - 2];
    double nim = fma(re, Y, im * X) + e.ks[m - 2];
    re = nre; im = nim;
  }
  by = fma(re, X, -im * Y);
  bx = fma(re, Y, im * X);
}

// a9 for straight elements (h = 0):  Omega = -(1/Ps)[a1 b - a2 (u.b) u],  b = (bx, by, 0)
__device__ __forceinline__ void omega_straight(double Px, double Py, double iPs, double bx, double by, const PCon& c,
                                               double& ox, double& oy, double& os) {
  double pb = c.a2p * fma(Px, bx, Py * by);
  ox = -iPs * fma(c.a1, bx, -pb * Px);
  oy = -iPs * fma(c.a1, by, -pb * Py);
  os = pb;
}

// ---------------------------------------------------------------------------------------------
// thick elements
// ---------------------------------------------------------------------------------------------

// a4: exact sector bend (10) in N slices, spin from the slice-edge Omega (6b).
// With c = cos(h ds), s = sin(h ds), A = sqrt(Pa^2 - Px^2), g = A - eta(1 + hX):
//   Px_f = Px + [g s - Px (1-c)]                                                    (10b)
//   X_f  = X + g (ck - sk r) + Px (sk + ck r),  r = (Px + Px_f)/(A + A_f)           (10a) rearranged
// Y and T do not feed back into the motion or Omega, so they are advanced once per element from
// the total asin difference (group property of the flow).
template <int DEPTH>
__device__ __forceinline__ bool sbend_exact(State& z, const DevElem& e, const PCon& c, const Ref& r) {
  const double ea = fma(-z.Py, z.Py, c.e0);   // Pa^2 - 1                                  (8)
  const double Pa2 = 1.0 + ea;
  double a2 = fma(-z.Px, z.Px, Pa2);
  if (!(a2 > 0.0)) return false;
  double A = sqrt(a2);
  double Am1 = fma(-z.Px, z.Px, ea) / (A + 1.0);   // A - 1 without cancellation
  const double A0 = A, Am1_0 = Am1, Px0 = z.Px;
  const double q2 = c.a2p * e.k0 * z.Py;           // G(gamma-1) (u.b)/P  /  (Py... ) see Omega below
  const double a1k = c.a1 * e.k0 - q2 * z.Py;
  SpinAcc<DEPTH> acc;
  acc.reset();
  const int N = e.N;
  const double ds = e.ds;
  {
    double f = fma(e.h, z.X, 1.0) / A;
    double w = 0.5 * ds;
    acc.edge(0, w * (f * q2 * z.Px), w * (e.h - f * a1k), w * (f * q2 * A));
  }
  for (int i = 1; i <= N; ++i) {
    double g = (Am1 + e.ome) - e.k0 * z.X;
    double dPx = fma(g, e.sn, -z.Px * e.cm);
    double Pxf = z.Px + dPx;
    double f2 = fma(-Pxf, Pxf, Pa2);
    if (!(f2 > 0.0)) return false;
    double Af = sqrt(f2);
    double t = 1.0 / (Af * (Af + A));
    double iAf = t * (Af + A);
    double rr = (z.Px + Pxf) * (t * Af);
    z.X += fma(g, fma(-e.sk, rr, e.ck), z.Px * fma(e.ck, rr, e.sk));
    Am1 = fma(-dPx, rr, Am1);
    z.Px = Pxf;
    A = Af;
    double f = fma(e.h, z.X, 1.0) * iAf;
    double w = (i == N) ? 0.5 * ds : ds;
    acc.edge(i, w * (f * q2 * z.Px), w * (e.h - f * a1k), w * (f * q2 * A));
  }
  // asin(Px0/Pa) - asin(PxN/Pa) = asin((Px0 A_N - Px_N A_0)/Pa^2)
  double arg = fma(Px0, Am1 - Am1_0, -(z.Px - Px0) * A0) / Pa2;
  double dasin = asin(arg);
  double dh = dasin * e.inv_h;
  z.Y = fma(z.Py * e.inv_eta, e.L + dh, z.Y);
  z.T += e.inv_eta * (fma(-z.Pt, e.L, -c.ibpt * dh) - e.ome * e.L * r.ibeta0);
  acc.finish(z.Sx, z.Sy, z.Ss);
  return true;
}

// a5: TEAPOT sector bend (30)(31): half curved drift, kick -ds k0 (1+hX), half curved drift.
// The curved drift is a straight line seen from the rotating frame, so (Px,Ps) simply rotate by
// phi = h ds/2; X, Y, T use rho(sec phi - 1), rho tan phi and rho(tan phi - phi) from the host.
__device__ __forceinline__ bool curved_half_drift(State& z, double& Ps, const DevElem& e, const PCon& c) {
  double iPs = 1.0 / Ps;
  double xp = z.Px * iPs;
  double D = fma(-xp, e.ht, 1.0);
  if (!(D > 0.0)) return false;
  double iD = 1.0 / D;
  double hs2 = 0.5 * e.ds;
  // delta q = [(rho+X) tan phi - s Ps D]/(Ps D),  s = ds/2
  double num = e.r_tanmphi + fma(z.X, e.ht, hs2 * fma(z.Px, e.ht, -(Ps - 1.0)));
  double dq = num * iPs * iD;
  z.X = (e.r_secm1 + fma(z.X, e.hsec, e.r_tan * xp)) * iD;
  z.Y = fma(z.Py, hs2 + dq, z.Y);
  z.T += fma(-z.Pt, hs2, -c.ibpt * dq);
  double Pxn = fma(z.Px, e.hc, Ps * e.hs);
  Ps = fma(Ps, e.hc, -z.Px * e.hs);
  z.Px = Pxn;
  return Ps > 0.0;
}
template <int DEPTH>
__device__ __forceinline__ bool sbend_teapot(State& z, const DevElem& e, const PCon& c) {
  const double pa2 = fma(-z.Py, z.Py, 1.0 + c.e0);
  double ps2 = fma(-z.Px, z.Px, pa2);
  if (!(ps2 > 0.0)) return false;
  double Ps = sqrt(ps2);
  const double q2 = c.a2p * e.k0 * z.Py;
  const double a1k = c.a1 * e.k0 - q2 * z.Py;
  SpinAcc<DEPTH> acc;
  acc.reset();
  const int N = e.N;
  const double ds = e.ds;
  {
    double f = fma(e.h, z.X, 1.0) / Ps;
    double w = 0.5 * ds;
    acc.edge(0, w * (f * q2 * z.Px), w * (e.h - f * a1k), w * (f * q2 * Ps));
  }
  for (int i = 1; i <= N; ++i) {
    if (!curved_half_drift(z, Ps, e, c)) return false;
    z.Px = fma(-ds * e.k0, fma(e.h, z.X, 1.0), z.Px);
    ps2 = fma(-z.Px, z.Px, pa2);
    if (!(ps2 > 0.0)) return false;
    Ps = sqrt(ps2);
    if (!curved_half_drift(z, Ps, e, c)) return false;
    double f = fma(e.h, z.X, 1.0) / Ps;
    double w = (i == N) ? 0.5 * ds : ds;
    acc.edge(i, w * (f * q2 * z.Px), w * (e.h - f * a1k), w * (f * q2 * Ps));
  }
  acc.finish(z.Sx, z.Sy, z.Ss);
  return true;
}

// a7: drift-kick multipole (29): half drift, kick (28), half drift.  The momenta are constant
// between kicks, so one 1/Ps serves the second half drift, the edge Omega and the next first half.
template <int DEPTH>
__device__ __forceinline__ bool mult_dk(State& z, const DevElem& e, const PCon& c, const Ref& r) {
  SpinAcc<DEPTH> acc;
  acc.reset();
  const int N = e.N;
  const double ds = e.ds, hds = 0.5 * e.ds;
  double pt2 = fma(z.Px, z.Px, z.Py * z.Py);
  double ps2m1 = c.e0 - pt2;
  if (!(1.0 + ps2m1 > 0.0)) return false;
  double Ps = sqrt(1.0 + ps2m1);
  double rr = 1.0 / (Ps * (Ps + 1.0));
  double iPs = rr * (Ps + 1.0), iPs1 = rr * Ps;
  double tnum = (c.tA - pt2 * r.ibeta0 - z.Pt * ps2m1 * iPs1) * iPs1 * iPs;   // T' of the drift
  double bx, by, ox, oy, os;
  mult_field(e, z.X, z.Y, bx, by);
  omega_straight(z.Px, z.Py, iPs, bx, by, c, ox, oy, os);
  acc.edge(0, hds * ox, hds * oy, hds * os);
  for (int i = 1; i <= N; ++i) {
    z.X = fma(hds * iPs, z.Px, z.X);
    z.Y = fma(hds * iPs, z.Py, z.Y);
    z.T = fma(hds, tnum, z.T);
    mult_field(e, z.X, z.Y, bx, by);
    z.Px = fma(-ds, by, z.Px);
    z.Py = fma(ds, bx, z.Py);
    pt2 = fma(z.Px, z.Px, z.Py * z.Py);
    ps2m1 = c.e0 - pt2;
    if (!(1.0 + ps2m1 > 0.0)) return false;
    Ps = sqrt(1.0 + ps2m1);
    rr = 1.0 / (Ps * (Ps + 1.0));
    iPs = rr * (Ps + 1.0); iPs1 = rr * Ps;
    tnum = (c.tA - pt2 * r.ibeta0 - z.Pt * ps2m1 * iPs1) * iPs1 * iPs;
    z.X = fma(hds * iPs, z.Px, z.X);
    z.Y = fma(hds * iPs, z.Py, z.Y);
    z.T = fma(hds, tnum, z.T);
    mult_field(e, z.X, z.Y, bx, by);
    omega_straight(z.Px, z.Py, iPs, bx, by, c, ox, oy, os);
    double w = (i == N) ? hds : ds;
    acc.edge(i, w * ox, w * oy, w * os);
  }
  acc.finish(z.Sx, z.Sy, z.Ss);
  return true;
}

// a6: quadrupole matrix-kick (24)(25)(27).  kappa^2 = |k1|/P (23); with u = (kappa ds/2)^2 the four
// functions cos, sin(x)/x, cosh, sinh(x)/x are power series in u (no sqrt of kappa is needed).
struct QuadLin {
  double C, S, Ch, Sh;        // cos x, s*sin(x)/x ... see build()
  double kS, kSh;             // |k1| s sin(x)/x,  |k1| s sinh(x)/x
  double tpp_f, txx_f, txp_f; // (24e) coefficients of Px^2, X^2, X Px in the focusing plane
  double tpp_d, txx_d, txp_d; // ... of Py^2, Y^2, Y Py in the defocusing plane
};
__device__ __forceinline__ void quadlin_build(QuadLin& q, double ak1, double s, const PCon& c) {
  double kap2 = ak1 * c.iP;
  double u = kap2 * s * s;
  double C, Sx, Ch, Shx;
  if (u <= 0.25) {
    double a = 1.0 / 87178291200.0, b = 1.0 / 1307674368000.0;   // 14!, 15!
    double ca = a, sa = b, ha = a, hb = b;
    ca = fma(ca, -u, 1.0 / 479001600.0); sa = fma(sa, -u, 1.0 / 6227020800.0);
    ha = fma(ha, u, 1.0 / 479001600.0);  hb = fma(hb, u, 1.0 / 6227020800.0);
    ca = fma(ca, -u, 1.0 / 3628800.0);   sa = fma(sa, -u, 1.0 / 39916800.0);
    ha = fma(ha, u, 1.0 / 3628800.0);    hb = fma(hb, u, 1.0 / 39916800.0);
    ca = fma(ca, -u, 1.0 / 40320.0);     sa = fma(sa, -u, 1.0 / 362880.0);
    ha = fma(ha, u, 1.0 / 40320.0);      hb = fma(hb, u, 1.0 / 362880.0);
    ca = fma(ca, -u, 1.0 / 720.0);       sa = fma(sa, -u, 1.0 / 5040.0);
    ha = fma(ha, u, 1.0 / 720.0);        hb = fma(hb, u, 1.0 / 5040.0);
    ca = fma(ca, -u, 1.0 / 24.0);        sa = fma(sa, -u, 1.0 / 120.0);
    ha = fma(ha, u, 1.0 / 24.0);         hb = fma(hb, u, 1.0 / 120.0);
    ca = fma(ca, -u, 0.5);               sa = fma(sa, -u, 1.0 / 6.0);
    ha = fma(ha, u, 0.5);                hb = fma(hb, u, 1.0 / 6.0);
    C = fma(ca, -u, 1.0);  Sx = fma(sa, -u, 1.0);
    Ch = fma(ha, u, 1.0);  Shx = fma(hb, u, 1.0);
  } else {
    double x = sqrt(u), sn, cs;
    sincos(x, &sn, &cs);
    C = cs; Sx = sn / x; Ch = cosh(x); Shx = sinh(x) / x;
  }
  q.C = C; q.Ch = Ch;
  q.S = s * c.iP * Sx;  q.Sh = s * c.iP * Shx;       // X += (s/P) Px sin(x)/x
  q.kS = ak1 * s * Sx;  q.kSh = ak1 * s * Shx;       // Px -= kappa^2 P s X sin(x)/x,  kappa^2 P = |k1|
  double s4 = 0.25 * s, iP2 = c.iP * c.iP;
  double SC = Sx * C, ShC = Shx * Ch;                // sin(2x)/(2x), sinh(2x)/(2x)
  q.tpp_f = s4 * iP2 * (1.0 + SC);
  q.txx_f = s4 * kap2 * (1.0 - SC);
  q.txp_f = -0.5 * u * Sx * Sx * c.iP;
  q.tpp_d = s4 * iP2 * (1.0 + ShC);
  q.txx_d = s4 * kap2 * (ShC - 1.0);
  q.txp_d = 0.5 * u * Shx * Shx * c.iP;
}
// flow of H_qL over s = ds/2: (uf,pf) is the focusing plane, (ud,pd) the defocusing one (A11)
__device__ __forceinline__ void quadlin_apply(const QuadLin& q, double& uf, double& pf, double& ud, double& pd, double& T,
                                              double tfac) {
  double curly = fma(q.tpp_f, pf * pf, fma(q.txx_f, uf * uf, q.txp_f * uf * pf)) +
                 fma(q.tpp_d, pd * pd, fma(q.txx_d, ud * ud, q.txp_d * ud * pd));
  T = fma(-tfac, curly, T);
  double nu = fma(uf, q.C, q.S * pf);
  pf = fma(pf, q.C, -q.kS * uf);
  uf = nu;
  nu = fma(ud, q.Ch, q.Sh * pd);
  pd = fma(pd, q.Ch, q.kSh * ud);
  ud = nu;
}
template <int DEPTH>
__device__ __forceinline__ bool quad_mk(State& z, const DevElem& e, const PCon& c) {
  const double k1 = e.kn[0];
  const bool foc = k1 > 0.0;
  const int N = e.N;
  const double ds = e.ds, hds = 0.5 * e.ds;
  QuadLin ql;
  quadlin_build(ql, fabs(k1), hds, c);
  const double tfac = c.iP * c.ibpt;
  const double P2 = 1.0 + c.e0;
  const double hiP3 = 0.5 * c.iP * c.iP * c.iP;
  SpinAcc<DEPTH> acc;
  acc.reset();
  double ox, oy, os;
  {
    double ps2 = P2 - fma(z.Px, z.Px, z.Py * z.Py);
    if (!(ps2 > 0.0)) return false;
    double iPs = rsqrt(ps2);
    omega_straight(z.Px, z.Py, iPs, k1 * z.Y, k1 * z.X, c, ox, oy, os);
    acc.edge(0, hds * ox, hds * oy, hds * os);
  }
  for (int i = 1; i <= N; ++i) {
    if (foc) quadlin_apply(ql, z.X, z.Px, z.Y, z.Py, z.T, tfac);
    else     quadlin_apply(ql, z.Y, z.Py, z.X, z.Px, z.T, tfac);
    {   // (25): X += ds Px (1/Ps - 1/P), 1/Ps - 1/P = pt2/(P Ps (P+Ps))
      double pt2 = fma(z.Px, z.Px, z.Py * z.Py);
      double ps2 = P2 - pt2;
      if (!(ps2 > 0.0)) return false;
      double Ps = sqrt(ps2);
      double t = 1.0 / (Ps * (c.P + Ps));           // 1/(Ps (P+Ps))
      double d = pt2 * c.iP * t;
      z.X = fma(ds * d, z.Px, z.X);
      z.Y = fma(ds * d, z.Py, z.Y);
      // T' = -(1/beta0+Pt)[1/Ps - 1/P - pt2/(2P^3)] + tq,  bracket = pt2^2 (2P+Ps)/(2 P^3 Ps (P+Ps)^2)
      double br = pt2 * pt2 * fma(2.0, c.P, Ps) * hiP3 * t * (t * Ps);
      z.T = fma(ds, fma(-c.ibpt, br, c.tq), z.T);
    }
    if (foc) quadlin_apply(ql, z.X, z.Px, z.Y, z.Py, z.T, tfac);
    else     quadlin_apply(ql, z.Y, z.Py, z.X, z.Px, z.T, tfac);
    double ps2 = P2 - fma(z.Px, z.Px, z.Py * z.Py);
    if (!(ps2 > 0.0)) return false;
    double iPs = rsqrt(ps2);
    omega_straight(z.Px, z.Py, iPs, k1 * z.Y, k1 * z.X, c, ox, oy, os);
    double w = (i == N) ? hds : ds;
    acc.edge(i, w * ox, w * oy, w * os);
  }
  acc.finish(z.Sx, z.Sy, z.Ss);
  return true;
}

// ---------------------------------------------------------------------------------------------
// the kernel
// ---------------------------------------------------------------------------------------------
constexpr int TRACK_BLOCK = 64;

template <int SPLIT, int DEPTH>
__global__ void __launch_bounds__(TRACK_BLOCK) track_kernel(const TrackArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  DevElem* tab = reinterpret_cast<DevElem*>(smem_raw);
  const uint16_t* seq = a.seq;
  {   // a0: stage the unique-element table (and the sequence when it fits) into shared memory
    const int nw = a.n_unique * (int)(sizeof(DevElem) / sizeof(double));
    const double* src = reinterpret_cast<const double*>(a.tab);
    double* dst = reinterpret_cast<double*>(smem_raw);
    for (int i = threadIdx.x; i < nw; i += blockDim.x) dst[i] = src[i];
    if (a.use_smem_seq) {
      uint16_t* sseq = reinterpret_cast<uint16_t*>(smem_raw + (size_t)a.n_unique * sizeof(DevElem));
      for (int i = threadIdx.x; i < a.n_seq; i += blockDim.x) sseq[i] = a.seq[i];
      seq = sseq;
    }
    __syncthreads();
  }
  const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= a.n) return;
  if (a.lost[j]) return;
  State z;
  z.X = a.p[0][j]; z.Px = a.p[1][j]; z.Y = a.p[2][j]; z.Py = a.p[3][j]; z.T = a.p[4][j]; z.Pt = a.p[5][j];
  z.Sx = a.p[6][j]; z.Sy = a.p[7][j]; z.Ss = a.p[8][j];
  Ref ref;
  ref_set(ref, a.E0, a.mass);
  PCon pc;
  pcon_set(pc, z.Pt, ref, a.G);
  bool alive = true;
  for (long long turn = 0; turn < a.n_turns && alive; ++turn) {
    for (int ie = 0; ie < a.n_seq && alive; ++ie) {
      const DevElem& e = tab[seq[ie]];
      switch (e.type) {
        case K_DRIFT: alive = drift(z, e.L, pc, ref); break;
        case K_SBEND:
          if (SPLIT == SPLIT_DK) alive = sbend_teapot<DEPTH>(z, e, pc);
          else alive = sbend_exact<DEPTH>(z, e, pc, ref);
          break;
        case K_QUAD:
          if (SPLIT == SPLIT_MK) alive = quad_mk<DEPTH>(z, e, pc);
          else alive = mult_dk<DEPTH>(z, e, pc, ref);
          break;
        case K_MULT: alive = mult_dk<DEPTH>(z, e, pc, ref); break;
        case K_THIN: {   // A10: half kick, spin, half kick
          double bx, by, ox, oy, os;
          mult_field(e, z.X, z.Y, bx, by);
          z.Px = fma(-0.5, by, z.Px);
          z.Py = fma(0.5, bx, z.Py);
          double ps2 = 1.0 + pc.e0 - fma(z.Px, z.Px, z.Py * z.Py);
          if (!(ps2 > 0.0)) { alive = false; break; }
          omega_straight(z.Px, z.Py, rsqrt(ps2), bx, by, pc, ox, oy, os);
          Quat q = quat_from_rotvec(ox, oy, os);
          quat_rotate(q, z.Sx, z.Sy, z.Ss);
          z.Px = fma(-0.5, by, z.Px);
          z.Py = fma(0.5, bx, z.Py);
          break;
        }
        case K_RF: {     // A12, A13
          double krf = e.krf_over_beta * ref.beta0;
          double dE = e.volt * sin(fma(e.sign * krf, z.T, e.phi_s));
          // E - E0' = p0c Pt + dE - dEs: the O(E0) terms are never formed
          double num = fma(ref.p0c, z.Pt, dE - e.dEs);
          if (e.dEs != 0.0) {
            double p0_old = ref.p0c;
            ref_set(ref, ref.E0 + e.dEs, ref.mass);
            double sc = p0_old / ref.p0c;
            z.Px *= sc; z.Py *= sc;
          }
          z.Pt = num / ref.p0c;
          pcon_set(pc, z.Pt, ref, a.G);
          break;
        }
        case K_SNAKE: {
          Quat q{e.qw, e.qx, e.qy, e.qs};
          quat_rotate(q, z.Sx, z.Sy, z.Ss);
          break;
        }
        default: break;
      }
    }
  }
  if (!alive) a.lost[j] = 1;
  a.p[0][j] = z.X; a.p[1][j] = z.Px; a.p[2][j] = z.Y; a.p[3][j] = z.Py; a.p[4][j] = z.T; a.p[5][j] = z.Pt;
  a.p[6][j] = z.Sx; a.p[7][j] = z.Sy; a.p[8][j] = z.Ss;
}

}  // namespace gst
