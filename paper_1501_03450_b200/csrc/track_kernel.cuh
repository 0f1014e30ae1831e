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
//
// Scheduling: the kernel runs at ~3.5 warps per SM sub-partition, so the FP64
// pipe is fed by instruction-level parallelism inside a thread.  The slice loop is software
// pipelined -- orbit slice i+1 is independent of the quaternion work of edge i and sits in the same
// basic block -- and the loop body is branch-free: reciprocal and reciprocal square root are
// MUFU seeds + Newton steps without slow-path calls, domain errors set a sticky flag, and the
// Romberg-level membership of an edge is resolved at compile time for odd edges.
#pragma once
#include <cstdint>

namespace gst {

enum : int { K_DRIFT = 0, K_SBEND = 1, K_QUAD = 2, K_MULT = 3, K_THIN = 4, K_RF = 5, K_SNAKE = 6, K_MARKER = 7, K_FRINGE = 8, K_SOLENOID = 9, K_RBEND = 10 };
enum : int { SPLIT_DK = 0, SPLIT_BK = 1, SPLIT_MK = 2 };

// Fourth-order symmetric composition of a second-order slice map S2 (R5):
//   S4(ds) = S2(x1 ds) S2(x0 ds) S2(x1 ds),  x1 = 1/(2 - 2^(1/3)),  x0 = 1 - 2 x1.
// Neighbouring exact pieces (half drifts, curved drifts, linear quadrupole flows) are merged by their
// group property: A(x1/2) B(x1) A((x1+x0)/2) B(x0) A((x1+x0)/2) B(x1) A(x1/2).
#define GST_YOSHIDA_X1 1.3512071919596576340476878089715
#define GST_YOSHIDA_X0 (-1.7024143839193152680953756179429)

// constants of one curved drift (31) of length `len` in a bend of curvature h: phi = h len
struct TeapotHalf {
  double len;
  double c, s, t, sec;   // cos phi, sin phi, tan phi, 1/cos phi
  double r_secm1;        // rho (sec phi - 1)
  double r_tan;          // rho tan phi
  double r_tanmphi;      // rho (tan phi - phi)
};

// Unique-element record, derived on the host for one value of n_slices (a0).
struct __align__(16) DevElem {
  int type;
  int N;          // slices of this element (thick), else 1
  int order;      // highest multipole order present (2..5); 2 if none
  int pure_quad;  // 1 when only kn[0] is non-zero
  double L;       // length
  double Lpre;    // length of the drift space in front of this element that the lattice compiler merged into it (0: none)
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
  // sector bend, TEAPOT curved drifts (31): [0] over ds/2 (second order), [1] over x1 ds/2 and [2] over
  // (x1 + x0) ds/2 < 0 (the merged neighbours of the fourth-order composition, see Yoshida above), [3] over ds
  // (the whole drifts of the DKSKD ordering, whose table is derived for half slices)
  TeapotHalf th[4];
  // rectangular bend (section 3.2): rotations (17) by phi_entr [0] and by -phi_exit [1]
  double rb_c[2], rb_s[2], rb_t[2], rb_sec[2];   // cos, sin, tan, sec of the rotation angle
  double rb_qw[2], rb_qy[2];                     // the same rotation of the spin components: (cos, sin)(angle/2) about y
  double rb_rho;                                 // rho_b = 1/k0 (12)
  double rb_xoff;                                // (18): rho_b (cos phi_exit - cos phi_entr)
  double rb_arc;                                 // rho_b (phi_entr - phi_exit), (19)
  double rb_cd, rb_sd;                           // cos, sin of phi_entr - phi_exit
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
  const uint32_t* seq;     // element sequence: (index into tab) << 8 | type, see seq_pack()
  int n_unique;
  int n_seq;
  long long n;
  long long n_turns;
  double E0, E0lo, mass, G;   // reference energy = E0 + E0lo (compensated sum of the cavity gains)
  const int* err;           // the bunch's error word: non-zero = an earlier launch on this bunch failed and nobody has been
                            // told yet; the kernel then leaves everything as it is (include/gst.h, "Errors")
};

// One sequence entry carries the element type next to the table index, so that the per-element dispatch
// needs one (prefetched) load instead of the chain seq -> table -> type.
__host__ __device__ inline uint32_t seq_pack(uint32_t index, int type) { return (index << 8) | (uint32_t)type; }

struct Quat { double w, x, y, s; };

// ---------------------------------------------------------------------------------------------
// branch-free reciprocal and reciprocal square root: 20-bit MUFU seed + Newton in FMAs.
// (CUDA's 1.0/x and sqrt() carry a slow-path call that splits the basic block.)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double rcp_nr(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));   // MUFU.RCP64H: relative error < 2^-20
  double e = fma(-x, y, 1.0);
  e = fma(e, e, e);                 // e + e^2: cubic step y (1 + e + e^2), residual e^3 < 2^-60
  return fma(y, e, y);              // ~1 ulp (gst_selftest_math measures it)
}
__device__ __forceinline__ double rsqrt_nr(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x)); // MUFU.RSQ64H: relative error < 2^-20
  double t = x * y;
  double e = fma(-t, y, 1.0);       // 1 - x y^2
  double c = fma(0.375, e, 0.5);
  return fma(y * e, c, y);          // cubic step y (1 + e/2 + 3e^2/8), residual (5/16) e^3 < 2^-58
}

// domain test of A15 (false for NaN).  Integer compares on the sign-and-exponent word instead of DSETP measured 0.5 %
// slower, although a DSETP takes two FP64 issue slots.
__device__ __forceinline__ bool is_pos(double x) { return x > 0.0; }

// reference-particle and per-particle constants that change only when Pt or E0 changes
struct Ref {
  double E0, mass, p0c, beta0, gamma0, ibeta0, ibg2;  // ibg2 = 1/(beta0 gamma0)^2 = 1/beta0^2 - 1
  double E0lo;                                        // E0 + E0lo = exact sum of the gains so far (ref_energy_add)
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

// A13: E_o <- E_o + dE_s once per turn and cavity.  The spin phase of a turn is 2 pi G gamma_o, so rounding errors of
// E_o that pile up over n turns grow as n^2 in the spin (7.6e-8 after 4000 turns against the long-double oracle,
// tests/test_gpu_parity.py::test_ramp_through_an_isolated_resonance).  The sum is therefore carried as an unevaluated
// pair (two-sum, renormalised): E0 is the correctly rounded exact sum at every turn, E0lo the remainder.
__host__ __device__ __forceinline__ void ref_energy_add(double& E0, double& E0lo, double dEs) {
  const double s = E0 + dEs;
  const double bb = s - E0;
  const double err = (E0 - (s - bb)) + (dEs - bb);   // s + err = E0 + dEs exactly
  const double lo = E0lo + err;
  const double hi = s + lo;
  E0lo = lo - (hi - s);
  E0 = hi;
}
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
// q = (cos(th/2), sin(th/2) w/th) for rotation vector w: both factors are even in th, so they are
// functions of v = th^2 -- no sqrt, no division, no sincos ("low-order polynomials", here
// taken to full double precision).  Three tiers by angle; the first is the straight-line path:
//   tier 1  v <= 1/8 (th <= 0.35 rad per edge: every magnet of the BASELINE rings at >= 8 slices): degree-4
//           polynomials in v that interpolate cos(sqrt(v)/2) and sin(sqrt(v)/2)/sqrt(v) at the five Chebyshev
//           nodes of [0, 1/8] (near-minimax; 50-digit fit, coefficients rounded to double, constant terms
//           1 and 1/2 exactly): error 3.2e-17 absolute on the cosine, 3.2e-18 relative on the sine factor
//           -- below half an ulp; the degree-6 Taylor pair it replaces costs four more DFMAs per edge
//   tier 2  v <= 2: Taylor, 10 terms;   tier 3: sincos.
// The coefficients sit in constant memory so that each DFMA takes its coefficient as a c[bank][offset]
// operand (a double literal would cost two extra UMOV/MOV instructions per use on sm_100).
//   QPOLY[2k] = coefficient of v^k in the cosine, QPOLY[2k+1] = in sin(x)/th, k = 1..4
#ifndef GST_QPOLY_DEG
#define GST_QPOLY_DEG 4
#endif
#if GST_QPOLY_DEG == 4
#define GST_QTIER1 0.125
static __constant__ double QPOLY[10] = {
    1.0, 0.5,
    -0.12499999999999359, -0.02083333333333304,
    0.0026041666662562613, 0.00026041666664801025,
    -2.1701379695306356e-05, -1.5500987884264741e-06,
    9.679713447825894e-08, 5.378467506662951e-09};
#else   // degree-6 Taylor pair, v <= 1/2: (-1/4)^k/(2k)! and (1/2)(-1/4)^k/(2k+1)!, remainder (v/4)^7/14! < 6e-18
#define GST_QTIER1 0.5
static __constant__ double QPOLY[14] = {
    1.0, 0.5,
    -1.0 / 8.0, -0.5 / 24.0,
    1.0 / (16.0 * 24.0), 0.5 / (16.0 * 120.0),
    -1.0 / (64.0 * 720.0), -0.5 / (64.0 * 5040.0),
    1.0 / (256.0 * 40320.0), 0.5 / (256.0 * 362880.0),
    -1.0 / (1024.0 * 3628800.0), -0.5 / (1024.0 * 39916800.0),
    1.0 / (4096.0 * 479001600.0), 0.5 / (4096.0 * 6227020800.0)};
#endif

// tiers 2 and 3 (large angle per edge), kept out of line: they are rare and would otherwise be
// replicated at every call site (instruction-cache footprint)
static __device__ __noinline__ double2 quat_cs_slow(double v) {
  double c, s;
  if (v <= 2.0) {
    // tier 2: u = v/4 <= 0.5, k = 0..9, remainder < 4e-20
    double u = 0.25 * v;
    c = -1.0 / 6402373705728000.0;  s = -1.0 / 121645100408832000.0;
    c = fma(c, u, 1.0 / 20922789888000.0);  s = fma(s, u, 1.0 / 355687428096000.0);
    c = fma(c, u, -1.0 / 87178291200.0);    s = fma(s, u, -1.0 / 1307674368000.0);
    c = fma(c, u, 1.0 / 479001600.0);       s = fma(s, u, 1.0 / 6227020800.0);
    c = fma(c, u, -1.0 / 3628800.0);        s = fma(s, u, -1.0 / 39916800.0);
    c = fma(c, u, 1.0 / 40320.0);           s = fma(s, u, 1.0 / 362880.0);
    c = fma(c, u, -1.0 / 720.0);            s = fma(s, u, -1.0 / 5040.0);
    c = fma(c, u, 1.0 / 24.0);              s = fma(s, u, 1.0 / 120.0);
    c = fma(c, u, -0.5);                    s = fma(s, u, -1.0 / 6.0);
    c = fma(c, u, 1.0);                     s = fma(s, u, 1.0);
    s *= 0.5;
  } else {
    double th = sqrt(v), sn, cs;
    sincos(0.5 * th, &sn, &cs);
    c = cs; s = sn / th;
  }
  return make_double2(c, s);
}

// Straight magnets (quadrupoles, multipoles) turn the spin by milliradians per slice edge: for them (SMALL = true) tier 1
// is v <= 1/128 (th <= 0.088 rad) with degree-3 interpolants (errors 5.6e-18 / 6.5e-19), two DFMAs per edge less;
// anything larger goes to the out-of-line tiers, whose Taylor polynomial is valid from v = 0.
static __constant__ double QPOLY3[8] = {
    1.0, 0.5,
    -0.12499999999998845, -0.02083333333333269,
    0.0026041666592755064, 0.00026041666625604374,
    -2.1699875165301865e-05, -1.5500151101381229e-06};
template <bool SMALL> __device__ __forceinline__ Quat quat_from_rotvec_t(double wx, double wy, double ws);
template <> __device__ __forceinline__ Quat quat_from_rotvec_t<true>(double wx, double wy, double ws) {
  const double v = fma(wx, wx, fma(wy, wy, ws * ws));
  double c = QPOLY3[6], s = QPOLY3[7];
  c = fma(c, v, QPOLY3[4]);  s = fma(s, v, QPOLY3[5]);
  c = fma(c, v, QPOLY3[2]);  s = fma(s, v, QPOLY3[3]);
  c = fma(c, v, 1.0);        s = fma(s, v, 0.5);
  if (__builtin_expect(v > 0.0078125, 0)) {
    const double2 cs = quat_cs_slow(v);
    c = cs.x; s = cs.y;
  }
  return Quat{c, s * wx, s * wy, s * ws};
}
__device__ __forceinline__ Quat quat_from_rotvec(double wx, double wy, double ws) {
  const double v = fma(wx, wx, fma(wy, wy, ws * ws));   // th^2;  x = th/2, x^2 = v/4
#if GST_QPOLY_DEG == 4
  double c = QPOLY[8], s = QPOLY[9];
#else
  double c = QPOLY[12], s = QPOLY[13];
  c = fma(c, v, QPOLY[10]); s = fma(s, v, QPOLY[11]);
  c = fma(c, v, QPOLY[8]);  s = fma(s, v, QPOLY[9]);
#endif
  c = fma(c, v, QPOLY[6]);  s = fma(s, v, QPOLY[7]);
  c = fma(c, v, QPOLY[4]);  s = fma(s, v, QPOLY[5]);
  c = fma(c, v, QPOLY[2]);  s = fma(s, v, QPOLY[3]);
  c = fma(c, v, 1.0);       s = fma(s, v, 0.5);
  if (__builtin_expect(v > GST_QTIER1, 0)) {     // (a warp vote in front of this branch measured 6 % slower)
    const double2 cs = quat_cs_slow(v);
    c = cs.x; s = cs.y;
  }
  return Quat{c, s * wx, s * wy, s * ws};
}
template <> __device__ __forceinline__ Quat quat_from_rotvec_t<false>(double wx, double wy, double ws) {
  return quat_from_rotvec(wx, wy, ws);
}
// a (x) b
__device__ __forceinline__ Quat quat_mul(const Quat& a, const Quat& b) {
  Quat r;
  r.w = fma(a.w, b.w, -fma(a.x, b.x, fma(a.y, b.y, a.s * b.s)));
  r.x = fma(a.w, b.x, fma(a.x, b.w, fma(a.y, b.s, -a.s * b.y)));
  r.y = fma(a.w, b.y, fma(-a.x, b.s, fma(a.y, b.w, a.s * b.x)));
  r.s = fma(a.w, b.s, fma(a.x, b.y, fma(-a.y, b.x, a.s * b.w)));
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

// S <- q S q* / |q|^2 for any q != 0 (the normalised Romberg result of P:546 applied to S without forming it)
__device__ __forceinline__ void quat_rotate_unnormalised(const Quat& q, double& Sx, double& Sy, double& Ss) {
  const double i2 = 2.0 * rcp_nr(fma(q.w, q.w, fma(q.x, q.x, fma(q.y, q.y, q.s * q.s))));
  double tx = i2 * fma(q.y, Ss, -q.s * Sy);
  double ty = i2 * fma(q.s, Sx, -q.x * Ss);
  double ts = i2 * fma(q.x, Sy, -q.y * Sx);
  Sx += fma(q.w, tx, fma(q.y, ts, -q.s * ty));
  Sy += fma(q.w, ty, fma(q.s, tx, -q.x * ts));
  Ss += fma(q.w, ts, fma(q.x, ty, -q.y * tx));
}

// Running products of the DEPTH trapezoid levels.  Level l has stride 2^l (l = 0 is the
// finest); edge i belongs to it when 2^l | i.  The rotation for weight 2^l is obtained from the
// finest one by angle doubling instead of a new sincos.
// The Romberg table (39b) is linear in its first column, so its bottom-right entry is a fixed linear
// combination of the DEPTH level products: row d-1 holds the weights of Q[0] (finest) .. Q[d-1] (coarsest),
// obtained by running (39b) on unit vectors (exact integers over a common denominator).
static __constant__ double ROMBERG_W[6][6] = {
    {1.0, 0.0, 0.0, 0.0, 0.0, 0.0},
    {4.0 / 3.0, -1.0 / 3.0, 0.0, 0.0, 0.0, 0.0},
    {64.0 / 45.0, -20.0 / 45.0, 1.0 / 45.0, 0.0, 0.0, 0.0},
    {4096.0 / 2835.0, -1344.0 / 2835.0, 84.0 / 2835.0, -1.0 / 2835.0, 0.0, 0.0},
    {1048576.0 / 722925.0, -348160.0 / 722925.0, 22848.0 / 722925.0, -340.0 / 722925.0, 1.0 / 722925.0, 0.0},
    {1073741824.0 / 739552275.0, -357564416.0 / 739552275.0, 23744512.0 / 739552275.0, -371008.0 / 739552275.0,
     1364.0 / 739552275.0, -1.0 / 739552275.0}};

// the same weights divided by the finest level's: row d-1 = ROMBERG_W[d-1][l] / ROMBERG_W[d-1][0]
static __constant__ double ROMBERG_REL[6][6] = {
    {1.0, 0.0, 0.0, 0.0, 0.0, 0.0},
    {1.0, -1.0 / 4.0, 0.0, 0.0, 0.0, 0.0},
    {1.0, -20.0 / 64.0, 1.0 / 64.0, 0.0, 0.0, 0.0},
    {1.0, -1344.0 / 4096.0, 84.0 / 4096.0, -1.0 / 4096.0, 0.0, 0.0},
    {1.0, -348160.0 / 1048576.0, 22848.0 / 1048576.0, -340.0 / 1048576.0, 1.0 / 1048576.0, 0.0},
    {1.0, -357564416.0 / 1073741824.0, 23744512.0 / 1073741824.0, -371008.0 / 1073741824.0, 1364.0 / 1073741824.0,
     -1.0 / 1073741824.0}};

template <int DEPTH> struct SpinAcc {
  Quat Q[DEPTH];
  // first edge of an element: every level starts from its own rotation (the product with the identity
  // is skipped; bit-identical apart from the sign of a zero)
  template <bool SMALL>
  __device__ __forceinline__ void init(double wx, double wy, double ws) {
    Quat q = quat_from_rotvec_t<SMALL>(wx, wy, ws);
    Q[0] = q;
#pragma unroll
    for (int l = 1; l < DEPTH; ++l) {
      q = quat_double(q);
      Q[l] = q;
    }
  }
  // fold rotation vector (weight * ds * Omega_i) into levels 0..NS-1, all known at compile time
  template <int NS, bool SMALL>
  __device__ __forceinline__ Quat fold_static(double wx, double wy, double ws) {
    Quat q = quat_from_rotvec_t<SMALL>(wx, wy, ws);
    Q[0] = quat_mul(q, Q[0]);
#pragma unroll
    for (int l = 1; l < NS; ++l) {
      q = quat_double(q);
      Q[l] = quat_mul(q, Q[l]);
    }
    return q;
  }
  // continue from level FROM upwards while 2^l | i (run-time, uniform across the grid)
  template <int FROM>
  __device__ __forceinline__ void fold_dynamic(int i, Quat q) {
#pragma unroll
    for (int l = FROM; l < DEPTH; ++l) {
      if ((i & ((1 << l) - 1)) != 0) return;
      q = quat_double(q);
      Q[l] = quat_mul(q, Q[l]);
    }
  }
  // Romberg limit (39b) P:542 of the level products, normalised, applied to S (a11).
  // Q[l] holds step h*2^l, i.e. column entry k = DEPTH-1-l of (38).
  // The normalisation is a common positive factor, so the weights are taken relative to the finest level's (its
  // product enters with weight one) and the rotation divides by |q|^2 instead of normalising q first: a reciprocal
  // instead of a reciprocal square root and eight multiplications less per element.
  __device__ __forceinline__ void finish(double& Sx, double& Sy, double& Ss) {
    Quat q = Q[0];
#pragma unroll
    for (int l = 1; l < DEPTH; ++l) {
      q.w = fma(ROMBERG_REL[DEPTH - 1][l], Q[l].w, q.w); q.x = fma(ROMBERG_REL[DEPTH - 1][l], Q[l].x, q.x);
      q.y = fma(ROMBERG_REL[DEPTH - 1][l], Q[l].y, q.y); q.s = fma(ROMBERG_REL[DEPTH - 1][l], Q[l].s, q.s);
    }
    quat_rotate_unnormalised(q, Sx, Sy, Ss);
  }
};

// ---------------------------------------------------------------------------------------------
// particle state in registers
// ---------------------------------------------------------------------------------------------
struct State {
  double X, Px, Y, Py, T, Pt, Sx, Sy, Ss;
};

// Longitudinal momentum at the particle's present transverse momenta: what a drift, the entrance of a bend and the
// entrance of a drift-kick magnet all start from.  The lattice compiler (gst_api.cu) merges every drift space into
// the element behind it (DevElem::Lpre), so that this one square root serves the drift AND that element.
struct Mom {
  double pt2;     // Px^2 + Py^2
  double ps2m1;   // Ps^2 - 1, without cancellation
  double iPs, Ps;
  bool ok;        // Ps^2 > 0 (A15)
};
__device__ __forceinline__ Mom mom_of(const State& z, const PCon& c) {
  Mom m;
  m.pt2 = fma(z.Px, z.Px, z.Py * z.Py);
  m.ps2m1 = c.e0 - m.pt2;
  const double ps2 = 1.0 + m.ps2m1;
  m.ok = is_pos(ps2);
  m.iPs = rsqrt_nr(ps2);
  m.Ps = ps2 * m.iPs;
  return m;
}
// a3: exact drift (29b) over L.  T' = 1/beta0 - (1/beta0+Pt)/Ps is evaluated as [(Ps-1)/beta0 - Pt]/Ps with
// Ps-1 = (Ps^2-1)/(Ps+1) and the O(Pt) terms combined analytically; iPs1 = 1/(Ps+1).
__device__ __forceinline__ void drift_with(State& z, double L, const Mom& m, double iPs1, const PCon& c, const Ref& r) {
  const double num = (fma(-m.pt2, r.ibeta0, c.tA) - z.Pt * m.ps2m1 * iPs1) * iPs1;
  const double LiPs = L * m.iPs;
  z.X = fma(LiPs, z.Px, z.X);
  z.Y = fma(LiPs, z.Py, z.Y);
  z.T = fma(LiPs, num, z.T);
}
__device__ __forceinline__ bool drift(State& z, double L, const PCon& c, const Ref& r) {
  const Mom m = mom_of(z, c);
  drift_with(z, L, m, rcp_nr(m.Ps + 1.0), c, r);
  return m.ok;
}

// ---------------------------------------------------------------------------------------------
// thick elements: a "stepper" advances the orbit by one slice and evaluates weight*ds*Omega at the
// current point; the spin policy's run() drives it through the N slices with the spin work software-pipelined.
// ---------------------------------------------------------------------------------------------
// The spin side of a thick element is a policy object with one method, run(stepper, N, ds):
//   FusedSpin<DEPTH>  -- the trapezoid / Romberg scheme (38)(39): every edge is folded into DEPTH level products
//   MidSpin<KIND>     -- the mid-slice comparison integrators (37)
// ROLLED: the matrix-kick kernels take the edges one per iteration with the level membership tested at run time
// (uniform branches).  Their two-edge loop body would be 6 kB for the quadrupole (160 fp64 instructions per
// slice), as much as the L0 instruction cache: rolled, matrix-kick runs 2 % faster (12-18 % before the quadrupole's
// two polarities shared one loop, see QuadPlane), while the drift-/bend-kick kernels, whose two-edge bodies are 3 kB,
// lose 4 %.
template <int DEPTH, bool ROLLED = false> struct FusedSpin {
  double &Sx, &Sy, &Ss;
  __device__ __forceinline__ FusedSpin(State& z) : Sx(z.Sx), Sy(z.Sy), Ss(z.Ss) {}
  template <class Stepper>
  __device__ __forceinline__ void run(Stepper& s, int N, double ds) {
    constexpr bool SM = Stepper::SMALL_ANGLE;      // (in the rolled matrix-kick kernels it measured 4 % slower)
    SpinAcc<DEPTH> acc;
    const double hds = 0.5 * ds;
    double wx, wy, ws;
    s.omega(hds, wx, wy, ws);                       // pending edge 0, half weight
    s.advance();                                    // orbit slice 1 ...
    acc.template init<SM>(wx, wy, ws);                           // ... independent of the spin work of edge 0
    if (DEPTH > 1 && ROLLED) {
      s.omega(ds, wx, wy, ws);                                 // pending edge 1 (N >= 2 when DEPTH >= 2)
#pragma unroll 1
      for (int i = 1; i < N; ++i) {
        s.advance();                                           // slice i+1 next to the fold of edge i
        Quat q = acc.template fold_static<1, SM>(wx, wy, ws);
        acc.template fold_dynamic<1>(i, q);
        s.omega(i + 1 == N ? hds : ds, wx, wy, ws);
      }
      acc.template fold_static<DEPTH, SM>(wx, wy, ws);             // edge N: every level
    } else if (DEPTH == 1) {
      s.omega(N == 1 ? hds : ds, wx, wy, ws);
      for (int i = 2; i <= N; ++i) {
        s.advance();                                // slice i next to the fold of edge i-1
        acc.template fold_static<1, SM>(wx, wy, ws);
        s.omega(i == N ? hds : ds, wx, wy, ws);
      }
      acc.template fold_static<1, SM>(wx, wy, ws);
    } else {
      // DEPTH >= 2: N is even (A4).  Edges are taken in pairs (odd, even): the odd edge belongs to
      // level 0 only, the even edge to levels 0 and 1 and, where 4 | i, 8 | i, ..., to higher ones.
      s.omega(ds, wx, wy, ws);                                 // pending edge 1
      for (int i = 1; i + 1 < N; i += 2) {
        s.advance();                                           // slice i+1
        acc.template fold_static<1, SM>(wx, wy, ws);               // odd edge i
        s.omega(ds, wx, wy, ws);
        s.advance();                                           // slice i+2
        {
          Quat q = acc.template fold_static<2, SM>(wx, wy, ws);    // even edge i+1
          acc.template fold_dynamic<2>(i + 1, q);
        }
        s.omega(ds, wx, wy, ws);
      }
      s.advance();                                             // slice N
      acc.template fold_static<1, SM>(wx, wy, ws);                 // odd edge N-1
      s.omega(hds, wx, wy, ws);
      acc.template fold_static<DEPTH, SM>(wx, wy, ws);             // edge N: every level (2^(DEPTH-1) | N)
    }
    acc.finish(Sx, Sy, Ss);
  }
  // thin element (A10): one rotation, no Romberg
  __device__ __forceinline__ void thin(double wx, double wy, double ws) {
    Quat q = quat_from_rotvec(wx, wy, ws);
    quat_rotate(q, Sx, Sy, Ss);
  }
  __device__ __forceinline__ void snake(const Quat& q) { quat_rotate(q, Sx, Sy, Ss); }
};

// Mid-slice piece-wise-constant precession (37) P:470-482, the comparison integrator of Figs. 7 and 14.
// KIND = 0: half slice map, rotation by ds*Omega(mid), half slice map ("DKDSDKD"); KIND = -1: half drift,
// half kick, rotation, half kick, half drift ("DKSKD") in drift-kick-mapped elements.  The element table is
// derived for HALF slices: N2 = 2 N maps of length ds2 = ds/2, one rotation of weight 2 ds2 per pair.
template <int KIND> struct MidSpin {
  double &Sx, &Sy, &Ss;
  __device__ __forceinline__ MidSpin(State& z) : Sx(z.Sx), Sy(z.Sy), Ss(z.Ss) {}
  template <class Stepper>
  __device__ __forceinline__ void run(Stepper& s, int N2, double ds2) {
    constexpr bool DKSKD = KIND == -1;
    const double w = 2.0 * ds2;
    double wx, wy, ws;
    s.template pwc_first<DKSKD>();
    s.omega(w, wx, wy, ws);
    Quat Q = quat_from_rotvec(wx, wy, ws);
    s.template pwc_second<DKSKD>();
    for (int i = 2; i < N2; i += 2) {
      s.template pwc_first<DKSKD>();
      s.omega(w, wx, wy, ws);
      Q = quat_mul(quat_from_rotvec(wx, wy, ws), Q);        // later rotations on the left (37b)
      s.template pwc_second<DKSKD>();
    }
    quat_rotate_unnormalised(Q, Sx, Sy, Ss);
  }
  __device__ __forceinline__ void thin(double wx, double wy, double ws) {
    Quat q = quat_from_rotvec(wx, wy, ws);
    quat_rotate(q, Sx, Sy, Ss);
  }
  __device__ __forceinline__ void snake(const Quat& q) { quat_rotate(q, Sx, Sy, Ss); }
};
// FAT: the kernel variant for bunches that leave most of the chip empty (see track_kernel below); there the matrix-kick
// loops keep their two-edge bodies.
template <int DEPTH, int SPLIT, bool FAT> struct SpinPolicy { using type = FusedSpin<DEPTH, SPLIT == SPLIT_MK && !FAT>; };
template <int SPLIT, bool FAT> struct SpinPolicy<0, SPLIT, FAT> { using type = MidSpin<0>; };
template <int SPLIT, bool FAT> struct SpinPolicy<-1, SPLIT, FAT> { using type = MidSpin<-1>; };

// a4: exact sector bend (10), spin from the slice-edge Omega (6b).
// With c = cos(h ds), s = sin(h ds), A = sqrt(Pa^2 - Px^2), g = A - eta(1 + hX):
//   Px_f = Px + [g s - Px (1-c)]                                                    (10b)
//   X_f  = X + g (ck - sk r) + Px (sk + ck r),  r = (Px + Px_f)/(A + A_f)           (10a) rearranged
// Y and T do not feed back into the motion or Omega, so they are advanced once per element from
// the total asin difference (group property of the flow).
struct BendExact {
  static constexpr bool SMALL_ANGLE = false;
  double &X, &Px;
  double A, Am1, iA;
  double Pa2, q2, a1k;
  double h, k0, cm, sn, ck, sk, ome;
  bool bad;
  // A = sqrt(Pa^2 - Px^2) is Ps: the drift space merged in front of the magnet (e.Lpre) shares its square root
  // and its 1/(Ps + 1) with the entrance values A, 1/A and A - 1
  __device__ __forceinline__ BendExact(State& z, const DevElem& e, const PCon& c, const Ref& r)
      : X(z.X), Px(z.Px), h(e.h), k0(e.k0), cm(e.cm), sn(e.sn), ck(e.ck), sk(e.sk), ome(e.ome) {
    const Mom m = mom_of(z, c);
    const double iPs1 = rcp_nr(m.Ps + 1.0);
    if (e.Lpre != 0.0) drift_with(z, e.Lpre, m, iPs1, c, r);
    Pa2 = 1.0 + fma(-z.Py, z.Py, c.e0);            // (8)
    bad = !m.ok;
    iA = m.iPs;
    A = m.Ps;
    Am1 = m.ps2m1 * iPs1;                          // A - 1 without cancellation
    q2 = c.a2p * e.k0 * z.Py;                      // G(gamma-1) (u.b) / P  per unit momentum component
    a1k = fma(c.a1, e.k0, -q2 * z.Py);
  }
  __device__ __forceinline__ void advance() {
    const double g = (Am1 + ome) - k0 * X;
    const double dPx = fma(g, sn, -Px * cm);
    const double Pxf = Px + dPx;
    const double f2 = fma(-Pxf, Pxf, Pa2);
    bad |= !is_pos(f2);
    const double y = rsqrt_nr(f2);
    const double Af = f2 * y;
    const double rr = (Px + Pxf) * rcp_nr(Af + A);
    X = fma(g, fma(-sk, rr, ck), fma(Px, fma(ck, rr, sk), X));
    Am1 = fma(-dPx, rr, Am1);
    Px = Pxf; A = Af; iA = y;
  }
  template <bool DKSKD> __device__ __forceinline__ void pwc_first() { advance(); }     // exact map: half slice
  template <bool DKSKD> __device__ __forceinline__ void pwc_second() { advance(); }
  // Omega = -(1+hX)/Ps [a1 b - a2 (u.b) u] + h y-hat with b = (0, k0, 0), Ps = A
  __device__ __forceinline__ void omega(double w, double& wx, double& wy, double& ws) const {
    const double fw = fma(h, X, 1.0) * iA * w;
    const double fq = fw * q2;
    wx = fq * Px;
    wy = fma(-fw, a1k, w * h);
    ws = fq * A;
  }
};

static __constant__ double APOLY[6] = {1.0 / 6.0, 3.0 / 40.0, 15.0 / 336.0, 105.0 / 3456.0, 945.0 / 42240.0, 10395.0 / 599040.0};

// asin(x): polynomial for the small arguments of differences of nearby angles, the library routine otherwise
__device__ __forceinline__ double asin_small(double x) {
  const double v = x * x;
  if (v < 2.5e-3) {     // asin(x)/x = 1 + v/6 + 3v^2/40 + 15v^3/336 + 105v^4/3456 + 945v^5/42240 + 10395v^6/599040
    double p = APOLY[5];
    p = fma(p, v, APOLY[4]);
    p = fma(p, v, APOLY[3]);
    p = fma(p, v, APOLY[2]);
    p = fma(p, v, APOLY[1]);
    p = fma(p, v, APOLY[0]);
    return fma(p * v, x, x);
  }
  return asin(x);
}

template <class Spin>
__device__ __forceinline__ bool sbend_exact(State& z, const DevElem& e, const PCon& c, const Ref& r, Spin& spin) {
  BendExact s(z, e, c, r);
  const double A0 = s.A, Am1_0 = s.Am1, Px0 = z.Px;
  spin.run(s, e.N, e.ds);
  // asin(Px0/Pa) - asin(PxN/Pa) = asin(x),  x = (Px0 A_N - Px_N A_0)/Pa^2  (no cancellation)
  const double x = fma(Px0, s.Am1 - Am1_0, -(z.Px - Px0) * A0) * rcp_nr(s.Pa2);
  const double dasin = asin_small(x);
  const double dh = dasin * e.inv_h;
  z.Y = fma(z.Py * e.inv_eta, e.L + dh, z.Y);
  z.T += e.inv_eta * (fma(-z.Pt, e.L, -c.ibpt * dh) - e.ome * e.L * r.ibeta0);
  return !s.bad;
}

// a5: TEAPOT sector bend (30)(31): half curved drift, kick -ds k0 (1+hX), half curved drift.
// The curved drift is a straight line seen from the rotating frame, so (Px,Ps) simply rotate by
// phi = h ds/2; X, Y, T use rho(sec phi - 1), rho tan phi and rho(tan phi - phi) from the host.
template <int ORDER> struct BendTeapot {
  static constexpr bool SMALL_ANGLE = false;
  State& z;
  const DevElem& e;
  const PCon& c;
  double Ps, iPs, pa2, q2, a1k;
  bool bad;
  __device__ __forceinline__ BendTeapot(State& z_, const DevElem& e_, const PCon& c_, const Ref& r) : z(z_), e(e_), c(c_) {
    const Mom m = mom_of(z, c);
    if (e.Lpre != 0.0) drift_with(z, e.Lpre, m, rcp_nr(m.Ps + 1.0), c, r);
    pa2 = fma(-z.Py, z.Py, 1.0 + c.e0);
    bad = !m.ok;
    iPs = m.iPs;
    Ps = m.Ps;
    q2 = c.a2p * e.k0 * z.Py;
    a1k = fma(c.a1, e.k0, -q2 * z.Py);
  }
  // curved drift (31) of length t.len; on entry iPs = 1/Ps
  __device__ __forceinline__ void curved_drift(const TeapotHalf& t) {
    const double xp = z.Px * iPs;
    const double D = fma(-xp, t.t, 1.0);
    bad |= !is_pos(D);
    const double iD = rcp_nr(D);
    // delta q = [(rho+X) tan phi - len Ps D]/(Ps D)
    const double num = t.r_tanmphi + fma(z.X, t.t, t.len * fma(z.Px, t.t, -(Ps - 1.0)));
    const double dq = num * iPs * iD;
    z.X = (t.r_secm1 + fma(z.X, t.sec, t.r_tan * xp)) * iD;
    z.Y = fma(z.Py, t.len + dq, z.Y);
    z.T += fma(-z.Pt, t.len, -c.ibpt * dq);
    const double Pxn = fma(z.Px, t.c, Ps * t.s);
    Ps = fma(Ps, t.c, -z.Px * t.s);
    z.Px = Pxn;
    bad |= !is_pos(Ps);
  }
  // kick of (30c) over `len`, then the new longitudinal momentum
  __device__ __forceinline__ void kick(double len) {
    z.Px = fma(-len * e.k0, fma(e.h, z.X, 1.0), z.Px);
    const double ps2 = fma(-z.Px, z.Px, pa2);
    bad |= !is_pos(ps2);
    iPs = rsqrt_nr(ps2);
    Ps = ps2 * iPs;
  }
  __device__ __forceinline__ void advance() {
    iPs = rcp_nr(Ps);
    if (ORDER == 2) {
      curved_drift(e.th[0]);
      kick(e.ds);
      curved_drift(e.th[0]);
    } else {
      curved_drift(e.th[1]);
      kick(GST_YOSHIDA_X1 * e.ds);
      curved_drift(e.th[2]);
      kick(GST_YOSHIDA_X0 * e.ds);
      curved_drift(e.th[2]);
      kick(GST_YOSHIDA_X1 * e.ds);
      curved_drift(e.th[1]);
    }
  }
  // mid-slice PWC (37): the element table is derived for HALF slices (e.ds = half the spin slice)
  template <bool DKSKD> __device__ __forceinline__ void pwc_first() {
    if (DKSKD) { iPs = rcp_nr(Ps); curved_drift(e.th[3]); kick(e.ds); } else advance();
  }
  template <bool DKSKD> __device__ __forceinline__ void pwc_second() {
    if (DKSKD) { kick(e.ds); curved_drift(e.th[3]); } else advance();
  }
  __device__ __forceinline__ void omega(double w, double& wx, double& wy, double& ws) const {
    const double fw = fma(e.h, z.X, 1.0) * rcp_nr(Ps) * w;
    const double fq = fw * q2;
    wx = fq * z.Px;
    wy = fma(-fw, a1k, w * e.h);
    ws = fq * Ps;
  }
};
template <int ORDER, class Spin>
__device__ __forceinline__ bool sbend_teapot(State& z, const DevElem& e, const PCon& c, const Ref& r, Spin& spin) {
  BendTeapot<ORDER> s(z, e, c, r);
  spin.run(s, e.N, e.ds);
  return !s.bad;
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

// a9 for straight elements (h = 0):  w Omega = -(w/Ps)[a1 b - a2 (u.b) u],  b = (bx, by, 0)
__device__ __forceinline__ void omega_straight(double w, double Px, double Py, double iPs, double bx, double by,
                                               const PCon& c, double& wx, double& wy, double& ws) {
  const double pb = c.a2p * fma(Px, bx, Py * by);
  const double wi = -w * iPs;
  wx = wi * fma(c.a1, bx, -pb * Px);
  wy = wi * fma(c.a1, by, -pb * Py);
  ws = w * pb;
}

// a7: drift-kick multipole (29): half drift, kick (28), half drift.  The momenta are constant
// between kicks, so one 1/Ps serves the second half drift, the edge Omega and the next first half.
// PURE = quadrupole term only (the common case): field and kick collapse to two FMAs.
template <bool PURE, int ORDER> struct MultDK {
  static constexpr bool SMALL_ANGLE = true;
  State& z;
  const DevElem& e;
  const PCon& c;
  double iPs, tnum, hds, k1, dsk, a1k, a2k, ibeta0, P2;
  bool bad;
  // T' = 1/beta0 - (1/beta0+Pt)/Ps is formed directly here: its rounding error is 2^-53 * (ds/2) per half
  // drift in ABSOLUTE terms (a few 1e-18 m), far below 1e-12 of any bunch length;
  // the cancellation-free form (one more MUFU + 14 FP64 instructions per slice) is kept for whole drifts.
  __device__ __forceinline__ void momenta() {
    const double ps2 = P2 - fma(z.Px, z.Px, z.Py * z.Py);
    bad |= !is_pos(ps2);
    iPs = rsqrt_nr(ps2);
    tnum = fma(-c.ibpt, iPs, ibeta0);
  }
  __device__ __forceinline__ MultDK(State& z_, const DevElem& e_, const PCon& c_, const Ref& r) : z(z_), e(e_), c(c_) {
    hds = 0.5 * e.ds;
    k1 = e.kn[0];
    dsk = e.ds * k1;
    a1k = c.a1 * k1;
    a2k = c.a2p * k1;
    ibeta0 = r.ibeta0;
    P2 = 1.0 + c.e0;
    const Mom m = mom_of(z, c);                    // shared with the drift space merged in front of the magnet
    if (e.Lpre != 0.0) drift_with(z, e.Lpre, m, rcp_nr(m.Ps + 1.0), c, r);
    bad = !m.ok;
    iPs = m.iPs;
    tnum = fma(-c.ibpt, iPs, ibeta0);
  }
  __device__ __forceinline__ void drift_by(double len) {
    const double l = len * iPs;
    z.X = fma(l, z.Px, z.X);
    z.Y = fma(l, z.Py, z.Y);
    z.T = fma(len, tnum, z.T);
  }
  __device__ __forceinline__ void kick_by(double len, double lenk) {    // lenk = len * k1
    if (PURE) {
      z.Px = fma(-lenk, z.X, z.Px);
      z.Py = fma(lenk, z.Y, z.Py);
    } else {
      double bx, by;
      mult_field(e, z.X, z.Y, bx, by);
      z.Px = fma(-len, by, z.Px);
      z.Py = fma(len, bx, z.Py);
    }
    momenta();
  }
  __device__ __forceinline__ void advance() {
    if (ORDER == 2) {
      drift_by(hds);
      kick_by(e.ds, dsk);
      drift_by(hds);
    } else {
      drift_by(GST_YOSHIDA_X1 * hds);
      kick_by(GST_YOSHIDA_X1 * e.ds, GST_YOSHIDA_X1 * dsk);
      drift_by((GST_YOSHIDA_X1 + GST_YOSHIDA_X0) * hds);
      kick_by(GST_YOSHIDA_X0 * e.ds, GST_YOSHIDA_X0 * dsk);
      drift_by((GST_YOSHIDA_X1 + GST_YOSHIDA_X0) * hds);
      kick_by(GST_YOSHIDA_X1 * e.ds, GST_YOSHIDA_X1 * dsk);
      drift_by(GST_YOSHIDA_X1 * hds);
    }
  }
  template <bool DKSKD> __device__ __forceinline__ void pwc_first() {
    if (DKSKD) { drift_by(e.ds); kick_by(e.ds, dsk); } else advance();
  }
  template <bool DKSKD> __device__ __forceinline__ void pwc_second() {
    if (DKSKD) { kick_by(e.ds, dsk); drift_by(e.ds); } else advance();
  }
  __device__ __forceinline__ void omega(double w, double& wx, double& wy, double& ws) const {
    if (PURE) {     // (6b) with b = k1 (Y, X, 0): w Omega = -(w a1 k1/Ps)(Y, X, 0) + (w g d/Ps)(Px, Py, Ps), g d = a2' (u.b) P
      const double d = fma(z.Px, z.Y, z.Py * z.X);
      const double wa = (w * a1k) * iPs, wg = (w * a2k) * d;
      const double t = wg * iPs;
      wx = fma(t, z.Px, -wa * z.Y);
      wy = fma(t, z.Py, -wa * z.X);
      ws = wg;
    } else {
      double bx, by;
      mult_field(e, z.X, z.Y, bx, by);
      omega_straight(w, z.Px, z.Py, iPs, bx, by, c, wx, wy, ws);
    }
  }
};
template <int ORDER, class Spin>
__device__ __forceinline__ bool mult_dk(State& z, const DevElem& e, const PCon& c, const Ref& r, Spin& spin) {
  if (e.pure_quad) {
    MultDK<true, ORDER> s(z, e, c, r);
    spin.run(s, e.N, e.ds);
    return !s.bad;
  }
  MultDK<false, ORDER> s(z, e, c, r);
  spin.run(s, e.N, e.ds);
  return !s.bad;
}

// a6: quadrupole matrix-kick (24)(25)(27).  kappa^2 = |k1|/P (23); with u = (kappa ds/2)^2 the four
// functions cos, sin(x)/x, cosh, sinh(x)/x are power series in u (no sqrt of kappa is needed).
// One plane of the linear flow (24a-d) and of its time-of-flight form (24e):
//   u' = C u + S p,  p' = C p - k u;   T' contribution -(1/beta_o + Pt)/P (pp p^2 + xx u^2 + xp u p).
// For the plane the magnet focuses C = cos x, S = (s/P) sin(x)/x, k = |k1| s sin(x)/x; for the other one the hyperbolic
// functions and k < 0 (A11: the paper's rotation by 90 degrees).  Which plane is which is decided by the sign of k1 when
// the coefficients are built, so that ONE copy of the slice loop serves both polarities: the loop instantiated once per
// polarity put the matrix-kick kernels over the instruction cache (19 % of the warp samples waited for instructions).
struct QuadPlane { double C, S, k, pp, xx, xp; };
struct QuadLin { QuadPlane x, y; };
__device__ __forceinline__ void quadlin_build(QuadLin& q, double k1, double s, const PCon& c) {
  const double ak1 = fabs(k1);
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
  const double s4 = 0.25 * s, iP2 = c.iP * c.iP;
  const double SC = Sx * C, ShC = Shx * Ch;          // sin(2x)/(2x), sinh(2x)/(2x)
  QuadPlane f, d;
  f.C = C;  f.S = s * c.iP * Sx;   f.k = ak1 * s * Sx;       // X += (s/P) Px sin(x)/x,  Px -= kappa^2 P s X sin(x)/x
  d.C = Ch; d.S = s * c.iP * Shx;  d.k = -ak1 * s * Shx;     // kappa^2 P = |k1|
  f.pp = s4 * iP2 * (1.0 + SC);   f.xx = s4 * kap2 * (1.0 - SC);   f.xp = -0.5 * u * Sx * Sx * c.iP;
  d.pp = s4 * iP2 * (1.0 + ShC);  d.xx = s4 * kap2 * (ShC - 1.0);  d.xp = 0.5 * u * Shx * Shx * c.iP;
  const bool foc_x = k1 > 0.0;
  q.x = foc_x ? f : d;
  q.y = foc_x ? d : f;
}
// flow of H_qL over the length the coefficients were built for
__device__ __forceinline__ void quadlin_apply(const QuadLin& q, State& z, double tfac) {
  const double curly = fma(q.x.pp, z.Px * z.Px, fma(q.x.xx, z.X * z.X, q.x.xp * z.X * z.Px)) +
                       fma(q.y.pp, z.Py * z.Py, fma(q.y.xx, z.Y * z.Y, q.y.xp * z.Y * z.Py));
  z.T = fma(-tfac, curly, z.T);
  double nu = fma(z.X, q.x.C, q.x.S * z.Px);
  z.Px = fma(z.Px, q.x.C, -q.x.k * z.X);
  z.X = nu;
  nu = fma(z.Y, q.y.C, q.y.S * z.Py);
  z.Py = fma(z.Py, q.y.C, -q.y.k * z.Y);
  z.Y = nu;
}
// 1/Ps for a particle of total momentum P and transverse momentum pt: with eps = pt^2/P^2,
//   1/Ps = (1/P)(1 - eps)^(-1/2) = (1/P)[1 + eps h(eps)],  h = 1/2 + 3/8 eps + 5/16 eps^2 + 35/128 eps^3 + ...
// In a quadrupole P is a constant of the element, so the kick of H_qNL (25) and the 1/Ps of Omega need neither a
// reciprocal square root nor a reciprocal while eps <= 2^-13 (angles up to 11 mrad; the truncation error of h is then
// 63/256 eps^4 = 5e-17, half an ulp): (25a) uses 1/Ps - 1/P = eps h/P, (25e)'s bracket 1/Ps - 1/P - pt^2/(2P^3) =
// eps^2 (3/8 + 5/16 eps + 35/128 eps^2)/P.  Larger angles take the exact forms, out of line.
#define GST_MK_EPS_MAX 1.220703125e-4   // 2^-13
struct QuadNL { double d, br, iPs; bool ok; };   // 1/Ps - 1/P, the bracket of (25e), 1/Ps
static __device__ __noinline__ QuadNL quadnl_exact(double pt2, double P, double iP) {
  QuadNL r;
  const double ps2 = fma(P, P, -pt2);
  r.ok = is_pos(ps2);
  r.iPs = rsqrt_nr(ps2);
  const double Ps = ps2 * r.iPs;
  const double t = r.iPs * rcp_nr(P + Ps);           // 1/(Ps (P+Ps))
  r.d = pt2 * iP * t;                                // 1/Ps - 1/P = pt2/(P Ps (P+Ps))
  r.br = pt2 * pt2 * fma(2.0, P, Ps) * (0.5 * iP * iP * iP) * t * (t * Ps);   // pt2^2 (2P+Ps)/(2 P^3 Ps (P+Ps)^2)
  return r;
}
template <int ORDER> struct QuadMK {
  static constexpr bool SMALL_ANGLE = true;
  State& z;
  const PCon& c;
  QuadLin ql;       // linear flow over ds/2 (second order) or x1 ds/2 (fourth order)
  QuadLin ql2;      // fourth order only: linear flow over (x1 + x0) ds/2 < 0
  double k1, ds, tfac, iP2, a1k;
  bool bad;
  __device__ __forceinline__ QuadMK(State& z_, const DevElem& e, const PCon& c_) : z(z_), c(c_) {
    k1 = e.kn[0];
    ds = e.ds;
    if (ORDER == 2) {
      quadlin_build(ql, k1, 0.5 * e.ds, c);
    } else {
      quadlin_build(ql, k1, (0.5 * GST_YOSHIDA_X1) * e.ds, c);
      quadlin_build(ql2, k1, (0.5 * (GST_YOSHIDA_X1 + GST_YOSHIDA_X0)) * e.ds, c);
    }
    tfac = c.iP * c.ibpt;
    iP2 = c.iP * c.iP;
    a1k = c.a1 * k1;
    bad = false;
  }
  __device__ __forceinline__ void lin(const QuadLin& q) { quadlin_apply(q, z, tfac); }
  // (25) over `len`: X += len Px (1/Ps - 1/P);  T' = -(1/beta0+Pt)[1/Ps - 1/P - pt2/(2P^3)] + tq
  __device__ __forceinline__ void nonlinear(double len) {
    const double pt2 = fma(z.Px, z.Px, z.Py * z.Py);
    const double eps = pt2 * iP2;
    const double ie = c.iP * eps;
    const double h2 = fma(fma(35.0 / 128.0, eps, 5.0 / 16.0), eps, 3.0 / 8.0);
    double d = ie * fma(h2, eps, 0.5);
    double br = ie * eps * h2;
    if (__builtin_expect(!(eps <= GST_MK_EPS_MAX), 0)) {
      const QuadNL x = quadnl_exact(pt2, c.P, c.iP);
      d = x.d; br = x.br;
      bad |= !x.ok;
    }
    z.X = fma(len * d, z.Px, z.X);
    z.Y = fma(len * d, z.Py, z.Y);
    z.T = fma(len, fma(-c.ibpt, br, c.tq), z.T);
  }
  __device__ __forceinline__ void advance() {
    if (ORDER == 2) {
      lin(ql);
      nonlinear(ds);
      lin(ql);
    } else {
      lin(ql);
      nonlinear(GST_YOSHIDA_X1 * ds);
      lin(ql2);
      nonlinear(GST_YOSHIDA_X0 * ds);
      lin(ql2);
      nonlinear(GST_YOSHIDA_X1 * ds);
      lin(ql);
    }
  }
  template <bool DKSKD> __device__ __forceinline__ void pwc_first() { advance(); }     // not a drift-kick map: half slice
  template <bool DKSKD> __device__ __forceinline__ void pwc_second() { advance(); }
  __device__ __forceinline__ void omega(double w, double& wx, double& wy, double& ws) {
    const double pt2 = fma(z.Px, z.Px, z.Py * z.Py);
    const double eps = pt2 * iP2;
    double iPs = fma(c.iP * eps, fma(fma(fma(35.0 / 128.0, eps, 5.0 / 16.0), eps, 3.0 / 8.0), eps, 0.5), c.iP);
    if (__builtin_expect(!(eps <= GST_MK_EPS_MAX), 0)) {
      const QuadNL x = quadnl_exact(pt2, c.P, c.iP);
      iPs = x.iPs;
      bad |= !x.ok;
    }
    const double pb = c.a2p * k1 * (z.Px * z.Y + z.Py * z.X);
    const double wi = -w * iPs;
    wx = wi * fma(a1k, z.Y, -pb * z.Px);
    wy = wi * fma(a1k, z.X, -pb * z.Py);
    ws = w * pb;
  }
};
template <int ORDER, class Spin>
__device__ __forceinline__ bool quad_mk(State& z, const DevElem& e, const PCon& c, Spin& spin) {
  QuadMK<ORDER> s(z, e, c);
  spin.run(s, e.N, e.ds);
  return !s.bad;
}

// ---------------------------------------------------------------------------------------------
// one element (the dispatch is uniform across the grid: every particle is in the same element)
// ---------------------------------------------------------------------------------------------
// f3: rectangular bend (section 3.2).  e.k0 = 1/rho_b; all coordinates between the two rotations are
// internal to the magnet (Cartesian frame along its axis).
struct BendRect {
  static constexpr bool SMALL_ANGLE = false;     // body (13): Px falls linearly, X follows sqrt(Pa^2 - Px^2); Y, T once per element
  State& z;
  double k0, ds, Pa2, A, iA, q2, a1k;
  bool bad;
  __device__ __forceinline__ BendRect(State& z_, const DevElem& e, const PCon& c) : z(z_), k0(e.k0), ds(e.ds) {
    Pa2 = fma(-z.Py, z.Py, 1.0 + c.e0);                    // (8)
    const double a2 = fma(-z.Px, z.Px, Pa2);
    bad = !is_pos(a2);
    iA = rsqrt_nr(a2);
    A = a2 * iA;
    q2 = c.a2p * e.k0 * z.Py;
    a1k = fma(c.a1, e.k0, -q2 * z.Py);
  }
  __device__ __forceinline__ void advance() {
    const double Pxf = fma(-ds, k0, z.Px);                 // (13b)
    const double f2 = fma(-Pxf, Pxf, Pa2);
    bad |= !is_pos(f2);
    const double y = rsqrt_nr(f2);
    const double Af = f2 * y;
    // (13a): rho_b (A_f - A) = rho_b (Px - Px_f)(Px + Px_f)/(A_f + A) = ds (Px + Px_f)/(A_f + A)
    z.X = fma(ds * (z.Px + Pxf), rcp_nr(Af + A), z.X);
    z.Px = Pxf; A = Af; iA = y;
  }
  template <bool DKSKD> __device__ __forceinline__ void pwc_first() { advance(); }
  template <bool DKSKD> __device__ __forceinline__ void pwc_second() { advance(); }
  // (6b) with h = 0, b = (0, k0, 0), Ps = A
  __device__ __forceinline__ void omega(double w, double& wx, double& wy, double& ws) const {
    const double fw = iA * w;
    const double fq = fw * q2;
    wx = fq * z.Px;
    wy = -fw * a1k;
    ws = fq * A;
  }
};
// dynamic rotation (17) about y-hat; k = 0: by phi_entr, k = 1: by -phi_exit (constants from the host)
__device__ __forceinline__ bool rbend_rotate(State& z, const DevElem& e, int k, const PCon& c) {
  const double ps2 = 1.0 + c.e0 - fma(z.Px, z.Px, z.Py * z.Py);
  const double iPs = rsqrt_nr(ps2);
  const double Ps = ps2 * iPs;
  const double den = fma(-z.Px * iPs, e.rb_t[k], 1.0);
  const double q = z.X * e.rb_t[k] * rcp_nr(den);
  z.Y = fma(z.Py * iPs, q, z.Y);                           // (17c)
  z.T = fma(-c.ibpt * iPs, q, z.T);                        // (17e), sign of reading A5
  z.X = z.X * e.rb_sec[k] * rcp_nr(den);                   // (17a)
  z.Px = fma(z.Px, e.rb_c[k], Ps * e.rb_s[k]);             // (17b)
  return is_pos(ps2) && is_pos(den);
}
// thin-fringe orbit map (15), b = +-k0
__device__ __forceinline__ bool rbend_fringe(State& z, double b, const PCon& c) {
  const double ps2 = 1.0 + c.e0 - fma(z.Px, z.Px, z.Py * z.Py);
  const double iPs = rsqrt_nr(ps2);
  const double xp = z.Px * iPs, yp = z.Py * iPs;
  const double id = rcp_nr(fma(yp, yp, 1.0));
  const double arg = fma(2.0 * b * xp * yp * id, z.Y, 1.0);
  const double Yf = 2.0 * z.Y * rcp_nr(1.0 + arg * rsqrt_nr(arg));                                  // (15c)
  const double Y2 = Yf * Yf;
  z.X = fma(0.5 * b * iPs * (fma(xp, xp, 1.0) * id - 2.0 * xp * xp * yp * yp * id * id), Y2, z.X);  // (15a)
  z.Py = fma(-b * xp * id, Yf, z.Py);                                                               // (15d)
  z.T = fma(-0.5 * b * c.ibpt * xp * iPs * iPs * fma(-yp, yp, 1.0) * id * id, Y2, z.T);             // (15e)
  z.Y = Yf;
  return is_pos(ps2) && is_pos(arg);
}
template <class Spin>
__device__ __forceinline__ bool rbend(State& z, const DevElem& e, const PCon& c, const Ref& r, double G, Spin& spin) {
  bool ok = rbend_rotate(z, e, 0, c);
  spin.snake(Quat{e.rb_qw[0], 0.0, e.rb_qy[0], 0.0});
  const double g1 = c.a2p * (1.0 + c.e0);                   // G (gamma - 1)
  // entrance: spin kick (42) (with the length Y in its x-hat term, R10), then the orbit map (15)
  spin.thin(e.k0 * g1 * z.Px * z.Y, 0.0, -e.k0 * (1.0 + G) * z.Y);
  ok &= rbend_fringe(z, e.k0, c);
  BendRect s(z, e, c);
  const double A0 = s.A, Px0 = z.Px;
  spin.run(s, e.N, e.ds);
  {   // Y (13c) and T (13e) + (19) over the whole body.  d = asin(Px0/Pa) - asin(PxN/Pa):
      //   sin d = (Px0 A_N - Px_N A_0)/Pa^2,  cos d = (A_0 A_N + Px0 Px_N)/Pa^2;
      // delta = d - (phi_entr - phi_exit) from sin delta = sin d cos D - cos d sin D, so that
      //   T: -(1/beta_o + Pt) rho_b d + L_arc/beta_o = -(1/beta_o + Pt) rho_b delta - Pt L_arc   (no O(1) cancellation)
    const double iPa2 = rcp_nr(s.Pa2);
    const double sd = fma(Px0, s.A, -z.Px * A0) * iPa2, cd = fma(A0, s.A, Px0 * z.Px) * iPa2;
    const double delta = asin_small(fma(sd, e.rb_cd, -cd * e.rb_sd));
    z.Y = fma(z.Py, fma(e.rb_rho, delta, e.rb_arc), z.Y);
    z.T = fma(-c.ibpt * e.rb_rho, delta, fma(-z.Pt, e.rb_arc, z.T));
  }
  ok &= !s.bad;
  ok &= rbend_fringe(z, -e.k0, c);
  spin.thin(-e.k0 * g1 * z.Px * z.Y, 0.0, e.k0 * (1.0 + G) * z.Y);
  z.X -= e.rb_xoff;                                         // (18)
  ok &= rbend_rotate(z, e, 1, c);
  spin.snake(Quat{e.rb_qw[1], 0.0, e.rb_qy[1], 0.0});
  (void)r;
  return ok;
}

// f4: solenoid with thin-pancake fringes (section 3.7).  e.k0 = b_0/(B rho)_o, eta = k0/2 (35).
// The body flow (34) is exact, so a slice is the same map over ds; Ps of (33) is an invariant of it, which
// makes kappa = eta/Ps and cos/sin(kappa ds) per-particle constants of the element, and lets T (34c) be
// applied once (cancellation-free as in drift()).  Omega (6b) takes u-hat from the kinetic momentum (36).
struct Solenoid {
  static constexpr bool SMALL_ANGLE = false;
  State& z;
  const PCon& c;
  double eta, cs, sn, sn_eta, eta_sn, iPs, Ps, two_eta;
  bool bad;
  __device__ __forceinline__ Solenoid(State& z_, const DevElem& e, const PCon& c_) : z(z_), c(c_) {
    eta = 0.5 * e.k0;
    two_eta = e.k0;
    const double kx = fma(eta, z.Y, z.Px), ky = fma(-eta, z.X, z.Py);
    const double ps2 = 1.0 + c.e0 - fma(kx, kx, ky * ky);
    bad = !is_pos(ps2);
    iPs = rsqrt_nr(bad ? 1.0 : ps2);
    Ps = ps2 * iPs;
    sincos(eta * iPs * e.ds, &sn, &cs);
    sn_eta = sn / eta;
    eta_sn = eta * sn;
  }
  __device__ __forceinline__ void advance() {      // R2 R1 of (34a)(34b)
    const double X1 = fma(cs, z.X, sn_eta * z.Px), P1 = fma(cs, z.Px, -eta_sn * z.X);
    const double Y1 = fma(cs, z.Y, sn_eta * z.Py), Q1 = fma(cs, z.Py, -eta_sn * z.Y);
    z.X = fma(cs, X1, sn * Y1);   z.Px = fma(cs, P1, sn * Q1);
    z.Y = fma(cs, Y1, -sn * X1);  z.Py = fma(cs, Q1, -sn * P1);
  }
  template <bool DKSKD> __device__ __forceinline__ void pwc_first() { advance(); }
  template <bool DKSKD> __device__ __forceinline__ void pwc_second() { advance(); }
  // w Omega, b = (0, 0, 2 eta):  (2 eta a2' kx, 2 eta a2' ky, 2 eta (a2' Ps - a1/Ps)),  a2' = G(gamma-1)/P^2
  __device__ __forceinline__ void omega(double w, double& wx, double& wy, double& ws) const {
    const double kx = fma(eta, z.Y, z.Px), ky = fma(-eta, z.X, z.Py);
    const double f = w * two_eta * c.a2p;
    wx = f * kx;
    wy = f * ky;
    ws = fma(f, Ps, -w * two_eta * c.a1 * iPs);
  }
  // thin-pancake fringe spin kick (40) P:553: sign = +1 entrance, -1 exit; kinetic momentum and Ps with A/2
  __device__ __forceinline__ void fringe(double sign, double& wx, double& wy, double& ws) {
    const double kx = fma(0.5 * eta, z.Y, z.Px), ky = fma(-0.5 * eta, z.X, z.Py);
    const double ps2 = 1.0 + c.e0 - fma(kx, kx, ky * ky);
    bad |= !is_pos(ps2);
    const double ips = rsqrt_nr(ps2);
    const double proj = c.a2p * fma(z.X, kx, z.Y * ky);       // G(gamma-1)(X kx + Y ky)/P^2
    const double pre = sign * eta * ips;
    wx = pre * fma(c.a1, z.X, -proj * kx);
    wy = pre * fma(c.a1, z.Y, -proj * ky);
    ws = -sign * eta * proj;                                   // pre * (-proj * Ps')
  }
};
template <class Spin>
__device__ __forceinline__ bool solenoid(State& z, const DevElem& e, const PCon& c, const Ref& r, Spin& spin) {
  Solenoid s(z, e, c);
  double wx, wy, ws;
  s.fringe(+1.0, wx, wy, ws);
  spin.thin(wx, wy, ws);
  spin.run(s, e.N, e.ds);
  s.fringe(-1.0, wx, wy, ws);
  spin.thin(wx, wy, ws);
  // (34c) over the whole length, with the kinetic transverse momentum (an invariant of the body flow)
  const double kx = fma(s.eta, z.Y, z.Px), ky = fma(-s.eta, z.X, z.Py);
  const double pt2 = fma(kx, kx, ky * ky);
  const double ps2m1 = c.e0 - pt2;
  const double iPs1 = rcp_nr(s.Ps + 1.0);
  const double num = (fma(-pt2, r.ibeta0, c.tA) - z.Pt * ps2m1 * iPs1) * iPs1;
  z.T = fma(e.L * s.iPs, num, z.T);
  return !s.bad;
}

static __constant__ double FRINGE_INV_M[4] = {1.0 / 2.0, 1.0 / 3.0, 1.0 / 4.0, 1.0 / 5.0};

// the element types that take a merged drift space in front of them the plain way (see element_step)
template <int SPLIT, int ORDER, class Spin>
__device__ __forceinline__ bool element_step_other(int type, State& z, const DevElem& e, PCon& pc, Ref& ref, double G, Spin& spin) {
  if (SPLIT == SPLIT_MK && type == K_QUAD) return quad_mk<ORDER>(z, e, pc, spin);   // the other splits never get here with a quadrupole
  if (type == K_THIN) {   // A10: half kick, spin, half kick
    double bx, by, wx, wy, ws;
    mult_field(e, z.X, z.Y, bx, by);
    z.Px = fma(-0.5, by, z.Px);
    z.Py = fma(0.5, bx, z.Py);
    const double ps2 = 1.0 + pc.e0 - fma(z.Px, z.Px, z.Py * z.Py);
    const bool ok = is_pos(ps2);
    omega_straight(1.0, z.Px, z.Py, rsqrt_nr(ok ? ps2 : 1.0), bx, by, pc, wx, wy, ws);
    spin.thin(wx, wy, ws);
    z.Px = fma(-0.5, by, z.Px);
    z.Py = fma(0.5, bx, z.Py);
    return ok;
  }
  if (type == K_RF) {     // A12, A13
    double krf = e.krf_over_beta * ref.beta0;
    double dE = e.volt * sin(fma(e.sign * krf, z.T, e.phi_s));
    // E - E0' = p0c Pt + dE - dEs: the O(E0) terms are never formed
    double num = fma(ref.p0c, z.Pt, dE - e.dEs);
    if (e.dEs != 0.0) {
      double p0_old = ref.p0c;
      double E0 = ref.E0;
      ref_energy_add(E0, ref.E0lo, e.dEs);
      ref_set(ref, E0, ref.mass);
      double sc = p0_old / ref.p0c;
      z.Px *= sc; z.Py *= sc;
    }
    z.Pt = num / ref.p0c;
    pcon_set(pc, z.Pt, ref, G);
    return true;
  }
  if (type == K_SNAKE) spin.snake(Quat{e.qw, e.qx, e.qy, e.qs});
  if (type == K_SOLENOID) return solenoid(z, e, pc, ref, spin);
  if (type == K_RBEND) return rbend(z, e, pc, ref, G, spin);
  if (type == K_FRINGE) {   // thin-fringe spin kick (41) P:561: rotation about s-hat, orbit untouched
    double re = z.X, im = z.Y;                       // (X + iY)^m
    double psi = e.k0 * im;                          // m = 1
    const int top = e.order;
    for (int m = 2; m <= top; ++m) {
      const double nre = fma(re, z.X, -im * z.Y), nim = fma(re, z.Y, im * z.X);
      re = nre; im = nim;
      psi = fma(fma(e.kn[m - 2], im, e.ks[m - 2] * re), FRINGE_INV_M[m - 2], psi);
    }
    spin.thin(0.0, 0.0, -e.sign * (1.0 + G) * psi);  // e.sign = +1 entering, -1 leaving
  }
  return true;
}

// One element of the COMPILED sequence (gst_api.cu: compile_lattice): drift spaces never come alone -- consecutive
// ones are merged and each run is handed to the element behind it as e.Lpre -- except at the end of the ring, and
// markers are gone.  Bends and drift-kick magnets take their Lpre themselves, sharing its square root with their own
// entrance values; every other type drifts first.  The tests are ordered by how often each type occurs in a ring.
template <int SPLIT, int ORDER, class Spin>
__device__ __forceinline__ bool element_step(int type, State& z, const DevElem& e, PCon& pc, Ref& ref, double G, Spin& spin) {
  if (type == K_QUAD && SPLIT != SPLIT_MK) return mult_dk<ORDER>(z, e, pc, ref, spin);
  if (type == K_SBEND) {
    if (SPLIT == SPLIT_DK) return sbend_teapot<ORDER>(z, e, pc, ref, spin);
    return sbend_exact(z, e, pc, ref, spin);
  }
  if (type == K_DRIFT) return drift(z, e.L, pc, ref);
  if (type == K_MULT) return mult_dk<ORDER>(z, e, pc, ref, spin);
  bool ok = true;
  if (e.Lpre != 0.0) ok = drift(z, e.Lpre, pc, ref);
  return element_step_other<SPLIT, ORDER>(type, z, e, pc, ref, G, spin) && ok;
}
// ---------------------------------------------------------------------------------------------
// the kernel
// ---------------------------------------------------------------------------------------------
// 64-thread blocks, <= 128 registers: the register file is split per SM sub-partition (16 384 each), so
// 128 registers allow 4 warps per sub-partition = 8 blocks per SM, and the 1024 blocks of a 65 536-
// particle bunch are resident in ONE wave (148 x 8 = 1184 slots).  With 144+ registers only 3 warps
// fit per sub-partition (888 slots) and the last 136 blocks run alone in a second wave (measured:
// 85 ms vs 53 ms per 20 turns, profiles/r01_notes.md).
constexpr int TRACK_BLOCK = 64;
constexpr int TRACK_MIN_BLOCKS = 8;
// The fourth-order matrix-kick and drift-kick maps (two coefficient tables; three kicks and four curved drifts per
// slice) spill 800 B per thread at 128 registers.  With 6 blocks per SM (3 warps per sub-partition, 168 registers) they
// measured 20 % and 5 % faster; fourth-order bend-kick is 3 % slower that way and stays at 8, like every second-order
// kernel.
// A bunch of at most two warps per sub-partition is not short of registers but of parallelism: one warp's dependency
// chains set the time.  The FAT variant is compiled for 4 blocks per SM (up to 255 registers; ptxas takes 170-190, no
// spills, more of the loop bodies in flight): measured +7 % (bend-kick) to +18 % (matrix-kick, with its two-edge loop
// bodies) on 4096-particle bunches, +7 % at 16 384.
constexpr int TRACK_FAT_BLOCKS = 4;
__host__ __device__ constexpr int track_min_blocks(int split, int order, bool fat) {
  return fat ? TRACK_FAT_BLOCKS : (order == 4 && split != SPLIT_BK) ? 6 : TRACK_MIN_BLOCKS;
}

// a0: the lattice is ALWAYS read from shared memory (LDS; element records and sequence entries through a pointer that
// may point to global or shared memory measured 3 % slower).  Two layouts of the dynamic shared memory, chosen on the
// host (track_launch.cuh: plan_smem) and compiled as two kernels:
//   RESIDENT   [unique-element table][sequence], staged once per block -- every BASELINE ring (12-20 records, <= 2.3 kB
//              of sequence); needs both to fit the block's budget
//   STREAMED   per warp [one DevElem][window of SEQ_WINDOW sequence entries]: the warp copies each element's record
//              from global memory before the element (3 coalesced loads per lane) and refills its window every
//              SEQ_WINDOW elements -- rings with hundreds of individually powered magnets or tens of thousands of elements
constexpr int SEQ_WINDOW = 64;
constexpr size_t STREAM_BYTES_PER_WARP = sizeof(DevElem) + SEQ_WINDOW * sizeof(uint32_t);

template <bool STREAMED>
__device__ __forceinline__ void stage_lattice(const TrackArgs& a, unsigned char* smem_raw) {
  if (!STREAMED) {
    const int nw = a.n_unique * (int)(sizeof(DevElem) / sizeof(double));
    const double* src = reinterpret_cast<const double*>(a.tab);
    double* dst = reinterpret_cast<double*>(smem_raw);
    for (int i = threadIdx.x; i < nw; i += blockDim.x) dst[i] = src[i];
    uint32_t* sseq = reinterpret_cast<uint32_t*>(smem_raw + (size_t)a.n_unique * sizeof(DevElem));
    for (int i = threadIdx.x; i < a.n_seq; i += blockDim.x) sseq[i] = a.seq[i];
  }
  __syncthreads();
}

// Turns [t0, t1) of the ring for one particle.  The turn and element loops run to the end for every thread of the
// warp (also for lanes without a particle, which carry a particle on the reference orbit), so that their counters, the
// sequence loads and the type dispatch are warp-uniform (uniform registers, no divergence bookkeeping) and the warp can
// copy element records together; a particle that is lost (A15) goes on with the reference orbit and nothing of it is
// stored (R6).
template <int SPLIT, int ORDER, bool STREAMED, class Spin>
__device__ __forceinline__ bool track_turns(State& z, Ref& ref, PCon& pc, Spin& spin, long long t0, long long t1,
                                            const TrackArgs& a, unsigned char* smem_raw) {
  bool lost = false;
  const int n_seq = a.n_seq;
  if (!STREAMED) {
    const DevElem* tab = reinterpret_cast<const DevElem*>(smem_raw);
    const uint32_t* seq = reinterpret_cast<const uint32_t*>(smem_raw + (size_t)a.n_unique * sizeof(DevElem));
    uint32_t nxt = seq[0];
    for (long long turn = t0; turn < t1; ++turn) {
#pragma unroll 1
      for (int ie = 0; ie < n_seq; ++ie) {
        const uint32_t cur = nxt;
        nxt = seq[ie + 1 < n_seq ? ie + 1 : 0];          // next element's entry, one element ahead
        const bool ok = element_step<SPLIT, ORDER>((int)(cur & 0xffu), z, tab[cur >> 8], pc, ref, a.G, spin);
        if (!ok) {
          lost = true;
          z.X = z.Px = z.Y = z.Py = z.T = z.Pt = 0.0;
          pcon_set(pc, 0.0, ref, a.G);
        }
      }
    }
  } else {
    const int lane = threadIdx.x & 31;
    unsigned char* mine = smem_raw + (threadIdx.x >> 5) * STREAM_BYTES_PER_WARP;
    double* rec = reinterpret_cast<double*>(mine);
    uint32_t* win = reinterpret_cast<uint32_t*>(mine + sizeof(DevElem));
    for (long long turn = t0; turn < t1; ++turn) {
#pragma unroll 1
      for (int ie = 0; ie < n_seq; ++ie) {
        if ((ie & (SEQ_WINDOW - 1)) == 0) {               // refill the window of sequence entries
          __syncwarp();
          for (int k = lane; k < SEQ_WINDOW && ie + k < n_seq; k += 32) win[k] = a.seq[ie + k];
          __syncwarp();
        }
        const uint32_t cur = win[ie & (SEQ_WINDOW - 1)];
        const double* src = reinterpret_cast<const double*>(a.tab + (cur >> 8));
        __syncwarp();                                     // everybody is done with the previous record
        for (int k = lane; k < (int)(sizeof(DevElem) / sizeof(double)); k += 32) rec[k] = src[k];
        __syncwarp();
        const bool ok = element_step<SPLIT, ORDER>((int)(cur & 0xffu), z, *reinterpret_cast<const DevElem*>(mine), pc, ref,
                                                   a.G, spin);
        if (!ok) {
          lost = true;
          z.X = z.Px = z.Y = z.Py = z.T = z.Pt = 0.0;
          pcon_set(pc, 0.0, ref, a.G);
        }
      }
    }
  }
  return lost;
}

template <int SPLIT, int DEPTH, int ORDER, bool STREAMED, bool FAT>
__global__ void __launch_bounds__(TRACK_BLOCK, track_min_blocks(SPLIT, ORDER, FAT)) track_kernel(const TrackArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  stage_lattice<STREAMED>(a, smem_raw);
  if (*a.err != 0) return;                               // an earlier launch on this bunch failed: leave everything (gst.h)
  const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = j < a.n && !a.lost[j];
  if (!__any_sync(0xffffffffu, valid)) return;           // a warp without particles (the other lanes keep in step)
  State z;
  z.X = z.Px = z.Y = z.Py = z.T = z.Pt = 0.0;
  z.Sx = 0.0; z.Sy = 1.0; z.Ss = 0.0;
  if (valid) {
    z.X = a.p[0][j]; z.Px = a.p[1][j]; z.Y = a.p[2][j]; z.Py = a.p[3][j]; z.T = a.p[4][j]; z.Pt = a.p[5][j];
    z.Sx = a.p[6][j]; z.Sy = a.p[7][j]; z.Ss = a.p[8][j];
  }
  Ref ref;
  ref_set(ref, a.E0, a.mass);
  ref.E0lo = a.E0lo;
  PCon pc;
  pcon_set(pc, z.Pt, ref, a.G);
  typename SpinPolicy<DEPTH, SPLIT, FAT>::type spin(z);
  const bool lost = track_turns<SPLIT, ORDER, STREAMED>(z, ref, pc, spin, 0, a.n_turns, a, smem_raw);
  if (!valid) return;
  if (lost) { a.lost[j] = 1; return; }
  a.p[0][j] = z.X; a.p[1][j] = z.Px; a.p[2][j] = z.Y; a.p[3][j] = z.Py; a.p[4][j] = z.T; a.p[5][j] = z.Pt;
  a.p[6][j] = z.Sx; a.p[7][j] = z.Sy; a.p[8][j] = z.Ss;
}

}  // namespace gst
