/* gst.h -- C ABI of the B200-native spin-orbit tracker (after arXiv:1501.03450, GPUSPINTRACK).
 *
 * The library tracks a bunch of spin-1/2 particles, one CUDA thread per particle, through
 * a ring lattice for many turns: symplectic orbital integration through every element
 * (section 3) followed by Thomas-BMT spin integration with quaternions and Romberg
 * extrapolation (section 4).  "P:nnn" cites /root/reference/PAPER.md line nnn; "(n)" an equation.
 *
 * Conventions
 *   - Phase space is MAD's canonical set (1) P:55: X, Px, Y, Py, T = -c dt, Pt = (E-E0)/(p0 c);
 *     momenta in units of the reference momentum p0.  Spin is a unit 3-vector with
 *     components along the local (x, y, s) axes: x radial-outward, y up, s along the beam.
 *   - All particle data are fp64, structure-of-arrays, in DEVICE memory owned by the caller
 *     (e.g. torch tensors); the library borrows the nine pointers and updates them in place.
 *   - Opaque handles; every call returns a gst_status; no exceptions or aborts cross the ABI.
 *     gst_last_error() gives a thread-local message for the last non-OK status.
 *   - Nothing here falls back to the CPU: without a CUDA device every compute call returns
 *     GST_ECUDA.
 *   - Devices: a lattice lives on the CUDA device that was current when it was created, a bunch on the
 *     device that owns its arrays; every entry point switches to that device for its own duration and
 *     restores the caller's, so several devices can be driven from one thread or from several.  A
 *     bunch can only be tracked through a lattice of its own device (GST_EINVAL); a stream argument
 *     must belong to that device.
 *   - Lost particles (R6): a particle is lost when a square-root argument or a
 *     curved-drift denominator of the maps below turns non-positive.  Its flag is set; from then on it
 *     is skipped by every gst_track and excluded from every reduction.  Its nine array entries keep
 *     the values they had when the gst_track call that lost it BEGAN (not the element-entrance values
 *     of SURVEY A15's wording): only the flag is specified.
 *   - Errors of an asynchronous launch: gst_track returns before its kernel runs, so a kernel that fails
 *     (the rotating launch of the same name, csrc/track_chain_kernel.cuh, gives up when the chip makes no
 *     progress for several seconds) cannot be reported by it.  The failure is recorded in the bunch:
 *     gst_track calls that are already enqueued behind it do nothing, and the NEXT call that
 *     synchronises (gst_bunch_status, gst_polarization, gst_emittance, gst_bunch_lost) returns
 *     GST_ECUDA once and clears the condition.  After that report the particle arrays are UNDEFINED
 *     (partly advanced) and the turn counter / reference energy are those of all calls enqueued: load a
 *     checkpoint into the arrays and call gst_bunch_set_reference before tracking on.
 */
#ifndef GST_H_
#define GST_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum { GST_OK = 0, GST_EINVAL = 1, GST_ENOMEM = 2, GST_ECUDA = 3, GST_ESTATE = 4 } gst_status;

/* element types: P:114-464 (orbit), P:585 (snake); RFCAV is DESIGN.md reading A12/A13 */
typedef enum {
  GST_DRIFT = 0,     /* exact drift, flow of H_drift (29b) P:371                                   */
  GST_SBEND = 1,     /* sector bend: exact flow (10) P:137, or TEAPOT drift-kick (30)(31) P:381     */
  GST_QUAD = 2,      /* quadrupole: matrix-kick (24)(25)(27) P:298-353, or drift-kick (29)          */
  GST_MULTIPOLE = 3, /* thick straight multipole, always drift-kick (28)(29) P:359-374              */
  GST_THINMULT = 4,  /* thin lens, "drift-kick without the drift" P:378                             */
  GST_RFCAV = 5,     /* thin RF cavity with optional reference-energy ramp                          */
  GST_SNAKE = 6,     /* Siberian snake: orbit-transparent thin spin rotation P:585                  */
  GST_MARKER = 7,
  GST_FRINGE = 8,    /* thin-fringe spin kick (41) P:561 of a magnet with body strengths k0 (dipole, m = 1), kn, ks
                        (m = 2..5, per unit length): rotation about s-hat by
                        -sign (1+G) [k0 Y + sum_m (kn Im (X+iY)^m + ks Re (X+iY)^m)/m]; sign = +1 at the
                        entrance, -1 at the exit; orbit-transparent (the paper gives no orbital fringe map)  */
  GST_SOLENOID = 9,  /* solenoid with thin-pancake fringes, section 3.7: k0 = b_0/(B rho)_o [1/m] (eta of (35)
                        is k0/2), L > 0; exact body flow (34) in n_slices*slice_mult slices for the spin scheme, Omega
                        with u-hat from the kinetic momentum (36), fringe spin kicks (40) at both ends; the orbit is
                        canonical throughout (the fringes leave the canonical momenta unchanged)             */
  GST_RBEND = 10     /* rectangular bend, section 3.2: L = magnet length along its axis, k0 = b_1/(B rho)_o =
                        1/rho_b, kn[0] = phi_entr, kn[1] = phi_exit (angles between the design orbit and the normals of
                        the two faces; sin(phi_entr) - sin(phi_exit) = L*k0, else GST_EINVAL).  Rotation (17) into the
                        magnet frame, fringe spin kick (42) and orbit map (15), body (13) in n_slices*slice_mult slices,
                        exit fringe, offset (18), rotation out, time offset (19)                                     */
} gst_elem_type;

/* which integrator each thick magnet uses (".apdf"; reading A16).  The *_4 values take the
 * same splits with every second-order slice map (27) replaced by the fourth-order symmetric composition
 * S2(x1 ds) S2(x0 ds) S2(x1 ds), x1 = 1/(2 - 2^(1/3)), x0 = 1 - 2 x1 ("higher-order versions of
 * (27)"; reading R5); exact maps (sector bends under bend-/matrix-kick, drifts) are unchanged, and the spin
 * integrator still samples Omega at the slice edges only.                                              */
typedef enum {
  GST_SPLIT_DRIFT_KICK = 0,    /* bends (30)(31), quads and multipoles (29)           */
  GST_SPLIT_BEND_KICK = 1,     /* bends exact (10), quads and multipoles (29)         */
  GST_SPLIT_MATRIX_KICK = 2,   /* bends exact (10), quads (24)(25)(27): paper's BK/MK */
  GST_SPLIT_DRIFT_KICK_4 = 3,
  GST_SPLIT_BEND_KICK_4 = 4,
  GST_SPLIT_MATRIX_KICK_4 = 5
} gst_split;

/* One lattice element.  Plain data, 144 bytes, HOST memory, copied by gst_lattice_create.
 * Strengths are normalised by the reference rigidity (B rho)_o = p0/q, so no rigidity is needed. */
typedef struct {
  int32_t type;       /* gst_elem_type                                                            */
  int32_t slice_mult; /* thick magnets: slices = n_slices * slice_mult ("4 n_b"); >= 1      */
  double L;           /* length [m]; > 0 for DRIFT/SBEND/QUAD/MULTIPOLE/SOLENOID/RBEND, ignored otherwise */
  double h;           /* SBEND: curvature of the local frame 1/rho_c = angle/L [1/m]; != 0 */
  double k0;          /* SBEND: b1/(B rho)_o = eta*h [1/m] (9); eta != 1 is a mis-powered magnet;
                         RBEND: 1/rho_b; SOLENOID: b_0/(B rho)_o; FRINGE: the magnet's dipole strength   */
  double kn[4];       /* normal  b_m/(B rho)_o, m = 2..5 -> kn[m-2], convention of (28): no 1/(m-1)!;
                         QUAD uses kn[0] only (!= 0); THINMULT: integrated (times L);
                         RBEND: kn[0] = phi_entr, kn[1] = phi_exit [rad]                          */
  double ks[4];       /* skew    a_m/(B rho)_o, same layout; must be 0 for QUAD                   */
  double volt_eV;     /* RFCAV: q*V peak energy gain [eV]                                         */
  double harmonic;    /* RFCAV: harmonic number; k_rf = 2 pi harmonic beta_o / C, C = sum of L    */
  double phi_s;       /* RFCAV: synchronous phase [rad]; reference energy += volt_eV*sin(phi_s)   */
  double sign;        /* RFCAV: +1/-1, dE = volt_eV*sin(phi_s + sign*k_rf*T)  (+1 above transition);
                         FRINGE: +1 entrance, -1 exit                                             */
  double snake_mu;    /* SNAKE: rotation angle [rad]                                              */
  double snake_phi;   /* SNAKE: axis (sin phi, 0, cos phi) in (x,y,s): angle from s-hat in the x-s plane */
} gst_element;

typedef struct {
  double G;       /* gyromagnetic anomaly (g-2)/2 (4) P:87 */
  double mass_eV; /* rest energy [eV]                       */
  double gamma0;  /* reference Lorentz factor at turn 0     */
} gst_beam; /* charge +1 */

typedef struct gst_lattice gst_lattice;
typedef struct gst_bunch gst_bunch;

/* Stage an element table (a0).  `elems` and `beam` are HOST pointers, copied.  The table is
 * de-duplicated to unique elements + a packed uint32 sequence and uploaded to the current CUDA device
 * (synchronously: the sequence is resident when the call returns).
 * GST_EINVAL: n == 0, unknown type, L <= 0 for a thick element, SBEND with h == 0 or k0 == 0, QUAD
 * with kn[0] == 0 or any skew/higher term, SOLENOID or RBEND with k0 == 0, RBEND whose angles do not
 * match L*k0, slice_mult < 1, more than 65535 unique elements.                                    */
gst_status gst_lattice_create(const gst_element* elems, size_t n, const gst_beam* beam, gst_lattice** out);
void gst_lattice_destroy(gst_lattice* lat);

/* particle-element-steps one particle makes per turn at `n_slices` (thick: n_slices*slice_mult,
 * everything else 1): the unit of BASELINE.json's metric.                                          */
int64_t gst_lattice_steps_per_turn(const gst_lattice* lat, int n_slices);

/* Bind nine DEVICE arrays of n doubles each (SoA; D1, D2 of DESIGN.md).  Borrowed, not copied: the
 * caller keeps them alive until gst_bunch_destroy.  Allocates the per-particle lost flags (A15) and a
 * few kB of scratch on the device that owns `x` (the current device when n == 0).  GST_EINVAL when
 * `x` is not device memory.                                                                          */
gst_status gst_bunch_init(double* x, double* px, double* y, double* py, double* t, double* pt, double* sx, double* sy,
                          double* ss, size_t n, gst_bunch** out);
void gst_bunch_destroy(gst_bunch* b);

/* Track the bunch for n_turns turns of `lat` in place (a1-a12, a14).  ASYNCHRONOUS on
 * `cuda_stream` (a cudaStream_t, NULL = default stream); never synchronises.  One launch of the
 * persistent turn-loop kernel.  The bunch carries the turn counter and the reference energy across
 * calls (first call takes gamma0 from the lattice's beam).
 *   n_slices      base number of orbital slices per thick magnet (n_b of P:585), >= 1
 *   romberg_depth number d of step-size levels in the Romberg table (39): 1 = trapezoid edge
 *                 product only; d = k+1 for the paper's "k Romberg iterations"; 1..6
 * GST_EINVAL if 2^(d-1) does not divide n_slices*slice_mult of some thick magnet (reading A4).   */
gst_status gst_track(gst_bunch* b, const gst_lattice* lat, int64_t n_turns, gst_split split, int n_slices,
                     int romberg_depth, void* cuda_stream);

/* The comparison integrators of the paper's section 4.1 (Figs. 7, 14): the same orbit maps, but the
 * spin is rotated once per slice by R(ds Omega) with Omega taken in the MIDDLE of the slice (37), no Romberg.
 *   GST_PWC_HALF_SLICE  half a slice map, spin rotation, half a slice map ("DKDSDKD"); any split
 *   GST_PWC_DKSKD       half drift, half kick, spin rotation, half kick, half drift ("DKSKD") in the
 *                       elements a drift-kick map integrates under `split`; the others as GST_PWC_HALF_SLICE
 * Second-order splits only (GST_EINVAL for GST_SPLIT_*_4).  Otherwise exactly like gst_track: asynchronous,
 * in place, one launch.                                                                              */
typedef enum { GST_PWC_HALF_SLICE = 0, GST_PWC_DKSKD = 1 } gst_pwc_order;
gst_status gst_track_pwc(gst_bunch* b, const gst_lattice* lat, int64_t n_turns, gst_split split, int n_slices,
                         gst_pwc_order order, void* cuda_stream);

/* How gst_track lays a bunch over the chip (per bunch; results are bit-identical):
 *   GST_LAUNCH_AUTO    default.  One thread per particle, orbit and spin work software-pipelined.  When the
 *                      bunch fits the chip in fewer than 1.5 waves but fills its sub-partitions unevenly (e.g. 65 536
 *                      particles = 3.46 warps each), the turns are cut into chunks and the warps of particles rotate
 *                      over all resident warp slots (csrc/track_chain_kernel.cuh, a cooperative launch)
 *                      Bunches of at most two warps per sub-partition take a kernel variant compiled with registers to
 *                      spare ("track_kernel_fat", see gst_bunch_last_kernel), and the smallest ones (at most 3 warps of
 *                      particles per SM: 14 208 particles on a B200; second-order splits, lattice resident in shared
 *                      memory) the kernel that gives a particle's orbit and its spin to two warps of a block
 *                      ("track_split_kernel", csrc/track_split_kernel.cuh)
 *   GST_LAUNCH_STATIC  never rotate, one thread per particle: every warp keeps its slot for the whole call
 *   GST_LAUNCH_LEAN    as GST_LAUNCH_STATIC, and always the occupancy-oriented kernel, whatever the bunch size        */
typedef enum { GST_LAUNCH_AUTO = 0, GST_LAUNCH_STATIC = 1, GST_LAUNCH_LEAN = 2 } gst_launch_mode;
gst_status gst_bunch_set_launch(gst_bunch* b, gst_launch_mode mode);

/* Synchronise `cuda_stream` and report whether every gst_track enqueued on this bunch so far ran to the end:
 * GST_OK, or GST_ECUDA once for a failed launch (see "Errors" above; the message names the kernel).  Cheap: one
 * 4-byte copy.  Callers that read the borrowed arrays themselves (the normal PyTorch use) call this first.        */
gst_status gst_bunch_status(gst_bunch* b, void* cuda_stream);

/* Bunch polarization (a13; reading A18): out = {Px, Py, Ps, |P|} over particles not lost;
 * out_lost (may be NULL) = number lost.  Enqueues the reduction on the stream and SYNCHRONISES it.
 * `out` and `out_lost` are HOST pointers.                                                           */
gst_status gst_polarization(gst_bunch* b, void* cuda_stream, double out[4], int64_t* out_lost);

/* Geometric rms emittances (a13; reading A19), HOST out = {eps_x, eps_y}; synchronises the stream. */
gst_status gst_emittance(gst_bunch* b, void* cuda_stream, double out_exy[2]);

/* The ADDITIVE record behind both reports, for bunches sharded over several GPUs (particles are
 * independent, so the only exchange of the method is the sum behind a bunch-wide report).  HOST out:
 *   [0..3]   sum Sx, sum Sy, sum Ss, number of particles not lost                                     (A18)
 *   [4..7]   sum X, sum Px, sum Y, sum Py
 *   [8..13]  central sums about THIS shard's means: dX dX, dPx dPx, dX dPx, dY dY, dPy dPy, dY dPy    (A19, two-pass)
 *   [14..19] n m m' of the same six pairs (m = this shard's means)
 * Records of disjoint shards add component by component (one all-reduce of GST_MOMENTS_LEN doubles); the central sums
 * of the union are [8..13] + [14..19] - (sum u)(sum u')/n of the summed record, which gst_moments_finish evaluates.
 * Synchronises the stream and reports a failed launch like gst_polarization.                                        */
#define GST_MOMENTS_LEN 20
gst_status gst_moments(gst_bunch* b, void* cuda_stream, double out[GST_MOMENTS_LEN]);

/* Polarization {Px, Py, Ps, |P|} (A18), geometric rms emittances {eps_x, eps_y} (A19) and particle count of a record
 * of gst_moments or of a component-wise sum of such records.  HOST pointers; any of the three outputs may be NULL.
 * Pure host arithmetic: needs no device.  For a single record it returns what gst_polarization / gst_emittance do.  */
gst_status gst_moments_finish(const double rec[GST_MOMENTS_LEN], double out_pol[4], double out_exy[2], int64_t* out_alive);

/* Name of the kernel the last gst_track / gst_track_pwc on this bunch launched ("" before the first call; static
 * storage): "track_kernel"; "track_chain_kernel" (the rotating launch); "track_kernel_fat": the same code compiled
 * with registers to spare, taken for bunches of at most two warps per SM sub-partition (37 888 particles on a B200),
 * where one warp's dependency chains set the time -- the same source compiled a second time, so results agree
 * with "track_kernel" to rounding (1e-13), not bit for bit; "track_chain_kernel" IS bit-identical to
 * "track_kernel"; "track_split_kernel": orbit and Omega of 32 particles in one warp, their quaternion work in a
 * second one (GST_LAUNCH_AUTO, the smallest bunches) -- the same functions compiled once more, so again equal to
 * the others to rounding.                                                                             */
const char* gst_bunch_last_kernel(const gst_bunch* b);

/* Copy the lost flags (1 = lost) to HOST memory, n bytes; synchronises the stream and reports a failed
 * launch like gst_bunch_status.                                                                       */
gst_status gst_bunch_lost(gst_bunch* b, void* cuda_stream, uint8_t* host_out);

/* Reference Lorentz factor and turn counter the bunch carries (host-side bookkeeping of A13).
 * The reference energy is summed with a remainder term (two doubles), so gamma0 is the correctly
 * rounded E_o(n)/m after any number of cavity passages; gst_bunch_set_reference clears the remainder. */
gst_status gst_bunch_reference(const gst_bunch* b, double* gamma0, int64_t* turn);
gst_status gst_bunch_set_reference(gst_bunch* b, const gst_beam* beam, int64_t turn);

/* End-to-end convenience with HOST buffers: allocates device arrays, copies the nine host arrays
 * (n doubles each, pinned or pageable) to the device, tracks, reduces, copies the state back into
 * the same host arrays.  out_pol = {Px,Py,Ps,|P|}, out_lost may be NULL.  Synchronous.  The device
 * workspace is kept in the lattice handle between calls of the same bunch size (freed by gst_lattice_destroy,
 * and dropped when a call fails); concurrent calls on one lattice serialise.  A failed launch is reported by
 * this call itself (GST_ECUDA); the host arrays are then left as they were.                           */
gst_status gst_track_host(const gst_lattice* lat, double* const host_state[9], size_t n, int64_t n_turns,
                          gst_split split, int n_slices, int romberg_depth, double out_pol[4], int64_t* out_lost);

/* Bunch polarization WITHOUT ANY ALLOCATION, for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it) and so cannot make a gst_bunch.  The same two-stage reduction as
 * gst_polarization, with its per-block partial sums in a fixed device array inside the library (128 KiB that every
 * GPU which loads the library holds until the process exits) instead of memory from gst_bunch_init.
 *   sx, sy, ss  DEVICE arrays of n doubles: the spin components (borrowed, read only)
 *   lost        DEVICE array of n bytes, non-zero = excluded (A15/A18), or NULL: nobody is lost
 *   n           particles; at most GST_NOALLOC_MAX_PARTICLES, else GST_EINVAL (the scratch array is what it is)
 *   out_dev     DEVICE array of 5 doubles: {Px, Py, Ps, |P|, number of particles counted}
 * ASYNCHRONOUS on `cuda_stream`: two kernels are enqueued, nothing is synchronised, nothing is copied to the host.
 * Calls no cudaMalloc, cudaFree or allocating library routine.  Runs on the device that owns out_dev; the inputs must
 * live there.  Every call on a device shares the one scratch array, which keeps the last call's contents (none of it
 * has to start at zero: a call overwrites every record it later reads): calls that OVERLAP on the GPU -- different
 * streams without an event between them, several host threads -- race on it and give wrong sums; calls on one stream
 * are safe.  (The first call on a device asks the driver for the array's address: make it before a capture begins.)  */
#define GST_NOALLOC_MAX_PARTICLES 1048576
gst_status gst_polarization_noalloc(const double* sx, const double* sy, const double* ss, const uint8_t* lost, size_t n,
                                    double* out_dev, void* cuda_stream);

/* Thread-local message for the last error on this thread; never NULL. */
const char* gst_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* GST_H_ */
