// track_split_kernel.cuh -- T1s: small bunches, a particle's orbit and its spin in two warps of one block.
//
// Why: a bunch of 4096 particles is 128 warps on the 592 SM sub-partitions of the chip.  Every warp has a
// sub-partition to itself, the FP64 pipe is idle half of the time (one warp's dependency chains set the time), and
// 464 sub-partitions do nothing.  More threads per warp or more particles per thread do not help: the time is the
// length of ONE instruction stream.  So the stream is cut in two.  The orbit does not depend on the spin (P:774:
// the paper's orbit and spin kernels), hence
//   warp 0 of a block (producer)  advances the orbit of 32 particles through the ring with the fused kernel's own
//                                 element code and evaluates w ds Omega at every slice edge (a9), nothing else;
//   warp 1 (consumer)             takes these rotation vectors and does all quaternion work for the same particles:
//                                 the level products (a10), Romberg, normalisation, rotation of S (a11), snakes (a12).
// Both walk the same element sequence, so the consumer knows what each vector is without tags.  The vectors travel
// through a ring in shared memory (2 x SPLIT_HALF entries of 3 doubles per lane, conflict-free), handed over half a
// ring at a time with the named-barrier producer / consumer protocol (bar.arrive on one side, bar.sync on the other):
// a waiting warp sleeps in the barrier unit and takes no issue slots.  The two warps sit on different
// sub-partitions, each with its own FP64 pipe.
//
// The arithmetic is the fused kernel's, function by function (the steppers' omega() / advance(), quat_from_rotvec,
// SpinAcc, FusedSpin::run), so the results agree with "track_kernel_fat" to rounding (the compiler contracts and
// orders the same source per kernel).  Lost particles: the producer goes on with the reference orbit as the fused
// kernel does; nothing of a lost particle is stored by either warp.
#pragma once
#include "track_kernel.cuh"

namespace gst {

constexpr int SPLIT_BLOCK = 64;
constexpr int SPLIT_HALF = 16;                                                    // entries per half of the ring
constexpr size_t SPLIT_RING_BYTES = 2 * SPLIT_HALF * 3 * 32 * sizeof(double);     // 24 576 per block
constexpr int SPLIT_MIN_BLOCKS = 4;                                               // registers to spare, as the FAT variant

// named barriers 1..4 of the block; barrier 0 is __syncthreads
enum : int { RING_FULL = 1, RING_EMPTY = 3 };
__device__ __forceinline__ void named_sync(int id) { asm volatile("bar.sync %0, 64;" ::"r"(id) : "memory"); }
__device__ __forceinline__ void named_arrive(int id) { asm volatile("bar.arrive %0, 64;" ::"r"(id) : "memory"); }

__device__ __forceinline__ void sts_f64(unsigned addr, double v) { asm volatile("st.shared.f64 [%0], %1;" ::"r"(addr), "d"(v) : "memory"); }
__device__ __forceinline__ double lds_f64(unsigned addr) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr) : "memory");
  return v;
}

// One lane's view of the ring: entry r, component k of lane l at byte r * 768 + k * 256 + l * 8 of the ring (shared
// state space, 32-bit addresses).  Half h is entries 16 h .. 16 h + 15.  The producer waits for "half h empty" before
// it writes the half's first entry and announces "half h full" after its last; the consumer the other way round.
// Nothing depends on the absolute count, so the 32-bit counter may wrap (it does after 4.3e9 edges, under a million
// turns of a large ring).
struct RotvecRing {
  unsigned mine;     // shared-space address of this lane's slot in entry 0
  unsigned s;        // entries pushed (producer) or popped (consumer) so far; both count the same sequence
  __device__ __forceinline__ void attach(const void* ring, int lane) {
    mine = (unsigned)__cvta_generic_to_shared(ring) + 8u * (unsigned)lane;
    s = 0;
  }
  // producer -------------------------------------------------------------------------------------------------
  __device__ __forceinline__ void push(double wx, double wy, double ws) {
    const unsigned t = s & (SPLIT_HALF - 1), h = (s / SPLIT_HALF) & 1;
    if (t == 0) named_sync(RING_EMPTY + h);              // wait until this half has been read
    const unsigned p = mine + (s & (2 * SPLIT_HALF - 1)) * 768u;
    sts_f64(p, wx); sts_f64(p + 256, wy); sts_f64(p + 512, ws);
    if (t == SPLIT_HALF - 1) named_arrive(RING_FULL + h);   // the half just written may be read
    ++s;
  }
  __device__ __forceinline__ void flush() {              // the last half, if it is a partial one
    if ((s & (SPLIT_HALF - 1)) != 0) named_arrive(RING_FULL + ((s / SPLIT_HALF) & 1));
  }
  // consumer -------------------------------------------------------------------------------------------------
  __device__ __forceinline__ void open() {               // both halves start empty
    named_arrive(RING_EMPTY);
    named_arrive(RING_EMPTY + 1);
  }
  __device__ __forceinline__ void pop(double& wx, double& wy, double& ws) {
    const unsigned t = s & (SPLIT_HALF - 1), h = (s / SPLIT_HALF) & 1;
    if (t == 0) named_sync(RING_FULL + h);
    const unsigned p = mine + (s & (2 * SPLIT_HALF - 1)) * 768u;
    wx = lds_f64(p); wy = lds_f64(p + 256); ws = lds_f64(p + 512);
    if (t == SPLIT_HALF - 1) named_arrive(RING_EMPTY + h);  // the half just read may be written again
    ++s;
  }
};

// The producer's spin policy (see the policies in track_kernel.cuh): the edges of a thick element in order, with the
// trapezoid weights of FusedSpin::run (half at both ends).
struct ProducerSpin {
  RotvecRing& ring;
  __device__ __forceinline__ ProducerSpin(RotvecRing& r) : ring(r) {}
  // Omega of edge i and the orbit slice behind it do not depend on each other: side by side in one loop body, so
  // that a lone warp has two dependency chains to issue from
  template <class Stepper>
  __device__ __forceinline__ void run(Stepper& s, int N, double ds) {
    const double hds = 0.5 * ds;
    double wx, wy, ws;
    s.omega(hds, wx, wy, ws);
    s.advance();
    ring.push(wx, wy, ws);
    for (int i = 1; i < N; ++i) {
      s.omega(ds, wx, wy, ws);
      s.advance();
      ring.push(wx, wy, ws);
    }
    s.omega(hds, wx, wy, ws);
    ring.push(wx, wy, ws);
  }
  __device__ __forceinline__ void thin(double wx, double wy, double ws) { ring.push(wx, wy, ws); }
  __device__ __forceinline__ void snake(const Quat&) {}          // constants of the element table: the consumer has them
};

// The consumer's "stepper": the next edge's rotation vector comes out of the ring, already weighted, so that
// FusedSpin::run itself does the consumer's side of a thick element.  (Converting each vector to a quaternion one edge
// ahead of the level products, in a loop of its own, measured 7 % slower on bend-kick bunches.)
template <bool SMALL> struct RingStepper {
  static constexpr bool SMALL_ANGLE = SMALL;
  RotvecRing& ring;
  __device__ __forceinline__ void advance() {}
  __device__ __forceinline__ void omega(double, double& wx, double& wy, double& ws) { ring.pop(wx, wy, ws); }
};

// The spin side of every element type, in the order element_step() / element_step_other() call their spin policy.
// Quadrupoles and multipoles take the small-angle quaternion polynomial in every split (MultDK, QuadMK), bends,
// solenoids and rectangular bends the general one.
template <int DEPTH>
__device__ __forceinline__ void spin_turns(FusedSpin<DEPTH, false>& spin, RotvecRing& ring, const TrackArgs& a,
                                           const unsigned char* smem_raw) {
  const DevElem* tab = reinterpret_cast<const DevElem*>(smem_raw);
  const uint32_t* seq = reinterpret_cast<const uint32_t*>(smem_raw + (size_t)a.n_unique * sizeof(DevElem));
  const int n_seq = a.n_seq;
  RingStepper<true> small{ring};
  RingStepper<false> large{ring};
  double wx, wy, ws;
  for (long long turn = 0; turn < a.n_turns; ++turn) {
#pragma unroll 1
    for (int ie = 0; ie < n_seq; ++ie) {
      const uint32_t cur = seq[ie];
      const int type = (int)(cur & 0xffu);
      const DevElem& e = tab[cur >> 8];
      if (type == K_QUAD || type == K_MULT) {
        spin.run(small, e.N, e.ds);
      } else if (type == K_SBEND) {
        spin.run(large, e.N, e.ds);
      } else if (type == K_THIN || type == K_FRINGE) {
        ring.pop(wx, wy, ws);
        spin.thin(wx, wy, ws);
      } else if (type == K_SNAKE) {
        spin.snake(Quat{e.qw, e.qx, e.qy, e.qs});
      } else if (type == K_SOLENOID) {
        ring.pop(wx, wy, ws);
        spin.thin(wx, wy, ws);
        spin.run(large, e.N, e.ds);
        ring.pop(wx, wy, ws);
        spin.thin(wx, wy, ws);
      } else if (type == K_RBEND) {
        spin.snake(Quat{e.rb_qw[0], 0.0, e.rb_qy[0], 0.0});
        ring.pop(wx, wy, ws);
        spin.thin(wx, wy, ws);
        spin.run(large, e.N, e.ds);
        ring.pop(wx, wy, ws);
        spin.thin(wx, wy, ws);
        spin.snake(Quat{e.rb_qw[1], 0.0, e.rb_qy[1], 0.0});
      }
    }
  }
}

// offset of the ring behind the resident lattice (track_kernel.cuh: stage_lattice)
__host__ __device__ inline size_t split_ring_offset(int n_unique, int n_seq) {
  return ((size_t)n_unique * sizeof(DevElem) + (size_t)n_seq * sizeof(uint32_t) + 15) & ~size_t(15);
}

template <int SPLIT, int DEPTH>
__global__ void __launch_bounds__(SPLIT_BLOCK, SPLIT_MIN_BLOCKS) track_split_kernel(const TrackArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ unsigned char s_lost[32];
  stage_lattice<false>(a, smem_raw);
  if (*a.err != 0) return;                               // an earlier launch on this bunch failed: leave everything (gst.h)
  const int lane = threadIdx.x & 31;
  const bool producer = threadIdx.x < 32;
  const long long j = (long long)blockIdx.x * 32 + lane;
  const bool valid = j < a.n && !a.lost[j];
  RotvecRing ring;
  ring.attach(smem_raw + split_ring_offset(a.n_unique, a.n_seq), lane);
  State z;
  z.X = z.Px = z.Y = z.Py = z.T = z.Pt = 0.0;
  z.Sx = 0.0; z.Sy = 1.0; z.Ss = 0.0;
  if (producer) {
    if (valid) {
      z.X = a.p[0][j]; z.Px = a.p[1][j]; z.Y = a.p[2][j]; z.Py = a.p[3][j]; z.T = a.p[4][j]; z.Pt = a.p[5][j];
    }
    Ref ref;
    ref_set(ref, a.E0, a.mass);
    ref.E0lo = a.E0lo;
    PCon pc;
    pcon_set(pc, z.Pt, ref, a.G);
    ProducerSpin spin(ring);
    const bool lost = track_turns<SPLIT, 2, false>(z, ref, pc, spin, 0, a.n_turns, a, smem_raw);
    ring.flush();
    s_lost[lane] = lost ? 1 : 0;
  } else {
    if (valid) { z.Sx = a.p[6][j]; z.Sy = a.p[7][j]; z.Ss = a.p[8][j]; }
    ring.open();
    FusedSpin<DEPTH, false> spin(z);
    spin_turns<DEPTH>(spin, ring, a, smem_raw);
  }
  __syncthreads();                                       // the consumer learns which particles were lost
  if (!valid) return;
  const bool lost = s_lost[lane] != 0;
  if (producer) {
    if (lost) { a.lost[j] = 1; return; }
    a.p[0][j] = z.X; a.p[1][j] = z.Px; a.p[2][j] = z.Y; a.p[3][j] = z.Py; a.p[4][j] = z.T; a.p[5][j] = z.Pt;
  } else if (!lost) {
    a.p[6][j] = z.Sx; a.p[7][j] = z.Sy; a.p[8][j] = z.Ss;
  }
}

}  // namespace gst
