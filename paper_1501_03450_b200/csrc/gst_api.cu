// gst_api.cu -- C ABI (include/gst.h) over the CUDA kernels: lattice staging (a0), bunch handles,
// the track launch (T1) and the reductions (T2).  The diagnostics of include/gst_diag.h are in gst_diag.cu.
#include "../../include/gst.h"
#include "../../include/gst_diag.h"

#include <cuda_runtime.h>

#include <cmath>
#include <algorithm>
#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <climits>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "gst_internal.h"
#include "reduce_kernel.cuh"
#include "track_launch.cuh"

namespace gst {
thread_local std::string g_err = "";

gst_status fail(gst_status s, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_err = buf;
  return s;
}
}  // namespace gst

namespace {
using gst::DeviceGuard;
using gst::fail;

bool is_thick(int t) { return t == GST_SBEND || t == GST_QUAD || t == GST_MULTIPOLE || t == GST_SOLENOID || t == GST_RBEND; }

// one derived unique-element table (a value of n_slices): pinned host copy, device copy, upload event
struct DevTable {
  gst::DevElem* h_tab = nullptr;
  gst::DevElem* d_tab = nullptr;
  cudaEvent_t ready = nullptr;
};

}  // namespace

// One element of the COMPILED lattice: a user element (never a drift except at the end of the ring, never a marker)
// together with the drift space in front of it.  See compile_lattice().
struct CompiledElem {
  gst_element e;
  double Lpre;     // summed length of the drifts (and skipped markers) between the previous compiled element and this one
};

struct gst_lattice {
  std::vector<gst_element> elems;   // as given: what gst_lattice_steps_per_turn counts
  std::vector<CompiledElem> uniq;   // compiled and de-duplicated
  std::vector<uint32_t> seq;        // gst::seq_pack(index into uniq, type) per position of the compiled sequence
  gst_beam beam;
  int device = 0;                   // the CUDA device the tables live on
  int sms = 0;                      // its SM count
  double C = 0;                     // circumference = sum of L
  uint32_t* d_seq = nullptr;
  mutable std::map<int, DevTable> tables;   // derived unique-element tables, keyed by n_slices
  mutable std::mutex mu;
  std::vector<double> cav_dEs;      // per cavity in lattice order: volt*sin(phi_s)
  // workspace of gst_track_host, kept between calls (device state, bunch handle, stream) so that the end-to-end
  // call costs two copies and the kernels, not allocations; guarded by mu_host (calls on one lattice serialise)
  mutable std::mutex mu_host;
  mutable double* ws_state = nullptr;
  mutable size_t ws_n = 0;
  mutable gst_bunch* ws_bunch = nullptr;
  mutable cudaStream_t ws_stream = nullptr;
};

struct gst_bunch {
  double* p[9];
  size_t n = 0;
  int device = 0;                 // the CUDA device that owns the arrays
  gst_launch_mode launch_mode = GST_LAUNCH_AUTO;
  long long poll_limit_override = 0;   // gst_diag_chain_poll_limit
  uint8_t* d_lost = nullptr;
  double* d_partials = nullptr;   // [RED_MAX_BLOCKS][RED_WIDTH]
  double* d_result = nullptr;     // [2*RED_WIDTH]
  double* h_result = nullptr;     // pinned
  bool have_ref = false;
  double E0 = 0, E0lo = 0, mass = 0;   // reference energy E0 + E0lo (gst::ref_energy_add)
  int64_t turn = 0;
  // chain rotation (track_chain_kernel.cuh): [scratch | per-chain progress flags], per-chain reference energies
  int* d_chain = nullptr;
  double* d_chain_E0 = nullptr;
  int* d_err = nullptr;           // error word: set by a kernel that gave up, cleared when the host has reported it
  int* h_err = nullptr;           // pinned landing place of its copies
  const char* last_kernel = "";
};

namespace {

// host-side derivation of the per-slice constants of one unique element (a0)
gst::DevElem derive(const CompiledElem& ce, int n_slices, double C) {
  const gst_element& e = ce.e;
  gst::DevElem d;
  std::memset(&d, 0, sizeof d);
  d.Lpre = ce.Lpre;
  d.type = e.type;
  d.N = is_thick(e.type) ? n_slices * e.slice_mult : 1;
  d.L = e.L;
  d.ds = e.L / d.N;
  d.h = e.h;
  d.k0 = e.k0;
  d.order = 2;
  for (int m = 2; m <= 5; ++m) {
    d.kn[m - 2] = e.kn[m - 2];
    d.ks[m - 2] = e.ks[m - 2];
    if (e.kn[m - 2] != 0.0 || e.ks[m - 2] != 0.0) d.order = m;
  }
  d.pure_quad = (d.order == 2 && e.ks[0] == 0.0) ? 1 : 0;
  if (e.type == GST_SBEND) {
    long double h = e.h, k0 = e.k0, ds = (long double)e.L / d.N;
    long double half = sinl(0.5L * h * ds);
    long double cm = 2.0L * half * half;
    d.cm = (double)cm;
    d.sn = (double)sinl(h * ds);
    d.ck = (double)(cm / k0);
    d.sk = (double)(sinl(h * ds) / k0);
    d.ome = (double)((h - k0) / h);
    d.inv_eta = (double)(h / k0);
    d.inv_h = (double)(1.0L / h);
    // TEAPOT curved drifts: ds/2 (second order), x1 ds/2 and (x1 + x0) ds/2 (fourth order, merged neighbours)
    const long double x1 = 1.0L / (2.0L - cbrtl(2.0L)), x0 = 1.0L - 2.0L * x1;
    const long double lens[4] = {0.5L * ds, 0.5L * x1 * ds, 0.5L * (x1 + x0) * ds, ds};
    for (int k = 0; k < 4; ++k) {
      gst::TeapotHalf& t = d.th[k];
      long double phi = h * lens[k];
      long double q = sinl(0.5L * phi);
      t.len = (double)lens[k];
      t.c = (double)cosl(phi);
      t.s = (double)sinl(phi);
      t.t = (double)tanl(phi);
      t.sec = (double)(1.0L / cosl(phi));
      t.r_secm1 = (double)((2.0L * q * q / cosl(phi)) / h);
      t.r_tan = (double)(tanl(phi) / h);
      // tan(phi) - phi: series for small phi (long double subtraction would lose digits)
      long double tmp;
      if (fabsl(phi) < 0.05L) {
        long double p2 = phi * phi;
        tmp = phi * p2 * (1.0L / 3 + p2 * (2.0L / 15 + p2 * (17.0L / 315 + p2 * (62.0L / 2835 + p2 * (1382.0L / 155925 +
              p2 * (21844.0L / 6081075 + p2 * (929569.0L / 638512875)))))));
      } else {
        tmp = tanl(phi) - phi;
      }
      t.r_tanmphi = (double)(tmp / h);
    }
  }
  if (e.type == GST_RFCAV) {
    d.volt = e.volt_eV;
    d.krf_over_beta = 2.0 * M_PI * e.harmonic / C;
    d.phi_s = e.phi_s;
    d.sign = e.sign;
    d.dEs = e.volt_eV * std::sin(e.phi_s);
  }
  if (e.type == GST_FRINGE) d.sign = e.sign;
  if (e.type == GST_RBEND) {
    const long double ang[2] = {(long double)e.kn[0], -(long double)e.kn[1]};
    for (int k = 0; k < 2; ++k) {
      d.rb_c[k] = (double)cosl(ang[k]);
      d.rb_s[k] = (double)sinl(ang[k]);
      d.rb_t[k] = (double)tanl(ang[k]);
      d.rb_sec[k] = (double)(1.0L / cosl(ang[k]));
      d.rb_qw[k] = (double)cosl(0.5L * ang[k]);
      d.rb_qy[k] = (double)sinl(0.5L * ang[k]);
    }
    const long double rho = 1.0L / (long double)e.k0, dphi = (long double)e.kn[0] - (long double)e.kn[1];
    d.rb_rho = (double)rho;
    d.rb_xoff = (double)(rho * (cosl(e.kn[1]) - cosl(e.kn[0])));
    d.rb_arc = (double)(rho * dphi);
    d.rb_cd = (double)cosl(dphi);
    d.rb_sd = (double)sinl(dphi);
    d.kn[0] = d.kn[1] = 0.0;          // the angles are not multipole strengths
    d.order = 2;
    d.pure_quad = 0;
  }
  if (e.type == GST_SNAKE) {
    double sh = std::sin(0.5 * e.snake_mu);
    d.qw = std::cos(0.5 * e.snake_mu);
    d.qx = sh * std::sin(e.snake_phi);
    d.qy = 0.0;
    d.qs = sh * std::cos(e.snake_phi);
  }
  return d;
}

// The derived table of one slicing: made on first use, uploaded on the caller's stream from a pinned copy that the
// lattice keeps alive; `ready` orders every other stream behind that upload.
gst_status get_table(const gst_lattice* lat, int n_slices, cudaStream_t st, const gst::DevElem** out) {
  std::lock_guard<std::mutex> lk(lat->mu);
  auto it = lat->tables.find(n_slices);
  if (it == lat->tables.end()) {
    const size_t bytes = lat->uniq.size() * sizeof(gst::DevElem);
    DevTable t;
    cudaError_t ce = cudaMallocHost(&t.h_tab, bytes);
    if (ce == cudaSuccess) {
      for (size_t i = 0; i < lat->uniq.size(); ++i) t.h_tab[i] = derive(lat->uniq[i], n_slices, lat->C);
      ce = cudaMalloc(&t.d_tab, bytes);
    }
    if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&t.ready, cudaEventDisableTiming);
    if (ce == cudaSuccess) ce = cudaMemcpyAsync(t.d_tab, t.h_tab, bytes, cudaMemcpyHostToDevice, st);
    if (ce == cudaSuccess) ce = cudaEventRecord(t.ready, st);
    if (ce != cudaSuccess) {
      if (t.ready) cudaEventDestroy(t.ready);
      if (t.d_tab) cudaFree(t.d_tab);
      if (t.h_tab) cudaFreeHost(t.h_tab);
      return fail(ce == cudaErrorMemoryAllocation ? GST_ENOMEM : GST_ECUDA, "staging the element table: %s", cudaGetErrorString(ce));
    }
    it = lat->tables.emplace(n_slices, t).first;
  } else {
    CUDA_TRY(cudaStreamWaitEvent(st, it->second.ready, 0));
  }
  *out = it->second.d_tab;
  return GST_OK;
}

gst_status validate_track(const gst_lattice* lat, int64_t n_turns, int split, int n_slices, int depth) {
  if (n_turns < 0) return fail(GST_EINVAL, "n_turns < 0");
  if (split < 0 || split > 5) return fail(GST_EINVAL, "unknown split %d", split);
  if (n_slices < 1 || n_slices > (1 << 20)) return fail(GST_EINVAL, "n_slices must be in 1..2^20");
  if (depth < 1 || depth > 6) return fail(GST_EINVAL, "romberg_depth must be in 1..6");
  for (const CompiledElem& ce : lat->uniq)
    if (const gst_element& e = ce.e; is_thick(e.type)) {
      const int64_t N = (int64_t)n_slices * e.slice_mult;          // 2 N must fit an int (half slices of gst_track_pwc)
      if (N > (int64_t)(1 << 30)) return fail(GST_EINVAL, "n_slices*slice_mult = %lld exceeds 2^30", (long long)N);
      if (N % (1LL << (depth - 1)) != 0)
        return fail(GST_EINVAL, "2^(depth-1) = %ld does not divide the %lld slices of a thick element", 1L << (depth - 1), (long long)N);
    }
  return GST_OK;
}

// Has a launch on this bunch failed since the last report?  Enqueues a 4-byte copy behind everything on `st`,
// synchronises, and on failure clears the word (so that the bunch is usable again) and names the failure.
gst_status sync_and_report(gst_bunch* b, cudaStream_t st) {
  CUDA_TRY(cudaMemcpyAsync(b->h_err, b->d_err, sizeof(int), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  if (*b->h_err != 0) {
    CUDA_TRY(cudaMemsetAsync(b->d_err, 0, sizeof(int), st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return fail(GST_ECUDA, "%s: a hand-off between warp slots timed out (the chip made no progress); the particle arrays "
                "of this bunch are undefined", b->last_kernel);
  }
  return GST_OK;
}

}  // namespace

extern "C" {

const char* gst_last_error(void) { return gst::g_err.c_str(); }

gst_status gst_lattice_create(const gst_element* elems, size_t n, const gst_beam* beam, gst_lattice** out) {
  if (!elems || !beam || !out || n == 0) return fail(GST_EINVAL, "null argument or empty lattice");
  if (n > (size_t)INT32_MAX) return fail(GST_EINVAL, "more than 2^31 - 1 elements");
  if (!(beam->gamma0 > 1.0) || !(beam->mass_eV > 0.0)) return fail(GST_EINVAL, "beam: need gamma0 > 1 and mass_eV > 0");
  for (size_t i = 0; i < n; ++i) {
    const gst_element& e = elems[i];
    if (e.type < 0 || e.type > GST_RBEND) return fail(GST_EINVAL, "element %zu: unknown type %d", i, e.type);
    if ((is_thick(e.type) || e.type == GST_DRIFT) && !(e.L > 0.0)) return fail(GST_EINVAL, "element %zu: L must be > 0", i);
    if (is_thick(e.type) && e.slice_mult < 1) return fail(GST_EINVAL, "element %zu: slice_mult must be >= 1", i);
    if (e.type == GST_SBEND && (e.h == 0.0 || e.k0 == 0.0)) return fail(GST_EINVAL, "element %zu: SBEND needs h != 0 and k0 != 0", i);
    if (e.type == GST_SOLENOID && e.k0 == 0.0) return fail(GST_EINVAL, "element %zu: SOLENOID needs k0 != 0", i);
    if (e.type == GST_RBEND) {
      if (e.k0 == 0.0) return fail(GST_EINVAL, "element %zu: RBEND needs k0 != 0", i);
      if (std::fabs(std::sin(e.kn[0]) - std::sin(e.kn[1]) - e.L * e.k0) > 1e-12 * (1.0 + std::fabs(e.L * e.k0)))
        return fail(GST_EINVAL, "element %zu: RBEND needs sin(phi_entr) - sin(phi_exit) = L*k0 (13b)", i);
    }
    if (e.type == GST_QUAD) {
      if (e.kn[0] == 0.0) return fail(GST_EINVAL, "element %zu: QUAD needs kn[0] != 0", i);
      for (int k = 0; k < 4; ++k)
        if (e.ks[k] != 0.0 || (k > 0 && e.kn[k] != 0.0)) return fail(GST_EINVAL, "element %zu: QUAD takes kn[0] only", i);
    }
  }
  gst_lattice* lat = new (std::nothrow) gst_lattice;
  if (!lat) return fail(GST_ENOMEM, "out of host memory");
  lat->elems.assign(elems, elems + n);
  lat->beam = *beam;
  // Lattice compilation.  A drift changes no momentum and is exact for any length (29b), so consecutive drifts are one
  // drift (group property; long straights are cut into many pieces), and a drift followed by a magnet needs the same
  // sqrt(P^2 - Px^2 - Py^2) as the magnet's own entrance: every run of drifts is folded into the element behind it
  // (CompiledElem::Lpre -> DevElem::Lpre) and costs that element a handful of multiply-adds instead of an element
  // dispatch, two reciprocal chains and a square root of its own.  Markers do nothing and are dropped.  The end of the
  // ring is a hard boundary (the state handed back after a turn is the state at the end of the user's lattice): drifts
  // that are left there stay one drift element.  The step count of the metric is that of the USER lattice.
  {
    double pending = 0.0;
    auto emit = [&](const gst_element& el, double Lpre) -> bool {
      CompiledElem ce;
      std::memset(&ce, 0, sizeof ce);
      ce.e = el;
      ce.Lpre = Lpre;
      size_t k = 0;
      for (; k < lat->uniq.size(); ++k)
        if (std::memcmp(&lat->uniq[k], &ce, sizeof ce) == 0) break;
      if (k == lat->uniq.size()) {
        if (k >= 65535) return false;
        lat->uniq.push_back(ce);
      }
      lat->seq.push_back(gst::seq_pack((uint32_t)k, el.type));
      return true;
    };
    bool fits = true;
    for (size_t i = 0; i < n && fits; ++i) {
      gst_element e = elems[i];
      if (!is_thick(e.type)) e.slice_mult = 1;
      if (e.type == GST_RBEND) lat->C += (e.kn[0] - e.kn[1]) / e.k0;   // design arc length (19)
      else if (e.type == GST_DRIFT || is_thick(e.type)) lat->C += e.L;
      else e.L = 0.0;
      if (e.type == GST_RFCAV) lat->cav_dEs.push_back(e.volt_eV * std::sin(e.phi_s));
      if (e.type == GST_DRIFT) { pending += e.L; continue; }
      if (e.type == GST_MARKER) continue;
      fits = emit(e, pending);
      pending = 0.0;
    }
    if (fits && (pending > 0.0 || lat->seq.empty())) {      // what is left at the end of the ring (or a ring of markers)
      gst_element tail;
      std::memset(&tail, 0, sizeof tail);
      tail.type = pending > 0.0 ? GST_DRIFT : GST_MARKER;
      tail.slice_mult = 1;
      tail.L = pending;
      fits = emit(tail, 0.0);
    }
    if (!fits) { delete lat; return fail(GST_EINVAL, "more than 65535 unique elements"); }
  }
  n = lat->seq.size();        // from here on: the compiled sequence
  // the sequence goes up through a pinned staging buffer on a stream of its own, complete when this call returns
  // (a blocking copy from pageable memory may return before its DMA has landed, and streams made with
  // cudaStreamNonBlocking -- torch's -- are not ordered behind the legacy stream)
  cudaError_t ce = cudaGetDevice(&lat->device);
  if (ce == cudaSuccess) ce = cudaDeviceGetAttribute(&lat->sms, cudaDevAttrMultiProcessorCount, lat->device);
  uint32_t* h_seq = nullptr;
  cudaStream_t up = nullptr;
  if (ce == cudaSuccess) ce = cudaMalloc(&lat->d_seq, n * sizeof(uint32_t));
  if (ce == cudaSuccess) ce = cudaMallocHost(&h_seq, n * sizeof(uint32_t));
  if (ce == cudaSuccess) ce = cudaStreamCreateWithFlags(&up, cudaStreamNonBlocking);
  if (ce == cudaSuccess) {
    std::memcpy(h_seq, lat->seq.data(), n * sizeof(uint32_t));
    ce = cudaMemcpyAsync(lat->d_seq, h_seq, n * sizeof(uint32_t), cudaMemcpyHostToDevice, up);
  }
  if (ce == cudaSuccess) ce = cudaStreamSynchronize(up);
  if (up) cudaStreamDestroy(up);
  if (h_seq) cudaFreeHost(h_seq);
  if (ce != cudaSuccess) {
    if (lat->d_seq) cudaFree(lat->d_seq);
    delete lat;
    return fail(ce == cudaErrorMemoryAllocation ? GST_ENOMEM : GST_ECUDA, "staging the element sequence: %s", cudaGetErrorString(ce));
  }
  *out = lat;
  return GST_OK;
}

static void drop_host_workspace(const gst_lattice* lat) {
  if (lat->ws_bunch) gst_bunch_destroy(lat->ws_bunch);
  if (lat->ws_state) cudaFree(lat->ws_state);
  lat->ws_bunch = nullptr;
  lat->ws_state = nullptr;
  lat->ws_n = 0;
}

void gst_lattice_destroy(gst_lattice* lat) {
  if (!lat) return;
  DeviceGuard guard(lat->device);
  drop_host_workspace(lat);
  if (lat->ws_stream) cudaStreamDestroy(lat->ws_stream);
  for (auto& kv : lat->tables) {
    cudaEventDestroy(kv.second.ready);
    cudaFree(kv.second.d_tab);
    cudaFreeHost(kv.second.h_tab);
  }
  cudaFree(lat->d_seq);
  delete lat;
}

int64_t gst_lattice_steps_per_turn(const gst_lattice* lat, int n_slices) {
  if (!lat || n_slices < 1) return 0;
  int64_t s = 0;
  for (const gst_element& e : lat->elems) s += is_thick(e.type) ? (int64_t)n_slices * e.slice_mult : 1;
  return s;
}

gst_status gst_bunch_init(double* x, double* px, double* y, double* py, double* t, double* pt, double* sx, double* sy,
                          double* ss, size_t n, gst_bunch** out) {
  if (!out) return fail(GST_EINVAL, "null out");
  double* p[9] = {x, px, y, py, t, pt, sx, sy, ss};
  for (int i = 0; i < 9; ++i)
    if (!p[i] && n > 0) return fail(GST_EINVAL, "null state pointer %d", i);
  int device = 0;
  CUDA_TRY(cudaGetDevice(&device));
  if (n > 0) {      // the bunch lives where its arrays live
    cudaPointerAttributes at;
    CUDA_TRY(cudaPointerGetAttributes(&at, x));
    if (at.type == cudaMemoryTypeDevice) device = at.device;
    else if (at.type != cudaMemoryTypeManaged) return fail(GST_EINVAL, "the state arrays must be device memory");
  }
  GUARD_DEVICE(device);
  gst_bunch* b = new (std::nothrow) gst_bunch;
  if (!b) return fail(GST_ENOMEM, "out of host memory");
  for (int i = 0; i < 9; ++i) b->p[i] = p[i];
  b->n = n;
  b->device = device;
  cudaError_t ce = cudaMalloc(&b->d_lost, n > 0 ? n : 1);
  if (ce == cudaSuccess) ce = cudaMemset(b->d_lost, 0, n > 0 ? n : 1);
  if (ce == cudaSuccess) ce = cudaMalloc(&b->d_partials, sizeof(double) * gst::RED_MAX_BLOCKS * gst::RED_WIDTH);
  if (ce == cudaSuccess) ce = cudaMalloc(&b->d_result, sizeof(double) * 2 * gst::RED_WIDTH);
  if (ce == cudaSuccess) ce = cudaMallocHost(&b->h_result, sizeof(double) * 2 * gst::RED_WIDTH);
  const size_t n_chains = (n + 31) / 32 + 1;
  // [scratch | chain flags], zeroed together before every rotating launch
  if (ce == cudaSuccess) ce = cudaMalloc(&b->d_chain, sizeof(int) * (n_chains + gst::CHAIN_SCRATCH_INTS));
  if (ce == cudaSuccess) ce = cudaMalloc(&b->d_chain_E0, sizeof(double) * 2 * n_chains);
  if (ce == cudaSuccess) ce = cudaMalloc(&b->d_err, sizeof(int));
  if (ce == cudaSuccess) ce = cudaMemset(b->d_err, 0, sizeof(int));
  if (ce == cudaSuccess) ce = cudaMallocHost(&b->h_err, sizeof(int));
  if (ce == cudaSuccess) ce = cudaDeviceSynchronize();     // the memsets ran on the legacy stream: done before any launch
  if (ce != cudaSuccess) {
    gst_bunch_destroy(b);
    return fail(ce == cudaErrorMemoryAllocation ? GST_ENOMEM : GST_ECUDA, "gst_bunch_init: %s", cudaGetErrorString(ce));
  }
  *out = b;
  return GST_OK;
}

void gst_bunch_destroy(gst_bunch* b) {
  if (!b) return;
  DeviceGuard guard(b->device);
  if (b->d_lost) cudaFree(b->d_lost);
  if (b->d_partials) cudaFree(b->d_partials);
  if (b->d_result) cudaFree(b->d_result);
  if (b->h_result) cudaFreeHost(b->h_result);
  if (b->d_chain) cudaFree(b->d_chain);
  if (b->d_chain_E0) cudaFree(b->d_chain_E0);
  if (b->d_err) cudaFree(b->d_err);
  if (b->h_err) cudaFreeHost(b->h_err);
  delete b;
}

gst_status gst_bunch_reference(const gst_bunch* b, double* gamma0, int64_t* turn) {
  if (!b) return fail(GST_EINVAL, "null bunch");
  if (!b->have_ref) return fail(GST_ESTATE, "the bunch has no reference energy yet (track it or set one)");
  if (gamma0) *gamma0 = b->E0 / b->mass;
  if (turn) *turn = b->turn;
  return GST_OK;
}

const char* gst_bunch_last_kernel(const gst_bunch* b) { return b ? b->last_kernel : ""; }

gst_status gst_bunch_set_reference(gst_bunch* b, const gst_beam* beam, int64_t turn) {
  if (!b || !beam || !(beam->gamma0 > 1.0) || !(beam->mass_eV > 0.0)) return fail(GST_EINVAL, "bad reference");
  b->E0 = beam->gamma0 * beam->mass_eV;
  b->E0lo = 0.0;
  b->mass = beam->mass_eV;
  b->turn = turn;
  b->have_ref = true;
  return GST_OK;
}

gst_status gst_bunch_set_launch(gst_bunch* b, gst_launch_mode mode) {
  if (!b || (mode != GST_LAUNCH_AUTO && mode != GST_LAUNCH_STATIC && mode != GST_LAUNCH_LEAN)) return fail(GST_EINVAL, "null bunch or unknown launch mode %d", (int)mode);
  b->launch_mode = mode;
  return GST_OK;
}

gst_status gst_diag_chain_poll_limit(gst_bunch* b, int64_t polls) {
  if (!b || polls < 0) return fail(GST_EINVAL, "null bunch or negative poll count");
  b->poll_limit_override = -(long long)polls;       // negative = absolute count (track_chain_kernel.cuh)
  return GST_OK;
}

// depth_code >= 1: trapezoid/Romberg scheme of that depth; 0 / -1: mid-slice PWC (half-slice / DKSKD ordering),
// for which the element table is derived for 2 n_slices half slices
static gst_status track_impl(gst_bunch* b, const gst_lattice* lat, int64_t n_turns, gst_split split, int n_slices,
                             int depth_code, void* cuda_stream) {
  if (!b || !lat) return fail(GST_EINVAL, "null handle");
  gst_status vs = validate_track(lat, n_turns, (int)split, n_slices, depth_code >= 1 ? depth_code : 1);
  if (vs != GST_OK) return vs;
  if (depth_code < 1 && (int)split > 2) return fail(GST_EINVAL, "gst_track_pwc takes the second-order splits only");
  if (b->n > 0 && b->device != lat->device)
    return fail(GST_EINVAL, "the bunch lives on device %d, the lattice on device %d", b->device, lat->device);
  GUARD_DEVICE(lat->device);
  const int romberg_depth = depth_code;
  const int table_slices = depth_code >= 1 ? n_slices : 2 * n_slices;
  if (!b->have_ref) {
    b->E0 = lat->beam.gamma0 * lat->beam.mass_eV;
    b->E0lo = 0.0;
    b->mass = lat->beam.mass_eV;
    b->have_ref = true;
  }
  if (b->n == 0 || n_turns == 0) return GST_OK;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const gst::DevElem* d_tab = nullptr;
  gst_status ts = get_table(lat, table_slices, st, &d_tab);
  if (ts != GST_OK) return ts;
  gst::LaunchRequest rq;
  gst::TrackArgs& a = rq.args;
  for (int i = 0; i < 9; ++i) a.p[i] = b->p[i];
  a.lost = b->d_lost;
  a.tab = d_tab;
  a.seq = lat->d_seq;
  a.n_unique = (int)lat->uniq.size();
  a.n_seq = (int)lat->seq.size();
  a.n = (long long)b->n;
  a.n_turns = n_turns;
  a.E0 = b->E0;
  a.E0lo = b->E0lo;
  a.mass = b->mass;
  a.G = lat->beam.G;
  a.err = b->d_err;
  rq.tab_bytes = lat->uniq.size() * sizeof(gst::DevElem);
  rq.seq_bytes = (lat->seq.size() * sizeof(uint32_t) + 15) & ~size_t(15);
  rq.steps_per_turn = gst_lattice_steps_per_turn(lat, table_slices);
  rq.sms = lat->sms;
  rq.allow_chain = b->launch_mode == GST_LAUNCH_AUTO;
  rq.allow_fat = b->launch_mode != GST_LAUNCH_LEAN;
  rq.allow_split = b->launch_mode == GST_LAUNCH_AUTO;
  rq.chain.scratch = b->d_chain;
  rq.chain.flag = b->d_chain + gst::CHAIN_SCRATCH_INTS;
  rq.chain.E0 = b->d_chain_E0;
  rq.chain.err = b->d_err;
  rq.poll_limit_override = b->poll_limit_override;
  const int order = (int)split >= 3 ? 4 : 2;
  const cudaError_t ce = gst::launch_tracking((int)split % 3, order, romberg_depth, rq, st);
  if (ce != cudaSuccess) return fail(GST_ECUDA, "track launch: %s", cudaGetErrorString(ce));
  b->last_kernel = rq.kernel;
  // host-side bookkeeping of the reference energy: the same IEEE operations the kernel performs
  for (int64_t t = 0; t < n_turns; ++t)
    for (double dEs : lat->cav_dEs)
      if (dEs != 0.0) gst::ref_energy_add(b->E0, b->E0lo, dEs);
  b->turn += n_turns;
  return GST_OK;
}

gst_status gst_track(gst_bunch* b, const gst_lattice* lat, int64_t n_turns, gst_split split, int n_slices,
                     int romberg_depth, void* cuda_stream) {
  if (romberg_depth < 1) return fail(GST_EINVAL, "romberg_depth must be in 1..6");
  return track_impl(b, lat, n_turns, split, n_slices, romberg_depth, cuda_stream);
}

gst_status gst_track_pwc(gst_bunch* b, const gst_lattice* lat, int64_t n_turns, gst_split split, int n_slices,
                         gst_pwc_order order, void* cuda_stream) {
  if (order != GST_PWC_HALF_SLICE && order != GST_PWC_DKSKD) return fail(GST_EINVAL, "unknown PWC ordering %d", (int)order);
  return track_impl(b, lat, n_turns, split, n_slices, order == GST_PWC_HALF_SLICE ? 0 : -1, cuda_stream);
}

gst_status gst_bunch_status(gst_bunch* b, void* cuda_stream) {
  if (!b) return fail(GST_EINVAL, "null bunch");
  GUARD_DEVICE(b->device);
  return sync_and_report(b, (cudaStream_t)cuda_stream);
}

static gst_status run_moments(gst_bunch* b, cudaStream_t st, bool second) {
  int blocks = (int)((b->n + gst::RED_BLOCK - 1) / gst::RED_BLOCK);
  if (blocks > gst::RED_MAX_BLOCKS) blocks = gst::RED_MAX_BLOCKS;
  if (blocks < 1) blocks = 1;
  gst::RedArgs a;
  for (int i = 0; i < 9; ++i) a.p[i] = b->p[i];
  a.lost = b->d_lost;
  a.n = (long long)b->n;
  a.partials = b->d_partials;
  a.result = b->d_result;
  gst::moments_kernel<false><<<blocks, gst::RED_BLOCK, 0, st>>>(a);
  gst::finalize_kernel<<<1, gst::RED_BLOCK, 0, st>>>(b->d_partials, blocks, b->d_result, 0);
  if (second) {
    gst::moments_kernel<true><<<blocks, gst::RED_BLOCK, 0, st>>>(a);
    gst::finalize_kernel<<<1, gst::RED_BLOCK, 0, st>>>(b->d_partials, blocks, b->d_result, 1);
  }
  CUDA_TRY(cudaGetLastError());
  CUDA_TRY(cudaMemcpyAsync(b->h_result, b->d_result, sizeof(double) * 2 * gst::RED_WIDTH, cudaMemcpyDeviceToHost, st));
  return sync_and_report(b, st);
}

gst_status gst_polarization(gst_bunch* b, void* cuda_stream, double out[4], int64_t* out_lost) {
  if (!b || !out) return fail(GST_EINVAL, "null argument");
  GUARD_DEVICE(b->device);
  gst_status s = run_moments(b, (cudaStream_t)cuda_stream, false);
  if (s != GST_OK) return s;
  const double* r = b->h_result;   // {sum Sx, Sy, Ss, alive, sum X, Px, Y, Py}
  double alive = r[3];
  double inv = alive > 0 ? 1.0 / alive : 0.0;
  out[0] = r[0] * inv; out[1] = r[1] * inv; out[2] = r[2] * inv;
  out[3] = std::sqrt(out[0] * out[0] + out[1] * out[1] + out[2] * out[2]);
  if (out_lost) *out_lost = (int64_t)b->n - (int64_t)alive;
  return GST_OK;
}

gst_status gst_emittance(gst_bunch* b, void* cuda_stream, double out_exy[2]) {
  if (!b || !out_exy) return fail(GST_EINVAL, "null argument");
  GUARD_DEVICE(b->device);
  gst_status s = run_moments(b, (cudaStream_t)cuda_stream, true);
  if (s != GST_OK) return s;
  const double* r = b->h_result;
  const double* c = b->h_result + gst::RED_WIDTH;   // {sxx, spp, sxp, syy, sqq, syq} central sums
  double alive = r[3];
  if (!(alive > 0)) { out_exy[0] = out_exy[1] = 0; return GST_OK; }
  for (int k = 0; k < 2; ++k) {
    double uu = c[3 * k] / alive, pp = c[3 * k + 1] / alive, up = c[3 * k + 2] / alive;
    double e2 = uu * pp - up * up;
    out_exy[k] = e2 > 0 ? std::sqrt(e2) : 0.0;
  }
  return GST_OK;
}

// 8(e): the additive record of a shard.  Central sums about the shard's own means (two-pass, moments_kernel<true>)
// plus n * mean * mean per pair, so that the records of disjoint shards add component by component and
//   central sum of the union = sum c + sum n m m' - (sum u)(sum u')/alive      (gst_moments_finish).
gst_status gst_moments(gst_bunch* b, void* cuda_stream, double out[GST_MOMENTS_LEN]) {
  if (!b || !out) return fail(GST_EINVAL, "null argument");
  GUARD_DEVICE(b->device);
  gst_status s = run_moments(b, (cudaStream_t)cuda_stream, true);
  if (s != GST_OK) return s;
  const double* r = b->h_result;                    // {sum Sx, Sy, Ss, alive, sum X, Px, Y, Py}
  const double* c = b->h_result + gst::RED_WIDTH;   // {sxx, spp, sxp, syy, sqq, syq} about this shard's means
  for (int k = 0; k < 8; ++k) out[k] = r[k];
  const double alive = r[3];
  const double inv = alive > 0 ? 1.0 / alive : 0.0;
  for (int k = 0; k < 2; ++k) {
    const double su = r[4 + 2 * k], sp = r[5 + 2 * k];
    out[8 + 3 * k] = alive > 0 ? c[3 * k] : 0.0;
    out[9 + 3 * k] = alive > 0 ? c[3 * k + 1] : 0.0;
    out[10 + 3 * k] = alive > 0 ? c[3 * k + 2] : 0.0;
    out[14 + 3 * k] = su * su * inv;
    out[15 + 3 * k] = sp * sp * inv;
    out[16 + 3 * k] = su * sp * inv;
  }
  return GST_OK;
}

gst_status gst_moments_finish(const double rec[GST_MOMENTS_LEN], double out_pol[4], double out_exy[2], int64_t* out_alive) {
  if (!rec) return fail(GST_EINVAL, "null argument");
  const double alive = rec[3];
  if (!(alive >= 0) || alive != std::floor(alive)) return fail(GST_EINVAL, "record with a particle count of %g", alive);
  const double inv = alive > 0 ? 1.0 / alive : 0.0;
  if (out_alive) *out_alive = (int64_t)alive;
  if (out_pol) {
    out_pol[0] = rec[0] * inv; out_pol[1] = rec[1] * inv; out_pol[2] = rec[2] * inv;
    out_pol[3] = std::sqrt(out_pol[0] * out_pol[0] + out_pol[1] * out_pol[1] + out_pol[2] * out_pol[2]);
  }
  if (out_exy) {
    for (int k = 0; k < 2; ++k) {
      const double su = rec[4 + 2 * k], sp = rec[5 + 2 * k];
      // between-shard part of the central sums: sum_r n_r m_r m_r' - n m m'  (zero for a single shard)
      const double uu = (rec[8 + 3 * k] + (rec[14 + 3 * k] - su * su * inv)) * inv;
      const double pp = (rec[9 + 3 * k] + (rec[15 + 3 * k] - sp * sp * inv)) * inv;
      const double up = (rec[10 + 3 * k] + (rec[16 + 3 * k] - su * sp * inv)) * inv;
      const double e2 = uu * pp - up * up;
      out_exy[k] = e2 > 0 ? std::sqrt(e2) : 0.0;
    }
  }
  return GST_OK;
}

gst_status gst_bunch_lost(gst_bunch* b, void* cuda_stream, uint8_t* host_out) {
  if (!b || !host_out) return fail(GST_EINVAL, "null argument");
  GUARD_DEVICE(b->device);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (b->n) CUDA_TRY(cudaMemcpyAsync(host_out, b->d_lost, b->n, cudaMemcpyDeviceToHost, st));
  return sync_and_report(b, st);
}

gst_status gst_track_host(const gst_lattice* lat, double* const host_state[9], size_t n, int64_t n_turns,
                          gst_split split, int n_slices, int romberg_depth, double out_pol[4], int64_t* out_lost) {
  if (!lat || !host_state || !out_pol) return fail(GST_EINVAL, "null argument");
  gst_status vs = validate_track(lat, n_turns, (int)split, n_slices, romberg_depth);
  if (vs != GST_OK) return vs;
  GUARD_DEVICE(lat->device);
  std::lock_guard<std::mutex> lk(lat->mu_host);
  if (!lat->ws_stream) CUDA_TRY(cudaStreamCreateWithFlags(&lat->ws_stream, cudaStreamNonBlocking));
  if (!lat->ws_bunch || lat->ws_n != n) {          // (re)build the workspace for this bunch size
    drop_host_workspace(lat);
    CUDA_TRY(cudaMalloc(&lat->ws_state, sizeof(double) * 9 * (n ? n : 1)));
    double* d0 = lat->ws_state;
    gst_status bs = gst_bunch_init(d0, d0 + n, d0 + 2 * n, d0 + 3 * n, d0 + 4 * n, d0 + 5 * n, d0 + 6 * n, d0 + 7 * n,
                                   d0 + 8 * n, n, &lat->ws_bunch);
    if (bs != GST_OK) { drop_host_workspace(lat); return bs; }
    lat->ws_n = n;
  }
  double* d = lat->ws_state;
  cudaStream_t st = lat->ws_stream;
  gst_bunch* b = lat->ws_bunch;
  b->have_ref = false;                             // a fresh bunch every call: reference energy from the lattice, turn 0
  b->turn = 0;
  gst_status s = GST_OK;
  cudaError_t ce = cudaMemsetAsync(b->d_lost, 0, n > 0 ? n : 1, st);
  for (int i = 0; i < 9 && ce == cudaSuccess; ++i)
    ce = cudaMemcpyAsync(d + i * n, host_state[i], sizeof(double) * n, cudaMemcpyHostToDevice, st);
  if (ce != cudaSuccess) s = fail(GST_ECUDA, "H2D: %s", cudaGetErrorString(ce));
  if (s == GST_OK) s = gst_track(b, lat, n_turns, split, n_slices, romberg_depth, st);
  if (s == GST_OK) s = gst_polarization(b, st, out_pol, out_lost);     // synchronises and reports a failed launch
  if (s == GST_OK) {
    for (int i = 0; i < 9 && ce == cudaSuccess; ++i)
      ce = cudaMemcpyAsync(host_state[i], d + i * n, sizeof(double) * n, cudaMemcpyDeviceToHost, st);
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
    if (ce != cudaSuccess) s = fail(GST_ECUDA, "D2H: %s", cudaGetErrorString(ce));
  }
  if (s != GST_OK) {                                // nothing of a failed call is kept for the next one
    const std::string msg = gst::g_err;
    cudaStreamSynchronize(st);
    drop_host_workspace(lat);
    gst::g_err = msg;
  }
  return s;
}

}  // extern "C"
