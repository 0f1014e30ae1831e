// gst_api.cu -- C ABI (include/gst.h) over the CUDA kernels: lattice staging (a0), bunch handles,
// the track launch (T1), reductions (T2) and the FP64-peak microbenchmark (T3).
#include "../../include/gst.h"

#include <cuda_runtime.h>

#include <cmath>
#include <algorithm>
#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "reduce_kernel.cuh"
#include "track_launch.cuh"

namespace {

thread_local std::string g_err = "";
std::atomic<int> g_variant{GST_KERNEL_FUSED};

gst_status fail(gst_status s, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_err = buf;
  return s;
}
#define CUDA_TRY(expr)                                                                      \
  do {                                                                                      \
    cudaError_t e_ = (expr);                                                                \
    if (e_ != cudaSuccess) return fail(GST_ECUDA, "%s: %s", #expr, cudaGetErrorString(e_)); \
  } while (0)

bool is_thick(int t) { return t == GST_SBEND || t == GST_QUAD || t == GST_MULTIPOLE || t == GST_SOLENOID || t == GST_RBEND; }

struct DevTable {
  gst::DevElem* d_tab = nullptr;
};

}  // namespace

struct gst_lattice {
  std::vector<gst_element> elems;   // as given
  std::vector<gst_element> uniq;    // de-duplicated
  std::vector<uint32_t> seq;        // gst::seq_pack(index into uniq, type) per lattice position
  gst_beam beam;
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
  uint8_t* d_lost = nullptr;
  double* d_partials = nullptr;   // [RED_MAX_BLOCKS][RED_WIDTH]
  double* d_result = nullptr;     // [2*RED_WIDTH]
  double* h_result = nullptr;     // pinned
  bool have_ref = false;
  double E0 = 0, E0lo = 0, mass = 0;   // reference energy E0 + E0lo (gst::ref_energy_add)
  int64_t turn = 0;
  // chain rotation (track_chain_kernel.cuh): per-chain progress flags and reference energies, error word
  int* d_chain_flag = nullptr;
  double* d_chain_E0 = nullptr;
  int* d_err = nullptr;
  const char* last_kernel = "";
};

namespace {

// host-side derivation of the per-slice constants of one unique element (a0)
gst::DevElem derive(const gst_element& e, int n_slices, double C) {
  gst::DevElem d;
  std::memset(&d, 0, sizeof d);
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

gst_status get_table(const gst_lattice* lat, int n_slices, const gst::DevElem** out) {
  std::lock_guard<std::mutex> lk(lat->mu);
  auto it = lat->tables.find(n_slices);
  if (it == lat->tables.end()) {
    std::vector<gst::DevElem> host(lat->uniq.size());
    for (size_t i = 0; i < lat->uniq.size(); ++i) host[i] = derive(lat->uniq[i], n_slices, lat->C);
    DevTable t;
    CUDA_TRY(cudaMalloc(&t.d_tab, host.size() * sizeof(gst::DevElem)));
    CUDA_TRY(cudaMemcpy(t.d_tab, host.data(), host.size() * sizeof(gst::DevElem), cudaMemcpyHostToDevice));
    it = lat->tables.emplace(n_slices, t).first;
  }
  *out = it->second.d_tab;
  return GST_OK;
}

// max relative error (in units of 2^-53) of the branch-free reciprocal / reciprocal square root
__global__ void math_selftest_kernel(unsigned long long* out, int n) {
  double worst_rcp = 0.0, worst_rsq = 0.0;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    double x = exp2(-2.0 + 4.0 * ((double)i + 0.37) / (double)n);     // [0.25, 4)
    double r = gst::rcp_nr(x), q = gst::rsqrt_nr(x);
    double er = fabs(fma(r, x, -1.0));                                 // |r x - 1|, exact residual
    double eq = fabs(fma(q * q, x, -1.0)) * 0.5;                       // ~ |q sqrt(x) - 1|
    worst_rcp = fmax(worst_rcp, er);
    worst_rsq = fmax(worst_rsq, eq);
  }
  atomicMax(out, (unsigned long long)__double_as_longlong(worst_rcp));
  atomicMax(out + 1, (unsigned long long)__double_as_longlong(worst_rsq));
}

gst_status validate_track(const gst_lattice* lat, int64_t n_turns, int split, int n_slices, int depth) {
  if (n_turns < 0) return fail(GST_EINVAL, "n_turns < 0");
  if (split < 0 || split > 5) return fail(GST_EINVAL, "unknown split %d", split);
  if (n_slices < 1 || n_slices > (1 << 20)) return fail(GST_EINVAL, "n_slices must be >= 1");
  if (depth < 1 || depth > 6) return fail(GST_EINVAL, "romberg_depth must be in 1..6");
  for (const gst_element& e : lat->uniq)
    if (is_thick(e.type)) {
      long N = (long)n_slices * e.slice_mult;
      if (N % (1L << (depth - 1)) != 0)
        return fail(GST_EINVAL, "2^(depth-1) = %ld does not divide the %ld slices of a thick element", 1L << (depth - 1), N);
    }
  return GST_OK;
}

}  // namespace

extern "C" {

const char* gst_last_error(void) { return g_err.c_str(); }

gst_status gst_set_kernel_variant(gst_kernel_variant v) {
  if (v != GST_KERNEL_FUSED && v != GST_KERNEL_PAIR && v != GST_KERNEL_FUSED_STATIC) return fail(GST_EINVAL, "unknown kernel variant %d", (int)v);
  g_variant.store((int)v);
  return GST_OK;
}

gst_status gst_lattice_create(const gst_element* elems, size_t n, const gst_beam* beam, gst_lattice** out) {
  if (!elems || !beam || !out || n == 0) return fail(GST_EINVAL, "null argument or empty lattice");
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
  lat->seq.resize(n);
  for (size_t i = 0; i < n; ++i) {
    gst_element e = elems[i];
    if (!is_thick(e.type)) e.slice_mult = 1;
    if (e.type == GST_RBEND) lat->C += (e.kn[0] - e.kn[1]) / e.k0;   // design arc length (19)
    else if (e.type == GST_DRIFT || is_thick(e.type)) lat->C += e.L;
    else e.L = 0.0;
    size_t k = 0;
    for (; k < lat->uniq.size(); ++k)
      if (std::memcmp(&lat->uniq[k], &e, sizeof e) == 0) break;
    if (k == lat->uniq.size()) {
      if (k >= 65535) { delete lat; return fail(GST_EINVAL, "more than 65535 unique elements"); }
      lat->uniq.push_back(e);
    }
    lat->seq[i] = gst::seq_pack((uint32_t)k, e.type);
    if (e.type == GST_RFCAV) lat->cav_dEs.push_back(e.volt_eV * std::sin(e.phi_s));
  }
  cudaError_t ce = cudaMalloc(&lat->d_seq, n * sizeof(uint32_t));
  if (ce == cudaSuccess) ce = cudaMemcpy(lat->d_seq, lat->seq.data(), n * sizeof(uint32_t), cudaMemcpyHostToDevice);
  if (ce != cudaSuccess) {
    if (lat->d_seq) cudaFree(lat->d_seq);
    delete lat;
    return fail(GST_ECUDA, "staging the element sequence: %s", cudaGetErrorString(ce));
  }
  *out = lat;
  return GST_OK;
}

void gst_lattice_destroy(gst_lattice* lat) {
  if (!lat) return;
  if (lat->ws_bunch) gst_bunch_destroy(lat->ws_bunch);
  if (lat->ws_state) cudaFree(lat->ws_state);
  if (lat->ws_stream) cudaStreamDestroy(lat->ws_stream);
  for (auto& kv : lat->tables) cudaFree(kv.second.d_tab);
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
  gst_bunch* b = new (std::nothrow) gst_bunch;
  if (!b) return fail(GST_ENOMEM, "out of host memory");
  for (int i = 0; i < 9; ++i) b->p[i] = p[i];
  b->n = n;
  cudaError_t ce = cudaMalloc(&b->d_lost, n > 0 ? n : 1);
  if (ce == cudaSuccess) ce = cudaMemset(b->d_lost, 0, n > 0 ? n : 1);
  if (ce == cudaSuccess) ce = cudaMalloc(&b->d_partials, sizeof(double) * gst::RED_MAX_BLOCKS * gst::RED_WIDTH);
  if (ce == cudaSuccess) ce = cudaMalloc(&b->d_result, sizeof(double) * 2 * gst::RED_WIDTH);
  if (ce == cudaSuccess) ce = cudaMallocHost(&b->h_result, sizeof(double) * 2 * gst::RED_WIDTH);
  const size_t n_chains = (n + 31) / 32 + 1;
  // [sm scratch | chain flags], zeroed together before every rotating launch
  if (ce == cudaSuccess) ce = cudaMalloc(&b->d_chain_flag, sizeof(int) * (n_chains + 2 * gst::CHAIN_MAX_SMID + 1));
  if (ce == cudaSuccess) ce = cudaMalloc(&b->d_chain_E0, sizeof(double) * 2 * n_chains);
  if (ce == cudaSuccess) ce = cudaMalloc(&b->d_err, sizeof(int));
  if (ce == cudaSuccess) ce = cudaMemset(b->d_err, 0, sizeof(int));
  if (ce != cudaSuccess) {
    gst_bunch_destroy(b);
    return fail(ce == cudaErrorMemoryAllocation ? GST_ENOMEM : GST_ECUDA, "gst_bunch_init: %s", cudaGetErrorString(ce));
  }
  *out = b;
  return GST_OK;
}

void gst_bunch_destroy(gst_bunch* b) {
  if (!b) return;
  if (b->d_lost) cudaFree(b->d_lost);
  if (b->d_partials) cudaFree(b->d_partials);
  if (b->d_result) cudaFree(b->d_result);
  if (b->h_result) cudaFreeHost(b->h_result);
  if (b->d_chain_flag) cudaFree(b->d_chain_flag);
  if (b->d_chain_E0) cudaFree(b->d_chain_E0);
  if (b->d_err) cudaFree(b->d_err);
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

// depth_code >= 1: trapezoid/Romberg scheme of that depth; 0 / -1: mid-slice PWC (half-slice / DKSKD ordering),
// for which the element table is derived for 2 n_slices half slices
static gst_status track_impl(gst_bunch* b, const gst_lattice* lat, int64_t n_turns, gst_split split, int n_slices,
                             int depth_code, void* cuda_stream) {
  if (!b || !lat) return fail(GST_EINVAL, "null handle");
  gst_status vs = validate_track(lat, n_turns, (int)split, n_slices, depth_code >= 1 ? depth_code : 1);
  if (vs != GST_OK) return vs;
  if (depth_code < 1 && (int)split > 2) return fail(GST_EINVAL, "gst_track_pwc takes the second-order splits only");
  const int romberg_depth = depth_code;
  const int table_slices = depth_code >= 1 ? n_slices : 2 * n_slices;
  if (!b->have_ref) {
    b->E0 = lat->beam.gamma0 * lat->beam.mass_eV;
    b->E0lo = 0.0;
    b->mass = lat->beam.mass_eV;
    b->have_ref = true;
  }
  if (b->n == 0 || n_turns == 0) return GST_OK;
  const gst::DevElem* d_tab = nullptr;
  gst_status ts = get_table(lat, table_slices, &d_tab);
  if (ts != GST_OK) return ts;
  gst::TrackArgs a;
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
  size_t tab_bytes = lat->uniq.size() * sizeof(gst::DevElem);
  size_t seq_bytes = (lat->seq.size() * sizeof(uint32_t) + 15) & ~size_t(15);
  const bool pair = g_variant.load() == GST_KERNEL_PAIR;
  gst::ChainLaunch chain_req;
  chain_req.args.sm_scratch = b->d_chain_flag;
  chain_req.args.flag = b->d_chain_flag + 2 * gst::CHAIN_MAX_SMID + 1;
  chain_req.args.E0 = b->d_chain_E0;
  chain_req.args.err = b->d_err;
  chain_req.steps_per_turn = gst_lattice_steps_per_turn(lat, table_slices);
  gst::ChainLaunch* chain = g_variant.load() == GST_KERNEL_FUSED ? &chain_req : nullptr;
  a.use_smem_seq = 0;
  a.use_smem_tab = 0;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  cudaError_t ce;
  const int order = (int)split >= 3 ? 4 : 2;
  switch ((int)split % 3) {
    case 0: ce = gst::launch_split_dk(order, romberg_depth, a, tab_bytes, seq_bytes, pair, st, chain); break;
    case 1: ce = gst::launch_split_bk(order, romberg_depth, a, tab_bytes, seq_bytes, pair, st, chain); break;
    default: ce = gst::launch_split_mk(order, romberg_depth, a, tab_bytes, seq_bytes, pair, st, chain); break;
  }
  if (ce != cudaSuccess) return fail(GST_ECUDA, "track launch: %s", cudaGetErrorString(ce));
  b->last_kernel = pair && romberg_depth >= 1 && (int)split < 3 ? "track_pair_kernel"
                   : (chain_req.taken ? "track_chain_kernel" : "track_kernel");
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
  int err = 0;
  CUDA_TRY(cudaMemcpyAsync(&err, b->d_err, sizeof(int), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  if (err) return fail(GST_ECUDA, "track_chain_kernel: a chain handoff timed out (not every warp slot was resident)");
  return GST_OK;
}

gst_status gst_polarization(gst_bunch* b, void* cuda_stream, double out[4], int64_t* out_lost) {
  if (!b || !out) return fail(GST_EINVAL, "null argument");
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

gst_status gst_bunch_lost(gst_bunch* b, void* cuda_stream, uint8_t* host_out) {
  if (!b || !host_out) return fail(GST_EINVAL, "null argument");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (b->n) CUDA_TRY(cudaMemcpyAsync(host_out, b->d_lost, b->n, cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  return GST_OK;
}

gst_status gst_track_host(const gst_lattice* lat, double* const host_state[9], size_t n, int64_t n_turns,
                          gst_split split, int n_slices, int romberg_depth, double out_pol[4], int64_t* out_lost) {
  if (!lat || !host_state || !out_pol) return fail(GST_EINVAL, "null argument");
  gst_status vs = validate_track(lat, n_turns, (int)split, n_slices, romberg_depth);
  if (vs != GST_OK) return vs;
  std::lock_guard<std::mutex> lk(lat->mu_host);
  if (!lat->ws_stream) CUDA_TRY(cudaStreamCreate(&lat->ws_stream));
  if (!lat->ws_bunch || lat->ws_n != n) {          // (re)build the workspace for this bunch size
    if (lat->ws_bunch) gst_bunch_destroy(lat->ws_bunch);
    if (lat->ws_state) cudaFree(lat->ws_state);
    lat->ws_bunch = nullptr;
    lat->ws_state = nullptr;
    CUDA_TRY(cudaMalloc(&lat->ws_state, sizeof(double) * 9 * (n ? n : 1)));
    double* d0 = lat->ws_state;
    gst_status bs = gst_bunch_init(d0, d0 + n, d0 + 2 * n, d0 + 3 * n, d0 + 4 * n, d0 + 5 * n, d0 + 6 * n, d0 + 7 * n,
                                   d0 + 8 * n, n, &lat->ws_bunch);
    if (bs != GST_OK) return bs;
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
  if (s == GST_OK) s = gst_polarization(b, st, out_pol, out_lost);
  if (s == GST_OK) {
    for (int i = 0; i < 9 && ce == cudaSuccess; ++i)
      ce = cudaMemcpyAsync(host_state[i], d + i * n, sizeof(double) * n, cudaMemcpyDeviceToHost, st);
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
    if (ce != cudaSuccess) s = fail(GST_ECUDA, "D2H: %s", cudaGetErrorString(ce));
  }
  return s;
}

gst_status gst_selftest_math(double out[2]) {
  if (!out) return fail(GST_EINVAL, "null argument");
  unsigned long long* d = nullptr;
  CUDA_TRY(cudaMalloc(&d, 16));
  CUDA_TRY(cudaMemset(d, 0, 16));
  math_selftest_kernel<<<296, 256>>>(d, 1 << 24);
  unsigned long long h[2];
  cudaError_t ce = cudaMemcpy(h, d, 16, cudaMemcpyDeviceToHost);
  cudaFree(d);
  if (ce != cudaSuccess) return fail(GST_ECUDA, "selftest: %s", cudaGetErrorString(ce));
  for (int k = 0; k < 2; ++k) {
    double v;
    std::memcpy(&v, &h[k], 8);
    out[k] = v / 1.1102230246251565e-16;      // in units of 2^-53
  }
  return GST_OK;
}

static gst_status fp64_peak_impl(bool three_registers, double* out_tflops, double* out_ms) {
  if (!out_tflops) return fail(GST_EINVAL, "null argument");
  int dev = 0, sms = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  double* d_out = nullptr;
  CUDA_TRY(cudaMalloc(&d_out, sizeof(double) * sms * 8 * gst::PEAK_BLOCK));
  cudaEvent_t e0, e1;
  CUDA_TRY(cudaEventCreate(&e0));
  CUDA_TRY(cudaEventCreate(&e1));
  const int iters = 1 << 14;
  float best = 1e30f;
  for (int rep = 0; rep < 6; ++rep) {
    cudaEventRecord(e0);
    if (three_registers) gst::dfma_rrr_kernel<<<sms * 8, gst::PEAK_BLOCK>>>(d_out, iters, 1.0 + 1e-9 * rep);
    else gst::dfma_peak_kernel<<<sms * 8, gst::PEAK_BLOCK>>>(d_out, iters, 1.0 + 1e-9 * rep);
    cudaEventRecord(e1);
    CUDA_TRY(cudaEventSynchronize(e1));
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d_out);
  CUDA_TRY(cudaGetLastError());
  double flops = 2.0 * gst::PEAK_CHAINS * (double)iters * gst::PEAK_UNROLL * (double)sms * 8 * gst::PEAK_BLOCK;
  *out_tflops = flops / (best * 1e-3) / 1e12;
  if (out_ms) *out_ms = best;
  return GST_OK;
}

gst_status gst_fp64_peak(double* out_tflops, double* out_ms) { return fp64_peak_impl(false, out_tflops, out_ms); }
gst_status gst_fp64_peak_rrr(double* out_tflops, double* out_ms) { return fp64_peak_impl(true, out_tflops, out_ms); }

}  // extern "C"
