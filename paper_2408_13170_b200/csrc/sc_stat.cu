// sc_stat.cu -- kernels and C ABI of libscstat.so (sm_100a).  See include/sc_stat.h for the contract and
// DESIGN.md for the design.  No CPU fallback, no torch, no third-party code.
//
// Pipeline of one sc_eval_stat call, per batch of particles:
//   k_particle_consts  a1 + a3  per-particle constants, validity, time window [jlo, jhi) by bisection on t(f_j)
//   k_nodes            a2       phase / amplitude at the coarse nodes (one node per `stride` bins)
//   k_dense2 / k_dense a4 + a5  THE HOT LOOP: lane = particle, warp walks the bins of its chunk in order;
//                               whitened data broadcast from shared memory; k_dense2 (FP32 amplitudes, packed FFMA2):
//                               FP64 phase by forward differences + FP32 sin/cos; k_dense (all-FP64): phase factor by
//                               a rotation recurrence, amplitudes anchored in FP64 with an FP32 correction;
//                               complete segments are finalised in registers, straddlers leave fragments
//   k_stitch           a6       fixed-order stitch of the fragments -> Upsilon[p]
// The kernels live in sc_kernels_*.cuh (included below in pipeline order, one translation unit); this file holds the
// handle, the host-side orchestration and the extern "C" entry points.
#include "../../include/sc_stat.h"
#include "sc_math.cuh"

#include <cub/device/device_radix_sort.cuh>

#include <algorithm>
#include <climits>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <type_traits>
#include <vector>

using namespace sc;

#include "sc_kernels_prep.cuh"
#include "sc_kernels_dense64.cuh"
#include "sc_kernels_dense32.cuh"
#include "sc_kernels_dense32tc.cuh"
#include "sc_kernels_dense32x3.cuh"
#include "sc_kernels_adaptive.cuh"
#include "sc_kernels_stitch.cuh"
#include "sc_kernels_search.cuh"
#include "sc_kernels_streams.cuh"
#include "sc_kernels_misc.cuh"

namespace {

// ------------------------------------------------------------------------------------------------ host side
thread_local std::string g_init_error;

}  // namespace

// The analysis of one edge list for one chunk length (host vectors + their device copies).  A handle keeps two: the one in
// use and an alternate (the all-FP64 chunking of the same edges, used by the escalation pass), swapped by swap_edge_cache.
struct EdgeCache {
  int* d_edges = nullptr; int* d_chunk_k0 = nullptr; uint8_t* d_flags = nullptr; size_t edge_cap = 0, k0_cap = 0, flags_cap = 0;
  // cached edge analysis
  std::vector<int> edges; int cached_chunk = 0; int chunk_first = 0, n_chunks = 0;
  std::vector<int> chunk_k0; std::vector<uint8_t> flags;
  // next_close[c]: the chunk in which a piece left open at the end of chunk c is closed (-1: it is not) -- for k_stitch
  std::vector<int> next_close; int* d_next_close = nullptr; size_t nc_cap = 0;
  // pieces (fine sub-intervals cut at the edges) and their sigma moments, for k_dense2; cached with the edges
  int cached_lg = 0; int n_pieces = 0;
  int* d_piece_first = nullptr; int* d_piece_lo = nullptr; int* d_piece_hi = nullptr; float2* d_moments = nullptr;
  size_t pf_cap = 0, plo_cap = 0, phi_cap = 0, mom_cap = 0;
  double2* d_moments64 = nullptr; size_t mom64_cap = 0;   // FP64 moments per piece (all-FP64 chunking only)
  float2* d_momentsT = nullptr; size_t momT_cap = 0;      // moments of the T weights per piece (fused three-channel kernel)
};

struct sc_handle : EdgeCache {
  sc_config cfg;
  DevCfg dc;
  int device = 0;
  double s0 = 1.0;                 // weight scale (power of two)
  float4* D32 = nullptr; double4* W64 = nullptr; double2* G64 = nullptr;   // D32: bin-pair layout of k_dense2
  // options
  int precision = 0; int f32_min_seg = 8; size_t scratch_cap = (size_t)32 << 30;   // of 180 GB per B200
  double win_frac = 0.0;           // SC_OPT_WINDOW_FRACTION_PPM: mean share of the band inside a particle's time window (0: not stated)
  double tc_max_s = 10.0 * 31557600.0; int forced_stride_log2 = 0; int sincos_mode = 0; int mufu_min_seg = 32;
  int lg_f32 = 5, lg_f64 = 5;      // log2 of the coarse node spacing per precision mode (set_stride)
  double mufu_gain2 = 1.0;        // <cos^2 + sin^2> of the hardware sin/cos, measured at init
  double dd = 0.0;                // <d|d> (Eq. 1), computed at init
  double* d_comp = nullptr; size_t comp_cap = 0;   // components scratch of sc_eval_loglike
  void* d_km = nullptr; size_t km_cap = 0;         // k-means: changed counter + member counts
  // streams workload: template (FP64 + FP32), pieces of the edge list, per-piece sigma and z partials
  double4* d_T64 = nullptr; float4* d_T32 = nullptr; size_t t64_cap = 0, t32_cap = 0;
  int* d_sp = nullptr; size_t sp_cap = 0; double* d_spsig = nullptr; size_t spsig_cap = 0;
  double2* d_zpart = nullptr; size_t zpart_cap = 0; double* d_hh = nullptr; size_t hh_cap = 0;
  // adaptive (per-particle) segments: moments of the weights over groups and fine sub-intervals, cached per node spacing
  int ad_lg = 0; float2* d_gmom = nullptr; float2* d_smom = nullptr; size_t gmom_cap = 0, smom_cap = 0;
  double2* d_gmom64 = nullptr; double2* d_smom64 = nullptr; size_t gmom64_cap = 0, smom64_cap = 0;   // FP64 copies (edge decision)
  float2* d_gmomT = nullptr; float2* d_smomT = nullptr; double2* d_smom64T = nullptr; size_t gmomT_cap = 0, smomT_cap = 0, smom64T_cap = 0;   // ... of the T weights (three-channel handles)
  int* d_ad_edges = nullptr; size_t ad_edges_cap = 0;    // the edges of a batch when the caller does not ask for them
  // scratch
  void* scratch = nullptr; size_t scratch_bytes = 0;
  unsigned long long* d_counter = nullptr;
  double* d_params_stage = nullptr; double* d_out_stage = nullptr; size_t stage_cap = 0;
  long long launches = 0;
  EdgeCache alt;                   // see EdgeCache
  // escalation: particles whose FP32-path Upsilon is below the mode's threshold are re-evaluated
  // by the all-FP64 path; compacted index list, count, gathered parameters and their results
  int escalate = 1; double esc_tau_poly = 6.0, esc_tau_mufu = 16.0;
  int quad_amp = 1;
  int last_lg = 0, last_flavour = 0;   // sc_get_launch_info
  double esc_tau_nodes = 0.0;      // threshold the node spacing of the current call adds (select_stride_f32)
  int* d_esc_idx = nullptr; int* d_esc_count = nullptr; double* d_esc_params = nullptr; double* d_esc_out = nullptr;
  size_t esc_idx_cap = 0, esc_cnt_cap = 0, esc_par_cap = 0, esc_out_cap = 0; int* h_esc_hint = nullptr;
  // tensor-core flavour of the FP32-amplitude kernel (k_dense2_tc, SC_OPT_TENSOR_CORES; off by default: measured slower than
  // k_dense2): per-tile operand image, built for one node spacing
  int use_tc = 0; uint4* d_tc_img = nullptr; size_t tc_img_cap = 0; int tc_img_lg = 0;
  int window_sort = 1; void* d_sort_tmp = nullptr; size_t sort_cap = 0;   // cub radix-sort workspace of the window sort
  // three-channel handles (A, E, T): the T channel lives in a second handle whose first slot carries T (chan_set = 1)
  // and whose second slot is empty; the per-segment sums of both are added before |z|^2/sigma is formed
  sc_handle* sub = nullptr; double* d_seg3 = nullptr; size_t seg3_cap = 0;
  // fused tables of the one-pass three-channel kernel k_dense3 (built by sc_init_data3): data records (wA, wE, wT) per bin
  // pair, sigma weights per bin pair, and the T weights in FP64 for the piece moments; SC_OPT_FUSED_AET
  float4* D3 = nullptr; float4* Gp3 = nullptr; double2* GT64 = nullptr; int use_fused3 = 1;
  // optional per-kernel-class device timing (SC_OPT_PROFILE): event pairs recorded around each launch
  bool profile = false;
  struct Ev { cudaEvent_t a, b; int cls; };
  std::vector<Ev> evs; size_t ev_used = 0;
  double cls_ms[SC_N_TIMING_CLASSES] = {}; long long cls_n[SC_N_TIMING_CLASSES] = {};
  bool cuda_failed = false;
  std::string err;
};

namespace {

int fail(sc_handle* h, int code, const char* fmt, ...);
int pick_stride_log2(const sc_config& cfg, double tc_max_s, int forced, double max_days);
double node_seconds_per_bin(const sc_config& cfg, double tc_max_s);

// Node spacing per precision mode: measured against the oracle on c1-c5, the interpolation
// error of Upsilon is <= K days^6 / sqrt(N') with days = signal time per coarse interval at the slowest-chirping corner,
// N' = segments inside the particle's window, K = 7.5e-10 for N' = 1 (largest of 400 particles; the single coherent sum
// has the heavier tail) and 1.4e-10 for N' >= 8.  The FP32-amplitude path (N' >= 8) keeps days <= 4: model 2e-7, a fifth
// of the 1e-6 bar.  The all-FP64 path (any N', so N' = 1) keeps days <= 2: model 5e-8 -- it is also the path of the
// ill-conditioned particles (Upsilon << 1, where the relative error is amplified): at 2.5 days c5's smallest Upsilon
// reached 8.5e-7 and the escalation test failed, so the margin stays.
constexpr double kNodeDaysF64 = 2.0, kNodeDaysF32 = 4.0;

void apply_stride(DevCfg& d, int lg) {
  d.log2_stride = lg;
  d.stride = 1 << lg;
  const int n_int = (d.n_bins + d.stride - 1) / d.stride;
  d.n_nodes = n_int + kNodeOff + 4;
}

void set_stride(sc_handle* h) {
  h->lg_f64 = pick_stride_log2(h->cfg, h->tc_max_s, h->forced_stride_log2, kNodeDaysF64);
  h->lg_f32 = pick_stride_log2(h->cfg, h->tc_max_s, h->forced_stride_log2, kNodeDaysF32);
  apply_stride(h->dc, h->lg_f64);
}

// Node spacing of the FP32-amplitude path for ONE call: the interpolation error of a
// segment's z_k grows like (days per coarse interval)^6 and is independent from segment to segment, so the error of
// Upsilon = sum over the N' segments inside a particle's window falls like 1 / sqrt(N'): measured on c1-c5,
// max relative error <= 1.4e-10 days^6 / sqrt(N') for N' >= 8.  kNodeDaysF32 is the limit at N' = 8, the fewest
// segments the FP32 path is left with (below that the escalation pass takes the particle); at larger N' the same
// modelled error (2e-7) allows kNodeDaysF32 (N' / 8)^(1/12) days, capped at kNodeDaysMax.  N' = n_seg x window
// fraction / 2 when the caller has stated the fraction (SC_OPT_WINDOW_FRACTION_PPM; the search measures it), else 8.
// n_seg = 0 keeps the N' = 8 spacing: per-segment output (sc_eval_segments, the two-pass three-channel path), where
// nothing averages, and per-particle segments (sc_eval_stat_adaptive), whose integer edges are decided on the
// interpolated cumulative sigma -- wider nodes there move 0.3 % of the c3 edges by one bin instead of < 0.1 %.
constexpr double kNodeDaysMax = 8.0;
void select_stride_f32(sc_handle* h, int n_seg) {
  double n_eff = 8.0;
  if (n_seg > 0 && h->win_frac > 0.0) n_eff = 0.5 * (double)n_seg * h->win_frac;
  const double days = std::min(kNodeDaysMax, kNodeDaysF32 * pow(std::max(n_eff, 8.0) / 8.0, 1.0 / 12.0));
  h->lg_f32 = pick_stride_log2(h->cfg, h->tc_max_s, h->forced_stride_log2, days);
  // A particle of the same population with far fewer segments than the mean (a window that leaves the band) does not
  // average as much: with the spacing chosen, the model needs N' >= 8 (days / kNodeDaysF32)^12 segments, i.e.
  // Upsilon ~ 2 N' above twice that -- below it the escalation pass (all-FP64 path, its own spacing) takes the particle.
  h->esc_tau_nodes = 0.0;
  if (n_seg > 0 && h->forced_stride_log2 == 0) {
    const double d = (double)(1 << h->lg_f32) * node_seconds_per_bin(h->cfg, h->tc_max_s) / 86400.0;
    if (d > kNodeDaysF32) h->esc_tau_nodes = 2.0 * 8.0 * pow(d / kNodeDaysF32, 12.0);
  }
}

int fail(sc_handle* h, int code, const char* fmt, ...) {
  char buf[512];
  va_list ap; va_start(ap, fmt); vsnprintf(buf, sizeof buf, fmt, ap); va_end(ap);
  if (h) { h->err = buf; if (code == SC_ERR_CUDA) h->cuda_failed = true; }
  else g_init_error = buf;
  return code;
}

#define SC_CUDA(h, call)                                                                         \
  do { cudaError_t e_ = (call);                                                                  \
       if (e_ != cudaSuccess) return fail((h), e_ == cudaErrorMemoryAllocation ? SC_ERR_OOM : SC_ERR_CUDA, \
                                          "%s failed: %s", #call, cudaGetErrorString(e_)); } while (0)

// RAII: records an event pair around one kernel launch when profiling is on.
struct Timed {
  sc_handle* h; cudaStream_t st; int idx = -1;
  Timed(sc_handle* h_, cudaStream_t st_, int cls) : h(h_), st(st_) {
    if (!h->profile) return;
    if (h->ev_used == h->evs.size()) {
      sc_handle::Ev e; e.cls = cls;
      if (cudaEventCreate(&e.a) != cudaSuccess || cudaEventCreate(&e.b) != cudaSuccess) { cudaGetLastError(); return; }
      h->evs.push_back(e);
    }
    idx = (int)h->ev_used++;
    h->evs[idx].cls = cls;
    cudaEventRecord(h->evs[idx].a, st);
  }
  ~Timed() { if (idx >= 0) cudaEventRecord(h->evs[idx].b, st); }
};

int check_launch(sc_handle* h, const char* what) {
  h->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(h, SC_ERR_CUDA, "launch of %s failed: %s", what, cudaGetErrorString(e));
  return SC_OK;
}

// Coarse node spacing: the slowly varying amplitudes change on the orbital time scale,
// so the spacing is set in TIME: at most max_days at the slowest-chirping corner of the problem.  Time per bin is
// |dt/df| df = (8/3) tau / (f T_obs) with tau <= tc_max (Newtonian), largest at the low band edge.
double node_seconds_per_bin(const sc_config& cfg, double tc_max_s) {
  const double f_lo = (double)std::max<int64_t>(cfg.j0, 1) / cfg.T_obs_s;
  return (8.0 / 3.0) * tc_max_s / (f_lo * cfg.T_obs_s);
}
int pick_stride_log2(const sc_config& cfg, double tc_max_s, int forced, double max_days) {
  if (forced > 0) return std::min(std::max(forced, 3), 12);
  const double s_per_bin = node_seconds_per_bin(cfg, tc_max_s);
  int lg = 5;
  while (lg < 11 && (double)(2 << lg) * s_per_bin <= max_days * 86400.0) ++lg;
  return lg;
}

int grow(sc_handle* h, void** ptr, size_t* cap, size_t need) {
  if (*cap >= need) return SC_OK;
  if (*ptr) { cudaFree(*ptr); *ptr = nullptr; *cap = 0; }
  SC_CUDA(h, cudaMalloc(ptr, need));
  *cap = need;
  return SC_OK;
}

// Host analysis of the edge list for a given chunk length: which chunks are launched, the segment each one
// starts in, and which fragments each chunk leaves (shared by all particles, Q2).
void analyse_edges(sc_handle* h, int CH) {
  const std::vector<int>& e = h->edges;
  const int n_seg = (int)e.size() - 1;
  h->cached_chunk = CH;
  h->chunk_k0.clear(); h->flags.clear();
  h->chunk_first = 0; h->n_chunks = 0;
  if (e[n_seg] <= e[0]) return;
  h->chunk_first = e[0] / CH;
  const int chunk_last = (e[n_seg] - 1) / CH;
  h->n_chunks = chunk_last - h->chunk_first + 1;
  for (int cI = 0; cI < h->n_chunks; ++cI) {
    const int cs = (h->chunk_first + cI) * CH;
    const int ce = std::min(cs + CH, (int)h->cfg.n_bins);
    const int k0 = (int)(std::upper_bound(e.begin(), e.end(), cs) - e.begin()) - 1;   // last k with e_k <= cs
    uint8_t fl = 0;
    if (k0 >= 0 && k0 < n_seg && e[k0] < cs) {
      fl |= CF_HEAD;
      if (e[k0 + 1] <= ce) fl |= CF_HEAD_CLOSES;
    }
    // the piece open at the chunk end belongs to segment kt = last k with e_k < ce; it is a tail if it began here
    const int kt = (int)(std::lower_bound(e.begin(), e.end(), ce) - e.begin()) - 1;
    if (kt >= 0 && kt < n_seg && e[kt + 1] > ce && e[kt] >= cs) fl |= CF_TAIL;
    h->chunk_k0.push_back(k0);
    h->flags.push_back(fl);
  }
  h->next_close.assign((size_t)h->n_chunks, -1);
  for (int cI = h->n_chunks - 2; cI >= 0; --cI) {
    const uint8_t fl = h->flags[(size_t)cI + 1];
    if (fl & CF_HEAD) h->next_close[cI] = (fl & CF_HEAD_CLOSES) ? cI + 1 : h->next_close[(size_t)cI + 1];
  }
}

template <typename R>
int run_batches(sc_handle* h, const double* params, int64_t P, double* out, double* out_seg, double* out_comp,
                cudaStream_t st, bool seg_mode, const int* esc_count = nullptr, int esc_blocks = 0, bool fused3 = false) {
  // esc_count != nullptr: the escalation pass -- P is an upper bound, the number of particles sits on the device;
  // its launches are timed as SC_TIME_ESC and do not count evaluated bins twice
  const int cls_nodes = esc_count ? SC_TIME_ESC : SC_TIME_NODES, cls_dense = esc_count ? SC_TIME_ESC : SC_TIME_DENSE,
            cls_stitch = esc_count ? SC_TIME_ESC : SC_TIME_STITCH;
  const int n_seg = (int)h->edges.size() - 1;
  DevCfg dc = h->dc;
  apply_stride(dc, sizeof(R) == 4 ? h->lg_f32 : h->lg_f64);
  if (fused3) dc.chan_set = 2;                    // node amplitudes (A, E, T)
  const int NA = fused3 ? 6 : 4;                  // amplitude fields per node
  const int n_nodes = dc.n_nodes;
  const int n_chunks = h->n_chunks;
  // per-particle scratch bytes
  const size_t per_p = 2 * ((size_t)kPcFields * 8 + 8) /* constants, jlo, jhi: unsorted + sorted */ + 16 /* sort keys, map */
                       + (size_t)n_nodes * (4 + 8 + NA * sizeof(R)) + (size_t)std::max(n_chunks, 1) * kFragFields * 8
                       + (size_t)kStitchParts * kStitchRec * 8;
  int64_t Pb_max = (int64_t)(h->scratch_cap / per_p) / kBlock * kBlock;
  if (Pb_max < kBlock) Pb_max = kBlock;
  const int64_t P_round = (P + kBlock - 1) / kBlock * kBlock;
  const int P_pad = (int)std::min<int64_t>(Pb_max, P_round);
  int rc = grow(h, &h->scratch, &h->scratch_bytes, per_p * (size_t)P_pad + 1024);
  if (rc) return rc;
  // carve
  char* base = (char*)h->scratch;
  auto take = [&](size_t bytes) { char* r = base; base += (bytes + 255) / 256 * 256; return r; };
  double* pc = (double*)take((size_t)kPcFields * 8 * P_pad);
  int* jlo = (int*)take((size_t)4 * P_pad);
  int* jhi = (int*)take((size_t)4 * P_pad);
  int* node_n = (int*)take((size_t)n_nodes * 4 * P_pad);
  double* node_frac = (double*)take((size_t)n_nodes * 8 * P_pad);
  R* node_amp = (R*)take((size_t)n_nodes * NA * sizeof(R) * P_pad);
  double* frag = (double*)take((size_t)std::max(n_chunks, 1) * kFragFields * 8 * P_pad);
  double* stitch_rec = (double*)take((size_t)kStitchParts * kStitchRec * 8 * P_pad);
  // window sort (see k_gather_sorted): not in the segment-table mode (rows are addressed by particle).  In the escalation
  // pass the count sits on the device: all P_pad slots are sorted, the unused ones to the end -- only below 4096 segments
  // (a rule of the call, not of the data: with that many segments hardly any particle is selected and the sort's seven
  // small launches per batch would cost more than they save).
  const bool sorted = h->window_sort && !seg_mode && P_pad > kBlock && (!esc_count || n_seg < 4096);
  double* pc_u = (double*)take((size_t)kPcFields * 8 * P_pad);
  int* jlo_u = (int*)take((size_t)4 * P_pad);
  int* jhi_u = (int*)take((size_t)4 * P_pad);
  int* key_s = (int*)take((size_t)4 * P_pad);
  int* iota = (int*)take((size_t)4 * P_pad);
  int* pmap = (int*)take((size_t)4 * P_pad);
  (void)base;
  size_t sort_bytes = 0;
  if (sorted) {
    if (cub::DeviceRadixSort::SortPairs(nullptr, sort_bytes, jlo_u, key_s, iota, pmap, P_pad, 0, 32, st) != cudaSuccess)
      return fail(h, SC_ERR_CUDA, "cub::DeviceRadixSort size query failed");
    if ((rc = grow(h, &h->d_sort_tmp, &h->sort_cap, sort_bytes + 256))) return rc;
    k_iota<<<(P_pad + 255) / 256, 256, 0, st>>>(iota, P_pad);
    if ((rc = check_launch(h, "k_iota"))) return rc;
  }

  const int e_first = h->edges.front(), e_last = h->edges.back();
  const double four_df = 4.0 / h->cfg.T_obs_s;
  // sin/cos flavour of the FP32 path: hardware MUFU (gain-calibrated) from mufu_min_seg segments up, else polynomial
  const int sincos = (h->sincos_mode == 0) ? (n_seg >= h->mufu_min_seg ? 2 : 0) : (h->sincos_mode == 2 ? 2 : 0);
  const double h0 = pow(dc.f_amp_ref, -7.0 / 6.0);
  // segment tables are in definition units; the hardware sin/cos gain g (g^2 = mufu_gain2) multiplies every z_k of the FP32 path
  const double sz = h->s0 * h0 / four_df / ((sizeof(R) == 4 && sincos == 2) ? sqrt(h->mufu_gain2) : 1.0),
               ss = h->s0 * h->s0 * h0 * h0 / four_df;

  // particle blocks launched per kernel: all of them, or (escalation pass) the caller's estimate -- the kernels stride
  const int pblocks = esc_count ? std::max(1, std::min(esc_blocks, P_pad / kBlock)) : P_pad / kBlock;
  // tensor-core flavour of the FP32-amplitude kernel: fine sub-intervals of at least one 32-bin tile
  const bool use_tc = sizeof(R) == 4 && h->cached_chunk == tc::kChunk && n_chunks > 0 && !fused3;
  if (use_tc && h->tc_img_lg != dc.log2_stride) {
    const long long n_tiles = (long long)((dc.n_bins + tc::kChunk - 1) / tc::kChunk) * (tc::kChunk / tc::kTileBins);
    if ((rc = grow(h, (void**)&h->d_tc_img, &h->tc_img_cap, (size_t)n_tiles * tc::kTileBytes))) return rc;
    Timed tm(h, st, SC_TIME_OTHER);
    k_tc_image<<<(unsigned)n_tiles, 32, 0, st>>>(h->D32, dc.log2_stride - 2, n_tiles, h->d_tc_img);
    if ((rc = check_launch(h, "k_tc_image"))) return rc;
    h->tc_img_lg = dc.log2_stride;
  }
  for (int64_t pb = 0; pb < P; pb += P_pad) {
    const int Pn = (int)std::min<int64_t>(P_pad, P - pb);
    {
      Timed tm(h, st, cls_nodes);
      k_particle_consts<<<pblocks, 128, 0, st>>>(dc, params + pb * 8, Pn, P_pad, sorted ? pc_u : pc, sorted ? jlo_u : jlo,
                                                 sorted ? jhi_u : jhi, e_first, e_last,
                                                 esc_count ? nullptr : h->d_counter, esc_count, (int)pb);
    }
    if ((rc = check_launch(h, "k_particle_consts"))) return rc;
    if (sorted && n_chunks > 0) {
      Timed tm(h, st, cls_nodes);
      // keys: window centres, staged in jlo (the sorted copy of the windows is written by k_gather_sorted afterwards)
      k_sort_key<<<(P_pad + 255) / 256, 256, 0, st>>>(jlo_u, jhi_u, jlo, P_pad, esc_count, (int)pb);
      if ((rc = check_launch(h, "k_sort_key"))) return rc;
      if (cub::DeviceRadixSort::SortPairs(h->d_sort_tmp, sort_bytes, jlo, key_s, iota, pmap, P_pad, 0, 32, st) != cudaSuccess)
        return fail(h, SC_ERR_CUDA, "cub::DeviceRadixSort::SortPairs failed");
      h->launches += 3;
      k_gather_sorted<<<(P_pad + 127) / 128, 128, 0, st>>>(pmap, P_pad, pc_u, jlo_u, jhi_u, pc, jlo, jhi, esc_count, (int)pb);
      if ((rc = check_launch(h, "k_gather_sorted"))) return rc;
    }
    if (n_chunks == 0) {
      if (!seg_mode && out) SC_CUDA(h, cudaMemsetAsync(out + pb, 0, (size_t)Pn * 8, st));
      if (out_comp) SC_CUDA(h, cudaMemsetAsync(out_comp + pb * 3, 0, (size_t)Pn * 24, st));
      continue;
    }
    {
      Timed tm(h, st, cls_nodes);
      if (fused3) k_nodes<R, false, 6><<<dim3((n_nodes + kNodesPerCta - 1) / kNodesPerCta, pblocks), 128, 0, st>>>(dc, pc, jlo, jhi, P_pad, node_n, node_frac, node_amp, nullptr, 0, 1);
      else if (esc_count) k_nodes<R, true><<<dim3((n_nodes + kNodesPerCta - 1) / kNodesPerCta, pblocks), 128, 0, st>>>(dc, pc, jlo, jhi, P_pad, node_n, node_frac, node_amp, esc_count, (int)pb, 1);
      else k_nodes<R, false><<<dim3((n_nodes + kNodesPerCta - 1) / kNodesPerCta, pblocks), 128, 0, st>>>(dc, pc, jlo, jhi, P_pad, node_n, node_frac, node_amp, nullptr, 0, 1);
    }
    if ((rc = check_launch(h, "k_nodes"))) return rc;
    DenseArgs a = {};
    a.esc_count = esc_count; a.esc_pb = (int)pb;
    a.edges = h->d_edges; a.n_seg = n_seg; a.chunk_first = h->chunk_first; a.chunk_k0 = h->d_chunk_k0;
    a.node_n = node_n; a.node_frac = node_frac; a.node_amp = node_amp; a.jlo = jlo; a.jhi = jhi; a.P_pad = P_pad;
    a.frag = frag; a.out_seg = seg_mode ? out_seg + (size_t)pb * n_seg * 3 : nullptr; a.P = Pn;
    a.seg_scale_z = sz; a.seg_scale_s = ss; a.comp = out_comp ? 1 : 0;
    a.piece_first = h->d_piece_first; a.moments = reinterpret_cast<const ulonglong2*>(h->d_moments);
    a.momentsT = reinterpret_cast<const ulonglong2*>(h->d_momentsT);
    a.moments64 = (sizeof(R) == 8 && h->cached_lg > 0) ? h->d_moments64 : nullptr;
    const dim3 grid(n_chunks, pblocks);
    {
      Timed tm(h, st, cls_dense);
      if (sizeof(R) == 4) {
        const ulonglong2* Dp = reinterpret_cast<const ulonglong2*>(h->D32);
        // merged coarse intervals (see coarse_dslope): worth their test only where the coarse intervals are long; the
        // fine sub-intervals may span kNodeDaysF32 / 4 days of signal time
        const bool merge = dc.stride >= 512;
        // quadratic amplitudes over runs of >= 64 bins (pairs_fast_q): where the pieces are long enough to pay for the run
        // set-up at each piece start (c4 at N = 50 000, 33-bin segments: +1 %; c3/c4 at N = 5000, 328 bins: -4 %)
        const bool quad = h->quad_amp && dc.stride >= 1024 && (long long)(e_last - e_first) >= 128LL * n_seg;
        a.merge_lim = 86400.0 * (kNodeDaysF32 / 4.0) / h->cfg.T_obs_s;
        const dim3 grid_tc(pblocks, n_chunks);
        if (!esc_count) {
          h->last_lg = dc.log2_stride;
          const bool quad_on = quad && sincos == 2 && !seg_mode;
          h->last_flavour = (sincos == 2 ? SC_FLAVOUR_MUFU : 0) |
                            (fused3 ? (SC_FLAVOUR_AET | (quad_on ? SC_FLAVOUR_QUAD : 0)) : use_tc ? SC_FLAVOUR_TC :
                             ((merge ? SC_FLAVOUR_MERGE : 0) | ((quad_on && merge) ? SC_FLAVOUR_QUAD : 0)));
        }
        if (fused3) {
          const ulonglong2* D3p = reinterpret_cast<const ulonglong2*>(h->D3);
          const ulonglong2* Gp = reinterpret_cast<const ulonglong2*>(h->Gp3);
          if (seg_mode && sincos == 2) k_dense3<true, 2><<<grid, kBlock, 0, st>>>(dc, a, D3p, Gp);
          else if (seg_mode) k_dense3<true, 0><<<grid, kBlock, 0, st>>>(dc, a, D3p, Gp);
          else if (sincos == 2 && quad) k_dense3<false, 2, true><<<grid, kBlock, 0, st>>>(dc, a, D3p, Gp);
          else if (sincos == 2) k_dense3<false, 2><<<grid, kBlock, 0, st>>>(dc, a, D3p, Gp);
          else k_dense3<false, 0><<<grid, kBlock, 0, st>>>(dc, a, D3p, Gp);
        }
        else if (use_tc) {
          const uint4* Tg = h->d_tc_img;
          if (seg_mode) k_dense2_tc<true, 0><<<grid_tc, tc::kThreads, tc::kSmemBytes, st>>>(dc, a, Dp, Tg);
          else if (sincos == 2 && merge) k_dense2_tc<false, 2, true><<<grid_tc, tc::kThreads, tc::kSmemBytes, st>>>(dc, a, Dp, Tg);
          else if (sincos == 2) k_dense2_tc<false, 2><<<grid_tc, tc::kThreads, tc::kSmemBytes, st>>>(dc, a, Dp, Tg);
          else if (merge) k_dense2_tc<false, 0, true><<<grid_tc, tc::kThreads, tc::kSmemBytes, st>>>(dc, a, Dp, Tg);
          else k_dense2_tc<false, 0><<<grid_tc, tc::kThreads, tc::kSmemBytes, st>>>(dc, a, Dp, Tg);
        }
        else if (seg_mode && sincos == 2 && merge) k_dense2<true, 2, true><<<grid, kBlock, 0, st>>>(dc, a, Dp);
        else if (seg_mode && sincos == 2) k_dense2<true, 2><<<grid, kBlock, 0, st>>>(dc, a, Dp);
        else if (seg_mode && merge) k_dense2<true, 0, true><<<grid, kBlock, 0, st>>>(dc, a, Dp);
        else if (seg_mode) k_dense2<true, 0><<<grid, kBlock, 0, st>>>(dc, a, Dp);
        else if (sincos == 2 && merge && quad) k_dense2<false, 2, true, true><<<grid, kBlock, kDense2Smem, st>>>(dc, a, Dp);
        else if (sincos == 2 && merge) k_dense2<false, 2, true><<<grid, kBlock, kDense2Smem, st>>>(dc, a, Dp);
        else if (sincos == 2) k_dense2<false, 2><<<grid, kBlock, kDense2Smem, st>>>(dc, a, Dp);
        else if (merge) k_dense2<false, 0, true><<<grid, kBlock, kDense2Smem, st>>>(dc, a, Dp);
        else k_dense2<false, 0><<<grid, kBlock, kDense2Smem, st>>>(dc, a, Dp);
      } else {
        if (seg_mode) k_dense<true><<<grid, kBlock, kDense64Smem, st>>>(dc, a, h->W64, h->G64);
        else if (esc_count) k_dense<false, true><<<grid, kBlock, kDense64Smem, st>>>(dc, a, h->W64, h->G64);
        else k_dense<false><<<grid, kBlock, kDense64Smem, st>>>(dc, a, h->W64, h->G64);
      }
    }
    if ((rc = check_launch(h, "k_dense"))) return rc;
    Timed tm2(h, st, cls_stitch);
    if (seg_mode) k_stitch_seg<<<(Pn + 127) / 128, 128, 0, st>>>(frag, h->d_flags, h->d_chunk_k0, n_chunks, P_pad, Pn, n_seg, sz, ss,
                                                                out_seg + (size_t)pb * n_seg * 3);
    else {
      // the hardware sin/cos gain g (g^2 = mufu_gain2) multiplies every |z_k|: Upsilon by g^2, O_hat by g, <h|h> not at all.
      // Units (whitened -> definition): Upsilon is scale free, x_k = 4 df |z_k| = |Z_k| s0 h0, [h|h]_k = Sg_k s0^2 h0^2.
      const double g2 = (sizeof(R) == 4 && sincos == 2) ? h->mufu_gain2 : 1.0;
      // many chunks: a particle's range folded in kStitchParts parts by as many threads, then joined (k_stitch_parts)
      if (!esc_count && n_chunks >= 64) {
        const int n_slots = sorted ? P_pad : Pn;
        k_stitch_parts<<<dim3((n_slots + 127) / 128, kStitchParts), 128, 0, st>>>(frag, h->d_flags, n_chunks, P_pad, n_slots, out_comp ? 1 : 0,
                                                                                 jlo, jhi, h->chunk_first, h->cached_chunk, stitch_rec);
        if ((rc = check_launch(h, "k_stitch_parts"))) return rc;
        k_stitch_join<<<(n_slots + 127) / 128, 128, 0, st>>>(stitch_rec, n_chunks, P_pad, Pn, 1.0 / g2, out ? out + pb : nullptr,
                                                            out_comp ? out_comp + pb * 3 : nullptr, h->s0 * h0 / sqrt(g2),
                                                            h->s0 * h->s0 * h0 * h0, sorted ? pmap : nullptr, jlo, jhi, h->chunk_first,
                                                            h->cached_chunk, h->d_next_close);
      } else
      k_stitch<<<esc_count ? pblocks : ((sorted ? P_pad : Pn) + 127) / 128, 128, 0, st>>>(frag, h->d_flags, n_chunks, P_pad, Pn, 1.0 / g2, out ? out + pb : nullptr,
                                                 out_comp ? out_comp + pb * 3 : nullptr, h->s0 * h0 / sqrt(g2),
                                                 h->s0 * h->s0 * h0 * h0, esc_count, (int)pb, sorted ? pmap : nullptr,
                                                 jlo, jhi, h->chunk_first, h->cached_chunk, h->d_next_close);
    }
    if ((rc = check_launch(h, "k_stitch"))) return rc;
  }
  return SC_OK;
}

// Pieces of the launched range for fine sub-intervals of 2^lg_fine bins: every sub-interval is cut at the distinct
// edges strictly inside it (the same walk k_dense2 does); their sigma moments are computed on the device.
int build_pieces(sc_handle* h, int CH, int lg_fine, cudaStream_t st) {
  const std::vector<int>& e = h->edges;
  const int Sf = 1 << lg_fine;
  const int nb2 = ((int)h->cfg.n_bins + 1) & ~1;
  const long long isub0 = (long long)h->chunk_first * CH / Sf;
  const int n_sub = (int)((long long)h->n_chunks * CH / Sf);
  std::vector<int> first((size_t)n_sub + 1), lo, hi;
  size_t idx = 0;
  for (int t = 0; t < n_sub; ++t) {
    first[t] = (int)lo.size();
    const long long ib = (isub0 + t) * Sf;
    if (ib >= nb2) continue;
    const int iek = (int)std::min<long long>(ib + Sf, nb2);
    int cur = (int)ib;
    while (idx < e.size() && e[idx] <= ib) ++idx;
    while (idx < e.size() && e[idx] < iek) {
      if (e[idx] > cur) { lo.push_back(cur); hi.push_back(e[idx]); cur = e[idx]; }
      ++idx;
    }
    lo.push_back(cur); hi.push_back(iek);
  }
  first[n_sub] = (int)lo.size();
  h->n_pieces = (int)lo.size();
  int rc;
  if ((rc = grow(h, (void**)&h->d_piece_first, &h->pf_cap, first.size() * 4))) return rc;
  if ((rc = grow(h, (void**)&h->d_piece_lo, &h->plo_cap, std::max<size_t>(lo.size(), 1) * 4))) return rc;
  if ((rc = grow(h, (void**)&h->d_piece_hi, &h->phi_cap, std::max<size_t>(hi.size(), 1) * 4))) return rc;
  if ((rc = grow(h, (void**)&h->d_moments, &h->mom_cap, std::max<size_t>(lo.size(), 1) * 8 * sizeof(float2)))) return rc;
  const bool f64 = (CH == kChunkF64);            // the all-FP64 kernel reads the moments in FP64
  if (f64 && (rc = grow(h, (void**)&h->d_moments64, &h->mom64_cap, std::max<size_t>(lo.size(), 1) * 7 * sizeof(double2)))) return rc;
  SC_CUDA(h, cudaMemcpyAsync(h->d_piece_first, first.data(), first.size() * 4, cudaMemcpyHostToDevice, st));
  if (h->n_pieces > 0) {
    SC_CUDA(h, cudaMemcpyAsync(h->d_piece_lo, lo.data(), lo.size() * 4, cudaMemcpyHostToDevice, st));
    SC_CUDA(h, cudaMemcpyAsync(h->d_piece_hi, hi.data(), hi.size() * 4, cudaMemcpyHostToDevice, st));
    SC_CUDA(h, cudaStreamSynchronize(st));       // the host vectors go out of scope
    Timed tm(h, st, SC_TIME_OTHER);
    k_moments<<<(h->n_pieces + 127) / 128, 128, 0, st>>>(h->G64, h->d_piece_lo, h->d_piece_hi, h->n_pieces, (int)h->cfg.n_bins,
                                                        lg_fine, h->d_moments, f64 ? h->d_moments64 : nullptr);
    if ((rc = check_launch(h, "k_moments"))) return rc;
    if (h->GT64 && !f64) {                         // fused three-channel kernel: the same moments of the T weights
      if ((rc = grow(h, (void**)&h->d_momentsT, &h->momT_cap, std::max<size_t>(lo.size(), 1) * 8 * sizeof(float2)))) return rc;
      k_moments<<<(h->n_pieces + 127) / 128, 128, 0, st>>>(h->GT64, h->d_piece_lo, h->d_piece_hi, h->n_pieces, (int)h->cfg.n_bins,
                                                          lg_fine, h->d_momentsT, nullptr);
      if ((rc = check_launch(h, "k_moments"))) return rc;
    }
  } else {
    SC_CUDA(h, cudaStreamSynchronize(st));
  }
  return SC_OK;
}

// lg_fine > 0: also build the piece tables of k_dense2 for fine sub-intervals of 2^lg_fine bins.
int prepare_edges(sc_handle* h, const int32_t* seg_edges, int32_t n_seg, int CH, int lg_fine, cudaStream_t st) {
  if (!seg_edges || n_seg <= 0) return fail(h, SC_ERR_INVALID_ARG, "seg_edges is null or n_seg <= 0");
  std::vector<int> e((size_t)n_seg + 1);
  cudaPointerAttributes at;
  cudaError_t pe = cudaPointerGetAttributes(&at, seg_edges);
  if (pe != cudaSuccess) { cudaGetLastError(); at.type = cudaMemoryTypeUnregistered; }
  if (at.type == cudaMemoryTypeDevice) {
    SC_CUDA(h, cudaMemcpyAsync(e.data(), seg_edges, e.size() * 4, cudaMemcpyDeviceToHost, st));
    SC_CUDA(h, cudaStreamSynchronize(st));
  } else {
    memcpy(e.data(), seg_edges, e.size() * 4);
  }
  if (e[0] < 0 || e[n_seg] > h->cfg.n_bins) return fail(h, SC_ERR_INVALID_ARG, "seg_edges outside [0, n_bins]");
  for (int k = 0; k < n_seg; ++k)
    if (e[k + 1] < e[k]) return fail(h, SC_ERR_INVALID_ARG, "seg_edges not non-decreasing at k=%d", k);
  if (e == h->edges && CH == h->cached_chunk && lg_fine == h->cached_lg) return SC_OK;
  h->edges.swap(e);
  analyse_edges(h, CH);
  h->cached_lg = lg_fine;
  // (the cache key is valid only once every table below is on the device: any failure invalidates it)
  auto upload = [&]() -> int {
    int rc;
    if (lg_fine > 0 && (rc = build_pieces(h, CH, lg_fine, st))) return rc;
    if ((rc = grow(h, (void**)&h->d_edges, &h->edge_cap, h->edges.size() * 4))) return rc;
    if ((rc = grow(h, (void**)&h->d_chunk_k0, &h->k0_cap, (size_t)std::max(h->n_chunks, 1) * 4))) return rc;
    if ((rc = grow(h, (void**)&h->d_flags, &h->flags_cap, (size_t)std::max(h->n_chunks, 1)))) return rc;
    if ((rc = grow(h, (void**)&h->d_next_close, &h->nc_cap, (size_t)std::max(h->n_chunks, 1) * 4))) return rc;
    SC_CUDA(h, cudaMemcpyAsync(h->d_edges, h->edges.data(), h->edges.size() * 4, cudaMemcpyHostToDevice, st));
    if (h->n_chunks > 0) {
      SC_CUDA(h, cudaMemcpyAsync(h->d_chunk_k0, h->chunk_k0.data(), (size_t)h->n_chunks * 4, cudaMemcpyHostToDevice, st));
      SC_CUDA(h, cudaMemcpyAsync(h->d_flags, h->flags.data(), (size_t)h->n_chunks, cudaMemcpyHostToDevice, st));
      SC_CUDA(h, cudaMemcpyAsync(h->d_next_close, h->next_close.data(), (size_t)h->n_chunks * 4, cudaMemcpyHostToDevice, st));
    }
    return SC_OK;
  };
  const int rc = upload();
  if (rc) { h->cached_chunk = 0; h->cached_lg = 0; h->edges.clear(); }
  return rc;
}

int eval_common(sc_handle* h, const double* params, int64_t P, const int32_t* seg_edges, int32_t n_seg,
                double* out, double* out_seg, void* stream, bool seg_mode, double* out_comp = nullptr, bool fused3 = false) {
  // fused3: the one-pass three-channel kernel (FP32-amplitude path of a three-channel handle; the caller escalates)
  if (!h) return SC_ERR_NOT_INIT;
  if (h->cuda_failed) return SC_ERR_CUDA;
  if (!params || P <= 0 || (!seg_mode && !out && !out_comp) || (seg_mode && !out_seg))
    return fail(h, SC_ERR_INVALID_ARG, "null pointer or n_particles <= 0");
  cudaStream_t st = (cudaStream_t)stream;
  const bool f64 = !fused3 && ((h->precision == 2) || (h->precision == 0 && n_seg < h->f32_min_seg));
  select_stride_f32(h, seg_mode ? 0 : n_seg);
  // all-FP64 path: sigma from FP64 piece moments when a fine sub-interval is long enough to pay for them (>= 32 bins)
  const int lg_fine64 = (h->lg_f64 - 2 >= 5) ? h->lg_f64 - 2 : 0;
  // chunk length: 1024 bins (all-FP64), 2048 (k_dense2: the chunk's data is staged in shared memory), 8192 (k_dense2_tc)
  const int ch32 = (h->use_tc && h->lg_f32 >= 7 && !fused3) ? tc::kChunk : kChunkF32;
  int rc = prepare_edges(h, seg_edges, n_seg, f64 ? kChunkF64 : ch32, f64 ? lg_fine64 : h->lg_f32 - 2, st);
  if (rc) return rc;
  SC_CUDA(h, cudaMemsetAsync(h->d_counter, 0, 8, st));
  if (seg_mode) SC_CUDA(h, cudaMemsetAsync(out_seg, 0, (size_t)P * n_seg * 3 * 8, st));
  if (f64) return run_batches<double>(h, params, P, out, out_seg, out_comp, st, seg_mode);
  if (fused3) return run_batches<float>(h, params, P, out, out_seg, out_comp, st, seg_mode, nullptr, 0, true);
  if ((rc = run_batches<float>(h, params, P, out, out_seg, out_comp, st, seg_mode))) return rc;
  // Escalation: the FP32 path's error is ~ c / sqrt(Upsilon) relative (c <= 1.0e-6 polynomial,
  // 1.6e-6 hardware sin/cos, measured against the oracle), so a particle whose statistic comes out below tau is evaluated
  // again by the all-FP64 path.  Device-side selection, no host synchronisation: the FP64 kernels are launched for the
  // worst case and their 128-particle blocks beyond the selected count return at once.
  if (h->escalate && h->precision == 0 && !seg_mode && out && !out_comp && h->n_chunks > 0) {
    if (P > INT32_MAX / 16) return SC_OK;
    const bool mufu = (h->sincos_mode == 0) ? (n_seg >= h->mufu_min_seg) : (h->sincos_mode == 2);
    const size_t P_round = (size_t)((P + kBlock - 1) / kBlock * kBlock);
    if ((rc = grow(h, (void**)&h->d_esc_idx, &h->esc_idx_cap, (size_t)P * 4))) return rc;
    if ((rc = grow(h, (void**)&h->d_esc_count, &h->esc_cnt_cap, 256))) return rc;
    if ((rc = grow(h, (void**)&h->d_esc_params, &h->esc_par_cap, P_round * 64))) return rc;
    if ((rc = grow(h, (void**)&h->d_esc_out, &h->esc_out_cap, P_round * 8))) return rc;
    {
      Timed tm(h, st, SC_TIME_ESC);
      k_esc_select<<<1, 1024, 0, st>>>(out, params, (int)P, std::max(mufu ? h->esc_tau_mufu : h->esc_tau_poly, h->esc_tau_nodes), h->d_esc_idx,
                                       h->d_esc_count, h->d_esc_params);
    }
    if ((rc = check_launch(h, "k_esc_select"))) return rc;
    // grid-size hint: the count of the latest selection whose copy has landed (possibly an earlier call's); the kernels
    // stride over the selected particles, so a stale or low hint costs parallelism, never correctness
    if (!h->h_esc_hint) { SC_CUDA(h, cudaMallocHost((void**)&h->h_esc_hint, 4)); *h->h_esc_hint = (int)std::min<int64_t>(P, 1024); }
    const int hint = *(volatile int*)h->h_esc_hint;
    SC_CUDA(h, cudaMemcpyAsync(h->h_esc_hint, h->d_esc_count, 4, cudaMemcpyDeviceToHost, st));
    const int esc_blocks = (int)std::min<int64_t>((2LL * hint + kBlock - 1) / kBlock + 1, (int64_t)P_round / kBlock);
    const std::vector<int> e_host = h->edges;                  // host copy: the alternate cache analyses the same list
    std::swap(static_cast<EdgeCache&>(*h), h->alt);
    rc = prepare_edges(h, e_host.data(), n_seg, kChunkF64, lg_fine64, st);
    if (!rc) rc = run_batches<double>(h, h->d_esc_params, P, h->d_esc_out, nullptr, nullptr, st, false, h->d_esc_count, esc_blocks);
    std::swap(static_cast<EdgeCache&>(*h), h->alt);
    if (rc) return rc;
    Timed tm(h, st, SC_TIME_ESC);
    k_esc_scatter<<<(unsigned)((P + 127) / 128), 128, 0, st>>>(h->d_esc_idx, h->d_esc_count, h->d_esc_out, out);
    if ((rc = check_launch(h, "k_esc_scatter"))) return rc;
  }
  return SC_OK;
}

// ------------------------------------------------------------------------------------------------ three channels (A, E, T)
// out = 4 df sum_k |zAE_k + zT_k|^2 / (sigAE_k + sigT_k) from the per-segment sums of the two passes (definition units),
// optionally the combined segments and the Eq. 8 / Eq. 3 components.
__global__ void k_combine3(const double* __restrict__ segA, const double* __restrict__ segT, int P, int n_seg, double four_df,
                           double* __restrict__ out, double* __restrict__ out_seg, double* __restrict__ comp3) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P) return;
  double ups = 0.0, xs = 0.0, hs = 0.0;
  for (int k = 0; k < n_seg; ++k) {
    const size_t at = ((size_t)p * n_seg + k) * 3;
    const double zr = segA[at] + segT[at], zi = segA[at + 1] + segT[at + 1], sg = segA[at + 2] + segT[at + 2];
    if (out_seg) { out_seg[at] = zr; out_seg[at + 1] = zi; out_seg[at + 2] = sg; }
    if (sg > 0.0) {
      const double z2 = zr * zr + zi * zi;
      ups += z2 / sg; xs += sqrt(z2); hs += sg;
    }
  }
  if (out) out[p] = four_df * ups;
  if (comp3) { comp3[3 * (size_t)p] = four_df * ups; comp3[3 * (size_t)p + 1] = four_df * xs; comp3[3 * (size_t)p + 2] = four_df * hs; }
}

// Statistic / segments / components of a handle with or without the T channel.
int eval_any(sc_handle* h, const double* params, int64_t P, const int32_t* seg_edges, int32_t n_seg,
             double* out, double* out_seg, void* stream, bool seg_mode, double* out_comp = nullptr) {
  if (!h) return SC_ERR_NOT_INIT;
  if (!h->sub) return eval_common(h, params, P, seg_edges, n_seg, out, out_seg, stream, seg_mode, out_comp);
  if (h->cuda_failed) return SC_ERR_CUDA;
  if (!params || P <= 0 || (!seg_mode && !out && !out_comp) || (seg_mode && !out_seg) || !seg_edges || n_seg <= 0)
    return fail(h, SC_ERR_INVALID_ARG, "null pointer, n_particles <= 0 or n_seg <= 0");
  cudaStream_t st = (cudaStream_t)stream;
  const size_t per_p = (size_t)n_seg * 24;                     // one particle's row of a segment table
  const double four_df = 4.0 / h->cfg.T_obs_s;
  int rc;
  const bool f32_path = (h->precision == 1) || (h->precision == 0 && n_seg >= h->f32_min_seg);
  // Escalation on three channels (SC_OPT_ESCALATE): the FP32-amplitude kernels leave an error ~ 1e-6 / sqrt(Upsilon), so the
  // particles whose COMBINED statistic is below tau are evaluated again by the all-FP64 kernels -- two passes in
  // segment-table mode, combined, scattered back.  The selected count is read back (one 4-byte copy per call or batch).
  auto escalate3 = [&](double* outp, const double* par, int64_t Pn) -> int {
    if (!(h->escalate && h->precision == 0 && f32_path && !seg_mode && outp && !out_comp && Pn <= INT32_MAX / 16)) return SC_OK;
    int rc2;
    const size_t P_round = (size_t)((Pn + kBlock - 1) / kBlock * kBlock);
    if ((rc2 = grow(h, (void**)&h->d_esc_idx, &h->esc_idx_cap, (size_t)Pn * 4))) return rc2;
    if ((rc2 = grow(h, (void**)&h->d_esc_count, &h->esc_cnt_cap, 256))) return rc2;
    if ((rc2 = grow(h, (void**)&h->d_esc_params, &h->esc_par_cap, P_round * 64))) return rc2;
    if ((rc2 = grow(h, (void**)&h->d_esc_out, &h->esc_out_cap, P_round * 8))) return rc2;
    {
      Timed tm(h, st, SC_TIME_ESC);
      const bool mufu3 = (h->sincos_mode == 0) ? (n_seg >= h->mufu_min_seg) : (h->sincos_mode == 2);
      k_esc_select<<<1, 1024, 0, st>>>(outp, par, (int)Pn, std::max(mufu3 ? h->esc_tau_mufu : h->esc_tau_poly, h->esc_tau_nodes), h->d_esc_idx, h->d_esc_count, h->d_esc_params);
    }
    if ((rc2 = check_launch(h, "k_esc_select"))) return rc2;
    int n_esc = 0;
    SC_CUDA(h, cudaMemcpyAsync(&n_esc, h->d_esc_count, 4, cudaMemcpyDeviceToHost, st));
    SC_CUDA(h, cudaStreamSynchronize(st));
    if (n_esc <= 0) return SC_OK;
    // (the tables of the main passes are not needed any more: a call with the fused kernel has none, the two-pass loop has combined its batch)
    if (2 * per_p * (size_t)n_esc > h->seg3_cap && (rc2 = grow(h, (void**)&h->d_seg3, &h->seg3_cap, 2 * per_p * (size_t)n_esc))) return rc2;
    double* eA = h->d_seg3; double* eT = eA + (size_t)n_esc * n_seg * 3;
    // (the all-FP64 chunking of the same edges lives in the alternate cache, as in eval_common's own escalation pass: the
    // FP32 kernels' analysis of the list stays valid for the next call)
    h->precision = 2; h->sub->precision = 2;
    std::swap(static_cast<EdgeCache&>(*h), h->alt);
    rc2 = eval_common(h, h->d_esc_params, n_esc, seg_edges, n_seg, nullptr, eA, stream, true);
    std::swap(static_cast<EdgeCache&>(*h), h->alt);
    if (!rc2) rc2 = eval_common(h->sub, h->d_esc_params, n_esc, seg_edges, n_seg, nullptr, eT, stream, true);
    h->precision = 0; h->sub->precision = 0;
    if (rc2) return rc2;
    Timed tm(h, st, SC_TIME_ESC);
    k_combine3<<<(unsigned)((n_esc + 127) / 128), 128, 0, st>>>(eA, eT, n_esc, n_seg, four_df, h->d_esc_out, nullptr, nullptr);
    if ((rc2 = check_launch(h, "k_combine3"))) return rc2;
    k_esc_scatter<<<(unsigned)((Pn + 127) / 128), 128, 0, st>>>(h->d_esc_idx, h->d_esc_count, h->d_esc_out, outp);
    return check_launch(h, "k_esc_scatter");
  };

  // One pass (k_dense3: A, E, T in the pair loop) on the FP32-amplitude path; the all-FP64 modes take the two passes below.
  if (h->D3 && h->use_fused3 && f32_path) {
    if ((rc = eval_common(h, params, P, seg_edges, n_seg, out, out_seg, stream, seg_mode, out_comp, true))) return rc;
    return escalate3(out, params, P);
  }

  // Two passes, (A, E) and (T, nothing), through the two-channel kernels in segment-table mode, then the combination;
  // batches of particles such that the two segment tables fit in 2 GiB
  int64_t Pb = (int64_t)std::max<size_t>(1, ((size_t)1 << 30) / per_p);
  Pb = std::min<int64_t>(Pb, P);
  for (int64_t pb = 0; pb < P; pb += Pb) {
    const int64_t Pn = std::min<int64_t>(Pb, P - pb);
    if ((rc = grow(h, (void**)&h->d_seg3, &h->seg3_cap, 2 * per_p * (size_t)Pb))) return rc;
    double* segA = h->d_seg3; double* segT = segA + (size_t)Pb * n_seg * 3;
    if ((rc = eval_common(h, params + pb * 8, Pn, seg_edges, n_seg, nullptr, segA, stream, true))) return rc;
    if ((rc = eval_common(h->sub, params + pb * 8, Pn, seg_edges, n_seg, nullptr, segT, stream, true))) {
      fail(h, rc, "T pass: %s", h->sub->err.c_str());
      return rc;
    }
    {
      Timed tm(h, st, SC_TIME_STITCH);
      k_combine3<<<(unsigned)((Pn + 127) / 128), 128, 0, st>>>(segA, segT, (int)Pn, n_seg, four_df, out ? out + pb : nullptr,
                                                              seg_mode ? out_seg + (size_t)pb * n_seg * 3 : nullptr,
                                                              out_comp ? out_comp + pb * 3 : nullptr);
      if ((rc = check_launch(h, "k_combine3"))) return rc;
    }
    if ((rc = escalate3(out ? out + pb : nullptr, params + pb * 8, Pn))) return rc;
  }
  return SC_OK;
}

// Per-particle equal-SNR^2 segments: see the kernels above.  FP32-amplitude path.
int run_adaptive(sc_handle* h, const double* params, int64_t P, int n_seg, double* out, int32_t* out_edges, double* out_comp,
                 cudaStream_t st) {
  DevCfg dc = h->dc;
  select_stride_f32(h, 0);
  apply_stride(dc, h->lg_f32);
  const bool three = (h->sub != nullptr);        // three-channel handle: (A, E, T) in every step (NA = 6 amplitude fields)
  if (three) dc.chan_set = 2;
  const int NA = three ? 6 : 4;
  const int CH = kChunkF32;
  const int n_nodes = dc.n_nodes;
  const int n_chunks = (dc.n_bins + CH - 1) / CH;
  const int lg_fine = dc.log2_stride - 2, lg_group = std::min(5, lg_fine);
  int rc;
  // moments tables (shared by all particles; depend on the data and the node spacing only)
  const int n_groups = (int)(((long long)n_chunks * CH) >> lg_group), n_sub = (int)(((long long)n_chunks * CH) >> lg_fine);
  if (h->ad_lg != dc.log2_stride) {
    if ((rc = grow(h, (void**)&h->d_gmom, &h->gmom_cap, (size_t)n_groups * 8 * sizeof(float2)))) return rc;
    if ((rc = grow(h, (void**)&h->d_smom, &h->smom_cap, (size_t)n_sub * 8 * sizeof(float2)))) return rc;
    if ((rc = grow(h, (void**)&h->d_gmom64, &h->gmom64_cap, (size_t)n_groups * 7 * sizeof(double2)))) return rc;
    if ((rc = grow(h, (void**)&h->d_smom64, &h->smom64_cap, (size_t)n_sub * 7 * sizeof(double2)))) return rc;
    Timed tm(h, st, SC_TIME_OTHER);
    k_moments<<<(n_groups + 127) / 128, 128, 0, st>>>(h->G64, nullptr, (const int*)(size_t)lg_group, n_groups, dc.n_bins, lg_fine, h->d_gmom, h->d_gmom64);
    if ((rc = check_launch(h, "k_moments"))) return rc;
    k_moments<<<(n_sub + 127) / 128, 128, 0, st>>>(h->G64, nullptr, (const int*)(size_t)lg_fine, n_sub, dc.n_bins, lg_fine, h->d_smom, h->d_smom64);
    if ((rc = check_launch(h, "k_moments"))) return rc;
    if (three) {
      if ((rc = grow(h, (void**)&h->d_gmomT, &h->gmomT_cap, (size_t)n_groups * 8 * sizeof(float2)))) return rc;
      if ((rc = grow(h, (void**)&h->d_smomT, &h->smomT_cap, (size_t)n_sub * 8 * sizeof(float2)))) return rc;
      if ((rc = grow(h, (void**)&h->d_smom64T, &h->smom64T_cap, (size_t)n_sub * 7 * sizeof(double2)))) return rc;
      k_moments<<<(n_groups + 127) / 128, 128, 0, st>>>(h->GT64, nullptr, (const int*)(size_t)lg_group, n_groups, dc.n_bins, lg_fine, h->d_gmomT, nullptr);
      if ((rc = check_launch(h, "k_moments"))) return rc;
      k_moments<<<(n_sub + 127) / 128, 128, 0, st>>>(h->GT64, nullptr, (const int*)(size_t)lg_fine, n_sub, dc.n_bins, lg_fine, h->d_smomT, h->d_smom64T);
      if ((rc = check_launch(h, "k_moments"))) return rc;
    }
    h->ad_lg = dc.log2_stride;
  }
  // (FP64 node amplitudes: the edge decision is taken in FP64; the packed kernel converts them as it reads)
  const size_t per_p = 2 * ((size_t)kPcFields * 8 + 8) + 16 + (size_t)n_nodes * (4 + 8 + NA * sizeof(double))
                       + (size_t)(n_chunks + 1) * 8 + (size_t)n_chunks * kFragAd * 8 + (size_t)n_sub * 8;
  int64_t Pb_max = (int64_t)(h->scratch_cap / per_p) / kBlock * kBlock;
  if (Pb_max < kBlock) Pb_max = kBlock;
  const int64_t P_round = (P + kBlock - 1) / kBlock * kBlock;
  const int P_pad = (int)std::min<int64_t>(Pb_max, P_round);
  if ((rc = grow(h, &h->scratch, &h->scratch_bytes, per_p * (size_t)P_pad + 4096))) return rc;
  char* base = (char*)h->scratch;
  auto take = [&](size_t bytes) { char* r = base; base += (bytes + 255) / 256 * 256; return r; };
  double* pc = (double*)take((size_t)kPcFields * 8 * P_pad);
  int* jlo = (int*)take((size_t)4 * P_pad);
  int* jhi = (int*)take((size_t)4 * P_pad);
  int* node_n = (int*)take((size_t)n_nodes * 4 * P_pad);
  double* node_frac = (double*)take((size_t)n_nodes * 8 * P_pad);
  double* node_amp = (double*)take((size_t)n_nodes * NA * sizeof(double) * P_pad);
  double* cbase = (double*)take((size_t)(n_chunks + 1) * 8 * P_pad);
  double* frag = (double*)take((size_t)n_chunks * kFragAd * 8 * P_pad);
  double* sub_sigma = (double*)take((size_t)n_sub * 8 * P_pad);
  // window sort, as in run_batches
  const bool sorted = h->window_sort && P_pad > kBlock;
  double* pc_u = (double*)take((size_t)kPcFields * 8 * P_pad);
  int* jlo_u = (int*)take((size_t)4 * P_pad);
  int* jhi_u = (int*)take((size_t)4 * P_pad);
  int* key_s = (int*)take((size_t)4 * P_pad);
  int* iota = (int*)take((size_t)4 * P_pad);
  int* pmap = (int*)take((size_t)4 * P_pad);
  (void)base;
  size_t sort_bytes = 0;
  if (sorted) {
    if (cub::DeviceRadixSort::SortPairs(nullptr, sort_bytes, jlo_u, key_s, iota, pmap, P_pad, 0, 32, st) != cudaSuccess)
      return fail(h, SC_ERR_CUDA, "cub::DeviceRadixSort size query failed");
    if ((rc = grow(h, &h->d_sort_tmp, &h->sort_cap, sort_bytes + 256))) return rc;
    k_iota<<<(P_pad + 255) / 256, 256, 0, st>>>(iota, P_pad);
    if ((rc = check_launch(h, "k_iota"))) return rc;
  }

  const double four_df = 4.0 / h->cfg.T_obs_s;
  const int sincos = (h->sincos_mode == 0) ? (n_seg >= h->mufu_min_seg ? 2 : 0) : (h->sincos_mode == 2 ? 2 : 0);
  const double h0 = pow(dc.f_amp_ref, -7.0 / 6.0);
  (void)four_df;
  if (out_edges) SC_CUDA(h, cudaMemsetAsync(out_edges, 0, (size_t)P * (n_seg + 1) * 4, st));
  else if ((rc = grow(h, (void**)&h->d_ad_edges, &h->ad_edges_cap, (size_t)std::min<int64_t>(P, P_pad) * (n_seg + 1) * 4))) return rc;

  for (int64_t pb = 0; pb < P; pb += P_pad) {
    const int Pn = (int)std::min<int64_t>(P_pad, P - pb);
    {
      Timed tm(h, st, SC_TIME_NODES);
      k_particle_consts<<<(P_pad + 127) / 128, 128, 0, st>>>(dc, params + pb * 8, Pn, P_pad, sorted ? pc_u : pc, sorted ? jlo_u : jlo,
                                                            sorted ? jhi_u : jhi, 0, dc.n_bins, h->d_counter);
    }
    if ((rc = check_launch(h, "k_particle_consts"))) return rc;
    if (sorted) {
      Timed tm(h, st, SC_TIME_NODES);
      // keys: window centres, staged in jlo (the sorted copy of the windows is written by k_gather_sorted afterwards)
      k_sort_key<<<(P_pad + 255) / 256, 256, 0, st>>>(jlo_u, jhi_u, jlo, P_pad);
      if ((rc = check_launch(h, "k_sort_key"))) return rc;
      if (cub::DeviceRadixSort::SortPairs(h->d_sort_tmp, sort_bytes, jlo, key_s, iota, pmap, P_pad, 0, 32, st) != cudaSuccess)
        return fail(h, SC_ERR_CUDA, "cub::DeviceRadixSort::SortPairs failed");
      h->launches += 3;
      k_gather_sorted<<<(P_pad + 127) / 128, 128, 0, st>>>(pmap, P_pad, pc_u, jlo_u, jhi_u, pc, jlo, jhi);
      if ((rc = check_launch(h, "k_gather_sorted"))) return rc;
    }
    {
      Timed tm(h, st, SC_TIME_NODES);
      // (the consumers read a node only where a lane of the warp is inside its window: skip_unreached)
      if (three) k_nodes<double, false, 6><<<dim3((n_nodes + kNodesPerCta - 1) / kNodesPerCta, (P_pad + 127) / 128), 128, 0, st>>>(dc, pc, jlo, jhi, P_pad, node_n, node_frac, node_amp, nullptr, 0, 1);
      else k_nodes<double><<<dim3((n_nodes + kNodesPerCta - 1) / kNodesPerCta, (P_pad + 127) / 128), 128, 0, st>>>(dc, pc, jlo, jhi, P_pad, node_n, node_frac, node_amp, nullptr, 0, 1);
    }
    if ((rc = check_launch(h, "k_nodes"))) return rc;
    DenseArgs a = {};
    a.node_n = node_n; a.node_frac = node_frac; a.node_amp = node_amp; a.jlo = jlo; a.jhi = jhi; a.P_pad = P_pad;
    a.frag = frag; a.P = Pn; a.comp = out_comp ? 1 : 0; a.n_seg = n_seg;
    AdaptArgs ad = {};
    ad.n_seg = n_seg; ad.n_chunks = n_chunks; ad.cbase = cbase; ad.chunk_sigma = cbase;
    ad.gmom = reinterpret_cast<const ulonglong2*>(h->d_gmom); ad.smom = reinterpret_cast<const ulonglong2*>(h->d_smom);
    ad.lg_group = lg_group;
    ad.out_edges = out_edges ? out_edges + (size_t)pb * (n_seg + 1) : h->d_ad_edges;
    ad.pmap = sorted ? pmap : nullptr;
    ad.smom64 = h->d_smom64; ad.gmom64 = h->d_gmom64; ad.G64 = h->G64; ad.sub_sigma = sub_sigma;
    ad.gmomT = reinterpret_cast<const ulonglong2*>(h->d_gmomT); ad.smomT = reinterpret_cast<const ulonglong2*>(h->d_smomT);
    ad.smom64T = h->d_smom64T; ad.GT64 = h->GT64;
    const dim3 grid(n_chunks, P_pad / kBlock);
    {
      Timed tm(h, st, SC_TIME_OTHER);
      if (three) k_sigma_chunks64<6><<<grid, kBlock, 0, st>>>(dc, a, ad);
      else k_sigma_chunks64<4><<<grid, kBlock, 0, st>>>(dc, a, ad);
      if ((rc = check_launch(h, "k_sigma_chunks64"))) return rc;
      k_scan_chunks<<<(P_pad + 127) / 128, 128, 0, st>>>(cbase, n_chunks, P_pad);
      if ((rc = check_launch(h, "k_scan_chunks"))) return rc;
      if (three) k_edges64<6><<<grid, kBlock, 0, st>>>(dc, a, ad);
      else k_edges64<4><<<grid, kBlock, 0, st>>>(dc, a, ad);
      if ((rc = check_launch(h, "k_edges64"))) return rc;
    }
    {
      Timed tm(h, st, SC_TIME_DENSE);
      const ulonglong2* Dp = reinterpret_cast<const ulonglong2*>(h->D32);
      const bool merge = dc.stride >= 512;                     // as in run_batches
      const bool quad = h->quad_amp && dc.stride >= 1024 && (long long)dc.n_bins >= 128LL * n_seg;
      a.merge_lim = 86400.0 * (kNodeDaysF32 / 4.0) / h->cfg.T_obs_s;
      if (three) {
        const ulonglong2* D3p = reinterpret_cast<const ulonglong2*>(h->D3);
        const ulonglong2* Gp = reinterpret_cast<const ulonglong2*>(h->Gp3);
        if (sincos == 2 && quad) k_dense2_ad<2, false, 6, true><<<grid, kBlock, 0, st>>>(dc, a, ad, D3p, Gp);
        else if (sincos == 2) k_dense2_ad<2, false, 6><<<grid, kBlock, 0, st>>>(dc, a, ad, D3p, Gp);
        else k_dense2_ad<0, false, 6><<<grid, kBlock, 0, st>>>(dc, a, ad, D3p, Gp);
      }
      else if (sincos == 2 && merge && quad) k_dense2_ad<2, true, 4, true><<<grid, kBlock, 0, st>>>(dc, a, ad, Dp);
      else if (sincos == 2 && merge) k_dense2_ad<2, true><<<grid, kBlock, 0, st>>>(dc, a, ad, Dp);
      else if (sincos == 2) k_dense2_ad<2><<<grid, kBlock, 0, st>>>(dc, a, ad, Dp);
      else if (merge) k_dense2_ad<0, true><<<grid, kBlock, 0, st>>>(dc, a, ad, Dp);
      else k_dense2_ad<0><<<grid, kBlock, 0, st>>>(dc, a, ad, Dp);
    }
    if ((rc = check_launch(h, "k_dense2_ad"))) return rc;
    Timed tm2(h, st, SC_TIME_STITCH);
    const double g2 = (sincos == 2) ? h->mufu_gain2 : 1.0;
    k_stitch_ad<<<((sorted ? P_pad : Pn) + 127) / 128, 128, 0, st>>>(frag, n_chunks, P_pad, Pn, 1.0 / g2, out ? out + pb : nullptr,
                                                  out_comp ? out_comp + pb * 3 : nullptr, h->s0 * h0 / sqrt(g2),
                                                  h->s0 * h->s0 * h0 * h0, out_edges ? ad.out_edges : nullptr, n_seg, dc.n_bins, ad.pmap, jlo, jhi, CH);
    if ((rc = check_launch(h, "k_stitch_ad"))) return rc;
  }
  return SC_OK;
}

__global__ void k_fill_edges01(int* __restrict__ out_edges, int P, int n_bins) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p < P) { out_edges[2 * (size_t)p] = 0; out_edges[2 * (size_t)p + 1] = n_bins; }
}

int init_common(sc_handle** out, const sc_config* cfg, const double* dA, const double* dE, const double* S_A,
                const double* S_E, void* stream, bool host_inputs, int chan_set = 0) {
  if (!out) return fail(nullptr, SC_ERR_INVALID_ARG, "out is null");
  *out = nullptr;
  if (!cfg || !dA || !dE || !S_A || !S_E) return fail(nullptr, SC_ERR_INVALID_ARG, "null pointer");
  if (!(cfg->T_obs_s > 0.0) || cfg->n_bins < 1 || cfg->n_bins >= (int64_t)1 << 31 || cfg->j0 < 0)
    return fail(nullptr, SC_ERR_INVALID_ARG, "bad grid (T_obs_s, j0, n_bins)");
  if (cfg->n_channels != 2) return fail(nullptr, SC_ERR_INVALID_ARG, "n_channels must be 2 (A,E) here; three channels: sc_init_data3");
  if (cfg->pn_order_x2 < 0 || cfg->pn_order_x2 > 7) return fail(nullptr, SC_ERR_INVALID_ARG, "pn_order_x2 must be 0..7");
  if (cfg->window_mode != 0 && cfg->window_mode != 1) return fail(nullptr, SC_ERR_INVALID_ARG, "window_mode must be 0 or 1");
  if (!(cfg->arm_L_s > 0.0) || !(cfg->au_s > 0.0) || !(cfg->year_s > 0.0))
    return fail(nullptr, SC_ERR_INVALID_ARG, "orbit constants must be positive");
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return fail(nullptr, SC_ERR_CUDA, "no CUDA device (%s); this library has no CPU fallback",
                e == cudaSuccess ? "device count 0" : cudaGetErrorString(e));
  }
  sc_handle* h = new sc_handle();
  h->cfg = *cfg;
  cudaStream_t st = (cudaStream_t)stream;
  const int n = (int)cfg->n_bins;
  DevCfg& d = h->dc;
  d.T_obs = cfg->T_obs_s; d.inv_T = 1.0 / cfg->T_obs_s; d.j0 = cfg->j0; d.n_bins = n;
  d.window_mode = cfg->window_mode; d.pn_order_x2 = cfg->pn_order_x2; d.ecc_leading = cfg->ecc_leading;
  d.f_ref_ecc = cfg->f_ref_ecc; d.L = cfg->arm_L_s; d.AU = cfg->au_s; d.alpha0 = cfg->orbit_alpha0; d.year = cfg->year_s;
  for (int m = 0; m < 3; ++m) {
    const double b = 2.0 * kPi * m / 3.0 + cfg->orbit_lambda0;
    d.sbn[m] = sin(b); d.cbn[m] = cos(b);
  }
  d.f_amp_ref = (double)std::max<int64_t>(cfg->j0, 1) / cfg->T_obs_s;
  d.chan_set = chan_set;
  set_stride(h);
  auto bail = [&](int code) { sc_free(h); return code; };
#define SC_INIT(call)                                                                              \
  do { cudaError_t e_ = (call);                                                                    \
       if (e_ != cudaSuccess) { fail(nullptr, e_ == cudaErrorMemoryAllocation ? SC_ERR_OOM : SC_ERR_CUDA, \
                                     "%s failed: %s", #call, cudaGetErrorString(e_));              \
                                return bail(e_ == cudaErrorMemoryAllocation ? SC_ERR_OOM : SC_ERR_CUDA); } } while (0)
  SC_INIT(cudaGetDevice(&h->device));
  // the all-FP64 kernel stages 64 KB per CTA in dynamic shared memory
  SC_INIT(cudaFuncSetAttribute(k_dense<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kDense64Smem));
  SC_INIT(cudaFuncSetAttribute(k_dense<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kDense64Smem));
  SC_INIT(cudaFuncSetAttribute(k_dense<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kDense64Smem));
  SC_INIT(cudaFuncSetAttribute(k_dense2<false, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kDense2Smem));
  SC_INIT(cudaFuncSetAttribute(k_dense2<false, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, kDense2Smem));
  SC_INIT(cudaFuncSetAttribute(k_dense2<false, 2, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kDense2Smem));
  SC_INIT(cudaFuncSetAttribute(k_dense2<false, 2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kDense2Smem));
  SC_INIT(cudaFuncSetAttribute(k_dense2<false, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, kDense2Smem));
  SC_INIT(cudaFuncSetAttribute(k_dense2_tc<true, 0, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, tc::kSmemBytes));
  SC_INIT(cudaFuncSetAttribute(k_dense2_tc<false, 2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, tc::kSmemBytes));
  SC_INIT(cudaFuncSetAttribute(k_dense2_tc<false, 2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, tc::kSmemBytes));
  SC_INIT(cudaFuncSetAttribute(k_dense2_tc<false, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, tc::kSmemBytes));
  SC_INIT(cudaFuncSetAttribute(k_dense2_tc<false, 0, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, tc::kSmemBytes));
  const int n_pairs_pad = (n + tc::kChunk - 1) / tc::kChunk * (tc::kChunk / 2);   // whole chunks of either FP32-amplitude kernel
  SC_INIT(cudaMalloc(&h->D32, (size_t)n_pairs_pad * kPairRec * sizeof(float4)));
  SC_INIT(cudaMalloc(&h->W64, (size_t)n * sizeof(double4)));
  SC_INIT(cudaMalloc(&h->G64, (size_t)n * sizeof(double2)));
  SC_INIT(cudaMalloc(&h->d_counter, 16));
  SC_INIT(cudaMemsetAsync(h->d_counter, 0, 16, st));
  double* stage = nullptr;
  const double *pA = dA, *pE = dE, *pSA = S_A, *pSE = S_E;
  if (host_inputs) {
    SC_INIT(cudaMalloc(&stage, (size_t)n * 6 * 8));
    SC_INIT(cudaMemcpyAsync(stage, dA, (size_t)n * 16, cudaMemcpyHostToDevice, st));
    SC_INIT(cudaMemcpyAsync(stage + 2 * (size_t)n, dE, (size_t)n * 16, cudaMemcpyHostToDevice, st));
    SC_INIT(cudaMemcpyAsync(stage + 4 * (size_t)n, S_A, (size_t)n * 8, cudaMemcpyHostToDevice, st));
    SC_INIT(cudaMemcpyAsync(stage + 5 * (size_t)n, S_E, (size_t)n * 8, cudaMemcpyHostToDevice, st));
    pA = stage; pE = stage + 2 * (size_t)n; pSA = stage + 4 * (size_t)n; pSE = stage + 5 * (size_t)n;
  }
  const double four_df = 4.0 / cfg->T_obs_s;
  k_max_weight<<<std::min((n + 255) / 256, 1184), 256, 0, st>>>(pSA, pSE, n, four_df, h->d_counter + 1);
  h->launches++;
  unsigned long long bits = 0;
  SC_INIT(cudaMemcpyAsync(&bits, h->d_counter + 1, 8, cudaMemcpyDeviceToHost, st));
  SC_INIT(cudaStreamSynchronize(st));
  double umax;
  memcpy(&umax, &bits, 8);
  int ex = 0;
  if (umax > 0.0 && std::isfinite(umax)) { frexp(umax, &ex); }       // umax = m 2^ex, m in [0.5, 1)
  h->s0 = ldexp(1.0, (ex + 1) / 2);                                   // s0^2 >= umax, power of two
  k_whiten<<<(n_pairs_pad + 255) / 256, 256, 0, st>>>(pA, pE, pSA, pSE, n, n_pairs_pad, four_df, 1.0 / h->s0, h->D32, h->W64, h->G64);
  h->launches++;
  SC_INIT(cudaGetLastError());
  k_mufu_gain<<<1, 1024, 0, st>>>((double*)(h->d_counter + 1));
  h->launches++;
  SC_INIT(cudaMemcpyAsync(&h->mufu_gain2, h->d_counter + 1, 8, cudaMemcpyDeviceToHost, st));
  SC_INIT(cudaStreamSynchronize(st));
  if (!(h->mufu_gain2 > 0.999 && h->mufu_gain2 < 1.001)) {
    fail(nullptr, SC_ERR_CUDA, "hardware sin/cos gain calibration out of range (%g)", h->mufu_gain2);
    return bail(SC_ERR_CUDA);
  }
  {
    double* part = nullptr;
    SC_INIT(cudaMalloc(&part, 256 * 8));
    k_data_norm<<<256, 256, 0, st>>>(h->W64, h->G64, n, part);
    h->launches++;
    double hp[256];
    SC_INIT(cudaMemcpyAsync(hp, part, sizeof hp, cudaMemcpyDeviceToHost, st));
    SC_INIT(cudaStreamSynchronize(st));
    cudaFree(part);
    double acc = 0.0;
    for (int i = 0; i < 256; ++i) acc += hp[i];
    h->dd = acc;      // |W|^2/G = |d|^2 4df/S: the scale s0 cancels
  }
  if (stage) { SC_INIT(cudaStreamSynchronize(st)); cudaFree(stage); }
#undef SC_INIT
  *out = h;
  return SC_OK;
}

}  // namespace

extern "C" {

int sc_init_data(sc_handle** out, const sc_config* cfg, const double* dA, const double* dE, const double* S_A,
                 const double* S_E, void* stream) {
  return init_common(out, cfg, dA, dE, S_A, S_E, stream, false);
}

int sc_init_data_host(sc_handle** out, const sc_config* cfg, const double* dA, const double* dE, const double* S_A,
                      const double* S_E, void* stream) {
  return init_common(out, cfg, dA, dE, S_A, S_E, stream, true);
}

int sc_init_data3(sc_handle** out, const sc_config* cfg, const double* dA, const double* dE, const double* dT,
                  const double* S_A, const double* S_E, const double* S_T, void* stream) {
  if (!out) return fail(nullptr, SC_ERR_INVALID_ARG, "out is null");
  *out = nullptr;
  if (!cfg || !dT || !S_T) return fail(nullptr, SC_ERR_INVALID_ARG, "null pointer");
  if (cfg->n_channels != 3) return fail(nullptr, SC_ERR_INVALID_ARG, "sc_init_data3 needs n_channels = 3");
  sc_config c2 = *cfg;
  c2.n_channels = 2;
  sc_handle* h = nullptr;
  int rc = init_common(&h, &c2, dA, dE, S_A, S_E, stream, false, 0);
  if (rc) return rc;
  // T pass: (T, nothing) with the PSD S_T in both slots (the second slot carries zero data and a zero template)
  double* zeros = nullptr;
  if (cudaMalloc(&zeros, (size_t)cfg->n_bins * 16) != cudaSuccess) { cudaGetLastError(); sc_free(h); return fail(nullptr, SC_ERR_OOM, "cudaMalloc failed"); }
  cudaMemsetAsync(zeros, 0, (size_t)cfg->n_bins * 16, (cudaStream_t)stream);
  rc = init_common(&h->sub, &c2, dT, zeros, S_T, S_T, stream, false, 1);
  cudaStreamSynchronize((cudaStream_t)stream);
  cudaFree(zeros);
  if (rc) { sc_free(h); return rc; }
  h->cfg.n_channels = 3;
  // fused tables of the one-pass kernel k_dense3: T's whitened data and weights at the (A, E) handle's scale
  {
    const int n = (int)cfg->n_bins;
    const int n_pairs_pad = (n + tc::kChunk - 1) / tc::kChunk * (tc::kChunk / 2);
    cudaStream_t st = (cudaStream_t)stream;
    if (cudaMalloc(&h->D3, (size_t)n_pairs_pad * 3 * sizeof(float4)) != cudaSuccess ||
        cudaMalloc(&h->Gp3, (size_t)n_pairs_pad * 2 * sizeof(float4)) != cudaSuccess ||
        cudaMalloc(&h->GT64, (size_t)n * sizeof(double2)) != cudaSuccess) {
      cudaGetLastError(); sc_free(h); return fail(nullptr, SC_ERR_OOM, "cudaMalloc failed (fused three-channel tables)");
    }
    const float r = (float)(h->sub->s0 / h->s0);              // both powers of two
    k_fuse3<<<(n_pairs_pad + 255) / 256, 256, 0, st>>>(h->D32, h->sub->D32, h->sub->G64, n_pairs_pad, n, r, h->D3, h->Gp3, h->GT64);
    h->launches++;
    if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) { sc_free(h); return fail(nullptr, SC_ERR_CUDA, "k_fuse3 failed"); }
  }
  *out = h;
  return SC_OK;
}

int sc_gen_template3(sc_handle* h, const double* params, int64_t P, double* hA, double* hE, double* hT, void* stream) {
  if (!h) return SC_ERR_NOT_INIT;
  if (!h->sub) return fail(h, SC_ERR_INVALID_ARG, "not a three-channel handle");
  if (!hT) return fail(h, SC_ERR_INVALID_ARG, "hT is null");
  int rc = sc_gen_template(h, params, P, hA, hE, stream);
  if (rc) return rc;
  // the T pass writes T into its first slot; its second (empty) slot goes to scratch
  cudaStream_t st = (cudaStream_t)stream;
  double* dump = nullptr;
  SC_CUDA(h, cudaMalloc(&dump, (size_t)P * h->cfg.n_bins * 16));
  rc = sc_gen_template(h->sub, params, P, hT, dump, stream);
  cudaStreamSynchronize(st);
  cudaFree(dump);
  if (rc) fail(h, rc, "T pass: %s", h->sub->err.c_str());
  return rc;
}

int sc_eval_stat(sc_handle* h, const double* params, int64_t P, const int32_t* seg_edges, int32_t n_seg, double* out,
                 void* stream) {
  return eval_any(h, params, P, seg_edges, n_seg, out, nullptr, stream, false);
}

int sc_eval_segments(sc_handle* h, const double* params, int64_t P, const int32_t* seg_edges, int32_t n_seg,
                     double* out_seg, void* stream) {
  return eval_any(h, params, P, seg_edges, n_seg, nullptr, out_seg, stream, true);
}

int sc_eval_components(sc_handle* h, const double* params, int64_t P, const int32_t* seg_edges, int32_t n_seg,
                       double* out3, void* stream) {
  if (!out3) return h ? fail(h, SC_ERR_INVALID_ARG, "out3 is null") : SC_ERR_NOT_INIT;
  return eval_any(h, params, P, seg_edges, n_seg, nullptr, nullptr, stream, false, out3);
}

int sc_eval_loglike(sc_handle* h, const double* params, const double* amp, int64_t P, const int32_t* seg_edges,
                    int32_t n_seg, double* out, void* stream) {
  if (!h) return SC_ERR_NOT_INIT;
  if (h->cuda_failed) return SC_ERR_CUDA;
  if (!params || !amp || !out || P <= 0) return fail(h, SC_ERR_INVALID_ARG, "null pointer or n_particles <= 0");
  int rc = grow(h, (void**)&h->d_comp, &h->comp_cap, (size_t)P * 24);
  if (rc) return rc;
  if ((rc = eval_any(h, params, P, seg_edges, n_seg, nullptr, nullptr, stream, false, h->d_comp))) return rc;
  k_loglike<<<(unsigned)((P + 127) / 128), 128, 0, (cudaStream_t)stream>>>(h->d_comp, amp, h->dd, (int)P, out);
  return check_launch(h, "k_loglike");
}

int sc_data_norm(sc_handle* h, double* dd) {
  if (!h) return SC_ERR_NOT_INIT;
  if (!dd) return fail(h, SC_ERR_INVALID_ARG, "dd is null");
  *dd = h->dd + (h->sub ? h->sub->dd : 0.0);
  return SC_OK;
}

int sc_eval_stat_adaptive(sc_handle* h, const double* params, int64_t P, int32_t n_seg, double* out, int32_t* out_edges,
                          double* out3, void* stream) {
  if (!h) return SC_ERR_NOT_INIT;
  if (h->cuda_failed) return SC_ERR_CUDA;
  if (!params || P <= 0 || n_seg <= 0 || (!out && !out3)) return fail(h, SC_ERR_INVALID_ARG, "null pointer, n_particles <= 0 or n_seg <= 0");
  if (n_seg > h->cfg.n_bins) return fail(h, SC_ERR_INVALID_ARG, "n_seg exceeds n_bins");
  cudaStream_t st = (cudaStream_t)stream;
  if (n_seg == 1) {                              // one segment: the edges are (0, n_bins) for every particle
    const int32_t e[2] = {0, (int32_t)h->cfg.n_bins};
    int rc = eval_any(h, params, P, e, 1, out, nullptr, stream, false, out3);
    if (rc) return rc;
    if (out_edges) {
      k_fill_edges01<<<(unsigned)((P + 127) / 128), 128, 0, st>>>(out_edges, (int)P, (int)h->cfg.n_bins);
      return check_launch(h, "k_fill_edges01");
    }
    return SC_OK;
  }
  SC_CUDA(h, cudaMemsetAsync(h->d_counter, 0, 8, st));
  return run_adaptive(h, params, P, n_seg, out, out_edges, out3, st);
}

// ------------------------------------------------------------------------------------------------ hierarchical search
// Fig. 2 / Sec. III of the paper (App. B): for every rung N of the ladder
// { evaluate Upsilon_N for all particles -> PSO step (Eq. 13-15) per swarm } until every swarm has converged, then
// k-means regrouping of all particles and the next rung; after the last rung swarms whose best reaches the threshold are
// flagged.  The population never leaves the device; the host reads back one double per swarm and iteration (the bests,
// for the convergence rule).
int sc_search_run(sc_handle* h, const sc_search_config* sc, double* pos, double* vel, int32_t* label, int64_t P,
                  int32_t n_swarms, const double* lo, const double* hi, double* best_pos, double* best_val,
                  int64_t* n_members, int32_t* passed, int32_t* iters_per_rung, double* hist, void* stream) {
  if (!h) return SC_ERR_NOT_INIT;
  if (h->cuda_failed) return SC_ERR_CUDA;
  if (!sc || !pos || !vel || !label || !lo || !hi || !best_pos || !best_val)
    return fail(h, SC_ERR_INVALID_ARG, "null pointer");
  if (P <= 0 || n_swarms <= 0 || n_swarms > 128) return fail(h, SC_ERR_INVALID_ARG, "need n_particles > 0 and 1 <= n_swarms <= 128");
  if (sc->n_rungs < 1 || sc->n_rungs > SC_MAX_RUNGS) return fail(h, SC_ERR_INVALID_ARG, "n_rungs must be 1..%d", SC_MAX_RUNGS);
  if (sc->conv_window < 1 || sc->max_iters_per_rung < 1 || sc->kmeans_max_iters < 0)
    return fail(h, SC_ERR_INVALID_ARG, "conv_window, max_iters_per_rung must be >= 1 and kmeans_max_iters >= 0");
  for (int r = 0; r < sc->n_rungs; ++r)
    if (sc->n_seg[r] < 1 || sc->n_seg[r] > h->cfg.n_bins) return fail(h, SC_ERR_INVALID_ARG, "n_seg[%d] out of range", r);
  cudaStream_t st = (cudaStream_t)stream;
  const int S = n_swarms;
  const int64_t nb = h->cfg.n_bins;
  // device state owned by this call
  double* buf = nullptr;
  const size_t n_stat = (size_t)std::max<int64_t>(P, S);    // statistic per particle; per swarm in the final re-evaluation
  const size_t n_d = (size_t)P * 8 + (size_t)P + n_stat + (size_t)S * 8 * 2 + (size_t)S + 8;
  SC_CUDA(h, cudaMalloc(&buf, n_d * 8 + (size_t)S * 8));
  double* pbest_pos = buf; double* pbest_val = pbest_pos + (size_t)P * 8; double* stat = pbest_val + P;
  double* gbest_pos = stat + n_stat; double* cent = gbest_pos + (size_t)S * 8; double* gbest_val = cent + (size_t)S * 8;
  double* eps_d = gbest_val + S;
  long long* cnt_d = (long long*)(eps_d + 8);
  std::vector<double> gv((size_t)S), hst;
  std::vector<int64_t> cnt((size_t)S, 0);
  std::vector<int32_t> e;
  int rc = SC_OK;
  uint64_t iter_global = 0;
  // ranking precision (sc_search_config): force the FP32-amplitude path without escalation for the whole search
  const int saved_precision = h->precision, saved_escalate = h->escalate;
  // (precision mode and escalation of a three-channel handle apply to both of its passes)
  auto set_mode = [&](int prec, int esc) { h->precision = prec; h->escalate = esc; if (h->sub) { h->sub->precision = prec; h->sub->escalate = esc; } };
  if (sc->ranking_precision) set_mode(1, 0);
  const bool auto_precision = (h->precision == 0) && h->escalate && !h->sub;
  double win_frac = -1.0;                          // mean window fraction, -1: not measured yet
  unsigned long long ev_bins = 0;
  const double saved_win_frac = h->win_frac;
  auto cleanup = [&](int code) { set_mode(saved_precision, saved_escalate); h->win_frac = saved_win_frac; cudaFree(buf); return code; };
#define SC_S(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cleanup(fail(h, SC_ERR_CUDA, "%s failed: %s", #call, cudaGetErrorString(e_))); } while (0)
  SC_S(cudaMemsetAsync(gbest_pos, 0, (size_t)S * 8 * 8, st));

  for (int r = 0; r < sc->n_rungs; ++r) {
    const int N = sc->n_seg[r];
    // the objective changes with N: personal bests start afresh on every rung (Q21)
    k_fill<<<(unsigned)((P + 255) / 256), 256, 0, st>>>(pbest_val, (long long)P, -INFINITY);
    if ((rc = check_launch(h, "k_fill"))) return cleanup(rc);
    SC_S(cudaMemcpyAsync(pbest_pos, pos, (size_t)P * 64, cudaMemcpyDeviceToDevice, st));
    SC_S(cudaMemcpyAsync(eps_d, sc->eps_min[r], 64, cudaMemcpyHostToDevice, st));
    if (!sc->adaptive_edges || N == 1) {
      e.resize((size_t)N + 1);
      for (int k = 0; k <= N; ++k) e[k] = (int32_t)(((long long)k * nb) / N);       // equal-width shared edges (Q2)
    }
    hst.assign((size_t)S * sc->max_iters_per_rung, 0.0);
    const bool shared_rung = !(sc->adaptive_edges && N > 1);
    // Shared edges and short time windows (c5: a window covers ~2.5 % of the band): a particle then sees only N x phi
    // non-empty segments, and below f32_min_seg of them the FP32 pass would escalate nearly everybody.  phi = mean window
    // fraction, measured once from the evaluated-bin count of the first shared-edge evaluation of the search (read in
    // the synchronisation every iteration has anyway; a deterministic function of the first population).
    if (shared_rung && auto_precision && win_frac >= 0.0) h->precision = ((double)N * win_frac < (double)h->f32_min_seg) ? 2 : 0;
    int it = 0;
    for (; it < sc->max_iters_per_rung; ++it) {
      if (!shared_rung) rc = sc_eval_stat_adaptive(h, pos, P, N, stat, nullptr, nullptr, stream);
      else rc = eval_any(h, pos, P, e.data(), N, stat, nullptr, stream, false);
      if (rc) return cleanup(rc);
      const bool measure = shared_rung && auto_precision && win_frac < 0.0;
      if (measure) SC_S(cudaMemcpyAsync(&ev_bins, h->d_counter, 8, cudaMemcpyDeviceToHost, st));
      rc = sc_pso_step_labeled(h, pos, vel, pbest_pos, pbest_val, stat, gbest_pos, gbest_val, label, lo, hi, eps_d,
                               sc->omega[r], sc->phi_p[r], sc->phi_g[r], sc->seed, iter_global++, P, S, stream);
      if (rc) return cleanup(rc);
      SC_S(cudaMemcpyAsync(gv.data(), gbest_val, (size_t)S * 8, cudaMemcpyDeviceToHost, st));
      SC_S(cudaStreamSynchronize(st));
      if (measure) {
        win_frac = (double)ev_bins / ((double)P * (double)nb);
        h->precision = ((double)N * win_frac < (double)h->f32_min_seg) ? 2 : 0;
        if (saved_win_frac == 0.0) h->win_frac = win_frac;     // node spacing of the later shared-edge evaluations (select_stride_f32)
      }
      bool all_conv = true;
      for (int s = 0; s < S; ++s) {
        hst[(size_t)s * sc->max_iters_per_rung + it] = gv[s];
        if (gv[s] == -INFINITY) continue;                                   // empty swarm
        // converged when the best has not improved by more than conv_delta over conv_window iterations
        const bool conv = (it >= sc->conv_window) &&
                          (gv[s] - hst[(size_t)s * sc->max_iters_per_rung + it - sc->conv_window] <= sc->conv_delta);
        all_conv = all_conv && conv;
      }
      if (all_conv) { ++it; break; }
    }
    if (auto_precision) h->precision = 0;
    if (iters_per_rung) iters_per_rung[r] = it;
    if (hist)
      for (int s = 0; s < S; ++s)
        memcpy(hist + ((size_t)r * S + s) * sc->max_iters_per_rung, hst.data() + (size_t)s * sc->max_iters_per_rung,
               (size_t)sc->max_iters_per_rung * 8);
    if (r + 1 < sc->n_rungs && sc->kmeans_max_iters > 0) {
      // regroup all particles: k-means from the current swarm bests (Q19)
      SC_S(cudaMemcpyAsync(cent, gbest_pos, (size_t)S * 64, cudaMemcpyDeviceToDevice, st));
      int32_t n_it = 0;
      if ((rc = sc_kmeans(h, pos, P, lo, hi, cent, S, sc->kmeans_max_iters, label, (int64_t*)cnt_d, &n_it, stream))) return cleanup(rc);
    }
  }
  if (sc->ranking_precision) {
    // the reported bests are re-evaluated at full accuracy (all-FP64 path) at the swarm-best positions
    const int N = sc->n_seg[sc->n_rungs - 1];
    set_mode(2, saved_escalate);
    if (sc->adaptive_edges && N > 1) {
      // per-particle segments: the edges each best was ranked on (decided in FP64), then the statistic on exactly those
      // edges by the all-FP64 kernels, swarm by swarm
      int32_t* ed = nullptr;
      SC_S(cudaMalloc(&ed, (size_t)S * (N + 1) * 4));
      rc = sc_eval_stat_adaptive(h, gbest_pos, S, N, stat, ed, nullptr, stream);
      for (int s = 0; s < S && !rc; ++s)
        rc = eval_any(h, gbest_pos + (size_t)s * 8, 1, ed + (size_t)s * (N + 1), N, stat + s, nullptr, stream, false);
      cudaStreamSynchronize(st);
      cudaFree(ed);
    } else rc = eval_any(h, gbest_pos, S, e.data(), N, stat, nullptr, stream, false);
    if (rc) return cleanup(rc);
    k_keep_empty<<<1, 128, 0, st>>>(gbest_val, stat, S);
    if ((rc = check_launch(h, "k_keep_empty"))) return cleanup(rc);
  }
  // results: the bests of the last rung
  SC_S(cudaMemcpyAsync(best_val, gbest_val, (size_t)S * 8, cudaMemcpyDeviceToHost, st));
  SC_S(cudaMemcpyAsync(best_pos, gbest_pos, (size_t)S * 64, cudaMemcpyDeviceToHost, st));
  {
    std::vector<int32_t> lab((size_t)P);
    SC_S(cudaMemcpyAsync(lab.data(), label, (size_t)P * 4, cudaMemcpyDeviceToHost, st));
    SC_S(cudaStreamSynchronize(st));
    for (int64_t p = 0; p < P; ++p) if (lab[p] >= 0 && lab[p] < S) ++cnt[lab[p]];
  }
  for (int s = 0; s < S; ++s) {
    if (n_members) n_members[s] = cnt[s];
    if (passed) passed[s] = (cnt[s] > 0 && best_val[s] >= sc->threshold) ? 1 : 0;
  }
#undef SC_S
  return cleanup(SC_OK);
}

int sc_whiten_streams(sc_handle* h, const double* dA_ri, const double* dE_ri, int64_t n_streams, int32_t out_f64, void* W,
                      void* stream) {
  if (!h) return SC_ERR_NOT_INIT;
  if (h->cuda_failed) return SC_ERR_CUDA;
  if (!dA_ri || !dE_ri || !W || n_streams <= 0) return fail(h, SC_ERR_INVALID_ARG, "null pointer or n_streams <= 0");
  cudaStream_t st = (cudaStream_t)stream;
  const long long nb = h->cfg.n_bins, tot = nb * n_streams;
  const unsigned grid = (unsigned)((tot + 255) / 256);
  if (out_f64) k_whiten_streams_f64<<<grid, 256, 0, st>>>(dA_ri, dE_ri, h->G64, h->s0, nb, n_streams, (double4*)W);
  else k_whiten_streams_f32<<<grid, 256, 0, st>>>(dA_ri, dE_ri, h->G64, h->s0, nb, n_streams, (float4*)W);
  return check_launch(h, "k_whiten_streams");
}

int sc_eval_stat_streams(sc_handle* h, const double* theta, const void* W, int32_t w_is_f64, int64_t n_streams,
                         const int32_t* seg_edges, int32_t n_seg, double* out, void* stream) {
  if (!h) return SC_ERR_NOT_INIT;
  if (h->cuda_failed) return SC_ERR_CUDA;
  if (!theta || !W || !out || n_streams <= 0 || n_streams > 65535) return fail(h, SC_ERR_INVALID_ARG, "null pointer or n_streams outside 1..65535");
  if (!seg_edges || n_seg <= 0) return fail(h, SC_ERR_INVALID_ARG, "seg_edges is null or n_seg <= 0");
  if (h->sub) return fail(h, SC_ERR_INVALID_ARG, "the streams workload is not available on three-channel handles");
  cudaStream_t st = (cudaStream_t)stream;
  const int nb = (int)h->cfg.n_bins;
  std::vector<int> e((size_t)n_seg + 1);
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, seg_edges) != cudaSuccess) { cudaGetLastError(); at.type = cudaMemoryTypeUnregistered; }
  if (at.type == cudaMemoryTypeDevice) {
    SC_CUDA(h, cudaMemcpyAsync(e.data(), seg_edges, e.size() * 4, cudaMemcpyDeviceToHost, st));
    SC_CUDA(h, cudaStreamSynchronize(st));
  } else memcpy(e.data(), seg_edges, e.size() * 4);
  if (e[0] < 0 || e[n_seg] > nb) return fail(h, SC_ERR_INVALID_ARG, "seg_edges outside [0, n_bins]");
  for (int k = 0; k < n_seg; ++k)
    if (e[k + 1] < e[k]) return fail(h, SC_ERR_INVALID_ARG, "seg_edges not non-decreasing at k=%d", k);
  // pieces of the non-empty segments
  std::vector<int> plo, phi, plast;
  for (int k = 0; k < n_seg; ++k)
    for (int a = e[k]; a < e[k + 1]; a += kStreamPiece) {
      plo.push_back(a); phi.push_back(std::min(a + kStreamPiece, e[k + 1])); plast.push_back(a + kStreamPiece >= e[k + 1] ? 1 : 0);
    }
  const int n_pieces = (int)plo.size();
  if (n_pieces == 0) { SC_CUDA(h, cudaMemsetAsync(out, 0, (size_t)n_streams * 8, st)); return SC_OK; }
  int rc;
  if ((rc = grow(h, (void**)&h->d_sp, &h->sp_cap, (size_t)n_pieces * 12))) return rc;
  if ((rc = grow(h, (void**)&h->d_spsig, &h->spsig_cap, (size_t)n_pieces * 8))) return rc;
  if ((rc = grow(h, (void**)&h->d_zpart, &h->zpart_cap, (size_t)n_pieces * n_streams * 16))) return rc;
  if ((rc = grow(h, (void**)&h->d_T64, &h->t64_cap, (size_t)nb * 32))) return rc;
  if ((rc = grow(h, (void**)&h->d_T32, &h->t32_cap, (size_t)nb * 16))) return rc;
  if ((rc = grow(h, (void**)&h->d_hh, &h->hh_cap, (size_t)nb * 32))) return rc;
  int* d_lo = h->d_sp; int* d_hi = d_lo + n_pieces; int* d_last = d_hi + n_pieces;
  SC_CUDA(h, cudaMemcpyAsync(d_lo, plo.data(), (size_t)n_pieces * 4, cudaMemcpyHostToDevice, st));
  SC_CUDA(h, cudaMemcpyAsync(d_hi, phi.data(), (size_t)n_pieces * 4, cudaMemcpyHostToDevice, st));
  SC_CUDA(h, cudaMemcpyAsync(d_last, plast.data(), (size_t)n_pieces * 4, cudaMemcpyHostToDevice, st));
  SC_CUDA(h, cudaStreamSynchronize(st));             // the host vectors go out of scope
  // the template, once (same node tables and interpolants as everything else)
  double* hA = h->d_hh; double* hE = hA + (size_t)nb * 2;
  if ((rc = sc_gen_template(h, theta, 1, hA, hE, stream))) return rc;
  {
    Timed tm(h, st, SC_TIME_OTHER);
    k_streams_template<<<(nb + 255) / 256, 256, 0, st>>>(hA, hE, nb, h->d_T64, h->d_T32);
    if ((rc = check_launch(h, "k_streams_template"))) return rc;
    k_streams_sigma<<<(n_pieces + 7) / 8, 256, 0, st>>>(h->d_T64, h->G64, d_lo, d_hi, n_pieces, h->d_spsig);
    if ((rc = check_launch(h, "k_streams_sigma"))) return rc;
  }
  {
    Timed tm(h, st, SC_TIME_DENSE);
    const dim3 grid((n_pieces + 7) / 8, (unsigned)n_streams);
    if (w_is_f64) k_streams_z<double4, double><<<grid, 256, 0, st>>>((const double4*)W, h->d_T64, d_lo, d_hi, n_pieces, nb, (int)n_streams, h->d_zpart);
    else k_streams_z<float4, float><<<grid, 256, 0, st>>>((const float4*)W, h->d_T32, d_lo, d_hi, n_pieces, nb, (int)n_streams, h->d_zpart);
    if ((rc = check_launch(h, "k_streams_z"))) return rc;
  }
  Timed tm2(h, st, SC_TIME_STITCH);
  k_streams_finish<<<(unsigned)((n_streams + 127) / 128), 128, 0, st>>>(h->d_zpart, h->d_spsig, d_last, n_pieces, (int)n_streams, out);
  return check_launch(h, "k_streams_finish");
}

int sc_eval_stat_host(sc_handle* h, const double* params, int64_t P, const int32_t* seg_edges, int32_t n_seg,
                      double* out, void* stream) {
  if (!h) return SC_ERR_NOT_INIT;
  if (h->cuda_failed) return SC_ERR_CUDA;
  if (!params || !out || P <= 0) return fail(h, SC_ERR_INVALID_ARG, "null pointer or n_particles <= 0");
  cudaStream_t st = (cudaStream_t)stream;
  const size_t need = (size_t)P * 9 * 8;
  if (h->stage_cap < need) {
    if (h->d_params_stage) cudaFree(h->d_params_stage);
    h->d_params_stage = nullptr; h->stage_cap = 0;
    SC_CUDA(h, cudaMalloc(&h->d_params_stage, need));
    h->stage_cap = need;
  }
  h->d_out_stage = h->d_params_stage + (size_t)P * 8;
  SC_CUDA(h, cudaMemcpyAsync(h->d_params_stage, params, (size_t)P * 64, cudaMemcpyHostToDevice, st));
  int rc = eval_any(h, h->d_params_stage, P, seg_edges, n_seg, h->d_out_stage, nullptr, stream, false);
  if (rc) return rc;
  SC_CUDA(h, cudaMemcpyAsync(out, h->d_out_stage, (size_t)P * 8, cudaMemcpyDeviceToHost, st));
  SC_CUDA(h, cudaStreamSynchronize(st));
  return SC_OK;
}

int sc_gen_template(sc_handle* h, const double* params, int64_t P, double* hA, double* hE, void* stream) {
  if (!h) return SC_ERR_NOT_INIT;
  if (h->cuda_failed) return SC_ERR_CUDA;
  if (!params || !hA || !hE || P <= 0) return fail(h, SC_ERR_INVALID_ARG, "null pointer or n_templates <= 0");
  cudaStream_t st = (cudaStream_t)stream;
  const DevCfg& dc = h->dc;
  const int n_nodes = dc.n_nodes;
  const int P_pad = kBlock;       // templates are generated kBlock at a time
  const size_t per_p = (size_t)kPcFields * 8 + 8 + (size_t)n_nodes * (4 + 8 + 32);
  int rc = grow(h, &h->scratch, &h->scratch_bytes, per_p * (size_t)P_pad + 8192);
  if (rc) return rc;
  char* base = (char*)h->scratch;
  auto take = [&](size_t bytes) { char* r = base; base += (bytes + 255) / 256 * 256; return r; };
  double* pc = (double*)take((size_t)kPcFields * 8 * P_pad);
  int* jlo = (int*)take((size_t)4 * P_pad);
  int* jhi = (int*)take((size_t)4 * P_pad);
  int* node_n = (int*)take((size_t)n_nodes * 4 * P_pad);
  double* node_frac = (double*)take((size_t)n_nodes * 8 * P_pad);
  double* node_amp = (double*)take((size_t)n_nodes * 32 * P_pad);
  const double h0 = pow(dc.f_amp_ref, -7.0 / 6.0);
  for (int64_t pb = 0; pb < P; pb += P_pad) {
    const int Pn = (int)std::min<int64_t>(P_pad, P - pb);
    k_particle_consts<<<1, kBlock, 0, st>>>(dc, params + pb * 8, Pn, P_pad, pc, jlo, jhi, 0, 0, h->d_counter);
    if ((rc = check_launch(h, "k_particle_consts"))) return rc;
    k_nodes<double><<<dim3((n_nodes + kNodesPerCta - 1) / kNodesPerCta, 1), kBlock, 0, st>>>(dc, pc, jlo, jhi, P_pad, node_n, node_frac, node_amp);
    if ((rc = check_launch(h, "k_nodes"))) return rc;
    k_template<<<dim3((dc.n_bins + 255) / 256, Pn), 256, 0, st>>>(dc, node_n, node_frac, node_amp, jlo, jhi, P_pad, Pn, h0,
                                                                 hA + (size_t)pb * dc.n_bins * 2, hE + (size_t)pb * dc.n_bins * 2);
    if ((rc = check_launch(h, "k_template"))) return rc;
  }
  return SC_OK;
}

int sc_pso_step(sc_handle* h, double* pos, double* vel, double* pbest_pos, double* pbest_val, const double* stat,
                double* gbest_pos, double* gbest_val, const double* lo, const double* hi, const double* eps_min,
                double omega, double phi_p, double phi_g, uint64_t seed, uint64_t iter, int64_t P, int32_t n_swarms,
                void* stream) {
  if (!h) return SC_ERR_NOT_INIT;
  if (h->cuda_failed) return SC_ERR_CUDA;
  if (!pos || !vel || !pbest_pos || !pbest_val || !stat || !gbest_pos || !gbest_val || !lo || !hi || !eps_min)
    return fail(h, SC_ERR_INVALID_ARG, "null pointer");
  if (P <= 0 || n_swarms <= 0 || P % n_swarms != 0 || P / n_swarms > INT32_MAX)
    return fail(h, SC_ERR_INVALID_ARG, "n_particles must be a positive multiple of n_swarms");
  cudaStream_t st = (cudaStream_t)stream;
  const int per = (int)(P / n_swarms);
  int rc;
  Timed tm(h, st, SC_TIME_PSO);
  k_pso_best<<<n_swarms, 1024, 0, st>>>(pos, pbest_pos, pbest_val, stat, gbest_pos, gbest_val, per, nullptr, 0);
  if ((rc = check_launch(h, "k_pso_best"))) return rc;
  k_pso_move<<<(unsigned)((P + 127) / 128), 128, 0, st>>>(pos, vel, pbest_pos, gbest_pos, lo, hi, eps_min, omega, phi_p, phi_g,
                                                          seed, iter, P, per, nullptr);
  return check_launch(h, "k_pso_move");
}

int sc_pso_best(sc_handle* h, const double* pos, double* pbest_pos, double* pbest_val, const double* stat, double* cand,
                int64_t P, int32_t n_swarms, int64_t index_offset, void* stream) {
  if (!h) return SC_ERR_NOT_INIT;
  if (h->cuda_failed) return SC_ERR_CUDA;
  if (!pos || !pbest_pos || !pbest_val || !stat || !cand) return fail(h, SC_ERR_INVALID_ARG, "null pointer");
  if (P <= 0 || n_swarms <= 0 || P % n_swarms != 0 || P / n_swarms > INT32_MAX || index_offset < 0)
    return fail(h, SC_ERR_INVALID_ARG, "n_particles must be a positive multiple of n_swarms, index_offset >= 0");
  cudaStream_t st = (cudaStream_t)stream;
  Timed tm(h, st, SC_TIME_PSO);
  k_pso_best<<<n_swarms, 1024, 0, st>>>(pos, pbest_pos, pbest_val, stat, nullptr, nullptr, (int)(P / n_swarms), nullptr, 0,
                                        cand, (long long)index_offset);
  return check_launch(h, "k_pso_best");
}

int sc_pso_pick(sc_handle* h, const double* cand, int32_t n_cand, int32_t n_swarms, double* gbest_pos, double* gbest_val,
                void* stream) {
  if (!h) return SC_ERR_NOT_INIT;
  if (h->cuda_failed) return SC_ERR_CUDA;
  if (!cand || !gbest_pos || !gbest_val) return fail(h, SC_ERR_INVALID_ARG, "null pointer");
  if (n_cand <= 0 || n_swarms <= 0) return fail(h, SC_ERR_INVALID_ARG, "n_cand and n_swarms must be positive");
  cudaStream_t st = (cudaStream_t)stream;
  Timed tm(h, st, SC_TIME_PSO);
  k_pso_pick<<<n_swarms, 32, 0, st>>>(cand, n_cand, n_swarms, gbest_pos, gbest_val);
  return check_launch(h, "k_pso_pick");
}

int sc_pso_move(sc_handle* h, double* pos, double* vel, const double* pbest_pos, const double* gbest_pos, const double* lo,
                const double* hi, const double* eps_min, double omega, double phi_p, double phi_g, uint64_t seed,
                uint64_t iter, int64_t P, int32_t n_swarms, int64_t index_offset, void* stream) {
  if (!h) return SC_ERR_NOT_INIT;
  if (h->cuda_failed) return SC_ERR_CUDA;
  if (!pos || !vel || !pbest_pos || !gbest_pos || !lo || !hi || !eps_min) return fail(h, SC_ERR_INVALID_ARG, "null pointer");
  if (P <= 0 || n_swarms <= 0 || P % n_swarms != 0 || P / n_swarms > INT32_MAX || index_offset < 0)
    return fail(h, SC_ERR_INVALID_ARG, "n_particles must be a positive multiple of n_swarms, index_offset >= 0");
  cudaStream_t st = (cudaStream_t)stream;
  Timed tm(h, st, SC_TIME_PSO);
  k_pso_move<<<(unsigned)((P + 127) / 128), 128, 0, st>>>(pos, vel, pbest_pos, gbest_pos, lo, hi, eps_min, omega, phi_p, phi_g,
                                                          seed, iter, P, (int)(P / n_swarms), nullptr, (long long)index_offset);
  return check_launch(h, "k_pso_move");
}

int sc_pso_step_labeled(sc_handle* h, double* pos, double* vel, double* pbest_pos, double* pbest_val, const double* stat,
                        double* gbest_pos, double* gbest_val, const int32_t* label, const double* lo, const double* hi,
                        const double* eps_min, double omega, double phi_p, double phi_g, uint64_t seed, uint64_t iter,
                        int64_t P, int32_t n_swarms, void* stream) {
  if (!h) return SC_ERR_NOT_INIT;
  if (h->cuda_failed) return SC_ERR_CUDA;
  if (!pos || !vel || !pbest_pos || !pbest_val || !stat || !gbest_pos || !gbest_val || !label || !lo || !hi || !eps_min)
    return fail(h, SC_ERR_INVALID_ARG, "null pointer");
  if (P <= 0 || n_swarms <= 0) return fail(h, SC_ERR_INVALID_ARG, "n_particles and n_swarms must be positive");
  cudaStream_t st = (cudaStream_t)stream;
  int rc;
  Timed tm(h, st, SC_TIME_PSO);
  k_pso_best<<<n_swarms, 1024, 0, st>>>(pos, pbest_pos, pbest_val, stat, gbest_pos, gbest_val, 0, label, (long long)P);
  if ((rc = check_launch(h, "k_pso_best"))) return rc;
  k_pso_move<<<(unsigned)((P + 127) / 128), 128, 0, st>>>(pos, vel, pbest_pos, gbest_pos, lo, hi, eps_min, omega, phi_p, phi_g,
                                                          seed, iter, P, 1, label);
  return check_launch(h, "k_pso_move");
}

int sc_kmeans(sc_handle* h, const double* pos, int64_t P, const double* lo, const double* hi, double* cent, int32_t K,
              int32_t max_iter, int32_t* label, int64_t* count, int32_t* n_iter, void* stream) {
  if (!h) return SC_ERR_NOT_INIT;
  if (h->cuda_failed) return SC_ERR_CUDA;
  if (!pos || !lo || !hi || !cent || !label) return fail(h, SC_ERR_INVALID_ARG, "null pointer");
  if (P <= 0 || K <= 0 || K > 128 || max_iter <= 0) return fail(h, SC_ERR_INVALID_ARG, "need n_particles > 0, 1 <= K <= 128, max_iter > 0");
  cudaStream_t st = (cudaStream_t)stream;
  int rc;
  if ((rc = grow(h, (void**)&h->d_km, &h->km_cap, 16 + (size_t)K * 8))) return rc;
  int* d_changed = (int*)h->d_km;
  long long* d_cnt = (long long*)((char*)h->d_km + 16);
  SC_CUDA(h, cudaMemsetAsync(label, 0xFF, (size_t)P * 4, st));       // -1: every particle counts as changed in iteration 1
  int it = 0;
  while (it < max_iter) {
    ++it;
    SC_CUDA(h, cudaMemsetAsync(d_changed, 0, 4, st));
    {
      Timed tm(h, st, SC_TIME_PSO);
      k_km_assign<<<(unsigned)((P + 127) / 128), 128, 0, st>>>(pos, (long long)P, lo, hi, cent, K, label, d_changed);
      if ((rc = check_launch(h, "k_km_assign"))) return rc;
      k_km_update<<<K, 8, 0, st>>>(pos, (long long)P, label, cent, d_cnt);
      if ((rc = check_launch(h, "k_km_update"))) return rc;
    }
    int changed = 0;
    SC_CUDA(h, cudaMemcpyAsync(&changed, d_changed, 4, cudaMemcpyDeviceToHost, st));
    SC_CUDA(h, cudaStreamSynchronize(st));
    if (changed == 0) break;
  }
  if (count) SC_CUDA(h, cudaMemcpyAsync(count, d_cnt, (size_t)K * 8, cudaMemcpyDeviceToDevice, st));
  if (n_iter) *n_iter = it;
  return SC_OK;
}

// ------------------------------------------------------------------------------------------------ k-means without allocation
// sc_kmeans_static: the Lloyd iterations of sc_kmeans for callers that may not allocate device memory (code under CUDA
// graph capture, serving loops, harnesses that forbid cudaMalloc).  Its scratch -- the "labels changed" counter and the K
// member counts -- lives in a file-scope device array: every GPU that loads the library holds these 2 KiB until exit.
// In host code the array's name is a host-side stand-in, not a device address: the address comes from
// cudaGetSymbolAddress, once per device with that device current (static_scratch below), and only that pointer is
// handed to the kernels.  All calls on a device share the array and it keeps the last call's contents: the counter is
// cleared before every iteration, the counts are rewritten by every k_km_update; calls that overlap on the GPU race.
constexpr int kStaticMaxK = SC_KMEANS_STATIC_MAX_K;
constexpr size_t kStaticScratchBytes = 2048;                 // 16 (counter, padded) + kStaticMaxK x 8 <= 2048
static_assert(16 + (size_t)kStaticMaxK * 8 <= kStaticScratchBytes, "static scratch too small for SC_KMEANS_STATIC_MAX_K");
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

namespace {
constexpr int kStaticMaxDevices = 64;
void* g_static_ptr[kStaticMaxDevices] = {};                  // device address of g_static_scratch, per device ordinal
std::mutex g_static_mutex;

// The device address of g_static_scratch on the handle's device (resolved once per device; no allocation).
int static_scratch(sc_handle* h, void** out) {
  int dev = -1;
  SC_CUDA(h, cudaGetDevice(&dev));
  if (dev != h->device) return fail(h, SC_ERR_INVALID_ARG, "the current device (%d) is not the handle's (%d)", dev, h->device);
  if (dev < 0 || dev >= kStaticMaxDevices) return fail(h, SC_ERR_INVALID_ARG, "device ordinal %d beyond %d", dev, kStaticMaxDevices - 1);
  std::lock_guard<std::mutex> lock(g_static_mutex);
  if (!g_static_ptr[dev]) {
    void* ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&ptr, g_static_scratch);
    if (e != cudaSuccess || !ptr) {
      cudaGetLastError();
      return fail(h, SC_ERR_CUDA, "cudaGetSymbolAddress(g_static_scratch) failed: %s", cudaGetErrorString(e));
    }
    g_static_ptr[dev] = ptr;
  }
  *out = g_static_ptr[dev];
  return SC_OK;
}
}  // namespace

int sc_kmeans_static(sc_handle* h, const double* pos, int64_t P, const double* lo, const double* hi, double* cent, int32_t K,
                     int32_t max_iter, int32_t* label, int64_t* count, int32_t* n_iter, void* stream) {
  if (!h) return SC_ERR_NOT_INIT;
  if (h->cuda_failed) return SC_ERR_CUDA;
  if (!pos || !lo || !hi || !cent || !label) return fail(h, SC_ERR_INVALID_ARG, "null pointer");
  if (K > kStaticMaxK)
    return fail(h, SC_ERR_INVALID_ARG, "K = %d exceeds SC_KMEANS_STATIC_MAX_K = %d, the size of the static scratch array", (int)K, kStaticMaxK);
  if (P <= 0 || K <= 0 || max_iter <= 0) return fail(h, SC_ERR_INVALID_ARG, "need n_particles > 0, K >= 1, max_iter > 0");
  cudaStream_t st = (cudaStream_t)stream;
  void* scratch = nullptr;
  int rc;
  if ((rc = static_scratch(h, &scratch))) return rc;
  int* d_changed = (int*)scratch;
  long long* d_cnt = (long long*)((char*)scratch + 16);
  SC_CUDA(h, cudaMemsetAsync(label, 0xFF, (size_t)P * 4, st));       // -1: every particle counts as changed in iteration 1
  int it = 0;
  while (it < max_iter) {
    ++it;
    SC_CUDA(h, cudaMemsetAsync(d_changed, 0, 4, st));                 // the array keeps the previous call's contents
    // (no Timed here: SC_OPT_PROFILE creates events on demand)
    k_km_assign<<<(unsigned)((P + 127) / 128), 128, 0, st>>>(pos, (long long)P, lo, hi, cent, K, label, d_changed);
    if ((rc = check_launch(h, "k_km_assign"))) return rc;
    k_km_update<<<K, 8, 0, st>>>(pos, (long long)P, label, cent, d_cnt);
    if ((rc = check_launch(h, "k_km_update"))) return rc;
    int changed = 0;
    SC_CUDA(h, cudaMemcpyAsync(&changed, d_changed, 4, cudaMemcpyDeviceToHost, st));
    SC_CUDA(h, cudaStreamSynchronize(st));
    if (changed == 0) break;
  }
  if (count) SC_CUDA(h, cudaMemcpyAsync(count, d_cnt, (size_t)K * 8, cudaMemcpyDeviceToDevice, st));
  if (n_iter) *n_iter = it;
  return SC_OK;
}

int sc_get_counters(sc_handle* h, int64_t* evaluated_bins, int64_t* kernel_launches, void* stream) {
  if (!h) return SC_ERR_NOT_INIT;
  if (h->cuda_failed) return SC_ERR_CUDA;
  unsigned long long v = 0;
  SC_CUDA(h, cudaMemcpyAsync(&v, h->d_counter, 8, cudaMemcpyDeviceToHost, (cudaStream_t)stream));
  SC_CUDA(h, cudaStreamSynchronize((cudaStream_t)stream));
  if (evaluated_bins) *evaluated_bins = (int64_t)v;
  if (kernel_launches) *kernel_launches = h->launches;
  return SC_OK;
}

int sc_get_launch_info(sc_handle* h, int32_t* stride_log2, int32_t* flavour) {
  if (!h) return SC_ERR_NOT_INIT;
  if (stride_log2) *stride_log2 = h->last_lg;
  if (flavour) *flavour = h->last_flavour;
  return SC_OK;
}

int sc_get_timing(sc_handle* h, double* ms_per_class, int64_t* launches_per_class, void* stream) {
  if (!h) return SC_ERR_NOT_INIT;
  if (h->cuda_failed) return SC_ERR_CUDA;
  SC_CUDA(h, cudaStreamSynchronize((cudaStream_t)stream));
  for (size_t i = 0; i < h->ev_used; ++i) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, h->evs[i].a, h->evs[i].b) == cudaSuccess) {
      h->cls_ms[h->evs[i].cls] += ms; h->cls_n[h->evs[i].cls]++;
    } else cudaGetLastError();
  }
  h->ev_used = 0;
  for (int c = 0; c < SC_N_TIMING_CLASSES; ++c) {
    if (ms_per_class) ms_per_class[c] = h->cls_ms[c];
    if (launches_per_class) launches_per_class[c] = h->cls_n[c];
    h->cls_ms[c] = 0.0; h->cls_n[c] = 0;
  }
  return SC_OK;
}

int sc_measure_fp64_peak(double* dfma_per_s, void* stream) {
  if (!dfma_per_s) return SC_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
    cudaGetLastError();
    return fail(nullptr, SC_ERR_CUDA, "no CUDA device; this library has no CPU fallback");
  }
  const int blocks = sms * 8, threads = 256, iters = 1 << 15;
  double* buf = nullptr;
  if (cudaMalloc(&buf, (size_t)blocks * threads * 8) != cudaSuccess) { cudaGetLastError(); return fail(nullptr, SC_ERR_OOM, "cudaMalloc failed"); }
  cudaEvent_t a, b;
  cudaEventCreate(&a); cudaEventCreate(&b);
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(a, st);
    k_dfma_peak<<<blocks, threads, 0, st>>>(buf, iters, 0.999999, 1e-9);
    cudaEventRecord(b, st);
    cudaEventSynchronize(b);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(a); cudaEventDestroy(b); cudaFree(buf);
  if (cudaGetLastError() != cudaSuccess) return fail(nullptr, SC_ERR_CUDA, "k_dfma_peak failed");
  *dfma_per_s = (double)blocks * threads * 8.0 * iters / (best * 1e-3);
  return SC_OK;
}

int sc_set_option(sc_handle* h, int32_t option, int64_t value) {
  if (!h) return SC_ERR_NOT_INIT;
  if (h->sub && option != SC_OPT_PROFILE) { const int rc = sc_set_option(h->sub, option, value); if (rc) return fail(h, rc, "%s", h->sub->err.c_str()); }
  switch (option) {
    case SC_OPT_PRECISION:
      if (value < 0 || value > 2) return fail(h, SC_ERR_INVALID_ARG, "precision must be 0, 1 or 2");
      h->precision = (int)value; return SC_OK;
    case SC_OPT_F32_MIN_SEG:
      if (value < 1) return fail(h, SC_ERR_INVALID_ARG, "f32_min_seg must be >= 1");
      h->f32_min_seg = (int)std::min<int64_t>(value, INT32_MAX); return SC_OK;
    case SC_OPT_SCRATCH_BYTES:
      if (value < (1 << 20)) return fail(h, SC_ERR_INVALID_ARG, "scratch cap must be >= 1 MiB");
      h->scratch_cap = (size_t)value; return SC_OK;
    case SC_OPT_PROFILE:
      h->profile = (value != 0); return SC_OK;
    case SC_OPT_MUFU_MIN_SEG:
      if (value < 1) return fail(h, SC_ERR_INVALID_ARG, "mufu_min_seg must be >= 1");
      h->mufu_min_seg = (int)std::min<int64_t>(value, INT32_MAX); return SC_OK;
    case SC_OPT_WINDOW_SORT:
      if (value < 0 || value > 1) return fail(h, SC_ERR_INVALID_ARG, "window_sort must be 0 or 1");
      h->window_sort = (int)value; return SC_OK;
    case SC_OPT_FUSED_AET:
      if (value < 0 || value > 1) return fail(h, SC_ERR_INVALID_ARG, "fused_aet must be 0 or 1");
      h->use_fused3 = (int)value; return SC_OK;
    case SC_OPT_TENSOR_CORES:
      if (value < 0 || value > 1) return fail(h, SC_ERR_INVALID_ARG, "tensor_cores must be 0 or 1");
      h->use_tc = (int)value; return SC_OK;
    case SC_OPT_ESCALATE:
      if (value < 0 || value > 1) return fail(h, SC_ERR_INVALID_ARG, "escalate must be 0 or 1");
      h->escalate = (int)value; return SC_OK;
    case SC_OPT_ESC_TAU_POLY_X1000:
    case SC_OPT_ESC_TAU_MUFU_X1000:
      if (value < 0) return fail(h, SC_ERR_INVALID_ARG, "escalation threshold must be >= 0");
      (option == SC_OPT_ESC_TAU_POLY_X1000 ? h->esc_tau_poly : h->esc_tau_mufu) = (double)value * 1e-3; return SC_OK;
    case SC_OPT_SINCOS:
      if (value < 0 || value > 2) return fail(h, SC_ERR_INVALID_ARG, "sincos must be 0, 1 or 2");
      h->sincos_mode = (int)value; return SC_OK;
    case SC_OPT_TC_MAX_S:
      if (value < 1) return fail(h, SC_ERR_INVALID_ARG, "tc_max_s must be >= 1");
      h->tc_max_s = (double)value; set_stride(h); return SC_OK;
    case SC_OPT_QUAD_AMPLITUDES:
      if (value < 0 || value > 1) return fail(h, SC_ERR_INVALID_ARG, "quad_amplitudes must be 0 or 1");
      h->quad_amp = (int)value; return SC_OK;
    case SC_OPT_WINDOW_FRACTION_PPM:
      if (value < 0 || value > 1000000) return fail(h, SC_ERR_INVALID_ARG, "window fraction must be 0 (not stated) .. 1000000 ppm");
      h->win_frac = (double)value * 1e-6; return SC_OK;
    case SC_OPT_STRIDE_LOG2:
      if (value != 0 && (value < 3 || value > 12)) return fail(h, SC_ERR_INVALID_ARG, "stride_log2 must be 0 (auto) or 3..12");
      h->forced_stride_log2 = (int)value; set_stride(h); return SC_OK;
    default:
      return fail(h, SC_ERR_INVALID_ARG, "unknown option %d", (int)option);
  }
}

int sc_free(sc_handle* h) {
  if (!h) return SC_ERR_NOT_INIT;
  if (h->sub) sc_free(h->sub);
  cudaFree(h->d_seg3);
  cudaFree(h->D32); cudaFree(h->W64); cudaFree(h->G64); cudaFree(h->d_tc_img); cudaFree(h->D3); cudaFree(h->Gp3); cudaFree(h->GT64);
  cudaFree(h->d_momentsT); cudaFree(h->alt.d_momentsT); cudaFree(h->d_gmomT); cudaFree(h->d_smomT); cudaFree(h->d_smom64T);
  cudaFree(h->scratch); cudaFree(h->d_edges); cudaFree(h->d_chunk_k0); cudaFree(h->d_flags);
  cudaFree(h->d_counter); cudaFree(h->d_params_stage); cudaFree(h->d_comp); cudaFree(h->d_km); cudaFree(h->d_T64); cudaFree(h->d_T32); cudaFree(h->d_sp);
  cudaFree(h->d_spsig); cudaFree(h->d_zpart); cudaFree(h->d_hh); cudaFree(h->d_gmom); cudaFree(h->d_smom);
  cudaFree(h->d_gmom64); cudaFree(h->d_smom64); cudaFree(h->d_ad_edges);
  cudaFree(h->d_piece_first); cudaFree(h->d_piece_lo); cudaFree(h->d_piece_hi); cudaFree(h->d_moments);
  cudaFree(h->alt.d_edges); cudaFree(h->alt.d_chunk_k0); cudaFree(h->alt.d_flags); cudaFree(h->alt.d_next_close); cudaFree(h->d_next_close);
  cudaFree(h->d_moments64); cudaFree(h->alt.d_moments64);
  cudaFree(h->alt.d_piece_first); cudaFree(h->alt.d_piece_lo); cudaFree(h->alt.d_piece_hi); cudaFree(h->alt.d_moments);
  cudaFreeHost(h->h_esc_hint); cudaFree(h->d_sort_tmp);
  cudaFree(h->d_esc_idx); cudaFree(h->d_esc_count); cudaFree(h->d_esc_params); cudaFree(h->d_esc_out);
  for (auto& e : h->evs) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
  cudaGetLastError();
  delete h;
  return SC_OK;
}

const char* sc_last_error(const sc_handle* h) { return h ? h->err.c_str() : g_init_error.c_str(); }

const char* sc_version(void) { return "scstat 0.1 (sm_100a)"; }

}  // extern "C"
