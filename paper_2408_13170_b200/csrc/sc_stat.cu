// sc_stat.cu -- kernels and C ABI of libscstat.so (sm_100a).  See include/sc_stat.h for the contract and
// DESIGN.md for the design.  No CPU fallback, no torch, no third-party code.
//
// Pipeline of one sc_eval_stat call, per batch of particles:
//   k_particle_consts  a1 + a3  per-particle constants, validity, time window [jlo, jhi) by bisection on t(f_j)
//   k_nodes            a2       phase / amplitude at the coarse nodes (one node per `stride` bins)
//   k_dense<R, SEG>    a4 + a5  THE HOT LOOP: lane = particle, warp walks the bins of its chunk in order;
//                               whitened data broadcast from shared memory; FP64 phase by forward differences;
//                               complete segments are finalised in registers, straddlers leave fragments
//   k_stitch           a6       fixed-order stitch of the fragments -> Upsilon[p]
#include "../../include/sc_stat.h"
#include "sc_math.cuh"

#include <cub/device/device_radix_sort.cuh>

#include <algorithm>
#include <climits>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <string>
#include <type_traits>
#include <vector>

using namespace sc;

namespace {

constexpr int kBlock = 128;            // threads per CTA of the dense kernel = particles per CTA
constexpr int kChunkF32 = 2048;        // bins per CTA, FP32 amplitude path (24 B/bin of shared memory)
constexpr int kChunkF64 = 1024;        // bins per CTA, all-FP64 path (48 B/bin)
constexpr int kFlushBins = 32;         // FP32 partial sums are folded into the FP64 accumulators this often
constexpr int kFragFields = 9;         // partial Upsilon, head (zr, zi, sg), tail (zr, zi, sg), partial sum|z|, partial sum sigma
constexpr double kMagic = 6755399441055744.0;   // 1.5 * 2^52: (x + kMagic) - kMagic = rint(x), low word = int

// chunk flags (host-built from the edges, shared by all particles)
enum : uint8_t { CF_HEAD = 1, CF_HEAD_CLOSES = 2, CF_TAIL = 4 };

// ------------------------------------------------------------------------------------------------ whitening (a0)
__global__ void k_max_weight(const double* __restrict__ S_A, const double* __restrict__ S_E, int n, double four_df,
                             unsigned long long* __restrict__ out_max_bits) {
  double m = 0.0;
  for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < n; j += gridDim.x * blockDim.x) {
    const double a = S_A[j], e = S_E[j];
    if (isfinite(a) && a > 0.0) m = fmax(m, four_df / a);
    if (isfinite(e) && e > 0.0) m = fmax(m, four_df / e);
  }
  for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0 && isfinite(m)) atomicMax(out_max_bits, (unsigned long long)__double_as_longlong(m));
}

// W_a = d_a * (4 df / S_a) / s0,  G_a = (4 df / S_a) / s0^2  with s0 a power of two (exact rescaling).
// FP64 copies per bin (all-FP64 path) and the FP32 copy in the bin-pair layout of k_dense2: for pair m = bins
// (2m, 2m+1) three 16-byte records (wAr, wAi), (wEr, wEi), (gA, gE), each field as (even bin, odd bin); bins past
// n_bins (padding up to a whole chunk) are zero.
__device__ __forceinline__ void whiten_bin(const double* __restrict__ dA, const double* __restrict__ dE,
                                           const double* __restrict__ S_A, const double* __restrict__ S_E, int j, int n,
                                           double four_df, double inv_s0, double4& w, double2& g) {
  w = make_double4(0.0, 0.0, 0.0, 0.0); g = make_double2(0.0, 0.0);
  if (j >= n) return;
  const double a = S_A[j], e = S_E[j];
  const double ua = (isfinite(a) && a > 0.0) ? four_df / a : 0.0;
  const double ue = (isfinite(e) && e > 0.0) ? four_df / e : 0.0;
  w.x = dA[2 * j] * ua * inv_s0; w.y = dA[2 * j + 1] * ua * inv_s0;
  w.z = dE[2 * j] * ue * inv_s0; w.w = dE[2 * j + 1] * ue * inv_s0;
  if (!(isfinite(w.x) && isfinite(w.y))) { w.x = 0.0; w.y = 0.0; }
  if (!(isfinite(w.z) && isfinite(w.w))) { w.z = 0.0; w.w = 0.0; }
  g.x = ua * inv_s0 * inv_s0; g.y = ue * inv_s0 * inv_s0;
}
__global__ void k_whiten(const double* __restrict__ dA, const double* __restrict__ dE,
                         const double* __restrict__ S_A, const double* __restrict__ S_E, int n, int n_pairs_pad,
                         double four_df, double inv_s0, float4* __restrict__ D32,
                         double4* __restrict__ W64, double2* __restrict__ G64) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= n_pairs_pad) return;
  double4 w0, w1; double2 g0, g1;
  whiten_bin(dA, dE, S_A, S_E, 2 * m, n, four_df, inv_s0, w0, g0);
  whiten_bin(dA, dE, S_A, S_E, 2 * m + 1, n, four_df, inv_s0, w1, g1);
  if (2 * m < n) { W64[2 * m] = w0; G64[2 * m] = g0; }
  if (2 * m + 1 < n) { W64[2 * m + 1] = w1; G64[2 * m + 1] = g1; }
  D32[3 * (size_t)m + 0] = make_float4((float)w0.x, (float)w1.x, (float)w0.y, (float)w1.y);
  D32[3 * (size_t)m + 1] = make_float4((float)w0.z, (float)w1.z, (float)w0.w, (float)w1.w);
  D32[3 * (size_t)m + 2] = make_float4((float)g0.x, (float)g1.x, (float)g0.y, (float)g1.y);
}

// <d|d> = 4 df sum_a sum_j |d_a|^2 / S_a = sum |W|^2 / G over the bins with non-zero weight (Eq. 1 with a = b = d;
// the constant of Eq. 9).  Fixed grid and a fixed-order tree: deterministic.  part: [gridDim.x] partial sums.
__global__ void k_data_norm(const double4* __restrict__ W64, const double2* __restrict__ G64, int n, double* __restrict__ part) {
  __shared__ double sh[256];
  double acc = 0.0;
  for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < n; j += gridDim.x * blockDim.x) {
    const double4 w = W64[j]; const double2 g = G64[j];
    if (g.x > 0.0) acc += (w.x * w.x + w.y * w.y) / g.x;
    if (g.y > 0.0) acc += (w.z * w.z + w.w * w.w) / g.y;
  }
  sh[threadIdx.x] = acc;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) part[blockIdx.x] = sh[0];
}

// Eq. 9: log L_hat_N = -1/2 <d|d> - 1/2 A^2 <h|h> + A O_hat_N for a template of amplitude A times the
// unit-amplitude template the components refer to.
__global__ void k_loglike(const double* __restrict__ comp3, const double* __restrict__ amp, double dd, int P,
                          double* __restrict__ out) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P) return;
  const double A = amp[p];
  out[p] = -0.5 * dd - 0.5 * A * A * comp3[3 * (size_t)p + 2] + A * comp3[3 * (size_t)p + 1];
}

__global__ void k_fill(double* __restrict__ x, long long n, double v) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) x[i] = v;
}

// ------------------------------------------------------------------------------------------------ a1 + a3
__global__ void k_particle_consts(DevCfg c, const double* __restrict__ params, int P, int P_pad,
                                  double* __restrict__ pc, int* __restrict__ jlo_out, int* __restrict__ jhi_out,
                                  int e_first, int e_last, unsigned long long* __restrict__ eval_bins,
                                  const int* __restrict__ esc_count = nullptr, int esc_pb = 0) {
  // escalation pass: the number of particles is known on the device only; the launched blocks stride over the
  // 128-particle blocks below it (the grid is sized from a host-side hint, correctness does not depend on it)
  if (esc_count) P = min(P, *esc_count - esc_pb);
  for (int pblk = blockIdx.x; ; pblk += gridDim.x) {
  if (esc_count && pblk * (int)blockDim.x >= P) return;
  const int p = pblk * blockDim.x + threadIdx.x;
  if (p >= P_pad) return;
  int jlo = 0, jhi = 0;
  Particle q = {};
  if (p < P) {
    double th[8];
    bool ok = true;
#pragma unroll
    for (int i = 0; i < 8; ++i) { th[i] = params[(size_t)p * 8 + i]; ok = ok && isfinite(th[i]); }
    ok = ok && (th[0] > 0.0) && (th[1] > 0.0) && (th[1] <= 0.25);
    if (ok) {
      const double M = th[0] * kMsunSec * pow(th[1], -0.6);
      q.piM = kPi * M; q.eta = th[1]; q.tc = th[2];
      q.tau_hi = th[2] * c.inv_T;
      q.tau_lo = fma(-q.tau_hi, c.T_obs, th[2]) * c.inv_T;
      sincos(th[3], &q.sl, &q.cl);
      sincos(th[4], &q.sb, &q.cb);
      sincos(2.0 * th[6], &q.s2p, &q.c2p);
      q.ci = cos(th[5]);
      q.ecc = 0.0;
      if (c.ecc_leading) q.ecc = (2355.0 / 1462.0) * th[7] * th[7] * pow(cbrt(q.piM * c.f_ref_ecc), 19.0 / 3.0);
      if (c.window_mode == 1) {
        // Q4: the template lives where 0 <= t(f_j) <= T_obs; t(f) is monotone, so bisect on the bin index
        // with t(f_j) evaluated directly at the bin frequencies (same expression the definition uses).
        int lo = 0, hi = c.n_bins;       // first j with t(f_j) >= 0
        while (lo < hi) {
          const int mid = (lo + hi) >> 1;
          if (tf_direct(c, q, (double)(c.j0 + mid) / c.T_obs) >= 0.0) hi = mid; else lo = mid + 1;
        }
        jlo = lo;
        lo = jlo; hi = c.n_bins;          // first j with t(f_j) > T_obs
        while (lo < hi) {
          const int mid = (lo + hi) >> 1;
          if (tf_direct(c, q, (double)(c.j0 + mid) / c.T_obs) > c.T_obs) hi = mid; else lo = mid + 1;
        }
        jhi = lo;
      } else {
        jlo = 0; jhi = c.n_bins;
      }
    }
    const int a = max(jlo, e_first), b = min(jhi, e_last);
    if (b > a && eval_bins) atomicAdd(eval_bins, (unsigned long long)(b - a));
  }
  pc[PC_PIM * (size_t)P_pad + p] = q.piM;       pc[PC_ETA * (size_t)P_pad + p] = q.eta;
  pc[PC_TC * (size_t)P_pad + p] = q.tc;         pc[PC_TAU_HI * (size_t)P_pad + p] = q.tau_hi;
  pc[PC_TAU_LO * (size_t)P_pad + p] = q.tau_lo; pc[PC_CL * (size_t)P_pad + p] = q.cl;
  pc[PC_SL * (size_t)P_pad + p] = q.sl;         pc[PC_CB * (size_t)P_pad + p] = q.cb;
  pc[PC_SB * (size_t)P_pad + p] = q.sb;         pc[PC_C2P * (size_t)P_pad + p] = q.c2p;
  pc[PC_S2P * (size_t)P_pad + p] = q.s2p;       pc[PC_CI * (size_t)P_pad + p] = q.ci;
  pc[PC_ECC * (size_t)P_pad + p] = q.ecc;
  jlo_out[p] = jlo; jhi_out[p] = jhi;
  if (!esc_count) return;
  }
}

// ------------------------------------------------------------------------------------------------ a2
// One thread per (node, particle), particle fastest -> coalesced [node][particle] tables; a CTA takes 128 particles and
// a group of kNodesPerCta consecutive nodes (one CTA per node is launch-bound when most of the table is out of reach).
constexpr int kNodesPerCta = 16;
template <typename R, bool ESC = false>
__global__ void k_nodes(DevCfg c, const double* __restrict__ pc, const int* __restrict__ jlo, const int* __restrict__ jhi,
                        int P_pad, int* __restrict__ node_n, double* __restrict__ node_frac,
                        R* __restrict__ node_amp /* [node][4][P_pad] */, const int* __restrict__ esc_count = nullptr,
                        int esc_pb = 0, int skip_unreached = 0) {
  const int i_first = blockIdx.x * kNodesPerCta;            // nodes i_first .. i_last-1  <->  node index i - kNodeOff
  const int i_last = min(i_first + kNodesPerCta, c.n_nodes);
  const int esc_lim = ESC ? min(*esc_count - esc_pb, P_pad) : 0;
  for (int pblk = blockIdx.y; ; pblk += gridDim.y) {   // one pass, except in the escalation pass (see k_particle_consts)
    if (ESC && pblk * (int)blockDim.x >= esc_lim) return;
    const int p = pblk * blockDim.x + threadIdx.x;
    if (p >= P_pad) return;
    const int lo = jlo[p], hi = jhi[p];
    // nodes farther than the stencils reach from the particle's window are never read
    const long long reach = 4LL << c.log2_stride;
    const long long r_lo = (long long)lo - reach, r_hi = (long long)hi + reach;
    // skip_unreached (k_dense / k_dense2 as consumers): a warp reads a node only where one of its particles' windows is
    // within reach of it, and then for all its lanes -- so a block none of whose particles reaches the node need not write
    // it at all (with the batch sorted by window start that is most of the table when the windows are short)
    const long long g_lo = ((long long)i_first - kNodeOff) << c.log2_stride, g_hi = ((long long)i_last - 1 - kNodeOff) << c.log2_stride;
    const bool group_reached = hi > lo && g_hi >= r_lo && g_lo <= r_hi;
    if (!(skip_unreached && !__syncthreads_or(group_reached))) {
      Particle q = {};
      if (group_reached) q = load_particle(pc, P_pad, p);
      for (int i = i_first; i < i_last; ++i) {
        const long long pos = ((long long)i - kNodeOff) << c.log2_stride;   // bin position of the node
        const bool reached = hi > lo && pos >= r_lo && pos <= r_hi && c.j0 + pos > 0;
        if (skip_unreached && !__syncthreads_or(reached)) continue;
        NodeOut o = {};
        if (reached) o = eval_node(c, q, c.j0 + pos);
        const size_t at = (size_t)i * P_pad + p;
        node_n[at] = o.n_turns;
        node_frac[at] = o.frac;
        R* a = node_amp + (size_t)i * 4 * P_pad + p;
        a[0] = (R)o.Ar; a[(size_t)P_pad] = (R)o.Ai; a[2 * (size_t)P_pad] = (R)o.Er; a[3 * (size_t)P_pad] = (R)o.Ei;
      }
    }
    if (!ESC) return;
  }
}

// ------------------------------------------------------------------------------------------------ a4 + a5
// sin, cos of 2 pi x for |x| <= 1/8 turn (Taylor in x^2, coefficients (2 pi)^k / k!).
__device__ __forceinline__ void sincos_2pi_small(float x, float& s, float& c) {
  const float x2 = x * x;
  float ps = fmaf(x2, 42.0586939448976531f, -76.7058597530613858f);  // (2pi)^9/9!, -(2pi)^7/7!
  ps = fmaf(ps, x2, 81.6052492760750542f);                            // (2pi)^5/5!
  ps = fmaf(ps, x2, -41.3417022403997602f);                           // -(2pi)^3/3!
  ps = fmaf(ps, x2, 6.28318530717958648f);
  s = ps * x;
  float pc = fmaf(x2, -26.4262567833743975f, 60.2446413718766604f);  // -(2pi)^10/10!, (2pi)^8/8!
  pc = fmaf(pc, x2, -85.4568172066937277f);                           // -(2pi)^6/6!
  pc = fmaf(pc, x2, 64.9393940226682915f);                            // (2pi)^4/4!
  pc = fmaf(pc, x2, -19.7392088021787172f);                           // -(2pi)^2/2!
  c = fmaf(pc, x2, 1.0f);
}
__device__ __forceinline__ void sincos_2pi_small(double x, double& s, double& c) {
  const double x2 = x * x;
  double ps = fma(x2, -0.71812230177850051223, 3.8199525848482821277);     // -(2pi)^15/15!, (2pi)^13/13!
  ps = fma(ps, x2, -15.094642576822990392);                                 // -(2pi)^11/11!
  ps = fma(ps, x2, 42.058693944897653145);
  ps = fma(ps, x2, -76.705859753061385842);
  ps = fma(ps, x2, 81.605249276075054203);
  ps = fma(ps, x2, -41.341702240399760234);
  ps = fma(ps, x2, 6.2831853071795864769);
  s = ps * x;
  double pc = fma(x2, 0.28200596845579121507, -1.7143907110886720654);     // (2pi)^16/16!, -(2pi)^14/14!
  pc = fma(pc, x2, 7.9035363713184688042);                                  // (2pi)^12/12!
  pc = fma(pc, x2, -26.426256783374397453);
  pc = fma(pc, x2, 60.244641371876660363);
  pc = fma(pc, x2, -85.456817206693727736);
  pc = fma(pc, x2, 64.939394022668291491);
  pc = fma(pc, x2, -19.739208802178717238);
  c = fma(pc, x2, 1.0);
}

template <typename R> struct DataT;
template <> struct DataT<double> { using W = double4; using G = double2; static constexpr int chunk = kChunkF64; };

struct DenseArgs {
  const int* edges;            // [n_seg + 1]
  int n_seg;
  int chunk_first;             // first chunk launched (global chunk index)
  const int* chunk_k0;         // [n_chunks_launched] last k with e_k <= chunk start (-1 .. n_seg)
  const int* node_n;           // [n_nodes][P_pad]
  const double* node_frac;
  const void* node_amp;        // R [n_nodes][4][P_pad]
  const int* jlo; const int* jhi;
  int P_pad;
  double* frag;                // [n_chunks_launched][kFragFields][P_pad]
  double* out_seg;             // SEG mode: [P][n_seg][3] (already offset to this batch), else nullptr
  int P;                       // particles in this batch
  double seg_scale_z, seg_scale_s;
  int comp;                    // also accumulate sum_k |z_k| and sum_k sigma_k (Eq. 8, 9 components)
  // k_dense2 only: pieces = fine sub-intervals cut at the segment edges, with the moments of the sigma weights
  const int* piece_first;      // [n_sub_launched + 1] first piece of each launched fine sub-interval
  const ulonglong2* moments;   // [n_pieces][4] = 8 packed (A, E) pairs: sum_j g_a(j) s_j^m, m = 0..6, pad
  // escalation pass (k_dense only): device-side particle count and this batch's offset; nullptr otherwise
  const int* esc_count; int esc_pb;
};

// All-FP64 flavour (few segments, N_seg < 8 by default): one bin per step, quintic phase by 5 forward differences,
// FP64 polynomial sin/cos, FP64 amplitudes and accumulation.
template <bool SEG, bool ESC = false>
__global__ void __launch_bounds__(kBlock) k_dense(DevCfg c, DenseArgs a, const double4* __restrict__ Wg,
                                                  const double2* __restrict__ Gg) {
  using R = double;
  constexpr int SC = 0;
  using WT = typename DataT<R>::W;
  using GT = typename DataT<R>::G;
  constexpr int CH = DataT<R>::chunk;
  __shared__ WT sW[CH];
  __shared__ GT sG[CH];

  const int chunk_l = blockIdx.x;                              // launched-chunk index
  const int cs = (a.chunk_first + chunk_l) * CH;
  const int ce = min(cs + CH, c.n_bins);
  const int esc_lim = ESC ? min(*a.esc_count - a.esc_pb, a.P_pad) : 0;
  if (ESC && (int)(blockIdx.y * kBlock) >= esc_lim) return;
  if (!ESC) {                                                  // as in k_dense2: nothing of this block lives in this chunk
    const int p0 = blockIdx.y * kBlock + threadIdx.x;
    if (!__syncthreads_or((a.jhi[p0] > cs) && (a.jlo[p0] < ce))) {
      double* fz = a.frag + (size_t)chunk_l * kFragFields * a.P_pad + p0;
#pragma unroll
      for (int m = 0; m < kFragFields; ++m) fz[(size_t)m * a.P_pad] = 0.0;
      return;
    }
  }

  for (int t = threadIdx.x; t < ce - cs; t += kBlock) { sW[t] = Wg[cs + t]; sG[t] = Gg[cs + t]; }
  __syncthreads();

  // one pass over the block's 128 particles; in the escalation pass the blocks stride over the selected particles
  for (int pblk = blockIdx.y; ; pblk += gridDim.y) {
  if (ESC && pblk * kBlock >= esc_lim) return;
  const int p = pblk * kBlock + threadIdx.x;                   // particle within the batch (P_pad is a multiple of kBlock)

  const int jlo = a.jlo[p], jhi = a.jhi[p];
  const int S = c.stride, Sf = S >> 2;
  const R hS = R(1.0) / R(Sf);
  const R* __restrict__ namp = reinterpret_cast<const R*>(a.node_amp);

  int k = a.chunk_k0[chunk_l];
  int next_edge = (k + 1 <= a.n_seg) ? a.edges[k + 1] : INT_MAX;
  bool open_at_edge = (k >= 0 && k < a.n_seg) ? (a.edges[k] == cs) : true;
  double Zr = 0.0, Zi = 0.0, Sg = 0.0, ups = 0.0, xs = 0.0, hs = 0.0;
  double* frag = a.frag + (size_t)chunk_l * kFragFields * a.P_pad + p;

  auto close_piece = [&](bool at_edge_end) {
    // at_edge_end: the piece ends at e_{k+1}.  open_at_edge: it began at e_k.
    if (open_at_edge && at_edge_end) {
      if (SEG) {
        if (p < a.P) {
          double* o = a.out_seg + ((size_t)p * a.n_seg + k) * 3;
          o[0] = Zr * a.seg_scale_z; o[1] = Zi * a.seg_scale_z; o[2] = Sg * a.seg_scale_s;
        }
      } else if (Sg > 0.0) {
        const double z2 = Zr * Zr + Zi * Zi;
        ups += z2 / Sg;
        if (a.comp) { xs += sqrt(z2); hs += Sg; }
      }
    } else if (!open_at_edge) {          // began in an earlier chunk: head fragment (closed or running through)
      frag[(size_t)1 * a.P_pad] = Zr; frag[(size_t)2 * a.P_pad] = Zi; frag[(size_t)3 * a.P_pad] = Sg;
    } else {                             // began here, continues into the next chunk: tail fragment
      frag[(size_t)4 * a.P_pad] = Zr; frag[(size_t)5 * a.P_pad] = Zi; frag[(size_t)6 * a.P_pad] = Sg;
    }
    Zr = 0.0; Zi = 0.0; Sg = 0.0;
  };

  int fd_pos = -1;                   // bin the forward-difference state is positioned at (-1: none)
  double phi = 0.0, d1 = 0.0, d2 = 0.0, d3 = 0.0, d4 = 0.0, d5 = 0.0;
  int quad = 0;
  for (int ib = cs; ib < ce; ib += Sf) {
    const int ie = min(ib + Sf, ce);
    const bool lane_in = (ib >= jlo) && (ie <= jhi);
    const bool lane_out = (ie <= jlo) || (ib >= jhi);
    const bool all_in = __all_sync(0xffffffffu, lane_in);
    const bool all_out = __all_sync(0xffffffffu, lane_out);

    R cf[4][4];        // cubic coefficients of (Ar, Ai, Er, Ei) in t = (u - u_sub)/fine_stride
    if (!all_out) {
      const int ic = ib >> c.log2_stride;                      // coarse interval
      const int i0 = ic + kNodeOff;                            // table row of its left node
      const int q = (ib >> (c.log2_stride - 2)) & 3;           // fine sub-interval within the coarse one
      if (fd_pos != ib || q == 0) {
        // (re)build the phase forward differences at u0 = ib - ic*stride from the 6-node quintic
        const size_t base = (size_t)i0 * a.P_pad + p;
        const int n0 = a.node_n[base];
        const double r0 = a.node_frac[base];
        double Y[6];
#pragma unroll
        for (int m = -2; m <= 3; ++m) {
          const size_t at = (size_t)(i0 + m) * a.P_pad + p;
          Y[m + 2] = (double)(a.node_n[at] - n0) + (a.node_frac[at] - r0);
        }
        double b[6], d[6];
        quintic_coeffs(Y, 1.0 / (double)S, b);
        const int u0 = ib - (ic << c.log2_stride);
        if (u0) taylor_shift(b, (double)u0);
        forward_diffs(b, d);
        phi = r0 + b[0]; d1 = d[1]; d2 = d[2]; d3 = d[3]; d4 = d[4]; d5 = d[5];
        quad = 0;
        fd_pos = ib;
      }
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const R* col = namp + ((size_t)i0 * 4 + r) * a.P_pad + p;
        const ptrdiff_t st = (ptrdiff_t)4 * a.P_pad;
        R nd[6];
#pragma unroll
        for (int m = -2; m <= 3; ++m) nd[m + 2] = col[m * st];
        fine_cubic<R>(nd, q, cf[r][0], cf[r][1], cf[r][2], cf[r][3]);
      }
    }
    R s = R(0.0);

    // one bin: phase step + reduction (FP64), sincos, amplitude cubic, multiply-accumulate
    auto bin = [&](int j, bool masked, R& zr, R& zi, R& sg) {
      R cr, sr;
      if (SC == 2 && sizeof(R) == 4) {
        // The phase is never reduced in FP64: adding 1.5 * 2^20 leaves rint(phi * 2^32) mod 2^32 in the low word,
        // i.e. the fraction of a turn in [-1/2, 1/2) as an int32; hardware sin/cos (MUFU) of that angle.
        const int n = __double2loint(phi + 1572864.0);
        const float xr = (float)n * 1.4629180792671596e-09f;          // 2 pi / 2^32
        cr = (R)__cosf(xr); sr = (R)__sinf(xr);
      } else {
        // reduce phi to |x| <= 1/8 turn, carrying the quadrant
        const double t = fma(phi, 4.0, kMagic);
        quad += __double2loint(t);
        const double kf = t - kMagic;
        phi = fma(kf, -0.25, phi);
        R sn, cn;
        sincos_2pi_small((R)phi, sn, cn);
        // rotate by quad * 90 degrees
        const bool swp = quad & 1;
        cr = swp ? sn : cn; sr = swp ? cn : sn;
        cr = ((quad + 1) & 2) ? -cr : cr;
        sr = (quad & 2) ? -sr : sr;
      }
      // advance the forward differences to the next bin
      phi += d1; d1 += d2; d2 += d3; d3 += d4; d4 += d5;
      // amplitudes
      const R Ar = fma(fma(fma(cf[0][3], s, cf[0][2]), s, cf[0][1]), s, cf[0][0]);
      const R Ai = fma(fma(fma(cf[1][3], s, cf[1][2]), s, cf[1][1]), s, cf[1][0]);
      const R Er = fma(fma(fma(cf[2][3], s, cf[2][2]), s, cf[2][1]), s, cf[2][0]);
      const R Ei = fma(fma(fma(cf[3][3], s, cf[3][2]), s, cf[3][1]), s, cf[3][0]);
      s += hS;
      const WT w = sW[j - cs];
      const GT g = sG[j - cs];
      // q = W_A conj(c_A) + W_E conj(c_E)
      R qr = fma(w.x, Ar, fma(w.y, Ai, fma(w.z, Er, w.w * Ei)));
      R qi = fma(w.y, Ar, fma(-w.x, Ai, fma(w.w, Er, -(w.z * Ei))));
      R ss = fma(g.x, fma(Ar, Ar, Ai * Ai), g.y * fma(Er, Er, Ei * Ei));
      if (masked) {
        const bool in = (j >= jlo) && (j < jhi);
        qr = in ? qr : R(0.0); qi = in ? qi : R(0.0); ss = in ? ss : R(0.0);
      }
      // z += q e^{+2 pi i Phi}
      zr = fma(qr, cr, fma(-qi, sr, zr));
      zi = fma(qr, sr, fma(qi, cr, zi));
      sg += ss;
    };

    int j = ib;
    while (j < ie) {
      const int b = min(next_edge, ie);
      const bool live = (k >= 0) && (k < a.n_seg);
      if (b > j) {
        if (all_out) {
          // nothing to add; the forward-difference state is rebuilt at the next interval
        } else if (!live) {
          for (int jj = j; jj < b; ++jj) { phi += d1; d1 += d2; d2 += d3; d3 += d4; d4 += d5; s += hS; }
          fd_pos = b;
        } else {
          for (int jj = j; jj < b;) {
            const int e2 = min(jj + kFlushBins, b);
            R zr = R(0.0), zi = R(0.0), sg = R(0.0);
            if (all_in) { for (; jj < e2; ++jj) bin(jj, false, zr, zi, sg); }
            else        { for (; jj < e2; ++jj) bin(jj, true, zr, zi, sg); }
            Zr += (double)zr; Zi += (double)zi; Sg += (double)sg;
          }
          fd_pos = b;
        }
        j = b;
      }
      if (j == next_edge) {
        if (live) close_piece(true);
        ++k;
        next_edge = (k + 1 <= a.n_seg) ? a.edges[k + 1] : INT_MAX;
        open_at_edge = true;
      }
    }
  }
  // the piece still open at the chunk end
  if (k >= 0 && k < a.n_seg) close_piece(false);
  if (!SEG) {
    frag[0] = ups;
    if (a.comp) { frag[(size_t)7 * a.P_pad] = xs; frag[(size_t)8 * a.P_pad] = hs; }
  }
  if (!ESC) return;
  }
}


// ------------------------------------------------------------------------------------------------ a4 + a5, FP32x2
// The FP32-amplitude flavour of the hot loop, written for the packed FP32 pipe of sm_100a (FFMA2 / FMUL2 / FADD2:
// one issue slot carries two FP32 operations).  Each lane (= particle) walks its chunk two bins at a time: the low
// half of every packed register belongs to the even bin 2m, the high half to the odd bin 2m+1, so the whole
// per-bin arithmetic (amplitude cubics, the complex multiply-accumulate with the data, |h|^2) is element-wise and
// needs no swizzle.  Segment edges on odd bins split a pair between two segments (the pair is evaluated once).
// Phase: per fine sub-interval the 6-node quintic is economised (Chebyshev) to a cubic and advanced by forward
// differences, 3 FP64 adds per bin; the fraction of a turn is read from the low word of phi + 1.5 * 2^20.
typedef unsigned long long u64;
__device__ __forceinline__ u64 f2pack(float lo, float hi) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void f2unpack(u64 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ u64 f2fma(u64 a, u64 b, u64 c) { u64 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ u64 f2mul(u64 a, u64 b) { u64 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 f2add(u64 a, u64 b) { u64 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 f2neg(u64 a) { float lo, hi; f2unpack(a, lo, hi); return f2pack(-lo, -hi); }   // folded into FFMA2 by ptxas
__device__ __forceinline__ u64 f2bcast(float v) { return f2pack(v, v); }

__device__ __forceinline__ u64 f2sub(u64 a, u64 b) { u64 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }

// Cubic coefficients on fine sub-interval q for two amplitude components at once (the halves of the packed registers):
// kFineM applied to node[m] - node[2], so that the rounding of the matrix entries acts on small differences only.
__device__ __forceinline__ void fine_cubic2(const u64 nd[6], int q, u64 out[4]) {
  u64 dl[6];
#pragma unroll
  for (int m = 0; m < 6; ++m) dl[m] = f2sub(nd[m], nd[2]);
#pragma unroll
  for (int kk = 0; kk < 4; ++kk) {
    u64 acc = (kk == 0) ? nd[2] : 0ull;
#pragma unroll
    for (int m = 0; m < 6; ++m)
      if (m != 2) acc = f2fma(f2bcast(kFineM[q][kk][m]), dl[m], acc);
    out[kk] = acc;
  }
}

#ifndef SC_DENSE2_MINB
#define SC_DENSE2_MINB 4     /* CTAs per SM the register allocation aims at (128 registers/thread) */
#endif

constexpr int kPairRec = 3;

// Moments of the sigma weights over one piece (a fine sub-interval cut at the segment edges; shared by all particles):
//   M_a,m = sum_{j in piece} G_a(j) s_j^m,  s_j = (j - sub-interval start)/Sf,  m = 0..6,  a = A, E.
// On a fine sub-interval the amplitudes are cubics in s, so |c_a(s)|^2 is a polynomial of degree 6 and
// sigma_piece = sum_m (e_A,m M_A,m + e_E,m M_E,m) -- the per-bin evaluation of |h|^2 leaves the hot loop.
__global__ void k_moments(const double2* __restrict__ G64, const int* __restrict__ piece_lo, const int* __restrict__ piece_hi,
                          int n_pieces, int n_bins, int log2_fine, float2* __restrict__ out /* [n_pieces][8] */) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_pieces) return;
  // piece_lo == nullptr: uniform pieces of 2^(int)(size_t)piece_hi bins (the groups / sub-intervals of the adaptive path)
  const int lg_u = (int)(size_t)piece_hi;
  const int lo = piece_lo ? piece_lo[i] : (i << lg_u);
  const int hi = min(piece_lo ? piece_hi[i] : ((i + 1) << lg_u), n_bins);
  const int ib = (lo >> log2_fine) << log2_fine;
  const double hS = 1.0 / (double)(1 << log2_fine);
  double mA[7] = {0, 0, 0, 0, 0, 0, 0}, mE[7] = {0, 0, 0, 0, 0, 0, 0};
  for (int j = lo; j < hi; ++j) {
    const double2 g = G64[j];
    const double sj = (double)(j - ib) * hS;
    double pw = 1.0;
#pragma unroll
    for (int m = 0; m < 7; ++m) { mA[m] = fma(g.x, pw, mA[m]); mE[m] = fma(g.y, pw, mE[m]); pw *= sj; }
  }
#pragma unroll
  for (int m = 0; m < 7; ++m) out[(size_t)i * 8 + m] = make_float2((float)mA[m], (float)mE[m]);
  out[(size_t)i * 8 + 7] = make_float2(0.f, 0.f);
}            // ulonglong2 records per bin pair: (wAr, wAi), (wEr, wEi), (gA, gE), each (even, odd)

// FP32 sin/cos of a phase given as a signed 32-bit fraction of a turn: polynomial flavour (SC = 0).
__device__ __forceinline__ void sincos_frac32(int n, float& sr, float& cr) {
  const int q = (n + (1 << 29)) >> 30;                       // nearest quarter turn
  const float x = (float)(n - (q << 30)) * 2.3283064365386963e-10f;   // |x| <= 1/8 turn
  float sn, cn;
  sincos_2pi_small(x, sn, cn);
  const bool swp = q & 1;
  cr = swp ? sn : cn; sr = swp ? cn : sn;
  cr = ((q + 1) & 2) ? -cr : cr;
  sr = (q & 2) ? -sr : sr;
}

// ---- pieces of the packed hot loop shared by k_dense2 (shared edges) and k_dense2_ad (per-particle edges) ----
struct PhaseFD { double phi, d1, d2, d3; };   // phase in turns at the next bin and its forward differences (unit steps)
__device__ __forceinline__ void phase_next_pair(PhaseFD& ph, int& n0, int& n1) {
  n0 = __double2loint(ph.phi);
  ph.phi += ph.d1; ph.d1 += ph.d2; ph.d2 += ph.d3;
  n1 = __double2loint(ph.phi);
  ph.phi += ph.d1; ph.d1 += ph.d2; ph.d2 += ph.d3;
}
__device__ __forceinline__ void phase_skip_pair(PhaseFD& ph) {
  ph.phi += ph.d1; ph.d1 += ph.d2; ph.d2 += ph.d3;
  ph.phi += ph.d1; ph.d1 += ph.d2; ph.d2 += ph.d3;
}
__device__ __forceinline__ void phase_set(PhaseFD& ph, double p0, const double b[6]) {
  // phi carries the bias 1.5 * 2^20: in that binade the unit in the last place is 2^-32 turn, so the low word of phi IS the
  // fraction of a turn as an int32 -- no separate biasing add per bin.  Every step then rounds to 2^-32 turn (1.5e-9 rad): a
  // random walk of < 1e-8 rad over a fine sub-interval (<= 512 steps), far below the FP32 amplitudes' 1e-7 per bin.
  ph.phi = p0 + 1572864.0;
  ph.d1 = b[1] + b[2] + b[3];
  ph.d2 = 2.0 * b[2] + 6.0 * b[3];
  ph.d3 = 6.0 * b[3];
}

// Phase on fine sub-interval [ib, ib + Sf): quintic through 6 nodes -> Taylor shift to the centre of the sub-interval ->
// Chebyshev economisation to a cubic on [-H, H] -> shift to the start -> forward differences for unit steps.
__device__ __forceinline__ void sub_phase(const DevCfg& c, const DenseArgs& a, int p, int ib, PhaseFD& ph) {
  const int ic = ib >> c.log2_stride;
  const int i0 = ic + kNodeOff;
  const int S = c.stride, Sf = S >> 2;
  const size_t base = (size_t)i0 * a.P_pad + p;
  const int n0 = a.node_n[base];
  const double r0 = a.node_frac[base];
  double Y[6];
#pragma unroll
  for (int m = -2; m <= 3; ++m) {
    const size_t at = (size_t)(i0 + m) * a.P_pad + p;
    Y[m + 2] = (double)(a.node_n[at] - n0) + (a.node_frac[at] - r0);
  }
  double b[6];
  quintic_coeffs(Y, 1.0 / (double)S, b);
  const double H = 0.5 * (double)Sf;
  taylor_shift(b, (double)(ib - (ic << c.log2_stride)) + H);
  const double H2 = H * H, H4 = H2 * H2;
  b[0] = fma(-0.125 * H4, b[4], b[0]);
  b[2] = fma(H2, b[4], b[2]);
  b[1] = fma(-0.3125 * H4, b[5], b[1]);
  b[3] = fma(1.25 * H2, b[5], b[3]);
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 2; j >= i; --j) b[j] = fma(-H, b[j + 1], b[j]);
  phase_set(ph, r0 + b[0], b);
}

// Cubic coefficients of (Ar, Ai, Er, Ei) on that sub-interval in s = (j - ib)/Sf.
__device__ __forceinline__ void sub_amps(const DevCfg& c, const DenseArgs& a, int p, int ib, float (&cf)[4][4]) {
  const int i0 = (ib >> c.log2_stride) + kNodeOff;
  const int q = (ib >> (c.log2_stride - 2)) & 3;
  const float* __restrict__ namp = reinterpret_cast<const float*>(a.node_amp);
#pragma unroll
  for (int r = 0; r < 4; r += 2) {                          // (Ar, Ai) then (Er, Ei) as packed halves
    const float* col = namp + ((size_t)i0 * 4 + r) * a.P_pad + p;
    const ptrdiff_t st = (ptrdiff_t)4 * a.P_pad;
    u64 nd[6], o[4];
#pragma unroll
    for (int m = -2; m <= 3; ++m) nd[m + 2] = f2pack(col[m * st], col[m * st + a.P_pad]);
    fine_cubic2(nd, q, o);
#pragma unroll
    for (int kk = 0; kk < 4; ++kk) f2unpack(o[kk], cf[r][kk], cf[r + 1][kk]);
  }
}

// One bin pair (j, j+1): FP64 phase steps, sin/cos, amplitude cubics, multiply-accumulate into packed sums (low half =
// even bin, high half = odd bin).  MASKED: apply the particle's time window per bin.  WITH_SG: accumulate |h|^2 per
// bin (otherwise sigma comes from the moments).  s2 = (s_j, s_{j+1}), rec = the pair's data record; both advance.
template <bool MASKED, bool WITH_SG, int SC>
__device__ __forceinline__ void pair_eval(PhaseFD& ph, const float (&cf)[4][4], u64& s2, const ulonglong2*& rec, int j,
                                          int jlo, int jhi, u64 h2, u64 K2, u64& zr2, u64& zi2, u64& sg2) {
  int n0, n1;
  phase_next_pair(ph, n0, n1);
  float c0, c1, s0, s1;
  if (SC == 2) {
    float x0, x1;
    f2unpack(f2mul(f2pack((float)n0, (float)n1), K2), x0, x1);
    c0 = __cosf(x0); s0 = __sinf(x0); c1 = __cosf(x1); s1 = __sinf(x1);
  } else {
    sincos_frac32(n0, s0, c0);
    sincos_frac32(n1, s1, c1);
  }
  u64 cr2 = f2pack(c0, c1), sr2 = f2pack(s0, s1);
  const u64 Ar = f2fma(f2fma(f2fma(f2bcast(cf[0][3]), s2, f2bcast(cf[0][2])), s2, f2bcast(cf[0][1])), s2, f2bcast(cf[0][0]));
  const u64 Ai = f2fma(f2fma(f2fma(f2bcast(cf[1][3]), s2, f2bcast(cf[1][2])), s2, f2bcast(cf[1][1])), s2, f2bcast(cf[1][0]));
  const u64 Er = f2fma(f2fma(f2fma(f2bcast(cf[2][3]), s2, f2bcast(cf[2][2])), s2, f2bcast(cf[2][1])), s2, f2bcast(cf[2][0]));
  const u64 Ei = f2fma(f2fma(f2fma(f2bcast(cf[3][3]), s2, f2bcast(cf[3][2])), s2, f2bcast(cf[3][1])), s2, f2bcast(cf[3][0]));
  s2 = f2add(s2, h2);
  const ulonglong2 wA = rec[0], wE = rec[1];
  u64 m2 = 0;
  if (MASKED) {
    m2 = f2pack((j >= jlo && j < jhi) ? 1.0f : 0.0f, (j + 1 >= jlo && j + 1 < jhi) ? 1.0f : 0.0f);
    cr2 = f2mul(cr2, m2); sr2 = f2mul(sr2, m2);
  }
  // q = W_A conj(c_A) + W_E conj(c_E)
  const u64 qr = f2fma(wA.x, Ar, f2fma(wA.y, Ai, f2fma(wE.x, Er, f2mul(wE.y, Ei))));
  const u64 qi = f2fma(wA.y, Ar, f2fma(f2neg(wA.x), Ai, f2fma(wE.y, Er, f2neg(f2mul(wE.x, Ei)))));
  if (WITH_SG) {
    ulonglong2 g = rec[2];
    if (MASKED) { g.x = f2mul(g.x, m2); g.y = f2mul(g.y, m2); }
    sg2 = f2fma(g.x, f2fma(Ar, Ar, f2mul(Ai, Ai)), f2fma(g.y, f2fma(Er, Er, f2mul(Ei, Ei)), sg2));
  }
  rec += kPairRec;
  // z += q e^{+2 pi i Phi}
  zr2 = f2fma(qr, cr2, f2fma(f2neg(qi), sr2, zr2));
  zi2 = f2fma(qr, sr2, f2fma(qi, cr2, zi2));
}

// sigma of a run of bins from the moments of its weights: |c_a(s)|^2 = sum_m e_a,m s^m with the cubic coefficients of
// the sub-interval; both channels at once (A in the low half, E in the high half).  mp: 4 records = 8 (A, E) pairs.
__device__ __forceinline__ double sigma_moments(const float (&cf)[4][4], const ulonglong2* __restrict__ mp) {
  const ulonglong2 m01 = mp[0], m23 = mp[1], m45 = mp[2], m6 = mp[3];
  u64 R[4], I[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) { R[i] = f2pack(cf[0][i], cf[2][i]); I[i] = f2pack(cf[1][i], cf[3][i]); }
  const u64 two = f2bcast(2.0f);
  const u64 R0x2 = f2mul(R[0], two), I0x2 = f2mul(I[0], two), R1x2 = f2mul(R[1], two), I1x2 = f2mul(I[1], two);
  const u64 R2x2 = f2mul(R[2], two), I2x2 = f2mul(I[2], two);
  const u64 e0 = f2fma(R[0], R[0], f2mul(I[0], I[0]));
  const u64 e1 = f2fma(R0x2, R[1], f2mul(I0x2, I[1]));
  const u64 e2 = f2fma(R0x2, R[2], f2fma(I0x2, I[2], f2fma(R[1], R[1], f2mul(I[1], I[1]))));
  const u64 e3 = f2fma(R0x2, R[3], f2fma(I0x2, I[3], f2fma(R1x2, R[2], f2mul(I1x2, I[2]))));
  const u64 e4 = f2fma(R1x2, R[3], f2fma(I1x2, I[3], f2fma(R[2], R[2], f2mul(I[2], I[2]))));
  const u64 e5 = f2fma(R2x2, R[3], f2mul(I2x2, I[3]));
  const u64 e6 = f2fma(R[3], R[3], f2mul(I[3], I[3]));
  u64 acc = f2mul(e0, m01.x);
  acc = f2fma(e1, m01.y, acc); acc = f2fma(e2, m23.x, acc); acc = f2fma(e3, m23.y, acc);
  acc = f2fma(e4, m45.x, acc); acc = f2fma(e5, m45.y, acc); acc = f2fma(e6, m6.x, acc);
  float l, h;
  f2unpack(acc, l, h);
  return (double)l + (double)h;
}

// sin, cos of the phase at the next two bins as packed halves; advances the phase by two bins.
template <int SC>
__device__ __forceinline__ void sincos_pair(PhaseFD& ph, u64 K2, u64& cr2, u64& sr2) {
  int n0, n1;
  phase_next_pair(ph, n0, n1);
  float c0, c1, s0, s1;
  if (SC == 2) {
    float x0, x1;
    f2unpack(f2mul(f2pack((float)n0, (float)n1), K2), x0, x1);
    c0 = __cosf(x0); s0 = __sinf(x0); c1 = __cosf(x1); s1 = __sinf(x1);
  } else {
    sincos_frac32(n0, s0, c0);
    sincos_frac32(n1, s1, c1);
  }
  cr2 = f2pack(c0, c1); sr2 = f2pack(s0, s1);
}
// amplitude cubics at (s_j, s_{j+1}), q = W_A conj(c_A) + W_E conj(c_E), z += q e^{+2 pi i Phi}
__device__ __forceinline__ void mac_pair(const float (&cf)[4][4], u64& s2, const ulonglong2 wA, const ulonglong2 wE, u64 h2,
                                         u64 cr2, u64 sr2, u64& zr2, u64& zi2) {
  const u64 Ar = f2fma(f2fma(f2fma(f2bcast(cf[0][3]), s2, f2bcast(cf[0][2])), s2, f2bcast(cf[0][1])), s2, f2bcast(cf[0][0]));
  const u64 Ai = f2fma(f2fma(f2fma(f2bcast(cf[1][3]), s2, f2bcast(cf[1][2])), s2, f2bcast(cf[1][1])), s2, f2bcast(cf[1][0]));
  const u64 Er = f2fma(f2fma(f2fma(f2bcast(cf[2][3]), s2, f2bcast(cf[2][2])), s2, f2bcast(cf[2][1])), s2, f2bcast(cf[2][0]));
  const u64 Ei = f2fma(f2fma(f2fma(f2bcast(cf[3][3]), s2, f2bcast(cf[3][2])), s2, f2bcast(cf[3][1])), s2, f2bcast(cf[3][0]));
  s2 = f2add(s2, h2);
  const u64 qr = f2fma(wA.x, Ar, f2fma(wA.y, Ai, f2fma(wE.x, Er, f2mul(wE.y, Ei))));
  const u64 qi = f2fma(wA.y, Ar, f2fma(f2neg(wA.x), Ai, f2fma(wE.y, Er, f2neg(f2mul(wE.x, Ei)))));
  zr2 = f2fma(qr, cr2, f2fma(f2neg(qi), sr2, zr2));
  zi2 = f2fma(qr, sr2, f2fma(qi, cr2, zi2));
}
// n >= 1 consecutive unmasked pairs, software-pipelined by hand: the sin/cos (FP64 step, conversion, MUFU) and the
// shared-memory loads of pair i+1 are issued before the multiply-accumulate of pair i.
template <int SC>
__device__ __forceinline__ void pairs_fast(PhaseFD& ph, const float (&cf)[4][4], u64& s2, const ulonglong2*& rec, int n,
                                           u64 h2, u64 K2, u64& zr2, u64& zi2) {
  u64 cr, sr;
  sincos_pair<SC>(ph, K2, cr, sr);
  ulonglong2 wA = rec[0], wE = rec[1];
#pragma unroll 1
  for (int i = 1; i < n; ++i) {
    u64 crn, srn;
    sincos_pair<SC>(ph, K2, crn, srn);
    rec += kPairRec;
    const ulonglong2 wAn = rec[0], wEn = rec[1];
    mac_pair(cf, s2, wA, wE, h2, cr, sr, zr2, zi2);
    cr = crn; sr = srn; wA = wAn; wE = wEn;
  }
  rec += kPairRec;
  mac_pair(cf, s2, wA, wE, h2, cr, sr, zr2, zi2);
}

template <bool SEG, int SC>
__global__ void __launch_bounds__(kBlock, SC_DENSE2_MINB) k_dense2(DevCfg c, DenseArgs a, const ulonglong2* __restrict__ Dg) {
  constexpr int CH = kChunkF32;
  __shared__ ulonglong2 sD[CH / 2 * kPairRec];                 // 48 KB

  const int chunk_l = blockIdx.x;
  const int cs = (a.chunk_first + chunk_l) * CH;
  const int ce = min(cs + CH, c.n_bins);
  const int ce2 = (ce + 1) & ~1;                               // pair-aligned end (data beyond n_bins is zero)
  const int p = blockIdx.y * kBlock + threadIdx.x;

  // no particle of this block has its time window in this chunk (common once the batch is sorted by window start):
  // leave empty fragments and skip the staging of the data
  if (!__syncthreads_or((a.jhi[p] > cs) && (a.jlo[p] < ce))) {
    double* fz = a.frag + (size_t)chunk_l * kFragFields * a.P_pad + p;
#pragma unroll
    for (int m = 0; m < kFragFields; ++m) fz[(size_t)m * a.P_pad] = 0.0;
    return;
  }

  {
    const ulonglong2* src = Dg + (size_t)(cs >> 1) * kPairRec;
#pragma unroll 4
    for (int t = threadIdx.x; t < CH / 2 * kPairRec; t += kBlock) sD[t] = src[t];
  }
  __syncthreads();

  const int jlo = a.jlo[p], jhi = a.jhi[p];
  const int S = c.stride, Sf = S >> 2;
  const float hS = 1.0f / (float)Sf;
  const u64 h2 = f2bcast(2.0f * hS);
  const u64 K2 = f2bcast(1.4629180792671596e-09f);            // 2 pi / 2^32

  int k = a.chunk_k0[chunk_l];
  int next_edge = (k + 1 <= a.n_seg) ? a.edges[k + 1] : INT_MAX;
  bool open_at_edge = (k >= 0 && k < a.n_seg) ? (a.edges[k] == cs) : true;
  double Zr = 0.0, Zi = 0.0, Sg = 0.0, ups = 0.0, xs = 0.0, hs = 0.0;
  double* frag = a.frag + (size_t)chunk_l * kFragFields * a.P_pad + p;

  auto close_piece = [&](bool at_edge_end) {
    if (open_at_edge && at_edge_end) {
      if (SEG) {
        if (p < a.P) {
          double* o = a.out_seg + ((size_t)p * a.n_seg + k) * 3;
          o[0] = Zr * a.seg_scale_z; o[1] = Zi * a.seg_scale_z; o[2] = Sg * a.seg_scale_s;
        }
      } else if (Sg > 0.0) {
        const double z2 = Zr * Zr + Zi * Zi;
        ups += z2 / Sg;
        if (a.comp) { xs += sqrt(z2); hs += Sg; }
      }
    } else if (!open_at_edge) {
      frag[(size_t)1 * a.P_pad] = Zr; frag[(size_t)2 * a.P_pad] = Zi; frag[(size_t)3 * a.P_pad] = Sg;
    } else {
      frag[(size_t)4 * a.P_pad] = Zr; frag[(size_t)5 * a.P_pad] = Zi; frag[(size_t)6 * a.P_pad] = Sg;
    }
    Zr = 0.0; Zi = 0.0; Sg = 0.0;
  };
  auto next_segment = [&]() {
    ++k;
    next_edge = (k + 1 <= a.n_seg) ? a.edges[k + 1] : INT_MAX;
    open_at_edge = true;
  };

  PhaseFD fd = {};
  for (int ib = cs; ib < ce2; ib += Sf) {
    const int ie = min(ib + Sf, ce2);
    const bool lane_in = (ib >= jlo) && (ie <= jhi);
    const bool lane_out = (ie <= jlo) || (ib >= jhi);
    const bool all_in = __all_sync(0xffffffffu, lane_in);
    const bool all_out = __all_sync(0xffffffffu, lane_out);

    float cf[4][4];    // cubic coefficients of (Ar, Ai, Er, Ei) in s = (j - ib)/Sf (FFMA2 broadcasts a scalar operand)
    if (!all_out) {
      sub_phase(c, a, p, ib, fd);
      sub_amps(c, a, p, ib, cf);
    }

    u64 s2 = 0;        // (s_j, s_{j+1}) of the next pair
    const ulonglong2* rec = sD;   // its data record
    auto pair = [&](int j, auto masked_c, auto with_sg_c, u64& zr2, u64& zi2, u64& sg2) {
      pair_eval<decltype(masked_c)::value, decltype(with_sg_c)::value, SC>(fd, cf, s2, rec, j, jlo, jhi, h2, K2, zr2, zi2, sg2);
    };
    auto sigma_piece = [&](int piece) { Sg += sigma_moments(cf, a.moments + (size_t)piece * 4); };
    using T_ = std::true_type; using F_ = std::false_type;

    // Walk the pieces of this sub-interval (it is cut at every distinct edge inside it).  Pairs are evaluated once:
    // when a piece ends on an odd bin the straddling pair forms a flush group of its own, its low half goes to the
    // piece that ends and its high half is carried into the next piece.
    const bool use_mom = all_in;      // all lanes inside their windows: sigma from the piece moments, unmasked pairs
    int piece = use_mom ? a.piece_first[(ib >> (c.log2_stride - 2)) - ((a.chunk_first * CH) >> (c.log2_stride - 2))] : 0;
    float car_zr = 0.f, car_zi = 0.f, car_sg = 0.f;
    bool carry = false;
    int pl = ib;
    while (pl < ie) {
      const int ph = min(next_edge, ie);                       // next_edge > pl: edges <= pl are consumed
      const bool live = (k >= 0) && (k < a.n_seg);
      int jj = pl;
      if (carry) {
        if (live) { Zr += (double)car_zr; Zi += (double)car_zi; Sg += (double)car_sg; }
        carry = false;
        jj = pl + 1;
      }
      const int jfull = ph & ~1;                               // full pairs end here; a straddling pair follows if ph is odd
      if (!all_out) {
        if (!live && jj < jfull) {
          for (int t = jj; t < jfull; t += 2) phase_skip_pair(fd);
          jj = jfull;
        }
        s2 = f2pack((float)(jj - ib) * hS, (float)(jj + 1 - ib) * hS);
        rec = sD + ((jj - cs) >> 1) * kPairRec;
        while (jj < ph) {
          const bool split = (jj == jfull);                    // the pair (ph - 1, ph)
          const int e2 = split ? jj + 2 : min(jj + kFlushBins, jfull);
          u64 zr2 = 0, zi2 = 0, sg2 = 0;
          if (use_mom) { pairs_fast<SC>(fd, cf, s2, rec, (e2 - jj) >> 1, h2, K2, zr2, zi2); jj = e2; }
          else         { for (; jj < e2; jj += 2) pair(jj, T_{}, T_{}, zr2, zi2, sg2); }
          float zrl, zrh, zil, zih, sgl, sgh;
          f2unpack(zr2, zrl, zrh); f2unpack(zi2, zil, zih); f2unpack(sg2, sgl, sgh);
          if (split) { car_zr = zrh; car_zi = zih; car_sg = sgh; carry = true; zrh = 0.f; zih = 0.f; sgh = 0.f; }
          if (live) { Zr += (double)(zrl + zrh); Zi += (double)(zil + zih); Sg += (double)(sgl + sgh); }
        }
      } else if (ph & 1) {
        car_zr = 0.f; car_zi = 0.f; car_sg = 0.f; carry = true;   // keep the bookkeeping of the walk uniform
      }
      if (use_mom && live) sigma_piece(piece);
      ++piece;
      while (next_edge == ph) {                                // segments that end here (incl. empty ones)
        if (k >= 0 && k < a.n_seg) close_piece(true);
        next_segment();
      }
      pl = ph;
    }
  }
  // (a segment that ends exactly on the chunk end was closed by the walk: the host's CF_HEAD_CLOSES rule says the same)
  // the piece still open at the chunk end
  if (k >= 0 && k < a.n_seg) close_piece(false);
  if (!SEG) {
    frag[0] = ups;
    if (a.comp) { frag[(size_t)7 * a.P_pad] = xs; frag[(size_t)8 * a.P_pad] = hs; }
  }
}

// ------------------------------------------------------------------------------------------------ per-particle segments
// Equal squared-SNR segments re-evaluated for every particle (App. A):
//   s_j = sum_a |h_a(f_j)|^2 / S_a(f_j),  C = sum_j s_j,  e_0 = 0, e_N = n_bins,
//   e_n = min{ j : sum_{j' < j} s_j' >= C n / N }   (n = 1 .. N-1),
// then Upsilon_N on those edges.  Three steps, all with lane = particle:
//   k_sigma_chunks   sigma of every (chunk, particle) from the moments of the weights (no per-bin work inside the window)
//   k_scan_chunks    prefix sum over chunks -> cumulative sigma at every chunk start, and C
//   k_dense2_ad      the hot loop of k_dense2 with a running cumulative sigma per lane: groups of <= 32 bins in which
//                    no lane of the warp reaches its next target (decided from the group's moments) take the unmasked
//                    packed path; the others are walked bin by bin and the segments are closed where the running sum
//                    crosses the target.  The number of edges closed inside a chunk is fixed by the scanned sums
//                    (k0 = K(cbase[chunk]), k1 = K(cbase[chunk + 1])), so neighbouring chunks always agree.
constexpr int kFragAd = 10;    // partial Upsilon, head (zr, zi, sg), tail (zr, zi, sg), head-closes flag, partial sum|z|, sum sigma

struct AdaptArgs {
  int n_seg, n_chunks;
  const double* cbase;         // [n_chunks + 1][P_pad]: cumulative sigma at the chunk starts; row n_chunks = C
  const ulonglong2* gmom;      // [n_groups][4] moments of the weights over groups of 2^lg_group bins
  const ulonglong2* smom;      // [n_sub][4]    ... over the fine sub-intervals
  int lg_group;
  int* out_edges;              // [P][n_seg + 1] of this batch, or nullptr
  double* chunk_sigma;         // = cbase (written by k_sigma_chunks before the scan)
};

__device__ __forceinline__ double seg_target(double C, int n, int N) { return C * (double)n / (double)N; }
// K(c) = max{ n in [0, N-1] : C n / N <= c }: the segment that contains the first bin whose cumulative sum is c.
__device__ __forceinline__ int seg_index(double cum, double C, int N) {
  if (!(C > 0.0)) return 0;
  int n = (int)(cum / C * (double)N);
  n = min(max(n, 0), N - 1);
  while (n + 1 <= N - 1 && seg_target(C, n + 1, N) <= cum) ++n;
  while (n > 0 && seg_target(C, n, N) > cum) --n;
  return n;
}

__global__ void __launch_bounds__(kBlock) k_sigma_chunks(DevCfg c, DenseArgs a, AdaptArgs ad, const float4* __restrict__ D32) {
  constexpr int CH = kChunkF32;
  const int chunk = blockIdx.x;
  const int cs = chunk * CH;
  const int ce = min(cs + CH, c.n_bins);
  const int ce2 = (ce + 1) & ~1;
  const int p = blockIdx.y * kBlock + threadIdx.x;
  const int jlo = a.jlo[p], jhi = a.jhi[p];
  const int Sf = c.stride >> 2;
  const float hS = 1.0f / (float)Sf;
  double tot = 0.0;
  for (int ib = cs; ib < ce2; ib += Sf) {
    const int ie = min(ib + Sf, ce2);
    const bool lane_in = (ib >= jlo) && (ie <= jhi);
    const bool lane_out = (ie <= jlo) || (ib >= jhi);
    const bool all_in = __all_sync(0xffffffffu, lane_in);
    const bool all_out = __all_sync(0xffffffffu, lane_out);
    if (all_out) continue;
    float cf[4][4];
    sub_amps(c, a, p, ib, cf);
    if (all_in) {
      tot += sigma_moments(cf, ad.smom + (size_t)(ib >> (c.log2_stride - 2)) * 4);
    } else {
      // a window border of some lane falls in this sub-interval: bin by bin, masked (two sub-intervals per particle)
      for (int j = ib; j < ie; ++j) {
        const float sj = (float)(j - ib) * hS;
        const float Ar = fmaf(fmaf(fmaf(cf[0][3], sj, cf[0][2]), sj, cf[0][1]), sj, cf[0][0]);
        const float Ai = fmaf(fmaf(fmaf(cf[1][3], sj, cf[1][2]), sj, cf[1][1]), sj, cf[1][0]);
        const float Er = fmaf(fmaf(fmaf(cf[2][3], sj, cf[2][2]), sj, cf[2][1]), sj, cf[2][0]);
        const float Ei = fmaf(fmaf(fmaf(cf[3][3], sj, cf[3][2]), sj, cf[3][1]), sj, cf[3][0]);
        const float4 g = D32[(size_t)(j >> 1) * kPairRec + 2];            // (gA even, gA odd, gE even, gE odd)
        const float gA = (j & 1) ? g.y : g.x, gE = (j & 1) ? g.w : g.z;
        const float sg = fmaf(gA, fmaf(Ar, Ar, Ai * Ai), gE * fmaf(Er, Er, Ei * Ei));
        if (j >= jlo && j < jhi) tot += (double)sg;
      }
    }
  }
  ad.chunk_sigma[(size_t)(chunk + 1) * a.P_pad + p] = tot;
}

__global__ void k_scan_chunks(double* __restrict__ cbase, int n_chunks, int P_pad) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P_pad) return;
  double acc = 0.0;
  cbase[p] = 0.0;
  for (int i = 1; i <= n_chunks; ++i) {
    acc += cbase[(size_t)i * P_pad + p];
    cbase[(size_t)i * P_pad + p] = acc;
  }
}

template <int SC>
__global__ void __launch_bounds__(kBlock, SC_DENSE2_MINB) k_dense2_ad(DevCfg c, DenseArgs a, AdaptArgs ad,
                                                                      const ulonglong2* __restrict__ Dg) {
  constexpr int CH = kChunkF32;
  __shared__ ulonglong2 sD[CH / 2 * kPairRec];
  const int chunk = blockIdx.x;
  const int cs = chunk * CH;
  const int ce = min(cs + CH, c.n_bins);
  const int ce2 = (ce + 1) & ~1;
  const int p = blockIdx.y * kBlock + threadIdx.x;
  {
    const ulonglong2* src = Dg + (size_t)(cs >> 1) * kPairRec;
#pragma unroll 4
    for (int t = threadIdx.x; t < CH / 2 * kPairRec; t += kBlock) sD[t] = src[t];
  }
  __syncthreads();

  const int jlo = a.jlo[p], jhi = a.jhi[p];
  const int Sf = c.stride >> 2;
  const float hS = 1.0f / (float)Sf;
  const u64 h2 = f2bcast(2.0f * hS);
  const u64 K2 = f2bcast(1.4629180792671596e-09f);
  const int N = ad.n_seg;
  const int Gs = 1 << ad.lg_group;

  const double C = ad.cbase[(size_t)ad.n_chunks * a.P_pad + p];
  const double cb0 = ad.cbase[(size_t)chunk * a.P_pad + p];
  const double cb1 = ad.cbase[(size_t)(chunk + 1) * a.P_pad + p];
  int k = seg_index(cb0, C, N);                 // segment open at the chunk start
  const int k1 = seg_index(cb1, C, N);          // edges k+1 .. k1 are closed inside this chunk, no more, no fewer
  double t_next = (k < k1) ? seg_target(C, k + 1, N) - cb0 : INFINITY;
  double crel = 0.0, c_open = 0.0;              // cumulative sigma relative to the chunk start; its value where the open piece began
  double Zr = 0.0, Zi = 0.0, ups = 0.0, xs = 0.0, hs = 0.0;
  bool closed_any = false;
  double* frag = a.frag + (size_t)chunk * kFragAd * a.P_pad + p;

  auto close_at = [&](int j) {                  // edge k+1 lies at bin j
    const double Sg = crel - c_open;
    if (!closed_any) {                          // the piece that was open at the chunk start: head fragment
      frag[(size_t)1 * a.P_pad] = Zr; frag[(size_t)2 * a.P_pad] = Zi; frag[(size_t)3 * a.P_pad] = Sg;
      closed_any = true;
    } else if (Sg > 0.0) {
      const double z2 = Zr * Zr + Zi * Zi;
      ups += z2 / Sg;
      if (a.comp) { xs += sqrt(z2); hs += Sg; }
    }
    Zr = 0.0; Zi = 0.0; c_open = crel;
    ++k;
    if (ad.out_edges && p < a.P) ad.out_edges[(size_t)p * (N + 1) + k] = j;
    t_next = (k < k1) ? seg_target(C, k + 1, N) - cb0 : INFINITY;
  };

  PhaseFD ph = {};
  for (int ib = cs; ib < ce2; ib += Sf) {
    const int ie = min(ib + Sf, ce2);
    const bool lane_in = (ib >= jlo) && (ie <= jhi);
    const bool lane_out = (ie <= jlo) || (ib >= jhi);
    const bool all_in = __all_sync(0xffffffffu, lane_in);
    const bool all_out = __all_sync(0xffffffffu, lane_out);
    if (all_out) continue;
    float cf[4][4];
    sub_phase(c, a, p, ib, ph);
    sub_amps(c, a, p, ib, cf);
    u64 s2 = f2pack(0.0f, hS);
    const ulonglong2* rec = sD + ((ib - cs) >> 1) * kPairRec;
    for (int gs = ib; gs < ie; gs += Gs) {
      const int ge = min(gs + Gs, ie);
      const double sg_m = sigma_moments(cf, ad.gmom + (size_t)(gs >> ad.lg_group) * 4);
      // would the running sum reach this lane's next target inside the group?  (margin: the per-bin and the moment sums
      // differ by FP32 rounding; a group flagged needlessly only takes the slower path)
      const bool cross = (k < k1) && (crel + sg_m * 1.0001 >= t_next);
      const bool slow = !all_in || __any_sync(0xffffffffu, cross);
      if (!slow) {
        u64 zr2 = 0, zi2 = 0;
        pairs_fast<SC>(ph, cf, s2, rec, (ge - gs) >> 1, h2, K2, zr2, zi2);
        float zrl, zrh, zil, zih;
        f2unpack(zr2, zrl, zrh); f2unpack(zi2, zil, zih);
        Zr += (double)(zrl + zrh); Zi += (double)(zil + zih);
        crel += sg_m;
      } else {
        for (int jj = gs; jj < ge; jj += 2) {
          u64 zr2 = 0, zi2 = 0, sg2 = 0;
          pair_eval<true, true, SC>(ph, cf, s2, rec, jj, jlo, jhi, h2, K2, zr2, zi2, sg2);
          float zrl, zrh, zil, zih, sgl, sgh;
          f2unpack(zr2, zrl, zrh); f2unpack(zi2, zil, zih); f2unpack(sg2, sgl, sgh);
          while (k < k1 && crel >= t_next) close_at(jj);          // e_n = first bin whose cumulative sum reached the target
          Zr += (double)zrl; Zi += (double)zil; crel += (double)sgl;
          while (k < k1 && crel >= t_next) close_at(jj + 1);
          Zr += (double)zrh; Zi += (double)zih; crel += (double)sgh;
        }
      }
    }
  }
  while (k < k1) close_at(ce);                  // targets the scanned sums place in this chunk (rounding): at its end
  const double Sg = crel - c_open;
  if (!closed_any) {
    frag[(size_t)1 * a.P_pad] = Zr; frag[(size_t)2 * a.P_pad] = Zi; frag[(size_t)3 * a.P_pad] = Sg;
    frag[(size_t)4 * a.P_pad] = 0.0; frag[(size_t)5 * a.P_pad] = 0.0; frag[(size_t)6 * a.P_pad] = 0.0;
  } else {
    frag[(size_t)4 * a.P_pad] = Zr; frag[(size_t)5 * a.P_pad] = Zi; frag[(size_t)6 * a.P_pad] = Sg;
  }
  frag[(size_t)7 * a.P_pad] = closed_any ? 1.0 : 0.0;
  frag[0] = ups;
  if (a.comp) { frag[(size_t)8 * a.P_pad] = xs; frag[(size_t)9 * a.P_pad] = hs; }
}

__global__ void k_stitch_ad(const double* __restrict__ frag, int n_chunks, int P_pad, int P, double scale,
                            double* __restrict__ out, double* __restrict__ comp3, double x_scale, double h_scale,
                            int* __restrict__ out_edges, int n_seg, int n_bins) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P) return;
  double ups = 0.0, zr = 0.0, zi = 0.0, sg = 0.0, xs = 0.0, hs = 0.0;
  auto finish = [&]() {
    if (sg > 0.0) {
      const double z2 = zr * zr + zi * zi;
      ups += z2 / sg;
      if (comp3) { xs += sqrt(z2); hs += sg; }
    }
  };
  // serial fold in chunk order (bitwise reproducible), loads of kU chunks in flight (as in k_stitch)
  constexpr int kU = 8;
  for (int c0 = 0; c0 < n_chunks; c0 += kU) {
    double v[kU][8], w8[kU], w9[kU];
#pragma unroll
    for (int u = 0; u < kU; ++u) {
      const double* f = frag + (size_t)min(c0 + u, n_chunks - 1) * kFragAd * P_pad + p;
#pragma unroll
      for (int m = 0; m < 8; ++m) v[u][m] = f[(size_t)m * P_pad];
      w8[u] = comp3 ? f[(size_t)8 * P_pad] : 0.0; w9[u] = comp3 ? f[(size_t)9 * P_pad] : 0.0;
    }
#pragma unroll
    for (int u = 0; u < kU; ++u) {
      if (c0 + u >= n_chunks) break;
      zr += v[u][1]; zi += v[u][2]; sg += v[u][3];
      if (v[u][7] != 0.0) {
        finish();
        zr = v[u][4]; zi = v[u][5]; sg = v[u][6];
      }
      ups += v[u][0];
      if (comp3) { xs += w8[u]; hs += w9[u]; }
    }
  }
  finish();                                     // the last segment closes at e_N = n_bins
  if (out) out[p] = ups * scale;
  if (comp3) { comp3[3 * (size_t)p] = ups * scale; comp3[3 * (size_t)p + 1] = xs * x_scale; comp3[3 * (size_t)p + 2] = hs * h_scale; }
  if (out_edges) { out_edges[(size_t)p * (n_seg + 1)] = 0; out_edges[(size_t)p * (n_seg + 1) + n_seg] = n_bins; }
}

// ------------------------------------------------------------------------------------------------ a6
// out[p] = Upsilon.  comp3 != nullptr: also comp3[p] = (Upsilon, X = sum_k |z_k| x_scale, H = sum_k sigma_k h_scale).
__global__ void k_stitch(const double* __restrict__ frag, const uint8_t* __restrict__ flags, int n_chunks, int P_pad,
                         int P, double scale, double* __restrict__ out, double* __restrict__ comp3, double x_scale,
                         double h_scale, const int* __restrict__ esc_count = nullptr, int esc_pb = 0,
                         const int* __restrict__ pmap = nullptr, const int* __restrict__ jlo = nullptr,
                         const int* __restrict__ jhi = nullptr, int chunk_first = 0, int chunk_len = 1,
                         const int* __restrict__ next_close = nullptr) {
  if (esc_count) P = min(P, *esc_count - esc_pb);
  // pmap != nullptr: slot p of the tables holds particle pmap[p] of the batch (window sort); all P_pad slots are visited
  for (int p = blockIdx.x * blockDim.x + threadIdx.x; p < (pmap ? P_pad : P); p += gridDim.x * blockDim.x) {
  const int q = pmap ? pmap[p] : p;
  if (q >= P) continue;
  double ups = 0.0, zr = 0.0, zi = 0.0, sg = 0.0, xs = 0.0, hs = 0.0;
  // The walk is serial per particle (fixed order = bitwise reproducible); the loads are not: the fragments of kU chunks
  // are fetched unconditionally (fields a chunk did not write are never used) before they are folded in.
  // Chunks that lie wholly outside the particle's time window hold empty fragments: only [c_lo, c_hi] is read; what
  // the skipped chunks could still do is close the piece left open at c_hi (flags are shared by all particles).
  int c_lo = 0, c_hi = n_chunks - 1;
  if (jlo) {
    const int lo = jlo[p], hi = jhi[p];
    if (hi <= lo) { c_lo = 0; c_hi = -1; }
    else {
      c_lo = max(lo / chunk_len - chunk_first, 0);
      c_hi = min((hi - 1) / chunk_len - chunk_first, n_chunks - 1);
    }
  }
  constexpr int kU = 8;
  for (int c0 = c_lo; c0 <= c_hi; c0 += kU) {
    double v[kU][7], w7[kU], w8[kU];
#pragma unroll
    for (int u = 0; u < kU; ++u) {
      const int cI = min(c0 + u, c_hi);
      const double* f = frag + (size_t)cI * kFragFields * P_pad + p;
#pragma unroll
      for (int m = 0; m < 7; ++m) v[u][m] = f[(size_t)m * P_pad];
      w7[u] = comp3 ? f[(size_t)7 * P_pad] : 0.0; w8[u] = comp3 ? f[(size_t)8 * P_pad] : 0.0;
    }
#pragma unroll
    for (int u = 0; u < kU; ++u) {
      if (c0 + u > c_hi) break;
      const uint8_t fl = flags[c0 + u];
      if (fl & CF_HEAD) {
        zr += v[u][1]; zi += v[u][2]; sg += v[u][3];
        if (fl & CF_HEAD_CLOSES) {
          if (sg > 0.0) {
            const double z2 = zr * zr + zi * zi;
            ups += z2 / sg;
            if (comp3) { xs += sqrt(z2); hs += sg; }
          }
          zr = 0.0; zi = 0.0; sg = 0.0;
        }
      }
      ups += v[u][0];
      if (comp3) { xs += w7[u]; hs += w8[u]; }
      if (fl & CF_TAIL) { zr = v[u][4]; zi = v[u][5]; sg = v[u][6]; }
    }
  }
  // the piece left open at c_hi runs on through empty chunks until one closes it (next_close, shared by all particles)
  if (sg > 0.0 && next_close && c_hi >= 0 && c_hi < n_chunks - 1 && next_close[c_hi] >= 0) {
    const double z2 = zr * zr + zi * zi;
    ups += z2 / sg;
    if (comp3) { xs += sqrt(z2); hs += sg; }
  }
  if (out) out[q] = ups * scale;
  if (comp3) { comp3[3 * (size_t)q] = ups * scale; comp3[3 * (size_t)q + 1] = xs * x_scale; comp3[3 * (size_t)q + 2] = hs * h_scale; }
  }
}

__global__ void k_stitch_seg(const double* __restrict__ frag, const uint8_t* __restrict__ flags,
                             const int* __restrict__ chunk_k0, int n_chunks, int P_pad, int P, int n_seg,
                             double sz, double ss, double* __restrict__ out_seg) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P) return;
  double zr = 0.0, zi = 0.0, sg = 0.0;
  for (int cI = 0; cI < n_chunks; ++cI) {
    const double* f = frag + (size_t)cI * kFragFields * P_pad + p;
    const uint8_t fl = flags[cI];
    if (fl & CF_HEAD) {
      zr += f[(size_t)1 * P_pad]; zi += f[(size_t)2 * P_pad]; sg += f[(size_t)3 * P_pad];
      if (fl & CF_HEAD_CLOSES) {
        double* o = out_seg + ((size_t)p * n_seg + chunk_k0[cI]) * 3;
        o[0] = zr * sz; o[1] = zi * sz; o[2] = sg * ss;
        zr = 0.0; zi = 0.0; sg = 0.0;
      }
    }
    if (fl & CF_TAIL) { zr = f[(size_t)4 * P_pad]; zi = f[(size_t)5 * P_pad]; sg = f[(size_t)6 * P_pad]; }
  }
}

// ------------------------------------------------------------------------------------------------ template generation
// h_alpha(f_j) through the same node tables and interpolants (polynomials evaluated directly instead of by
// forward differences).  One thread per (bin, template).
__global__ void k_template(DevCfg c, const int* __restrict__ node_n, const double* __restrict__ node_frac,
                           const double* __restrict__ node_amp, const int* __restrict__ jlo, const int* __restrict__ jhi,
                           int P_pad, int P, double amp_scale, double* __restrict__ hA, double* __restrict__ hE) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  const int p = blockIdx.y;
  if (j >= c.n_bins || p >= P) return;
  double2 oA = make_double2(0.0, 0.0), oE = oA;
  if (j >= jlo[p] && j < jhi[p]) {
    const int i0 = (j >> c.log2_stride) + kNodeOff;
    const double u = (double)(j - ((j >> c.log2_stride) << c.log2_stride));
    const size_t base = (size_t)i0 * P_pad + p;
    const int n0 = node_n[base];
    const double r0 = node_frac[base];
    double Y[6], b[6];
    for (int m = -2; m <= 3; ++m) {
      const size_t at = (size_t)(i0 + m) * P_pad + p;
      Y[m + 2] = (double)(node_n[at] - n0) + (node_frac[at] - r0);
    }
    quintic_coeffs(Y, 1.0 / (double)c.stride, b);
    double phi = r0 + u * (b[1] + u * (b[2] + u * (b[3] + u * (b[4] + u * b[5]))));
    phi -= rint(phi);
    double sn, cn;
    sincospi(2.0 * phi, &sn, &cn);
    const int Sf = c.stride >> 2;
    const int q = (int)u / Sf;
    const double s = (u - (double)(q * Sf)) / (double)Sf;
    double v[4];
    for (int r = 0; r < 4; ++r) {
      const double* col = node_amp + ((size_t)i0 * 4 + r) * P_pad + p;
      const ptrdiff_t st = (ptrdiff_t)4 * P_pad;
      double nd[6];
      for (int m = -2; m <= 3; ++m) nd[m + 2] = col[m * st];
      double a0, a1, a2, a3;
      fine_cubic<double>(nd, q, a0, a1, a2, a3);
      v[r] = (a0 + s * (a1 + s * (a2 + s * a3))) * amp_scale;
    }
    // h = amp * e^{-2 pi i Phi}
    oA = make_double2(v[0] * cn + v[1] * sn, v[1] * cn - v[0] * sn);
    oE = make_double2(v[2] * cn + v[3] * sn, v[3] * cn - v[2] * sn);
  }
  reinterpret_cast<double2*>(hA)[(size_t)p * c.n_bins + j] = oA;
  reinterpret_cast<double2*>(hE)[(size_t)p * c.n_bins + j] = oE;
}

// ------------------------------------------------------------------------------------------------ a7 PSO
// (1)+(2): one CTA per swarm.  label == nullptr: swarm s = particles [s per_swarm, (s+1) per_swarm); else swarm s = the
// particles with label[p] == s (n_scan = n_particles; a swarm without members gets gbest_val = -inf, gbest_pos untouched).
__global__ void k_pso_best(const double* __restrict__ pos, double* __restrict__ pbest_pos, double* __restrict__ pbest_val,
                           const double* __restrict__ stat, double* __restrict__ gbest_pos, double* __restrict__ gbest_val,
                           int per_swarm, const int* __restrict__ label, long long n_scan) {
  const int s = blockIdx.x;
  const long long p0 = label ? 0 : (long long)s * per_swarm;
  const long long n_t = label ? n_scan : per_swarm;
  double best = -INFINITY;
  long long besti = LLONG_MAX;
  bool any = false;
  for (long long t = threadIdx.x; t < n_t; t += blockDim.x) {
    const long long p = p0 + t;
    if (label && label[p] != s) continue;
    double pv = pbest_val[p];
    const double st = stat[p];
    if (st > pv) {
      pv = st;
      pbest_val[p] = st;
#pragma unroll
      for (int m = 0; m < 8; ++m) pbest_pos[p * 8 + m] = pos[p * 8 + m];
    }
    // arg max with lowest index on ties; NaN never wins; the first element seeds the comparison like a serial scan
    if (!any || pv > best) { best = pv; besti = p; any = true; }
  }
  __shared__ double sv[32];
  __shared__ long long si[32];
  __shared__ int sa[32];
  // serial-scan semantics: candidate (v, i) beats (w, j) if v > w, or (v == w or both not comparable) and i < j.
  auto better = [](double v, long long i, bool av, double w, long long j, bool aw) {
    if (!aw) return av;
    if (!av) return false;
    if (v > w) return true;
    if (w > v) return false;
    return i < j;
  };
  for (int o = 16; o > 0; o >>= 1) {
    const double ov = __shfl_xor_sync(0xffffffffu, best, o);
    const long long oi = __shfl_xor_sync(0xffffffffu, besti, o);
    const int oa = __shfl_xor_sync(0xffffffffu, (int)any, o);
    if (better(ov, oi, oa, best, besti, any)) { best = ov; besti = oi; any = oa; }
  }
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
  if (l == 0) { sv[w] = best; si[w] = besti; sa[w] = any; }
  __syncthreads();
  if (w == 0) {
    const int nw = (blockDim.x + 31) >> 5;
    best = (l < nw) ? sv[l] : -INFINITY; besti = (l < nw) ? si[l] : LLONG_MAX; any = (l < nw) ? sa[l] : false;
    for (int o = 16; o > 0; o >>= 1) {
      const double ov = __shfl_xor_sync(0xffffffffu, best, o);
      const long long oi = __shfl_xor_sync(0xffffffffu, besti, o);
      const int oa = __shfl_xor_sync(0xffffffffu, (int)any, o);
      if (better(ov, oi, oa, best, besti, any)) { best = ov; besti = oi; any = oa; }
    }
    if (l == 0) { si[0] = besti; sa[0] = any; }
  }
  __syncthreads();
  const long long bi = si[0];
  if (!sa[0]) {                                  // no members (labelled swarms only)
    if (threadIdx.x == 8) gbest_val[s] = -INFINITY;
    return;
  }
  if (threadIdx.x < 8) gbest_pos[s * 8 + threadIdx.x] = pbest_pos[bi * 8 + threadIdx.x];
  if (threadIdx.x == 8) gbest_val[s] = pbest_val[bi];
}

// (3)-(6): one thread per particle.
__global__ void k_pso_move(double* __restrict__ pos, double* __restrict__ vel, const double* __restrict__ pbest_pos,
                           const double* __restrict__ gbest_pos, const double* __restrict__ lo, const double* __restrict__ hi,
                           const double* __restrict__ eps_min, double omega, double phi_p, double phi_g,
                           uint64_t seed, uint64_t iter, long long P, int per_swarm, const int* __restrict__ label) {
  const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P) return;
  const int s = label ? label[p] : (int)(p / per_swarm);
  uint32_t w[16];
#pragma unroll
  for (uint32_t b = 0; b < 4; ++b)
    philox4x32_10((uint32_t)p, (uint32_t)iter, b, 0u, (uint32_t)seed, (uint32_t)(seed >> 32), w + 4 * b);
#pragma unroll
  for (int m = 0; m < 8; ++m) {
    const double rP = ((double)w[m] + 0.5) * 0x1p-32, rG = ((double)w[8 + m] + 0.5) * 0x1p-32;
    const double th = pos[p * 8 + m];
    // Eq. 14, same association as written: (Omega v + Phi_P r_P (Psi - theta)) + Phi_G r_G (Xi - theta), no contraction
    const double t1 = __dmul_rn(omega, vel[p * 8 + m]);
    const double t2 = __dmul_rn(__dmul_rn(phi_p, rP), __dsub_rn(pbest_pos[p * 8 + m], th));
    const double t3 = __dmul_rn(__dmul_rn(phi_g, rG), __dsub_rn(gbest_pos[s * 8 + m], th));
    const double u = __dadd_rn(__dadd_rn(t1, t2), t3);
    const double au = fabs(u), eps = eps_min[m];
    double v;
    if (au > 0.0) v = (eps > au ? eps : au) * (u / au);      // Eq. 15
    else v = (eps > 0.0) ? eps : 0.0;                        // Q9: sign(0) = +1
    double x = th + v;                                       // Eq. 13
    if (x < lo[m]) { x = lo[m]; v = -v; }                    // Q9: reflect
    else if (x > hi[m]) { x = hi[m]; v = -v; }
    pos[p * 8 + m] = x;
    vel[p * 8 + m] = v;
  }
}

// ------------------------------------------------------------------------------------------------ k-means regrouping
// Lloyd's algorithm on the particle positions in prior-box units (reading Q19).  Same arithmetic order
// as the definition: squared distance accumulated over the dimensions in order without contraction, lowest k on ties;
// centroid sums in particle order (one thread per (cluster, dimension) walks all particles: K * 8 threads, a few MB of
// L2-resident reads -- k-means runs once per rung of the ladder).
__global__ void k_km_assign(const double* __restrict__ pos, long long P, const double* __restrict__ lo,
                            const double* __restrict__ hi, const double* __restrict__ cent, int K, int* __restrict__ label,
                            int* __restrict__ changed) {
  extern __shared__ double sc_[];
  const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P) return;
  double w[8], x[8];
#pragma unroll
  for (int m = 0; m < 8; ++m) { w[m] = (hi[m] > lo[m]) ? 1.0 / (hi[m] - lo[m]) : 0.0; x[m] = pos[p * 8 + m]; }
  int bk = 0;
  double bd = INFINITY;
  for (int k = 0; k < K; ++k) {
    double d = 0.0;
#pragma unroll
    for (int m = 0; m < 8; ++m) { const double t = __dmul_rn(__dsub_rn(x[m], cent[k * 8 + m]), w[m]); d = __dadd_rn(d, __dmul_rn(t, t)); }
    if (d < bd) { bd = d; bk = k; }
  }
  if (label[p] != bk) { label[p] = bk; atomicAdd(changed, 1); }
}
__global__ void k_km_update(const double* __restrict__ pos, long long P, const int* __restrict__ label,
                            double* __restrict__ cent, long long* __restrict__ count) {
  const int k = blockIdx.x, m = threadIdx.x;
  double sum = 0.0;
  long long n = 0;
  for (long long p = 0; p < P; ++p)
    if (label[p] == k) { sum = __dadd_rn(sum, pos[p * 8 + m]); ++n; }
  if (n > 0) cent[k * 8 + m] = sum / (double)n;
  if (m == 0) count[k] = n;
}

// ------------------------------------------------------------------------------------------------ many data streams x one template
// Second workload (the 5000 noise realisations of Fig. 3): Upsilon_N of ONE template
// against many data streams that share the PSD.  The template and its sigma_k are computed once; per stream and bin
// the work is one 16-byte (FP32) or 32-byte (FP64) load and 8 multiply-adds, so this path is HBM-bound.
//   W_d(j)  = d_d(j) 4df/S(j) / s0  (whitened streams, [stream][bin][(A re, A im, E re, E im)])
//   z_k[d]  = sum_{j in segment k} W_d(j) . conj(h(j)),   sigma_k = sum_j (|h_A|^2 G_A + |h_E|^2 G_E),  Upsilon[d] = sum_k |z_k[d]|^2 / sigma_k
// Segments are cut into pieces of <= kStreamPiece bins; one warp per (piece, stream), lanes stride over the bins
// (coalesced), shuffle reduction, partial z in [piece][stream] order; k_streams_finish walks the pieces in order.
constexpr int kStreamPiece = 1024;

__global__ void k_whiten_streams_f32(const double* __restrict__ dA, const double* __restrict__ dE, const double2* __restrict__ G64,
                                     double s0, long long n_bins, long long n_streams, float4* __restrict__ W) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_bins * n_streams) return;
  const double2 g = G64[i % n_bins];
  W[i] = make_float4((float)(dA[2 * i] * g.x * s0), (float)(dA[2 * i + 1] * g.x * s0),
                     (float)(dE[2 * i] * g.y * s0), (float)(dE[2 * i + 1] * g.y * s0));
}
__global__ void k_whiten_streams_f64(const double* __restrict__ dA, const double* __restrict__ dE, const double2* __restrict__ G64,
                                     double s0, long long n_bins, long long n_streams, double4* __restrict__ W) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_bins * n_streams) return;
  const double2 g = G64[i % n_bins];
  W[i] = make_double4(dA[2 * i] * g.x * s0, dA[2 * i + 1] * g.x * s0, dE[2 * i] * g.y * s0, dE[2 * i + 1] * g.y * s0);
}
// template of the streams path: (h_A re, im, h_E re, im) in FP64 and FP32, from the k_template output
__global__ void k_streams_template(const double* __restrict__ hA, const double* __restrict__ hE, int n_bins,
                                   double4* __restrict__ T64, float4* __restrict__ T32) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n_bins) return;
  const double4 t = make_double4(hA[2 * j], hA[2 * j + 1], hE[2 * j], hE[2 * j + 1]);
  T64[j] = t;
  T32[j] = make_float4((float)t.x, (float)t.y, (float)t.z, (float)t.w);
}
// sigma of every piece (template only): one warp per piece, fixed-order reduction
__global__ void k_streams_sigma(const double4* __restrict__ T64, const double2* __restrict__ G64, const int* __restrict__ piece_lo,
                                const int* __restrict__ piece_hi, int n_pieces, double* __restrict__ piece_sigma) {
  const int piece = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (piece >= n_pieces) return;
  const int lane = threadIdx.x & 31;
  double acc = 0.0;
  for (int j = piece_lo[piece] + lane; j < piece_hi[piece]; j += 32) {
    const double4 t = T64[j]; const double2 g = G64[j];
    acc += (t.x * t.x + t.y * t.y) * g.x + (t.z * t.z + t.w * t.w) * g.y;
  }
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (lane == 0) piece_sigma[piece] = acc;
}
// streaming (evict-first) loads: every stream byte is read exactly once
__device__ __forceinline__ float4 ld_stream(const float4* p) { return __ldcs(p); }
__device__ __forceinline__ double4 ld_stream(const double4* p) {
  const double2 a = __ldcs(reinterpret_cast<const double2*>(p)), b = __ldcs(reinterpret_cast<const double2*>(p) + 1);
  return make_double4(a.x, a.y, b.x, b.y);
}
template <typename W4, typename R>
__global__ void __launch_bounds__(256) k_streams_z(const W4* __restrict__ W, const W4* __restrict__ T, const int* __restrict__ piece_lo,
                                                   const int* __restrict__ piece_hi, int n_pieces, long long n_bins, int n_streams,
                                                   double2* __restrict__ zpart /* [n_pieces][n_streams] */) {
  const int piece = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (piece >= n_pieces) return;
  const int d = blockIdx.y;
  const int lane = threadIdx.x & 31;
  const W4* __restrict__ Wd = W + (size_t)d * n_bins;
  const int lo = piece_lo[piece], hi = piece_hi[piece];
  R zr0 = 0, zi0 = 0, zr1 = 0, zi1 = 0;
  int j = lo + lane;
  for (; j + 32 < hi; j += 64) {                      // two independent loads in flight per lane
    const W4 w0 = ld_stream(Wd + j), w1 = ld_stream(Wd + j + 32);
    const W4 t0 = T[j], t1 = T[j + 32];
    zr0 += w0.x * t0.x + w0.y * t0.y + w0.z * t0.z + w0.w * t0.w;     // Re (w conj t)
    zi0 += w0.y * t0.x - w0.x * t0.y + w0.w * t0.z - w0.z * t0.w;     // Im (w conj t)
    zr1 += w1.x * t1.x + w1.y * t1.y + w1.z * t1.z + w1.w * t1.w;
    zi1 += w1.y * t1.x - w1.x * t1.y + w1.w * t1.z - w1.z * t1.w;
  }
  if (j < hi) {
    const W4 w0 = ld_stream(Wd + j); const W4 t0 = T[j];
    zr0 += w0.x * t0.x + w0.y * t0.y + w0.z * t0.z + w0.w * t0.w;
    zi0 += w0.y * t0.x - w0.x * t0.y + w0.w * t0.z - w0.z * t0.w;
  }
  double zr = (double)zr0 + (double)zr1, zi = (double)zi0 + (double)zi1;
  for (int o = 16; o > 0; o >>= 1) { zr += __shfl_xor_sync(0xffffffffu, zr, o); zi += __shfl_xor_sync(0xffffffffu, zi, o); }
  if (lane == 0) zpart[(size_t)piece * n_streams + d] = make_double2(zr, zi);
}
__global__ void k_streams_finish(const double2* __restrict__ zpart, const double* __restrict__ piece_sigma,
                                 const int* __restrict__ piece_last /* 1 = last piece of its segment */, int n_pieces,
                                 int n_streams, double* __restrict__ out) {
  const int d = blockIdx.x * blockDim.x + threadIdx.x;
  if (d >= n_streams) return;
  double ups = 0.0, zr = 0.0, zi = 0.0, sg = 0.0;
  for (int i = 0; i < n_pieces; ++i) {
    const double2 z = zpart[(size_t)i * n_streams + d];
    zr += z.x; zi += z.y; sg += piece_sigma[i];
    if (piece_last[i]) {
      if (sg > 0.0) ups += (zr * zr + zi * zi) / sg;
      zr = 0.0; zi = 0.0; sg = 0.0;
    }
  }
  out[d] = ups;
}

// ------------------------------------------------------------------------------------------------ MUFU gain
// The hardware sin/cos (MUFU) used by the fast FP32 path has a small systematic gain: <cos^2 + sin^2> over uniformly
// distributed angles is not exactly 1.  It is measured once per handle with the very instruction sequence of the
// dense kernel (2^20 equispaced angles, fixed-order reduction => deterministic) and divided out of Upsilon.
// ------------------------------------------------------------------------------------------------ window sort
// Lanes of a warp are particles; a warp works on a fine sub-interval as soon as ONE of its particles' time windows
// (Q4) overlaps it.  Where the windows cover only part of the band (c5: ~25 %) particles in input order waste most of the
// lanes, so each batch is processed in the order of the window starts j_lo (stable radix sort of (j_lo, index)):
// k_gather_sorted re-orders the per-particle constants and windows, k_stitch scatters through the same map.
__global__ void k_iota(int* __restrict__ v, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) v[i] = i;
}
__global__ void k_gather_sorted(const int* __restrict__ map, int P_pad, const double* __restrict__ pc_u,
                                const int* __restrict__ jlo_u, const int* __restrict__ jhi_u, double* __restrict__ pc,
                                int* __restrict__ jlo, int* __restrict__ jhi) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P_pad) return;
  const int q = map[p];
#pragma unroll
  for (int f = 0; f < kPcFields; ++f) pc[(size_t)f * P_pad + p] = pc_u[(size_t)f * P_pad + q];
  jlo[p] = jlo_u[q]; jhi[p] = jhi_u[q];
}

// ------------------------------------------------------------------------------------------------ escalation
// Particles whose FP32-path statistic is below tau (0 < Upsilon < tau): ascending index list, count and gathered
// parameter rows.  One CTA of 1024 threads scans the population in order (deterministic).
__global__ void __launch_bounds__(1024) k_esc_select(const double* __restrict__ ups, const double* __restrict__ params, int P,
                                                     double tau, int* __restrict__ idx, int* __restrict__ count,
                                                     double* __restrict__ params_c) {
  __shared__ int wsum[32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  int base = 0;
  for (int t0 = 0; t0 < P; t0 += 1024) {
    const int p = t0 + threadIdx.x;
    const double u = (p < P) ? ups[p] : 0.0;
    const bool f = (u > 0.0) && (u < tau);
    const unsigned b = __ballot_sync(0xffffffffu, f);
    if (lane == 0) wsum[w] = __popc(b);
    __syncthreads();
    int off = 0, tot = 0;
#pragma unroll
    for (int i = 0; i < 32; ++i) { const int v = wsum[i]; off += (i < w) ? v : 0; tot += v; }
    if (f) {
      const int at = base + off + __popc(b & ((1u << lane) - 1u));
      idx[at] = p;
#pragma unroll
      for (int i = 0; i < 8; ++i) params_c[(size_t)at * 8 + i] = params[(size_t)p * 8 + i];
    }
    base += tot;
    __syncthreads();
  }
  if (threadIdx.x == 0) *count = base;
}
__global__ void k_esc_scatter(const int* __restrict__ idx, const int* __restrict__ count, const double* __restrict__ ups_c,
                              double* __restrict__ ups) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < *count) ups[idx[i]] = ups_c[i];
}

// gbest_val[s] = re-evaluated value, except for empty swarms (-inf stays)
__global__ void k_keep_empty(double* __restrict__ gbest_val, const double* __restrict__ re, int S) {
  const int s = threadIdx.x;
  if (s < S && gbest_val[s] != -INFINITY) gbest_val[s] = re[s];
}

__global__ void k_mufu_gain(double* __restrict__ out) {
  __shared__ double sh[1024];
  double acc = 0.0;
  for (int i = 0; i < 1024; ++i) {
    const int n = (int)(((unsigned)(i * 1024 + threadIdx.x) << 12) + 2048u);
    const float xr = (float)n * 1.4629180792671596e-09f;
    const float cr = __cosf(xr), sr = __sinf(xr);
    acc += (double)cr * (double)cr + (double)sr * (double)sr;
  }
  sh[threadIdx.x] = acc;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) {
    if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) out[0] = sh[0] / 1048576.0;
}

// ------------------------------------------------------------------------------------------------ peaks
// FP64 FMA throughput probe for the roofline denominator: 8 independent DFMA chains per thread.
__global__ void k_dfma_peak(double* __restrict__ out, int iters, double a, double b) {
  double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
  for (int i = 0; i < iters; ++i) {
    x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
    x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

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
};

struct sc_handle : EdgeCache {
  sc_config cfg;
  DevCfg dc;
  int device = 0;
  double s0 = 1.0;                 // weight scale (power of two)
  float4* D32 = nullptr; double4* W64 = nullptr; double2* G64 = nullptr;   // D32: bin-pair layout of k_dense2
  // options
  int precision = 0; int f32_min_seg = 8; size_t scratch_cap = (size_t)8 << 30;
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
  // scratch
  void* scratch = nullptr; size_t scratch_bytes = 0;
  unsigned long long* d_counter = nullptr;
  double* d_params_stage = nullptr; double* d_out_stage = nullptr; size_t stage_cap = 0;
  long long launches = 0;
  EdgeCache alt;                   // see EdgeCache
  // escalation: particles whose FP32-path Upsilon is below the mode's threshold are re-evaluated
  // by the all-FP64 path; compacted index list, count, gathered parameters and their results
  int escalate = 1; double esc_tau_poly = 6.0, esc_tau_mufu = 16.0;
  int* d_esc_idx = nullptr; int* d_esc_count = nullptr; double* d_esc_params = nullptr; double* d_esc_out = nullptr;
  size_t esc_idx_cap = 0, esc_cnt_cap = 0, esc_par_cap = 0, esc_out_cap = 0; int* h_esc_hint = nullptr;
  int window_sort = 1; void* d_sort_tmp = nullptr; size_t sort_cap = 0;   // cub radix-sort workspace of the window sort
  // three-channel handles (A, E, T): the T channel lives in a second handle whose first slot carries T (chan_set = 1)
  // and whose second slot is empty; the per-segment sums of both are added before |z|^2/sigma is formed
  sc_handle* sub = nullptr; double* d_seg3 = nullptr; size_t seg3_cap = 0;
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

// Node spacing per precision mode: the all-FP64 path (N_seg < 8, where 1e-8 rad matters)
// keeps the nodes <= 2 days of signal time apart, the FP32-amplitude path (error floor ~1e-8 relative) <= 4 days.
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
int pick_stride_log2(const sc_config& cfg, double tc_max_s, int forced, double max_days) {
  if (forced > 0) return std::min(std::max(forced, 3), 12);
  const double f_lo = (double)std::max<int64_t>(cfg.j0, 1) / cfg.T_obs_s;
  const double s_per_bin = (8.0 / 3.0) * tc_max_s / (f_lo * cfg.T_obs_s);
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
                cudaStream_t st, bool seg_mode, const int* esc_count = nullptr, int esc_blocks = 0) {
  // esc_count != nullptr: the escalation pass -- P is an upper bound, the number of particles sits on the device;
  // its launches are timed as SC_TIME_ESC and do not count evaluated bins twice
  const int cls_nodes = esc_count ? SC_TIME_ESC : SC_TIME_NODES, cls_dense = esc_count ? SC_TIME_ESC : SC_TIME_DENSE,
            cls_stitch = esc_count ? SC_TIME_ESC : SC_TIME_STITCH;
  const int n_seg = (int)h->edges.size() - 1;
  DevCfg dc = h->dc;
  apply_stride(dc, sizeof(R) == 4 ? h->lg_f32 : h->lg_f64);
  const int n_nodes = dc.n_nodes;
  const int n_chunks = h->n_chunks;
  // per-particle scratch bytes
  const size_t per_p = 2 * ((size_t)kPcFields * 8 + 8) /* constants, jlo, jhi: unsorted + sorted */ + 16 /* sort keys, map */
                       + (size_t)n_nodes * (4 + 8 + 4 * sizeof(R)) + (size_t)std::max(n_chunks, 1) * kFragFields * 8;
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
  R* node_amp = (R*)take((size_t)n_nodes * 4 * sizeof(R) * P_pad);
  double* frag = (double*)take((size_t)std::max(n_chunks, 1) * kFragFields * 8 * P_pad);
  // window sort (see k_gather_sorted): not in the segment-table mode (rows are addressed by particle) nor in the
  // escalation pass (few particles, count on the device)
  const bool sorted = h->window_sort && !seg_mode && !esc_count && P_pad > kBlock;
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
  const double sz = h->s0 * h0 / four_df, ss = h->s0 * h->s0 * h0 * h0 / four_df;

  // particle blocks launched per kernel: all of them, or (escalation pass) the caller's estimate -- the kernels stride
  const int pblocks = esc_count ? std::max(1, std::min(esc_blocks, P_pad / kBlock)) : P_pad / kBlock;
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
      if (cub::DeviceRadixSort::SortPairs(h->d_sort_tmp, sort_bytes, jlo_u, key_s, iota, pmap, P_pad, 0, 32, st) != cudaSuccess)
        return fail(h, SC_ERR_CUDA, "cub::DeviceRadixSort::SortPairs failed");
      h->launches += 3;
      k_gather_sorted<<<(P_pad + 127) / 128, 128, 0, st>>>(pmap, P_pad, pc_u, jlo_u, jhi_u, pc, jlo, jhi);
      if ((rc = check_launch(h, "k_gather_sorted"))) return rc;
    }
    if (n_chunks == 0) {
      if (!seg_mode && out) SC_CUDA(h, cudaMemsetAsync(out + pb, 0, (size_t)Pn * 8, st));
      if (out_comp) SC_CUDA(h, cudaMemsetAsync(out_comp + pb * 3, 0, (size_t)Pn * 24, st));
      continue;
    }
    {
      Timed tm(h, st, cls_nodes);
      if (esc_count) k_nodes<R, true><<<dim3((n_nodes + kNodesPerCta - 1) / kNodesPerCta, pblocks), 128, 0, st>>>(dc, pc, jlo, jhi, P_pad, node_n, node_frac, node_amp, esc_count, (int)pb);
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
    const dim3 grid(n_chunks, pblocks);
    {
      Timed tm(h, st, cls_dense);
      if (sizeof(R) == 4) {
        const ulonglong2* Dp = reinterpret_cast<const ulonglong2*>(h->D32);
        if (seg_mode) k_dense2<true, 0><<<grid, kBlock, 0, st>>>(dc, a, Dp);
        else if (sincos == 2) k_dense2<false, 2><<<grid, kBlock, 0, st>>>(dc, a, Dp);
        else k_dense2<false, 0><<<grid, kBlock, 0, st>>>(dc, a, Dp);
      } else {
        if (seg_mode) k_dense<true><<<grid, kBlock, 0, st>>>(dc, a, h->W64, h->G64);
        else if (esc_count) k_dense<false, true><<<grid, kBlock, 0, st>>>(dc, a, h->W64, h->G64);
        else k_dense<false><<<grid, kBlock, 0, st>>>(dc, a, h->W64, h->G64);
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
      k_stitch<<<esc_count ? pblocks : ((sorted ? P_pad : Pn) + 127) / 128, 128, 0, st>>>(frag, h->d_flags, n_chunks, P_pad, Pn, 1.0 / g2, out ? out + pb : nullptr,
                                                 out_comp ? out_comp + pb * 3 : nullptr, h->s0 * h0 / sqrt(g2),
                                                 h->s0 * h->s0 * h0 * h0, esc_count, (int)pb, sorted ? pmap : nullptr,
                                                 jlo, jhi, h->chunk_first, sizeof(R) == 4 ? kChunkF32 : kChunkF64, h->d_next_close);
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
  SC_CUDA(h, cudaMemcpyAsync(h->d_piece_first, first.data(), first.size() * 4, cudaMemcpyHostToDevice, st));
  if (h->n_pieces > 0) {
    SC_CUDA(h, cudaMemcpyAsync(h->d_piece_lo, lo.data(), lo.size() * 4, cudaMemcpyHostToDevice, st));
    SC_CUDA(h, cudaMemcpyAsync(h->d_piece_hi, hi.data(), hi.size() * 4, cudaMemcpyHostToDevice, st));
    SC_CUDA(h, cudaStreamSynchronize(st));       // the host vectors go out of scope
    Timed tm(h, st, SC_TIME_OTHER);
    k_moments<<<(h->n_pieces + 127) / 128, 128, 0, st>>>(h->G64, h->d_piece_lo, h->d_piece_hi, h->n_pieces, (int)h->cfg.n_bins,
                                                        lg_fine, h->d_moments);
    if ((rc = check_launch(h, "k_moments"))) return rc;
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
  int rc;
  if (lg_fine > 0 && (rc = build_pieces(h, CH, lg_fine, st))) { h->cached_chunk = 0; return rc; }
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
}

int eval_common(sc_handle* h, const double* params, int64_t P, const int32_t* seg_edges, int32_t n_seg,
                double* out, double* out_seg, void* stream, bool seg_mode, double* out_comp = nullptr) {
  if (!h) return SC_ERR_NOT_INIT;
  if (h->cuda_failed) return SC_ERR_CUDA;
  if (!params || P <= 0 || (!seg_mode && !out && !out_comp) || (seg_mode && !out_seg))
    return fail(h, SC_ERR_INVALID_ARG, "null pointer or n_particles <= 0");
  cudaStream_t st = (cudaStream_t)stream;
  const bool f64 = (h->precision == 2) || (h->precision == 0 && n_seg < h->f32_min_seg);
  int rc = prepare_edges(h, seg_edges, n_seg, f64 ? kChunkF64 : kChunkF32, f64 ? 0 : h->lg_f32 - 2, st);
  if (rc) return rc;
  SC_CUDA(h, cudaMemsetAsync(h->d_counter, 0, 8, st));
  if (seg_mode) SC_CUDA(h, cudaMemsetAsync(out_seg, 0, (size_t)P * n_seg * 3 * 8, st));
  if (f64) return run_batches<double>(h, params, P, out, out_seg, out_comp, st, seg_mode);
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
      k_esc_select<<<1, 1024, 0, st>>>(out, params, (int)P, mufu ? h->esc_tau_mufu : h->esc_tau_poly, h->d_esc_idx,
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
    rc = prepare_edges(h, e_host.data(), n_seg, kChunkF64, 0, st);
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
  // batches of particles such that the two segment tables fit in 2 GiB
  const size_t per_p = (size_t)n_seg * 24;
  int64_t Pb = (int64_t)std::max<size_t>(1, ((size_t)1 << 30) / per_p);
  Pb = std::min<int64_t>(Pb, P);
  int rc = grow(h, (void**)&h->d_seg3, &h->seg3_cap, 2 * per_p * (size_t)Pb);
  if (rc) return rc;
  double* segA = h->d_seg3; double* segT = segA + (size_t)Pb * n_seg * 3;
  const double four_df = 4.0 / h->cfg.T_obs_s;
  for (int64_t pb = 0; pb < P; pb += Pb) {
    const int64_t Pn = std::min<int64_t>(Pb, P - pb);
    if ((rc = eval_common(h, params + pb * 8, Pn, seg_edges, n_seg, nullptr, segA, stream, true))) return rc;
    if ((rc = eval_common(h->sub, params + pb * 8, Pn, seg_edges, n_seg, nullptr, segT, stream, true))) {
      fail(h, rc, "T pass: %s", h->sub->err.c_str());
      return rc;
    }
    Timed tm(h, st, SC_TIME_STITCH);
    k_combine3<<<(unsigned)((Pn + 127) / 128), 128, 0, st>>>(segA, segT, (int)Pn, n_seg, four_df, out ? out + pb : nullptr,
                                                            seg_mode ? out_seg + (size_t)pb * n_seg * 3 : nullptr,
                                                            out_comp ? out_comp + pb * 3 : nullptr);
    if ((rc = check_launch(h, "k_combine3"))) return rc;
  }
  return SC_OK;
}

// Per-particle equal-SNR^2 segments: see the kernels above.  FP32-amplitude path.
int run_adaptive(sc_handle* h, const double* params, int64_t P, int n_seg, double* out, int32_t* out_edges, double* out_comp,
                 cudaStream_t st) {
  DevCfg dc = h->dc;
  apply_stride(dc, h->lg_f32);
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
    Timed tm(h, st, SC_TIME_OTHER);
    k_moments<<<(n_groups + 127) / 128, 128, 0, st>>>(h->G64, nullptr, (const int*)(size_t)lg_group, n_groups, dc.n_bins, lg_fine, h->d_gmom);
    if ((rc = check_launch(h, "k_moments"))) return rc;
    k_moments<<<(n_sub + 127) / 128, 128, 0, st>>>(h->G64, nullptr, (const int*)(size_t)lg_fine, n_sub, dc.n_bins, lg_fine, h->d_smom);
    if ((rc = check_launch(h, "k_moments"))) return rc;
    h->ad_lg = dc.log2_stride;
  }
  const size_t per_p = (size_t)kPcFields * 8 + 8 + (size_t)n_nodes * (4 + 8 + 4 * sizeof(float))
                       + (size_t)(n_chunks + 1) * 8 + (size_t)n_chunks * kFragAd * 8;
  int64_t Pb_max = (int64_t)(h->scratch_cap / per_p) / kBlock * kBlock;
  if (Pb_max < kBlock) Pb_max = kBlock;
  const int64_t P_round = (P + kBlock - 1) / kBlock * kBlock;
  const int P_pad = (int)std::min<int64_t>(Pb_max, P_round);
  if ((rc = grow(h, &h->scratch, &h->scratch_bytes, per_p * (size_t)P_pad + 2048))) return rc;
  char* base = (char*)h->scratch;
  auto take = [&](size_t bytes) { char* r = base; base += (bytes + 255) / 256 * 256; return r; };
  double* pc = (double*)take((size_t)kPcFields * 8 * P_pad);
  int* jlo = (int*)take((size_t)4 * P_pad);
  int* jhi = (int*)take((size_t)4 * P_pad);
  int* node_n = (int*)take((size_t)n_nodes * 4 * P_pad);
  double* node_frac = (double*)take((size_t)n_nodes * 8 * P_pad);
  float* node_amp = (float*)take((size_t)n_nodes * 4 * sizeof(float) * P_pad);
  double* cbase = (double*)take((size_t)(n_chunks + 1) * 8 * P_pad);
  double* frag = (double*)take((size_t)n_chunks * kFragAd * 8 * P_pad);
  (void)base;

  const double four_df = 4.0 / h->cfg.T_obs_s;
  const int sincos = (h->sincos_mode == 0) ? (n_seg >= h->mufu_min_seg ? 2 : 0) : (h->sincos_mode == 2 ? 2 : 0);
  const double h0 = pow(dc.f_amp_ref, -7.0 / 6.0);
  (void)four_df;
  if (out_edges) SC_CUDA(h, cudaMemsetAsync(out_edges, 0, (size_t)P * (n_seg + 1) * 4, st));

  for (int64_t pb = 0; pb < P; pb += P_pad) {
    const int Pn = (int)std::min<int64_t>(P_pad, P - pb);
    {
      Timed tm(h, st, SC_TIME_NODES);
      k_particle_consts<<<(P_pad + 127) / 128, 128, 0, st>>>(dc, params + pb * 8, Pn, P_pad, pc, jlo, jhi, 0, dc.n_bins, h->d_counter);
    }
    if ((rc = check_launch(h, "k_particle_consts"))) return rc;
    {
      Timed tm(h, st, SC_TIME_NODES);
      k_nodes<float><<<dim3((n_nodes + kNodesPerCta - 1) / kNodesPerCta, (P_pad + 127) / 128), 128, 0, st>>>(dc, pc, jlo, jhi, P_pad, node_n, node_frac, node_amp);
    }
    if ((rc = check_launch(h, "k_nodes"))) return rc;
    DenseArgs a = {};
    a.node_n = node_n; a.node_frac = node_frac; a.node_amp = node_amp; a.jlo = jlo; a.jhi = jhi; a.P_pad = P_pad;
    a.frag = frag; a.P = Pn; a.comp = out_comp ? 1 : 0; a.n_seg = n_seg;
    AdaptArgs ad = {};
    ad.n_seg = n_seg; ad.n_chunks = n_chunks; ad.cbase = cbase; ad.chunk_sigma = cbase;
    ad.gmom = reinterpret_cast<const ulonglong2*>(h->d_gmom); ad.smom = reinterpret_cast<const ulonglong2*>(h->d_smom);
    ad.lg_group = lg_group;
    ad.out_edges = out_edges ? out_edges + (size_t)pb * (n_seg + 1) : nullptr;
    const dim3 grid(n_chunks, P_pad / kBlock);
    {
      Timed tm(h, st, SC_TIME_OTHER);
      k_sigma_chunks<<<grid, kBlock, 0, st>>>(dc, a, ad, h->D32);
      if ((rc = check_launch(h, "k_sigma_chunks"))) return rc;
      k_scan_chunks<<<(P_pad + 127) / 128, 128, 0, st>>>(cbase, n_chunks, P_pad);
      if ((rc = check_launch(h, "k_scan_chunks"))) return rc;
    }
    {
      Timed tm(h, st, SC_TIME_DENSE);
      const ulonglong2* Dp = reinterpret_cast<const ulonglong2*>(h->D32);
      if (sincos == 2) k_dense2_ad<2><<<grid, kBlock, 0, st>>>(dc, a, ad, Dp);
      else k_dense2_ad<0><<<grid, kBlock, 0, st>>>(dc, a, ad, Dp);
    }
    if ((rc = check_launch(h, "k_dense2_ad"))) return rc;
    Timed tm2(h, st, SC_TIME_STITCH);
    const double g2 = (sincos == 2) ? h->mufu_gain2 : 1.0;
    k_stitch_ad<<<(Pn + 127) / 128, 128, 0, st>>>(frag, n_chunks, P_pad, Pn, 1.0 / g2, out ? out + pb : nullptr,
                                                  out_comp ? out_comp + pb * 3 : nullptr, h->s0 * h0 / sqrt(g2),
                                                  h->s0 * h->s0 * h0 * h0, ad.out_edges, n_seg, dc.n_bins);
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
  const int n_pairs_pad = (n + kChunkF32 - 1) / kChunkF32 * (kChunkF32 / 2);
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
  if (h->sub && n_seg > 1) return fail(h, SC_ERR_INVALID_ARG, "per-particle segments are not available on three-channel handles");
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
  if (h->sub && sc->adaptive_edges) return fail(h, SC_ERR_INVALID_ARG, "per-particle segments are not available on three-channel handles");
  cudaStream_t st = (cudaStream_t)stream;
  const int S = n_swarms;
  const int64_t nb = h->cfg.n_bins;
  // device state owned by this call
  double* buf = nullptr;
  const size_t n_d = (size_t)P * 8 + (size_t)P * 2 + (size_t)S * 8 * 2 + (size_t)S + 8;
  SC_CUDA(h, cudaMalloc(&buf, n_d * 8 + (size_t)S * 8));
  double* pbest_pos = buf; double* pbest_val = pbest_pos + (size_t)P * 8; double* stat = pbest_val + P;
  double* gbest_pos = stat + P; double* cent = gbest_pos + (size_t)S * 8; double* gbest_val = cent + (size_t)S * 8;
  double* eps_d = gbest_val + S;
  long long* cnt_d = (long long*)(eps_d + 8);
  std::vector<double> gv((size_t)S), hst;
  std::vector<int64_t> cnt((size_t)S, 0);
  std::vector<int32_t> e;
  int rc = SC_OK;
  uint64_t iter_global = 0;
  // ranking precision (sc_search_config): force the FP32-amplitude path without escalation for the whole search
  const int saved_precision = h->precision, saved_escalate = h->escalate;
  if (sc->ranking_precision) { h->precision = 1; h->escalate = 0; }
  auto cleanup = [&](int code) { h->precision = saved_precision; h->escalate = saved_escalate; cudaFree(buf); return code; };
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
    int it = 0;
    for (; it < sc->max_iters_per_rung; ++it) {
      if (sc->adaptive_edges && N > 1) rc = sc_eval_stat_adaptive(h, pos, P, N, stat, nullptr, nullptr, stream);
      else rc = eval_any(h, pos, P, e.data(), N, stat, nullptr, stream, false);
      if (rc) return cleanup(rc);
      rc = sc_pso_step_labeled(h, pos, vel, pbest_pos, pbest_val, stat, gbest_pos, gbest_val, label, lo, hi, eps_d,
                               sc->omega[r], sc->phi_p[r], sc->phi_g[r], sc->seed, iter_global++, P, S, stream);
      if (rc) return cleanup(rc);
      SC_S(cudaMemcpyAsync(gv.data(), gbest_val, (size_t)S * 8, cudaMemcpyDeviceToHost, st));
      SC_S(cudaStreamSynchronize(st));
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
    h->precision = 2;
    if (sc->adaptive_edges && N > 1) rc = sc_eval_stat_adaptive(h, gbest_pos, S, N, stat, nullptr, nullptr, stream);
    else rc = eval_any(h, gbest_pos, S, e.data(), N, stat, nullptr, stream, false);
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
  cudaFree(h->D32); cudaFree(h->W64); cudaFree(h->G64);
  cudaFree(h->scratch); cudaFree(h->d_edges); cudaFree(h->d_chunk_k0); cudaFree(h->d_flags);
  cudaFree(h->d_counter); cudaFree(h->d_params_stage); cudaFree(h->d_comp); cudaFree(h->d_km); cudaFree(h->d_T64); cudaFree(h->d_T32); cudaFree(h->d_sp);
  cudaFree(h->d_spsig); cudaFree(h->d_zpart); cudaFree(h->d_hh); cudaFree(h->d_gmom); cudaFree(h->d_smom);
  cudaFree(h->d_piece_first); cudaFree(h->d_piece_lo); cudaFree(h->d_piece_hi); cudaFree(h->d_moments);
  cudaFree(h->alt.d_edges); cudaFree(h->alt.d_chunk_k0); cudaFree(h->alt.d_flags); cudaFree(h->alt.d_next_close); cudaFree(h->d_next_close);
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
