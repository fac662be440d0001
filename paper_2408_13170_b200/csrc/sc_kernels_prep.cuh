// sc_kernels_prep.cuh -- a0 whitening, a1 + a3 per-particle constants and time window, a2 coarse nodes.
// Part of libscstat.so (one translation unit: sc_stat.cu includes the kernel files in pipeline order).
#pragma once
#include "sc_common.cuh"

namespace {

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
        const int j_first = (c.j0 == 0) ? 1 : 0;   // (f = 0 carries no template: t(f) diverges there)
        int lo = j_first, hi = c.n_bins;  // first j with t(f_j) >= 0
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
        // The bisection assumes t(f) increasing over the band (true for the PN terms; the leading eccentric term can
        // break it for large e_0 or far below f_ref_ecc).  Probe the window: t must increase from its first to its last
        // bin through seven interior bins, all inside [0, T_obs]; a particle that fails has no contiguous window and is
        // treated as invalid input (Upsilon = 0, include/sc_stat.h).
        if (jhi > jlo + 1) {
          double t_prev = tf_direct(c, q, (double)(c.j0 + jlo) / c.T_obs);
          bool mono = (t_prev >= 0.0);
          for (int s = 1; s <= 8 && mono; ++s) {
            const int j = jlo + (int)(((long long)(jhi - 1 - jlo) * s) / 8);
            const double t = tf_direct(c, q, (double)(c.j0 + j) / c.T_obs);
            mono = (t >= t_prev) && (t <= c.T_obs);
            t_prev = t;
          }
          if (!mono) { jlo = 0; jhi = 0; }
        }
      } else {
        jlo = (c.j0 == 0) ? 1 : 0; jhi = c.n_bins;
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
#ifndef SC_NODES_MINB
#define SC_NODES_MINB 4   /* CTAs per SM: 128 registers instead of 143 at 3 (same 40 B of spills) -- the kernel is FP64-latency bound;
                             c3 0.63 -> 0.57 ms, c5 1.36 -> 1.18 ms; 5 CTAs / 96 registers the same */
#endif
template <typename R, bool ESC = false, int NA = 4 /* amplitude fields per node: 4 = (A, E) or (T, 0); 6 = (A, E, T) */>
__global__ void __launch_bounds__(128, SC_NODES_MINB) k_nodes(DevCfg c, const double* __restrict__ pc, const int* __restrict__ jlo, const int* __restrict__ jhi,
                        int P_pad, int* __restrict__ node_n, double* __restrict__ node_frac,
                        R* __restrict__ node_amp /* [node][NA][P_pad] */, const int* __restrict__ esc_count = nullptr,
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
    // it at all (with the batch sorted by window centre that is most of the table when the windows are short)
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
        R* a = node_amp + (size_t)i * NA * P_pad + p;
        a[0] = (R)o.Ar; a[(size_t)P_pad] = (R)o.Ai; a[2 * (size_t)P_pad] = (R)o.Er; a[3 * (size_t)P_pad] = (R)o.Ei;
        if (NA == 6) { a[4 * (size_t)P_pad] = (R)o.Tr; a[5 * (size_t)P_pad] = (R)o.Ti; }
      }
    }
    if (!ESC) return;
  }
}

}  // namespace
