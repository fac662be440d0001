// sc_kernels_misc.cuh -- MUFU gain calibration, window sort, escalation selection, FP64 peak probe.
// Part of libscstat.so (one translation unit: sc_stat.cu includes the kernel files in pipeline order).
#pragma once
#include "sc_common.cuh"

namespace {

// ------------------------------------------------------------------------------------------------ MUFU gain
// The hardware sin/cos (MUFU) used by the fast FP32 path has a small systematic gain: <cos^2 + sin^2> over uniformly
// distributed angles is not exactly 1.  It is measured once per handle with the very instruction sequence of the
// dense kernel (2^20 equispaced angles, fixed-order reduction => deterministic) and divided out of Upsilon.
// ------------------------------------------------------------------------------------------------ window sort
// Lanes of a warp are particles; a warp works on a fine sub-interval as soon as ONE of its particles' time windows
// (Q4) overlaps it.  Where the windows cover only part of the band (c5: ~25 %) particles in input order waste most of the
// lanes, so each batch is processed in the order of the window centres j_lo + j_hi (stable radix sort of (key, index)):
// k_gather_sorted re-orders the per-particle constants and windows, k_stitch scatters through the same map.
// Why the centre and not the start: the windows differ in length as well as in position (two degrees of freedom, M_c and
// t_c); neighbours in j_lo share their starts but not their ends, neighbours in the centre differ by half the length
// spread at either end.  On c5 the sub-intervals a warp walks with some lane outside its window drop from 27 % to 2 %.
__global__ void k_iota(int* __restrict__ v, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) v[i] = i;
}
// Escalation pass (esc_count != nullptr): only the first *esc_count - esc_pb slots of the unsorted arrays were written; the
// others get the largest key (they sort to the end, stable) and an empty window.
__global__ void k_sort_key(const int* __restrict__ jlo_u, const int* __restrict__ jhi_u, int* __restrict__ key, int n,
                           const int* __restrict__ esc_count = nullptr, int esc_pb = 0) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const bool live = !esc_count || i < *esc_count - esc_pb;
  key[i] = live ? (jlo_u[i] >> 1) + (jhi_u[i] >> 1) : INT_MAX;  // the centre (no overflow for n_bins < 2^31)
}
__global__ void k_gather_sorted(const int* __restrict__ map, int P_pad, const double* __restrict__ pc_u,
                                const int* __restrict__ jlo_u, const int* __restrict__ jhi_u, double* __restrict__ pc,
                                int* __restrict__ jlo, int* __restrict__ jhi, const int* __restrict__ esc_count = nullptr,
                                int esc_pb = 0) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P_pad) return;
  const int q = map[p];
  if (esc_count && q >= *esc_count - esc_pb) { jlo[p] = 0; jhi[p] = 0; return; }
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

}  // namespace
