// sc_kernels_streams.cuh -- second workload: many data streams x one template (Fig. 3).
// Part of libscstat.so (one translation unit: sc_stat.cu includes the kernel files in pipeline order).
#pragma once
#include "sc_common.cuh"

namespace {

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

}  // namespace
