// sc_kernels_stitch.cuh -- a6 statistic from the chunk fragments; template generation.
// Part of libscstat.so (one translation unit: sc_stat.cu includes the kernel files in pipeline order).
#pragma once
#include "sc_common.cuh"

namespace {

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

// The same fold with a particle's chunk range cut in kStitchParts contiguous parts, one thread each (k_stitch is a serial
// chain of ~n_chunks / 8 rounds of loads per particle: latency-bound when the windows cover many chunks).  A part folds its
// chunks from an empty carry and records what the serial walk would need to continue through it: the sums before its first
// reset event (a head that closes, or a tail that begins a piece), which event that was, the open piece at its end, and the
// closed segments in between.  k_stitch_join walks a particle's parts in order.  Same terms as k_stitch, other association.
constexpr int kStitchParts = 8;
constexpr int kStitchRec = 10;          // ups, xs, hs, head (zr, zi, sg), open piece at the end (zr, zi, sg), first event
__device__ __forceinline__ void stitch_range(const int* __restrict__ jlo, const int* __restrict__ jhi, int p, int chunk_first,
                                             int chunk_len, int n_chunks, int& c_lo, int& c_hi) {
  c_lo = 0; c_hi = n_chunks - 1;
  if (jlo) {
    const int lo = jlo[p], hi = jhi[p];
    if (hi <= lo) { c_lo = 0; c_hi = -1; }
    else {
      c_lo = max(lo / chunk_len - chunk_first, 0);
      c_hi = min((hi - 1) / chunk_len - chunk_first, n_chunks - 1);
    }
  }
}
__global__ void k_stitch_parts(const double* __restrict__ frag, const uint8_t* __restrict__ flags, int n_chunks, int P_pad, int n_slots,
                               int with_comp, const int* __restrict__ jlo, const int* __restrict__ jhi, int chunk_first,
                               int chunk_len, double* __restrict__ rec) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  const int part = blockIdx.y;
  if (p >= n_slots) return;
  int c_lo, c_hi;
  stitch_range(jlo, jhi, p, chunk_first, chunk_len, n_chunks, c_lo, c_hi);
  const int n = c_hi - c_lo + 1;
  const int len = (max(n, 0) + kStitchParts - 1) / kStitchParts;
  const int a = c_lo + part * len, b = min(a + len - 1, c_hi);
  double ups = 0.0, xs = 0.0, hs = 0.0, zr = 0.0, zi = 0.0, sg = 0.0, hzr = 0.0, hzi = 0.0, hsg = 0.0;
  int ev = 0;                            // 0: no reset event in this part, 1: a head closed first, 2: a tail began first
  constexpr int kU = 8;
  for (int c0 = a; c0 <= b; c0 += kU) {
    double v[kU][7], w7[kU], w8[kU];
#pragma unroll
    for (int u = 0; u < kU; ++u) {
      const int cI = min(c0 + u, b);
      const double* f = frag + (size_t)cI * kFragFields * P_pad + p;
#pragma unroll
      for (int m = 0; m < 7; ++m) v[u][m] = f[(size_t)m * P_pad];
      w7[u] = with_comp ? f[(size_t)7 * P_pad] : 0.0; w8[u] = with_comp ? f[(size_t)8 * P_pad] : 0.0;
    }
#pragma unroll
    for (int u = 0; u < kU; ++u) {
      if (c0 + u > b) break;
      const uint8_t fl = flags[c0 + u];
      if (fl & CF_HEAD) {
        zr += v[u][1]; zi += v[u][2]; sg += v[u][3];
        if (fl & CF_HEAD_CLOSES) {
          if (ev == 0) { hzr = zr; hzi = zi; hsg = sg; ev = 1; }
          else if (sg > 0.0) {
            const double z2 = zr * zr + zi * zi;
            ups += z2 / sg;
            if (with_comp) { xs += sqrt(z2); hs += sg; }
          }
          zr = 0.0; zi = 0.0; sg = 0.0;
        }
      }
      ups += v[u][0];
      if (with_comp) { xs += w7[u]; hs += w8[u]; }
      if (fl & CF_TAIL) {
        if (ev == 0) { hzr = zr; hzi = zi; hsg = sg; ev = 2; }
        zr = v[u][4]; zi = v[u][5]; sg = v[u][6];
      }
    }
  }
  double* r = rec + (size_t)part * kStitchRec * P_pad + p;
  r[0] = ups; r[(size_t)1 * P_pad] = xs; r[(size_t)2 * P_pad] = hs;
  r[(size_t)3 * P_pad] = hzr; r[(size_t)4 * P_pad] = hzi; r[(size_t)5 * P_pad] = hsg;
  r[(size_t)6 * P_pad] = zr; r[(size_t)7 * P_pad] = zi; r[(size_t)8 * P_pad] = sg;
  r[(size_t)9 * P_pad] = (double)ev;
}
__global__ void k_stitch_join(const double* __restrict__ rec, int n_chunks, int P_pad, int P, double scale, double* __restrict__ out,
                              double* __restrict__ comp3, double x_scale, double h_scale, const int* __restrict__ pmap,
                              const int* __restrict__ jlo, const int* __restrict__ jhi, int chunk_first, int chunk_len,
                              const int* __restrict__ next_close) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= (pmap ? P_pad : P)) return;
  const int q = pmap ? pmap[p] : p;
  if (q >= P) return;
  int c_lo, c_hi;
  stitch_range(jlo, jhi, p, chunk_first, chunk_len, n_chunks, c_lo, c_hi);
  double ups = 0.0, xs = 0.0, hs = 0.0, zr = 0.0, zi = 0.0, sg = 0.0;
  auto close = [&](double cr, double ci, double cs_) {
    if (cs_ > 0.0) {
      const double z2 = cr * cr + ci * ci;
      ups += z2 / cs_;
      if (comp3) { xs += sqrt(z2); hs += cs_; }
    }
  };
#pragma unroll
  for (int part = 0; part < kStitchParts; ++part) {
    const double* r = rec + (size_t)part * kStitchRec * P_pad + p;
    const int ev = (int)r[(size_t)9 * P_pad];
    if (ev == 0) { zr += r[(size_t)6 * P_pad]; zi += r[(size_t)7 * P_pad]; sg += r[(size_t)8 * P_pad]; }
    else {
      if (ev == 1) close(zr + r[(size_t)3 * P_pad], zi + r[(size_t)4 * P_pad], sg + r[(size_t)5 * P_pad]);
      zr = r[(size_t)6 * P_pad]; zi = r[(size_t)7 * P_pad]; sg = r[(size_t)8 * P_pad];
    }
    ups += r[0];
    if (comp3) { xs += r[(size_t)1 * P_pad]; hs += r[(size_t)2 * P_pad]; }
  }
  // the piece left open at c_hi runs on through empty chunks until one closes it (as in k_stitch)
  if (sg > 0.0 && next_close && c_hi >= 0 && c_hi < n_chunks - 1 && next_close[c_hi] >= 0) close(zr, zi, sg);
  if (out) out[q] = ups * scale;
  if (comp3) { comp3[3 * (size_t)q] = ups * scale; comp3[3 * (size_t)q + 1] = xs * x_scale; comp3[3 * (size_t)q + 2] = hs * h_scale; }
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

}  // namespace
