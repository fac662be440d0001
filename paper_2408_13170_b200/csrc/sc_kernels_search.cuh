// sc_kernels_search.cuh -- a7 PSO update (Eq. 13-15) and k-means regrouping.
// Part of libscstat.so (one translation unit: sc_stat.cu includes the kernel files in pipeline order).
#pragma once
#include "sc_common.cuh"

namespace {

// ------------------------------------------------------------------------------------------------ a7 PSO
// (1)+(2): one CTA per swarm.  label == nullptr: swarm s = particles [s per_swarm, (s+1) per_swarm); else swarm s = the
// particles with label[p] == s (n_scan = n_particles; a swarm without members gets gbest_val = -inf, gbest_pos untouched).
// cand != nullptr (sc_pso_best: a swarm sharded over ranks): instead of (gbest_pos, gbest_val) the block's best is left as a
// candidate record cand[s][10] = (value, GLOBAL particle index = index_offset + local index, position[8]) for k_pso_pick.
__global__ void k_pso_best(const double* __restrict__ pos, double* __restrict__ pbest_pos, double* __restrict__ pbest_val,
                           const double* __restrict__ stat, double* __restrict__ gbest_pos, double* __restrict__ gbest_val,
                           int per_swarm, const int* __restrict__ label, long long n_scan,
                           double* __restrict__ cand = nullptr, long long index_offset = 0) {
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
  if (cand) {
    if (threadIdx.x < 8) cand[s * 10 + 2 + threadIdx.x] = pbest_pos[bi * 8 + threadIdx.x];
    if (threadIdx.x == 8) { cand[s * 10] = pbest_val[bi]; cand[s * 10 + 1] = (double)(index_offset + bi); }
    return;
  }
  if (threadIdx.x < 8) gbest_pos[s * 8 + threadIdx.x] = pbest_pos[bi * 8 + threadIdx.x];
  if (threadIdx.x == 8) gbest_val[s] = pbest_val[bi];
}

// (2) across shards: among n_cand candidate records per swarm (cand [n_cand][n_swarms][10], e.g. all-gathered over the
// ranks that share the swarms) the arg max of the value, lowest global particle index on ties -- the rule of k_pso_best,
// so a swarm cut into shards gets the same best as the swarm in one piece.  One warp per swarm.
__global__ void k_pso_pick(const double* __restrict__ cand, int n_cand, int n_swarms, double* __restrict__ gbest_pos,
                           double* __restrict__ gbest_val) {
  const int s = blockIdx.x, l = threadIdx.x;
  double best = -INFINITY, bidx = INFINITY;
  int bc = -1;
  for (int c = l; c < n_cand; c += 32) {
    const double* r = cand + ((size_t)c * n_swarms + s) * 10;
    const double v = r[0], i = r[1];
    if (bc < 0 || v > best || (v == best && i < bidx)) { best = v; bidx = i; bc = c; }
  }
  for (int o = 16; o > 0; o >>= 1) {
    const double ov = __shfl_xor_sync(0xffffffffu, best, o), oi = __shfl_xor_sync(0xffffffffu, bidx, o);
    const int oc = __shfl_xor_sync(0xffffffffu, bc, o);
    if (oc >= 0 && (bc < 0 || ov > best || (ov == best && oi < bidx))) { best = ov; bidx = oi; bc = oc; }
  }
  if (bc < 0) return;
  const double* r = cand + ((size_t)bc * n_swarms + s) * 10;
  if (l < 8) gbest_pos[s * 8 + l] = r[2 + l];
  if (l == 8) gbest_val[s] = r[0];
}

// (3)-(6): one thread per particle.
__global__ void k_pso_move(double* __restrict__ pos, double* __restrict__ vel, const double* __restrict__ pbest_pos,
                           const double* __restrict__ gbest_pos, const double* __restrict__ lo, const double* __restrict__ hi,
                           const double* __restrict__ eps_min, double omega, double phi_p, double phi_g,
                           uint64_t seed, uint64_t iter, long long P, int per_swarm, const int* __restrict__ label,
                           long long index_offset = 0 /* global index of local particle 0: the Philox counter */) {
  const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P) return;
  const int s = label ? label[p] : (int)(p / per_swarm);
  uint32_t w[16];
#pragma unroll
  for (uint32_t b = 0; b < 4; ++b)
    philox4x32_10((uint32_t)(p + index_offset), (uint32_t)iter, b, 0u, (uint32_t)seed, (uint32_t)(seed >> 32), w + 4 * b);
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

}  // namespace
