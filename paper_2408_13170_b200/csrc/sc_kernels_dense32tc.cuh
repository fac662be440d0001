// sc_kernels_dense32tc.cuh -- a4 + a5, FP32-amplitude hot loop with the amplitude x data contraction on the 5th-generation
// tensor cores (tcgen05.mma kind::tf32, accumulators in TMEM).  Part of libscstat.so (one translation unit).
//
// What goes where.  z_k = sum_j q_j e^{2 pi i Phi_j} with the per-bin factor q_j = sum_a W_a(j) conj(c_a(j)), a = A, E.  On a
// fine sub-interval the node amplitudes are cubics; about its centre (x = s - 1/2, |x| <= 1/2)
//     c_a(x) = g0_a + g1_a x + g2_a x^2 + g3_a x^3      =>      q_j = sum_a sum_{m=0..3} conj(g_m,a) [W_a(j) x_j^m].
// That is a dense contraction, [128 particles x K] times [K x bins], whose data side (the brackets) is shared by ALL
// particles: the bin grid and the sub-interval grid are shared.  It runs on the tensor cores in split TF32 -- every FP32
// factor v = hi + lo with hi = tf32(v), lo = tf32(v - hi), representing v to 2^-24 |v| like FP32 itself:
//     m = 0 (the leading term):      hi*hi + hi*lo + lo*hi + lo*lo      -- error of the products <= 2^-24 relative
//     m = 1, 2 (<= 4e-2, 6e-4 |c|):  hi*hi + hi*lo + lo*hi              -- dropped lo*lo <= 2^-22 of a small term
//     m = 3 (<= 7e-6 |c|):           hi*hi
// 11 x 4 = 44 of K = 48 columns, smallest terms first so that the FP32 accumulator in TMEM takes the leading products last.
// The CUDA cores keep what is NOT a contraction: the FP64 phase by forward differences, sin/cos, the rotation
// z += q e^{2 pi i Phi} (4 packed FMAs per bin pair), the segment bookkeeping.  Against k_dense2 the 12 amplitude and 8
// data FMAs per bin and the shared-memory data records leave the loop (26 -> 5 packed-pipe slots per bin pair).
//
// Mechanics per CTA (128 particles x one chunk of 2048 bins, 4 CTAs per SM, 128 TMEM columns each):
//   * the data side is precomputed once per data stream and node spacing by k_tc_image: per 16-bin tile a 6 KB K-major
//     operand image (canonical no-swizzle core-matrix order), 32 rows = (pair, real/imaginary output, even/odd bin) so that
//     an accumulator row reads (q_r even, q_r odd, q_i even, q_i odd) per bin pair -- the packed registers of the loop;
//     one cp.async.bulk (UBLKCP) per tile into a 4-stage ring, completion on an mbarrier;
//   * per fine sub-interval every thread writes its particle's coefficient row (TF32 hi/lo) into the A tile (24 KB);
//   * one elected lane issues 6 tcgen05.mma (M = 128, N = 32, K = 8) per tile into one of four TMEM buffers and commits to
//     mbarriers.  The tiles a chunk needs form one list; tile g is issued by the LAST of the four warps to release its
//     trigger tile (g - 4 inside a sub-interval: the buffer it reuses; an acq_rel counter in shared memory), so no warp
//     waits for another except through the data it needs;
//   * the coefficient rows of the NEXT sub-interval are written when a warp enters the last tile of the current one (its
//     MMAs have completed by then, so one A tile is enough): the pipeline runs through sub-interval borders.  Only the
//     first tensor-core sub-interval after a gap (chunk start, a band-edge sub-interval) is a rendezvous;
//   * each thread reads its own row (TMEM lane = particle) with tcgen05.ld: a whole tile (32 columns) at once where no
//     segment edge cuts it, and releases the buffer before the arithmetic.
// Sub-intervals that are not "all 128 lanes inside their time windows" take the k_dense2 code path with the records read
// from global memory (band edges; a few per cent of the work on the short-window configurations).
#pragma once
#include "sc_common.cuh"

namespace {

namespace tc {
constexpr int kTileBins = 16;
constexpr int kKC = 12;                                   // 16-byte K chunks per row: K = 48 TF32
constexpr int kRowGroup = kKC * 128;                      // bytes per 8-row group of an operand tile (SBO)
constexpr int kTileBytes = 4 * kRowGroup;                 // operand image of one tile: 32 rows x K = 48 -> 6144 B
constexpr int kABytes = 16 * kRowGroup;                   // coefficient tile: 128 rows -> 24576 B
constexpr int kStages = 4, kBufs = 4;
constexpr int kOffA = 0;
constexpr int kOffT = kABytes;                            // ring
constexpr int kOffBar = kOffT + kStages * kTileBytes;     // b_full[4], s_free[4], d_full[4], buf_free[4], a_ready
constexpr int kBarFull = 0, kBarSFree = 4, kBarDFull = 8, kBarBufFree = 12, kBarAReady = 16, kNumBars = 17;
constexpr int kOffU = kOffBar + kNumBars * 8;             // tmem base, i_lo (max), i_hi (min), merge mask
constexpr int kSmemBytes = kOffU + 24;
constexpr int kChunk = 8192;                              // bins per CTA (nothing but the tiles in flight is staged)
constexpr int kThreads = kBlock + 32;                     // four consumer warps (lane = particle) and the producer warp
// instruction descriptor: D = F32, A = B = TF32, both K-major, N = 32, M = 128
constexpr uint32_t kIdesc = (1u << 4) | (2u << 7) | (2u << 10) | ((32u >> 3) << 17) | ((128u >> 4) << 24);

// (all shared-memory operands are 32-bit shared-window addresses: sb = address of the CTA's dynamic shared memory)
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t b, uint32_t cnt) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(b), "r"(cnt));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t b, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(b), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t b, uint32_t parity) {
  asm volatile("{\n.reg .pred P1;\nLAB_WAIT:\nmbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n@P1 bra DONE;\nbra LAB_WAIT;\nDONE:\n}"
               :: "r"(b), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               :: "r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ bool elect_one() {
  uint32_t pred = 0;
  asm volatile("{\n.reg .pred P1;\nelect.sync _|P1, 0xffffffff;\nselp.u32 %0, 1, 0, P1;\n}" : "=r"(pred));
  return pred != 0;
}
// K-major, no swizzle: a core matrix is 8 rows x 16 B, contiguous; LBO = distance between the two core matrices of one
// K = 8 step (128 B), SBO = distance between 8-row groups (kRowGroup), for both operands.
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr) {
  return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)(128 >> 4) << 16) | ((uint64_t)(kRowGroup >> 4) << 32) | (1ull << 46);
}
__device__ __forceinline__ void mma_tf32(uint32_t d_tmem, uint64_t da, uint64_t db, uint32_t acc) {
  asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}"
               :: "r"(d_tmem), "l"(da), "l"(db), "r"(kIdesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void mma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t b) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(b) : "memory");
}
__device__ __forceinline__ uint32_t lds_u8(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ float tf32_rna(float v) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(v));
  return __uint_as_float(r);
}
__device__ __forceinline__ void tld4(uint32_t taddr, uint32_t (&d)[4]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(d[0]), "=r"(d[1]), "=r"(d[2]), "=r"(d[3]) : "r"(taddr));
}
__device__ __forceinline__ void tld16(uint32_t taddr, uint32_t* d) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
               : "=r"(d[0]), "=r"(d[1]), "=r"(d[2]), "=r"(d[3]), "=r"(d[4]), "=r"(d[5]), "=r"(d[6]), "=r"(d[7]),
                 "=r"(d[8]), "=r"(d[9]), "=r"(d[10]), "=r"(d[11]), "=r"(d[12]), "=r"(d[13]), "=r"(d[14]), "=r"(d[15]) : "r"(taddr));
}
// the wait names the registers it protects, so that no use of them can be scheduled above it
__device__ __forceinline__ void tld_wait4(uint32_t (&d)[4]) {
  asm volatile("tcgen05.wait::ld.sync.aligned;" : "+r"(d[0]), "+r"(d[1]), "+r"(d[2]), "+r"(d[3]) :: "memory");
}
__device__ __forceinline__ void tld_wait16(uint32_t* d) {
  asm volatile("tcgen05.wait::ld.sync.aligned;"
               : "+r"(d[0]), "+r"(d[1]), "+r"(d[2]), "+r"(d[3]), "+r"(d[4]), "+r"(d[5]), "+r"(d[6]), "+r"(d[7]),
                 "+r"(d[8]), "+r"(d[9]), "+r"(d[10]), "+r"(d[11]), "+r"(d[12]), "+r"(d[13]), "+r"(d[14]), "+r"(d[15]) :: "memory");
}
__device__ __forceinline__ void pin16(uint32_t* d) {    // (no instruction: orders the uses of d after the preceding wait)
  asm volatile("" : "+r"(d[0]), "+r"(d[1]), "+r"(d[2]), "+r"(d[3]), "+r"(d[4]), "+r"(d[5]), "+r"(d[6]), "+r"(d[7]),
                    "+r"(d[8]), "+r"(d[9]), "+r"(d[10]), "+r"(d[11]), "+r"(d[12]), "+r"(d[13]), "+r"(d[14]), "+r"(d[15]) :: "memory");
}

// The producer (one thread of the fifth warp): for every tile of the tensor-core range [i_lo, i_hi) of sub-intervals, in
// walking order (g = 0, 1, ...), wait for its trigger (the four consumer warps have released the TMEM buffer it reuses /
// have written the coefficient rows it needs) and for its operand image, issue the 6 MMAs (M128 N32 K8) into TMEM buffer
// g & 3, commit to d_full (consumers) and s_free (the ring stage), then start the load of tile g + 2 into the stage tile
// g - 2 has vacated.  Triggers: tile t >= 4 of a sub-interval -- tile g - 4 (its buffer); t < 4 of a sub-interval that
// follows another -- the last tile of that one (the rows are rewritten when it is entered); the very first tile -- the rows.
__device__ __noinline__ void producer(uint32_t sb, uint32_t tmem, const uint4* __restrict__ Tc, int i_lo, int i_hi, int lg_tps,
                                      int n_last /* tiles of sub-interval i_hi - 1 */) {
  const uint32_t bar = sb + kOffBar;
  const int tps = 1 << lg_tps;                                // tiles per (full) sub-interval
  const int n_list = ((i_hi - i_lo - 1) << lg_tps) + n_last;
  const int tile0 = i_lo << lg_tps;                           // listed tile g is tile tile0 + g of the chunk
  for (int g = 0; g < min(n_list, 2); ++g) {
    mbar_expect_tx(bar + (kBarFull + g) * 8, kTileBytes);
    bulk_g2s(sb + kOffT + g * kTileBytes, Tc + (size_t)(tile0 + g) * (kTileBytes / 16), kTileBytes, bar + (kBarFull + g) * 8);
  }
  for (int g = 0; g < n_list; ++g) {
    const int stg = g & 3, t = g & (tps - 1);
    if (g == 0) mbar_wait(bar + kBarAReady * 8, 0u);
    else if (g >= tps || g >= 4) {
      const int tr = (g < tps || t >= 4) ? g - 4 : g - t - 1;
      mbar_wait(bar + (kBarBufFree + (tr & 3)) * 8, (uint32_t)((tr >> 2) & 1));
    }
    mbar_wait(bar + (kBarFull + stg) * 8, (uint32_t)((g >> 2) & 1));
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t aA = sb + kOffA, bB = sb + kOffT + stg * kTileBytes;
#ifndef SC_TC_NMMA
#define SC_TC_NMMA (kKC / 2)
#endif
#pragma unroll
    for (int k = 0; k < SC_TC_NMMA; ++k) mma_tf32(tmem + stg * 32, make_desc(aA + k * 256), make_desc(bB + k * 256), k > 0);
    mma_commit(bar + (kBarDFull + stg) * 8);
    mma_commit(bar + (kBarSFree + stg) * 8);
    if (g + 2 < n_list) {
      const int x = g + 2, s2 = x & 3;
      if (x >= 4) mbar_wait(bar + (kBarSFree + s2) * 8, (uint32_t)(((x >> 2) - 1) & 1));   // the MMAs of tile x - 4 have read the stage
      mbar_expect_tx(bar + (kBarFull + s2) * 8, kTileBytes);
      bulk_g2s(sb + kOffT + s2 * kTileBytes, Tc + (size_t)(tile0 + x) * (kTileBytes / 16), kTileBytes, bar + (kBarFull + s2) * 8);
    }
  }
}
}  // namespace tc

// The data side of the contraction (see the header), one CTA of 32 threads per 16-bin tile; thread n = row of the K-major
// image: pair = n / 4, n & 1 = odd bin of the pair, n & 2 = imaginary output.  With v = (wAr, wAi, wEr, wEi) for the real and
// (wAi, -wAr, wEi, -wEr) for the imaginary output, Pm = v x^m, the 16-byte chunks of a row are
//   hi(P3) | hi(P2) lo(P2) hi(P2) | hi(P1) lo(P1) hi(P1) | lo(P0) hi(P0) lo(P0) hi(P0) | 0      against the coefficient row
//   hi(g3) | lo(g2) hi(g2) hi(g2) | lo(g1) hi(g1) hi(g1) | lo(g0) lo(g0) hi(g0) hi(g0) | 0      written by k_dense2_tc.
__global__ void __launch_bounds__(32) k_tc_image(const float4* __restrict__ D32, int lg_fine, long long n_tiles,
                                                 uint4* __restrict__ img) {
  const long long tile = blockIdx.x;
  if (tile >= n_tiles) return;
  const int n = threadIdx.x;
  const long long j = tile * tc::kTileBins + 2 * (n >> 2) + (n & 1);
  const float4 ra = D32[(size_t)(j >> 1) * kPairRec], re = D32[(size_t)(j >> 1) * kPairRec + 1];
  const bool odd = (j & 1);
  const float w[4] = {odd ? ra.y : ra.x, odd ? ra.w : ra.z, odd ? re.y : re.x, odd ? re.w : re.z};
  float v[4] = {w[0], w[1], w[2], w[3]};
  if (n & 2) { v[0] = w[1]; v[1] = -w[0]; v[2] = w[3]; v[3] = -w[2]; }
  const int Sf = 1 << lg_fine;
  const double x = (double)(j & (Sf - 1)) / (double)Sf - 0.5;
  uint4* row = img + (size_t)tile * (tc::kTileBytes / 16) + (n >> 3) * (tc::kRowGroup / 16) + (n & 7);   // + chunk * 8
  float hi[4][4], lo[4][4];
  double xm = 1.0;
#pragma unroll
  for (int m = 0; m < 4; ++m) {
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const float P = (float)((double)v[r] * xm);
      hi[m][r] = tc::tf32_rna(P);
      lo[m][r] = tc::tf32_rna(P - hi[m][r]);
    }
    xm *= x;
  }
  auto pack = [](const float (&q)[4]) { return make_uint4(__float_as_uint(q[0]), __float_as_uint(q[1]), __float_as_uint(q[2]), __float_as_uint(q[3])); };
  row[0 * 8] = pack(hi[3]);
  row[1 * 8] = pack(hi[2]); row[2 * 8] = pack(lo[2]); row[3 * 8] = pack(hi[2]);
  row[4 * 8] = pack(hi[1]); row[5 * 8] = pack(lo[1]); row[6 * 8] = pack(hi[1]);
  row[7 * 8] = pack(lo[0]); row[8 * 8] = pack(hi[0]); row[9 * 8] = pack(lo[0]); row[10 * 8] = pack(hi[0]);
  row[11 * 8] = make_uint4(0u, 0u, 0u, 0u);
}

// one bin pair: z += q e^{2 pi i Phi} with q = (q_r, q_i) from the accumulator row
template <int SC>
__device__ __forceinline__ void tc_pair(PhaseFD& ph, u64 K2, u64 qr2, u64 qi2, u64& zr2, u64& zi2) {
  u64 cr2, sr2;
#if defined(SC_TC_EXP) && SC_TC_EXP == 1      /* timing experiment: no FP64 phase steps */
  { int n0 = __double2loint(ph.phi), n1 = __double2hiint(ph.d1) + n0; ph.phi = __hiloint2double(__double2hiint(ph.phi), n1 * 3 + 7);
    float x0, x1; f2unpack(f2mul(f2pack((float)n0, (float)n1), K2), x0, x1);
    cr2 = f2pack(__cosf(x0), __cosf(x1)); sr2 = f2pack(__sinf(x0), __sinf(x1)); }
#elif defined(SC_TC_EXP) && SC_TC_EXP == 2    /* timing experiment: no MUFU */
  { int n0, n1; phase_next_pair(ph, n0, n1);
    const u64 x = f2mul(f2pack((float)n0, (float)n1), K2); cr2 = x; sr2 = f2mul(x, x); }
#else
  sincos_pair<SC>(ph, K2, cr2, sr2);
#endif
  zr2 = f2fma(qr2, cr2, f2fma(f2neg(qi2), sr2, zr2));
  zi2 = f2fma(qr2, sr2, f2fma(qi2, cr2, zi2));
}


#ifndef SC_DENSE2TC_MINB
#define SC_DENSE2TC_MINB 4
#endif
template <bool SEG, int SC, bool MERGE = false>
__global__ void __launch_bounds__(tc::kThreads, SC_DENSE2TC_MINB) k_dense2_tc(DevCfg c, DenseArgs a, const ulonglong2* __restrict__ Dg,
                                                                             const uint4* __restrict__ Tg) {
  constexpr int CH = tc::kChunk;
  extern __shared__ __align__(128) unsigned char smem[];
  uint4* sA = reinterpret_cast<uint4*>(smem + tc::kOffA);
  uint32_t* sU = reinterpret_cast<uint32_t*>(smem + tc::kOffU);
  const uint32_t sb = tc::smem_u32(smem);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int chunk_l = blockIdx.y;                              // particle block fastest: the CTAs in flight share their tiles in L2
  const int cs = (a.chunk_first + chunk_l) * CH;
  const int ce = min(cs + CH, c.n_bins);
  const int ce2 = (ce + 1) & ~1;                               // pair-aligned end (data beyond n_bins is zero)
  const bool is_prod = (warp == 4);                            // the producer warp owns no particles
  const int p = blockIdx.x * kBlock + (is_prod ? 0 : tid);
  const int jlo = a.jlo[p], jhi = a.jhi[p];

  if (!__syncthreads_or(!is_prod && (jhi > cs) && (jlo < ce))) {
    if (!is_prod) {
      double* fz = a.frag + (size_t)chunk_l * kFragFields * a.P_pad + p;
#pragma unroll
      for (int m = 0; m < kFragFields; ++m) fz[(size_t)m * a.P_pad] = 0.0;
    }
    return;
  }

  if (tid == 0) {
#pragma unroll
    for (int i = 0; i < tc::kNumBars; ++i) tc::mbar_init(sb + tc::kOffBar + i * 8, (i >= tc::kBarBufFree) ? 4 : 1);
    sU[1] = 0u; sU[2] = 0x7fffffffu; sU[3] = 0xffffffffu;
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) {
    __syncwarp();
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(sb + tc::kOffU), "r"(128u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = sU[0];
  const uint32_t tm_lane = tmem + ((uint32_t)(warp * 32) << 16);

  const int S = c.stride, Sf = S >> 2, lgSf = c.log2_stride - 2;
  const int n_sub = (ce2 - cs + Sf - 1) >> lgSf;              // sub-intervals of this chunk (the last one may be cut by the band end)
  const float hS = 1.0f / (float)Sf;
  const u64 h2 = f2bcast(2.0f * hS);
  const u64 K2 = f2bcast(1.4629180792671596e-09f);            // 2 pi / 2^32

  // The sub-intervals all 128 lanes spend inside their time windows form one range [i_lo, i_hi) (every window is an
  // interval): the tensor-core range.  Which coarse intervals merge (see k_dense2) is decided for the CTA as well.
  if (!is_prod) {
    const int lo_l = max(0, (jlo - cs + Sf - 1) >> lgSf);
    const int hi_l = (ce2 <= jhi) ? n_sub : min(max(jhi - cs, 0) >> lgSf, n_sub - 1);
    uint32_t mm = 0u;
    if constexpr (MERGE) {
      const int n_co = CH >> c.log2_stride;                    // <= 16 (stride >= 512)
      for (int ic = 0; ic < n_co; ++ic) {
        const int ib = cs + (ic << c.log2_stride);
        const bool win = (ib >= jlo) && (ib + S <= jhi) && (ib + S <= ce2);
        if (win && coarse_dslope(c, a, p, ib >> c.log2_stride) <= a.merge_lim) mm |= 1u << ic;
      }
    }
    const int lo_w = __reduce_max_sync(0xffffffffu, lo_l), hi_w = __reduce_min_sync(0xffffffffu, hi_l);
    mm = __reduce_and_sync(0xffffffffu, mm);
    if (lane == 0) { atomicMax(&sU[1], (uint32_t)lo_w); atomicMin(&sU[2], (uint32_t)hi_w); atomicAnd(&sU[3], mm); }
  }
  __syncthreads();
  const int i_lo = (int)sU[1], i_hi = max((int)sU[2], i_lo);   // (empty range: i_hi = i_lo)
  const uint32_t mergemask = MERGE ? sU[3] : 0u;
  const uint4* Tc = Tg + (size_t)(cs >> 4) * (tc::kTileBytes / 16);   // this chunk's tiles
  const int lg_tps = lgSf - 4;                                 // tiles per sub-interval
  auto tiles_of = [&](int i) { const int ib = cs + (i << lgSf); return (min(ib + Sf, ce2) - ib + 15) >> 4; };
  if (is_prod) {
    if (lane == 0 && i_hi > i_lo) tc::producer(sb, tmem, Tc, i_lo, i_hi, lg_tps, tiles_of(i_hi - 1));
    __syncwarp();
  }

  if (!is_prod) {
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

  float cc[MERGE ? 4 : 1][4];  // merged coarse interval: cubic of the amplitudes in t = (j - coarse start)/stride
  // set-up of the sub-interval starting at bin ibx: phase differences (fresh unless a merged coarse interval runs on) and
  // the cubic coefficients of (Ar, Ai, Er, Ei) in s = (j - ibx)/Sf
  auto setup = [&](int ibx, PhaseFD& fdx, bool& fresh, float (&cfx)[4][4]) {
    const bool merged = MERGE && ((mergemask >> ((ibx - cs) >> c.log2_stride)) & 1u);
    fresh = true;
    if (merged) {
      if constexpr (MERGE) {
        if ((ibx & (S - 1)) == 0) { coarse_phase(c, a, p, ibx, fdx); coarse_amps(c, a, p, ibx, cc); }
        else fresh = false;                                    // the phase differences run on
        coarse_to_fine(cc, (ibx >> lgSf) & 3, cfx);
      }
    } else {
      sub_phase(c, a, p, ibx, fdx);
      sub_amps(c, a, p, ibx, cfx);
    }
  };
  // the particle's coefficient row about the centre of the sub-interval (x = s - 1/2), TF32 hi / lo (see k_tc_image)
  auto write_row = [&](const float (&cfx)[4][4]) {
    uint4 H[4], L[4];          // per power m: hi and lo of (Ar, Ai, Er, Ei)
    {
      float g[4][4];
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const float c0 = cfx[r][0], c1 = cfx[r][1], c2 = cfx[r][2], c3 = cfx[r][3];
        g[0][r] = fmaf(0.5f, c1, c0) + fmaf(0.125f, c3, 0.25f * c2);
        g[1][r] = fmaf(0.75f, c3, c1 + c2); g[2][r] = fmaf(1.5f, c3, c2); g[3][r] = c3;
      }
#pragma unroll
      for (int m = 0; m < 4; ++m) {
        float h[4], l[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) { h[r] = tc::tf32_rna(g[m][r]); l[r] = tc::tf32_rna(g[m][r] - h[r]); }
        H[m] = make_uint4(__float_as_uint(h[0]), __float_as_uint(h[1]), __float_as_uint(h[2]), __float_as_uint(h[3]));
        L[m] = make_uint4(__float_as_uint(l[0]), __float_as_uint(l[1]), __float_as_uint(l[2]), __float_as_uint(l[3]));
      }
    }
    uint4* row = sA + (tid >> 3) * (tc::kRowGroup / 16) + (tid & 7);
    row[0 * 8] = H[3];
    row[1 * 8] = L[2]; row[2 * 8] = H[2]; row[3 * 8] = H[2];
    row[4 * 8] = L[1]; row[5 * 8] = H[1]; row[6 * 8] = H[1];
    row[7 * 8] = L[0]; row[8 * 8] = L[0]; row[9 * 8] = H[0]; row[10 * 8] = H[0];
    row[11 * 8] = make_uint4(0u, 0u, 0u, 0u);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  };

  PhaseFD fd = {}, fd_n = {};
  float cf[4][4], cf_n[4][4];
  bool fresh_n = false, prepared = false;   // the next sub-interval's set-up has been made (and its row written)
  const uint32_t bar_d = sb + tc::kOffBar + tc::kBarDFull * 8, bar_f = sb + tc::kOffBar + tc::kBarBufFree * 8;

  // this warp is done with listed tile g (its accumulator row is in registers or consumed): one arrival per warp
  auto leave = [&](int g) {
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    asm volatile("{\n.reg .pred P1;\nsetp.eq.u32 P1, %1, 0;\n@P1 mbarrier.arrive.shared::cta.b64 _, [%0];\n}"
                 :: "r"(bar_f + (uint32_t)(g & 3) * 8), "r"(lane) : "memory");
  };

  for (int ib = cs; ib < ce2; ib += Sf) {
    const int ie = min(ib + Sf, ce2);
    const int i_sub = (ib - cs) >> lgSf;
    const bool fast = (i_sub >= i_lo) && (i_sub < i_hi);       // CTA-uniform

    if (fast) {
      // ---------------------------------------------------------------- tensor-core sub-interval, tile by tile
      const int n_t = (ie - ib + 15) >> 4;
      const int g_base = (i_sub - i_lo) << lg_tps;             // listed tiles that belong to earlier sub-intervals
      const bool chain_next = (i_sub + 1 < i_hi);
      if (prepared) {
        if (fresh_n) fd = fd_n;
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
          for (int m = 0; m < 4; ++m) cf[r][m] = cf_n[r][m];
        prepared = false;
      } else {
        bool fresh;
        setup(ib, fd, fresh, cf);
        write_row(cf);
        __syncwarp();
        if (lane == 0) tc::mbar_arrive(sb + tc::kOffBar + tc::kBarAReady * 8);   // the producer waits for the four rows
      }
      int piece = a.piece_first[(ib >> lgSf) - ((a.chunk_first * CH) >> lgSf)];
      u64 zr2 = 0, zi2 = 0;    // FP32 partial sums (even bins, odd bins) of the open piece since the last fold
      bool live = (k >= 0) && (k < a.n_seg);
      bool carry = false;      // the odd bin of a pair that straddled an edge waits in car_* for the piece it belongs to
      float car_zr = 0.f, car_zi = 0.f;
      auto fold = [&]() {
        float zrl, zrh, zil, zih;
        f2unpack(zr2, zrl, zrh); f2unpack(zi2, zil, zih);
        if (live) { Zr += (double)(zrl + zrh); Zi += (double)(zil + zih); }
        zr2 = 0; zi2 = 0;
      };
      for (int t = 0; t < n_t; ++t) {
        const int tb = ib + (t << 4), te = min(tb + 16, ie), g = g_base + t;
        tc::mbar_wait(bar_d + (uint32_t)(g & 3) * 8, (uint32_t)((g >> 2) & 1));
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        if (t == n_t - 1 && chain_next) {
          // every MMA of this sub-interval has completed: the row of the next one may be written now
          setup(ib + Sf, fd_n, fresh_n, cf_n);
          write_row(cf_n);
          prepared = true;
        }
        const uint32_t tbuf = tm_lane + (uint32_t)((g & 3) * 32);
        if (next_edge >= te && live && !carry && te - tb == 16) {
          // a whole tile inside one live piece: all 32 accumulator columns at once, the buffer is released before the arithmetic
          uint32_t d[32];
          tc::tld16(tbuf, d); tc::tld16(tbuf + 16, d + 16);
          tc::tld_wait16(d); tc::pin16(d + 16);
          leave(g);
#if defined(SC_TC_EXP) && SC_TC_EXP == 5   /* timing experiment: pipeline only, no per-bin arithmetic */
#pragma unroll
          for (int i = 0; i < 8; ++i) { zr2 ^= (u64)d[4 * i] | ((u64)d[4 * i + 1] << 32); zi2 ^= (u64)d[4 * i + 2] | ((u64)d[4 * i + 3] << 32); }
#else
#pragma unroll
          for (int i = 0; i < 8; ++i)
            tc_pair<SC>(fd, K2, f2pack(__uint_as_float(d[4 * i]), __uint_as_float(d[4 * i + 1])),
                        f2pack(__uint_as_float(d[4 * i + 2]), __uint_as_float(d[4 * i + 3])), zr2, zi2);
#endif
          if (t & 1) fold();                                   // every 32 bins
        } else {
          // a tile cut by segment edges, outside [e_0, e_N), or cut by the band end: piece by piece, pair by pair
          int jj = tb;
          while (jj < te) {
            const int ph = min(next_edge, te);                 // next_edge > jj (edges <= jj are consumed)
            if (carry) {                                       // jj is the odd bin of the straddling pair: already evaluated
              if (live) { Zr += (double)car_zr; Zi += (double)car_zi; }
              carry = false;
              ++jj;
            }
            const int jfull = ph & ~1;                         // full pairs end here; a straddling pair follows if ph is odd
            for (; jj < jfull; jj += 2) {
              if (live) {
                uint32_t d[4];
                tc::tld4(tbuf + (uint32_t)((jj & 15) * 2), d);
                tc::tld_wait4(d);
                tc_pair<SC>(fd, K2, f2pack(__uint_as_float(d[0]), __uint_as_float(d[1])), f2pack(__uint_as_float(d[2]), __uint_as_float(d[3])), zr2, zi2);
              } else {
                phase_skip_pair(fd);
              }
            }
            if (jj < ph) {
              // the pair (ph - 1, ph): even bin -> the piece that ends at ph, odd bin -> the next one
              fold();
              uint32_t d[4];
              tc::tld4(tbuf + (uint32_t)((jj & 15) * 2), d);
              tc::tld_wait4(d);
              tc_pair<SC>(fd, K2, f2pack(__uint_as_float(d[0]), __uint_as_float(d[1])), f2pack(__uint_as_float(d[2]), __uint_as_float(d[3])), zr2, zi2);
              float zrl, zil;
              f2unpack(zr2, zrl, car_zr); f2unpack(zi2, zil, car_zi);
              if (live) { Zr += (double)zrl; Zi += (double)zil; }
              zr2 = 0; zi2 = 0;
              carry = true;
              jj = ph;                                         // (the odd bin ph is taken at the top of the next piece)
            }
            if (ph == next_edge) {
              // the piece ends at an edge inside (or at the end of) the tile
              fold();
              if (ph < ie) {                                   // (an edge on the sub-interval end is handled below)
                if (live) Sg += sigma_moments(cf, a.moments + (size_t)piece * 4);
                ++piece;
                while (next_edge == ph) {
                  if (k >= 0 && k < a.n_seg) close_piece(true);
                  next_segment();
                }
                live = (k >= 0) && (k < a.n_seg);
              }
            }
          }
          leave(g);
          if (t & 1) fold();
        }
      }
      // the piece open at the end of the sub-interval
      fold();
      if (live) Sg += sigma_moments(cf, a.moments + (size_t)piece * 4);
      while (next_edge == ie) {                                // segments that end here (incl. empty ones)
        if (k >= 0 && k < a.n_seg) close_piece(true);
        next_segment();
      }
      continue;
    }

    // ------------------------------------------------------------------ band-edge sub-interval: the k_dense2 walk, records from global memory
    const bool lane_in = (ib >= jlo) && (ie <= jhi);
    const bool lane_out = (ie <= jlo) || (ib >= jhi);
    const bool all_in = __all_sync(0xffffffffu, lane_in);
    const bool all_out = __all_sync(0xffffffffu, lane_out);
    if (!all_out) { bool fresh; setup(ib, fd, fresh, cf); }

    u64 s2 = 0;        // (s_j, s_{j+1}) of the next pair
    const ulonglong2* rec = Dg;   // its data record
    auto pair = [&](int j, auto masked_c, auto with_sg_c, u64& zr2, u64& zi2, u64& sg2) {
      pair_eval<decltype(masked_c)::value, decltype(with_sg_c)::value, SC>(fd, cf, s2, rec, j, jlo, jhi, h2, K2, zr2, zi2, sg2);
    };
    using T_ = std::true_type;
    const bool use_mom = all_in;      // all lanes inside their windows: sigma from the piece moments, unmasked pairs
    int piece = use_mom ? a.piece_first[(ib >> lgSf) - ((a.chunk_first * CH) >> lgSf)] : 0;
    float car_zr = 0.f, car_zi = 0.f, car_sg = 0.f;
    bool carry = false;
    int pl = ib;
    while (pl < ie) {
      const int ph = min(next_edge, ie);
      const bool live = (k >= 0) && (k < a.n_seg);
      int jj = pl;
      if (carry) {
        if (live) { Zr += (double)car_zr; Zi += (double)car_zi; Sg += (double)car_sg; }
        carry = false;
        jj = pl + 1;
      }
      const int jfull = ph & ~1;
      if (!all_out) {
        if (!live && jj < jfull) {
          for (int t = jj; t < jfull; t += 2) phase_skip_pair(fd);
          jj = jfull;
        }
        s2 = f2pack((float)(jj - ib) * hS, (float)(jj + 1 - ib) * hS);
        rec = Dg + (size_t)(jj >> 1) * kPairRec;
        while (jj < ph) {
          const bool split = (jj == jfull);
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
      if (use_mom && live) Sg += sigma_moments(cf, a.moments + (size_t)piece * 4);
      ++piece;
      while (next_edge == ph) {
        if (k >= 0 && k < a.n_seg) close_piece(true);
        next_segment();
      }
      pl = ph;
    }
  }
  if (k >= 0 && k < a.n_seg) close_piece(false);
  if (!SEG) {
    frag[0] = ups;
    if (a.comp) { frag[(size_t)7 * a.P_pad] = xs; frag[(size_t)8 * a.P_pad] = hs; }
  }
  }  // consumer warps
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem), "r"(128u) : "memory");
  }
}

}  // namespace
