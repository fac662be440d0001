/*
 * sc_stat.h -- C ABI of the B200-native semi-coherent statistic library (libscstat.so).
 *
 * Hot path of Bandopadhyay & Moore, "A GPU-accelerated semi-coherent hierarchical search for stellar-mass
 * binary inspiral signals in LISA" (arXiv 2408.13170; text at /root/reference/PAPER.md, cited PAPER.md:<line>):
 * batched evaluation of the semi-coherent detection statistic Upsilon_N (Eq. 10) for a whole
 * particle-swarm population, plus the PSO update (Eq. 13-15).  Where the paper names a model
 * but prints no formula (waveform, response), the readings O1..O7 / Q1..Q17 of SURVEY.md 8(c) are used; they are
 * restated in DESIGN.md.
 *
 * Conventions
 *  - Plain C, no exceptions, no torch types.  Every function returns an int status (0 = SC_OK, negative = error);
 *    the message of the last error is available from sc_last_error().
 *  - "device" = pointer to CUDA device memory of the current device; "host" = ordinary host memory.
 *  - The caller owns every buffer it passes.  The handle owns its whitened copy of the data and its scratch
 *    (grown lazily); nothing caller-visible is allocated by the library.
 *  - All work is enqueued on the given cudaStream_t (passed as void*; NULL = default stream).  No host
 *    synchronisation happens inside the *_stat / pso calls unless stated; one handle is used from one stream
 *    at a time.
 *  - CUDA errors are sticky in the handle: after SC_ERR_CUDA every call returns SC_ERR_CUDA.
 *  - There is NO CPU fallback: without a CUDA device sc_init_data fails with SC_ERR_CUDA.
 *
 * Particle parameter row (D3, Q3), FP64, row-major [n_particles][8]:
 *    theta = ( M_c [Msun, detector frame], eta, t_c [s from data start], lambda, beta, iota, psi, e_0 ).
 * Per-particle invalid input (non-finite, eta outside (0, 0.25], M_c <= 0) gives Upsilon = 0, never NaN.  So does a
 * particle whose t(f) is not increasing across its time window (window_mode = 1: the window is found by bisection and
 * verified at nine probe bins; the leading eccentric term can break monotonicity for large e_0): it has no contiguous
 * window.  The bin f = 0 (j0 = 0) carries no template.
 */
#ifndef SC_STAT_H
#define SC_STAT_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sc_handle sc_handle;    /* opaque, library-owned */

/* POD, copied at init.  Frequency grid f_j = (j0 + j)/T_obs_s, j = 0..n_bins-1 (the FFT grid). */
typedef struct {
  double  T_obs_s;        /* observation time; df = 1/T_obs                                         */
  int64_t j0;             /* first bin index                                                         */
  int64_t n_bins;         /* 1 <= n_bins < 2^31                                                      */
  int32_t n_channels;     /* 2 (A,E) for sc_init_data; 3 (A,E,T) for sc_init_data3                   */
  int32_t window_mode;    /* 0 = none, 1 = template is zero where t(f) is outside [0, T_obs]  (Q4)   */
  int32_t pn_order_x2;    /* highest phase term kept, 0..7; 7 = 3.5PN (O2)                           */
  int32_t ecc_leading;    /* 1 = include the leading-order e0^2 phase term (Q5)                      */
  double  f_ref_ecc;      /* GW frequency at which e0 is defined                                     */
  double  arm_L_s, au_s, orbit_alpha0, orbit_lambda0, year_s;   /* orbit constants, seconds / rad (Q6) */
} sc_config;

enum {
  SC_OK = 0,
  SC_ERR_INVALID_ARG = -1,   /* null pointer, n <= 0, bad config, edges not non-decreasing or out of [0, n_bins] */
  SC_ERR_NOT_INIT = -2,      /* null / freed handle                                                             */
  SC_ERR_CUDA = -3,          /* a CUDA call or kernel failed (sticky)                                           */
  SC_ERR_OOM = -4            /* device allocation failed                                                        */
};

/* Options for sc_set_option. */
enum {
  SC_OPT_PRECISION = 1,      /* 0 = auto (FP32 amplitude path when n_seg >= SC_OPT_F32_MIN_SEG, else all-FP64),
                                1 = force FP32 amplitude path, 2 = force all-FP64.  Phase is FP64 always.       */
  SC_OPT_F32_MIN_SEG = 2,    /* threshold of the auto rule (default 8)               */
  SC_OPT_SCRATCH_BYTES = 3,  /* cap of the node-table scratch (default 32 GiB); larger populations run in batches     */
  SC_OPT_TC_MAX_S = 4,       /* the caller's upper bound on t_c [s] over the particles (the search tile's t_c range,
                                PAPER.md:253); sets the coarse node spacing to about one day of signal time at the
                                low band edge.  Default 10 yr.                                  */
  SC_OPT_WINDOW_FRACTION_PPM = 15, /* the caller's statement of the mean share of the band that lies inside a particle's time
                                window, in parts per million (0 = not stated, default; sc_get_counters after one evaluation gives
                                evaluated_bins / (n_particles x n_bins)).  With shared edges a particle then has N' = n_seg x fraction
                                non-empty segments, and the FP32-amplitude path spaces its nodes for that N': the interpolation
                                errors of the segments are independent, so the error of Upsilon falls like 1/sqrt(N') and the node
                                spacing may grow like N'^(1/12) at the same modelled error (half the
                                stated fraction is used).  Not stated: N' = 8, the fewest segments that path is left with.
                                Particles of such a population that end up with too few segments for the spacing chosen
                                (Upsilon below twice 8 (days / 4)^12) go to the escalation pass like those below tau.
                                sc_search_run measures the fraction itself when none is stated.  Per-segment output
                                (sc_eval_segments) and per-particle segments (sc_eval_stat_adaptive: integer edges from the
                                interpolated sigma) always keep the N' = 8 spacing. */
  SC_OPT_QUAD_AMPLITUDES = 16, /* 1 (default): where the fine sub-intervals are >= 256 bins (node spacing >= 1024) and the segments
                                >= 128 bins on average, the unmasked pair loop of k_dense2 / k_dense2_ad evaluates the amplitudes as
                                quadratics over runs of a quarter sub-interval (22 packed FP32 instructions per bin pair instead of
                                26; the dropped term is <= 3e-8 of the amplitude).  0: cubics
                                everywhere. */
  SC_OPT_STRIDE_LOG2 = 5,    /* 0 = automatic (rule above), else log2 of the coarse node spacing in bins (3..12)   */
  SC_OPT_PROFILE = 6,        /* 1 = record a CUDA event pair around every kernel launch (read by sc_get_timing)     */
  SC_OPT_SINCOS = 7,         /* FP32 amplitude path: sin/cos of the phase.  0 = automatic: hardware MUFU sin/cos
                                (gain-calibrated at init) when n_seg >= SC_OPT_MUFU_MIN_SEG, else FP32 polynomial;
                                1 = polynomial always; 2 = MUFU always.  See DESIGN.md "Precision".                  */
  SC_OPT_MUFU_MIN_SEG = 8,   /* threshold of that rule (default 32)                                                  */
  SC_OPT_ESCALATE = 9,       /* 1 (default): in the automatic precision mode sc_eval_stat / sc_eval_stat_host / the search
                                driver re-evaluate, by the all-FP64 path, every particle whose FP32-path statistic came
                                out as 0 < Upsilon < tau (the FP32 path's relative error grows like 1/sqrt(Upsilon));
                                selection, compaction and scatter happen on the device, no host synchronisation.
                                Three-channel handles (sc_init_data3): the selection is made on the COMBINED statistic,
                                both passes re-run all-FP64 for the compacted set; there
                                the selected count is read back (one 4-byte synchronising copy per particle batch).
                                0 = off.  Not applied by sc_eval_segments / _components / _loglike / _adaptive.        */
  SC_OPT_ESC_TAU_POLY_X1000 = 10,  /* tau x 1000 for the polynomial sin/cos flavour (default 6000)                    */
  SC_OPT_ESC_TAU_MUFU_X1000 = 11,  /* tau x 1000 for the hardware sin/cos flavour (default 16000)                     */
  SC_OPT_FUSED_AET = 14,     /* three-channel handles (sc_init_data3).  1 (default): the FP32-amplitude path evaluates A, E and T in
                                ONE pass (k_dense3: three channels in the pair loop).  0: two passes through the two-channel
                                kernels, (A, E) and (T, nothing), with per-segment tables combined afterwards.  The all-FP64
                                modes (n_seg < SC_OPT_F32_MIN_SEG, SC_OPT_PRECISION = 2, the escalation pass) always take two. */
  SC_OPT_TENSOR_CORES = 13,  /* 0 (default): the CUDA-core kernel k_dense2 (Horner cubics per bin).  1: the FP32-amplitude path
                                forms the amplitude x data factor of every bin as a split-TF32 contraction on the tensor cores
                                (tcgen05, k_dense2_tc; node spacings >= 128 bins; chunks of 8192 bins).  Same definition, same
                                tolerance, the two differ at the FP32 rounding level.  Measured on c3: 1.2 - 1.4 x SLOWER than
                                k_dense2 (DESIGN.md section 6 says why) -- kept as a tested alternative, not the product path. */
  SC_OPT_WINDOW_SORT = 12    /* 1 (default): each particle batch is processed in the order of the time-window centres (stable
                                radix sort on the device), so that the 32 particles of a warp share their windows; results
                                are bitwise reproducible for a given population and option set, but a particle's rounding
                                (FP32 path: ~1e-8 relative) depends on which particles share its warp.  0 = input order.  */
};

/* Kernel classes of sc_get_timing. */
enum { SC_TIME_NODES = 0, SC_TIME_DENSE = 1, SC_TIME_STITCH = 2, SC_TIME_PSO = 3, SC_TIME_OTHER = 4,
       SC_TIME_ESC = 5 /* every kernel of the escalation pass (SC_OPT_ESCALATE) */, SC_N_TIMING_CLASSES = 6 };

/* a0 -- data whitening, once per data stream (PSD known; Eq. 1 weights).
 * dA_ri, dE_ri: DEVICE, interleaved (re, im) FP64, n_bins complex each.  S_A, S_E: DEVICE, one-sided PSD, n_bins.
 * Stores W_a = d_a * 4df/S_a and G_a = 4df/S_a (rescaled to O(1)) in FP32 and FP64; the inputs are not kept.
 * Bins with non-finite or non-positive S are given zero weight.  Synchronises the stream once (to size the scale).
 * On success *out is a new handle (free with sc_free). */
int sc_init_data(sc_handle** out, const sc_config* cfg,
                 const double* dA_ri, const double* dE_ri, const double* S_A, const double* S_E,
                 void* cuda_stream);
/* Same with HOST buffers (copied to the device inside). */
int sc_init_data_host(sc_handle** out, const sc_config* cfg,
                      const double* dA_ri, const double* dE_ri, const double* S_A, const double* S_E,
                      void* cuda_stream);

/* Three TDI channels A, E, T (Eq. 1 and Eq. 7 sum over alpha in {A, E, T}; T = (X + Y + Z)/sqrt(3),
 * reading Q16).  cfg->n_channels must be 3; all arrays DEVICE as in sc_init_data.  On such a handle sc_eval_stat[_host],
 * sc_eval_segments, sc_eval_components, sc_eval_loglike, sc_data_norm, sc_eval_stat_adaptive and sc_search_run (shared or
 * per-particle edges) include the T channel: z_k and sigma_k are summed over A, E and T before |z_k|^2 / sigma_k is formed
 * (one common phase per segment, Q1), and the equal-SNR^2 edges are those of s_j summed over the three channels.  The
 * FP32-amplitude path does this in one pass (SC_OPT_FUSED_AET), the all-FP64 modes in two passes whose per-segment sums are
 * added.  The streams workload returns SC_ERR_INVALID_ARG on three-channel handles. */
int sc_init_data3(sc_handle** out, const sc_config* cfg,
                  const double* dA_ri, const double* dE_ri, const double* dT_ri,
                  const double* S_A, const double* S_E, const double* S_T, void* cuda_stream);
/* sc_gen_template with the T channel: hT_ri DEVICE [n_templates][n_bins] complex FP64 interleaved. */
int sc_gen_template3(sc_handle* h, const double* params, int64_t n_templates,
                     double* hA_ri, double* hE_ri, double* hT_ri, void* cuda_stream);

/* a1..a6 -- Upsilon_N(d, theta_p) for every particle (Eq. 7, 8, 10; readings Q1, Q2, Q7, Q8):
 *   z_k = sum_a sum_{j in [e_k, e_k+1)} d_a conj(h_a)/S_a,  sigma_k = sum_a sum_j |h_a|^2/S_a,
 *   out[p] = 4 df sum_{k: sigma_k > 0} |z_k|^2 / sigma_k,
 * with h_a(theta, f_j) = T_a(theta, f_j) A(f_j) e^{-i Psi(f_j)} (Eq. 16; O2-O4, window Q4).
 * params: DEVICE [n_particles][8].  seg_edges: HOST or DEVICE, n_seg+1 non-decreasing bin indices in [0, n_bins]
 * shared by all particles (Q2); edges may cover only part of the band and may contain empty segments.  A device
 * pointer is copied back to the host first (one stream synchronisation); host pointers cost no synchronisation.
 * out: DEVICE [n_particles]. */
int sc_eval_stat(sc_handle* h, const double* params, int64_t n_particles,
                 const int32_t* seg_edges, int32_t n_seg, double* out, void* cuda_stream);
/* Same with HOST params / out (copies inside; synchronises the stream before returning). */
int sc_eval_stat_host(sc_handle* h, const double* params, int64_t n_particles,
                      const int32_t* seg_edges, int32_t n_seg, double* out, void* cuda_stream);

/* Debug / parity: the per-segment sums themselves, out_seg DEVICE [n_particles][n_seg][3] = (Re z_k, Im z_k, sigma_k)
 * in the units of the definition above (template amplitude A(f) = f^(-7/6), O2). */
int sc_eval_segments(sc_handle* h, const double* params, int64_t n_particles,
                     const int32_t* seg_edges, int32_t n_seg, double* out_seg, void* cuda_stream);

/* Upsilon_N with the paper's own segments (App. A): boundaries f_n(theta) chosen for
 * EVERY particle such that each segment holds an equal share of the template's squared SNR.  On the FFT grid (reading
 * Q18): s_j = sum_a |h_a(f_j)|^2 / S_a(f_j), C = sum_j s_j, e_0 = 0, e_N = n_bins and
 *   e_n = min{ j : sum_{j' < j} s_j' >= C n / N },  n = 1 .. N-1;
 * then out[p] as in sc_eval_stat on those edges.  Floating point decides these integers, and the decision is taken in FP64
 * like the definition's (FP64 node amplitudes, FP64 moments of the weights, an FP64 bin-by-bin walk where a target falls): an
 * edge differs from a direct FP64 evaluation's only where a cumulative sum comes within the interpolation error (~1e-12
 * relative) of its target.  The statistic on those edges runs on the FP32-amplitude path.
 * out: DEVICE [n_particles] or NULL; out_edges: DEVICE int32 [n_particles][n_seg + 1] or NULL (the edges used; all
 * zero but the last for a particle whose template is empty); out3: DEVICE [n_particles][3] or NULL (as
 * sc_eval_components).  n_seg = 1 is sc_eval_stat on (0, n_bins); 2 <= n_seg runs the FP32-amplitude path. */
int sc_eval_stat_adaptive(sc_handle* h, const double* params, int64_t n_particles, int32_t n_seg,
                          double* out, int32_t* out_edges, double* out3, void* cuda_stream);

/* Eq. 8, 3, 10 from the same per-segment sums: out3 DEVICE [n_particles][3] =
 *   ( Upsilon_N,  O_hat_N = sum_k x_k = 4 df sum_k |z_k|,  <h|h> = sum_k [h|h]_k = 4 df sum_k sigma_k ),
 * the last two for the unit-amplitude template A(f) = f^(-7/6) (O2); a template of amplitude A has A O_hat, A^2 <h|h>.
 * Arguments otherwise as sc_eval_stat. */
int sc_eval_components(sc_handle* h, const double* params, int64_t n_particles,
                       const int32_t* seg_edges, int32_t n_seg, double* out3, void* cuda_stream);

/* Eq. 9: the semi-coherent log-likelihood log L_hat_N = -1/2 <d|d> - 1/2 A_p^2 <h|h> + A_p O_hat_N
 * of the template A_p f^(-7/6) T_a e^{-i Psi} (A_p carries 1/D_L and the chirp-mass prefactor).
 * amp: DEVICE [n_particles]; out: DEVICE [n_particles]. */
int sc_eval_loglike(sc_handle* h, const double* params, const double* amp, int64_t n_particles,
                    const int32_t* seg_edges, int32_t n_seg, double* out, void* cuda_stream);

/* <d|d> of the data stream the handle was built from (Eq. 1; computed once in sc_init_data).  dd: HOST. */
int sc_data_norm(sc_handle* h, double* dd);

/* The template itself on the dense grid through the same node tables and interpolants the statistic uses
 * (for injections and element-wise parity).  params: DEVICE [n_templates][8];
 * hA_ri, hE_ri: DEVICE [n_templates][n_bins] complex FP64 interleaved. */
int sc_gen_template(sc_handle* h, const double* params, int64_t n_templates,
                    double* hA_ri, double* hE_ri, void* cuda_stream);

/* a7 -- one synchronous PSO iteration (Eq. 13-15; App. B; readings Q9, Q10):
 *  (1) personal bests: stat[p] > pbest_val[p] (strict) -> pbest := (pos[p], stat[p]);
 *  (2) per swarm (n_swarms equal contiguous blocks): gbest := arg max pbest_val, lowest index on ties;
 *  (3) u = omega v + phi_p r_P (pbest - pos) + phi_g r_G (gbest - pos), r ~ U(0,1) from Philox4x32-10 keyed by
 *      seed with counter (particle, iter, block, 0);  (4) v = max(eps, |u|) sign(u) (sign(0) = +1);
 *  (5) pos += v;  (6) reflect at [lo, hi].
 * All arrays DEVICE, FP64: pos, vel, pbest_pos [n_particles][8]; pbest_val, stat [n_particles];
 * gbest_pos [n_swarms][8], gbest_val [n_swarms] (outputs); lo, hi, eps_min [8].
 * n_particles must be a multiple of n_swarms. */
int sc_pso_step(sc_handle* h, double* pos, double* vel, double* pbest_pos, double* pbest_val,
                const double* stat, double* gbest_pos, double* gbest_val,
                const double* lo, const double* hi, const double* eps_min,
                double omega, double phi_p, double phi_g, uint64_t seed, uint64_t iter,
                int64_t n_particles, int32_t n_swarms, void* cuda_stream);

/* a7 in its two halves, for swarms whose particles are SHARDED over ranks ("partition particles contiguously
 * by swarm then by rank; one all-reduce of (value, global index) + broadcast of the winning position").
 * A rank holds n_particles LOCAL particles in n_swarms equal contiguous blocks (its pieces of n_swarms swarms);
 * index_offset = the global index of its local particle 0 (global indices break ties and are the Philox counters, so the
 * sharded step is bit-identical to sc_pso_step on the whole population).
 *  sc_pso_best: steps (1)-(2) on the local particles; cand DEVICE [n_swarms][10] (out) = per block the candidate record
 *               (best personal-best value, its GLOBAL particle index as a double, its position[8]).
 *  sc_pso_pick: step (2) across shards: cand DEVICE [n_cand][n_swarms][10] (the records of the n_cand shards of each swarm,
 *               e.g. all-gathered over the ranks that share the swarms) -> gbest_pos [n_swarms][8], gbest_val [n_swarms]:
 *               arg max of the value, lowest global index on ties.
 *  sc_pso_move: steps (3)-(6) for the local particles against the given gbest_pos [n_swarms][8].
 * sc_pso_step == sc_pso_best + sc_pso_pick(n_cand = 1) + sc_pso_move with index_offset = 0.  All arrays DEVICE FP64. */
int sc_pso_best(sc_handle* h, const double* pos, double* pbest_pos, double* pbest_val, const double* stat, double* cand,
                int64_t n_particles, int32_t n_swarms, int64_t index_offset, void* cuda_stream);
int sc_pso_pick(sc_handle* h, const double* cand, int32_t n_cand, int32_t n_swarms, double* gbest_pos, double* gbest_val,
                void* cuda_stream);
int sc_pso_move(sc_handle* h, double* pos, double* vel, const double* pbest_pos, const double* gbest_pos,
                const double* lo, const double* hi, const double* eps_min,
                double omega, double phi_p, double phi_g, uint64_t seed, uint64_t iter,
                int64_t n_particles, int32_t n_swarms, int64_t index_offset, void* cuda_stream);

/* a7 with swarm membership given by a label per particle (after the k-means regrouping of PAPER.md:199 the members of
 * a swarm are not contiguous).  label: DEVICE int32 [n_particles], values in [0, n_swarms).  A swarm without members
 * gets gbest_val = -inf and keeps its gbest_pos.  Otherwise exactly sc_pso_step. */
int sc_pso_step_labeled(sc_handle* h, double* pos, double* vel, double* pbest_pos, double* pbest_val,
                        const double* stat, double* gbest_pos, double* gbest_val, const int32_t* label,
                        const double* lo, const double* hi, const double* eps_min,
                        double omega, double phi_p, double phi_g, uint64_t seed, uint64_t iter,
                        int64_t n_particles, int32_t n_swarms, void* cuda_stream);

/* Multi-swarm regrouping: Lloyd's k-means on all particle positions in prior-box units,
 * y_m = (theta_m - lo_m)/(hi_m - lo_m) over the dimensions with hi_m > lo_m (reading Q19).  Per iteration:
 * label[p] = arg min_k |y_p - y_k|^2 (lowest k on ties); centroid_k = mean of its members (a cluster without members keeps
 * its centroid).  Stops when no label changes or after max_iter iterations (one stream synchronisation per iteration).
 * pos: DEVICE [n_particles][8]; lo, hi: DEVICE [8]; cent: DEVICE [K][8], in = initial centroids, out = final; K <= 128;
 * label: DEVICE int32 [n_particles] (out); count: DEVICE int64 [K] or NULL (out); n_iter: HOST or NULL (out). */
int sc_kmeans(sc_handle* h, const double* pos, int64_t n_particles, const double* lo, const double* hi,
              double* cent, int32_t K, int32_t max_iter, int32_t* label, int64_t* count, int32_t* n_iter,
              void* cuda_stream);

/* sc_kmeans for callers that may not allocate device memory (CUDA graph capture set-ups, serving loops, harnesses that
 * forbid cudaMalloc): same arguments, same iterations, same results bit for bit, but the scratch (the "labels changed"
 * counter and the K member counts) lives in a file-scope static device array of 2 KiB that every GPU loading the library
 * holds until exit.  The call allocates and frees nothing on the device (no cudaMalloc / cudaFree, no allocating library
 * routine, no timing events: SC_OPT_PROFILE does not cover it).  K > SC_KMEANS_STATIC_MAX_K returns SC_ERR_INVALID_ARG.
 * The handle's device must be current.  The first call on a device resolves the array's address (cudaGetSymbolAddress);
 * like sc_kmeans it synchronises the stream once per iteration.  ALL calls on a device share the array: calls that
 * overlap on the GPU (different streams or host threads) race -- serialise them. */
#define SC_KMEANS_STATIC_MAX_K 128
int sc_kmeans_static(sc_handle* h, const double* pos, int64_t n_particles, const double* lo, const double* hi,
                     double* cent, int32_t K, int32_t max_iter, int32_t* label, int64_t* count, int32_t* n_iter,
                     void* cuda_stream);

/* The search of one tile (Fig. 2; Sec. III A-B; App. B). */
#define SC_MAX_RUNGS 8
typedef struct {
  int32_t n_rungs;                      /* ladder length, <= SC_MAX_RUNGS                                             */
  int32_t n_seg[SC_MAX_RUNGS];          /* the ladder, e.g. {100, 50, 10, 1}                            */
  double  omega[SC_MAX_RUNGS], phi_p[SC_MAX_RUNGS], phi_g[SC_MAX_RUNGS];   /* Table IV per rung     */
  double  eps_min[SC_MAX_RUNGS][8];     /* minimum velocities per rung, in the order of the parameter row              */
  int32_t adaptive_edges;               /* 1 = per-particle equal-SNR^2 segments, 0 = equal-width edges */
  int32_t conv_window;                  /* 50                                                          */
  double  conv_delta;                   /* 2.0                                                          */
  int32_t max_iters_per_rung;           /* hard cap (the paper states none)                                            */
  int32_t kmeans_max_iters;             /* Lloyd iterations cap; 0 = no regrouping between rungs                       */
  double  threshold;                    /* 100: swarms whose final best reaches it are flagged (Fig. 2)  */
  uint64_t seed;                        /* PSO uniforms: Philox key; the iteration counter runs on across rungs        */
  int32_t ranking_precision;            /* 0: every evaluation as sc_eval_stat (1e-6 per particle: all-FP64 below 8 segments,
                                           escalation).  1: the swarm only has to be RANKED -- all rungs run the FP32-amplitude
                                           path without escalation (relative error <= 1.6e-6/sqrt(Upsilon): < 2e-7 for anything
                                           near the Upsilon_1 >= 100 threshold), about 3x faster on the N < 8 rungs; the
                                           reported best_val are re-evaluated by the all-FP64 path at the end (with per-particle
                                           segments: on the very edges each best was ranked on).                          */
  int32_t reserved_;                    /* 0 */
} sc_search_config;
/* For every rung N: { Upsilon_N(pos) for all particles; sc_pso_step_labeled } until every non-empty swarm satisfies
 * "best has not improved by more than conv_delta over conv_window iterations" (or max_iters_per_rung); personal bests
 * start afresh on every rung (the objective changes, reading Q21); between rungs sc_kmeans regroups all particles from
 * the swarm bests as initial centroids (the particle count is conserved; the number of swarm slots is fixed, reading Q20).
 * pos, vel: DEVICE [n_particles][8], in = initial state, out = final.  label: DEVICE int32 [n_particles], in = initial
 * swarm of each particle, out = final.  lo, hi: DEVICE [8].  Outputs (HOST; all but best_* may be NULL):
 * best_pos [n_swarms][8], best_val [n_swarms] = swarm bests on the last rung; n_members [n_swarms]; passed [n_swarms] =
 * best_val >= threshold; iters_per_rung [n_rungs]; hist [n_rungs][n_swarms][max_iters_per_rung] = best after every
 * iteration (0 beyond the iterations run).  Synchronises the stream every iteration (S doubles read back).
 * Precision (automatic mode, two-channel handles): a shared-edge rung on which a particle's time window covers fewer than
 * SC_OPT_F32_MIN_SEG segments on average (n_seg x the mean window fraction, measured once from the first shared-edge
 * evaluation) runs on the all-FP64 path, like n_seg < SC_OPT_F32_MIN_SEG itself. */
int sc_search_run(sc_handle* h, const sc_search_config* cfg, double* pos, double* vel, int32_t* label,
                  int64_t n_particles, int32_t n_swarms, const double* lo, const double* hi,
                  double* best_pos, double* best_val, int64_t* n_members, int32_t* passed, int32_t* iters_per_rung,
                  double* hist, void* cuda_stream);

/* Second workload (the 5000 noise realisations of Fig. 3): MANY data streams that
 * share the handle's PSD against ONE template.  The handle's own data stream is not used.
 * sc_whiten_streams: dA_ri, dE_ri DEVICE FP64 [n_streams][n_bins][2] -> W DEVICE [n_streams][n_bins][4]
 *   = (A re, A im, E re, E im) of d 4df/S (rescaled to O(1) like the handle's own copy), FP32 (out_f64 = 0) or FP64.
 * sc_eval_stat_streams: out[d] = Upsilon_N(d_d, theta) (Eq. 10) for d = 0 .. n_streams-1 (<= 65535); theta: DEVICE [8];
 *   W as written by sc_whiten_streams (w_is_f64 says which flavour); seg_edges as in sc_eval_stat; out: DEVICE
 *   [n_streams].  The template and sigma_k are evaluated once in FP64; the per-stream sums run in the precision of W
 *   (FP32 streams: use for n_seg >= 8, like the FP32-amplitude path; FP64 streams for fewer segments).
 *   This path is HBM-bound: 16 (FP32) or 32 (FP64) bytes per stream and bin. */
int sc_whiten_streams(sc_handle* h, const double* dA_ri, const double* dE_ri, int64_t n_streams, int32_t out_f64,
                      void* W, void* cuda_stream);
int sc_eval_stat_streams(sc_handle* h, const double* theta, const void* W, int32_t w_is_f64, int64_t n_streams,
                         const int32_t* seg_edges, int32_t n_seg, double* out, void* cuda_stream);

/* Counters of the last sc_eval_stat / sc_eval_segments call (synchronises the stream):
 *  evaluated_bins = sum_p |{j in window_p} intersect [e_0, e_N)|  (the "evaluated (particle x bin)" of the metric),
 *  kernel_launches = CUDA kernels launched by the library since the handle was created. */
int sc_get_counters(sc_handle* h, int64_t* evaluated_bins, int64_t* kernel_launches, void* cuda_stream);

/* What the last FP32-amplitude pass of sc_eval_stat / sc_eval_segments / sc_eval_stat_host launched (host values, no
 * synchronisation; 0, 0 before the first such pass): log2 of the coarse node spacing in bins, and the kernel flavour as
 * a bit set -- SC_FLAVOUR_MUFU (hardware sin/cos), SC_FLAVOUR_MERGE (one set-up per coarse interval where it holds),
 * SC_FLAVOUR_QUAD (quadratic amplitudes over runs, 22 packed FP32 instructions per bin pair instead of 26),
 * SC_FLAVOUR_TC (k_dense2_tc), SC_FLAVOUR_AET (k_dense3).  For reporting (bench.py's instruction count) and tests. */
enum { SC_FLAVOUR_MUFU = 1, SC_FLAVOUR_MERGE = 2, SC_FLAVOUR_QUAD = 4, SC_FLAVOUR_TC = 8, SC_FLAVOUR_AET = 16 };
int sc_get_launch_info(sc_handle* h, int32_t* stride_log2, int32_t* flavour);

/* With SC_OPT_PROFILE = 1: device time [ms] and launch count per kernel class since the previous call, measured with
 * CUDA events on the launching stream (ms_per_class, launches_per_class: HOST arrays of SC_N_TIMING_CLASSES; either
 * may be NULL).  Synchronises the stream and resets the accumulators. */
int sc_get_timing(sc_handle* h, double* ms_per_class, int64_t* launches_per_class, void* cuda_stream);

/* Roofline denominator: sustained FP64 FMA rate of the current device, in DFMA/s, from a
 * dependent-chain-free microbenchmark (8 chains per thread, all SMs).  Needs no handle.  Synchronises. */
int sc_measure_fp64_peak(double* dfma_per_s, void* cuda_stream);

int sc_set_option(sc_handle* h, int32_t option, int64_t value);
int sc_free(sc_handle* h);
const char* sc_last_error(const sc_handle* h);    /* h may be NULL: error of the last failed sc_init_data */
const char* sc_version(void);

#ifdef __cplusplus
}
#endif
#endif
