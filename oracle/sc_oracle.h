/*
 * sc_oracle.h -- CPU ORACLE for the semi-coherent statistic (TEST INFRASTRUCTURE, NOT THE PRODUCT).
 *
 * Plain, slow, double-precision, direct evaluation of what the hot path of
 * arxiv 2408.13170 (Bandopadhyay & Moore) computes.  Written from the paper text
 * (/root/reference/PAPER.md, cited as PAPER.md:<line>) and from the readings of
 * SURVEY.md section 8(c) (cited as O1..O7, Q1..Q17) where the paper prints no formula.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may use anything in this directory.  It shares no code with the CUDA path under
 * paper_2408_13170_b200/ and neither includes the other.
 *
 * Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`):
 *   sco_stat_from_arrays : brute-force phase-grid maximisation of Eq. 7/10 on tiny grids; d=h identities;
 *                          phase/rescale invariance; refinement monotonicity; Cauchy-Schwarz; impulse indexing;
 *                          Monte-Carlo moments of Eq. 11-12.
 *   sco_phase / sco_tf   : Newtonian closed form; Table I / III t_c values;
 *                          finite-difference identity t(f) = Psi'(f)/2pi in long double; cycle count; the published
 *                          TaylorT2 timing series through 3.5PN (pins psi_2 .. psi_7); Peters' small-e equations
 *                          (pin the leading eccentric coefficient).
 *                          PARITY WITH THE LALSimulation / TaylorF2Ecc [49] CODE ITSELF IS UNPINNED (not in the container).
 *   sco_phase_ld / sco_tf_ld (truth mode): every pin of sco_phase / sco_tf above is run on them as well (Newtonian closed
 *                          form, TaylorT2 series, finite-difference identity, Peters); they agree with the FP64 functions to
 *                          the FP64 rounding of a 1e7-rad phase; f t_c against exact integer arithmetic (Python fractions);
 *                          truth-mode statistic = FP64-mode statistic to the predicted 3e-8/sqrt(Upsilon).
 *   sco_eval_stat_levels : level by level equal to sco_eval_stat and to a numpy bin sum over the oracle's template.
 *   sco_orbit/sco_template: arm lengths = L, centroid on the 1-AU circle; two-pulse single-link identity;
 *                          long-wavelength Michelson limit; T-combination -> 0; beta = +-pi/2 kills the Doppler term.
 *                          PARITY WITH BBHx [56] IS UNPINNED (not in the container).
 *   sco_components_from_seg / sco_loglike : noise-free d = A0 h gives log L_hat(A0) = 0; N = 1: max over a phase grid;
 *                          max over the amplitude gives -1/2<d|d> + 1/2 X^2/H, = Upsilon_1/2 - <d|d>/2 at N = 1.
 *   sco_equal_snr_edges  : flat s_j -> e_n = ceil(n n_bins/N); power-law s_j against the closed-form quantiles;
 *                          every segment holds C/N to within one bin's s_j; App. A: linear chirp +
 *                          white PSD -> equal-duration segments.
 *   sco_philox4x32_10    : known-answer vectors of the published algorithm (Salmon et al. 2011), moments.
 *   sco_pso_step         : hand-computed one-particle examples of Eq. 14 -> 15 -> 13.
 *   sco_pso_step_labeled : equals sco_pso_step when the labels are the contiguous blocks; invariant under a permutation
 *                          of the particles that carries the labels along (uniforms are keyed by the particle index).
 *   sco_kmeans           : well-separated blobs recover the generating partition; fixed point (nearest-centroid labels,
 *                          centroids = member means); within-cluster sum of squares never increases; a hand-computed
 *                          1-D example; scikit-learn's Lloyd KMeans from the same initial centroids gives the same labels.
 *   sco_converged        : the rule of PAPER.md:508 on hand-written histories.
 *   sco_*3 (A, E, T)     : reduce to the two-channel functions when the T data and template vanish; T template = the
 *                          (X+Y+Z)/sqrt(3) of sco_tdi (pinned above: T -> 0 in the long-wavelength limit); d = h gives rho^2
 *                          = <h|h>_A + <h|h>_E + <h|h>_T for any edges; brute-force phase grid on tiny grids.
 */
#ifndef SC_ORACLE_H
#define SC_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Field-for-field the same information the product's config carries; declared independently. */
typedef struct {
  double  T_obs_s;        /* observation time; df = 1/T_obs                   */
  int64_t j0;             /* f_j = (j0 + j)/T_obs_s                                          */
  int64_t n_bins;
  int32_t n_channels;     /* 2 = A,E  (Q16)                                                  */
  int32_t window_mode;    /* 1 = h(f)=0 where t(f) outside [0,T_obs]  (Q4)                   */
  int32_t pn_order_x2;    /* highest PN term kept in the phase sum, 7 = 3.5PN (O2)           */
  int32_t ecc_leading;    /* 1 = leading-order e0^2 phase term (Q5)                          */
  double  f_ref_ecc;      /* GW frequency at which e0 is defined                             */
  double  arm_L_s, au_s, orbit_alpha0, orbit_lambda0, year_s;   /* orbit constants (Q6)      */
  int32_t truth_mode;     /* 1 = "truth" mode: frequency, phase and its sin/cos in long double */
  int32_t reserved_;
} sco_config;

/* theta = (M_c [Msun, detector frame], eta, t_c [s from data start], lambda, beta, iota, psi, e_0)  (D3, Q3) */

/* O2: stationary-phase TaylorF2 phase Psi(f) [rad], h ~ A e^{-i Psi}. */
double sco_phase(const sco_config* c, const double theta[8], double f);
/* O3: t(f) = Psi'(f)/(2 pi) [s], analytic term-by-term derivative of O2. */
double sco_tf(const sco_config* c, const double theta[8], double f);
/* Truth mode: O2 / O3 line for line in x87 long double, f = j_abs / T_obs formed in long
 * double.  sco_phase_truth: out = (Psi rounded to double, the remainder Psi - that, cos Psi, sin Psi). */
long double sco_phase_ld(const sco_config* c, const double theta[8], long double f);
long double sco_tf_ld(const sco_config* c, const double theta[8], long double f);
void sco_phase_truth(const sco_config* c, const double theta[8], int64_t j_abs, double out[4]);
double sco_tf_truth(const sco_config* c, const double theta[8], int64_t j_abs);
/* O4: spacecraft positions p[0]=centroid p0, p[1..3]=spacecraft 1..3, in light-seconds, at time t [s]. */
void sco_orbit(const sco_config* c, double t, double p[4][3]);
/* O4: single-link response y_sr(f) for link s->r (1-based), WITHOUT the factor A(f) e^{-i Psi(f)}:
 * out = -i pi f L sinc[pi f L (1 - k.n_sr)] exp[-i pi f (L + k.(p_r+p_s))] zeta_sr ; orbit evaluated at time t. */
void sco_link(const sco_config* c, const double theta[8], double f, double t, int s, int r, double out_ri[2]);
/* O4: TDI transfer functions (X,Y,Z,A,E,T)(f) at orbit time t, without A(f) e^{-i Psi}; out_ri[6][2]. */
void sco_tdi(const sco_config* c, const double theta[8], double f, double t, double out_ri[6][2]);
/* O2+O3+O4 (+Q4 window): h_A, h_E on bins [j_begin, j_begin+n); interleaved re/im, n each.
 * Returns the number of bins inside the time window. Invalid theta -> all zeros, returns 0. */
int64_t sco_template(const sco_config* c, const double theta[8], int64_t j_begin, int64_t n,
                     double* hA_ri, double* hE_ri);

/* O1: Eq. 1/7/8/10 on arrays.  d,h interleaved re/im per channel (E pointers may be NULL for one channel),
 * S one-sided PSD per bin, edges[n_seg+1] bin indices, df = 1/T_obs.
 * out_seg (may be NULL) = [n_seg][3] = (Re z_k, Im z_k, sigma_k) with
 *   z_k = sum_a sum_j d_a conj(h_a)/S_a ,  sigma_k = sum_a sum_j |h_a|^2/S_a ;
 * returns Upsilon_N = 4 df sum_{k: sigma_k>0} |z_k|^2/sigma_k. */
double sco_stat_from_arrays(const double* dA_ri, const double* dE_ri, const double* hA_ri, const double* hE_ri,
                            const double* S_A, const double* S_E, double df,
                            const int64_t* edges, int64_t n_seg, double* out_seg);
/* Eq. 1 coherent inner product <a|b> over bins [0,n) (A3: rho^2 = <h|h>). */
double sco_inner(const double* aA_ri, const double* aE_ri, const double* bA_ri, const double* bE_ri,
                 const double* S_A, const double* S_E, double df, int64_t n);

/* Whole-population statistic: for each particle, sco_template then sco_stat_from_arrays (OpenMP over particles).
 * out[n_particles]; out_seg (may be NULL) [n_particles][n_seg][3]; n_inwin (may be NULL) [n_particles]. */
void sco_eval_stat(const sco_config* c, const double* dA_ri, const double* dE_ri, const double* S_A, const double* S_E,
                   const double* params, int64_t n_particles, const int64_t* edges, int64_t n_seg,
                   double* out, double* out_seg, int64_t* n_inwin);
/* Same templates, several edge lists at once (hierarchy levels): edges_cat = concatenated lists, n_segs[n_levels];
 * out [n_levels][n_particles]. */
void sco_eval_stat_levels(const sco_config* c, const double* dA_ri, const double* dE_ri, const double* S_A, const double* S_E,
                          const double* params, int64_t n_particles, const int64_t* edges_cat, const int64_t* n_segs,
                          int64_t n_levels, double* out);
/* Eq. 8, 3, 10 from the per-segment sums: out3 = (Upsilon_N, O_hat_N = sum_n x_n, <h|h> = sum_n [h|h]_n). */
void sco_components_from_seg(const double* seg, int64_t n_seg, double df, double out3[3]);
/* Eq. 9: log L_hat_N = -1/2 <d|d> - 1/2 amp^2 <h|h> + amp O_hat_N (hh, ohat of the unit-amplitude template). */
double sco_loglike(double dd, double hh, double ohat, double amp);
/* PAPER.md:120 (reading Q18): equal squared-SNR segment edges of one template on the FFT grid:
 * e_0 = 0, e_N = n_bins, e_n = min{ j : sum_{j'<j} s_j' >= (n/N) sum_j s_j },  s_j = sum_a |h_a|^2/S_a. */
void sco_equal_snr_edges(const double* hA_ri, const double* hE_ri, const double* S_A, const double* S_E,
                         int64_t n_bins, int64_t n_seg, int64_t* edges);
/* Upsilon_N with per-particle equal-SNR^2 edges; in_edges / out_edges [P][n_seg+1] and out_comp3 [P][3] may be NULL. */
void sco_eval_stat_adaptive(const sco_config* c, const double* dA_ri, const double* dE_ri, const double* S_A,
                            const double* S_E, const double* params, int64_t n_particles, int64_t n_seg,
                            const int64_t* in_edges, double* out, int64_t* out_edges, double* out_comp3);
int sco_num_threads(void);

/* Q10: Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11). */
void sco_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* Q10: the 16 uniforms of (seed, particle, iter): r_P[0..7], r_G[0..7], u = (word + 0.5) 2^-32. */
void sco_pso_uniforms(uint64_t seed, uint64_t particle, uint64_t iter, double rP[8], double rG[8]);
/* O7: one synchronous PSO step, Eq. 13-15 + best bookkeeping + reflecting boundary (Q9). */
void sco_pso_step(double* pos, double* vel, double* pbest_pos, double* pbest_val, const double* stat,
                  double* gbest_pos, double* gbest_val, const double* lo, const double* hi, const double* eps_min,
                  double omega, double phi_p, double phi_g, uint64_t seed, uint64_t iter,
                  int64_t n_particles, int32_t n_swarms);

/* Three channels A, E, T: the same definitions with one more term in every channel sum. */
int64_t sco_template3(const sco_config* c, const double theta[8], int64_t j_begin, int64_t n,
                      double* hA_ri, double* hE_ri, double* hT_ri);
double sco_stat_from_arrays3(const double* dA_ri, const double* dE_ri, const double* dT_ri, const double* hA_ri,
                             const double* hE_ri, const double* hT_ri, const double* S_A, const double* S_E,
                             const double* S_T, double df, const int64_t* edges, int64_t n_seg, double* out_seg);
double sco_inner3(const double* aA, const double* aE, const double* aT, const double* bA, const double* bE, const double* bT,
                  const double* S_A, const double* S_E, const double* S_T, double df, int64_t n);
/* Three-channel versions of sco_equal_snr_edges / sco_eval_stat_adaptive (s_j summed over A, E, T).  Pins: hT == NULL gives
 * sco_equal_snr_edges; every segment holds C/N to within one bin's s_j; d = h over three channels gives rho^2 on its own
 * edges; in_edges = the shared equal-width list gives sco_eval_stat3 (tests/test_oracle_three_channels.py). */
void sco_equal_snr_edges3(const double* hA_ri, const double* hE_ri, const double* hT_ri, const double* S_A, const double* S_E,
                          const double* S_T, int64_t n_bins, int64_t n_seg, int64_t* edges);
void sco_eval_stat_adaptive3(const sco_config* c, const double* dA_ri, const double* dE_ri, const double* dT_ri,
                             const double* S_A, const double* S_E, const double* S_T, const double* params, int64_t P,
                             int64_t n_seg, const int64_t* in_edges, double* out, int64_t* out_edges, double* out_comp3);
void sco_eval_stat3(const sco_config* c, const double* dA_ri, const double* dE_ri, const double* dT_ri, const double* S_A,
                    const double* S_E, const double* S_T, const double* params, int64_t n_particles,
                    const int64_t* edges, int64_t n_seg, double* out, double* out_seg);

/* O7 with a swarm label per particle (members need not be contiguous; PAPER.md:199 regrouping). */
void sco_pso_step_labeled(double* pos, double* vel, double* pbest_pos, double* pbest_val, const double* stat,
                          double* gbest_pos, double* gbest_val, const int32_t* label, const double* lo, const double* hi,
                          const double* eps_min, double omega, double phi_p, double phi_g, uint64_t seed, uint64_t iter,
                          int64_t n_particles, int32_t n_swarms);
/* Lloyd's k-means on the particle positions in prior-box units (Q19); returns the iterations run. */
int32_t sco_kmeans(const double* pos, int64_t n_particles, const double* lo, const double* hi, double* cent, int32_t K,
                   int32_t max_iter, int32_t* label, int64_t* count);
/* convergence rule "best does not improve by more than delta in `window` iterations". */
int32_t sco_converged(const double* hist, int64_t n_iter, int32_t window, double delta);

#ifdef __cplusplus
}
#endif
#endif
