/*
 * sc_oracle.c -- CPU ORACLE (TEST INFRASTRUCTURE, NOT THE PRODUCT).  See sc_oracle.h for scope and pins.
 *
 * Everything is evaluated directly at every FFT bin in plain FP64, in the order the paper / SURVEY.md 8(c)
 * states it: no interpolation, no blocking, no fusion.  Build: gcc -O2 -ffp-contract=off -fopenmp.
 * "Truth" mode (sco_config.truth_mode = 1): the same formulas with the frequency, the
 * phase Psi(f) and its sin/cos in x87 long double (64-bit mantissa: 1e-12 rad at Psi = 1e7 rad instead of the 3e-9 rad
 * of FP64) -- for the corner where the FP64 rounding of the phase is the larger error (N = 1 at small Upsilon).  The
 * bin sums stay plain FP64 (relative rounding ~1e-13 over 4e6 bins: four orders below the phase term).
 * The time-window decision (Q4) stays in FP64 in both modes: it decides an integer, and both sides take it in FP64.
 *
 * Citations: PAPER.md:<line> = /root/reference/PAPER.md; "O1..O7" and "Q1..Q17" = SURVEY.md section 8(c) readings
 * (listed again in DESIGN.md), used where the paper names a model but prints no formula.
 */
#include "sc_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define SCO_PI      3.141592653589793238462643383279502884
#define SCO_EULER   0.577215664901532860606512090082402431
#define SCO_MSUN_S  4.925491025543576e-06   /* G Msun / c^3 in seconds (O2) */

/* ------------------------------------------------------------------------------------------------
 * O2 -- phase.  PAPER.md:219 names "TaylorF2Ecc" [49] and prints no formula; the reading is the textbook
 * non-spinning TaylorF2 stationary-phase phase to 3.5PN plus the leading-order e0^2 term:
 *   v = (pi M f)^(1/3),  M = M_c eta^(-3/5)
 *   Psi(f) = 2 pi f t_c - phi_c - pi/4 + 3/(128 eta) v^-5 sum_{k=0}^{7} psi_k v^k ,   phi_c = 0.
 * ------------------------------------------------------------------------------------------------ */
static int theta_valid(const double th[8]) {
  for (int i = 0; i < 8; ++i) if (!isfinite(th[i])) return 0;
  if (!(th[0] > 0.0)) return 0;
  if (!(th[1] > 0.0 && th[1] <= 0.25)) return 0;
  return 1;
}

/* psi_k(eta, v) for k = 0..7 (psi_5 and psi_6 carry ln v). */
static void pn_coeffs(double eta, double v, double psi[8]) {
  const double pi = SCO_PI, eta2 = eta * eta, eta3 = eta2 * eta;
  psi[0] = 1.0;
  psi[1] = 0.0;
  psi[2] = 3715.0 / 756.0 + 55.0 * eta / 9.0;
  psi[3] = -16.0 * pi;
  psi[4] = 15293365.0 / 508032.0 + 27145.0 * eta / 504.0 + 3085.0 * eta2 / 72.0;
  psi[5] = pi * (38645.0 / 756.0 - 65.0 * eta / 9.0) * (1.0 + 3.0 * log(v));
  psi[6] = 11583231236531.0 / 4694215680.0 - 640.0 * pi * pi / 3.0 - 6848.0 * SCO_EULER / 21.0
           - (6848.0 / 21.0) * log(4.0 * v)
           + (-15737765635.0 / 3048192.0 + 2255.0 * pi * pi / 12.0) * eta
           + 76055.0 * eta2 / 1728.0 - 127825.0 * eta3 / 1296.0;
  psi[7] = pi * (77096675.0 / 254016.0 + 378515.0 * eta / 1512.0 - 74045.0 * eta2 / 756.0);
}

double sco_phase(const sco_config* c, const double th[8], double f) {
  const double pi = SCO_PI;
  const double Mc = th[0] * SCO_MSUN_S, eta = th[1], tc = th[2], e0 = th[7];
  const double M = Mc * pow(eta, -0.6);
  const double v = cbrt(pi * M * f);
  double psi[8];
  pn_coeffs(eta, v, psi);
  double sum = 0.0;
  for (int k = 0; k <= c->pn_order_x2 && k <= 7; ++k) sum += psi[k] * pow(v, (double)(k - 5));
  double Psi = 2.0 * pi * f * tc - pi / 4.0 + 3.0 / (128.0 * eta) * sum;
  if (c->ecc_leading) {
    /* Q5: Delta Psi = -(3/(128 eta)) v^-5 (2355/1462) e0^2 (v_ref/v)^(19/3) */
    const double vref = cbrt(pi * M * c->f_ref_ecc);
    Psi += -3.0 / (128.0 * eta) * pow(v, -5.0) * (2355.0 / 1462.0) * e0 * e0 * pow(vref / v, 19.0 / 3.0);
  }
  return Psi;
}

/* O3 -- t(f) = (1/2pi) dPsi/df, term by term with dv/df = v/(3f):
 *   d/df[psi_k v^(k-5)] = (k-5) psi_k v^(k-5)/(3f)           (k != 5, 6)
 *   d/df[psi_5]         = P5 * 3 * (1/(3f)),   P5 = pi(38645/756 - 65 eta/9)
 *   d/df[psi_6 v]       = (psi_6 - 6848/21) v/(3f)
 * Newtonian limit: t_c - t(f) = (5/256) M_c^(-5/3) (pi f)^(-8/3). */
double sco_tf(const sco_config* c, const double th[8], double f) {
  const double pi = SCO_PI;
  const double Mc = th[0] * SCO_MSUN_S, eta = th[1], tc = th[2], e0 = th[7];
  const double M = Mc * pow(eta, -0.6);
  const double v = cbrt(pi * M * f);
  double psi[8];
  pn_coeffs(eta, v, psi);
  double sum = 0.0;
  for (int k = 0; k <= c->pn_order_x2 && k <= 7; ++k) {
    if (k == 5) sum += 3.0 * pi * (38645.0 / 756.0 - 65.0 * eta / 9.0);
    else if (k == 6) sum += (psi[6] - 6848.0 / 21.0) * v;
    else sum += (double)(k - 5) * psi[k] * pow(v, (double)(k - 5));
  }
  double dPsi = 2.0 * pi * tc + 3.0 / (128.0 * eta) * sum / (3.0 * f);
  if (c->ecc_leading) {
    /* the eccentric term scales as f^(-34/9) */
    const double vref = cbrt(pi * M * c->f_ref_ecc);
    const double dPsi_e = -3.0 / (128.0 * eta) * pow(v, -5.0) * (2355.0 / 1462.0) * e0 * e0 * pow(vref / v, 19.0 / 3.0);
    dPsi += dPsi_e * (-34.0 / 9.0) / f;
  }
  return dPsi / (2.0 * pi);
}

/* ---- truth mode: O2 / O3 once more, line for line, in long double (f arrives in long double as well: the FP64
 * rounding of f alone moves 2 pi f t_c by 2e-9 rad). ---- */
#define SCO_PIL    3.141592653589793238462643383279502884L
#define SCO_EULERL 0.577215664901532860606512090082402431L
static void pn_coeffs_ld(long double eta, long double v, long double psi[8]) {
  const long double pi = SCO_PIL, eta2 = eta * eta, eta3 = eta2 * eta;
  psi[0] = 1.0L;
  psi[1] = 0.0L;
  psi[2] = 3715.0L / 756.0L + 55.0L * eta / 9.0L;
  psi[3] = -16.0L * pi;
  psi[4] = 15293365.0L / 508032.0L + 27145.0L * eta / 504.0L + 3085.0L * eta2 / 72.0L;
  psi[5] = pi * (38645.0L / 756.0L - 65.0L * eta / 9.0L) * (1.0L + 3.0L * logl(v));
  psi[6] = 11583231236531.0L / 4694215680.0L - 640.0L * pi * pi / 3.0L - 6848.0L * SCO_EULERL / 21.0L
           - (6848.0L / 21.0L) * logl(4.0L * v)
           + (-15737765635.0L / 3048192.0L + 2255.0L * pi * pi / 12.0L) * eta
           + 76055.0L * eta2 / 1728.0L - 127825.0L * eta3 / 1296.0L;
  psi[7] = pi * (77096675.0L / 254016.0L + 378515.0L * eta / 1512.0L - 74045.0L * eta2 / 756.0L);
}

long double sco_phase_ld(const sco_config* c, const double th[8], long double f) {
  const long double pi = SCO_PIL;
  const long double Mc = (long double)th[0] * (long double)SCO_MSUN_S, eta = th[1], tc = th[2], e0 = th[7];
  const long double M = Mc * powl(eta, -0.6L);
  const long double v = cbrtl(pi * M * f);
  long double psi[8];
  pn_coeffs_ld(eta, v, psi);
  long double sum = 0.0L;
  for (int k = 0; k <= c->pn_order_x2 && k <= 7; ++k) sum += psi[k] * powl(v, (long double)(k - 5));
  long double Psi = 2.0L * pi * f * tc - pi / 4.0L + 3.0L / (128.0L * eta) * sum;
  if (c->ecc_leading) {
    const long double vref = cbrtl(pi * M * (long double)c->f_ref_ecc);
    Psi += -3.0L / (128.0L * eta) * powl(v, -5.0L) * (2355.0L / 1462.0L) * e0 * e0 * powl(vref / v, 19.0L / 3.0L);
  }
  return Psi;
}

long double sco_tf_ld(const sco_config* c, const double th[8], long double f) {
  const long double pi = SCO_PIL;
  const long double Mc = (long double)th[0] * (long double)SCO_MSUN_S, eta = th[1], tc = th[2], e0 = th[7];
  const long double M = Mc * powl(eta, -0.6L);
  const long double v = cbrtl(pi * M * f);
  long double psi[8];
  pn_coeffs_ld(eta, v, psi);
  long double sum = 0.0L;
  for (int k = 0; k <= c->pn_order_x2 && k <= 7; ++k) {
    if (k == 5) sum += 3.0L * pi * (38645.0L / 756.0L - 65.0L * eta / 9.0L);
    else if (k == 6) sum += (psi[6] - 6848.0L / 21.0L) * v;
    else sum += (long double)(k - 5) * psi[k] * powl(v, (long double)(k - 5));
  }
  long double dPsi = 2.0L * pi * tc + 3.0L / (128.0L * eta) * sum / (3.0L * f);
  if (c->ecc_leading) {
    const long double vref = cbrtl(pi * M * (long double)c->f_ref_ecc);
    const long double dPsi_e = -3.0L / (128.0L * eta) * powl(v, -5.0L) * (2355.0L / 1462.0L) * e0 * e0 * powl(vref / v, 19.0L / 3.0L);
    dPsi += dPsi_e * (-34.0L / 9.0L) / f;
  }
  return dPsi / (2.0L * pi);
}
/* ctypes-friendly wrappers (x87 long double does not cross the binding): f = j_abs / T_obs formed in long double;
 * out = (Psi rounded to double, Psi - that in double, cos Psi, sin Psi). */
void sco_phase_truth(const sco_config* c, const double th[8], int64_t j_abs, double out[4]) {
  const long double f = (long double)j_abs / (long double)c->T_obs_s;
  const long double Psi = sco_phase_ld(c, th, f);
  out[0] = (double)Psi; out[1] = (double)(Psi - (long double)out[0]);
  out[2] = (double)cosl(Psi); out[3] = (double)sinl(Psi);
}
double sco_tf_truth(const sco_config* c, const double th[8], int64_t j_abs) {
  return (double)sco_tf_ld(c, th, (long double)j_abs / (long double)c->T_obs_s);
}

/* ------------------------------------------------------------------------------------------------
 * O4 -- orbits and response.  PAPER.md:233-241 (Eq. 16) cites the BBHx implementation of [56] and prints
 * no formula; the reading is the leading-order frequency-domain response with the orbit frozen at t_f.
 * Equal-arm orbits to first order in e = L/(2 sqrt3 AU) (Q6); positions in light-seconds.
 * ------------------------------------------------------------------------------------------------ */
void sco_orbit(const sco_config* c, double t, double p[4][3]) {
  const double pi = SCO_PI;
  const double AU = c->au_s, L = c->arm_L_s;
  const double e = L / (2.0 * sqrt(3.0) * AU);
  const double alpha = 2.0 * pi * t / c->year_s + c->orbit_alpha0;
  const double sa = sin(alpha), ca = cos(alpha);
  p[0][0] = AU * ca; p[0][1] = AU * sa; p[0][2] = 0.0;
  for (int n = 1; n <= 3; ++n) {
    const double bn = 2.0 * pi * (double)(n - 1) / 3.0 + c->orbit_lambda0;
    const double sb = sin(bn), cb = cos(bn);
    p[n][0] = p[0][0] + AU * e * (sa * ca * sb - (1.0 + sa * sa) * cb);
    p[n][1] = p[0][1] + AU * e * (sa * ca * cb - (1.0 + ca * ca) * sb);
    p[n][2] = -sqrt(3.0) * AU * e * cos(alpha - bn);
  }
}

static double dot3(const double a[3], const double b[3]) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

/* sky basis (O4): n_hat source direction, k = -n_hat propagation, (u, v, k) right-handed (Q17). */
static void sky_basis(const double th[8], double k[3], double u[3], double v[3]) {
  const double lam = th[3], bet = th[4];
  const double cl = cos(lam), sl = sin(lam), cb = cos(bet), sb = sin(bet);
  k[0] = -cb * cl; k[1] = -cb * sl; k[2] = -sb;
  u[0] = -sb * cl; u[1] = -sb * sl; u[2] = cb;
  v[0] = -sl;      v[1] = cl;       v[2] = 0.0;
}

/* single link s->r given the orbit p[][] (at t_f) and the sky basis */
static void link_core(const sco_config* c, const double th[8], double f, double p[4][3],
                      const double k[3], const double u[3], const double v[3], int s, int r, double out[2]) {
  const double pi = SCO_PI, L = c->arm_L_s;
  const double iota = th[5], pol = th[6];
  double n[3];
  for (int i = 0; i < 3; ++i) n[i] = p[r][i] - p[s][i];
  const double nn = sqrt(dot3(n, n));
  for (int i = 0; i < 3; ++i) n[i] /= nn;
  /* polarisation: e+ = u(x)u - v(x)v, ex = u(x)v + v(x)u; eps+ = cos2psi e+ + sin2psi ex, epsx = -sin2psi e+ + cos2psi ex */
  const double nu = dot3(n, u), nv = dot3(n, v);
  const double nep = nu * nu - nv * nv, nex = 2.0 * nu * nv;
  const double c2 = cos(2.0 * pol), s2 = sin(2.0 * pol);
  const double Fp = c2 * nep + s2 * nex, Fx = -s2 * nep + c2 * nex;
  /* zeta_sr = (1+cos^2 iota)/2 (n.eps+.n) - i cos(iota) (n.epsx.n)   [h+ = (1+cos^2 i)/2 A e^-iPsi, hx = -i cos i A e^-iPsi] */
  const double ci = cos(iota);
  const double zr = 0.5 * (1.0 + ci * ci) * Fp, zi = -ci * Fx;
  /* y_sr = -i pi f L sinc[pi f L (1 - k.n)] exp[-i pi f (L + k.(p_r + p_s))] zeta */
  const double kn = dot3(k, n);
  const double x = pi * f * L * (1.0 - kn);
  const double sinc = (x == 0.0) ? 1.0 : sin(x) / x;
  double prs[3];
  for (int i = 0; i < 3; ++i) prs[i] = p[r][i] + p[s][i];
  const double ph = -pi * f * (L + dot3(k, prs));
  const double er = cos(ph), ei = sin(ph);
  /* (-i a)(er + i ei)(zr + i zi), a = pi f L sinc */
  const double a = pi * f * L * sinc;
  const double wr = er * zr - ei * zi, wi = er * zi + ei * zr;   /* e * zeta */
  out[0] = a * wi;      /* -i (wr + i wi) = wi - i wr */
  out[1] = -a * wr;
}

void sco_link(const sco_config* c, const double th[8], double f, double t, int s, int r, double out[2]) {
  double p[4][3], k[3], u[3], v[3];
  sco_orbit(c, t, p);
  sky_basis(th, k, u, v);
  link_core(c, th, f, p, k, u, v, s, r, out);
}

void sco_tdi(const sco_config* c, const double th[8], double f, double t, double out[6][2]) {
  const double pi = SCO_PI, L = c->arm_L_s;
  /* y[s][r], 1-based */
  double y[4][4][2], p[4][3], k[3], u[3], v[3];
  sco_orbit(c, t, p);
  sky_basis(th, k, u, v);
  for (int s = 1; s <= 3; ++s)
    for (int r = 1; r <= 3; ++r)
      if (s != r) link_core(c, th, f, p, k, u, v, s, r, y[s][r]);
  const double Dr = cos(2.0 * pi * f * L), Di = -sin(2.0 * pi * f * L);   /* D = e^{-2 pi i f L} */
  const double D2r = Dr * Dr - Di * Di, D2i = 2.0 * Dr * Di;
  const double gr = 1.0 - D2r, gi = -D2i;                                 /* 1 - D^2 */
  /* TDI 1st generation (Q6): X = (1-D^2)[(y31 + D y13) - (y21 + D y12)], Y and Z by cyclic 1->2->3->1 */
  double XYZ[3][2];
  for (int m = 0; m < 3; ++m) {
    const int a = 1 + m % 3, b = 1 + (m + 1) % 3, cc = 1 + (m + 2) % 3;   /* (a,b,c) = (1,2,3),(2,3,1),(3,1,2) */
    /* [(y_ca + D y_ac) - (y_ba + D y_ab)] */
    const double tr = (y[cc][a][0] + Dr * y[a][cc][0] - Di * y[a][cc][1]) - (y[b][a][0] + Dr * y[a][b][0] - Di * y[a][b][1]);
    const double ti = (y[cc][a][1] + Dr * y[a][cc][1] + Di * y[a][cc][0]) - (y[b][a][1] + Dr * y[a][b][1] + Di * y[a][b][0]);
    XYZ[m][0] = gr * tr - gi * ti;
    XYZ[m][1] = gr * ti + gi * tr;
  }
  for (int q = 0; q < 2; ++q) {
    const double X = XYZ[0][q], Y = XYZ[1][q], Z = XYZ[2][q];
    out[0][q] = X; out[1][q] = Y; out[2][q] = Z;
    out[3][q] = (Z - X) / sqrt(2.0);                 /* A */
    out[4][q] = (X - 2.0 * Y + Z) / sqrt(6.0);       /* E */
    out[5][q] = (X + Y + Z) / sqrt(3.0);             /* T */
  }
}

/* O2+O3+O4: h_alpha(f_j) = T_alpha(theta, f_j; t_f) * f^(-7/6) * e^{-i Psi(f_j)}  (Eq. 16),
 * zero outside the time window 0 <= t(f_j) <= T_obs when window_mode = 1 (Q4). */
int64_t sco_template3(const sco_config* c, const double th[8], int64_t j_begin, int64_t n, double* hA, double* hE,
                      double* hT);
int64_t sco_template(const sco_config* c, const double th[8], int64_t j_begin, int64_t n, double* hA, double* hE) {
  return sco_template3(c, th, j_begin, n, hA, hE, NULL);
}
/* The same with the third TDI channel T = (X + Y + Z)/sqrt(3) (the paper uses A, E and T; Q16). */
int64_t sco_template3(const sco_config* c, const double th[8], int64_t j_begin, int64_t n, double* hA, double* hE,
                      double* hT) {
  memset(hA, 0, (size_t)n * 2 * sizeof(double));
  if (hE) memset(hE, 0, (size_t)n * 2 * sizeof(double));
  if (hT) memset(hT, 0, (size_t)n * 2 * sizeof(double));
  if (!theta_valid(th)) return 0;
  int64_t inwin = 0;
  for (int64_t i = 0; i < n; ++i) {
    const double f = (double)(c->j0 + j_begin + i) / c->T_obs_s;
    const double t = sco_tf(c, th, f);
    if (c->window_mode == 1 && !(t >= 0.0 && t <= c->T_obs_s)) continue;
    ++inwin;
    const double amp = pow(f, -7.0 / 6.0);
    double tdi[6][2];
    sco_tdi(c, th, f, t, tdi);
    double cP, sP;                                               /* cos Psi, sin Psi */
    if (c->truth_mode) {
      const long double Psi = sco_phase_ld(c, th, (long double)(c->j0 + j_begin + i) / (long double)c->T_obs_s);
      cP = (double)cosl(Psi); sP = (double)sinl(Psi);
    } else {
      const double Psi = sco_phase(c, th, f);
      cP = cos(Psi); sP = sin(Psi);
    }
    const double er = amp * cP, ei = -amp * sP;                  /* A e^{-i Psi} */
    hA[2 * i]     = tdi[3][0] * er - tdi[3][1] * ei;
    hA[2 * i + 1] = tdi[3][0] * ei + tdi[3][1] * er;
    if (hE) {
      hE[2 * i]     = tdi[4][0] * er - tdi[4][1] * ei;
      hE[2 * i + 1] = tdi[4][0] * ei + tdi[4][1] * er;
    }
    if (hT) {
      hT[2 * i]     = tdi[5][0] * er - tdi[5][1] * ei;
      hT[2 * i + 1] = tdi[5][0] * ei + tdi[5][1] * er;
    }
  }
  return inwin;
}

/* ------------------------------------------------------------------------------------------------
 * O1 -- statistic core.  Eq. 7: [a|b]_n = sum_alpha 4 Re int_{f_n}^{f_n+1} a b^dagger / S df,
 * evaluated as a Riemann sum over FFT bins (Q7: half-open segments, no end-point weights).
 * Eq. 10: x_n = max_phi [d | h e^{i phi}]_n = 4 df |z_n| with ONE complex z_n summed over
 * channels (Q1);  [h|h]_n = 4 df sigma_n;  Upsilon_N = sum_n x_n^2/[h|h]_n = 4 df sum_n |z_n|^2/sigma_n.
 * Segments with sigma_n = 0 contribute 0 (Q8).
 * ------------------------------------------------------------------------------------------------ */
double sco_stat_from_arrays(const double* dA, const double* dE, const double* hA, const double* hE,
                            const double* SA, const double* SE, double df,
                            const int64_t* edges, int64_t n_seg, double* out_seg) {
  double ups = 0.0;
  for (int64_t k = 0; k < n_seg; ++k) {
    double zr = 0.0, zi = 0.0, sig = 0.0;
    for (int64_t j = edges[k]; j < edges[k + 1]; ++j) {
      /* d conj(h) / S */
      zr += (dA[2 * j] * hA[2 * j] + dA[2 * j + 1] * hA[2 * j + 1]) / SA[j];
      zi += (dA[2 * j + 1] * hA[2 * j] - dA[2 * j] * hA[2 * j + 1]) / SA[j];
      sig += (hA[2 * j] * hA[2 * j] + hA[2 * j + 1] * hA[2 * j + 1]) / SA[j];
      if (dE && hE && SE) {
        zr += (dE[2 * j] * hE[2 * j] + dE[2 * j + 1] * hE[2 * j + 1]) / SE[j];
        zi += (dE[2 * j + 1] * hE[2 * j] - dE[2 * j] * hE[2 * j + 1]) / SE[j];
        sig += (hE[2 * j] * hE[2 * j] + hE[2 * j + 1] * hE[2 * j + 1]) / SE[j];
      }
    }
    if (out_seg) { out_seg[3 * k] = zr; out_seg[3 * k + 1] = zi; out_seg[3 * k + 2] = sig; }
    if (sig > 0.0) {
      const double x = 4.0 * df * sqrt(zr * zr + zi * zi);     /* x_n, Eq. 10 */
      const double hh = 4.0 * df * sig;                        /* [h|h]_n */
      ups += x * x / hh;
    }
  }
  return ups;
}

/* Eq. 1: <a|b> = sum_alpha 4 Re sum_j a b^dagger / S df. */
double sco_inner(const double* aA, const double* aE, const double* bA, const double* bE,
                 const double* SA, const double* SE, double df, int64_t n) {
  double acc = 0.0;
  for (int64_t j = 0; j < n; ++j) {
    acc += (aA[2 * j] * bA[2 * j] + aA[2 * j + 1] * bA[2 * j + 1]) / SA[j];
    if (aE && bE && SE) acc += (aE[2 * j] * bE[2 * j] + aE[2 * j + 1] * bE[2 * j + 1]) / SE[j];
  }
  return 4.0 * df * acc;
}

/* ------------------------------------------------------------------------------------------------
 * Eq. 8: O_hat_N(d,h) = sum_n max_phi [d|h e^{i phi}]_n = sum_n x_n = 4 df sum_n |z_n|;
 * Eq. 3: <h|h> = sum_n [h|h]_n = 4 df sum_n sigma_n;  Eq. 10: Upsilon_N.
 * seg = [n_seg][3] = (Re z_n, Im z_n, sigma_n) as sco_stat_from_arrays writes it.  out3 = (Upsilon_N, O_hat_N, <h|h>).
 * Segments with sigma_n = 0 have z_n = 0 as well and contribute nothing to any of the three (Q8).
 * ------------------------------------------------------------------------------------------------ */
void sco_components_from_seg(const double* seg, int64_t n_seg, double df, double out3[3]) {
  double ups = 0.0, ohat = 0.0, hh = 0.0;
  for (int64_t n = 0; n < n_seg; ++n) {
    const double zr = seg[3 * n], zi = seg[3 * n + 1], sig = seg[3 * n + 2];
    if (sig > 0.0) {
      const double x = 4.0 * df * sqrt(zr * zr + zi * zi);
      const double h_n = 4.0 * df * sig;
      ups += x * x / h_n;
      ohat += x;
      hh += h_n;
    }
  }
  out3[0] = ups; out3[1] = ohat; out3[2] = hh;
}

/* Eq. 9: log L_hat_N = -1/2 <d|d> - 1/2 <h|h> + O_hat_N(d,h) for the template amp * h, with
 * hh = <h|h> and ohat = O_hat_N(d,h) of the unit-amplitude template (both are homogeneous in the amplitude). */
double sco_loglike(double dd, double hh, double ohat, double amp) {
  return -0.5 * dd - 0.5 * amp * amp * hh + amp * ohat;
}

/* ------------------------------------------------------------------------------------------------
 * "the segment boundaries are chosen such that each of the N segments contains an equal amount of
 * squared SNR ... f_n is reevaluated for every new value of theta".  On the FFT grid (reading Q18):
 *   s_j = sum_alpha |h_alpha(f_j)|^2 / S_alpha(f_j)     (the integrand of <h|h>, Eq. 1/3)
 *   C_j = sum_{j' < j} s_j'  (C_0 = 0, C_n_bins = C, summed in bin order),
 *   e_0 = 0,  e_N = n_bins,  e_n = min{ j : C_j >= C n / N }  for 0 < n < N.
 * If C = 0 (empty template) every interior edge is 0.
 * ------------------------------------------------------------------------------------------------ */
void sco_equal_snr_edges(const double* hA, const double* hE, const double* SA, const double* SE,
                         int64_t n_bins, int64_t n_seg, int64_t* edges) {
  double total = 0.0;
  for (int64_t j = 0; j < n_bins; ++j) {
    total += (hA[2 * j] * hA[2 * j] + hA[2 * j + 1] * hA[2 * j + 1]) / SA[j];
    if (hE && SE) total += (hE[2 * j] * hE[2 * j] + hE[2 * j + 1] * hE[2 * j + 1]) / SE[j];
  }
  edges[0] = 0; edges[n_seg] = n_bins;
  double cum = 0.0;            /* C_j */
  int64_t j = 0;
  for (int64_t n = 1; n < n_seg; ++n) {
    const double target = total * (double)n / (double)n_seg;
    while (j < n_bins && !(cum >= target)) {
      cum += (hA[2 * j] * hA[2 * j] + hA[2 * j + 1] * hA[2 * j + 1]) / SA[j];
      if (hE && SE) cum += (hE[2 * j] * hE[2 * j] + hE[2 * j + 1] * hE[2 * j + 1]) / SE[j];
      ++j;
    }
    edges[n] = (total > 0.0) ? j : 0;
  }
}

/* Upsilon_N with per-particle equal-SNR^2 edges.  in_edges (may be NULL): [P][n_seg+1] edges to use
 * instead of computing them (the parity tests pass the edges the device chose: where floating point decides an
 * integer the decision is taken once).  out_edges (may be NULL): [P][n_seg+1] the edges used. */
void sco_eval_stat_adaptive(const sco_config* c, const double* dA, const double* dE, const double* SA, const double* SE,
                            const double* params, int64_t P, int64_t n_seg, const int64_t* in_edges,
                            double* out, int64_t* out_edges, double* out_comp3) {
  const int64_t n = c->n_bins;
  const double df = 1.0 / c->T_obs_s;
  const int two = (c->n_channels >= 2);
#pragma omp parallel
  {
    double* hA = (double*)malloc((size_t)n * 2 * sizeof(double));
    double* hE = (double*)malloc((size_t)n * 2 * sizeof(double));
    int64_t* e = (int64_t*)malloc((size_t)(n_seg + 1) * sizeof(int64_t));
    double* seg = (double*)malloc((size_t)n_seg * 3 * sizeof(double));
#pragma omp for schedule(dynamic, 1)
    for (int64_t p = 0; p < P; ++p) {
      sco_template(c, params + 8 * p, 0, n, hA, two ? hE : NULL);
      if (in_edges) memcpy(e, in_edges + p * (n_seg + 1), (size_t)(n_seg + 1) * sizeof(int64_t));
      else sco_equal_snr_edges(hA, two ? hE : NULL, SA, two ? SE : NULL, n, n_seg, e);
      out[p] = sco_stat_from_arrays(dA, two ? dE : NULL, hA, two ? hE : NULL, SA, two ? SE : NULL, df, e, n_seg, seg);
      if (out_edges) memcpy(out_edges + p * (n_seg + 1), e, (size_t)(n_seg + 1) * sizeof(int64_t));
      if (out_comp3) sco_components_from_seg(seg, n_seg, df, out_comp3 + 3 * p);
    }
    free(hA); free(hE); free(e); free(seg);
  }
}

int sco_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void sco_eval_stat_levels(const sco_config* c, const double* dA, const double* dE, const double* SA, const double* SE,
                          const double* params, int64_t P, const int64_t* edges_cat, const int64_t* n_segs,
                          int64_t n_levels, double* out) {
  const int64_t n = c->n_bins;
  const double df = 1.0 / c->T_obs_s;
  const int two = (c->n_channels >= 2);
#pragma omp parallel
  {
    double* hA = (double*)malloc((size_t)n * 2 * sizeof(double));
    double* hE = (double*)malloc((size_t)n * 2 * sizeof(double));
#pragma omp for schedule(dynamic, 1)
    for (int64_t p = 0; p < P; ++p) {
      sco_template(c, params + 8 * p, 0, n, hA, two ? hE : NULL);
      const int64_t* e = edges_cat;
      for (int64_t l = 0; l < n_levels; ++l) {
        out[l * P + p] = sco_stat_from_arrays(dA, two ? dE : NULL, hA, two ? hE : NULL, SA, two ? SE : NULL, df, e, n_segs[l], NULL);
        e += n_segs[l] + 1;
      }
    }
    free(hA); free(hE);
  }
}

void sco_eval_stat(const sco_config* c, const double* dA, const double* dE, const double* SA, const double* SE,
                   const double* params, int64_t P, const int64_t* edges, int64_t n_seg,
                   double* out, double* out_seg, int64_t* n_inwin) {
  const int64_t n = c->n_bins;
  const double df = 1.0 / c->T_obs_s;
  const int two = (c->n_channels >= 2);
#pragma omp parallel
  {
    double* hA = (double*)malloc((size_t)n * 2 * sizeof(double));
    double* hE = (double*)malloc((size_t)n * 2 * sizeof(double));
#pragma omp for schedule(dynamic, 1)
    for (int64_t p = 0; p < P; ++p) {
      const int64_t w = sco_template(c, params + 8 * p, 0, n, hA, two ? hE : NULL);
      if (n_inwin) n_inwin[p] = w;
      out[p] = sco_stat_from_arrays(dA, two ? dE : NULL, hA, two ? hE : NULL, SA, two ? SE : NULL, df, edges, n_seg,
                                    out_seg ? out_seg + (size_t)p * (size_t)n_seg * 3 : NULL);
    }
    free(hA); free(hE);
  }
}

/* ------------------------------------------------------------------------------------------------
 * Q10 -- Philox4x32-10, restated from the published algorithm (Salmon et al., SC'11).
 * ------------------------------------------------------------------------------------------------ */
void sco_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

void sco_pso_uniforms(uint64_t seed, uint64_t particle, uint64_t iter, double rP[8], double rG[8]) {
  const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  uint32_t w[16];
  for (uint32_t b = 0; b < 4; ++b) {
    const uint32_t ctr[4] = {(uint32_t)particle, (uint32_t)iter, b, 0u};
    sco_philox4x32_10(ctr, key, w + 4 * b);
  }
  for (int m = 0; m < 8; ++m) {
    rP[m] = ((double)w[m] + 0.5) * 0x1p-32;
    rG[m] = ((double)w[8 + m] + 0.5) * 0x1p-32;
  }
}

/* ------------------------------------------------------------------------------------------------
 * O7 -- one synchronous PSO step.  Eq. 14, Eq. 15, Eq. 13;
 * bests use iteration i-1 quantities; reflecting boundary and sign(0) = +1 per Q9.
 * Swarms are n_swarms equal contiguous blocks of particles.
 * ------------------------------------------------------------------------------------------------ */
void sco_pso_step(double* pos, double* vel, double* pbest_pos, double* pbest_val, const double* stat,
                  double* gbest_pos, double* gbest_val, const double* lo, const double* hi, const double* eps_min,
                  double omega, double phi_p, double phi_g, uint64_t seed, uint64_t iter,
                  int64_t P, int32_t n_swarms) {
  /* (1) personal bests: strict improvement */
  for (int64_t p = 0; p < P; ++p)
    if (stat[p] > pbest_val[p]) {
      pbest_val[p] = stat[p];
      for (int m = 0; m < 8; ++m) pbest_pos[8 * p + m] = pos[8 * p + m];
    }
  /* (2) swarm bests: arg max of the personal bests, lowest index on ties */
  const int64_t per = P / n_swarms;
  for (int32_t s = 0; s < n_swarms; ++s) {
    int64_t best = (int64_t)s * per;
    for (int64_t p = best + 1; p < (int64_t)(s + 1) * per; ++p)
      if (pbest_val[p] > pbest_val[best]) best = p;
    gbest_val[s] = pbest_val[best];
    for (int m = 0; m < 8; ++m) gbest_pos[8 * s + m] = pbest_pos[8 * best + m];
  }
  /* (3)-(6) */
  for (int64_t p = 0; p < P; ++p) {
    const int32_t s = (int32_t)(p / per);
    double rP[8], rG[8];
    sco_pso_uniforms(seed, (uint64_t)p, iter, rP, rG);
    for (int m = 0; m < 8; ++m) {
      const double th = pos[8 * p + m];
      const double u = omega * vel[8 * p + m] + phi_p * rP[m] * (pbest_pos[8 * p + m] - th)
                       + phi_g * rG[m] * (gbest_pos[8 * s + m] - th);                         /* Eq. 14 */
      const double au = fabs(u), eps = eps_min[m];
      double v;
      if (au > 0.0) v = (eps > au ? eps : au) * (u / au);                                     /* Eq. 15 */
      else v = (eps > 0.0) ? eps : 0.0;                                                       /* Q9: sign(0) = +1 */
      double x = th + v;                                                                      /* Eq. 13 */
      if (x < lo[m]) { x = lo[m]; v = -v; }                                                   /* Q9: reflect */
      else if (x > hi[m]) { x = hi[m]; v = -v; }
      pos[8 * p + m] = x;
      vel[8 * p + m] = v;
    }
  }
}


/* ------------------------------------------------------------------------------------------------
 * Multi-swarm bookkeeping of the hierarchical search (readings Q19-Q21 of DESIGN.md).
 * ------------------------------------------------------------------------------------------------ */

/* O7 with swarm membership given by a label per particle (after k-means regrouping the members of a swarm are no
 * longer contiguous).  A swarm without members gets gbest_val = -inf and keeps its gbest_pos. */
void sco_pso_step_labeled(double* pos, double* vel, double* pbest_pos, double* pbest_val, const double* stat,
                          double* gbest_pos, double* gbest_val, const int32_t* label, const double* lo, const double* hi,
                          const double* eps_min, double omega, double phi_p, double phi_g, uint64_t seed, uint64_t iter,
                          int64_t P, int32_t n_swarms) {
  for (int64_t p = 0; p < P; ++p)
    if (stat[p] > pbest_val[p]) {
      pbest_val[p] = stat[p];
      for (int m = 0; m < 8; ++m) pbest_pos[8 * p + m] = pos[8 * p + m];
    }
  for (int32_t s = 0; s < n_swarms; ++s) {
    int64_t best = -1;
    for (int64_t p = 0; p < P; ++p)
      if (label[p] == s && (best < 0 || pbest_val[p] > pbest_val[best])) best = p;
    if (best < 0) { gbest_val[s] = -INFINITY; continue; }
    gbest_val[s] = pbest_val[best];
    for (int m = 0; m < 8; ++m) gbest_pos[8 * s + m] = pbest_pos[8 * best + m];
  }
  for (int64_t p = 0; p < P; ++p) {
    const int32_t s = label[p];
    double rP[8], rG[8];
    sco_pso_uniforms(seed, (uint64_t)p, iter, rP, rG);
    for (int m = 0; m < 8; ++m) {
      const double th = pos[8 * p + m];
      const double u = omega * vel[8 * p + m] + phi_p * rP[m] * (pbest_pos[8 * p + m] - th)
                       + phi_g * rG[m] * (gbest_pos[8 * s + m] - th);                         /* Eq. 14 */
      const double au = fabs(u), eps = eps_min[m];
      double v;
      if (au > 0.0) v = (eps > au ? eps : au) * (u / au);                                     /* Eq. 15 */
      else v = (eps > 0.0) ? eps : 0.0;
      double x = th + v;                                                                      /* Eq. 13 */
      if (x < lo[m]) { x = lo[m]; v = -v; }
      else if (x > hi[m]) { x = hi[m]; v = -v; }
      pos[8 * p + m] = x;
      vel[8 * p + m] = v;
    }
  }
}

/* k-means (Lloyd's algorithm) on the particle positions, in coordinates scaled by the prior box:
 * y_m = (theta_m - lo_m)/(hi_m - lo_m) for the dimensions with hi_m > lo_m, others ignored (Q19).
 * cent [K][8] in: initial centroids (theta units), out: final.  Each iteration: (a) label[p] = arg min_k |y_p - y_k|^2,
 * lowest k on ties; (b) centroid_k = mean of its members (sums in particle order), a cluster without members keeps its
 * centroid.  Stops when no label changes or after max_iter iterations; returns the number of iterations run.
 * count [K] (may be NULL) = members per cluster. */
int32_t sco_kmeans(const double* pos, int64_t P, const double* lo, const double* hi, double* cent, int32_t K,
                   int32_t max_iter, int32_t* label, int64_t* count) {
  double w[8];
  for (int m = 0; m < 8; ++m) w[m] = (hi[m] > lo[m]) ? 1.0 / (hi[m] - lo[m]) : 0.0;
  for (int64_t p = 0; p < P; ++p) label[p] = -1;
  int32_t it = 0;
  double* sum = (double*)malloc((size_t)K * 8 * sizeof(double));
  int64_t* cnt = (int64_t*)malloc((size_t)K * sizeof(int64_t));
  while (it < max_iter) {
    ++it;
    int64_t changed = 0;
    for (int64_t p = 0; p < P; ++p) {
      int32_t bk = 0; double bd = INFINITY;
      for (int32_t k = 0; k < K; ++k) {
        double d = 0.0;
        for (int m = 0; m < 8; ++m) { const double t = (pos[8 * p + m] - cent[8 * k + m]) * w[m]; d += t * t; }
        if (d < bd) { bd = d; bk = k; }
      }
      if (label[p] != bk) { label[p] = bk; ++changed; }
    }
    for (int32_t k = 0; k < K; ++k) { cnt[k] = 0; for (int m = 0; m < 8; ++m) sum[8 * k + m] = 0.0; }
    for (int64_t p = 0; p < P; ++p) {
      const int32_t k = label[p];
      ++cnt[k];
      for (int m = 0; m < 8; ++m) sum[8 * k + m] += pos[8 * p + m];
    }
    for (int32_t k = 0; k < K; ++k)
      if (cnt[k] > 0) for (int m = 0; m < 8; ++m) cent[8 * k + m] = sum[8 * k + m] / (double)cnt[k];
    if (changed == 0) break;
  }
  if (count) for (int32_t k = 0; k < K; ++k) count[k] = cnt[k];
  free(sum); free(cnt);
  return it;
}

/* App. B: a swarm has converged when the best value in its history has not improved by more than delta
 * over the last `window` iterations.  hist [n_iter] = best-so-far after each iteration of the rung. */
int32_t sco_converged(const double* hist, int64_t n_iter, int32_t window, double delta) {
  if (n_iter <= window) return 0;
  return (hist[n_iter - 1] - hist[n_iter - 1 - window] <= delta) ? 1 : 0;
}


/* ------------------------------------------------------------------------------------------------
 * Three TDI channels A, E, T (Eq. 1 and 7 sum over alpha in {A, E, T}).  Same definitions as above
 * with one more term in every channel sum.
 * ------------------------------------------------------------------------------------------------ */
double sco_stat_from_arrays3(const double* dA, const double* dE, const double* dT, const double* hA, const double* hE,
                             const double* hT, const double* SA, const double* SE, const double* ST, double df,
                             const int64_t* edges, int64_t n_seg, double* out_seg) {
  const double* d[3] = {dA, dE, dT};
  const double* h[3] = {hA, hE, hT};
  const double* S[3] = {SA, SE, ST};
  double ups = 0.0;
  for (int64_t k = 0; k < n_seg; ++k) {
    double zr = 0.0, zi = 0.0, sig = 0.0;
    for (int64_t j = edges[k]; j < edges[k + 1]; ++j)
      for (int a = 0; a < 3; ++a) {
        zr += (d[a][2 * j] * h[a][2 * j] + d[a][2 * j + 1] * h[a][2 * j + 1]) / S[a][j];
        zi += (d[a][2 * j + 1] * h[a][2 * j] - d[a][2 * j] * h[a][2 * j + 1]) / S[a][j];
        sig += (h[a][2 * j] * h[a][2 * j] + h[a][2 * j + 1] * h[a][2 * j + 1]) / S[a][j];
      }
    if (out_seg) { out_seg[3 * k] = zr; out_seg[3 * k + 1] = zi; out_seg[3 * k + 2] = sig; }
    if (sig > 0.0) {
      const double x = 4.0 * df * sqrt(zr * zr + zi * zi);
      const double hh = 4.0 * df * sig;
      ups += x * x / hh;
    }
  }
  return ups;
}

double sco_inner3(const double* aA, const double* aE, const double* aT, const double* bA, const double* bE, const double* bT,
                  const double* SA, const double* SE, const double* ST, double df, int64_t n) {
  return sco_inner(aA, aE, bA, bE, SA, SE, df, n) + sco_inner(aT, NULL, bT, NULL, ST, NULL, df, n);
}

void sco_eval_stat3(const sco_config* c, const double* dA, const double* dE, const double* dT, const double* SA,
                    const double* SE, const double* ST, const double* params, int64_t P, const int64_t* edges,
                    int64_t n_seg, double* out, double* out_seg) {
  const int64_t n = c->n_bins;
  const double df = 1.0 / c->T_obs_s;
#pragma omp parallel
  {
    double* hA = (double*)malloc((size_t)n * 2 * sizeof(double));
    double* hE = (double*)malloc((size_t)n * 2 * sizeof(double));
    double* hT = (double*)malloc((size_t)n * 2 * sizeof(double));
#pragma omp for schedule(dynamic, 1)
    for (int64_t p = 0; p < P; ++p) {
      sco_template3(c, params + 8 * p, 0, n, hA, hE, hT);
      out[p] = sco_stat_from_arrays3(dA, dE, dT, hA, hE, hT, SA, SE, ST, df, edges, n_seg,
                                     out_seg ? out_seg + (size_t)p * (size_t)n_seg * 3 : NULL);
    }
    free(hA); free(hE); free(hT);
  }
}

/* Per-particle equal-SNR^2 segments over three channels (PAPER.md:120 with the channel sums of PAPER.md:36, 59):
 *   s_j = sum_{a in A,E,T} |h_a(f_j)|^2 / S_a(f_j),  then exactly the rule of sco_equal_snr_edges.  hT == NULL: two channels. */
void sco_equal_snr_edges3(const double* hA, const double* hE, const double* hT, const double* SA, const double* SE,
                          const double* ST, int64_t n_bins, int64_t n_seg, int64_t* edges) {
  double total = 0.0;
  for (int64_t j = 0; j < n_bins; ++j) {
    total += (hA[2 * j] * hA[2 * j] + hA[2 * j + 1] * hA[2 * j + 1]) / SA[j];
    total += (hE[2 * j] * hE[2 * j] + hE[2 * j + 1] * hE[2 * j + 1]) / SE[j];
    if (hT && ST) total += (hT[2 * j] * hT[2 * j] + hT[2 * j + 1] * hT[2 * j + 1]) / ST[j];
  }
  edges[0] = 0; edges[n_seg] = n_bins;
  double cum = 0.0;            /* C_j */
  int64_t j = 0;
  for (int64_t n = 1; n < n_seg; ++n) {
    const double target = total * (double)n / (double)n_seg;
    while (j < n_bins && !(cum >= target)) {
      cum += (hA[2 * j] * hA[2 * j] + hA[2 * j + 1] * hA[2 * j + 1]) / SA[j];
      cum += (hE[2 * j] * hE[2 * j] + hE[2 * j + 1] * hE[2 * j + 1]) / SE[j];
      if (hT && ST) cum += (hT[2 * j] * hT[2 * j] + hT[2 * j + 1] * hT[2 * j + 1]) / ST[j];
      ++j;
    }
    edges[n] = (total > 0.0) ? j : 0;
  }
}

/* Upsilon_N over three channels with per-particle equal-SNR^2 edges; in_edges / out_edges / out_comp3 as in
 * sco_eval_stat_adaptive. */
void sco_eval_stat_adaptive3(const sco_config* c, const double* dA, const double* dE, const double* dT, const double* SA,
                             const double* SE, const double* ST, const double* params, int64_t P, int64_t n_seg,
                             const int64_t* in_edges, double* out, int64_t* out_edges, double* out_comp3) {
  const int64_t n = c->n_bins;
  const double df = 1.0 / c->T_obs_s;
#pragma omp parallel
  {
    double* hA = (double*)malloc((size_t)n * 2 * sizeof(double));
    double* hE = (double*)malloc((size_t)n * 2 * sizeof(double));
    double* hT = (double*)malloc((size_t)n * 2 * sizeof(double));
    int64_t* e = (int64_t*)malloc((size_t)(n_seg + 1) * sizeof(int64_t));
    double* seg = (double*)malloc((size_t)n_seg * 3 * sizeof(double));
#pragma omp for schedule(dynamic, 1)
    for (int64_t p = 0; p < P; ++p) {
      sco_template3(c, params + 8 * p, 0, n, hA, hE, hT);
      if (in_edges) memcpy(e, in_edges + p * (n_seg + 1), (size_t)(n_seg + 1) * sizeof(int64_t));
      else sco_equal_snr_edges3(hA, hE, hT, SA, SE, ST, n, n_seg, e);
      out[p] = sco_stat_from_arrays3(dA, dE, dT, hA, hE, hT, SA, SE, ST, df, e, n_seg, seg);
      if (out_edges) memcpy(out_edges + p * (n_seg + 1), e, (size_t)(n_seg + 1) * sizeof(int64_t));
      if (out_comp3) sco_components_from_seg(seg, n_seg, df, out_comp3 + 3 * p);
    }
    free(hA); free(hE); free(hT); free(e); free(seg);
  }
}
