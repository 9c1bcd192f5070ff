/* ORACLE (test infrastructure).  Closed-form cross sections and stopping powers
 * that fill the tables ("tabulated discrete interaction cross
 * sections"; Table 2 names the models; the formulas are the
 * textbook readings listed in DESIGN.md section 3, R-C5).
 * kappa = E/me (photons); tau = T/me, gamma = tau+1, beta2 = 1-1/gamma^2 (e+-).
 */
#include <math.h>
#include "emo.h"

/* Coulomb correction f_c(Z) (Davies-Bethe-Maximon, 4-term form) */
double emo_fc(int Z) {
    double a = EMO_ALPHA * Z, a2 = a * a;
    return a2 * (1.0 / (1.0 + a2) + 0.20206 - 0.0369 * a2 + 0.0083 * a2 * a2 - 0.002 * a2 * a2 * a2);
}

/* radiation length of an element, g/cm2 (Tsai 1974 / PDG "Passage of particles") */
double emo_X0_elem_gcm2(int Z, double A) {
    double Lrad, Lprad;
    switch (Z) {
        case 1: Lrad = 5.31; Lprad = 6.144; break;
        case 2: Lrad = 4.79; Lprad = 5.621; break;
        case 3: Lrad = 4.74; Lprad = 5.805; break;
        case 4: Lrad = 4.71; Lprad = 5.924; break;
        default:
            Lrad = log(184.15 * pow((double)Z, -1.0 / 3.0));
            Lprad = log(1194.0 * pow((double)Z, -2.0 / 3.0));
    }
    double inv = 4.0 * EMO_ALPHA * EMO_RE * EMO_RE * (EMO_NA / A) *
                 ((double)Z * Z * (Lrad - emo_fc(Z)) + (double)Z * Lprad);
    return 1.0 / inv;
}

/* Klein-Nishina total cross section per electron, cm2.  The closed form
 * cancels badly at small kappa in fp64, so it is evaluated in x87 extended
 * precision (the definition itself, no series). */
double emo_sigma_kn(double E) {
    long double k = (long double)E / (long double)EMO_ME;
    long double L = log1pl(2.0L * k);
    long double a = (1.0L + k) / (k * k) * (2.0L * (1.0L + k) / (1.0L + 2.0L * k) - L / k);
    long double b = L / (2.0L * k);
    long double c = (1.0L + 3.0L * k) / ((1.0L + 2.0L * k) * (1.0L + 2.0L * k));
    long double s = 2.0L * 3.14159265358979323846264338327950288L * (long double)EMO_RE * (long double)EMO_RE * (a + b - c);
    return (double)s;
}

/* Photoelectric stand-in (R22): Born K-shell x 5/4, per atom, cm2 */
double emo_sigma_pe(int Z, double E) {
    double sT = 8.0 * EMO_PI * EMO_RE * EMO_RE / 3.0;
    double a4 = EMO_ALPHA * EMO_ALPHA * EMO_ALPHA * EMO_ALPHA;
    double z5 = (double)Z * Z * Z * Z * Z;
    return 1.25 * 4.0 * sqrt(2.0) * a4 * z5 * sT * pow(EMO_ME / E, 3.5);
}

/* Bethe-Heitler screening functions (Butcher-Messel parametrisation) */
static void screening(double delta, double *phi1, double *phi2) {
    if (delta <= 1.0) {
        *phi1 = 20.867 - 3.242 * delta + 0.625 * delta * delta;
        *phi2 = 20.209 - 1.930 * delta - 0.086 * delta * delta;
    } else {
        *phi1 = *phi2 = 21.12 - 4.184 * log(delta + 0.952);
    }
}
static double pair_F(int Z, double E) {
    double F = (8.0 / 3.0) * log((double)Z);
    if (E >= 50.0) F += 8.0 * emo_fc(Z);
    return F;
}
static double pair_xi(int Z) {
    return log(1440.0 * pow((double)Z, -2.0 / 3.0)) / (log(183.0 * pow((double)Z, -1.0 / 3.0)) - emo_fc(Z));
}

/* dsigma/deps per atom (eps = total lepton energy / E), clipped at 0 */
double emo_pair_dcs(int Z, double E, double eps) {
    double eps0 = EMO_ME / E;
    if (eps <= eps0 || eps >= 1.0 - eps0) return 0.0;
    double delta = 136.0 * pow((double)Z, -1.0 / 3.0) * eps0 / (eps * (1.0 - eps));
    double p1, p2;
    screening(delta, &p1, &p2);
    double F = pair_F(Z, E);
    double br = (eps * eps + (1.0 - eps) * (1.0 - eps)) * (p1 - 0.5 * F) +
                (2.0 / 3.0) * eps * (1.0 - eps) * (p2 - 0.5 * F);
    if (br < 0.0) br = 0.0;
    return EMO_ALPHA * EMO_RE * EMO_RE * (double)Z * ((double)Z + pair_xi(Z)) * br;
}

/* Gauss-Legendre nodes/weights on [-1,1] by Newton iteration on P_n */
void emo_gauss_legendre(int n, double *x, double *w) {
    for (int i = 0; i < n; ++i) {
        double z = cos(EMO_PI * (i + 0.75) / (n + 0.5));
        double pp = 0.0;
        for (int it = 0; it < 100; ++it) {
            double p1 = 1.0, p2 = 0.0;
            for (int j = 1; j <= n; ++j) {
                double p3 = p2; p2 = p1;
                p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j;
            }
            pp = n * (z * p1 - p2) / (z * z - 1.0);
            double dz = p1 / pp;
            z -= dz;
            if (fabs(dz) < 1e-16) break;
        }
        /* recompute derivative at the converged node */
        double p1 = 1.0, p2 = 0.0;
        for (int j = 1; j <= n; ++j) { double p3 = p2; p2 = p1; p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j; }
        pp = n * (z * p1 - p2) / (z * z - 1.0);
        x[n - 1 - i] = z;                 /* ascending order */
        w[n - 1 - i] = 2.0 / ((1.0 - z * z) * pp * pp);
    }
}

/* sigma_pair(Z,E) := 2 x (32-point Gauss-Legendre sum over eps in [eps0, 1/2]) -- table value by definition */
double emo_sigma_pair(int Z, double E) {
    static double gx[32], gw[32];
    static int init = 0;
    if (!init) {
#pragma omp critical(emo_gl32)
        { if (!init) { emo_gauss_legendre(32, gx, gw); init = 1; } }
    }
    if (E <= 2.0 * EMO_ME) return 0.0;
    double eps0 = EMO_ME / E;
    double half = 0.5 * (0.5 - eps0);
    double sum = 0.0;
    for (int q = 0; q < 32; ++q) {
        double eps = eps0 + half * (1.0 + gx[q]);
        sum += gw[q] * emo_pair_dcs(Z, E, eps);
    }
    return 2.0 * half * sum;
}

/* Moller, per electron; eps = T_delta/T in [x, 1/2] */
double emo_moller_dcs(double T, double eps) {
    double g = T / EMO_ME + 1.0, g2 = g * g, b2 = 1.0 - 1.0 / g2;
    double c = (2.0 * g - 1.0) / g2;
    double pre = 2.0 * EMO_PI * EMO_RE * EMO_RE / (b2 * (g - 1.0));
    return pre * ((g - 1.0) * (g - 1.0) / g2 + (1.0 / eps) * (1.0 / eps - c) +
                  (1.0 / (1.0 - eps)) * (1.0 / (1.0 - eps) - c));
}
double emo_sigma_moller(double T, double Tcut) {
    if (!(T > 2.0 * Tcut)) return 0.0;
    double x = Tcut / T;
    double g = T / EMO_ME + 1.0, g2 = g * g, b2 = 1.0 - 1.0 / g2;
    double pre = 2.0 * EMO_PI * EMO_RE * EMO_RE / (b2 * (g - 1.0));
    return pre * ((g - 1.0) * (g - 1.0) / g2 * (0.5 - x) + 1.0 / x - 1.0 / (1.0 - x) -
                  (2.0 * g - 1.0) / g2 * log((1.0 - x) / x));
}

/* Bhabha, per electron; eps in [x, 1] */
static void bhabha_B(double g, double *B1, double *B2, double *B3, double *B4) {
    double y = 1.0 / (g + 1.0), t = 1.0 - 2.0 * y;
    *B1 = 2.0 - y * y;
    *B2 = t * (3.0 + y * y);
    *B4 = t * t * t;
    *B3 = t * t + *B4;
}
double emo_bhabha_dcs(double T, double eps) {
    double g = T / EMO_ME + 1.0, b2 = 1.0 - 1.0 / (g * g), B1, B2, B3, B4;
    bhabha_B(g, &B1, &B2, &B3, &B4);
    double pre = 2.0 * EMO_PI * EMO_RE * EMO_RE / (g - 1.0);
    return pre * (1.0 / (b2 * eps * eps) - B1 / eps + B2 - B3 * eps + B4 * eps * eps);
}
double emo_sigma_bhabha(double T, double Tcut) {
    if (!(T > Tcut)) return 0.0;
    double x = Tcut / T;
    double g = T / EMO_ME + 1.0, b2 = 1.0 - 1.0 / (g * g), B1, B2, B3, B4;
    bhabha_B(g, &B1, &B2, &B3, &B4);
    double pre = 2.0 * EMO_PI * EMO_RE * EMO_RE / (g - 1.0);
    return pre * ((1.0 / b2) * (1.0 / x - 1.0) + B1 * log(x) + B2 * (1.0 - x) -
                  0.5 * B3 * (1.0 - x * x) + (B4 / 3.0) * (1.0 - x * x * x));
}

/* two-photon annihilation in flight (Heitler), per electron */
double emo_sigma_annih(double T) {
    double g = T / EMO_ME + 1.0, s = sqrt(g * g - 1.0);
    return EMO_PI * EMO_RE * EMO_RE / (g + 1.0) *
           ((g * g + 4.0 * g + 1.0) / (g * g - 1.0) * log(g + s) - (g + 3.0) / s);
}

/* complete-screening bremsstrahlung (R22): dSigma/dk = (1/X0)(1/k)(4/3 - 4y/3 + y^2) */
double emo_brems_Sigma(double T, double kc, double X0) {
    if (!(T > kc)) return 0.0;
    double u = kc / T;
    return (1.0 / X0) * ((4.0 / 3.0) * log(1.0 / u) - (4.0 / 3.0) * (1.0 - u) + 0.5 * (1.0 - u * u));
}
double emo_brems_dedx(double T, double kc, double X0) {
    double u = (kc <= 0.0 || kc > T) ? 1.0 : kc / T;     /* kc<=0: unrestricted */
    return (T / X0) * ((4.0 / 3.0) * u - (2.0 / 3.0) * u * u + (1.0 / 3.0) * u * u * u);
}

/* restricted collision stopping power (Berger-Seltzer / ICRU 37), MeV/cm.
 * Tcut <= 0 means unrestricted (tau_up = tau/2 for e-, tau for e+). */
double emo_dedx_col(const emo_material *m, int ptype, double T, double Tcut) {
    double tau = T / EMO_ME, g = tau + 1.0, g2 = g * g, b2 = 1.0 - 1.0 / g2;
    double tmax = (ptype == EMO_ELECTRON) ? 0.5 * tau : tau;
    double tup = tmax;
    if (Tcut > 0.0) { double tc = Tcut / EMO_ME; if (tc < tup) tup = tc; }
    double Im = m->I / EMO_ME;
    double lg = log(2.0 * (g + 1.0) / (Im * Im));
    double F;
    if (ptype == EMO_ELECTRON) {
        F = -1.0 - b2 + log((tau - tup) * tup) + tau / (tau - tup) +
            (1.0 / g2) * (0.5 * tup * tup + (2.0 * tau + 1.0) * log(1.0 - tup / tau));
    } else {
        double y = 1.0 / (g + 1.0);
        double t2 = tup * tup, t3 = t2 * tup, t4 = t3 * tup;
        F = log(tau * tup) - (b2 / tau) * (tau + 2.0 * tup - 1.5 * t2 * y - (tup - t3 / 3.0) * y * y -
                                           (0.5 * t2 - tau * t3 / 3.0 + 0.25 * t4) * y * y * y);
    }
    /* density effect: truncated high-energy asymptote (R23) */
    double bg = sqrt(b2) * g;
    double del = 2.0 * log(m->hwp * bg / m->I) - 1.0;
    if (del < 0.0) del = 0.0;
    return 2.0 * EMO_PI * EMO_RE * EMO_RE * EMO_ME * m->n_e / b2 * (lg + F - del);
}

/* ---- multiple scattering of e+- (PAPER.md:111 names Urban / WentzelVI, "in progress", no formulas;
 * DESIGN.md R-MSC is the reading) ----
 * Single elastic scattering: screened Rutherford (Wentzel) per atom,
 *   dsigma/dOmega = Z (Z + 1) r_e^2 (m_e c^2 / (beta p c))^2 / (1 - cos(theta) + 2 A)^2
 * (Z + 1 instead of Z: scattering off the atomic electrons), with Moliere's screening parameter
 *   A = (hbar / (2 p a_TF))^2 (1.13 + 3.76 (alpha Z / beta)^2),  a_TF = 0.88534 a_0 Z^(-1/3),
 * i.e. hbar / (p a_TF) = alpha Z^(1/3) m_e c^2 / (0.88534 p c). */
double emo_msc_screening(int Z, double T) {
    double pc2 = T * (T + 2.0 * EMO_ME);                 /* (p c)^2 */
    double Et = T + EMO_ME;
    double beta2 = pc2 / (Et * Et);
    double h = EMO_ALPHA * cbrt((double)Z) * EMO_ME / 0.88534;
    double az = EMO_ALPHA * Z;
    return 0.25 * h * h / pc2 * (1.13 + 3.76 * az * az / beta2);
}

/* first transport cross section sigma_1 = Int (1 - cos(theta)) dsigma over 0 <= t = 1 - cos(theta) <= t_m.
 * The finite nucleus ends the Rutherford law at theta_max = hbar / (p R_N), R_N = 1.4 fm A^(1/3) (the sharp
 * cutoff of the textbook treatment, Jackson section 13.6): t_m = min(2, theta_max^2 / 2).  With
 * Int_0^t_m t / (t + 2A)^2 dt = ln(1 + t_m / (2A)) - t_m / (t_m + 2A):
 *   sigma_1 = 2 pi Z (Z + 1) r_e^2 (m_e c^2 / (beta p c))^2 (ln(1 + t_m / (2A)) - t_m / (t_m + 2A)) */
double emo_msc_sigma1(int Z, double Amass, double T) {
    double pc2 = T * (T + 2.0 * EMO_ME);
    double bpc = pc2 / (T + EMO_ME);                     /* beta p c */
    double A = emo_msc_screening(Z, T);
    double c = EMO_RE * EMO_ME / bpc;
    double lam = EMO_RE * EMO_ME / EMO_ALPHA;            /* hbar c, MeV cm */
    double RN = 1.4e-13 * cbrt(Amass);
    double tm = 0.5 * lam * lam / (pc2 * RN * RN);
    if (tm > 2.0) tm = 2.0;
    return 2.0 * EMO_PI * (double)Z * (Z + 1.0) * c * c * (log1p(tm / (2.0 * A)) - tm / (tm + 2.0 * A));
}

/* ---- DESIGN.md R-MSC2: what Lewis' theory (H. W. Lewis, Phys. Rev. 78 (1950) 526) fixes about the SPATIAL
 * displacement of a true path t in an unbounded medium of constant transport mean free paths lambda_1, lambda_2
 * (lambda_l^-1 = n Int (1 - P_l(cos theta)) dsigma), start at the origin along +z, tau = t / lambda_1,
 * kappa = lambda_1 / lambda_2:
 *   <z>         = lambda_1 (1 - exp(-tau))
 *   <x^2 + y^2> = (4 lambda_1^2 / 3) [ tau - (kappa + 1) / kappa + kappa / (kappa - 1) exp(-tau)
 *                                      - exp(-kappa tau) / (kappa (kappa - 1)) ]
 * Both hold for ANY single-scattering law.  The multiple-scattering step of the transport moves the track by <z>
 * along its direction instead of by t, and displaces it sideways so that the mean square displacement is Lewis'. */

/* second transport cross section of the screened Rutherford law of emo_msc_sigma1, same cutoff t_m:
 * 1 - P_2(mu) = (3/2)(1 - mu^2) = 3 t - (3/2) t^2, t = 1 - mu, and with
 *   I_1 = Int_0^t_m t   / (t + 2A)^2 dt = ln(1 + t_m / 2A) - t_m / (t_m + 2A)
 *   I_2 = Int_0^t_m t^2 / (t + 2A)^2 dt = t_m - 4A ln(1 + t_m / 2A) + 2A t_m / (t_m + 2A)
 * sigma_2 = 2 pi Z (Z + 1) r_e^2 (m_e c^2 / (beta p c))^2 (3 I_1 - (3/2) I_2) */
double emo_msc_sigma2(int Z, double Amass, double T) {
    double pc2 = T * (T + 2.0 * EMO_ME);
    double bpc = pc2 / (T + EMO_ME);
    double A = emo_msc_screening(Z, T);
    double c = EMO_RE * EMO_ME / bpc;
    double lam = EMO_RE * EMO_ME / EMO_ALPHA;
    double RN = 1.4e-13 * cbrt(Amass);
    double tm = 0.5 * lam * lam / (pc2 * RN * RN);
    if (tm > 2.0) tm = 2.0;
    double lg = log1p(tm / (2.0 * A)), fr = tm / (tm + 2.0 * A);
    double I1 = lg - fr;
    double I2 = tm - 4.0 * A * lg + 2.0 * A * fr;
    return 2.0 * EMO_PI * (double)Z * (Z + 1.0) * c * c * (3.0 * I1 - 1.5 * I2);
}

/* phi_3(x) = (x^2/2 - x + 1 - exp(-x)) / x^3 = 1/6 - x/24 + x^2/120 - ...: the plain expression loses everything to
 * cancellation for small x, so below x = 0.5 the series is summed (terms x^n / (n + 3)!, n <= 14: the next is below
 * 1e-19) */
double emo_msc_phi3(double x) {
    if (x < 0.5) {
        double s = 0.0, term = 1.0 / 6.0;
        for (int n = 0; n <= 14; ++n) { s += term; term *= -x / (double)(n + 4); }
        return s;
    }
    return (0.5 * x * x - x - expm1(-x)) / (x * x * x);
}

/* <z> = lambda_1 (1 - exp(-tau)) = t (1 - exp(-tau)) / tau */
double emo_msc_geom_length(double t, double il1) {
    double tau = t * il1;
    if (!(tau > 0.0)) return t;
    return t * (-expm1(-tau) / tau);
}

/* Lewis' <x^2 + y^2>.  The bracket is O(tau^3) for small tau: written with phi_3 it is
 *   tau^3 (kappa / (kappa - 1)) (kappa phi_3(kappa tau) - phi_3(tau)),
 * which does not cancel there (kappa > 1 for every forward-peaked law), and lambda_1^2 tau^3 = t^2 tau.  For
 * tau >= 1 it is the other way round -- the two phi_3 agree in their leading 1 / (2 x) and the printed form is the
 * well-conditioned one. */
double emo_msc_lateral_r2(double t, double il1, double il2) {
    double tau = t * il1;
    if (!(tau > 0.0) || !(il2 > il1)) return 0.0;
    double kap = il2 / il1;
    if (tau < 1.0)
        return (4.0 / 3.0) * t * t * tau * (kap / (kap - 1.0)) * (kap * emo_msc_phi3(kap * tau) - emo_msc_phi3(tau));
    double br = tau - (kap + 1.0) / kap + (kap * exp(-tau) - exp(-kap * tau) / kap) / (kap - 1.0);
    return (4.0 / 3.0) * br / (il1 * il1);
}

/* Deflection after a path s = tau lambda_1: Lewis' theory gives <cos(theta)> = exp(-tau) exactly; the angle is
 * drawn from the Henyey-Greenstein density p(mu) ~ (1 - g^2) / (1 + g^2 - 2 g mu)^(3/2), whose mean cosine is
 * g, with g = exp(-tau).  Inverse of its distribution function, xi = F(mu), written for 1 - mu so that nothing
 * cancels as g -> 1:  a = 1 - g,  S = (1 + g) a / (a + 2 g xi),  1 - mu = a (1 - xi) (S + a) / (a + 2 g xi). */
double emo_msc_one_minus_mu(double tau, double xi) {
    double g = exp(-tau), a = -expm1(-tau);
    double den = a + 2.0 * g * xi;
    double S = (1.0 + g) * a / den;
    double t = a * (1.0 - xi) * (S + a) / den;
    return t < 0.0 ? 0.0 : (t > 2.0 ? 2.0 : t);
}

/* ---- energy-loss fluctuations of e+- (DESIGN.md R-FLUCT; PAPER.md:111 lists "energy loss" with the e+-
 * processes, PAPER.md:114 (ii) continuous slowing down) ----
 * The collisions with energy transfer W below the production threshold make up the continuous loss; the
 * variance of their sum over a path s is s n_e Int_0^Tup W^2 (dsigma/dW) dW (Bohr; the collisions are
 * independent).  With eps = W/T and the Moller / Bhabha laws above (x = Tup/T):
 *   Moller:  T^2 pre [c0 x^3/3 + x + (x/(1-x) + x + 2 ln(1-x)) + c (x + ln(1-x))],  c0 = (g-1)^2/g^2, c = (2g-1)/g^2
 *   Bhabha:  T^2 pre [x/b2 - B1 x^2/2 + B2 x^3/3 - B3 x^4/4 + B4 x^5/5]
 * (term by term the integrals of eps^2 times the laws; leading term pre T^2 x = 2 pi re^2 me Tup / beta^2). */
double emo_loss_second_moment(int ptype, double T, double Tcut) {
    double g = T / EMO_ME + 1.0, g2 = g * g, b2 = 1.0 - 1.0 / g2;
    if (ptype == EMO_ELECTRON) {
        double x = Tcut / T;
        if (x > 0.5) x = 0.5;
        double pre = 2.0 * EMO_PI * EMO_RE * EMO_RE / (b2 * (g - 1.0));
        double c0 = (g - 1.0) * (g - 1.0) / g2, c = (2.0 * g - 1.0) / g2;
        double L = log1p(-x);
        return T * T * pre * (c0 * x * x * x / 3.0 + x + (x / (1.0 - x) + x + 2.0 * L) + c * (x + L));
    } else {
        double x = Tcut / T, B1, B2, B3, B4;
        if (x > 1.0) x = 1.0;
        bhabha_B(g, &B1, &B2, &B3, &B4);
        double pre = 2.0 * EMO_PI * EMO_RE * EMO_RE / (g - 1.0);
        double x2 = x * x;
        return T * T * pre * (x / b2 - 0.5 * B1 * x2 + B2 * x2 * x / 3.0 - 0.25 * B3 * x2 * x2 + 0.2 * B4 * x2 * x2 * x);
    }
}

/* The fluctuated loss of a step: normal about the mean dE with variance V (Box-Muller from the two uniforms:
 * z = sqrt(-2 ln xi1) cos(2 pi xi2)), kept inside [0, min(2 dE, E)] by clamping -- symmetric about the mean
 * unless the mean is more than half of E, so the mean loss stays dE. */
double emo_fluctuate_loss(double dE, double V, double E, double xi1, double xi2) {
    double z = sqrt(-2.0 * log(xi1)) * cos(2.0 * EMO_PI * xi2);
    double d = dE + sqrt(V) * z;
    double hi = 2.0 * dE < E ? 2.0 * dE : E;
    return d < 0.0 ? 0.0 : (d > hi ? hi : d);
}
