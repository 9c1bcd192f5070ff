// emx_xs.h -- closed-form cross sections and stopping powers evaluated by the table-builder kernels
// (step A11 of DESIGN.md; "tabulated discrete interaction cross sections"; PAPER.md:128
// imports them from Geant4, BASELINE.json configs[0] says "tabulated from closed forms").
// Formulas: DESIGN.md C3 (materials) and C5.1-C5.9.  kappa = E/me; tau = T/me, gamma = tau + 1.
#pragma once
#include "emx_core.h"
#include "emx_gl.h"

namespace emx {

// Coulomb correction f_c(Z), Davies-Bethe-Maximon 4-term form (C3)
EMX_HD double coulomb_fc(int Z) {
    const double a = kAlpha * Z, a2 = a * a;
    return a2 * (1.0 / (1.0 + a2) + 0.20206 - 0.0369 * a2 + 0.0083 * a2 * a2 - 0.002 * a2 * a2 * a2);
}

// radiation length of one element in g/cm2 (Tsai 1974; C3)
EMX_HD double X0_element(int Z, double A) {
    double Lrad, Lprad;
    if (Z == 1) { Lrad = 5.31; Lprad = 6.144; }
    else if (Z == 2) { Lrad = 4.79; Lprad = 5.621; }
    else if (Z == 3) { Lrad = 4.74; Lprad = 5.805; }
    else if (Z == 4) { Lrad = 4.71; Lprad = 5.924; }
    else {
        Lrad = log(184.15 * pow((double)Z, -1.0 / 3.0));
        Lprad = log(1194.0 * pow((double)Z, -2.0 / 3.0));
    }
    const double zz = (double)Z;
    return 1.0 / (4.0 * kAlpha * kRe * kRe * (kNa / A) * (zz * zz * (Lrad - coulomb_fc(Z)) + zz * Lprad));
}

// Klein-Nishina total cross section per electron, cm2 (C5.1).
// The closed form loses 1/kappa^2 digits to cancellation, so below kappa = 1 the same number is obtained
// as the integral of the Klein-Nishina differential cross section over eps = E'/E in [1/(1+2 kappa), 1],
//   dsigma/deps = pi re^2 / kappa * (eps + 1/eps - t (2 - t)),  t = (1 - eps) / (kappa eps),
// with the 32-point Gauss-Legendre rule (integrand analytic on the interval: converged far below 1 ulp).
EMX_HD double sigma_kn(double E) {
    const double k = E / kMe;
    if (k < 1.0) {
        const double e0 = 1.0 / (1.0 + 2.0 * k);
        const double half = 0.5 * (1.0 - e0);
        double sum = 0.0;
        for (int q = 0; q < 32; ++q) {
            const double eps = e0 + half * (1.0 + gl32_x(q));
            const double t = (1.0 - eps) / (k * eps);
            sum += gl32_w(q) * (eps + 1.0 / eps - t * (2.0 - t));
        }
        return kPi * kRe * kRe / k * (half * sum);
    }
    const double L = log1p(2.0 * k);
    const double a = (1.0 + k) / (k * k) * (2.0 * (1.0 + k) / (1.0 + 2.0 * k) - L / k);
    const double b = L / (2.0 * k);
    const double c = (1.0 + 3.0 * k) / ((1.0 + 2.0 * k) * (1.0 + 2.0 * k));
    return 2.0 * kPi * kRe * kRe * (a + b - c);
}

// photoelectric stand-in, per atom, cm2 (C5.2; R22)
EMX_HD double sigma_pe(int Z, double E) {
    const double sT = 8.0 * kPi * kRe * kRe / 3.0;
    const double a4 = kAlpha * kAlpha * kAlpha * kAlpha;
    const double zz = (double)Z;
    const double z5 = zz * zz * zz * zz * zz;
    return 1.25 * 4.0 * sqrt(2.0) * a4 * z5 * sT * pow(kMe / E, 3.5);
}

// Butcher-Messel screening functions (C5.3)
EMX_HD void screening(double d, double &phi1, double &phi2) {
    if (d <= 1.0) {
        phi1 = 20.867 - 3.242 * d + 0.625 * d * d;
        phi2 = 20.209 - 1.930 * d - 0.086 * d * d;
    } else {
        phi1 = phi2 = 21.12 - 4.184 * m_log(d + 0.952);
    }
}
EMX_HD double pair_F(int Z, double E) {
    double F = (8.0 / 3.0) * m_log((double)Z);
    if (E >= 50.0) F += 8.0 * coulomb_fc(Z);
    return F;
}

// Bethe-Heitler pair production per atom: 2 x GL32 sum of the clipped DCS over eps in [eps0, 1/2] (C5.3)
EMX_HD double sigma_pair(int Z, double E) {
    if (E <= 2.0 * kMe) return 0.0;
    const double zz = (double)Z;
    const double eps0 = kMe / E;
    const double c136 = 136.0 * pow(zz, -1.0 / 3.0) * eps0;
    const double F = pair_F(Z, E);
    const double xi = log(1440.0 * pow(zz, -2.0 / 3.0)) / (log(183.0 * pow(zz, -1.0 / 3.0)) - coulomb_fc(Z));
    const double pre = kAlpha * kRe * kRe * zz * (zz + xi);
    const double half = 0.5 * (0.5 - eps0);
    double sum = 0.0;
    for (int q = 0; q < 32; ++q) {
        const double eps = eps0 + half * (1.0 + gl32_x(q));
        double dcs = 0.0;
        if (eps > eps0 && eps < 1.0 - eps0) {
            const double delta = c136 / (eps * (1.0 - eps));
            double p1, p2;
            screening(delta, p1, p2);
            double br = (eps * eps + (1.0 - eps) * (1.0 - eps)) * (p1 - 0.5 * F) +
                        (2.0 / 3.0) * eps * (1.0 - eps) * (p2 - 0.5 * F);
            if (br < 0.0) br = 0.0;
            dcs = pre * br;
        }
        sum += gl32_w(q) * dcs;
    }
    return 2.0 * half * sum;
}

// Moller total per electron for delta-ray energies in [Tcut, T/2] (C5.5)
EMX_HD double sigma_moller(double T, double Tcut) {
    if (!(T > 2.0 * Tcut)) return 0.0;
    const double x = Tcut / T;
    const double g = T / kMe + 1.0, g2 = g * g, b2 = 1.0 - 1.0 / g2;
    const double pre = 2.0 * kPi * kRe * kRe / (b2 * (g - 1.0));
    return pre * ((g - 1.0) * (g - 1.0) / g2 * (0.5 - x) + 1.0 / x - 1.0 / (1.0 - x) -
                  (2.0 * g - 1.0) / g2 * log((1.0 - x) / x));
}

// Bhabha total per electron for delta-ray energies in [Tcut, T] (C5.6)
EMX_HD double sigma_bhabha(double T, double Tcut) {
    if (!(T > Tcut)) return 0.0;
    const double x = Tcut / T;
    const double g = T / kMe + 1.0, b2 = 1.0 - 1.0 / (g * g);
    const double y = 1.0 / (g + 1.0), t = 1.0 - 2.0 * y;
    const double B1 = 2.0 - y * y, B2 = t * (3.0 + y * y), B4 = t * t * t, B3 = t * t + B4;
    const double pre = 2.0 * kPi * kRe * kRe / (g - 1.0);
    return pre * ((1.0 / b2) * (1.0 / x - 1.0) + B1 * log(x) + B2 * (1.0 - x) - 0.5 * B3 * (1.0 - x * x) +
                  (B4 / 3.0) * (1.0 - x * x * x));
}

// two-photon annihilation in flight, Heitler, per electron (C5.7)
EMX_HD double sigma_annih(double T) {
    const double g = T / kMe + 1.0, s = sqrt(g * g - 1.0);
    return kPi * kRe * kRe / (g + 1.0) * ((g * g + 4.0 * g + 1.0) / (g * g - 1.0) * log(g + s) - (g + 3.0) / s);
}

// complete-screening bremsstrahlung: macroscopic cross section above kc and restricted radiative loss (C5.4)
EMX_HD double brems_Sigma(double T, double kc, double X0) {
    if (!(T > kc)) return 0.0;
    const double u = kc / T;
    return (1.0 / X0) * ((4.0 / 3.0) * log(1.0 / u) - (4.0 / 3.0) * (1.0 - u) + 0.5 * (1.0 - u * u));
}
EMX_HD double brems_dedx(double T, double kc, double X0) {
    const double u = (kc <= 0.0 || kc > T) ? 1.0 : kc / T;  // kc <= 0: unrestricted
    return (T / X0) * ((4.0 / 3.0) * u - (2.0 / 3.0) * u * u + (1.0 / 3.0) * u * u * u);
}

// restricted collision stopping power, Berger-Seltzer / ICRU 37, MeV/cm (C5.8).  Tcut <= 0: unrestricted.
EMX_HD double dedx_col(const Material &m, int ptype, double T, double Tcut) {
    const double tau = T / kMe, g = tau + 1.0, g2 = g * g, b2 = 1.0 - 1.0 / g2;
    double tup = (ptype == kElectron) ? 0.5 * tau : tau;
    if (Tcut > 0.0) {
        const double tc = Tcut / kMe;
        if (tc < tup) tup = tc;
    }
    const double Im = m.I / kMe;
    const double lg = log(2.0 * (g + 1.0) / (Im * Im));
    double F;
    if (ptype == kElectron) {
        F = -1.0 - b2 + log((tau - tup) * tup) + tau / (tau - tup) +
            (1.0 / g2) * (0.5 * tup * tup + (2.0 * tau + 1.0) * log(1.0 - tup / tau));
    } else {
        const double y = 1.0 / (g + 1.0);
        const double t2 = tup * tup, t3 = t2 * tup, t4 = t3 * tup;
        F = log(tau * tup) - (b2 / tau) * (tau + 2.0 * tup - 1.5 * t2 * y - (tup - t3 / 3.0) * y * y -
                                           (0.5 * t2 - tau * t3 / 3.0 + 0.25 * t4) * y * y * y);
    }
    // density effect: truncated high-energy asymptote (R23)
    const double bg = sqrt(b2) * g;
    double del = 2.0 * log(m.hwp * bg / m.I) - 1.0;
    if (del < 0.0) del = 0.0;
    return 2.0 * kPi * kRe * kRe * kMe * m.n_e / b2 * (lg + F - del);
}

// ---- energy-loss fluctuations (DESIGN.md R-FLUCT): second moment of the transfers W = eps T below the
// production threshold, Int_0^x eps^2 (dsigma/deps) deps T^2, cm2 MeV2 per electron, x = min(Tcut/T, 1/2 | 1).
// Moller law pre (c0 + 1/eps^2 - c/eps + 1/(1-eps)^2 - c/(1-eps)), Bhabha law pre (1/(b2 eps^2) - B1/eps + B2
// - B3 eps + B4 eps^2) (C5.5, C5.6), integrated term by term.
EMX_HD double loss_second_moment(int ptype, double T, double Tcut) {
    const double g = T / kMe + 1.0, g2 = g * g, b2 = 1.0 - 1.0 / g2;
    double x = Tcut / T;
    if (ptype == kElectron) {
        if (x > 0.5) x = 0.5;
        const double pre = 2.0 * kPi * kRe * kRe / (b2 * (g - 1.0));
        const double c0 = (g - 1.0) * (g - 1.0) / g2, c = (2.0 * g - 1.0) / g2;
        const double L = log1p(-x);
        return T * T * pre * (c0 * x * x * x / 3.0 + x + (x / (1.0 - x) + x + 2.0 * L) + c * (x + L));
    }
    if (x > 1.0) x = 1.0;
    const double y = 1.0 / (g + 1.0), t = 1.0 - 2.0 * y;
    const double B1 = 2.0 - y * y, B2 = t * (3.0 + y * y), B4 = t * t * t, B3 = t * t + B4;
    const double pre = 2.0 * kPi * kRe * kRe / (g - 1.0);
    const double x2 = x * x;
    return T * T * pre * (x / b2 - 0.5 * B1 * x2 + B2 * x2 * x / 3.0 - 0.25 * B3 * x2 * x2 + 0.2 * B4 * x2 * x2 * x);
}

// ---- multiple scattering of e+- (DESIGN.md R-MSC; PAPER.md:111 names the models, prints no formula) ----
// Screened Rutherford law per atom, dsigma/dOmega = Z (Z + 1) re^2 (me / (beta p))^2 / (t + 2 A)^2 with
// t = 1 - cos(theta); Moliere: 4 A = chi_0^2 (1.13 + 3.76 (alpha Z / beta)^2), chi_0 = hbar / (p a_TF),
// a_TF = 0.88534 a_0 Z^(-1/3).  Lengths via hbar c = re me / alpha and a_0 = re / alpha^2.
EMX_HD double msc_screening(int Z, double T) {
    const double p2 = T * (T + 2.0 * kMe);
    const double inv_beta2 = (T + kMe) * (T + kMe) / p2;
    const double az = kAlpha * (double)Z;
    const double chi0 = kAlpha * kMe * cbrt((double)Z) / (0.88534 * sqrt(p2));
    return 0.25 * chi0 * chi0 * (1.13 + 3.76 * az * az * inv_beta2);
}
// first transport cross section, cm2 per atom: the law integrated with weight t up to
// t_m = min(2, theta_max^2 / 2), theta_max = hbar / (p R_N), R_N = 1.4e-13 cm A^(1/3) (finite nucleus):
//   sigma_1 = 2 pi Z (Z + 1) (re me / (beta p))^2 (ln(1 + t_m / 2A) - t_m / (t_m + 2A))
EMX_HD double msc_sigma1(int Z, double Amass, double T) {
    const double p2 = T * (T + 2.0 * kMe);
    const double A2 = 2.0 * msc_screening(Z, T);
    const double hbarc = kRe * kMe / kAlpha;
    const double th_max = hbarc / (sqrt(p2) * 1.4e-13 * cbrt(Amass));
    double tm = 0.5 * th_max * th_max;
    if (tm > 2.0) tm = 2.0;
    const double c = kRe * kMe * (T + kMe) / p2;
    const double zz = (double)Z;
    return 2.0 * kPi * zz * (zz + 1.0) * c * c * (log1p(tm / A2) - tm / (tm + A2));
}

// ---- DESIGN.md R-MSC2: the spatial moments of Lewis' theory (Phys. Rev. 78 (1950) 526) for a true path t,
// tau = t / lambda_1, kappa = lambda_1 / lambda_2:  <z> = lambda_1 (1 - exp(-tau)),
// <x^2 + y^2> = (4 lambda_1^2 / 3) (tau - (kappa + 1) / kappa + kappa exp(-tau) / (kappa - 1) - exp(-kappa tau) / (kappa (kappa - 1)))
// second transport cross section, cm2 per atom: the law of msc_sigma1 integrated with weight
// 1 - P_2 = 3 t - (3/2) t^2 up to t_m:  I_1 = ln(1 + t_m / 2A) - t_m / (t_m + 2A),
// I_2 = t_m - 4A ln(1 + t_m / 2A) + 2A t_m / (t_m + 2A),  sigma_2 = 2 pi Z (Z + 1) (re me / (beta p))^2 (3 I_1 - 3 I_2 / 2)
EMX_HD double msc_sigma2(int Z, double Amass, double T) {
    const double p2 = T * (T + 2.0 * kMe);
    const double A2 = 2.0 * msc_screening(Z, T);
    const double hbarc = kRe * kMe / kAlpha;
    const double th_max = hbarc / (sqrt(p2) * 1.4e-13 * cbrt(Amass));
    double tm = 0.5 * th_max * th_max;
    if (tm > 2.0) tm = 2.0;
    const double c = kRe * kMe * (T + kMe) / p2;
    const double zz = (double)Z;
    const double lg = log1p(tm / A2), fr = tm / (tm + A2);
    const double I1 = lg - fr;
    const double I2 = tm - 2.0 * A2 * lg + A2 * fr;
    return 2.0 * kPi * zz * (zz + 1.0) * c * c * (3.0 * I1 - 1.5 * I2);
}
// phi_3(x) = (x^2 / 2 - x + 1 - exp(-x)) / x^3: series below x = 1/2 (the plain form cancels), 15 terms
EMX_HD double msc_phi3(double x) {
    if (x < 0.5) {
        double s = 0.0, term = 1.0 / 6.0;
        for (int n = 0; n <= 14; ++n) {
            s += term;
            term *= -x / (double)(n + 4);
        }
        return s;
    }
    return (0.5 * x * x - x - expm1(-x)) / (x * x * x);
}
EMX_HD double msc_geom_length(double t, double il1) {
    const double tau = t * il1;
    if (!(tau > 0.0)) return t;
    return t * (-expm1(-tau) / tau);
}
// <x^2 + y^2>: with phi_3 for tau < 1 (the printed bracket is O(tau^3) and cancels), as printed for tau >= 1
EMX_HD double msc_lateral_r2(double t, double il1, double il2) {
    const double tau = t * il1;
    if (!(tau > 0.0) || !(il2 > il1)) return 0.0;
    const double kap = il2 / il1;
    if (tau < 1.0) return (4.0 / 3.0) * t * t * tau * (kap / (kap - 1.0)) * (kap * msc_phi3(kap * tau) - msc_phi3(tau));
    const double br = tau - (kap + 1.0) / kap + (kap * exp(-tau) - exp(-kap * tau) / kap) / (kap - 1.0);
    return (4.0 / 3.0) * br / (il1 * il1);
}

EMX_HD double dedx_total(const Material &m, int ptype, double T, double Tcut, double kcut) {
    return dedx_col(m, ptype, T, Tcut) + brems_dedx(T, kcut, m.X0);
}

}  // namespace emx
