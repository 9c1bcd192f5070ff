// emx_interact.h -- the six discrete interactors of PAPER.md:110-111 (Table 2): Klein-Nishina Compton,
// photoelectric, Bethe-Heitler pair production, bremsstrahlung, Moller / Bhabha ionisation and
// two-photon annihilation (step A7 of DESIGN.md).  The paper names the models only; the samplers are
// the readings of DESIGN.md C6.  Uniforms are consumed strictly in the order written there.
#pragma once
#include "emx_core.h"
#include "emx_xs.h"

namespace emx {

EMX_HD void normalise(Vec3 &v, const Vec3 &fallback) {
    const double n = norm(v);
    if (n > 0.0) {
        v.x /= n;
        v.y /= n;
        v.z /= n;
    } else {
        v = fallback;
    }
}

EMX_HD void sincos_(double a, double &s, double &c) { m_sincos(a, s, c); }

// rotate u by polar cosine mu (sine s) and azimuth (cphi, sphi) -- C6 "Common"
EMX_NI Vec3 rotate(const Vec3 &u, double mu, double s, double cphi, double sphi) {
    Vec3 o;
    const double rho2 = u.x * u.x + u.y * u.y;
    if (rho2 > 1e-30) {
        const double rho = sqrt(rho2);
        o.x = u.x * mu + s * (u.x * u.z * cphi - u.y * sphi) / rho;
        o.y = u.y * mu + s * (u.y * u.z * cphi + u.x * sphi) / rho;
        o.z = u.z * mu - s * rho * cphi;
    } else {
        o.x = s * cphi;
        o.y = s * sphi;
        o.z = (u.z > 0.0 ? mu : -mu);
    }
    normalise(o, u);
    return o;
}
EMX_HD Vec3 rotate_mu_phi(const Vec3 &u, double mu, double phi) {
    double sp, cp;
    sincos_(phi, sp, cp);
    return rotate(u, mu, sqrt((1.0 - mu) * (1.0 + mu)), cp, sp);
}

EMX_HD double beta_of(double T) { return sqrt(T * (T + 2.0 * kMe)) / (T + kMe); }
EMX_HD double clamp1(double m) { return m > 1.0 ? 1.0 : (m < -1.0 ? -1.0 : m); }
// Exact inverse CDF of p(mu) ~ (1 - beta mu)^-2 (R30) for a lepton of kinetic energy T, as t = 1 - mu:
// mu = (v + beta) / (beta v + 1), v = 2 xi - 1  =>  t = (1 - beta)(1 - v) / (1 + beta v)
//    = 2 (1 - beta)(1 - xi) / ((1 - beta) + 2 beta xi),  1 - beta = 1 / (gamma^2 (1 + beta)).
// Nothing cancels, so the emission angle (~1/gamma) keeps its relative precision at every energy.
EMX_HD double boosted_iso_t(double xi, double T) {
    const double g = T / kMe + 1.0, b = beta_of(T);
    const double omb = 1.0 / (g * g * (1.0 + b));
    const double t = 2.0 * omb * (1.0 - xi) / (omb + 2.0 * b * xi);
    return t < 0.0 ? 0.0 : (t > 2.0 ? 2.0 : t);
}
EMX_HD double sin_of_t(double t) {
    const double s2 = t * (2.0 - t);
    return s2 > 0.0 ? sqrt(s2) : 0.0;
}

// ---- fluctuated continuous loss of a step (R-FLUCT): normal about the mean dE with variance V (Box-Muller:
// z = sqrt(-2 ln xi1) cos(2 pi xi2)), clamped to [0, min(2 dE, E)]
EMX_NI double fluctuate_loss(double dE, double V, double E, double xi1, double xi2) {
    double sp, cp;
    sincos_(2.0 * kPi * xi2, sp, cp);
    const double d = dE + sqrt(V) * (sqrt(-2.0 * m_log(xi1)) * cp);
    const double hi = 2.0 * dE < E ? 2.0 * dE : E;
    return d < 0.0 ? 0.0 : (d > hi ? hi : d);
}

// ---- multiple-scattering deflection after a path of tau transport mean free paths (R-MSC): polar angle from
// the Henyey-Greenstein law with mean cosine g = exp(-tau) (Lewis: <cos> = exp(-tau) exactly), azimuth uniform.
// Inverse distribution function written for t = 1 - mu so that nothing cancels as g -> 1:
//   a = 1 - g, S = (1 + g) a / (a + 2 g xi), t = a (1 - xi) (S + a) / (a + 2 g xi).   Draws: polar, azimuth.
EMX_HD double msc_one_minus_mu(double tau, double xi) {
    const double g = m_exp(-tau), a = -expm1(-tau);
    const double den = a + 2.0 * g * xi;
    const double S = (1.0 + g) * a / den;
    const double t = a * (1.0 - xi) * (S + a) / den;
    return t < 0.0 ? 0.0 : (t > 2.0 ? 2.0 : t);
}
EMX_NI Vec3 msc_deflect(Rng &r, double tau, const Vec3 &u) {
    const double x1 = r.next(), x2 = r.next();
    const double t = msc_one_minus_mu(tau, x1);
    const double s2 = t * (2.0 - t);
    double sp, cp;
    sincos_(2.0 * kPi * x2, sp, cp);
    return rotate(u, 1.0 - t, s2 > 0.0 ? sqrt(s2) : 0.0, cp, sp);
}

// ---- Compton, Klein-Nishina (C6.1): photon E -> E1 along u1, electron Te along ue
EMX_NI void compton(Rng &r, double E, const Vec3 &u, double &E1, Vec3 &u1, double &Te, Vec3 &ue) {
    const double k = E / kMe;
    const double e0 = 1.0 / (1.0 + 2.0 * k);
    const double a1 = -m_log(e0), a2 = 0.5 * (1.0 - e0 * e0);
    double eps, t;
    for (;;) {
        const double x1 = r.next(), x2 = r.next(), x3 = r.next();
        if (x1 * (a1 + a2) < a1) eps = m_exp(-a1 * x2);
        else eps = sqrt(e0 * e0 + (1.0 - e0 * e0) * x2);
        t = (1.0 - eps) / (k * eps);
        if (x3 <= 1.0 - eps * t * (2.0 - t) / (1.0 + eps * eps)) break;
    }
    const double mu = 1.0 - t;
    const double s2 = t * (2.0 - t);
    const double s = s2 > 0.0 ? sqrt(s2) : 0.0;
    double sp, cp;
    sincos_(2.0 * kPi * r.next(), sp, cp);
    u1 = rotate(u, mu, s, cp, sp);
    E1 = eps * E;
    Te = E - E1;
    // momentum balance E u = E1 u1 + p_e u_e with u1 = mu u + s e: p_e u_e = (E - E1 mu) u - E1 s e, and
    // E - E1 mu = Te + E1 t carries no cancellation
    ue = rotate(u, Te + E1 * t, -E1 * s, cp, sp);
}

// ---- photoelectron direction, leading Sauter term p(mu) ~ (1 - mu^2) / (1 - beta mu)^4 (C6.2)
EMX_NI Vec3 photo_dir(Rng &r, double E, const Vec3 &u) {
    const double g = E / kMe + 1.0;
    const double b = beta_of(E);
    const double A = 1.0 / (g * g * b * (1.0 + b));
    double nu;
    for (;;) {
        const double x1 = r.next(), x2 = r.next();
        nu = 1.0 / (1.0 / A - x1 * (1.0 / A - 1.0 / (A + 2.0))) - A;
        if (x2 <= A * (2.0 + A) * nu * (2.0 - nu) / ((A + nu) * (A + nu))) break;
    }
    const double s2 = nu * (2.0 - nu);
    double sp, cp;
    sincos_(2.0 * kPi * r.next(), sp, cp);
    return rotate(u, 1.0 - nu, s2 > 0.0 ? sqrt(s2) : 0.0, cp, sp);
}

// ---- Bethe-Heitler pair production on element Z (C6.3).  false = null interaction.
EMX_HD double pair_F1(double d, double F) {
    double a, b;
    screening(d, a, b);
    return 3.0 * a - b - F;
}
EMX_HD double pair_F2(double d, double F) {
    double a, b;
    screening(d, a, b);
    return 1.5 * a + 0.5 * b - F;
}
EMX_NI bool pair_production(Rng &r, int Z, double E, const Vec3 &u, double &Tm, Vec3 &um, double &Tp, Vec3 &up) {
    const double e0 = kMe / E;
    const double c = 136.0 * m_pow((double)Z, -1.0 / 3.0) * e0;
    const double F = pair_F(Z, E);
    const double dmin = 4.0 * c;
    const double dmax = m_exp((42.24 - F) / 8.368) - 0.952;
    if (!(E > 2.0 * kMe) || dmin >= dmax) return false;
    const double e1 = 0.5 - 0.5 * sqrt(1.0 - dmin / dmax);
    const double emin = e0 > e1 ? e0 : e1;
    const double F10 = pair_F1(dmin, F), F20 = pair_F2(dmin, F);
    const double N1 = (0.5 - emin) * (0.5 - emin) * F10, N2 = 1.5 * F20;
    double eps;
    for (;;) {
        const double x1 = r.next(), x2 = r.next(), x3 = r.next();
        if (x1 * (N1 + N2) < N1) {
            eps = 0.5 - (0.5 - emin) * m_cbrt(x2);
            if (x3 * F10 <= pair_F1(c / (eps * (1.0 - eps)), F)) break;
        } else {
            eps = emin + (0.5 - emin) * x2;
            if (x3 * F20 <= pair_F2(c / (eps * (1.0 - eps)), F)) break;
        }
    }
    const double x4 = r.next();
    const double ee = (x4 < 0.5) ? eps : 1.0 - eps;  // the electron's share
    double tm = ee * E - kMe;
    if (tm < 0.0) tm = 0.0;
    double tp = E - tm - 2.0 * kMe;
    if (tp < 0.0) tp = 0.0;
    Tm = tm;
    Tp = tp;
    const double t_m = boosted_iso_t(r.next(), tm);
    const double t_p = boosted_iso_t(r.next(), tp);
    double sp, cp;
    sincos_(2.0 * kPi * r.next(), sp, cp);
    um = rotate(u, 1.0 - t_m, sin_of_t(t_m), cp, sp);
    up = rotate(u, 1.0 - t_p, sin_of_t(t_p), -cp, -sp);
    return true;
}

// ---- bremsstrahlung, complete-screening shape (C6.4).  false = null (T <= kc).
EMX_NI bool bremsstrahlung(Rng &r, double T, double kc, const Vec3 &u, double &k, Vec3 &ug, double &T1, Vec3 &u1) {
    if (!(T > kc)) return false;
    const double lr = m_log(T / kc);
    double kk;
    for (;;) {
        const double x1 = r.next(), x2 = r.next();
        kk = kc * m_exp(x1 * lr);
        if (kk > T) kk = T;
        const double y = kk / T;
        if ((4.0 / 3.0) * x2 <= 4.0 / 3.0 - 4.0 * y / 3.0 + y * y) break;
    }
    const double t = boosted_iso_t(r.next(), T), sn = sin_of_t(t);
    double sp, cp;
    sincos_(2.0 * kPi * r.next(), sp, cp);
    ug = rotate(u, 1.0 - t, sn, cp, sp);
    const double p = sqrt(T * (T + 2.0 * kMe));
    k = kk;
    T1 = T - kk;
    // recoil p u - k u_gamma = (p - k mu) u - k s e, with p - k mu = (p - T) + T1 + k t and
    // p - T = 2 me T / (p + T): no difference of nearly equal numbers
    u1 = rotate(u, 2.0 * kMe * T / (p + T) + T1 + kk * t, -kk * sn, cp, sp);
    return true;
}

// exact two-body kinematics of a knock-on electron of energy Td on a free electron at rest (C6.5)
EMX_NI void knock_on(Rng &r, double T, double Td, const Vec3 &u, Vec3 &ud, double &T1, Vec3 &u1) {
    const double p = sqrt(T * (T + 2.0 * kMe)), pd = sqrt(Td * (Td + 2.0 * kMe));
    const double mu = clamp1(Td * (T + 2.0 * kMe) / (p * pd));
    // sin^2 = 1 - mu^2 = 2 me (T - Td) / (T (Td + 2 me)) in closed form
    const double s2 = 2.0 * kMe * (T - Td) / (T * (Td + 2.0 * kMe));
    const double sn = s2 > 0.0 ? sqrt(s2) : 0.0;
    double sp, cp;
    sincos_(2.0 * kPi * r.next(), sp, cp);
    ud = rotate(u, mu, sn, cp, sp);
    T1 = T - Td;
    // primary: p u - pd u_delta = (p - pd mu) u - pd s e, p - pd mu = (T - Td)(T + 2 me) / p
    u1 = rotate(u, T1 * (T + 2.0 * kMe) / p, -pd * sn, cp, sp);
}

EMX_NI bool moller(Rng &r, double T, double Tcut, const Vec3 &u, double &Td, Vec3 &ud, double &T1, Vec3 &u1) {
    if (!(T > 2.0 * Tcut)) return false;
    const double x = Tcut / T, g = T / kMe + 1.0, g2 = g * g;
    const double c = (2.0 * g - 1.0) / g2, a = (g - 1.0) * (g - 1.0) / g2;
    const double whalf = 0.25 * (a + 8.0 - 4.0 * c);
    double eps;
    for (;;) {
        const double x1 = r.next(), x2 = r.next();
        eps = x / (1.0 - x1 * (1.0 - 2.0 * x));
        const double w = eps * eps * (a + (1.0 / eps) * (1.0 / eps - c) + (1.0 / (1.0 - eps)) * (1.0 / (1.0 - eps) - c));
        if (x2 * whalf <= w) break;
    }
    Td = eps * T;
    knock_on(r, T, Td, u, ud, T1, u1);
    return true;
}

EMX_NI bool bhabha(Rng &r, double T, double Tcut, const Vec3 &u, double &Td, Vec3 &ud, double &T1, Vec3 &u1) {
    if (!(T > Tcut)) return false;
    const double x = Tcut / T, g = T / kMe + 1.0, b2 = 1.0 - 1.0 / (g * g);
    const double y = 1.0 / (g + 1.0), t = 1.0 - 2.0 * y;
    const double B1 = 2.0 - y * y, B2 = t * (3.0 + y * y), B4 = t * t * t, B3 = t * t + B4;
    double eps;
    for (;;) {
        const double x1 = r.next(), x2 = r.next();
        eps = x / (1.0 - x1 * (1.0 - x));
        if (x2 <= 1.0 - b2 * (B1 * eps - B2 * eps * eps + B3 * eps * eps * eps - B4 * eps * eps * eps * eps)) break;
    }
    Td = eps * T;
    knock_on(r, T, Td, u, ud, T1, u1);
    return true;
}

// ---- two-photon annihilation in flight, Heitler (C6.6)
EMX_NI void annih_flight(Rng &r, double T, const Vec3 &u, double &k1, Vec3 &u1, double &k2, Vec3 &u2) {
    const double g = T / kMe + 1.0;
    const double rr = sqrt((g - 1.0) / (g + 1.0));
    const double elo = 0.5 * (1.0 - rr), ehi = 0.5 * (1.0 + rr);
    const double lr = m_log(ehi / elo);
    double eps;
    for (;;) {
        const double x1 = r.next(), x2 = r.next();
        eps = elo * m_exp(x1 * lr);
        if (x2 <= 1.0 - eps + (2.0 * g * eps - 1.0) / (eps * (g + 1.0) * (g + 1.0))) break;
    }
    const double Etot = T + 2.0 * kMe;
    const double kk = eps * Etot;
    const double pg = sqrt(g * g - 1.0);  // p / me
    const double mu = clamp1((eps * (g + 1.0) - 1.0) / (eps * pg));
    // sin^2 = 1 - mu^2 = (2 (g + 1) eps (1 - eps) - 1) / (eps^2 (g^2 - 1)) in closed form
    const double s2 = (2.0 * (g + 1.0) * eps * (1.0 - eps) - 1.0) / (eps * eps * (g * g - 1.0));
    const double sn = s2 > 0.0 ? sqrt(s2) : 0.0;
    double sp, cp;
    sincos_(2.0 * kPi * r.next(), sp, cp);
    u1 = rotate(u, mu, sn, cp, sp);
    k1 = kk;
    k2 = Etot - kk;
    // second photon: p u - k1 u1 = (p - k1 mu) u - k1 s e, p - k1 mu = me (g + 1) ((1 - eps)(g + 1) - 1) / sqrt(g^2 - 1)
    u2 = rotate(u, kMe * (g + 1.0) * ((1.0 - eps) * (g + 1.0) - 1.0) / pg, -kk * sn, cp, sp);
}

// ---- annihilation at rest: two back-to-back me photons, isotropic (C6.6, R12/R25)
EMX_NI void annih_rest(Rng &r, Vec3 &u1, Vec3 &u2) {
    const double xi = r.next();
    const double mu = 2.0 * xi - 1.0;
    double sp, cp;
    sincos_(2.0 * kPi * r.next(), sp, cp);
    const double s = 2.0 * sqrt(xi * (1.0 - xi));  // sqrt((1 - mu)(1 + mu)) without the cancellation
    u1 = {s * cp, s * sp, mu};
    u2 = {-u1.x, -u1.y, -u1.z};
}

}  // namespace emx
