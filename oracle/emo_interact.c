/* ORACLE (test infrastructure).  Discrete interactors named in PAPER.md:110-111
 * (Table 2): Klein-Nishina Compton, photoelectric, Bethe-Heitler pair production,
 * bremsstrahlung, Moller/Bhabha ionisation, two-photon annihilation.  The paper
 * names the models only; each sampler below is the reading fixed in DESIGN.md
 * R-C6.  Draws are consumed strictly in the order written.
 */
#include <math.h>
#include "emo.h"

static void normalise(double v[3], const double fallback[3]) {
    double n = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
    if (n > 0.0) { v[0] /= n; v[1] /= n; v[2] /= n; }
    else { v[0] = fallback[0]; v[1] = fallback[1]; v[2] = fallback[2]; }
}

/* rotate u by polar cosine mu (sine s) and azimuth (cos cphi, sin sphi) */
static void rotate_cs(const double u[3], double mu, double s, double cphi, double sphi, double out[3]) {
    double rho2 = u[0] * u[0] + u[1] * u[1];
    if (rho2 > 1e-30) {
        double rho = sqrt(rho2);
        out[0] = u[0] * mu + s * (u[0] * u[2] * cphi - u[1] * sphi) / rho;
        out[1] = u[1] * mu + s * (u[1] * u[2] * cphi + u[0] * sphi) / rho;
        out[2] = u[2] * mu - s * rho * cphi;
    } else {
        out[0] = s * cphi; out[1] = s * sphi; out[2] = (u[2] > 0.0 ? mu : -mu);
    }
    normalise(out, u);
}

void emo_rotate(const double u[3], double mu, double phi, double out[3]) {
    double s = sqrt((1.0 - mu) * (1.0 + mu));
    rotate_cs(u, mu, s, cos(phi), sin(phi), out);
}

static double beta_of(double T) { return sqrt(T * (T + 2.0 * EMO_ME)) / (T + EMO_ME); }
static double clamp1(double m) { return m > 1.0 ? 1.0 : (m < -1.0 ? -1.0 : m); }

/* Exact inverse CDF of p(mu) ~ (1 - beta mu)^-2 (R30), returned as t = 1 - mu for a lepton of kinetic energy T:
 * mu = (v + beta) / (beta v + 1), v = 2 xi - 1, gives 1 - mu = (1 - beta)(1 - v) / (1 + beta v).  With
 * 1 - beta = 1 / (gamma^2 (1 + beta)) and 1 + beta v = (1 - beta) + 2 beta xi nothing cancels: the emission angle,
 * which is ~1/gamma, keeps full relative precision at every energy (forming 1 - mu from a
 * rounded mu loses a factor gamma^2). */
static double boosted_iso_t(double xi, double T) {
    double g = T / EMO_ME + 1.0, b = beta_of(T);
    double omb = 1.0 / (g * g * (1.0 + b));
    double t = 2.0 * omb * (1.0 - xi) / (omb + 2.0 * b * xi);
    return t < 0.0 ? 0.0 : (t > 2.0 ? 2.0 : t);
}
static double sin_of_t(double t) { double s2 = t * (2.0 - t); return s2 > 0.0 ? sqrt(s2) : 0.0; }

/* ---- Compton (Klein-Nishina) ---- */
void emo_compton(emo_rng *r, double E, const double u[3], double *E1, double u1[3], double *Te, double ue[3]) {
    double k = E / EMO_ME;
    double e0 = 1.0 / (1.0 + 2.0 * k);
    double a1 = -log(e0), a2 = 0.5 * (1.0 - e0 * e0);
    double eps, t;
    for (;;) {
        double x1 = emo_next(r), x2 = emo_next(r), x3 = emo_next(r);
        if (x1 * (a1 + a2) < a1) eps = exp(-a1 * x2);
        else eps = sqrt(e0 * e0 + (1.0 - e0 * e0) * x2);
        t = (1.0 - eps) / (k * eps);
        if (x3 <= 1.0 - eps * t * (2.0 - t) / (1.0 + eps * eps)) break;
    }
    double mu = 1.0 - t;
    double s2 = t * (2.0 - t);
    double s = s2 > 0.0 ? sqrt(s2) : 0.0;
    double phi = 2.0 * EMO_PI * emo_next(r);
    rotate_cs(u, mu, s, cos(phi), sin(phi), u1);
    *E1 = eps * E;
    *Te = E - *E1;
    /* momentum balance E u = E1 u1 + p_e u_e with u1 = mu u + s e: p_e u_e = (E - E1 mu) u - E1 s e, and
     * E - E1 mu = Te + E1 t carries no cancellation */
    rotate_cs(u, *Te + (*E1) * t, -(*E1) * s, cos(phi), sin(phi), ue);
}

/* ---- photoelectron direction: p(mu) ~ (1-mu^2)/(1-beta mu)^4 (Sauter, leading term) ---- */
void emo_photo_dir(emo_rng *r, double E, const double u[3], double ue[3]) {
    double g = E / EMO_ME + 1.0;
    double b = beta_of(E);
    double A = 1.0 / (g * g * b * (1.0 + b));
    double nu;
    for (;;) {
        double x1 = emo_next(r), x2 = emo_next(r);
        nu = 1.0 / (1.0 / A - x1 * (1.0 / A - 1.0 / (A + 2.0))) - A;
        if (x2 <= A * (2.0 + A) * nu * (2.0 - nu) / ((A + nu) * (A + nu))) break;
    }
    double s2 = nu * (2.0 - nu);
    double phi = 2.0 * EMO_PI * emo_next(r);
    rotate_cs(u, 1.0 - nu, s2 > 0.0 ? sqrt(s2) : 0.0, cos(phi), sin(phi), ue);
}

/* ---- Bethe-Heitler pair production on element Z ---- */
static void scr(double d, double *p1, double *p2) {
    if (d <= 1.0) { *p1 = 20.867 - 3.242 * d + 0.625 * d * d; *p2 = 20.209 - 1.930 * d - 0.086 * d * d; }
    else { *p1 = *p2 = 21.12 - 4.184 * log(d + 0.952); }
}
static double F1(double d, double F) { double a, b; scr(d, &a, &b); return 3.0 * a - b - F; }
static double F2(double d, double F) { double a, b; scr(d, &a, &b); return 1.5 * a + 0.5 * b - F; }

int emo_pair(emo_rng *r, int Z, double E, const double u[3], double *Tm, double um[3], double *Tp, double up[3]) {
    double e0 = EMO_ME / E;
    double c = 136.0 * pow((double)Z, -1.0 / 3.0) * e0;
    double F = (8.0 / 3.0) * log((double)Z);
    if (E >= 50.0) F += 8.0 * emo_fc(Z);
    double dmin = 4.0 * c;
    double dmax = exp((42.24 - F) / 8.368) - 0.952;
    if (!(E > 2.0 * EMO_ME) || dmin >= dmax) return 0;            /* null interaction */
    double e1 = 0.5 - 0.5 * sqrt(1.0 - dmin / dmax);
    double emin = e0 > e1 ? e0 : e1;
    double F10 = F1(dmin, F), F20 = F2(dmin, F);
    double N1 = (0.5 - emin) * (0.5 - emin) * F10, N2 = 1.5 * F20;
    double eps;
    for (;;) {
        double x1 = emo_next(r), x2 = emo_next(r), x3 = emo_next(r);
        if (x1 * (N1 + N2) < N1) {
            eps = 0.5 - (0.5 - emin) * cbrt(x2);
            if (x3 * F10 <= F1(c / (eps * (1.0 - eps)), F)) break;
        } else {
            eps = emin + (0.5 - emin) * x2;
            if (x3 * F20 <= F2(c / (eps * (1.0 - eps)), F)) break;
        }
    }
    double x4 = emo_next(r);
    double ee = (x4 < 0.5) ? eps : 1.0 - eps;                      /* electron's share */
    double tm = ee * E - EMO_ME;
    if (tm < 0.0) tm = 0.0;
    double tp = E - tm - 2.0 * EMO_ME;
    if (tp < 0.0) tp = 0.0;
    *Tm = tm; *Tp = tp;
    double t_m = boosted_iso_t(emo_next(r), tm);
    double t_p = boosted_iso_t(emo_next(r), tp);
    double phi = 2.0 * EMO_PI * emo_next(r);
    double cp = cos(phi), sp = sin(phi);
    rotate_cs(u, 1.0 - t_m, sin_of_t(t_m), cp, sp, um);
    rotate_cs(u, 1.0 - t_p, sin_of_t(t_p), -cp, -sp, up);
    return 1;
}

/* ---- bremsstrahlung, complete screening shape ---- */
int emo_brems(emo_rng *r, double T, double kc, const double u[3], double *k, double ug[3], double *T1, double u1[3]) {
    if (!(T > kc)) return 0;
    double lr = log(T / kc), kk;
    for (;;) {
        double x1 = emo_next(r), x2 = emo_next(r);
        kk = kc * exp(x1 * lr);
        if (kk > T) kk = T;
        double y = kk / T;
        if ((4.0 / 3.0) * x2 <= 4.0 / 3.0 - 4.0 * y / 3.0 + y * y) break;
    }
    double t = boosted_iso_t(emo_next(r), T), sn = sin_of_t(t);
    double phi = 2.0 * EMO_PI * emo_next(r);
    double cp = cos(phi), sp = sin(phi);
    rotate_cs(u, 1.0 - t, sn, cp, sp, ug);
    double p = sqrt(T * (T + 2.0 * EMO_ME));
    *k = kk; *T1 = T - kk;
    /* recoil p u - k u_gamma = (p - k mu) u - k s e, with p - k mu = (p - T) + T1 + k t and
     * p - T = 2 me T / (p + T): no difference of nearly equal numbers */
    rotate_cs(u, 2.0 * EMO_ME * T / (p + T) + *T1 + kk * t, -kk * sn, cp, sp, u1);
    return 1;
}

/* shared two-body kinematics for a knock-on electron of energy Td */
static void knock_on(emo_rng *r, double T, double Td, const double u[3], double ud[3], double *T1, double u1[3]) {
    double p = sqrt(T * (T + 2.0 * EMO_ME)), pd = sqrt(Td * (Td + 2.0 * EMO_ME));
    double mu = clamp1(Td * (T + 2.0 * EMO_ME) / (p * pd));
    /* sin^2 = 1 - mu^2 = 2 me (T - Td) / (T (Td + 2 me)) in closed form */
    double s2 = 2.0 * EMO_ME * (T - Td) / (T * (Td + 2.0 * EMO_ME));
    double sn = s2 > 0.0 ? sqrt(s2) : 0.0;
    double phi = 2.0 * EMO_PI * emo_next(r);
    double cp = cos(phi), sp = sin(phi);
    rotate_cs(u, mu, sn, cp, sp, ud);
    *T1 = T - Td;
    /* primary: p u - pd u_delta = (p - pd mu) u - pd s e, p - pd mu = (T - Td)(T + 2 me) / p */
    rotate_cs(u, (*T1) * (T + 2.0 * EMO_ME) / p, -pd * sn, cp, sp, u1);
}

/* ---- Moller ---- */
int emo_moller(emo_rng *r, double T, double Tcut, const double u[3], double *Td, double ud[3], double *T1, double u1[3]) {
    if (!(T > 2.0 * Tcut)) return 0;
    double x = Tcut / T, g = T / EMO_ME + 1.0, g2 = g * g;
    double c = (2.0 * g - 1.0) / g2, a = (g - 1.0) * (g - 1.0) / g2;
    double whalf = 0.25 * (a + 8.0 - 4.0 * c);
    double eps;
    for (;;) {
        double x1 = emo_next(r), x2 = emo_next(r);
        eps = x / (1.0 - x1 * (1.0 - 2.0 * x));
        double w = eps * eps * (a + (1.0 / eps) * (1.0 / eps - c) + (1.0 / (1.0 - eps)) * (1.0 / (1.0 - eps) - c));
        if (x2 * whalf <= w) break;
    }
    *Td = eps * T;
    knock_on(r, T, *Td, u, ud, T1, u1);
    return 1;
}

/* ---- Bhabha ---- */
int emo_bhabha(emo_rng *r, double T, double Tcut, const double u[3], double *Td, double ud[3], double *T1, double u1[3]) {
    if (!(T > Tcut)) return 0;
    double x = Tcut / T, g = T / EMO_ME + 1.0, b2 = 1.0 - 1.0 / (g * g);
    double y = 1.0 / (g + 1.0), t = 1.0 - 2.0 * y;
    double B1 = 2.0 - y * y, B2 = t * (3.0 + y * y), B4 = t * t * t, B3 = t * t + B4;
    double eps;
    for (;;) {
        double x1 = emo_next(r), x2 = emo_next(r);
        eps = x / (1.0 - x1 * (1.0 - x));
        if (x2 <= 1.0 - b2 * (B1 * eps - B2 * eps * eps + B3 * eps * eps * eps - B4 * eps * eps * eps * eps)) break;
    }
    *Td = eps * T;
    knock_on(r, T, *Td, u, ud, T1, u1);
    return 1;
}

/* ---- two-photon annihilation in flight (Heitler) ---- */
void emo_annih_flight(emo_rng *r, double T, const double u[3], double *k1, double u1[3], double *k2, double u2[3]) {
    double g = T / EMO_ME + 1.0;
    double rr = sqrt((g - 1.0) / (g + 1.0));
    double elo = 0.5 * (1.0 - rr), ehi = 0.5 * (1.0 + rr);
    double lr = log(ehi / elo), eps;
    for (;;) {
        double x1 = emo_next(r), x2 = emo_next(r);
        eps = elo * exp(x1 * lr);
        if (x2 <= 1.0 - eps + (2.0 * g * eps - 1.0) / (eps * (g + 1.0) * (g + 1.0))) break;
    }
    double Etot = T + 2.0 * EMO_ME;
    double kk = eps * Etot;
    double pg = sqrt(g * g - 1.0);                                  /* p / me */
    double mu = clamp1((eps * (g + 1.0) - 1.0) / (eps * pg));
    /* sin^2 = 1 - mu^2 = (2 (g + 1) eps (1 - eps) - 1) / (eps^2 (g^2 - 1)) in closed form */
    double s2 = (2.0 * (g + 1.0) * eps * (1.0 - eps) - 1.0) / (eps * eps * (g * g - 1.0));
    double sn = s2 > 0.0 ? sqrt(s2) : 0.0;
    double phi = 2.0 * EMO_PI * emo_next(r);
    double cp = cos(phi), sp = sin(phi);
    rotate_cs(u, mu, sn, cp, sp, u1);
    *k1 = kk; *k2 = Etot - kk;
    /* second photon: p u - k1 u1 = (p - k1 mu) u - k1 s e, p - k1 mu = me (g + 1) ((1 - eps)(g + 1) - 1) / sqrt(g^2 - 1) */
    rotate_cs(u, EMO_ME * (g + 1.0) * ((1.0 - eps) * (g + 1.0) - 1.0) / pg, -kk * sn, cp, sp, u2);
}

/* ---- annihilation at rest: two back-to-back me photons, isotropic ---- */
void emo_annih_rest(emo_rng *r, double u1[3], double u2[3]) {
    double xi = emo_next(r);
    double mu = 2.0 * xi - 1.0;
    double phi = 2.0 * EMO_PI * emo_next(r);
    double s = 2.0 * sqrt(xi * (1.0 - xi));                        /* sqrt((1 - mu)(1 + mu)) without the cancellation */
    u1[0] = s * cos(phi); u1[1] = s * sin(phi); u1[2] = mu;
    u2[0] = -u1[0]; u2[1] = -u1[1]; u2[2] = -u1[2];
}

/* ---- multiple-scattering deflection (DESIGN.md R-MSC) ----
 * tau = path length in units of the first transport mean free path.  Draws: xi_1 (polar), xi_2 (azimuth).
 * The sine comes from t = 1 - mu as sqrt(t (2 - t)), never from sqrt(1 - mu^2). */
void emo_msc_deflect(emo_rng *r, double tau, const double u[3], double out[3]) {
    double x1 = emo_next(r), x2 = emo_next(r);
    double t = emo_msc_one_minus_mu(tau, x1);
    double s2 = t * (2.0 - t);
    double phi = 2.0 * EMO_PI * x2;
    rotate_cs(u, 1.0 - t, s2 > 0.0 ? sqrt(s2) : 0.0, cos(phi), sin(phi), out);
}
