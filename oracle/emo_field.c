/* ORACLE (test infrastructure).  Charged-track propagation in a uniform magnetic
 * field, or in a solenoid field with a fringe ("on-device propagation of particles through arbitrary
 * magnetic fields ... different integration algorithms"; BASELINE.json
 * configs[3]: "adaptive RK4 (1e-6 mm miss-distance tolerance)").  The paper gives
 * no algorithm: classical RK4 with step doubling (Press et al.) plus a chord /
 * secant boundary search -> DESIGN.md R-C9.
 * State y = (x, u);  dy/ds = (u, kappa u x Bhat),  kappa = q*CB*|B|/p.
 */
#include <math.h>
#include "emo.h"

static void rhs(const double u[3], double kappa, const double B[3], double dx[3], double du[3]) {
    dx[0] = u[0]; dx[1] = u[1]; dx[2] = u[2];
    du[0] = kappa * (u[1] * B[2] - u[2] * B[1]);
    du[1] = kappa * (u[2] * B[0] - u[0] * B[2]);
    du[2] = kappa * (u[0] * B[1] - u[1] * B[0]);
}

static void rk4(const double x[3], const double u[3], double kappa, const double B[3], double h,
                double xo[3], double uo[3]) {
    double k1x[3], k1u[3], k2x[3], k2u[3], k3x[3], k3u[3], k4x[3], k4u[3], ut[3];
    rhs(u, kappa, B, k1x, k1u);
    for (int i = 0; i < 3; ++i) ut[i] = u[i] + 0.5 * h * k1u[i];
    rhs(ut, kappa, B, k2x, k2u);
    for (int i = 0; i < 3; ++i) ut[i] = u[i] + 0.5 * h * k2u[i];
    rhs(ut, kappa, B, k3x, k3u);
    for (int i = 0; i < 3; ++i) ut[i] = u[i] + h * k3u[i];
    rhs(ut, kappa, B, k4x, k4u);
    for (int i = 0; i < 3; ++i) {
        xo[i] = x[i] + (h / 6.0) * (k1x[i] + 2.0 * k2x[i] + 2.0 * k3x[i] + k4x[i]);
        uo[i] = u[i] + (h / 6.0) * (k1u[i] + 2.0 * k2u[i] + 2.0 * k3u[i] + k4u[i]);
    }
}

/* one step of h versus two of h/2; err = |x_full - x_half|; result = the two-half-step
 * state with u renormalised */
void emo_rk4_doubling(const double x[3], const double u[3], double kappa, const double B[3], double h,
                      double x1[3], double u1[3], double *err) {
    double xf[3], uf[3], xm[3], um[3];
    rk4(x, u, kappa, B, h, xf, uf);
    rk4(x, u, kappa, B, 0.5 * h, xm, um);
    rk4(xm, um, kappa, B, 0.5 * h, x1, u1);
    double dx = xf[0] - x1[0], dy = xf[1] - x1[1], dz = xf[2] - x1[2];
    *err = sqrt(dx * dx + dy * dy + dz * dz);
    double n = sqrt(u1[0] * u1[0] + u1[1] * u1[1] + u1[2] * u1[2]);
    u1[0] /= n; u1[1] /= n; u1[2] /= n;
}

/* ---- non-uniform field: the same integrator with the field taken at the stage positions ---- */
void emo_field_profile(const emo_problem *p, const double x[3], double g[3]) {
    if (p->field_kind == 0) { g[0] = p->Bhat[0]; g[1] = p->Bhat[1]; g[2] = p->Bhat[2]; return; }
    const double az = fabs(x[2]);
    const double f = 1.0 / (1.0 + exp((az - p->fringe_z0) / p->fringe_a));
    const double sg = x[2] > 0.0 ? 1.0 : (x[2] < 0.0 ? -1.0 : 0.0);
    const double fp = -sg * f * (1.0 - f) / p->fringe_a;
    g[0] = -0.5 * x[0] * fp * p->Bhat[2];
    g[1] = -0.5 * x[1] * fp * p->Bhat[2];
    g[2] = f * p->Bhat[2];
}

static void rk4_map(const emo_problem *p, const double x[3], const double u[3], double kappa, double h,
                    double xo[3], double uo[3]) {
    double g[3], k1x[3], k1u[3], k2x[3], k2u[3], k3x[3], k3u[3], k4x[3], k4u[3], xt[3], ut[3];
    emo_field_profile(p, x, g);
    rhs(u, kappa, g, k1x, k1u);
    for (int i = 0; i < 3; ++i) { xt[i] = x[i] + 0.5 * h * k1x[i]; ut[i] = u[i] + 0.5 * h * k1u[i]; }
    emo_field_profile(p, xt, g);
    rhs(ut, kappa, g, k2x, k2u);
    for (int i = 0; i < 3; ++i) { xt[i] = x[i] + 0.5 * h * k2x[i]; ut[i] = u[i] + 0.5 * h * k2u[i]; }
    emo_field_profile(p, xt, g);
    rhs(ut, kappa, g, k3x, k3u);
    for (int i = 0; i < 3; ++i) { xt[i] = x[i] + h * k3x[i]; ut[i] = u[i] + h * k3u[i]; }
    emo_field_profile(p, xt, g);
    rhs(ut, kappa, g, k4x, k4u);
    for (int i = 0; i < 3; ++i) {
        xo[i] = x[i] + (h / 6.0) * (k1x[i] + 2.0 * k2x[i] + 2.0 * k3x[i] + k4x[i]);
        uo[i] = u[i] + (h / 6.0) * (k1u[i] + 2.0 * k2u[i] + 2.0 * k3u[i] + k4u[i]);
    }
}

void emo_rk4_doubling_map(const emo_problem *p, const double x[3], const double u[3], double kappa, double h,
                          double x1[3], double u1[3], double *err) {
    double xf[3], uf[3], xm[3], um[3];
    rk4_map(p, x, u, kappa, h, xf, uf);
    rk4_map(p, x, u, kappa, 0.5 * h, xm, um);
    rk4_map(p, xm, um, kappa, 0.5 * h, x1, u1);
    double dx = xf[0] - x1[0], dy = xf[1] - x1[1], dz = xf[2] - x1[2];
    *err = sqrt(dx * dx + dy * dy + dz * dz);
    double n = sqrt(u1[0] * u1[0] + u1[1] * u1[1] + u1[2] * u1[2]);
    u1[0] /= n; u1[1] /= n; u1[2] /= n;
}

/* ---- second integrator (DESIGN.md R-INT; "different integration algorithms"): the embedded pair of
 * Dormand and Prince, J. Comput. Appl. Math. 6 (1980) 19, RK5(4)7M.  Seven stages (the seventh is the fifth-order
 * solution itself), the fifth-order solution is advanced, err = |x_5 - x_4| = h |sum_i e_i k_i^x| (positions only, as
 * for the step doubling), u renormalised.  The field is taken at the stage positions (emo_field_profile returns the
 * constant direction of a uniform field).  Sums run over j ascending from 0.0. */
static const double DP_A[7][6] = {
    { 0.0, 0.0, 0.0, 0.0, 0.0, 0.0 },
    { 1.0 / 5.0, 0.0, 0.0, 0.0, 0.0, 0.0 },
    { 3.0 / 40.0, 9.0 / 40.0, 0.0, 0.0, 0.0, 0.0 },
    { 44.0 / 45.0, -56.0 / 15.0, 32.0 / 9.0, 0.0, 0.0, 0.0 },
    { 19372.0 / 6561.0, -25360.0 / 2187.0, 64448.0 / 6561.0, -212.0 / 729.0, 0.0, 0.0 },
    { 9017.0 / 3168.0, -355.0 / 33.0, 46732.0 / 5247.0, 49.0 / 176.0, -5103.0 / 18656.0, 0.0 },
    { 35.0 / 384.0, 0.0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 11.0 / 84.0 } };
static const double DP_E[7] = { 71.0 / 57600.0, 0.0, -71.0 / 16695.0, 71.0 / 1920.0, -17253.0 / 339200.0, 22.0 / 525.0,
                                -1.0 / 40.0 };

void emo_dp45(const emo_problem *p, const double x[3], const double u[3], double kappa, double h,
              double x1[3], double u1[3], double *err) {
    double kx[7][3], ku[7][3], xs[3], us[3], g[3];
    for (int s = 0; s < 7; ++s) {
        for (int i = 0; i < 3; ++i) {
            double ax = 0.0, au = 0.0;
            for (int j = 0; j < s; ++j) { ax += DP_A[s][j] * kx[j][i]; au += DP_A[s][j] * ku[j][i]; }
            xs[i] = x[i] + h * ax;
            us[i] = u[i] + h * au;
        }
        emo_field_profile(p, xs, g);
        rhs(us, kappa, g, kx[s], ku[s]);
    }
    /* xs, us of the seventh stage are the fifth-order solution */
    double e[3];
    for (int i = 0; i < 3; ++i) {
        double a = 0.0;
        for (int j = 0; j < 7; ++j) a += DP_E[j] * kx[j][i];
        e[i] = h * a;
        x1[i] = xs[i];
        u1[i] = us[i];
    }
    *err = sqrt(e[0] * e[0] + e[1] * e[1] + e[2] * e[2]);
    double n = sqrt(u1[0] * u1[0] + u1[1] * u1[1] + u1[2] * u1[2]);
    u1[0] /= n; u1[1] /= n; u1[2] /= n;
}

/* propagate up to s_max inside cell `vol`; returns the arc length travelled,
 * *hit = surface reached (-1: none).  x, u are updated in place. */
double emo_propagate_field(const emo_problem *p, int vol, int *surf_io, double x[3], double u[3],
                           double kappa, double s_max, int *hit) {
    int n_sub;
    return emo_propagate_field_n(p, vol, surf_io, x, u, kappa, s_max, hit, &n_sub);
}

/* the same, also counting the substep attempts (passes of the loop) in *n_sub: instrumentation for the level-2
 * parity bound (the rounding of a step grows with its substeps), no arithmetic of its own */
double emo_propagate_field_n(const emo_problem *p, int vol, int *surf_io, double x[3], double u[3],
                             double kappa, double s_max, int *hit, int *n_sub) {
    const double eps = p->ph.field_eps;
    double s_done = 0.0;
    int surf = *surf_io;
    double h = 0.25 / fabs(kappa);
    if (s_max < h) h = s_max;
    *hit = -1;
    *n_sub = 0;
    for (int attempt = 0; attempt < p->ph.max_substeps; ++attempt) {
        *n_sub += 1;
        double rem = s_max - s_done;
        if (h > rem) h = rem;
        double x1[3], u1[3], err;
        if (p->ph.integrator == 1) emo_dp45(p, x, u, kappa, h, x1, u1, &err);
        else if (p->field_kind == 0) emo_rk4_doubling(x, u, kappa, p->Bhat, h, x1, u1, &err);
        else emo_rk4_doubling_map(p, x, u, kappa, h, x1, u1, &err);
        if (err > eps && h > 1e-9) {
            double f = 0.9 * pow(eps / err, 0.2);
            h *= (f > 0.2 ? f : 0.2);
            continue;
        }
        double c[3] = { x1[0] - x[0], x1[1] - x[1], x1[2] - x[2] };
        double L = sqrt(c[0] * c[0] + c[1] * c[1] + c[2] * c[2]);
        if (!(L > 0.0)) { s_done += h; break; }
        double cd[3] = { c[0] / L, c[1] / L, c[2] / L };
        int S;
        double d = emo_distance(p, vol, x, cd, surf, &S);
        if (d <= eps) {
            /* chord bends back across the surface the track sits on: shorten and retry */
            if (d == 0.0 && S == surf && h > 1e-9) { h *= 0.5; continue; }
            *hit = S;                                  /* immediate (re-)crossing, nothing travelled */
            *surf_io = surf;
            return s_done;
        }
        if (d > L + eps) {                             /* chord ends inside the cell, clear of S: accept */
            x[0] = x1[0]; x[1] = x1[1]; x[2] = x1[2];
            u[0] = u1[0]; u[1] = u1[1]; u[2] = u1[2];
            s_done += h; surf = -1;
            if (s_done >= s_max * (1.0 - 1e-14)) break;
            double e = err > eps / 3125.0 ? err : eps / 3125.0;
            double f = 0.9 * pow(eps / e, 0.2);
            h *= (f < 5.0 ? f : 5.0);
            continue;
        }
        if (L - d <= eps) {                            /* |L - d| <= eps: landed on S within tolerance, whether just
                                                          past it or just short of it.  (A point accepted as "inside"
                                                          a hair short of S can round onto S unflagged, and the next
                                                          chord then sees S at distance 0 and walks through it.) */
            x[0] = x1[0]; x[1] = x1[1]; x[2] = x1[2];
            u[0] = u1[0]; u[1] = u1[1]; u[2] = u1[2];
            *hit = S;
            *surf_io = S;
            return s_done + h;
        }
        h *= d / L;                                    /* secant: aim the chord end at S */
    }
    *surf_io = surf;
    return s_done;
}
