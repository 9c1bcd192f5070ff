// emx_field.h -- charged-track propagation in a magnetic field, uniform or a solenoid with a fringe (step A5
// of DESIGN.md).
// PAPER.md:144 "on-device propagation of particles through arbitrary magnetic fields ... different
// integration algorithms"; BASELINE.json configs[3]: "adaptive RK4 (1e-6 mm miss-distance tolerance)".
// Algorithm (C9): classical RK4 with step doubling for the local error, plus a chord /
// secant search for the boundary landing point.  y = (x, u), dy/ds = (u, kappa u x Bhat).
#pragma once
#include "emx_core.h"
#include "emx_geom.h"

namespace emx {

EMX_HD Vec3 lorentz(const Vec3 &u, double kappa, const double B[3]) {
    return {kappa * (u.y * B[2] - u.z * B[1]), kappa * (u.z * B[0] - u.x * B[2]), kappa * (u.x * B[1] - u.y * B[0])};
}

// one classical RK4 step of length h.  dx/ds = u, so the x-stages are the u-stage arguments.
EMX_HD void rk4_step(const Vec3 &x, const Vec3 &u, double kappa, const double B[3], double h, Vec3 &xo, Vec3 &uo) {
    const Vec3 k1u = lorentz(u, kappa, B);
    const Vec3 u2 = u + (0.5 * h) * k1u;
    const Vec3 k2u = lorentz(u2, kappa, B);
    const Vec3 u3 = u + (0.5 * h) * k2u;
    const Vec3 k3u = lorentz(u3, kappa, B);
    const Vec3 u4 = u + h * k3u;
    const Vec3 k4u = lorentz(u4, kappa, B);
    const double h6 = h / 6.0;
    xo.x = x.x + h6 * (u.x + 2.0 * u2.x + 2.0 * u3.x + u4.x);
    xo.y = x.y + h6 * (u.y + 2.0 * u2.y + 2.0 * u3.y + u4.y);
    xo.z = x.z + h6 * (u.z + 2.0 * u2.z + 2.0 * u3.z + u4.z);
    uo.x = u.x + h6 * (k1u.x + 2.0 * k2u.x + 2.0 * k3u.x + k4u.x);
    uo.y = u.y + h6 * (k1u.y + 2.0 * k2u.y + 2.0 * k3u.y + k4u.y);
    uo.z = u.z + h6 * (k1u.z + 2.0 * k2u.z + 2.0 * k3u.z + k4u.z);
}

// ---- non-uniform field (include/emx.h: emx_set_field_fringe): B(x) = Bmag g(x), a solenoid along z whose
// field falls off towards its ends, with the radial part that keeps div B = 0 to first order in r
EMX_HD void field_profile(const Params &P, const Vec3 &x, double g[3]) {
    const double az = fabs(x.z);
    const double f = 1.0 / (1.0 + m_exp((az - P.fringe_z0) / P.fringe_a));
    const double sg = x.z > 0.0 ? 1.0 : (x.z < 0.0 ? -1.0 : 0.0);
    const double fp = -sg * f * (1.0 - f) / P.fringe_a;
    g[0] = -0.5 * x.x * fp * P.Bhat[2];
    g[1] = -0.5 * x.y * fp * P.Bhat[2];
    g[2] = f * P.Bhat[2];
}

// classical RK4 with the field taken at the stage positions (x-stages: dx/ds = u)
EMX_HD void rk4_step_map(const Params &P, const Vec3 &x, const Vec3 &u, double kappa, double h, Vec3 &xo, Vec3 &uo) {
    double g[3];
    field_profile(P, x, g);
    const Vec3 k1u = lorentz(u, kappa, g);
    const Vec3 x2 = x + (0.5 * h) * u;
    const Vec3 u2 = u + (0.5 * h) * k1u;
    field_profile(P, x2, g);
    const Vec3 k2u = lorentz(u2, kappa, g);
    const Vec3 x3 = x + (0.5 * h) * u2;
    const Vec3 u3 = u + (0.5 * h) * k2u;
    field_profile(P, x3, g);
    const Vec3 k3u = lorentz(u3, kappa, g);
    const Vec3 x4 = x + h * u3;
    const Vec3 u4 = u + h * k3u;
    field_profile(P, x4, g);
    const Vec3 k4u = lorentz(u4, kappa, g);
    const double h6 = h / 6.0;
    xo.x = x.x + h6 * (u.x + 2.0 * u2.x + 2.0 * u3.x + u4.x);
    xo.y = x.y + h6 * (u.y + 2.0 * u2.y + 2.0 * u3.y + u4.y);
    xo.z = x.z + h6 * (u.z + 2.0 * u2.z + 2.0 * u3.z + u4.z);
    uo.x = u.x + h6 * (k1u.x + 2.0 * k2u.x + 2.0 * k3u.x + k4u.x);
    uo.y = u.y + h6 * (k1u.y + 2.0 * k2u.y + 2.0 * k3u.y + k4u.y);
    uo.z = u.z + h6 * (k1u.z + 2.0 * k2u.z + 2.0 * k3u.z + k4u.z);
}

// one step of h against two of h/2: err = |x_full - x_half|, result = half-step state, u renormalised.
// MAP: the field is evaluated at the stage positions (non-uniform field); else it is P.Bhat everywhere
template <bool MAP>
EMX_NI void rk4_doubling(const Params &P, const Vec3 &x, const Vec3 &u, double kappa, double h, Vec3 &x1, Vec3 &u1,
                         double &err) {
    Vec3 xf, uf, xm, um;
    if (MAP) {
        rk4_step_map(P, x, u, kappa, h, xf, uf);
        rk4_step_map(P, x, u, kappa, 0.5 * h, xm, um);
        rk4_step_map(P, xm, um, kappa, 0.5 * h, x1, u1);
    } else {
        rk4_step(x, u, kappa, P.Bhat, h, xf, uf);
        rk4_step(x, u, kappa, P.Bhat, 0.5 * h, xm, um);
        rk4_step(xm, um, kappa, P.Bhat, 0.5 * h, x1, u1);
    }
    err = norm(xf - x1);
    const double n = norm(u1);
    u1.x /= n;
    u1.y /= n;
    u1.z /= n;
}

// Progress of a propagation that is spread over several iterations of the loop: the
// arc length done, the current trial step and the substep attempts used.  attempt == 0: none in progress.
struct FieldState {
    double s_done, h;
    int attempt;
};

// Propagate up to s_max inside cell `vol`.  Returns the arc length travelled so far; hit = surface reached
// (-1 none).  x, u are updated; on_surf is the surface the track sits on (updated when suspended).
// The substep loop of C9 runs for at most `budget` attempts per call; if it is not finished by then,
// `suspended` is set and fs holds the loop variables, so that the next call continues the SAME sequence of
// substeps: slicing changes when the work is done, never its result.  budget >= max_substeps: one call.
template <bool MAP>
EMX_NI double propagate_field(const Params &P, int vol, int &on_surf, Vec3 &x, Vec3 &u, double kappa, double s_max,
                              int &hit, FieldState &fs, int budget, bool &suspended) {
    const double eps = P.ph.field_eps;
    double s_done;
    int surf = on_surf;
    double h;
    int attempt;
    if (fs.attempt > 0) {  // resume
        s_done = fs.s_done;
        h = fs.h;
        attempt = fs.attempt;
    } else {
        s_done = 0.0;
        h = 0.25 / fabs(kappa);
        if (s_max < h) h = s_max;
        attempt = 0;
    }
    hit = -1;
    suspended = false;
    const int max_attempts = P.ph.max_substeps;
    const int stop_at = (budget < max_attempts - attempt) ? attempt + budget : max_attempts;
    for (; attempt < max_attempts; ++attempt) {
        if (attempt >= stop_at) {  // out of budget for this iteration: park the loop variables
            fs.s_done = s_done;
            fs.h = h;
            fs.attempt = attempt;
            on_surf = surf;
            suspended = true;
            return s_done;
        }
        const double rem = s_max - s_done;
        if (h > rem) h = rem;
        Vec3 x1, u1;
        double err;
        rk4_doubling<MAP>(P, x, u, kappa, h, x1, u1, err);
        if (err > eps && h > 1e-9) {  // too inaccurate: shrink and retry
            const double f = 0.9 * m_pow(eps / err, 0.2);
            h *= (f > 0.2 ? f : 0.2);
            continue;
        }
        const Vec3 c = x1 - x;
        const double L = norm(c);
        if (!(L > 0.0)) {
            s_done += h;
            break;
        }
        const Vec3 cd = {c.x / L, c.y / L, c.z / L};
        int S;
        const double d = distance_to_boundary(P, vol, x, cd, surf, S);
        if (d <= eps) {
            // chord bends back across the surface the track sits on: shorten and retry
            if (d == 0.0 && S == surf && h > 1e-9) {
                h *= 0.5;
                continue;
            }
            hit = S;  // immediate (re-)crossing, nothing more travelled
            fs.attempt = 0;
            return s_done;
        }
        if (d > L + eps) {  // chord ends inside the cell, clear of S: accept
            x = x1;
            u = u1;
            s_done += h;
            surf = -1;
            if (s_done >= s_max * (1.0 - 1e-14)) break;
            const double e = err > eps / 3125.0 ? err : eps / 3125.0;
            const double f = 0.9 * m_pow(eps / e, 0.2);
            h *= (f < 5.0 ? f : 5.0);
            continue;
        }
        if (L - d <= eps) {  // |L - d| <= eps: landed on S, just past it or just short of it
            x = x1;
            u = u1;
            hit = S;
            fs.attempt = 0;
            return s_done + h;
        }
        h *= d / L;  // secant: aim the chord end at S
    }
    fs.attempt = 0;
    return s_done;
}

}  // namespace emx
