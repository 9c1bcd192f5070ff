// emx_field.h -- charged-track propagation in a magnetic field, uniform or a solenoid with a fringe (step A5
// of DESIGN.md).
// PAPER.md:144 "on-device propagation of particles through arbitrary magnetic fields ... different
// integration algorithms"; BASELINE.json configs[3]: "adaptive RK4 (1e-6 mm miss-distance tolerance)".
// Algorithm (C9): classical RK4 with step doubling for the local error, plus a chord /
// secant search for the boundary landing point.  y = (x, u), dy/ds = (u, kappa u x Bhat).
//
// The substep loop of C9 is written as ONE ATTEMPT per call (field_attempt): the propagation kernel keeps every
// lane of a warp busy with one attempt of SOME track and hands a lane a new track as soon as its own is done,
// so tracks that need 1 and tracks that need 1000 attempts share a warp without idling it.
#pragma once
#include "emx_core.h"
#include "emx_geom.h"

namespace emx {

// AX: direction of a uniform field.  0 / 1 / 2: along +-x / +-y / +-z, the sign folded into kappa by the caller
// (Bhat = b e_a, b = +-1: kappa (u x Bhat) = (kappa b)(u x e_a) exactly, every product with the zero components
// of Bhat being an exact zero) -- the same numbers as the general formula with a third of the arithmetic;
// 3: any direction.
constexpr int kAxisAny = 3;

template <int AX>
EMX_HD Vec3 lorentz(const Vec3 &u, double kappa, const double B[3]) {
    if (AX == 0) return {0.0, kappa * u.z, -(kappa * u.y)};
    if (AX == 1) return {-(kappa * u.z), 0.0, kappa * u.x};
    if (AX == 2) return {kappa * u.y, -(kappa * u.x), 0.0};
    return {kappa * (u.y * B[2] - u.z * B[1]), kappa * (u.z * B[0] - u.x * B[2]), kappa * (u.x * B[1] - u.y * B[0])};
}

// u + f k, leaving the component along an axis-aligned field alone (its k is an exact zero)
template <int AX>
EMX_HD Vec3 stage_u(const Vec3 &u, double f, const Vec3 &k) {
    return {AX == 0 ? u.x : u.x + f * k.x, AX == 1 ? u.y : u.y + f * k.y, AX == 2 ? u.z : u.z + f * k.z};
}

// one classical RK4 step of length h.  dx/ds = u, so the x-stages are the u-stage arguments.
// h6 = h / 6 (the caller divides once per substep: (h / 2) / 6 = (h / 6) / 2 exactly)
template <int AX>
EMX_HD void rk4_step(const Vec3 &x, const Vec3 &u, double kappa, const double B[3], double h, double h6, Vec3 &xo, Vec3 &uo) {
    const Vec3 k1u = lorentz<AX>(u, kappa, B);
    const Vec3 u2 = stage_u<AX>(u, 0.5 * h, k1u);
    const Vec3 k2u = lorentz<AX>(u2, kappa, B);
    const Vec3 u3 = stage_u<AX>(u, 0.5 * h, k2u);
    const Vec3 k3u = lorentz<AX>(u3, kappa, B);
    const Vec3 u4 = stage_u<AX>(u, h, k3u);
    const Vec3 k4u = lorentz<AX>(u4, kappa, B);
    xo.x = x.x + h6 * (u.x + 2.0 * u2.x + 2.0 * u3.x + u4.x);
    xo.y = x.y + h6 * (u.y + 2.0 * u2.y + 2.0 * u3.y + u4.y);
    xo.z = x.z + h6 * (u.z + 2.0 * u2.z + 2.0 * u3.z + u4.z);
    uo.x = AX == 0 ? u.x : u.x + h6 * (k1u.x + 2.0 * k2u.x + 2.0 * k3u.x + k4u.x);
    uo.y = AX == 1 ? u.y : u.y + h6 * (k1u.y + 2.0 * k2u.y + 2.0 * k3u.y + k4u.y);
    uo.z = AX == 2 ? u.z : u.z + h6 * (k1u.z + 2.0 * k2u.z + 2.0 * k3u.z + k4u.z);
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
    const Vec3 k1u = lorentz<kAxisAny>(u, kappa, g);
    const Vec3 x2 = x + (0.5 * h) * u;
    const Vec3 u2 = u + (0.5 * h) * k1u;
    field_profile(P, x2, g);
    const Vec3 k2u = lorentz<kAxisAny>(u2, kappa, g);
    const Vec3 x3 = x + (0.5 * h) * u2;
    const Vec3 u3 = u + (0.5 * h) * k2u;
    field_profile(P, x3, g);
    const Vec3 k3u = lorentz<kAxisAny>(u3, kappa, g);
    const Vec3 x4 = x + h * u3;
    const Vec3 u4 = u + h * k3u;
    field_profile(P, x4, g);
    const Vec3 k4u = lorentz<kAxisAny>(u4, kappa, g);
    const double h6 = h / 6.0;
    xo.x = x.x + h6 * (u.x + 2.0 * u2.x + 2.0 * u3.x + u4.x);
    xo.y = x.y + h6 * (u.y + 2.0 * u2.y + 2.0 * u3.y + u4.y);
    xo.z = x.z + h6 * (u.z + 2.0 * u2.z + 2.0 * u3.z + u4.z);
    uo.x = u.x + h6 * (k1u.x + 2.0 * k2u.x + 2.0 * k3u.x + k4u.x);
    uo.y = u.y + h6 * (k1u.y + 2.0 * k2u.y + 2.0 * k3u.y + k4u.y);
    uo.z = u.z + h6 * (k1u.z + 2.0 * k2u.z + 2.0 * k3u.z + k4u.z);
}

// one step of h against two of h/2: err = |x_full - x_half|, result = half-step state, u renormalised.
// MAP: the field is evaluated at the stage positions (non-uniform field); else it is uniform along AX
template <bool MAP, int AX>
EMX_NI void rk4_doubling(const Params &P, const Vec3 &x, const Vec3 &u, double kappa, double h, Vec3 &x1, Vec3 &u1,
                         double &err) {
    Vec3 xf, uf, xm, um;
    if (MAP) {
        rk4_step_map(P, x, u, kappa, h, xf, uf);
        rk4_step_map(P, x, u, kappa, 0.5 * h, xm, um);
        rk4_step_map(P, xm, um, kappa, 0.5 * h, x1, u1);
    } else {
        const double h6 = h / 6.0, hh6 = 0.5 * h6;
        rk4_step<AX>(x, u, kappa, P.Bhat, h, h6, xf, uf);
        rk4_step<AX>(x, u, kappa, P.Bhat, 0.5 * h, hh6, xm, um);
        rk4_step<AX>(xm, um, kappa, P.Bhat, 0.5 * h, hh6, x1, u1);
    }
    err = norm(xf - x1);
    const double n = norm(u1);
    u1.x /= n;
    u1.y /= n;
    u1.z /= n;
}

// ---- second integrator (DESIGN.md R-INT; "different integration algorithms"): the embedded pair of Dormand
// and Prince (RK5(4)7M, J. Comput. Appl. Math. 6 (1980) 19).  Seven stages with the field at the stage positions, the
// fifth-order solution (= the state of the seventh stage) is advanced, err = |x_5 - x_4| = h |sum_i e_i k_i^x|, u
// renormalised.  Stage sums in ascending order (terms with a zero coefficient left out: they add a signed zero).
template <bool MAP, int AX>
EMX_NI void dp45_step(const Params &P, const Vec3 &x, const Vec3 &u, double kappa, double h, Vec3 &x1, Vec3 &u1, double &err) {
    constexpr double A[7][6] = {{0.0, 0.0, 0.0, 0.0, 0.0, 0.0},
                                {1.0 / 5.0, 0.0, 0.0, 0.0, 0.0, 0.0},
                                {3.0 / 40.0, 9.0 / 40.0, 0.0, 0.0, 0.0, 0.0},
                                {44.0 / 45.0, -56.0 / 15.0, 32.0 / 9.0, 0.0, 0.0, 0.0},
                                {19372.0 / 6561.0, -25360.0 / 2187.0, 64448.0 / 6561.0, -212.0 / 729.0, 0.0, 0.0},
                                {9017.0 / 3168.0, -355.0 / 33.0, 46732.0 / 5247.0, 49.0 / 176.0, -5103.0 / 18656.0, 0.0},
                                {35.0 / 384.0, 0.0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 11.0 / 84.0}};
    constexpr double E[7] = {71.0 / 57600.0, 0.0, -71.0 / 16695.0, 71.0 / 1920.0, -17253.0 / 339200.0, 22.0 / 525.0, -1.0 / 40.0};
    Vec3 kx[7], ku[7];  // dx/ds = the stage direction, du/ds = kappa u x Bhat at the stage
    Vec3 xs = x, us = u;
#pragma unroll
    for (int s = 0; s < 7; ++s) {
        if (s > 0) {
            Vec3 ax = {0.0, 0.0, 0.0}, au = {0.0, 0.0, 0.0};
#pragma unroll
            for (int j = 0; j < s; ++j) {
                if (A[s][j] == 0.0) continue;
                ax.x += A[s][j] * kx[j].x;
                ax.y += A[s][j] * kx[j].y;
                ax.z += A[s][j] * kx[j].z;
                if (AX != 0) au.x += A[s][j] * ku[j].x;
                if (AX != 1) au.y += A[s][j] * ku[j].y;
                if (AX != 2) au.z += A[s][j] * ku[j].z;
            }
            xs = {x.x + h * ax.x, x.y + h * ax.y, x.z + h * ax.z};
            us = {AX == 0 ? u.x : u.x + h * au.x, AX == 1 ? u.y : u.y + h * au.y, AX == 2 ? u.z : u.z + h * au.z};
        }
        kx[s] = us;
        if (MAP) {
            double g[3];
            field_profile(P, xs, g);
            ku[s] = lorentz<kAxisAny>(us, kappa, g);
        } else {
            ku[s] = lorentz<AX>(us, kappa, P.Bhat);
        }
    }
    Vec3 e = {0.0, 0.0, 0.0};
#pragma unroll
    for (int j = 0; j < 7; ++j) {
        if (E[j] == 0.0) continue;
        e.x += E[j] * kx[j].x;
        e.y += E[j] * kx[j].y;
        e.z += E[j] * kx[j].z;
    }
    e = {h * e.x, h * e.y, h * e.z};
    err = norm(e);
    x1 = xs;
    const double n = norm(us);
    u1 = {us.x / n, us.y / n, us.z / n};
}

// one substep with integrator INTEG (0: step doubling, 1: Dormand-Prince)
template <bool MAP, int AX, int INTEG>
EMX_HD void field_substep(const Params &P, const Vec3 &x, const Vec3 &u, double kappa, double h, Vec3 &x1, Vec3 &u1, double &err) {
    if (INTEG == 1) dp45_step<MAP, AX>(P, x, u, kappa, h, x1, u1, err);
    else rk4_doubling<MAP, AX>(P, x, u, kappa, h, x1, u1, err);
}

// x^(1/5) for the step-size control, x in [1e-30, 1e30], within 1 ulp: r ~ x^(-1/5) from a single-precision seed of
// the special-function unit (relative error below 1e-5) and two Newton steps r <- r (6 - x r^5) / 5 (each squares the
// error times 3: 3e-10, then below rounding), y = x r^4, and one Newton step of y^5 = x with 1 / (5 y^4) = r^4 / 5
// whose residual comes out of one fused multiply-add.  30 instructions against the 110 of exp(log(x) / 5), which was
// 30 % of all instructions of the propagation kernel (profiles/r2_field_hotspots.md).
EMX_HD double fifth_root(double x) {
#if defined(__CUDA_ARCH__)
    double r = (double)__powf((float)x, -0.2f);
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        const double r2 = r * r, r4 = r2 * r2;
        r = r * (0.2 * fma(-x, r4 * r, 6.0));
    }
    const double r2 = r * r, r4 = r2 * r2;
    const double y = x * r4;
    const double y2 = y * y;
    return fma(-0.2 * r4, fma(y2 * y2, y, -x), y);
#else
    return pow(x, 0.2);
#endif
}

// Loop variables of a propagation: the arc length done, the current trial step and the substep attempts used.
// They live in registers while a lane works on the track and in the slot while the track is parked between two
// iterations of the loop; either way the SAME sequence of substeps is taken: when the attempts are made never
// changes a result.
struct FieldState {
    double s_done, h;
    int attempt;
};

EMX_HD void field_begin(double kappa, double s_max, FieldState &fs) {
    fs.s_done = 0.0;
    fs.h = 0.25 / fabs(kappa);
    if (s_max < fs.h) fs.h = s_max;
    fs.attempt = 0;
}

// ONE attempt of the substep loop of C9 inside one cell, towards the arc length s_max.  x, u, on_surf (the surface
// the track sits on) and fs are updated.  Returns true when the propagation is over: s = arc length travelled,
// hit = surface reached (-1 none: s_max travelled, or the max_substeps attempts of the step are used up).
// cell = the faces of the track's cell (Params::faces, or the kernel's copy of it in shared memory).
template <bool MAP, int AX, int INTEG = 0>
EMX_NI bool field_attempt(const Params &P, const Face *cell, int &on_surf, Vec3 &x, Vec3 &u, double kappa, double s_max,
                          FieldState &fs, int &hit, double &s) {
    const double eps = P.ph.field_eps;
    const double rem = s_max - fs.s_done;
    double h = fs.h;
    if (h > rem) h = rem;
    Vec3 x1, u1;
    double err;
    field_substep<MAP, AX, INTEG>(P, x, u, kappa, h, x1, u1, err);
    hit = -1;
    // the two places of C9 that rescale h by 0.9 (eps / e)^(1/5) -- shrink after a rejected substep, grow after an
    // accepted one -- share ONE evaluation of the power, so that lanes which shrink and lanes which grow do not
    // run it one after the other
    double ratio = 0.0;
    int rescale = 0;  // 1 shrink, 2 grow
    if (err > eps && h > 1e-9) {  // too inaccurate: shrink and retry
        ratio = eps / err;
        rescale = 1;
    } else {
        const Vec3 c = x1 - x;
        const double L = norm(c);
        if (!(L > 0.0)) {
            fs.s_done += h;
            s = fs.s_done;
            return true;
        }
        const Vec3 cd = {c.x / L, c.y / L, c.z / L};
        int S;
        const double d = distance_to_faces(cell, x, cd, on_surf, S);
        if (d <= eps) {
            // chord bends back across the surface the track sits on: shorten and retry
            if (d == 0.0 && S == on_surf && h > 1e-9) {
                h *= 0.5;
            } else {
                hit = S;  // immediate (re-)crossing, nothing more travelled
                s = fs.s_done;
                return true;
            }
        } else if (d > L + eps) {  // chord ends inside the cell, clear of S: accept
            x = x1;
            u = u1;
            fs.s_done += h;
            on_surf = -1;
            if (fs.s_done >= s_max * (1.0 - 1e-14)) {
                s = fs.s_done;
                return true;
            }
            const double e = err > P.field_eps_floor ? err : P.field_eps_floor;
            ratio = eps / e;
            rescale = 2;
        } else if (L - d <= eps) {  // |L - d| <= eps: landed on S, just past it or just short of it
            x = x1;
            u = u1;
            hit = S;
            s = fs.s_done + h;
            return true;
        } else {
            h *= d / L;  // secant: aim the chord end at S
        }
    }
    if (rescale) {
        const double f = 0.9 * fifth_root(ratio);
        if (rescale == 1) h *= (f > 0.2 ? f : 0.2);
        else h *= (f < 5.0 ? f : 5.0);
    }
    fs.h = h;
    fs.attempt += 1;
    if (fs.attempt >= P.ph.max_substeps) {  // the step's attempts are used up: whatever was travelled
        s = fs.s_done;
        return true;
    }
    return false;
}

// the axis of a uniform field (host and device): 0 / 1 / 2 with sign b = Bhat[axis], or kAxisAny
EMX_HD int field_axis(const double Bhat[3]) {
    for (int a = 0; a < 3; ++a) {
        const int i = (a + 1) % 3, j = (a + 2) % 3;
        if (Bhat[i] == 0.0 && Bhat[j] == 0.0 && (Bhat[a] == 1.0 || Bhat[a] == -1.0)) return a;
    }
    return kAxisAny;
}

// The whole propagation in one call (level-2 hook; the loop's kernel calls field_attempt itself).
template <bool MAP>
EMX_NI double propagate_field(const Params &P, int vol, int &on_surf, Vec3 &x, Vec3 &u, double kappa, double s_max,
                              int &hit, int &n_attempts) {
    FieldState fs;
    field_begin(kappa, s_max, fs);
    double s = 0.0;
    const int ax = MAP ? kAxisAny : field_axis(P.Bhat);
    const double kb = ax == kAxisAny ? kappa : kappa * P.Bhat[ax];
    bool done = false;
    n_attempts = 0;
    const Face *cell = P.faces + (size_t)vol * EMX_MAX_FACES;
    while (!done) {
        if (P.ph.integrator == 1) {
            if (MAP || ax == kAxisAny) done = field_attempt<MAP, kAxisAny, 1>(P, cell, on_surf, x, u, kappa, s_max, fs, hit, s);
            else if (ax == 0) done = field_attempt<false, 0, 1>(P, cell, on_surf, x, u, kb, s_max, fs, hit, s);
            else if (ax == 1) done = field_attempt<false, 1, 1>(P, cell, on_surf, x, u, kb, s_max, fs, hit, s);
            else done = field_attempt<false, 2, 1>(P, cell, on_surf, x, u, kb, s_max, fs, hit, s);
        } else if (MAP || ax == kAxisAny) done = field_attempt<MAP, kAxisAny>(P, cell, on_surf, x, u, kappa, s_max, fs, hit, s);
        else if (ax == 0) done = field_attempt<false, 0>(P, cell, on_surf, x, u, kb, s_max, fs, hit, s);
        else if (ax == 1) done = field_attempt<false, 1>(P, cell, on_surf, x, u, kb, s_max, fs, hit, s);
        else done = field_attempt<false, 2>(P, cell, on_surf, x, u, kb, s_max, fs, hit, s);
        ++n_attempts;
    }
    return s;
}

}  // namespace emx
