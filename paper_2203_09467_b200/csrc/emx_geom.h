// emx_geom.h -- boundary navigation in the plane / z-cylinder CSG (steps A4, A6 of DESIGN.md).
// "quadric surface representations ... cell volumes as CSG combinations of those
// surfaces ... single geometry level"; restricted to axis planes and z-cylinders, cells = AND of
// half-spaces (C8).  f = x_a - v (planes), x^2 + y^2 - v^2 (CZ); sense -1 where f < 0.
#pragma once
#include "emx_core.h"

namespace emx {

// f(x) and grad f . u of surface (type, v)
EMX_HD double surf_f(int type, double v, const Vec3 &x) {
    if (type == EMX_S_CZ) return x.x * x.x + x.y * x.y - v * v;
    return comp(x, type) - v;
}
EMX_HD double surf_g(int type, const Vec3 &x, const Vec3 &u) {
    if (type == EMX_S_CZ) return 2.0 * (x.x * u.x + x.y * u.y);
    return comp(u, type);
}

// Distance along u from x to the nearest face of the cell whose faces are cell[0 .. cell[0].n); on_surf = surface
// the track is flagged on (-1 none).  Returns +inf and hit = -1 when no face is ahead.  Ties -> lowest surface id.
EMX_NI double distance_to_faces(const Face *cell, const Vec3 &x, const Vec3 &u, int on_surf, int &hit) {
    double best = kInf;
    int bs = -1;
    const int nn = cell[0].n;
    const int nf = nn & 0xff, np = (nn >> 8) & 0xff;
    // planes (the table lists them first): one division each, the iterations are independent of one another
#pragma unroll 2
    for (int i = 0; i < np; ++i) {
        const Face f = cell[i];
        const int S = f.S;
        const int type = f.type;
        double d = -1.0;
        bool have = false;
        const double ua = comp(u, type);
        if (S == on_surf) {
            const int ns = ua > 0.0 ? 1 : -1;
            if (ns != f.sense) {  // heading back across the surface it sits on
                d = 0.0;
                have = true;
            }
        } else if (ua != 0.0) {
            const double t = (f.v - comp(x, type)) / ua;
            if (t > 0.0) { d = t; have = true; }
        }
        if (have && (d < best || (d == best && S < bs))) {
            best = d;
            bs = S;
        }
    }
    // z-cylinders: coefficients shared by all of them
    const double a = u.x * u.x + u.y * u.y;
    const double b = x.x * u.x + x.y * u.y;
    const double rr = x.x * x.x + x.y * x.y;
#pragma unroll 2
    for (int i = np; i < nf; ++i) {
        const Face f = cell[i];
        const int S = f.S;
        const double v = f.v;
        double d = -1.0;
        bool have = false;
        if (S == on_surf) {
            const double g = 2.0 * b;
            const int ns = g > 0.0 ? 1 : -1;
            if (ns != f.sense) {  // heading back across the surface it sits on
                d = 0.0;
                have = true;
            } else if (a > 0.0) {  // on the cylinder: c0 = 0 exactly, roots 0 and -2b/a
                const double r = -2.0 * b / a;
                if (r > 0.0) { d = r; have = true; }
            }
        } else if (a > 0.0) {
            const double c0 = rr - v * v;
            const double disc = b * b - a * c0;
            if (disc >= 0.0) {
                const double sq = sqrt(disc);
                const double q = (b >= 0.0) ? -(b + sq) : -(b - sq);  // cancellation-free pair q/a, c0/q
                const double r1 = q / a;
                const double r2 = (q != 0.0) ? c0 / q : -1.0;
                const double lo = r1 < r2 ? r1 : r2, hi = r1 < r2 ? r2 : r1;
                if (lo > 0.0) { d = lo; have = true; }
                else if (hi > 0.0) { d = hi; have = true; }
            }
        }
        if (have && (d < best || (d == best && S < bs))) {
            best = d;
            bs = S;
        }
    }
    hit = bs;
    return best;
}
EMX_HD double distance_to_boundary(const Params &P, int vol, const Vec3 &x, const Vec3 &u, int on_surf, int &hit) {
    return distance_to_faces(P.faces + (size_t)vol * EMX_MAX_FACES, x, u, on_surf, hit);
}

// does cell c contain the point just across S (entered with sense `newsense`)?  Faces within the
// tolerance take their sense from the direction of motion (C8).
EMX_HD bool cell_matches(const Params &P, int cid, const Vec3 &x, const Vec3 &u, int S, int newsense) {
    const Face *cell = P.faces + (size_t)cid * EMX_MAX_FACES;
    const int nf = cell[0].n & 0xff;
    for (int i = 0; i < nf; ++i) {
        const Face fc = cell[i];
        int sn;
        if (fc.S == S) {
            sn = newsense;
        } else {
            const int type = fc.type;
            const double v = fc.v;
            const double f = surf_f(type, v, x);
            const double tol = (type == EMX_S_CZ) ? 2e-9 * v : 1e-9;
            if (fabs(f) <= tol) sn = surf_g(type, x, u) > 0.0 ? 1 : -1;
            else sn = f > 0.0 ? 1 : -1;
        }
        if (sn != fc.sense) return false;
    }
    return true;
}

// Cell entered when crossing surface S at x with direction u; -1 = left the world.
// Definition (C8): the lowest cell id whose faces all agree.  A cell that lists S with the other
// sense can never agree, so only two precomputed lists (ascending id) have to be looked at: the cells that
// list (S, newsense) -- in a world tiled without overlap the answer is one of them -- and, if none of those
// matches (edges and corners where another surface lies within the tolerance), the cells that do not list S
// at all.  For a world tiled without overlap this returns the id of the full scan in id order.  Both lists leave
// out the cells that a parallel face of their own keeps on the other side of S (emx_host.h never_across): the
// scan would reject them anyway, and a track leaving the world finds nothing to test.
EMX_NI int neighbour(const Params &P, const Vec3 &x, const Vec3 &u, int S) {
    const int newsense = surf_g(P.surf_type[S], x, u) > 0.0 ? 1 : -1;
    const int k = 2 * S + (newsense > 0 ? 1 : 0);
    for (int j = P.nb_off[k], e = P.nb_off[k + 1]; j < e; ++j) {
        const int cid = P.nb_list[j];
        if (cell_matches(P, cid, x, u, S, newsense)) return cid;
    }
    for (int j = P.nb2_off[k], e = P.nb2_off[k + 1]; j < e; ++j) {
        const int cid = P.nb2_list[j];
        if (cell_matches(P, cid, x, u, S, newsense)) return cid;
    }
    return -1;
}

}  // namespace emx
