/* ORACLE (test infrastructure).  Surface/cell geometry ("quadric
 * surface representations ... cell volumes as CSG combinations of those
 * surfaces ... single geometry level"), restricted to axis-aligned planes and
 * z-cylinders, cells = conjunction of half-spaces (DESIGN.md R-C8).
 * Surfaces: PX/PY/PZ(c): f = x_a - c;  CZ(r): f = x^2 + y^2 - r^2.
 * Sense -1 where f < 0.  sign(g) := (g > 0 ? +1 : -1) everywhere.
 */
#include <math.h>
#include "emo.h"

static double surf_f(const emo_surface *s, const double x[3]) {
    if (s->type == EMO_S_CZ) return x[0] * x[0] + x[1] * x[1] - s->v * s->v;
    return x[s->type] - s->v;
}
/* grad f . u */
static double surf_g(const emo_surface *s, const double x[3], const double u[3]) {
    if (s->type == EMO_S_CZ) return 2.0 * (x[0] * u[0] + x[1] * u[1]);
    return u[s->type];
}
static double surf_tol(const emo_surface *s) {
    return s->type == EMO_S_CZ ? 2e-9 * s->v : 1e-9;
}

/* distance along u from x to the nearest face of cell `vol`; `surf` = surface
 * the track is flagged on (-1 none).  Returns +inf and *hit = -1 if none. */
double emo_distance(const emo_problem *p, int vol, const double x[3], const double u[3], int surf, int *hit) {
    const emo_volume *v = &p->vol[vol];
    double best = INFINITY;
    int bs = -1;
    for (int i = 0; i < v->n_faces; ++i) {
        int S = v->surf[i];
        const emo_surface *s = &p->surf[S];
        double d = -1.0;
        int have = 0;
        if (S == surf) {
            double g = surf_g(s, x, u);
            int ns = g > 0.0 ? 1 : -1;
            if (ns != v->sense[i]) { d = 0.0; have = 1; }          /* points back across it */
            else if (s->type == EMO_S_CZ) {                          /* on the cylinder: c0 = 0 exactly */
                double a = u[0] * u[0] + u[1] * u[1];
                double b = x[0] * u[0] + x[1] * u[1];
                if (a > 0.0) { double r = -2.0 * b / a; if (r > 0.0) { d = r; have = 1; } }
            }
        } else if (s->type == EMO_S_CZ) {
            double a = u[0] * u[0] + u[1] * u[1];
            double b = x[0] * u[0] + x[1] * u[1];
            double c0 = x[0] * x[0] + x[1] * x[1] - s->v * s->v;
            if (a > 0.0) {
                double disc = b * b - a * c0;
                if (disc >= 0.0) {
                    double sq = sqrt(disc);
                    double q = (b >= 0.0) ? -(b + sq) : -(b - sq);
                    double r1 = q / a;
                    double r2 = (q != 0.0) ? c0 / q : -1.0;
                    double lo = r1 < r2 ? r1 : r2, hi = r1 < r2 ? r2 : r1;
                    if (lo > 0.0) { d = lo; have = 1; }
                    else if (hi > 0.0) { d = hi; have = 1; }
                }
            }
        } else {
            double ua = u[s->type];
            if (ua != 0.0) {
                double t = (s->v - x[s->type]) / ua;
                if (t > 0.0) { d = t; have = 1; }
            }
        }
        if (have && (d < best || (d == best && S < bs))) { best = d; bs = S; }
    }
    *hit = bs;
    return best;
}

/* cell entered when crossing surface S at x with direction u; -1 = left the world */
int emo_neighbour(const emo_problem *p, const double x[3], const double u[3], int S) {
    int newsense = surf_g(&p->surf[S], x, u) > 0.0 ? 1 : -1;
    for (int c = 0; c < p->n_vol; ++c) {
        const emo_volume *v = &p->vol[c];
        int ok = 1;
        for (int i = 0; i < v->n_faces && ok; ++i) {
            int Sf = v->surf[i];
            int sn;
            if (Sf == S) sn = newsense;
            else {
                const emo_surface *s = &p->surf[Sf];
                double f = surf_f(s, x);
                if (fabs(f) <= surf_tol(s)) sn = surf_g(s, x, u) > 0.0 ? 1 : -1;
                else sn = f > 0.0 ? 1 : -1;
            }
            if (sn != v->sense[i]) ok = 0;
        }
        if (ok) return c;
    }
    return -1;
}

/* first cell containing x by sign(f) alone (start-volume helper) */
int emo_locate(const emo_problem *p, const double x[3]) {
    for (int c = 0; c < p->n_vol; ++c) {
        const emo_volume *v = &p->vol[c];
        int ok = 1;
        for (int i = 0; i < v->n_faces && ok; ++i) {
            double f = surf_f(&p->surf[v->surf[i]], x);
            if ((f > 0.0 ? 1 : -1) != v->sense[i]) ok = 0;
        }
        if (ok) return c;
    }
    return -1;
}
