// emx_batch.h -- AoS <-> register conversion for the level-2 parity hook emx_step_batch (include/emx.h):
// the hook runs the SAME step<PT>() the transport kernels run and writes out everything a step produced.
#pragma once
#include "emx_step.h"

namespace emx {

EMX_HD void put3(double *d, const Vec3 &v) {
    d[0] = v.x;
    d[1] = v.y;
    d[2] = v.z;
}

EMX_HD void pack_secondary(const Params &P, uint64_t seed, const Track &t, uint32_t step0, emx_step_result &r,
                           int pt, double E, const Vec3 &u, int ord) {
    emx_track &s = r.sec[r.n_sec];
    put3(s.x, t.x);
    put3(s.u, u);
    s.E = E;
    s.tid = child_tid((uint32_t)seed, t.prim, t.tid, step0, (uint32_t)ord);
    s.prim = t.prim;
    s.step = 0;
    s.vol = t.vol;
    s.surf = -1;
    s.ptype = pt;
    s.alive = 1;
    r.sec_ord[r.n_sec] = ord;
    r.n_sec += 1;
    (void)P;
}

// one step of in -> out
EMX_HD void step_one(const Params &P, uint64_t seed, const emx_track &in, emx_step_result &r) {
    Track t;
    t.x = {in.x[0], in.x[1], in.x[2]};
    t.u = {in.u[0], in.u[1], in.u[2]};
    t.E = in.E;
    t.tid = in.tid;
    t.prim = in.prim;
    t.step = in.step;
    t.vol = in.vol;
    t.surf = in.surf;
    t.alive = 1;
    StepOut o;
    int n_sub = 0;
    const int pt = in.ptype;
    if (pt == kGamma) step<false>(P, seed, pt, t, o, n_sub);
    else if (!P.ph.msc && !P.ph.fluct) {
        if (P.field_kind == 0) step<true, false, false>(P, seed, pt, t, o, n_sub);
        else step<true, true, false>(P, seed, pt, t, o, n_sub);
    } else {
        if (P.field_kind == 0) step<true, false, true>(P, seed, pt, t, o, n_sub);
        else step<true, true, true>(P, seed, pt, t, o, n_sub);
    }

    put3(r.trk.x, t.x);
    put3(r.trk.u, t.u);
    r.trk.E = t.E;
    r.trk.tid = t.tid;
    r.trk.prim = t.prim;
    r.trk.step = t.step;
    r.trk.vol = t.vol;
    r.trk.surf = t.surf;
    r.trk.ptype = in.ptype;
    r.trk.alive = t.alive;
    r.action = o.action;
    r.process = o.process;
    r.n_sec = 0;
    for (int k = 0; k < 4; ++k) {
        r.sec_ord[k] = 0;
        emx_track &s = r.sec[k];
        s.x[0] = s.x[1] = s.x[2] = s.u[0] = s.u[1] = s.u[2] = s.E = 0.0;
        s.tid = 0;
        s.prim = s.step = 0;
        s.vol = s.surf = s.ptype = s.alive = 0;
    }
    // secondaries carry the step number the parent had when it produced them; a surviving parent has
    // already advanced, so undo that for the id
    const uint32_t step0 = in.step;
    if (o.s0.ptype >= 0) pack_secondary(P, seed, t, step0, r, o.s0.ptype, o.s0.E, o.s0.u, o.s0.ord);
    if (o.s1.ptype >= 0) pack_secondary(P, seed, t, step0, r, o.s1.ptype, o.s1.E, o.s1.u, o.s1.ord);
    if (o.rest_alloc) {
        const Vec3 m = {-o.rest_u.x, -o.rest_u.y, -o.rest_u.z};
        pack_secondary(P, seed, t, step0, r, kGamma, kMe, o.rest_u, 2);
        pack_secondary(P, seed, t, step0, r, kGamma, kMe, m, 3);
    }
    r.edep = o.edep;
    r.edep_vol = in.vol;
    r.below_cut = o.below_cut;
    r.escaped = o.escaped;
    r.looper = o.looper;
    r.s = o.s;
    r.msc_tau = o.msc_tau;
    r.n_draws = o.n_draws;
    r.null_int = o.null_int;
    r.rest = o.rest;
    r.n_sub = n_sub;
}

}  // namespace emx
