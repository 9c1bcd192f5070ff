// emx_step.h -- one step of one track (C7; PAPER.md:114 lists what a step must do:
// material-dependent properties, continuous slowing down, competition among discrete processes,
// scattering / absorption, secondary emission, energy cutoffs).
//
// The step is written in STAGES so that the loop can run each as its own kernel with its own register
// budget and regroup the tracks in between:
//   step_a0   items 1-4 of C7: tracking cut, table lookup, interaction length and step limits (draw 0);
//   a1        item 5, the move: move_straight(), or the adaptive RK4 of emx_field.h one attempt at a time
//             (field_attempt; it may be spread over several iterations), closed by field_move_done();
//   step_a2   items 6-7 and the SELECTION of item 8: continuous loss, cut kill, boundary relocation, multiple
//             scattering, choice of the discrete process (the remaining phase-A draws);
//   step_interact  item 8 (the interactor, draws 2...) and item 9 for a track whose interaction is pending.
// What a1 hands to a2 is the `Carry` (action, path travelled, surface hit); a2 looks the tables up again at the
// unchanged pre-step energy (same arithmetic, same values) instead of carrying eight doubles through memory.
// step<>() = the three back to back: the level-2 hook.  Photons (CH = false) and e+- (CH = true; the type is a
// run-time value: e- and e+ share a pool and differ in charge sign, tables and the rest-mass bookkeeping).
#pragma once
#include "emx_core.h"
#include "emx_geom.h"
#include "emx_field.h"
#include "emx_interact.h"

namespace emx {

// per-track state held in registers during a step (the SoA store is the HBM form)
struct Track {
    Vec3 x, u;
    double E;
    uint64_t tid;
    uint32_t prim, step;
    int vol, surf;
    int alive;
};

// a secondary produced by this step; position / cell / primary are the parent's (C10)
struct Sec {
    Vec3 u;
    double E;
    int ptype;  // -1: not allocated
    int ord;
};

struct StepOut {
    int action, process;
    Sec s0, s1;          // interaction products, ordinals 0 and 1
    int rest_alloc;      // at-rest annihilation photons allocated (ordinals 2, 3), directions +-rest_u
    Vec3 rest_u;
    double edep, below_cut, escaped, looper, s;
    double msc_tau;      // path / lambda_1 of this step's multiple-scattering deflection (level-2 hook)
    int n_draws, null_int, rest;
    int suspended;       // field propagation parked for the next iteration: nothing else of the step happened
};

// what stage a1 hands to stage a2
constexpr int kActCut = 7;  // internal action code: the track was below the tracking cut at the start of the step
struct Carry {
    double s_phys;  // limit of the move: the step limit of the physics (R-MSC2: its geometric length); kept while a
                    // propagation is parked
    double s;       // path travelled by the move
    int action;     // EMX_A_* after the move (BOUNDARY / TRUNC override the physics limit), or kActCut
    int hit;        // surface reached, -1 none
};

EMX_HD void clear_out(StepOut &o) {
    o.action = EMX_A_NONE;
    o.process = -1;
    o.s0.ptype = -1;
    o.s1.ptype = -1;
    o.rest_alloc = 0;
    o.edep = o.below_cut = o.escaped = o.looper = o.s = 0.0;
    o.msc_tau = 0.0;
    o.n_draws = o.null_int = o.rest = 0;
    o.suspended = 0;
}

// grid lookup (C4): bin j and fraction f of ln E, shared by every table of the step
struct GridPos {
    int j;
    double f;
};
EMX_HD GridPos grid_pos(const Params &P, double E) {
    const double t = (m_log(E) - P.lnE0) * P.inv_dlnE;
    int j = (int)floor(t);
    const int n = P.ph.n_E;
    if (j < 0) j = 0;
    if (j > n - 2) j = n - 2;
    double f = t - j;
    if (f < 0.0) f = 0.0;
    if (f > 1.0) f = 1.0;
    return {j, f};
}
EMX_HD double interp(const double *T, const GridPos &g) { return (1.0 - g.f) * T[g.j] + g.f * T[g.j + 1]; }
EMX_HD const double *table(const Params &P, int mat, int kind) {
    return P.tab + ((size_t)mat * EMX_NTABLE + (size_t)kind) * (size_t)P.ph.n_E;
}

// C7 item 3: everything the step reads from the tables at the pre-step energy, fixed process order
struct Lookup {
    double Sig0, Sig1, Sig2, Stot, D, R;
    double iL0;   // 1 / lambda_1 (R-MSC)
    double iL20;  // 1 / lambda_2 (R-MSC2)
    double var0;  // variance of the loss per unit path (R-FLUCT)
    const double *Rtab;
};
// gtab: the photon kernel's shared-memory copy of its three tables per material ([mat][3][n_E], emx_schedule entry 7
// bit 1; nullptr: the tables are read from global memory through L1)
template <bool CH, bool EXT>
EMX_HD void lookup_tables(const Params &P, int pt, int mat, double E, Lookup &L, const double *gtab = nullptr) {
    const GridPos g = grid_pos(P, E);
    L.D = L.R = L.iL0 = L.iL20 = L.var0 = 0.0;
    L.Rtab = nullptr;
    if (!CH) {
        const size_t nE = (size_t)P.ph.n_E;
        const double *T0 = gtab ? gtab + (size_t)mat * 3 * nE : table(P, mat, EMX_T_COMPTON);  // kinds 0, 1, 2 are adjacent
        L.Sig0 = interp(T0, g);
        L.Sig1 = interp(T0 + nE, g);
        L.Sig2 = interp(T0 + 2 * nE, g);
        L.Stot = L.Sig0 + L.Sig1 + L.Sig2;
    } else {
        const bool em = (pt == kElectron);
        L.Sig0 = interp(table(P, mat, em ? EMX_T_MOLLER : EMX_T_BHABHA), g);
        L.Sig1 = interp(table(P, mat, em ? EMX_T_BREMS_EM : EMX_T_BREMS_EP), g);
        L.Sig2 = em ? 0.0 : interp(table(P, mat, EMX_T_ANNIH), g);
        L.D = interp(table(P, mat, em ? EMX_T_DEDX_EM : EMX_T_DEDX_EP), g);
        L.Rtab = table(P, mat, em ? EMX_T_RANGE_EM : EMX_T_RANGE_EP);
        L.R = interp(L.Rtab, g);
        L.Stot = em ? (L.Sig0 + L.Sig1) : (L.Sig0 + L.Sig1 + L.Sig2);
        if (EXT && P.ph.fluct) L.var0 = interp(table(P, mat, em ? EMX_T_VAR_EM : EMX_T_VAR_EP), g);
        if (EXT && P.ph.msc) L.iL0 = interp(table(P, mat, EMX_T_MSC), g);
        if (EXT && P.ph.msc == 2) L.iL20 = interp(table(P, mat, EMX_T_MSC2), g);
    }
}

// C7 item 4: interaction length resampled every step (R27, draw 0 = xi); continuous-loss step function (R9);
// multiple-scattering step limit (R-MSC)
template <bool CH, bool EXT>
EMX_HD void step_limits(const Params &P, const Lookup &L, double xi, double &s_phys, int &action) {
    const emx_physics &ph = P.ph;
    s_phys = L.Stot > 0.0 ? -m_log(xi) / L.Stot : kInf;
    action = EMX_A_DISCRETE;
    if (CH) {
        double s_loss;
        if (L.R <= ph.rho_R) s_loss = L.R;
        else s_loss = ph.alpha_R * L.R + ph.rho_R * (1.0 - ph.alpha_R) * (2.0 - ph.rho_R / L.R);
        if (s_loss < s_phys) {
            s_phys = s_loss;
            action = EMX_A_LOSS;
        }
        if (EXT && ph.msc) {  // s <= max(f_r max(R, lambda_1), s_min)
            const double big = (L.iL0 > 0.0 && 1.0 / L.iL0 > L.R) ? 1.0 / L.iL0 : L.R;
            double s_msc = ph.msc_fr * big;
            if (s_msc < ph.msc_smin) s_msc = ph.msc_smin;
            if (s_msc < s_phys) {
                s_phys = s_msc;
                action = EMX_A_MSC;
            }
        }
    }
}

// exact inverse of the forward lookup on a range table (C5.9)
EMX_NI double range_inverse(const Params &P, const double *R, double r) {
    const int n = P.ph.n_E;
    if (r <= R[0]) return m_exp(P.lnE0) * (r / R[0]);  // constant dE/dx below the grid (R24)
    if (r >= R[n - 1]) return m_exp(P.lnE0 + (n - 1) * P.dlnE);
    int lo = 0, hi = n - 1;  // R[lo] <= r < R[hi]
    while (hi - lo > 1) {
        const int mid = (lo + hi) / 2;
        if (R[mid] <= r) lo = mid;
        else hi = mid;
    }
    const double f = (r - R[lo]) / (R[lo + 1] - R[lo]);
    return m_exp(P.lnE0 + (lo + f) * P.dlnE);
}

// C10: a secondary of type pt; deposited locally instead when below the tracking cut (gamma, e-) or when
// electrons are deposited at creation (BASELINE configs[0])
EMX_HD void add_secondary(const Params &P, StepOut &o, Sec &slot, int pt, double E, const Vec3 &d, int ord) {
    if (pt == kElectron && P.ph.deposit_e_at_creation) {
        o.edep += E;
        return;
    }
    if (pt != kPositron && E < P.ph.E_trk) {
        o.edep += E;
        o.below_cut += E;
        return;
    }
    slot.u = d;
    slot.E = E;
    slot.ptype = pt;
    slot.ord = ord;
}

// tracking-cut kill: deposit E locally; an e+ annihilates at rest (R12 / R25)
EMX_HD void kill_below(const Params &P, int pt, Rng &rng, Track &t, StepOut &o, double E) {
    o.edep += E;
    o.below_cut += E;
    if (pt == kPositron) {
        Vec3 u1, u2;
        annih_rest(rng, u1, u2);
        o.rest = 1;
        if (kMe < P.ph.E_trk) {  // the photons themselves are below the cut
            o.edep += kMe;
            o.below_cut += kMe;
            o.edep += kMe;
            o.below_cut += kMe;
        } else {
            o.rest_alloc = 1;
            o.rest_u = u1;
        }
    }
    t.E = 0.0;
    t.alive = 0;
}

// 9. step counter, looper cap (R14)
EMX_HD void finish_step(const Params &P, int pt, Track &t, StepOut &o) {
    if (t.alive) {
        t.step += 1;
        if ((int)t.step >= P.ph.max_steps) {
            o.looper += t.E + (pt == kPositron ? 2.0 * kMe : 0.0);
            t.alive = 0;
        }
    }
}

// ---- stage a0: items 1-4 (tracking cut, lookup, limits; draw 0).  Fills c.s_phys and c.action.
// EXT: multiple scattering and / or energy-loss fluctuations are on.
// L receives the table values of item 3 (left alone below the cut and in vacuum) for a caller that runs stage a2 next.
template <bool CH, bool EXT>
EMX_HD void step_a0(const Params &P, uint64_t seed, int pt, const Track &t, Carry &c, Lookup &L, const double *gtab = nullptr) {
    const emx_physics &ph = P.ph;
    const int mat = P.vol[t.vol].material;
    c.s = 0.0;
    c.hit = -1;
    if (t.E < ph.E_trk) {  // 1. tracking cut at step start
        c.s_phys = 0.0;
        c.action = kActCut;
    } else if (mat < 0) {  // 2. vacuum: no physics, capped flight
        c.s_phys = ph.vacuum_step;
        c.action = EMX_A_TRUNC;
    } else {  // 3. lookup, 4. limits
        lookup_tables<CH, EXT>(P, pt, mat, t.E, L, gtab);
        const double xi = draw_at(seed, t.prim, t.tid, t.step, 0u);
        step_limits<CH, EXT>(P, L, xi, c.s_phys, c.action);
        // R-MSC2: the limits are true path lengths; what the move is limited by is the geometric length of the step
        if (CH && EXT && ph.msc == 2) c.s_phys = msc_geom_length(c.s_phys, L.iL0);
    }
}

// ---- stage a1, item 5 without a field (photons always): distance to the boundary, straight move
EMX_HD void move_straight(const Params &P, Track &t, Carry &c) {
    int hit;
    const double d = distance_to_boundary(P, t.vol, t.x, t.u, t.surf, hit);
    double s;
    if (d <= c.s_phys) {  // boundary wins ties (R10)
        s = d;
        c.action = EMX_A_BOUNDARY;
        c.hit = hit;
    } else {
        s = c.s_phys;
        c.hit = -1;
    }
    t.x.x += s * t.u.x;
    t.x.y += s * t.u.y;
    t.x.z += s * t.u.z;
    c.s = s;
}

// ---- stage a1, item 5 in a field: curvature of the track, and what the finished propagation means for the step
EMX_HD double curvature(const Params &P, int pt, double E) {
    const double pm = sqrt(E * (E + 2.0 * kMe));
    const double q = (pt == kElectron) ? -1.0 : 1.0;
    return q * kCB * P.Bmag / pm;
}
EMX_HD void field_move_done(Carry &c, double s, int hit) {
    c.s = s;
    c.hit = hit;
    if (hit >= 0) c.action = EMX_A_BOUNDARY;
    else if (!(s >= c.s_phys * (1.0 - 1e-14))) c.action = EMX_A_TRUNC;
}

// ---- stage a2: items 6, 7, 7b and the selection of item 8.  t.E is still the pre-step energy.  Returns the process
// id (EMX_P_*) if an interaction is pending (step_interact finishes the step), else -1 and the step is complete.
// HAVE_L: L already holds the table values of stage a0 (same slot, same energy); else they are looked up again.
template <bool CH, bool EXT, bool HAVE_L = false>
EMX_HD int step_a2(const Params &P, uint64_t seed, int pt, Track &t, StepOut &o, const Carry &c, Lookup &L) {
    const emx_physics &ph = P.ph;
    clear_out(o);
    Rng rng;
    rng.init(seed, t.prim, t.tid, t.step);
    if (c.action == kActCut) {
        kill_below(P, pt, rng, t, o, t.E);
        o.n_draws = (int)rng.n;
        return -1;
    }
    const int mat = P.vol[t.vol].material;
    const int action = c.action;
    double s = c.s;
    const double E = t.E;
    if (!HAVE_L) {
        L.Sig0 = L.Sig1 = L.Sig2 = L.Stot = L.D = L.R = L.iL0 = L.iL20 = L.var0 = 0.0;
        L.Rtab = nullptr;
    }
    double xi0 = 0.5;
    if (mat >= 0) {
        if (!HAVE_L) lookup_tables<CH, EXT>(P, pt, mat, E, L);
        xi0 = rng.next();  // draw 0 was the interaction length (stage a1); this also restores the block's second half
    }
    const bool msc = CH && EXT && ph.msc && mat >= 0;  // multiple scattering applies (R-MSC)
    if (msc && ph.msc == 2) {
        // R-MSC2: c.s is the geometric length of the move; from here on s is the TRUE path length -- the limit of the
        // physics (the same evaluation as stage a0's) if the move was completed, else in proportion
        double t_phys;
        int a0;
        step_limits<CH, EXT>(P, L, xi0, t_phys, a0);
        const bool full = action != EMX_A_BOUNDARY && action != EMX_A_TRUNC;
        s = full ? t_phys : t_phys * (c.s / msc_geom_length(t_phys, L.iL0));
    }
    o.s = s;

    // 6. continuous loss (e+- in matter)
    if (CH && mat >= 0) {
        double dE, f1 = 0.0, f2 = 0.0;
        const bool fl = EXT && ph.fluct;  // energy-loss fluctuations (R-FLUCT): two draws, always consumed
        if (fl) {
            f1 = rng.next();
            f2 = rng.next();
        }
        if (action == EMX_A_LOSS && L.R <= ph.rho_R) {
            dE = E;  // range stop: the whole loss-limited step was travelled (a cut-short step has another action)
        } else {
            if (s * L.D <= ph.lin_loss * E) {
                dE = s * L.D;
            } else {
                const double E2 = range_inverse(P, L.Rtab, L.R - s);
                dE = E - E2;
                if (dE < 0.0) dE = 0.0;
                if (dE > E) dE = E;
            }
            if (fl && dE > 0.0) {
                dE = fluctuate_loss(dE, s * L.var0, E, f1, f2);
            }
        }
        t.E = E - dE;
        o.edep += dE;
        if (t.E < ph.E_trk) {
            o.action = action;
            kill_below(P, pt, rng, t, o, t.E);
            o.n_draws = (int)rng.n;
            return -1;
        }
    }
    o.action = action;

    // 7. boundary crossing / relocation
    if (action == EMX_A_BOUNDARY) {
        const int nv = neighbour(P, t.x, t.u, c.hit);
        t.surf = c.hit;
        if (nv < 0) {  // left the world: escape (an e+ carries its rest-mass credit, R13)
            o.escaped += t.E + (pt == kPositron ? 2.0 * kMe : 0.0);
            t.alive = 0;
            o.n_draws = (int)rng.n;
            return -1;
        }
        t.vol = nv;
    } else {
        t.surf = -1;
    }

    // 7b. multiple-scattering deflection at the end of the step (R-MSC): <cos> = exp(-Int ds / lambda_1), the
    // integral by the trapezoid rule over the pre-step and post-loss energies; two draws, always consumed
    if (msc) {
        const GridPos g1 = grid_pos(P, t.E);
        const double iL1 = interp(table(P, mat, EMX_T_MSC), g1);
        const double tau = 0.5 * (L.iL0 + iL1) * s;
        const Vec3 u0 = t.u;
        t.u = msc_deflect(rng, tau, u0);
        o.msc_tau = tau;
        // R-MSC2 lateral displacement along the transverse part d of the new direction (|d| = sin(theta)) by
        // rho = sqrt(3 <r^2> / (2 (1 - g^2))) |d|: <rho^2> = Lewis' <x^2 + y^2> for the Henyey-Greenstein angle
        // (<sin^2> = (2/3)(1 - g^2), g = exp(-tau)); at most 0.9 of the way to the cell's boundary; none after a
        // step that ended on a boundary
        if (ph.msc == 2 && action != EMX_A_BOUNDARY) {
            const double il1 = 0.5 * (L.iL0 + iL1);
            const double il2 = 0.5 * (L.iL20 + interp(table(P, mat, EMX_T_MSC2), g1));
            const double r2 = msc_lateral_r2(s, il1, il2);
            const double om = -expm1(-2.0 * tau);
            const double mu = u0.x * t.u.x + u0.y * t.u.y + u0.z * t.u.z;
            const Vec3 d = {t.u.x - mu * u0.x, t.u.y - mu * u0.y, t.u.z - mu * u0.z};
            const double dn = norm(d);
            if (r2 > 0.0 && om > 0.0 && dn > 0.0) {
                double rho = sqrt(1.5 * r2 / om) * dn;
                const Vec3 dh = {d.x / dn, d.y / dn, d.z / dn};
                int hs;
                const double lim = 0.9 * distance_to_boundary(P, t.vol, t.x, dh, -1, hs);
                if (rho > lim) rho = lim;
                t.x.x += rho * dh.x;
                t.x.y += rho * dh.y;
                t.x.z += rho * dh.z;
            }
        }
    }

    // 8. discrete interaction: select with the pre-step cross sections, interact at the post-loss energy (R21)
    if (action == EMX_A_DISCRETE) {
        const double target = rng.next() * L.Stot;
        int k;
        if (CH && pt == kElectron) {
            k = (L.Sig0 > target) ? 0 : 1;
            if (k == 1 && L.Sig1 <= 0.0) k = 0;
        } else {
            const double c1 = L.Sig0 + L.Sig1;
            k = (L.Sig0 > target) ? 0 : ((c1 > target) ? 1 : 2);
            if (k == 2 && L.Sig2 <= 0.0) k = 1;
            if (k == 1 && L.Sig1 <= 0.0) k = 0;
        }
        int proc;  // k-th process of this particle type -> process id
        if (!CH) proc = (k == 0) ? EMX_P_COMPTON : (k == 1 ? EMX_P_PHOTO : EMX_P_PAIR);
        else if (pt == kElectron) proc = (k == 0) ? EMX_P_MOLLER : EMX_P_BREMS;
        else proc = (k == 0) ? EMX_P_BHABHA : (k == 1 ? EMX_P_BREMS : EMX_P_ANNIH);
        o.n_draws = (int)rng.n;
        return proc;  // interaction pending: the step is finished by step_interact
    }
    finish_step(P, pt, t, o);
    o.n_draws = (int)rng.n;
    return -1;
}

// Item 8 of C7 for a track whose interaction `proc` was selected by step_a2: the interactor runs at the
// post-loss energy t.E with draws 2, 3, ... of the step, then item 9.
template <bool CH>
EMX_HD void step_interact(const Params &P, uint64_t seed, int pt, Track &t, StepOut &o, int proc) {
    const emx_physics &ph = P.ph;
    Rng rng;
    rng.init(seed, t.prim, t.tid, t.step);
    const int mat = P.vol[t.vol].material;
    // draws 0 (interaction length) and the process selection were used by stages a1 / a2, and in between two each
    // by the energy-loss fluctuation (R-FLUCT) and the multiple-scattering deflection (R-MSC) of an e+-
    rng.n = CH ? 2u + (ph.fluct ? 2u : 0u) + (ph.msc ? 2u : 0u) : 2u;
    const Material &m = P.mat[mat];
    const double E1 = t.E;
    const Vec3 u0 = t.u;
    o.process = proc;
    if (!CH) {
        if (proc == EMX_P_COMPTON) {
            double Eg, Te;
            Vec3 ug, ue;
            compton(rng, E1, u0, Eg, ug, Te, ue);
            add_secondary(P, o, o.s0, kElectron, Te, ue, 0);
            t.E = Eg;
            t.u = ug;
        } else if (proc == EMX_P_PHOTO) {
            if (ph.deposit_e_at_creation) {
                o.edep += E1;
            } else {
                const Vec3 ue = photo_dir(rng, E1, u0);
                add_secondary(P, o, o.s0, kElectron, E1, ue, 0);
            }
            t.E = 0.0;
            t.alive = 0;
        } else {
            int ie = 0;
            if (m.n_elem > 1) {  // element selection (R4)
                const double xe = rng.next();
                const GridPos g1 = grid_pos(P, E1);
                double se[EMX_MAX_ELEM], st = 0.0;
                for (int i = 0; i < m.n_elem; ++i) {
                    se[i] = interp(table(P, mat, EMX_T_PAIR_ELEM0 + i), g1);
                    st += se[i];
                }
                double cc = 0.0;
                ie = m.n_elem - 1;
                for (int i = 0; i < m.n_elem; ++i) {
                    cc += se[i];
                    if (cc > xe * st) {
                        ie = i;
                        break;
                    }
                }
            }
            double Tm, Tp;
            Vec3 um, up;
            if (pair_production(rng, m.Z[ie], E1, u0, Tm, um, Tp, up)) {
                add_secondary(P, o, o.s0, kElectron, Tm, um, 0);
                add_secondary(P, o, o.s1, kPositron, Tp, up, 1);
                t.E = 0.0;
                t.alive = 0;
            } else {
                o.null_int = 1;
            }
        }
    } else {
        const bool ioni = (proc == EMX_P_MOLLER || proc == EMX_P_BHABHA), brem = (proc == EMX_P_BREMS);
        if (ioni) {
            double Td, T1;
            Vec3 ud, u1;
            const bool ok = (proc == EMX_P_MOLLER) ? moller(rng, E1, m.Tcut, u0, Td, ud, T1, u1)
                                                   : bhabha(rng, E1, m.Tcut, u0, Td, ud, T1, u1);
            if (ok) {
                add_secondary(P, o, o.s0, kElectron, Td, ud, 0);
                t.E = T1;
                t.u = u1;
            } else {
                o.null_int = 1;
            }
        } else if (brem) {
            double k1, T1;
            Vec3 ug, u1;
            if (bremsstrahlung(rng, E1, m.kcut, u0, k1, ug, T1, u1)) {
                add_secondary(P, o, o.s0, kGamma, k1, ug, 0);
                t.E = T1;
                t.u = u1;
            } else {
                o.null_int = 1;
            }
        } else {
            double k1, k2;
            Vec3 u1, u2;
            annih_flight(rng, E1, u0, k1, u1, k2, u2);
            add_secondary(P, o, o.s0, kGamma, k1, u1, 0);
            add_secondary(P, o, o.s1, kGamma, k2, u2, 1);
            t.E = 0.0;
            t.alive = 0;
        }
    }
    if (t.alive && t.E < ph.E_trk) kill_below(P, pt, rng, t, o, t.E);
    finish_step(P, pt, t, o);
    o.n_draws = (int)rng.n;
}

// the whole step in one call (level-2 hook): the propagation is run to its end.  n_sub = substep attempts of the
// field propagation (0 without one)
template <bool CH, bool MAP = false, bool EXT = false>
EMX_HD void step(const Params &P, uint64_t seed, int pt, Track &t, StepOut &o, int &n_sub) {
    Carry c;
    Lookup L;
    L.Sig0 = L.Sig1 = L.Sig2 = L.Stot = L.D = L.R = L.iL0 = L.iL20 = L.var0 = 0.0;
    L.Rtab = nullptr;
    n_sub = 0;
    step_a0<CH, EXT>(P, seed, pt, t, c, L);
    if (c.action != kActCut) {
        if (!CH || P.Bmag == 0.0) {
            move_straight(P, t, c);
        } else {
            int hit, on_surf = t.surf;  // the slot's flag is rewritten by stage a2, not by the propagation
            const double s = propagate_field<MAP>(P, t.vol, on_surf, t.x, t.u, curvature(P, pt, t.E), c.s_phys, hit, n_sub);
            field_move_done(c, s, hit);
        }
    }
    const int proc = step_a2<CH, EXT, true>(P, seed, pt, t, o, c, L);
    if (proc >= 0) step_interact<CH>(P, seed, pt, t, o, proc);
}

}  // namespace emx
