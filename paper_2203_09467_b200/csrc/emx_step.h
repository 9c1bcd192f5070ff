// emx_step.h -- one step of one track (C7; PAPER.md:114 lists what a step must do:
// material-dependent properties, continuous slowing down, competition among discrete processes,
// scattering / absorption, secondary emission, energy cutoffs).  Steps A1-A8 of DESIGN.md section 2
// fused into one device function so that a track's state is read once and written once per step.
// step<PT>() is instantiated per particle type: each type has its own slot pool and kernel.
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
template <int PT>
EMX_HD void kill_below(const Params &P, Rng &rng, Track &t, StepOut &o, double E) {
    o.edep += E;
    o.below_cut += E;
    if (PT == kPositron) {
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

// One step of a live track of type PT (C7).  `t` is updated in place; `o` receives everything else.
// The step is written in two parts so that the loop can regroup tracks between them:
//   step_pre      items 1-7 of C7 plus the SELECTION of the discrete process (draws 0 and 1); returns the
//                 process id (EMX_P_*) if an interaction is pending, else -1 and the step is complete;
//   step_interact item 8 (the interactor, draws 2...) and item 9 for a track whose interaction is pending.
// step() = both, back to back (the level-2 hook).  `fs` / `budget`: time slicing of the field propagation
// (emx_field.h); pass attempt = 0 and a budget >= max_substeps to run the whole propagation in one call.
template <int PT>
EMX_HD void finish_step(const Params &P, Track &t, StepOut &o) {
    // 9. step counter, looper cap (R14)
    if (t.alive) {
        t.step += 1;
        if ((int)t.step >= P.ph.max_steps) {
            o.looper += t.E + (PT == kPositron ? 2.0 * kMe : 0.0);
            t.alive = 0;
        }
    }
}

// MAP: the magnetic field is non-uniform (evaluated at the stage positions of the integrator)
// EXT: the condensed-history extensions of e+- -- multiple scattering (emx_physics.msc) and / or energy-loss
// fluctuations (emx_physics.fluct) -- are switched on (their own instantiation, so that the kernels of a problem
// without them carry none of their registers)
template <int PT, bool MAP = false, bool EXT = false>
EMX_HD int step_pre(const Params &P, uint64_t seed, Track &t, StepOut &o, FieldState &fs, int budget) {
    const emx_physics &ph = P.ph;
    o.action = EMX_A_NONE;
    o.process = -1;
    o.s0.ptype = -1;
    o.s1.ptype = -1;
    o.rest_alloc = 0;
    o.edep = o.below_cut = o.escaped = o.looper = o.s = 0.0;
    o.msc_tau = 0.0;
    o.n_draws = o.null_int = o.rest = 0;
    o.suspended = 0;
    Rng rng;
    rng.init(seed, t.prim, t.tid, t.step);
    const int vol = t.vol;
    const int mat = P.vol[vol].material;

    // 1. tracking cut at step start
    if (t.E < ph.E_trk) {
        kill_below<PT>(P, rng, t, o, t.E);
        o.n_draws = (int)rng.n;
        return -1;
    }

    double Sig0 = 0.0, Sig1 = 0.0, Sig2 = 0.0, Stot = 0.0, D = 0.0, R = 0.0, s_phys;
    const bool msc = EXT && (PT != kGamma) && ph.msc && mat >= 0;  // multiple scattering applies (R-MSC)
    double iL0 = 0.0;                                       // 1 / lambda_1 at the pre-step energy
    double var0 = 0.0;                                      // variance of the loss per unit path at the pre-step energy
    const double *Rtab = nullptr;
    int action;
    const double E = t.E;
    if (mat < 0) {
        // 2. vacuum: no physics, capped flight
        s_phys = ph.vacuum_step;
        action = EMX_A_TRUNC;
    } else {
        // 3. lookup (C4), fixed process order
        const GridPos g = grid_pos(P, E);
        if (PT == kGamma) {
            Sig0 = interp(table(P, mat, EMX_T_COMPTON), g);
            Sig1 = interp(table(P, mat, EMX_T_PHOTO), g);
            Sig2 = interp(table(P, mat, EMX_T_PAIR), g);
        } else if (PT == kElectron) {
            Sig0 = interp(table(P, mat, EMX_T_MOLLER), g);
            Sig1 = interp(table(P, mat, EMX_T_BREMS_EM), g);
            D = interp(table(P, mat, EMX_T_DEDX_EM), g);
            Rtab = table(P, mat, EMX_T_RANGE_EM);
            R = interp(Rtab, g);
        } else {
            Sig0 = interp(table(P, mat, EMX_T_BHABHA), g);
            Sig1 = interp(table(P, mat, EMX_T_BREMS_EP), g);
            Sig2 = interp(table(P, mat, EMX_T_ANNIH), g);
            D = interp(table(P, mat, EMX_T_DEDX_EP), g);
            Rtab = table(P, mat, EMX_T_RANGE_EP);
            R = interp(Rtab, g);
        }
        Stot = (PT == kElectron) ? (Sig0 + Sig1) : (Sig0 + Sig1 + Sig2);
        // 4. limits: interaction length resampled every step (R27); continuous-loss step function (R9)
        const double xi = rng.next();
        s_phys = Stot > 0.0 ? -m_log(xi) / Stot : kInf;
        action = EMX_A_DISCRETE;
        if (PT != kGamma) {
            double s_loss;
            if (R <= ph.rho_R) s_loss = R;
            else s_loss = ph.alpha_R * R + ph.rho_R * (1.0 - ph.alpha_R) * (2.0 - ph.rho_R / R);
            if (s_loss < s_phys) {
                s_phys = s_loss;
                action = EMX_A_LOSS;
            }
            if (EXT && ph.fluct) var0 = interp(table(P, mat, PT == kElectron ? EMX_T_VAR_EM : EMX_T_VAR_EP), g);
            if (msc) {  // R-MSC step limit: s <= max(f_r max(R, lambda_1), s_min)
                iL0 = interp(table(P, mat, EMX_T_MSC), g);
                const double big = (iL0 > 0.0 && 1.0 / iL0 > R) ? 1.0 / iL0 : R;
                double s_msc = ph.msc_fr * big;
                if (s_msc < ph.msc_smin) s_msc = ph.msc_smin;
                if (s_msc < s_phys) {
                    s_phys = s_msc;
                    action = EMX_A_MSC;
                }
            }
        }
    }

    // 5. geometry / move
    double s;
    int hit = -1;
    bool full = true;  // the whole s_phys was travelled
    if (PT == kGamma || P.Bmag == 0.0) {
        const double d = distance_to_boundary(P, vol, t.x, t.u, t.surf, hit);
        if (d <= s_phys) {  // boundary wins ties (R10)
            s = d;
            action = EMX_A_BOUNDARY;
            full = false;
        } else {
            s = s_phys;
            hit = -1;
        }
        t.x.x += s * t.u.x;
        t.x.y += s * t.u.y;
        t.x.z += s * t.u.z;
    } else {
        const double pm = sqrt(E * (E + 2.0 * kMe));
        const double q = (PT == kElectron) ? -1.0 : 1.0;
        const double kappa = q * kCB * P.Bmag / pm;
        bool susp;
        s = propagate_field<MAP>(P, vol, t.surf, t.x, t.u, kappa, s_phys, hit, fs, budget, susp);
        if (susp) {  // x, u, surf and fs hold the progress; the step continues in the next iteration
            o.suspended = 1;
            return -1;
        }
        if (hit >= 0) {
            action = EMX_A_BOUNDARY;
            full = false;
        } else if (!(s >= s_phys * (1.0 - 1e-14))) {
            action = EMX_A_TRUNC;
            full = false;
        }
    }
    o.s = s;

    // 6. continuous loss (e+- in matter)
    if (PT != kGamma && mat >= 0) {
        double dE, f1 = 0.0, f2 = 0.0;
        const bool fl = EXT && ph.fluct;  // energy-loss fluctuations (R-FLUCT): two draws, always consumed
        if (fl) {
            f1 = rng.next();
            f2 = rng.next();
        }
        if (action == EMX_A_LOSS && R <= ph.rho_R && full) {
            dE = E;  // range stop
        } else {
            if (s * D <= ph.lin_loss * E) {
                dE = s * D;
            } else {
                const double E2 = range_inverse(P, Rtab, R - s);
                dE = E - E2;
                if (dE < 0.0) dE = 0.0;
                if (dE > E) dE = E;
            }
            if (fl && dE > 0.0) {
                dE = fluctuate_loss(dE, s * var0, E, f1, f2);
            }
        }
        t.E = E - dE;
        o.edep += dE;
        if (t.E < ph.E_trk) {
            o.action = action;
            kill_below<PT>(P, rng, t, o, t.E);
            o.n_draws = (int)rng.n;
            return -1;
        }
    }
    o.action = action;

    // 7. boundary crossing / relocation
    if (action == EMX_A_BOUNDARY) {
        const int nv = neighbour(P, t.x, t.u, hit);
        t.surf = hit;
        if (nv < 0) {  // left the world: escape (an e+ carries its rest-mass credit, R13)
            o.escaped += t.E + (PT == kPositron ? 2.0 * kMe : 0.0);
            t.alive = 0;
            o.n_draws = (int)rng.n;
            return -1;
        }
        t.vol = nv;
    } else {
        t.surf = -1;
    }

    // 7b. multiple-scattering deflection at the end of the step (R-MSC): <cos> = exp(-Int ds / lambda_1), the
    // integral by the trapezoid rule over the pre-step and post-loss energies; draws 1 and 2, always consumed
    if (msc) {
        const double iL1 = interp(table(P, mat, EMX_T_MSC), grid_pos(P, t.E));
        const double tau = 0.5 * (iL0 + iL1) * s;
        t.u = msc_deflect(rng, tau, t.u);
        o.msc_tau = tau;
    }

    // 8. discrete interaction: select with the pre-step cross sections, interact at the post-loss energy (R21)
    if (action == EMX_A_DISCRETE) {
        const double target = rng.next() * Stot;
        int k;
        if (PT == kElectron) {
            k = (Sig0 > target) ? 0 : 1;
            if (k == 1 && Sig1 <= 0.0) k = 0;
        } else {
            const double c1 = Sig0 + Sig1;
            k = (Sig0 > target) ? 0 : ((c1 > target) ? 1 : 2);
            if (k == 2 && Sig2 <= 0.0) k = 1;
            if (k == 1 && Sig1 <= 0.0) k = 0;
        }
        // k-th process of this particle type -> process id
        int proc;
        if (PT == kGamma) proc = (k == 0) ? EMX_P_COMPTON : (k == 1 ? EMX_P_PHOTO : EMX_P_PAIR);
        else if (PT == kElectron) proc = (k == 0) ? EMX_P_MOLLER : EMX_P_BREMS;
        else proc = (k == 0) ? EMX_P_BHABHA : (k == 1 ? EMX_P_BREMS : EMX_P_ANNIH);
        o.n_draws = (int)rng.n;
        return proc;  // interaction pending: the step is finished by step_interact
    }
    finish_step<PT>(P, t, o);
    o.n_draws = (int)rng.n;
    return -1;
}

// Item 8 of C7 for a track whose interaction `proc` was selected by step_pre: the interactor runs at the
// post-loss energy t.E with draws 2, 3, ... of the step, then item 9.
template <int PT>
EMX_HD void step_interact(const Params &P, uint64_t seed, Track &t, StepOut &o, int proc) {
    const emx_physics &ph = P.ph;
    Rng rng;
    rng.init(seed, t.prim, t.tid, t.step);
    const int mat = P.vol[t.vol].material;
    // draws 0 (interaction length) and the process selection were used by step_pre, and in between two each by
    // the energy-loss fluctuation (R-FLUCT) and the multiple-scattering deflection (R-MSC) of an e+-
    rng.n = (PT != kGamma) ? 2u + (ph.fluct ? 2u : 0u) + (ph.msc ? 2u : 0u) : 2u;
    const Material &m = P.mat[mat];
    const double E1 = t.E;
    const Vec3 u0 = t.u;
    o.process = proc;
    {
        if (PT == kGamma) {
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
                const bool ok = (PT == kElectron) ? moller(rng, E1, m.Tcut, u0, Td, ud, T1, u1)
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
        if (t.alive && t.E < ph.E_trk) kill_below<PT>(P, rng, t, o, t.E);
    }
    finish_step<PT>(P, t, o);
    o.n_draws = (int)rng.n;
}

// the whole step in one call
template <int PT, bool MAP = false, bool EXT = false>
EMX_HD void step(const Params &P, uint64_t seed, Track &t, StepOut &o, FieldState &fs, int budget) {
    const int proc = step_pre<PT, MAP, EXT>(P, seed, t, o, fs, budget);
    if (proc >= 0) step_interact<PT>(P, seed, t, o, proc);
}

}  // namespace emx
