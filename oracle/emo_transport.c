/* ORACLE (test infrastructure).  One step of one track, and the one-track-at-a-
 * time transport loop with a LIFO stack per primary.
 * Paper: PAPER.md:114 lists what a step must do (material-dependent properties,
 * continuous slowing down, selection among competing discrete processes,
 * scattering/absorption, secondary emission, energy cutoffs); PAPER.md:70 the
 * secondary stack; PAPER.md:204-212 the loop until no tracks/initializers
 * remain.  The order of operations, draw order and tie-breaks are the readings
 * of DESIGN.md R-C7, R-C10, R-C11.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include "emo.h"

typedef struct {
    const emo_problem *p;
    uint64_t seed;
    emo_rng rng;
    emo_step_result *o;
} ctx_t;

/* C10: secondary of type pt, energy E, direction d, ordinal ord, born at the track's position */
static void add_sec(ctx_t *c, int pt, double E, const double d[3], int ord) {
    emo_step_result *o = c->o;
    const emo_physics *ph = &c->p->ph;
    if (pt == EMO_ELECTRON && ph->deposit_e_at_creation) { o->edep += E; return; }
    if (pt != EMO_POSITRON && E < ph->E_trk) { o->edep += E; o->below_cut += E; return; }
    emo_track *s = &o->sec[o->n_sec];
    memset(s, 0, sizeof(*s));
    for (int i = 0; i < 3; ++i) { s->x[i] = o->trk.x[i]; s->u[i] = d[i]; }
    s->E = E;
    s->tid = emo_child_tid(c->seed, o->trk.prim, o->trk.tid, o->trk.step, (uint32_t)ord);
    s->prim = o->trk.prim; s->step = 0;
    s->vol = o->trk.vol; s->surf = -1; s->ptype = pt; s->alive = 1;
    o->sec_ord[o->n_sec] = ord;
    o->n_sec++;
}

/* tracking-cut kill: deposit E locally; e+ annihilates at rest (R12/R25) */
static void kill_below(ctx_t *c, double E) {
    emo_step_result *o = c->o;
    o->edep += E; o->below_cut += E;
    if (o->trk.ptype == EMO_POSITRON) {
        double u1[3], u2[3];
        emo_annih_rest(&c->rng, u1, u2);
        add_sec(c, EMO_GAMMA, EMO_ME, u1, 2);
        add_sec(c, EMO_GAMMA, EMO_ME, u2, 3);
        o->rest = 1;
    }
    o->trk.E = 0.0;
    o->trk.alive = 0;
}

void emo_step(const emo_problem *p, uint64_t seed, const emo_track *in, emo_step_result *out) {
    const emo_physics *ph = &p->ph;
    memset(out, 0, sizeof(*out));
    out->trk = *in;
    out->process = -1;
    out->edep_vol = in->vol;
    emo_track *t = &out->trk;
    ctx_t c; c.p = p; c.seed = seed; c.o = out;
    c.rng.seed = seed; c.rng.prim = t->prim; c.rng.tid = t->tid; c.rng.step = t->step; c.rng.n = 0;
    const int pt = t->ptype;
    const int vol = t->vol;
    const int mat = p->vol[vol].material;

    /* 1. tracking cut at step start */
    if (t->E < ph->E_trk) { kill_below(&c, t->E); out->n_draws = (int)c.rng.n; return; }

    double Sig[3] = {0, 0, 0}, Stot = 0.0, D = 0.0, R = 0.0, s_phys, s_loss = INFINITY;
    const int msc = (ph->msc && pt != EMO_GAMMA && mat >= 0);   /* multiple scattering applies (R-MSC) */
    const int msc2 = (msc && ph->msc == 2);                      /* ... with Lewis' spatial moments (R-MSC2) */
    double iL0 = 0.0;                                            /* 1/lambda_1 at the pre-step energy */
    int nproc = 0, procs[3] = {-1, -1, -1};
    int action;
    const double E = t->E;
    if (mat < 0) {
        /* 2. vacuum */
        s_phys = ph->vacuum_step; action = EMO_A_TRUNC;
    } else {
        /* 3. lookup (C4), fixed process order */
        if (pt == EMO_GAMMA) {
            nproc = 3; procs[0] = EMO_P_COMPTON; procs[1] = EMO_P_PHOTO; procs[2] = EMO_P_PAIR;
            Sig[0] = emo_lookup(p, mat, EMO_T_COMPTON, E);
            Sig[1] = emo_lookup(p, mat, EMO_T_PHOTO, E);
            Sig[2] = emo_lookup(p, mat, EMO_T_PAIR, E);
        } else if (pt == EMO_ELECTRON) {
            nproc = 2; procs[0] = EMO_P_MOLLER; procs[1] = EMO_P_BREMS;
            Sig[0] = emo_lookup(p, mat, EMO_T_MOLLER, E);
            Sig[1] = emo_lookup(p, mat, EMO_T_BREMS_EM, E);
            D = emo_lookup(p, mat, EMO_T_DEDX_EM, E);
            R = emo_lookup(p, mat, EMO_T_RANGE_EM, E);
        } else {
            nproc = 3; procs[0] = EMO_P_BHABHA; procs[1] = EMO_P_BREMS; procs[2] = EMO_P_ANNIH;
            Sig[0] = emo_lookup(p, mat, EMO_T_BHABHA, E);
            Sig[1] = emo_lookup(p, mat, EMO_T_BREMS_EP, E);
            Sig[2] = emo_lookup(p, mat, EMO_T_ANNIH, E);
            D = emo_lookup(p, mat, EMO_T_DEDX_EP, E);
            R = emo_lookup(p, mat, EMO_T_RANGE_EP, E);
        }
        for (int k = 0; k < nproc; ++k) Stot += Sig[k];
        /* 4. limits */
        double xi = emo_next(&c.rng);
        double s_int = Stot > 0.0 ? -log(xi) / Stot : INFINITY;
        s_phys = s_int; action = EMO_A_DISCRETE;
        if (pt != EMO_GAMMA) {
            if (R <= ph->rho_R) s_loss = R;
            else s_loss = ph->alpha_R * R + ph->rho_R * (1.0 - ph->alpha_R) * (2.0 - ph->rho_R / R);
            if (s_loss < s_phys) { s_phys = s_loss; action = EMO_A_LOSS; }
        }
        if (msc) {
            /* R-MSC step limit: s <= max(f_r max(R, lambda_1), s_min) */
            iL0 = emo_lookup(p, mat, EMO_T_MSC, E);
            double big = (iL0 > 0.0 && 1.0 / iL0 > R) ? 1.0 / iL0 : R;
            double s_msc = ph->msc_fr * big;
            if (s_msc < ph->msc_smin) s_msc = ph->msc_smin;
            if (s_msc < s_phys) { s_phys = s_msc; action = EMO_A_MSC; }
        }
    }

    /* 5. geometry / move.  R-MSC2: s_phys is the TRUE path length t of the step; the track is moved by the mean
     * geometric length z(t) = lambda_1 (1 - exp(-t / lambda_1)) of Lewis' theory (lambda_1 at the pre-step energy).
     * A move cut short after the geometric length g < z(t) stands for the true length t g / z(t). */
    double s_move = msc2 ? emo_msc_geom_length(s_phys, iL0) : s_phys;
    double s;
    int hit = -1;
    int full = 1;                         /* the full s_phys was travelled */
    if (pt == EMO_GAMMA || p->Bmag == 0.0) {
        double d = emo_distance(p, vol, t->x, t->u, t->surf, &hit);
        if (d <= s_move) { s = d; action = EMO_A_BOUNDARY; full = 0; }
        else { s = s_move; hit = -1; }
        for (int i = 0; i < 3; ++i) t->x[i] += s * t->u[i];
    } else {
        double pm = sqrt(E * (E + 2.0 * EMO_ME));
        double q = (pt == EMO_ELECTRON) ? -1.0 : 1.0;
        double kappa = q * EMO_CB * p->Bmag / pm;
        int sf = t->surf;
        s = emo_propagate_field_n(p, vol, &sf, t->x, t->u, kappa, s_move, &hit, &out->n_sub);
        if (hit >= 0) { action = EMO_A_BOUNDARY; full = 0; }
        else if (!(s >= s_move * (1.0 - 1e-14))) { action = EMO_A_TRUNC; full = 0; }
    }
    if (msc2) s = full ? s_phys : s_phys * (s / s_move);   /* from here on s is the true path length */
    out->s = s;

    /* 6. continuous loss (e+- in matter) */
    if (pt != EMO_GAMMA && mat >= 0) {
        double dE, f1 = 0.0, f2 = 0.0;
        if (ph->fluct) { f1 = emo_next(&c.rng); f2 = emo_next(&c.rng); }          /* R-FLUCT: always consumed */
        if (action == EMO_A_LOSS && R <= ph->rho_R && full) dE = E;              /* range stop */
        else {
            if (s * D <= ph->lin_loss * E) dE = s * D;
            else {
                double E2 = emo_range_inverse(p, mat, pt == EMO_ELECTRON ? EMO_T_RANGE_EM : EMO_T_RANGE_EP, R - s);
                dE = E - E2;
                if (dE < 0.0) dE = 0.0;
                if (dE > E) dE = E;
            }
            if (ph->fluct && dE > 0.0) {                                         /* R-FLUCT */
                double V = s * emo_lookup(p, mat, pt == EMO_ELECTRON ? EMO_T_VAR_EM : EMO_T_VAR_EP, E);
                dE = emo_fluctuate_loss(dE, V, E, f1, f2);
            }
        }
        t->E = E - dE;
        out->edep += dE;
        if (t->E < ph->E_trk) { out->action = action; kill_below(&c, t->E); out->n_draws = (int)c.rng.n; return; }
    }
    out->action = action;

    /* 7. boundary */
    if (action == EMO_A_BOUNDARY) {
        int nv = emo_neighbour(p, t->x, t->u, hit);
        t->surf = hit;
        if (nv < 0) {
            out->escaped += t->E + (pt == EMO_POSITRON ? 2.0 * EMO_ME : 0.0);
            t->alive = 0;
            out->n_draws = (int)c.rng.n;
            return;
        }
        t->vol = nv;
    } else {
        t->surf = -1;
    }

    /* 7b. multiple-scattering deflection at the end of the step (R-MSC): <cos> = exp(-Int ds / lambda_1), the
     * integral by the trapezoid rule over the pre-step and post-loss energies; two draws, always consumed */
    if (msc) {
        double iL1 = emo_lookup(p, mat, EMO_T_MSC, t->E);
        double tau = 0.5 * (iL0 + iL1) * s;
        double u0[3] = { t->u[0], t->u[1], t->u[2] }, u1[3];
        emo_msc_deflect(&c.rng, tau, u0, u1);
        t->u[0] = u1[0]; t->u[1] = u1[1]; t->u[2] = u1[2];
        out->msc_tau = tau;
        /* R-MSC2 lateral displacement: along the transverse part of the new direction, d = u1 - (u0.u1) u0 with
         * |d| = sin(theta), by rho = sqrt(3 <r^2> / (2 (1 - g^2))) sin(theta): for the Henyey-Greenstein angle
         * <sin^2(theta)> = (2/3)(1 - g^2), g = exp(-tau), so <rho^2> is Lewis' <x^2 + y^2> of the true path s
         * (lambda_1, lambda_2 averaged over the pre-step and post-loss energies like tau).  No draw of its own.
         * The track stays inside its cell: rho <= 0.9 x the distance to the cell's boundary along d; a step that
         * ended ON a boundary is not displaced. */
        if (msc2 && action != EMO_A_BOUNDARY) {
            double il1 = 0.5 * (iL0 + iL1);
            double il2 = 0.5 * (emo_lookup(p, mat, EMO_T_MSC2, E) + emo_lookup(p, mat, EMO_T_MSC2, t->E));
            double r2 = emo_msc_lateral_r2(s, il1, il2);
            double om = -expm1(-2.0 * tau);
            double mu = u0[0] * u1[0] + u0[1] * u1[1] + u0[2] * u1[2];
            double d[3] = { u1[0] - mu * u0[0], u1[1] - mu * u0[1], u1[2] - mu * u0[2] };
            double dn = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            if (r2 > 0.0 && om > 0.0 && dn > 0.0) {
                double rho = sqrt(1.5 * r2 / om) * dn;
                double dh[3] = { d[0] / dn, d[1] / dn, d[2] / dn };
                int hs;
                double lim = 0.9 * emo_distance(p, t->vol, t->x, dh, -1, &hs);
                if (rho > lim) rho = lim;
                for (int i = 0; i < 3; ++i) t->x[i] += rho * dh[i];
            }
        }
    }

    /* 8. discrete */
    if (action == EMO_A_DISCRETE) {
        double xi = emo_next(&c.rng);
        double target = xi * Stot, cum = 0.0;
        int k = nproc - 1;
        for (int i = 0; i < nproc; ++i) { cum += Sig[i]; if (cum > target) { k = i; break; } }
        while (k > 0 && Sig[k] <= 0.0) --k;               /* rounding fallback never picks a disabled process */
        int proc = procs[k];
        out->process = proc;
        const double E1 = t->E;                            /* post-loss energy */
        const emo_material *m = &p->mat[mat];
        double u0[3] = { t->u[0], t->u[1], t->u[2] };
        switch (proc) {
        case EMO_P_COMPTON: {
            double Eg, ug[3], Te, ue[3];
            emo_compton(&c.rng, E1, u0, &Eg, ug, &Te, ue);
            add_sec(&c, EMO_ELECTRON, Te, ue, 0);
            t->E = Eg; t->u[0] = ug[0]; t->u[1] = ug[1]; t->u[2] = ug[2];
        } break;
        case EMO_P_PHOTO: {
            if (ph->deposit_e_at_creation) out->edep += E1;
            else { double ue[3]; emo_photo_dir(&c.rng, E1, u0, ue); add_sec(&c, EMO_ELECTRON, E1, ue, 0); }
            t->E = 0.0; t->alive = 0;
        } break;
        case EMO_P_PAIR: {
            int ie = 0;
            if (m->n_elem > 1) {                           /* element selection (R4) */
                double xe = emo_next(&c.rng);
                double se[EMO_MAX_ELEM], st = 0.0;
                for (int i = 0; i < m->n_elem; ++i) { se[i] = emo_lookup(p, mat, EMO_T_PAIR_ELEM0 + i, E1); st += se[i]; }
                double cc = 0.0; ie = m->n_elem - 1;
                for (int i = 0; i < m->n_elem; ++i) { cc += se[i]; if (cc > xe * st) { ie = i; break; } }
            }
            double Tm, um[3], Tp, up[3];
            if (emo_pair(&c.rng, m->Z[ie], E1, u0, &Tm, um, &Tp, up)) {
                add_sec(&c, EMO_ELECTRON, Tm, um, 0);
                add_sec(&c, EMO_POSITRON, Tp, up, 1);
                t->E = 0.0; t->alive = 0;
            } else out->null_int = 1;
        } break;
        case EMO_P_MOLLER: case EMO_P_BHABHA: {
            double Td, ud[3], T1, u1[3];
            int ok = (proc == EMO_P_MOLLER) ? emo_moller(&c.rng, E1, m->Tcut, u0, &Td, ud, &T1, u1)
                                            : emo_bhabha(&c.rng, E1, m->Tcut, u0, &Td, ud, &T1, u1);
            if (ok) {
                add_sec(&c, EMO_ELECTRON, Td, ud, 0);
                t->E = T1; t->u[0] = u1[0]; t->u[1] = u1[1]; t->u[2] = u1[2];
            } else out->null_int = 1;
        } break;
        case EMO_P_BREMS: {
            double k1, ug[3], T1, u1[3];
            if (emo_brems(&c.rng, E1, m->kcut, u0, &k1, ug, &T1, u1)) {
                add_sec(&c, EMO_GAMMA, k1, ug, 0);
                t->E = T1; t->u[0] = u1[0]; t->u[1] = u1[1]; t->u[2] = u1[2];
            } else out->null_int = 1;
        } break;
        case EMO_P_ANNIH: {
            double k1, u1[3], k2, u2[3];
            emo_annih_flight(&c.rng, E1, u0, &k1, u1, &k2, u2);
            add_sec(&c, EMO_GAMMA, k1, u1, 0);
            add_sec(&c, EMO_GAMMA, k2, u2, 1);
            t->E = 0.0; t->alive = 0;
        } break;
        default: break;
        }
        if (t->alive && t->E < ph->E_trk) kill_below(&c, t->E);
    }

    /* 9. step counter, looper cap (R14) */
    if (t->alive) {
        t->step += 1;
        if ((int)t->step >= ph->max_steps) {
            out->looper += t->E + (pt == EMO_POSITRON ? 2.0 * EMO_ME : 0.0);
            t->alive = 0;
        }
    }
    out->n_draws = (int)c.rng.n;
}

int emo_step_batch(const emo_problem *p, uint64_t seed, long n, const emo_track *in, emo_step_result *out) {
    if (!p->built) return -1;
#pragma omp parallel for schedule(dynamic, 64)
    for (long i = 0; i < n; ++i) emo_step(p, seed, &in[i], &out[i]);
    return 0;
}

int emo_step_bin(uint64_t n) {
    int b;
    if (n < 16) b = (int)n;
    else {
        int e = 0;
        while ((n >> e) > 1) ++e;                        /* e = floor(log2 n) >= 4 */
        b = 16 + 4 * (e - 4) + (int)((n >> (e - 2)) & 3);
    }
    return b < EMO_NHIST ? b : EMO_NHIST - 1;
}

typedef struct { emo_track *v; size_t n, cap; } stack_t;
static int push(stack_t *s, const emo_track *t) {
    if (s->n == s->cap) {
        size_t nc = s->cap ? 2 * s->cap : 256;
        emo_track *nv = (emo_track *)realloc(s->v, nc * sizeof(emo_track));
        if (!nv) return -1;
        s->v = nv; s->cap = nc;
    }
    s->v[s->n++] = *t;
    return 0;
}

/* transport: per primary a LIFO stack; secondaries pushed in ordinal order, popped until empty (C10) */
int emo_transport(const emo_problem *p, long n_prim, const int *ptype, const double *E,
                  const double *pos3, const double *dir3, const int *start_vol, const int *start_surf,
                  uint64_t seed, int n_threads, double *edep, emo_scalars *sc,
                  double *per_prim, double *per_prim_tally) {
    if (!p->built) return -1;
    const int nt = p->n_tally;
    memset(sc, 0, sizeof(*sc));
    for (int i = 0; i < nt; ++i) edep[i] = 0.0;
    int fail = 0;
    (void)n_threads;
#pragma omp parallel num_threads(n_threads > 0 ? n_threads : 1)
    {
        stack_t st = { NULL, 0, 0 };
        double *led = (double *)calloc((size_t)(nt > 0 ? nt : 1), sizeof(double));   /* thread-local sums */
        double *ped = (double *)calloc((size_t)(nt > 0 ? nt : 1), sizeof(double));   /* this primary */
        emo_scalars ls; memset(&ls, 0, sizeof(ls));
        emo_step_result *r = (emo_step_result *)malloc(sizeof(emo_step_result));
#pragma omp for schedule(dynamic, 1)
        for (long ip = 0; ip < n_prim; ++ip) {
            if (!led || !ped || !r) { fail = 1; continue; }
            emo_track t0; memset(&t0, 0, sizeof(t0));
            for (int i = 0; i < 3; ++i) { t0.x[i] = pos3[3 * ip + i]; t0.u[i] = dir3[3 * ip + i]; }
            t0.E = E[ip]; t0.tid = 0; t0.prim = (uint32_t)ip; t0.step = 0;
            t0.vol = start_vol[ip]; t0.surf = start_surf ? start_surf[ip] : -1;
            t0.ptype = ptype[ip]; t0.alive = 1;
            double pe_tot = 0.0, pe_esc = 0.0, pe_loop = 0.0, pe_bc = 0.0;
            double pst[3] = {0, 0, 0}, ptr[3] = {0, 0, 0};
            double Ein = t0.E + (t0.ptype == EMO_POSITRON ? 2.0 * EMO_ME : 0.0);
            for (int i = 0; i < nt; ++i) ped[i] = 0.0;
            st.n = 0;
            if (push(&st, &t0)) { fail = 1; continue; }
            ls.tracks[t0.ptype]++; ptr[t0.ptype] += 1.0;
            while (st.n > 0) {
                emo_track t = st.v[--st.n];
                uint64_t taken = 0;                       /* steps of this track */
                while (t.alive) {
                    emo_step(p, seed, &t, r);
                    ++taken;
                    ls.steps[t.ptype]++; ls.track_steps++; pst[t.ptype] += 1.0;
                    if (r->edep != 0.0) {
                        int tl = p->vol[r->edep_vol].tally;
                        if (tl >= 0) ped[tl] += r->edep;
                        pe_tot += r->edep;
                    }
                    pe_bc += r->below_cut; pe_esc += r->escaped; pe_loop += r->looper;
                    if (r->process >= 0) { if (r->null_int) ls.null_int++; else ls.inter[r->process]++; }
                    if (r->rest) ls.inter[EMO_P_REST]++;
                    for (int k = 0; k < r->n_sec; ++k) {
                        if (push(&st, &r->sec[k])) { fail = 1; break; }
                        ls.tracks[r->sec[k].ptype]++; ptr[r->sec[k].ptype] += 1.0;
                    }
                    t = r->trk;
                }
                ls.step_hist[t.ptype][emo_step_bin(taken)]++;
            }
            for (int i = 0; i < nt; ++i) led[i] += ped[i];
            ls.below_cut += pe_bc; ls.escaped += pe_esc; ls.looper += pe_loop; ls.E_in += Ein;
            if (per_prim) {
                double *q = &per_prim[(size_t)EMO_PER_PRIM * ip];
                q[0] = pe_tot; q[1] = pe_esc; q[2] = pe_loop; q[3] = pe_bc; q[4] = Ein;
                q[5] = pst[0]; q[6] = pst[1]; q[7] = pst[2]; q[8] = ptr[0]; q[9] = ptr[1]; q[10] = ptr[2];
            }
            if (per_prim_tally) for (int i = 0; i < nt; ++i) per_prim_tally[(size_t)nt * ip + i] = ped[i];
        }
#pragma omp critical(emo_merge)
        {
            if (led) for (int i = 0; i < nt; ++i) edep[i] += led[i];
            sc->escaped += ls.escaped; sc->below_cut += ls.below_cut; sc->looper += ls.looper; sc->E_in += ls.E_in;
            for (int i = 0; i < 3; ++i) { sc->steps[i] += ls.steps[i]; sc->tracks[i] += ls.tracks[i]; }
            for (int i = 0; i < EMO_NPROC; ++i) sc->inter[i] += ls.inter[i];
            sc->null_int += ls.null_int; sc->track_steps += ls.track_steps;
            for (int i = 0; i < 3; ++i)
                for (int b = 0; b < EMO_NHIST; ++b) sc->step_hist[i][b] += ls.step_hist[i][b];
        }
        free(st.v); free(led); free(ped); free(r);
    }
    return fail ? -2 : 0;
}
