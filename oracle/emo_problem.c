/* ORACLE (test infrastructure).  Problem description, material properties and
 * the physics tables on the log-spaced energy grid (PAPER.md:116, PAPER.md:128:
 * the paper imports tables from Geant4; BASELINE.json configs[0] says "cross
 * sections tabulated from closed forms" -> DESIGN.md R-C3, R-C4, R-C5.9, R-C5.10).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include "emo.h"

emo_problem *emo_create(void) {
    emo_problem *p = (emo_problem *)calloc(1, sizeof(emo_problem));
    if (!p) return NULL;
    emo_physics *ph = &p->ph;
    ph->process_mask = 63u;
    ph->E_min = 1e-3; ph->E_max = 1e4; ph->n_E = 256;
    ph->E_trk = 1e-3; ph->prod_cut_cm = 0.07;
    ph->alpha_R = 0.2; ph->rho_R = 0.1; ph->lin_loss = 0.01;
    ph->field_eps = 1e-7; ph->max_substeps = 1000; ph->vacuum_step = 1e3;
    ph->max_steps = 10000; ph->deposit_e_at_creation = 0;
    ph->msc = 0; ph->msc_fr = 0.2; ph->msc_smin = 1e-3; ph->fluct = 0; ph->integrator = 0;
    return p;
}

void emo_destroy(emo_problem *p) {
    if (!p) return;
    for (int i = 0; i < p->n_mat; ++i) free(p->mat[i].tab);
    free(p->mat); free(p->surf); free(p->vol); free(p);
}

/* I_eV is the material's mean excitation energy (compounds: the Bragg-additivity value
 * from DESIGN.md's material table is passed in by the caller). */
int emo_add_material(emo_problem *p, int n_elem, const int *Z, const double *A, const double *w,
                     double rho, double I_eV) {
    if (n_elem < 1 || n_elem > EMO_MAX_ELEM || rho <= 0.0 || I_eV <= 0.0) return -1;
    emo_material *nm = (emo_material *)realloc(p->mat, (size_t)(p->n_mat + 1) * sizeof(emo_material));
    if (!nm) return -2;
    p->mat = nm;
    emo_material *m = &p->mat[p->n_mat];
    memset(m, 0, sizeof(*m));
    m->n_elem = n_elem; m->rho = rho; m->I = I_eV * 1e-6;
    double invX0 = 0.0;
    for (int i = 0; i < n_elem; ++i) {
        m->Z[i] = Z[i]; m->A[i] = A[i]; m->w[i] = w[i];
        m->n_i[i] = rho * EMO_NA * w[i] / A[i];
        m->n_e += m->n_i[i] * Z[i];
        invX0 += rho * w[i] / emo_X0_elem_gcm2(Z[i], A[i]);
    }
    m->X0 = 1.0 / invX0;
    m->hwp = (EMO_ME / EMO_ALPHA) * sqrt(4.0 * EMO_PI * m->n_e * EMO_RE * EMO_RE * EMO_RE);
    m->Tcut = -1.0; m->kcut = -1.0;
    p->built = 0;
    return p->n_mat++;
}

int emo_add_surface(emo_problem *p, int type, double v) {
    if (type < EMO_S_PX || type > EMO_S_CZ) return -1;
    emo_surface *ns = (emo_surface *)realloc(p->surf, (size_t)(p->n_surf + 1) * sizeof(emo_surface));
    if (!ns) return -2;
    p->surf = ns;
    p->surf[p->n_surf].type = type; p->surf[p->n_surf].v = v;
    return p->n_surf++;
}

int emo_add_volume(emo_problem *p, int n_faces, const int *surf, const int *sense, int material, int tally) {
    if (n_faces < 0 || n_faces > EMO_MAX_FACES) return -1;
    emo_volume *nv = (emo_volume *)realloc(p->vol, (size_t)(p->n_vol + 1) * sizeof(emo_volume));
    if (!nv) return -2;
    p->vol = nv;
    emo_volume *v = &p->vol[p->n_vol];
    memset(v, 0, sizeof(*v));
    v->n_faces = n_faces;
    for (int i = 0; i < n_faces; ++i) {
        if (surf[i] < 0 || surf[i] >= p->n_surf || (sense[i] != 1 && sense[i] != -1)) return -1;
        v->surf[i] = surf[i]; v->sense[i] = sense[i];
    }
    v->material = material; v->tally = tally;
    if (tally + 1 > p->n_tally) p->n_tally = tally + 1;
    return p->n_vol++;
}

int emo_set_field(emo_problem *p, double Bx, double By, double Bz) {
    p->B[0] = Bx; p->B[1] = By; p->B[2] = Bz;
    p->Bmag = sqrt(Bx * Bx + By * By + Bz * Bz);
    for (int i = 0; i < 3; ++i) p->Bhat[i] = p->Bmag > 0.0 ? p->B[i] / p->Bmag : 0.0;
    p->field_kind = 0;
    return 0;
}

int emo_set_field_fringe(emo_problem *p, double z0_cm, double a_cm) {
    if (!(p->Bmag > 0.0) || p->B[0] != 0.0 || p->B[1] != 0.0 || !(z0_cm > 0.0) || !(a_cm > 0.0)) return -1;
    p->field_kind = 1; p->fringe_z0 = z0_cm; p->fringe_a = a_cm;
    return 0;
}

int emo_set_physics(emo_problem *p, const emo_physics *ph) {
    if (ph->n_E < 2 || !(ph->E_max > ph->E_min) || !(ph->E_min > 0.0)) return -1;
    if (ph->msc < 0 || ph->msc > 2) return -1;
    if (ph->integrator < 0 || ph->integrator > 1) return -1;
    if (ph->msc && (!(ph->msc_fr > 0.0) || !(ph->msc_smin > 0.0))) return -1;
    p->ph = *ph; p->built = 0;
    return 0;
}

int emo_set_cuts(emo_problem *p, int material, double Tcut, double kcut) {
    if (material < 0 || material >= p->n_mat) return -1;
    p->mat[material].Tcut = Tcut; p->mat[material].kcut = kcut; p->built = 0;
    return 0;
}

/* 4-point Gauss-Legendre on [0,1] */
static void gl4_unit(double t[4], double w[4]) {
    double x[4], ww[4];
    emo_gauss_legendre(4, x, ww);
    for (int q = 0; q < 4; ++q) { t[q] = 0.5 * (1.0 + x[q]); w[q] = 0.5 * ww[q]; }
}

static double dedx_total(const emo_material *m, int ptype, double T, double Tcut, double kcut) {
    return emo_dedx_col(m, ptype, T, Tcut) + emo_brems_dedx(T, kcut, m->X0);
}

/* range table: R_0 = E_0/dedx(E_0) (R24); R_j = R_{j-1} + Delta * sum_q w_q E_q / dedx(E_q) */
static void build_range(const emo_problem *p, const emo_material *m, int ptype, double Tcut, double kcut, double *R) {
    double t[4], w[4];
    gl4_unit(t, w);
    int n = p->ph.n_E;
    double E0 = exp(p->lnE0);
    R[0] = E0 / dedx_total(m, ptype, E0, Tcut, kcut);
    for (int j = 1; j < n; ++j) {
        double xl = p->lnE0 + (j - 1) * p->dlnE, sum = 0.0;
        for (int q = 0; q < 4; ++q) {
            double Eq = exp(xl + p->dlnE * t[q]);
            sum += w[q] * Eq * p->dlnE / dedx_total(m, ptype, Eq, Tcut, kcut);
        }
        R[j] = R[j - 1] + sum;
    }
}

int emo_build_tables(emo_problem *p) {
    const emo_physics *ph = &p->ph;
    int n = ph->n_E;
    p->lnE0 = log(ph->E_min);
    p->dlnE = log(ph->E_max / ph->E_min) / (n - 1);
    p->inv_dlnE = (n - 1) / log(ph->E_max / ph->E_min);
    double *Ru = (double *)malloc((size_t)n * sizeof(double));
    if (!Ru) return -2;
    for (int im = 0; im < p->n_mat; ++im) {
        emo_material *m = &p->mat[im];
        free(m->tab);
        m->tab = (double *)calloc((size_t)EMO_NTABLE * n, sizeof(double));
        if (!m->tab) { free(Ru); return -2; }
        double *T = m->tab;
        /* photon tables */
        for (int j = 0; j < n; ++j) {
            double E = exp(p->lnE0 + j * p->dlnE);
            if (ph->process_mask & EMO_M_COMPTON) T[EMO_T_COMPTON * n + j] = m->n_e * emo_sigma_kn(E);
            if (ph->process_mask & EMO_M_PHOTO) {
                double s = 0.0;
                for (int i = 0; i < m->n_elem; ++i) s += m->n_i[i] * emo_sigma_pe(m->Z[i], E);
                T[EMO_T_PHOTO * n + j] = s;
            }
            if (ph->process_mask & EMO_M_PAIR) {
                double s = 0.0;
                for (int i = 0; i < m->n_elem; ++i) {
                    double v = m->n_i[i] * emo_sigma_pair(m->Z[i], E);
                    T[(EMO_T_PAIR_ELEM0 + i) * n + j] = v;
                    s += v;
                }
                T[EMO_T_PAIR * n + j] = s;
            }
            if (ph->process_mask & EMO_M_ANNIH) T[EMO_T_ANNIH * n + j] = m->n_e * emo_sigma_annih(E);
        }
        /* production cuts from the cut length (R11 / C5.10) unless given explicitly */
        if (ph->prod_cut_cm > 0.0 && (m->Tcut < 0.0 || m->kcut < 0.0)) {
            double cut = ph->prod_cut_cm;
            build_range(p, m, EMO_ELECTRON, -1.0, -1.0, Ru);   /* unrestricted CSDA */
            double Tc;
            if (cut <= Ru[0]) Tc = ph->E_min;
            else if (cut >= Ru[n - 1]) Tc = ph->E_max;
            else {
                int j = 0;
                while (j < n - 2 && Ru[j + 1] <= cut) ++j;
                double f = (cut - Ru[j]) / (Ru[j + 1] - Ru[j]);
                Tc = exp(p->lnE0 + (j + f) * p->dlnE);
            }
            double kc = ph->E_max;
            for (int j = 0; j < n; ++j) {
                double S = T[EMO_T_COMPTON * n + j] + T[EMO_T_PHOTO * n + j] + T[EMO_T_PAIR * n + j];
                if (S > 0.0 && 5.0 / S >= cut) { kc = exp(p->lnE0 + j * p->dlnE); break; }
            }
            if (m->Tcut < 0.0) m->Tcut = Tc;
            if (m->kcut < 0.0) m->kcut = kc;
        }
        if (m->Tcut < 0.0 || m->kcut < 0.0) { free(Ru); return -3; }
        /* charged tables */
        for (int j = 0; j < n; ++j) {
            double E = exp(p->lnE0 + j * p->dlnE);
            if (ph->process_mask & EMO_M_IONI) {
                T[EMO_T_MOLLER * n + j] = m->n_e * emo_sigma_moller(E, m->Tcut);
                T[EMO_T_BHABHA * n + j] = m->n_e * emo_sigma_bhabha(E, m->Tcut);
            }
            if (ph->process_mask & EMO_M_BREMS) {
                double s = emo_brems_Sigma(E, m->kcut, m->X0);
                T[EMO_T_BREMS_EM * n + j] = s;
                T[EMO_T_BREMS_EP * n + j] = s;
            }
            if (ph->msc) {                                 /* 1/lambda_1 = sum_i n_i sigma_1(Z_i, E) (R-MSC) */
                double s = 0.0;
                for (int i = 0; i < m->n_elem; ++i) s += m->n_i[i] * emo_msc_sigma1(m->Z[i], m->A[i], E);
                T[EMO_T_MSC * n + j] = s;
                if (ph->msc == 2) {                        /* 1/lambda_2 (R-MSC2) */
                    double s2 = 0.0;
                    for (int i = 0; i < m->n_elem; ++i) s2 += m->n_i[i] * emo_msc_sigma2(m->Z[i], m->A[i], E);
                    T[EMO_T_MSC2 * n + j] = s2;
                }
            }
            if (ph->fluct) {                               /* variance of the loss per unit path (R-FLUCT) */
                T[EMO_T_VAR_EM * n + j] = m->n_e * emo_loss_second_moment(EMO_ELECTRON, E, m->Tcut);
                T[EMO_T_VAR_EP * n + j] = m->n_e * emo_loss_second_moment(EMO_POSITRON, E, m->Tcut);
            }
            T[EMO_T_DEDX_EM * n + j] = dedx_total(m, EMO_ELECTRON, E, m->Tcut, m->kcut);
            T[EMO_T_DEDX_EP * n + j] = dedx_total(m, EMO_POSITRON, E, m->Tcut, m->kcut);
        }
        build_range(p, m, EMO_ELECTRON, m->Tcut, m->kcut, &T[EMO_T_RANGE_EM * n]);
        build_range(p, m, EMO_POSITRON, m->Tcut, m->kcut, &T[EMO_T_RANGE_EP * n]);
    }
    free(Ru);
    p->built = 1;
    return 0;
}

int emo_get_table(const emo_problem *p, int material, int kind, double *out, int n) {
    if (!p->built || material < 0 || material >= p->n_mat || kind < 0 || kind >= EMO_NTABLE || n != p->ph.n_E) return -1;
    memcpy(out, &p->mat[material].tab[(size_t)kind * n], (size_t)n * sizeof(double));
    return 0;
}

int emo_get_material_info(const emo_problem *p, int material, double *o) {
    if (material < 0 || material >= p->n_mat) return -1;
    const emo_material *m = &p->mat[material];
    o[0] = m->n_e; o[1] = m->I; o[2] = m->hwp; o[3] = m->X0; o[4] = m->Tcut; o[5] = m->kcut; o[6] = m->rho; o[7] = m->n_elem;
    return 0;
}

/* C4: linear interpolation in ln E, clamped */
double emo_lookup(const emo_problem *p, int material, int kind, double E) {
    int n = p->ph.n_E;
    const double *T = &p->mat[material].tab[(size_t)kind * n];
    double t = (log(E) - p->lnE0) * p->inv_dlnE;
    int j = (int)floor(t);
    if (j < 0) j = 0;
    if (j > n - 2) j = n - 2;
    double f = t - j;
    if (f < 0.0) f = 0.0;
    if (f > 1.0) f = 1.0;
    return (1.0 - f) * T[j] + f * T[j + 1];
}

/* exact inverse of the forward rule on a range table (C5.9) */
double emo_range_inverse(const emo_problem *p, int material, int kind_range, double r) {
    int n = p->ph.n_E;
    const double *R = &p->mat[material].tab[(size_t)kind_range * n];
    if (r <= R[0]) return exp(p->lnE0) * (r / R[0]);          /* constant dE/dx below the grid */
    if (r >= R[n - 1]) return exp(p->lnE0 + (n - 1) * p->dlnE);
    int lo = 0, hi = n - 1;                                   /* R[lo] <= r < R[hi] */
    while (hi - lo > 1) {
        int mid = (lo + hi) / 2;
        if (R[mid] <= r) lo = mid; else hi = mid;
    }
    double f = (r - R[lo]) / (R[lo + 1] - R[lo]);
    return exp(p->lnE0 + (lo + f) * p->dlnE);
}
