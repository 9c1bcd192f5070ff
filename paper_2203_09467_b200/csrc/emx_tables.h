// emx_tables.h -- per-entry work of the physics-table builder (step A11 of DESIGN.md).
// PAPER.md:128 imports every table from Geant4 through a ROOT file; BASELINE.json configs[0] asks for
// "cross sections tabulated from closed forms", so the tables are computed on the device by the kernels in
// emx_kernels.cu, one thread per (material, grid point), from the closed forms of emx_xs.h.
// Layout: tab[(mat * EMX_NTABLE + kind) * n_E + j], value at E_j = exp(lnE0 + j dlnE) (C4).
#pragma once
#include "emx_core.h"
#include "emx_xs.h"

namespace emx {

struct TableCtx {
    emx_physics ph;
    double lnE0, dlnE;
    int n_mat;
    Material *mat;   // device, writable: the builder fills in Tcut / kcut
    double *tab;     // device
    double *scratch; // device, n_mat * n_E doubles (unrestricted CSDA range for the cut conversion)
};

EMX_HD double grid_E(const TableCtx &c, int j) { return exp(c.lnE0 + j * c.dlnE); }

// range increment of bin (j-1, j): Delta * sum_q w_q E_q / dedx(E_q), 4-point Gauss-Legendre in ln E on the
// closed forms (C5.9); j = 0 gives R_0 = E_0 / dedx(E_0) (R24)
EMX_HD double range_bin(const TableCtx &c, const Material &m, int ptype, double Tcut, double kcut, int j) {
    if (j == 0) {
        const double E0 = exp(c.lnE0);
        return E0 / dedx_total(m, ptype, E0, Tcut, kcut);
    }
    const double xl = c.lnE0 + (j - 1) * c.dlnE;
    double sum = 0.0;
    for (int q = 0; q < 4; ++q) {
        const double tq = 0.5 * (1.0 + gl4_x(q)), wq = 0.5 * gl4_w(q);
        const double Eq = exp(xl + c.dlnE * tq);
        sum += wq * Eq * c.dlnE / dedx_total(m, ptype, Eq, Tcut, kcut);
    }
    return sum;
}

// pass 1: photon tables, annihilation, and the unrestricted e- range increments
EMX_HD void table_pass1(const TableCtx &c, int im, int j) {
    const Material &m = c.mat[im];
    const int n = c.ph.n_E;
    double *T = c.tab + (size_t)im * EMX_NTABLE * n;
    const double E = grid_E(c, j);
    const unsigned mask = c.ph.process_mask;
    T[EMX_T_COMPTON * n + j] = (mask & EMX_M_COMPTON) ? m.n_e * sigma_kn(E) : 0.0;
    double pe = 0.0;
    if (mask & EMX_M_PHOTO)
        for (int i = 0; i < m.n_elem; ++i) pe += m.n_i[i] * sigma_pe(m.Z[i], E);
    T[EMX_T_PHOTO * n + j] = pe;
    double pr = 0.0;
    for (int i = 0; i < EMX_MAX_ELEM; ++i) {
        double v = 0.0;
        if ((mask & EMX_M_PAIR) && i < m.n_elem) {
            v = m.n_i[i] * sigma_pair(m.Z[i], E);
            pr += v;
        }
        T[(EMX_T_PAIR_ELEM0 + i) * n + j] = v;
    }
    T[EMX_T_PAIR * n + j] = pr;
    T[EMX_T_ANNIH * n + j] = (mask & EMX_M_ANNIH) ? m.n_e * sigma_annih(E) : 0.0;
    c.scratch[(size_t)im * n + j] = range_bin(c, m, kElectron, -1.0, -1.0, j);
}

// pass 2 (one thread per material): production thresholds from the cut length (C5.10, R11)
EMX_HD void table_cuts(const TableCtx &c, int im) {
    Material &m = c.mat[im];
    const int n = c.ph.n_E;
    const double *T = c.tab + (size_t)im * EMX_NTABLE * n;
    double *Ru = c.scratch + (size_t)im * n;
    if (!(c.ph.prod_cut_cm > 0.0) || (m.Tcut >= 0.0 && m.kcut >= 0.0)) return;
    const double cut = c.ph.prod_cut_cm;
    for (int j = 1; j < n; ++j) Ru[j] = Ru[j - 1] + Ru[j];  // sequential prefix sum: fixed summation order
    double Tc;
    if (cut <= Ru[0]) Tc = c.ph.E_min;
    else if (cut >= Ru[n - 1]) Tc = c.ph.E_max;
    else {
        int j = 0;
        while (j < n - 2 && Ru[j + 1] <= cut) ++j;
        const double f = (cut - Ru[j]) / (Ru[j + 1] - Ru[j]);
        Tc = exp(c.lnE0 + (j + f) * c.dlnE);
    }
    double kc = c.ph.E_max;
    for (int j = 0; j < n; ++j) {
        const double S = T[EMX_T_COMPTON * n + j] + T[EMX_T_PHOTO * n + j] + T[EMX_T_PAIR * n + j];
        if (S > 0.0 && 5.0 / S >= cut) {
            kc = grid_E(c, j);
            break;
        }
    }
    if (m.Tcut < 0.0) m.Tcut = Tc;
    if (m.kcut < 0.0) m.kcut = kc;
}

// pass 3: charged-particle tables and restricted range increments
EMX_HD void table_pass3(const TableCtx &c, int im, int j) {
    const Material &m = c.mat[im];
    const int n = c.ph.n_E;
    double *T = c.tab + (size_t)im * EMX_NTABLE * n;
    const double E = grid_E(c, j);
    const unsigned mask = c.ph.process_mask;
    T[EMX_T_MOLLER * n + j] = (mask & EMX_M_IONI) ? m.n_e * sigma_moller(E, m.Tcut) : 0.0;
    T[EMX_T_BHABHA * n + j] = (mask & EMX_M_IONI) ? m.n_e * sigma_bhabha(E, m.Tcut) : 0.0;
    const double sb = (mask & EMX_M_BREMS) ? brems_Sigma(E, m.kcut, m.X0) : 0.0;
    T[EMX_T_BREMS_EM * n + j] = sb;
    T[EMX_T_BREMS_EP * n + j] = sb;
    double il = 0.0;  // 1 / lambda_1 = sum_i n_i sigma_1(Z_i) (R-MSC)
    if (c.ph.msc)
        for (int i = 0; i < m.n_elem; ++i) il += m.n_i[i] * msc_sigma1(m.Z[i], m.A[i], E);
    T[EMX_T_MSC * n + j] = il;
    double il2 = 0.0;  // 1 / lambda_2 (R-MSC2)
    if (c.ph.msc == 2)
        for (int i = 0; i < m.n_elem; ++i) il2 += m.n_i[i] * msc_sigma2(m.Z[i], m.A[i], E);
    T[EMX_T_MSC2 * n + j] = il2;
    T[EMX_T_VAR_EM * n + j] = c.ph.fluct ? m.n_e * loss_second_moment(kElectron, E, m.Tcut) : 0.0;  // R-FLUCT
    T[EMX_T_VAR_EP * n + j] = c.ph.fluct ? m.n_e * loss_second_moment(kPositron, E, m.Tcut) : 0.0;
    T[EMX_T_DEDX_EM * n + j] = dedx_total(m, kElectron, E, m.Tcut, m.kcut);
    T[EMX_T_DEDX_EP * n + j] = dedx_total(m, kPositron, E, m.Tcut, m.kcut);
    T[EMX_T_RANGE_EM * n + j] = range_bin(c, m, kElectron, m.Tcut, m.kcut, j);
    T[EMX_T_RANGE_EP * n + j] = range_bin(c, m, kPositron, m.Tcut, m.kcut, j);
}

// pass 4 (one thread per (material, e-/e+)): range = sequential prefix sum of the increments
EMX_HD void table_range_sum(const TableCtx &c, int im, int which) {
    const int n = c.ph.n_E;
    double *R = c.tab + ((size_t)im * EMX_NTABLE + (which ? EMX_T_RANGE_EP : EMX_T_RANGE_EM)) * n;
    for (int j = 1; j < n; ++j) R[j] = R[j - 1] + R[j];
}

}  // namespace emx
