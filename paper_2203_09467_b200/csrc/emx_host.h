// emx_host.h -- host-side problem description behind the C-ABI (include/emx.h): materials, surfaces,
// cells, field and physics switches (the inputs PAPER.md:235-237 lists), plus the derived quantities that
// are computed once on the host: material constants (C3), grid constants (C4) and the
// per-surface neighbour candidate lists used by emx_geom.h.
#pragma once
#include <string>
#include <vector>
#include "emx_core.h"
#include "emx_xs.h"

namespace emx {

struct HostProblem {
    std::vector<Material> mat;
    std::vector<int> surf_type;
    std::vector<double> surf_v;
    std::vector<Volume> vol;
    emx_physics ph;
    double B[3] = {0.0, 0.0, 0.0};
    int field_kind = 0;  // 0 uniform, 1 solenoid with fringe
    double fringe_z0 = 0.0, fringe_a = 0.0;
    int n_tally = 0;
    bool built = false;
    std::string err;

    HostProblem() {
        ph.process_mask = 63u;
        ph.E_min = 1e-3;
        ph.E_max = 1e4;
        ph.n_E = 256;
        ph.E_trk = 1e-3;
        ph.prod_cut_cm = 0.07;
        ph.alpha_R = 0.2;   // R9
        ph.rho_R = 0.1;     // R9
        ph.lin_loss = 0.01; // R9
        ph.field_eps = 1e-7;   // R14: 1e-6 mm
        ph.max_substeps = 1000;
        ph.vacuum_step = 1e3;
        ph.max_steps = 10000;
        ph.deposit_e_at_creation = 0;
        ph.msc = 0;
        ph.msc_fr = 0.2;
        ph.msc_smin = 1e-3;
        ph.integrator = 0;
        ph.fluct = 0;
    }
};

// material constants of C3: number densities, electron density, plasma energy, radiation length
inline bool derive_material(Material &m, int n_elem, const int *Z, const double *A, const double *w, double rho,
                            double I_eV) {
    if (n_elem < 1 || n_elem > EMX_MAX_ELEM || !(rho > 0.0) || !(I_eV > 0.0)) return false;
    m = Material();
    m.n_elem = n_elem;
    m.rho = rho;
    m.I = I_eV * 1e-6;
    m.n_e = 0.0;
    double invX0 = 0.0;
    for (int i = 0; i < EMX_MAX_ELEM; ++i) {
        m.Z[i] = 0;
        m.A[i] = m.w[i] = m.n_i[i] = 0.0;
    }
    for (int i = 0; i < n_elem; ++i) {
        if (Z[i] < 1 || !(A[i] > 0.0) || !(w[i] >= 0.0)) return false;
        m.Z[i] = Z[i];
        m.A[i] = A[i];
        m.w[i] = w[i];
        m.n_i[i] = rho * kNa * w[i] / A[i];
        m.n_e += m.n_i[i] * Z[i];
        invX0 += rho * w[i] / X0_element(Z[i], A[i]);
    }
    m.X0 = 1.0 / invX0;
    m.hwp = (kMe / kAlpha) * sqrt(4.0 * kPi * m.n_e * kRe * kRe * kRe);
    m.Tcut = -1.0;
    m.kcut = -1.0;
    return true;
}

// Can cell c hold points just across S on its `sense` side?  Not if one of its own faces is a surface of the same
// family (same axis plane, or z-cylinder) that keeps the cell on the other side of S by more than `margin`: with
// sense = +1 the point has f_S >= -eps, and a face (v_f <= v_S - margin, sense -1) wants f_f < 0 where
// f_f >= margin - eps > 0 (mirror image for sense = -1).  The point crossing S lies within the landing tolerance
// eps = field_eps of S (C9), margin = max(1e-6, 10 eps) cm, so cell_matches() would reject exactly
// these cells at that face: leaving them out of the candidate lists cannot change what neighbour() returns.
inline bool never_across(const HostProblem &hp, int c, int S, int sense, double margin) {
    const Volume &v = hp.vol[c];
    const int tS = hp.surf_type[S];
    const double vS = hp.surf_v[S];
    for (int i = 0; i < v.n_faces; ++i) {
        const int Sf = v.surf[i];
        if (Sf == S || hp.surf_type[Sf] != tS) continue;
        const double vf = hp.surf_v[Sf];
        if (sense > 0 && v.sense[i] < 0 && vf <= vS - margin) return true;
        if (sense < 0 && v.sense[i] > 0 && vf >= vS + margin) return true;
    }
    return false;
}

// nb_off[2 S + (sense > 0)] .. nb_off[2 S + (sense > 0) + 1]: cells listing (S, sense), ascending id, without the
// cells that can never lie across S on that side
inline void build_neighbour_lists(const HostProblem &hp, std::vector<int> &off, std::vector<int> &list) {
    const int ns = (int)hp.surf_type.size();
    const double margin = fmax(1e-6, 10.0 * hp.ph.field_eps);
    off.assign(2 * ns + 1, 0);
    list.clear();
    for (int k = 0; k < 2 * ns; ++k) {
        const int S = k / 2, sense = (k & 1) ? 1 : -1;
        off[k] = (int)list.size();
        for (int c = 0; c < (int)hp.vol.size(); ++c) {
            const Volume &v = hp.vol[c];
            for (int i = 0; i < v.n_faces; ++i)
                if (v.surf[i] == S && v.sense[i] == sense) {
                    if (!never_across(hp, c, S, sense, margin)) list.push_back(c);
                    break;
                }
        }
    }
    off[2 * ns] = (int)list.size();
}

// off2[2 S + (sense > 0)] .. off2[2 S + (sense > 0) + 1]: cells that do not list S with either sense, ascending id,
// again without the cells that can never lie across S on that side (a track leaving the world through an outer
// surface finds both lists empty instead of testing every cell of the problem)
inline void build_nonlisting_lists(const HostProblem &hp, std::vector<int> &off2, std::vector<int> &list2) {
    const int ns = (int)hp.surf_type.size();
    const double margin = fmax(1e-6, 10.0 * hp.ph.field_eps);
    off2.assign(2 * ns + 1, 0);
    list2.clear();
    for (int k = 0; k < 2 * ns; ++k) {
        const int S = k / 2, sense = (k & 1) ? 1 : -1;
        off2[k] = (int)list2.size();
        for (int c = 0; c < (int)hp.vol.size(); ++c) {
            const Volume &v = hp.vol[c];
            bool lists = false;
            for (int i = 0; i < v.n_faces; ++i) lists = lists || (v.surf[i] == S);
            if (!lists && !never_across(hp, c, S, sense, margin)) list2.push_back(c);
        }
    }
    off2[2 * ns] = (int)list2.size();
}

struct GridConsts {
    double lnE0, dlnE, inv_dlnE;
};
inline GridConsts grid_consts(const emx_physics &ph) {
    GridConsts g;
    g.lnE0 = log(ph.E_min);
    g.dlnE = log(ph.E_max / ph.E_min) / (ph.n_E - 1);
    g.inv_dlnE = (ph.n_E - 1) / log(ph.E_max / ph.E_min);
    return g;
}

}  // namespace emx
