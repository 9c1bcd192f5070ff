/* emo.h -- ORACLE for the EM-shower step loop (arxiv 2203.09467, "Celeritas").
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  A plain, slow, one-track-at-a-
 * time fp64 CPU transport of a coupled gamma/e-/e+ shower, written from the
 * paper's description of the loop ("six characteristics",
 * PAPER.md:110-111 Table 2 model names, PAPER.md:116 tabulated cross sections,
 * PAPER.md:70 secondary stack, PAPER.md:142 surfaces+CSG cells
 * field propagation) and the readings listed in DESIGN.md section 3 (the paper
 * prints no formulas; every formula is a stated textbook reading).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference leg may load this library.  It shares no source, header,
 * table or constant generator with the CUDA path in paper_2203_09467_b200/.
 *
 * Units: MeV, cm, g/cm3, tesla.  Particle codes 0 = gamma, 1 = e-, 2 = e+.
 *
 * Parity status: every function below is pinned by tests/test_oracle_*.py.
 * Of the aggregate shower shapes the longitudinal profile is pinned (maximum at
 * ln(E/Ec) - 0.5 radiation lengths and the 95 % containment length of the PDG
 * review, tests/test_oracle_transport.py) and, with multiple scattering on, the
 * lateral containment in Moliere radii (tests/test_oracle_msc2.py); sampling fractions and
 * multiplicities remain "parity unpinned" beyond energy conservation: the paper
 * prints no number for them and no independent code exists in this container.
 * emo_sigma_pe is a definitional stand-in (R3): its pin is its own
 * definition.
 */
#ifndef EMO_H
#define EMO_H
#include <stdint.h>
#include <stddef.h>

#define EMO_MAX_ELEM 4
#define EMO_MAX_FACES 8
#define EMO_GAMMA 0
#define EMO_ELECTRON 1
#define EMO_POSITRON 2

/* physical constants, CODATA 2018 (DESIGN.md R-C1) */
#define EMO_ME 0.51099895000          /* MeV */
#define EMO_RE 2.8179403262e-13       /* cm */
#define EMO_ALPHA 7.2973525693e-3
#define EMO_NA 6.02214076e23          /* 1/mol */
#define EMO_CB 2.99792458             /* curvature: kappa[1/cm] = q*CB*B[T]/p[MeV/c]: r = p/(qB), 1e6 eV/c / (c * 1 T) = 0.333564 cm */
#define EMO_PI 3.14159265358979323846

/* process bits (process_mask) and process ids (counters, step results) */
enum { EMO_P_COMPTON = 0, EMO_P_PHOTO = 1, EMO_P_PAIR = 2, EMO_P_MOLLER = 3,
       EMO_P_BHABHA = 4, EMO_P_BREMS = 5, EMO_P_ANNIH = 6, EMO_P_REST = 7, EMO_NPROC = 8 };
/* mask bits: compton 1, photo 2, pair 4, ionisation (Moller+Bhabha) 8, brems 16, annihilation 32 */
#define EMO_M_COMPTON 1u
#define EMO_M_PHOTO 2u
#define EMO_M_PAIR 4u
#define EMO_M_IONI 8u
#define EMO_M_BREMS 16u
#define EMO_M_ANNIH 32u

/* step limiter ("action") */
enum { EMO_A_NONE = 0, EMO_A_DISCRETE = 1, EMO_A_LOSS = 2, EMO_A_BOUNDARY = 3, EMO_A_TRUNC = 4,
       EMO_A_MSC = 5 /* the multiple-scattering step limit (DESIGN.md R-MSC) */ };

/* table kinds per material (each n_E doubles) */
enum { EMO_T_COMPTON = 0, EMO_T_PHOTO, EMO_T_PAIR, EMO_T_MOLLER, EMO_T_BREMS_EM,
       EMO_T_DEDX_EM, EMO_T_RANGE_EM, EMO_T_BHABHA, EMO_T_BREMS_EP, EMO_T_ANNIH,
       EMO_T_DEDX_EP, EMO_T_RANGE_EP, EMO_T_PAIR_ELEM0, /* + element index */
       EMO_T_MSC = EMO_T_PAIR_ELEM0 + EMO_MAX_ELEM,     /* 1/lambda_1, inverse first transport mean free path of e+- */
       EMO_T_VAR_EM, EMO_T_VAR_EP,                      /* d(variance of the restricted collision loss)/ds, MeV2/cm */
       EMO_T_MSC2,                                      /* 1/lambda_2, inverse second transport mean free path (msc = 2) */
       EMO_NTABLE };

/* surface types */
enum { EMO_S_PX = 0, EMO_S_PY = 1, EMO_S_PZ = 2, EMO_S_CZ = 3 };

typedef struct {
    int n_elem;
    int Z[EMO_MAX_ELEM];
    double A[EMO_MAX_ELEM];
    double w[EMO_MAX_ELEM];      /* mass fractions */
    double rho;                  /* g/cm3 */
    double I;                    /* mean excitation energy, MeV */
    double n_i[EMO_MAX_ELEM];    /* atoms/cm3 */
    double n_e;                  /* electrons/cm3 */
    double hwp;                  /* plasma energy, MeV */
    double X0;                   /* radiation length, cm */
    double Tcut;                 /* e-/e+ production threshold (delta rays), MeV */
    double kcut;                 /* photon production threshold (brems), MeV */
    double *tab;                 /* EMO_NTABLE * n_E doubles */
} emo_material;

typedef struct { int type; double v; } emo_surface;  /* v: plane position or cylinder radius */

typedef struct {
    int n_faces;
    int surf[EMO_MAX_FACES];
    int sense[EMO_MAX_FACES];    /* -1: f<0 side, +1: f>0 side */
    int material;                /* -1 vacuum */
    int tally;                   /* -1 none */
} emo_volume;

typedef struct {
    unsigned process_mask;
    double E_min, E_max;         /* grid */
    int n_E;
    double E_trk;                /* tracking cut, MeV */
    double prod_cut_cm;          /* >0: derive Tcut/kcut per material from this length */
    double alpha_R, rho_R;       /* step function */
    double lin_loss;             /* linear-loss limit (fraction of E) */
    double field_eps;            /* cm: RK4 local error and landing tolerance */
    int max_substeps;            /* field substep attempts per step */
    double vacuum_step;          /* cm */
    int max_steps;               /* per track */
    int deposit_e_at_creation;   /* config 0: every e- is deposited at birth */
    int msc;                     /* 1: multiple scattering of e+- (DESIGN.md R-MSC); 2: also the path-length
                                  * correction and the lateral displacement of Lewis' theory (DESIGN.md R-MSC2) */
    double msc_fr;               /* step limit s <= max(msc_fr * max(R, lambda_1), msc_smin) */
    double msc_smin;             /* cm */
    int fluct;                   /* 1: energy-loss fluctuations of e+- (DESIGN.md R-FLUCT) */
    int integrator;              /* field propagation: 0 classical RK4 with step doubling (R-C9), 1 Dormand-Prince 5(4) (R-INT) */
} emo_physics;

typedef struct {
    int n_mat, n_surf, n_vol, n_tally;
    emo_material *mat;
    emo_surface *surf;
    emo_volume *vol;
    emo_physics ph;
    double B[3];                 /* tesla */
    double Bmag, Bhat[3];
    int field_kind;              /* 0 uniform; 1 solenoid with fringe (emo_set_field_fringe) */
    double fringe_z0, fringe_a;  /* cm */
    double lnE0, dlnE, inv_dlnE; /* grid: x_j = lnE0 + j*dlnE */
    int built;
} emo_problem;

typedef struct {
    double x[3], u[3], E;
    uint64_t tid;
    uint32_t prim, step;
    int vol, surf, ptype, alive;
} emo_track;

/* everything one step produces (level-2 parity object) */
typedef struct {
    emo_track trk;               /* updated track (alive=0 if killed) */
    int action, process;         /* limiter; process id or -1 */
    int n_sec;
    emo_track sec[4];            /* allocated secondaries in ordinal order */
    int sec_ord[4];
    double edep;                 /* energy deposited into tally[vol_pre or vol at deposit] */
    int edep_vol;                /* volume the deposit belongs to */
    double below_cut;            /* part of edep that came from tracking-cut kills/births */
    double escaped, looper;
    double s;                    /* step length travelled */
    double msc_tau;              /* path length / lambda_1 used for the deflection of this step (0: none) */
    int n_draws;                 /* uniform draws consumed */
    int null_int;                /* 1 if the discrete interaction was kinematically null */
    int rest;                    /* 1 if an e+ annihilated at rest in this step */
    int n_sub;                   /* substep attempts of the field propagation (0: straight move) */
} emo_step_result;

#define EMO_NHIST 96
typedef struct {
    double escaped, below_cut, looper, E_in;
    uint64_t steps[3], tracks[3], inter[EMO_NPROC], null_int, track_steps;
    uint64_t step_hist[3][EMO_NHIST];   /* tracks by particle type and by emo_step_bin(steps the track took) */
} emo_scalars;

/* ---- philox.c ---- */
void emo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
double emo_u01(uint32_t wa, uint32_t wb);
double emo_draw(uint64_t seed, uint32_t prim, uint64_t tid, uint32_t step, uint32_t n);
uint64_t emo_child_tid(uint64_t seed, uint32_t prim, uint64_t tid, uint32_t step, uint32_t ordinal);

/* ---- xs.c : closed-form cross sections / stopping powers ---- */
double emo_fc(int Z);
double emo_X0_elem_gcm2(int Z, double A);
double emo_sigma_kn(double E);                          /* cm2 per electron */
double emo_sigma_pe(int Z, double E);                   /* cm2 per atom */
double emo_pair_dcs(int Z, double E, double eps);       /* cm2 per atom per unit eps, clipped at 0 */
double emo_sigma_pair(int Z, double E);                 /* 2*GL32 over [eps0,1/2] */
double emo_sigma_moller(double T, double Tcut);         /* cm2 per electron */
double emo_sigma_bhabha(double T, double Tcut);
double emo_sigma_annih(double T);
double emo_moller_dcs(double T, double eps);            /* dsigma/deps, cm2 */
double emo_bhabha_dcs(double T, double eps);
double emo_brems_Sigma(double T, double kc, double X0); /* 1/cm */
double emo_brems_dedx(double T, double kc, double X0);  /* MeV/cm */
double emo_dedx_col(const emo_material *m, int ptype, double T, double Tcut); /* MeV/cm; Tcut<=0: unrestricted */
void   emo_gauss_legendre(int n, double *x, double *w); /* nodes/weights on [-1,1] */
/* second moment of the energy transfers below the production threshold, Int_0^Tup W^2 dsigma, MeV2 cm2 per
 * electron (DESIGN.md R-FLUCT); ptype EMO_ELECTRON: Moller, Tup = min(Tcut, T/2); EMO_POSITRON: Bhabha, min(Tcut, T) */
double emo_loss_second_moment(int ptype, double T, double Tcut);
/* fluctuated loss: mean dE, variance V, the two uniforms; energy E bounds it (DESIGN.md R-FLUCT) */
double emo_fluctuate_loss(double dE, double V, double E, double xi1, double xi2);
/* multiple scattering (DESIGN.md R-MSC) */
double emo_msc_screening(int Z, double T);              /* Moliere screening parameter A */
double emo_msc_sigma1(int Z, double Amass, double T);   /* first transport cross section, cm2 per atom */
double emo_msc_one_minus_mu(double tau, double xi);     /* 1 - cos(theta) of a step of s = tau * lambda_1 */
/* DESIGN.md R-MSC2: second transport cross section; Lewis' mean geometric length <z> and mean square lateral
 * displacement <x^2 + y^2> of a true path t (il1 = 1/lambda_1, il2 = 1/lambda_2, both 1/cm) */
double emo_msc_sigma2(int Z, double Amass, double T);   /* Int (1 - P_2(cos theta)) dsigma, cm2 per atom */
double emo_msc_phi3(double x);                          /* (x^2/2 - x + 1 - exp(-x)) / x^3 */
double emo_msc_geom_length(double t, double il1);       /* cm */
double emo_msc_lateral_r2(double t, double il1, double il2); /* cm2 */

/* ---- problem.c ---- */
emo_problem *emo_create(void);
void emo_destroy(emo_problem *p);
int emo_add_material(emo_problem *p, int n_elem, const int *Z, const double *A, const double *w,
                     double rho, double I_eV);
int emo_add_surface(emo_problem *p, int type, double v);
int emo_add_volume(emo_problem *p, int n_faces, const int *surf, const int *sense, int material, int tally);
int emo_set_field(emo_problem *p, double Bx, double By, double Bz);
/* Non-uniform field ("propagation of particles through arbitrary magnetic fields"): a solenoid
 * along z whose field falls off towards its ends, B(x) = |B| g(x) with
 *   f(z) = 1 / (1 + exp((|z| - z0) / a)),   g = (-x f'(z) / 2, -y f'(z) / 2, f(z)),   f' = -sign(z) f (1 - f) / a
 * (the radial part makes div B = 0 to first order in r).  Needs a field set along +-z; returns -1 otherwise. */
int emo_set_field_fringe(emo_problem *p, double z0_cm, double a_cm);
/* g(x) of the field set on p (Bhat for the uniform field) */
void emo_field_profile(const emo_problem *p, const double x[3], double g[3]);
/* Dormand-Prince 5(4) step (DESIGN.md R-INT): x1, u1 = fifth-order solution (u1 normalised), err = |x_5 - x_4| */
void emo_dp45(const emo_problem *p, const double x[3], const double u[3], double kappa, double h,
              double x1[3], double u1[3], double *err);
/* step doubling as emo_rk4_doubling, the field evaluated at the stage positions */
void emo_rk4_doubling_map(const emo_problem *p, const double x[3], const double u[3], double kappa, double h,
                          double x1[3], double u1[3], double *err);
int emo_set_physics(emo_problem *p, const emo_physics *ph);
int emo_set_cuts(emo_problem *p, int material, double Tcut, double kcut); /* explicit energies */
int emo_build_tables(emo_problem *p);
int emo_get_table(const emo_problem *p, int material, int kind, double *out, int n);
int emo_get_material_info(const emo_problem *p, int material, double *out8); /* n_e,I,hwp,X0,Tcut,kcut,rho,n_elem */
double emo_lookup(const emo_problem *p, int material, int kind, double E);
double emo_range_inverse(const emo_problem *p, int material, int kind_range, double r);

/* ---- geom.c ---- */
double emo_distance(const emo_problem *p, int vol, const double x[3], const double u[3], int surf, int *hit);
int emo_neighbour(const emo_problem *p, const double x[3], const double u[3], int S);
int emo_locate(const emo_problem *p, const double x[3]);

/* ---- field.c ---- */
void emo_rk4_doubling(const double x[3], const double u[3], double kappa, const double Bhat[3], double h,
                      double x1[3], double u1[3], double *err);
double emo_propagate_field(const emo_problem *p, int vol, int *surf_io, double x[3], double u[3],
                           double kappa, double s_max, int *hit);
double emo_propagate_field_n(const emo_problem *p, int vol, int *surf_io, double x[3], double u[3],
                             double kappa, double s_max, int *hit, int *n_sub);

/* ---- interact.c : samplers; draws come from a callback-free draw cursor ---- */
typedef struct { uint64_t seed; uint32_t prim; uint64_t tid; uint32_t step; uint32_t n; } emo_rng;
double emo_next(emo_rng *r);
void emo_rotate(const double u[3], double mu, double phi, double out[3]);
void emo_compton(emo_rng *r, double E, const double u[3], double *E1, double u1[3], double *Te, double ue[3]);
void emo_photo_dir(emo_rng *r, double E, const double u[3], double ue[3]);
int  emo_pair(emo_rng *r, int Z, double E, const double u[3], double *Tm, double um[3], double *Tp, double up[3]);
int  emo_brems(emo_rng *r, double T, double kc, const double u[3], double *k, double ug[3], double *T1, double u1[3]);
int  emo_moller(emo_rng *r, double T, double Tcut, const double u[3], double *Td, double ud[3], double *T1, double u1[3]);
int  emo_bhabha(emo_rng *r, double T, double Tcut, const double u[3], double *Td, double ud[3], double *T1, double u1[3]);
void emo_annih_flight(emo_rng *r, double T, const double u[3], double *k1, double u1[3], double *k2, double u2[3]);
void emo_annih_rest(emo_rng *r, double u1[3], double u2[3]);
void emo_msc_deflect(emo_rng *r, double tau, const double u[3], double out[3]);

/* ---- transport.c ---- */
void emo_step(const emo_problem *p, uint64_t seed, const emo_track *in, emo_step_result *out);
int emo_step_batch(const emo_problem *p, uint64_t seed, long n, const emo_track *in, emo_step_result *out);
/* transport n primaries; per_prim (optional) receives, for each primary,
 * [edep_total, escaped, looper, below_cut, E_in, steps_g, steps_em, steps_ep, trk_g, trk_em, trk_ep]
 * (11 doubles); per_prim_tally (optional) receives n_prim*n_tally doubles. */
#define EMO_PER_PRIM 11
/* Steps-per-track histogram ("steps per track ... by particle type", one of the paper's two
 * verification observables).  Bin of a track that took n >= 1 steps: n itself below 16, then four bins per
 * octave: 16 + 4 (e - 4) + (the two bits of n below its leading bit), e = floor(log2 n); the last bin
 * collects everything beyond. */
int emo_step_bin(uint64_t n);
int emo_transport(const emo_problem *p, long n_prim, const int *ptype, const double *E,
                  const double *pos3, const double *dir3, const int *start_vol, const int *start_surf,
                  uint64_t seed, int n_threads, double *edep, emo_scalars *sc,
                  double *per_prim, double *per_prim_tally);
#endif
