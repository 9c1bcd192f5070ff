// emx_api.cu -- the C-ABI of include/emx.h: problem object, table build, transport driver, tallies, hooks.
// Host logic only; every computation of the path runs in the kernels of emx_kernels.cu / emx_transport.cu.
#include <cuda_runtime.h>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>
#include "emx_host.h"
#include "emx_kernels.h"
#include "emx_tables.h"

using namespace emx;

struct emx_problem {
    HostProblem hp;
    // the one device block the library owns: materials, geometry, tables, tallies
    void *dev = nullptr;
    size_t dev_bytes = 0;
    Material *d_mat = nullptr;
    int *d_surf_type = nullptr;
    double *d_surf_v = nullptr;
    Volume *d_vol = nullptr;
    Face *d_faces = nullptr;
    double *d_tab = nullptr;
    double *d_scratch = nullptr;
    int *d_nb_off = nullptr, *d_nb_list = nullptr, *d_nb2_off = nullptr, *d_nb2_list = nullptr;
    double *d_tally = nullptr;
    Params P;
    // results of the last transport
    Ctl last_ctl;
    bool have_ctl = false;
    double last_ms = -1.0;
    std::vector<uint32_t> iter_log;
    std::string err;
    // pinned staging for the control block
    Ctl *h_ctl = nullptr;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    // optional per-kernel timing of the loop (emx_set_profile)
    bool profile = false;
    std::vector<cudaEvent_t> prof_ev;
    double prof_ms[kNStages + 2] = {0};  // the step kernels by stage (emx_kernels.h), refill, all step kernels
    int n_sm = 148;
    long launches = 0, iterations_launched = 0;
    std::vector<float> iter_ms;  // per iteration: refill ms, step ms (profiling on)
    // iteration graph: internal streams (the caller's stream may be the legacy stream, which cannot be captured)
    cudaStream_t s0 = nullptr, s1 = nullptr, s2 = nullptr;
    cudaEvent_t evFork = nullptr, evJ1 = nullptr, evJ2 = nullptr, evIn = nullptr, evOut = nullptr;
    long long prim_first = 0;  // primary index of the first element passed to emx_transport
    // the instantiated iteration graph is kept for the next emx_transport with the same kernel arguments
    // (workspace, primaries, seed, tables): capture + instantiation cost about 2 ms
    cudaGraphExec_t graph_exec = nullptr;
    Work graph_w;
    Primaries graph_pr;
    uint64_t graph_seed = 0;
    unsigned long long graph_gen = 0, params_gen = 1;
    bool graph_is_loop = false;
    bool use_graph = true;
    emx_schedule sched;        // emx_set_schedule: when work is done, never what it computes
    // production thresholds given with emx_set_cuts (< 0: derive from the cut length at every build)
    std::vector<double> user_Tcut, user_kcut;
};

namespace {

thread_local std::string g_err;

int fail(emx_problem *p, int code, const char *msg) {
    if (p) p->err = msg;
    g_err = msg;
    return code;
}
int fail_cuda(emx_problem *p, cudaError_t e, const char *where) {
    char buf[256];
    snprintf(buf, sizeof buf, "%s: %s", where, cudaGetErrorString(e));
    if (p) p->err = buf;
    g_err = buf;
    return EMX_E_CUDA;
}
#define CU(call)                                                  \
    do {                                                          \
        cudaError_t e_ = (call);                                  \
        if (e_ != cudaSuccess) return fail_cuda(p, e_, #call);    \
    } while (0)

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

void free_device(emx_problem *p) {
    if (p->dev) cudaFree(p->dev);
    p->dev = nullptr;
    p->d_tally = nullptr;
    p->hp.built = false;
}

struct Carve {
    char *base;
    size_t off = 0;
    template <typename T>
    T *take(size_t n) {
        off = align_up(off, 256);
        T *r = base ? (T *)(base + off) : nullptr;
        off += n * sizeof(T);
        return r;
    }
};

// carve the caller's workspace; with base == nullptr only the size is computed
size_t carve_work(char *base, long n_slots, long qcap, Work &w, int max_log) {
    Carve c{base};
    int nch = (int)((n_slots + kChunk - 1) / kChunk);
    if (nch < 2) nch = 2;  // one chunk per pool at least
    w.n_chunks = nch;
    w.slot_cap = nch * kChunk;
    w.pool_reserve = nch / 32 > 1 ? nch / 32 : 1;
    w.qtotal = (int)qcap;
    w.ctl = c.take<Ctl>(1);
    w.log = c.take<uint32_t>(2 * (size_t)max_log);
    w.max_log = max_log;
    const size_t n = (size_t)nch * kChunk;
    Store &t = w.st;
    t.xy = c.take<double2>(n); t.zu = c.take<double2>(n); t.uu = c.take<double2>(n);
    t.Et = c.take<double2>(n);
    t.id = c.take<int4>(n);
    t.alive = c.take<uint8_t>(n); t.stage = c.take<uint8_t>(n); t.ptype = c.take<uint8_t>(n); t.act = c.take<uint8_t>(n);
    t.s_phys = c.take<double>(n); t.s_done = c.take<double>(n); t.h_try = c.take<double>(n);
    t.att = c.take<int>(n);
    t.kap = c.take<double>(n);
    w.free_list = c.take<int>((size_t)nch);
    w.rtab = c.take<int>((size_t)nch);
    for (int p = 0; p < kPools; ++p) {
        w.ctab[p] = c.take<int>((size_t)nch);
        w.chunk_dead[p] = c.take<int>((size_t)nch + 1);
        w.chunk_off[p] = c.take<int>((size_t)nch + 1);
        w.hole_idx[p] = c.take<int>(n);
        for (int k = 0; k < kMaxLists; ++k) w.ilist[p][k] = (p == kPoolGamma && k == 3) ? nullptr : c.take<int>(n);
    }
    // everything above (track store, scan arrays, interaction lists: about 150 MB of addresses at 2^20 slots, of
    // which an iteration touches what the live tracks need) is kept together; the stacks follow
    {
        const size_t q = (size_t)w.qtotal;
        Stack &s = w.q;
        s.xy = c.take<double2>(q); s.zu = c.take<double2>(q); s.uu = c.take<double2>(q);
        s.Et = c.take<double2>(q);
        s.id = c.take<int4>(q);
    }
    return align_up(c.off, 256);
}

// staging area of emx_transport_host behind the workspace proper: the six primary arrays (4 + 8 + 24 + 24 + 4 + 4
// bytes per primary)
size_t staging_bytes(long n) {
    const size_t nn = (size_t)(n > 0 ? n : 1);
    return align_up(nn * 4, 256) * 3 + align_up(nn * 8, 256) + 2 * align_up(nn * 24, 256);
}

constexpr int kMaxLog = 1 << 16;

}  // namespace

extern "C" {

const char *emx_version(void) { return "emx 0.1 (sm_100a)"; }

const char *emx_last_error(const emx_problem *p) { return p ? p->err.c_str() : g_err.c_str(); }

int emx_create(emx_problem **out) {
    if (!out) return fail(nullptr, EMX_E_ARG, "emx_create: null output");
    emx_problem *p = new (std::nothrow) emx_problem();
    if (!p) return fail(nullptr, EMX_E_NOMEM, "emx_create: out of memory");
    p->sched.loop_node = 1;
    p->sched.slice_min = 2;
    p->sched.slice_max = 16;
    p->sched.slice_above = -1;
    p->sched.admit_below = 0;
    p->sched.mev_per_slot = 0;
    p->sched.reserved = 0;
    for (int k = 0; k < 8; ++k) p->sched.blocks_per_sm[k] = 0;
    *out = p;
    return EMX_OK;
}

void emx_destroy(emx_problem *p) {
    if (!p) return;
    free_device(p);
    if (p->graph_exec) cudaGraphExecDestroy(p->graph_exec);
    if (p->h_ctl) cudaFreeHost(p->h_ctl);
    if (p->ev0) cudaEventDestroy(p->ev0);
    if (p->ev1) cudaEventDestroy(p->ev1);
    for (cudaEvent_t e : p->prof_ev) cudaEventDestroy(e);
    for (cudaEvent_t e : {p->evFork, p->evJ1, p->evJ2, p->evIn, p->evOut})
        if (e) cudaEventDestroy(e);
    for (cudaStream_t s : {p->s0, p->s1, p->s2})
        if (s) cudaStreamDestroy(s);
    delete p;
}

int emx_add_material(emx_problem *p, int n_elem, const int *Z, const double *A, const double *mass_frac,
                     double density_g_cm3, double mean_exc_energy_eV) {
    if (!p || !Z || !A || !mass_frac) return fail(p, EMX_E_ARG, "emx_add_material: null argument");
    Material m;
    if (!derive_material(m, n_elem, Z, A, mass_frac, density_g_cm3, mean_exc_energy_eV))
        return fail(p, EMX_E_ARG, "emx_add_material: invalid element list, density or mean excitation energy");
    p->hp.mat.push_back(m);
    p->user_Tcut.push_back(-1.0);
    p->user_kcut.push_back(-1.0);
    p->hp.built = false;
    return (int)p->hp.mat.size() - 1;
}

int emx_add_surface(emx_problem *p, int type, double value_cm) {
    if (!p || type < EMX_S_PX || type > EMX_S_CZ) return fail(p, EMX_E_ARG, "emx_add_surface: invalid type");
    if (type == EMX_S_CZ && !(value_cm > 0.0)) return fail(p, EMX_E_ARG, "emx_add_surface: radius must be > 0");
    p->hp.surf_type.push_back(type);
    p->hp.surf_v.push_back(value_cm);
    p->hp.built = false;
    return (int)p->hp.surf_v.size() - 1;
}

int emx_add_volume(emx_problem *p, int n_faces, const int *surf, const int *sense, int material, int tally) {
    if (!p || n_faces < 0 || n_faces > EMX_MAX_FACES || (n_faces > 0 && (!surf || !sense)))
        return fail(p, EMX_E_ARG, "emx_add_volume: invalid face list");
    if (material < -1 || material >= (int)p->hp.mat.size() || tally < -1)
        return fail(p, EMX_E_ARG, "emx_add_volume: unknown material or invalid tally id");
    Volume v;
    memset(&v, 0, sizeof v);
    v.n_faces = n_faces;
    for (int i = 0; i < n_faces; ++i) {
        if (surf[i] < 0 || surf[i] >= (int)p->hp.surf_v.size() || (sense[i] != 1 && sense[i] != -1))
            return fail(p, EMX_E_ARG, "emx_add_volume: unknown surface or sense not +-1");
        v.surf[i] = surf[i];
        v.sense[i] = sense[i];
    }
    v.material = material;
    v.tally = tally;
    p->hp.vol.push_back(v);
    if (tally + 1 > p->hp.n_tally) p->hp.n_tally = tally + 1;
    p->hp.built = false;
    return (int)p->hp.vol.size() - 1;
}

int emx_set_field(emx_problem *p, double Bx, double By, double Bz) {
    if (!p) return fail(p, EMX_E_ARG, "emx_set_field: null problem");
    p->hp.B[0] = Bx;
    p->hp.B[1] = By;
    p->hp.B[2] = Bz;
    p->hp.field_kind = 0;
    p->hp.built = false;
    return EMX_OK;
}

int emx_set_field_fringe(emx_problem *p, double z0_cm, double a_cm) {
    if (!p) return fail(p, EMX_E_ARG, "emx_set_field_fringe: null problem");
    if (p->hp.B[0] != 0.0 || p->hp.B[1] != 0.0 || p->hp.B[2] == 0.0)
        return fail(p, EMX_E_ARG, "emx_set_field_fringe: set a field along z first (emx_set_field)");
    if (!(z0_cm > 0.0) || !(a_cm > 0.0)) return fail(p, EMX_E_ARG, "emx_set_field_fringe: z0 and a must be > 0");
    p->hp.field_kind = 1;
    p->hp.fringe_z0 = z0_cm;
    p->hp.fringe_a = a_cm;
    p->hp.built = false;
    return EMX_OK;
}

int emx_get_physics(const emx_problem *p, emx_physics *out) {
    if (!p || !out) return EMX_E_ARG;
    *out = p->hp.ph;
    return EMX_OK;
}

int emx_set_physics(emx_problem *p, const emx_physics *ph) {
    if (!p || !ph) return fail(p, EMX_E_ARG, "emx_set_physics: null argument");
    if (ph->n_E < 2 || !(ph->E_max > ph->E_min) || !(ph->E_min > 0.0) || ph->max_steps < 1 || ph->max_substeps < 1 ||
        !(ph->field_eps > 0.0) || !(ph->vacuum_step > 0.0))
        return fail(p, EMX_E_ARG, "emx_set_physics: invalid grid or limits");
    if (ph->msc < 0 || ph->msc > 2) return fail(p, EMX_E_ARG, "emx_set_physics: msc is 0, 1 or 2");
    if (ph->integrator < 0 || ph->integrator > 1) return fail(p, EMX_E_ARG, "emx_set_physics: integrator is 0 or 1");
    if (ph->msc && (!(ph->msc_fr > 0.0) || !(ph->msc_smin > 0.0)))
        return fail(p, EMX_E_ARG, "emx_set_physics: multiple scattering needs msc_fr > 0 and msc_smin > 0");
    p->hp.ph = *ph;
    p->hp.built = false;
    return EMX_OK;
}

int emx_set_cuts(emx_problem *p, int material, double Tcut, double kcut) {
    if (!p || material < 0 || material >= (int)p->hp.mat.size()) return fail(p, EMX_E_ARG, "emx_set_cuts: unknown material");
    p->user_Tcut[material] = Tcut;  // < 0: back to the cut-length conversion
    p->user_kcut[material] = kcut;
    p->hp.built = false;
    return EMX_OK;
}

int emx_n_tally(const emx_problem *p) { return p ? p->hp.n_tally : EMX_E_ARG; }

int emx_build_tables(emx_problem *p, void *stream) {
    if (!p) return fail(p, EMX_E_ARG, "emx_build_tables: null problem");
    HostProblem &hp = p->hp;
    if (hp.vol.empty()) return fail(p, EMX_E_STATE, "emx_build_tables: no volume defined");
    // every build starts from what the caller set: the thresholds a previous build derived from another cut length
    // or another grid must not survive it
    for (size_t im = 0; im < hp.mat.size(); ++im) {
        hp.mat[im].Tcut = p->user_Tcut[im];
        hp.mat[im].kcut = p->user_kcut[im];
        if (!(hp.ph.prod_cut_cm > 0.0) && (hp.mat[im].Tcut < 0.0 || hp.mat[im].kcut < 0.0))
            return fail(p, EMX_E_STATE, "emx_build_tables: no production cut length and no explicit cut energies");
    }
    cudaStream_t st = (cudaStream_t)stream;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1)
        return fail(p, EMX_E_CUDA, "emx_build_tables: no CUDA device (this library has no CPU path)");
    free_device(p);

    std::vector<int> nb_off, nb_list;
    build_neighbour_lists(hp, nb_off, nb_list);
    std::vector<int> nb2_off, nb2_list;
    build_nonlisting_lists(hp, nb2_off, nb2_list);
    const size_t n = (size_t)hp.ph.n_E, nm = hp.mat.size(), ns = hp.surf_v.size(), nv = hp.vol.size();
    Carve c{nullptr};
    auto layout = [&](Carve &cv) {
        p->d_mat = cv.take<Material>(nm ? nm : 1);
        p->d_surf_type = cv.take<int>(ns ? ns : 1);
        p->d_surf_v = cv.take<double>(ns ? ns : 1);
        p->d_vol = cv.take<Volume>(nv);
        p->d_faces = cv.take<Face>(nv * EMX_MAX_FACES);
        p->d_tab = cv.take<double>((nm ? nm : 1) * EMX_NTABLE * n);
        p->d_scratch = cv.take<double>((nm ? nm : 1) * n);
        p->d_nb_off = cv.take<int>(nb_off.size());
        p->d_nb_list = cv.take<int>(nb_list.size() ? nb_list.size() : 1);
        p->d_nb2_off = cv.take<int>(nb2_off.size());
        p->d_nb2_list = cv.take<int>(nb2_list.size() ? nb2_list.size() : 1);
        p->d_tally = cv.take<double>(hp.n_tally ? hp.n_tally : 1);
    };
    layout(c);
    p->dev_bytes = align_up(c.off, 256);
    CU(cudaMalloc(&p->dev, p->dev_bytes));
    Carve c2{(char *)p->dev};
    layout(c2);
    CU(cudaMemsetAsync(p->dev, 0, p->dev_bytes, st));
    if (nm) CU(cudaMemcpyAsync(p->d_mat, hp.mat.data(), nm * sizeof(Material), cudaMemcpyHostToDevice, st));
    if (ns) {
        CU(cudaMemcpyAsync(p->d_surf_type, hp.surf_type.data(), ns * sizeof(int), cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(p->d_surf_v, hp.surf_v.data(), ns * sizeof(double), cudaMemcpyHostToDevice, st));
    }
    CU(cudaMemcpyAsync(p->d_vol, hp.vol.data(), nv * sizeof(Volume), cudaMemcpyHostToDevice, st));
    std::vector<Face> faces(nv * EMX_MAX_FACES);  // the cells' face lists resolved against the surface table
    memset(faces.data(), 0, faces.size() * sizeof(Face));
    for (size_t iv = 0; iv < nv; ++iv) {
        const Volume &v = hp.vol[iv];
        // planes first, cylinders after (each group in the cell's own order): the distance routine runs one uniform loop
        // per kind; the result does not depend on the order (ties go to the lowest surface id)
        int k = 0, n_plane = 0;
        for (int pass = 0; pass < 2; ++pass)
            for (int i = 0; i < v.n_faces; ++i) {
                const bool cyl = hp.surf_type[v.surf[i]] == EMX_S_CZ;
                if (cyl != (pass == 1)) continue;
                Face &f = faces[iv * EMX_MAX_FACES + k++];
                f.S = v.surf[i];
                f.v = hp.surf_v[v.surf[i]];
                f.type = (int8_t)hp.surf_type[v.surf[i]];
                f.sense = (int8_t)v.sense[i];
                if (!cyl) n_plane += 1;
            }
        faces[iv * EMX_MAX_FACES].n = (int16_t)(v.n_faces | (n_plane << 8));  // low byte: faces, high byte: planes among them
    }
    CU(cudaMemcpyAsync(p->d_faces, faces.data(), faces.size() * sizeof(Face), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(p->d_nb_off, nb_off.data(), nb_off.size() * sizeof(int), cudaMemcpyHostToDevice, st));
    if (!nb_list.empty())
        CU(cudaMemcpyAsync(p->d_nb_list, nb_list.data(), nb_list.size() * sizeof(int), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(p->d_nb2_off, nb2_off.data(), nb2_off.size() * sizeof(int), cudaMemcpyHostToDevice, st));
    if (!nb2_list.empty())
        CU(cudaMemcpyAsync(p->d_nb2_list, nb2_list.data(), nb2_list.size() * sizeof(int), cudaMemcpyHostToDevice, st));

    const GridConsts g = grid_consts(hp.ph);
    if (nm) {
        TableCtx tc;
        tc.ph = hp.ph;
        tc.lnE0 = g.lnE0;
        tc.dlnE = g.dlnE;
        tc.n_mat = (int)nm;
        tc.mat = p->d_mat;
        tc.tab = p->d_tab;
        tc.scratch = p->d_scratch;
        CU(launch_build_tables(tc, st));
        // the builder derived the production thresholds on the device: mirror them on the host
        CU(cudaMemcpyAsync(hp.mat.data(), p->d_mat, nm * sizeof(Material), cudaMemcpyDeviceToHost, st));
    }
    CU(cudaStreamSynchronize(st));

    Params &P = p->P;
    P.ph = hp.ph;
    P.n_mat = (int)nm;
    P.n_surf = (int)ns;
    P.n_vol = (int)nv;
    P.n_tally = hp.n_tally;
    P.mat = p->d_mat;
    P.surf_type = p->d_surf_type;
    P.surf_v = p->d_surf_v;
    P.vol = p->d_vol;
    P.faces = p->d_faces;
    P.tab = p->d_tab;
    P.nb_off = p->d_nb_off;
    P.nb_list = p->d_nb_list;
    P.nb2_off = p->d_nb2_off;
    P.nb2_list = p->d_nb2_list;
    const double bm = sqrt(hp.B[0] * hp.B[0] + hp.B[1] * hp.B[1] + hp.B[2] * hp.B[2]);
    P.Bmag = bm;
    P.field_eps_floor = hp.ph.field_eps / 3125.0;
    for (int i = 0; i < 3; ++i) P.Bhat[i] = bm > 0.0 ? hp.B[i] / bm : 0.0;
    P.field_kind = hp.field_kind;
    P.fringe_z0 = hp.fringe_z0;
    P.fringe_a = hp.fringe_a;
    P.lnE0 = g.lnE0;
    P.dlnE = g.dlnE;
    P.inv_dlnE = g.inv_dlnE;
    {
        int dev = 0, sms = 0;
        CU(cudaGetDevice(&dev));
        CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        p->n_sm = sms > 0 ? sms : 148;
    }
    if (!p->h_ctl) CU(cudaMallocHost(&p->h_ctl, sizeof(Ctl)));
    if (!p->ev0) CU(cudaEventCreate(&p->ev0));
    if (!p->ev1) CU(cudaEventCreate(&p->ev1));
    if (!p->s0) {
        CU(cudaStreamCreateWithFlags(&p->s0, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&p->s1, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&p->s2, cudaStreamNonBlocking));
        for (cudaEvent_t *e : {&p->evFork, &p->evJ1, &p->evJ2, &p->evIn, &p->evOut})
            CU(cudaEventCreateWithFlags(e, cudaEventDisableTiming));
    }
    hp.built = true;
    p->params_gen += 1;  // kernel nodes hold Params by value: a kept graph is stale now
    p->have_ctl = false;
    return EMX_OK;
}

int emx_get_table(const emx_problem *cp, int material, int kind, double *host_out, int n) {
    emx_problem *p = const_cast<emx_problem *>(cp);
    if (!p || !p->hp.built) return fail(p, EMX_E_STATE, "emx_get_table: tables not built");
    if (material < 0 || material >= (int)p->hp.mat.size() || kind < 0 || kind >= EMX_NTABLE || n != p->hp.ph.n_E || !host_out)
        return fail(p, EMX_E_ARG, "emx_get_table: invalid material, kind or length");
    CU(cudaMemcpy(host_out, p->d_tab + ((size_t)material * EMX_NTABLE + kind) * n, (size_t)n * sizeof(double),
                  cudaMemcpyDeviceToHost));
    return EMX_OK;
}

int emx_get_material_info(const emx_problem *p, int material, double *o) {
    if (!p || !o || material < 0 || material >= (int)p->hp.mat.size()) return EMX_E_ARG;
    const Material &m = p->hp.mat[material];
    o[0] = m.n_e; o[1] = m.I; o[2] = m.hwp; o[3] = m.X0; o[4] = m.Tcut; o[5] = m.kcut; o[6] = m.rho; o[7] = m.n_elem;
    return EMX_OK;
}

static bool sizes_ok(long n_slots, long queue_capacity) {
    return n_slots >= 1 && queue_capacity >= 1 && n_slots <= (1L << 22) && queue_capacity <= (1L << 30);
}

size_t emx_workspace_bytes(const emx_problem *p, long n_slots, long queue_capacity) {
    if (!p || !sizes_ok(n_slots, queue_capacity)) return 0;
    Work w;
    return carve_work(nullptr, n_slots, queue_capacity, w, kMaxLog);
}

size_t emx_staging_bytes(long n_primaries) { return n_primaries < 0 ? 0 : staging_bytes(n_primaries); }

int emx_reset_tallies(emx_problem *p, void *stream) {
    if (!p || !p->hp.built) return fail(p, EMX_E_STATE, "emx_reset_tallies: tables not built");
    CU(cudaMemsetAsync(p->d_tally, 0, sizeof(double) * (size_t)(p->hp.n_tally ? p->hp.n_tally : 1), (cudaStream_t)stream));
    return EMX_OK;
}

// blocks of the persistent step kernels: blocks_per_sm of the schedule, else what the compiled kernel's launch
// bounds allow, shared between the chains that run side by side
static void size_grids(const emx_problem *p, Work &w) {
    // defaults per stage (kStage*): 128-thread blocks per SM
    static const int kDefault[kNStages] = {5, 4, 6, 5, 5, 4, 4};
    for (int k = 0; k < kNStages; ++k) {
        int b = p->sched.blocks_per_sm[k] > 0 ? p->sched.blocks_per_sm[k] : kDefault[k];
        // the propagation kernels of a uniform field are compiled for 6 blocks per SM (80 registers), that of a field map for 5
        if (k == kStageField && p->sched.blocks_per_sm[k] <= 0 && p->P.field_kind == 0) b = 6;
        if (b > 16) b = 16;
        w.grid[k] = p->n_sm * b;
    }
    w.grid[7] = 0;
    // what all resident warps of the step kernels can ask of a stack at the same time: 64 warps per SM,
    // 32 lanes x 4 records each
    w.reserve_slack = p->n_sm * 64 * 128;
}

static int transport_device(emx_problem *p, const Primaries &pr, uint64_t seed, long n_slots, long queue_capacity,
                            void *workspace, size_t workspace_bytes, cudaStream_t st) {
    if (pr.first + pr.n > 0x100000000LL) return fail(p, EMX_E_ARG, "emx_transport: primary indices beyond 2^32");
    if (!sizes_ok(n_slots, queue_capacity))
        return fail(p, EMX_E_ARG, "emx_transport: n_slots must be in [1, 2^22] and queue_capacity in [1, 2^30]");
    Work w;
    memset(&w, 0, sizeof(w));  // compared bytewise with the arguments of the kept graph
    const size_t need = carve_work((char *)workspace, n_slots, queue_capacity, w, kMaxLog);
    if (need > workspace_bytes) return fail(p, EMX_E_CAPACITY, "emx_transport: workspace smaller than emx_workspace_bytes()");
    // admission limits (R8): the shower energy in flight is what fills the slots and then the queue
    w.n_primaries = pr.n;
    w.wave = (int)(n_slots / 256 < 256 ? 256 : (n_slots / 256 > 4096 ? 4096 : n_slots / 256));
    w.inflight_cap = (p->sched.mev_per_slot > 0 ? (double)p->sched.mev_per_slot : 20.0) * (double)n_slots;
    w.admit_below = p->sched.admit_below > 0 ? p->sched.admit_below : 2 * n_slots;
    w.slice_above = p->sched.slice_above >= 0 ? p->sched.slice_above : n_slots / 32;
    w.slice_min = p->sched.slice_min > 0 ? p->sched.slice_min : 1;
    w.slice_max = p->sched.slice_max >= w.slice_min ? p->sched.slice_max : w.slice_min;
    size_grids(p, w);
    w.stage_faces = p->sched.blocks_per_sm[7] & 3;  // entry 7 of the schedule: staging switches (bit 0 faces, bit 1 photon tables)
    const bool field = p->P.Bmag != 0.0;
    const int per_iter = launches_per_iteration(field);
    CU(cudaEventRecord(p->ev0, st));
    CU(launch_init(w, pr, st));
    p->launches = 1;
    p->iterations_launched = 0;
    for (double &v : p->prof_ms) v = 0.0;
    p->iter_ms.clear();
    if (p->use_graph && !p->profile) {
        // ---- device-driven path: kIterPerGraph iterations captured once as a CUDA graph; inside an iteration
        // the two pools' chains are parallel branches.  The host only looks at the done flag between graph launches.
        constexpr int kIterPerGraph = 8;
        CU(cudaEventRecord(p->evIn, st));
        CU(cudaStreamWaitEvent(p->s0, p->evIn, 0));
        cudaError_t ce = cudaSuccess;
        Primaries prz;
        memset(&prz, 0, sizeof(prz));
        prz.n = pr.n; prz.ptype = pr.ptype; prz.E = pr.E; prz.pos3 = pr.pos3; prz.dir3 = pr.dir3;
        prz.vol = pr.vol; prz.surf = pr.surf; prz.first = pr.first;
        const bool want_loop = p->sched.loop_node != 0;
        const bool keep = p->graph_exec && p->graph_gen == p->params_gen && p->graph_seed == seed &&
                          p->graph_is_loop == want_loop &&
                          memcmp(&p->graph_w, &w, sizeof(Work)) == 0 && memcmp(&p->graph_pr, &prz, sizeof(Primaries)) == 0;
        // kIterPerGraph iterations of the loop, captured from s0 (fork / join over s1)
        auto capture_iterations = [&]() -> cudaError_t {
            cudaError_t e = cudaSuccess;
            for (int k = 0; k < kIterPerGraph && e == cudaSuccess; ++k) {
                e = launch_refill(w, pr, p->s0);
                if (e == cudaSuccess) e = cudaEventRecord(p->evFork, p->s0);
                if (e == cudaSuccess) e = cudaStreamWaitEvent(p->s1, p->evFork, 0);
                if (e == cudaSuccess) e = launch_step_pool(kPoolCharged, p->P, w, seed, p->d_tally, p->s1);
                if (e == cudaSuccess) e = launch_step_pool(kPoolGamma, p->P, w, seed, p->d_tally, p->s0);
                if (e == cudaSuccess) e = cudaEventRecord(p->evJ1, p->s1);
                if (e == cudaSuccess) e = cudaStreamWaitEvent(p->s0, p->evJ1, 0);
            }
            return e;
        };
        if (!keep) {
            if (p->graph_exec) cudaGraphExecDestroy(p->graph_exec);
            p->graph_exec = nullptr;
            cudaGraph_t graph = nullptr;
            bool looped = false;
            if (want_loop) {
                // the whole loop as ONE graph: a WHILE node whose body is kIterPerGraph iterations followed by
                // a one-thread kernel that sets the node's condition from the done flag -- nothing returns to
                // the host until the transport is over
                cudaGraphConditionalHandle handle = 0;
                cudaGraphNode_t node = nullptr;
                cudaGraphNodeParams np = {cudaGraphNodeTypeConditional};
                ce = cudaGraphCreate(&graph, 0);
                if (ce == cudaSuccess) ce = cudaGraphConditionalHandleCreate(&handle, graph, 1, cudaGraphCondAssignDefault);
                if (ce == cudaSuccess) {
                    np.type = cudaGraphNodeTypeConditional;
                    np.conditional.handle = handle;
                    np.conditional.type = cudaGraphCondTypeWhile;
                    np.conditional.size = 1;
                    ce = cudaGraphAddNode(&node, graph, nullptr, 0, &np);
                }
                if (ce == cudaSuccess)
                    ce = cudaStreamBeginCaptureToGraph(p->s0, np.conditional.phGraph_out[0], nullptr, nullptr, 0,
                                                       cudaStreamCaptureModeThreadLocal);
                if (ce == cudaSuccess) {
                    ce = capture_iterations();
                    if (ce == cudaSuccess) ce = launch_loop_condition(w, (unsigned long long)handle, p->s0);
                    cudaGraph_t body = nullptr;
                    const cudaError_t ce2 = cudaStreamEndCapture(p->s0, &body);
                    if (ce == cudaSuccess) ce = ce2;
                }
                if (ce == cudaSuccess) ce = cudaGraphInstantiate(&p->graph_exec, graph, 0);
                if (ce == cudaSuccess) looped = true;
                else {  // no conditional nodes on this driver: fall back to flat graphs
                    cudaGetLastError();
                    if (graph) cudaGraphDestroy(graph);
                    graph = nullptr;
                    p->graph_exec = nullptr;
                    p->sched.loop_node = 0;
                    ce = cudaSuccess;
                }
            }
            if (!looped) {
                CU(cudaStreamBeginCapture(p->s0, cudaStreamCaptureModeThreadLocal));
                ce = capture_iterations();
                cudaError_t ce2 = cudaStreamEndCapture(p->s0, &graph);
                if (ce != cudaSuccess) { if (graph) cudaGraphDestroy(graph); return fail_cuda(p, ce, "emx_transport: graph capture"); }
                CU(ce2);
                ce = cudaGraphInstantiate(&p->graph_exec, graph, 0);
            }
            cudaGraphDestroy(graph);
            if (ce != cudaSuccess) { p->graph_exec = nullptr; return fail_cuda(p, ce, "cudaGraphInstantiate"); }
            p->graph_w = w;
            p->graph_pr = prz;
            p->graph_seed = seed;
            p->graph_gen = p->params_gen;
            p->graph_is_loop = looped;
        }
        cudaGraphExec_t exec = p->graph_exec;
        if (p->graph_is_loop) {
            ce = cudaGraphLaunch(exec, p->s0);
            if (ce == cudaSuccess) ce = cudaMemcpyAsync(p->h_ctl, w.ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, p->s0);
            if (ce == cudaSuccess) ce = cudaStreamSynchronize(p->s0);
            if (ce == cudaSuccess) {
                const long bodies = (long)((p->h_ctl->iter + kIterPerGraph) / kIterPerGraph);  // the last one finds done
                p->launches += bodies * (kIterPerGraph * per_iter + 1);
                p->iterations_launched += bodies * kIterPerGraph;
            }
        } else {
            int batch = 1;
            for (;;) {
                for (int k = 0; k < batch && ce == cudaSuccess; ++k) ce = cudaGraphLaunch(exec, p->s0);
                p->launches += (long)batch * kIterPerGraph * per_iter;
                p->iterations_launched += (long)batch * kIterPerGraph;
                if (ce == cudaSuccess) ce = cudaMemcpyAsync(p->h_ctl, w.ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, p->s0);
                if (ce == cudaSuccess) ce = cudaStreamSynchronize(p->s0);
                if (ce != cudaSuccess || p->h_ctl->done || p->h_ctl->error) break;
                if (batch < 8) batch *= 2;
            }
        }
        if (ce != cudaSuccess) {
            cudaGraphExecDestroy(p->graph_exec);
            p->graph_exec = nullptr;
            return fail_cuda(p, ce, "emx_transport: iteration graph");
        }
        CU(cudaEventRecord(p->evOut, p->s0));
        CU(cudaStreamWaitEvent(st, p->evOut, 0));
    } else {
        // ---- plain stream launches, kernel by kernel on the caller's stream (what a profiler can list); with
        // profiling on every kernel is bracketed by CUDA events
        static const int kNoField[] = {kStageACharged, kStageBCharged, kStageAGamma, kStageBGamma};
        static const int kField[] = {kStageA0, kStageField, kStageA2, kStageBCharged, kStageAGamma, kStageBGamma};
        const int *order = field ? kField : kNoField;
        const int n_stage = field ? 6 : 4;
        const int ev_per_iter = n_stage + 2;
        int batch = 8;
        for (;;) {
            size_t ne = 0;
            if (p->profile) {
                while (p->prof_ev.size() < (size_t)batch * ev_per_iter) {
                    cudaEvent_t e;
                    CU(cudaEventCreate(&e));
                    p->prof_ev.push_back(e);
                }
            }
            for (int k = 0; k < batch; ++k) {
                if (p->profile) CU(cudaEventRecord(p->prof_ev[ne++], st));
                CU(launch_refill(w, pr, st));
                for (int q = 0; q < n_stage; ++q) {
                    if (p->profile) CU(cudaEventRecord(p->prof_ev[ne++], st));
                    CU(launch_stage(order[q], p->P, w, seed, p->d_tally, st));
                }
                if (p->profile) CU(cudaEventRecord(p->prof_ev[ne++], st));
            }
            p->launches += (long)batch * per_iter;
            p->iterations_launched += batch;
            CU(cudaMemcpyAsync(p->h_ctl, w.ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, st));
            CU(cudaStreamSynchronize(st));
            if (p->profile)
                for (int k = 0; k < batch; ++k) {
                    float ms;
                    const cudaEvent_t *e = &p->prof_ev[(size_t)k * ev_per_iter];
                    CU(cudaEventElapsedTime(&ms, e[0], e[1])); p->prof_ms[kNStages] += ms; p->iter_ms.push_back(ms);
                    for (int q = 0; q < n_stage; ++q) {
                        CU(cudaEventElapsedTime(&ms, e[1 + q], e[2 + q]));
                        p->prof_ms[order[q]] += ms;
                    }
                    CU(cudaEventElapsedTime(&ms, e[1], e[1 + n_stage])); p->prof_ms[kNStages + 1] += ms; p->iter_ms.push_back(ms);
                }
            if (p->h_ctl->done || p->h_ctl->error) break;
            if (batch < 64) batch *= 2;
        }
    }
    CU(cudaEventRecord(p->ev1, st));
    CU(cudaEventSynchronize(p->ev1));
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, p->ev0, p->ev1));
    p->last_ms = ms;
    p->last_ctl = *p->h_ctl;
    p->have_ctl = true;
    const size_t nlog = (size_t)(p->last_ctl.iter < (unsigned long long)kMaxLog ? p->last_ctl.iter : kMaxLog);
    p->iter_log.resize(2 * nlog);
    if (nlog) CU(cudaMemcpy(p->iter_log.data(), w.log, 2 * nlog * sizeof(uint32_t), cudaMemcpyDeviceToHost));
    if (p->last_ctl.error == EMX_E_ARG) return fail(p, EMX_E_ARG, "emx_transport: a primary's particle code is outside 0..2");
    if (p->last_ctl.error) return fail(p, p->last_ctl.error, "emx_transport: secondary stacks full, no track can be stepped");
    return EMX_OK;
}

int emx_transport(emx_problem *p, long n, const int *ptype, const double *E, const double *pos3, const double *dir3,
                  const int *start_vol, const int *start_surf, uint64_t seed, long n_slots, long queue_capacity,
                  void *workspace, size_t workspace_bytes, void *stream) {
    if (!p || !p->hp.built) return fail(p, EMX_E_STATE, "emx_transport: tables not built");
    if (n < 0 || (n > 0 && (!ptype || !E || !pos3 || !dir3 || !start_vol)) || !workspace || n_slots < 1 || queue_capacity < 1)
        return fail(p, EMX_E_ARG, "emx_transport: invalid argument");
    Primaries pr{n, ptype, E, pos3, dir3, start_vol, start_surf, p->prim_first};
    return transport_device(p, pr, seed, n_slots, queue_capacity, workspace, workspace_bytes, (cudaStream_t)stream);
}

int emx_transport_host(emx_problem *p, long n, const int *ptype, const double *E, const double *pos3,
                       const double *dir3, const int *start_vol, const int *start_surf, uint64_t seed, long n_slots,
                       long queue_capacity, void *workspace, size_t workspace_bytes, void *stream) {
    if (!p || !p->hp.built) return fail(p, EMX_E_STATE, "emx_transport_host: tables not built");
    if (n < 0 || (n > 0 && (!ptype || !E || !pos3 || !dir3 || !start_vol)) || !workspace)
        return fail(p, EMX_E_ARG, "emx_transport_host: invalid argument");
    if (!sizes_ok(n_slots, queue_capacity))
        return fail(p, EMX_E_ARG, "emx_transport_host: n_slots must be in [1, 2^22] and queue_capacity in [1, 2^30]");
    cudaStream_t st = (cudaStream_t)stream;
    // the primaries are staged in the caller's workspace, behind the part emx_workspace_bytes() describes
    Work w0;
    const size_t body = carve_work(nullptr, n_slots, queue_capacity, w0, kMaxLog);
    if (body + staging_bytes(n) > workspace_bytes)
        return fail(p, EMX_E_CAPACITY, "emx_transport_host: workspace smaller than emx_workspace_bytes() + emx_staging_bytes()");
    const size_t nn = (size_t)(n ? n : 1);
    Carve c{(char *)workspace + body};
    int *d_pt = c.take<int>(nn), *d_vol = c.take<int>(nn), *d_surf = c.take<int>(nn);
    double *d_E = c.take<double>(nn), *d_pos = c.take<double>(3 * nn), *d_dir = c.take<double>(3 * nn);
    cudaError_t e = cudaSuccess;
    auto up = [&](void *dst, const void *src, size_t b) {
        if (e == cudaSuccess && b) e = cudaMemcpyAsync(dst, src, b, cudaMemcpyHostToDevice, st);
    };
    up(d_pt, ptype, (size_t)n * 4);
    up(d_vol, start_vol, (size_t)n * 4);
    if (start_surf) up(d_surf, start_surf, (size_t)n * 4);
    up(d_E, E, (size_t)n * 8);
    up(d_pos, pos3, (size_t)n * 24);
    up(d_dir, dir3, (size_t)n * 24);
    if (e != cudaSuccess) return fail_cuda(p, e, "emx_transport_host: upload");
    Primaries pr{n, d_pt, d_E, d_pos, d_dir, d_vol, start_surf ? d_surf : nullptr, p->prim_first};
    return transport_device(p, pr, seed, n_slots, queue_capacity, workspace, body, st);
}

int emx_set_primary_offset(emx_problem *p, long first) {
    if (!p) return fail(p, EMX_E_ARG, "emx_set_primary_offset: null problem");
    if (first < 0 || first > 0xffffffffL) return fail(p, EMX_E_ARG, "emx_set_primary_offset: offset outside [0, 2^32)");
    p->prim_first = first;
    return EMX_OK;
}

int emx_neighbour_candidates(const emx_problem *cp, int surface, int sense, int which, int32_t *host_out, int cap) {
    emx_problem *p = const_cast<emx_problem *>(cp);
    if (!p || surface < 0 || surface >= (int)p->hp.surf_type.size() || (sense != 1 && sense != -1) || (which != 0 && which != 1) ||
        cap < 0 || (cap > 0 && !host_out))
        return fail(p, EMX_E_ARG, "emx_neighbour_candidates: invalid argument");
    std::vector<int> off, list;
    if (which == 0) build_neighbour_lists(p->hp, off, list);
    else build_nonlisting_lists(p->hp, off, list);
    const int k = 2 * surface + (sense > 0 ? 1 : 0);
    const int n = off[k + 1] - off[k];
    for (int j = 0; j < n && j < cap; ++j) host_out[j] = list[off[k] + j];
    return n;
}

int emx_get_schedule(const emx_problem *p, emx_schedule *out) {
    if (!p || !out) return EMX_E_ARG;
    *out = p->sched;
    return EMX_OK;
}

int emx_set_schedule(emx_problem *p, const emx_schedule *in) {
    if (!p || !in) return fail(p, EMX_E_ARG, "emx_set_schedule: null argument");
    if (in->slice_min < 1 || in->slice_max < in->slice_min)
        return fail(p, EMX_E_ARG, "emx_set_schedule: need 1 <= slice_min <= slice_max");
    for (int k = 0; k < 8; ++k)
        if (in->blocks_per_sm[k] < 0 || in->blocks_per_sm[k] > 16)
            return fail(p, EMX_E_ARG, "emx_set_schedule: blocks_per_sm outside 0..16");
    p->sched = *in;
    return EMX_OK;
}

int emx_read_tallies(const emx_problem *cp, double *edep_host, emx_scalars *out) {
    emx_problem *p = const_cast<emx_problem *>(cp);
    if (!p || !p->hp.built) return fail(p, EMX_E_STATE, "emx_read_tallies: tables not built");
    if (edep_host && p->hp.n_tally)
        CU(cudaMemcpy(edep_host, p->d_tally, sizeof(double) * (size_t)p->hp.n_tally, cudaMemcpyDeviceToHost));
    if (out) {
        memset(out, 0, sizeof(*out));
        if (p->have_ctl) {
            const Ctl &c = p->last_ctl;
            out->escaped = c.escaped; out->below_cut = c.below_cut; out->looper = c.looper; out->E_in = c.E_in;
            for (int k = 0; k < 3; ++k) { out->steps[k] = c.steps[k]; out->tracks[k] = c.tracks[k]; }
            for (int k = 0; k < EMX_NPROC; ++k) out->inter[k] = c.inter[k];
            out->null_int = c.null_int;
            out->track_steps = c.steps[0] + c.steps[1] + c.steps[2];
            out->stalls = c.stalls; out->iterations = c.iter; out->peak_live = c.peak_live; out->peak_queue = c.peak_queue;
        }
    }
    return EMX_OK;
}

double emx_last_transport_ms(const emx_problem *p) { return p ? p->last_ms : -1.0; }

int emx_set_profile(emx_problem *p, int on) {
    if (!p) return EMX_E_ARG;
    p->profile = (on & 1) != 0;
    p->use_graph = (on & 2) == 0;  // bit 1: plain stream launches without profiling (diagnostics)
    return EMX_OK;
}

int emx_get_profile(const emx_problem *p, double *ms9, long *launches, long *iterations_launched) {
    if (!p) return EMX_E_ARG;
    if (ms9) for (int k = 0; k < kNStages + 2; ++k) ms9[k] = p->prof_ms[k];
    if (launches) *launches = p->launches;
    if (iterations_launched) *iterations_launched = p->iterations_launched;
    return EMX_OK;
}

long emx_get_iteration_log(const emx_problem *p, uint32_t *host_out, long max_iter) {
    if (!p || !host_out || max_iter < 0) return EMX_E_ARG;
    long n = (long)(p->iter_log.size() / 2);
    if (n > max_iter) n = max_iter;
    if (n) memcpy(host_out, p->iter_log.data(), (size_t)n * 2 * sizeof(uint32_t));
    return n;
}

int emx_get_lanes(const emx_problem *p, uint64_t *lanes8) {
    if (!p || !lanes8 || !p->have_ctl) return EMX_E_ARG;
    const Ctl &c = p->last_ctl;
    const bool field = p->P.Bmag != 0.0;
    lanes8[kStageAGamma] = c.lanes[2][kPoolGamma];
    lanes8[kStageACharged] = field ? 0ull : c.lanes[2][kPoolCharged];
    lanes8[kStageA0] = c.lanes[0][kPoolCharged];
    lanes8[kStageField] = c.lanes[1][kPoolCharged];
    lanes8[kStageA2] = field ? c.lanes[2][kPoolCharged] : 0ull;
    lanes8[kStageBGamma] = c.lanes[3][kPoolGamma];
    lanes8[kStageBCharged] = c.lanes[3][kPoolCharged];
    lanes8[7] = c.attempts;
    return EMX_OK;
}

int emx_read_step_hist(const emx_problem *cp, uint64_t *hist_host) {
    emx_problem *p = const_cast<emx_problem *>(cp);
    if (!p || !hist_host) return fail(p, EMX_E_ARG, "emx_read_step_hist: null argument");
    if (!p->have_ctl) return fail(p, EMX_E_STATE, "emx_read_step_hist: no transport yet");
    for (int pt = 0; pt < 3; ++pt)
        for (int b = 0; b < EMX_NHIST; ++b) hist_host[pt * EMX_NHIST + b] = p->last_ctl.hist[pt][b];
    return EMX_OK;
}

long emx_get_iteration_times(const emx_problem *p, float *host_out, long max_iter) {
    if (!p || !host_out || max_iter < 0) return EMX_E_ARG;
    long n = (long)(p->iter_ms.size() / 2);
    if (n > max_iter) n = max_iter;
    if (n) memcpy(host_out, p->iter_ms.data(), (size_t)n * 2 * sizeof(float));
    return n;
}

int emx_step_batch(emx_problem *p, uint64_t seed, long n, const emx_track *in, emx_step_result *out, void *stream) {
    if (!p || !p->hp.built) return fail(p, EMX_E_STATE, "emx_step_batch: tables not built");
    if (n < 0 || (n > 0 && (!in || !out))) return fail(p, EMX_E_ARG, "emx_step_batch: invalid argument");
    CU(launch_step_batch(p->P, seed, n, in, out, (cudaStream_t)stream));
    return EMX_OK;
}

int emx_field_substep_batch(emx_problem *p, long n, const double *x3, const double *u3, const double *kappa,
                            const double *h, double *x1, double *u1, double *err, void *stream) {
    if (!p || !p->hp.built) return fail(p, EMX_E_STATE, "emx_field_substep_batch: tables not built");
    if (n < 0 || (n > 0 && (!x3 || !u3 || !kappa || !h || !x1 || !u1 || !err)))
        return fail(p, EMX_E_ARG, "emx_field_substep_batch: invalid argument");
    if (p->P.Bmag <= 0.0) return fail(p, EMX_E_STATE, "emx_field_substep_batch: no field set");
    CU(launch_field_substep_batch(p->P, n, x3, u3, kappa, h, x1, u1, err, (cudaStream_t)stream));
    return EMX_OK;
}

int emx_philox_batch(long n, const uint32_t *ctr4, const uint32_t *key2, uint32_t *out4, void *stream) {
    emx_problem *p = nullptr;
    if (n < 0 || (n > 0 && (!ctr4 || !key2 || !out4))) return fail(p, EMX_E_ARG, "emx_philox_batch: invalid argument");
    CU(launch_philox_batch(n, ctr4, key2, out4, (cudaStream_t)stream));
    return EMX_OK;
}

int emx_draw_batch(uint64_t seed, long n, const uint32_t *prim, const uint64_t *tid, const uint32_t *step,
                   const uint32_t *nn, double *u, uint64_t *child, void *stream) {
    emx_problem *p = nullptr;
    if (n < 0 || (n > 0 && (!prim || !tid || !step || !nn))) return fail(p, EMX_E_ARG, "emx_draw_batch: invalid argument");
    CU(launch_draw_batch(seed, n, prim, tid, step, nn, u, child, (cudaStream_t)stream));
    return EMX_OK;
}

int emx_refill_plan(long n_live, long capacity, long n_queue, const uint8_t *alive, int32_t *src, long *counts_host,
                    void *stream) {
    emx_problem *p = nullptr;
    if (n_live < 0 || capacity < n_live || capacity < 1 || n_queue < 0 || (n_live > 0 && !alive) || !src || !counts_host ||
        capacity > (1L << 30) || n_queue > (1L << 30))
        return fail(p, EMX_E_ARG, "emx_refill_plan: invalid argument");
    cudaStream_t st = (cudaStream_t)stream;
    int *scratch = nullptr;
    const size_t ints = refill_plan_scratch_ints(capacity);
    CU(cudaMalloc(&scratch, ints * sizeof(int)));
    const Ctl *d_ctl = nullptr;
    cudaError_t e = launch_refill_plan(n_live, capacity, n_queue, alive, src, scratch, &d_ctl, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    Ctl hc;
    if (e == cudaSuccess) e = cudaMemcpy(&hc, d_ctl, sizeof(Ctl), cudaMemcpyDeviceToHost);
    cudaFree(scratch);
    if (e != cudaSuccess) return fail_cuda(p, e, "emx_refill_plan");
    counts_host[0] = hc.plan[0].n_final;
    counts_host[1] = hc.plan[0].q_new;
    counts_host[2] = hc.plan[0].h - hc.plan[0].a;
    return EMX_OK;
}

}  // extern "C"

// ---- emx_refill_plan_static: the refill hook for callers that cannot allocate (include/emx.h) ----
// Same kernels as emx_refill_plan; their scratch (chunk tables, hole list, control block, a padded copy of the alive
// flags) lives in ONE file-scope device array instead of a cudaMalloc'ed block.  Every GPU that loads libemx holds the
// array until the process exits; every call shares it.
namespace {
constexpr long kStaticPlanMaxCapacity = 1L << 16;  // slots: what emx_refill_plan_static accepts
constexpr size_t static_plan_ints(long capacity) {  // the layout of launch_refill_plan (emx_transport.cu)
    return 7 * ((size_t)(capacity + kChunk - 1) / kChunk + 1) + (size_t)capacity + (sizeof(Ctl) + 3) / 4 + 64 +
           (((size_t)(capacity + kChunk - 1) / kChunk + 1) * kChunk + 3) / 4 + 64;
}
constexpr size_t kStaticPlanInts = static_plan_ints(kStaticPlanMaxCapacity);  // 345 KB
}  // namespace

static __device__ __align__(256) int g_static_plan_scratch[kStaticPlanInts];

namespace {
constexpr int kMaxDevices = 64;
int *g_static_plan_ptr[kMaxDevices];  // device address of the array on each device, looked up once
std::mutex g_static_plan_mu;

// The array's name is a host-side stand-in in host code: its device address comes from the runtime, once per device,
// with that device current.
int static_plan_scratch(int **out) {
    emx_problem *p = nullptr;
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return fail(p, EMX_E_ARG, "emx_refill_plan_static: device ordinal above 63");
    std::lock_guard<std::mutex> lock(g_static_plan_mu);
    if (!g_static_plan_ptr[dev]) {
        void *a = nullptr;
        CU(cudaGetSymbolAddress(&a, g_static_plan_scratch));
        if (!a) return fail(p, EMX_E_CUDA, "emx_refill_plan_static: no device address for the scratch array");
        g_static_plan_ptr[dev] = static_cast<int *>(a);
    }
    *out = g_static_plan_ptr[dev];
    return EMX_OK;
}
}  // namespace

extern "C" {

long emx_refill_plan_static_max(void) { return kStaticPlanMaxCapacity; }

int emx_refill_plan_static_setup(void) {
    int *scratch = nullptr;
    return static_plan_scratch(&scratch);
}

int emx_refill_plan_static(long n_live, long capacity, long n_queue, const uint8_t *alive, int32_t *src,
                           long *counts_host, void *stream) {
    emx_problem *p = nullptr;
    if (n_live < 0 || capacity < n_live || capacity < 1 || n_queue < 0 || (n_live > 0 && !alive) || !src || !counts_host ||
        n_queue > (1L << 30))
        return fail(p, EMX_E_ARG, "emx_refill_plan_static: invalid argument");
    if (capacity > kStaticPlanMaxCapacity || refill_plan_scratch_ints(capacity) > kStaticPlanInts) {
        char buf[160];
        snprintf(buf, sizeof buf, "emx_refill_plan_static: capacity %ld is above the %ld slots the static scratch holds "
                 "(use emx_refill_plan)", capacity, kStaticPlanMaxCapacity);
        g_err = buf;
        return EMX_E_CAPACITY;
    }
    int *scratch = nullptr;
    const int rc = static_plan_scratch(&scratch);
    if (rc != EMX_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    // the array keeps what the last call left in it: everything this call uses starts from zero
    CU(cudaMemsetAsync(scratch, 0, refill_plan_scratch_ints(capacity) * sizeof(int), st));
    const Ctl *d_ctl = nullptr;
    cudaError_t e = launch_refill_plan(n_live, capacity, n_queue, alive, src, scratch, &d_ctl, st);
    PoolPlan plan = PoolPlan();  // three counts come back through a plain host struct: no staging buffer of ours
    if (e == cudaSuccess) e = cudaMemcpyAsync(&plan, &d_ctl->plan[0], sizeof(PoolPlan), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return fail_cuda(p, e, "emx_refill_plan_static");
    counts_host[0] = plan.n_final;
    counts_host[1] = plan.q_new;
    counts_host[2] = plan.h - plan.a;
    return EMX_OK;
}

}  // extern "C"
