// emx_api.cu -- the C-ABI of include/emx.h: problem object, table build, transport driver, tallies, hooks.
// Host logic only; every computation of the path runs in the kernels of emx_kernels.cu / emx_transport.cu.
#include <cuda_runtime.h>
#include <cstdio>
#include <cstdlib>
#include <cstring>
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
    double prof_ms[8] = {0, 0, 0, 0, 0, 0, 0, 0};  // phase A gamma, e-, e+; phase B gamma, e-, e+; refill; all step kernels
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
    int loop_node = 1;         // 1: the whole loop is one graph with a WHILE node; 0: flat graphs + host polling
    bool graph_is_loop = false;
    bool use_graph = true;
    long slice_above = -1;  // < 0: n_slots / 32
    int slice_budget = 2;
    int warps_per_sm[3] = {16, 16, 8};  // gamma, e-, e+ (the e+ pool holds 8 % of the slots)
    double pool_frac[3] = {0.0, 0.0, 0.0};  // EMX_POOL_FRAC: share of the slots per pool (0: the default split)
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

// split n into three pool sizes (gamma, e-, e+), each a multiple of kChunk
void split3(long n, const double f[3], int out[3]) {
    long used = 0;
    for (int k = 0; k < 3; ++k) {
        long v = (long)((double)n * f[k]) / kChunk * kChunk;
        if (v < kChunk) v = kChunk;
        out[k] = (int)v;
        used += v;
    }
    (void)used;
}

const double kPoolFrac[3] = {0.50, 0.42, 0.08};   // measured live mix of the workloads
const double kQueueFrac[3] = {0.30, 0.60, 0.10};  // e- secondaries dominate the queued records in every config

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

// with multiple scattering the charged tracks take ~7x the steps: measured on config 7, +24 % over the split above
const double kPoolFracMsc[3] = {0.25, 0.63, 0.12};
// share of the track slots per pool: the knob if set, else the default split for the physics of the problem
// (the split decides when a step is taken, never its result)
static const double *pool_split(const emx_problem *p) {
    return p->pool_frac[0] > 0.0 ? p->pool_frac : (p->hp.ph.msc ? kPoolFracMsc : kPoolFrac);
}

// carve the caller's workspace; with base == nullptr only the size is computed
size_t carve_work(char *base, long n_slots, long qcap, Work &w, int max_log, const double *pool_frac) {
    Carve c{base};
    split3(n_slots, pool_frac, w.cap);
    split3(qcap, kQueueFrac, w.qcap);
    w.ctl = c.take<Ctl>(1);
    w.log = c.take<uint32_t>(2 * (size_t)max_log);
    w.max_log = max_log;
    for (int p = 0; p < 3; ++p) {
        const size_t n = (size_t)w.cap[p], nch = n / kChunk + 1;
        TrackSoA &t = w.trk[p];
        t.x = c.take<double>(n); t.y = c.take<double>(n); t.z = c.take<double>(n);
        t.ux = c.take<double>(n); t.uy = c.take<double>(n); t.uz = c.take<double>(n);
        t.E = c.take<double>(n);
        t.tid = c.take<uint64_t>(n);
        t.prim = c.take<uint32_t>(n); t.step = c.take<uint32_t>(n);
        t.vol = c.take<int>(n); t.surf = c.take<int>(n);
        t.alive = c.take<uint8_t>(n);
        t.pend = c.take<uint8_t>(n);
        if (p != 0) {
            t.fs_s = c.take<double>(n);
            t.fs_h = c.take<double>(n);
            t.fs_a = c.take<int>(n);
        } else {
            t.fs_s = t.fs_h = nullptr;
            t.fs_a = nullptr;
        }
        w.chunk_dead[p] = c.take<int>(nch);
        w.chunk_off[p] = c.take<int>(nch);
        w.hole_idx[p] = c.take<int>(n);
        for (int k = 0; k < 3; ++k) w.ilist[p][k] = c.take<int>(n);
    }
    // everything above (track store, scan arrays, interaction lists: about 110 MB at 2^20 slots) is touched in
    // every iteration and is kept together; the stacks follow.  (A persisting-L2 access-policy window over
    // this region was tried: 83 MB can be set aside on B200, and it was 9 % slower.)
    w.hot_bytes = align_up(c.off, 256);
    for (int p = 0; p < 3; ++p) {
        const size_t q = (size_t)w.qcap[p];
        QueueSoA &s = w.q[p];
        s.x = c.take<double>(q); s.y = c.take<double>(q); s.z = c.take<double>(q);
        s.ux = c.take<double>(q); s.uy = c.take<double>(q); s.uz = c.take<double>(q);
        s.E = c.take<double>(q);
        s.tid = c.take<uint64_t>(q);
        s.prim = c.take<uint32_t>(q);
        s.vol = c.take<int>(q); s.surf = c.take<int>(q);
    }
    return align_up(c.off, 256);
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
    // tuning knobs of the scheduler (they never change a result, only when work is done)
    if (const char *e = getenv("EMX_SLICE_BUDGET")) p->slice_budget = atoi(e) > 0 ? atoi(e) : p->slice_budget;
    if (const char *e = getenv("EMX_SLICE_ABOVE")) p->slice_above = atol(e);
    if (const char *e = getenv("EMX_LOOP_NODE")) p->loop_node = atoi(e);
    if (const char *e = getenv("EMX_POOL_FRAC")) {
        double f[3] = {0, 0, 0};
        if (sscanf(e, "%lf,%lf,%lf", &f[0], &f[1], &f[2]) == 3 && f[0] > 0 && f[1] > 0 && f[2] > 0)
            for (int k = 0; k < 3; ++k) p->pool_frac[k] = f[k] / (f[0] + f[1] + f[2]);
    }
    if (const char *e = getenv("EMX_WARPS_PER_SM")) sscanf(e, "%d,%d,%d", &p->warps_per_sm[0], &p->warps_per_sm[1], &p->warps_per_sm[2]);
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
    if (ph->msc && (!(ph->msc_fr > 0.0) || !(ph->msc_smin > 0.0)))
        return fail(p, EMX_E_ARG, "emx_set_physics: multiple scattering needs msc_fr > 0 and msc_smin > 0");
    p->hp.ph = *ph;
    p->hp.built = false;
    return EMX_OK;
}

int emx_set_cuts(emx_problem *p, int material, double Tcut, double kcut) {
    if (!p || material < 0 || material >= (int)p->hp.mat.size()) return fail(p, EMX_E_ARG, "emx_set_cuts: unknown material");
    p->hp.mat[material].Tcut = Tcut;
    p->hp.mat[material].kcut = kcut;
    p->hp.built = false;
    return EMX_OK;
}

int emx_n_tally(const emx_problem *p) { return p ? p->hp.n_tally : EMX_E_ARG; }

int emx_build_tables(emx_problem *p, void *stream) {
    if (!p) return fail(p, EMX_E_ARG, "emx_build_tables: null problem");
    HostProblem &hp = p->hp;
    if (hp.vol.empty()) return fail(p, EMX_E_STATE, "emx_build_tables: no volume defined");
    for (const Material &m : hp.mat)
        if (!(hp.ph.prod_cut_cm > 0.0) && (m.Tcut < 0.0 || m.kcut < 0.0))
            return fail(p, EMX_E_STATE, "emx_build_tables: no production cut length and no explicit cut energies");
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
    P.tab = p->d_tab;
    P.nb_off = p->d_nb_off;
    P.nb_list = p->d_nb_list;
    P.nb2_off = p->d_nb2_off;
    P.nb2_list = p->d_nb2_list;
    const double bm = sqrt(hp.B[0] * hp.B[0] + hp.B[1] * hp.B[1] + hp.B[2] * hp.B[2]);
    P.Bmag = bm;
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

size_t emx_workspace_bytes(const emx_problem *p, long n_slots, long queue_capacity) {
    // pools hold fewer than 2^21 slots each (packed list counters): n_slots <= 2^21
    if (!p || n_slots < 1 || queue_capacity < 1 || n_slots > (1L << 21) || queue_capacity > (1L << 30)) return 0;
    Work w;
    return carve_work(nullptr, n_slots, queue_capacity, w, kMaxLog, pool_split(p));
}

int emx_reset_tallies(emx_problem *p, void *stream) {
    if (!p || !p->hp.built) return fail(p, EMX_E_STATE, "emx_reset_tallies: tables not built");
    CU(cudaMemsetAsync(p->d_tally, 0, sizeof(double) * (size_t)(p->hp.n_tally ? p->hp.n_tally : 1), (cudaStream_t)stream));
    return EMX_OK;
}

static int transport_device(emx_problem *p, const Primaries &pr, uint64_t seed, long n_slots, long queue_capacity,
                            void *workspace, size_t workspace_bytes, cudaStream_t st) {
    if (pr.first + pr.n > 0x100000000LL) return fail(p, EMX_E_ARG, "emx_transport: primary indices beyond 2^32");
    Work w;
    memset(&w, 0, sizeof(w));  // compared bytewise with the arguments of the kept graph
    const size_t need = carve_work((char *)workspace, n_slots, queue_capacity, w, kMaxLog, pool_split(p));
    if (need > workspace_bytes) return fail(p, EMX_E_CAPACITY, "emx_transport: workspace smaller than emx_workspace_bytes()");
    // admission limits (R8): about 20 MeV of shower energy in flight per queued record at the peak of
    // the queue (measured on configs 1-4), with a factor 4 of headroom below the capacity
    w.n_primaries = pr.n;
    w.wave = (int)(n_slots / 256 < 256 ? 256 : (n_slots / 256 > 4096 ? 4096 : n_slots / 256));
    w.inflight_cap = 5.0 * (double)queue_capacity;
    w.slice_above = p->slice_above >= 0 ? p->slice_above : n_slots / 32;
    w.slice_budget = p->slice_budget;
    for (int k = 0; k < 3; ++k) w.warps_per_sm[k] = p->warps_per_sm[k];
    CU(cudaEventRecord(p->ev0, st));
    CU(launch_init(w, pr, st));
    p->launches = 1;
    p->iterations_launched = 0;
    for (double &v : p->prof_ms) v = 0.0;
    p->iter_ms.clear();
    if (p->use_graph && !p->profile) {
        // ---- device-driven path: kIterPerGraph iterations captured once as a CUDA graph; inside an iteration
        // the three step kernels are parallel branches, so the tail of one pool overlaps the start of the next.
        // The host only looks at the done flag between graph launches.
        constexpr int kIterPerGraph = 8;
        CU(cudaEventRecord(p->evIn, st));
        CU(cudaStreamWaitEvent(p->s0, p->evIn, 0));
        cudaError_t ce = cudaSuccess;
        Primaries prz;
        memset(&prz, 0, sizeof(prz));
        prz.n = pr.n; prz.ptype = pr.ptype; prz.E = pr.E; prz.pos3 = pr.pos3; prz.dir3 = pr.dir3;
        prz.vol = pr.vol; prz.surf = pr.surf; prz.first = pr.first;
        const bool keep = p->graph_exec && p->graph_gen == p->params_gen && p->graph_seed == seed &&
                          p->graph_is_loop == (p->loop_node != 0) &&
                          memcmp(&p->graph_w, &w, sizeof(Work)) == 0 && memcmp(&p->graph_pr, &prz, sizeof(Primaries)) == 0;
        // kIterPerGraph iterations of the loop, captured from s0 (fork / join over s1, s2)
        auto capture_iterations = [&]() -> cudaError_t {
            cudaError_t e = cudaSuccess;
            for (int k = 0; k < kIterPerGraph && e == cudaSuccess; ++k) {
                e = launch_refill(w, pr, p->s0);
                if (e == cudaSuccess) e = cudaEventRecord(p->evFork, p->s0);
                if (e == cudaSuccess) e = cudaStreamWaitEvent(p->s1, p->evFork, 0);
                if (e == cudaSuccess) e = cudaStreamWaitEvent(p->s2, p->evFork, 0);
                if (e == cudaSuccess) e = launch_step_pool(kPositron, p->P, w, seed, p->d_tally, p->n_sm, p->s1);
                if (e == cudaSuccess) e = launch_step_pool(kElectron, p->P, w, seed, p->d_tally, p->n_sm, p->s2);
                if (e == cudaSuccess) e = launch_step_pool(kGamma, p->P, w, seed, p->d_tally, p->n_sm, p->s0);
                if (e == cudaSuccess) e = cudaEventRecord(p->evJ1, p->s1);
                if (e == cudaSuccess) e = cudaEventRecord(p->evJ2, p->s2);
                if (e == cudaSuccess) e = cudaStreamWaitEvent(p->s0, p->evJ1, 0);
                if (e == cudaSuccess) e = cudaStreamWaitEvent(p->s0, p->evJ2, 0);
            }
            return e;
        };
        if (!keep) {
            if (p->graph_exec) cudaGraphExecDestroy(p->graph_exec);
            p->graph_exec = nullptr;
            cudaGraph_t graph = nullptr;
            bool looped = false;
            if (p->loop_node) {
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
                    p->loop_node = 0;
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
                p->launches += bodies * (kIterPerGraph * kLaunchesPerIteration + 1);
                p->iterations_launched += bodies * kIterPerGraph;
            }
        } else {
            int batch = 1;
            for (;;) {
                for (int k = 0; k < batch && ce == cudaSuccess; ++k) ce = cudaGraphLaunch(exec, p->s0);
                p->launches += (long)batch * kIterPerGraph * kLaunchesPerIteration;
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
    int batch = 8;
    for (;;) {
        size_t ne = 0;
        if (p->profile) {
            while (p->prof_ev.size() < (size_t)batch * 8) {
                cudaEvent_t e;
                CU(cudaEventCreate(&e));
                p->prof_ev.push_back(e);
            }
        }
        for (int k = 0; k < batch; ++k) {
            if (p->profile) CU(cudaEventRecord(p->prof_ev[ne++], st));
            CU(launch_refill(w, pr, st));
            if (p->profile) {
                for (int pt = 2; pt >= 0; --pt)
                    for (int ph = 0; ph < 2; ++ph) {
                        CU(cudaEventRecord(p->prof_ev[ne++], st));
                        CU(launch_phase(pt, ph, p->P, w, seed, p->d_tally, p->n_sm, st));
                    }
                CU(cudaEventRecord(p->prof_ev[ne++], st));
            } else {
                CU(launch_step(p->P, w, seed, p->d_tally, p->n_sm, st));
            }
        }
        p->launches += (long)batch * kLaunchesPerIteration;
        p->iterations_launched += batch;
        CU(cudaMemcpyAsync(p->h_ctl, w.ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        if (p->profile)
            for (int k = 0; k < batch; ++k) {
                float ms;
                const cudaEvent_t *e = &p->prof_ev[(size_t)k * 8];
                CU(cudaEventElapsedTime(&ms, e[0], e[1])); p->prof_ms[6] += ms; p->iter_ms.push_back(ms);
                int q = 1;
                for (int pt = 2; pt >= 0; --pt)
                    for (int ph = 0; ph < 2; ++ph, ++q) {
                        CU(cudaEventElapsedTime(&ms, e[q], e[q + 1]));
                        p->prof_ms[3 * ph + pt] += ms;
                    }
                CU(cudaEventElapsedTime(&ms, e[1], e[7])); p->prof_ms[7] += ms; p->iter_ms.push_back(ms);
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
    cudaStream_t st = (cudaStream_t)stream;
    // staging area for the primaries: 4 + 8 + 24 + 24 + 4 + 4 bytes each
    const size_t nn = (size_t)(n ? n : 1);
    char *d = nullptr;
    const size_t bytes = align_up(nn * 4, 256) * 3 + align_up(nn * 8, 256) + 2 * align_up(nn * 24, 256);
    CU(cudaMalloc(&d, bytes));
    Carve c{d};
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
    int rc;
    if (e != cudaSuccess) rc = fail_cuda(p, e, "emx_transport_host: upload");
    else {
        Primaries pr{n, d_pt, d_E, d_pos, d_dir, d_vol, start_surf ? d_surf : nullptr, p->prim_first};
        rc = transport_device(p, pr, seed, n_slots, queue_capacity, workspace, workspace_bytes, st);
    }
    cudaFree(d);
    return rc;
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

int emx_set_pool_split(emx_problem *p, double fg, double fe, double fp) {
    if (!p) return fail(p, EMX_E_ARG, "emx_set_pool_split: null problem");
    if (fg == 0.0 && fe == 0.0 && fp == 0.0) {
        p->pool_frac[0] = p->pool_frac[1] = p->pool_frac[2] = 0.0;
        return EMX_OK;
    }
    if (!(fg > 0.0) || !(fe > 0.0) || !(fp > 0.0)) return fail(p, EMX_E_ARG, "emx_set_pool_split: every share must be > 0");
    const double s = fg + fe + fp;
    p->pool_frac[0] = fg / s;
    p->pool_frac[1] = fe / s;
    p->pool_frac[2] = fp / s;
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

int emx_get_profile(const emx_problem *p, double *ms4, long *launches, long *iterations_launched) {  // ms4: 8 doubles
    if (!p) return EMX_E_ARG;
    if (ms4) for (int k = 0; k < 8; ++k) ms4[k] = p->prof_ms[k];
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

int emx_get_lanes(const emx_problem *p, uint64_t *lanes6) {
    if (!p || !lanes6 || !p->have_ctl) return EMX_E_ARG;
    for (int ph = 0; ph < 2; ++ph)
        for (int pt = 0; pt < 3; ++pt) lanes6[3 * ph + pt] = p->last_ctl.lanes[ph][pt];
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
    cudaError_t e = launch_refill_plan(n_live, capacity, n_queue, alive, src, scratch, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    Ctl hc;
    if (e == cudaSuccess) {
        // the control block sits behind the three int arrays (see launch_refill_plan)
        const size_t nch = (size_t)(capacity + kChunk - 1) / kChunk + 1;
        int *q = scratch + 2 * nch + capacity;
        q += (16 - ((uintptr_t)q / 4) % 16) % 16;
        e = cudaMemcpy(&hc, q, sizeof(Ctl), cudaMemcpyDeviceToHost);
    }
    cudaFree(scratch);
    if (e != cudaSuccess) return fail_cuda(p, e, "emx_refill_plan");
    counts_host[0] = hc.plan[0].n_final;
    counts_host[1] = hc.plan[0].q_new;
    counts_host[2] = hc.plan[0].h - hc.plan[0].a;
    return EMX_OK;
}

}  // extern "C"
