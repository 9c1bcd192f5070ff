// emx_kernels.h -- launchers of the CUDA kernels (emx_kernels.cu, emx_transport.cu), called by emx_api.cu.
#pragma once
#include <cuda_runtime.h>
#include "emx_core.h"
#include "emx_work.h"

namespace emx {

struct TableCtx;

cudaError_t launch_build_tables(const TableCtx &c, cudaStream_t st);
cudaError_t launch_step_batch(const Params &P, uint64_t seed, long n, const emx_track *in, emx_step_result *out,
                              cudaStream_t st);
cudaError_t launch_field_substep_batch(const Params &P, long n, const double *x3, const double *u3, const double *kappa,
                                       const double *h, double *x1, double *u1, double *err, cudaStream_t st);
cudaError_t launch_philox_batch(long n, const uint32_t *ctr, const uint32_t *key, uint32_t *out, cudaStream_t st);
cudaError_t launch_draw_batch(uint64_t seed, long n, const uint32_t *prim, const uint64_t *tid, const uint32_t *step,
                              const uint32_t *nn, double *u, uint64_t *child, cudaStream_t st);

// primaries in DEVICE memory (AoS xyz as in include/emx.h)
struct Primaries {
    long n;
    const int *ptype;
    const double *E, *pos3, *dir3;
    const int *vol, *surf;  // surf may be null
    long long first;        // primary index of element 0 (emx_set_primary_offset): element i is primary first + i
};

// the step kernels by stage (index of Work::grid, of emx_get_profile's milliseconds and of emx_get_lanes)
enum : int {
    kStageAGamma = 0,    // k_a<gamma>: limits + straight move + finish
    kStageACharged = 1,  // k_a<charged>: the same for e+- when there is no field
    kStageA0 = 2,        // k_a0: limits of e+- (field)
    kStageField = 3,     // k_field: adaptive RK4 propagation of e+-
    kStageA2 = 4,        // k_a2: finish of e+- (field)
    kStageBGamma = 5,    // k_b<gamma>: Compton, photoelectric, pair production
    kStageBCharged = 6,  // k_b<charged>: Moller, Bhabha, bremsstrahlung, annihilation
    kNStages = 7
};

// resets the control block, totals the injected energy
cudaError_t launch_init(const Work &w, const Primaries &pr, cudaStream_t st);
// one iteration of the loop = launch_refill (k_plan, k_fill, k_move) then the two pools' chains
// (launch_step_pool, or stage by stage with launch_stage); tally = device edep array
cudaError_t launch_refill(const Work &w, const Primaries &pr, cudaStream_t st);
// sets the condition of a graph WHILE node (handle from cudaGraphConditionalHandleCreate): go on unless done
cudaError_t launch_loop_condition(const Work &w, unsigned long long handle, cudaStream_t st);
cudaError_t launch_stage(int stage, const Params &P, const Work &w, uint64_t seed, double *tally, cudaStream_t st);
cudaError_t launch_step_pool(int pool, const Params &P, const Work &w, uint64_t seed, double *tally, cudaStream_t st);
cudaError_t step_kernel_regs(int stage, bool field, int *regs);
// kernels launched per iteration: 3 refill kernels + the stages of the two chains
inline int launches_per_iteration(bool field) { return 3 + 2 + (field ? 4 : 2); }
// level-1 hook: the refill index logic alone on a caller-supplied alive[] (see include/emx.h)
cudaError_t launch_refill_plan(long n_live, long capacity, long n_queue, const uint8_t *alive, int32_t *src,
                               int *scratch, const Ctl **ctl_out, cudaStream_t st);
size_t refill_plan_scratch_ints(long capacity);

}  // namespace emx
