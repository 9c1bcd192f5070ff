// emx_work.h -- layout of the caller-provided device workspace: the SoA track store ("state" in the paper's
// params/state split), the secondary stacks ("stack allocator", PAPER.md:204
// "track initializers"), and the loop's control block.  DESIGN.md section 5.
//
// The store is split into one POOL per particle type (gamma, e-, e+): a track never changes type, so each
// pool is stepped by a kernel instantiated for that type -- particle type is the coarsest "next action"
// and partitioning by it removes the largest source of warp divergence.  Inside a pool the live tracks
// always occupy the dense prefix [0, n_live): the refill pass fills holes from the pool's LIFO stack and,
// when the stack runs dry, from the tail of the pool, so every field access is a coalesced 8-byte stream.
#pragma once
#include "emx_core.h"

namespace emx {

constexpr int kChunk = 128;  // slots per thread block of the step / refill kernels

struct TrackSoA {
    double *x, *y, *z, *ux, *uy, *uz, *E;
    uint64_t *tid;
    uint32_t *prim, *step;
    int *vol, *surf;
    uint8_t *alive;
    uint8_t *pend;  // 0, or 1 + process id of the interaction selected by phase A and not yet run
    // field propagation in progress (charged pools only; null for gamma): arc length done, trial step,
    // substep attempts used (0 = none in progress)
    double *fs_s, *fs_h;
    int *fs_a;
};

struct QueueSoA {  // secondary / primary initializer records (76 B per record)
    double *x, *y, *z, *ux, *uy, *uz, *E;
    uint64_t *tid;
    uint32_t *prim;
    int *vol, *surf;
};

struct PoolPlan {
    int n_old;    // live range before the refill
    int h;        // holes (dead slots) in [0, n_old)
    int a;        // holes filled from the stack
    int n_new;    // live range after tail compaction
    int extra;    // records appended beyond n_old
    int n_final;  // live range after the refill
    int q_old, q_new;
};

struct Ctl {
    int n_live[3];
    int q_top[3];
    int m_step[3];  // tracks to step this iteration (= n_live)
    int q_safe[3];  // set by k_plan: stack p cannot overflow in this iteration whatever the step kernels push
    PoolPlan plan[3];
    int done, error, had_live;
    int idle_iters;  // consecutive iterations without progress although tracks are live (R7)
    int work_ctr3[3];  // next 32-slot chunk of each pool's step kernel (phase A)
    int work_ctrB[3];  // next 32-entry chunk of each pool's interaction lists (phase B)
    unsigned long long icount64[3];  // entries in the interaction lists of each pool, 3 x 21 bits packed
    int field_budget;  // substep attempts per track and iteration (time slicing of the field propagation)
    unsigned long long iter;
    unsigned long long progress;  // steps committed + tombstones retired in the current iteration (R7)
    long long next_primary;       // primaries [0, next_primary) have been admitted
    double E_admitted;            // energy of the admitted primaries (e+ with their 2 me)
    double edep_total;            // all energy deposited so far (every cell, tallied or not)
    double escaped, below_cut, looper, E_in;
    unsigned long long steps[3], tracks[3], inter[EMX_NPROC], null_int, stalls, peak_live, peak_queue;
    unsigned long long lanes[2][3];  // track slots processed by phase A / phase B kernels, per pool
    unsigned long long hist[3][EMX_NHIST];  // tracks by type and by the bin of the steps they took
};

struct Work {
    TrackSoA trk[3];
    QueueSoA q[3];
    int cap[3];   // slots per pool
    int qcap[3];  // records per stack
    int *chunk_dead[3];
    int *chunk_off[3];
    int *hole_idx[3];
    int *ilist[3][3];  // slots waiting for an interactor, [pool][process slot], capacity cap[pool] each
    Ctl *ctl;
    uint32_t *log;  // per iteration: live, queued
    int max_log;
    // admission of primaries (R8): up to `wave` primaries enter per iteration while the energy in
    // flight (admitted - deposited - escaped) is below inflight_cap and no stack is more than a quarter full
    long long n_primaries;
    int wave;
    double inflight_cap;
    size_t hot_bytes;       // leading part of the workspace that holds the track store, scan arrays and lists
    int warps_per_sm[3];    // persistent step-kernel warps per SM, per pool
    long long slice_above;  // live tracks above which the field propagation is time-sliced
    int slice_budget;       // substep attempts per track and iteration while sliced
};

// bytes of one slot / one record, for the workspace carve-up and the roofline arithmetic
constexpr size_t kSlotBytes = 7 * 8 + 8 + 4 + 4 + 4 + 4 + 1;  // + 20 B in the charged pools (field progress)
constexpr size_t kRecordBytes = 7 * 8 + 8 + 4 + 4 + 4;

}  // namespace emx
