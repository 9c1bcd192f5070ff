// emx_work.h -- layout of the caller-provided device workspace: the SoA track store ("state" in the paper's
// params/state split), the secondary stacks ("stack allocator", PAPER.md:204
// "track initializers"), and the loop's control block.  DESIGN.md section 5.
//
// Two POOLS share one physical store: photons, and e- / e+ ("charged": the two differ in the sign of the
// curvature, in which tables they read and in the rest-mass bookkeeping, not in the shape of their step).  A
// track never changes pool, so each pool is stepped by kernels instantiated for it -- the pool is the coarsest
// "next action", and partitioning by it removes the largest source of warp divergence.  The store is cut into
// chunks of 128 slots; a pool OWNS a set of chunks through its chunk table (pool-local chunk -> physical chunk)
// and k_plan moves free chunks to the pool that needs them, so the split of the slots follows the live mix of
// the workload by itself.  In pool-local numbering the live tracks always occupy the dense prefix [0, n_live):
// the refill fills holes from the pool's LIFO stack and, when the stack runs dry, from the tail of the pool, so
// every access of a warp is a coalesced 16-byte-per-lane stream inside one chunk.
#pragma once
#include <cuda_runtime.h>
#include <cstddef>
#include "emx_core.h"

namespace emx {

constexpr int kChunk = 128;  // slots per chunk (and per thread block of the refill kernels)
constexpr int kPools = 2;
enum : int { kPoolGamma = 0, kPoolCharged = 1 };
EMX_HD int pool_of(int ptype) { return ptype == kGamma ? kPoolGamma : kPoolCharged; }

// where a live track is in its step
enum : int {
    kStFresh = 0,   // needs limits (stage a0)
    kStParked = 2,  // charged pool in a field: limits known, propagation not started or in progress
    kStMoved = 3,   // move done, needs stage a2
    kStPend = 8     // + process id: interaction selected, waits for the interactor (or stalled on a full stack)
};

// Track store, indexed by PHYSICAL slot.  Fields that are read and written together share a 16-byte word, so a
// lane moves its slot with five vector accesses: (x, y), (z, ux), (uy, uz), (E, track id), (prim, step, vol, surf).
struct Store {
    double2 *xy, *zu, *uu;
    double2 *Et;  // .x = E (MeV), .y = the 64 bits of the track id
    int4 *id;     // .x prim, .y step, .z vol, .w surf
    uint8_t *alive;  // 0 dead, 1 alive, 2 filled / moved in this refill pass
    uint8_t *stage;  // kSt*
    uint8_t *ptype;  // charged pool: kElectron / kPositron
    uint8_t *act;    // EMX_A_* of the current step (from stage a0, overridden by the move), or kActCut
    // the move of the current step: step limit of the physics; arc length done (after the move: path travelled);
    // trial step of the propagation; substep attempts used (after the move: surface hit, -1 none)
    double *s_phys, *s_done, *h_try;
    int *att;
    double *kap;     // curvature of the current step (sign of the charge and of an axis-aligned field folded in)
};

// secondary / primary initializer record (80 bytes): same packing, .id = (prim, vol, surf, ptype)
struct Stack {
    double2 *xy, *zu, *uu, *Et;
    int4 *id;
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

constexpr int kMaxLists = 4;  // interaction lists per pool: gamma Compton / photo / pair; charged Moller / Bhabha / brems / annihilation

struct Ctl {
    int n_live[kPools];
    int q_top[kPools];   // records on each stack; the pair is also updated as ONE 64-bit word (8-byte aligned here)
    int m_step[kPools];  // tracks to step this iteration (= n_live)
    int q_safe[kPools];  // set by k_plan: stack p cannot overflow in this iteration whatever the step kernels push
    PoolPlan plan[kPools];
    int owned[kPools];   // chunks in each pool's chunk table
    int n_free;          // chunks on the free list
    int done, error, had_live;
    int idle_iters;      // consecutive iterations without progress although tracks are live (R7)
    int work_f;          // next slot of the charged pool for the propagation kernel (the dense kernels stride)
    int icount[kPools][kMaxLists];  // entries in the interaction lists
    int field_min;       // substep attempts a track is given per iteration before it may be parked
    unsigned long long iter;
    unsigned long long progress;  // steps committed + propagations advanced in the current iteration (R7)
    long long next_primary;       // primaries [0, next_primary) have been admitted
    double E_admitted;            // energy of the admitted primaries (e+ with their 2 me)
    double edep_total;            // all energy deposited so far (every cell, tallied or not)
    double escaped, below_cut, looper, E_in;
    unsigned long long peak_live, peak_queue;
    // ---- everything above is the loop state k_plan works on (it copies it to shared memory and back: kCtlHead);
    // below are run totals that only the step kernels add to
    unsigned long long steps[3], tracks[3], inter[EMX_NPROC], null_int, stalls;
    unsigned long long lanes[4][kPools];  // slots processed by the kernels a0 / field / a (or a2) / b, per pool
    unsigned long long attempts;          // substep attempts of the field propagation
    unsigned long long hist[3][EMX_NHIST];  // tracks by type and by the bin of the steps they took
};

constexpr size_t kCtlHead = offsetof(Ctl, steps);  // bytes of the loop state at the start of Ctl (a multiple of 8)

struct Work {
    Store st;
    Stack q;              // ONE arena for both stacks: photons grow up from record 0, e+- down from the last record
    int n_chunks;         // physical chunks of the store
    int qtotal;           // records in the arena (what the two stacks may hold together)
    int *ctab[kPools];    // chunk tables, n_chunks entries each
    int *free_list;       // n_chunks entries
    int *rtab;            // physical chunk -> its index in the owning pool's chunk table
    int *chunk_dead[kPools];  // per pool-local chunk: slots that died in the last iteration
    int *chunk_off[kPools];   // ... exclusive prefix sum of it
    int *hole_idx[kPools];
    int *ilist[kPools][kMaxLists];  // PHYSICAL slots waiting for an interactor, n_slots entries each
    Ctl *ctl;
    uint32_t *log;  // per iteration: live, queued
    int max_log;
    // admission of primaries (R8): up to `wave` primaries enter per iteration while the energy in
    // flight (admitted - deposited - escaped) is below inflight_cap, fewer than admit_below records are queued and
    // the arena is less than a quarter full
    long long n_primaries;
    int wave;
    long long admit_below;  // no primaries are admitted while this many records are queued
    double inflight_cap;
    long long slice_above;  // live tracks above which the field propagation is time-sliced
    int slice_min;          // substep attempts per track and iteration before parking while sliced
    int slice_max;          // ... after which a track is parked even if the pool still has work
    int grid[8];            // blocks of the persistent step kernels, by stage (emx_kernels.h: kStage*)
    int reserve_slack;      // records all resident warps can request at the same time (see reserve())
    int slot_cap;           // slots a pool may hold at most (= n_chunks * kChunk; smaller in the refill hook)
    int stage_faces;        // shared-memory staging switches (emx_schedule entry 7): bit 0 the face table in k_field, bit 1
                            // the photon tables in k_a<gamma>
    int pool_reserve;       // chunks a pool never takes, so that the other pool can always start (n_chunks / 32, >= 1)
};

// record r (counted from the bottom of its stack) of pool's stack in the shared arena
__device__ __forceinline__ int qrec(const Work &w, int pool, int r) { return pool == kPoolGamma ? r : w.qtotal - 1 - r; }

// physical slot of pool-local slot i
__device__ __forceinline__ int phys_slot(const Work &w, int pool, int i) {
    return (w.ctab[pool][i / kChunk] * kChunk) | (i % kChunk);
}

// bytes of one slot / one record, for the roofline arithmetic
constexpr size_t kSlotBytes = 5 * 16 + 4;   // + 28 B of propagation state in the charged pool
constexpr size_t kRecordBytes = 5 * 16;

}  // namespace emx
