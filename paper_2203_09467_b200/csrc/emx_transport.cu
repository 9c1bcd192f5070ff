// emx_transport.cu -- the loop kernels: primary loading, refill / compaction (A0, A9), the per-type step
// kernels (A1-A8, A10) and loop control (A12).  DESIGN.md section 5.
//
// One ITERATION = k_plan (admission + refill plan) -> k_fill -> k_move -> per pool (e+, e-, gamma):
// k_step_pool<PT> (phase A) -> k_interact<PT> (phase B).  Eight iterations and k_loop_condition form the body
// of a graph WHILE node: nothing returns to the host during a transport; pool sizes, stack tops and the done
// flag live in the device control block.
#include <cuda_runtime.h>
#include "emx_kernels.h"
#include "emx_step.h"

namespace emx {

// stack records are written once and read once: streaming stores / loads (evict-first) keep them from
// displacing the track store in L2
#ifndef EMX_STREAM_HINTS
#define EMX_STREAM_HINTS 1
#endif
#if EMX_STREAM_HINTS
#define EMX_ST(p, v) __stcs((p), (v))
#define EMX_LD(p) __ldcs((p))
#else
#define EMX_ST(p, v) (*(p) = (v))
#define EMX_LD(p) (*(p))
#endif

__device__ __forceinline__ void load_record(const QueueSoA &q, int r, const TrackSoA &t, int i) {
    t.x[i] = EMX_LD(&q.x[r]);
    t.y[i] = EMX_LD(&q.y[r]);
    t.z[i] = EMX_LD(&q.z[r]);
    t.ux[i] = EMX_LD(&q.ux[r]);
    t.uy[i] = EMX_LD(&q.uy[r]);
    t.uz[i] = EMX_LD(&q.uz[r]);
    t.E[i] = EMX_LD(&q.E[r]);
    t.tid[i] = (uint64_t)EMX_LD((const unsigned long long *)&q.tid[r]);
    t.prim[i] = EMX_LD(&q.prim[r]);
    t.step[i] = 0u;
    t.vol[i] = EMX_LD(&q.vol[r]);
    t.surf[i] = EMX_LD(&q.surf[r]);
    t.alive[i] = 2;  // 2 = filled in this refill pass (k_move still ranks it as a hole)
    if (t.fs_a) t.fs_a[i] = 0;
    if (t.pend) t.pend[i] = 0;
}

__device__ __forceinline__ void move_slot(const TrackSoA &t, int from, int to) {
    t.x[to] = t.x[from];
    t.y[to] = t.y[from];
    t.z[to] = t.z[from];
    t.ux[to] = t.ux[from];
    t.uy[to] = t.uy[from];
    t.uz[to] = t.uz[from];
    t.E[to] = t.E[from];
    t.tid[to] = t.tid[from];
    t.prim[to] = t.prim[from];
    t.step[to] = t.step[from];
    t.vol[to] = t.vol[from];
    t.surf[to] = t.surf[from];
    t.alive[to] = 2;
    if (t.pend) t.pend[to] = t.pend[from];
    if (t.fs_a) {
        t.fs_s[to] = t.fs_s[from];
        t.fs_h[to] = t.fs_h[from];
        t.fs_a[to] = t.fs_a[from];
    }
}

// Optional timeline of the iteration graph (diagnostics, -DEMX_TIMELINE): first block start / last block end
// of every kernel node, from %globaltimer, for iterations [EMX_TL_FIRST, EMX_TL_FIRST + kTlN).
#ifdef EMX_TIMELINE
#ifndef EMX_TL_FIRST
#define EMX_TL_FIRST 2500
#endif
constexpr int kTlN = 64;
__device__ unsigned long long g_tl[kTlN][9][4];  // min start, max end, sum of block times, blocks
__device__ __forceinline__ void tl_mark(const Work &w, int node, int which, int iter_off) {
    __shared__ unsigned long long s_t0;
    if (threadIdx.x != 0) return;
    const long long it = (long long)w.ctl->iter - iter_off - EMX_TL_FIRST;
    if (it < 0 || it >= kTlN) return;
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    atomicMax(&g_tl[it][node][which], which == 0 ? ~t : t);
    if (which == 0) s_t0 = t;
    else {
        atomicAdd(&g_tl[it][node][2], t - s_t0);
        atomicAdd(&g_tl[it][node][3], 1ull);
    }
}
#define EMX_TL(w, node, which, off) tl_mark(w, node, which, off)
#else
#define EMX_TL(w, node, which, off) ((void)0)
#endif

// ------------------------------------------------------------------------------------------------
// Loop start: clear the control block, total the injected energy and the primaries per type.
__global__ void __launch_bounds__(1024) k_init(Work w, Primaries pr) {
    __shared__ int s_cnt[3][32];
    __shared__ double s_E[32];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    Ctl *c = w.ctl;
    int cnt[3] = {0, 0, 0};
    double ein = 0.0;
    for (long i = tid; i < pr.n; i += blockDim.x) {
        const int pt = pr.ptype[i];
        cnt[0] += (pt == 0);
        cnt[1] += (pt == 1);
        cnt[2] += (pt == 2);
        ein += pr.E[i] + (pt == kPositron ? 2.0 * kMe : 0.0);
    }
    for (int p = 0; p < 3; ++p) {
        int v = cnt[p];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (lane == 0) s_cnt[p][wid] = v;
    }
    for (int o = 16; o > 0; o >>= 1) ein += __shfl_down_sync(0xffffffffu, ein, o);
    if (lane == 0) s_E[wid] = ein;
    __syncthreads();
    if (tid == 0) {
        Ctl z = Ctl();
        double e = 0.0;
        for (int k = 0; k < 32; ++k) e += s_E[k];
        for (int p = 0; p < 3; ++p) {
            int t = 0;
            for (int k = 0; k < 32; ++k) t += s_cnt[p][k];
            z.tracks[p] = (unsigned long long)t;
        }
        z.E_in = e;
        *c = z;
    }
    for (int p = 0; p < 3; ++p)
        for (int k = tid; k <= w.cap[p] / kChunk; k += blockDim.x) w.chunk_dead[p][k] = 0;
}

// A0, first half: admission of primaries (R8).  Done by the one block of k_plan at the start of every iteration.  While the
// shower energy in flight and the stacks are below their soft limits, the next `wave` primaries are pushed
// onto the stacks of their types, lowest index on top, so they enter the pools in ascending order at the
// refill that follows.  Histories do not depend on when a primary is admitted (keyed RNG, C2); admission only
// bounds the number of queued records (the queue had to hold 2.5e7 initializers).
__device__ __forceinline__ void admit_block(const Work &w, const Primaries &pr) {
    __shared__ int s_cnt[3][32];
    __shared__ int s_total[3], s_base[3];
    __shared__ double s_E[32];
    __shared__ int s_go;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, nw = blockDim.x >> 5;
    Ctl *c = w.ctl;
    if (c->done) return;
    const long long next = c->next_primary;
    if (next >= pr.n) return;
    const double inflight = c->E_admitted - (c->edep_total + c->escaped + c->looper);
    if (inflight >= w.inflight_cap) return;
    for (int p = 0; p < 3; ++p)
        if (4LL * c->q_top[p] >= (long long)w.qcap[p]) return;  // a stack is a quarter full: let it drain first
    const long long A = (pr.n - next) < (long long)w.wave ? (pr.n - next) : (long long)w.wave;
    // pass 1: counts per type and energy of the window
    int cnt[3] = {0, 0, 0};
    double ein = 0.0;
    for (long long k = tid; k < A; k += blockDim.x) {
        const int pt = pr.ptype[next + k];
        cnt[0] += (pt == 0);
        cnt[1] += (pt == 1);
        cnt[2] += (pt == 2);
        ein += pr.E[next + k] + (pt == kPositron ? 2.0 * kMe : 0.0);
    }
    for (int p = 0; p < 3; ++p) {
        int v = cnt[p];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (lane == 0) s_cnt[p][wid] = v;
    }
    for (int o = 16; o > 0; o >>= 1) ein += __shfl_down_sync(0xffffffffu, ein, o);
    if (lane == 0) s_E[wid] = ein;
    __syncthreads();
    if (tid == 0) {
        int go = 1;
        for (int p = 0; p < 3; ++p) {
            int t = 0;
            for (int k = 0; k < nw; ++k) t += s_cnt[p][k];
            s_total[p] = t;
            s_base[p] = 0;
            if (c->q_top[p] + t > w.qcap[p]) go = 0;  // no room: try again in a later iteration
        }
        s_go = go;
    }
    __syncthreads();
    if (!s_go) return;
    // pass 2: stable rank of each primary inside its type, tile by tile
    for (long long base = 0; base < A; base += blockDim.x) {
        const long long k = base + tid;
        const long long i = next + k;
        const int pt = (k < A) ? pr.ptype[i] : -1;
        int rank = 0;
        for (int p = 0; p < 3; ++p) {
            const unsigned b = __ballot_sync(0xffffffffu, pt == p);
            if (lane == 0) s_cnt[p][wid] = __popc(b);
            if (pt == p) rank = __popc(b & ((1u << lane) - 1u));
        }
        __syncthreads();
        if (pt >= 0) {
            int before = s_base[pt];
            for (int q = 0; q < wid; ++q) before += s_cnt[pt][q];
            const int r = c->q_top[pt] + s_total[pt] - 1 - (before + rank);  // lowest index on top
            const QueueSoA &q = w.q[pt];
            q.x[r] = pr.pos3[3 * i];
            q.y[r] = pr.pos3[3 * i + 1];
            q.z[r] = pr.pos3[3 * i + 2];
            q.ux[r] = pr.dir3[3 * i];
            q.uy[r] = pr.dir3[3 * i + 1];
            q.uz[r] = pr.dir3[3 * i + 2];
            q.E[r] = pr.E[i];
            q.tid[r] = 0ull;
            q.prim[r] = (uint32_t)(pr.first + i);
            q.vol[r] = pr.vol[i];
            q.surf[r] = pr.surf ? pr.surf[i] : -1;
        }
        __syncthreads();
        if (tid < 3) {
            int t = 0;
            for (int q = 0; q < nw; ++q) t += s_cnt[tid][q];
            s_base[tid] += t;
        }
        __syncthreads();
    }
    if (tid == 0) {
        double e = 0.0;
        for (int k = 0; k < nw; ++k) e += s_E[k];
        for (int p = 0; p < 3; ++p) c->q_top[p] += s_total[p];
        c->next_primary = next + A;
        c->E_admitted += e;
    }
}

cudaError_t launch_init(const Work &w, const Primaries &pr, cudaStream_t st) {
    k_init<<<1, 1024, 0, st>>>(w, pr);
    return cudaGetLastError();
}

constexpr int kPlanThreads = 1024;
constexpr int kPatience = 64;  // iterations without progress before the loop gives up (R7)

// ------------------------------------------------------------------------------------------------
// A9 / A12: refill plan and loop control.  One block.  Per pool: exclusive prefix sum of the per-chunk
// dead counts the step kernel left behind -> rank of every hole; then the sizes of the refill:
//   a      holes filled from the stack (hole k, ascending slot index, takes record [q - 1 - k]),
//   h - a  holes left when the stack is dry: the live range shrinks to n_new and the live tracks above
//          n_new move into the remaining holes below it (j-th live track from the end -> j-th such hole),
//   extra  records appended above the old range when the stack holds more than the holes.
__global__ void __launch_bounds__(1024) k_plan(Work w, Primaries pr) {
    constexpr int kGroupWarps = 10;  // warps 0-9 scan the gamma pool, 10-19 e-, 20-29 e+ (side by side)
    __shared__ int s_warp[3][kGroupWarps];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    Ctl *c = w.ctl;
    if (c->done) return;
    EMX_TL(w, 0, 0, 0);
    admit_block(w, pr);
    __syncthreads();
    const int p = wid / kGroupWarps, wig = wid % kGroupWarps;  // pool of this warp, warp index in its group
    if (p < 3) {
        const int gt = wig * 32 + lane;  // thread index in the group
        const int n_old = c->n_live[p];
        const int nch = (n_old + kChunk - 1) / kChunk;
        constexpr int kPer = 8;  // chunks per thread: one pass of a group covers 2560 chunks
        int carry = 0;           // dead slots before this pass (every thread of the group keeps its own copy)
        for (int base = 0; base < nch; base += kGroupWarps * 32 * kPer) {
            const int k0 = base + gt * kPer;
            int d[kPer], v = 0;
#pragma unroll
            for (int q = 0; q < kPer; ++q) {
                d[q] = (k0 + q < nch) ? w.chunk_dead[p][k0 + q] : 0;
                v += d[q];
            }
            int inc = v;  // inclusive warp scan of the per-thread sums
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += t;
            }
            if (lane == 31) s_warp[p][wig] = inc;
            asm volatile("bar.sync %0, %1;" ::"r"(p + 1), "r"(kGroupWarps * 32) : "memory");
            int before = 0, total = 0;
#pragma unroll
            for (int k = 0; k < kGroupWarps; ++k) {
                const int x = s_warp[p][k];
                before += k < wig ? x : 0;
                total += x;
            }
            int off = carry + before + inc - v;
#pragma unroll
            for (int q = 0; q < kPer; ++q) {
                if (k0 + q < nch) {
                    w.chunk_off[p][k0 + q] = off;
                    w.chunk_dead[p][k0 + q] = 0;  // the step kernels count the next iteration's deaths into it
                }
                off += d[q];
            }
            carry += total;
            asm volatile("bar.sync %0, %1;" ::"r"(p + 1), "r"(kGroupWarps * 32) : "memory");
        }
        if (gt == 0) {
            const int h = carry;
            const int q = c->q_top[p];
            const int a = h < q ? h : q;
            const int n_new = n_old - (h - a);
            int extra = 0;
            if (h == a) {
                extra = q - a;
                const int room = w.cap[p] - n_old;
                if (extra > room) extra = room;
            }
            PoolPlan pl;
            pl.n_old = n_old;
            pl.h = h;
            pl.a = a;
            pl.n_new = n_new;
            pl.extra = extra;
            pl.n_final = n_new + extra;
            pl.q_old = q;
            pl.q_new = q - a - extra;
            c->plan[p] = pl;
            c->n_live[p] = pl.n_final;
            c->q_top[p] = pl.q_new;
        }
    }
    __syncthreads();
    if (tid == 0) {
        const long long ng = c->n_live[0], ne = c->n_live[1], np = c->n_live[2];
        const long long live = ng + ne + np;
        const long long queued = (long long)c->q_top[0] + c->q_top[1] + c->q_top[2];
        // a track pushes at most 4 records in an iteration (two products and two at-rest photons): where even that
        // fits, the step kernels reserve with one atomic and no look at the top first
        for (int p = 0; p < 3; ++p) c->q_safe[p] = ((long long)c->q_top[p] + 4LL * live <= (long long)w.qcap[p]) ? 1 : 0;
        if ((unsigned long long)live > c->peak_live) c->peak_live = (unsigned long long)live;
        if ((unsigned long long)queued > c->peak_queue) c->peak_queue = (unsigned long long)queued;
        if (c->iter < (unsigned long long)w.max_log) {
            w.log[2 * c->iter] = (uint32_t)live;
            w.log[2 * c->iter + 1] = (uint32_t)queued;
        }
        if (live == 0 && c->next_primary >= w.n_primaries) {
            c->done = 1;
            c->m_step[0] = c->m_step[1] = c->m_step[2] = 0;
        } else {
            c->iter += 1;
            // R7: a step whose secondaries do not fit on the stacks is not committed and is re-executed in a
            // later iteration with the same (tid, step) and hence the same draws.  Progress = steps committed or
            // field propagations advanced; retiring a tombstone is none (stalled warps can push and retire
            // tombstones for ever).  kPatience iterations in a row without progress although tracks are live:
            // the stacks are too small for this problem
            c->m_step[0] = (int)ng;
            c->m_step[1] = (int)ne;
            c->m_step[2] = (int)np;
            EMX_TL(w, 0, 1, 1);
            c->idle_iters = (c->had_live && c->progress == 0ull) ? c->idle_iters + 1 : 0;
            if (c->idle_iters >= kPatience) {
                c->error = EMX_E_CAPACITY;
                c->done = 1;
            }
            c->had_live = live > 0 ? 1 : 0;
            // time slicing of the field propagation: with many tracks in flight a track may use only a few
            // substep attempts per iteration (the rest of its step continues next iteration), so that no warp
            // holds an iteration open for hundreds of substeps; with few tracks left latency matters more
            c->field_budget = live > w.slice_above ? w.slice_budget : 0x7fffffff;
            c->progress = 0ull;
            c->work_ctr3[0] = c->work_ctr3[1] = c->work_ctr3[2] = 0;
            c->work_ctrB[0] = c->work_ctrB[1] = c->work_ctrB[2] = 0;
            for (int a = 0; a < 3; ++a) c->icount64[a] = 0ull;
        }
    }
}

// rank of slot i among the dead slots of its chunk (exclusive), for a block that covers one chunk
__device__ __forceinline__ int rank_in_chunk(bool dead, int *s_w) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const unsigned b = __ballot_sync(0xffffffffu, dead);
    if (lane == 0) s_w[wid] = __popc(b);
    __syncthreads();
    int r = __popc(b & ((1u << lane) - 1u));
    for (int k = 0; k < wid; ++k) r += s_w[k];
    __syncthreads();
    return r;
}

constexpr int kRefillBlocks = 1184;  // per pool: 8 x 148 blocks, grid-stride over the chunks

// A0: fill holes from the stack, list the holes that are left, append records above the old range
__global__ void __launch_bounds__(kChunk) k_fill(Work w, int32_t *dbg_src) {
    __shared__ int s_w[kChunk / 32];
    const int p = blockIdx.y;
    const Ctl *c = w.ctl;
    if (c->done) return;
    const PoolPlan pl = c->plan[p];
    const int top = pl.n_old > pl.n_final ? pl.n_old : pl.n_final;
    const int nch_old = (pl.n_old + kChunk - 1) / kChunk;
    const TrackSoA &t = w.trk[p];
    EMX_TL(w, 1, 0, 1);
    for (int ch = blockIdx.x; ch * kChunk < top; ch += gridDim.x) {  // grid-stride over 128-slot chunks
        const int base = ch * kChunk;
        if (ch < nch_old && base + kChunk <= pl.n_old) {  // chunk inside the old range: skip it if nothing died
            const int d0 = w.chunk_off[p][ch];
            const int d1 = (ch + 1 < nch_old) ? w.chunk_off[p][ch + 1] : pl.h;
            if (d1 == d0) continue;
        }
        const int i = base + threadIdx.x;
        const bool dead = (i < pl.n_old) && (t.alive[i] == 0);
        const int k = w.chunk_off[p][ch < nch_old ? ch : 0] + rank_in_chunk(dead, s_w);
        if (dead) {
            if (k < pl.a) {
                const int r = pl.q_old - 1 - k;
                if (dbg_src) { dbg_src[i] = r; t.alive[i] = 2; }
                else load_record(w.q[p], r, t, i);
            } else {
                w.hole_idx[p][k - pl.a] = i;
            }
        } else if (i >= pl.n_old && i < pl.n_old + pl.extra) {
            const int r = pl.q_old - 1 - pl.a - (i - pl.n_old);
            if (dbg_src) { dbg_src[i] = r; t.alive[i] = 2; }
            else load_record(w.q[p], r, t, i);
        }
    }
    EMX_TL(w, 1, 1, 1);
}

// A9: tail compaction when the stack ran dry: live tracks at or above n_new move into the holes below it
__global__ void __launch_bounds__(kChunk) k_move(Work w, int32_t *dbg_src) {
    __shared__ int s_w[kChunk / 32];
    const int p = blockIdx.y;
    const Ctl *c = w.ctl;
    if (c->done) return;
    const PoolPlan pl = c->plan[p];
    EMX_TL(w, 2, 0, 1);
    if (pl.h == pl.a) {  // nothing to compact
        EMX_TL(w, 2, 1, 1);
        return;
    }
    const TrackSoA &t = w.trk[p];
    // grid-stride over the chunks that overlap the tail [n_new, n_old)
    for (int ch = pl.n_new / kChunk + blockIdx.x; ch * kChunk < pl.n_old; ch += gridDim.x) {
        const int i = ch * kChunk + threadIdx.x;
        const bool in = i < pl.n_old;
        const uint8_t al = in ? t.alive[i] : (uint8_t)1;
        const bool dead = al != 1;  // holes of this pass, whether k_fill has refilled them (2) or not (0)
        const int dead_before = w.chunk_off[p][ch] + rank_in_chunk(dead, s_w);
        if (in && !dead && i >= pl.n_new) {
            const int dead_after = pl.h - dead_before;      // dead slots in (i, n_old)
            const int j = (pl.n_old - 1 - i) - dead_after;  // live tracks in (i, n_old)
            const int dest = w.hole_idx[p][j];
            if (dbg_src) { dbg_src[dest] = -2 - i; t.alive[dest] = 2; }
            else move_slot(t, i, dest);
        }
    }
    EMX_TL(w, 2, 1, 1);
}

// ------------------------------------------------------------------------------------------------
// A1-A8 + A10: one step of every live track.  One PERSISTENT launch per pool and phase: the grid is a fixed
// number of 128-thread blocks (16 warps per SM: what 128 registers per thread allow) whose four warps work
// independently, each pulling 32-slot chunks of the pool from a device-side work counter until none are
// left.  A warp never waits for another warp: there is no block-wide barrier and no shared memory.  One pool per launch keeps the code of a
// single particle type in the instruction caches (a merged kernel for the three types was instruction-fetch
// bound: profiles/r1_v2_*); the three launches are parallel branches of the iteration graph.
//   per lane: the track is read once, stepped in registers (step<PT>) and written once;
//   secondaries go straight onto the typed stacks: the warp counts its records per type with ballots, one
//   lane reserves the range with one atomic per type ("atomic addition to unambiguously reserve
//   one or more items") and the lanes write consecutive records;
//   tallies: lanes that deposit into the same tally are reduced with warp shuffles and one lane issues the
//   fp64 atomic (north_star "warp-shuffle reductions for tallies"); run counters are kept in registers, one
//   counter per lane, across all chunks of the warp and flushed once at the end of the launch.
#ifndef EMX_WARPS_PER_SM
#define EMX_WARPS_PER_SM 16
#endif
constexpr int kStepWarpsPerSM = EMX_WARPS_PER_SM;
// warps of a step-kernel block are independent (no barrier, no shared memory); they are grouped four to a
// block only because block dispatch is what an idle iteration costs (~2.4 ns per block, 21 000 single-warp
// blocks per iteration = 50 us)
#ifndef EMX_STEP_BLOCK
#define EMX_STEP_BLOCK 128
#endif
constexpr int kStepBlock = EMX_STEP_BLOCK;

__device__ __forceinline__ void push_record(const QueueSoA &q, int r, const Vec3 &x, const Vec3 &u, double E,
                                            uint64_t tid, uint32_t prim, int vol) {
    EMX_ST(&q.x[r], x.x);
    EMX_ST(&q.y[r], x.y);
    EMX_ST(&q.z[r], x.z);
    EMX_ST(&q.ux[r], u.x);
    EMX_ST(&q.uy[r], u.y);
    EMX_ST(&q.uz[r], u.z);
    EMX_ST(&q.E[r], E);
    EMX_ST((unsigned long long *)&q.tid[r], (unsigned long long)tid);
    EMX_ST(&q.prim[r], prim);
    EMX_ST(&q.vol[r], vol);
    EMX_ST(&q.surf[r], -1);
}

__device__ __forceinline__ double warp_sum(double v) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// per-warp accumulators, spread over the lanes: lane k owns integer counter k (0..7 interactions by process,
// 8 null interactions, 9..11 tracks created by type, 12..14 steps by type, 15 progress, 16 stalls) and lanes
// 0..3 own the doubles escaped, below_cut, looper, deposited
struct WarpAcc {
    unsigned long long n;
    double d;
};

// Reserve `cnt` records (warp total) on stack ty; returns the base index or -1 when the stack is full.
// Far from the capacity one atomicAdd does it: kReserveSlack bounds what all resident warps of
// the three step kernels can request at the same time (one outstanding reservation of <= 96 records each), so
// the top cannot pass the capacity.  Near the capacity a small stack (tests) is reserved by compare-and-swap,
// which never moves the top past the capacity; a large stack is simply treated as full.  Nothing is ever rolled back: an add-then-subtract scheme lets a
// reservation succeed above a top that a concurrent failure has inflated, and strands its records.
constexpr int kReserveSlack = 148 * 3 * 32 * 96;

__device__ __forceinline__ int reserve(Ctl *c, const Work &w, int ty, int cnt, int lane) {
    int r0 = -1;
    if (lane == 0) {
        const int cap = w.qcap[ty];
        if (__ldg(&c->q_safe[ty])) {
            // k_plan's guarantee for this iteration: one round trip to the top instead of two
            r0 = atomicAdd(&c->q_top[ty], cnt);
        } else {
            int old = *(volatile int *)&c->q_top[ty];
            if ((long long)old + cnt + kReserveSlack <= (long long)cap) {
                r0 = atomicAdd(&c->q_top[ty], cnt);
            } else if (cap < 8 * kReserveSlack) {
                // small stack: exact accounting by compare-and-swap
                while (old + cnt <= cap) {
                    const int prev = atomicCAS(&c->q_top[ty], old, old + cnt);
                    if (prev == old) {
                        r0 = old;
                        break;
                    }
                    old = prev;
                }
            }
            // large stack within kReserveSlack of its capacity: treated as full (thousands of warps spinning on
            // one compare-and-swap cost 10x the iteration; the last 2 % of a large stack are not worth it)
        }
    }
    return __shfl_sync(0xffffffffu, r0, 0);
}

// bin of the steps-per-track histogram (include/emx.h: EMX_NHIST)
__device__ __forceinline__ int step_bin(uint32_t n) {
    int b = (int)n;
    if (n >= 16u) {
        const int e = 31 - __clz(n);
        b = 16 + 4 * (e - 4) + (int)((n >> (e - 2)) & 3u);
    }
    return b < EMX_NHIST ? b : EMX_NHIST - 1;
}

// index of process `proc` among the processes of particle type PT (the order of C7.8), and back
template <int PT>
__device__ __forceinline__ int proc_slot(int proc) {
    if (PT == kGamma) return proc == EMX_P_COMPTON ? 0 : (proc == EMX_P_PHOTO ? 1 : 2);
    if (PT == kElectron) return proc == EMX_P_MOLLER ? 0 : 1;
    return proc == EMX_P_BHABHA ? 0 : (proc == EMX_P_BREMS ? 1 : 2);
}
template <int PT>
__device__ __forceinline__ int slot_proc(int k) {
    if (PT == kGamma) return k == 0 ? EMX_P_COMPTON : (k == 1 ? EMX_P_PHOTO : EMX_P_PAIR);
    if (PT == kElectron) return k == 0 ? EMX_P_MOLLER : EMX_P_BREMS;
    return k == 0 ? EMX_P_BHABHA : (k == 1 ? EMX_P_BREMS : EMX_P_ANNIH);
}

// What both step kernels do with a lane's result: reserve and write the secondaries (A8), write the track
// back, tally (A10), count.  `pend` >= 0: the lane's step is not finished -- its interaction `pend` was
// selected and waits for k_interact; only what has happened so far (move, continuous loss) is committed.
template <int PT, bool CONSEC>
__device__ __forceinline__ WarpAcc epilogue(const Params &P, const Work &w, uint64_t seed, double *tally, int i,
                                            bool active, bool tomb, bool parked, int pend, Track &t, StepOut &o,
                                            int vol0, uint32_t step0) {
    WarpAcc acc;
    acc.n = 0ull;
    acc.d = 0.0;
    Ctl *c = w.ctl;
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    const TrackSoA &ts = w.trk[PT];
    // ---- A8: secondaries -> typed stacks.  When a stack cannot take the warp's records the lanes that needed
    // it STALL: nothing of their step is committed (R7).  Records a stalled lane did obtain
    // for another type become tombstones (E < 0), which the next refill loads and this kernel retires.
    const int ng = (o.s0.ptype == kGamma) + (o.s1.ptype == kGamma) + 2 * o.rest_alloc;
    const int ne = (o.s0.ptype == kElectron);  // only ordinal 0 is ever an electron
    const int np = (o.s1.ptype == kPositron);  // only the pair positron
    bool stall = false;
    int r_e = -1, r_p = -1, r_g = -1;
    unsigned b = __ballot_sync(0xffffffffu, ne);
    if (b) {
        const int r0 = reserve(c, w, kElectron, __popc(b), lane);
        if (ne) {
            if (r0 < 0) stall = true;
            else r_e = r0 + __popc(b & lt);
        }
    }
    if (PT == kGamma) {  // only photons make positrons
        b = __ballot_sync(0xffffffffu, np);
        if (b) {
            const int r0 = reserve(c, w, kPositron, __popc(b), lane);
            if (np) {
                if (r0 < 0) stall = true;
                else r_p = r0 + __popc(b & lt);
            }
        }
    }
    if (PT != kGamma) {  // only e+- make photons: 0..3 per lane -> inclusive warp scan of the counts
        b = __ballot_sync(0xffffffffu, ng > 0);
        if (b) {
            int inc = ng;
            for (int d = 1; d < 32; d <<= 1) {
                const int v = __shfl_up_sync(0xffffffffu, inc, d);
                if (lane >= d) inc += v;
            }
            const int r0 = reserve(c, w, kGamma, __shfl_sync(0xffffffffu, inc, 31), lane);
            if (ng) {
                if (r0 < 0) stall = true;
                else r_g = r0 + inc - ng;
            }
        }
    }
    if (stall) {
        if (r_e >= 0) w.q[kElectron].E[r_e] = -1.0;
        if (r_p >= 0) w.q[kPositron].E[r_p] = -1.0;
        if (r_g >= 0)
            for (int k = 0; k < ng; ++k) w.q[kGamma].E[r_g + k] = -1.0;
    } else {
        if (ne) push_record(w.q[kElectron], r_e, t.x, o.s0.u, o.s0.E, child_tid((uint32_t)seed, t.prim, t.tid, step0, 0u),
                            t.prim, t.vol);
        if (np) push_record(w.q[kPositron], r_p, t.x, o.s1.u, o.s1.E, child_tid((uint32_t)seed, t.prim, t.tid, step0, 1u),
                            t.prim, t.vol);
        if (ng) {
            const QueueSoA &q = w.q[kGamma];
            int r = r_g;
            if (o.s0.ptype == kGamma)
                push_record(q, r++, t.x, o.s0.u, o.s0.E, child_tid((uint32_t)seed, t.prim, t.tid, step0, 0u), t.prim, t.vol);
            if (o.s1.ptype == kGamma)
                push_record(q, r++, t.x, o.s1.u, o.s1.E, child_tid((uint32_t)seed, t.prim, t.tid, step0, 1u), t.prim, t.vol);
            if (o.rest_alloc) {
                const Vec3 mu = {-o.rest_u.x, -o.rest_u.y, -o.rest_u.z};
                push_record(q, r++, t.x, o.rest_u, kMe, child_tid((uint32_t)seed, t.prim, t.tid, step0, 2u), t.prim, t.vol);
                push_record(q, r++, t.x, mu, kMe, child_tid((uint32_t)seed, t.prim, t.tid, step0, 3u), t.prim, t.vol);
            }
        }
    }
    const bool commit = active && !tomb && !stall && !parked;

    // ---- write the track back (A5-A7 results); tid and prim never change
    if (commit) {
        ts.x[i] = t.x.x;
        ts.y[i] = t.x.y;
        ts.z[i] = t.x.z;
        ts.ux[i] = t.u.x;
        ts.uy[i] = t.u.y;
        ts.uz[i] = t.u.z;
        ts.E[i] = t.E;
        ts.step[i] = t.step;
        ts.vol[i] = t.vol;
        ts.surf[i] = t.surf;
        if (PT != kGamma) ts.fs_a[i] = 0;
        ts.pend[i] = (uint8_t)(pend >= 0 ? 1 + pend : 0);
    }
    const bool died = active && (tomb || (commit && !t.alive));
    if (active) ts.alive[i] = (uint8_t)(died ? 0 : 1);
    // steps-per-track histogram: a track that ends here took step0 + 1 steps; lanes with the same bin share
    // one atomic (most tracks end after a few steps: per-lane atomics on those few bins cost 70 % more time)
    {
        const bool ended = died && !tomb;
        const unsigned be = __ballot_sync(0xffffffffu, ended);
        if (ended) {
            const int hb = step_bin(step0 + 1u);
            const unsigned m = __match_any_sync(be, hb);
            if (lane == __ffs(m) - 1) atomicAdd(&c->hist[PT][hb], (unsigned long long)__popc(m));
        }
    }
    // dead slots per 128-slot chunk, for the refill plan (A9)
    if (CONSEC) {  // the warp's lanes are 32 consecutive slots of one chunk
        const unsigned bd = __ballot_sync(0xffffffffu, died);
        if (bd && lane == 0) atomicAdd(&w.chunk_dead[PT][i / kChunk], __popc(bd));
    } else if (died) {
        atomicAdd(&w.chunk_dead[PT][i / kChunk], 1);
    }

    // ---- A10: per-volume tally.  Lanes with the same tally id are summed with shuffles; one atomic per group.
    // (Letting the lanes of a warp that is spread over many ids add their deposits one by one saves the reductions
    // -- +2 % on configs 2 and 7 -- but serialises on the few tally addresses of configs 4 and 5: -40 %.)
    {
        const int tl = (commit && o.edep != 0.0) ? P.vol[vol0].tally : -1;
        unsigned m = __ballot_sync(0xffffffffu, tl >= 0);
        while (m) {
            const int leader = __ffs(m) - 1;
            const int key = __shfl_sync(0xffffffffu, tl, leader);
            const bool mine = (tl == key);
            const unsigned grp = __ballot_sync(0xffffffffu, mine);
            const double s = warp_sum(mine ? o.edep : 0.0);
            if (lane == leader) atomicAdd(&tally[key], s);
            m &= ~grp;
        }
    }
    // ---- run totals, accumulated in registers (lane k owns counter k)
    {
        const double e0 = commit ? o.escaped : 0.0, e1 = commit ? o.below_cut : 0.0, e2 = commit ? o.looper : 0.0,
                     e3 = commit ? o.edep : 0.0;
        // escapes, cut kills and loopers are rare: a warp reduction only for the totals that have something to add
        if (__ballot_sync(0xffffffffu, e0 != 0.0)) {
            const double s0 = warp_sum(e0);
            if (lane == 0) acc.d += s0;
        }
        if (__ballot_sync(0xffffffffu, e1 != 0.0)) {
            const double s1 = warp_sum(e1);
            if (lane == 1) acc.d += s1;
        }
        if (__ballot_sync(0xffffffffu, e2 != 0.0)) {
            const double s2 = warp_sum(e2);
            if (lane == 2) acc.d += s2;
        }
        if (__ballot_sync(0xffffffffu, e3 != 0.0)) {
            const double s3 = warp_sum(e3);
            if (lane == 3) acc.d += s3;
        }
        const int proc = (commit && o.process >= 0) ? (o.null_int ? 8 : o.process) : -1;
        unsigned add = 0;
        for (int k = 0; k < 9; ++k) {
            const unsigned cnt = __popc(__ballot_sync(0xffffffffu, proc == k));
            if (lane == k) add = cnt;
        }
        const unsigned n_rest = __popc(__ballot_sync(0xffffffffu, commit && o.rest));
        if (lane == EMX_P_REST) add += n_rest;
        const unsigned n_e = __popc(__ballot_sync(0xffffffffu, commit && ne));
        const unsigned n_p = __popc(__ballot_sync(0xffffffffu, commit && np));
        unsigned n_g = commit ? (unsigned)ng : 0u;
        for (int o2 = 16; o2 > 0; o2 >>= 1) n_g += __shfl_xor_sync(0xffffffffu, n_g, o2);
        const unsigned n_commit = __popc(__ballot_sync(0xffffffffu, commit));
        const unsigned n_done = __popc(__ballot_sync(0xffffffffu, commit && pend < 0));  // completed steps
        const unsigned n_parked = __popc(__ballot_sync(0xffffffffu, parked));
        const unsigned n_stall = __popc(__ballot_sync(0xffffffffu, active && stall));
        const unsigned n_active = __popc(__ballot_sync(0xffffffffu, active));
        if (lane == 9) add = n_g;
        if (lane == 10) add = n_e;
        if (lane == 11) add = n_p;
        if (lane == 12 + PT) add = n_done;
        if (lane == 15) add = n_commit + n_parked;
        if (lane == 16) add = n_stall;
        if (lane == 17) add = n_active;
        acc.n += add;
    }
    return acc;
}

// one pool per launch: the code of a single particle type stays resident in the instruction caches

// Phase A of a chunk: items 1-7 of C7 and the selection of the discrete process for 32 consecutive slots.
// Lanes whose step ends here (boundary, loss-limited, truncated, killed) are committed; lanes with an
// interaction pending are committed as far as they got and filed in the list of their process, so that
// k_interact runs every interactor on full warps (B:north_star "partitioned by next action").
template <int PT, bool MAP, bool EXT>
__device__ __forceinline__ WarpAcc pre_chunk(const Params &P, const Work &w, uint64_t seed, double *tally, int base,
                                             int n_live, int budget) {
    Ctl *c = w.ctl;
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    const int i = base + lane;
    const TrackSoA &ts = w.trk[PT];
    const bool active = i < n_live;
    Track t;
    StepOut o;
    int vol0 = 0;
    uint32_t step0 = 0;
    // every field of the slot is loaded up front, whether or not the lane turns out to need it (tombstone, stalled
    // interaction, no propagation in progress): one round trip to L2 instead of a chain of four dependent ones
    double E0 = 0.0;
    uint8_t pend_b = 0;
    FieldState fs;
    fs.s_done = fs.h = 0.0;
    fs.attempt = 0;
    if (active) {
        E0 = ts.E[i];
        pend_b = ts.pend[i];
        t.x = {ts.x[i], ts.y[i], ts.z[i]};
        t.u = {ts.ux[i], ts.uy[i], ts.uz[i]};
        t.tid = ts.tid[i];
        t.prim = ts.prim[i];
        t.step = ts.step[i];
        t.vol = ts.vol[i];
        t.surf = ts.surf[i];
        if (PT != kGamma) {
            fs.attempt = ts.fs_a[i];
            fs.s_done = ts.fs_s[i];
            fs.h = ts.fs_h[i];
        }
    }
    const bool tomb = active && E0 < 0.0;  // tombstone record: retire the slot without stepping
    const int pend_in = (active && !tomb) ? (int)pend_b - 1 : -1;  // interaction still waiting (stalled)
    int pend = -1;
    if (active && !tomb && pend_in < 0) {
        t.E = E0;
        t.alive = 1;
        vol0 = t.vol;
        step0 = t.step;
        pend = step_pre<PT, MAP, EXT>(P, seed, t, o, fs, budget);
        if (PT != kGamma && o.suspended) {
            // the propagation continues in the next iteration: park position, direction, surface flag and the
            // loop variables; nothing else of the step has happened yet
            ts.x[i] = t.x.x;
            ts.y[i] = t.x.y;
            ts.z[i] = t.x.z;
            ts.ux[i] = t.u.x;
            ts.uy[i] = t.u.y;
            ts.uz[i] = t.u.z;
            ts.surf[i] = t.surf;
            ts.fs_s[i] = fs.s_done;
            ts.fs_h[i] = fs.h;
            ts.fs_a[i] = fs.attempt;
            o.s0.ptype = o.s1.ptype = -1;
            o.rest_alloc = 0;
            o.process = -1;
            o.edep = o.below_cut = o.escaped = o.looper = 0.0;
            o.null_int = o.rest = 0;
            t.alive = 1;
        }
    } else {
        o.s0.ptype = o.s1.ptype = -1;
        o.rest_alloc = 0;
        o.process = -1;
        o.edep = o.below_cut = o.escaped = o.looper = 0.0;
        o.null_int = o.rest = 0;
        o.suspended = 0;
        t.alive = 1;
    }
    const bool parked = active && !tomb && (PT != kGamma) && o.suspended;
    const bool waiting = pend_in >= 0;  // nothing to do in this phase

    // file the lanes with a pending interaction (new or stalled) in the list of their process.  The three list
    // counters of a pool are packed into one 64-bit word (21 bits each; pools hold fewer than 2^21 slots, checked
    // by the host), so one atomic per warp reserves the entries of all three lists.  It is issued BEFORE the
    // epilogue and its result is used after it: the round trip to L2 runs under the epilogue's work.
    const int pk = waiting ? proc_slot<PT>(pend_in) : (pend >= 0 && !parked ? proc_slot<PT>(pend) : -1);
    const unsigned b0 = __ballot_sync(0xffffffffu, pk == 0);
    const unsigned b1 = __ballot_sync(0xffffffffu, pk == 1);
    const unsigned b2 = __ballot_sync(0xffffffffu, pk == 2);
    unsigned long long lbase = 0ull;
    if ((b0 | b1 | b2) && lane == 0)
        lbase = atomicAdd(&c->icount64[PT], (unsigned long long)__popc(b0) | ((unsigned long long)__popc(b1) << 21) |
                                               ((unsigned long long)__popc(b2) << 42));

    WarpAcc acc = epilogue<PT, true>(P, w, seed, tally, i, active && !waiting, tomb, parked, pend, t, o, vol0, step0);

    if (b0 | b1 | b2) {
        lbase = __shfl_sync(0xffffffffu, lbase, 0);
        if (pk >= 0) {
            const unsigned bk = pk == 0 ? b0 : (pk == 1 ? b1 : b2);
            const int r0 = (int)((lbase >> (21 * pk)) & 0x1fffffull);
            w.ilist[PT][pk][r0 + __popc(bk & lt)] = i;
        }
    }
    return acc;
}

// Phase B of a chunk: 32 tracks of pool PT waiting for the same interactor (list k of the pool).
template <int PT>
__device__ __forceinline__ WarpAcc interact_chunk(const Params &P, const Work &w, uint64_t seed, double *tally, int k,
                                                  int first, int n_list) {
    const int lane = threadIdx.x & 31;
    const int idx = first + lane;
    const TrackSoA &ts = w.trk[PT];
    const bool active = idx < n_list;
    const int i = active ? w.ilist[PT][k][idx] : 0;
    Track t;
    StepOut o;
    o.action = EMX_A_DISCRETE;
    o.process = -1;
    o.s0.ptype = o.s1.ptype = -1;
    o.rest_alloc = 0;
    o.edep = o.below_cut = o.escaped = o.looper = o.s = 0.0;
    o.n_draws = o.null_int = o.rest = o.suspended = 0;
    int vol0 = 0;
    uint32_t step0 = 0;
    t.alive = 1;
    if (active) {
        t.x = {ts.x[i], ts.y[i], ts.z[i]};
        t.u = {ts.ux[i], ts.uy[i], ts.uz[i]};
        t.E = ts.E[i];
        t.tid = ts.tid[i];
        t.prim = ts.prim[i];
        t.step = ts.step[i];
        t.vol = ts.vol[i];
        t.surf = -1;
        vol0 = t.vol;
        step0 = t.step;
        step_interact<PT>(P, seed, t, o, slot_proc<PT>(k));
    }
    return epilogue<PT, false>(P, w, seed, tally, i, active, false, false, -1, t, o, vol0, step0);
}

template <int PT, bool MAP, bool EXT = false>
__global__ void __launch_bounds__(kStepBlock, kStepWarpsPerSM * 32 / kStepBlock) k_step_pool(const __grid_constant__ Params P,
                                                                  const __grid_constant__ Work w, uint64_t seed,
                                                                  double *tally) {
    Ctl *c = w.ctl;
    const int lane = threadIdx.x & 31;
    const int nl = c->m_step[PT];
    const int total = (nl + 31) >> 5;
    const int budget = c->field_budget;
    EMX_TL(w, 3 + PT, 0, 1);
    WarpAcc acc;
    acc.n = 0ull;
    acc.d = 0.0;
    int k_next = 0;
    if (lane == 0) k_next = atomicAdd(&c->work_ctr3[PT], 1);
    for (;;) {
        const int k = __shfl_sync(0xffffffffu, k_next, 0);
        if (k >= total) break;
        if (lane == 0) k_next = atomicAdd(&c->work_ctr3[PT], 1);
        const WarpAcc d = pre_chunk<PT, MAP, EXT>(P, w, seed, tally, k << 5, nl, budget);
        acc.n += d.n;
        acc.d += d.d;
    }
    if (acc.n) {
        unsigned long long *dst = lane < 8    ? &c->inter[lane]
                                  : lane == 8 ? &c->null_int
                                  : lane < 12 ? &c->tracks[lane - 9]
                                  : lane < 15 ? &c->steps[lane - 12]
                                  : lane == 15 ? &c->progress
                                               : &c->stalls;
        if (lane <= 16) atomicAdd(dst, acc.n);
        if (lane == 17) atomicAdd(&c->lanes[0][PT], acc.n);
    }
    EMX_TL(w, 3 + PT, 1, 1);
    if (acc.d != 0.0 && lane < 4) {
        double *dst = lane == 0 ? &c->escaped : lane == 1 ? &c->below_cut : lane == 2 ? &c->looper : &c->edep_total;
        atomicAdd(dst, acc.d);
    }
}

// Phase B: the interactors.  Persistent single-warp blocks pull 32-entry chunks of the pool's process lists;
// a warp runs ONE interactor on (up to) 32 tracks that all selected it.
#ifndef EMX_WARPS_B
#define EMX_WARPS_B EMX_WARPS_PER_SM
#endif
template <int PT>
__global__ void __launch_bounds__(kStepBlock, EMX_WARPS_B * 32 / kStepBlock) k_interact(const __grid_constant__ Params P,
                                                                 const __grid_constant__ Work w, uint64_t seed,
                                                                 double *tally) {
    Ctl *c = w.ctl;
    const int lane = threadIdx.x & 31;
    constexpr int nk = (PT == kElectron) ? 2 : 3;
    // order in which the lists are worked off.  The stacks are LIFO, so what is pushed LAST is refilled
    // first: photons run pair production first (its leptons are the most energetic secondaries and go to the
    // bottom of this iteration's records) and photoelectric absorption last.  Keeping low-energy tracks on top
    // is what keeps the queue short ("preferentially selecting lower-energy particles").
    const int ord0 = (PT == kGamma) ? 2 : 0, ord1 = (PT == kGamma) ? 0 : 1, ord2 = (PT == kGamma) ? 1 : 2;
    int n[3], cb[4];
    cb[0] = 0;
    const unsigned long long packed = c->icount64[PT];
    n[0] = (int)((packed >> (21 * ord0)) & 0x1fffffull);
    n[1] = (int)((packed >> (21 * ord1)) & 0x1fffffull);
    n[2] = ord2 < nk ? (int)((packed >> (21 * ord2)) & 0x1fffffull) : 0;
#pragma unroll
    for (int k = 0; k < 3; ++k) cb[k + 1] = cb[k] + ((n[k] + 31) >> 5);
    const int total = cb[3];
    EMX_TL(w, 6 + PT, 0, 1);
    WarpAcc acc;
    acc.n = 0ull;
    acc.d = 0.0;
    int k_next = 0;
    if (lane == 0 && total > 0) k_next = atomicAdd(&c->work_ctrB[PT], 1);
    for (;;) {
        const int ch = __shfl_sync(0xffffffffu, k_next, 0);
        if (ch >= total) break;
        if (lane == 0) k_next = atomicAdd(&c->work_ctrB[PT], 1);
        // one call site: the interactor code exists once per kernel
        const int sel = ch < cb[1] ? 0 : (ch < cb[2] ? 1 : 2);
        const int kk = sel == 0 ? ord0 : (sel == 1 ? ord1 : ord2);
        const WarpAcc d = interact_chunk<PT>(P, w, seed, tally, kk, (ch - cb[sel]) << 5, n[sel]);
        acc.n += d.n;
        acc.d += d.d;
    }
    if (acc.n) {
        unsigned long long *dst = lane < 8    ? &c->inter[lane]
                                  : lane == 8 ? &c->null_int
                                  : lane < 12 ? &c->tracks[lane - 9]
                                  : lane < 15 ? &c->steps[lane - 12]
                                  : lane == 15 ? &c->progress
                                               : &c->stalls;
        if (lane <= 16) atomicAdd(dst, acc.n);
        if (lane == 17) atomicAdd(&c->lanes[1][PT], acc.n);
    }
    EMX_TL(w, 6 + PT, 1, 1);
    if (acc.d != 0.0 && lane < 4) {
        double *dst = lane == 0 ? &c->escaped : lane == 1 ? &c->below_cut : lane == 2 ? &c->looper : &c->edep_total;
        atomicAdd(dst, acc.d);
    }
}

#ifdef EMX_TIMELINE
extern "C" int emx_debug_timeline(unsigned long long *host, int clear) {
    if (clear) {
        void *a = nullptr;
        cudaGetSymbolAddress(&a, g_tl);
        return (int)cudaMemset(a, 0, sizeof(g_tl));
    }
    return (int)cudaMemcpyFromSymbol(host, g_tl, sizeof(g_tl));
}
#endif

// phase A of a charged pool: the instantiation for the kind of field set on the problem, with or without the
// condensed-history extensions (multiple scattering, energy-loss fluctuations)
template <int PT>
static void launch_phase_a(const Params &P, const Work &w, uint64_t seed, double *tally, int g, cudaStream_t st) {
    if (!P.ph.msc && !P.ph.fluct) {
        if (P.field_kind == 0) k_step_pool<PT, false><<<g, kStepBlock, 0, st>>>(P, w, seed, tally);
        else k_step_pool<PT, true><<<g, kStepBlock, 0, st>>>(P, w, seed, tally);
    } else {
        if (P.field_kind == 0) k_step_pool<PT, false, true><<<g, kStepBlock, 0, st>>>(P, w, seed, tally);
        else k_step_pool<PT, true, true><<<g, kStepBlock, 0, st>>>(P, w, seed, tally);
    }
}

cudaError_t launch_refill(const Work &w, const Primaries &pr, cudaStream_t st) {
    k_plan<<<1, kPlanThreads, 0, st>>>(w, pr);
    const dim3 g3(kRefillBlocks, 3);
    k_fill<<<g3, kChunk, 0, st>>>(w, nullptr);
    k_move<<<g3, kChunk, 0, st>>>(w, nullptr);
    return cudaGetLastError();
}

// A12 when the loop is a graph WHILE node: after the last iteration of the body, continue unless done
__global__ void k_loop_condition(Work w, cudaGraphConditionalHandle handle) {
    cudaGraphSetConditional(handle, w.ctl->done ? 0u : 1u);
}
cudaError_t launch_loop_condition(const Work &w, unsigned long long handle, cudaStream_t st) {
    k_loop_condition<<<1, 1, 0, st>>>(w, (cudaGraphConditionalHandle)handle);
    return cudaGetLastError();
}

cudaError_t launch_step_pool(int pt, const Params &P, const Work &w, uint64_t seed, double *tally, int n_sm,
                             cudaStream_t st);

// blocks of a pool's persistent step kernels: warps_per_sm warps per SM, which pull chunks until the pool is done
static int step_grid(const Work &w, int pt, int n_sm) {
    return n_sm * (w.warps_per_sm[pt] > 0 ? w.warps_per_sm[pt] : kStepWarpsPerSM) * 32 / kStepBlock;
}

cudaError_t launch_step(const Params &P, const Work &w, uint64_t seed, double *tally, int n_sm, cudaStream_t st) {
    for (int pt = 2; pt >= 0; --pt) {
        const cudaError_t e = launch_step_pool(pt, P, w, seed, tally, n_sm, st);
        if (e != cudaSuccess) return e;
    }
    return cudaGetLastError();
}

// one phase of one pool (profiling path: every kernel bracketed by events)
cudaError_t launch_phase(int pt, int phase, const Params &P, const Work &w, uint64_t seed, double *tally, int n_sm,
                         cudaStream_t st) {
    const int g = step_grid(w, pt, n_sm);
    if (phase == 0) {
        if (pt == kGamma) k_step_pool<kGamma, false><<<g, kStepBlock, 0, st>>>(P, w, seed, tally);
        else if (pt == kElectron) launch_phase_a<kElectron>(P, w, seed, tally, g, st);
        else launch_phase_a<kPositron>(P, w, seed, tally, g, st);
    } else {
        if (pt == kGamma) k_interact<kGamma><<<g, kStepBlock, 0, st>>>(P, w, seed, tally);
        else if (pt == kElectron) k_interact<kElectron><<<g, kStepBlock, 0, st>>>(P, w, seed, tally);
        else k_interact<kPositron><<<g, kStepBlock, 0, st>>>(P, w, seed, tally);
    }
    return cudaGetLastError();
}

// the step kernels of one pool on its own stream (fork / join branches of the iteration graph)
cudaError_t launch_step_pool(int pt, const Params &P, const Work &w, uint64_t seed, double *tally, int n_sm,
                             cudaStream_t st) {
    // persistent single-warp blocks per SM for this pool: the three pools' kernels run side by side, so each
    // gets a share of the 16 warps per SM that fit
    const int g = step_grid(w, pt, n_sm);
    if (pt == kGamma) {
        k_step_pool<kGamma, false><<<g, kStepBlock, 0, st>>>(P, w, seed, tally);
        k_interact<kGamma><<<g, kStepBlock, 0, st>>>(P, w, seed, tally);
    } else if (pt == kElectron) {
        launch_phase_a<kElectron>(P, w, seed, tally, g, st);
        k_interact<kElectron><<<g, kStepBlock, 0, st>>>(P, w, seed, tally);
    } else {
        launch_phase_a<kPositron>(P, w, seed, tally, g, st);
        k_interact<kPositron><<<g, kStepBlock, 0, st>>>(P, w, seed, tally);
    }
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// level-1 hook: the refill index logic (k_plan, k_fill, k_move) on a caller-supplied alive[] array
__global__ void k_hook_init(Work w, int n_live, int n_queue) {
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        Ctl z = Ctl();
        z.n_live[0] = n_live;
        z.q_top[0] = n_queue;
        *w.ctl = z;
    }
}
__global__ void __launch_bounds__(kChunk) k_count_dead(Work w, int n_live) {
    const int i = blockIdx.x * kChunk + threadIdx.x;
    const int n = __syncthreads_count(i < n_live && w.trk[0].alive[i] == 0);
    if (threadIdx.x == 0) w.chunk_dead[0][blockIdx.x] = n;
}

size_t refill_plan_scratch_ints(long capacity) {
    const size_t nch = (size_t)(capacity + kChunk - 1) / kChunk + 1;
    return 2 * nch + (size_t)capacity + (sizeof(Ctl) + 3) / 4 + 64 + ((size_t)capacity + 3) / 4 + 64;
}

cudaError_t launch_refill_plan(long n_live, long capacity, long n_queue, const uint8_t *alive, int32_t *src,
                               int *scratch, cudaStream_t st) {
    const size_t nch = (size_t)(capacity + kChunk - 1) / kChunk + 1;
    Work w = Work();
    int *p = scratch;
    w.chunk_dead[0] = p; p += nch;
    w.chunk_off[0] = p; p += nch;
    w.hole_idx[0] = p; p += capacity;
    p += (16 - ((uintptr_t)p / 4) % 16) % 16;  // 64-byte alignment for the control block
    w.ctl = (Ctl *)p; p += (sizeof(Ctl) + 3) / 4;
    w.trk[0].alive = (uint8_t *)p;
    w.cap[0] = (int)capacity;
    w.cap[1] = w.cap[2] = 0;
    w.qcap[0] = w.qcap[1] = w.qcap[2] = 0x7fffffff;
    w.log = nullptr;
    w.max_log = 0;
    w.n_primaries = 0;
    cudaMemsetAsync(w.trk[0].alive, 0, (size_t)capacity, st);
    if (n_live > 0) cudaMemcpyAsync(w.trk[0].alive, alive, (size_t)n_live, cudaMemcpyDeviceToDevice, st);
    cudaMemsetAsync(src, 0xFF, (size_t)capacity * sizeof(int32_t), st);
    k_hook_init<<<1, 32, 0, st>>>(w, (int)n_live, (int)n_queue);
    const unsigned g = (unsigned)((n_live + kChunk - 1) / kChunk);
    if (g) k_count_dead<<<g, kChunk, 0, st>>>(w, (int)n_live);
    Primaries none = Primaries();
    k_plan<<<1, 1024, 0, st>>>(w, none);
    const dim3 g3(kRefillBlocks, 1);
    k_fill<<<g3, kChunk, 0, st>>>(w, src);
    k_move<<<g3, kChunk, 0, st>>>(w, src);
    return cudaGetLastError();
}

}  // namespace emx
