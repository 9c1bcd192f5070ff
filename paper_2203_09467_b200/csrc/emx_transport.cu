// emx_transport.cu -- the loop kernels: primary loading, refill / compaction (A0, A9), the step kernels
// (A1-A8, A10) and loop control (A12).  DESIGN.md section 5.
//
// One ITERATION = k_plan (admission, refill plan, chunk trading) -> k_fill -> k_move -> per pool
//   photons:          k_a<gamma>  (limits + straight move + finish)                        -> k_b<gamma>
//   e+-, no field:    k_a<charged>                                                        -> k_b<charged>
//   e+-, in a field:  k_a0 (limits) -> k_field (adaptive RK4, lanes refilled) -> k_a2 (finish) -> k_b<charged>
// The two pools' chains are parallel branches of the iteration graph.  Eight iterations and k_loop_condition form
// the body of a graph WHILE node: nothing returns to the host during a transport; pool sizes, stack tops and
// the done flag live in the device control block.
#include <cuda_runtime.h>
#include "emx_kernels.h"
#include "emx_step.h"
#include "emx_diag.h"

namespace emx {

// stack records are written once and read once: streaming stores / loads (evict-first) keep them from
// displacing the track store in L2
__device__ __forceinline__ void st_cs(double2 *p, double2 v) { __stcs(p, v); }
__device__ __forceinline__ void st_cs(int4 *p, int4 v) { __stcs(p, v); }
__device__ __forceinline__ double2 ld_cs(const double2 *p) { return __ldcs(p); }
__device__ __forceinline__ int4 ld_cs(const int4 *p) { return __ldcs(p); }

__device__ __forceinline__ double2 pack_Et(double E, uint64_t tid) { return make_double2(E, __longlong_as_double((long long)tid)); }
__device__ __forceinline__ uint64_t tid_of(double2 Et) { return (uint64_t)__double_as_longlong(Et.y); }

// A0: record r of stack `pool` becomes the track in physical slot s
template <int POOL>
__device__ __forceinline__ void load_record(const Work &w, int r_stack, int s) {
    const Stack &q = w.q;
    const int r = qrec(w, POOL, r_stack);
    const Store &t = w.st;
    t.xy[s] = ld_cs(&q.xy[r]);
    t.zu[s] = ld_cs(&q.zu[r]);
    t.uu[s] = ld_cs(&q.uu[r]);
    t.Et[s] = ld_cs(&q.Et[r]);
    const int4 id = ld_cs(&q.id[r]);  // prim, vol, surf, ptype
    t.id[s] = make_int4(id.x, 0, id.y, id.z);
    if (POOL == kPoolCharged) t.ptype[s] = (uint8_t)id.w;
    t.alive[s] = 2;  // 2 = filled in this refill pass (k_move still ranks it as a hole)
    t.stage[s] = kStFresh;
}

template <int POOL>
__device__ __forceinline__ void move_slot(const Work &w, int from, int to) {
    const Store &t = w.st;
    t.xy[to] = t.xy[from];
    t.zu[to] = t.zu[from];
    t.uu[to] = t.uu[from];
    t.Et[to] = t.Et[from];
    t.id[to] = t.id[from];
    t.stage[to] = t.stage[from];
    t.alive[to] = 2;
    if (POOL == kPoolCharged) {  // a propagation may be parked in the slot
        t.ptype[to] = t.ptype[from];
        t.act[to] = t.act[from];
        t.s_phys[to] = t.s_phys[from];
        t.s_done[to] = t.s_done[from];
        t.h_try[to] = t.h_try[from];
        t.att[to] = t.att[from];
        t.kap[to] = t.kap[from];
    }
}

// ------------------------------------------------------------------------------------------------
// Loop start: clear the control block, total the injected energy and the primaries per type, hand every
// chunk of the store to the free list.
__global__ void __launch_bounds__(1024) k_init(Work w, Primaries pr) {
    __shared__ int s_cnt[3][32];
    __shared__ double s_E[32];
    __shared__ int s_bad;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    Ctl *c = w.ctl;
    if (tid == 0) s_bad = 0;
    __syncthreads();
    int cnt[3] = {0, 0, 0};
    double ein = 0.0;
    for (long i = tid; i < pr.n; i += blockDim.x) {
        const int pt = pr.ptype[i];
        if (pt < 0 || pt > 2) s_bad = 1;
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
        z.n_free = w.n_chunks;
        if (s_bad) {  // a particle code outside 0..2: nothing is transported
            z.error = EMX_E_ARG;
            z.done = 1;
        }
        *c = z;
    }
    for (int k = tid; k < w.n_chunks; k += blockDim.x) w.free_list[k] = w.n_chunks - 1 - k;  // chunk 0 on top
    for (int p = 0; p < kPools; ++p)
        for (int k = tid; k <= w.n_chunks; k += blockDim.x) w.chunk_dead[p][k] = 0;
}

// A0, first half: admission of primaries (R8).  Done by the one block of k_plan at the start of every iteration.  While the
// shower energy in flight and the stacks are below their soft limits, the next `wave` primaries are pushed
// onto the stacks of their pools, lowest index on top, so they enter the pools in ascending order at the
// refill that follows.  Histories do not depend on when a primary is admitted (keyed RNG, C2); admission only
// bounds the number of queued records (the queue had to hold 2.5e7 initializers).
// Returns (to every thread) the number of primaries admitted.
__device__ __forceinline__ int admit_block(const Work &w, const Primaries &pr, Ctl *c) {
    __shared__ int s_cnt[kPools][32];
    __shared__ int s_total[kPools], s_base[kPools];
    __shared__ double s_E[32];
    __shared__ long long s_A;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, nw = blockDim.x >> 5;
    if (c->done) return 0;
    const long long next = c->next_primary;
    if (next >= pr.n) return 0;
    const double inflight = c->E_admitted - (c->edep_total + c->escaped + c->looper);
    if (inflight >= w.inflight_cap) return 0;
    long long A = (pr.n - next) < (long long)w.wave ? (pr.n - next) : (long long)w.wave;
    {
        const long long queued = (long long)c->q_top[0] + c->q_top[1];
        if (queued > 0 && 4LL * queued >= (long long)w.qtotal) return 0;  // the arena is a quarter full: let it drain first
        if (queued >= w.admit_below) return 0;  // enough records wait to keep every slot busy: more would only sit in HBM
        const long long room = (long long)w.qtotal - queued;
        if (A > room) A = room;  // a wave never asks for more than the arena can hold
    }
    if (A <= 0) return 0;
    // pass 1: energy of the window and its primaries per pool
    int cnt[kPools] = {0, 0};
    double ein = 0.0;
    for (long long k = tid; k < A; k += blockDim.x) {
        const int pt = pr.ptype[next + k];
        cnt[pool_of(pt)] += 1;
        ein += pr.E[next + k] + (pt == kPositron ? 2.0 * kMe : 0.0);
    }
    for (int p = 0; p < kPools; ++p) {
        int v = cnt[p];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (lane == 0) s_cnt[p][wid] = v;
    }
    for (int o = 16; o > 0; o >>= 1) ein += __shfl_down_sync(0xffffffffu, ein, o);
    if (lane == 0) s_E[wid] = ein;
    __syncthreads();
    if (tid == 0) {
        for (int p = 0; p < kPools; ++p) {
            int t = 0;
            for (int k = 0; k < nw; ++k) t += s_cnt[p][k];
            s_total[p] = t;
            s_base[p] = 0;
        }
        s_A = A;
    }
    __syncthreads();
    // pass 2: stable rank of each primary inside its pool, tile by tile
    for (long long base = 0; base < A; base += blockDim.x) {
        const long long k = base + tid;
        const long long i = next + k;
        const int pt = (k < A) ? pr.ptype[i] : -1;
        const int pl = pt >= 0 ? pool_of(pt) : -1;
        int rank = 0;
        for (int p = 0; p < kPools; ++p) {
            const unsigned b = __ballot_sync(0xffffffffu, pl == p);
            if (lane == 0) s_cnt[p][wid] = __popc(b);
            if (pl == p) rank = __popc(b & ((1u << lane) - 1u));
        }
        __syncthreads();
        if (pl >= 0) {
            int before = s_base[pl];
            for (int q = 0; q < wid; ++q) before += s_cnt[pl][q];
            const int r = qrec(w, pl, c->q_top[pl] + s_total[pl] - 1 - (before + rank));  // lowest index on top
            const Stack &q = w.q;
            q.xy[r] = make_double2(pr.pos3[3 * i], pr.pos3[3 * i + 1]);
            q.zu[r] = make_double2(pr.pos3[3 * i + 2], pr.dir3[3 * i]);
            q.uu[r] = make_double2(pr.dir3[3 * i + 1], pr.dir3[3 * i + 2]);
            q.Et[r] = pack_Et(pr.E[i], 0ull);
            q.id[r] = make_int4((int)(uint32_t)(pr.first + i), pr.vol[i], pr.surf ? pr.surf[i] : -1, pt);
        }
        __syncthreads();
        if (tid < kPools) {
            int t = 0;
            for (int q = 0; q < nw; ++q) t += s_cnt[tid][q];
            s_base[tid] += t;
        }
        __syncthreads();
    }
    if (tid == 0) {
        double e = 0.0;
        for (int k = 0; k < nw; ++k) e += s_E[k];
        for (int p = 0; p < kPools; ++p) c->q_top[p] += s_total[p];
        c->next_primary = next + A;
        c->E_admitted += e;
    }
    return (int)s_A;
}

cudaError_t launch_init(const Work &w, const Primaries &pr, cudaStream_t st) {
    k_init<<<1, 1024, 0, st>>>(w, pr);
    return cudaGetLastError();
}

constexpr int kPlanThreads = 1024;
constexpr int kPatience = 64;  // iterations without progress before the loop gives up (R7)

// ------------------------------------------------------------------------------------------------
// A9 / A12: refill plan and loop control.  One block.  Per pool: exclusive prefix sum of the per-chunk
// dead counts the step kernels left behind -> rank of every hole; then the sizes of the refill:
//   a      holes filled from the stack (hole k, ascending slot index, takes record [q - 1 - k]),
//   h - a  holes left when the stack is dry: the live range shrinks to n_new and the live tracks above
//          n_new move into the remaining holes below it (j-th live track from the end -> j-th such hole),
//   extra  records appended above the old range when the stack holds more than the holes -- as far as the pool
//          has room, and room is what the pools TRADE here: chunks beyond a pool's range go to the free list, and
//          the free chunks go to the pools in proportion to what their stacks could fill (the
//          track slots are the resource; no per-workload split of them is needed).
__global__ void __launch_bounds__(1024) k_plan(Work w, Primaries pr) {
    constexpr int kGroupWarps = 16;  // warps 0-15 scan the photon pool, 16-31 the charged pool (side by side)
    __shared__ int s_warp[kPools][kGroupWarps];
    __shared__ int s_h[kPools], s_grant[kPools], s_owned[kPools], s_free;
    // the loop state is worked on in shared memory: one coalesced read and one write of the head of the control block
    // instead of a chain of dependent round trips to L2 for every field thread 0 touches
    __shared__ unsigned long long s_head[kCtlHead / 8];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (w.ctl->done) return;
    for (int k = tid; k < (int)(kCtlHead / 8); k += blockDim.x) s_head[k] = reinterpret_cast<const unsigned long long *>(w.ctl)[k];
    __syncthreads();
    Ctl *c = reinterpret_cast<Ctl *>(s_head);
    EMX_TL(w, 0, 0, 0);
    const int admitted = admit_block(w, pr, c);
    __syncthreads();
    {
        const int p = wid / kGroupWarps, wig = wid % kGroupWarps;  // pool of this warp, warp index in its group
        const int gt = wig * 32 + lane;                            // thread index in the group
        const int n_old = c->n_live[p];
        const int nch = (n_old + kChunk - 1) / kChunk;
        constexpr int kPer = 8;  // chunks per thread: one pass of a group covers 4096 chunks
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
        if (gt == 0) s_h[p] = carry;
    }
    __syncthreads();
    if (tid == 0) {
        // the two refills, and how many chunks each pool holds after this iteration
        int a[kPools], n_new[kPools], want_extra[kPools], base[kPools], d[kPools], g[kPools];
        for (int p = 0; p < kPools; ++p) {
            const int n_old = c->n_live[p], h = s_h[p], q = c->q_top[p];
            a[p] = h < q ? h : q;
            n_new[p] = n_old - (h - a[p]);
            want_extra[p] = (h == a[p]) ? q - a[p] : 0;
            // a pool keeps the chunks of its old range through this iteration (k_move still reads its tail)
            base[p] = (n_old + kChunk - 1) / kChunk;
            // ... and never grows into the last pool_reserve chunks of the store, so that the other pool can always start
            const long long top = (long long)n_new[p] + want_extra[p];
            long long want = (top + kChunk - 1) / kChunk;
            if (want > w.n_chunks - w.pool_reserve) want = w.n_chunks - w.pool_reserve;
            d[p] = want > base[p] ? (int)want - base[p] : 0;
        }
        const int avail = w.n_chunks - base[0] - base[1];
        if (d[0] + d[1] <= avail) {
            g[0] = d[0];
            g[1] = d[1];
        } else {
            g[0] = (int)((long long)avail * d[0] / (d[0] + d[1]));
            g[1] = avail - g[0];
        }
        for (int p = 0; p < kPools; ++p) {
            const int n_old = c->n_live[p], h = s_h[p], q = c->q_top[p];
            const int grant = base[p] + g[p];
            int extra = want_extra[p];
            long long room = (long long)grant * kChunk;
            if (room > w.slot_cap) room = w.slot_cap;
            room -= n_old;
            if (extra > room) extra = (int)room;
            PoolPlan pl;
            pl.n_old = n_old;
            pl.h = h;
            pl.a = a[p];
            pl.n_new = n_new[p];
            pl.extra = extra;
            pl.n_final = n_new[p] + extra;
            pl.q_old = q;
            pl.q_new = q - a[p] - extra;
            c->plan[p] = pl;
            c->n_live[p] = pl.n_final;
            c->q_top[p] = pl.q_new;
            s_grant[p] = grant;
            s_owned[p] = c->owned[p];
        }
        s_free = c->n_free;
    }
    __syncthreads();
    // chunk trading: first every pool returns what it holds beyond its grant, then takes what it is short of
    for (int p = 0; p < kPools; ++p) {
        const int own = s_owned[p], grant = s_grant[p], nf = s_free;
        for (int k = tid; k < own - grant; k += blockDim.x) w.free_list[nf + k] = w.ctab[p][grant + k];
        __syncthreads();
        if (tid == 0 && own > grant) {
            s_free = nf + (own - grant);
            s_owned[p] = grant;
        }
        __syncthreads();
    }
    for (int p = 0; p < kPools; ++p) {
        const int own = s_owned[p], grant = s_grant[p], nf = s_free;
        for (int k = tid; k < grant - own; k += blockDim.x) {
            const int ch = w.free_list[nf - 1 - k];
            w.ctab[p][own + k] = ch;
            w.rtab[ch] = own + k;
        }
        __syncthreads();
        if (tid == 0 && grant > own) {
            s_free = nf - (grant - own);
            s_owned[p] = grant;
        }
        __syncthreads();
    }
    if (tid == 0) {
        for (int p = 0; p < kPools; ++p) c->owned[p] = s_owned[p];
        c->n_free = s_free;
        const long long ng = c->n_live[0], nc = c->n_live[1];
        const long long live = ng + nc;
        const long long queued = (long long)c->q_top[0] + c->q_top[1];
        // a track pushes at most 4 records in an iteration (two products and two at-rest photons): where even that
        // fits, the step kernels reserve with one atomic and no look at the top first
        c->q_safe[0] = c->q_safe[1] = (queued + 4LL * live <= (long long)w.qtotal) ? 1 : 0;
        if ((unsigned long long)live > c->peak_live) c->peak_live = (unsigned long long)live;
        if ((unsigned long long)queued > c->peak_queue) c->peak_queue = (unsigned long long)queued;
        if (c->iter < (unsigned long long)w.max_log) {
            w.log[2 * c->iter] = (uint32_t)live;
            w.log[2 * c->iter + 1] = (uint32_t)queued;
        }
        if (live == 0 && c->next_primary >= w.n_primaries) {
            c->done = 1;
            c->m_step[0] = c->m_step[1] = 0;  // the iterations still queued behind this one find nothing to do
            for (int p = 0; p < kPools; ++p)
                for (int k = 0; k < kMaxLists; ++k) c->icount[p][k] = 0;
        } else {
            c->iter += 1;
            // R7: a step whose secondaries do not fit on the stacks is not committed and is re-executed in a
            // later iteration with the same (tid, step) and hence the same draws.  Progress = steps committed or
            // field propagations advanced; retiring a tombstone is none (stalled warps can push and retire
            // tombstones for ever).  kPatience iterations in a row without progress although tracks are live --
            // or with nothing live, nothing queued and no primary admitted -- : the stacks are too small
            c->m_step[0] = (int)ng;
            c->m_step[1] = (int)nc;
            EMX_TL(w, 0, 1, 1);
            const bool stuck = (c->had_live && c->progress == 0ull) || (live == 0 && admitted == 0);
            c->idle_iters = stuck ? c->idle_iters + 1 : 0;
            if (c->idle_iters >= kPatience) {
                c->error = EMX_E_CAPACITY;
                c->done = 1;
                c->m_step[0] = c->m_step[1] = 0;  // nothing more is stepped (k_plan returns at once from now on)
            }
            c->had_live = live > 0 ? 1 : 0;
            // time slicing of the field propagation: with many tracks in flight a track may be parked after a few
            // substep attempts (the rest of its step continues next iteration), so that no propagation holds an
            // iteration open; with few tracks left latency matters more and every propagation runs to its end
            c->field_min = live > w.slice_above ? w.slice_min : 0x7fffffff;
            c->progress = 0ull;
            c->work_f = 0;
            for (int p = 0; p < kPools; ++p)
                for (int k = 0; k < kMaxLists; ++k) c->icount[p][k] = 0;
        }
    }
    __syncthreads();
    for (int k = tid; k < (int)(kCtlHead / 8); k += blockDim.x) reinterpret_cast<unsigned long long *>(w.ctl)[k] = s_head[k];
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
template <int POOL>
__device__ __forceinline__ void fill_pool(const Work &w, int32_t *dbg_src, int *s_w) {
    const Ctl *c = w.ctl;
    const PoolPlan pl = c->plan[POOL];
    const int top = pl.n_old > pl.n_final ? pl.n_old : pl.n_final;
    const int nch_old = (pl.n_old + kChunk - 1) / kChunk;
    const Store &t = w.st;
    for (int ch = blockIdx.x; ch * kChunk < top; ch += gridDim.x) {  // grid-stride over 128-slot chunks
        const int base = ch * kChunk;
        if (ch < nch_old && base + kChunk <= pl.n_old) {  // chunk inside the old range: skip it if nothing died
            const int d0 = w.chunk_off[POOL][ch];
            const int d1 = (ch + 1 < nch_old) ? w.chunk_off[POOL][ch + 1] : pl.h;
            if (d1 == d0) continue;
        }
        const int i = base + threadIdx.x;
        const int s = w.ctab[POOL][ch] * kChunk + threadIdx.x;
        const bool dead = (i < pl.n_old) && (t.alive[s] == 0);
        const int k = w.chunk_off[POOL][ch < nch_old ? ch : 0] + rank_in_chunk(dead, s_w);
        if (dead) {
            if (k < pl.a) {
                const int r = pl.q_old - 1 - k;
                if (dbg_src) { dbg_src[i] = r; t.alive[s] = 2; }
                else load_record<POOL>(w, r, s);
            } else {
                w.hole_idx[POOL][k - pl.a] = i;
            }
        } else if (i >= pl.n_old && i < pl.n_old + pl.extra) {
            const int r = pl.q_old - 1 - pl.a - (i - pl.n_old);
            if (dbg_src) { dbg_src[i] = r; t.alive[s] = 2; }
            else load_record<POOL>(w, r, s);
        }
    }
}
__global__ void __launch_bounds__(kChunk) k_fill(Work w, int32_t *dbg_src) {
    __shared__ int s_w[kChunk / 32];
    if (w.ctl->done) return;
    EMX_TL(w, 1, 0, 1);
    if (blockIdx.y == 0) fill_pool<kPoolGamma>(w, dbg_src, s_w);
    else fill_pool<kPoolCharged>(w, dbg_src, s_w);
    EMX_TL(w, 1, 1, 1);
}

// A9: tail compaction when the stack ran dry: live tracks at or above n_new move into the holes below it
template <int POOL>
__device__ __forceinline__ void move_pool(const Work &w, int32_t *dbg_src, int *s_w) {
    const Ctl *c = w.ctl;
    const PoolPlan pl = c->plan[POOL];
    if (pl.h == pl.a) return;  // nothing to compact
    const Store &t = w.st;
    // grid-stride over the chunks that overlap the tail [n_new, n_old)
    for (int ch = pl.n_new / kChunk + blockIdx.x; ch * kChunk < pl.n_old; ch += gridDim.x) {
        const int i = ch * kChunk + threadIdx.x;
        const int s = w.ctab[POOL][ch] * kChunk + threadIdx.x;
        const bool in = i < pl.n_old;
        const uint8_t al = in ? t.alive[s] : (uint8_t)1;
        const bool dead = al != 1;  // holes of this pass, whether k_fill has refilled them (2) or not (0)
        const int dead_before = w.chunk_off[POOL][ch] + rank_in_chunk(dead, s_w);
        if (in && !dead && i >= pl.n_new) {
            const int dead_after = pl.h - dead_before;      // dead slots in (i, n_old)
            const int j = (pl.n_old - 1 - i) - dead_after;  // live tracks in (i, n_old)
            const int dest = w.hole_idx[POOL][j];
            if (dbg_src) { dbg_src[dest] = -2 - i; t.alive[phys_slot(w, POOL, dest)] = 2; }
            else move_slot<POOL>(w, s, phys_slot(w, POOL, dest));
        }
    }
}
__global__ void __launch_bounds__(kChunk) k_move(Work w, int32_t *dbg_src) {
    __shared__ int s_w[kChunk / 32];
    if (w.ctl->done) return;
    EMX_TL(w, 2, 0, 1);
    if (blockIdx.y == 0) move_pool<kPoolGamma>(w, dbg_src, s_w);
    else move_pool<kPoolCharged>(w, dbg_src, s_w);
    EMX_TL(w, 2, 1, 1);
}

// ------------------------------------------------------------------------------------------------
// A1-A8 + A10: one step of every live track.  PERSISTENT launches: a fixed number of 128-thread blocks whose
// four warps work independently, each pulling 32-slot groups of the pool from a device-side work counter until
// none are left.  A warp never waits for another warp: no block-wide barrier, no shared memory.  One pool and
// one stage per kernel keeps its code in the instruction caches and its registers few enough for 20-32 warps
// per SM (the fused kernel of round 1 held 128 registers and 16 warps; profiles/r2_*).
//   secondaries go straight onto the stacks: the warp counts its records per pool, one lane reserves the range
//   with one atomic ("atomic addition to unambiguously reserve one or more items") and the lanes
//   write consecutive records;
//   tallies: lanes that deposit into the same tally are reduced with warp shuffles and one lane issues the
//   fp64 atomic (north_star "warp-shuffle reductions for tallies"); run counters are kept in registers, one
//   counter per lane, across all groups of the warp and flushed once at the end of the launch.
constexpr int kStepBlock = 128;

template <int POOL>
__device__ __forceinline__ void push_record(const Work &w, int r, const Vec3 &x, const Vec3 &u, double E, uint64_t tid,
                                            uint32_t prim, int vol, int ptype) {
    const Stack &q = w.q;
    r = qrec(w, POOL, r);
    st_cs(&q.xy[r], make_double2(x.x, x.y));
    st_cs(&q.zu[r], make_double2(x.z, u.x));
    st_cs(&q.uu[r], make_double2(u.y, u.z));
    st_cs(&q.Et[r], pack_Et(E, tid));
    st_cs(&q.id[r], make_int4((int)prim, vol, -1, ptype));
}

__device__ __forceinline__ double warp_sum(double v) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ int warp_scan_incl(int v, int lane) {
    for (int d = 1; d < 32; d <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v += t;
    }
    return v;
}

// per-warp accumulators, spread over the lanes: lane k owns integer counter k (0..7 interactions by process,
// 8 null interactions, 9..11 tracks created by type, 12..14 steps by type, 15 progress, 16 stalls, 17 slots
// processed) and lanes 0..3 own the doubles escaped, below_cut, looper, deposited
struct WarpAcc {
    unsigned long long n;
    double d;
};
__device__ __forceinline__ void flush_acc(Ctl *c, const WarpAcc &acc, int lane, unsigned long long *lanes_ctr) {
    if (acc.n) {
        unsigned long long *dst = lane < 8    ? &c->inter[lane]
                                  : lane == 8 ? &c->null_int
                                  : lane < 12 ? &c->tracks[lane - 9]
                                  : lane < 15 ? &c->steps[lane - 12]
                                  : lane == 15 ? &c->progress
                                               : &c->stalls;
        if (lane <= 16) atomicAdd(dst, acc.n);
        if (lane == 17) atomicAdd(lanes_ctr, acc.n);
    }
    if (acc.d != 0.0 && lane < 4) {
        double *dst = lane == 0 ? &c->escaped : lane == 1 ? &c->below_cut : lane == 2 ? &c->looper : &c->edep_total;
        atomicAdd(dst, acc.d);
    }
}

// Reserve `cnt` records (warp total) on stack `pool`; returns the base index or -1 when the arena is full.
// Far from the capacity one atomicAdd does it: w.reserve_slack bounds what all resident warps of
// the step kernels can request at the same time (one outstanding reservation of <= 128 records each), so
// the stacks cannot meet.  Near the capacity a small arena (tests) is reserved by compare-and-swap,
// which never lets the two tops pass the capacity; a large arena is simply treated as full.  Nothing is ever rolled
// back: an add-then-subtract scheme lets a reservation succeed above a top that a concurrent failure has
// inflated, and strands its records.
__device__ __forceinline__ int reserve(Ctl *c, const Work &w, int pool, int cnt, bool safe) {
    // the two tops are the halves of one 64-bit word: one atomic moves one of them and returns both, so "do the two
    // stacks still fit the arena" is always decided on a consistent pair
    unsigned long long *tops = reinterpret_cast<unsigned long long *>(&c->q_top[0]);
    const int sh = 32 * pool;
    const unsigned long long inc = (unsigned long long)cnt << sh;
    const long long cap = w.qtotal;
    if (safe) return (int)((atomicAdd(tops, inc) >> sh) & 0xffffffffull);  // k_plan's guarantee for this iteration
    unsigned long long old = *(volatile unsigned long long *)tops;
    long long used = (long long)(old & 0xffffffffull) + (long long)(old >> 32);
    if (used + cnt + w.reserve_slack <= cap) return (int)((atomicAdd(tops, inc) >> sh) & 0xffffffffull);
    if (cap < 8LL * w.reserve_slack) {
        // small arena: exact accounting by compare-and-swap
        while (used + cnt <= cap) {
            const unsigned long long prev = atomicCAS(tops, old, old + inc);
            if (prev == old) return (int)((old >> sh) & 0xffffffffull);
            old = prev;
            used = (long long)(old & 0xffffffffull) + (long long)(old >> 32);
        }
    }
    // large arena within the slack of its capacity: treated as full (thousands of warps spinning on
    // one compare-and-swap cost 10x the iteration; the last 2 % of a large arena are not worth it)
    return -1;
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

// index of process `proc` among the interaction lists of its pool, and back
template <int POOL>
__device__ __forceinline__ int proc_slot(int proc) {
    if (POOL == kPoolGamma) return proc == EMX_P_COMPTON ? 0 : (proc == EMX_P_PHOTO ? 1 : 2);
    return proc == EMX_P_MOLLER ? 0 : (proc == EMX_P_BHABHA ? 1 : (proc == EMX_P_BREMS ? 2 : 3));
}
template <int POOL>
__device__ __forceinline__ int slot_proc(int k) {
    if (POOL == kPoolGamma) return k == 0 ? EMX_P_COMPTON : (k == 1 ? EMX_P_PHOTO : EMX_P_PAIR);
    return k == 0 ? EMX_P_MOLLER : (k == 1 ? EMX_P_BHABHA : (k == 2 ? EMX_P_BREMS : EMX_P_ANNIH));
}

// what of the slot a kernel's epilogue has to write back
enum : int { kWrX = 1, kWrU = 2, kWrE = 4 };

// What the finishing kernels do with a lane's result: reserve and write the secondaries (A8), write the track
// back, tally (A10), count.  `pend` >= 0: the lane's step is not finished -- its interaction `pend` was
// selected and waits for k_b; only what has happened so far (move, continuous loss) is committed.
// i = pool-local slot, s = physical slot, pt = particle type of the lane's track.
template <int POOL, int WR, bool CONSEC>
__device__ __forceinline__ WarpAcc epilogue(const Params &P, const Work &w, uint64_t seed, double *tally, int i, int s,
                                            int pt, bool active, bool tomb, int pend, Track &t, StepOut &o, int vol0,
                                            uint32_t step0, int safe) {
    WarpAcc acc;
    acc.n = 0ull;
    acc.d = 0.0;
    Ctl *c = w.ctl;
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    const Store &ts = w.st;
    // ---- A8: secondaries -> stacks.  When a stack cannot take the warp's records the lanes that needed
    // it STALL: nothing of their step is committed (R7).  Records a stalled lane did obtain
    // on the other stack become tombstones (E < 0), which the next refill loads and the step kernels retire.
    const int ng = (o.s0.ptype == kGamma) + (o.s1.ptype == kGamma) + 2 * o.rest_alloc;
    const int nc = (o.s0.ptype == kElectron) + (o.s1.ptype == kPositron);  // ordinal 0 an e-, ordinal 1 the pair e+
    bool stall = false;
    int r_c = -1, r_g = -1;
    {
        // warp totals and each lane's offset: charged records 0..2 per lane from photons (pair production), 0..1
        // from e+-; photons 0..3 per lane, from e+- only.  Lane 0 reserves on the charged stack and lane 1 on the
        // photon stack in the same instruction, so the two round trips overlap.
        const unsigned bc = __ballot_sync(0xffffffffu, nc > 0);
        const unsigned bg = POOL == kPoolCharged ? __ballot_sync(0xffffffffu, ng > 0) : 0u;
        if (bc | bg) {
            int inc_c = 0, tot_c = 0, inc_g = 0, tot_g = 0;
            if (bc) {
                if (POOL == kPoolGamma) {
                    inc_c = warp_scan_incl(nc, lane);
                    tot_c = __shfl_sync(0xffffffffu, inc_c, 31);
                } else {
                    inc_c = __popc(bc & lt) + nc;
                    tot_c = __popc(bc);
                }
            }
            if (bg) {
                inc_g = warp_scan_incl(ng, lane);
                tot_g = __shfl_sync(0xffffffffu, inc_g, 31);
            }
            int r0 = -1;
            const int my_cnt = lane == 0 ? tot_c : (lane == 1 ? tot_g : 0);
            if (my_cnt) r0 = reserve(c, w, 1 - lane, my_cnt, (safe >> (1 - lane)) & 1);  // lane 0: kPoolCharged, lane 1: kPoolGamma
            const int r0c = __shfl_sync(0xffffffffu, r0, 0), r0g = __shfl_sync(0xffffffffu, r0, 1);
            if (nc) {
                if (r0c < 0) stall = true;
                else r_c = r0c + inc_c - nc;
            }
            if (ng) {
                if (r0g < 0) stall = true;
                else r_g = r0g + inc_g - ng;
            }
        }
    }
    if (stall) {
        if (r_c >= 0)
            for (int k = 0; k < nc; ++k) w.q.Et[qrec(w, kPoolCharged, r_c + k)] = make_double2(-1.0, 0.0);
        if (r_g >= 0)
            for (int k = 0; k < ng; ++k) w.q.Et[qrec(w, kPoolGamma, r_g + k)] = make_double2(-1.0, 0.0);
    } else {
        const uint32_t k0 = (uint32_t)seed;
        if (nc) {
            int r = r_c;
            if (o.s0.ptype == kElectron)
                push_record<kPoolCharged>(w, r++, t.x, o.s0.u, o.s0.E, child_tid(k0, t.prim, t.tid, step0, 0u), t.prim, t.vol, kElectron);
            if (o.s1.ptype == kPositron)
                push_record<kPoolCharged>(w, r++, t.x, o.s1.u, o.s1.E, child_tid(k0, t.prim, t.tid, step0, 1u), t.prim, t.vol, kPositron);
        }
        if (POOL == kPoolCharged && ng) {
            int r = r_g;
            if (o.s0.ptype == kGamma)
                push_record<kPoolGamma>(w, r++, t.x, o.s0.u, o.s0.E, child_tid(k0, t.prim, t.tid, step0, 0u), t.prim, t.vol, kGamma);
            if (o.s1.ptype == kGamma)
                push_record<kPoolGamma>(w, r++, t.x, o.s1.u, o.s1.E, child_tid(k0, t.prim, t.tid, step0, 1u), t.prim, t.vol, kGamma);
            if (o.rest_alloc) {
                const Vec3 mu = {-o.rest_u.x, -o.rest_u.y, -o.rest_u.z};
                push_record<kPoolGamma>(w, r++, t.x, o.rest_u, kMe, child_tid(k0, t.prim, t.tid, step0, 2u), t.prim, t.vol, kGamma);
                push_record<kPoolGamma>(w, r++, t.x, mu, kMe, child_tid(k0, t.prim, t.tid, step0, 3u), t.prim, t.vol, kGamma);
            }
        }
    }
    const bool commit = active && !tomb && !stall;

    // ---- write the track back (A5-A7 results); tid and prim never change
    if (commit) {
        if (WR & kWrX) ts.xy[s] = make_double2(t.x.x, t.x.y);
        if (WR & (kWrX | kWrU)) ts.zu[s] = make_double2(t.x.z, t.u.x);
        if (WR & kWrU) ts.uu[s] = make_double2(t.u.y, t.u.z);
        if (WR & kWrE) ts.Et[s] = pack_Et(t.E, t.tid);
        ts.id[s] = make_int4((int)t.prim, (int)t.step, t.vol, t.surf);
        ts.stage[s] = (uint8_t)(pend >= 0 ? kStPend + pend : kStFresh);
    }
    const bool died = active && (tomb || (commit && !t.alive));
    if (active) ts.alive[s] = (uint8_t)(died ? 0 : 1);
    // steps-per-track histogram: a track that ends here took step0 + 1 steps; lanes with the same bin share
    // one atomic (most tracks end after a few steps: per-lane atomics on those few bins cost 70 % more time)
    {
        const bool ended = died && !tomb;
        const unsigned be = __ballot_sync(0xffffffffu, ended);
        if (ended) {
            const int hb = step_bin(step0 + 1u) + EMX_NHIST * pt;
            const unsigned m = __match_any_sync(be, hb);
            if (lane == __ffs(m) - 1) atomicAdd(&c->hist[0][hb], (unsigned long long)__popc(m));
        }
    }
    // dead slots per 128-slot chunk, for the refill plan (A9)
    if (CONSEC) {  // the warp's lanes are 32 consecutive slots of one chunk
        const unsigned bd = __ballot_sync(0xffffffffu, died);
        if (bd && lane == 0) atomicAdd(&w.chunk_dead[POOL][i / kChunk], __popc(bd));
    } else if (died) {  // phase B works on physical slots: the chunk's place in the pool comes from the reverse table
        atomicAdd(&w.chunk_dead[POOL][w.rtab[s / kChunk]], 1);
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
            const double sum = warp_sum(mine ? o.edep : 0.0);
            if (lane == leader) atomicAdd(&tally[key], sum);
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
        const unsigned n_e = __popc(__ballot_sync(0xffffffffu, commit && o.s0.ptype == kElectron));
        const unsigned n_p = __popc(__ballot_sync(0xffffffffu, commit && o.s1.ptype == kPositron));
        unsigned n_g = commit ? (unsigned)ng : 0u;
        for (int o2 = 16; o2 > 0; o2 >>= 1) n_g += __shfl_xor_sync(0xffffffffu, n_g, o2);
        const bool stepped = commit && pend < 0;  // completed steps
        const unsigned n_commit = __popc(__ballot_sync(0xffffffffu, commit));
        const unsigned n_s0 = __popc(__ballot_sync(0xffffffffu, stepped && pt == kGamma));
        const unsigned n_s1 = __popc(__ballot_sync(0xffffffffu, stepped && pt == kElectron));
        const unsigned n_s2 = __popc(__ballot_sync(0xffffffffu, stepped && pt == kPositron));
        const unsigned n_stall = __popc(__ballot_sync(0xffffffffu, active && stall));
        const unsigned n_active = __popc(__ballot_sync(0xffffffffu, active));
        if (lane == 9) add = n_g;
        if (lane == 10) add = n_e;
        if (lane == 11) add = n_p;
        if (lane == 12) add = n_s0;
        if (lane == 13) add = n_s1;
        if (lane == 14) add = n_s2;
        if (lane == 15) add = n_commit;
        if (lane == 16) add = n_stall;
        if (lane == 17) add = n_active;
        acc.n += add;
    }
    return acc;
}

// ---- phase A of a group of 32 consecutive slots.
// FUSED: stages a0, a1 (straight move) and a2 in registers (photons; e+- without a field).
// else:  stage a2 alone, for the slots whose move the propagation kernel has finished.
// Lanes whose step ends here (boundary, loss-limited, truncated, killed) are committed; lanes with an
// interaction pending are committed as far as they got and filed in the list of their process, so that
// k_b runs every interactor on full warps (B:north_star "partitioned by next action").
template <int POOL, bool EXT, bool FUSED>
__device__ __forceinline__ WarpAcc a_group(const Params &P, const Work &w, uint64_t seed, double *tally, int base,
                                           int n_live, int safe, const double *gtab = nullptr) {
    constexpr bool CH = POOL == kPoolCharged;
    Ctl *c = w.ctl;
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    const int i = base + lane;
    const Store &ts = w.st;
    const int s = w.ctab[POOL][base / kChunk] * kChunk + (i % kChunk);
    const bool in = i < n_live;
    Track t;
    StepOut o;
    int vol0 = 0, pt = CH ? kElectron : kGamma;
    uint32_t step0 = 0;
    int stage = kStFresh, al = 1;
    double E0 = 0.0;
    if (in) {
        al = ts.alive[s];
        stage = ts.stage[s];
        const double2 Et = ts.Et[s];
        E0 = Et.x;
        t.tid = tid_of(Et);
        if (CH) pt = ts.ptype[s];
    }
    const bool tomb = in && E0 < 0.0;  // tombstone record: retire the slot without stepping
    const bool waiting = in && !tomb && stage >= kStPend;  // interaction selected earlier and stalled: file it again
    const bool go = in && !tomb && (FUSED ? stage == kStFresh : stage == kStMoved);
    int pend = -1;
    clear_out(o);
    t.alive = 1;
    if (go) {
        const int4 id = ts.id[s];
        const double2 xy = ts.xy[s], zu = ts.zu[s], uu = ts.uu[s];
        t.x = {xy.x, xy.y, zu.x};
        t.u = {zu.y, uu.x, uu.y};
        t.E = E0;
        t.prim = (uint32_t)id.x;
        t.step = (uint32_t)id.y;
        t.vol = id.z;
        t.surf = id.w;
        vol0 = t.vol;
        step0 = t.step;
        Carry cy;
        Lookup L;
        L.Sig0 = L.Sig1 = L.Sig2 = L.Stot = L.D = L.R = L.iL0 = L.iL20 = L.var0 = 0.0;
        L.Rtab = nullptr;
        if (FUSED) {
            step_a0<CH, EXT>(P, seed, pt, t, cy, L, gtab);
            if (cy.action != kActCut) move_straight(P, t, cy);
        } else {
            cy.action = ts.act[s];
            cy.s = ts.s_done[s];
            cy.hit = ts.att[s];
            cy.s_phys = 0.0;
        }
        pend = step_a2<CH, EXT, FUSED>(P, seed, pt, t, o, cy, L);
    }
    // file the lanes with a pending interaction (new or stalled) in the list of their process: one atomic per
    // warp and non-empty list
    const int pk = waiting ? proc_slot<POOL>(stage - kStPend) : (pend >= 0 ? proc_slot<POOL>(pend) : -1);
    // (lane k reserves the entries of list k; the atomics are in flight while the epilogue runs)
    constexpr int nk = CH ? 4 : 3;
    unsigned my_mask = 0;
    int list_cnt = 0, list_r0 = 0;
#pragma unroll
    for (int k = 0; k < nk; ++k) {
        const unsigned b = __ballot_sync(0xffffffffu, pk == k);
        if (pk == k) my_mask = b;
        if (lane == k) list_cnt = __popc(b);
    }
    if (list_cnt) list_r0 = atomicAdd(&c->icount[POOL][lane], list_cnt);
    // FUSED: position moved here; a2: position and direction were written by the propagation kernel and change
    // again only through multiple scattering (deflection; lateral displacement of R-MSC2)
    constexpr int WR = FUSED ? (kWrX | (CH ? kWrE : 0) | (CH && EXT ? kWrU : 0)) : (kWrE | (EXT ? (kWrU | kWrX) : 0));
    WarpAcc acc = epilogue<POOL, WR, true>(P, w, seed, tally, i, s, pt, go || tomb, tomb, pend, t, o, vol0, step0, safe);
    const int my_base = __shfl_sync(0xffffffffu, list_r0, pk >= 0 ? pk : 0);
    if (pk >= 0) w.ilist[POOL][pk][my_base + __popc(my_mask & lt)] = s;
    // a track the refill has just moved and that no kernel finishes in this iteration (parked propagation, stalled
    // interaction) still carries the mark of the refill pass
    if (in && !(go || tomb) && al == 2) ts.alive[s] = 1;
    return acc;
}

// the persistent loop of the dense phase-A kernels
template <int POOL, bool EXT, bool FUSED>
__device__ __forceinline__ void a_kernel_body(const Params &P, const Work &w, uint64_t seed, double *tally, int node,
                                              const double *gtab = nullptr) {
    Ctl *c = w.ctl;
    const int lane = threadIdx.x & 31;
    const int nl = c->m_step[POOL];
    const int total = (nl + 31) >> 5;
    const int safe = c->q_safe[0] | (c->q_safe[1] << 1);
    EMX_TL(w, node, 0, 1);
    WarpAcc acc;
    acc.n = 0ull;
    acc.d = 0.0;
    // the groups of a dense kernel cost about the same: a fixed stride per warp, no work counter
    const int n_warps = gridDim.x * (kStepBlock / 32);
    for (int k = blockIdx.x * (kStepBlock / 32) + (threadIdx.x >> 5); k < total; k += n_warps) {
        const WarpAcc d = a_group<POOL, EXT, FUSED>(P, w, seed, tally, k << 5, nl, safe, gtab);
        acc.n += d.n;
        acc.d += d.d;
    }
    flush_acc(c, acc, lane, &c->lanes[2][POOL]);
    EMX_TL(w, node, 1, 1);
}

#ifndef EMX_BLOCKS_A
#define EMX_BLOCKS_A 4   // resident 128-thread blocks per SM the dense phase-A kernels are compiled for
#endif
#ifndef EMX_BLOCKS_AG
#define EMX_BLOCKS_AG 5  // the photon instantiation of k_a: 102 registers (measured: -7 % for the kernel); e+- keep 4 blocks (128)
#endif
#ifndef EMX_BLOCKS_A2
#define EMX_BLOCKS_A2 5
#endif
#ifndef EMX_BLOCKS_B
#define EMX_BLOCKS_B 4
#endif
#ifndef EMX_BLOCKS_F
#define EMX_BLOCKS_F 6  // uniform field: 80 registers; the field-map instantiations keep 96 (5 blocks)
#endif
#ifndef EMX_BLOCKS_0
#define EMX_BLOCKS_0 8
#endif

template <int POOL, bool EXT>
__global__ void __launch_bounds__(kStepBlock, POOL == kPoolGamma ? EMX_BLOCKS_AG : EMX_BLOCKS_A) k_a(const __grid_constant__ Params P, const __grid_constant__ Work w,
                                                                uint64_t seed, double *tally, int stage_tab) {
    // photon pool, emx_schedule entry 7 bit 1: the three tables a photon step interpolates (Compton, photoelectric, pair:
    // 3 x n_E doubles per material, adjacent kinds) are copied to shared memory first (B:north_star "shared-memory ...
    // staging of the hot table slices"; measured, profiles/r2_staging.md)
    extern __shared__ double s_gtab[];
    const double *gtab = nullptr;
    if (POOL == kPoolGamma && stage_tab) {
        const int nE = P.ph.n_E, per = 3 * nE;
        for (int k = threadIdx.x; k < P.n_mat * per; k += blockDim.x)
            s_gtab[k] = P.tab[(size_t)(k / per) * EMX_NTABLE * nE + (k % per)];
        __syncthreads();
        gtab = s_gtab;
    }
    a_kernel_body<POOL, EXT, true>(P, w, seed, tally, 3 + POOL, gtab);
}
template <bool EXT>
__global__ void __launch_bounds__(kStepBlock, EMX_BLOCKS_A2) k_a2(const __grid_constant__ Params P, const __grid_constant__ Work w,
                                                                  uint64_t seed, double *tally) {
    a_kernel_body<kPoolCharged, EXT, false>(P, w, seed, tally, 4);
}

// ---- stage a0 of the charged pool when there is a field: limits of every fresh track (dense, nothing but
// per-lane work).  A track below the tracking cut goes straight to stage a2.
template <bool EXT>
__global__ void __launch_bounds__(kStepBlock, EMX_BLOCKS_0) k_a0(const __grid_constant__ Params P, const __grid_constant__ Work w,
                                                                 uint64_t seed) {
    Ctl *c = w.ctl;
    const int lane = threadIdx.x & 31;
    const int nl = c->m_step[kPoolCharged];
    const int total = (nl + 31) >> 5;
    const Store &ts = w.st;
    const int ax = P.field_kind == 0 ? field_axis(P.Bhat) : kAxisAny;
    EMX_TL(w, 7, 0, 1);
    unsigned long long n_done = 0;
    const int n_warps = gridDim.x * (kStepBlock / 32);
    for (int k = blockIdx.x * (kStepBlock / 32) + (threadIdx.x >> 5); k < total; k += n_warps) {
        const int i = (k << 5) + lane;
        if (i >= nl) continue;
        const int s = phys_slot(w, kPoolCharged, i);
        if (ts.stage[s] != kStFresh) continue;
        const double2 Et = ts.Et[s];
        if (Et.x < 0.0) continue;  // tombstone: stage a2 retires it
        const int4 id = ts.id[s];
        Track t;
        t.E = Et.x;
        t.tid = tid_of(Et);
        t.prim = (uint32_t)id.x;
        t.step = (uint32_t)id.y;
        t.vol = id.z;
        Carry cy;
        Lookup L;
        const int pt = ts.ptype[s];
        step_a0<true, EXT>(P, seed, pt, t, cy, L);
        ts.act[s] = (uint8_t)cy.action;
        if (cy.action == kActCut) {
            ts.stage[s] = kStMoved;
        } else {  // the propagation starts here: curvature and the first trial step (C9)
            double kappa = curvature(P, pt, t.E);
            if (ax != kAxisAny) kappa *= P.Bhat[ax];
            FieldState fs;
            field_begin(kappa, cy.s_phys, fs);
            ts.s_phys[s] = cy.s_phys;
            ts.kap[s] = kappa;
            ts.s_done[s] = fs.s_done;
            ts.h_try[s] = fs.h;
            ts.att[s] = fs.attempt;
            ts.stage[s] = kStParked;
        }
        n_done += 1;
    }
    for (int o = 16; o > 0; o >>= 1) n_done += __shfl_xor_sync(0xffffffffu, n_done, o);
    if (lane == 0 && n_done) atomicAdd(&c->lanes[0][kPoolCharged], n_done);
    EMX_TL(w, 7, 1, 1);
}

// ---- stage a1 of the charged pool in a field: the adaptive RK4 of C9, ONE ATTEMPT of the substep loop per pass
// of the warp.  A lane whose track is done (or parked) takes the next track of the pool in the same pass, so the
// warp stays full whether a propagation needs 1 attempt or 1000 (a lane that runs the whole loop of its own
// track idles 31 others for as long as the longest of them lasts: the e- kernel of round 1 spent 212 of the 311 us
// of an iteration that way once the field had its true strength).  A track may be parked after field_min
// attempts once the pool has no track left to hand out (or after slice_max attempts): its loop variables go to
// the slot and the next iteration continues the SAME sequence of substeps.
template <bool MAP, int AX, int INTEG = 0>
__global__ void __launch_bounds__(kStepBlock, MAP ? 5 : EMX_BLOCKS_F) k_field(const __grid_constant__ Params P, const __grid_constant__ Work w,
                                                                    int stage_faces) {
    // the face table of the whole geometry (16 B per face) is staged in shared memory when it fits: every attempt
    // reads the faces of its cell (B:north_star "shared-memory ... staging of the hot table slices")
    extern __shared__ double2 s_faces2[];
    const Face *faces = P.faces;
    if (stage_faces) {
        const double2 *src = reinterpret_cast<const double2 *>(P.faces);
        for (int k = threadIdx.x; k < P.n_vol * EMX_MAX_FACES; k += blockDim.x) s_faces2[k] = src[k];
        __syncthreads();
        faces = reinterpret_cast<const Face *>(s_faces2);
    }
    Ctl *c = w.ctl;
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    const int nl = c->m_step[kPoolCharged];
    const int min_att = c->field_min, max_att = w.slice_max;
    const Store &ts = w.st;
    EMX_TL(w, 8, 0, 1);
    bool have = false, dry = false;
    int s = 0, vol = 0, surf = -1, used = 0, act = 0;
    Vec3 x = {0.0, 0.0, 0.0}, u = {0.0, 0.0, 1.0};
    double kappa = 1.0, s_max = 0.0;
    FieldState fs;
    fs.s_done = fs.h = 0.0;
    fs.attempt = 0;
    unsigned n_att = 0, n_trk = 0;
    for (;;) {
        // hand the idle lanes the next slots of the pool
        unsigned need = __ballot_sync(0xffffffffu, !have && !dry);
        while (need) {
            const int leader = __ffs(need) - 1;
            int i0 = 0;
            if (lane == leader) i0 = atomicAdd(&c->work_f, __popc(need));
            i0 = __shfl_sync(0xffffffffu, i0, leader);
            if (!have && !dry) {
                const int i = i0 + __popc(need & lt);
                if (i >= nl) {
                    dry = true;
                } else {
                    s = phys_slot(w, kPoolCharged, i);
                    if (ts.stage[s] == kStParked) {
                        const double2 xy = ts.xy[s], zu = ts.zu[s], uu = ts.uu[s];
                        const int4 id = ts.id[s];
                        x = {xy.x, xy.y, zu.x};
                        u = {zu.y, uu.x, uu.y};
                        vol = id.z;
                        surf = id.w;
                        s_max = ts.s_phys[s];
                        act = ts.act[s];
                        kappa = ts.kap[s];
                        fs.s_done = ts.s_done[s];
                        fs.h = ts.h_try[s];
                        fs.attempt = ts.att[s];
                        have = true;
                        used = 0;
                        n_trk += 1;
                    }
                }
            }
            need = __ballot_sync(0xffffffffu, !have && !dry);
        }
        if (!__ballot_sync(0xffffffffu, have)) break;
        const bool pool_dry = __ballot_sync(0xffffffffu, dry) != 0u;
        if (have) {
            int hit;
            double sres;
            const bool done = field_attempt<MAP, AX, INTEG>(P, faces + vol * EMX_MAX_FACES, surf, x, u, kappa, s_max, fs, hit, sres);
            used += 1;
            n_att += 1;
            if (done) {
                Carry cy;
                cy.s_phys = s_max;
                cy.action = act;
                field_move_done(cy, sres, hit);
                ts.xy[s] = make_double2(x.x, x.y);
                ts.zu[s] = make_double2(x.z, u.x);
                ts.uu[s] = make_double2(u.y, u.z);
                ts.s_done[s] = cy.s;
                ts.att[s] = cy.hit;
                ts.act[s] = (uint8_t)cy.action;
                ts.stage[s] = kStMoved;
                have = false;
            } else if (used >= min_att && (pool_dry || used >= max_att)) {
                ts.xy[s] = make_double2(x.x, x.y);
                ts.zu[s] = make_double2(x.z, u.x);
                ts.uu[s] = make_double2(u.y, u.z);
                reinterpret_cast<int *>(ts.id)[4 * (size_t)s + 3] = surf;
                ts.s_done[s] = fs.s_done;
                ts.h_try[s] = fs.h;
                ts.att[s] = fs.attempt;
                ts.stage[s] = kStParked;
                have = false;
            }
        }
    }
    unsigned long long a = n_att, b = n_trk;
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, o);
        b += __shfl_xor_sync(0xffffffffu, b, o);
    }
    if (lane == 0 && a) {
        atomicAdd(&c->progress, a);
        atomicAdd(&c->attempts, a);
        atomicAdd(&c->lanes[1][kPoolCharged], b);
    }
    EMX_TL(w, 8, 1, 1);
}

// ---- phase B of a group: 32 tracks of a pool waiting for the same interactor (list k of the pool).
template <int POOL>
__device__ __forceinline__ WarpAcc b_group(const Params &P, const Work &w, uint64_t seed, double *tally, int k, int first,
                                           int n_list, int safe) {
    constexpr bool CH = POOL == kPoolCharged;
    const int lane = threadIdx.x & 31;
    const int idx = first + lane;
    const Store &ts = w.st;
    const bool active = idx < n_list;
    const int s = active ? w.ilist[POOL][k][idx] : 0;
    const int i = 0;  // phase B does not need the pool-local index
    Track t;
    StepOut o;
    clear_out(o);
    o.action = EMX_A_DISCRETE;
    int vol0 = 0, pt = CH ? kElectron : kGamma;
    uint32_t step0 = 0;
    t.alive = 1;
    if (active) {
        const double2 xy = ts.xy[s], zu = ts.zu[s], uu = ts.uu[s], Et = ts.Et[s];
        const int4 id = ts.id[s];
        if (CH) pt = ts.ptype[s];
        t.x = {xy.x, xy.y, zu.x};
        t.u = {zu.y, uu.x, uu.y};
        t.E = Et.x;
        t.tid = tid_of(Et);
        t.prim = (uint32_t)id.x;
        t.step = (uint32_t)id.y;
        t.vol = id.z;
        t.surf = -1;
        vol0 = t.vol;
        step0 = t.step;
        step_interact<CH>(P, seed, pt, t, o, slot_proc<POOL>(k));
    }
    return epilogue<POOL, kWrU | kWrE, false>(P, w, seed, tally, i, s, pt, active, false, -1, t, o, vol0, step0, safe);
}

// Phase B: the interactors.  Persistent warps pull 32-entry groups of the pool's process lists; a warp runs ONE
// interactor on (up to) 32 tracks that all selected it.
template <int POOL>
__global__ void __launch_bounds__(kStepBlock, EMX_BLOCKS_B) k_b(const __grid_constant__ Params P, const __grid_constant__ Work w,
                                                                uint64_t seed, double *tally) {
    Ctl *c = w.ctl;
    const int lane = threadIdx.x & 31;
    constexpr int nk = (POOL == kPoolCharged) ? 4 : 3;
    // order in which the lists are worked off.  The stacks are LIFO, so what is pushed LAST is refilled
    // first: photons run pair production first (its leptons are the most energetic secondaries and go to the
    // bottom of this iteration's records) and photoelectric absorption last; e+- run bremsstrahlung and
    // annihilation before the knock-on electrons.  Keeping low-energy tracks on top is what keeps the queue
    // short ("preferentially selecting lower-energy particles").
    const int ord[4] = {POOL == kPoolGamma ? 2 : 2, POOL == kPoolGamma ? 0 : 3, POOL == kPoolGamma ? 1 : 0, 1};
    int n[4], cb[5];
    cb[0] = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        n[k] = k < nk ? c->icount[POOL][ord[k]] : 0;
        cb[k + 1] = cb[k] + ((n[k] + 31) >> 5);
    }
    const int total = cb[4];
    const int safe = c->q_safe[0] | (c->q_safe[1] << 1);
    EMX_TL(w, 5 + POOL, 0, 1);
    WarpAcc acc;
    acc.n = 0ull;
    acc.d = 0.0;
    const int n_warps = gridDim.x * (kStepBlock / 32);
    for (int ch = blockIdx.x * (kStepBlock / 32) + (threadIdx.x >> 5); ch < total; ch += n_warps) {
        // one call site: the interactor code exists once per kernel
        const int sel = ch < cb[1] ? 0 : (ch < cb[2] ? 1 : (ch < cb[3] ? 2 : 3));
        const WarpAcc d = b_group<POOL>(P, w, seed, tally, ord[sel], (ch - cb[sel]) << 5, n[sel], safe);
        acc.n += d.n;
        acc.d += d.d;
    }
    flush_acc(c, acc, lane, &c->lanes[3][POOL]);
    EMX_TL(w, 5 + POOL, 1, 1);
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

// ------------------------------------------------------------------------------------------------
// launchers

cudaError_t launch_refill(const Work &w, const Primaries &pr, cudaStream_t st) {
    k_plan<<<1, kPlanThreads, 0, st>>>(w, pr);
    const dim3 g3(kRefillBlocks, kPools);
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

static bool ext_on(const Params &P) { return P.ph.msc || P.ph.fluct; }

// the kernels of one pool's chain, one by one (kStage*: emx_kernels.h)
cudaError_t launch_stage(int stage, const Params &P, const Work &w, uint64_t seed, double *tally, cudaStream_t st) {
    const int g = w.grid[stage];
    const bool ext = ext_on(P);
    switch (stage) {
    case kStageAGamma: {
        // shared-memory copy of the photon tables: 3 x n_E doubles per material, up to 40 KB per block
        const size_t tb = (size_t)P.n_mat * 3 * (size_t)P.ph.n_E * sizeof(double);
        const int stage_tab = ((w.stage_faces & 2) && tb <= 40 * 1024) ? 1 : 0;
        k_a<kPoolGamma, false><<<g, kStepBlock, stage_tab ? tb : 0, st>>>(P, w, seed, tally, stage_tab);
        break;
    }
    case kStageACharged:  // no field: limits + straight move + finish
        if (ext) k_a<kPoolCharged, true><<<g, kStepBlock, 0, st>>>(P, w, seed, tally, 0);
        else k_a<kPoolCharged, false><<<g, kStepBlock, 0, st>>>(P, w, seed, tally, 0);
        break;
    case kStageA0:
        if (ext) k_a0<true><<<g, kStepBlock, 0, st>>>(P, w, seed);
        else k_a0<false><<<g, kStepBlock, 0, st>>>(P, w, seed);
        break;
    case kStageField: {
        const int ax = P.field_kind == 0 ? field_axis(P.Bhat) : kAxisAny;
        // shared-memory copy of the face table: up to 40 KB per block (5 blocks per SM stay resident)
        const size_t fb = (size_t)P.n_vol * EMX_MAX_FACES * sizeof(Face);
        const int stage = ((w.stage_faces & 1) && fb <= 40 * 1024) ? 1 : 0;
        const size_t sm = stage ? fb : 0;
        if (P.ph.integrator == 1) {  // Dormand-Prince 5(4) (DESIGN.md R-INT): instantiations of their own
            if (P.field_kind != 0) k_field<true, kAxisAny, 1><<<g, kStepBlock, sm, st>>>(P, w, stage);
            else if (ax == 0) k_field<false, 0, 1><<<g, kStepBlock, sm, st>>>(P, w, stage);
            else if (ax == 1) k_field<false, 1, 1><<<g, kStepBlock, sm, st>>>(P, w, stage);
            else if (ax == 2) k_field<false, 2, 1><<<g, kStepBlock, sm, st>>>(P, w, stage);
            else k_field<false, kAxisAny, 1><<<g, kStepBlock, sm, st>>>(P, w, stage);
        } else if (P.field_kind != 0) k_field<true, kAxisAny><<<g, kStepBlock, sm, st>>>(P, w, stage);
        else if (ax == 0) k_field<false, 0><<<g, kStepBlock, sm, st>>>(P, w, stage);
        else if (ax == 1) k_field<false, 1><<<g, kStepBlock, sm, st>>>(P, w, stage);
        else if (ax == 2) k_field<false, 2><<<g, kStepBlock, sm, st>>>(P, w, stage);
        else k_field<false, kAxisAny><<<g, kStepBlock, sm, st>>>(P, w, stage);
        break;
    }
    case kStageA2:
        if (ext) k_a2<true><<<g, kStepBlock, 0, st>>>(P, w, seed, tally);
        else k_a2<false><<<g, kStepBlock, 0, st>>>(P, w, seed, tally);
        break;
    case kStageBGamma:
        k_b<kPoolGamma><<<g, kStepBlock, 0, st>>>(P, w, seed, tally);
        break;
    case kStageBCharged:
        k_b<kPoolCharged><<<g, kStepBlock, 0, st>>>(P, w, seed, tally);
        break;
    default:
        return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

// the step kernels of one pool on its stream (fork / join branches of the iteration graph)
cudaError_t launch_step_pool(int pool, const Params &P, const Work &w, uint64_t seed, double *tally, cudaStream_t st) {
    cudaError_t e = cudaSuccess;
    if (pool == kPoolGamma) {
        e = launch_stage(kStageAGamma, P, w, seed, tally, st);
        if (e == cudaSuccess) e = launch_stage(kStageBGamma, P, w, seed, tally, st);
    } else {
        if (P.Bmag == 0.0) {
            e = launch_stage(kStageACharged, P, w, seed, tally, st);
        } else {
            e = launch_stage(kStageA0, P, w, seed, tally, st);
            if (e == cudaSuccess) e = launch_stage(kStageField, P, w, seed, tally, st);
            if (e == cudaSuccess) e = launch_stage(kStageA2, P, w, seed, tally, st);
        }
        if (e == cudaSuccess) e = launch_stage(kStageBCharged, P, w, seed, tally, st);
    }
    return e;
}

// registers per thread of the step kernels as compiled (for sizing the persistent grids)
cudaError_t step_kernel_regs(int stage, bool field, int *regs) {
    cudaFuncAttributes a;
    cudaError_t e;
    switch (stage) {
    case kStageAGamma: e = cudaFuncGetAttributes(&a, k_a<kPoolGamma, false>); break;
    case kStageACharged: e = cudaFuncGetAttributes(&a, k_a<kPoolCharged, false>); break;
    case kStageA0: e = cudaFuncGetAttributes(&a, k_a0<false>); break;
    case kStageField: e = cudaFuncGetAttributes(&a, k_field<false, 2>); break;
    case kStageA2: e = cudaFuncGetAttributes(&a, k_a2<false>); break;
    case kStageBGamma: e = cudaFuncGetAttributes(&a, k_b<kPoolGamma>); break;
    default: e = cudaFuncGetAttributes(&a, k_b<kPoolCharged>); break;
    }
    (void)field;
    if (e == cudaSuccess) *regs = a.numRegs;
    return e;
}

// ------------------------------------------------------------------------------------------------
// level-1 hook: the refill index logic (k_plan, k_fill, k_move) on a caller-supplied alive[] array
__global__ void k_hook_init(Work w, int n_live, int n_queue) {
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid == 0) {
        Ctl z = Ctl();
        z.n_live[0] = n_live;
        z.q_top[0] = n_queue;
        z.owned[0] = w.n_chunks;  // the one pool of the hook owns every chunk, in order
        *w.ctl = z;
    }
    for (int k = tid; k < w.n_chunks; k += gridDim.x * blockDim.x) {
        w.ctab[0][k] = k;
        w.ctab[1][k] = 0;
        w.rtab[k] = k;
    }
}
__global__ void __launch_bounds__(kChunk) k_count_dead(Work w, int n_live) {
    const int i = blockIdx.x * kChunk + threadIdx.x;
    const int n = __syncthreads_count(i < n_live && w.st.alive[i] == 0);
    if (threadIdx.x == 0) w.chunk_dead[0][blockIdx.x] = n;
}

size_t refill_plan_scratch_ints(long capacity) {
    const size_t nch = (size_t)(capacity + kChunk - 1) / kChunk + 1;
    return 7 * nch + (size_t)capacity + (sizeof(Ctl) + 3) / 4 + 64 + (nch * kChunk + 3) / 4 + 64;
}

cudaError_t launch_refill_plan(long n_live, long capacity, long n_queue, const uint8_t *alive, int32_t *src,
                               int *scratch, const Ctl **ctl_out, cudaStream_t st) {
    const size_t nch = (size_t)(capacity + kChunk - 1) / kChunk + 1;
    Work w = Work();
    int *p = scratch;
    w.chunk_dead[0] = p; p += nch;
    w.chunk_off[0] = p; p += nch;
    w.chunk_dead[1] = w.chunk_dead[0];  // the second pool of the hook is empty
    w.chunk_off[1] = w.chunk_off[0];
    w.ctab[0] = p; p += nch;
    w.ctab[1] = p; p += nch;
    w.free_list = p; p += 2 * nch;
    w.rtab = p; p += nch;
    w.hole_idx[0] = p; p += capacity;
    w.hole_idx[1] = w.hole_idx[0];
    p += (16 - ((uintptr_t)p / 4) % 16) % 16;  // 64-byte alignment for the control block
    w.ctl = (Ctl *)p; p += (sizeof(Ctl) + 3) / 4;
    *ctl_out = w.ctl;
    w.st.alive = (uint8_t *)p;
    w.n_chunks = (int)((capacity + kChunk - 1) / kChunk);
    w.slot_cap = (int)capacity;
    w.pool_reserve = 0;
    w.qtotal = 0x7fffffff;
    w.log = nullptr;
    w.max_log = 0;
    w.n_primaries = 0;
    cudaMemsetAsync(w.st.alive, 0, nch * kChunk, st);
    if (n_live > 0) cudaMemcpyAsync(w.st.alive, alive, (size_t)n_live, cudaMemcpyDeviceToDevice, st);
    cudaMemsetAsync(src, 0xFF, (size_t)capacity * sizeof(int32_t), st);
    cudaMemsetAsync(w.chunk_dead[0], 0, 2 * nch * sizeof(int), st);
    k_hook_init<<<8, 256, 0, st>>>(w, (int)n_live, (int)n_queue);
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
