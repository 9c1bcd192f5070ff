// emx_diag.h -- DIAGNOSTICS ONLY, compiled in with -DEMX_TIMELINE (paper_2203_09467_b200/diagnostics/timeline.py):
// first block start / last block end of every kernel node of the iteration graph, from %globaltimer, for
// iterations [EMX_TL_FIRST, EMX_TL_FIRST + kTlN).  Without the flag EMX_TL() expands to nothing and the product
// library carries none of this.  Nodes: 0 k_plan, 1 k_fill, 2 k_move, 3 k_a<gamma>, 4 k_a<charged> / k_a2,
// 5 k_b<gamma>, 6 k_b<charged>, 7 k_a0, 8 k_field.
#pragma once
#include "emx_work.h"

namespace emx {
#ifdef EMX_TIMELINE
#ifndef EMX_TL_FIRST
#define EMX_TL_FIRST 2500
#endif
constexpr int kTlN = 64;
constexpr int kTlNodes = 9;
__device__ unsigned long long g_tl[kTlN][kTlNodes][4];  // min start, max end, sum of block times, blocks
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
}  // namespace emx
