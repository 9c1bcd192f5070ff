// emx_kernels.cu -- every __global__ kernel of the path (sm_100a) and its launcher.
// DESIGN.md section 5 describes each kernel with its algorithmic bytes and the roofline that bounds it.
#include <cuda_runtime.h>
#include "emx_kernels.h"
#include "emx_tables.h"
#include "emx_batch.h"

namespace emx {

// ------------------------------------------------------------------------------------------------
// A11: table builder (runs once per problem)
__global__ void k_table_pass1(TableCtx c) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j < c.ph.n_E) table_pass1(c, blockIdx.y, j);
}
__global__ void k_table_cuts(TableCtx c) {
    if (threadIdx.x == 0) table_cuts(c, blockIdx.x);
}
__global__ void k_table_pass3(TableCtx c) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j < c.ph.n_E) table_pass3(c, blockIdx.y, j);
}
__global__ void k_table_range(TableCtx c) {
    if (threadIdx.x < 2) table_range_sum(c, blockIdx.x, threadIdx.x);
}

cudaError_t launch_build_tables(const TableCtx &c, cudaStream_t st) {
    const int n = c.ph.n_E, tb = 64;
    const dim3 g((n + tb - 1) / tb, c.n_mat);
    k_table_pass1<<<g, tb, 0, st>>>(c);
    k_table_cuts<<<c.n_mat, 32, 0, st>>>(c);
    k_table_pass3<<<g, tb, 0, st>>>(c);
    k_table_range<<<c.n_mat, 32, 0, st>>>(c);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// parity hooks (include/emx.h)
__global__ void k_step_batch(Params P, uint64_t seed, long n, const emx_track *in, emx_step_result *out) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) step_one(P, seed, in[i], out[i]);
}
cudaError_t launch_step_batch(const Params &P, uint64_t seed, long n, const emx_track *in, emx_step_result *out,
                              cudaStream_t st) {
    if (n <= 0) return cudaSuccess;
    const int tb = 64;
    k_step_batch<<<(unsigned)((n + tb - 1) / tb), tb, 0, st>>>(P, seed, n, in, out);
    return cudaGetLastError();
}

// ONE substep of the field propagation (rk4_doubling as k_field runs it: the axis specialisation of a uniform
// field with the sign of the field folded into the curvature, or the field map at the stage positions)
__global__ void k_field_substep_batch(Params P, long n, const double *x3, const double *u3, const double *kappa,
                                      const double *h, double *x1, double *u1, double *err) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const Vec3 x = {x3[3 * i], x3[3 * i + 1], x3[3 * i + 2]}, u = {u3[3 * i], u3[3 * i + 1], u3[3 * i + 2]};
    Vec3 xo, uo;
    double e;
    const int ax = P.field_kind == 0 ? field_axis(P.Bhat) : kAxisAny;
    if (P.ph.integrator == 1) {
        if (P.field_kind != 0) dp45_step<true, kAxisAny>(P, x, u, kappa[i], h[i], xo, uo, e);
        else if (ax == 0) dp45_step<false, 0>(P, x, u, kappa[i] * P.Bhat[0], h[i], xo, uo, e);
        else if (ax == 1) dp45_step<false, 1>(P, x, u, kappa[i] * P.Bhat[1], h[i], xo, uo, e);
        else if (ax == 2) dp45_step<false, 2>(P, x, u, kappa[i] * P.Bhat[2], h[i], xo, uo, e);
        else dp45_step<false, kAxisAny>(P, x, u, kappa[i], h[i], xo, uo, e);
    } else if (P.field_kind != 0) rk4_doubling<true, kAxisAny>(P, x, u, kappa[i], h[i], xo, uo, e);
    else if (ax == 0) rk4_doubling<false, 0>(P, x, u, kappa[i] * P.Bhat[0], h[i], xo, uo, e);
    else if (ax == 1) rk4_doubling<false, 1>(P, x, u, kappa[i] * P.Bhat[1], h[i], xo, uo, e);
    else if (ax == 2) rk4_doubling<false, 2>(P, x, u, kappa[i] * P.Bhat[2], h[i], xo, uo, e);
    else rk4_doubling<false, kAxisAny>(P, x, u, kappa[i], h[i], xo, uo, e);
    put3(x1 + 3 * i, xo);
    put3(u1 + 3 * i, uo);
    err[i] = e;
}
cudaError_t launch_field_substep_batch(const Params &P, long n, const double *x3, const double *u3, const double *kappa,
                                       const double *h, double *x1, double *u1, double *err, cudaStream_t st) {
    if (n <= 0) return cudaSuccess;
    k_field_substep_batch<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(P, n, x3, u3, kappa, h, x1, u1, err);
    return cudaGetLastError();
}

__global__ void k_philox_batch(long n, const uint32_t *ctr, const uint32_t *key, uint32_t *out) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const Philox4 b = philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], key[2 * i], key[2 * i + 1]);
    for (int k = 0; k < 4; ++k) out[4 * i + k] = b.w[k];
}
__global__ void k_draw_batch(uint64_t seed, long n, const uint32_t *prim, const uint64_t *tid, const uint32_t *step,
                             const uint32_t *nn, double *u, uint64_t *child) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    if (u) u[i] = draw_at(seed, prim[i], tid[i], step[i], nn[i]);
    if (child) child[i] = child_tid((uint32_t)seed, prim[i], tid[i], step[i], nn[i]);
}
cudaError_t launch_philox_batch(long n, const uint32_t *ctr, const uint32_t *key, uint32_t *out, cudaStream_t st) {
    if (n <= 0) return cudaSuccess;
    k_philox_batch<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(n, ctr, key, out);
    return cudaGetLastError();
}
cudaError_t launch_draw_batch(uint64_t seed, long n, const uint32_t *prim, const uint64_t *tid, const uint32_t *step,
                              const uint32_t *nn, double *u, uint64_t *child, cudaStream_t st) {
    if (n <= 0) return cudaSuccess;
    k_draw_batch<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(seed, n, prim, tid, step, nn, u, child);
    return cudaGetLastError();
}

}  // namespace emx
