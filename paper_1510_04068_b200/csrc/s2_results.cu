// s2_results.cu -- a9 for device-resident callers: the 96-byte result records of the last force call unpacked into
// the caller's device arrays (same layouts as s2_get_results), so that a consumer on the GPU -- the block-step
// integrator kernels, an NCCL combine of j-sharded partial results (sec 2.2.3) -- never goes through
// the host.  Pure data movement: one thread per i reads its record (three 32-byte sectors) and writes the fields.
#include "s2_force_sweep.cuh"

namespace s2 {

__global__ void __launch_bounds__(256) unpack_records_kernel(const double *rec, int ni, int order, double *acc, double *jerk,
                                                             double *snap, double *pot, int *nn_id, double *nn_r2, int *ngb_count)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= ni) return;
    const double2 *r = reinterpret_cast<const double2 *>(rec + (size_t)i * REC);
    const double2 r0 = r[0], r1 = r[1], r2 = r[2], r3 = r[3], r4 = r[4];
    if (acc) { acc[3 * (size_t)i] = r0.x; acc[3 * (size_t)i + 1] = r0.y; acc[3 * (size_t)i + 2] = r1.x; }
    if (jerk) { jerk[3 * (size_t)i] = r1.y; jerk[3 * (size_t)i + 1] = r2.x; jerk[3 * (size_t)i + 2] = r2.y; }
    if (pot) pot[i] = r3.x;
    if (nn_r2) nn_r2[i] = r3.y;
    if (nn_id) nn_id[i] = __double2loint(r4.x);
    if (ngb_count) ngb_count[i] = __double2hiint(r4.x);
    if (snap && order == 6) {
        const double2 r5 = r[5];
        snap[3 * (size_t)i] = r4.y; snap[3 * (size_t)i + 1] = r5.x; snap[3 * (size_t)i + 2] = r5.y;
    }
}

cudaError_t launch_unpack_records(const double *rec, int ni, int order, double *acc, double *jerk, double *snap, double *pot,
                                  int *nn_id, double *nn_r2, int *ngb_count, cudaStream_t st)
{
    if (ni <= 0) return cudaSuccess;
    unpack_records_kernel<<<(ni + 255) / 256, 256, 0, st>>>(rec, ni, order, acc, jerk, snap, pot, nn_id, nn_r2, ngb_count);
    return cudaGetLastError();
}

// fp32 path, reading R-F32: flag the i-particles whose jerk is a strongly cancelling sum (fp32_flag_warp,
// s2_force_sweep.cuh) for the launch shapes whose final records are not written by reduce_kernel (which flags inline):
// single-slice sweeps, the fused combine, reduce_thread_kernel.  One warp per i.
__global__ void __launch_bounds__(256) fp32_flag_kernel(const double *rec, F32Flag f, int ni)
{
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");   // chained by programmatic dependent launch:
    asm volatile("griddepcontrol.wait;" ::: "memory");                // sweep (-> reduce) -> flag -> fix-up
    const int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (i >= ni) return;
    fp32_flag_warp(f, rec, i, ni, threadIdx.x & 31);
}

cudaError_t launch_fp32_flag(const double *rec, const F32Flag &f, int ni, cudaStream_t st)
{
    if (ni <= 0) return cudaSuccess;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(((long long)ni * 32 + 255) / 256)); cfg.blockDim = dim3(256); cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, fp32_flag_kernel, rec, f, ni);
}

// Self-test of the uniform-operand sweep (s2_api.cu bank_selftest): do two sets of records hold the same sums?
// Per i: ||a - b|| <= tol ||a|| for acc, jerk, snap and |a - b| <= tol |a| for pot; NaNs count as a difference.
__global__ void __launch_bounds__(256) compare_records_kernel(const double *a, const double *b, int ni, int order, double tol, int *bad)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= ni) return;
    const double *x = a + (size_t)i * REC, *y = b + (size_t)i * REC;
    bool ok = true;
    for (int v = 0; v < (order == 6 ? 3 : 2); ++v) {
        const int o = v == 2 ? 9 : 3 * v;
        double num = 0.0, den = 0.0;
        for (int c = 0; c < 3; ++c) {
            const double d = x[o + c] - y[o + c];
            num += d * d;
            den += x[o + c] * x[o + c];
        }
        ok = ok && num <= tol * tol * den;   // false for NaN
    }
    ok = ok && fabs(x[6] - y[6]) <= tol * fabs(x[6]);
    if (!ok) *bad = 1;
}

cudaError_t launch_compare_records(const double *a, const double *b, int ni, int order, double tol, int *bad, cudaStream_t st)
{
    if (ni <= 0) return cudaSuccess;
    compare_records_kernel<<<(ni + 255) / 256, 256, 0, st>>>(a, b, ni, order, tol, bad);
    return cudaGetLastError();
}

}  // namespace s2
