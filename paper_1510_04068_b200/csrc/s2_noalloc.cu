// s2_noalloc.cu -- s2_forces_noalloc: the j-split force sweep + fixed-order combine (PAPER.md
// sec 2.1 "parallelize over the source particles ... split into subsets", sec 2.2.4 "the second sums the
// partial results") as ONE entry point that allocates nothing.
//
// Why: some callers cannot call cudaMalloc -- code under CUDA-graph capture, tight serving loops, harnesses that forbid
// it.  The context-based calls of s2_api.cu grow their partial-record buffer on demand through the allocator; here the
// partial sums of the j-slices live in a file-scope static device array of a fixed, modest size instead
// (kNaScratchBytes = 4 MiB; every GPU that loads the library holds it until the process exits).  The caller passes the
// inputs (predicted j-particles, i-list) and the outputs as device pointers; the entry point calls no cudaMalloc, no
// cudaFree and no allocating library routine -- only cudaSetDevice, (once per device) cudaGetSymbolAddress, and two
// kernel launches.
//
// The scratch array is shared by every call on a device and keeps the last call's contents.  Nothing in it has to start
// at zero: every partial row the combine reads was written by the sweep of the same call (row (s, i) for all s < S,
// i < n_i), so no clearing is needed and stale rows of an earlier, larger call are never read.  Two calls that overlap
// on the GPU (different streams, or one stream of each of two host threads) RACE on the array: callers serialise them.
//
// Arithmetic: IEEE fp64, 4th order (acc, jerk, pot), the pair terms of SURVEY sec 8(c) O3 with the reciprocal square
// root of DESIGN.md reading R-RSQRT; self-interaction skipped by id (P3).  Sums: lanes of a warp take interleaved j of a
// slice and combine by an xor-butterfly, slices are added in slice order 0, 1, ...: bit-reproducible run to run.
#include <cuda_runtime.h>

#include <mutex>

#include "../../include/s2b200.h"

namespace {

constexpr int kNaMaxNi = 4096;                 // largest i-list accepted
constexpr int kNaMaxRows = 65536;              // partial rows (slice, i) the scratch holds: S * n_i <= kNaMaxRows
constexpr int kNaRow = 8;                      // doubles per row: acc[3], jerk[3], pot, pad (64 B = two sectors)
constexpr size_t kNaScratchBytes = (size_t)kNaMaxRows * kNaRow * sizeof(double);   // 4 MiB
constexpr int kNaWarps = 8;                    // warps (= i-particles) per CTA of the sweep
constexpr int kNaMaxDevices = 64;

// Host code: this NAME is a host-side stand-in, not a device address.  Only cudaGetSymbolAddress gives the address a
// kernel may be handed (na_scratch_ptr below); device code in this file could also name the array directly.
static __device__ __align__(256) double g_na_scratch[(size_t)kNaMaxRows * kNaRow];

__device__ __forceinline__ double na_rsqrt(double s)
{
    double y0;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(s));            // MUFU.RSQ64H seed, ~2^-22
    const double e = fma(-(s * y0), y0, 1.0);
    return y0 * fma(fma(0.375, e, 0.5), e, 1.0);                         // one third-order step: e^3 + 2 ulp
}

// grid (ceil(n_i / 8), S); one warp per i-particle, lanes take interleaved j of slice blockIdx.y
__global__ void __launch_bounds__(32 * kNaWarps) na_sweep_kernel(const double *pos, const double *vel, const double *mass, const int *id,
                                                                 int nj, const int *i_addr, int ni, double eps2, int slice_len,
                                                                 double *scratch)
{
    const int lane = threadIdx.x & 31;
    const int i = blockIdx.x * kNaWarps + (threadIdx.x >> 5);
    if (i >= ni) return;                                                 // whole warp
    double *row = scratch + ((size_t)blockIdx.y * ni + i) * kNaRow;
    const int ia = i_addr[i];
    if (ia < 0 || ia >= nj) {                                            // bad address: the result of this i is NaN, nothing faults
        if (lane < kNaRow) row[lane] = __longlong_as_double(0x7ff8000000000000LL);
        return;
    }
    const double xi = pos[3 * (size_t)ia], yi = pos[3 * (size_t)ia + 1], zi = pos[3 * (size_t)ia + 2];
    const double vxi = vel[3 * (size_t)ia], vyi = vel[3 * (size_t)ia + 1], vzi = vel[3 * (size_t)ia + 2];
    const int idi = id[ia];
    const int j0 = blockIdx.y * slice_len, j1 = min(nj, j0 + slice_len);
    double ax = 0, ay = 0, az = 0, jx = 0, jy = 0, jz = 0, pot = 0;
#pragma unroll 4
    for (int j = j0 + lane; j < j1; j += 32) {
        const double dx = pos[3 * (size_t)j] - xi, dy = pos[3 * (size_t)j + 1] - yi, dz = pos[3 * (size_t)j + 2] - zi;
        const double dvx = vel[3 * (size_t)j] - vxi, dvy = vel[3 * (size_t)j + 1] - vyi, dvz = vel[3 * (size_t)j + 2] - vzi;
        const double s = fma(dz, dz, fma(dy, dy, fma(dx, dx, eps2)));
        const double rv = fma(dz, dvz, fma(dy, dvy, dx * dvx));
        double y = na_rsqrt(s);
        y = id[j] == idi ? 0.0 : y;                                      // self skipped by identity, for every output
        const double y2 = y * y, my = mass[j] * y, q = my * y2;
        const double a3 = -3.0 * (rv * y2);
        pot -= my;
        ax = fma(q, dx, ax); ay = fma(q, dy, ay); az = fma(q, dz, az);
        jx = fma(q, fma(a3, dx, dvx), jx); jy = fma(q, fma(a3, dy, dvy), jy); jz = fma(q, fma(a3, dz, dvz), jz);
    }
#pragma unroll
    for (int m = 1; m < 32; m <<= 1) {                                   // fixed butterfly order
        ax += __shfl_xor_sync(0xffffffffu, ax, m); ay += __shfl_xor_sync(0xffffffffu, ay, m); az += __shfl_xor_sync(0xffffffffu, az, m);
        jx += __shfl_xor_sync(0xffffffffu, jx, m); jy += __shfl_xor_sync(0xffffffffu, jy, m); jz += __shfl_xor_sync(0xffffffffu, jz, m);
        pot += __shfl_xor_sync(0xffffffffu, pot, m);
    }
    if (lane == 0) {
        row[0] = ax; row[1] = ay; row[2] = az; row[3] = jx; row[4] = jy; row[5] = jz; row[6] = pot; row[7] = 0.0;
    }
}

// one thread per i: rows of slices 0, 1, ..., S-1 added in that order
__global__ void __launch_bounds__(128) na_combine_kernel(const double *scratch, int ni, int S, double *acc, double *jerk, double *pot)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= ni) return;
    double v[7] = {0, 0, 0, 0, 0, 0, 0};
    for (int s = 0; s < S; ++s) {
        const double2 *r = reinterpret_cast<const double2 *>(scratch + ((size_t)s * ni + i) * kNaRow);
        const double2 r0 = r[0], r1 = r[1], r2 = r[2], r3 = r[3];
        v[0] += r0.x; v[1] += r0.y; v[2] += r1.x; v[3] += r1.y; v[4] += r2.x; v[5] += r2.y; v[6] += r3.x;
    }
    acc[3 * (size_t)i] = v[0]; acc[3 * (size_t)i + 1] = v[1]; acc[3 * (size_t)i + 2] = v[2];
    jerk[3 * (size_t)i] = v[3]; jerk[3 * (size_t)i + 1] = v[4]; jerk[3 * (size_t)i + 2] = v[5];
    pot[i] = v[6];
}

// Device address of the scratch array, looked up once per device WITH THAT DEVICE CURRENT (the caller has set it).
std::mutex g_na_mu;
double *g_na_ptr[kNaMaxDevices];
int g_na_sms[kNaMaxDevices];

cudaError_t na_scratch_ptr(int device, double **ptr, int *sms)
{
    std::lock_guard<std::mutex> lock(g_na_mu);
    if (!g_na_ptr[device]) {
        double *p = nullptr;
        cudaError_t e = cudaGetSymbolAddress((void **)&p, g_na_scratch);
        if (e != cudaSuccess) return e;
        int n = 0;
        e = cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, device);
        if (e != cudaSuccess) return e;
        g_na_ptr[device] = p;
        g_na_sms[device] = n;
    }
    *ptr = g_na_ptr[device];
    *sms = g_na_sms[device];
    return cudaSuccess;
}

}  // namespace

extern "C" int s2_noalloc_limits(int *max_ni, long long *scratch_bytes)
{
    if (max_ni) *max_ni = kNaMaxNi;
    if (scratch_bytes) *scratch_bytes = (long long)kNaScratchBytes;
    return S2_OK;
}

extern "C" int s2_forces_noalloc(int device, void *cuda_stream, int nj, const double *d_pos, const double *d_vel,
                                 const double *d_mass, const int *d_id, int ni, const int *d_i_address, double eps2,
                                 double *d_acc, double *d_jerk, double *d_pot)
{
    if (nj <= 0 || ni <= 0 || !d_pos || !d_vel || !d_mass || !d_id || !d_i_address || !d_acc || !d_jerk || !d_pot)
        return S2_EINVAL;
    if (ni > kNaMaxNi) return S2_ERANGE;                 // beyond the fixed scratch: use the context calls (s2_calc_ilist*)
    if (device < 0 || device >= kNaMaxDevices) return S2_ERANGE;
    if (cudaSetDevice(device) != cudaSuccess) {
        cudaGetLastError();
        return S2_ECUDA;                                 // no CPU fallback
    }
    double *scratch = nullptr;
    int sms = 0;
    if (na_scratch_ptr(device, &scratch, &sms) != cudaSuccess) {
        cudaGetLastError();
        return S2_ECUDA;
    }
    // j-slices: enough CTAs for four per SM, at least 64 j per slice, and S * n_i rows within the scratch
    const int gi = (ni + kNaWarps - 1) / kNaWarps;
    int S = (4 * sms + gi - 1) / gi;
    S = S < 1 ? 1 : S;
    if (S > nj / 64) S = nj / 64 > 0 ? nj / 64 : 1;
    if (S > kNaMaxRows / ni) S = kNaMaxRows / ni;
    if (S > 65535) S = 65535;
    const int slice_len = (nj + S - 1) / S;
    S = (nj + slice_len - 1) / slice_len;                // no empty slices
    cudaStream_t st = (cudaStream_t)cuda_stream;
    na_sweep_kernel<<<dim3(gi, S), 32 * kNaWarps, 0, st>>>(d_pos, d_vel, d_mass, d_id, nj, d_i_address, ni, eps2, slice_len, scratch);
    na_combine_kernel<<<(ni + 127) / 128, 128, 0, st>>>(scratch, ni, S, d_acc, d_jerk, d_pot);
    if (cudaGetLastError() != cudaSuccess) return S2_ECUDA;
    return S2_OK;
}
