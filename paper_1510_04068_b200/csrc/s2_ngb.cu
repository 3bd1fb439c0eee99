// s2_ngb.cu -- a8 / a9: device-side compaction of the neighbour lists of one force call into CSR form
// ("count -> scan -> fill"; sec 3 "a list of particles within a given radius").
//
// The sweep (and the reduce) leave the lists in a fixed-stride buffer list[n_i][ngb_cap] with the true counts in the
// result records.  At config 5 that buffer is 1 GiB for ~135 MB of members (mean 32 of cap 256), so reading it back
// as it stands moves 8x the payload over the host link.  Here:
//   csr_len_kernel      len[i] = min(count_i, cap) from the records, plus one partial sum per block of 2048 i
//   csr_scan_kernel     exclusive scan of the block sums (one CTA), total
//   csr_offsets_kernel  per-block exclusive scan of len -> offsets[i] (64-bit), offsets[n_i] = total
//   csr_fill_kernel     one warp per i copies its segment to out[offsets[i] ..]   (coalesced 128-byte rows)
// All four stream their inputs once: HBM-bound, algorithmic bytes = 8 B (count word) + 4 B (len) + 8 B (offset) per i
// + 8 B per list member (4 read + 4 written).
#include "s2_internal.h"

namespace s2 {

constexpr int kCsrThreads = 256;
constexpr int kCsrPerThread = 8;
constexpr int kCsrPerBlock = kCsrThreads * kCsrPerThread;   // 2048 i-particles per block

__device__ __forceinline__ int warp_incl_scan(int v, int lane)
{
#pragma unroll
    for (int m = 1; m < 32; m <<= 1) {
        const int o = __shfl_up_sync(0xffffffffu, v, m);
        if (lane >= m) v += o;
    }
    return v;
}

// thread t of block b owns the consecutive i-particles b * 2048 + t * 8 .. + 7
__global__ void __launch_bounds__(kCsrThreads) csr_len_kernel(const double *rec, int ni, int cap, int *len, long long *block_sum)
{
    __shared__ int s_w[kCsrThreads / 32];
    const int i0 = blockIdx.x * kCsrPerBlock + threadIdx.x * kCsrPerThread;
    int sum = 0;
#pragma unroll
    for (int k = 0; k < kCsrPerThread; ++k) {
        const int i = i0 + k;
        int l = 0;
        if (i < ni) {
            l = min(__double2hiint(rec[(size_t)i * REC + 8]), cap);   // record word 8 = {nn id, neighbour count}
            len[i] = l;
        }
        sum += l;
    }
#pragma unroll
    for (int m = 16; m > 0; m >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, m);
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = sum;
    __syncthreads();
    if (threadIdx.x == 0) {
        long long t = 0;
        for (int w = 0; w < kCsrThreads / 32; ++w) t += s_w[w];
        block_sum[blockIdx.x] = t;
    }
}

// one CTA: block_sum[b] <- sum of block_sum[0 .. b-1]; *total <- sum of all (sequential over chunks of 1024)
__global__ void __launch_bounds__(1024) csr_scan_kernel(long long *block_sum, int nb, long long *total)
{
    __shared__ long long s_w[32];
    __shared__ long long s_carry;
    if (threadIdx.x == 0) s_carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int b0 = 0; b0 < nb; b0 += 1024) {
        const int b = b0 + threadIdx.x;
        const long long v = b < nb ? block_sum[b] : 0;
        long long incl = v;
#pragma unroll
        for (int m = 1; m < 32; m <<= 1) {
            const long long o = __shfl_up_sync(0xffffffffu, incl, m);
            if (lane >= m) incl += o;
        }
        if (lane == 31) s_w[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            long long w = s_w[lane];
#pragma unroll
            for (int m = 1; m < 32; m <<= 1) {
                const long long o = __shfl_up_sync(0xffffffffu, w, m);
                if (lane >= m) w += o;
            }
            s_w[lane] = w;   // inclusive scan of the warp totals
        }
        __syncthreads();
        const long long base = s_carry + (warp ? s_w[warp - 1] : 0);
        if (b < nb) block_sum[b] = base + incl - v;
        __syncthreads();
        if (threadIdx.x == 1023) s_carry = base + incl;
        __syncthreads();
    }
    if (threadIdx.x == 0) *total = s_carry;
}

__global__ void __launch_bounds__(kCsrThreads) csr_offsets_kernel(const int *len, int ni, const long long *block_off,
                                                                  const long long *total, long long *offsets)
{
    __shared__ int s_w[kCsrThreads / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int i0 = blockIdx.x * kCsrPerBlock + threadIdx.x * kCsrPerThread;
    int l[kCsrPerThread], sum = 0;
#pragma unroll
    for (int k = 0; k < kCsrPerThread; ++k) {
        l[k] = i0 + k < ni ? len[i0 + k] : 0;
        sum += l[k];
    }
    const int incl = warp_incl_scan(sum, lane);
    if (lane == 31) s_w[warp] = incl;
    __syncthreads();
    int wbase = 0;
    for (int w = 0; w < warp; ++w) wbase += s_w[w];
    long long off = block_off[blockIdx.x] + wbase + incl - sum;
#pragma unroll
    for (int k = 0; k < kCsrPerThread; ++k) {
        if (i0 + k < ni) offsets[i0 + k] = off;
        off += l[k];
    }
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) offsets[ni] = *total;
}

// one warp per kFillPerWarp consecutive i: each segment (<= cap addresses) is read with all its loads issued before the
// stores of the group, so that a warp keeps several rows in flight (rows are a fixed stride apart: a row of ~32
// members is four sectors of its own)
constexpr int kFillPerWarp = 4;
__global__ void __launch_bounds__(256) csr_fill_kernel(const int *list, const int *len, const long long *offsets, int ni, int cap,
                                                       int *out)
{
    const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    const int i0 = w * kFillPerWarp;
    if (i0 >= ni) return;
    int n[kFillPerWarp], v[kFillPerWarp];
    long long off[kFillPerWarp];
#pragma unroll
    for (int u = 0; u < kFillPerWarp; ++u) {
        const int i = i0 + u;
        n[u] = i < ni ? len[i] : 0;
        off[u] = i < ni ? offsets[i] : 0;
    }
#pragma unroll
    for (int u = 0; u < kFillPerWarp; ++u)
        v[u] = lane < n[u] ? list[(size_t)(i0 + u) * cap + lane] : 0;
#pragma unroll
    for (int u = 0; u < kFillPerWarp; ++u) {
        int *dst = out + off[u];
        if (lane < n[u]) dst[lane] = v[u];
        const int *src = list + (size_t)(i0 + u) * cap;
        for (int k = lane + 32; k < n[u]; k += 32) dst[k] = src[k];   // segments longer than a warp (rare)
    }
}

cudaError_t launch_csr_scan(const double *rec, int ni, int cap, int *len, long long *block_sum, long long *total,
                            long long *offsets, cudaStream_t st)
{
    if (ni <= 0) return cudaSuccess;
    const int nb = (ni + kCsrPerBlock - 1) / kCsrPerBlock;
    csr_len_kernel<<<nb, kCsrThreads, 0, st>>>(rec, ni, cap, len, block_sum);
    csr_scan_kernel<<<1, 1024, 0, st>>>(block_sum, nb, total);
    csr_offsets_kernel<<<nb, kCsrThreads, 0, st>>>(len, ni, block_sum, total, offsets);
    return cudaGetLastError();
}

cudaError_t launch_csr_fill(const int *list, const int *len, const long long *offsets, int ni, int cap, int *out, cudaStream_t st)
{
    if (ni <= 0) return cudaSuccess;
    const long long threads = (long long)((ni + kFillPerWarp - 1) / kFillPerWarp) * 32;
    csr_fill_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(list, len, offsets, ni, cap, out);
    return cudaGetLastError();
}

int csr_blocks(int ni) { return (ni + kCsrPerBlock - 1) / kCsrPerBlock; }

}  // namespace s2
