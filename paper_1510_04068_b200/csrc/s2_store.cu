// s2_store.cu -- a1 (commit: scatter staged particles into the fp64 SoA j-store) and
// a2 (Taylor predictor) kernels.  PAPER.md L88: "one copy kernel to move particles from CPU
// buffers to GPU buffers, one kernel to predict the particles to the new time-step".
// Both are pure streaming kernels: HBM-bound.
#include "s2_internal.h"
#include "s2_predict.cuh"

namespace s2 {

// One thread per staged particle; a warp reads contiguous rows of the staged arrays and writes to `address`
// (contiguous when the host sends address-ordered sets).
__global__ void __launch_bounds__(256) scatter_kernel(ScatterArgs a)
{
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= a.n) return;
    int addr = a.address[p];
    if (addr < 0 || addr >= a.nj_cap) {
        *a.erange_flag = 1;
        return;
    }
    a.dst_id[addr] = a.id[p];
#pragma unroll
    for (int f = 0; f < kMaxFields; ++f) {
        if (f < a.nfields) {
            // scalars (t, m): plain length-n arrays; vector components: (n,3) row-major, src already offset by the
            // component, so the three loads of a thread cover one contiguous 24-byte row
            // a missing field (2nd-order context committed without acc / jerk) is stored as zero
            const double v = !a.src[f] ? 0.0 : (f < 2 ? a.src[f][p] : a.src[f][(size_t)3 * p]);
            a.dst[f][addr] = v;
        }
    }
}

cudaError_t launch_scatter(const ScatterArgs &a, cudaStream_t st)
{
    if (a.n <= 0) return cudaSuccess;
    scatter_kernel<<<(a.n + 255) / 256, 256, 0, st>>>(a);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// Predictor (a2): one thread per j, arithmetic in predict_one (s2_predict.cuh).

template <int ORDER>
__global__ void __launch_bounds__(256) predict_kernel(PredictArgs a)
{
    asm volatile("griddepcontrol.wait;" ::: "memory");   // no-op unless launched with programmatic stream serialisation
    int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= a.nj) return;
    predict_one<ORDER>(a, j, a.t_dev ? *a.t_dev : a.t);
}

cudaError_t launch_predict(const PredictArgs &a, cudaStream_t st)
{
    if (a.nj <= 0) return cudaSuccess;
    const int grid = (a.nj + 255) / 256;
    if (a.pdl) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(grid); cfg.blockDim = dim3(256); cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        return a.order == 6 ? cudaLaunchKernelEx(&cfg, predict_kernel<6>, a) : cudaLaunchKernelEx(&cfg, predict_kernel<4>, a);
    }
    if (a.order == 6)
        predict_kernel<6><<<grid, 256, 0, st>>>(a);
    else
        predict_kernel<4><<<grid, 256, 0, st>>>(a);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// Peak microbenchmarks (roofline denominators and the FP64 operand-path model of DESIGN.md 5.2):
// 8 independent chains per thread, 64 warps per SM.
//   kind 0  DFMA  a = fma(a, c1, c2), c1/c2 compile-time constants       (nominal FP64 rate)
//   kind 1  FFMA  same in fp32
//   kind 2  DFMA  a_k = fma(b_k, b_k+1, a_k): three distinct 64-bit register operands
//   kind 3  DFMA  a_k = fma(q, b_k, a_k): one operand shared by consecutive instructions (reuse cache)
//   kind 4  DADD  a_k = a_k + b_k: two distinct register operands
template <typename T, int MODE>
__global__ void __launch_bounds__(256) peak_fma_kernel(T *out, int iters, T seed)
{
    T a[8], b[8];
    const T q = (T)0.999999 + seed * (T)1e-9;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        a[k] = seed + (T)(threadIdx.x + k);
        b[k] = (T)1.0 + (T)1e-9 * (T)(threadIdx.x + k) * seed;
    }
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                if (MODE == 0) a[k] = fma(a[k], (T)0.999999, (T)1e-7);
                if (MODE == 2) a[k] = fma(b[k], b[(k + 1) & 7], a[k]);
                if (MODE == 3) a[k] = fma(q, b[k], a[k]);
                if (MODE == 4) a[k] = a[k] + b[k];
            }
        }
    }
    T s = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += a[k] + b[k];
    if (s == (T)123456.789) out[blockIdx.x * blockDim.x + threadIdx.x] = s;   // never true; keeps the chains live
}

// Packed FP32 (FFMA2 / FADD2, PTX fma/add.rn.f32x2): the same 8 chains per thread, each a register PAIR, so one
// instruction carries two lane-operations; *fma_per_s counts lane-operations (2 per lane and instruction).
//   kind 5  FFMA2  a = fma2(a, c1, c2), constants                       (packed rate with free operands)
//   kind 6  FFMA2  a_k = fma2(b_k, b_k+1, a_k): three distinct register pairs
//   kind 7  FFMA2  a_k = fma2(q, b_k, a_k), q a 32-bit register broadcast to both halves (the j operand of the sweep)
//   kind 8  FADD2  a_k = a_k + b_k: two distinct register pairs
typedef unsigned long long pk_f32x2;
__device__ __forceinline__ pk_f32x2 pk_make(float lo, float hi)
{
    pk_f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ pk_f32x2 pk_fma(pk_f32x2 a, pk_f32x2 b, pk_f32x2 c)
{
    pk_f32x2 d;
    asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ pk_f32x2 pk_add(pk_f32x2 a, pk_f32x2 b)
{
    pk_f32x2 d;
    asm volatile("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
template <int MODE>
__global__ void __launch_bounds__(256) peak_fma2_kernel(float *out, int iters, float seed)
{
    pk_f32x2 a[8], b[8];
    const float qs = 0.999999f + seed * 1e-9f;
    const pk_f32x2 q = pk_make(qs, qs);
    const pk_f32x2 c1 = pk_make(0.999999f, 0.999999f), c2 = pk_make(1e-7f, 1e-7f);
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        a[k] = pk_make(seed + (float)(threadIdx.x + k), seed + (float)(threadIdx.x + k + 8));
        b[k] = pk_make(1.0f + 1e-7f * (float)(threadIdx.x + k) * seed, 1.0f + 1e-7f * (float)(threadIdx.x + k + 8) * seed);
    }
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                if (MODE == 5) a[k] = pk_fma(a[k], c1, c2);
                if (MODE == 6) a[k] = pk_fma(b[k], b[(k + 1) & 7], a[k]);
                if (MODE == 7) a[k] = pk_fma(q, b[k], a[k]);
                if (MODE == 8) a[k] = pk_add(a[k], b[k]);
            }
        }
    }
    pk_f32x2 s = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s ^= a[k] ^ b[k];
    if (s == 0x123456789abcdefull) out[blockIdx.x * blockDim.x + threadIdx.x] = 1.f;   // never true; keeps the chains live
}

cudaError_t run_peak_fma(int kind, int iters, int sm_count, cudaStream_t st, double *fma_per_s)
{
    cudaEvent_t e0, e1;
    cudaError_t err;
    if ((err = cudaEventCreate(&e0)) != cudaSuccess) return err;
    if ((err = cudaEventCreate(&e1)) != cudaSuccess) return err;
    const int grid = sm_count * 8, block = 256;   // 64 warps per SM
    void *dummy = nullptr;
    for (int rep = 0; rep < 2; ++rep) {           // first pass warms up
        if (rep == 1) cudaEventRecord(e0, st);
        switch (kind) {
        case 0: peak_fma_kernel<double, 0><<<grid, block, 0, st>>>((double *)dummy, iters, 1.0); break;
        case 1: peak_fma_kernel<float, 0><<<grid, block, 0, st>>>((float *)dummy, iters, 1.0f); break;
        case 2: peak_fma_kernel<double, 2><<<grid, block, 0, st>>>((double *)dummy, iters, 1.0); break;
        case 3: peak_fma_kernel<double, 3><<<grid, block, 0, st>>>((double *)dummy, iters, 1.0); break;
        case 5: peak_fma2_kernel<5><<<grid, block, 0, st>>>((float *)dummy, iters, 1.0f); break;
        case 6: peak_fma2_kernel<6><<<grid, block, 0, st>>>((float *)dummy, iters, 1.0f); break;
        case 7: peak_fma2_kernel<7><<<grid, block, 0, st>>>((float *)dummy, iters, 1.0f); break;
        case 8: peak_fma2_kernel<8><<<grid, block, 0, st>>>((float *)dummy, iters, 1.0f); break;
        default: peak_fma_kernel<double, 4><<<grid, block, 0, st>>>((double *)dummy, iters, 1.0); break;
        }
    }
    cudaEventRecord(e1, st);
    err = cudaEventSynchronize(e1);
    if (err == cudaSuccess) err = cudaGetLastError();
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (err != cudaSuccess) return err;
    const double fmas = (double)grid * block * (double)iters * 16.0 * 8.0 * (kind >= 5 && kind <= 8 ? 2.0 : 1.0);
    *fma_per_s = fmas / (ms * 1e-3);
    return cudaSuccess;
}

// ---- hop latency between SMs through L2 (s2_hop_latency, s2b200_test.h) --------------------------------------
// CTA 0 stores a 64-bit word; every other CTA polls that word and answers in a word of its own (128 bytes apart);
// CTA 0 polls all answers (one thread each): one round trip = one store fanned out to all SMs + one gather = two hops.
// Relaxed gpu-scope loads and stores, no fences: the floor of any exchange between CTAs that live on different SMs.
__global__ void __launch_bounds__(256) hop_kernel(unsigned long long *buf, int iters, long long *cycles)
{
    const int cta = blockIdx.x, G = gridDim.x, tid = threadIdx.x;
    unsigned long long *flag = buf, *rep = buf + 16;
    auto ld = [](const unsigned long long *p) {
        unsigned long long v;
        asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
        return v;
    };
    auto st = [](unsigned long long *p, unsigned long long v) { asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory"); };
    const long long t0 = clock64();
    for (int i = 1; i <= iters; ++i) {
        if (cta == 0) {
            if (tid == 0) st(flag, (unsigned long long)i);
            for (int c = 1 + tid; c < G; c += blockDim.x) {
                unsigned spins = 0;
                while (ld(rep + (size_t)c * 16) != (unsigned long long)i && ++spins < (1u << 22)) {}
            }
            __syncthreads();
        } else if (tid == 0) {
            unsigned spins = 0;
            while (ld(flag) != (unsigned long long)i && ++spins < (1u << 22)) {}
            st(rep + (size_t)cta * 16, (unsigned long long)i);
        }
    }
    if (cta == 0 && tid == 0) *cycles = clock64() - t0;
}

cudaError_t run_hop_latency(int ctas, int iters, unsigned long long *buf, long long *d_cycles, cudaStream_t st)
{
    void *args[3] = {(void *)&buf, (void *)&iters, (void *)&d_cycles};
    return cudaLaunchCooperativeKernel((const void *)hop_kernel, dim3(ctas), dim3(256), args, 0, st);
}

}  // namespace s2
