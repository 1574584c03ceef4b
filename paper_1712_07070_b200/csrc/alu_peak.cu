// alu_peak.cu -- measurement helper (include/gamer_hydro.h: gamer_alu_peak): dependent-free instruction streams
// that give the plain-ALU roofs the hydro kernels are measured against ("measure with an FMA
// micro-benchmark at the clock the hydro kernel actually sustains").  Not part of the solver.
//
// Every thread carries NCH independent chains; operands come from memory so that nothing folds at compile time,
// and the result is stored behind a condition that never holds so that nothing is dead.  148 SMs x 2 CTAs x 1024
// threads = 16 warps per sub-partition: latency is fully hidden, the number is the issue / pipe limit.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/gamer_hydro.h"

namespace gamer {

constexpr int NCH = 8;        // independent chains per thread
constexpr int UNROLL = 16;    // stream instructions per chain and loop trip

template <int KIND> struct Stream;

// fp32 FMA, three register operands (FFMA R, R, R, R)
template <> struct Stream<GAMER_ALU_FFMA> {
    typedef float T;
    static constexpr double FLOPS = 2.0, INSTS = 1.0;
    static __device__ __forceinline__ void op(float& a, float b, float c) { a = fmaf(a, b, c); }
};
// fp32 multiply then add, kept apart (FMUL + FADD): 1 FLOP per issue slot -- the mix of a kernel whose products and
// sums do not pair up
template <> struct Stream<GAMER_ALU_FMUL_FADD> {
    typedef float T;
    static constexpr double FLOPS = 2.0, INSTS = 2.0;
    static __device__ __forceinline__ void op(float& a, float b, float c) {
        a = __fadd_rn(__fmul_rn(a, b), c);
    }
};
// fp32 FMA + min/max (FFMA on the FMA pipe, FMNMX on the ALU pipe): do the two pipes issue in the same clock?
template <> struct Stream<GAMER_ALU_FFMA_FMNMX> {
    typedef float T;
    static constexpr double FLOPS = 2.0, INSTS = 2.0;
    static __device__ __forceinline__ void op(float& a, float b, float c) { a = fminf(fmaf(a, b, c), b); }
};
// packed fp32 FMA (fma.rn.f32x2, Blackwell): two FMAs per instruction
template <> struct Stream<GAMER_ALU_FFMA2> {
    typedef float2 T;
    static constexpr double FLOPS = 4.0, INSTS = 1.0;
    static __device__ __forceinline__ void op(float2& a, float2 b, float2 c) {
        uint64_t ra, rb, rc;
        asm("mov.b64 %0, {%1, %2};" : "=l"(ra) : "f"(a.x), "f"(a.y));
        asm("mov.b64 %0, {%1, %2};" : "=l"(rb) : "f"(b.x), "f"(b.y));
        asm("mov.b64 %0, {%1, %2};" : "=l"(rc) : "f"(c.x), "f"(c.y));
        asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(ra) : "l"(ra), "l"(rb), "l"(rc));
        asm("mov.b64 {%0, %1}, %2;" : "=f"(a.x), "=f"(a.y) : "l"(ra));
    }
};
// packed fp32 FMA + min/max
template <> struct Stream<GAMER_ALU_FFMA2_FMNMX> {
    typedef float2 T;
    static constexpr double FLOPS = 4.0, INSTS = 3.0;
    static __device__ __forceinline__ void op(float2& a, float2 b, float2 c) {
        Stream<GAMER_ALU_FFMA2>::op(a, b, c);
        a.x = fminf(a.x, b.x);
        a.y = fminf(a.y, b.y);
    }
};
// one packed FMA to two plain ones: 4 FMAs in 3 issue slots
template <> struct Stream<GAMER_ALU_FFMA2_FFMA> {
    typedef float2 T;
    static constexpr double FLOPS = 8.0, INSTS = 3.0;
    static __device__ __forceinline__ void op(float2& a, float2 b, float2 c) {
        Stream<GAMER_ALU_FFMA2>::op(a, b, c);
        a.x = fmaf(a.x, b.x, c.x);
        a.y = fmaf(a.y, b.y, c.y);
    }
};
// packed FMA + one integer add (IADD3 on the ALU pipe) on a side chain
template <> struct Stream<GAMER_ALU_FFMA2_IADD> {
    typedef float2 T;
    static constexpr double FLOPS = 4.0, INSTS = 2.0;
    static __device__ __forceinline__ void op(float2& a, float2 b, float2 c) {
        Stream<GAMER_ALU_FFMA2>::op(a, b, c);
        a.y = __int_as_float(__float_as_int(a.y) + __float_as_int(b.y));      // the .y lane carries integer garbage: only rates matter
    }
};
// fp64 FMA
template <> struct Stream<GAMER_ALU_DFMA> {
    typedef double T;
    static constexpr double FLOPS = 2.0, INSTS = 1.0;
    static __device__ __forceinline__ void op(double& a, double b, double c) { a = fma(a, b, c); }
};
// fp32 reciprocal approximation (MUFU.RCP) interleaved 1:8 with FMAs: the special-function unit beside the FMA pipe
template <> struct Stream<GAMER_ALU_FFMA_MUFU> {
    typedef float T;
    static constexpr double FLOPS = 2.0 * 8.0 / 9.0, INSTS = 1.0;      // per stream slot, averaged
    static __device__ __forceinline__ void op(float& a, float b, float c) { a = fmaf(a, b, c); }
};

__device__ __forceinline__ float make_val(const float* p, int i, float*) { return p[i]; }
__device__ __forceinline__ double make_val(const float* p, int i, double*) { return (double)p[i]; }
__device__ __forceinline__ float2 make_val(const float* p, int i, float2*) { return make_float2(p[i], p[i + 1]); }
__device__ __forceinline__ bool is_magic(float v) { return v == 123456.0f; }
__device__ __forceinline__ bool is_magic(double v) { return v == 123456.0; }
__device__ __forceinline__ bool is_magic(float2 v) { return v.x == 123456.0f && v.y == 654321.0f; }
__device__ __forceinline__ float to_float(float v) { return v; }
__device__ __forceinline__ float to_float(double v) { return (float)v; }
__device__ __forceinline__ float to_float(float2 v) { return v.x + v.y; }

template <int KIND>
__global__ void __launch_bounds__(1024, 2) alu_stream_kernel(const float* __restrict__ seed, float* __restrict__ sink, int trips) {
    typedef typename Stream<KIND>::T T;
    T a[NCH];
    const T b = make_val(seed, 0, (T*)nullptr), c = make_val(seed, 2, (T*)nullptr);
#pragma unroll
    for (int k = 0; k < NCH; ++k) a[k] = make_val(seed, 4 + ((threadIdx.x + k) & 7), (T*)nullptr);
    for (int t = 0; t < trips; ++t) {
#pragma unroll
        for (int u = 0; u < UNROLL; ++u) {
#pragma unroll
            for (int k = 0; k < NCH; ++k) {
                if (KIND == GAMER_ALU_FFMA_MUFU && ((u * NCH + k) % 9) == 8) {
                    float r;
                    float x = to_float(a[k]);
                    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
                    a[k] = make_val(&r, 0, (T*)nullptr);      // KIND's T is float here
                } else {
                    Stream<KIND>::op(a[k], b, c);
                }
            }
        }
    }
    bool hit = false;
#pragma unroll
    for (int k = 0; k < NCH; ++k) hit = hit || is_magic(a[k]);
    if (hit) {
        float s = 0.f;
#pragma unroll
        for (int k = 0; k < NCH; ++k) s += to_float(a[k]);
        sink[blockIdx.x * blockDim.x + threadIdx.x] = s;
    }
}

template <int KIND>
static int run_stream(double* tflops, double* ginst, cudaStream_t st) {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return GAMER_ECUDA;
    const int grid = sms * 2, block = 1024, trips = 2048;
    float h[16] = {0.999f, 0.998f, 1e-3f, 2e-3f, 1.0f, 1.1f, 1.2f, 1.3f, 1.4f, 1.5f, 1.6f, 1.7f, 1.8f, 0, 0, 0};
    float *seed = nullptr, *sink = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = GAMER_ECUDA;
    float best = 0.f;
    if (cudaMalloc(&seed, sizeof(h)) != cudaSuccess) goto done;
    if (cudaMalloc(&sink, sizeof(float) * grid * block) != cudaSuccess) goto done;
    if (cudaMemcpyAsync(seed, h, sizeof(h), cudaMemcpyHostToDevice, st) != cudaSuccess) goto done;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) goto done;
    alu_stream_kernel<KIND><<<grid, block, 0, st>>>(seed, sink, trips / 8);      // warm-up, clocks up
    for (int rep = 0; rep < 5; ++rep) {
        float ms = 0.f;
        cudaEventRecord(e0, st);
        alu_stream_kernel<KIND><<<grid, block, 0, st>>>(seed, sink, trips);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess || cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess) goto done;
        if (rep == 0 || ms < best) best = ms;
    }
    if (cudaGetLastError() != cudaSuccess) goto done;
    {
        const double slots = (double)grid * block * (double)trips * UNROLL * NCH;
        if (tflops) *tflops = slots * Stream<KIND>::FLOPS / (best * 1e-3) / 1e12;
        if (ginst) *ginst = slots * Stream<KIND>::INSTS / 32.0 / (best * 1e-3) / 1e9;
        rc = GAMER_OK;
    }
done:
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (seed) cudaFree(seed);
    if (sink) cudaFree(sink);
    return rc;
}

}  // namespace gamer

extern "C" int gamer_alu_peak(int kind, double* tflops_out, double* gwarpinst_out, void* stream) {
    using namespace gamer;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    switch (kind) {
    case GAMER_ALU_FFMA: return run_stream<GAMER_ALU_FFMA>(tflops_out, gwarpinst_out, st);
    case GAMER_ALU_FMUL_FADD: return run_stream<GAMER_ALU_FMUL_FADD>(tflops_out, gwarpinst_out, st);
    case GAMER_ALU_FFMA_FMNMX: return run_stream<GAMER_ALU_FFMA_FMNMX>(tflops_out, gwarpinst_out, st);
    case GAMER_ALU_FFMA2: return run_stream<GAMER_ALU_FFMA2>(tflops_out, gwarpinst_out, st);
    case GAMER_ALU_FFMA2_FMNMX: return run_stream<GAMER_ALU_FFMA2_FMNMX>(tflops_out, gwarpinst_out, st);
    case GAMER_ALU_DFMA: return run_stream<GAMER_ALU_DFMA>(tflops_out, gwarpinst_out, st);
    case GAMER_ALU_FFMA_MUFU: return run_stream<GAMER_ALU_FFMA_MUFU>(tflops_out, gwarpinst_out, st);
    case GAMER_ALU_FFMA2_FFMA: return run_stream<GAMER_ALU_FFMA2_FFMA>(tflops_out, gwarpinst_out, st);
    case GAMER_ALU_FFMA2_IADD: return run_stream<GAMER_ALU_FFMA2_IADD>(tflops_out, gwarpinst_out, st);
    default: return GAMER_EINVAL;
    }
}
