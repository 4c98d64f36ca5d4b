// libnbody.so, translation unit 3: micro-probes of the instruction classes K_force is made of (include/nbody_bench.h).
// They give the "measured" denominators beside the nominal FP32 peak: thread-operations
// per second of FFMA, DADD, F2F (fp64 -> fp32), MUFU.RSQ, the DADD+F2F pair and packed FFMA2, each on every SM at
// once, and the issue-port probes (kinds 7..9): one packed FFMA2 next to one instruction of another pipe, which
// show whether that instruction is hidden behind the FFMA2's second pipe cycle or costs an issue cycle of its own.
#include "nbody_bench.h"
#include "nbody_internal.h"

namespace nbody {
namespace {

constexpr int kProbeIters = 4096;
constexpr int kProbeChains = 8;

template <int KIND>
__global__ void __launch_bounds__(256) k_probe(float *sink, float seed, unsigned long long *clk) {
    unsigned long long c0 = 0, g0 = 0;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
        c0 = clock64();
    }
    float f[kProbeChains];
    double d[kProbeChains];
    unsigned x[kProbeChains];
    __shared__ uint4 sm[64];
    if (KIND == 9) {
        if (threadIdx.x < 64) sm[threadIdx.x] = make_uint4(threadIdx.x, 1u, 2u, 3u);
        __syncthreads();
    }
    const unsigned sm_base = (unsigned)__cvta_generic_to_shared(sm);
#pragma unroll
    for (int c = 0; c < kProbeChains; ++c) {
        f[c] = seed + (float)(threadIdx.x + c);
        d[c] = (double)seed + (double)(threadIdx.x * 3 + c);
        x[c] = threadIdx.x * 7u + c;
    }
    unsigned long long p2[kProbeChains], p2c[kProbeChains], p2d[kProbeChains], p2b;
#pragma unroll
    for (int c = 0; c < kProbeChains; ++c) {
        asm("mov.b64 %0, {%1, %2};" : "=l"(p2[c]) : "f"(seed + c), "f"(seed - c));
        asm("mov.b64 %0, {%1, %2};" : "=l"(p2c[c]) : "f"(1e-3f * c + seed), "f"(2e-3f));
        asm("mov.b64 %0, {%1, %2};" : "=l"(p2d[c]) : "f"(0.999f + seed * c), "f"(0.998f + seed * c));
    }
    asm("mov.b64 %0, {%1, %2};" : "=l"(p2b) : "f"(0.999f + seed), "f"(0.998f + seed));
    const float b = 0.999f + seed, cc = 1e-3f;
    const double db = 1e-3 + (double)seed;
#pragma unroll 8
    for (int it = 0; it < kProbeIters; ++it) {
#pragma unroll
        for (int c = 0; c < kProbeChains; ++c) {
            if (KIND == 0) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[c]) : "f"(b), "f"(cc));
            if (KIND == 1) asm volatile("add.rn.f64 %0, %0, %1;" : "+d"(d[c]) : "d"(db));
            if (KIND == 2) {  // dependent round trip fp64 -> fp32 -> fp64 (two conversions)
                asm volatile("cvt.rn.f32.f64 %0, %1;" : "=f"(f[c]) : "d"(d[c]));
                asm volatile("cvt.f64.f32 %0, %1;" : "=d"(d[c]) : "f"(f[c]));
            }
            if (KIND == 3) asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(f[c]));
            if (KIND == 5)  // packed FFMA2, two fresh 64-bit operands (one shared): the pair loop's common form
                asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(p2[c]) : "l"(p2b), "l"(p2c[c]));
            if (KIND == 6)  // packed FFMA2, three fresh 64-bit operands
                asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(p2[c]) : "l"(p2d[c]), "l"(p2c[c]));
            if (KIND >= 7 && KIND <= 9) {  // one packed FFMA2 + one instruction of another pipe (independent chains)
                asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(p2[c]) : "l"(p2b), "l"(p2c[c]));
                if (KIND == 7) asm volatile("shf.l.wrap.b32 %0, %0, %1, 3;" : "+r"(x[c]) : "r"(x[(c + 1) % kProbeChains]));
                if (KIND == 8) asm volatile("add.rn.f64 %0, %0, %1;" : "+d"(d[c]) : "d"(db));
                if (KIND == 9) {
                    unsigned a0, a1, a2, a3;
                    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                                 : "=r"(a0), "=r"(a1), "=r"(a2), "=r"(a3)
                                 : "r"(sm_base + (((unsigned)it + c) & 63u) * 16u));
                    x[c] ^= a0 ^ a1 ^ a2 ^ a3;
                }
            }
            if (KIND == 4) {  // the literal difference pattern: DADD, F2F, and an FADD that consumes it
                double t;
                float g;
                asm volatile("add.rn.f64 %0, %1, %2;" : "=d"(t) : "d"(d[c]), "d"(db));
                asm volatile("cvt.rn.f32.f64 %0, %1;" : "=f"(g) : "d"(t));
                asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(f[c]) : "f"(g));
                d[c] = t;
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < kProbeChains; ++c) {
        float lo, hi, lo2, hi2, lo3, hi3;
        asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(p2[c]));
        asm("mov.b64 {%0, %1}, %2;" : "=f"(lo2), "=f"(hi2) : "l"(p2c[c]));
        asm("mov.b64 {%0, %1}, %2;" : "=f"(lo3), "=f"(hi3) : "l"(p2d[c]));
        s += f[c] + (float)d[c] + lo + hi + lo2 + hi2 + lo3 + hi3 + __uint_as_float(x[c]);
    }
    if (s == 123.456f) sink[0] = s;  // never true in practice; keeps the chains live
    if (blockIdx.x == 0 && threadIdx.x == 0) {  // SM cycles and nanoseconds this CTA ran: the SM clock under this load
        unsigned long long g1;
        const unsigned long long c1 = clock64();
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
        clk[0] = c1 - c0;
        clk[1] = g1 - g0;
    }
}

typedef void (*probe_fn)(float *, float, unsigned long long *);
const probe_fn kProbes[10] = {k_probe<0>, k_probe<1>, k_probe<2>, k_probe<3>, k_probe<4>,
                              k_probe<5>, k_probe<6>, k_probe<7>, k_probe<8>, k_probe<9>};

}  // namespace

int probe_peak(Ctx *c, int kind, int millis, double *tera_ops) {
    DeviceGuard guard(c->device);
    float *sink = nullptr;
    NB_CUDA(c, cudaMalloc(&sink, sizeof(float) + 2 * sizeof(unsigned long long) + 8));
    unsigned long long *clk = reinterpret_cast<unsigned long long *>(reinterpret_cast<char *>(sink) + 8);
    unsigned long long hclk[2] = {0, 0};
    double best_mhz = 0.0;
    cudaEvent_t e0, e1;
    NB_CUDA(c, cudaEventCreate(&e0));
    NB_CUDA(c, cudaEventCreate(&e1));
    const int grid = c->sm_count * 8;  // 2048 threads per SM
    const double ops_per_launch = (double)grid * 256.0 * kProbeIters * kProbeChains * (kind == 4 ? 3.0 : kind == 2 ? 2.0 : 1.0);
    double best = 0.0, spent = 0.0;
    int rc = NBODY_OK;
    for (int rep = 0; rep < 100000 && spent < (double)millis; ++rep) {
        cudaEventRecord(e0, 0);
        kProbes[kind]<<<grid, 256>>>(sink, 0.0f, clk);
        c->launches += 1;
        cudaEventRecord(e1, 0);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { rc = cuda_fail(c, e); break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        spent += ms;
        if (rep > 0 && ms > 0.f) {
            const double rate = ops_per_launch / (ms * 1e-3) / 1e12;
            if (rate > best) {
                best = rate;
                if (cudaMemcpy(hclk, clk, sizeof(hclk), cudaMemcpyDeviceToHost) == cudaSuccess && hclk[1] > 0)
                    best_mhz = (double)hclk[0] / (double)hclk[1] * 1e3;
            }
        }
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    tera_ops[0] = best;
    tera_ops[1] = best_mhz;
    return rc;
}

}  // namespace nbody

extern "C" int nbody_probe_peak(nbody_ctx *h, int kind, int millis, double *tera_ops_host) {
    if (!h || !tera_ops_host || kind < 0 || kind > 9 || millis < 1 || millis > 20000) return NBODY_EINVAL;
    return nbody::probe_peak(&h->c, kind, millis, tera_ops_host);
}
