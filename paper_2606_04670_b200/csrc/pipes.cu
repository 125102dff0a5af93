// pipes.cu -- diagnostic: measured issue rate of the fp32 instruction classes the pair kernels are made of
// (lipfit_pipe_throughput, bench.py --pipes).  DESIGN.md §7 derives the "alu" roofline peak from the unit
// counts of the guide (128 fp32 lanes per SM x clocks.max.sm); this probe is the measurement that says what
// that peak means for each SASS instruction on sm_100a: which pipe it occupies, whether the packed f32x2
// forms double the lane rate, what a 3-input FMNMX3 costs, and how far FMA-pipe and ALU-pipe instructions
// overlap.  Not on the hot path; never called by the compute entry points.
//
// Method: every resident warp runs CHAINS independent dependency chains of one instruction (inline PTX, so the
// instruction is the one named), ITER x UNROLL times; cycles = clock64() span of the slowest CTA of an SM-filling
// grid; result = lane-results per clock per SM.
#include "kernels.h"

namespace lipfit {

namespace {

constexpr int kProbeThreads = 512;
constexpr int kChains = 8;
constexpr int kUnroll = 8;

enum ProbeOp { P_FFMA = 0, P_FADD, P_FADD2, P_FFMA2, P_FMNMX, P_FMNMX3, P_MUFU_SQRT, P_FFMA_FMNMX, P_FADD2_FMNMX3,
               P_FADD_ABS, P_FADD2_FMNMX, P_FFMA_FMNMX3, P_2FADD2_FMNMX3, P_FADD2_2FMNMX3, P_FADD2_FADD,
               P_2FFMA_FMNMX3, P_COUNT };

template <int OP>
__global__ void __launch_bounds__(kProbeThreads)
pipe_probe_kernel(int iters, float seed, float* __restrict__ sink, long long* __restrict__ cycles) {
    float a[kChains], b[kChains];
    unsigned long long p[kChains];
#pragma unroll
    for (int c = 0; c < kChains; ++c) {
        a[c] = seed + static_cast<float>(threadIdx.x + c);
        b[c] = seed * 0.5f + static_cast<float>(c);
        p[c] = (static_cast<unsigned long long>(__float_as_uint(a[c])) << 32) | __float_as_uint(b[c]);
    }
    const float k1 = seed * 1.0000001f, k2 = seed * 0.9999999f;
    const unsigned long long kp = (static_cast<unsigned long long>(__float_as_uint(k1)) << 32) | __float_as_uint(k2);
    __syncthreads();
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < kUnroll; ++u) {
#pragma unroll
            for (int c = 0; c < kChains; ++c) {
                if (OP == P_FFMA) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[c]) : "f"(k1), "f"(k2));
                if (OP == P_FADD) asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(a[c]) : "f"(k1));
                if (OP == P_FADD_ABS) asm volatile("{.reg .f32 t; abs.f32 t, %0; add.rn.f32 %0, t, %1;}" : "+f"(a[c]) : "f"(k1));
                if (OP == P_FADD2) asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(p[c]) : "l"(kp));
                if (OP == P_FFMA2) asm volatile("fma.rn.f32x2 %0, %0, %1, %1;" : "+l"(p[c]) : "l"(kp));
                // (the second operand is a neighbouring chain: every result has two consumers, so ptxas cannot
                // merge two dependent 2-input minima into one FMNMX3)
                if (OP == P_FMNMX) asm volatile("min.f32 %0, %0, %1;" : "+f"(a[c]) : "f"(a[(c + 1) % kChains]));
                if (OP == P_FMNMX3) asm volatile("min.f32 %0, %0, %1, %2;" : "+f"(a[c]) : "f"(b[c]), "f"(k1));
                if (OP == P_MUFU_SQRT) asm volatile("sqrt.approx.ftz.f32 %0, %0;" : "+f"(a[c]));
                if (OP == P_FFMA_FMNMX) {  // one FMA-pipe and one ALU-pipe instruction per slot pair
                    asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[c]) : "f"(k1), "f"(k2));
                    asm volatile("min.f32 %0, %0, %1;" : "+f"(b[c]) : "f"(b[(c + 1) % kChains]));
                }
                if (OP == P_FADD2_FMNMX3) {
                    asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(p[c]) : "l"(kp));
                    asm volatile("min.f32 %0, %0, %1, %2;" : "+f"(a[c]) : "f"(b[c]), "f"(k1));
                }
                if (OP == P_FADD2_FMNMX) {
                    asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(p[c]) : "l"(kp));
                    asm volatile("min.f32 %0, %0, %1;" : "+f"(b[c]) : "f"(b[(c + 1) % kChains]));
                }
                if (OP == P_FFMA_FMNMX3) {
                    asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(b[c]) : "f"(k1), "f"(k2));
                    asm volatile("min.f32 %0, %0, %1, %2;" : "+f"(a[c]) : "f"(k2), "f"(k1));
                }
                if (OP == P_2FADD2_FMNMX3) {
                    asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(p[c]) : "l"(kp));
                    asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(p[c]) : "l"(kp));
                    asm volatile("min.f32 %0, %0, %1, %2;" : "+f"(a[c]) : "f"(b[c]), "f"(k1));
                }
                if (OP == P_FADD2_2FMNMX3) {
                    asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(p[c]) : "l"(kp));
                    asm volatile("min.f32 %0, %0, %1, %2;" : "+f"(a[c]) : "f"(k2), "f"(k1));
                    asm volatile("min.f32 %0, %0, %1, %2;" : "+f"(b[c]) : "f"(k2), "f"(k1));
                }
                if (OP == P_FADD2_FADD) {
                    asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(p[c]) : "l"(kp));
                    asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(a[c]) : "f"(k1));
                }
                if (OP == P_2FFMA_FMNMX3) {
                    asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(b[c]) : "f"(k1), "f"(k2));
                    asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(b[c]) : "f"(k1), "f"(k2));
                    asm volatile("min.f32 %0, %0, %1, %2;" : "+f"(a[c]) : "f"(k2), "f"(k1));
                }
            }
        }
    }
    const long long t1 = clock64();
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < kChains; ++c)
        s += a[c] + b[c] + __uint_as_float(static_cast<uint32_t>(p[c])) + __uint_as_float(static_cast<uint32_t>(p[c] >> 32));
    if (s == 12345.678f) sink[0] = s;  // keeps the chains alive
    if (threadIdx.x == 0) atomicMax(reinterpret_cast<unsigned long long*>(cycles), static_cast<unsigned long long>(t1 - t0));
}

template <int OP>
int run_probe(const Ctx& c, int iters, int ctas_per_sm, float* sink, long long* cycles) {
    pipe_probe_kernel<OP><<<c.num_sms * ctas_per_sm, kProbeThreads, 0, c.stream>>>(iters, 1.25f, sink, cycles);
    ++g_launches;
    LIPFIT_CUDA(cudaGetLastError());
    return LIPFIT_OK;
}

}  // namespace

// lane-results per instruction: packed forms retire 2 per lane, FMNMX3 folds two comparisons, the mixes issue both
static const double kProbeResults[P_COUNT] = {1, 1, 2, 2, 1, 2, 1, 2, 4, 1, 3, 3, 6, 6, 3, 4};
static const double kProbeInstr[P_COUNT] = {1, 1, 1, 1, 1, 1, 1, 2, 2, 1, 2, 2, 3, 3, 2, 3};

int pipe_throughput(const Ctx& c, int which, double* lane_results_per_clk_sm, double* warp_instr_per_clk_sm) {
    if (which < 0 || which >= P_COUNT) return LIPFIT_E_PARAM;
    Workspace w;
    int rc = w.alloc(sizeof(long long) + sizeof(float), c.stream);
    if (rc) return rc;
    long long* cycles = w.as<long long>();
    float* sink = reinterpret_cast<float*>(cycles + 1);
    const int iters = 2000, ctas_per_sm = 2;  // 2 x 512 threads = 32 warps per SM, 8 per sub-partition
    double best = 0.0;
    for (int rep = 0; rep < 3; ++rep) {  // first repetition warms the instruction cache
        LIPFIT_CUDA(cudaMemsetAsync(cycles, 0, sizeof(long long), c.stream));
        switch (which) {
#define PROBE_CASE(OP) case OP: rc = run_probe<OP>(c, iters, ctas_per_sm, sink, cycles); break;
            PROBE_CASE(P_FFMA) PROBE_CASE(P_FADD) PROBE_CASE(P_FADD2) PROBE_CASE(P_FFMA2) PROBE_CASE(P_FMNMX)
            PROBE_CASE(P_FMNMX3) PROBE_CASE(P_MUFU_SQRT) PROBE_CASE(P_FFMA_FMNMX) PROBE_CASE(P_FADD2_FMNMX3)
            PROBE_CASE(P_FADD_ABS) PROBE_CASE(P_FADD2_FMNMX) PROBE_CASE(P_FFMA_FMNMX3) PROBE_CASE(P_2FADD2_FMNMX3)
            PROBE_CASE(P_FADD2_2FMNMX3) PROBE_CASE(P_FADD2_FADD) PROBE_CASE(P_2FFMA_FMNMX3)
#undef PROBE_CASE
        }
        if (rc) return rc;
        long long h = 0;
        LIPFIT_CUDA(cudaMemcpyAsync(&h, cycles, sizeof(h), cudaMemcpyDeviceToHost, c.stream));
        LIPFIT_CUDA(cudaStreamSynchronize(c.stream));
        if (h <= 0) return LIPFIT_E_CUDA;
        const double slots = static_cast<double>(iters) * kUnroll * kChains * kProbeThreads * ctas_per_sm;  // per SM
        const double rate = slots * kProbeResults[which] / static_cast<double>(h);
        if (rate > best) best = rate;
    }
    if (lane_results_per_clk_sm) *lane_results_per_clk_sm = best;
    if (warp_instr_per_clk_sm) *warp_instr_per_clk_sm = best / kProbeResults[which] * kProbeInstr[which] / 32.0;
    return LIPFIT_OK;
}

}  // namespace lipfit
