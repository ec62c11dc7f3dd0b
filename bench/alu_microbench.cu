// alu_microbench.cu — register-only pipe-rate microbenchmarks for sm_100a.
//
// MEASURED_PEAKS.json holds HBM and bf16 tensor peaks only; the shooting kernel is bound by the plain ALUs
// (FP32 FMA pipe, MUFU pipe, issue slots).  This program measures, per SM sub-partition (SMSP), how many warp-wide
// instructions per clock each instruction mix sustains, with the SM clock read from clock64() inside the kernel and
// the wall time from CUDA events (their ratio is the SM frequency during the run).
//
// Build:  nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -o alu_microbench alu_microbench.cu
//         (paper_1406_0559_b200/build.py: build_microbench(); not part of libmlens.so)
// Run:    ./alu_microbench              every mix + the RED patterns (prints one JSON object)
//         ./alu_microbench --fp32-peak [device]  the scalar-FFMA rate alone, ~0.1 s: the MEASURED FP32 peak bench.py reports
//                                       beside the derived one ("measure it ... and report the clock")
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <cstring>

#define CK(x)                                                                             \
    do {                                                                                  \
        cudaError_t e_ = (x);                                                             \
        if (e_ != cudaSuccess) {                                                          \
            fprintf(stderr, "%s: %s\n", #x, cudaGetErrorString(e_));                      \
            exit(1);                                                                      \
        }                                                                                 \
    } while (0)

constexpr int kIters = 16384;
constexpr int kChains = 16;
static double g_clock_hz = 1.965e9;  // set from cudaDeviceProp::clockRate (the maximum SM clock) in main()

__device__ __forceinline__ float rcp_mufu(float x) {
    float r;
    asm volatile("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

enum Mix { FFMA = 0, FFMA2, MUFU, FFMA_MUFU_41, KERNEL_MIX, PAIRED_MIX, DFMA, FADD2_ONLY, LDS128, FFMA2_FMUL, FFMA2_MUFU_INDEP, FFMA2_3PAIRS, FFMA2_UBCAST, FFMA_3REGS, SHARED_MIX, KERNEL_NOMUFU, N_MIX };
static const char* kMixName[N_MIX] = {"ffma", "ffma2", "mufu_rcp", "ffma4_mufu1", "kernel_mix_6ffma2_2mufu",
                                      "paired_mix_6ffma2_3fmul_1mufu", "dfma", "fadd2", "lds128_broadcast",
                                      "ffma2x12_fmulx6", "ffma2x12_mufux4_independent",
                                      "ffma2_three_distinct_pairs", "ffma2_uniform_bcast_operand", "ffma_three_distinct_regs",
                                      "shared_mix_12ffma2_3fmul2_2mufu_per_4rays", "kernel_mix_without_mufu_6_packed_per_pair"};
// warp-instructions issued per inner iteration per thread, FP32 flops per iteration per thread
static const int kInstr[N_MIX] = {kChains, kChains, kChains, 20, 64, 80, kChains, kChains, kChains, 18, 16, kChains, kChains, kChains, 68, 48};

template <int MIX>
__global__ void __launch_bounds__(256) bench_kernel(float* out, long long* cycles, float seed, float useed) {
    __shared__ float4 sm[256];
    sm[threadIdx.x] = make_float4(seed, seed * 0.5f, seed * 0.25f, 1.0f);
    __syncthreads();
    float a[kChains];
    float2 p[kChains / 2], s2[kChains / 2];
    double dd[kChains];
#pragma unroll
    for (int k = 0; k < kChains; ++k) {
        a[k] = seed + 0.001f * (float)(k + threadIdx.x);
        dd[k] = (double)a[k];
    }
#pragma unroll
    for (int k = 0; k < kChains / 2; ++k) { p[k] = make_float2(a[2 * k], a[2 * k + 1]); s2[k] = make_float2(0.f, 0.f); }
    const float b = 0.999f + seed * 1e-6f, c = seed * 1e-3f;
    const float2 b2 = make_float2(b, b), c2 = make_float2(c, c);
    float2 xx[kChains / 2], yy[kChains / 2];
    float xs[kChains], ys[kChains];
#pragma unroll
    for (int k = 0; k < kChains / 2; ++k) {
        xx[k] = make_float2(seed + 0.01f * (float)(k + threadIdx.x), seed - 0.02f * k);
        yy[k] = make_float2(0.5f * seed + 0.003f * (float)(threadIdx.x - k), 1.f + 1e-3f * k);
    }
#pragma unroll
    for (int k = 0; k < kChains; ++k) { xs[k] = xx[k >> 1].x + k; ys[k] = yy[k >> 1].y - k; }
    const float2 u2 = make_float2(useed, useed);  // kernel parameter: lives in a uniform register
    unsigned long long g0 = 0, g1 = 0;
    if (threadIdx.x == 0) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
    const long long t0 = clock64();
    for (int it = 0; it < kIters; ++it) {
        if (MIX == FFMA) {
#pragma unroll
            for (int k = 0; k < kChains; ++k) a[k] = fmaf(a[k], b, c);
        } else if (MIX == FFMA2) {
#pragma unroll
            for (int r = 0; r < 2; ++r)
#pragma unroll
                for (int k = 0; k < kChains / 2; ++k) p[k] = __ffma2_rn(p[k], b2, c2);
        } else if (MIX == FADD2_ONLY) {
#pragma unroll
            for (int r = 0; r < 2; ++r)
#pragma unroll
                for (int k = 0; k < kChains / 2; ++k) p[k] = __fadd2_rn(p[k], c2);
        } else if (MIX == MUFU) {
#pragma unroll
            for (int k = 0; k < kChains; ++k)  // the LOP3 (ALU pipe) keeps nvcc from folding rcp(rcp(x)) to x
                a[k] = __int_as_float(__float_as_int(rcp_mufu(a[k])) ^ 1);
        } else if (MIX == FFMA_MUFU_41) {
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                a[k] = rcp_mufu(a[k]);
                a[4 + k] = fmaf(a[4 + k], b, c);
                a[8 + k] = fmaf(a[8 + k], b, c);
                a[12 + k] = fmaf(a[12 + k], b, a[k]);
                a[k] = fmaf(a[k], b, c);
            }
        } else if (MIX == KERNEL_MIX) {
            // the difference-form interaction for 8 ray pairs: 1 FADD2 + 5 FFMA2 + 2 MUFU per pair
#pragma unroll
            for (int k = 0; k < kChains / 2; ++k) {
                const float2 dx = __fadd2_rn(p[k], c2);
                const float2 r2 = __ffma2_rn(dx, dx, b2);
                const float2 rc = make_float2(rcp_mufu(r2.x), rcp_mufu(r2.y));
                const float2 pr = __ffma2_rn(b2, dx, c2);
                const float2 pi = __ffma2_rn(c2, dx, b2);
                p[k] = __ffma2_rn(pr, rc, p[k]);
                s2[k] = __ffma2_rn(pi, rc, s2[k]);
            }
        } else if (MIX == KERNEL_NOMUFU) {
            // the FMA side of the production loop alone (r2 stands in for its reciprocal): 6 packed per ray pair
#pragma unroll
            for (int k = 0; k < kChains / 2; ++k) {
                const float2 dx = __fadd2_rn(p[k], c2);
                const float2 r2 = __ffma2_rn(dx, dx, b2);
                const float2 pr = __ffma2_rn(b2, dx, c2);
                const float2 pi = __ffma2_rn(c2, dx, b2);
                p[k] = __ffma2_rn(pr, r2, p[k]);
                s2[k] = __ffma2_rn(pi, r2, s2[k]);
            }
        } else if (MIX == PAIRED_MIX) {
            // one reciprocal per ray pair: rc = 1/(r2.x*r2.y); 1/r2.x = rc*r2.y, 1/r2.y = rc*r2.x
#pragma unroll
            for (int k = 0; k < kChains / 2; ++k) {
                const float2 dx = __fadd2_rn(p[k], c2);
                const float2 r2 = __ffma2_rn(dx, dx, b2);
                const float q = rcp_mufu(r2.x * r2.y);
                const float2 rc = make_float2(q * r2.y, q * r2.x);
                const float2 pr = __ffma2_rn(b2, dx, c2);
                const float2 pi = __ffma2_rn(c2, dx, b2);
                p[k] = __ffma2_rn(pr, rc, p[k]);
                s2[k] = __ffma2_rn(pi, rc, s2[k]);
            }
        } else if (MIX == FFMA2_FMUL) {
            // does a scalar FP32 op cost one FMA-pipe cycle or two inside a packed stream?
#pragma unroll
            for (int k = 0; k < 6; ++k) {
                p[k] = __ffma2_rn(p[k], b2, c2);
                a[k] = a[k] * b;
                s2[k] = __ffma2_rn(s2[k], b2, c2);
            }
        } else if (MIX == FFMA2_MUFU_INDEP) {
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                p[k] = __ffma2_rn(p[k], b2, c2);
                a[k] = __int_as_float(__float_as_int(rcp_mufu(a[k])) ^ 1);
                s2[k] = __ffma2_rn(s2[k], b2, c2);
                p[k + 4] = __ffma2_rn(p[k + 4], b2, c2);
            }
        } else if (MIX == FFMA2_3PAIRS) {
            // accumulate form S += X*Y: three distinct register pairs per instruction (register-file read bound)
#pragma unroll
            for (int r = 0; r < 2; ++r)
#pragma unroll
                for (int k = 0; k < kChains / 2; ++k) s2[k] = __ffma2_rn(xx[k], yy[(k + r) & (kChains / 2 - 1)], s2[k]);
        } else if (MIX == FFMA2_UBCAST) {
#pragma unroll
            for (int r = 0; r < 2; ++r)
#pragma unroll
                for (int k = 0; k < kChains / 2; ++k) s2[k] = __ffma2_rn(u2, xx[(k + r) & (kChains / 2 - 1)], s2[k]);
        } else if (MIX == FFMA_3REGS) {
#pragma unroll
            for (int k = 0; k < kChains; ++k) a[k] = fmaf(xs[k], ys[k], a[k]);
        } else if (MIX == SHARED_MIX) {
            // the shared_rcp group: 4 rays (pairs A, B) take 4 reciprocals from 2 MUFU + 3 FMUL2
#pragma unroll
            for (int k = 0; k < kChains / 2; k += 2) {
                const float2 dxa = __fadd2_rn(p[k], c2), dxc = __fadd2_rn(p[k + 1], c2);
                const float2 ra = __ffma2_rn(dxa, dxa, b2), rb = __ffma2_rn(dxc, dxc, b2);
                const float2 qq = __fmul2_rn(ra, rb);
                const float2 t = make_float2(rcp_mufu(qq.x), rcp_mufu(qq.y));
                const float2 rca = __fmul2_rn(t, rb), rcb = __fmul2_rn(t, ra);
                p[k] = __ffma2_rn(__ffma2_rn(b2, dxa, c2), rca, p[k]);
                s2[k] = __ffma2_rn(__ffma2_rn(c2, dxa, b2), rca, s2[k]);
                p[k + 1] = __ffma2_rn(__ffma2_rn(b2, dxc, c2), rcb, p[k + 1]);
                s2[k + 1] = __ffma2_rn(__ffma2_rn(c2, dxc, b2), rcb, s2[k + 1]);
            }
        } else if (MIX == DFMA) {
#pragma unroll
            for (int k = 0; k < kChains; ++k) dd[k] = fma(dd[k], (double)b, (double)c);
        } else if (MIX == LDS128) {
#pragma unroll
            for (int k = 0; k < kChains; ++k) {
                const float4 q = sm[(it * kChains + k) & 255];  // same address in every lane: broadcast
                a[k] += q.x + q.w;
            }
        }
    }
    const long long t1 = clock64();
    if (threadIdx.x == 0) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < kChains; ++k) s += a[k] + (float)dd[k];
#pragma unroll
    for (int k = 0; k < kChains / 2; ++k) s += p[k].x + p[k].y + s2[k].x + s2[k].y + xx[k].x + yy[k].y;
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0) {
        cycles[blockIdx.x] = t1 - t0;
        if (blockIdx.x == 0) cycles[gridDim.x] = (long long)(g1 - g0);  // ns on the global timer over the same span
    }
}

template <int MIX>
void run(int sms, int ctas_req, float* out, long long* cyc_dev, bool last) {
    // exactly one resident wave: every CTA runs concurrently for the whole kernel, so CTA 0's clock64() span is the
    // kernel's span and instr/cycles is a true per-SMSP rate
    int occ = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, bench_kernel<MIX>, 256, 0));
    const int ctas_per_sm = occ < ctas_req ? occ : ctas_req;
    const int grid = sms * ctas_per_sm;
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    for (int w = 0; w < 3; ++w) bench_kernel<MIX><<<grid, 256>>>(out, cyc_dev, 1.0f, 0.5f);  // warm-up (clock ramp)
    CK(cudaDeviceSynchronize());
    float best = 1e30f;
    long long cyc_best = 0;
    for (int rep = 0; rep < 5; ++rep) {
        CK(cudaEventRecord(e0));
        bench_kernel<MIX><<<grid, 256>>>(out, cyc_dev, 1.0f, 0.5f);
        CK(cudaEventRecord(e1));
        CK(cudaEventSynchronize(e1));
        float ms;
        CK(cudaEventElapsedTime(&ms, e0, e1));
        long long c0;
        CK(cudaMemcpy(&c0, cyc_dev, sizeof(c0), cudaMemcpyDeviceToHost));
        if (ms < best) { best = ms; cyc_best = c0; }
    }
    // Throughput = total work / total (event) time.  CTA 0's own clock64() span must NOT be used: the warp scheduler
    // favours the oldest warps, so co-resident CTAs finish one after another (CTA 0 of 4 ends after 1/4 of the
    // kernel) and its span overstates the per-SMSP rate by up to the number of resident CTAs.
    const double warps_per_smsp = ctas_per_sm * 8 / 4.0;
    const double instr = (double)kIters * kInstr[MIX] * warps_per_smsp;
    const double clk = best * 1e-3 * g_clock_hz;  // SM cycles of the whole launch at the maximum SM clock
    const double ipc = instr / clk;
    printf("  \"%s\": {\"ctas_per_sm\": %d, \"warp_instr_per_clk_per_smsp\": %.4f, \"clk_per_warp_instr\": %.3f, "
           "\"cta0_cycles\": %lld, \"ms\": %.4f}%s\n",
           kMixName[MIX], ctas_per_sm, ipc, 1.0 / ipc, cyc_best, best, last ? "" : ",");
    CK(cudaEventDestroy(e0));
    CK(cudaEventDestroy(e1));
}

// ---------------------------------------------------------------------------------------------------------------
// binning sub-roof: throughput of integer REDs into an int32 map, by address pattern
//   0 random over the whole map   1 one address per warp (32-way same address)   2 neighbouring addresses (coalesced)
//   3 random within a 32x32 window per CTA (the footprint of a 64x64-ray tile, App. A.3)
// ---------------------------------------------------------------------------------------------------------------
template <int PATTERN>
__global__ void __launch_bounds__(256) red_kernel(int* map, unsigned n_pix_mask, int reps) {
    unsigned x = (blockIdx.x * 256u + threadIdx.x) * 2654435761u + 12345u;
    const unsigned win = (blockIdx.x * 40503u) & n_pix_mask;
    for (int r = 0; r < reps; ++r) {
        x = x * 1664525u + 1013904223u;  // LCG
        unsigned a;
        if (PATTERN == 0) a = (x >> 4) & n_pix_mask;
        else if (PATTERN == 1) a = (((blockIdx.x * 8u + (threadIdx.x >> 5)) * 977u + r) * 64u) & n_pix_mask;
        else if (PATTERN == 2) a = ((blockIdx.x * 256u + threadIdx.x) + (unsigned)r * 65536u) & n_pix_mask;
        else a = (win + ((x >> 8) & 1023u)) & n_pix_mask;
        atomicAdd(map + a, 1);  // result unused -> RED.E.ADD
    }
}

template <int PATTERN>
void run_red(const char* name, int sms, int* map, unsigned mask, bool last) {
    const int reps = 2048, grid = sms * 8;
    red_kernel<PATTERN><<<grid, 256>>>(map, mask, 64);
    CK(cudaDeviceSynchronize());
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    float best = 1e30f;
    for (int rep = 0; rep < 3; ++rep) {
        CK(cudaEventRecord(e0));
        red_kernel<PATTERN><<<grid, 256>>>(map, mask, reps);
        CK(cudaEventRecord(e1));
        CK(cudaEventSynchronize(e1));
        float ms;
        CK(cudaEventElapsedTime(&ms, e0, e1));
        if (ms < best) best = ms;
    }
    printf("  \"%s\": {\"reds_per_s\": %.4e, \"ms\": %.4f}%s\n", name, (double)grid * 256 * reps / (best * 1e-3), best,
           last ? "" : ",");
}

// --fp32-peak: scalar FFMA, 16 independent chains per thread, 4 CTAs x 256 threads per SM (8 warps per SMSP), best of
// 10 launches after a 20-launch warm-up (clock ramp).  flops = 2 per FFMA lane.  The SM clock is observed INSIDE the
// timed kernel: CTA 0's clock64() span over its %globaltimer span.
static int fp32_peak(int sms, float* out, long long* cyc) {
    const int grid = sms * 4;
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    for (int w = 0; w < 20; ++w) bench_kernel<FFMA><<<grid, 256>>>(out, cyc, 1.0f, 0.5f);
    CK(cudaDeviceSynchronize());
    float best = 1e30f;
    double mhz = 0.0;
    for (int rep = 0; rep < 10; ++rep) {
        CK(cudaEventRecord(e0));
        bench_kernel<FFMA><<<grid, 256>>>(out, cyc, 1.0f, 0.5f);
        CK(cudaEventRecord(e1));
        CK(cudaEventSynchronize(e1));
        float ms;
        CK(cudaEventElapsedTime(&ms, e0, e1));
        long long c0, ns;
        CK(cudaMemcpy(&c0, cyc, sizeof(c0), cudaMemcpyDeviceToHost));
        CK(cudaMemcpy(&ns, cyc + grid, sizeof(ns), cudaMemcpyDeviceToHost));
        if (ms < best) { best = ms; mhz = ns > 0 ? 1e3 * (double)c0 / (double)ns : 0.0; }
    }
    const double flops = 2.0 * (double)kIters * kChains * 256.0 * grid;
    printf("{\"fp32_tflops\": %.4f, \"ms\": %.4f, \"sm_mhz_observed\": %.1f, \"sms\": %d, "
           "\"how\": \"scalar FFMA, 16 chains/thread, 4x256 threads/SM, best of 10, CUDA events\"}\n",
           flops / (best * 1e-3) / 1e12, best, mhz, sms);
    return 0;
}

int main(int argc, char** argv) {
    const bool peak_only = argc > 1 && !strcmp(argv[1], "--fp32-peak");
    int ctas = (argc > 1 && !peak_only) ? atoi(argv[1]) : 4;
    const int dev = (peak_only && argc > 2) ? atoi(argv[2]) : 0;
    CK(cudaSetDevice(dev));
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, dev));
    const int sms = prop.multiProcessorCount;
    g_clock_hz = 1e3 * (double)prop.clockRate;
    float* out;
    long long* cyc;
    CK(cudaMalloc(&out, sizeof(float) * sms * 8 * 256));
    CK(cudaMalloc(&cyc, sizeof(long long) * (sms * 8 + 1)));
    if (peak_only) return fp32_peak(sms, out, cyc);
    printf("{\n  \"device\": \"%s\", \"sms\": %d, \"clock_rate_khz\": %d,\n", prop.name, sms, prop.clockRate);
    run<FFMA>(sms, ctas, out, cyc, false);
    run<FFMA2>(sms, ctas, out, cyc, false);
    run<FADD2_ONLY>(sms, ctas, out, cyc, false);
    run<MUFU>(sms, ctas, out, cyc, false);
    run<FFMA_MUFU_41>(sms, ctas, out, cyc, false);
    run<KERNEL_MIX>(sms, ctas, out, cyc, false);
    run<PAIRED_MIX>(sms, ctas, out, cyc, false);
    run<DFMA>(sms, ctas, out, cyc, false);
    run<LDS128>(sms, ctas, out, cyc, false);
    run<FFMA2_FMUL>(sms, ctas, out, cyc, false);
    run<FFMA2_MUFU_INDEP>(sms, ctas, out, cyc, false);
    run<FFMA2_3PAIRS>(sms, ctas, out, cyc, false);
    run<FFMA2_UBCAST>(sms, ctas, out, cyc, false);
    run<FFMA_3REGS>(sms, ctas, out, cyc, false);
    run<SHARED_MIX>(sms, ctas, out, cyc, false);
    run<KERNEL_NOMUFU>(sms, ctas, out, cyc, false);
    int* map;  // 4096^2 int32 = 64 MB (config 3's map; fits the 126 MB L2) and 16384^2 = 1 GB (larger than L2)
    for (int big = 0; big < 2; ++big) {
        const unsigned n_pix = big ? (1u << 28) : (1u << 24);
        CK(cudaMalloc(&map, sizeof(int) * (size_t)n_pix));
        CK(cudaMemset(map, 0, sizeof(int) * (size_t)n_pix));
        run_red<0>(big ? "red_random_1GB_map" : "red_random_64MB_map", sms, map, n_pix - 1, false);
        run_red<3>(big ? "red_window32x32_1GB_map" : "red_window32x32_64MB_map", sms, map, n_pix - 1, false);
        if (!big) {
            run_red<1>("red_same_address_per_warp", sms, map, n_pix - 1, false);
            run_red<2>("red_coalesced_neighbours", sms, map, n_pix - 1, false);
        }
        CK(cudaFree(map));
    }
    printf("  \"note\": \"rates are total work / event time at the maximum SM clock\"\n");
    printf("}\n");
    return 0;
}
