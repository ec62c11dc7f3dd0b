// umma_probe.cu — probe of the tensor pipe for the next kernel generation.
//
// The quantities the shooting loop forms before its reciprocal (r^2, Re and Im of c conj(w)) are bilinear in (ray, lens)
// and fit ONE tcgen05.mma.kind::tf32 with M = 128 rays, N = 192 = 64 lenses x 3, K = 8 (TF32 hi/lo pairs).  This program
// answers the two questions that plan depends on, on the actual hardware:
//   1. arithmetic: with TF32-exact operands (products exact in FP32), how far is the tensor pipe's K = 8 sum from the
//      exactly rounded FP32 sum?  (operands with the dynamic range of the real problem: |zeta|^2 ~ 1e5 next to lo parts ~1e-3)
//   2. rate: clocks per M128 x N192 x K8 TF32 MMA issued back to back by one thread of one CTA per SM.
// Not on the product path.  Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o umma_probe umma_probe.cu
#include <cuda_runtime.h>
#include <stdint.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#define CK(x)                                                                \
    do {                                                                     \
        cudaError_t e_ = (x);                                                \
        if (e_ != cudaSuccess) {                                             \
            fprintf(stderr, "%s: %s\n", #x, cudaGetErrorString(e_));         \
            exit(1);                                                         \
        }                                                                    \
    } while (0)

constexpr int kM = 128, kN = 192, kK = 8, kCols = 256;  // TMEM columns allocated (power of two >= kN)

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// canonical K-major, no-swizzle UMMA layout for 4-byte elements: 8-row x 16-byte core matrices; the second 16-byte chunk
// along K follows its core matrix (LBO = 128 B), the next 8 rows follow both chunks (SBO = 256 B)
__host__ __device__ inline int umma_off_bytes(int r, int k) { return (r % 8) * 16 + (r / 8) * 256 + (k / 4) * 128 + (k % 4) * 4; }

__device__ __forceinline__ uint64_t make_smem_desc(uint32_t saddr) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFF) >> 4);   // start address, 16-byte units
    d |= (uint64_t)(128 >> 4) << 16;           // leading byte offset (between the two K chunks)
    d |= (uint64_t)(256 >> 4) << 32;           // stride byte offset (between 8-row groups)
    d |= (uint64_t)1 << 46;                    // descriptor version 1 (Blackwell)
    return d;                                  // layout type 0 = no swizzle, base offset 0
}

__global__ void __launch_bounds__(128, 1) umma_probe_kernel(const float* __restrict__ A, const float* __restrict__ B,
                                                            float* __restrict__ D, int reps, long long* __restrict__ cycles) {
    __shared__ __align__(1024) unsigned char sA[kM * kK * 4];
    __shared__ __align__(1024) unsigned char sB[kN * kK * 4];
    __shared__ __align__(8) uint64_t bar;
    __shared__ uint32_t tmem_base_sh;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    for (int e = tid; e < kM * kK; e += 128) *reinterpret_cast<float*>(sA + umma_off_bytes(e / kK, e % kK)) = A[e];
    for (int e = tid; e < kN * kK; e += 128) *reinterpret_cast<float*>(sB + umma_off_bytes(e / kK, e % kK)) = B[e];
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // generic-proxy writes -> visible to the tensor pipe
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&bar)) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_sh)), "n"(kCols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = tmem_base_sh;

    // instruction descriptor: D = F32, A = B = TF32, both K-major, N >> 3, M >> 4
    const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(kN >> 3) << 17) | ((uint32_t)(kM >> 4) << 24);
    long long t0 = 0, t1 = 0;
    if (tid == 0) {
        const uint64_t da = make_smem_desc(smem_u32(sA)), db = make_smem_desc(smem_u32(sB));
        t0 = clock64();
        for (int r = 0; r < reps; ++r) {
            asm volatile(
                "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}\n" ::"r"(tmem_base),
                "l"(da), "l"(db), "r"(idesc), "r"(0u)
                : "memory");
        }
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(&bar)) : "memory");
    }
    // everybody waits for the tensor pipe (phase 0 of the barrier)
    {
        uint32_t done = 0;
        while (!done) {
            asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
                         : "=r"(done) : "r"(smem_u32(&bar)), "r"(0u) : "memory");
        }
    }
    if (tid == 0) { t1 = clock64(); cycles[blockIdx.x] = t1 - t0; }
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");

    // TMEM -> registers -> global: warp w owns lanes 32w..32w+31 (= rows of D), 32 columns per load
    for (int c0 = 0; c0 < kN; c0 += 32) {
        uint32_t v[32];
        const uint32_t taddr = tmem_base + ((uint32_t)(warp * 32) << 16) + (uint32_t)c0;
        asm volatile(
            "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
            "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
            "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
            : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
              "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]),
              "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]),
              "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
            : "r"(taddr)
            : "memory");
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        if (blockIdx.x == 0)
            for (int j = 0; j < 32; ++j) D[(size_t)(warp * 32 + lane) * kN + c0 + j] = __uint_as_float(v[j]);
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kCols) : "memory");
}

static float tf32_rna(float x) {  // round to 10 mantissa bits, ties away from zero (cvt.rna.tf32.f32)
    uint32_t b;
    memcpy(&b, &x, 4);
    b = (b + 0x1000u) & 0xffffe000u;
    memcpy(&x, &b, 4);
    return x;
}

int main() {
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, 0));
    std::vector<float> A((size_t)kM * kK), B((size_t)kN * kK);
    // ray rows: [1, 1, dx', dx', dy', dy', |delta|^2_hi, |delta|^2_lo] with d = 4.9e-4 (config 4), offsets in lattice steps
    const double d = 5.0 / 1024 / 10;
    for (int r = 0; r < kM; ++r) {
        const double dx = (r % 64) - 31.5, dy = (r / 64) * 17 - 31.5, q = (dx * dx + dy * dy) * d * d;
        const float qh = tf32_rna((float)q), ql = tf32_rna((float)(q - (double)qh));
        const float row[kK] = {1.f, 1.f, (float)dx, (float)dx, (float)dy, (float)dy, qh, ql};
        for (int k = 0; k < kK; ++k) A[(size_t)r * kK + k] = row[k];
    }
    // lens rows, three per lens: r^2 row [|z|^2 hi, lo, 2 d zx hi, lo, 2 d zy hi, lo, 1, 1]; Re row; Im row
    unsigned s = 12345u;
    auto rnd = [&]() { s = s * 1664525u + 1013904223u; return (double)(s >> 8) / 16777216.0; };
    std::vector<double> Bd((size_t)kN * kK, 0.0);
    for (int l = 0; l < kN / 3; ++l) {
        const double zx = (rnd() - 0.5) * 400, zy = (rnd() - 0.5) * 400, m = 0.3 + 3 * rnd();
        const double r2 = zx * zx + zy * zy, cr = m * zx / r2, ci = -m * zy / r2;
        const double v[3][4] = {{r2, 2 * d * zx, 2 * d * zy, 1.0}, {cr * zx + ci * zy, d * cr, d * ci, 0.0}, {ci * zx - cr * zy, d * ci, -d * cr, 0.0}};
        for (int q = 0; q < 3; ++q)
            for (int j = 0; j < 4; ++j) {
                const float hi = tf32_rna((float)v[q][j]);
                const float lo = (j == 3) ? (float)v[q][j] - 0.f * hi : tf32_rna((float)(v[q][j] - (double)hi));
                float h2 = hi, l2 = lo;
                if (j == 3) { h2 = (float)v[q][j]; l2 = (float)v[q][j]; }  // multiplies |delta|^2 hi and lo: both 1 (or 0)
                B[(size_t)(3 * l + q) * kK + 2 * j] = h2;
                B[(size_t)(3 * l + q) * kK + 2 * j + 1] = l2;
            }
    }
    float *dA, *dB, *dD;
    long long* dcyc;
    CK(cudaMalloc(&dA, A.size() * 4)); CK(cudaMalloc(&dB, B.size() * 4)); CK(cudaMalloc(&dD, (size_t)kM * kN * 4));
    CK(cudaMalloc(&dcyc, 8 * 256));
    CK(cudaMemcpy(dA, A.data(), A.size() * 4, cudaMemcpyHostToDevice));
    CK(cudaMemcpy(dB, B.data(), B.size() * 4, cudaMemcpyHostToDevice));
    CK(cudaMemset(dD, 0, (size_t)kM * kN * 4));
    umma_probe_kernel<<<1, 128>>>(dA, dB, dD, 1, dcyc);
    CK(cudaDeviceSynchronize());
    std::vector<float> D((size_t)kM * kN);
    CK(cudaMemcpy(D.data(), dD, D.size() * 4, cudaMemcpyDeviceToHost));
    // (1) arithmetic: against the exact sum of the 8 (exact) products, in units of the FP32 ulp of the result
    double max_ulp = 0, sum_ulp = 0, max_rel_r2 = 0;
    long long n_bad = 0;
    for (int r = 0; r < kM; ++r)
        for (int c = 0; c < kN; ++c) {
            double ex = 0, mag = 0;
            for (int k = 0; k < kK; ++k) { const double t = (double)A[(size_t)r * kK + k] * (double)B[(size_t)c * kK + k]; ex += t; mag = fmax(mag, fabs(t)); }
            const double got = D[(size_t)r * kN + c];
            const double ulp = ldexp(1.0, ilogb(fmax(mag, 1e-300)) - 23);  // ulp of the largest addend: the natural scale of the sum
            const double e = fabs(got - ex) / ulp;
            max_ulp = fmax(max_ulp, e); sum_ulp += e;
            if (c % 3 == 0) max_rel_r2 = fmax(max_rel_r2, fabs(got - ex) / fabs(ex));
            if (!(e < 64)) ++n_bad;
        }
    printf("{\n  \"device\": \"%s\",\n  \"mma\": \"tcgen05.mma.cta_group::1.kind::tf32 M%d N%d K%d\",\n", prop.name, kM, kN, kK);
    printf("  \"error_vs_exact_sum_in_ulp_of_largest_addend\": {\"max\": %.3f, \"mean\": %.4f, \"entries_off_by_64ulp_or_more\": %lld},\n", max_ulp,
           sum_ulp / (kM * kN), n_bad);
    printf("  \"max_relative_error_of_r2\": %.3e,\n", max_rel_r2);
    printf("  \"sample\": {\"D[5][0]\": %.9g, \"D[5][1]\": %.9g, \"D[5][2]\": %.9g},\n", D[5 * kN], D[5 * kN + 1], D[5 * kN + 2]);
    // (2) rate: back-to-back MMAs from one thread, one CTA per SM
    const int reps = 4096;
    umma_probe_kernel<<<prop.multiProcessorCount, 128>>>(dA, dB, dD, reps, dcyc);
    CK(cudaDeviceSynchronize());
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    CK(cudaEventRecord(e0));
    umma_probe_kernel<<<prop.multiProcessorCount, 128>>>(dA, dB, dD, reps, dcyc);
    CK(cudaEventRecord(e1));
    CK(cudaDeviceSynchronize());
    float ms;
    CK(cudaEventElapsedTime(&ms, e0, e1));
    long long cyc;
    CK(cudaMemcpy(&cyc, dcyc, 8, cudaMemcpyDeviceToHost));
    const double clk = (double)cyc / reps;
    printf("  \"clocks_per_mma\": %.2f, \"interactions_per_mma\": %d, \"tensor_clocks_per_interaction_warp\": %.4f,\n", clk, kM * kN / 3,
           clk / (kM * kN / 3 / 32.0));
    printf("  \"tf32_tflops_all_sms\": %.1f, \"kernel_ms\": %.4f\n}\n", 2.0 * kM * kN * kK * reps * prop.multiProcessorCount / (ms * 1e-3) / 1e12, ms);
    return 0;
}
