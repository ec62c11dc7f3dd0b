// shoot_umma_kernel.cuh — EXPERIMENTAL second-generation shooting kernel (mlens_set_option("kernel", 3)).
//
// Same sum as shoot_fp32_kernel (Eq. 1, directly over all lenses, difference form around the tile centre),
// but the three quantities formed before the reciprocal are taken from the tensor pipe (DESIGN.md "The lever that is
// left"): with w = zeta_l + delta_k and delta' = delta/d (in-tile offsets in lattice steps, exact in TF32)
//   r^2          = [1,1,dx',dx',dy',dy',|delta|^2_hi,|delta|^2_lo]_k . [|zeta|^2_hi,_lo,(2 d zx)_hi,_lo,(2 d zy)_hi,_lo,1,1]_l
//   Re(c conj w) = [1,1,dx',dx',dy',dy',0,0]_k . [(cr zx + ci zy)_hi,_lo,(d cr)_hi,_lo,(d ci)_hi,_lo,0,0]_l      (Im alike)
// One tcgen05.mma.kind::tf32 (M = 128 rays, N = 192 = 64 lenses x 3, K = 8) gives all three for 8192 interactions; the
// accumulator lives in TMEM with one ray per lane, so a consumer thread reads its own ray's values (tcgen05.ld.32x32b)
// and is left with the reciprocal — shared between two lenses: 3 FMUL + 1 MUFU per pair — and S += (Re, Im) * rc.
//
// Structure: one CTA per SM, 8 consumer warps + 1 control warp.  The ray matrix (32 blocks of 128 rays = one 64x64 tile,
// 128 KB, identical for every tile) stays in shared memory; lenses are processed in super-chunks of 512 (48 KB of TF32
// hi/lo rows written by an FP64 transform per tile); the control warp's lane 0 issues the MMAs into a double-buffered
// TMEM accumulator, mbarriers hand buffers back and forth; per-ray sums are accumulated in shared memory across
// super-chunks, then the same FP64 epilogue and integer-RED binning as the first kernel.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "shoot_kernel.cuh"

namespace mlk {

constexpr int kUmRays = 128;        // rays per MMA (M)
constexpr int kUmLenses = 64;       // lenses per MMA (N = 3 * 64)
constexpr int kUmN = 3 * kUmLenses;
constexpr int kUmSuperMax = 512;    // lenses per super-chunk resident in shared memory (template parameter kSuper: 512 or 256)
constexpr int kUmBlocks = kTile * kTile / kUmRays;  // 32 ray blocks per tile
constexpr int kUmConsumersMax = 16;  // consumer warps (template parameter kCons): 16 = 2 groups x 4 TMEM lane quadrants x 2 halves of
                                    // a chunk's lenses; 8 = 2 groups x 4 quadrants, every warp takes the whole chunk (the slim variant
                                    // that can share an SM with a CTA of the production kernel: 288 threads, 96 registers)
constexpr int kUmChunkBytes = kUmN * 8 * 4;         // 6144: one B chunk (192 rows x K = 8)
constexpr int kUmABlockBytes = kUmRays * 8 * 4;     // 4096: one A block

// canonical K-major no-swizzle UMMA layout for 4-byte elements (probed in round 1: profiles/r1e_umma_probe.md)
__host__ __device__ inline int umma_off_bytes(int r, int k) { return (r % 8) * 16 + (r / 8) * 256 + (k / 4) * 128 + (k % 4) * 4; }

__device__ __forceinline__ uint64_t umma_smem_desc(uint32_t saddr) {
    return (uint64_t)((saddr & 0x3FFFF) >> 4) | ((uint64_t)(128 >> 4) << 16) | ((uint64_t)(256 >> 4) << 32) | ((uint64_t)1 << 46);
}
__device__ __forceinline__ float tf32_rna(float x) {
    uint32_t r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
    return __uint_as_float(r);
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait_parity(uint64_t* bar, uint32_t parity) {
    uint32_t done = 0;
    while (!done)
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
                     : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float* v) {
    uint32_t r[16];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
          "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
#pragma unroll
    for (int j = 0; j < 16; ++j) v[j] = __uint_as_float(r[j]);
}

struct __align__(16) UmmaShared {
    uint64_t full[2], empty[2];          // TMEM accumulator hand-over
    uint32_t tmem_base;
    int near_n;
    long long next_tile;
    double part[kUmConsumersMax + 1][2];
    double near_zx[kNearMax], near_zy[kNearMax], near_m[kNearMax];
    unsigned long long ctr[3];
};


template <int kCons, int kSuper>
__global__ void __maxnreg__(kCons == 8 ? 112 : 96) shoot_umma_kernel(const ShootParams P) {
    constexpr int kUmConsumers = kCons, kUmThreads = 32 * (kCons + 1), kUmSuper = kSuper;
    constexpr int kParts = kCons / 8;        // warps that share one TMEM lane quadrant of a group
    constexpr int kHf = 4 / kParts;          // 16-lens sub-blocks of a chunk per warp
    constexpr int kBarThreads = 32 * kCons;  // both consumer groups take part in each named barrier
    extern __shared__ __align__(1024) unsigned char um_smem[];
    unsigned char* sA = um_smem;                                                     // 32 ray blocks x 4 KB
    unsigned char* sB = sA + kUmBlocks * kUmABlockBytes;                             // 8 lens chunks x 6 KB
    float2* sS = reinterpret_cast<float2*>(sB + (kUmSuper / kUmLenses) * kUmChunkBytes);  // per-ray sums of the tile
    UmmaShared& sh = *reinterpret_cast<UmmaShared*>(reinterpret_cast<unsigned char*>(sS) + kTile * kTile * sizeof(float2));
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const bool is_control = warp == kUmConsumers;

    for (int e = tid; e < kUmBlocks * kUmABlockBytes / 16; e += kUmThreads)
        reinterpret_cast<float4*>(sA)[e] = __ldg(reinterpret_cast<const float4*>(P.umma_A) + e);
    if (tid == 0) {
        mbar_init(&sh.full[0], 1); mbar_init(&sh.full[1], 1);
        mbar_init(&sh.empty[0], kUmConsumers / 2); mbar_init(&sh.empty[1], kUmConsumers / 2);
        mbar_fence_init();
        sh.ctr[0] = sh.ctr[1] = sh.ctr[2] = 0ull;
        sh.near_n = 0;
    }
    if (is_control) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(&sh.tmem_base)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = sh.tmem_base;
    const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(kUmN >> 3) << 17) | ((uint32_t)(kUmRays >> 4) << 24);

    // Ping-pong of the arithmetic phase between the two consumer groups (named barriers 1 and 2, 512 threads each):
    // a group may only do its MUFU/FMA work while the other one waits for / reads its next accumulator, so the two can
    // never fall into lock-step (both computing, then both waiting, with the MUFU idle a third of the time).
    if (!is_control && warp / (4 * kParts) == 1) asm volatile("bar.arrive 1, %0;" ::"n"(kBarThreads) : "memory");
    const long long n_tiles = (long long)P.tiles_x * P.tiles_y;
    const int n_super = P.n_lens > 0 ? (P.n_lens + kUmSuper - 1) / kUmSuper : 0;
    uint32_t seq = 0;  // MMA sequence number: buffer seq & 1, use (seq >> 1) of that buffer; same count in every warp
    long long nxt = 0;
    for (long long tile = blockIdx.x; tile < n_tiles;) {
        if (tid == 0) nxt = (long long)atomicAdd(P.tile_counter, 1ull) + gridDim.x;
        const int tJ = (int)(tile / P.tiles_x), tI = (int)(tile - (long long)tJ * P.tiles_x);
        const long long ti0 = P.i0 + (long long)tI * kTile, tj0 = P.j0 + (long long)tJ * kTile;
        const double Zcx = ((double)(ti0 + kTile / 2) - P.half_n1) * P.d;
        const double Zcy = ((double)(tj0 + kTile / 2) - P.half_n2) * P.d;
        for (int q = tid; q < kTile * kTile; q += kUmThreads) sS[q] = make_float2(0.f, 0.f);
        double pr_ = 0.0, pi_ = 0.0;

        for (int sc = 0; sc < n_super; ++sc) {
            const int l0 = sc * kUmSuper;
            const int n_sc = min(kUmSuper, P.n_lens - l0);
            const int n_chunks = (n_sc + kUmLenses - 1) / kUmLenses;
            // (1) FP64 transform of this super-chunk into TF32 hi/lo rows (three rows per lens, quantity-major per chunk)
            for (int t = tid; t < n_chunks * kUmLenses; t += kUmThreads) {
                double v[9] = {1.0e16, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};  // neutral lens: far away, no mass
                if (t < n_sc) {
                    const float4 q = __ldg(P.lens_raw + l0 + t);
                    const double zx = Zcx - (double)q.x, zy = Zcy - (double)q.y, m = (double)q.z;
                    const double r2 = zx * zx + zy * zy;
                    bool near = r2 < fmax(P.rho2 * fmax(m, 1.0), P.rho2_tile);
                    if (near) {
                        const int slot = atomicAdd(&sh.near_n, 1);
                        if (slot < kNearMax) { sh.near_zx[slot] = zx; sh.near_zy[slot] = zy; sh.near_m[slot] = m; }
                        else near = false;
                    }
                    if (!near) {
                        const double inv = m / r2;
                        const double cr = zx * inv, ci = -zy * inv;
                        pr_ += cr; pi_ += ci;
                        v[0] = r2; v[1] = 2.0 * P.d * zx; v[2] = 2.0 * P.d * zy;
                        v[3] = cr * zx + ci * zy; v[4] = P.d * cr; v[5] = P.d * ci;
                        v[6] = ci * zx - cr * zy; v[7] = P.d * ci; v[8] = -P.d * cr;
                    }
                }
                unsigned char* chunk = sB + (t / kUmLenses) * kUmChunkBytes;
#pragma unroll
                for (int qn = 0; qn < 3; ++qn) {
                    float h[3], l[3];
#pragma unroll
                    for (int j = 0; j < 3; ++j) {
                        h[j] = tf32_rna((float)v[3 * qn + j]);
                        l[j] = tf32_rna((float)(v[3 * qn + j] - (double)h[j]));
                    }
                    const float e = qn == 0 ? 1.f : 0.f;
                    // rows of a chunk: r^2 of the 64 lenses, then (Re, Im) interleaved per lens, so that a consumer's
                    // tcgen05.ld puts each lens's (Re, Im) into an adjacent register pair (packed FFMA2 accumulate)
                    const int row = qn == 0 ? (t % kUmLenses) : kUmLenses + 2 * (t % kUmLenses) + (qn - 1);
                    *reinterpret_cast<float4*>(chunk + umma_off_bytes(row, 0)) = make_float4(h[0], l[0], h[1], l[1]);
                    *reinterpret_cast<float4*>(chunk + umma_off_bytes(row, 4)) = make_float4(h[2], l[2], e, e);
                }
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncthreads();

            // (2) 32 ray blocks x n_chunks lens chunks: the control thread issues, the consumer warps drain
            if (is_control) {
                if (lane == 0) {
                    for (int rb = 0; rb < kUmBlocks; ++rb) {
                        const uint64_t da = umma_smem_desc(smem_u32(sA + rb * kUmABlockBytes));
                        for (int c = 0; c < n_chunks; ++c, ++seq) {
                            const uint32_t buf = seq & 1u, use = seq >> 1;
                            if (use >= 1) mbar_wait_parity(&sh.empty[buf], (use - 1) & 1u);
                            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                            const uint64_t db = umma_smem_desc(smem_u32(sB + c * kUmChunkBytes));
                            asm volatile(
                                "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                                "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}\n" ::"r"(tmem_base + buf * kUmN),
                                "l"(da), "l"(db), "r"(idesc), "r"(0u)
                                : "memory");
                            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(
                                             smem_u32(&sh.full[buf]))
                                         : "memory");
                        }
                    }
                } else {
                    seq += (uint32_t)(kUmBlocks * n_chunks);
                }
                __syncwarp();
            } else {
                // Two consumer groups of 8 warps work on alternate chunks (TMEM buffer = group): while one group is in its
                // TMEM-read phase (64 B/clk per sub-partition: the binding resource of this kernel) the other is in its
                // MUFU/FMA phase.  Within a group: 4 lane quadrants x 2 halves of the chunk's 64 lenses.
                const int group = warp / (4 * kParts), quad = warp & 3, part = (warp >> 2) % kParts;
                for (int rb = 0; rb < kUmBlocks; ++rb) {
                    float2 S[4];  // (S_re, S_im) partial sums, four independent chains
#pragma unroll
                    for (int a = 0; a < 4; ++a) S[a] = make_float2(0.f, 0.f);
                    for (int c = 0; c < n_chunks; ++c, ++seq) {
                        const uint32_t buf = seq & 1u, use = seq >> 1;
                        if ((int)buf != group) continue;
                        mbar_wait_parity(&sh.full[buf], use & 1u);
                        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                        const uint32_t tbase = tmem_base + ((uint32_t)(quad * 32) << 16) + buf * kUmN;
#pragma unroll(kHf == 2 ? 2 : 1)
                        for (int hf = 0; hf < kHf; ++hf) {
                            const int l16 = part * kHf + hf;  // which 16 of the chunk's 64 lenses
                            float r2[16], pq[32];
                            tmem_ld16(tbase + l16 * 16, r2);
                            tmem_ld16(tbase + kUmLenses + l16 * 32, pq);
                            tmem_ld16(tbase + kUmLenses + l16 * 32 + 16, pq + 16);
                            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                            if (hf == 0) {
                                if (group == 0) asm volatile("bar.sync 1, %0;" ::"n"(kBarThreads) : "memory");
                                else asm volatile("bar.sync 2, %0;" ::"n"(kBarThreads) : "memory");
                            }
                            if (hf == kHf - 1) {
                                // everything of this buffer is in registers: hand it back before the arithmetic
                                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                                __syncwarp();
                                if (lane == 0) mbar_arrive(&sh.empty[buf]);
                            }
#pragma unroll
                            for (int j = 0; j < 16; j += 4) {
                                // four lenses, two MUFU: lens j shares with j+2, lens j+1 with j+3 (all products packed)
                                const float2 Ra = make_float2(r2[j], r2[j + 1]), Rb = make_float2(r2[j + 2], r2[j + 3]);
                                const float2 Q = __fmul2_rn(Ra, Rb);
                                const float2 T = make_float2(rcp_mufu(Q.x), rcp_mufu(Q.y));
                                const float2 RCa = __fmul2_rn(T, Rb), RCb = __fmul2_rn(T, Ra);
                                S[0] = __ffma2_rn(make_float2(pq[2 * j], pq[2 * j + 1]), make_float2(RCa.x, RCa.x), S[0]);
                                S[1] = __ffma2_rn(make_float2(pq[2 * j + 2], pq[2 * j + 3]), make_float2(RCa.y, RCa.y), S[1]);
                                S[2] = __ffma2_rn(make_float2(pq[2 * j + 4], pq[2 * j + 5]), make_float2(RCb.x, RCb.x), S[2]);
                                S[3] = __ffma2_rn(make_float2(pq[2 * j + 6], pq[2 * j + 7]), make_float2(RCb.y, RCb.y), S[3]);
                            }
                        }
                        if (group == 0) asm volatile("bar.arrive 2, %0;" ::"n"(kBarThreads) : "memory");
                        else asm volatile("bar.arrive 1, %0;" ::"n"(kBarThreads) : "memory");
                    }
                    const int ray = rb * kUmRays + quad * 32 + lane;
                    atomicAdd(&sS[ray].x, (S[0].x + S[1].x) + (S[2].x + S[3].x));
                    atomicAdd(&sS[ray].y, (S[0].y + S[1].y) + (S[2].y + S[3].y));
                }
            }
            __syncthreads();  // the lens rows may be overwritten; all partial sums of this super-chunk are in sS
        }

        // (3) A_c = sum of c_i over the lenses of the FP32/TF32 list (FP64), block reduction
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            pr_ += __shfl_xor_sync(0xffffffffu, pr_, off);
            pi_ += __shfl_xor_sync(0xffffffffu, pi_, off);
        }
        if (lane == 0) { sh.part[warp][0] = pr_; sh.part[warp][1] = pi_; }
        __syncthreads();
        double Acr = 0.0, Aci = 0.0;
#pragma unroll
        for (int w = 0; w < kUmThreads / 32; ++w) { Acr += sh.part[w][0]; Aci += sh.part[w][1]; }

        // (4) per-ray epilogue and binning: 256 threads x 16 consecutive rays of one row (same arithmetic as
        //     shoot_fp32_kernel: conj(alpha) = A_c - delta*S, Eq. 1 in pixel units, run-combined integer REDs)
        int n_in = 0, n_out = 0, n_lost = 0;
        if (tid < kTile * kTile / 16) {
            const int n_near = min(sh.near_n, kNearMax);
            const bool near_overflow = sh.near_n > kNearMax;
            const int iy = tid / 4, ix0 = (tid % 4) * 16;
            const long long jray = tj0 + iy;
            const bool row_ok = jray < P.j0 + P.nj;
            const double x2 = ((double)jray + 0.5 - P.half_n2) * P.d;
            const double dyd = ((double)iy - 31.5) * P.d;
            const float dyf = (float)dyd;
            const double U1c = (P.f1 * Zcx - Acr + P.half_L) * P.inv_p;
            const double U2c = (P.f2 * Zcy + Aci + P.half_L) * P.inv_p;
            const double npix_d = (double)P.npix;
            int run_pix = -1, run_n = 0;
            for (int k = 0; k < 16; ++k) {
                const int ix = ix0 + k;
                const float2 S = sS[iy * kTile + ix];
                const long long iray = ti0 + ix;
                const bool ok = row_ok && iray < P.i0 + P.ni;
                const double dxd = ((double)ix - 31.5) * P.d;
                const float dxf = (float)dxd;
                const float ds_re = dxf * S.x - dyf * S.y;
                const float ds_im = dxf * S.y + dyf * S.x;
                double al1 = Acr - (double)ds_re;
                double al2 = -(Aci - (double)ds_im);
                for (int q = 0; q < n_near; ++q) {
                    const double wx = sh.near_zx[q] + dxd, wy = sh.near_zy[q] + dyd;
                    const double f = sh.near_m[q] / (wx * wx + wy * wy);
                    al1 += f * wx;
                    al2 += f * wy;
                }
                const double x1 = ((double)iray + 0.5 - P.half_n1) * P.d;
                if (near_overflow) {
                    al1 = al2 = 0.0;
                    for (int q = 0; q < P.n_lens; ++q) {
                        const float4 l = __ldg(P.lens_raw + q);
                        const double wx = x1 - (double)l.x, wy = x2 - (double)l.y;
                        const double f = (double)l.z / (wx * wx + wy * wy);
                        al1 += f * wx;
                        al2 += f * wy;
                    }
                }
                double u1 = (P.f1 * x1 - al1 + P.half_L) * P.inv_p;
                double u2 = (P.f2 * x2 - al2 + P.half_L) * P.inv_p;
                if (n_near == 0 && !near_overflow) {  // common case: same folding as the first kernel
                    u1 = fma(fma(P.f1, dxd, (double)ds_re), P.inv_p, U1c);
                    u2 = fma(fma(P.f2, dyd, -(double)ds_im), P.inv_p, U2c);
                }
                int pix;
                if (!(fabs(u1) <= 1.7976931348623157e308 && fabs(u2) <= 1.7976931348623157e308)) pix = -2;
                else if (u1 >= 0.0 && u1 < npix_d && u2 >= 0.0 && u2 < npix_d) pix = (int)u2 * P.npix + (int)u1;
                else pix = -1;
                if (ok) {
                    n_in += (pix >= 0); n_out += (pix == -1); n_lost += (pix == -2);
                    if (P.ray_y || P.ray_pix) {
                        const long long qidx = (jray - P.j0) * P.ni + (iray - P.i0);
                        if (P.ray_y) { P.ray_y[2 * qidx] = u1 * P.p - P.half_L; P.ray_y[2 * qidx + 1] = u2 * P.p - P.half_L; }
                        if (P.ray_pix) P.ray_pix[qidx] = pix;
                    }
                }
                if (P.count) {
                    const int bp = ok ? pix : -1;
                    if (bp != run_pix) {
                        if (run_pix >= 0) red_add(P.count + run_pix, run_n);
                        run_pix = bp; run_n = 1;
                    } else {
                        ++run_n;
                    }
                }
            }
            if (P.count && run_pix >= 0) red_add(P.count + run_pix, run_n);
        }
        n_in = __reduce_add_sync(0xffffffffu, n_in);
        n_out = __reduce_add_sync(0xffffffffu, n_out);
        n_lost = __reduce_add_sync(0xffffffffu, n_lost);
        if (lane == 0) {
            if (n_in) atomicAdd(&sh.ctr[0], (unsigned long long)n_in);
            if (n_out) atomicAdd(&sh.ctr[1], (unsigned long long)n_out);
            if (n_lost) atomicAdd(&sh.ctr[2], (unsigned long long)n_lost);
        }
        __syncthreads();
        if (tid == 0) { sh.near_n = 0; sh.next_tile = nxt; }
        __syncthreads();
        tile = sh.next_tile;
    }

    if (tid == 0) {
        if (sh.ctr[0]) atomicAdd(&P.counters[0], sh.ctr[0]);
        if (sh.ctr[1]) atomicAdd(&P.counters[1], sh.ctr[1]);
        if (sh.ctr[2]) atomicAdd(&P.counters[2], sh.ctr[2]);
        const unsigned long long tot = sh.ctr[0] + sh.ctr[1] + sh.ctr[2];
        if (tot) atomicAdd(&P.counters[3], tot);
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (is_control) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
}
}  // namespace mlk
