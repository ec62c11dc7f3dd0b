// shoot_ablation_kernels.cuh — compiled ONLY with -DMLENS_ABLATIONS (libmlens_ablations.so: tests and profiling runs).
//
//   shoot_fp32_r1_kernel   the round-1 production kernel, kept as the A/B baseline of the current one: same difference
//                          form around the TILE centre, two accumulators (S_re, S_im) per ray, 1 FADD2 + 5 FFMA2 per ray
//                          pair and one MUFU.RCP per ray ("kernel" 4; its loop variants "shared_rcp", "rays_per_thread")
//   shoot_plain_fp32_kernel  Eq. (1) in plain FP32 in global coordinates — misses the parity tolerances ("kernel" 2)
//   shoot_fp64_kernel      Eq. (1) in plain FP64, one ray per thread — plumbing / debug ("kernel" 0)
#pragma once
#include "shoot_kernel.cuh"

namespace mlk {

// kShared = number of the thread's 4-ray groups (two packed ray pairs A, B) per lens whose four reciprocals come from
// TWO MUFU.RCP instead of four, with packed multiplies only:
//   q = r2A * r2B (FMUL2);  t = (rcp q.x, rcp q.y);  1/r2A = t * r2B (FMUL2);  1/r2B = t * r2A (FMUL2)
// Kept as an ablation switch only: measured on B200 it LOSES (150.7 -> 159.2 -> 175.8 ms for 0/1/2 shared groups,
// round-1 measurement; the register-pair operand rates are in profiles/r2_alu_microbench.txt:
// ffma2_three_distinct_pairs).  Packed FP32 instructions with three distinct register-pair operands are bound by
// register-file read bandwidth (3.0 clk, not 2.0), so the three extra FMUL2 cost more than the two MUFU they save.
// kBin >= 0 fixes the binning route at compile time (the production instantiation: BIN_RUNS); kBin < 0 reads P.bin_mode.
template <int kR, int kShared, int kBin>
__global__ void __launch_bounds__(kTile * kTile / kR, 2) shoot_fp32_r1_kernel(const ShootParams P) {
    const int bin_mode = kBin >= 0 ? kBin : P.bin_mode;
    constexpr int kThreads = kTile * kTile / kR;
    constexpr int kTx = kTile / kR;  // threads along x1
    extern __shared__ __align__(128) unsigned char smem_raw_bytes[];
    TileShared& sh = *reinterpret_cast<TileShared*>(smem_raw_bytes);
    float4* xf = reinterpret_cast<float4*>(smem_raw_bytes + sizeof(TileShared));  // transformed chunk
    float4* raw0 = xf + P.chunk;                                                   // raw staging buffer(s)

    const int tid = threadIdx.x;
    const int lane = tid & 31, warp = tid >> 5;
    const int tx = tid % kTx, ty = tid / kTx;  // kTx threads x kR rays along x1, 64 rows along x2

    if (tid == 0) {
        mbar_init(&sh.bar[0], 1);
        mbar_init(&sh.bar[1], 1);
        mbar_fence_init();
        sh.ctr[0] = sh.ctr[1] = sh.ctr[2] = 0ull;
        sh.near_n = 0;
    }
    __syncthreads();

    // in-tile offsets delta (FP32), identical for every tile
    const float dyf = (float)(((double)ty - 31.5) * P.d);
    float2 dxb[kR / 2];
#pragma unroll
    for (int j = 0; j < kR / 2; ++j) {
        dxb[j].x = (float)(((double)(tx * kR + 2 * j) - 31.5) * P.d);
        dxb[j].y = (float)(((double)(tx * kR + 2 * j + 1) - 31.5) * P.d);
    }

    const double dxt0 = (double)(tx * kR) - 31.5;  // in-tile offset of the thread's first ray, in lattice steps
    const long long n_tiles = (long long)P.tiles_x * P.tiles_y;
    long long g = 0;  // sequence number of the raw-chunk load being consumed: buffer g&1, barrier phase (g>>1)&1

    // single-chunk case: the raw list is staged once and reused by every tile
    if (P.n_lens > 0 && tid == 0 && blockIdx.x < n_tiles) {
        const uint32_t bytes = (uint32_t)min(P.chunk, P.n_lens) * 16u;
        mbar_arrive_expect_tx(&sh.bar[0], bytes);
        bulk_copy_g2s(raw0, P.lens_raw, bytes, &sh.bar[0]);
    }

    // DYNAMIC tile scheduling.  Tiles are equal work, but the warp scheduler favours the older of an SM's two CTAs: with a
    // static split the older one finished its share after ~65 % of the kernel and the other ran the rest alone, with its
    // per-tile bookkeeping exposed (alone: 84 % of the paired rate at N* = 430, 92 % at N* = 2333).  Every CTA takes its
    // first tile by index and every further one from a global counter, fetched one tile ahead by thread 0 so that the
    // atomic's latency is hidden; all CTAs now finish within one tile of each other.  (Which CTA shoots a tile does not
    // affect its arithmetic, and the map is built from integer REDs, so the result is unchanged.)
    long long nxt = 0;  // thread 0 only
    for (long long tile = blockIdx.x; tile < n_tiles;) {
        if (tid == 0) nxt = (long long)atomicAdd(P.tile_counter, 1ull) + gridDim.x;
        const int tJ = (int)(tile / P.tiles_x), tI = (int)(tile - (long long)tJ * P.tiles_x);
        const long long ti0 = P.i0 + (long long)tI * kTile, tj0 = P.j0 + (long long)tJ * kTile;
        const double Zcx = ((double)(ti0 + kTile / 2) - P.half_n1) * P.d;
        const double Zcy = ((double)(tj0 + kTile / 2) - P.half_n2) * P.d;

        float2 Sr[kR / 2], Si[kR / 2];
#pragma unroll
        for (int j = 0; j < kR / 2; ++j) Sr[j] = Si[j] = make_float2(0.f, 0.f);
        double Acr = 0.0, Aci = 0.0;

        for (int c = 0; c < P.n_chunks && P.n_lens > 0; ++c) {
            const int l0 = c * P.chunk;
            const int n_c = min(P.chunk, P.n_lens - l0);
            const int buf = (int)(g & 1);
            float4* raw = raw0 + (size_t)buf * P.chunk;
            // (1) raw chunk landed?  (single-chunk lists are staged once and stay resident: only load 0 is waited for)
            if (P.n_chunks > 1 || tile == (long long)blockIdx.x) mbar_wait(&sh.bar[buf], (uint32_t)((g >> 1) & 1));
            // (2) per-tile FP64 transform: zeta = Z_c - z_i, c = m/zeta; near lenses go to the FP64 list
            double pr_ = 0.0, pi_ = 0.0;
            const int n_pad = (n_c + 3) & ~3;
            for (int t = tid; t < n_pad; t += kThreads) {
                float4 o = make_float4(kFar, kFar, 0.f, 0.f);
                if (t < n_c) {
                    const float4 q = raw[t];
                    const double zx = Zcx - (double)q.x, zy = Zcy - (double)q.y, m = (double)q.z;
                    const double r2 = zx * zx + zy * zy;
                    bool near = r2 < fmax(P.rho2 * fmax(m, 1.0), P.rho2_tile);
                    if (near) {
                        const int slot = atomicAdd(&sh.near_n, 1);
                        if (slot < kNearMax) {
                            sh.near_zx[slot] = zx; sh.near_zy[slot] = zy; sh.near_m[slot] = m;
                        } else {
                            near = false;  // list full: keep the lens in the FP32 list (still summed, less accurate)
                        }
                    }
                    if (!near) {
                        const double inv = m / r2;
                        const double cr = zx * inv, ci = -zy * inv;
                        pr_ += cr; pi_ += ci;
                        o = make_float4((float)zx, (float)zy, (float)cr, (float)ci);
                    }
                }
                xf[t] = o;
            }
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) {
                pr_ += __shfl_xor_sync(0xffffffffu, pr_, off);
                pi_ += __shfl_xor_sync(0xffffffffu, pi_, off);
            }
            if (lane == 0) { sh.part[warp][0] = pr_; sh.part[warp][1] = pi_; }
            __syncthreads();
            // (3) prefetch the next raw chunk (multi-chunk only): the buffer it overwrites was consumed one chunk ago
            if (P.n_chunks > 1 && tid == 0) {
                int cn = c + 1;
                long long tn = tile;
                if (cn == P.n_chunks) { cn = 0; tn = nxt; }
                if (tn < n_tiles) {
                    const int nb = (int)((g + 1) & 1);
                    const uint32_t bytes = (uint32_t)min(P.chunk, P.n_lens - cn * P.chunk) * 16u;
                    mbar_arrive_expect_tx(&sh.bar[nb], bytes);
                    bulk_copy_g2s(raw0 + (size_t)nb * P.chunk, P.lens_raw + (size_t)cn * P.chunk, bytes, &sh.bar[nb]);
                }
            }
            if (P.n_chunks > 1) ++g;
#pragma unroll
            for (int w = 0; w < kThreads / 32; ++w) { Acr += sh.part[w][0]; Aci += sh.part[w][1]; }

            // (4) HOT LOOP: all lenses of the chunk x this thread's kR rays
            float4 qn = xf[0];
#pragma unroll kHotUnroll
            for (int l = 0; l < n_pad; ++l) {
                const float4 q = qn;  // (zeta_x, zeta_y, c_r, c_i)
                qn = xf[l + 1];       // broadcast LDS.128 one lens ahead (xf[n_pad] is readable: raw0 follows xf)
                const float dy = dyf + q.y;
                const float dy2 = dy * dy;
                const float a = q.w * dy;    //  c_i * dy
                const float b = -q.z * dy;   // -c_r * dy
                const float2 NX = make_float2(q.x, q.x), DY2 = make_float2(dy2, dy2);
                const float2 AA = make_float2(a, a), BB = make_float2(b, b);
                const float2 CR = make_float2(q.z, q.z), CI = make_float2(q.w, q.w);
float2 dx[kR / 2], r2[kR / 2], rc[kR / 2];
#pragma unroll
                for (int j = 0; j < kR / 2; ++j) {
                    dx[j] = __fadd2_rn(dxb[j], NX);
                    r2[j] = __ffma2_rn(dx[j], dx[j], DY2);
                }
#pragma unroll
                for (int j = 0; j < kR / 2; j += 2) {
                    if (j / 2 < kShared) {
                        const float2 qq = __fmul2_rn(r2[j], r2[j + 1]);
                        const float2 t = make_float2(rcp_mufu(qq.x), rcp_mufu(qq.y));
                        rc[j] = __fmul2_rn(t, r2[j + 1]);
                        rc[j + 1] = __fmul2_rn(t, r2[j]);
                    } else {
                        rc[j] = make_float2(rcp_mufu(r2[j].x), rcp_mufu(r2[j].y));
                        rc[j + 1] = make_float2(rcp_mufu(r2[j + 1].x), rcp_mufu(r2[j + 1].y));
                    }
                }
#pragma unroll
                for (int j = 0; j < kR / 2; ++j) {
                    const float2 pr = __ffma2_rn(CR, dx[j], AA);
                    const float2 pi = __ffma2_rn(CI, dx[j], BB);
                    Sr[j] = __ffma2_rn(pr, rc[j], Sr[j]);
                    Si[j] = __ffma2_rn(pi, rc[j], Si[j]);
                }
            }
            __syncthreads();  // xf (and sh.part) may be overwritten by the next chunk / tile
        }

        // (5) per-ray FP64 epilogue: alpha, Eq. (1), pixel id; (6) binning
        const int n_near = min(sh.near_n, kNearMax);
        const bool near_overflow = sh.near_n > kNearMax;
        const long long jray = tj0 + ty;
        const bool row_ok = jray < P.j0 + P.nj;
        const double x2 = ((double)jray + 0.5 - P.half_n2) * P.d;
        int n_in = 0, n_out = 0, n_lost = 0;
        int run_pix = -1, run_n = 0;

        if (bin_mode == BIN_WINDOW) {
            // window origin: pixel of the tile centre under the macro-model plus the tile-centre deflection
            if (tid == 0) {
                const double yc1 = P.f1 * Zcx - Acr, yc2 = P.f2 * Zcy + Aci;
                const double u1 = (yc1 + P.half_L) / P.p, u2 = (yc2 + P.half_L) / P.p;
                sh.win_ix0 = (u1 > -1e9 && u1 < 1e9) ? (int)floor(u1) - kWin / 2 : -(1 << 30);
                sh.win_iy0 = (u2 > -1e9 && u2 < 1e9) ? (int)floor(u2) - kWin / 2 : -(1 << 30);
            }
            for (int t = tid; t < kWin * kWin; t += kThreads) sh.win[t] = 0;
            __syncthreads();
        }

        // Source position in PIXEL units, u = (y + L/2)/p.  Everything large is folded into one FP64 constant per tile,
        //   U_c = (f * Z_c -+ A_c + L/2) / p,
        // and a ray adds only its small in-tile part: u = U_c + (f*delta_true -+ delta*S)/p, where delta*S is formed in
        // FP32 (its own rounding, ~1e-9 R_E, is below that of the S accumulators) and delta_true is the exact FP64
        // in-tile offset.  One multiply by 1/p replaces the divide; against the oracle's (y + L/2)/p this moves u by
        // a few ulp (1e-13 px), far inside the 1e-3 px exemption band of the parity tolerance.
        const double U1c = (P.f1 * Zcx - Acr + P.half_L) * P.inv_p;
        const double U2c = (P.f2 * Zcy + Aci + P.half_L) * P.inv_p;
        const double dyt = ((double)ty - 31.5) * P.d;
        const double row2 = P.f2 * dyt;
        const bool special = n_near > 0 || near_overflow;  // tile-uniform: near-lens list or FP64 fallback in play
        const bool want_rays = P.ray_y != nullptr || P.ray_pix != nullptr;
        const double npix_d = (double)P.npix;
        // u1 of ray k = B1 + k*s1 + (delta*S)_re / p  with the thread's first in-tile offset folded into B1
        const double s1 = P.f1 * P.d * P.inv_p;
        const double B1 = fma(dxt0, s1, U1c);
        const double B2 = fma(row2, P.inv_p, U2c);

#pragma unroll
        for (int k = 0; k < kR; ++k) {
            const int j = k >> 1;
            const float srf = (k & 1) ? Sr[j].y : Sr[j].x;
            const float sif = (k & 1) ? Si[j].y : Si[j].x;
            const float dxf = (k & 1) ? dxb[j].y : dxb[j].x;
            const long long iray = ti0 + tx * kR + k;
            const bool ok = row_ok && iray < P.i0 + P.ni;
            // conj(alpha) = A_c - delta*S ; alpha = (Re, -Im);  y1 = f1 x1 - alpha1,  y2 = f2 x2 - alpha2
            const float ds_re = dxf * srf - dyf * sif;
            const float ds_im = dxf * sif + dyf * srf;
            double u1 = fma(f32_to_f64_bits(ds_re), P.inv_p, fma((double)k, s1, B1));
            double u2 = fma(-f32_to_f64_bits(ds_im), P.inv_p, B2);
            bool finite = fabsf(ds_re) <= 3.4028234663852886e38f && fabsf(ds_im) <= 3.4028234663852886e38f;
            if (special) {
                // exact FP64 in-tile offsets here: the float-rounded ones are off by ~1e-9 R_E, which a ray 1e-4 R_E from
                // a lens (deflection gradient m/r^2 ~ 1e8) turns into tens of pixels
                const double dxd = (dxt0 + (double)k) * P.d;
                double al1 = Acr - (double)ds_re;
                double al2 = -(Aci - (double)ds_im);
                for (int q = 0; q < n_near; ++q) {
                    const double wx = sh.near_zx[q] + dxd, wy = sh.near_zy[q] + dyt;
                    const double f = sh.near_m[q] / (wx * wx + wy * wy);
                    al1 += f * wx;
                    al2 += f * wy;
                }
                const double x1 = ((double)iray + 0.5 - P.half_n1) * P.d;
                if (near_overflow) {
                    // more than kNearMax lenses within rho of this tile: the FP32 list then holds lenses it cannot sum
                    // accurately (or at all: r2 = 0), so the tile's rays take Eq. (1) in plain FP64 from global memory
                    al1 = al2 = 0.0;
                    for (int q = 0; q < P.n_lens; ++q) {
                        const float4 l = __ldg(P.lens_raw + q);
                        const double wx = x1 - (double)l.x, wy = x2 - (double)l.y;
                        const double f = (double)l.z / (wx * wx + wy * wy);
                        al1 += f * wx;
                        al2 += f * wy;
                    }
                }
                u1 = (P.f1 * x1 - al1 + P.half_L) * P.inv_p;
                u2 = (P.f2 * x2 - al2 + P.half_L) * P.inv_p;
                finite = fabs(u1) <= 1.7976931348623157e308 && fabs(u2) <= 1.7976931348623157e308;
            }
            int pix;
            if (!finite) {
                pix = -2;  // non-finite source position (ray on a lens): lost
            } else if (u1 >= 0.0 && u1 < npix_d && u2 >= 0.0 && u2 < npix_d) {
                pix = floor_to_int(u2) * P.npix + floor_to_int(u1);
            } else {
                pix = -1;
            }
            if (ok) {
                n_in += (pix >= 0); n_out += (pix == -1); n_lost += (pix == -2);
                if (want_rays) {
                    const long long qidx = (jray - P.j0) * P.ni + (iray - P.i0);
                    if (P.ray_y) { P.ray_y[2 * qidx] = u1 * P.p - P.half_L; P.ray_y[2 * qidx + 1] = u2 * P.p - P.half_L; }
                    if (P.ray_pix) P.ray_pix[qidx] = pix;
                }
            }
            if (P.count) {
                const int bp = ok ? pix : -1;
                if (bin_mode == BIN_PER_RAY) {
                    if (bp >= 0) red_add(P.count + bp, 1);
                } else {
                    // thread-local run-combine: consecutive rays of a thread mostly share a pixel
                    const bool flush = (bp != run_pix);
                    flush_run(P, sh, bin_mode, run_pix, run_n, flush && run_pix >= 0);
                    if (flush) { run_pix = bp; run_n = 1; } else { ++run_n; }
                }
            }
        }
        if (P.count && bin_mode != BIN_PER_RAY) flush_run(P, sh, bin_mode, run_pix, run_n, run_pix >= 0);
        n_in = __reduce_add_sync(0xffffffffu, n_in);
        n_out = __reduce_add_sync(0xffffffffu, n_out);
        n_lost = __reduce_add_sync(0xffffffffu, n_lost);
        if (lane == 0) {
            if (n_in) atomicAdd(&sh.ctr[0], (unsigned long long)n_in);
            if (n_out) atomicAdd(&sh.ctr[1], (unsigned long long)n_out);
            if (n_lost) atomicAdd(&sh.ctr[2], (unsigned long long)n_lost);
        }
        __syncthreads();  // all epilogues done: near list and window are complete
        if (bin_mode == BIN_WINDOW && P.count) {
            for (int t = tid; t < kWin * kWin; t += kThreads) {
                const int v = sh.win[t];
                if (v) {
                    const int ix = sh.win_ix0 + (t % kWin), iy = sh.win_iy0 + (t / kWin);
                    red_add(P.count + (size_t)iy * P.npix + ix, v);
                }
            }
        }
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
}

// ---------------------------------------------------------------------------------------------------------------
// ABLATION ONLY (mlens_set_option("kernel", 2)): the "obvious" FP32 kernel — Eq. (1) summed in plain FP32 in global
// coordinates, same tiling, register blocking, packed arithmetic and MUFU reciprocal as the production kernel but no
// difference form (5 packed FP32 instructions per ray pair instead of 6, no per-tile transform).  It exists to show
// what the difference form buys: this kernel misses the north_star tolerances by 1-2 orders of magnitude
// (tests/test_gpu_parity.py::test_plain_fp32_ablation_fails_the_tolerances).
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(512, 2) shoot_plain_fp32_kernel(const ShootParams P) {
    constexpr int kR = 8, kThreads = 512, kTx = kTile / kR;
    extern __shared__ __align__(128) unsigned char smem_raw_bytes[];
    float4* ls = reinterpret_cast<float4*>(smem_raw_bytes);  // whole lens list (x, y, m, 0), padded to a multiple of 4
    const int tid = threadIdx.x, lane = tid & 31;
    const int tx = tid % kTx, ty = tid / kTx;
    const int n_pad = (P.n_lens + 3) & ~3;
    for (int t = tid; t < n_pad; t += kThreads) ls[t] = t < P.n_lens ? P.lens_raw[t] : make_float4(kFar, kFar, 0.f, 0.f);
    __syncthreads();
    const long long n_tiles = (long long)P.tiles_x * P.tiles_y;
    unsigned long long c_in = 0, c_out = 0, c_lost = 0;
    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const int tJ = (int)(tile / P.tiles_x), tI = (int)(tile - (long long)tJ * P.tiles_x);
        const long long jray = P.j0 + (long long)tJ * kTile + ty;
        const long long iray0 = P.i0 + (long long)tI * kTile + tx * kR;
        const double x2 = ((double)jray + 0.5 - P.half_n2) * P.d;
        const float x2f = (float)x2;
        float2 xf[kR / 2], ax[kR / 2], ay[kR / 2];
#pragma unroll
        for (int j = 0; j < kR / 2; ++j) {
            xf[j].x = (float)(((double)(iray0 + 2 * j) + 0.5 - P.half_n1) * P.d);
            xf[j].y = (float)(((double)(iray0 + 2 * j + 1) + 0.5 - P.half_n1) * P.d);
            ax[j] = ay[j] = make_float2(0.f, 0.f);
        }
#pragma unroll 4
        for (int l = 0; l < n_pad; ++l) {
            const float4 q = ls[l];
            const float dy = x2f - q.y, dy2 = dy * dy;
            const float2 NX = make_float2(-q.x, -q.x), DY2 = make_float2(dy2, dy2), M = make_float2(q.z, q.z);
            const float2 DY = make_float2(dy, dy);
#pragma unroll
            for (int j = 0; j < kR / 2; ++j) {
                const float2 dx = __fadd2_rn(xf[j], NX);
                const float2 r2 = __ffma2_rn(dx, dx, DY2);
                const float2 w = __fmul2_rn(M, make_float2(rcp_mufu(r2.x), rcp_mufu(r2.y)));
                ax[j] = __ffma2_rn(w, dx, ax[j]);
                ay[j] = __ffma2_rn(w, DY, ay[j]);
            }
        }
        int n_in = 0, n_out = 0, n_lost = 0;
#pragma unroll
        for (int k = 0; k < kR; ++k) {
            const int j = k >> 1;
            const long long iray = iray0 + k;
            const bool ok = jray < P.j0 + P.nj && iray < P.i0 + P.ni;
            const double x1 = ((double)iray + 0.5 - P.half_n1) * P.d;
            const double y1 = P.f1 * x1 - (double)((k & 1) ? ax[j].y : ax[j].x);
            const double y2 = P.f2 * x2 - (double)((k & 1) ? ay[j].y : ay[j].x);
            int pix;
            if (!(isfinite(y1) && isfinite(y2))) {
                pix = -2;
            } else {
                const double u1 = (y1 + P.half_L) / P.p, u2 = (y2 + P.half_L) / P.p;
                pix = (u1 >= 0.0 && u1 < (double)P.npix && u2 >= 0.0 && u2 < (double)P.npix)
                          ? (int)floor(u2) * P.npix + (int)floor(u1) : -1;
            }
            if (ok) {
                n_in += (pix >= 0); n_out += (pix == -1); n_lost += (pix == -2);
                if (P.ray_y || P.ray_pix) {
                    const long long qidx = (jray - P.j0) * P.ni + (iray - P.i0);
                    if (P.ray_y) { P.ray_y[2 * qidx] = y1; P.ray_y[2 * qidx + 1] = y2; }
                    if (P.ray_pix) P.ray_pix[qidx] = pix;
                }
                if (P.count && pix >= 0) red_add(P.count + pix, 1);
            }
        }
        n_in = __reduce_add_sync(0xffffffffu, n_in);
        n_out = __reduce_add_sync(0xffffffffu, n_out);
        n_lost = __reduce_add_sync(0xffffffffu, n_lost);
        c_in += n_in; c_out += n_out; c_lost += n_lost;
    }
    if (lane == 0) {
        if (c_in) atomicAdd(&P.counters[0], c_in);
        if (c_out) atomicAdd(&P.counters[1], c_out);
        if (c_lost) atomicAdd(&P.counters[2], c_lost);
        if (c_in + c_out + c_lost) atomicAdd(&P.counters[3], c_in + c_out + c_lost);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// plumbing / debug kernel: Eq. (1) in plain FP64, one ray per thread, lenses read from global memory
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) shoot_fp64_kernel(const ShootParams P) {
    const long long n_rays = P.ni * P.nj;
    int n_in = 0, n_out = 0, n_lost = 0;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n_rays; q += (long long)gridDim.x * blockDim.x) {
        const long long jj = q / P.ni, ii = q - jj * P.ni;
        const double x1 = ((double)(P.i0 + ii) + 0.5 - P.half_n1) * P.d;
        const double x2 = ((double)(P.j0 + jj) + 0.5 - P.half_n2) * P.d;
        double a1 = 0.0, a2 = 0.0;
        for (int k = 0; k < P.n_lens; ++k) {
            const float4 l = __ldg(P.lens_raw + k);
            const double dx = x1 - (double)l.x, dy = x2 - (double)l.y;
            const double w = (double)l.z / (dx * dx + dy * dy);
            a1 += w * dx;
            a2 += w * dy;
        }
        const double y1 = P.f1 * x1 - a1, y2 = P.f2 * x2 - a2;
        int pix;
        if (!(isfinite(y1) && isfinite(y2))) {
            pix = -2;
        } else {
            const double u1 = (y1 + P.half_L) / P.p, u2 = (y2 + P.half_L) / P.p;
            pix = (u1 >= 0.0 && u1 < (double)P.npix && u2 >= 0.0 && u2 < (double)P.npix)
                      ? (int)floor(u2) * P.npix + (int)floor(u1) : -1;
        }
        n_in += (pix >= 0); n_out += (pix == -1); n_lost += (pix == -2);
        if (P.ray_y) { P.ray_y[2 * q] = y1; P.ray_y[2 * q + 1] = y2; }
        if (P.ray_pix) P.ray_pix[q] = pix;
        if (P.count && pix >= 0) red_add(P.count + pix, 1);
    }
    n_in = __reduce_add_sync(0xffffffffu, n_in);
    n_out = __reduce_add_sync(0xffffffffu, n_out);
    n_lost = __reduce_add_sync(0xffffffffu, n_lost);
    if ((threadIdx.x & 31) == 0) {
        if (n_in) atomicAdd(&P.counters[0], (unsigned long long)n_in);
        if (n_out) atomicAdd(&P.counters[1], (unsigned long long)n_out);
        if (n_lost) atomicAdd(&P.counters[2], (unsigned long long)n_lost);
        if (n_in + n_out + n_lost) atomicAdd(&P.counters[3], (unsigned long long)(n_in + n_out + n_lost));
    }
}


}  // namespace mlk
