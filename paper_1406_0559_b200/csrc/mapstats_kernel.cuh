// mapstats_kernel.cuh — on-device map statistics: the full magnification probability
// distribution and the map means that GERLUMPH stores next to every map.
//
//   PAPER.md:307  mpd.dat: "the frequency of each magnification value in a map is counted and then divided by the
//                 total number of pixels".  Magnification is count/N_avg (Eq. 4) and counts are
//                 integers, so the full MPD is the histogram of the int32 ray counts: hist[c] = #pixels with count c.
//   PAPER.md:299  mapmeta.dat: average number of rays per pixel <N> and average magnification <mu> = <N>/N_avg.
//
// Integer work throughout (bit-exact against the oracle).  HBM-bound: 4 bytes read per pixel, int4-vectorised
// grid-stride loads by one persistent 1024-thread CTA per SM; a CTA-private shared-memory histogram (up to 48 Ki bins =
// 192 KB) takes the counts below `smem_bins` (a warp whose 32 lanes hold one value adds it once), larger counts go
// straight to the global 64-bit bins.  The CTA histograms are written to private slices of a scratch buffer and summed
// by mpd_reduce_kernel: flushing them with global atomics instead puts ~600 same-address atomics on every bin and
// costs 6x the whole streaming pass (measured 0.45 ms vs 0.08 ms on a 10000^2 map).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mlk {

constexpr int kMpdSmemBinsMax = 49152;  // 192 KB of u32 bins per CTA (1 CTA per SM)
constexpr int kMpdThreads = 1024;

struct MapStatsDev {               // device-side accumulator, zeroed (memset) before the launch
    unsigned long long sum_count;  // sum of all pixel counts
    unsigned long long n_clamped;  // pixels whose count was >= n_bins-1 (they all sit in the last bin)
    int max_count;
    int inv_min_count;             // INT_MAX - min(count), so that an all-zero struct is the neutral element
};

// One pixel.  `lim` = min(smem_bins, n_bins-1): a single unsigned compare sends the common case (0 <= c < lim) to the
// shared-memory bin; negative values (corrupt input -> bin 0), clamped counts (>= n_bins-1 -> last bin) and counts
// beyond the shared-memory bins take the slow path.
__device__ __forceinline__ void mpd_add(unsigned int* sh, unsigned lim, int smem_bins, unsigned long long* hist, int n_bins,
                                        int c, unsigned long long& clamped) {
    if ((unsigned)c < lim) {
        atomicAdd(&sh[c], 1u);
    } else {
        int b = c < 0 ? 0 : c;
        if (b >= n_bins - 1) { b = n_bins - 1; ++clamped; }
        if (b < smem_bins) atomicAdd(&sh[b], 1u);
        else atomicAdd(&hist[b], 1ull);
    }
}

__global__ void __launch_bounds__(kMpdThreads, 1) mpd_kernel(const int* __restrict__ count, long long n,
                                                             unsigned long long* __restrict__ hist, int n_bins,
                                                             int smem_bins, unsigned int* __restrict__ partial,
                                                             MapStatsDev* __restrict__ out) {
    extern __shared__ unsigned int sh[];  // smem_bins bins
    for (int t = threadIdx.x; t < smem_bins; t += kMpdThreads) sh[t] = 0u;
    __syncthreads();

    unsigned long long sum = 0ull, clamped = 0ull;
    int vmax = 0, vmin = 0x7fffffff;
    const unsigned lim = (unsigned)min(smem_bins, n_bins - 1);
    const long long n4 = n >> 2;
    const long long stride = (long long)gridDim.x * kMpdThreads;
    // the loop bound is warp-uniform (rounded up to whole warps) so that the warp votes always see converged warps
    const long long base0 = (long long)blockIdx.x * kMpdThreads + (threadIdx.x & ~31);
    constexpr int kInFlight = 4;  // independent 16-byte loads per thread: 64 KB in flight per SM covers HBM latency
    for (long long qb = base0; qb < n4; qb += kInFlight * stride) {
        int4 v[kInFlight];
        bool ok[kInFlight];
#pragma unroll
        for (int u = 0; u < kInFlight; ++u) {
            const long long q = qb + (threadIdx.x & 31) + u * stride;
            ok[u] = q < n4;
            v[u] = make_int4(0, 0, 0, 0);
            if (ok[u]) v[u] = __ldg(reinterpret_cast<const int4*>(count) + q);
        }
#pragma unroll
        for (int u = 0; u < kInFlight; ++u) {
            const int4 w = v[u];
            // flat regions (smooth-matter maps, the no-lens closed form): all 128 pixels of the warp's 512-byte row
            // segment hold one value, which would serialise the shared-memory atomic 32 ways -> one vote per int4,
            // one add of 128.  Elsewhere neighbouring counts differ (Poisson-like scatter) and conflicts are rare.
            const int w0 = __shfl_sync(0xffffffffu, w.x, 0);
            const bool flat = __all_sync(0xffffffffu, ok[u] && w.x == w0 && w.y == w0 && w.z == w0 && w.w == w0);
            if (ok[u]) {
                sum += (unsigned long long)((long long)w.x + w.y + w.z + w.w);
                vmax = max(max(vmax, max(w.x, w.y)), max(w.z, w.w));
                vmin = min(min(vmin, min(w.x, w.y)), min(w.z, w.w));
            }
            if (flat && (unsigned)w0 < lim) {
                if ((threadIdx.x & 31) == 0) atomicAdd(&sh[w0], 128u);
            } else if (ok[u]) {
                mpd_add(sh, lim, smem_bins, hist, n_bins, w.x, clamped);
                mpd_add(sh, lim, smem_bins, hist, n_bins, w.y, clamped);
                mpd_add(sh, lim, smem_bins, hist, n_bins, w.z, clamped);
                mpd_add(sh, lim, smem_bins, hist, n_bins, w.w, clamped);
            }
        }
    }
    if (blockIdx.x == 0 && threadIdx.x < (int)(n - (n4 << 2))) {  // ragged tail (< 4 pixels): plain global atomics
        const int c = count[(n4 << 2) + threadIdx.x];
        sum += (unsigned long long)c;
        vmax = max(vmax, c);
        vmin = min(vmin, c);
        int b = c < 0 ? 0 : c;
        if (b >= n_bins - 1) { b = n_bins - 1; ++clamped; }
        atomicAdd(&hist[b], 1ull);
    }
    __syncthreads();
    // this CTA's histogram -> its private slice (plain coalesced stores); mpd_reduce_kernel sums the slices
    for (int t = threadIdx.x; t < smem_bins; t += kMpdThreads) partial[(size_t)blockIdx.x * smem_bins + t] = sh[t];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        sum += __shfl_xor_sync(0xffffffffu, sum, off);
        clamped += __shfl_xor_sync(0xffffffffu, clamped, off);
    }
    vmax = __reduce_max_sync(0xffffffffu, vmax);
    vmin = __reduce_min_sync(0xffffffffu, vmin);
    if ((threadIdx.x & 31) == 0) {
        if (sum) atomicAdd(&out->sum_count, sum);
        if (clamped) atomicAdd(&out->n_clamped, clamped);
        atomicMax(&out->max_count, vmax);
        atomicMax(&out->inv_min_count, 0x7fffffff - vmin);
    }
}

// hist[t] += sum over CTAs of partial[cta][t].  32 bins x 8 slice-groups per 256-thread block: reads are coalesced
// across the 32 bins, every thread has ~n_ctas/8 independent loads (a single thread walking all 148 slices is
// latency-bound: ~90 us), no contended atomics.
__global__ void __launch_bounds__(256) mpd_reduce_kernel(const unsigned int* __restrict__ partial, int n_ctas, int smem_bins,
                                                         unsigned long long* __restrict__ hist, int n_bins) {
    __shared__ unsigned long long part[8][32];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int t = blockIdx.x * 32 + tx;
    unsigned long long v = 0ull;
    if (t < smem_bins && t < n_bins) {
#pragma unroll 4
        for (int g = ty; g < n_ctas; g += 8) v += partial[(size_t)g * smem_bins + t];
    }
    part[ty][tx] = v;
    __syncthreads();
    if (ty == 0 && t < smem_bins && t < n_bins) {
#pragma unroll
        for (int k = 1; k < 8; ++k) v += part[k][tx];
        if (v) atomicAdd(&hist[t], v);  // ragged-tail pixels and counts >= smem_bins were added atomically by mpd_kernel
    }
}

}  // namespace mlk
