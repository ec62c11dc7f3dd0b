// mapstats_kernel.cuh — on-device map statistics: the full magnification probability
// distribution and the map means that GERLUMPH stores next to every map.
//
//   PAPER.md:307  mpd.dat: "the frequency of each magnification value in a map is counted and then divided by the
//                 total number of pixels".  Magnification is count/N_avg (Eq. 4) and counts are
//                 integers, so the full MPD is the histogram of the int32 ray counts: hist[c] = #pixels with count c.
//   PAPER.md:299  mapmeta.dat: average number of rays per pixel <N> and average magnification <mu> = <N>/N_avg.
//
// Integer work throughout (bit-exact against the oracle).  HBM-bound: 4 bytes read per pixel, int4-vectorised
// grid-stride loads; a CTA-private shared-memory histogram takes the counts below kMpdSmemBins, equal counts of a warp
// are combined first (match.any), the few larger counts go straight to the global 64-bit bins.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mlk {

constexpr int kMpdSmemBins = 8192;  // 32 KB of u32 bins per CTA
constexpr int kMpdThreads = 256;

struct MapStatsDev {               // device-side accumulator, zeroed (memset) before the launch
    unsigned long long sum_count;  // sum of all pixel counts
    unsigned long long n_clamped;  // pixels whose count was >= n_bins-1 (they all sit in the last bin)
    int max_count;
    int inv_min_count;             // INT_MAX - min(count), so that an all-zero struct is the neutral element
};

// Called convergently by all 32 lanes of a warp; `valid` = this lane holds a pixel.
__device__ __forceinline__ void mpd_add(unsigned int* sh, unsigned long long* hist, int n_bins, int c, bool valid,
                                        unsigned long long& clamped) {
    // counts are >= 0 by construction; a negative value (corrupt input) is put in bin 0 rather than written out of range
    int b = c < 0 ? 0 : c;
    if (valid && b >= n_bins - 1) { b = n_bins - 1; ++clamped; }
    const bool in_smem = valid && b < kMpdSmemBins;
    // warp aggregation: lanes holding the same shared-memory bin elect one leader (smooth maps put most pixels in a few
    // bins, which would otherwise serialise the shared-memory atomic 32 ways); other lanes get a unique key
    const int key = in_smem ? b : -1 - (int)(threadIdx.x & 31);
    const unsigned peers = __match_any_sync(0xffffffffu, key);
    if (in_smem) {
        if ((int)(threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(&sh[b], (unsigned)__popc(peers));
    } else if (valid) {
        atomicAdd(&hist[b], 1ull);
    }
}

__global__ void __launch_bounds__(kMpdThreads) mpd_kernel(const int* __restrict__ count, long long n,
                                                          unsigned long long* __restrict__ hist, int n_bins,
                                                          MapStatsDev* __restrict__ out) {
    __shared__ unsigned int sh[kMpdSmemBins];
    for (int t = threadIdx.x; t < kMpdSmemBins; t += kMpdThreads) sh[t] = 0u;
    __syncthreads();

    unsigned long long sum = 0ull, clamped = 0ull;
    int vmax = 0, vmin = 0x7fffffff;
    const long long n4 = n >> 2;
    const long long stride = (long long)gridDim.x * kMpdThreads;
    // the loop bound is warp-uniform (rounded up to whole warps) so that match.any always sees converged warps
    const long long base0 = (long long)blockIdx.x * kMpdThreads + (threadIdx.x & ~31);
    for (long long qb = base0; qb < n4; qb += stride) {
        const long long q = qb + (threadIdx.x & 31);
        const bool valid = q < n4;
        int4 c = make_int4(0, 0, 0, 0);
        if (valid) {
            c = __ldg(reinterpret_cast<const int4*>(count) + q);
            sum += (unsigned long long)((long long)c.x + c.y + c.z + c.w);
            vmax = max(max(vmax, max(c.x, c.y)), max(c.z, c.w));
            vmin = min(min(vmin, min(c.x, c.y)), min(c.z, c.w));
        }
        mpd_add(sh, hist, n_bins, c.x, valid, clamped);
        mpd_add(sh, hist, n_bins, c.y, valid, clamped);
        mpd_add(sh, hist, n_bins, c.z, valid, clamped);
        mpd_add(sh, hist, n_bins, c.w, valid, clamped);
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
    for (int t = threadIdx.x; t < kMpdSmemBins && t < n_bins; t += kMpdThreads) {
        const unsigned v = sh[t];
        if (v) atomicAdd(&hist[t], (unsigned long long)v);
    }
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

}  // namespace mlk
