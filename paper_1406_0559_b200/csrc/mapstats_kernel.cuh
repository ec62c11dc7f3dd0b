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
// shared-memory bin and does NOTHING else — the sum, minimum and maximum of those pixels are read off the finished
// histogram by mpd_reduce_kernel (sum = sum_t t*hist[t], min/max = first/last non-empty bin), which takes a dozen
// integer instructions per int4 out of the streaming loop.  Negative values (corrupt input -> bin 0), clamped counts
// (>= n_bins-1 -> last bin) and counts beyond the shared-memory bins take the slow path, which keeps its own statistics.
__device__ __forceinline__ void mpd_add(unsigned int* sh, unsigned lim, int smem_bins, unsigned long long* hist, int n_bins,
                                        int c, unsigned long long& clamped, unsigned long long& sum, int& vmax, int& vmin) {
    if ((unsigned)c < lim) {
        atomicAdd(&sh[c], 1u);
    } else {
        sum += (unsigned long long)(long long)c;
        vmax = max(vmax, c);
        vmin = min(vmin, c);
        int b = c < 0 ? 0 : c;
        if (b >= n_bins - 1) { b = n_bins - 1; ++clamped; }
        if (b < smem_bins) atomicAdd(&sh[b], 1u);  // only the slow path puts pixels into shared bins >= lim (the last bin)
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
    // kInFlight independent 16-byte loads per thread, DOUBLE-BUFFERED: the next batch is requested before the current one
    // is binned, so loads stay in flight during the shared-memory atomics too (ncu of the single-buffered loop: 4.6
    // long-scoreboard stall cycles per issued instruction, 54 % issue-slot use — latency-bound, not bandwidth-bound).
    constexpr int kInFlight = 4;
    const int lane = threadIdx.x & 31;
    auto load_batch = [&](long long qb, int4 (&v)[kInFlight], unsigned& okmask) {
        okmask = 0u;
#pragma unroll
        for (int u = 0; u < kInFlight; ++u) {
            const long long q = qb + lane + u * stride;
            v[u] = make_int4(0, 0, 0, 0);
            if (qb < n4 && q < n4) {
                v[u] = __ldg(reinterpret_cast<const int4*>(count) + q);
                okmask |= 1u << u;
            }
        }
    };
    int4 cur[kInFlight], nxt[kInFlight];
    unsigned ok_cur, ok_nxt;
    load_batch(base0, cur, ok_cur);
    for (long long qb = base0; qb < n4; qb += kInFlight * stride) {
        load_batch(qb + kInFlight * stride, nxt, ok_nxt);
#pragma unroll
        for (int u = 0; u < kInFlight; ++u) {
            const int4 w = cur[u];
            const bool ok = (ok_cur >> u) & 1u;
            // flat regions (smooth-matter maps, the no-lens closed form): all 128 pixels of the warp's 512-byte row
            // segment hold one value, which would serialise the shared-memory atomic 32 ways -> one vote per int4,
            // one add of 128.  Elsewhere neighbouring counts differ (Poisson-like scatter) and conflicts are rare.
            const int w0 = __shfl_sync(0xffffffffu, w.x, 0);
            const bool flat = __all_sync(0xffffffffu, ok && w.x == w0 && w.y == w0 && w.z == w0 && w.w == w0);
            if (flat && (unsigned)w0 < lim) {
                if (lane == 0) atomicAdd(&sh[w0], 128u);
            } else if (ok) {
                mpd_add(sh, lim, smem_bins, hist, n_bins, w.x, clamped, sum, vmax, vmin);
                mpd_add(sh, lim, smem_bins, hist, n_bins, w.y, clamped, sum, vmax, vmin);
                mpd_add(sh, lim, smem_bins, hist, n_bins, w.z, clamped, sum, vmax, vmin);
                mpd_add(sh, lim, smem_bins, hist, n_bins, w.w, clamped, sum, vmax, vmin);
            }
        }
#pragma unroll
        for (int u = 0; u < kInFlight; ++u) cur[u] = nxt[u];
        ok_cur = ok_nxt;
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
// The statistics of the fast-path pixels (count < lim = min(smem_bins, n_bins-1)) come from here: bin t holds v pixels of
// count t, so they add t*v to the sum and, if v > 0, make t a candidate for the minimum and the maximum.
__global__ void __launch_bounds__(256) mpd_reduce_kernel(const unsigned int* __restrict__ partial, int n_ctas, int smem_bins,
                                                         unsigned long long* __restrict__ hist, int n_bins,
                                                         MapStatsDev* __restrict__ out) {
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
    if (ty == 0) {  // warp 0: statistics of the fast-path bins of this block
        const bool fast = t < min(smem_bins, n_bins - 1);
        unsigned long long s = fast ? v * (unsigned long long)t : 0ull;
        int lo = (fast && v) ? t : 0x7fffffff, hi = (fast && v) ? t : 0;
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
        lo = __reduce_min_sync(0xffffffffu, lo);
        hi = __reduce_max_sync(0xffffffffu, hi);
        if (tx == 0) {
            if (s) atomicAdd(&out->sum_count, s);
            if (hi > 0) atomicMax(&out->max_count, hi);
            if (lo != 0x7fffffff) atomicMax(&out->inv_min_count, 0x7fffffff - lo);
        }
    }
}

}  // namespace mlk

// ---------------------------------------------------------------------------------------------------------------
// Indexed maps: "convert a map with ray-counts to an indexed map and an index
// file.  The index file will hold all the distinct ray-count values, each matched to an index running from zero ...
// The indexed map will have its pixel ray-count values replaced by the appropriate index", stored in 16 bits.
// The distinct values are the non-empty bins of the MPD histogram, so the index file is a stream compaction of it.
// ---------------------------------------------------------------------------------------------------------------
namespace mlk {

// One CTA: exclusive scan of (hist[b] != 0) over all bins -> lut[b] = index of count value b (or -1), values[index] = b
// in ascending order, *n_distinct = number of non-empty bins.  n_bins <= ~1e6, so a single 1024-thread CTA walking the
// bins in 1024-wide strips with a running offset is enough (a few tens of microseconds).
__global__ void __launch_bounds__(1024, 1) index_build_kernel(const unsigned long long* __restrict__ hist, int n_bins,
                                                              int* __restrict__ lut, int* __restrict__ values,
                                                              int max_values, int* __restrict__ n_distinct) {
    __shared__ int warp_sums[32];
    __shared__ int base;
    if (threadIdx.x == 0) base = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int b0 = 0; b0 < n_bins; b0 += 1024) {
        const int b = b0 + threadIdx.x;
        const int flag = (b < n_bins && hist[b] != 0ull) ? 1 : 0;
        int incl = flag;  // inclusive warp scan
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, off);
            if (lane >= off) incl += t;
        }
        if (lane == 31) warp_sums[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            int w = warp_sums[lane], wi = w;
#pragma unroll
            for (int off = 1; off < 32; off <<= 1) {
                const int t = __shfl_up_sync(0xffffffffu, wi, off);
                if (lane >= off) wi += t;
            }
            warp_sums[lane] = wi - w;  // exclusive offsets of the warps
        }
        __syncthreads();
        const int idx = base + warp_sums[warp] + incl - flag;
        if (b < n_bins) {
            lut[b] = flag ? idx : -1;
            if (flag && idx < max_values) values[idx] = b;
        }
        __syncthreads();
        if (threadIdx.x == 1023) base = idx + flag;
        __syncthreads();
    }
    if (threadIdx.x == 0) *n_distinct = base;
}

// indexed[q] = lut[count[q]] as 16-bit; 4 pixels per thread per iteration (int4 in, 8 bytes out): 6 B/pixel of HBM
// traffic, the LUT (4 B x n_bins) is served from L1/L2.
__global__ void __launch_bounds__(256) index_apply_kernel(const int* __restrict__ count, long long n, const int* __restrict__ lut,
                                                          unsigned short* __restrict__ indexed) {
    const long long n4 = n >> 2, stride = (long long)gridDim.x * 256;
    for (long long q = (long long)blockIdx.x * 256 + threadIdx.x; q < n4; q += stride) {
        const int4 c = __ldg(reinterpret_cast<const int4*>(count) + q);
        ushort4 o;
        // counts are >= 0 by construction; max(c, 0) keeps a corrupt negative from reading outside the table
        o.x = (unsigned short)__ldg(lut + max(c.x, 0)); o.y = (unsigned short)__ldg(lut + max(c.y, 0));
        o.z = (unsigned short)__ldg(lut + max(c.z, 0)); o.w = (unsigned short)__ldg(lut + max(c.w, 0));
        reinterpret_cast<ushort4*>(indexed)[q] = o;
    }
    for (long long q = (n4 << 2) + (long long)blockIdx.x * 256 + threadIdx.x; q < n; q += stride)
        indexed[q] = (unsigned short)__ldg(lut + max(count[q], 0));
}

// count[q] = values[indexed[q]] (the decode direction)
__global__ void __launch_bounds__(256) index_decode_kernel(const unsigned short* __restrict__ indexed, long long n,
                                                           const int* __restrict__ values, int n_values, int* __restrict__ count) {
    const long long n4 = n >> 2, stride = (long long)gridDim.x * 256;
    for (long long q = (long long)blockIdx.x * 256 + threadIdx.x; q < n4; q += stride) {
        const ushort4 i = __ldg(reinterpret_cast<const ushort4*>(indexed) + q);
        int4 c;
        c.x = i.x < n_values ? __ldg(values + i.x) : -1; c.y = i.y < n_values ? __ldg(values + i.y) : -1;
        c.z = i.z < n_values ? __ldg(values + i.z) : -1; c.w = i.w < n_values ? __ldg(values + i.w) : -1;
        reinterpret_cast<int4*>(count)[q] = c;
    }
    for (long long q = (n4 << 2) + (long long)blockIdx.x * 256 + threadIdx.x; q < n; q += stride)
        count[q] = indexed[q] < n_values ? __ldg(values + indexed[q]) : -1;
}

// ---------------------------------------------------------------------------------------------------------------
// Minimal-bit-width storage (Table B.6): "rather than using the standard 16-bit and 32-bit data
// types, we could define our own data types, using in each case the minimum required number of bits to represent a
// particular map".  Value q (masked to `bits` bits) occupies bits [q*bits, (q+1)*bits) of a little-endian bit stream
// held in 32-bit words.  HBM-bound: src bytes in, bits/8 bytes out per value.
// ---------------------------------------------------------------------------------------------------------------
//
// pack: 32 values fill exactly `bits` words, so the bit layout repeats with a period of `bits` words.  A CTA takes a
// chunk of n_sub x K whole periods (K = 256 / bits, about 8192 values): the values come in with coalesced 16-byte loads
// into shared memory (several per thread in flight), then thread t < K*bits builds word r = t % bits of period t / bits of
// every one of the n_sub sub-blocks — the first value that touches its word, the bit offset inside that value and the
// number of values it needs are the same each time and computed once.  (One output word per thread straight from global
// memory ran at 28 % of the copy peak: a 64-bit division per word and three dependent 2-byte loads per thread in flight.)
constexpr int kPackChunkValues = 8192;  // upper bound of the values of one chunk (shared memory: 16 KB / 32 KB)

template <typename SrcT>
__global__ void __launch_bounds__(256) pack_bits_kernel(const SrcT* __restrict__ src, long long n, int bits,
                                                        unsigned int* __restrict__ packed, long long n_words, int n_sub) {
    __shared__ __align__(16) SrcT sv[kPackChunkValues];
    const unsigned int mask = bits >= 32 ? 0xffffffffu : ((1u << bits) - 1u);
    const int periods = 256 / bits;                 // per sub-block (bits <= 32 -> >= 8)
    const int words_per_sub = periods * bits, vals_per_sub = periods * 32;
    const int chunk_vals = n_sub * vals_per_sub;    // <= kPackChunkValues, a multiple of 32 values (>= 64 bytes)
    const long long chunk_words = (long long)n_sub * words_per_sub;
    const int t = threadIdx.x;
    const int r = t % bits, g = t / bits;           // word r of period g of each sub-block
    const int q_in = (32 * r) / bits;               // first value of the period that has bits in word r
    const int off = 32 * r - q_in * bits;           // bits of that value that went into word r - 1
    const int n_vals = (off + 31) / bits + 1;       // values with bits in word r (the last may lie beyond a ragged end)
    constexpr int kVec = 16 / (int)sizeof(SrcT);
    const unsigned int mask_vec = sizeof(SrcT) == 2 ? (mask & 0xffffu) * 0x10001u : mask;  // two 16-bit lanes per word
    const long long n_chunks = (n + chunk_vals - 1) / chunk_vals;
    for (long long c = blockIdx.x; c < n_chunks; c += gridDim.x) {
        const long long base = c * chunk_vals;
        __syncthreads();                            // the previous chunk has been consumed
        if (base + chunk_vals <= n) {               // values are masked to `bits` bits here, 4 or 8 at a time
            const uint4* gsrc = reinterpret_cast<const uint4*>(src + base);
            for (int v = t; v < chunk_vals / kVec; v += 256) {
                uint4 x = __ldg(gsrc + v);
                x.x &= mask_vec; x.y &= mask_vec; x.z &= mask_vec; x.w &= mask_vec;
                reinterpret_cast<uint4*>(sv)[v] = x;
            }
        } else {                                    // ragged end: zero-filled
            for (int v = t; v < chunk_vals; v += 256) sv[v] = base + v < n ? (SrcT)((unsigned int)src[base + v] & mask) : (SrcT)0;
        }
        __syncthreads();
        if (t < words_per_sub) {
            const SrcT* mine = sv + g * 32 + q_in;
            long long w = c * chunk_words + t;
            for (int sub = 0; sub < n_sub && w < n_words; ++sub, w += words_per_sub, mine += vals_per_sub) {
                // value k starts at bit k*bits - off of the word: the first one loses its low `off` bits to the previous
                // word, the others are shifted up by less than 32 (they overlap the word) — 32-bit shifts only
                unsigned int acc = (unsigned int)mine[0] >> off;
#pragma unroll 4
                for (int k = 1; k < n_vals; ++k) acc |= (unsigned int)mine[k] << (k * bits - off);
                packed[w] = acc;
            }
        }
    }
}

// unpack: 16 bytes of output per thread (4 int32 or 8 uint16 values).  Their bits span at most five consecutive words:
// five loads per thread, then the 160-bit window is shifted down by `bits` per value (funnel shifts) — a two-word window
// per value costs 16 loads per thread and was bound by L1 wavefronts (51 % of the copy peak).
template <typename DstT>
__global__ void __launch_bounds__(256) unpack_bits_kernel(const unsigned int* __restrict__ packed, long long n, int bits,
                                                          DstT* __restrict__ dst, long long n_words) {
    constexpr int kPer = 16 / (int)sizeof(DstT);
    const unsigned int mask = bits >= 32 ? 0xffffffffu : ((1u << bits) - 1u);
    const long long stride = (long long)gridDim.x * 256, n_vec = n / kPer;
    for (long long v = (long long)blockIdx.x * 256 + threadIdx.x; v < n_vec; v += stride) {
        const long long bit0 = v * kPer * bits;
        const long long w0 = bit0 >> 5;
        const int sh = (int)(bit0 & 31);
        unsigned int x0 = __ldg(packed + w0);
        unsigned int x1 = w0 + 1 < n_words ? __ldg(packed + w0 + 1) : 0u;
        unsigned int x2 = w0 + 2 < n_words ? __ldg(packed + w0 + 2) : 0u;
        unsigned int x3 = w0 + 3 < n_words ? __ldg(packed + w0 + 3) : 0u;
        unsigned int x4 = w0 + 4 < n_words ? __ldg(packed + w0 + 4) : 0u;
        x0 = __funnelshift_rc(x0, x1, sh); x1 = __funnelshift_rc(x1, x2, sh); x2 = __funnelshift_rc(x2, x3, sh);
        x3 = __funnelshift_rc(x3, x4, sh); x4 >>= sh;
        alignas(16) DstT out[kPer];
#pragma unroll
        for (int k = 0; k < kPer; ++k) {
            out[k] = (DstT)(x0 & mask);
            x0 = __funnelshift_rc(x0, x1, bits); x1 = __funnelshift_rc(x1, x2, bits); x2 = __funnelshift_rc(x2, x3, bits);
            x3 = __funnelshift_rc(x3, x4, bits); x4 = bits >= 32 ? 0u : x4 >> bits;
        }
        reinterpret_cast<uint4*>(dst)[v] = *reinterpret_cast<const uint4*>(out);
    }
    for (long long q = n_vec * kPer + (long long)blockIdx.x * 256 + threadIdx.x; q < n; q += stride) {  // < kPer values
        const long long bit0 = q * bits;
        const long long w = bit0 >> 5;
        const int sh = (int)(bit0 & 31);
        unsigned long long window = (unsigned long long)__ldg(packed + w);
        if (sh + bits > 32) window |= (unsigned long long)__ldg(packed + w + 1) << 32;
        dst[q] = (DstT)((unsigned int)(window >> sh) & mask);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Re-binned view of the MPD (the tools bin mpd.dat "into a histogram before they are returned ... By
// default, the number of bins is set to 100, with a maximum limit of 400").  Reading S20: n_out bins of
// equal width in log10(mu) on [mu_min, mu_max), mu = count/N_avg; out[k] = (pixels whose mu falls in bin k)/n_pixels;
// count 0 (mu = 0) and magnifications outside the range are left out.
//
// Integer-exact and deterministic: the bin of a count value is monotone in the count, so the host turns the n_out + 1
// bin boundaries into the smallest COUNT of each bin (RebinEdges, found by bisection on the FP64 expression of reading
// S20 — mlens.cu) and the device only compares integers, adds 64-bit pixel counts (order-independent) and divides each
// bin once.  The out array is used as 64-bit integer storage until mpd_rebin_finish_kernel converts it in place.
// ---------------------------------------------------------------------------------------------------------------
constexpr int kRebinMaxOut = 400;
struct RebinEdges {
    int lo[kRebinMaxOut + 1];  // lo[k] = smallest count whose bin index is >= k, k = 0..n_out (n_bins if there is none)
};

__global__ void __launch_bounds__(256) mpd_rebin_kernel(const unsigned long long* __restrict__ hist, int n_bins, int n_out,
                                                        const RebinEdges edges, unsigned long long* __restrict__ out_pixels) {
    __shared__ unsigned long long acc[kRebinMaxOut];
    __shared__ int lo[kRebinMaxOut + 1];
    for (int k = threadIdx.x; k <= n_out; k += 256) lo[k] = edges.lo[k];
    for (int k = threadIdx.x; k < n_out; k += 256) acc[k] = 0ull;
    __syncthreads();
    const int first = lo[0], last = lo[n_out];  // counts in [first, last) have a bin
    for (long long c = (long long)first + (long long)blockIdx.x * 256 + threadIdx.x; c < n_bins && c < last; c += (long long)gridDim.x * 256) {
        const unsigned long long pixels = hist[c];
        if (pixels == 0ull) continue;
        int a = 0, b = n_out;  // largest k with lo[k] <= c
        while (b - a > 1) {
            const int mid = (a + b) >> 1;
            if (lo[mid] <= (int)c) a = mid; else b = mid;
        }
        atomicAdd(&acc[a], pixels);
    }
    __syncthreads();
    for (int k = threadIdx.x; k < n_out; k += 256)
        if (acc[k]) atomicAdd(&out_pixels[k], acc[k]);
}

__global__ void __launch_bounds__(512) mpd_rebin_finish_kernel(double* __restrict__ out, int n_out, double n_pixels) {
    const int k = threadIdx.x;
    if (k < n_out) {
        const unsigned long long pixels = reinterpret_cast<const unsigned long long*>(out)[k];
        out[k] = (double)pixels / n_pixels;
    }
}

}  // namespace mlk
