// mlens.cu — host side of libmlens.so: the C ABI declared in include/mlens.h.
// Argument checking, the derived lattice (DESIGN.md "Readings" S2), the device copy of the lens list, kernel launches.
// No torch types, no CPU fallback: every step of the hot path runs in the kernels of shoot_kernel.cuh.
#include "../../include/mlens.h"

#include <cuda_runtime.h>
#include <cufft.h>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdint>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "convolve_kernel.cuh"
#include "mapstats_kernel.cuh"
#include "shoot_kernel.cuh"
#ifdef MLENS_ABLATIONS
#include "shoot_ablation_kernels.cuh"
#endif

namespace {

thread_local char g_err[512] = "";

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is state of the FUNCTION, not of the launch: two host threads (one
// handle each, e.g. the workers of survey.py) that set it to different sizes and then launch would race — the launch with
// the larger request fails with "invalid argument" when the other thread's smaller value is the current one.  Every
// set-attribute + launch pair of a kernel with dynamic shared memory runs under this mutex (microseconds of host time).
std::mutex g_launch_mutex;

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define MLENS_CUDA(call)                                                                              \
    do {                                                                                              \
        cudaError_t e_ = (call);                                                                      \
        if (e_ != cudaSuccess)                                                                        \
            return fail(e_ == cudaErrorMemoryAllocation ? MLENS_ENOMEM : MLENS_ECUDA, "%s: %s", #call, \
                        cudaGetErrorString(e_));                                                      \
    } while (0)

// Device memory of the handles comes from ONE library-owned stream-ordered pool per device that keeps freed blocks
// (release threshold = max): mlens_create / mlens_shoot_host / mlens_destroy of map after map then recycle the same
// blocks.  Measured on the B200 box: cudaFree of the 64 MB result buffers took 20 ... 1500 ms on one call in three, i.e.
// up to 1.6x the whole 0.88 s map of config 3 (profiles/r2_summary.md, "e2e"); cudaFreeAsync into the pool returns at once.
// mlens_trim_memory() hands the cached blocks back to the driver.
struct DevPool {
    cudaMemPool_t pool = nullptr;
    cudaStream_t stream = nullptr;
    int state = 0;  // 0 = not tried, 1 = pool in use, -1 = unavailable: plain cudaMalloc / cudaFree
};
std::mutex g_pool_mutex;
DevPool g_pools[64];

DevPool* device_pool() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
    DevPool* dp = &g_pools[dev];
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    if (dp->state == 0) {
        cudaMemPoolProps props;
        memset(&props, 0, sizeof(props));
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        unsigned long long keep = ~0ull;
        if (cudaMemPoolCreate(&dp->pool, &props) == cudaSuccess &&
            cudaMemPoolSetAttribute(dp->pool, cudaMemPoolAttrReleaseThreshold, &keep) == cudaSuccess &&
            cudaStreamCreateWithFlags(&dp->stream, cudaStreamNonBlocking) == cudaSuccess) {
            dp->state = 1;
        } else {
            (void)cudaGetLastError();
            dp->state = -1;
        }
    }
    return dp->state == 1 ? dp : nullptr;
}

template <typename T>
cudaError_t dev_alloc(T** p, size_t bytes) {
    if (DevPool* dp = device_pool()) {
        cudaError_t e = cudaMallocFromPoolAsync(reinterpret_cast<void**>(p), bytes, dp->pool, dp->stream);
        if (e == cudaErrorMemoryAllocation) {
            // the pool keeps the blocks of destroyed handles (of other map sizes, too): give them back and try once more
            (void)cudaGetLastError();
            cudaStreamSynchronize(dp->stream);
            cudaMemPoolTrimTo(dp->pool, 0);
            e = cudaMallocFromPoolAsync(reinterpret_cast<void**>(p), bytes, dp->pool, dp->stream);
        }
        if (e == cudaSuccess) e = cudaStreamSynchronize(dp->stream);  // usable from any stream from here on
        return e;
    }
    return cudaMalloc(reinterpret_cast<void**>(p), bytes);
}

// The caller has made sure that no work still uses the block (mlens_destroy synchronises the device first).
void dev_free(void* p) {
    if (!p) return;
    if (DevPool* dp = device_pool()) cudaFreeAsync(p, dp->stream);
    else cudaFree(p);
}

// The handles' small pinned host mirrors (64-byte blocks) are recycled the same way: cudaMallocHost costs 2-10 ms.
constexpr size_t kPinnedBlock = 64;
std::vector<void*> g_pinned_free;

cudaError_t pinned_alloc(void** p) {
    {
        std::lock_guard<std::mutex> lock(g_pool_mutex);
        if (!g_pinned_free.empty()) { *p = g_pinned_free.back(); g_pinned_free.pop_back(); return cudaSuccess; }
    }
    return cudaMallocHost(p, kPinnedBlock);
}

void pinned_free(void* p) {
    if (!p) return;
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    try { g_pinned_free.push_back(p); } catch (...) { cudaFreeHost(p); }
}

constexpr int kChunkMax = 2048;        // lenses per chunk when the list is streamed in several chunks
constexpr int kChunkSingleMax = 3072;  // largest list kept resident as one chunk
// The production instantiation of shoot_fp32_kernel (chosen by the sweep in profiles/): tile width,
// ray pairs per lens that share a reciprocal, resident CTAs per SM.
#ifndef MLENS_PROD_TILE_X
#define MLENS_PROD_TILE_X 64
#endif
#ifndef MLENS_PROD_RAYS
#define MLENS_PROD_RAYS 16
#endif
#ifndef MLENS_PROD_SHARED_PAIRS
#define MLENS_PROD_SHARED_PAIRS 2
#endif
constexpr int kProdTileX = MLENS_PROD_TILE_X, kProdRays = MLENS_PROD_RAYS, kProdSharedPairs = MLENS_PROD_SHARED_PAIRS;
constexpr int kProdCtas = 2;
constexpr int kTileCtrSlots = 256;     // ring of dynamic tile counters: one per launch in flight (see launch_block)
static_assert(kTileCtrSlots == 256, "mlens::slot_done holds one event per ring slot");

}  // namespace

static_assert(sizeof(mlk::MapStatsDev) <= kPinnedBlock && 8 * sizeof(unsigned long long) <= kPinnedBlock, "pinned mirror block");

struct mlens {
    // parameters
    double kappa, gamma, s, L, d;
    int npix;
    long long n_lens;
    mlens_geometry geo;
    // device state
    int device;
    int sm_count;
    float4* lens_dev;                  // (x, y, m, 0)
    unsigned long long* counters_dev;  // in_map, outside, lost, total
    unsigned long long* tile_ctr_dev;  // ring of kTileCtrSlots dynamic tile counters; launch number n uses slot n % kTileCtrSlots
    unsigned long long launch_seq;
    cudaEvent_t slot_done[256];        // per ring slot: recorded after the launch that used it (created on first use)
    int* max_count_dev;
    mlk::MapStatsDev* mapstats_dev;    // scratch of mlens_mpd (lazily allocated)
    mlk::MapStatsDev* mapstats_host;   // pinned mirror
    // convolution (lazily created): cuFFT plans, spectra of the map and of the kernel, profile normalisation scratch
    cufftHandle plan_r2c, plan_c2r;
    int have_plans;
    float2 *spec_map, *spec_ker, *spec_prep;  // spectra of the map, of the kernel given to mlens_convolve, of the prepared kernel
    int have_prep;
    double* prof_sum;
    unsigned long long* idx_hist;      // scratch of mlens_index_map: histogram, LUT, distinct counter
    int* idx_lut;
    long long idx_bins_cap;
    int* idx_n_dev;
    unsigned int* mpd_partial;         // sm_count x kMpdSmemBinsMax per-CTA histogram slices (lazily allocated)
    unsigned long long* counters_host;  // pinned mirror (4 counters + max_count)
    // host-buffer path
    int* count_own;
    float* mag_own;
    cudaStream_t own_stream;
    cudaEvent_t ev0, ev1, evk0, evk1;
    float last_ms, last_kernel_ms;
    // options
    int opt_kernel, opt_binning, opt_ctas_per_sm, opt_shared, opt_rays, opt_tile_x, opt_shared_pairs;
    double lens_extent;                // max |coordinate| over the lens list (guards the shared-reciprocal products)
    double mass_max;                   // largest lens mass (guards the FP32 range of the lattice-unit loop)
};

namespace {

// NULL handle, or a handle whose device is not the calling thread's current device (its buffers, plans and the
// caller's DEVICE pointers all belong to h->device: launching from another device would fault or silently misbehave)
int check_handle(const mlens_t* h) {
    if (!h) return fail(MLENS_EINVAL, "NULL handle");
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return fail(MLENS_ECUDA, "cudaGetDevice failed");
    if (dev != h->device)
        return fail(MLENS_EINVAL, "current CUDA device is %d but the handle was created on device %d", dev, h->device);
    return MLENS_OK;
}

int launch_block(mlens_t* h, long long i0, long long j0, long long ni, long long nj, int* count, double* ray_y,
                 int* ray_pix, cudaStream_t st) {
    if (ni == 0 || nj == 0) return MLENS_OK;
    mlk::ShootParams P;
    memset(&P, 0, sizeof(P));
    P.i0 = i0; P.j0 = j0; P.ni = ni; P.nj = nj;
    P.half_n1 = (double)h->geo.n1 / 2.0;
    P.half_n2 = (double)h->geo.n2 / 2.0;
    P.d = h->d;
    // tile width: the production kernel's is an option; every other kernel walks 64 x 64 tiles
    const int tile_x = h->opt_kernel == 1 ? h->opt_tile_x : mlk::kTile;
    P.tiles_x = (int)((ni + tile_x - 1) / tile_x);
    P.tiles_y = (int)((nj + mlk::kTile - 1) / mlk::kTile);
    P.f1 = 1.0 - h->geo.kappa_s - h->gamma;
    P.f2 = 1.0 - h->geo.kappa_s + h->gamma;
    P.half_L = h->L / 2.0;
    P.p = h->geo.p;
    P.inv_p = 1.0 / h->geo.p;
    P.npix = h->npix;
    P.lens_raw = h->lens_dev;
    P.n_lens = (int)h->n_lens;
    P.rho2 = 0.25;  // rho = 0.5 sqrt(max(m,1))
    {
        const double hd = 0.5 * h->d * std::sqrt((double)tile_x * tile_x + (double)mlk::kTile * mlk::kTile);  // tile half-diagonal
        P.rho2_tile = 4.0 * hd * hd;
    }
    P.count = count; P.ray_y = ray_y; P.ray_pix = ray_pix;
    P.counters = h->counters_dev;
    // Every launch gets its OWN dynamic tile counter, zeroed on the launch's stream: launches of one handle issued to
    // different streams may then overlap without stealing or re-zeroing each other's tiles (the ray counters are
    // plain atomic sums and do not care).  A slot is reused after kTileCtrSlots further launches.
    // The launch that used the slot kTileCtrSlots launches ago may still run on ANOTHER stream: this launch's stream first
    // waits for the event that launch recorded, so a live counter is never re-zeroed (no duplicated tiles).
    const int slot = (int)(h->launch_seq++ % kTileCtrSlots);
    P.tile_counter = h->tile_ctr_dev + slot;
    if (h->slot_done[slot]) MLENS_CUDA(cudaStreamWaitEvent(st, h->slot_done[slot], 0));
    MLENS_CUDA(cudaMemsetAsync(P.tile_counter, 0, sizeof(unsigned long long), st));
    struct SlotRelease {  // every return path below records "this slot's launch is done" on the launch's stream
        mlens_t* h; int slot; cudaStream_t st;
        ~SlotRelease() {
            if (!h->slot_done[slot] && cudaEventCreateWithFlags(&h->slot_done[slot], cudaEventDisableTiming) != cudaSuccess) {
                h->slot_done[slot] = nullptr;
                (void)cudaGetLastError();
                return;
            }
            cudaEventRecord(h->slot_done[slot], st);
        }
    } slot_release{h, slot, st};
    P.bin_mode = h->opt_binning;

#ifdef MLENS_ABLATIONS
    if (h->opt_kernel == 0) {
        const long long n_rays = ni * nj;
        long long blocks = (n_rays + 255) / 256;
        const long long cap = (long long)h->sm_count * 16;
        if (blocks > cap) blocks = cap;
        mlk::shoot_fp64_kernel<<<(unsigned)blocks, 256, 0, st>>>(P);
        MLENS_CUDA(cudaGetLastError());
        return MLENS_OK;
    }

    if (h->opt_kernel == 2) {  // ablation: plain-form FP32 (whole list resident in shared memory)
        if (P.n_lens > 12000) return fail(MLENS_EINVAL, "kernel 2 (plain FP32 ablation) holds at most 12000 lenses");
        const size_t smem = (size_t)(((P.n_lens + 3) & ~3) + 4) * 16;
        const long long n_tiles = (long long)P.tiles_x * P.tiles_y;
        long long grid = (long long)h->sm_count * (smem > 100 * 1024 ? 1 : 2);
        if (grid > n_tiles) grid = n_tiles;
        MLENS_CUDA(cudaFuncSetAttribute(mlk::shoot_plain_fp32_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        mlk::shoot_plain_fp32_kernel<<<(unsigned)grid, 512, smem, st>>>(P);
        MLENS_CUDA(cudaGetLastError());
        return MLENS_OK;
    }

#endif  // MLENS_ABLATIONS

    int chunk, n_chunks;
    if (P.n_lens <= kChunkSingleMax) {
        chunk = (P.n_lens + 3) & ~3;
        if (chunk < 4) chunk = 4;
        n_chunks = 1;
    } else {
        chunk = kChunkMax;
        n_chunks = (P.n_lens + chunk - 1) / chunk;
    }
    P.chunk = chunk; P.n_chunks = n_chunks;
    const size_t smem = sizeof(mlk::TileShared) + (size_t)chunk * 16 * (n_chunks > 1 ? 3 : 2);
    const long long n_tiles = (long long)P.tiles_x * P.tiles_y;
    void (*kern)(const mlk::ShootParams) = nullptr;
    int threads = 0, ctas = 0;

#ifdef MLENS_ABLATIONS
    if (h->opt_kernel == 4) {  // the round-1 production kernel (A/B baseline) and its shared-reciprocal variants
        switch (h->opt_shared) {
            case 0: kern = mlk::shoot_fp32_r1_kernel<8, 0, -1>; break;
            case 1: kern = mlk::shoot_fp32_r1_kernel<8, 1, -1>; break;
            case 2: kern = mlk::shoot_fp32_r1_kernel<8, 2, -1>; break;
            default: return fail(MLENS_EINVAL, "kernel 4 has shared_rcp 0..2");
        }
        threads = 512; ctas = 2;
    }
#endif
    if (!kern) {
        // Shared reciprocals multiply two squared distances in lattice units: keep the product inside FP32 (the lattice
        // has < 2^31 rays per axis, but the caller's lenses may lie anywhere).  Beyond that, one MUFU.RCP per ray.
        int shared = h->opt_shared_pairs;
        const double zmax = (h->lens_extent + std::fmax(h->geo.a1, h->geo.a2)) / h->d;  // per axis, lattice units
        if (shared > 0 && 4.0 * zmax * zmax * zmax * zmax > 1.0e37) shared = 0;
        // the loop itself forms |w|^2 <= 2 zmax^2 and c conj(w) ~ m / d^2 in FP32
        if (P.n_lens > 0 && (2.0 * zmax * zmax > 1.0e37 || h->mass_max / (h->d * h->d) > 1.0e37))
            return fail(MLENS_ERANGE, "ray_spacing %g is too small for the FP32 lattice-unit loop (lens distances / spacing up to %g)", h->d, zmax);
        const int code = h->opt_rays * 10000 + h->opt_tile_x * 10 + shared;
        // the default launch (run-combining REDs into a count map, no per-ray outputs) has its own, leaner instantiation
        const bool runs = h->opt_binning == mlk::BIN_RUNS && count != nullptr && ray_y == nullptr && ray_pix == nullptr;
        switch (code) {
#define MLENS_VARIANT(TX, R, SP, NC)                                                                                       \
    case R * 10000 + TX * 10 + SP:                                                                                          \
        kern = runs ? mlk::shoot_fp32_kernel<TX, R, SP, NC, mlk::BIN_RUNS> : mlk::shoot_fp32_kernel<TX, R, SP, NC, -1>;     \
        threads = TX / R * mlk::kTile; ctas = NC;                                                                           \
        break;
#ifdef MLENS_ABLATIONS  // the sweep grid: rays per thread x tile width x shared pairs (profiles/)
#define MLENS_SWEEP(SP) MLENS_VARIANT(64, 8, SP, 2) MLENS_VARIANT(48, 8, SP, 2) MLENS_VARIANT(32, 8, SP, 3) MLENS_VARIANT(64, 16, SP, 2)
            MLENS_SWEEP(0) MLENS_SWEEP(1) MLENS_SWEEP(2)
            MLENS_VARIANT(64, 8, 3, 2) MLENS_VARIANT(64, 8, 4, 2) MLENS_VARIANT(64, 16, 3, 2) MLENS_VARIANT(64, 16, 4, 2)
#undef MLENS_SWEEP
#else                   // the shipped library: the production instantiation and its one-reciprocal-per-ray fallback
            MLENS_VARIANT(kProdTileX, kProdRays, 0, kProdCtas)
#if MLENS_PROD_SHARED_PAIRS != 0
            MLENS_VARIANT(kProdTileX, kProdRays, kProdSharedPairs, kProdCtas)
#endif
#endif
#undef MLENS_VARIANT
            default: return fail(MLENS_EINVAL, "no kernel variant rays_per_thread=%d tile_x=%d shared_pairs=%d in this build", h->opt_rays, h->opt_tile_x, shared);
        }
    }
    if (h->opt_ctas_per_sm > 0) ctas = h->opt_ctas_per_sm;
    long long grid = (long long)h->sm_count * ctas;
    if (grid > n_tiles) grid = n_tiles;
    std::lock_guard<std::mutex> launch_lock(g_launch_mutex);
    MLENS_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    MLENS_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
    kern<<<(unsigned)grid, threads, smem, st>>>(P);
    MLENS_CUDA(cudaGetLastError());
    return MLENS_OK;
}

int launch_magnification(mlens_t* h, const int* count, float* mag, cudaStream_t st) {
    const long long n = (long long)h->npix * h->npix;
    MLENS_CUDA(cudaMemsetAsync(h->max_count_dev, 0, sizeof(int), st));
    long long blocks = (n / 4 + 255) / 256;
    const long long cap = (long long)h->sm_count * 8;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    mlk::magnification_kernel<<<(unsigned)blocks, 256, 0, st>>>(count, mag, n, h->geo.n_avg, h->max_count_dev);
    MLENS_CUDA(cudaGetLastError());
    return MLENS_OK;
}

int read_stats(mlens_t* h, cudaStream_t st, mlens_stats* out) {
    MLENS_CUDA(cudaMemcpyAsync(h->counters_host, h->counters_dev, 4 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    MLENS_CUDA(cudaMemcpyAsync(h->counters_host + 4, h->max_count_dev, sizeof(int), cudaMemcpyDeviceToHost, st));
    MLENS_CUDA(cudaStreamSynchronize(st));
    out->rays_in_map = (long long)h->counters_host[0];
    out->rays_outside = (long long)h->counters_host[1];
    out->rays_lost = (long long)h->counters_host[2];
    out->rays_total = (long long)h->counters_host[3];
    out->n_lens = h->n_lens;
    int mc;
    memcpy(&mc, h->counters_host + 4, sizeof(int));
    out->max_count = mc;
    out->elapsed_ms = h->last_ms;
    out->kernel_ms = h->last_kernel_ms;
    return MLENS_OK;
}

}  // namespace

extern "C" {

const char* mlens_last_error(void) { return g_err; }

int mlens_create(mlens_t** out, double kappa, double gamma, double s, double map_side, int npix, double ray_spacing,
                 const float* lens_xy, const float* lens_m, long long n_lens) {
    if (!out) return fail(MLENS_EINVAL, "out is NULL");
    *out = nullptr;
    if (!std::isfinite(kappa) || !std::isfinite(gamma) || !std::isfinite(s) || !std::isfinite(map_side) ||
        !std::isfinite(ray_spacing))
        return fail(MLENS_EINVAL, "non-finite parameter");
    if (kappa < 0) return fail(MLENS_EINVAL, "kappa < 0");
    if (s < 0 || s > 1) return fail(MLENS_EINVAL, "s outside [0,1]");
    if (!(map_side > 0) || npix <= 0 || !(ray_spacing > 0)) return fail(MLENS_EINVAL, "map_side, npix, ray_spacing must be > 0");
    if (n_lens < 0) return fail(MLENS_EINVAL, "n_lens < 0");
    if (n_lens > 0 && !lens_xy) return fail(MLENS_EINVAL, "lens_xy is NULL");
    if (n_lens > (1ll << 30)) return fail(MLENS_ERANGE, "n_lens too large");
    const double f1 = std::fabs(1.0 - kappa - gamma), f2 = std::fabs(1.0 - kappa + gamma);
    if (f1 < 1e-6 || f2 < 1e-6) return fail(MLENS_EINVAL, "macro-model on the critical line: |1-kappa-+gamma| < 1e-6");
    if ((long long)npix * npix >= (1ll << 31)) return fail(MLENS_ERANGE, "npix^2 >= 2^31");

    mlens_geometry g;
    g.kappa_s = s * kappa;
    g.kappa_star = kappa - g.kappa_s;
    g.p = map_side / npix;
    g.d = ray_spacing;
    g.a1 = 1.2 * (map_side / 2.0) / f1;
    g.a2 = 1.2 * (map_side / 2.0) / f2;
    const double c1 = std::ceil(g.a1 / ray_spacing - 1e-9), c2 = std::ceil(g.a2 / ray_spacing - 1e-9);
    if (!(c1 < 1073741824.0) || !(c2 < 1073741824.0)) return fail(MLENS_ERANGE, "lattice has >= 2^31 rays along an axis");
    g.n1 = 2 * (long long)c1;
    g.n2 = 2 * (long long)c2;
    g.n_avg = (g.p / ray_spacing) * (g.p / ray_spacing);

    std::vector<float4> packed;
    try {
        packed.resize((size_t)n_lens);
    } catch (...) {  // nothing may throw across the C ABI
        return fail(MLENS_ENOMEM, "host allocation of %lld lenses failed", n_lens);
    }
    for (long long k = 0; k < n_lens; ++k) {
        const float x = lens_xy[2 * k], y = lens_xy[2 * k + 1], m = lens_m ? lens_m[k] : 1.0f;
        if (!std::isfinite(x) || !std::isfinite(y)) return fail(MLENS_EINVAL, "lens %lld has a non-finite coordinate", k);
        if (!std::isfinite(m) || !(m > 0)) return fail(MLENS_EINVAL, "lens %lld has a mass that is not finite and > 0", k);
        packed[(size_t)k] = make_float4(x, y, m, 0.f);
    }

    int dev = 0;
    MLENS_CUDA(cudaGetDevice(&dev));
    // three attributes, not cudaGetDeviceProperties: that call alone costs milliseconds, more than config 1's whole map
    int cc_major = 0, cc_minor = 0, sm_count = 0;
    MLENS_CUDA(cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, dev));
    MLENS_CUDA(cudaDeviceGetAttribute(&cc_minor, cudaDevAttrComputeCapabilityMinor, dev));
    MLENS_CUDA(cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev));
    if (cc_major != 10) return fail(MLENS_ECUDA, "device %d is sm_%d%d; this library is built for sm_100a only", dev, cc_major, cc_minor);

    mlens* h = new (std::nothrow) mlens();
    if (!h) return fail(MLENS_ENOMEM, "host allocation failed");
    memset(h, 0, sizeof(*h));
    h->kappa = kappa; h->gamma = gamma; h->s = s; h->L = map_side; h->d = ray_spacing;
    h->npix = npix; h->n_lens = n_lens; h->geo = g;
    h->device = dev; h->sm_count = sm_count;
    h->opt_kernel = 1; h->opt_binning = mlk::BIN_RUNS; h->opt_ctas_per_sm = 0; h->opt_shared = 0; h->opt_rays = kProdRays;
    h->opt_tile_x = kProdTileX; h->opt_shared_pairs = kProdSharedPairs;
    for (long long k = 0; k < n_lens; ++k) {
        h->lens_extent = std::fmax(h->lens_extent, std::fmax(std::fabs((double)packed[(size_t)k].x), std::fabs((double)packed[(size_t)k].y)));
        h->mass_max = std::fmax(h->mass_max, (double)packed[(size_t)k].z);
    }

    cudaError_t e = cudaSuccess;
    if (e == cudaSuccess) e = dev_alloc(&h->lens_dev, sizeof(float4) * (size_t)(n_lens > 0 ? n_lens : 1));
    // The blocks are recycled ones (they hold a previous handle's lens list and counters) and the shooting streams are
    // not ordered with the legacy default stream: initialise them on the pool's own stream and wait for it, so that the
    // handle is complete before any stream can use it.
    DevPool* dp = device_pool();
    cudaStream_t init_st = dp ? dp->stream : (cudaStream_t)0;
    if (e == cudaSuccess && n_lens > 0)
        e = cudaMemcpyAsync(h->lens_dev, packed.data(), sizeof(float4) * (size_t)n_lens, cudaMemcpyHostToDevice, init_st);
    // one block for the small device state: 8 ray counters, the ring of tile counters, max_count
    if (e == cudaSuccess) e = dev_alloc(&h->counters_dev, (8 + kTileCtrSlots + 1) * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMemsetAsync(h->counters_dev, 0, (8 + kTileCtrSlots + 1) * sizeof(unsigned long long), init_st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(init_st);
    if (e == cudaSuccess) {
        h->tile_ctr_dev = h->counters_dev + 8;
        h->max_count_dev = reinterpret_cast<int*>(h->counters_dev + 8 + kTileCtrSlots);
    }
    if (e == cudaSuccess) e = pinned_alloc(reinterpret_cast<void**>(&h->counters_host));
    if (e == cudaSuccess) e = cudaEventCreate(&h->ev0);
    if (e == cudaSuccess) e = cudaEventCreate(&h->ev1);
    if (e == cudaSuccess) e = cudaEventCreate(&h->evk0);
    if (e == cudaSuccess) e = cudaEventCreate(&h->evk1);
    if (e != cudaSuccess) {
        const int code = fail(e == cudaErrorMemoryAllocation ? MLENS_ENOMEM : MLENS_ECUDA, "mlens_create: %s", cudaGetErrorString(e));
        mlens_destroy(h);
        return code;
    }
    *out = h;
    return MLENS_OK;
}

namespace {
// device_wide: wait for every stream of the device (the handle may have been used on any of them); otherwise only for `st`
void destroy_impl(mlens_t* h, bool device_wide, cudaStream_t st);
}

void mlens_destroy(mlens_t* h) { destroy_impl(h, true, nullptr); }

void mlens_destroy_on_stream(mlens_t* h, void* cuda_stream) { destroy_impl(h, false, (cudaStream_t)cuda_stream); }

namespace {
void destroy_impl(mlens_t* h, bool device_wide, cudaStream_t st) {
    if (!h) return;
    // the handle's blocks go back to ITS device's pool: make that device current for the duration, and let every kernel
    // that may still use them finish first (what cudaFree used to do implicitly)
    int cur = -1;
    cudaGetDevice(&cur);
    if (cur != h->device) cudaSetDevice(h->device);
    if (device_wide) cudaDeviceSynchronize();
    else cudaStreamSynchronize(st);
    dev_free(h->lens_dev);
    dev_free(h->counters_dev);  // also holds the tile counters and max_count
    dev_free(h->mapstats_dev);
    pinned_free(h->mapstats_host);
    dev_free(h->mpd_partial);
    dev_free(h->idx_hist);
    dev_free(h->idx_lut);
    dev_free(h->idx_n_dev);
    if (h->have_plans) { cufftDestroy(h->plan_r2c); cufftDestroy(h->plan_c2r); }
    dev_free(h->spec_map);
    dev_free(h->spec_ker);
    dev_free(h->spec_prep);
    dev_free(h->prof_sum);
    pinned_free(h->counters_host);
    dev_free(h->count_own);
    dev_free(h->mag_own);
    if (h->own_stream) cudaStreamDestroy(h->own_stream);
    for (cudaEvent_t ev : h->slot_done)
        if (ev) cudaEventDestroy(ev);
    if (h->ev0) cudaEventDestroy(h->ev0);
    if (h->ev1) cudaEventDestroy(h->ev1);
    if (h->evk0) cudaEventDestroy(h->evk0);
    if (h->evk1) cudaEventDestroy(h->evk1);
    if (cur >= 0 && cur != h->device) cudaSetDevice(cur);
    delete h;
}
}  // namespace

int mlens_trim_memory(void) {
    if (DevPool* dp = device_pool()) {
        MLENS_CUDA(cudaStreamSynchronize(dp->stream));
        MLENS_CUDA(cudaMemPoolTrimTo(dp->pool, 0));
    }
    std::vector<void*> pinned;
    {
        std::lock_guard<std::mutex> lock(g_pool_mutex);
        pinned.swap(g_pinned_free);
    }
    for (void* p : pinned) cudaFreeHost(p);
    return MLENS_OK;
}

int mlens_get_geometry(const mlens_t* h, mlens_geometry* g) {
    if (!h || !g) return fail(MLENS_EINVAL, "NULL argument");
    *g = h->geo;
    return MLENS_OK;
}

int mlens_set_option(mlens_t* h, const char* key, long long value) {
    if (!h || !key) return fail(MLENS_EINVAL, "NULL argument");
#ifndef MLENS_ABLATIONS
    // the shipped library holds the production kernel only: the debug / ablation / experimental kernels and loop variants
    // exist in the MLENS_ABLATIONS build (libmlens_ablations.so, used by the tests and the profiling runs)
    if ((!strcmp(key, "kernel") && value != 1) || (!strcmp(key, "shared_rcp") && value != 0) ||
        (!strcmp(key, "tile_x") && value != kProdTileX) || (!strcmp(key, "rays_per_thread") && value != kProdRays) ||
        (!strcmp(key, "shared_pairs") && value != 0 && value != kProdSharedPairs))
        return fail(MLENS_EINVAL, "option %s=%lld needs the MLENS_ABLATIONS build of the library", key, value);
#endif
    if (!strcmp(key, "kernel")) {
        if (value != 0 && value != 1 && value != 2 && value != 4) return fail(MLENS_EINVAL, "kernel must be 0, 1, 2 or 4");
        h->opt_kernel = (int)value;
    } else if (!strcmp(key, "tile_x")) {
        if (value != 64 && value != 48 && value != 32) return fail(MLENS_EINVAL, "tile_x must be 64, 48 or 32");
        h->opt_tile_x = (int)value;
    } else if (!strcmp(key, "rays_per_thread")) {
        if (value != 8 && value != 16) return fail(MLENS_EINVAL, "rays_per_thread must be 8 or 16");
        h->opt_rays = (int)value;
    } else if (!strcmp(key, "shared_pairs")) {
        if (value < 0 || value > 4) return fail(MLENS_EINVAL, "shared_pairs must be 0..4");
        h->opt_shared_pairs = (int)value;
    } else if (!strcmp(key, "binning")) {
        if (value < 0 || value > 3) return fail(MLENS_EINVAL, "binning must be 0..3");
        h->opt_binning = (int)value;
    } else if (!strcmp(key, "ctas_per_sm")) {
        if (value < 0 || value > 8) return fail(MLENS_EINVAL, "ctas_per_sm must be 0 (the kernel's own) or 1..8");
        h->opt_ctas_per_sm = (int)value;
    } else if (!strcmp(key, "shared_rcp")) {
        if (value < 0 || value > 2) return fail(MLENS_EINVAL, "shared_rcp must be 0..2");
        h->opt_shared = (int)value;
    } else {
        return fail(MLENS_EINVAL, "unknown option '%s'", key);
    }
    return MLENS_OK;
}

int mlens_reset_stats(mlens_t* h, void* cuda_stream) {
    if (int rc = check_handle(h)) return rc;
    MLENS_CUDA(cudaMemsetAsync(h->counters_dev, 0, 4 * sizeof(unsigned long long), (cudaStream_t)cuda_stream));
    return MLENS_OK;
}

int mlens_get_stats(mlens_t* h, void* cuda_stream, mlens_stats* stats) {
    if (!h || !stats) return fail(MLENS_EINVAL, "NULL argument");
    if (int rc = check_handle(h)) return rc;
    return read_stats(h, (cudaStream_t)cuda_stream, stats);
}

int mlens_shoot_block(mlens_t* h, long long i0, long long j0, long long ni, long long nj, int* count_dev,
                      double* ray_y_dev, int* ray_pix_dev, void* cuda_stream) {
    if (int rc = check_handle(h)) return rc;
    if (i0 < 0 || j0 < 0 || ni < 0 || nj < 0 || i0 + ni > h->geo.n1 || j0 + nj > h->geo.n2)
        return fail(MLENS_EINVAL, "block [%lld,+%lld) x [%lld,+%lld) is outside the %lld x %lld lattice", i0, ni, j0, nj,
                    h->geo.n1, h->geo.n2);
    return launch_block(h, i0, j0, ni, nj, count_dev, ray_y_dev, ray_pix_dev, (cudaStream_t)cuda_stream);
}

int mlens_magnification(mlens_t* h, const int* count_dev, float* mag_dev, void* cuda_stream) {
    if (!h || !count_dev) return fail(MLENS_EINVAL, "NULL argument");
    if (int rc = check_handle(h)) return rc;
    return launch_magnification(h, count_dev, mag_dev, (cudaStream_t)cuda_stream);
}

int mlens_mpd(mlens_t* h, const int* count_dev, unsigned long long* hist_dev, int n_bins, void* cuda_stream,
              mlens_map_stats* stats) {
    if (!h || !count_dev || !hist_dev) return fail(MLENS_EINVAL, "NULL argument");
    if (int rc = check_handle(h)) return rc;
    if (n_bins < 2) return fail(MLENS_EINVAL, "n_bins must be >= 2");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (!h->mapstats_dev) MLENS_CUDA(dev_alloc(&h->mapstats_dev, sizeof(mlk::MapStatsDev)));
    if (!h->mapstats_host) MLENS_CUDA(pinned_alloc(reinterpret_cast<void**>(&h->mapstats_host)));
    const long long n = (long long)h->npix * h->npix;
    MLENS_CUDA(cudaMemsetAsync(h->mapstats_dev, 0, sizeof(mlk::MapStatsDev), st));
    MLENS_CUDA(cudaMemsetAsync(hist_dev, 0, sizeof(unsigned long long) * (size_t)n_bins, st));
    if (!h->mpd_partial)
        MLENS_CUDA(dev_alloc(&h->mpd_partial, sizeof(unsigned int) * (size_t)h->sm_count * mlk::kMpdSmemBinsMax));
    // shared-memory bins: all of them when they fit (multiple of 1024 for the fill/flush loops), else the first 48 Ki
    int smem_bins = (n_bins + 1023) & ~1023;
    if (smem_bins > mlk::kMpdSmemBinsMax) smem_bins = mlk::kMpdSmemBinsMax;
    long long blocks = (n / 4 + mlk::kMpdThreads - 1) / mlk::kMpdThreads;
    if (blocks > h->sm_count) blocks = h->sm_count;  // one persistent 1024-thread CTA per SM
    if (blocks < 1) blocks = 1;
    const size_t smem = sizeof(unsigned int) * (size_t)smem_bins;
    {
        std::lock_guard<std::mutex> launch_lock(g_launch_mutex);
        MLENS_CUDA(cudaFuncSetAttribute(mlk::mpd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        mlk::mpd_kernel<<<(unsigned)blocks, mlk::kMpdThreads, smem, st>>>(count_dev, n, hist_dev, n_bins, smem_bins,
                                                                           h->mpd_partial, h->mapstats_dev);
        MLENS_CUDA(cudaGetLastError());
    }
    mlk::mpd_reduce_kernel<<<(smem_bins + 31) / 32, 256, 0, st>>>(h->mpd_partial, (int)blocks, smem_bins, hist_dev, n_bins, h->mapstats_dev);
    MLENS_CUDA(cudaGetLastError());
    if (stats) {
        MLENS_CUDA(cudaMemcpyAsync(h->mapstats_host, h->mapstats_dev, sizeof(mlk::MapStatsDev), cudaMemcpyDeviceToHost, st));
        MLENS_CUDA(cudaStreamSynchronize(st));
        stats->n_pixels = n;
        stats->sum_count = (long long)h->mapstats_host->sum_count;
        stats->n_clamped = (long long)h->mapstats_host->n_clamped;
        stats->min_count = 0x7fffffff - h->mapstats_host->inv_min_count;
        stats->max_count = h->mapstats_host->max_count;
        stats->mean_count = (double)stats->sum_count / (double)n;
        stats->mean_mu = stats->mean_count / h->geo.n_avg;
    }
    return MLENS_OK;
}

int mlens_index_map(mlens_t* h, const int* count_dev, int* values_dev, int max_values, unsigned short* indexed_dev,
                    void* cuda_stream, int* n_distinct) {
    if (!h || !count_dev || !values_dev || !indexed_dev || !n_distinct) return fail(MLENS_EINVAL, "NULL argument");
    if (int rc = check_handle(h)) return rc;
    if (max_values < 1) return fail(MLENS_EINVAL, "max_values must be >= 1");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long long n = (long long)h->npix * h->npix;
    // The histogram needs max(count) + 2 bins, which is not known yet.  Instead of a pass over the map to find it (and a
    // host round trip), take the capacity the handle already has (at least 16 Ki bins), and let the MPD pass itself say
    // whether it was enough: its statistics count the pixels clamped into the last bin.  Only then is the histogram
    // re-made with max_count + 2 bins (the capacity is kept, so the next map of a survey does not pay this again).
    long long n_bins = h->idx_bins_cap > 0 ? h->idx_bins_cap : 16384;
    int nd = 0;
    for (int attempt = 0;; ++attempt) {
        if (n_bins > h->idx_bins_cap) {
            dev_free(h->idx_hist);
            dev_free(h->idx_lut);
            h->idx_hist = nullptr; h->idx_lut = nullptr; h->idx_bins_cap = 0;
            MLENS_CUDA(dev_alloc(&h->idx_hist, sizeof(unsigned long long) * (size_t)n_bins));
            MLENS_CUDA(dev_alloc(&h->idx_lut, sizeof(int) * (size_t)n_bins));
            h->idx_bins_cap = n_bins;
        }
        if (!h->idx_n_dev) MLENS_CUDA(dev_alloc(&h->idx_n_dev, sizeof(int)));
        // (1) the MPD histogram: its non-empty bins are the distinct ray-count values
        if (int rc = mlens_mpd(h, count_dev, h->idx_hist, (int)n_bins, cuda_stream, nullptr)) return rc;
        // (2) compaction -> index file (values, ascending) and the count -> index table
        mlk::index_build_kernel<<<1, 1024, 0, st>>>(h->idx_hist, (int)n_bins, h->idx_lut, values_dev, max_values, h->idx_n_dev);
        MLENS_CUDA(cudaGetLastError());
        // (3) ONE host round trip: the number of distinct values and whether any count was clamped
        MLENS_CUDA(cudaMemcpyAsync(h->counters_host + 5, h->idx_n_dev, sizeof(int), cudaMemcpyDeviceToHost, st));
        MLENS_CUDA(cudaMemcpyAsync(h->mapstats_host, h->mapstats_dev, sizeof(mlk::MapStatsDev), cudaMemcpyDeviceToHost, st));
        MLENS_CUDA(cudaStreamSynchronize(st));
        memcpy(&nd, h->counters_host + 5, sizeof(int));
        if (h->mapstats_host->n_clamped == 0ull) break;  // every count had its own bin
        const long long need = (long long)h->mapstats_host->max_count + 2;
        if (need > 2147483647LL) return fail(MLENS_ERANGE, "largest count %d: the histogram would need more than 2^31-1 bins", h->mapstats_host->max_count);
        if (attempt > 0 || need <= n_bins) return fail(MLENS_ECUDA, "mlens_index_map: histogram of %lld bins still clamps (largest count %d)", n_bins, h->mapstats_host->max_count);
        n_bins = need;
    }
    *n_distinct = nd;
    if (nd > 65536) return fail(MLENS_ERANGE, "%d distinct ray-count values do not fit a 16-bit index", nd);
    if (nd > max_values) return fail(MLENS_ERANGE, "%d distinct ray-count values, values_dev holds %d", nd, max_values);
    // (4) the indexed map
    long long blocks = (n / 4 + 255) / 256;
    if (blocks > (long long)h->sm_count * 8) blocks = (long long)h->sm_count * 8;
    if (blocks < 1) blocks = 1;
    mlk::index_apply_kernel<<<(unsigned)blocks, 256, 0, st>>>(count_dev, n, h->idx_lut, indexed_dev);
    MLENS_CUDA(cudaGetLastError());
    return MLENS_OK;
}

int mlens_unindex_map(mlens_t* h, const unsigned short* indexed_dev, const int* values_dev, int n_values, int* count_dev,
                      void* cuda_stream) {
    if (!h || !indexed_dev || !values_dev || !count_dev) return fail(MLENS_EINVAL, "NULL argument");
    if (int rc = check_handle(h)) return rc;
    if (n_values < 1 || n_values > 65536) return fail(MLENS_EINVAL, "n_values must be 1..65536");
    const long long n = (long long)h->npix * h->npix;
    long long blocks = (n / 4 + 255) / 256;
    if (blocks > (long long)h->sm_count * 8) blocks = (long long)h->sm_count * 8;
    if (blocks < 1) blocks = 1;
    mlk::index_decode_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)cuda_stream>>>(indexed_dev, n, values_dev, n_values, count_dev);
    MLENS_CUDA(cudaGetLastError());
    return MLENS_OK;
}

int mlens_bits_needed(unsigned long long max_value) {
    int b = 1;
    while (b < 64 && (max_value >> b) != 0ull) ++b;
    return b;
}

long long mlens_packed_words(long long n_values, int bits) {
    if (n_values < 0 || bits < 1 || bits > 32) return -1;
    return (n_values * bits + 31) / 32;
}

int mlens_pack_map(mlens_t* h, const void* src_dev, int src_bits, int bits, unsigned int* packed_dev, void* cuda_stream) {
    if (!h || !src_dev || !packed_dev) return fail(MLENS_EINVAL, "NULL argument");
    if (int rc = check_handle(h)) return rc;
    if (src_bits != 16 && src_bits != 32) return fail(MLENS_EINVAL, "src_bits must be 16 or 32");
    if (bits < 1 || bits > src_bits) return fail(MLENS_EINVAL, "bits must be 1..src_bits");
    const long long n = (long long)h->npix * h->npix, n_words = mlens_packed_words(n, bits);
    // a chunk = n_sub sub-blocks of 256/bits whole 32-value periods, at most kPackChunkValues values
    const int vals_per_sub = (256 / bits) * 32;
    int n_sub = mlk::kPackChunkValues / vals_per_sub;
    if (n_sub < 1) n_sub = 1;
    const long long chunk_vals = (long long)n_sub * vals_per_sub;
    long long blocks = (n + chunk_vals - 1) / chunk_vals;
    if (blocks > (long long)h->sm_count * 32) blocks = (long long)h->sm_count * 32;
    if (blocks < 1) blocks = 1;
    if (src_bits == 32)
        mlk::pack_bits_kernel<int><<<(unsigned)blocks, 256, 0, (cudaStream_t)cuda_stream>>>((const int*)src_dev, n, bits, packed_dev, n_words, n_sub);
    else
        mlk::pack_bits_kernel<unsigned short><<<(unsigned)blocks, 256, 0, (cudaStream_t)cuda_stream>>>((const unsigned short*)src_dev, n, bits, packed_dev, n_words, n_sub);
    MLENS_CUDA(cudaGetLastError());
    return MLENS_OK;
}

int mlens_unpack_map(mlens_t* h, const unsigned int* packed_dev, int bits, void* dst_dev, int dst_bits, void* cuda_stream) {
    if (!h || !packed_dev || !dst_dev) return fail(MLENS_EINVAL, "NULL argument");
    if (int rc = check_handle(h)) return rc;
    if (dst_bits != 16 && dst_bits != 32) return fail(MLENS_EINVAL, "dst_bits must be 16 or 32");
    if (bits < 1 || bits > dst_bits) return fail(MLENS_EINVAL, "bits must be 1..dst_bits");
    const long long n = (long long)h->npix * h->npix;
    long long blocks = (n / (dst_bits == 32 ? 4 : 8) + 255) / 256;  // 16 bytes of output per thread
    if (blocks > (long long)h->sm_count * 16) blocks = (long long)h->sm_count * 16;
    if (blocks < 1) blocks = 1;
    if (dst_bits == 32)
        mlk::unpack_bits_kernel<int><<<(unsigned)blocks, 256, 0, (cudaStream_t)cuda_stream>>>(packed_dev, n, bits, (int*)dst_dev, mlens_packed_words(n, bits));
    else
        mlk::unpack_bits_kernel<unsigned short><<<(unsigned)blocks, 256, 0, (cudaStream_t)cuda_stream>>>(packed_dev, n, bits, (unsigned short*)dst_dev, mlens_packed_words(n, bits));
    MLENS_CUDA(cudaGetLastError());
    return MLENS_OK;
}

int mlens_mpd_rebin(mlens_t* h, const unsigned long long* hist_dev, int n_bins, int n_out, double mu_min, double mu_max,
                    double* prob_dev, void* cuda_stream) {
    if (!h || !hist_dev || !prob_dev) return fail(MLENS_EINVAL, "NULL argument");
    if (int rc = check_handle(h)) return rc;
    if (n_bins < 2) return fail(MLENS_EINVAL, "n_bins must be >= 2");
    if (n_out < 1 || n_out > 400) return fail(MLENS_EINVAL, "n_out must be 1..400 (PAPER.md:453: 'a maximum limit of 400')");
    if (!std::isfinite(mu_min) || !std::isfinite(mu_max) || !(mu_min > 0) || !(mu_max > mu_min))
        return fail(MLENS_EINVAL, "0 < mu_min < mu_max required");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    MLENS_CUDA(cudaMemsetAsync(prob_dev, 0, sizeof(double) * (size_t)n_out, st));  // 64-bit integer zeros, too
    // Reading S20: bin(c) = floor((log10(c / N_avg) - log10(mu_min)) / width), width = (log10(mu_max) - log10(mu_min)) / n_out,
    // kept when 0 <= bin < n_out.  The expression is monotone in c, so each bin is a range of counts: find the first count of
    // every bin here, by bisection on that very expression, and let the device work on integers only.
    const double log_min = std::log10(mu_min), width = (std::log10(mu_max) - log_min) / n_out, n_avg = h->geo.n_avg;
    auto position = [&](long long c) { return (std::log10((double)c / n_avg) - log_min) / width; };
    mlk::RebinEdges edges;
    for (int k = 0; k <= n_out; ++k) {
        long long a = 0, b = n_bins;  // position(a) < k (or a = 0: no logarithm), position(b) >= k (or b = n_bins: none)
        while (b - a > 1) {
            const long long mid = a + (b - a) / 2;
            if (position(mid) >= (double)k) b = mid; else a = mid;
        }
        edges.lo[k] = (int)b;
    }
    long long blocks = ((long long)n_bins + 255) / 256;
    if (blocks > (long long)h->sm_count * 8) blocks = (long long)h->sm_count * 8;
    mlk::mpd_rebin_kernel<<<(unsigned)blocks, 256, 0, st>>>(hist_dev, n_bins, n_out, edges, reinterpret_cast<unsigned long long*>(prob_dev));
    MLENS_CUDA(cudaGetLastError());
    mlk::mpd_rebin_finish_kernel<<<1, 512, 0, st>>>(prob_dev, n_out, (double)h->npix * (double)h->npix);
    MLENS_CUDA(cudaGetLastError());
    return MLENS_OK;
}

int mlens_profile_kernel(mlens_t* h, int shape, double size_pixels, float* kernel_dev, void* cuda_stream) {
    if (!h || !kernel_dev) return fail(MLENS_EINVAL, "NULL argument");
    if (int rc = check_handle(h)) return rc;
    if (shape != mlk::PROFILE_UNIFORM_DISC && shape != mlk::PROFILE_GAUSSIAN) return fail(MLENS_EINVAL, "unknown profile shape %d", shape);
    if (!std::isfinite(size_pixels) || !(size_pixels > 0)) return fail(MLENS_EINVAL, "profile size must be finite and > 0");
    const double half = shape == mlk::PROFILE_GAUSSIAN ? std::ceil(4.0 * size_pixels) : std::ceil(size_pixels);
    if (2.0 * half + 1.0 > (double)h->npix) return fail(MLENS_EINVAL, "profile support (%g pixels) does not fit the %d-pixel map", 2.0 * half + 1.0, h->npix);
    const int R = (int)half;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (!h->prof_sum) MLENS_CUDA(dev_alloc(&h->prof_sum, sizeof(double)));
    MLENS_CUDA(cudaMemsetAsync(h->prof_sum, 0, sizeof(double), st));
    const long long ns = (2LL * R + 1) * (2LL * R + 1);
    long long b1 = (ns + 255) / 256;
    if (b1 > (long long)h->sm_count * 8) b1 = (long long)h->sm_count * 8;
    mlk::profile_sum_kernel<<<(unsigned)b1, 256, 0, st>>>(shape, size_pixels, R, h->prof_sum);
    MLENS_CUDA(cudaGetLastError());
    const long long n = (long long)h->npix * h->npix;
    long long b2 = (n + 255) / 256;
    if (b2 > (long long)h->sm_count * 8) b2 = (long long)h->sm_count * 8;
    mlk::profile_fill_kernel<<<(unsigned)b2, 256, 0, st>>>(shape, size_pixels, R, h->npix, h->prof_sum, kernel_dev);
    MLENS_CUDA(cudaGetLastError());
    return MLENS_OK;
}

#define MLENS_CUFFT(call)                                                                   \
    do {                                                                                    \
        cufftResult r_ = (call);                                                            \
        if (r_ != CUFFT_SUCCESS)                                                            \
            return fail(r_ == CUFFT_ALLOC_FAILED ? MLENS_ENOMEM : MLENS_ECUDA, "%s: cuFFT error %d", #call, (int)r_); \
    } while (0)

namespace {
// cuFFT plans (created once per handle) bound to `st`
int convolve_plans(mlens_t* h, cudaStream_t st) {
    const int N = h->npix;
    if (!h->have_plans) {
        MLENS_CUFFT(cufftPlan2d(&h->plan_r2c, N, N, CUFFT_R2C));
        cufftResult r = cufftPlan2d(&h->plan_c2r, N, N, CUFFT_C2R);
        if (r != CUFFT_SUCCESS) { cufftDestroy(h->plan_r2c); return fail(MLENS_ECUDA, "cufftPlan2d(C2R): cuFFT error %d", (int)r); }
        h->have_plans = 1;
    }
    MLENS_CUFFT(cufftSetStream(h->plan_r2c, st));
    MLENS_CUFFT(cufftSetStream(h->plan_c2r, st));
    return MLENS_OK;
}
}  // namespace

int mlens_convolve_prepare(mlens_t* h, const float* kernel_dev, void* cuda_stream) {
    if (!h || !kernel_dev) return fail(MLENS_EINVAL, "NULL argument");
    if (int rc = check_handle(h)) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long long nc = (long long)h->npix * (h->npix / 2 + 1);
    if (int rc = convolve_plans(h, st)) return rc;
    if (!h->spec_prep) MLENS_CUDA(dev_alloc(&h->spec_prep, sizeof(float2) * (size_t)nc));
    h->have_prep = 0;
    MLENS_CUFFT(cufftExecR2C(h->plan_r2c, const_cast<float*>(kernel_dev), reinterpret_cast<cufftComplex*>(h->spec_prep)));
    h->have_prep = 1;
    return MLENS_OK;
}

int mlens_convolve(mlens_t* h, const float* map_dev, const float* kernel_dev, float* out_dev, void* cuda_stream) {
    if (!h || !map_dev || !out_dev) return fail(MLENS_EINVAL, "NULL argument");
    if (int rc = check_handle(h)) return rc;
    if (!kernel_dev && !h->have_prep) return fail(MLENS_EINVAL, "kernel_dev is NULL and no kernel was prepared (mlens_convolve_prepare)");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int N = h->npix;
    const long long nc = (long long)N * (N / 2 + 1);  // complex elements of an R2C spectrum
    if (int rc = convolve_plans(h, st)) return rc;
    if (!h->spec_map) MLENS_CUDA(dev_alloc(&h->spec_map, sizeof(float2) * (size_t)nc));
    // out-of-place R2C leaves its real input untouched; cuFFT takes non-const pointers
    MLENS_CUFFT(cufftExecR2C(h->plan_r2c, const_cast<float*>(map_dev), reinterpret_cast<cufftComplex*>(h->spec_map)));
    const float2* spec_k = h->spec_prep;  // the prepared spectrum, unless a kernel is given
    if (kernel_dev) {
        if (!h->spec_ker) MLENS_CUDA(dev_alloc(&h->spec_ker, sizeof(float2) * (size_t)nc));
        MLENS_CUFFT(cufftExecR2C(h->plan_r2c, const_cast<float*>(kernel_dev), reinterpret_cast<cufftComplex*>(h->spec_ker)));
        spec_k = h->spec_ker;
    }
    long long blocks = (nc / 2 + 255) / 256;
    if (blocks > (long long)h->sm_count * 8) blocks = (long long)h->sm_count * 8;
    if (blocks < 1) blocks = 1;
    mlk::spectral_product_kernel<<<(unsigned)blocks, 256, 0, st>>>(h->spec_map, spec_k, nc, 1.0f / ((float)N * (float)N));
    MLENS_CUDA(cudaGetLastError());
    MLENS_CUFFT(cufftExecC2R(h->plan_c2r, reinterpret_cast<cufftComplex*>(h->spec_map), out_dev));
    return MLENS_OK;
}

int mlens_shoot(mlens_t* h, int* count_dev, float* mag_dev, void* cuda_stream, mlens_stats* stats) {
    if (!h || !count_dev) return fail(MLENS_EINVAL, "NULL argument");
    if (int rc = check_handle(h)) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t n = (size_t)h->npix * h->npix;
    if (stats) MLENS_CUDA(cudaEventRecord(h->ev0, st));
    MLENS_CUDA(cudaMemsetAsync(count_dev, 0, n * sizeof(int), st));
    MLENS_CUDA(cudaMemsetAsync(h->counters_dev, 0, 4 * sizeof(unsigned long long), st));
    if (stats) MLENS_CUDA(cudaEventRecord(h->evk0, st));
    if (int rc = launch_block(h, 0, 0, h->geo.n1, h->geo.n2, count_dev, nullptr, nullptr, st)) return rc;
    if (stats) MLENS_CUDA(cudaEventRecord(h->evk1, st));
    if (int rc = launch_magnification(h, count_dev, mag_dev, st)) return rc;
    if (stats) {
        MLENS_CUDA(cudaEventRecord(h->ev1, st));
        MLENS_CUDA(cudaEventSynchronize(h->ev1));
        MLENS_CUDA(cudaEventElapsedTime(&h->last_ms, h->ev0, h->ev1));
        MLENS_CUDA(cudaEventElapsedTime(&h->last_kernel_ms, h->evk0, h->evk1));
        return read_stats(h, st, stats);
    }
    return MLENS_OK;
}

int mlens_shoot_host(mlens_t* h, int* count_host, float* mag_host, mlens_stats* stats) {
    if (!h || !count_host) return fail(MLENS_EINVAL, "NULL argument");
    if (int rc = check_handle(h)) return rc;
    const size_t n = (size_t)h->npix * h->npix;
    if (!h->own_stream) MLENS_CUDA(cudaStreamCreateWithFlags(&h->own_stream, cudaStreamNonBlocking));
    if (!h->count_own) MLENS_CUDA(dev_alloc(&h->count_own, n * sizeof(int)));
    if (mag_host && !h->mag_own) MLENS_CUDA(dev_alloc(&h->mag_own, n * sizeof(float)));
    mlens_stats local;
    if (int rc = mlens_shoot(h, h->count_own, mag_host ? h->mag_own : nullptr, h->own_stream, &local)) return rc;
    MLENS_CUDA(cudaMemcpyAsync(count_host, h->count_own, n * sizeof(int), cudaMemcpyDeviceToHost, h->own_stream));
    if (mag_host) MLENS_CUDA(cudaMemcpyAsync(mag_host, h->mag_own, n * sizeof(float), cudaMemcpyDeviceToHost, h->own_stream));
    MLENS_CUDA(cudaStreamSynchronize(h->own_stream));
    if (stats) *stats = local;
    return MLENS_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------
// mlens_mpd_static: the MPD of a count map for callers that must not allocate (include/mlens.h has the full contract).
//
// mlens_mpd needs a handle (mlens_create allocates the lens list, counters, events) and on first use takes its per-CTA
// histogram slices and a pinned statistics mirror from cudaMalloc / cudaMallocHost.  A process whose device memory is
// already spoken for — everything handed to one caching allocator at start-up, a fixed budget set by a job scheduler —
// or that computes map statistics next to running shooting kernels, where an allocation's device-wide synchronisation
// would stall them, cannot afford that.  Here the same two kernels (mpd_kernel, mpd_reduce_kernel) run with their
// scratch in the file-scope array below, which exists on every GPU that loads the library from load to exit.
//
// Size: kStaticMaxCtas slices of kStaticMaxBins 32-bit bins (148 x 8192 x 4 B = 4.6 MiB) + one MapStatsDev.
// ---------------------------------------------------------------------------------------------------------------
namespace {
constexpr int kStaticMaxBins = MLENS_MPD_STATIC_MAX_BINS;  // multiple of 1024 (the kernels' fill / flush loops)
constexpr int kStaticMaxCtas = 148;                        // one persistent CTA per SM of a B200
constexpr size_t kStaticSliceWords = (size_t)kStaticMaxCtas * kStaticMaxBins;
static_assert(kStaticMaxBins % 1024 == 0 && kStaticMaxBins <= mlk::kMpdSmemBinsMax, "static MPD bins");
static_assert(sizeof(mlk::MapStatsDev) <= 64 && (kStaticSliceWords * 4) % 256 == 0, "static MPD scratch layout");
}  // namespace

// [0, kStaticSliceWords): per-CTA histogram slices; then 16 words for the MapStatsDev accumulator.
// In HOST code this name is only a stand-in for the symbol: the device address comes from cudaGetSymbolAddress below.
static __device__ __align__(256) unsigned int g_mpd_static_scratch[kStaticSliceWords + 16];

namespace {
std::mutex g_static_mutex;
unsigned int* g_static_ptr[64];  // device address of g_mpd_static_scratch on each device, looked up once per device
int g_static_sm_count[64];

// Once per device, with that device current: look up the array's device address.  No allocation; the first call on a
// device may make the runtime load the library's module, which is why it should happen outside any stream capture.
int static_scratch(unsigned int** ptr, int* sm_count) {
    int dev = -1;
    MLENS_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return fail(MLENS_ECUDA, "device ordinal %d is outside 0..63", dev);
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {
        int cc_major = 0, cc_minor = 0, sms = 0;
        MLENS_CUDA(cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, dev));
        MLENS_CUDA(cudaDeviceGetAttribute(&cc_minor, cudaDevAttrComputeCapabilityMinor, dev));
        MLENS_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        if (cc_major != 10) return fail(MLENS_ECUDA, "device %d is sm_%d%d; this library is built for sm_100a only", dev, cc_major, cc_minor);
        void* p = nullptr;
        MLENS_CUDA(cudaGetSymbolAddress(&p, g_mpd_static_scratch));
        if (!p) return fail(MLENS_ECUDA, "cudaGetSymbolAddress returned a NULL address for the static MPD scratch");
        g_static_sm_count[dev] = sms;
        g_static_ptr[dev] = static_cast<unsigned int*>(p);
    }
    *ptr = g_static_ptr[dev];
    *sm_count = g_static_sm_count[dev];
    return MLENS_OK;
}
}  // namespace

extern "C" int mlens_mpd_static(const int* count_dev, long long n_pixels, double n_avg, unsigned long long* hist_dev,
                                int n_bins, void* cuda_stream, mlens_map_stats* stats) {
    if (!count_dev || !hist_dev) return fail(MLENS_EINVAL, "NULL argument");
    if (n_pixels < 1) return fail(MLENS_EINVAL, "n_pixels must be >= 1");
    if (n_bins < 2) return fail(MLENS_EINVAL, "n_bins must be >= 2");
    if (n_bins > kStaticMaxBins)
        return fail(MLENS_ERANGE, "n_bins = %d is beyond the %d bins that the static scratch of mlens_mpd_static holds; "
                    "use mlens_mpd (which allocates) for finer histograms", n_bins, kStaticMaxBins);
    if (stats && (!std::isfinite(n_avg) || !(n_avg > 0))) return fail(MLENS_EINVAL, "n_avg must be finite and > 0 when stats are requested");
    unsigned int* scratch = nullptr;
    int sm_count = 0;
    if (int rc = static_scratch(&scratch, &sm_count)) return rc;
    unsigned int* partial = scratch;
    mlk::MapStatsDev* st_dev = reinterpret_cast<mlk::MapStatsDev*>(scratch + kStaticSliceWords);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // What must start at zero: the statistics accumulator (atomic sums / maxima) and the caller's bins.  The slices need
    // no clearing although they keep the previous call's contents: every CTA overwrites its whole slice [0, smem_bins)
    // and the reduction reads exactly the slices of the CTAs of THIS launch.
    MLENS_CUDA(cudaMemsetAsync(st_dev, 0, sizeof(mlk::MapStatsDev), st));
    MLENS_CUDA(cudaMemsetAsync(hist_dev, 0, sizeof(unsigned long long) * (size_t)n_bins, st));
    const int smem_bins = (n_bins + 1023) & ~1023;  // <= kStaticMaxBins: all bins live in shared memory
    long long blocks = (n_pixels / 4 + mlk::kMpdThreads - 1) / mlk::kMpdThreads;
    if (blocks > sm_count) blocks = sm_count;
    if (blocks > kStaticMaxCtas) blocks = kStaticMaxCtas;
    if (blocks < 1) blocks = 1;
    const size_t smem = sizeof(unsigned int) * (size_t)smem_bins;
    {
        std::lock_guard<std::mutex> launch_lock(g_launch_mutex);
        MLENS_CUDA(cudaFuncSetAttribute(mlk::mpd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        mlk::mpd_kernel<<<(unsigned)blocks, mlk::kMpdThreads, smem, st>>>(count_dev, n_pixels, hist_dev, n_bins, smem_bins, partial, st_dev);
        MLENS_CUDA(cudaGetLastError());
    }
    mlk::mpd_reduce_kernel<<<(smem_bins + 31) / 32, 256, 0, st>>>(partial, (int)blocks, smem_bins, hist_dev, n_bins, st_dev);
    MLENS_CUDA(cudaGetLastError());
    if (stats) {
        mlk::MapStatsDev host;  // pageable stack memory: the copy is staged by the driver, nothing is allocated here
        MLENS_CUDA(cudaMemcpyAsync(&host, st_dev, sizeof(host), cudaMemcpyDeviceToHost, st));
        MLENS_CUDA(cudaStreamSynchronize(st));
        stats->n_pixels = n_pixels;
        stats->sum_count = (long long)host.sum_count;
        stats->n_clamped = (long long)host.n_clamped;
        stats->min_count = 0x7fffffff - host.inv_min_count;
        stats->max_count = host.max_count;
        stats->mean_count = (double)stats->sum_count / (double)n_pixels;
        stats->mean_mu = stats->mean_count / n_avg;
    }
    return MLENS_OK;
}
