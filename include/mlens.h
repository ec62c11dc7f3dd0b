/* mlens.h — C ABI of libmlens.so: direct inverse ray-shooting for quasar-microlensing magnification maps on one
 * NVIDIA B200 (sm_100a).
 *
 * The operation (Vernardos & Fluke 2014, arXiv:1406.0559; line numbers are of /root/reference/PAPER.md):
 *   - PAPER.md:71   rays on a regular image-plane lattice are projected through the lens plane, "each deflected by
 *                   N_* individual lenses ... and accumulated on a gridded source plane";
 *   - PAPER.md:73   Eq. (1): y = diag(1-gamma, 1+gamma) x - kappa_s x - sum_{i=1..N_*} m_i (x - x_i)/|x - x_i|^2,
 *                   summed DIRECTLY over all N_* point lenses for every ray (GPU-D);
 *   - PAPER.md:75-77 Eq. (2): kappa = kappa_s + kappa_*, s = kappa_s/kappa;
 *   - PAPER.md:85-87 Eq. (4): mu_ij = N_ij / N_avg;  here N_avg = (pixel/ray_spacing)^2 (BASELINE.json north_star);
 *   - PAPER.md:294  the count map is 32-bit integers, Npix*Npix, row-major.
 * Conventions the paper leaves open are listed in DESIGN.md ("Readings"): cell-centred symmetric lattice
 * x = (i + 1/2 - n/2) d with n1 = 2*ceil(a1/d - 1e-9), a1 = 1.2 (L/2)/|1-kappa-gamma| (a2, n2 with +gamma);
 * half-open pixels with floor, ix from y1, iy from y2, pixel id = iy*Npix + ix, corner of pixel (0,0) at
 * (-L/2, -L/2); no softening — a ray with a non-finite source position is counted as "lost" and not binned.
 *
 * All lengths are in Einstein radii of the mean lens mass, masses in units of the mean mass.
 *
 * Every function returns MLENS_OK (0) or a negative mlens_status; none throws or aborts.  After a failure
 * mlens_last_error() returns a thread-local description.  There is NO CPU fallback: without a CUDA device
 * mlens_create fails with MLENS_ECUDA.  Pointers are marked HOST or DEVICE; DEVICE pointers must belong to the device
 * that was current when mlens_create was called, and that device must be the calling thread's current device in every
 * later call on the handle (checked: MLENS_EINVAL otherwise).  DEVICE map pointers (count, mag, hist, indexed, values,
 * kernel, out) must be 16-byte aligned — the kernels use 128-bit accesses; any cudaMalloc'ed or torch-allocated buffer
 * is.  `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *
 * Concurrency.  Calls on one handle must not be issued concurrently from several host threads.  From ONE thread:
 *   - mlens_shoot_block launches of one handle MAY be issued to different streams and overlap on the device: each
 *     launch owns its tile counter (a ring of 256; launch n + 256 is made to wait, on the device, for launch n — an
 *     event per slot — so more launches in flight are safe, only no longer concurrent), the ray counters and the count
 *     map are atomic sums;
 *   - mlens_shoot, mlens_mpd, mlens_index_map, mlens_profile_kernel and mlens_convolve use per-handle scratch (events,
 *     histogram slices, spectra, cuFFT plans): calls of these on one handle must be ordered after one another — issue
 *     them to one stream, or order the streams with events.  Use one handle per stream for concurrent maps.
 */
#ifndef MLENS_H_
#define MLENS_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mlens mlens_t; /* opaque; owns the device copy of the lens list, device counters, scratch */

typedef enum {
    MLENS_OK = 0,
    MLENS_EINVAL = -1, /* bad argument (see each function) */
    MLENS_ENOMEM = -2, /* host or device allocation failed */
    MLENS_ECUDA = -3,  /* CUDA runtime error (no device, launch failure, ...) */
    MLENS_ERANGE = -4  /* lattice or map too large for the index types */
} mlens_status;

typedef struct {
    long long rays_total;   /* rays shot since the counters were last reset */
    long long rays_in_map;  /* rays binned into the count map */
    long long rays_outside; /* finite source position outside the map */
    long long rays_lost;    /* non-finite source position (ray exactly on a lens) */
    long long n_lens;
    int max_count;          /* largest pixel count seen by the last mlens_shoot / mlens_magnification (overflow guard,
                               PAPER.md:692-698: the paper's largest observed count is 998 878) */
    float elapsed_ms;       /* device time of the last mlens_shoot that was given a stats pointer, else 0 */
    float kernel_ms;        /* of which: the shooting kernel alone (steps a1-a4), CUDA events on `cuda_stream` */
} mlens_stats;

typedef struct {
    long long n1, n2;                  /* lattice ray counts along x1, x2 */
    double a1, a2;                     /* shooting-rectangle half-widths */
    double p, d;                       /* pixel size L/Npix, ray spacing */
    double kappa_s, kappa_star, n_avg; /* Eq. 2 split; N_avg = (p/d)^2 */
} mlens_geometry;

typedef struct {
    long long n_pixels;    /* npix*npix */
    long long sum_count;   /* sum of all pixel counts (= rays_in_map of the map's own shoot) */
    long long n_clamped;   /* pixels with count >= n_bins-1: they all sit in the last bin of the histogram */
    int min_count, max_count;
    double mean_count;     /* <N>  = sum_count / n_pixels           (mapmeta.dat) */
    double mean_mu;        /* <mu> = <N> / N_avg                    (Eq. 4) */
} mlens_map_stats;

/* Create a map context (a map is defined by kappa, gamma, s, width, resolution, N_avg and the
 * lens positions/masses).
 *   kappa, gamma, s    total convergence, shear, smooth-matter fraction (0 <= s <= 1)
 *   map_side, npix     L > 0 and Npix > 0: side of the square source-plane map and its pixel count per side
 *   ray_spacing        d > 0: image-plane lattice spacing
 *   lens_xy            HOST, 2*n_lens floats, interleaved x,y; copied — the caller keeps ownership
 *   lens_m             HOST, n_lens floats (> 0, finite), or NULL for m_i = 1
 *   n_lens             >= 0 (0 = macro-model only)
 * The lattice (n1, n2) and the rectangle are derived here (see mlens_get_geometry).
 * Errors: MLENS_EINVAL for non-finite or out-of-range parameters, |1-kappa-gamma| or |1-kappa+gamma| < 1e-6 (critical
 * line: the rectangle is unbounded), kappa < 0, NULL out / lens_xy (when n_lens > 0), a non-finite lens coordinate or a
 * mass that is not finite and > 0;  MLENS_ERANGE if n1 or n2 >= 2^31 or npix^2 >= 2^31;  MLENS_ECUDA / MLENS_ENOMEM. */
int mlens_create(mlens_t** out, double kappa, double gamma, double s, double map_side, int npix, double ray_spacing,
                 const float* lens_xy, const float* lens_m, long long n_lens);

/* Shoot the whole lattice (steps a1-a5 of the hot path): zero `count_dev` and the ray counters, shoot all n1*n2
 * rays, bin them, then — if `mag_dev` is not NULL — write mag = (float)((double)count / N_avg).
 *   count_dev   DEVICE, npix*npix int32, row-major [iy][ix], caller-owned
 *   mag_dev     DEVICE, npix*npix float32, or NULL
 *   stats       HOST or NULL.  NULL: all work is only enqueued on `cuda_stream` and the call returns at once.
 *               Non-NULL: the call synchronises the stream and fills *stats (elapsed_ms = device time of this call). */
int mlens_shoot(mlens_t* h, int* count_dev, float* mag_dev, void* cuda_stream, mlens_stats* stats);

/* Verification / partial shooting: rays i0 <= i < i0+ni, j0 <= j < j0+nj of the SAME lattice, through the SAME
 * kernel.  ACCUMULATES into count_dev and into the ray counters (zero them yourself / mlens_reset_stats).
 *   count_dev   DEVICE npix*npix int32, or NULL (no binning)
 *   ray_y_dev   DEVICE ni*nj*2 doubles or NULL: source position of ray (ii, jj) at [2*(jj*ni+ii)], [.. + 1]
 *   ray_pix_dev DEVICE ni*nj int32 or NULL: pixel id, -1 = outside the map, -2 = non-finite
 * Asynchronous on `cuda_stream`.  MLENS_EINVAL if the block is not inside [0,n1) x [0,n2); MLENS_ERANGE (also from
 * mlens_shoot) if ray_spacing is so small against the lens distances or masses that the FP32 loop, which works in units
 * of ray_spacing, would leave the FP32 range ((|lens coordinate| + rectangle)/ray_spacing > ~2e18, or m/ray_spacing^2 >
 * 1e37) — far outside any physical configuration. */
int mlens_shoot_block(mlens_t* h, long long i0, long long j0, long long ni, long long nj, int* count_dev,
                      double* ray_y_dev, int* ray_pix_dev, void* cuda_stream);

/* End-to-end convenience with HOST buffers: device buffers owned by the handle, mlens_shoot, copies back,
 * synchronises.  count_host: HOST npix*npix int32; mag_host: HOST npix*npix float32 or NULL; stats: HOST or NULL. */
int mlens_shoot_host(mlens_t* h, int* count_host, float* mag_host, mlens_stats* stats);

/* Step a5 alone (Eq. 4): mag = (float)((double)count / N_avg); also refreshes max_count.  Asynchronous. */
int mlens_magnification(mlens_t* h, const int* count_dev, float* mag_dev, void* cuda_stream);

/* Map statistics.  The full magnification probability distribution of PAPER.md:307 ("the
 * frequency of each magnification value in a map is counted and then divided by the total number of pixels"): since
 * mu = count/N_avg with integer counts, the MPD is the histogram of the counts, hist[c] = number of pixels whose count
 * is c (divide by n_pixels for the probability, c by N_avg for the magnification axis).  Also <N> and <mu>
 * (mapmeta.dat).
 *   count_dev  DEVICE npix*npix int32 (a finished count map)
 *   hist_dev   DEVICE n_bins unsigned 64-bit integers, caller-owned; ZEROED by the call, then filled.  Counts
 *              >= n_bins-1 are clamped into the last bin (use n_bins >= max_count+2 for the unclamped MPD)
 *   n_bins     >= 2
 *   stats      HOST or NULL.  NULL: asynchronous on `cuda_stream`.  Non-NULL: synchronises the stream and fills it.
 * Integer arithmetic only: the result is exact.  MLENS_EINVAL for NULL pointers or n_bins < 2. */
int mlens_mpd(mlens_t* h, const int* count_dev, unsigned long long* hist_dev, int n_bins, void* cuda_stream,
              mlens_map_stats* stats);

/* The MPD for callers that cannot allocate memory.
 *
 * mlens_mpd works on a handle, and both mlens_create and the first mlens_mpd on a handle allocate (device blocks for the
 * lens list, the counters and the per-CTA histogram slices; pinned host blocks for the statistics).  Some users of this
 * library cannot do that at the point where they want a map's statistics: a survey worker or a server that gave all of
 * its device memory to one allocator when it started (so that a later cudaMalloc fails, or breaks a memory budget its
 * scheduler enforces), or a loop that analyses finished maps while the next map is being shot on another stream (an
 * allocation synchronises the whole device and would stall the shooting kernel).  This entry point computes the same
 * histogram and the same statistics with the same kernels, takes no handle, and calls no cudaMalloc, cudaMallocHost,
 * cudaFree or other allocating routine: its scratch is a fixed array that is part of the library image.
 *
 *   count_dev  DEVICE n_pixels int32, 16-byte aligned (a finished count map; any shape — only the pixel count matters)
 *   n_pixels   >= 1
 *   n_avg      N_avg of the map, (pixel/ray_spacing)^2; only used for stats->mean_mu (must be > 0 if stats != NULL)
 *   hist_dev   DEVICE n_bins unsigned 64-bit, caller-owned; ZEROED by the call, then filled exactly as by mlens_mpd
 *              (counts >= n_bins-1 are clamped into the last bin)
 *   n_bins     2 .. MLENS_MPD_STATIC_MAX_BINS.  More bins: MLENS_ERANGE — use mlens_mpd, or clamp
 *   stats      HOST or NULL, as in mlens_mpd: NULL = asynchronous on `cuda_stream`; otherwise the stream is
 *              synchronised and *stats filled (copied into the caller's struct directly, no pinned mirror)
 *
 * The scratch: 148 x MLENS_MPD_STATIC_MAX_BINS 32-bit bins + 64 bytes = 4.6 MiB of device memory, held by EVERY GPU on
 * which the process uses this library, from the moment the library is loaded there until the process exits — whether or
 * not this function is ever called.  That is the price of never allocating, and the reason for the limit on n_bins.
 * ONE array per GPU is shared by all callers in the process, and it keeps what the last call left in it.  The call
 * clears the part that must start at zero itself (on `cuda_stream`), so calls that are ordered one after the other —
 * same stream, or streams ordered by events — are independent of each other.  Two calls that may run on the GPU at the
 * same time (different streams without ordering, different host threads) RACE on the array and return wrong
 * histograms; nothing detects this.  Order them, or use handles and mlens_mpd for concurrent work.
 *
 * The first call on each device looks up the array's device address (once per device, with that device current) and
 * checks that the device is an sm_100 part; make that first call during set-up, before any stream capture is begun.
 * Later calls only enqueue two memsets and two kernels.
 * Errors: MLENS_EINVAL (NULL pointers, n_pixels < 1, n_bins < 2, bad n_avg with stats), MLENS_ERANGE (n_bins beyond the
 * limit), MLENS_ECUDA (no sm_100 device, CUDA failure). */
#define MLENS_MPD_STATIC_MAX_BINS 8192
int mlens_mpd_static(const int* count_dev, long long n_pixels, double n_avg, unsigned long long* hist_dev, int n_bins,
                     void* cuda_stream, mlens_map_stats* stats);

/* Indexed maps: "The index file will hold all the distinct ray-count values,
 * each matched to an index running from zero to the maximum number of distinct ray-counts in the map.  The indexed map
 * will have its pixel ray-count values replaced by the appropriate index" — stored in 16 bits, halving the map.
 *   count_dev    DEVICE npix*npix int32 (a finished count map, counts >= 0)
 *   values_dev   DEVICE max_values int32, caller-owned: the index file, distinct counts in ASCENDING order
 *   indexed_dev  DEVICE npix*npix unsigned 16-bit, caller-owned: index of every pixel's count
 *   n_distinct   HOST out: number of distinct values (bits needed = ceil(log2(n_distinct)), PAPER.md Table B.6)
 * Synchronises `cuda_stream` once (the distinct count comes back to the host; a second pass and synchronisation only
 * if the map's largest count exceeds the histogram capacity the handle has, initially 16 Ki bins).  Integer-exact and lossless:
 * mlens_unindex_map(indexed, values) reproduces count_dev bit for bit.  MLENS_ERANGE if the map has more than 65536
 * distinct values (the paper's maximum over ~70 000 maps is 58 042, Table B.5) or more than max_values; *n_distinct is
 * set in both cases. */
int mlens_index_map(mlens_t* h, const int* count_dev, int* values_dev, int max_values, unsigned short* indexed_dev,
                    void* cuda_stream, int* n_distinct);

/* Decode: count_dev[q] = values_dev[indexed_dev[q]] (-1 for an index >= n_values).  Asynchronous. */
int mlens_unindex_map(mlens_t* h, const unsigned short* indexed_dev, const int* values_dev, int n_values, int* count_dev,
                      void* cuda_stream);

/* Minimal-bit-width storage (PAPER.md:704-712 and Table B.6): "rather than using the standard 16-bit and 32-bit data
 * types, we could define our own data types, using in each case the minimum required number of bits to represent a
 * particular map" — for a ray-count map (bits from its largest count) or an indexed map (bits from n_distinct - 1).
 *   mlens_bits_needed(v)      HOST helper: the smallest b >= 1 with v < 2^b (Table B.6: 16383 -> 14, 65535 -> 16,
 *                             1048575 -> 20, 16777215 -> 24)
 *   mlens_packed_words(n, b)  HOST helper: 32-bit words of a packed array of n b-bit values = ceil(n*b/32); -1 on bad
 *                             arguments.  (A 10000^2 map at 14/16/20/22/24/32 bits: 167/191/238/262/286/381 MiB, Table B.6.)
 *   mlens_pack_map            src_dev: DEVICE npix*npix values, 32-bit (int32 ray counts) or 16-bit (indexed map) as
 *                             given by src_bits; packed_dev: DEVICE mlens_packed_words(npix*npix, bits) 32-bit words,
 *                             caller-owned.  Value q occupies bits [q*bits, (q+1)*bits) of the little-endian bit stream
 *                             (bit i of the stream is bit i%32 of word i/32).  Values are MASKED to `bits` bits: choose
 *                             bits from mlens_bits_needed(max value).  1 <= bits <= src_bits.
 *   mlens_unpack_map          the inverse, into 32-bit or 16-bit values (bits <= dst_bits).
 * Integer-exact, asynchronous on `cuda_stream`.  MLENS_EINVAL for NULL pointers or widths outside those ranges. */
int mlens_bits_needed(unsigned long long max_value);
long long mlens_packed_words(long long n_values, int bits);
int mlens_pack_map(mlens_t* h, const void* src_dev, int src_bits, int bits, unsigned int* packed_dev, void* cuda_stream);
int mlens_unpack_map(mlens_t* h, const unsigned int* packed_dev, int bits, void* dst_dev, int dst_bits, void* cuda_stream);

/* Re-binned view of the MPD (the tools bin the stored MPD "into a histogram before they are returned
 * to the user.  By default, the number of bins is set to 100, with a maximum limit of 400").  Reading S20:
 * n_out bins of equal width in log10(mu) on [mu_min, mu_max), mu = count / N_avg.
 *   hist_dev   DEVICE n_bins unsigned 64-bit: the exact histogram written by mlens_mpd (unclamped: n_bins >= max_count+2)
 *   prob_dev   DEVICE n_out doubles, caller-owned, zeroed by the call: prob[k] = (number of pixels with
 *              floor(n_out*(log10(mu) - log10(mu_min))/(log10(mu_max) - log10(mu_min))) == k) / npix^2.  Pixels with
 *              count 0 (mu = 0 has no logarithm) or mu outside [mu_min, mu_max) are left out, so sum(prob) <= 1.
 * Asynchronous.  MLENS_EINVAL unless 1 <= n_out <= 400, n_bins >= 2 and 0 < mu_min < mu_max (finite). */
int mlens_mpd_rebin(mlens_t* h, const unsigned long long* hist_dev, int n_bins, int n_out, double mu_min, double mu_max,
                    double* prob_dev, void* cuda_stream);

/* Finite-source convolution (Eq. 6): C = M * K = F^-1[F(M) F(K)].
 *
 * mlens_profile_kernel writes the convolution kernel K of a source profile: the profile is sampled at pixel centres
 * ("binned in pixels of equal physical size to the map pixels"), normalised to sum 1 in FP64, and laid out over the
 * whole npix*npix array ("appended with empty (zero) pixels to match the pixel dimensions of the map") with the
 * profile centre on pixel (0,0) and negative offsets wrapped to the far edge, so that the convolution does not shift
 * the map.
 *   shape        0 = uniform disc of radius size_pixels, 1 = Gaussian of sigma size_pixels (cut at 4 sigma)
 *   size_pixels  > 0, in map pixels; the support (2*ceil(size)+1, or 2*ceil(4 sigma)+1) must fit in npix
 *   kernel_dev   DEVICE npix*npix float32, caller-owned, fully overwritten
 *
 * mlens_convolve computes the CIRCULAR convolution out[y][x] = sum_{y',x'} map[y'][x'] * kernel[(y-y') mod npix][(x-x')
 * mod npix] — what Eq. 6 evaluates — with two real-to-complex cuFFT transforms, one fused product-and-normalise kernel
 * and one complex-to-real transform, all FP32, asynchronous on `cuda_stream`.
 *   map_dev, kernel_dev  DEVICE npix*npix float32 (any real arrays of the map's shape), not modified
 *   out_dev              DEVICE npix*npix float32, caller-owned; must not alias the inputs
 * The handle keeps the two cuFFT plans and two npix*(npix/2+1) complex spectra between calls (0.8 GB for npix = 10000).
 * MLENS_EINVAL for NULL pointers / bad shape or size; MLENS_ECUDA / MLENS_ENOMEM for CUDA and cuFFT failures.
 *
 * mlens_convolve_prepare transforms a kernel ONCE and keeps its spectrum in the handle (another npix*(npix/2+1) complex
 * numbers); afterwards mlens_convolve may be called with kernel_dev == NULL to reuse it — a survey convolves many maps
 * with one source profile (~1e6 convolutions), which saves one of the three FFTs per map.  The result is
 * bit-identical to passing the kernel.  MLENS_EINVAL if kernel_dev is NULL and nothing was prepared. */
int mlens_profile_kernel(mlens_t* h, int shape, double size_pixels, float* kernel_dev, void* cuda_stream);
int mlens_convolve_prepare(mlens_t* h, const float* kernel_dev, void* cuda_stream);
int mlens_convolve(mlens_t* h, const float* map_dev, const float* kernel_dev, float* out_dev, void* cuda_stream);

/* Derived lattice and parameters (pure host data; valid from mlens_create on). */
int mlens_get_geometry(const mlens_t* h, mlens_geometry* g);

/* Synchronise `cuda_stream` and read the device ray counters. */
int mlens_get_stats(mlens_t* h, void* cuda_stream, mlens_stats* stats);

/* Zero the device ray counters (asynchronous). */
int mlens_reset_stats(mlens_t* h, void* cuda_stream);

/* Tuning switches.  Keys of the shipped library (libmlens.so):
 *   "binning"      0 = one global RED per ray, 1 = per-thread run-combine (default), 2 = + warp aggregation,
 *                  3 = + CTA-private shared-memory window — four routes to the same map, bit-identical results
 *   "ctas_per_sm"  persistent CTAs per SM; 0 (default) = the kernel's own choice (2)
 *   "shared_pairs" ray pairs per lens (of a thread's 8) whose reciprocals are shared: 2 (default) or 0 (one MUFU.RCP per
 *                  ray; also chosen automatically when lens coordinates / ray_spacing would overflow the FP32 products)
 *   "kernel" = 1, "rays_per_thread" = 16, "tile_x" = 64: accepted with these (production) values only
 * The debug / ablation / experimental kernels and the sweep grid are compiled only with -DMLENS_ABLATIONS
 * (libmlens_ablations.so, which the tests and profiling runs load; the shipped library returns MLENS_EINVAL for them, so
 * the public ABI cannot select a kernel that misses the parity tolerances):
 *   "kernel"       0 = plain FP64 one-ray-per-thread kernel (plumbing/debug), 2 = plain-form FP32 kernel (does NOT meet
 *                  the parity tolerances: the evidence for the difference form; <= 12000 lenses), 4 = the round-1
 *                  production kernel (A/B baseline; its loop variant "shared_rcp" 0..2).  (3 and 5 were the tensor-pipe
 *                  experiment of rounds 1-2: closed negative and removed.)
 *   "rays_per_thread" 8 | 16, "tile_x" 64 | 48 | 32 (8 rays only), "shared_pairs" 0..4: the sweep grid of kernel 1
 * Returns MLENS_EINVAL for an unknown key or value. */
int mlens_set_option(mlens_t* h, const char* key, long long value);

/* Thread-local message for the last failure on this thread ("" if none). */
const char* mlens_last_error(void);

/* Releases everything mlens_create and later calls on the handle allocated (never the caller's buffers), after
 * synchronising the handle's device.  NULL is allowed.
 * MEMORY RETENTION: the device blocks are NOT returned to the driver.  They go to a library-owned memory pool (one per
 * device) that KEEPS them for the next handle, so that creating / shooting / destroying map after map does not pay
 * cudaMalloc / cudaFree each time (cudaFree of a map-sized buffer was measured at up to 1.5 s on the B200 box).  For a
 * handle that used mlens_shoot_host and mlens_convolve at npix = 10000 that is about 2 GB (two maps, three spectra), and a
 * program that alternates map sizes accumulates one such set per size.  Other allocators in the process (torch's
 * caching allocator, cuFFT work areas, NCCL) cannot use that memory until mlens_trim_memory is called.  The library
 * itself trims the pool and retries once when one of its own allocations fails. */
void mlens_destroy(mlens_t* h);

/* mlens_destroy for a caller who issued ALL work on this handle to `cuda_stream` (or ordered it before that stream with
 * events): waits for that stream only, not for the whole device, then releases the handle as mlens_destroy does.  A
 * survey that runs several maps at once, one handle per stream (maps are produced in batches of
 * thousands), uses this so that finishing one map does not wait for the maps still running on the other streams.
 * Work of this handle still running on another, unordered stream is a use-after-free.  NULL handle allowed. */
void mlens_destroy_on_stream(mlens_t* h, void* cuda_stream);

/* Hand the device blocks cached by destroyed handles on the CURRENT device back to the driver, and free the recycled
 * pinned host blocks (blocks of live handles stay). */
int mlens_trim_memory(void);

#ifdef __cplusplus
}
#endif
#endif /* MLENS_H_ */
