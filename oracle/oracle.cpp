// ORACLE — TEST INFRASTRUCTURE ONLY.  Not part of the product path.
//
// Plain, slow, obviously-correct FP64 CPU implementation of direct inverse ray-shooting (GERLUMPH / GPU-D hot path,
// Vernardos & Fluke 2014, arXiv:1406.0559).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may load this library.  It shares NO code with the CUDA path (paper_1406_0559_b200/csrc):
// no headers, helpers, tables or constants.
//
// What it follows, in the paper's order and notation:
//   * PAPER.md:71   "large numbers (~10^9) of light rays are projected from the observer, through the lens plane,
//                    where they are each deflected by N_* individual lenses ... and accumulated on a gridded source
//                    plane"                                                        -> the three nested loops below
//   * PAPER.md:73   Eq. (1)  y = diag(1-gamma, 1+gamma) x - kappa_s x - sum_i m_i (x - x_i)/|x - x_i|^2
//   * PAPER.md:75-77 Eq. (2) kappa = kappa_s + kappa_*,  s = kappa_s/kappa
//   * PAPER.md:85-87 Eq. (4) mu_ij = N_ij / N_avg
//   * PAPER.md:103  Fig. 1: regular grid of rays on the lens plane; rectangular pixellated source-plane area.
// Where the paper is silent the readings S1-S17 of SURVEY.md §8(c) (restated in DESIGN.md "Readings") apply:
//   S2 cell-centred symmetric lattice  x = (i + 1/2 - n/2) d,  n = 2*ceil(a/d - 1e-9),
//      a1 = 1.2 (L/2)/|1-kappa-gamma|, a2 = 1.2 (L/2)/|1-kappa+gamma|          (BASELINE.json config rule)
//   S4 half-open pixels, floor; ix from y1, iy from y2; row-major iy*Npix+ix; corner of pixel (0,0) at (-L/2,-L/2)
//   S5 N_avg = (p/d)^2                                                            (BASELINE.json north_star)
//   S7 no softening; a non-finite source position counts as "lost" and is not binned
//   S8 lenses summed in input order, one FP64 accumulator per component
//   S14 lens arrays are FP32 at the interface and promoted exactly to double
//   S16 mag = (float)((double)count / N_avg)
//
// Pins (tests/test_oracle_pins.py, -m "not gpu"): P1 no-lens closed form, P2 single point lens A(u), P3 hand sums
// incl. the tolerance scale sum m/|x - x_i| (tests/golden/p3_hand_sums.txt), P4 ray conservation, P5 mean
// magnification, P6 mirror symmetry, P7 lens-order permutation, P8 mass-sheet transformation, P14 per-ray outputs of
// oracle_shoot_block / oracle_shoot_rays (y, alpha, scale, pixel) against oracle_map_points at lattice positions the
// TEST computes from reading S2, and against each other.  Parity status: pinned (the dense many-caustic regime itself
// has no closed form; there this code path, anchored by P1-P8 and P14, is the reference).
//
// Build: g++ -O3 -march=native -fopenmp -shared -fPIC oracle/oracle.cpp -o oracle/liboracle.so   (no fast-math)

#include <algorithm>
#include <cmath>
#include <vector>
#include <cstdint>
#include <cstring>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {

struct oracle_geometry {
    long long n1, n2;                       // lattice counts along x1, x2
    double a1, a2;                          // rectangle half-widths
    double p, d;                            // pixel size, ray spacing
    double kappa_s, kappa_star, n_avg;      // Eq. 2 split; N_avg = (p/d)^2
};

struct oracle_stats {
    long long rays_total, rays_in_map, rays_outside, rays_lost;
};

// Derived quantities (readings S2, S5).  Returns 0, or -1 on the critical line / bad arguments.
int oracle_derive_geometry(double kappa, double gamma, double s, double L, int npix, double d, oracle_geometry* g) {
    if (!(L > 0) || npix <= 0 || !(d > 0) || !(s >= 0 && s <= 1)) return -1;
    const double f1 = std::fabs(1.0 - kappa - gamma), f2 = std::fabs(1.0 - kappa + gamma);
    if (f1 < 1e-6 || f2 < 1e-6) return -1;
    g->kappa_s = s * kappa;
    g->kappa_star = kappa - g->kappa_s;
    g->p = L / npix;
    g->d = d;
    g->a1 = 1.2 * (L / 2.0) / f1;
    g->a2 = 1.2 * (L / 2.0) / f2;
    g->n1 = 2 * (long long)std::ceil(g->a1 / d - 1e-9);
    g->n2 = 2 * (long long)std::ceil(g->a2 / d - 1e-9);
    g->n_avg = (g->p / d) * (g->p / d);
    return 0;
}

// One ray, Eq. (1) written out.  alpha = sum_i m_i (x - x_i)/|x - x_i|^2 ; scale = sum_i m_i/|x - x_i| (the
// north_star's tolerance scale for the per-ray deflection check).
static inline void shoot_one(double x1, double x2, double kappa_s, double gamma, const float* lens_xy,
                             const float* lens_m, long long n_lens, double* y1, double* y2, double* al1, double* al2,
                             double* scale /* NULL: skip the sqrt */) {
    double a1s = 0.0, a2s = 0.0, sc = 0.0;
    for (long long k = 0; k < n_lens; ++k) {
        const double dx = x1 - (double)lens_xy[2 * k];
        const double dy = x2 - (double)lens_xy[2 * k + 1];
        const double r2 = dx * dx + dy * dy;
        const double m = lens_m ? (double)lens_m[k] : 1.0;
        const double w = m / r2;
        a1s += w * dx;
        a2s += w * dy;
        if (scale) sc += m / std::sqrt(r2);
    }
    *y1 = (1.0 - kappa_s - gamma) * x1 - a1s;
    *y2 = (1.0 - kappa_s + gamma) * x2 - a2s;
    *al1 = a1s;
    *al2 = a2s;
    if (scale) *scale = sc;
}

// Image-plane position of lattice index k along an axis with n rays (reading S2): cell-centred, symmetric about 0.
// The ONE place the lattice formula is written; oracle_shoot_block and oracle_shoot_rays both call it.
static inline double lattice_x(long long k, long long n, double d) { return ((double)k + 0.5 - (double)n / 2.0) * d; }

// Pixel id of a source position: >= 0 in map, -1 outside, -2 non-finite (readings S4, S7).
static inline int pixel_of(double y1, double y2, double L, double p, int npix) {
    if (!std::isfinite(y1) || !std::isfinite(y2)) return -2;
    const double u1 = (y1 + L / 2.0) / p;
    const double u2 = (y2 + L / 2.0) / p;
    if (u1 >= 0.0 && u1 < (double)npix && u2 >= 0.0 && u2 < (double)npix)
        return (int)std::floor(u2) * npix + (int)std::floor(u1);
    return -1;
}

// Rays i0 <= i < i0+ni, j0 <= j < j0+nj of the lattice.  count (npix*npix int32) is ACCUMULATED into (may be NULL).
// Optional per-ray outputs, ray (ii, jj) of the block at index q = jj*ni + ii:
//   ray_y[2q], ray_y[2q+1] source position; ray_alpha[2q..] deflection; ray_scale[q]; ray_pix[q].
int oracle_shoot_block(double kappa, double gamma, double s, double L, int npix, double d, const float* lens_xy,
                       const float* lens_m, long long n_lens, long long i0, long long j0, long long ni, long long nj,
                       int* count, double* ray_y, double* ray_alpha, double* ray_scale, int* ray_pix,
                       oracle_stats* stats, int n_threads) {
    oracle_geometry g;
    if (oracle_derive_geometry(kappa, gamma, s, L, npix, d, &g) != 0) return -1;
    if (i0 < 0 || j0 < 0 || ni < 0 || nj < 0 || i0 + ni > g.n1 || j0 + nj > g.n2) return -1;
    long long in_map = 0, outside = 0, lost = 0;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : in_map, outside, lost)
    for (long long jj = 0; jj < nj; ++jj) {
        const double x2 = lattice_x(j0 + jj, g.n2, d);
        for (long long ii = 0; ii < ni; ++ii) {
            const double x1 = lattice_x(i0 + ii, g.n1, d);
            double y1, y2, al1, al2, sc = 0.0;
            shoot_one(x1, x2, g.kappa_s, gamma, lens_xy, lens_m, n_lens, &y1, &y2, &al1, &al2, ray_scale ? &sc : nullptr);
            const int pix = pixel_of(y1, y2, L, g.p, npix);
            const long long q = jj * ni + ii;
            if (ray_y) { ray_y[2 * q] = y1; ray_y[2 * q + 1] = y2; }
            if (ray_alpha) { ray_alpha[2 * q] = al1; ray_alpha[2 * q + 1] = al2; }
            if (ray_scale) ray_scale[q] = sc;
            if (ray_pix) ray_pix[q] = pix;
            if (pix >= 0) {
                ++in_map;
                if (count) {
#pragma omp atomic
                    count[pix] += 1;
                }
            } else if (pix == -1) {
                ++outside;
            } else {
                ++lost;
            }
        }
    }
    if (stats) {
        stats->rays_total = ni * nj;
        stats->rays_in_map = in_map;
        stats->rays_outside = outside;
        stats->rays_lost = lost;
    }
    return 0;
}

// A list of individual lattice rays (ray_ij[2q] = i, ray_ij[2q+1] = j): sampled checks at the full-size configs.
int oracle_shoot_rays(double kappa, double gamma, double s, double L, int npix, double d, const float* lens_xy,
                      const float* lens_m, long long n_lens, const long long* ray_ij, long long n_rays, double* ray_y,
                      double* ray_alpha, double* ray_scale, int* ray_pix, int n_threads) {
    oracle_geometry g;
    if (oracle_derive_geometry(kappa, gamma, s, L, npix, d, &g) != 0) return -1;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic, 64)
    for (long long q = 0; q < n_rays; ++q) {
        const double x1 = lattice_x(ray_ij[2 * q], g.n1, d);
        const double x2 = lattice_x(ray_ij[2 * q + 1], g.n2, d);
        double y1, y2, al1, al2, sc = 0.0;
        shoot_one(x1, x2, g.kappa_s, gamma, lens_xy, lens_m, n_lens, &y1, &y2, &al1, &al2, ray_scale ? &sc : nullptr);
        if (ray_y) { ray_y[2 * q] = y1; ray_y[2 * q + 1] = y2; }
        if (ray_alpha) { ray_alpha[2 * q] = al1; ray_alpha[2 * q + 1] = al2; }
        if (ray_scale) ray_scale[q] = sc;
        if (ray_pix) ray_pix[q] = pixel_of(y1, y2, L, g.p, npix);
    }
    return 0;
}

// Arbitrary image-plane positions (not lattice rays): used by pin P3 (hand sums, Appendix D of SURVEY.md).
// scale (optional): the per-ray tolerance scale sum_i m_i/|x - x_i| of the same shoot_one call.
int oracle_map_points(double kappa, double gamma, double s, const float* lens_xy, const float* lens_m,
                      long long n_lens, const double* x, long long n_pts, double* y, double* alpha, double* scale) {
    const double kappa_s = s * kappa;
    for (long long q = 0; q < n_pts; ++q) {
        double y1, y2, al1, al2, sc = 0.0;
        shoot_one(x[2 * q], x[2 * q + 1], kappa_s, gamma, lens_xy, lens_m, n_lens, &y1, &y2, &al1, &al2,
                  scale ? &sc : nullptr);
        y[2 * q] = y1; y[2 * q + 1] = y2;
        if (alpha) { alpha[2 * q] = al1; alpha[2 * q + 1] = al2; }
        if (scale) scale[q] = sc;
    }
    return 0;
}

// Pixel ids for given source positions (exposes the S4 convention to the tests).
void oracle_pixels_of(const double* y, long long n_pts, double L, int npix, int* pix) {
    const double p = L / npix;
    for (long long q = 0; q < n_pts; ++q) pix[q] = pixel_of(y[2 * q], y[2 * q + 1], L, p, npix);
}

// Eq. (4) with N_avg = (p/d)^2 (readings S5, S16).
void oracle_magnification(const int* count, long long n_pixels, double n_avg, float* mag) {
    for (long long q = 0; q < n_pixels; ++q) mag[q] = (float)((double)count[q] / n_avg);
}

// Full magnification probability distribution ("the frequency of each magnification value in a map is
// counted and then divided by the total number of pixels") and the map means of mapmeta.dat.  mu is
// count/N_avg (Eq. 4) with integer counts, so the MPD is the histogram of the counts: hist[c] = #pixels with count c.
// Counts >= n_bins-1 are put in the last bin (same clamping convention as include/mlens.h).  One pixel at a time.
// out[0] = sum of counts, out[1] = number of clamped pixels, out[2] = min count, out[3] = max count.
void oracle_mpd(const int* count, long long n_pixels, unsigned long long* hist, int n_bins, long long* out) {
    for (int b = 0; b < n_bins; ++b) hist[b] = 0ull;
    long long sum = 0, clamped = 0, cmin = 2147483647LL, cmax = 0;
    for (long long q = 0; q < n_pixels; ++q) {
        const int c = count[q];
        sum += c;
        if (c < cmin) cmin = c;
        if (c > cmax) cmax = c;
        int b = c < 0 ? 0 : c;
        if (b >= n_bins - 1) { b = n_bins - 1; ++clamped; }
        hist[b] += 1ull;
    }
    out[0] = sum; out[1] = clamped; out[2] = cmin; out[3] = cmax;
}

// Source-profile convolution kernel K ("the projected two-dimensional source profile is binned in
// pixels of equal physical size to the map pixels, and then appended with empty (zero) pixels to match the pixel
// dimensions of the map").  Reading S19: the profile is sampled at pixel centres, normalised to sum 1, its
// centre sits on pixel (0,0) and negative offsets wrap to the far edge.  shape 0: uniform disc of radius `size`
// pixels; shape 1: Gaussian of sigma `size` pixels, cut at 4 sigma.
void oracle_profile_kernel(int shape, double size, int npix, float* K) {
    std::vector<double> v((size_t)npix * npix, 0.0);
    double sum = 0.0;
    for (int iy = 0; iy < npix; ++iy) {
        for (int ix = 0; ix < npix; ++ix) {
            const int dx = ix <= npix / 2 ? ix : ix - npix, dy = iy <= npix / 2 ? iy : iy - npix;
            const double r2 = (double)dx * dx + (double)dy * dy;
            double p = 0.0;
            if (shape == 0) p = (r2 <= size * size) ? 1.0 : 0.0;
            else p = (r2 <= 16.0 * size * size) ? std::exp(-r2 / (2.0 * size * size)) : 0.0;
            v[(size_t)iy * npix + ix] = p;
            sum += p;
        }
    }
    for (size_t q = 0; q < v.size(); ++q) K[q] = (float)(v[q] / sum);
}

// Eq. 6, C = M * K = F^-1[F(M) F(K)]: by the convolution theorem for the discrete transform this is the
// CIRCULAR convolution, written out here as its definition, one requested output pixel at a time, in FP64:
//   C[y][x] = sum_{y',x'} K[y'][x'] * M[(y - y') mod N][(x - x') mod N]
// (only non-zero K entries contribute; the loop skips zeros).  pts = n_pts (y, x) pairs; n_pts < 0 => all N*N pixels in
// row-major order.
void oracle_convolve_at(const float* M, const float* K, int npix, const long long* pts, long long n_pts, double* out) {
    std::vector<int> ky, kx;
    std::vector<double> kv;
    for (int y = 0; y < npix; ++y)
        for (int x = 0; x < npix; ++x)
            if (K[(size_t)y * npix + x] != 0.0f) { ky.push_back(y); kx.push_back(x); kv.push_back((double)K[(size_t)y * npix + x]); }
    const long long n = n_pts < 0 ? (long long)npix * npix : n_pts;
#pragma omp parallel for schedule(static)
    for (long long q = 0; q < n; ++q) {
        const int y = n_pts < 0 ? (int)(q / npix) : (int)pts[2 * q], x = n_pts < 0 ? (int)(q % npix) : (int)pts[2 * q + 1];
        double acc = 0.0;
        for (size_t t = 0; t < kv.size(); ++t) {
            int yy = y - ky[t], xx = x - kx[t];
            if (yy < 0) yy += npix;
            if (xx < 0) xx += npix;
            acc += kv[t] * (double)M[(size_t)yy * npix + xx];
        }
        out[q] = acc;
    }
}

// Indexed map: index file = the distinct ray-count values (ascending), indexed map = every pixel's
// count replaced by its position in the index file.  Plain sort + unique + binary search.  Returns the number of
// distinct values (values must hold n_pixels entries at most; indexed holds 32-bit indices here).
long long oracle_index_map(const int* count, long long n_pixels, int* values, int* indexed) {
    std::vector<int> v(count, count + n_pixels);
    std::sort(v.begin(), v.end());
    v.erase(std::unique(v.begin(), v.end()), v.end());
    for (size_t k = 0; k < v.size(); ++k) values[k] = v[k];
    for (long long q = 0; q < n_pixels; ++q)
        indexed[q] = (int)(std::lower_bound(v.begin(), v.end(), count[q]) - v.begin());
    return (long long)v.size();
}

// Minimal-bit-width storage (Table B.6).  Bit by bit, straight from the definition: bit k of value q
// is bit q*bits + k of the stream, and bit i of the stream is bit i%32 of 32-bit word i/32.
int oracle_bits_needed(unsigned long long max_value) {
    // the number of binary digits of max_value (halve until nothing is left); zero still takes one bit
    int digits = 0;
    for (unsigned long long v = max_value; v != 0ull; v /= 2ull) ++digits;
    return digits > 0 ? digits : 1;
}

void oracle_pack_bits(const unsigned int* values, long long n, int bits, unsigned int* packed, long long n_words) {
    for (long long w = 0; w < n_words; ++w) packed[w] = 0u;
    for (long long q = 0; q < n; ++q)
        for (int k = 0; k < bits; ++k)
            if ((values[q] >> k) & 1u) {
                const long long i = q * bits + k;
                packed[i >> 5] |= 1u << (i & 31);
            }
}

void oracle_unpack_bits(const unsigned int* packed, long long n, int bits, unsigned int* values) {
    for (long long q = 0; q < n; ++q) {
        unsigned int v = 0u;
        for (int k = 0; k < bits; ++k) {
            const long long i = q * bits + k;
            if ((packed[i >> 5] >> (i & 31)) & 1u) v |= 1u << k;
        }
        values[q] = v;
    }
}

// Re-binned MPD (reading S20): n_out equal-width bins in log10(mu) on [mu_min, mu_max), one count
// value at a time.
void oracle_mpd_rebin(const unsigned long long* hist, int n_bins, double n_avg, double n_pixels, int n_out, double mu_min,
                      double mu_max, double* prob) {
    // reading S20: prob[k] = (number of pixels whose mu falls in bin k) / n_pixels — count the pixels, divide once
    std::vector<unsigned long long> pixels((size_t)n_out, 0ull);
    const double log_min = std::log10(mu_min), width = (std::log10(mu_max) - log_min) / n_out;
    for (int c = 1; c < n_bins; ++c) {
        if (!hist[c]) continue;
        const double t = (std::log10((double)c / n_avg) - log_min) / width;
        if (t >= 0.0 && t < (double)n_out) pixels[(size_t)(int)t] += hist[c];
    }
    for (int k = 0; k < n_out; ++k) prob[k] = (double)pixels[(size_t)k] / n_pixels;
}

int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
