// convolve_kernel.cuh — device code of mlens_convolve / mlens_profile_kernel.
//
//   PAPER.md:143-150  "the projected two-dimensional source profile is binned in pixels of equal physical size to the
//                     map pixels, and then appended with empty (zero) pixels to match the pixel dimensions of the map
//                     ... C = M * K = F^-1[F(M) F(K)]" (Eq. 6), computed with cuFFT in the paper as well.
// The two FFTs and the inverse are cuFFT calls (a library FFT, as in the paper); the kernels here are the rest of the
// path: the source-profile kernel K written directly in its zero-padded, wrap-around layout, and the spectral product
// F(M) F(K) / N^2 fused with the normalisation of the unnormalised inverse transform.  Both are HBM-bound streams.
#pragma once
#include <cuda_runtime.h>

namespace mlk {

enum ProfileShape { PROFILE_UNIFORM_DISC = 0, PROFILE_GAUSSIAN = 1 };

// Unnormalised profile value of the pixel whose centre is (dx, dy) pixels from the profile centre.
//   uniform disc: 1 inside radius `size`, else 0;   Gaussian: exp(-r^2 / (2 size^2)), cut at 4 sigma (beyond: 0).
__device__ __forceinline__ double profile_value(int shape, double size, int dx, int dy) {
    const double r2 = (double)dx * dx + (double)dy * dy;
    if (shape == PROFILE_UNIFORM_DISC) return r2 <= size * size ? 1.0 : 0.0;
    return r2 <= 16.0 * size * size ? exp(-r2 / (2.0 * size * size)) : 0.0;
}

// Pass 1: sum of the unnormalised profile over its support [-R, R]^2 (R = support half-width in pixels), FP64.
__global__ void __launch_bounds__(256) profile_sum_kernel(int shape, double size, int R, double* __restrict__ sum) {
    const long long side = 2LL * R + 1, n = side * side;
    double acc = 0.0;
    for (long long q = (long long)blockIdx.x * 256 + threadIdx.x; q < n; q += (long long)gridDim.x * 256) {
        const int dy = (int)(q / side) - R, dx = (int)(q % side) - R;
        acc += profile_value(shape, size, dx, dy);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
    if ((threadIdx.x & 31) == 0 && acc != 0.0) atomicAdd(sum, acc);
}

// Pass 2: K[iy][ix] = profile(dx, dy) / sum with the profile centre on pixel (0,0) and negative offsets wrapped to the
// far edge (dx = ix for ix <= npix/2, ix - npix otherwise): the convolution then does not shift the map.  Every pixel
// is written (zeros outside the support = "appended with empty pixels").
__global__ void __launch_bounds__(256) profile_fill_kernel(int shape, double size, int R, int npix,
                                                           const double* __restrict__ sum, float* __restrict__ K) {
    const long long n = (long long)npix * npix;
    const double inv = 1.0 / *sum;
    for (long long q = (long long)blockIdx.x * 256 + threadIdx.x; q < n; q += (long long)gridDim.x * 256) {
        const int iy = (int)(q / npix), ix = (int)(q - (long long)iy * npix);
        const int dx = ix <= npix / 2 ? ix : ix - npix, dy = iy <= npix / 2 ? iy : iy - npix;
        float v = 0.f;
        if (dx >= -R && dx <= R && dy >= -R && dy <= R) v = (float)(profile_value(shape, size, dx, dy) * inv);
        K[q] = v;
    }
}

// A <- A * B * scale, elementwise over n complex numbers (float2), two per thread per iteration (float4 accesses).
// 24 bytes of HBM traffic per complex element (read A, read B, write A).
__global__ void __launch_bounds__(256) spectral_product_kernel(float2* __restrict__ A, const float2* __restrict__ B,
                                                               long long n, float scale) {
    const long long n2 = n >> 1;
    const long long stride = (long long)gridDim.x * 256;
    float4* A4 = reinterpret_cast<float4*>(A);
    const float4* B4 = reinterpret_cast<const float4*>(B);
    for (long long q = (long long)blockIdx.x * 256 + threadIdx.x; q < n2; q += stride) {
        const float4 a = A4[q], b = __ldg(B4 + q);
        float4 c;
        c.x = (a.x * b.x - a.y * b.y) * scale;
        c.y = (a.x * b.y + a.y * b.x) * scale;
        c.z = (a.z * b.z - a.w * b.w) * scale;
        c.w = (a.z * b.w + a.w * b.z) * scale;
        A4[q] = c;
    }
    if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
        const float2 a = A[n - 1], b = B[n - 1];
        A[n - 1] = make_float2((a.x * b.x - a.y * b.y) * scale, (a.x * b.y + a.y * b.x) * scale);
    }
}

}  // namespace mlk
