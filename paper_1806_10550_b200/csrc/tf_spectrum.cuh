// tf_spectrum.cuh -- radial Fourier transform, steps one to four of PAPER.md:760-776 (Appendix B).
//   1. magnitude of the 2-D DFT of zeta = h - H0: the transform itself is cuFFT (D2Z, a library FFT), these kernels
//      subtract H0 and expand the half spectrum to the full |Z| [ny][nx] array (|Z(-k)| = |Z(k)| for real input);
//   2. convolution with a separable Gaussian, truncated at ceil(3 sigma), normalised, periodic (R23);
//   3./4. (B.1): mean over the points of equal radius, i.e. equal key = kx^2 + ky^2 of the signed DFT indices on a
//      square domain, for keys <= kmax^2 (the paper restricts q to [0, 5 q_m]).
// Everything here is bandwidth-trivial next to the sweeps (three passes over one field).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tf {

constexpr int SP_THREADS = 256;
constexpr int SP_MAXW = 64;          // filter half-width limit: ceil(3 sigma) <= 64

__global__ void __launch_bounds__(SP_THREADS)
sp_subtract_kernel(size_t n, const double* __restrict__ h, double H0, double* __restrict__ zeta)
{
    for (size_t p = (size_t)blockIdx.x * SP_THREADS + threadIdx.x; p < n; p += (size_t)gridDim.x * SP_THREADS) zeta[p] = h[p] - H0;
}

// half spectrum Z[ky][kx], kx = 0 .. nx/2 (interleaved re, im) -> full magnitude [ny][nx]
__global__ void __launch_bounds__(SP_THREADS)
sp_magnitude_kernel(int nx, int ny, const double2* __restrict__ Z, double* __restrict__ mag)
{
    const int kx = blockIdx.x * SP_THREADS + threadIdx.x, ky = blockIdx.y;
    if (kx >= nx) return;
    const int nh = nx / 2 + 1;
    // real input: Z(ky, kx) = conj Z(-ky, -kx); the stored half has kx <= nx/2
    const int sx = kx < nh ? kx : nx - kx;
    const int sy = kx < nh ? ky : (ky == 0 ? 0 : ny - ky);
    const double2 z = Z[(size_t)sy * nh + sx];
    mag[(size_t)ky * nx + kx] = hypot(z.x, z.y);
}

struct SpWeights { double w[2 * SP_MAXW + 1]; int r; };

// out[ky][kx] = sum_m w[m] in[ky][kx - m] (ALONG_X) or in[ky - m][kx], indices modulo the size (periodic)
template <bool ALONG_X>
__global__ void __launch_bounds__(SP_THREADS)
sp_gauss_kernel(int nx, int ny, const double* __restrict__ in, double* __restrict__ out, const __grid_constant__ SpWeights W)
{
    const int kx = blockIdx.x * SP_THREADS + threadIdx.x, ky = blockIdx.y;
    if (kx >= nx) return;
    double acc = 0.0;
    for (int a = 0; a <= 2 * W.r; ++a) {             // fixed summation order a = 0 .. 2r
        const int m = a - W.r;
        int sx = kx, sy = ky;
        if (ALONG_X) { sx = (kx - m) % nx; if (sx < 0) sx += nx; }
        else { sy = (ky - m) % ny; if (sy < 0) sy += ny; }
        acc += W.w[a] * in[(size_t)sy * nx + sx];
    }
    out[(size_t)ky * nx + kx] = acc;
}

// sums[key] += value, counts[key] += 1 for key = kx~^2 + ky~^2 <= kmax2 (signed indices)
__global__ void __launch_bounds__(SP_THREADS)
sp_radial_kernel(int nx, int ny, const double* __restrict__ f, long long kmax2, double* __restrict__ sums,
                 unsigned long long* __restrict__ counts)
{
    const int kx = blockIdx.x * SP_THREADS + threadIdx.x, ky = blockIdx.y;
    if (kx >= nx) return;
    const long long sx = kx < (nx + 1) / 2 ? kx : kx - nx;      // signed DFT index (Nyquist counted negative)
    const long long sy = ky < (ny + 1) / 2 ? ky : ky - ny;
    const long long key = sx * sx + sy * sy;
    if (key > kmax2) return;
    atomicAdd(sums + key, f[(size_t)ky * nx + kx]);
    atomicAdd(counts + key, 1ull);
}

}  // namespace tf
