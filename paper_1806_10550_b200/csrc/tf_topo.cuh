// tf_topo.cuh -- Betti numbers b0, b1 of a thresholded film ("b0 counts the
// number of mountain peaks (components) above H*, and b1 counts the number of valleys (loops) surrounding the peaks").
// The paper runs CHomP on the host; here the counts come from one union-find labelling of the whole image on the GPU.
//
// Cubical-set conventions (R22): X = closed unit squares of the cells with h > H*.
//   b0 = components of X        : foreground cells connect through edges and corners (8-neighbourhood)
//   b1 = holes of X             : components of the complement (4-neighbourhood) that do not reach the image border
// One label array serves both classes: a cell is only ever united with neighbours of its own class.
//   topo_init_kernel    label = first cell of the cell's horizontal run inside its 32-cell warp segment (ballot),
//                       so that all unions along a row inside a segment are done before the first atomic
//   topo_merge_kernel   unions across segment seams, to the row above, and (foreground) across corners; a union is
//                       skipped when the two cells are already connected through a neighbour that makes the same union
//   topo_border_kernel  marks the root of every background component that has a cell on the image border
//   topo_count_kernel   roots (label == own index): foreground -> b0, unmarked background -> b1
// Union-find: roots only ever move to a smaller index (atomicMin), so a stale read returns an ancestor and the
// compare-and-retry loop of unite() repairs it; the counting kernels run after the merge kernel has completed.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tf {

constexpr int TOPO_THREADS = 256;    // threads per CTA, a multiple of 32: warp segments are aligned to 32 cells of a row

__device__ __forceinline__ int uf_find(int* L, int x)
{
    while (true) {
        const int p = __ldcg(L + x);
        if (p == x) return x;
        const int g = __ldcg(L + p);
        if (g == p) return p;
        L[x] = g;                     // path halving: g is an ancestor of x, whatever else happens concurrently
        x = g;
    }
}

__device__ __forceinline__ void uf_unite(int* L, int a, int b)
{
    while (true) {
        a = uf_find(L, a);
        b = uf_find(L, b);
        if (a == b) return;
        if (a > b) { const int t = a; a = b; b = t; }
        const int old = atomicMin(L + b, a);      // hang the larger root under the smaller one
        if (old == b) return;                      // b was still a root: done
        b = old;                                   // somebody moved b meanwhile: retry from where it points now
    }
}

// grid (ceil(nx / TOPO_THREADS), ny)
__global__ void __launch_bounds__(TOPO_THREADS)
topo_init_kernel(int nx, const double* __restrict__ h, double thr, int* __restrict__ L)
{
    const int i = blockIdx.x * TOPO_THREADS + threadIdx.x, j = blockIdx.y;
    const int lane = threadIdx.x & 31;
    const bool ok = i < nx;
    const size_t p = (size_t)j * nx + (ok ? i : nx - 1);
    const bool fg = ok && h[p] > thr;
    const unsigned bits = __ballot_sync(0xffffffffu, fg);
    // bit l of `starts`: cell l opens a run (segment start, or its class differs from the cell before it)
    const unsigned starts = (bits ^ (bits << 1)) | 1u;
    const unsigned below = starts & (0xffffffffu >> (31 - lane));
    const int run0 = 31 - __clz(below);
    if (ok) L[p] = (int)p - lane + run0;
}

// grid (ceil(nx / TOPO_THREADS), ny)
__global__ void __launch_bounds__(TOPO_THREADS)
topo_merge_kernel(int nx, int ny, const double* __restrict__ h, double thr, int* __restrict__ L)
{
    const int i = blockIdx.x * TOPO_THREADS + threadIdx.x, j = blockIdx.y;
    if (i >= nx) return;
    const int lane = threadIdx.x & 31;
    const int p = j * nx + i;
    const bool c = h[p] > thr;
    const bool hasW = i > 0, hasE = i < nx - 1, hasN = j > 0;
    const bool sameW = hasW && ((h[p - 1] > thr) == c);
    if (lane == 0 && sameW) uf_unite(L, p, p - 1);                 // seam between two warp segments of the row
    if (!hasN) return;
    const bool cN = h[p - nx] > thr;
    const bool cNW = hasW && (h[p - nx - 1] > thr), cNE = hasE && (h[p - nx + 1] > thr);
    const bool sameN = cN == c;
    // up: redundant if the cell to the left is in my run and its upper neighbour is in the upper run (it unites them)
    if (sameN && !(sameW && hasW && (cNW == c))) uf_unite(L, p, p - nx);
    if (c) {
        // corners, foreground only; skipped when an edge neighbour of mine (or of the corner cell) makes the connection
        const bool fW = hasW && sameW, fE = hasE && (h[p + 1] > thr);
        if (hasW && cNW && !cN && !fW) uf_unite(L, p, p - nx - 1);
        if (hasE && cNE && !cN && !fE) uf_unite(L, p, p - nx + 1);
    }
}

// one thread per border cell (2 nx + 2 ny, corners twice): background components that reach the border are not holes
__global__ void __launch_bounds__(TOPO_THREADS)
topo_border_kernel(int nx, int ny, const double* __restrict__ h, double thr, int* __restrict__ L, unsigned char* __restrict__ open)
{
    const int t = blockIdx.x * TOPO_THREADS + threadIdx.x;
    int i, j;
    if (t < nx) { i = t; j = 0; }
    else if (t < 2 * nx) { i = t - nx; j = ny - 1; }
    else if (t < 2 * nx + ny) { i = 0; j = t - 2 * nx; }
    else if (t < 2 * nx + 2 * ny) { i = nx - 1; j = t - 2 * nx - ny; }
    else return;
    const int p = j * nx + i;
    if (!(h[p] > thr)) open[uf_find(L, p)] = 1;
}

// grid-stride over all cells; cnt[0] += foreground roots, cnt[1] += background roots not marked open
__global__ void __launch_bounds__(TOPO_THREADS)
topo_count_kernel(size_t n, const double* __restrict__ h, double thr, const int* __restrict__ L,
                  const unsigned char* __restrict__ open, unsigned long long* __restrict__ cnt)
{
    unsigned n0 = 0, n1 = 0;
    for (size_t p = (size_t)blockIdx.x * TOPO_THREADS + threadIdx.x; p < n; p += (size_t)gridDim.x * TOPO_THREADS) {
        if (L[p] == (int)p) {
            if (h[p] > thr) ++n0;
            else if (!open[p]) ++n1;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        n0 += __shfl_xor_sync(0xffffffffu, n0, o);
        n1 += __shfl_xor_sync(0xffffffffu, n1, o);
    }
    if ((threadIdx.x & 31) == 0) {
        if (n0) atomicAdd(cnt, (unsigned long long)n0);
        if (n1) atomicAdd(cnt + 1, (unsigned long long)n1);
    }
}

}  // namespace tf
