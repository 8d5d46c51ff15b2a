/*
 * topo.c -- CPU oracle for the Betti numbers of a thresholded film (TEST INFRASTRUCTURE ONLY; see oracle/tfo.py).
 *
 * PAPER.md:457 (section 4.3): "consider a landscape sliced by a horizontal plane at the height H*.  Then, b0 counts
 * the number of mountain peaks (components) above H*, and b1 counts the number of valleys (loops) surrounding the
 * peaks."  The paper computes them with CHomP on cubical sets.  Written out for a 2-D image (R22):
 *   X(H*) = union of the closed unit squares of the cells with h > H*        (a cubical set)
 *   b0 = number of connected components of X: closed squares that share an edge OR a corner are connected
 *        (8-neighbourhood of cells)
 *   b1 = number of holes of X = bounded components of the complement (Alexander duality in the plane); the
 *        complement is open, so its cells connect through edges only (4-neighbourhood), and a component that
 *        reaches the border of the image is not bounded.
 * Plain flood fill with an explicit stack; no blocking, no union-find: nothing in common with the CUDA path.
 */
#include <stdlib.h>

/* labels components of cells with class `cls` (1: h > thr, 0: not) under the given neighbourhood;
 * returns the number of components; *touching = number of them with a cell on the image border */
static long long flood(const double* h, int nx, int ny, double thr, int cls, int eight, int* lab, int* stack,
                       long long* touching)
{
    long long ncomp = 0, ntouch = 0;
    const int dj[8] = {0, 0, 1, -1, 1, 1, -1, -1}, di[8] = {1, -1, 0, 0, 1, -1, 1, -1};
    const int nn = eight ? 8 : 4;
    for (int j0 = 0; j0 < ny; ++j0)
        for (int i0 = 0; i0 < nx; ++i0) {
            const int p0 = j0 * nx + i0;
            if (lab[p0] || ((h[p0] > thr) ? 1 : 0) != cls) continue;
            ++ncomp;
            int touch = 0, top = 0;
            stack[top++] = p0;
            lab[p0] = 1;
            while (top) {
                const int p = stack[--top];
                const int j = p / nx, i = p % nx;
                if (j == 0 || i == 0 || j == ny - 1 || i == nx - 1) touch = 1;
                for (int k = 0; k < nn; ++k) {
                    const int jj = j + dj[k], ii = i + di[k];
                    if (jj < 0 || ii < 0 || jj >= ny || ii >= nx) continue;
                    const int q = jj * nx + ii;
                    if (lab[q] || ((h[q] > thr) ? 1 : 0) != cls) continue;
                    lab[q] = 1;
                    stack[top++] = q;
                }
            }
            ntouch += touch;
        }
    *touching = ntouch;
    return ncomp;
}

/* b0[t], b1[t] for every threshold thr[t]; returns 0, or -1 if memory ran out */
int tfo_betti(const double* h, int nx, int ny, const double* thr, int nthr, long long* b0, long long* b1)
{
    const size_t n = (size_t)nx * ny;
    int* lab = (int*)malloc(n * sizeof(int));
    int* stack = (int*)malloc(n * sizeof(int));
    if (!lab || !stack) { free(lab); free(stack); return -1; }
    for (int t = 0; t < nthr; ++t) {
        long long touch;
        for (size_t p = 0; p < n; ++p) lab[p] = 0;
        b0[t] = flood(h, nx, ny, thr[t], 1, 1, lab, stack, &touch);
        const long long nbg = flood(h, nx, ny, thr[t], 0, 0, lab, stack, &touch);
        b1[t] = nbg - touch;
    }
    free(lab);
    free(stack);
    return 0;
}
