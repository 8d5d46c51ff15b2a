// tf_pcr.cuh -- CTA-cooperative parallel cyclic reduction for pentadiagonal systems stored along rows (the x-sweep's
// shape), the alternative BASELINE.json names for the x-sweep ("a warp-cooperative cyclic-reduction variant ... picked by
// measurement") and one of the two techniques the paper lists for parallelising a single system.
//
// A pentadiagonal system is block tridiagonal in pairs X_k = (x_2k, x_2k+1):  A_k X_{k-1} + B_k X_k + C_k X_{k+1} = Y_k
// with 2 x 2 blocks.  One PCR level with stride s replaces row k by  row_k - (A_k B_{k-s}^-1) row_{k-s} - (C_k B_{k+s}^-1) row_{k+s},
// which couples X_k to X_{k-2s}, X_{k+2s} only; after ceil(log2(nb)) levels every row reads B_k X_k = Y_k.  No pivoting
// (like the LU).  One CTA holds one whole system in shared memory (14 doubles per pair), one thread per
// pair; global traffic is the compulsory 56 B per unknown, the price is ~76 fp64 operations per pair and level against
// 17 per unknown for the LU.  Measured against the thread-per-line LU in DESIGN.md section 11.
#pragma once
#include <cuda_runtime.h>

namespace tf {

struct M2 { double a, b, c, d; };                     // [[a, b], [c, d]]
struct Blk { M2 A, B, C; double y0, y1; };

__device__ __forceinline__ M2 m2_mul(const M2& p, const M2& q)
{
    return M2{fma(p.a, q.a, p.b * q.c), fma(p.a, q.b, p.b * q.d), fma(p.c, q.a, p.d * q.c), fma(p.c, q.b, p.d * q.d)};
}
__device__ __forceinline__ M2 m2_inv(const M2& p)
{
    const double r = 1.0 / fma(p.a, p.d, -p.b * p.c);
    return M2{p.d * r, -p.b * r, -p.c * r, p.a * r};
}

constexpr int PCR_VALS = 14;

__device__ __forceinline__ Blk pcr_load(const double* sm, int k, int nb)
{
    if (k < 0 || k >= nb) return Blk{{0, 0, 0, 0}, {1, 0, 0, 1}, {0, 0, 0, 0}, 0.0, 0.0};   // a row that is not there
    const double* p = sm + k;                          // value v of pair k at sm[v * nb + k]: conflict-free
    Blk b;
    b.A = M2{p[0], p[nb], p[2 * nb], p[3 * nb]};
    b.B = M2{p[4 * nb], p[5 * nb], p[6 * nb], p[7 * nb]};
    b.C = M2{p[8 * nb], p[9 * nb], p[10 * nb], p[11 * nb]};
    b.y0 = p[12 * nb]; b.y1 = p[13 * nb];
    return b;
}

// one CTA per system (row), blockDim.x = nb rounded up to a warp; arrays [nrow][ncol] row-major, ncol = 2 nb
// MAXT: 512 (systems up to 1024 unknowns, 128 registers per thread) or 1024 (up to 2048 unknowns, 64 registers: spills)
template <int MAXT>
__global__ void __launch_bounds__(MAXT) penta_row_pcr_kernel(int ncol, const double* __restrict__ e, const double* __restrict__ c,
                                     const double* __restrict__ d, const double* __restrict__ a, const double* __restrict__ b,
                                     const double* __restrict__ rhs, double* __restrict__ x)
{
    extern __shared__ double sm[];
    const int nb = ncol / 2, k = threadIdx.x;
    const size_t row = (size_t)blockIdx.x * ncol;
    Blk me = {{0, 0, 0, 0}, {1, 0, 0, 1}, {0, 0, 0, 0}, 0.0, 0.0};
    if (k < nb) {
        const size_t o = row + 2 * k;
        const double2 E = *reinterpret_cast<const double2*>(e + o), Cc = *reinterpret_cast<const double2*>(c + o);
        const double2 D = *reinterpret_cast<const double2*>(d + o), Aa = *reinterpret_cast<const double2*>(a + o);
        const double2 Bb = *reinterpret_cast<const double2*>(b + o), Y = *reinterpret_cast<const double2*>(rhs + o);
        const bool first = (k == 0), last = (k == nb - 1);
        me.A = first ? M2{0, 0, 0, 0} : M2{E.x, Cc.x, 0.0, E.y};
        me.B = M2{D.x, Aa.x, Cc.y, D.y};
        me.C = last ? M2{0, 0, 0, 0} : M2{Bb.x, 0.0, Aa.y, Bb.y};
        me.y0 = Y.x; me.y1 = Y.y;
    }
    for (int s = 1; s < nb; s <<= 1) {
        if (k < nb) {
            double* p = sm + k;
            p[0] = me.A.a; p[nb] = me.A.b; p[2 * nb] = me.A.c; p[3 * nb] = me.A.d;
            p[4 * nb] = me.B.a; p[5 * nb] = me.B.b; p[6 * nb] = me.B.c; p[7 * nb] = me.B.d;
            p[8 * nb] = me.C.a; p[9 * nb] = me.C.b; p[10 * nb] = me.C.c; p[11 * nb] = me.C.d;
            p[12 * nb] = me.y0; p[13 * nb] = me.y1;
        }
        __syncthreads();
        if (k < nb) {
            const Blk lo = pcr_load(sm, k - s, nb), hi = pcr_load(sm, k + s, nb);
            const M2 al = m2_mul(me.A, m2_inv(lo.B)), ga = m2_mul(me.C, m2_inv(hi.B));
            const M2 t1 = m2_mul(al, lo.C), t2 = m2_mul(ga, hi.A);
            const M2 nA = m2_mul(al, lo.A), nC = m2_mul(ga, hi.C);
            me.B = M2{me.B.a - t1.a - t2.a, me.B.b - t1.b - t2.b, me.B.c - t1.c - t2.c, me.B.d - t1.d - t2.d};
            me.y0 = me.y0 - fma(al.a, lo.y0, al.b * lo.y1) - fma(ga.a, hi.y0, ga.b * hi.y1);
            me.y1 = me.y1 - fma(al.c, lo.y0, al.d * lo.y1) - fma(ga.c, hi.y0, ga.d * hi.y1);
            me.A = M2{-nA.a, -nA.b, -nA.c, -nA.d};
            me.C = M2{-nC.a, -nC.b, -nC.c, -nC.d};
        }
        __syncthreads();
    }
    if (k < nb) {
        const M2 Bi = m2_inv(me.B);
        double2 X;
        X.x = fma(Bi.a, me.y0, Bi.b * me.y1);
        X.y = fma(Bi.c, me.y0, Bi.d * me.y1);
        *reinterpret_cast<double2*>(x + row + 2 * k) = X;
    }
}

}  // namespace tf
