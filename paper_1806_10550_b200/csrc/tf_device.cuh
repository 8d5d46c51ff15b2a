// tf_device.cuh -- device-side arithmetic shared by the sweep kernels (sm_100a, fp64).
//
// What is computed (citations are PAPER.md lines of arXiv:1806.10550):
//   cell functions  f0 = h^3, f0' = 3h^2, f1 = h^3 Pi'(h), f1' = d f1/dh      (1.7)-(1.8), :84-91
//   face flux       F = fb0 * d(lap h)/ds + fb1 * dh/ds, fb = mean of 2 cells  (2.1), (2.27), :134, :290
//   directional Jacobian partials of the face flux                             (2.26), :274-278
//   pentadiagonal LU forward elimination / back substitution                   :729-734, (A.5)
// Everything is scaled by s = dt/2 and the grid spacings up front so that a row of the
// system matrix I + s*J costs the fewest fp64 instructions (the fp64 pipe is the co-limiter
// of this path next to HBM).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tf {

struct Params {
    int nx, ny;
    double dx, dy;
    double rdx2, rdy2;      // 1/dx^2, 1/dy^2
    int n, m;               // Pi exponents, n > m >= 1
    double cm, cn;          // kappa*m*hstar^m, kappa*n*hstar^n
    double mp[10];          // constants of the NLC / polymer pressures (tf_set_pressure), see cell_functions
};

// model selectors carried in the kernels' <N, M> template pair (N > 0: power law with exponents N, M; 0: runtime n, m)
constexpr int MODEL_NLC = -2, MODEL_POLYMER = -3;

// per-direction constants for one dt:  ca = s/(2 d^4),  cb = s/(2 d^2)
struct Dir { double ca, cb; };

__device__ __forceinline__ int refl(int k, int N) { return k < 0 ? -k - 1 : (k >= N ? 2 * N - 1 - k : k); }
__device__ __forceinline__ int clampi(int k, int lo, int hi) { return k < lo ? lo : (k > hi ? hi : k); }
// reflected then clamped: safe address for any k, exact ghost for k in [-N, 2N)
__device__ __forceinline__ int ghost(int k, int N) { return clampi(refl(k, N), 0, N - 1); }

// Reciprocal on the critical path of every recurrence (pivot 1/mu) and of every cell (1/h):
// MUFU.RCP64H seed (rel. error ~1.5e-7 measured) + one cubically convergent step y(1 + e + e^2):
// 20 + 3x8 cycles of dependent latency instead of ~72 for the IEEE division sequence, error <= 1 ulp.
// Arguments are positive normal numbers here (h > 0 is validated; pivots of I + sJ are ~1..2).
__device__ __forceinline__ double rcp(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    const double t = fma(e, e, e);
    return fma(y, t, y);
}

struct Cell { double f0, f1, g0, g1; };

// r^k for k >= 0, h^(-k) for k < 0 (small integer k; unrolled by the compiler when k is constant)
__device__ __forceinline__ double ipow_rh(double r, double h, int k)
{
    double b = k >= 0 ? r : h, p = 1.0;
    for (int t = (k >= 0 ? k : -k); t > 0; --t) p *= b;
    return p;
}

// Cell-centre functions.  With r = 1/h:  h^3 Pi'(h) = cm r^(m-2) - cn r^(n-2)  and its derivative
// (2-m) cm r^(m-1) + (n-2) cn r^(n-1)  (the same polynomials as 3h^2 Pi' + h^3 Pi'', summed exactly).
// NLC (1.8)-(1.9): Pi = K[(b/h)^3 - (b/h)^2] + (N/2) M^2, M = m(h)/h = g h/(h^2 + beta^2),
//   g = (1 + tanh((h - 2b)/w))/2.  mp = {cap0, cap1, K b^3, K b^2, N, beta^2, 1/w, 2b}.
// polymer (1.12): Pi = 8C/h^9 - A1/(6 pi h^3) + (A1 - A2)/(6 pi (h+d)^3).
//   mp = {cap0, cap1, C, A1/(2 pi), (A1 - A2)/(2 pi), d}.
// Both: f0 = cap0 h^3, f1 = cap1 h^3 Pi'(h) (1.7); the derivatives Pi', Pi'' are written out by hand below.
template <int N, int M>
__device__ __forceinline__ Cell cell_functions(double h, const Params& P)
{
    Cell c;
    const double r = rcp(h);
    const double h2 = h * h;
    if (N == MODEL_NLC || N == MODEL_POLYMER) {
        double P1, P2;
        if (N == MODEL_NLC) {
            const double Kb3 = P.mp[2], Kb2 = P.mp[3], Nn = P.mp[4], be2 = P.mp[5], iw = P.mp[6];
            // g = (1 + tanh x)/2 = 1/(1 + e^(-2x)); 1 - tanh^2 = 4 g (1 - g); tanh = 2g - 1 (one exp and one
            // reciprocal instead of the library tanh; x clamped so that e^(-2x) stays finite)
            const double x = fmin(fmax((h - P.mp[7]) * iw, -300.0), 300.0);
            const double g = rcp(1.0 + exp(-2.0 * x));
            const double t = fma(2.0, g, -1.0);
            const double s2 = 4.0 * g * (1.0 - g);
            const double g1 = 0.5 * s2 * iw, g2 = -t * s2 * iw * iw;
            const double rD = rcp(h2 + be2), bh = be2 - h2;
            const double Mm = g * h * rD;
            const double M1 = fma(g1, h, g * bh * rD) * rD;
            const double M2 = fma(g2, h, fma(2.0 * g1, bh, g * h * fma(2.0, h2, -6.0 * be2) * rD) * rD) * rD;
            const double r2 = r * r, r3 = r2 * r;
            P1 = fma(-3.0 * Kb3, r, 2.0 * Kb2) * r3 + Nn * Mm * M1;
            P2 = fma(12.0 * Kb3, r, -6.0 * Kb2) * r3 * r + Nn * fma(M1, M1, Mm * M2);
        } else {
            const double Cc = P.mp[2], a1 = P.mp[3], da = P.mp[4];
            const double rd = rcp(h + P.mp[5]);
            const double r2 = r * r, r4 = r2 * r2, r5 = r4 * r, r10 = r5 * r5;
            const double rd2 = rd * rd, rd4 = rd2 * rd2;
            P1 = fma(-72.0 * Cc, r10, fma(a1, r4, -da * rd4));
            P2 = fma(720.0 * Cc, r10 * r, fma(-4.0 * a1, r5, 4.0 * da * rd4 * rd));
        }
        const double h3 = h2 * h;
        c.f0 = P.mp[0] * h3;
        c.g0 = 3.0 * P.mp[0] * h2;
        c.f1 = P.mp[1] * h3 * P1;
        c.g1 = P.mp[1] * fma(3.0 * h2, P1, h3 * P2);
        return c;
    }
    c.f0 = h2 * h;
    c.g0 = 3.0 * h2;
    if (N == 3 && M == 2) {
        c.f1 = fma(-P.cn, r, P.cm);
        c.g1 = P.cn * r * r;
    } else {
        const int n = P.n, m = P.m;
        c.f1 = P.cm * ipow_rh(r, h, m - 2) - P.cn * ipow_rh(r, h, n - 2);
        c.g1 = (2 - m) * P.cm * ipow_rh(r, h, m - 1) + (n - 2) * P.cn * ipow_rh(r, h, n - 1);
    }
    return c;
}

// Scaled partials of one interior face between line points k and k+1 (spacing d):
//   A  = s/d * dF/dh_{k+2} = -s/d * dF/dh_{k-1} = ca*(f0_k + f0_{k+1})
//   p1 = s/d * dF/dh_k,  p2 = s/d * dF/dh_{k+1}            (unfolded)
struct Face { double A, p1, p2; };

// hm1..hp2 = h_{k-1}, h_k, h_{k+1}, h_{k+2};  sf0 = f0_k + f0_{k+1}, sf1 likewise;  dh = h_{k+1} - h_k
__device__ __forceinline__ Face face_partials(double hm1, double hp2, double dh, double sf0, double sf1,
                                              const Cell& ck, const Cell& ck1, const Dir& D)
{
    Face f;
    f.A = D.ca * sf0;
    const double B = D.cb * sf1;
    const double t = fma(-3.0, dh, hp2 - hm1);        // third difference * d^3
    const double tt = D.ca * t, gg = D.cb * dh;
    const double c3 = fma(3.0, f.A, -B);
    f.p1 = fma(ck.g0, tt, fma(ck.g1, gg, c3));
    f.p2 = fma(ck1.g0, tt, fma(ck1.g1, gg, -c3));
    return f;
}

// One row of the LU forward elimination.  State: (a1,b1,z1) = row i-1, (a2,b2,z2) = row i-2.
struct Elim { double a1, b1, z1, a2, b2, z2; };

__device__ __forceinline__ void elim_row(Elim& S, double e, double c, double q, double a, double b, double y,
                                         double& al, double& be, double& zz)
{
    const double gam = fma(-S.a2, e, c);
    const double mu = fma(-S.a1, gam, fma(-S.b2, e, q));
    const double rmu = rcp(mu);
    al = fma(-S.b1, gam, a) * rmu;
    be = b * rmu;
    zz = fma(-S.z1, gam, fma(-S.z2, e, y)) * rmu;
    S.a2 = S.a1; S.b2 = S.b1; S.z2 = S.z1;
    S.a1 = al; S.b1 = be; S.z1 = zz;
}

// ---------------------------------------------------------------------------------------------
// The same elimination with the shortest loop-carried dependency chain (measured on B200: DFMA 8.2
// cycles, MUFU.RCP64H 17.7; elim_row carries 75 cycles per row, this one 52).  Only 256 warps march
// an 8192^2 sweep, so the chain length x ny is a floor of the sweep time.
//   * row i-1 is carried UNFINISHED: its pivot reciprocal is r1 = y1 + y1*t1 (y1 the MUFU seed, t1 =
//     e + e^2 the cubic correction), its alpha, beta, z numerators are p1, b1, s1;
//   * the next pivot mu_i = T - (p1*gam) r1 is expanded as (T - g y1) - (g y1) t1, so that only ONE
//     fma follows the arrival of t1:  chain = fma(mu) -> MUFU -> fma(e) -> fma(t).
// A call consumes the bands of row i and emits the FINAL coefficients of row i-1 (the caller stores them
// one row behind and calls elim2_flush after the last row).  Same arithmetic as (A.5)/PAPER.md:729-734
// up to rounding (the reciprocal is applied in expanded form).
// ---------------------------------------------------------------------------------------------
struct Elim2 { double y1, t1, p1, b1, s1, a2, b2, z2; };

__device__ __forceinline__ Elim2 elim2_init() { Elim2 S = {0, 0, 0, 0, 0, 0, 0, 0}; return S; }

__device__ __forceinline__ void elim2_row(Elim2& S, double e, double c, double q, double a, double b, double y,
                                          double& al, double& be, double& zz)
{
    const double gam = fma(-S.a2, e, c);
    const double T = fma(-S.b2, e, q);
    const double g = S.p1 * gam;
    const double bg = S.b1 * gam;
    const double sy = fma(-S.z2, e, y);
    const double u1 = fma(-g, S.y1, T);
    const double G = g * S.y1;
    const double mu = fma(-G, S.t1, u1);             // the only op between t1 and the next seed
    double y0;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(mu));
    const double ee = fma(-mu, y0, 1.0);
    const double tt = fma(ee, ee, ee);
    const double r1 = fma(S.y1, S.t1, S.y1);         // finish row i-1, off the critical path
    al = S.p1 * r1; be = S.b1 * r1;
    zz = S.s1 * r1;
    const double s = fma(-zz, gam, sy);
    const double p = fma(-bg, r1, a);
    S.a2 = al; S.b2 = be; S.z2 = zz;
    S.y1 = y0; S.t1 = tt; S.p1 = p; S.b1 = b; S.s1 = s;
}

__device__ __forceinline__ void elim2_flush(const Elim2& S, double& al, double& be, double& zz)
{
    const double r1 = fma(S.y1, S.t1, S.y1);
    al = S.p1 * r1; be = S.b1 * r1; zz = S.s1 * r1;
}

// (No "memory" clobber on purpose: the stored fields are never read by the storing kernel, and a clobber
// would pin the next row's shared-memory loads behind this row's stores.)
// Predicated 8-byte store without a branch: the marching warps keep halo / out-of-range lanes alive, and a
// branch around the stores of every row would cut the row loop into basic blocks (no overlap of the next
// row's loads with this row's dependency chain).
__device__ __forceinline__ void st_if(int p, double* addr, double v)
{
    asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %2, 0;\n@q st.global.f64 [%0], %1;\n}\n" ::"l"(addr), "d"(v), "r"(p));
}

// three predicated stores under one predicate (alpha, beta, z of one row)
__device__ __forceinline__ void st3_if(int p, double* a0, double v0, double* a1, double v1, double* a2, double v2)
{
    asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %6, 0;\n@q st.global.f64 [%0], %3;\n@q st.global.f64 [%1], %4;\n"
                 "@q st.global.f64 [%2], %5;\n}\n" ::"l"(a0), "l"(a1), "l"(a2), "d"(v0), "d"(v1), "d"(v2), "r"(p));
}

// L2 prefetch hint (no register, no shared memory): the marching producers pull the rows they will need a
// few tiles from now into L2, so that their register loads one tile ahead see L2 latency, not HBM latency.
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// Speculative launch-ahead (S8): the host enqueues iteration k+1 before it has read the residual of iteration k.
// Every kernel of iteration k+1 first looks at iteration k's record {res, bad} (final: the writing kernel has
// completed in stream order) and returns at once if that iteration already converged (res < tol), produced a bad
// iterate, or a NaN -- so the iterate of the deciding iteration is left untouched.  p == nullptr: no gate.
// s != nullptr (on-device adaptive controller): the kernels take s = dt/2 of the current attempt from device memory
// and form their direction constants themselves, with the divisions of the host's make_dir (same bits).
struct Gate { const double* p; double tol; const double* s; };
__device__ __forceinline__ Dir dir_of(double s, double d)
{
    Dir D;
    D.ca = s / (2.0 * d * d * d * d);
    D.cb = s / (2.0 * d * d);
    return D;
}
__device__ __forceinline__ bool gate_closed(const Gate& g)
{
    if (g.p == nullptr) return false;
    const double r = __ldcg(g.p), b = __ldcg(g.p + 1);
    return !(r >= g.tol) || b != 0.0;
}

// warp index as a value the compiler knows to be warp-uniform (role branches then do not look divergent)
__device__ __forceinline__ int uniform_warp_idx() { return __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0); }

// order-preserving max for non-negative doubles (NaN bit patterns compare above +inf, so a NaN
// anywhere surfaces in the result)
__device__ __forceinline__ void atomic_max_nonneg(double* addr, double v)
{
    atomicMax(reinterpret_cast<unsigned long long*>(addr), (unsigned long long)__double_as_longlong(v));
}

__device__ __forceinline__ double warp_max_nonneg(double v)
{
    unsigned long long b = (unsigned long long)__double_as_longlong(v);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        unsigned long long t = __shfl_xor_sync(0xffffffffu, b, o);
        b = t > b ? t : b;
    }
    return __longlong_as_double((long long)b);
}

}  // namespace tf
