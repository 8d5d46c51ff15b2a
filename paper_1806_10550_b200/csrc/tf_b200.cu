// tf_b200.cu -- C-ABI (include/tf.h) and host step driver of the B200 thin-film ADI sweep.
// Host side only orders kernels on one stream and reads one 16-byte residual record per Newton
// iteration (the paper reads IJ/256 flag bytes per iteration; S8 of DESIGN.md).
#include "../../include/tf.h"
#include <cuda.h>
#include "tf_penta.cuh"
#include "tf_bwd.cuh"
#include "tf_fwd.cuh"
#include "tf_topo.cuh"
#include "tf_spectrum.cuh"
#include "tf_blocks.cuh"
#include "tf_control.cuh"
#include "tf_pcr.cuh"
#include <dlfcn.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

namespace {

using namespace tf;

constexpr int MAX_ITERS = 4096;
constexpr size_t ALIGN = 256;

std::atomic<unsigned long long> g_launches{0};
thread_local std::string g_err;

size_t align_up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }
size_t field_bytes(int nx, int ny) { return align_up((size_t)nx * ny * sizeof(double)); }
size_t scratch_bytes() { return align_up(sizeof(double) * (2 * (MAX_ITERS + 1) + RED_BLOCKS + 8 + CT_SIZE + 4 * CT_HIST_CAP)); }
constexpr int NFIELDS = 8;   // u, uk, bn, w, alpha, beta, z, a (second time derivative kept for the truncation criterion)

}  // namespace

struct tf_ctx {
    Params P;
    double kappa, hstar;
    int model;                                 // tf_pressure: TF_PI_POWER (create-time kappa, h*, n, m), TF_PI_NLC, TF_PI_POLYMER
    double tol;
    int max_iter, fixed_iters;
    bool have_state, owns_ws;
    cudaStream_t stream;
    char* ws;
    double *u, *uk, *bn, *w, *al, *be, *zz;    // fields
    double *red;                               // [2*(MAX_ITERS+1)] residual / bad flag per iteration
    double *part;                              // [RED_BLOCKS]
    double *scal;                              // [8] : scal[0] mass, (int*)(scal+1) flag
    double *ctl, *ctl_hist;                    // on-device adaptive controller: control block [CT_SIZE], history [4 * CT_HIST_CAP]
    double *pinned;                            // [4] host pinned readback
    double *pinned_red;                        // [2*MAX_ITERS] host pinned copy of the residual records
    double last_change;                        // max |u^{n+1} - u^n| / u^n of the last converged step (criterion on)
    double max_rel_change;                     // extra solution criterion (0 = off): reject a converged step that changed h by more
    double *acc;                               // a_{n-1/2} of the last accepted step (truncation criterion; swaps with w on acceptance)
    double max_trunc, last_trunc, dt_prev;     // truncation criterion: limit (0 = off), last estimate, step of the stored a
    bool have_acc;                             // acc holds a_{n-1/2} of the step that led to the current state
    int spec_batch, last_iters;                // speculative launch-ahead: batch size (0 = off), iterations of the last accepted step
    int mid_y, mid_x;                          // split rows / columns of the two-sided sweeps
    int num_sms;
    bool tma_y, tma_x;                         // TMA rings usable (row pitch multiple of 16 B, grid >= one box)
    CUtensorMap mY[3], mX[3];                  // alpha,beta,z as [ny][nx] (box RS x 32) and as [nx][ny] (box CS x 32)
    CUtensorMap mU[2];                         // the two state buffers as [ny][nx], box 32 x 16, 128-byte swizzle
    bool tma_yf;                               // y forward producers stage their inputs by TMA
    CUtensorMap mUy[2], mBn;                   // state buffers / b^n as [ny][nx], boxes (RP+4) x 32 and RP x 32
    double* ubuf[2];                           // buffer addresses mU[0], mU[1] were encoded for
    // CUDA graphs of launch-ahead batches (small grids are launch-bound): a batch {first iteration, count, which buffer
    // holds u^n, dt/2} that comes back is captured once and replayed; any setter that changes a launch argument clears them
    struct GraphEntry { int k0, n, parity; double s; cudaGraphExec_t exec; unsigned long long stamp; };
    std::vector<GraphEntry> graphs;
    std::vector<GraphEntry> misses;            // keys seen once (u and u_k swap every step, so keys alternate)
    bool use_graphs;
    cudaStream_t gstream;                      // capture stream (the caller's may be the legacy default stream)
    double* w0;                                // the buffer w started in (w and a swap when the truncation criterion accepts)
    unsigned long long gstamp, graph_replays;
    bool profiling;
    cudaEvent_t ev[65 * 5];                    // 5 events per iteration, up to 65 iterations in flight
    double prof_ms[TF_PROFILE_SLOTS];
    unsigned long long prof_n[TF_PROFILE_SLOTS];
    std::string err;
};

namespace {

tf_status fail(tf_ctx* c, tf_status st, const std::string& msg)
{
    if (c) c->err = msg; else g_err = msg;
    return st;
}

tf_status cuda_fail(tf_ctx* c, cudaError_t e, const char* what)
{
    return fail(c, TF_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define TF_CUDA(c, call)                                              \
    do {                                                              \
        cudaError_t e__ = (call);                                     \
        if (e__ != cudaSuccess) return cuda_fail((c), e__, #call);    \
    } while (0)

inline void count_launch(int n = 1) { g_launches.fetch_add((unsigned long long)n, std::memory_order_relaxed); }

Dir make_dir(double s, double d) { Dir D; D.ca = s / (2.0 * d * d * d * d); D.cb = s / (2.0 * d * d); return D; }

// ---- TMA tensor maps (driver entry point fetched through the runtime: no link-time libcuda dependency)
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn lookup_encode_tiled()
{
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
        return (EncodeTiledFn)p;
    return nullptr;
}

// contexts are created from several host threads (one per rank in the in-process multi-rank tests): the
// function-local static is initialised exactly once, thread-safely
EncodeTiledFn encode_tiled_fn()
{
    static const EncodeTiledFn fn = lookup_encode_tiled();
    return fn;
}

// fp64 matrix [outer][inner] (row pitch inner*8 bytes), box [box_outer][box_inner]
bool make_map2d(CUtensorMap* m, const double* base, int inner, int outer, int box_inner, int box_outer, bool swz128)
{
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return false;
    cuuint64_t dims[2] = {(cuuint64_t)inner, (cuuint64_t)outer};
    cuuint64_t strides[1] = {(cuuint64_t)inner * sizeof(double)};
    cuuint32_t box[2] = {(cuuint32_t)box_inner, (cuuint32_t)box_outer};
    cuuint32_t estr[2] = {1, 1};
    return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void*)base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
              swz128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// ---- ring-kernel launchers (dynamic shared memory above 48 KB needs the opt-in attribute once per kernel)
constexpr int YB_NST = 8, YB_RS = 16;     // 8 stages x 16 rows x 3 arrays x 256 B = 96 KiB per warp

// "has this kernel's shared-memory opt-in been done on the current device" (function attributes are per device)
struct DevOnce {
    std::atomic<unsigned long long> mask{0};
    static int dev() { int d = 0; cudaGetDevice(&d); return d & 63; }
    bool done() const { return (mask.load(std::memory_order_acquire) >> dev()) & 1ull; }
    void mark() { mask.fetch_or(1ull << dev(), std::memory_order_release); }   // setting the attribute twice is harmless
};

template <typename K>
cudaError_t opt_in_smem(K kernel, size_t bytes)
{
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

constexpr int YT_NST = 4, YT_RS = 16;     // TMA ring: 4 stages x 3 boxes of 16 x 32 doubles = 48 KiB per warp: all 512 CTAs resident (4 per SM)
constexpr int XT_NST = 3;                 // TMA ring: 3 stages x 16 KiB: all 512 CTAs resident (4 per SM)

// SM count of the CURRENT device (context-free entry points; a context keeps its own in c->num_sms)
int num_sms()
{
    static std::atomic<int> cache[64];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 148;
    int sms = cache[dev & 63].load(std::memory_order_relaxed);
    if (!sms) {
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) sms = 148;
        cache[dev & 63].store(sms, std::memory_order_relaxed);
    }
    return sms;
}

template <int NST>
cudaError_t launch_ybwd2_n(const CUtensorMap* m, dim3 g, int nx, int ny, int mid, const double* al, const double* be,
                           const double* zz, double* w, cudaStream_t st, Gate gate)
{
    constexpr size_t SM = (size_t)NST * 3 * YT_RS * 32 * 8 + 8 * NST + 1024;
    static DevOnce ready;
    if (!ready.done()) {
        cudaError_t e = opt_in_smem(ybwd2_tma_kernel<NST, YT_RS>, SM);
        if (e != cudaSuccess) return e;
        ready.mark();
    }
    ybwd2_tma_kernel<NST, YT_RS><<<g, 32, SM, st>>>(m[0], m[1], m[2], nx, ny, mid, al, be, zz, w, 1, gate);
    return cudaGetLastError();
}

template <int NST, bool UPDATE>
cudaError_t launch_xbwd2_n(const CUtensorMap* m, const CUtensorMap& uin, const CUtensorMap& uout, dim3 g, int nx, int ny,
                           int mid, const double* alT, const double* beT, const double* zzT, double* red, cudaStream_t st,
                           Gate gate = Gate{nullptr, 0.0})
{
    constexpr size_t SM = (size_t)NST * 4 * 16 * 32 * 8 + 8 * NST + 1024;
    static DevOnce ready;
    if (!ready.done()) {
        cudaError_t e = opt_in_smem(xbwd2_tma_kernel<NST, UPDATE>, SM);
        if (e != cudaSuccess) return e;
        ready.mark();
    }
    xbwd2_tma_kernel<NST, UPDATE><<<g, 32, SM, st>>>(m[0], m[1], m[2], uin, uout, nx, ny, mid, alT, beT, zzT, red, 1, gate);
    return cudaGetLastError();
}

// two-sided y back substitution (the y forward kernel is two-sided): TMA ring when the maps exist, else plain
cudaError_t launch_ybwd2(const CUtensorMap* m, bool tma, int nx, int ny, int mid, const double* al, const double* be,
                         const double* zz, double* w, cudaStream_t st, Gate gate = Gate{nullptr, 0.0})
{
    const dim3 g((nx + 31) / 32, 2);
    if (!tma) {
        ybwd2_plain_kernel<<<g, 32, 0, st>>>(nx, ny, mid, al, be, zz, w, gate);
        return cudaGetLastError();
    }
    return launch_ybwd2_n<YT_NST>(m, g, nx, ny, mid, al, be, zz, w, st, gate);
}

// two-sided x back substitution + update + residual
cudaError_t launch_xbwd2(const CUtensorMap* m, const CUtensorMap& uin, const CUtensorMap& uout, bool tma, int nx, int ny,
                         int mid, const double* alT, const double* beT, const double* zzT, const double* uk,
                         double* unew, double* red, cudaStream_t st, Gate gate, int sms)
{
    const dim3 g((ny + 31) / 32, 2);
    if (!tma) {
        xbwd2_plain_kernel<<<g, 32, 0, st>>>(nx, ny, mid, alT, beT, zzT, uk, unew, red, gate);
        return cudaGetLastError();
    }
    // ring depth: 3 stages when every CTA must fit at once (4 per SM); 6 when there are at most 2 CTAs per SM
    // (measured at 4096^2: 0.149 -> 0.138 ms; the y ring showed no gain from more stages)
    if ((int)(g.x * g.y) > 2 * sms)
        return launch_xbwd2_n<XT_NST, true>(m, uin, uout, g, nx, ny, mid, alT, beT, zzT, red, st, gate);
    return launch_xbwd2_n<2 * XT_NST, true>(m, uin, uout, g, nx, ny, mid, alT, beT, zzT, red, st, gate);
}

cudaError_t launch_ybwd(int nx, int ny, const double* al, const double* be, const double* zz, double* w,
                        cudaStream_t st)
{
    constexpr size_t SM = sizeof(double) * YB_NST * 3 * YB_RS * 32;
    static DevOnce ready;
    if (!ready.done()) {
        cudaError_t e = opt_in_smem(ybwd_ring_kernel<YB_NST, YB_RS, true>, SM);
        if (e == cudaSuccess) e = opt_in_smem(ybwd_ring_kernel<YB_NST, YB_RS, false>, SM);
        if (e != cudaSuccess) return e;
        ready.mark();
    }
    const int g = (nx + 31) / 32;
    if (nx % 2 == 0) ybwd_ring_kernel<YB_NST, YB_RS, true><<<g, 32, SM, st>>>(nx, ny, al, be, zz, w);
    else ybwd_ring_kernel<YB_NST, YB_RS, false><<<g, 32, SM, st>>>(nx, ny, al, be, zz, w);
    return cudaGetLastError();
}

constexpr int PC_NST = 3, PC_RS = 8;      // isolated solver, columns: 3 stages x 6 arrays x 8 rows x 256 B = 36 KiB per warp
constexpr int PR_NST = 2;                 // isolated solver, rows: 2 stages x 6 arrays x 4 KiB = 48 KiB per warp
#ifndef TF_YW_NP2
#define TF_YW_NP2 3
#endif
#ifndef TF_XW_NP2
#define TF_XW_NP2 7
#endif
#ifndef TF_YW_NP1
#define TF_YW_NP1 6
#endif
#ifndef TF_XW_NP1
#define TF_XW_NP1 7
#endif
#ifndef TF_NSUB1
#define TF_NSUB1 1
#endif
constexpr int YW_NP = 3, YW_RP = 8, YW_NSTG = 4;   // yfwd: consumer warp 0 + 3 producer warps, chunks of 8 rows, ring of 4 chunk slots (40 KiB)

#ifndef TF_XW_NP
#define TF_XW_NP 4
#endif
#ifndef TF_XW_NSTG
#define TF_XW_NSTG 3
#endif
constexpr int XW_NP = TF_XW_NP, XW_NSTG = TF_XW_NSTG;              // xfwd: per sub-problem 1 consumer + 4 producer warps, ring of 3 slots of 14 columns x 4 planes (38 KiB; 4 slots = two tiles were measured slower: 0.67 vs 0.53 ms -- the producers' unaligned row loads live on the L1 the carve-out leaves)

// forward kernels: NSUB sub-problems per CTA (4: two strips/blocks x two halves; 2: one x two halves)
template <int N, int M, bool FIRST, int NSUB>
cudaError_t launch_yfwd(tf_ctx* c, const CUtensorMap& mu, int tma, const Params& P, const Dir& DX, const Dir& DY,
                        const double* src, int grid, Gate gate)
{
    // producers per team: YW_NP with four teams per CTA; grids with two teams per CTA (sides <= ~4100) have SM capacity to spare
    constexpr int NP = NSUB == 2 ? TF_YW_NP2 : (NSUB == 1 ? TF_YW_NP1 : YW_NP);
    constexpr int NSTG = NP > YW_NSTG ? NP : YW_NSTG;                  // ring slots >= producers (see the kernel)
    constexpr size_t SM = NSUB * (size_t)NSTG * 5 * YW_RP * 32 * 8 + NSUB * NP * (size_t)(2 * YW_RP + 4) * 32 * 8 +
                          (2 * NSUB * NSTG + NSUB * NP) * 8;
    auto kern = yfwd_ws_kernel<N, M, FIRST, NP, YW_RP, NSTG, NSUB>;
    static DevOnce ready;
    if (!ready.done()) {
        cudaError_t e = opt_in_smem(kern, SM);
        if (e != cudaSuccess) return e;
        ready.mark();
    }
    kern<<<grid, 32 * fwd_warps(NSUB, NP), SM, c->stream>>>(mu, c->mBn, tma, P, DX, DY, c->mid_y, src, c->bn, c->al, c->be, c->zz, gate);
    return cudaGetLastError();
}

template <int N, int M, int NSUB>
cudaError_t launch_xfwd(tf_ctx* c, const Params& P, const Dir& DX, const double* src, int grid, Gate gate)
{
    constexpr size_t SM = NSUB * ((size_t)XW_NSTG * 4 * XW_CK * XW_LD * 8 + 16 * XW_NSTG);
    // two teams per CTA (sides <= ~4100, the paper's domain sizes): 7 producers of 4 rows each per team instead of 4 of 7
    // (measured at 4096^2: x forward 0.168 -> 0.153 ms; 6, 8, 9, 10 producers: 0.162 - 0.167; y forward with 4: slower)
    constexpr int NP = NSUB == 2 ? TF_XW_NP2 : (NSUB == 1 ? TF_XW_NP1 : XW_NP);
    auto kern = xfwd_ws_kernel<N, M, NP, XW_NSTG, NSUB>;
    static DevOnce ready;
    if (!ready.done()) {
        cudaError_t e = opt_in_smem(kern, SM);
        if (e != cudaSuccess) return e;
        ready.mark();
    }
    kern<<<grid, 32 * fwd_warps(NSUB, NP), SM, c->stream>>>(P, DX, c->mid_x, src, c->w, c->al, c->be, c->zz, gate);
    return cudaGetLastError();
}

// one pseudo-Newton iteration k: reads src (u^n if k == 0 else uk), writes uk, red[2k..2k+1].  gated: the four
// kernels return at once if iteration k-1's record says the step is already decided (speculative launch-ahead).
// which: 1 = the y-sweep (S1-S4: y forward + y backward -> w), 2 = the x-sweep (S5-S7 -> uk, red[2k]), 3 = both
// sdev != nullptr (on-device controller): s is read by the kernels from device memory, and iteration 0 is gated on gate0
template <int N, int M>
cudaError_t launch_iteration(tf_ctx* c, double s, int k, int slot, bool gated, int which = 3, const double* sdev = nullptr,
                             const double* gate0 = nullptr)
{
    const Params& P = c->P;
    Gate gate = (gated && k > 0) ? Gate{c->red + 2 * (k - 1), c->tol, sdev} : Gate{nullptr, 0.0, sdev};
    if (k == 0 && gate0) gate = Gate{gate0, c->tol, sdev};
    const Dir DX = make_dir(s, P.dx), DY = make_dir(s, P.dy);
    const double* src = (k == 0) ? c->u : c->uk;
    // one CTA = NSUB sub-problems: two strips x two halves, or one strip x two halves when that still leaves SMs idle
    const int nstrip = (P.nx + YW_VALID - 1) / YW_VALID;
    cudaEvent_t* ev = (c->profiling && slot >= 0) ? c->ev + 5 * slot : nullptr;
    if (ev) cudaEventRecord(ev[0], c->stream);
    if (which & 1) {
        const CUtensorMap& mu = c->mUy[src == c->ubuf[0] ? 0 : 1];
        const int tma = c->tma_yf ? 1 : 0;
        cudaError_t e;
        if (nstrip > c->num_sms)
            e = k == 0 ? launch_yfwd<N, M, true, 4>(c, mu, tma, P, DX, DY, src, (nstrip + 1) / 2, gate)
                       : launch_yfwd<N, M, false, 4>(c, mu, tma, P, DX, DY, src, (nstrip + 1) / 2, gate);
        else if (TF_NSUB1 && 2 * nstrip <= c->num_sms)      // one team per SM (sides <= ~2070): a whole SM per half line
            e = k == 0 ? launch_yfwd<N, M, true, 1>(c, mu, tma, P, DX, DY, src, 2 * nstrip, gate)
                       : launch_yfwd<N, M, false, 1>(c, mu, tma, P, DX, DY, src, 2 * nstrip, gate);
        else
            e = k == 0 ? launch_yfwd<N, M, true, 2>(c, mu, tma, P, DX, DY, src, nstrip, gate)
                       : launch_yfwd<N, M, false, 2>(c, mu, tma, P, DX, DY, src, nstrip, gate);
        if (e != cudaSuccess) return e;
    }
    if (ev) cudaEventRecord(ev[1], c->stream);
    cudaError_t le = cudaSuccess;
    if (which & 1) le = launch_ybwd2(c->mY, c->tma_y, P.nx, P.ny, c->mid_y, c->al, c->be, c->zz, c->w, c->stream, gate);
    if (le != cudaSuccess) return le;
    if (ev) cudaEventRecord(ev[2], c->stream);
    if (which & 2) {
        const int nblk = (P.ny + XW_R - 1) / XW_R;
        cudaError_t e = nblk > c->num_sms ? launch_xfwd<N, M, 4>(c, P, DX, src, (nblk + 1) / 2, gate)
                        : (TF_NSUB1 && 2 * nblk <= c->num_sms) ? launch_xfwd<N, M, 1>(c, P, DX, src, 2 * nblk, gate)
                                                               : launch_xfwd<N, M, 2>(c, P, DX, src, nblk, gate);
        if (e != cudaSuccess) return e;
    }
    if (ev) cudaEventRecord(ev[3], c->stream);
    if (which & 2)
        le = launch_xbwd2(c->mX, c->mU[src == c->ubuf[0] ? 0 : 1], c->mU[c->uk == c->ubuf[0] ? 0 : 1], c->tma_x, P.nx, P.ny,
                          c->mid_x, c->al, c->be, c->zz, src, c->uk, c->red + 2 * k, c->stream, gate, c->num_sms);
    if (le != cudaSuccess) return le;
    if (ev) cudaEventRecord(ev[4], c->stream);
    count_launch((which & 1 ? 2 : 0) + (which & 2 ? 2 : 0));
    return cudaGetLastError();
}

cudaError_t launch_iteration(tf_ctx* c, double s, int k, int slot, bool gated, int which = 3, const double* sdev = nullptr,
                             const double* gate0 = nullptr)
{
    if (c->model == TF_PI_NLC) return launch_iteration<MODEL_NLC, 0>(c, s, k, slot, gated, which, sdev, gate0);
    if (c->model == TF_PI_POLYMER) return launch_iteration<MODEL_POLYMER, 0>(c, s, k, slot, gated, which, sdev, gate0);
    if (!(c->P.n == 3 && c->P.m == 2)) return launch_iteration<0, 0>(c, s, k, slot, gated, which, sdev, gate0);
    return launch_iteration<3, 2>(c, s, k, slot, gated, which, sdev, gate0);
}

// after a stream sync: fold the event intervals of `niter` profiled iterations into the totals
void collect_profile(tf_ctx* c, int niter)
{
    if (!c->profiling) return;
    for (int it = 0; it < niter; ++it)
        for (int q = 0; q < TF_PROFILE_SLOTS; ++q) {
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, c->ev[5 * it + q], c->ev[5 * it + q + 1]) == cudaSuccess) {
                c->prof_ms[q] += ms;
                c->prof_n[q] += 1;
            }
        }
}

void clear_graphs(tf_ctx* c)
{
    for (auto& g : c->graphs) if (g.exec) cudaGraphExecDestroy(g.exec);
    c->graphs.clear();
    c->misses.clear();
}

// one launch-ahead batch: [clear the records] + iterations k0 .. k1-1 (gated) + the records of the batch to the host
cudaError_t enqueue_batch(tf_ctx* c, double s, int k0, int k1, int kmax)
{
    cudaError_t e = cudaSuccess;
    if (k0 == 0) e = cudaMemsetAsync(c->red, 0, sizeof(double) * 2 * (size_t)kmax, c->stream);
    for (int k = k0; k < k1 && e == cudaSuccess; ++k) e = launch_iteration(c, s, k, -1, true);
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(c->pinned_red + 2 * k0, c->red + 2 * k0, 2 * sizeof(double) * (size_t)(k1 - k0),
                            cudaMemcpyDeviceToHost, c->stream);
    return e;
}

// the same batch through a CUDA graph when its key {k0, count, buffer parity, s} has been seen before: captured on the
// second occurrence (the first ran plainly, so every kernel attribute is set), replayed from the third on
cudaError_t enqueue_batch_graphed(tf_ctx* c, double s, int k0, int k1, int kmax)
{
    const int n = k1 - k0, parity = ((c->u == c->ubuf[0]) ? 0 : 1) + ((c->w == c->w0) ? 0 : 2);
    if (!c->use_graphs) return enqueue_batch(c, s, k0, k1, kmax);
    for (auto& g : c->graphs)
        if (g.k0 == k0 && g.n == n && g.parity == parity && g.s == s) {
            g.stamp = ++c->gstamp;
            ++c->graph_replays;
            count_launch(4 * n);
            return cudaGraphLaunch(g.exec, c->stream);
        }
    size_t mi = 0;
    for (; mi < c->misses.size(); ++mi) {
        const auto& m = c->misses[mi];
        if (m.k0 == k0 && m.n == n && m.parity == parity && m.s == s) break;
    }
    if (mi == c->misses.size()) {                        // first occurrence: remember the key, launch plainly
        if (c->misses.size() >= 16) c->misses.erase(c->misses.begin());
        c->misses.push_back(tf_ctx::GraphEntry{k0, n, parity, s, nullptr, 0});
        return enqueue_batch(c, s, k0, k1, kmax);
    }
    c->misses.erase(c->misses.begin() + (long)mi);
    if (!c->gstream && cudaStreamCreateWithFlags(&c->gstream, cudaStreamNonBlocking) != cudaSuccess) {
        c->gstream = nullptr;
        c->use_graphs = false;
        return enqueue_batch(c, s, k0, k1, kmax);
    }
    cudaStream_t user = c->stream;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    cudaError_t e = cudaStreamBeginCapture(c->gstream, cudaStreamCaptureModeThreadLocal);
    if (e == cudaSuccess) {
        c->stream = c->gstream;
        e = enqueue_batch(c, s, k0, k1, kmax);
        c->stream = user;
        const cudaError_t e2 = cudaStreamEndCapture(c->gstream, &graph);
        if (e == cudaSuccess) e = e2;
    }
    if (e == cudaSuccess) e = cudaGraphInstantiate(&exec, graph, 0);
    if (graph) cudaGraphDestroy(graph);
    if (e != cudaSuccess) {                              // no graphs on this setup: fall back for good, run the batch plainly
        cudaGetLastError();
        c->use_graphs = false;
        return enqueue_batch(c, s, k0, k1, kmax);
    }
    if (c->graphs.size() >= 16) {                        // evict the least recently used
        size_t lru = 0;
        for (size_t i = 1; i < c->graphs.size(); ++i) if (c->graphs[i].stamp < c->graphs[lru].stamp) lru = i;
        cudaGraphExecDestroy(c->graphs[lru].exec);
        c->graphs.erase(c->graphs.begin() + (long)lru);
    }
    c->graphs.push_back(tf_ctx::GraphEntry{k0, n, parity, s, exec, ++c->gstamp});
    return cudaGraphLaunch(exec, c->stream);
}

tf_status create_common(tf_ctx** out, int nx, int ny, double dx, double dy, double kappa, double hstar,
                        int n, int m, tf_bc bc, void* dev_ws, size_t bytes, void* stream, bool own)
{
    if (!out) return fail(nullptr, TF_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (nx < 5 || ny < 5) return fail(nullptr, TF_ERR_INVALID_ARG, "nx, ny must be >= 5");
    if (((long long)nx + 1) * ((long long)ny + 1) >= (1LL << 31))
        return fail(nullptr, TF_ERR_INVALID_ARG, "(nx+1)*(ny+1) must be < 2^31 (32-bit element offsets)");
    if (!(dx > 0) || !(dy > 0) || !(kappa > 0) || !(hstar > 0) || !std::isfinite(dx) || !std::isfinite(dy) ||
        !std::isfinite(kappa) || !std::isfinite(hstar))
        return fail(nullptr, TF_ERR_INVALID_ARG, "dx, dy, kappa, hstar must be positive and finite");
    if (m < 1 || n <= m || n > 16) return fail(nullptr, TF_ERR_INVALID_ARG, "exponents must satisfy 16 >= n > m >= 1");
    if (bc != TF_BC_NOFLUX) return fail(nullptr, TF_ERR_UNSUPPORTED, "only TF_BC_NOFLUX (2.28) is defined");
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0)
        return fail(nullptr, TF_ERR_CUDA, std::string("no CUDA device: ") + cudaGetErrorString(e));
    tf_ctx* c = new (std::nothrow) tf_ctx();
    if (!c) return fail(nullptr, TF_ERR_ALLOC, "host allocation failed");
    Params& P = c->P;
    P.nx = nx; P.ny = ny; P.dx = dx; P.dy = dy;
    P.rdx2 = 1.0 / (dx * dx); P.rdy2 = 1.0 / (dy * dy);
    P.n = n; P.m = m;
    double hm = 1.0, hn = 1.0;
    for (int k = 0; k < m; ++k) hm *= hstar;
    for (int k = 0; k < n; ++k) hn *= hstar;
    P.cm = kappa * m * hm; P.cn = kappa * n * hn;
    c->kappa = kappa; c->hstar = hstar;
    c->model = TF_PI_POWER;
    for (double& v : P.mp) v = 0.0;
    c->tol = 1e-10; c->max_iter = 10; c->fixed_iters = 0;
    c->have_state = false; c->owns_ws = own;
    c->stream = (cudaStream_t)stream;
    const size_t need = tf_workspace_bytes(nx, ny);
    if (own) {
        void* p = nullptr;
        e = cudaMalloc(&p, need);
        if (e != cudaSuccess) { delete c; return fail(nullptr, TF_ERR_ALLOC, std::string("cudaMalloc: ") + cudaGetErrorString(e)); }
        c->ws = (char*)p;
    } else {
        if (!dev_ws || bytes < need || ((uintptr_t)dev_ws % ALIGN) != 0) {
            delete c;
            return fail(nullptr, TF_ERR_INVALID_ARG, "workspace NULL, misaligned (256 B) or smaller than tf_workspace_bytes");
        }
        c->ws = (char*)dev_ws;
    }
    const size_t fb = field_bytes(nx, ny);
    double** f[NFIELDS] = {&c->u, &c->uk, &c->bn, &c->w, &c->al, &c->be, &c->zz, &c->acc};
    for (int k = 0; k < NFIELDS; ++k) *f[k] = (double*)(c->ws + (size_t)k * fb);
    char* sc = c->ws + (size_t)NFIELDS * fb;
    c->red = (double*)sc;
    c->part = c->red + 2 * (MAX_ITERS + 1);
    c->scal = c->part + RED_BLOCKS;
    c->ctl = c->scal + 8;
    c->ctl_hist = c->ctl + CT_SIZE;
    e = cudaMallocHost((void**)&c->pinned, (4 + 2 * (size_t)MAX_ITERS) * sizeof(double));
    if (e != cudaSuccess) {
        if (own) cudaFree(c->ws);
        delete c;
        return fail(nullptr, TF_ERR_ALLOC, std::string("cudaMallocHost: ") + cudaGetErrorString(e));
    }
    c->pinned_red = c->pinned + 4;
    c->spec_batch = 2; c->last_iters = 1;
    c->max_rel_change = 0.0;
    c->max_trunc = 0.0; c->last_trunc = 0.0; c->dt_prev = 0.0; c->have_acc = false;
    c->ubuf[0] = c->u; c->ubuf[1] = c->uk;
    {
        int dev = 0, sms = 148;
        if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        c->num_sms = sms;
    }
    // split index of the two-sided sweeps: half the line, on a 16-row tile boundary when the line is long enough
    c->mid_y = ny >= 64 ? (ny / 2) / 16 * 16 : ny / 2;
    c->mid_x = nx >= 64 ? (nx / 2) / 16 * 16 : nx / 2;
    c->tma_y = (nx % 2 == 0) && nx >= 32 && ny >= YT_RS;
    c->tma_x = (nx % 2 == 0) && (ny % 2 == 0) && nx >= 64 && ny >= 32 && (c->mid_x % 16 == 0);
    if (c->tma_y) {
        const double* f3[3] = {c->al, c->be, c->zz};
        for (int k = 0; k < 3; ++k) c->tma_y = c->tma_y && make_map2d(&c->mY[k], f3[k], nx, ny, 32, YT_RS, false);
    }
    if (c->tma_x) {
        const double* f3[3] = {c->al, c->be, c->zz};
        for (int k = 0; k < 3; ++k) c->tma_x = c->tma_x && make_map2d(&c->mX[k], f3[k], ny, nx, 32, 16, false);
        for (int k = 0; k < 2; ++k) c->tma_x = c->tma_x && make_map2d(&c->mU[k], c->ubuf[k], nx, ny, 16, 32, true);
    }
    c->tma_yf = (nx % 2 == 0) && nx >= 32 && ny >= YW_RP + 4;
    if (c->tma_yf) {
        for (int k = 0; k < 2; ++k) c->tma_yf = c->tma_yf && make_map2d(&c->mUy[k], c->ubuf[k], nx, ny, 32, YW_RP + 4, false);
        c->tma_yf = c->tma_yf && make_map2d(&c->mBn, c->bn, nx, ny, 32, YW_RP, false);
    }
    if (!c->tma_yf) { memset(&c->mUy, 0, sizeof(c->mUy)); memset(&c->mBn, 0, sizeof(c->mBn)); }
    c->w0 = c->w;
    c->use_graphs = true; c->gstream = nullptr; c->gstamp = 0; c->graph_replays = 0;
    c->profiling = false;
    for (auto& ev : c->ev) ev = nullptr;
    for (int q = 0; q < TF_PROFILE_SLOTS; ++q) { c->prof_ms[q] = 0.0; c->prof_n[q] = 0; }
    *out = c;
    return TF_OK;
}

// sum + validity of a field on the context's stream; host gets (scale*sum, flag)
tf_status reduce_field(tf_ctx* c, const double* dev_field, double scale, double* sum, int* flag)
{
    const size_t n = (size_t)c->P.nx * c->P.ny;
    int* dflag = (int*)(c->scal + 1);
    TF_CUDA(c, cudaMemsetAsync(dflag, 0, sizeof(int), c->stream));
    sum_check_kernel<<<RED_BLOCKS, RED_THREADS, 0, c->stream>>>(n, dev_field, c->part, dflag);
    sum_final_kernel<<<1, 1024, 0, c->stream>>>(c->part, scale, c->scal);
    count_launch(2);
    TF_CUDA(c, cudaGetLastError());
    TF_CUDA(c, cudaMemcpyAsync(c->pinned, c->scal, 2 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    TF_CUDA(c, cudaStreamSynchronize(c->stream));
    if (sum) *sum = c->pinned[0];
    if (flag) std::memcpy(flag, &c->pinned[1], sizeof(int));
    return TF_OK;
}

// ---- partition variant of the isolated solver (tf_partition.cuh): interface pass, reduced system, chunk solves
constexpr int PART_MIN_LEN = 96;          // shortest admitted line length per chunk (chunks keep >= 81 rows)
constexpr int PART_MAX = 256;             // the reduced system is solved serially per line
constexpr int PI_NST = 4;                 // interface pass, columns: 4 stages x 12 KiB
constexpr int PJ_NST = 3;                 // interface pass, rows: 3 stages x 24 KiB

// phases: 1 = interface pass (-> iface, local chunks), 2 = reduced system over all Pg chunks (iface_all -> X),
// 4 = chunk solves (X -> x).  Single device: all three, Pg = P, p_off = 0, iface_all = iface.
tf_status penta_partition_phases(int phases, int nrow, int ncol, int dir, int P, int Pg, int p_off, const double* e,
                                 const double* c, const double* d, const double* a, const double* b, const double* rhs,
                                 double* x, double* al, double* be, double* zz, double* iface, const double* iface_all,
                                 double* rc, double* X, cudaStream_t st)
{
    const size_t nsys = (size_t)(dir ? ncol : nrow);
    const double* in6[6] = {e, c, d, a, b, rhs};
    bool ok = true;
    for (int k = 0; k < 6; ++k) ok = ok && ((uintptr_t)in6[k] % 16 == 0);
    if (phases & 4) ok = ok && ((uintptr_t)x % 16 == 0) && ((uintptr_t)al % 16 == 0);
    Maps6 M;
    CUtensorMap mw[3], mx;
    const double* w3[3] = {al, be, zz};
    if (dir == 1) {
        for (int k = 0; k < 6; ++k) ok = ok && make_map2d(&M.m[k], in6[k], ncol, nrow, 32, PC_RS, false);
        if (phases & 4) for (int k = 0; k < 3; ++k) ok = ok && make_map2d(&mw[k], w3[k], ncol, nrow, 32, YT_RS, false);
    } else {
        for (int k = 0; k < 6; ++k) ok = ok && make_map2d(&M.m[k], in6[k], ncol, nrow, 16, 32, true);
        if (phases & 4) {
            for (int k = 0; k < 3; ++k) ok = ok && make_map2d(&mw[k], w3[k], nrow, ncol, 32, 16, false);
            ok = ok && make_map2d(&mx, x, ncol, nrow, 16, 32, true);
        }
    }
    if (!ok) return fail(nullptr, TF_ERR_UNSUPPORTED, "partition variant: 16-byte aligned arrays and TMA tensor maps required");
    const dim3 g((unsigned)((nsys + 31) / 32), 2, (unsigned)P);
    int launches = 0;
    if (dir == 1) {
        constexpr size_t SMI = (size_t)PI_NST * 6 * PC_RS * 32 * 8 + 8 * PI_NST + 1024;
        constexpr size_t SMF = (size_t)PC_NST * 6 * PC_RS * 32 * 8 + 8 * PC_NST + 1024;
        constexpr size_t SMB = (size_t)YT_NST * 3 * YT_RS * 32 * 8 + 8 * YT_NST + 1024;
        static DevOnce ready;
        if (!ready.done()) {
            cudaError_t ee = opt_in_smem(penta_col_iface_kernel<PI_NST, PC_RS>, SMI);
            if (ee == cudaSuccess) ee = opt_in_smem(penta_col_fwd2_kernel<PC_NST, PC_RS>, SMF);
            if (ee == cudaSuccess) ee = opt_in_smem(ybwd2_tma_kernel<YT_NST, YT_RS, true>, SMB);
            if (ee != cudaSuccess) return cuda_fail(nullptr, ee, "cudaFuncSetAttribute");
            ready.mark();
        }
        if (phases & 1) { penta_col_iface_kernel<PI_NST, PC_RS><<<g, 32, SMI, st>>>(M, nrow, ncol, P, iface, Pg, p_off); ++launches; }
        if (phases & 2) { penta_reduced_kernel<<<(unsigned)((nsys + 31) / 32), 32, 0, st>>>((int)nsys, Pg, iface_all, rc, X); ++launches; }
        if (phases & 4) {
            penta_col_fwd2_kernel<PC_NST, PC_RS><<<g, 32, SMF, st>>>(M, nrow, ncol, chunk_mid(0, nrow), al, be, zz, P, X, Pg, p_off);
            ybwd2_tma_kernel<YT_NST, YT_RS, true><<<g, 32, SMB, st>>>(mw[0], mw[1], mw[2], ncol, nrow, 0, al, be, zz, x, P);
            launches += 2;
        }
    } else {
        constexpr size_t SMI = (size_t)PJ_NST * 6 * 32 * 16 * 8 + 8 * PJ_NST + 1024;
        constexpr size_t SMF = (size_t)PR_NST * 6 * 32 * 16 * 8 + 8 * PR_NST + 1024;
        constexpr size_t SMB = (size_t)XT_NST * 4 * 16 * 32 * 8 + 8 * XT_NST + 1024;
        static DevOnce ready;
        if (!ready.done()) {
            cudaError_t ee = opt_in_smem(penta_row_iface_kernel<PJ_NST>, SMI);
            if (ee == cudaSuccess) ee = opt_in_smem(penta_row_fwd2_kernel<PR_NST>, SMF);
            if (ee == cudaSuccess) ee = opt_in_smem(xbwd2_tma_kernel<XT_NST, false, true>, SMB);
            if (ee != cudaSuccess) return cuda_fail(nullptr, ee, "cudaFuncSetAttribute");
            ready.mark();
        }
        if (phases & 1) { penta_row_iface_kernel<PJ_NST><<<g, 32, SMI, st>>>(M, nrow, ncol, P, iface, Pg, p_off); ++launches; }
        if (phases & 2) { penta_reduced_kernel<<<(unsigned)((nsys + 31) / 32), 32, 0, st>>>((int)nsys, Pg, iface_all, rc, X); ++launches; }
        if (phases & 4) {
            penta_row_fwd2_kernel<PR_NST><<<g, 32, SMF, st>>>(M, nrow, ncol, chunk_mid(0, ncol), al, be, zz, P, X, Pg, p_off);
            xbwd2_tma_kernel<XT_NST, false, true><<<g, 32, SMB, st>>>(mw[0], mw[1], mw[2], mx, mx, ncol, nrow, 0, al, be, zz, nullptr, P);
            launches += 2;
        }
    }
    count_launch(launches);
    cudaError_t ee = cudaGetLastError();
    if (ee != cudaSuccess) return cuda_fail(nullptr, ee, "partition variant launch");
    return TF_OK;
}

tf_status penta_partition(int nrow, int ncol, int dir, int P, const double* e, const double* c, const double* d,
                          const double* a, const double* b, const double* rhs, double* x, char* ws, size_t fb,
                          cudaStream_t st)
{
    if ((uintptr_t)ws % 16) return fail(nullptr, TF_ERR_UNSUPPORTED, "partition variant: workspace must be 16-byte aligned");
    const size_t nsys = (size_t)(dir ? ncol : nrow);
    double* iface = (double*)(ws + 3 * fb);
    double* rc = iface + (size_t)P * 2 * IF_VALS * nsys;
    double* X = rc + (size_t)P * RC_VALS * nsys;
    return penta_partition_phases(7, nrow, ncol, dir, P, P, 0, e, c, d, a, b, rhs, x, (double*)ws, (double*)(ws + fb),
                                  (double*)(ws + 2 * fb), iface, iface, rc, X, st);
}

}  // namespace

extern "C" {

size_t tf_workspace_bytes(int nx, int ny)
{
    if (nx < 5 || ny < 5) return 0;
    return (size_t)NFIELDS * field_bytes(nx, ny) + scratch_bytes();
}

tf_status tf_create(tf_ctx** out, int nx, int ny, double dx, double dy, double kappa, double hstar, int n, int m,
                    tf_bc bc)
{
    return create_common(out, nx, ny, dx, dy, kappa, hstar, n, m, bc, nullptr, 0, nullptr, true);
}

tf_status tf_create_with_workspace(tf_ctx** out, int nx, int ny, double dx, double dy, double kappa, double hstar,
                                   int n, int m, tf_bc bc, void* dev_ws, size_t bytes, void* cuda_stream)
{
    return create_common(out, nx, ny, dx, dy, kappa, hstar, n, m, bc, dev_ws, bytes, cuda_stream, false);
}

void tf_destroy(tf_ctx* c)
{
    if (!c) return;
    cudaStreamSynchronize(c->stream);
    clear_graphs(c);
    if (c->gstream) cudaStreamDestroy(c->gstream);
    if (c->owns_ws) cudaFree(c->ws);
    for (auto& ev : c->ev) if (ev) cudaEventDestroy(ev);
    cudaFreeHost(c->pinned);
    delete c;
}

tf_status tf_set_newton(tf_ctx* c, double tol, int max_iter, int fixed_iters)
{
    if (!c) return TF_ERR_INVALID_ARG;
    if (!(tol >= 1e-14) || !std::isfinite(tol)) return fail(c, TF_ERR_INVALID_ARG, "tol must be >= 1e-14 (PAPER.md:338)");
    if (max_iter < 1 || max_iter > MAX_ITERS || fixed_iters < 0 || fixed_iters > MAX_ITERS)
        return fail(c, TF_ERR_INVALID_ARG, "max_iter in [1,4096], fixed_iters in [0,4096]");
    c->tol = tol; c->max_iter = max_iter; c->fixed_iters = fixed_iters;
    clear_graphs(c);
    return TF_OK;
}

tf_status tf_set_solution_criteria(tf_ctx* c, double max_rel_change)
{
    if (!c) return TF_ERR_INVALID_ARG;
    if (!(max_rel_change >= 0.0) || !std::isfinite(max_rel_change))
        return fail(c, TF_ERR_INVALID_ARG, "max_rel_change must be >= 0 and finite (0 = off)");
    c->max_rel_change = max_rel_change;
    return TF_OK;
}

tf_status tf_set_truncation_criterion(tf_ctx* c, double max_rel_truncation)
{
    if (!c) return TF_ERR_INVALID_ARG;
    if (!(max_rel_truncation >= 0.0) || !std::isfinite(max_rel_truncation))
        return fail(c, TF_ERR_INVALID_ARG, "max_rel_truncation must be >= 0 and finite (0 = off)");
    c->max_trunc = max_rel_truncation;
    return TF_OK;
}

tf_status tf_last_truncation_estimate(tf_ctx* c, double* estimate)
{
    if (!c || !estimate) return TF_ERR_INVALID_ARG;
    *estimate = c->last_trunc;
    return TF_OK;
}

tf_status tf_adaptive_run(tf_step_fn step, void* user, tf_adaptive* ctl, int n_accept, int max_attempts, double* t_advanced,
                          tf_step_record* hist, int hist_cap, int* nhist)
{
    if (!step || !ctl || n_accept < 0 || hist_cap < 0 || (hist_cap > 0 && !hist))
        return fail(nullptr, TF_ERR_INVALID_ARG, "tf_adaptive_run: NULL step/ctl or negative count");
    if (!(ctl->dt > 0) || !(ctl->shrink > 0 && ctl->shrink < 1) || !(ctl->grow >= 1) || ctl->grow_after < 1 ||
        !(ctl->dt_min > 0) || !(ctl->dt_max >= ctl->dt_min) || !std::isfinite(ctl->dt) || !std::isfinite(ctl->grow) ||
        !std::isfinite(ctl->dt_max))
        return fail(nullptr, TF_ERR_INVALID_ARG, "tf_adaptive_run: need dt > 0, 0 < shrink < 1, grow >= 1, grow_after >= 1, 0 < dt_min <= dt_max");
    if (max_attempts <= 0) max_attempts = 50 * std::max(n_accept, 1);
    double t = 0.0, dt = std::min(ctl->dt, ctl->dt_max);
    int accepted = 0, attempts = 0, streak = 0, nh = 0;
    tf_status out = TF_OK;
    while (accepted < n_accept) {
        if (attempts++ >= max_attempts) { out = TF_NOT_CONVERGED; fail(nullptr, out, "tf_adaptive_run: too many attempts"); break; }
        int it = 0;
        double res = 0.0;
        const int st = step(user, dt, &it, &res);
        if (nh < hist_cap) { hist[nh].dt = dt; hist[nh].status = st; hist[nh].newton_iters = it; hist[nh].residual = res; }
        ++nh;
        if (st < 0) { out = (tf_status)st; break; }                    // hard error of the step: stop, report it
        if (st == TF_OK) {
            ++accepted;
            t += dt;
            if (++streak >= ctl->grow_after) { dt = std::min(dt * ctl->grow, ctl->dt_max); streak = 0; }
        } else {                                                         // solution criteria not met: reduce the step
            streak = 0;
            dt *= ctl->shrink;
            if (dt < ctl->dt_min) { out = TF_NOT_CONVERGED; fail(nullptr, out, "tf_adaptive_run: dt fell below dt_min"); break; }
        }
    }
    ctl->dt = dt;
    if (t_advanced) *t_advanced = t;
    if (nhist) *nhist = nh;
    return out;
}

static int step_of_ctx(void* user, double dt, int* it, double* res) { return (int)tf_step((tf_ctx*)user, dt, it, res); }

tf_status tf_advance_adaptive(tf_ctx* c, tf_adaptive* ctl, int n_accept, int max_attempts, double* t_advanced,
                              tf_step_record* hist, int hist_cap, int* nhist)
{
    if (!c) return TF_ERR_INVALID_ARG;
    tf_status st = tf_adaptive_run(step_of_ctx, c, ctl, n_accept, max_attempts, t_advanced, hist, hist_cap, nhist);
    if (st != TF_OK && c->err.empty()) c->err = g_err;
    return st;
}

// Fig. 1 with every decision on the device (tf_control.cuh): attempts are enqueued a chunk at a time, each with max_iter
// gated iterations; the host reads the control block and the history once per chunk.
tf_status tf_advance_adaptive_device(tf_ctx* c, tf_adaptive* ctl, int n_accept, int max_attempts, double* t_advanced,
                                     tf_step_record* hist, int hist_cap, int* nhist)
{
    if (!c) return TF_ERR_INVALID_ARG;
    if (!ctl || n_accept < 0 || hist_cap < 0 || (hist_cap > 0 && !hist))
        return fail(c, TF_ERR_INVALID_ARG, "tf_advance_adaptive_device: NULL ctl or negative count");
    if (!(ctl->dt > 0) || !(ctl->shrink > 0 && ctl->shrink < 1) || !(ctl->grow >= 1) || ctl->grow_after < 1 ||
        !(ctl->dt_min > 0) || !(ctl->dt_max >= ctl->dt_min) || !std::isfinite(ctl->dt) || !std::isfinite(ctl->grow) ||
        !std::isfinite(ctl->dt_max))
        return fail(c, TF_ERR_INVALID_ARG, "tf_advance_adaptive_device: need dt > 0, 0 < shrink < 1, grow >= 1, grow_after >= 1, 0 < dt_min <= dt_max");
    if (!c->have_state) return fail(c, TF_ERR_STATE, "no state set");
    if (c->fixed_iters > 0)
        return fail(c, TF_ERR_UNSUPPORTED, "tf_advance_adaptive_device: fixed_iters needs the host controller");
    if (max_attempts <= 0) max_attempts = 50 * std::max(n_accept, 1);
    CtlParams P;
    P.shrink = ctl->shrink; P.grow = ctl->grow; P.dt_min = ctl->dt_min; P.dt_max = ctl->dt_max; P.tol = c->tol;
    P.grow_after = ctl->grow_after; P.n_accept = n_accept; P.max_attempts = max_attempts; P.kmax = c->max_iter;
    P.max_rel_change = c->max_rel_change; P.max_trunc = c->max_trunc;
    const bool crit_change = c->max_rel_change > 0.0, crit_trunc = c->max_trunc > 0.0;
    double init[CT_SIZE] = {0};
    init[CT_DT] = std::min(ctl->dt, ctl->dt_max);
    init[CT_HAVE_ACC] = (crit_trunc && c->have_acc) ? 1.0 : 0.0;         // the history of the host-side steps carries over
    init[CT_DT_PREV] = c->dt_prev;
    TF_CUDA(c, cudaMemcpyAsync(c->ctl, init, sizeof(init), cudaMemcpyHostToDevice, c->stream));
    TF_CUDA(c, cudaStreamSynchronize(c->stream));                        // `init` is on the stack
    const size_t n = (size_t)c->P.nx * c->P.ny;
    const unsigned gcopy = (unsigned)std::min<size_t>((n + 255) / 256, (size_t)c->num_sms * 16);
    std::vector<double> host(CT_SIZE + 4 * (size_t)CT_HIST_CAP);
    double* hc = host.data();
    int done = 0, attempts = 0, accepted = 0, drained = 0;
    // the device keeps the attempt records in a ring of CT_HIST_CAP entries; records [drained, upto) are copied out
    // before the next chunk (<= 16 attempts) could overwrite them, so a run may take any number of attempts
    auto drain = [&](int upto) -> cudaError_t {
        while (drained < upto) {
            const int at = drained % CT_HIST_CAP, cnt = std::min(upto - drained, CT_HIST_CAP - at);
            cudaError_t e = cudaMemcpyAsync(hc + CT_SIZE, c->ctl_hist + 4 * (size_t)at, sizeof(double) * 4 * (size_t)cnt,
                                            cudaMemcpyDeviceToHost, c->stream);
            if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
            if (e != cudaSuccess) return e;
            for (int a = drained; a < drained + cnt && a < hist_cap; ++a) {
                const double* r = hc + CT_SIZE + 4 * (size_t)(a - drained);
                hist[a].dt = r[0]; hist[a].status = (int)r[1]; hist[a].newton_iters = (int)r[2]; hist[a].residual = r[3];
            }
            drained += cnt;
        }
        return cudaSuccess;
    };
    while (!done) {
        const int chunk = std::max(1, std::min({n_accept - accepted + 1, 16, max_attempts - attempts + 1}));
        for (int a = 0; a < chunk; ++a) {
            ctl_begin_kernel<<<1, 256, 0, c->stream>>>(c->ctl, c->red, P);
            for (int k = 0; k < c->max_iter; ++k)
                TF_CUDA(c, launch_iteration(c, 1.0, k, -1, true, 3, c->ctl + CT_S, c->ctl + CT_GATE_RES));
            ctl_mid_kernel<<<1, 1, 0, c->stream>>>(c->ctl, c->red, P);
            if (crit_change)
                max_rel_change_ctl_kernel<<<RED_BLOCKS, RED_THREADS, 0, c->stream>>>(n, c->u, c->uk, c->ctl + CT_CONV, c->ctl + CT_CHANGE);
            if (crit_trunc)
                truncation_ctl_kernel<<<RED_BLOCKS, RED_THREADS, 0, c->stream>>>(n, c->u, c->uk, c->bn, c->acc, c->w, c->ctl + CT_CONV,
                                                                                  c->ctl + CT_DT, c->ctl + CT_DT_PREV,
                                                                                  c->ctl + CT_HAVE_ACC, c->ctl + CT_TRUNC);
            ctl_end_kernel<<<1, 1, 0, c->stream>>>(c->ctl, c->red, c->ctl_hist, P);
            ctl_commit_kernel<<<gcopy, 256, 0, c->stream>>>(n, c->uk, c->u, c->w, c->acc, c->ctl);
            count_launch(4 + (crit_change ? 1 : 0) + (crit_trunc ? 1 : 0));
        }
        TF_CUDA(c, cudaGetLastError());
        TF_CUDA(c, cudaMemcpyAsync(hc, c->ctl, sizeof(double) * CT_SIZE, cudaMemcpyDeviceToHost, c->stream));
        TF_CUDA(c, cudaStreamSynchronize(c->stream));
        attempts = (int)hc[CT_ATTEMPTS];
        accepted = (int)hc[CT_ACCEPTED];
        done = (int)hc[CT_DONE];
        if (!done && accepted >= n_accept) done = 1;
        if (!done && attempts >= max_attempts) done = 3;
        if (attempts - drained > CT_HIST_CAP - 32) TF_CUDA(c, drain(attempts));
    }
    TF_CUDA(c, drain(attempts));
    ctl->dt = hc[CT_DT];
    c->have_acc = crit_trunc && hc[CT_HAVE_ACC] != 0.0;                  // a_{n-1/2} of the last accepted step sits in c->acc
    if (c->have_acc) c->dt_prev = hc[CT_DT_PREV];
    if (crit_trunc) c->last_trunc = hc[CT_TRUNC];
    if (crit_change) c->last_change = hc[CT_CHANGE];
    if (t_advanced) *t_advanced = hc[CT_T];
    if (nhist) *nhist = attempts;
    if (done == 2) return fail(c, TF_NOT_CONVERGED, "tf_advance_adaptive_device: dt fell below dt_min");
    if (done == 3 && accepted < n_accept) return fail(c, TF_NOT_CONVERGED, "tf_advance_adaptive_device: too many attempts");
    return TF_OK;
}

tf_status tf_set_launch_ahead(tf_ctx* c, int batch)
{
    if (!c) return TF_ERR_INVALID_ARG;
    if (batch < 0 || batch > 64) return fail(c, TF_ERR_INVALID_ARG, "batch in [0,64]");
    c->spec_batch = batch;
    c->last_iters = 1;
    return TF_OK;
}

tf_status tf_set_cuda_graphs(tf_ctx* c, int on)
{
    if (!c) return TF_ERR_INVALID_ARG;
    c->use_graphs = on != 0;
    if (!on) clear_graphs(c);
    return TF_OK;
}

tf_status tf_graph_replays(tf_ctx* c, unsigned long long* replays)
{
    if (!c || !replays) return TF_ERR_INVALID_ARG;
    *replays = c->graph_replays;
    return TF_OK;
}

tf_status tf_set_pressure(tf_ctx* c, tf_pressure kind, const double* p, int np)
{
    if (!c) return TF_ERR_INVALID_ARG;
    double* mp = c->P.mp;
    const double PI = 3.14159265358979323846;
    clear_graphs(c);
    auto finite_pos = [](double v) { return v > 0 && std::isfinite(v); };
    if (kind == TF_PI_POWER) {
        c->model = TF_PI_POWER;
        return TF_OK;
    }
    if (!p) return fail(c, TF_ERR_INVALID_ARG, "params is NULL");
    for (int k = 0; k < np; ++k)
        if (!std::isfinite(p[k])) return fail(c, TF_ERR_INVALID_ARG, "non-finite parameter");
    if (kind == TF_PI_NLC) {
        if (np != 7) return fail(c, TF_ERR_INVALID_ARG, "NLC takes 7 parameters: cap0, cap1, K, b, N, beta, w");
        if (!finite_pos(p[0]) || !finite_pos(p[1]) || !finite_pos(p[3]) || !finite_pos(p[6]))
            return fail(c, TF_ERR_INVALID_ARG, "cap0, cap1, b, w must be positive");
        const double K = p[2], b = p[3];
        mp[0] = p[0]; mp[1] = p[1]; mp[2] = K * b * b * b; mp[3] = K * b * b; mp[4] = p[4]; mp[5] = p[5] * p[5];
        mp[6] = 1.0 / p[6]; mp[7] = 2.0 * b;
    } else if (kind == TF_PI_POLYMER) {
        if (np != 6) return fail(c, TF_ERR_INVALID_ARG, "polymer takes 6 parameters: cap0, cap1, C, A_SiOx, A_Si, d");
        if (!finite_pos(p[0]) || !finite_pos(p[1]) || !finite_pos(p[5]))
            return fail(c, TF_ERR_INVALID_ARG, "cap0, cap1, d must be positive");
        mp[0] = p[0]; mp[1] = p[1]; mp[2] = p[2]; mp[3] = p[3] / (2.0 * PI); mp[4] = (p[3] - p[4]) / (2.0 * PI); mp[5] = p[5];
    } else {
        return fail(c, TF_ERR_UNSUPPORTED, "unknown pressure kind");
    }
    c->model = kind;
    return TF_OK;
}

tf_status tf_set_state(tf_ctx* c, const double* h, int is_device_ptr)
{
    if (!c) return TF_ERR_INVALID_ARG;
    if (!h) return fail(c, TF_ERR_INVALID_ARG, "h is NULL");
    const size_t bytes = (size_t)c->P.nx * c->P.ny * sizeof(double);
    // stage in uk, validate on the device, then swap in (the previous state survives a rejection)
    TF_CUDA(c, cudaMemcpyAsync(c->uk, h, bytes, is_device_ptr ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice,
                               c->stream));
    int flag = 0;
    tf_status st = reduce_field(c, c->uk, 1.0, nullptr, &flag);
    if (st != TF_OK) return st;
    if (flag) return fail(c, TF_ERR_INVALID_ARG, "state has non-finite or non-positive values");
    std::swap(c->u, c->uk);
    c->have_state = true;
    c->have_acc = false;                             // a new film has no time-derivative history
    return TF_OK;
}

tf_status tf_get_state(tf_ctx* c, double* h_out, int is_device_ptr)
{
    if (!c) return TF_ERR_INVALID_ARG;
    if (!h_out) return fail(c, TF_ERR_INVALID_ARG, "h_out is NULL");
    if (!c->have_state) return fail(c, TF_ERR_STATE, "no state set");
    const size_t bytes = (size_t)c->P.nx * c->P.ny * sizeof(double);
    TF_CUDA(c, cudaMemcpyAsync(h_out, c->u, bytes, is_device_ptr ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost,
                               c->stream));
    TF_CUDA(c, cudaStreamSynchronize(c->stream));
    return TF_OK;
}

tf_status tf_step(tf_ctx* c, double dt, int* newton_iters, double* residual)
{
    if (!c) return TF_ERR_INVALID_ARG;
    if (!(dt > 0) || !std::isfinite(dt)) return fail(c, TF_ERR_INVALID_ARG, "dt must be positive and finite");
    if (!c->have_state) return fail(c, TF_ERR_STATE, "no state set");
    const double s = 0.5 * dt;
    const bool fixed = c->fixed_iters > 0;
    const int kmax = fixed ? c->fixed_iters : c->max_iter;
    int k = 0;
    double res = 0.0;
    tf_status status = TF_NOT_CONVERGED;
    if (fixed) {
        TF_CUDA(c, cudaMemsetAsync(c->red, 0, sizeof(double) * 2 * (size_t)kmax, c->stream));
        // parity mode: no host decision inside the step, one read at the end
        const bool prof = c->profiling && kmax <= 64;
        for (; k < kmax; ++k) TF_CUDA(c, launch_iteration(c, s, k, prof ? k : -1, false));
        TF_CUDA(c, cudaMemcpyAsync(c->pinned_red, c->red, 2 * sizeof(double) * (size_t)kmax, cudaMemcpyDeviceToHost,
                                   c->stream));
        TF_CUDA(c, cudaStreamSynchronize(c->stream));
        if (prof) collect_profile(c, kmax);
        res = c->pinned_red[2 * (kmax - 1)];
        status = TF_OK;
        // reading R18 also holds here: an iterate that was not finite or not positive must not become the state
        // (tf_set_state would refuse the same field, and the cell functions assume h > 0)
        for (int it = 0; it < kmax; ++it) {
            const double r = c->pinned_red[2 * it];
            if (c->pinned_red[2 * it + 1] != 0.0 || r != r) { status = TF_NOT_CONVERGED; res = r != r ? r : res; }
        }
    } else {
        // S8 with speculative launch-ahead: iterations are enqueued in batches -- the first as long as the previous
        // step's iteration count (the count changes slowly from step to step), then `spec_batch` at a time -- and the
        // host reads the residual records of a whole batch at once.  Iterations enqueued past the deciding one are
        // gated off on the device (gate_closed), so the result is exactly that of deciding after every iteration.
        const bool prof = c->profiling;
        int enq = 0, done = 0;
        int batch = c->spec_batch > 0 ? std::max(1, std::min(c->last_iters, prof ? 64 : kmax)) : 1;
        bool decided = false;
        while (!decided && done < kmax) {
            const int upto = std::min(kmax, enq + batch);
            if (prof) {
                if (enq == 0) TF_CUDA(c, cudaMemsetAsync(c->red, 0, sizeof(double) * 2 * (size_t)kmax, c->stream));
                for (; enq < upto; ++enq) TF_CUDA(c, launch_iteration(c, s, enq, enq - done, true));
                TF_CUDA(c, cudaMemcpyAsync(c->pinned_red + 2 * done, c->red + 2 * done, 2 * sizeof(double) * (size_t)(enq - done),
                                           cudaMemcpyDeviceToHost, c->stream));
            } else {
                TF_CUDA(c, enqueue_batch_graphed(c, s, enq, upto, kmax));
                enq = upto;
            }
            TF_CUDA(c, cudaStreamSynchronize(c->stream));
            const int first = done;
            for (; done < enq && !decided; ++done) {
                k = done + 1;
                res = c->pinned_red[2 * done];
                const bool bad = c->pinned_red[2 * done + 1] != 0.0;
                if (bad || res != res) decided = true;
                else if (res < c->tol) { status = TF_OK; decided = true; }
            }
            if (prof) collect_profile(c, done - first);
            batch = std::max(1, c->spec_batch);
        }
        if (status == TF_OK) c->last_iters = k;
    }
    if (status == TF_OK && c->max_rel_change > 0.0) {
        // "solution criteria" beyond convergence (PAPER.md:252 Note 2): here the largest relative change of h
        const size_t n = (size_t)c->P.nx * c->P.ny;
        TF_CUDA(c, cudaMemsetAsync(c->scal + 2, 0, sizeof(double), c->stream));
        max_rel_change_kernel<<<RED_BLOCKS, RED_THREADS, 0, c->stream>>>(n, c->u, c->uk, c->scal + 2);
        count_launch(1);
        TF_CUDA(c, cudaGetLastError());
        TF_CUDA(c, cudaMemcpyAsync(c->pinned, c->scal + 2, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        TF_CUDA(c, cudaStreamSynchronize(c->stream));
        c->last_change = c->pinned[0];
        if (!(c->last_change <= c->max_rel_change)) status = TF_REJECTED;
    }
    bool commit_acc = false;
    if (status == TF_OK && c->max_trunc > 0.0) {
        // second criterion (reading R25): estimated local truncation error of the trapezoidal rule, relative to h
        const size_t n = (size_t)c->P.nx * c->P.ny;
        const int have = c->have_acc ? 1 : 0;
        const double scale = have ? (dt * dt * dt / 12.0) / (0.5 * (dt + c->dt_prev)) : 0.0;
        TF_CUDA(c, cudaMemsetAsync(c->scal + 3, 0, sizeof(double), c->stream));
        truncation_kernel<<<RED_BLOCKS, RED_THREADS, 0, c->stream>>>(n, c->u, c->uk, c->bn, c->acc, c->w, 2.0 / (dt * dt), scale,
                                                                     have, c->scal + 3);
        count_launch(1);
        TF_CUDA(c, cudaGetLastError());
        TF_CUDA(c, cudaMemcpyAsync(c->pinned, c->scal + 3, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        TF_CUDA(c, cudaStreamSynchronize(c->stream));
        c->last_trunc = have ? c->pinned[0] : 0.0;
        if (have && !(c->last_trunc <= c->max_trunc)) status = TF_REJECTED;
        else commit_acc = true;
    }
    if (status == TF_OK && commit_acc) { std::swap(c->acc, c->w); c->dt_prev = dt; c->have_acc = true; }
    else if (status == TF_OK) c->have_acc = false;   // a step taken with the criterion off breaks the history
    if (status == TF_OK) std::swap(c->u, c->uk);     // pointer swap
    if (newton_iters) *newton_iters = k;
    if (residual) *residual = res;
    return status;
}

// ---- the rows of the path one by one (for callers that put an exchange step between the sweeps: section 8 of DESIGN.md)
tf_status tf_field(tf_ctx* c, int which, double** dev_ptr)
{
    if (!c || !dev_ptr) return TF_ERR_INVALID_ARG;
    double* f[5] = {c->u, c->uk, c->bn, c->w, c->red};
    if (which < 0 || which > 4) return fail(c, TF_ERR_INVALID_ARG, "tf_field: which in 0..4");
    *dev_ptr = f[which];
    return TF_OK;
}

tf_status tf_sweep(tf_ctx* c, double dt, int k, int which)
{
    if (!c) return TF_ERR_INVALID_ARG;
    if (!(dt > 0) || !std::isfinite(dt)) return fail(c, TF_ERR_INVALID_ARG, "dt must be positive and finite");
    if (k < 0 || k >= MAX_ITERS || (which & 3) == 0 || which > 7)
        return fail(c, TF_ERR_INVALID_ARG, "tf_sweep: k in [0,4096), which = 1, 2 or 3, + 4 for the gate");
    if (!c->have_state) return fail(c, TF_ERR_STATE, "no state set");
    if (which & 2) TF_CUDA(c, cudaMemsetAsync(c->red + 2 * k, 0, 2 * sizeof(double), c->stream));
    TF_CUDA(c, launch_iteration(c, 0.5 * dt, k, -1, (which & 4) != 0, which & 3));
    return TF_OK;
}

tf_status tf_residual(tf_ctx* c, int k, double* res, int* bad)
{
    if (!c || k < 0 || k >= MAX_ITERS) return TF_ERR_INVALID_ARG;
    TF_CUDA(c, cudaMemcpyAsync(c->pinned, c->red + 2 * k, 2 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    TF_CUDA(c, cudaStreamSynchronize(c->stream));
    if (res) *res = c->pinned[0];
    if (bad) *bad = (c->pinned[1] != 0.0 || c->pinned[0] != c->pinned[0]) ? 1 : 0;
    return TF_OK;
}

tf_status tf_accept(tf_ctx* c)
{
    if (!c) return TF_ERR_INVALID_ARG;
    if (!c->have_state) return fail(c, TF_ERR_STATE, "no state set");
    std::swap(c->u, c->uk);
    c->have_acc = false;
    return TF_OK;
}

// ---- exchange steps of the distributed time step: block pack / unpack and the record to be max-reduced
static tf_status blocks_common(const tf_rect* rects, int nrect, int ld, Rects* R, dim3* grid)
{
    if (!rects || nrect < 1 || nrect > BLK_MAX || ld < 1)
        return fail(nullptr, TF_ERR_INVALID_ARG, "tf_blocks_*: 1 <= nrect <= 64 blocks, ld >= 1");
    int maxr = 0, maxc = 0;
    for (int k = 0; k < nrect; ++k) {
        const tf_rect& q = rects[k];
        if (q.row0 < 0 || q.col0 < 0 || q.nrows < 0 || q.ncols < 0 || q.offset < 0 || q.col0 + q.ncols > ld)
            return fail(nullptr, TF_ERR_INVALID_ARG, "tf_blocks_*: block outside the field or negative offset");
        R->r[k] = Rect{q.row0, q.nrows, q.col0, q.ncols, q.offset};
        maxr = std::max(maxr, q.nrows);
        maxc = std::max(maxc, q.ncols);
    }
    R->n = nrect;
    const unsigned gy = (unsigned)((maxr + BLK_ROWS - 1) / BLK_ROWS);
    if (gy > 65535u) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_blocks_*: more than 524280 rows in a block");
    *grid = dim3((unsigned)std::max(1, std::min((maxc + BLK_THREADS - 1) / BLK_THREADS, 64)), std::max(gy, 1u), (unsigned)nrect);
    return TF_OK;
}

tf_status tf_blocks_gather(const double* field, int ld, const tf_rect* rects, int nrect, double* buf, void* cuda_stream)
{
    if (!field || !buf) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_blocks_gather: NULL pointer");
    Rects R;
    dim3 g;
    tf_status st = blocks_common(rects, nrect, ld, &R, &g);
    if (st != TF_OK) return st;
    blocks_gather_kernel<<<g, BLK_THREADS, 0, (cudaStream_t)cuda_stream>>>(field, ld, R, buf);
    count_launch(1);
    TF_CUDA(nullptr, cudaGetLastError());
    return TF_OK;
}

tf_status tf_blocks_scatter(const double* buf, const tf_rect* rects, int nrect, double* field, int ld, int reflect_left,
                            int reflect_right_at, void* cuda_stream)
{
    if (!field || !buf) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_blocks_scatter: NULL pointer");
    if (reflect_right_at >= 0 && (reflect_right_at < 2 || reflect_right_at + 2 > ld))
        return fail(nullptr, TF_ERR_INVALID_ARG, "tf_blocks_scatter: right ghost columns outside the field");
    if (reflect_left && ld < 4) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_blocks_scatter: field narrower than its ghosts");
    Rects R;
    dim3 g;
    tf_status st = blocks_common(rects, nrect, ld, &R, &g);
    if (st != TF_OK) return st;
    blocks_scatter_kernel<<<g, BLK_THREADS, 0, (cudaStream_t)cuda_stream>>>(buf, R, field, ld, reflect_left ? 1 : 0,
                                                                             reflect_right_at);
    count_launch(1);
    TF_CUDA(nullptr, cudaGetLastError());
    return TF_OK;
}

tf_status tf_block_copy(const double* src, int sld, int srow0, int scol0, double* dst, int dld, int drow0, int dcol0,
                        int nrows, int ncols, int reflect_left, int reflect_right_at, void* cuda_stream)
{
    if (!src || !dst) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_block_copy: NULL pointer");
    if (nrows < 0 || ncols < 0 || srow0 < 0 || scol0 < 0 || drow0 < 0 || dcol0 < 0 || scol0 + ncols > sld || dcol0 + ncols > dld)
        return fail(nullptr, TF_ERR_INVALID_ARG, "tf_block_copy: block outside a field");
    if (reflect_right_at >= 0 && (reflect_right_at < 2 || reflect_right_at + 2 > dld))
        return fail(nullptr, TF_ERR_INVALID_ARG, "tf_block_copy: right ghost columns outside the field");
    if (nrows == 0 || ncols == 0) return TF_OK;
    const unsigned gy = (unsigned)((nrows + BLK_ROWS - 1) / BLK_ROWS);
    if (gy > 65535u) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_block_copy: more than 524280 rows");
    const dim3 g((unsigned)std::max(1, std::min((ncols + BLK_THREADS - 1) / BLK_THREADS, 64)), gy);
    block_copy_kernel<<<g, BLK_THREADS, 0, (cudaStream_t)cuda_stream>>>(src, sld, srow0, scol0, dst, dld, drow0, dcol0, nrows,
                                                                         ncols, reflect_left ? 1 : 0, reflect_right_at);
    count_launch(1);
    TF_CUDA(nullptr, cudaGetLastError());
    return TF_OK;
}

tf_status tf_record_sanitize(tf_ctx* c, int k)
{
    if (!c || k < 0 || k >= MAX_ITERS) return TF_ERR_INVALID_ARG;
    record_sanitize_kernel<<<1, 1, 0, c->stream>>>(c->red + 2 * k);
    count_launch(1);
    TF_CUDA(c, cudaGetLastError());
    return TF_OK;
}

tf_status tf_mass(tf_ctx* c, double* mass)
{
    if (!c) return TF_ERR_INVALID_ARG;
    if (!mass) return fail(c, TF_ERR_INVALID_ARG, "mass is NULL");
    if (!c->have_state) return fail(c, TF_ERR_STATE, "no state set");
    return reduce_field(c, c->u, c->P.dx * c->P.dy, mass, nullptr);
}

tf_status tf_set_profiling(tf_ctx* c, int on)
{
    if (!c) return TF_ERR_INVALID_ARG;
    if (on)
        for (auto& ev : c->ev)
            if (!ev) TF_CUDA(c, cudaEventCreate(&ev));
    c->profiling = on != 0;
    for (int q = 0; q < TF_PROFILE_SLOTS; ++q) { c->prof_ms[q] = 0.0; c->prof_n[q] = 0; }
    return TF_OK;
}

tf_status tf_get_profile(tf_ctx* c, double ms[TF_PROFILE_SLOTS], unsigned long long launches[TF_PROFILE_SLOTS])
{
    if (!c) return TF_ERR_INVALID_ARG;
    for (int q = 0; q < TF_PROFILE_SLOTS; ++q) {
        if (ms) ms[q] = c->prof_ms[q];
        if (launches) launches[q] = c->prof_n[q];
    }
    return TF_OK;
}

size_t tf_penta_workspace_bytes(int nrow, int ncol)
{
    if (nrow < 1 || ncol < 1) return 0;
    return 3 * align_up((size_t)nrow * ncol * sizeof(double));
}

// ---- slabs of a line on different devices: the partition variant with an exchange step
static bool slab_shape_ok(int nrow, int ncol, int dir, int nparts)
{
    if (nrow < 1 || ncol < 1 || (dir != 0 && dir != 1) || nparts < 1 || nparts > PART_MAX) return false;
    const int len = dir ? nrow : ncol, nsys = dir ? ncol : nrow;
    return len / nparts >= PART_MIN_LEN && nsys >= 32 && nrow % 2 == 0 && ncol % 2 == 0;
}

size_t tf_penta_slab_interface_doubles(int nrow, int ncol, int dir, int nparts)
{
    if (!slab_shape_ok(nrow, ncol, dir, nparts)) return 0;
    return (size_t)nparts * 2 * IF_VALS * (size_t)(dir ? ncol : nrow);
}

size_t tf_penta_slab_workspace_bytes(int nrow, int ncol, int dir, int nparts, int nslabs)
{
    if (!slab_shape_ok(nrow, ncol, dir, nparts) || nslabs < 1 || (long long)nslabs * nparts > 65535) return 0;
    const size_t nsys = (size_t)(dir ? ncol : nrow);
    return tf_penta_workspace_bytes(nrow, ncol) + align_up((size_t)nslabs * nparts * (RC_VALS + 4) * nsys * sizeof(double));
}

tf_status tf_penta_slab_interface(int nrow, int ncol, int dir, int nparts, int slab, int nslabs, const double* e,
                                  const double* c, const double* d, const double* a, const double* b, const double* rhs,
                                  double* iface_local, void* cuda_stream)
{
    if (!slab_shape_ok(nrow, ncol, dir, nparts) || nslabs < 1 || slab < 0 || slab >= nslabs)
        return fail(nullptr, TF_ERR_INVALID_ARG, "tf_penta_slab_interface: bad shape, chunk count or slab index");
    if (!e || !c || !d || !a || !b || !rhs || !iface_local) return fail(nullptr, TF_ERR_INVALID_ARG, "NULL pointer");
    return penta_partition_phases(1, nrow, ncol, dir, nparts, nslabs * nparts, slab * nparts, e, c, d, a, b, rhs, nullptr,
                                  nullptr, nullptr, nullptr, iface_local, nullptr, nullptr, nullptr, (cudaStream_t)cuda_stream);
}

tf_status tf_penta_slab_solve(int nrow, int ncol, int dir, int nparts, int slab, int nslabs, const double* e,
                              const double* c, const double* d, const double* a, const double* b, const double* rhs,
                              const double* iface_all, double* x, void* dev_ws, void* cuda_stream)
{
    if (!slab_shape_ok(nrow, ncol, dir, nparts) || nslabs < 1 || slab < 0 || slab >= nslabs)
        return fail(nullptr, TF_ERR_INVALID_ARG, "tf_penta_slab_solve: bad shape, chunk count or slab index");
    if (!e || !c || !d || !a || !b || !rhs || !iface_all || !x || !dev_ws) return fail(nullptr, TF_ERR_INVALID_ARG, "NULL pointer");
    if ((uintptr_t)dev_ws % 16) return fail(nullptr, TF_ERR_UNSUPPORTED, "workspace must be 16-byte aligned");
    const size_t fb = align_up((size_t)nrow * ncol * sizeof(double));
    const size_t nsys = (size_t)(dir ? ncol : nrow);
    const int Pg = nslabs * nparts;
    char* ws = (char*)dev_ws;
    double* rc = (double*)(ws + 3 * fb);
    double* X = rc + (size_t)Pg * RC_VALS * nsys;
    return penta_partition_phases(2 | 4, nrow, ncol, dir, nparts, Pg, slab * nparts, e, c, d, a, b, rhs, x, (double*)ws,
                                  (double*)(ws + fb), (double*)(ws + 2 * fb), nullptr, iface_all, rc, X, (cudaStream_t)cuda_stream);
}

int tf_penta_partition_chunks(int nrow, int ncol, int dir, int nparts)
{
    if (nrow < 1 || ncol < 1 || (dir != 0 && dir != 1) || nparts < 0) return 0;
    const int len = dir ? nrow : ncol, nsys = dir ? ncol : nrow;
    const int pmax = std::min(len / PART_MIN_LEN, PART_MAX);          // every chunk keeps >= PART_MIN_LEN - 16 rows
    if (pmax < 2 || nsys < 32 || nrow % 2 || ncol % 2) return 1;      // the chunked kernels are the TMA ones only
    if (nparts > 0) return std::min(nparts, pmax);
    // auto: enough marching warps (2 per chunk and strip of 32 lines) for ~4 per SM, chunks not shorter than 256 rows
    const int strips = (nsys + 31) / 32;
    const int want = (2 * num_sms() + strips - 1) / strips;
    if (want < 6) return 1;               // >= ~1600 lines: thread-per-line is already HBM-bound (measured crossover ~2048)
    return std::max(1, std::min(std::min(want, len / 256), pmax));
}

size_t tf_penta_workspace_bytes_ex(int nrow, int ncol, int dir, int variant, int nparts)
{
    const size_t lu = tf_penta_workspace_bytes(nrow, ncol);
    if (lu == 0 || variant != TF_PENTA_PARTITION) return lu;
    const int P = tf_penta_partition_chunks(nrow, ncol, dir, nparts);
    const size_t nsys = (size_t)(dir ? ncol : nrow);
    return lu + align_up((size_t)P * (2 * IF_VALS + RC_VALS + 4) * nsys * sizeof(double));
}

tf_status tf_penta_solve(int nrow, int ncol, int dir, const double* e, const double* c, const double* d,
                         const double* a, const double* b, const double* rhs, double* x, void* dev_ws,
                         void* cuda_stream)
{
    return tf_penta_solve_ex(nrow, ncol, dir, TF_PENTA_LU, 0, e, c, d, a, b, rhs, x, dev_ws, cuda_stream);
}

tf_status tf_penta_solve_ex(int nrow, int ncol, int dir, int variant, int nparts, const double* e, const double* c,
                            const double* d, const double* a, const double* b, const double* rhs, double* x,
                            void* dev_ws, void* cuda_stream)
{
    if (nrow < 1 || ncol < 1 || (dir != 0 && dir != 1)) return fail(nullptr, TF_ERR_INVALID_ARG, "bad shape or dir");
    if ((dir ? nrow : ncol) < 3) return fail(nullptr, TF_ERR_INVALID_ARG, "system length must be >= 3");
    if (!e || !c || !d || !a || !b || !rhs || !x || !dev_ws) return fail(nullptr, TF_ERR_INVALID_ARG, "NULL pointer");
    if (variant != TF_PENTA_LU && variant != TF_PENTA_PARTITION && variant != TF_PENTA_PCR)
        return fail(nullptr, TF_ERR_UNSUPPORTED, "unknown variant");
    if (nparts < 0) return fail(nullptr, TF_ERR_INVALID_ARG, "nparts < 0");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (variant == TF_PENTA_PCR) {
        const double* in6[6] = {e, c, d, a, b, rhs};
        bool ok = dir == 0 && ncol % 2 == 0 && ncol >= 64 && ncol <= 2048 && ((uintptr_t)x % 16 == 0);
        for (int k = 0; k < 6; ++k) ok = ok && ((uintptr_t)in6[k] % 16 == 0);
        if (!ok) return fail(nullptr, TF_ERR_UNSUPPORTED, "TF_PENTA_PCR: dir = 0, even 64 <= ncol <= 2048, 16-byte aligned arrays");
        const int nb = ncol / 2;
        const size_t sm = (size_t)PCR_VALS * nb * sizeof(double);
        static DevOnce ready;
        if (!ready.done()) {
            cudaError_t ee = opt_in_smem(penta_row_pcr_kernel<512>, (size_t)PCR_VALS * 512 * sizeof(double));
            if (ee == cudaSuccess) ee = opt_in_smem(penta_row_pcr_kernel<1024>, (size_t)PCR_VALS * 1024 * sizeof(double));
            if (ee != cudaSuccess) return cuda_fail(nullptr, ee, "cudaFuncSetAttribute");
            ready.mark();
        }
        const unsigned nthr = (unsigned)((nb + 31) / 32 * 32);
        if (nb <= 512) penta_row_pcr_kernel<512><<<(unsigned)nrow, nthr, sm, st>>>(ncol, e, c, d, a, b, rhs, x);
        else penta_row_pcr_kernel<1024><<<(unsigned)nrow, nthr, sm, st>>>(ncol, e, c, d, a, b, rhs, x);
        count_launch(1);
        cudaError_t le = cudaGetLastError();
        if (le != cudaSuccess) return cuda_fail(nullptr, le, "penta_row_pcr launch");
        return TF_OK;
    }
    const size_t fb = align_up((size_t)nrow * ncol * sizeof(double));
    if (variant == TF_PENTA_PARTITION) {
        const int P = tf_penta_partition_chunks(nrow, ncol, dir, nparts);
        if (P > 1) return penta_partition(nrow, ncol, dir, P, e, c, d, a, b, rhs, x, (char*)dev_ws, fb, st);
    }
    double* al = (double*)dev_ws;
    double* be = (double*)((char*)dev_ws + fb);
    double* zz = (double*)((char*)dev_ws + 2 * fb);
    const double* in6[6] = {e, c, d, a, b, rhs};
    bool aligned = ((uintptr_t)dev_ws % 16 == 0) && ((uintptr_t)x % 16 == 0);
    for (int k = 0; k < 6; ++k) aligned = aligned && ((uintptr_t)in6[k] % 16 == 0);
    if (dir == 1) {
        // systems along columns: nsys = ncol, length = nrow
        const int mid = (nrow / 2) / 16 * 16;
        bool fast = aligned && (ncol % 2 == 0) && ncol >= 32 && nrow >= 64;
        Maps6 M;
        CUtensorMap mw[3];
        if (fast) {
            for (int k = 0; k < 6; ++k) fast = fast && make_map2d(&M.m[k], in6[k], ncol, nrow, 32, PC_RS, false);
            const double* w3[3] = {al, be, zz};
            for (int k = 0; k < 3; ++k) fast = fast && make_map2d(&mw[k], w3[k], ncol, nrow, 32, YT_RS, false);
        }
        if (fast) {
            constexpr size_t SM = (size_t)PC_NST * 6 * PC_RS * 32 * 8 + 8 * PC_NST + 1024;
            static DevOnce ready;
            if (!ready.done()) {
                cudaError_t ee = opt_in_smem(penta_col_fwd2_kernel<PC_NST, PC_RS>, SM);
                if (ee != cudaSuccess) return cuda_fail(nullptr, ee, "cudaFuncSetAttribute");
                ready.mark();
            }
            penta_col_fwd2_kernel<PC_NST, PC_RS><<<dim3((ncol + 31) / 32, 2), 32, SM, st>>>(M, nrow, ncol, mid, al, be, zz, 1, nullptr);
            cudaError_t le = launch_ybwd2(mw, true, ncol, nrow, mid, al, be, zz, x, st);
            if (le != cudaSuccess) return cuda_fail(nullptr, le, "ybwd2 launch");
        } else {
            const int g = (ncol + 31) / 32;
            penta_col_fwd_kernel<<<g, 32, 0, st>>>(nrow, ncol, e, c, d, a, b, rhs, al, be, zz);
            cudaError_t le = launch_ybwd(ncol, nrow, al, be, zz, x, st);
            if (le != cudaSuccess) return cuda_fail(nullptr, le, "ybwd launch");
        }
    } else {
        // systems along rows: nsys = nrow, length = ncol; coefficients transposed [col][row]
        const int mid = (ncol / 2) / 16 * 16;
        bool fast = aligned && (ncol % 2 == 0) && (nrow % 2 == 0) && ncol >= 64 && nrow >= 32;
        Maps6 M;
        CUtensorMap mw[3], mx;
        if (fast) {
            for (int k = 0; k < 6; ++k) fast = fast && make_map2d(&M.m[k], in6[k], ncol, nrow, 16, 32, true);
            const double* w3[3] = {al, be, zz};
            for (int k = 0; k < 3; ++k) fast = fast && make_map2d(&mw[k], w3[k], nrow, ncol, 32, 16, false);
            fast = fast && make_map2d(&mx, x, ncol, nrow, 16, 32, true);
        }
        if (fast) {
            constexpr size_t SMF = (size_t)PR_NST * 6 * 32 * 16 * 8 + 8 * PR_NST + 1024;
            static DevOnce ready;
            if (!ready.done()) {
                cudaError_t ee = opt_in_smem(penta_row_fwd2_kernel<PR_NST>, SMF);
                if (ee != cudaSuccess) return cuda_fail(nullptr, ee, "cudaFuncSetAttribute");
                ready.mark();
            }
            const dim3 g((nrow + 31) / 32, 2);
            penta_row_fwd2_kernel<PR_NST><<<g, 32, SMF, st>>>(M, nrow, ncol, mid, al, be, zz, 1, nullptr);
            cudaError_t le = launch_xbwd2_n<XT_NST, false>(mw, mx, mx, g, ncol, nrow, mid, al, be, zz, nullptr, st);
            if (le != cudaSuccess) return cuda_fail(nullptr, le, "xbwd2 launch");
        } else {
            const int g = (nrow + XT - 1) / XT;
            const size_t sm = sizeof(double) * PT_ARR * XT * XTP;
            static DevOnce attr_set;
            if (!attr_set.done()) {
                cudaError_t ee = cudaFuncSetAttribute(penta_row_fwd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
                if (ee != cudaSuccess) return cuda_fail(nullptr, ee, "cudaFuncSetAttribute");
                attr_set.mark();
            }
            penta_row_fwd_kernel<<<g, 32, sm, st>>>(nrow, ncol, e, c, d, a, b, rhs, al, be, zz);
            penta_row_bwd_kernel<<<g, 32, 0, st>>>(nrow, ncol, al, be, zz, x);
        }
    }
    count_launch(2);
    cudaError_t ee = cudaGetLastError();
    if (ee != cudaSuccess) return cuda_fail(nullptr, ee, "tf_penta_solve launch");
    return TF_OK;
}

// ---- tf_penta_solve_static: the isolated solve for callers that cannot allocate device memory (include/tf.h).
// The scratch (alpha, beta, z) is part of this library's device image.  Every device that loads the image keeps the
// array until the process ends, and every call on a device shares it.
static __device__ __align__(256) double g_penta_static_scratch[3 * (size_t)TF_PENTA_STATIC_MAX_ELEMS];

namespace {

// In host code `g_penta_static_scratch` is only a handle for the runtime, NOT a device address: a kernel given
// `&g_penta_static_scratch[0]` from the host would fault (or, on a system where the GPU can reach host memory, quietly
// work on the wrong bytes).  The device address is asked for once per device, with that device current, and kept.
std::mutex g_penta_static_mu;
double* g_penta_static_addr[64];      // by device ordinal; written under the mutex

tf_status penta_static_scratch(double** out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "tf_penta_solve_static: cudaGetDevice");
    if (dev < 0 || dev >= 64) return fail(nullptr, TF_ERR_UNSUPPORTED, "tf_penta_solve_static: device ordinal above 63");
    std::lock_guard<std::mutex> lock(g_penta_static_mu);
    if (!g_penta_static_addr[dev]) {
        double* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_penta_static_scratch);
        if (e != cudaSuccess) return cuda_fail(nullptr, e, "tf_penta_solve_static: cudaGetSymbolAddress");
        if (!p || (uintptr_t)p % ALIGN) return fail(nullptr, TF_ERR_CUDA, "tf_penta_solve_static: scratch address is null or misaligned");
        g_penta_static_addr[dev] = p;
    }
    *out = g_penta_static_addr[dev];
    return TF_OK;
}

}  // namespace

size_t tf_penta_static_max_elems(void) { return (size_t)TF_PENTA_STATIC_MAX_ELEMS; }

tf_status tf_penta_solve_static(int nrow, int ncol, int dir, const double* e, const double* c, const double* d,
                                const double* a, const double* b, const double* rhs, double* x, void* cuda_stream)
{
    // all argument checks come before the first CUDA call: a refused call touches no device
    if (nrow < 1 || ncol < 1 || (dir != 0 && dir != 1)) return fail(nullptr, TF_ERR_INVALID_ARG, "bad shape or dir");
    if ((unsigned long long)nrow * (unsigned long long)ncol > (unsigned long long)TF_PENTA_STATIC_MAX_ELEMS)
        return fail(nullptr, TF_ERR_INVALID_ARG,
                    "tf_penta_solve_static: nrow * ncol = " + std::to_string((unsigned long long)nrow * (unsigned long long)ncol) +
                        " exceeds the built-in scratch of TF_PENTA_STATIC_MAX_ELEMS = " + std::to_string((unsigned long long)TF_PENTA_STATIC_MAX_ELEMS) +
                        " elements; use tf_penta_solve with a caller-owned workspace");
    if ((dir ? nrow : ncol) < 3) return fail(nullptr, TF_ERR_INVALID_ARG, "system length must be >= 3");
    if (!e || !c || !d || !a || !b || !rhs || !x) return fail(nullptr, TF_ERR_INVALID_ARG, "NULL pointer");
    double* scratch = nullptr;
    const tf_status st = penta_static_scratch(&scratch);
    if (st != TF_OK) return st;
    // the three fields sit align_up(nrow * ncol * 8) <= 8 MiB apart: inside the array by the limit above.  The existing
    // thread-per-system path does the rest; it enqueues kernels and sets function attributes, and allocates nothing.
    return tf_penta_solve_ex(nrow, ncol, dir, TF_PENTA_LU, 0, e, c, d, a, b, rhs, x, scratch, cuda_stream);
}

// ---- tf_fp64_peak: DFMA micro-benchmark (the denominator of the "alu" roofline)
namespace {

constexpr int DFMA_CHAINS = 8, DFMA_ITERS = 16384;

__global__ void __launch_bounds__(256) dfma_probe_kernel(double* sink, double a, double b)
{
    double x[DFMA_CHAINS];
#pragma unroll
    for (int k = 0; k < DFMA_CHAINS; ++k) x[k] = 1.0 + 1e-3 * (double)(threadIdx.x + k);
#pragma unroll 4
    for (int it = 0; it < DFMA_ITERS; ++it) {
#pragma unroll
        for (int k = 0; k < DFMA_CHAINS; ++k) x[k] = fma(x[k], a, b);      // a, b are run-time values: nothing folds
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < DFMA_CHAINS; ++k) s += x[k];
    if (s == -1.2345e300) *sink = s;                                        // never true; keeps the chains alive
}

}  // namespace

tf_status tf_fp64_peak(int launches, double* best_dfma_per_s, double* mean_dfma_per_s, void* cuda_stream)
{
    if (launches < 1 || launches > 1000) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_fp64_peak: 1 <= launches <= 1000");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const unsigned grid = (unsigned)num_sms() * 16u;
    cudaEvent_t e0, e1;
    TF_CUDA(nullptr, cudaEventCreate(&e0));
    cudaError_t e = cudaEventCreate(&e1);
    if (e != cudaSuccess) { cudaEventDestroy(e0); return cuda_fail(nullptr, e, "cudaEventCreate"); }
    const double work = (double)grid * 256.0 * DFMA_CHAINS * DFMA_ITERS;
    double best = 0.0, total_ms = 0.0;
    for (int l = -1; l < launches && e == cudaSuccess; ++l) {                // l = -1: untimed warm-up
        cudaEventRecord(e0, st);
        dfma_probe_kernel<<<grid, 256, 0, st>>>(nullptr, 0.999999, 1e-6);
        cudaEventRecord(e1, st);
        count_launch(1);
        e = cudaEventSynchronize(e1);
        float ms = 0.0f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e == cudaSuccess && l >= 0) { total_ms += ms; best = std::max(best, work / (ms * 1e-3)); }
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "tf_fp64_peak");
    if (best_dfma_per_s) *best_dfma_per_s = best;
    if (mean_dfma_per_s) *mean_dfma_per_s = work * launches / (total_ms * 1e-3);
    return TF_OK;
}

size_t tf_betti_workspace_bytes(int nx, int ny, int nthr)
{
    if (nx < 1 || ny < 1 || nthr < 1) return 0;
    const size_t n = (size_t)nx * ny;
    return align_up(n * sizeof(int)) + align_up(n) + align_up(2 * sizeof(unsigned long long) * (size_t)nthr);
}

tf_status tf_betti(const double* h, int nx, int ny, const double* thresholds, int nthr, long long* b0, long long* b1,
                   void* dev_ws, void* cuda_stream)
{
    if (nx < 1 || ny < 1 || nthr < 1) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_betti: bad shape or threshold count");
    if ((long long)nx * ny >= (1LL << 31)) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_betti: nx*ny must be < 2^31 (32-bit labels)");
    if (!h || !thresholds || !b0 || !b1 || !dev_ws) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_betti: NULL pointer");
    for (int t = 0; t < nthr; ++t)
        if (thresholds[t] != thresholds[t]) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_betti: NaN threshold");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t n = (size_t)nx * ny;
    int* L = (int*)dev_ws;
    unsigned char* open = (unsigned char*)dev_ws + align_up(n * sizeof(int));
    unsigned long long* cnt = (unsigned long long*)(open + align_up(n));
    TF_CUDA(nullptr, cudaMemsetAsync(cnt, 0, 2 * sizeof(unsigned long long) * (size_t)nthr, st));
    const dim3 g((unsigned)((nx + TOPO_THREADS - 1) / TOPO_THREADS), (unsigned)ny);
    if (g.y > 65535u) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_betti: ny must be <= 65535");
    const unsigned gb = (unsigned)((2 * (size_t)nx + 2 * (size_t)ny + TOPO_THREADS - 1) / TOPO_THREADS);
    const unsigned gc = (unsigned)std::min<size_t>((n + TOPO_THREADS - 1) / TOPO_THREADS, (size_t)num_sms() * 16);
    for (int t = 0; t < nthr; ++t) {
        const double thr = thresholds[t];
        TF_CUDA(nullptr, cudaMemsetAsync(open, 0, n, st));
        topo_init_kernel<<<g, TOPO_THREADS, 0, st>>>(nx, h, thr, L);
        topo_merge_kernel<<<g, TOPO_THREADS, 0, st>>>(nx, ny, h, thr, L);
        topo_border_kernel<<<gb, TOPO_THREADS, 0, st>>>(nx, ny, h, thr, L, open);
        topo_count_kernel<<<gc, TOPO_THREADS, 0, st>>>(n, h, thr, L, open, cnt + 2 * t);
        count_launch(4);
        TF_CUDA(nullptr, cudaGetLastError());
    }
    std::vector<unsigned long long> host(2 * (size_t)nthr);
    TF_CUDA(nullptr, cudaMemcpyAsync(host.data(), cnt, host.size() * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    TF_CUDA(nullptr, cudaStreamSynchronize(st));
    for (int t = 0; t < nthr; ++t) { b0[t] = (long long)host[2 * t]; b1[t] = (long long)host[2 * t + 1]; }
    return TF_OK;
}

// ---- radial Fourier transform, App. B steps 1-4 (tf_spectrum.cuh); the FFT is cuFFT, loaded at run time
namespace {
struct CuFFT {
    void* lib = nullptr;
    int (*plan2d)(int*, int, int, int) = nullptr;
    int (*set_stream)(int, cudaStream_t) = nullptr;
    int (*exec_d2z)(int, double*, void*) = nullptr;
    int (*destroy)(int) = nullptr;
    int plan = -1, pnx = 0, pny = 0, pdev = -1;
    bool load()
    {
        if (lib) return true;
        const char* names[] = {"libcufft.so.11", "/usr/local/cuda/lib64/libcufft.so.11", "libcufft.so", "/usr/local/cuda/lib64/libcufft.so"};
        for (const char* n : names) {
            lib = dlopen(n, RTLD_NOW | RTLD_LOCAL);
            if (lib) break;
        }
        if (!lib) return false;
        plan2d = (int (*)(int*, int, int, int))dlsym(lib, "cufftPlan2d");
        set_stream = (int (*)(int, cudaStream_t))dlsym(lib, "cufftSetStream");
        exec_d2z = (int (*)(int, double*, void*))dlsym(lib, "cufftExecD2Z");
        destroy = (int (*)(int))dlsym(lib, "cufftDestroy");
        if (!plan2d || !set_stream || !exec_d2z || !destroy) { dlclose(lib); lib = nullptr; return false; }
        return true;
    }
    bool get_plan(int nx, int ny)
    {
        int dev = 0;
        cudaGetDevice(&dev);
        if (plan >= 0 && pnx == nx && pny == ny && pdev == dev) return true;
        if (plan >= 0) { destroy(plan); plan = -1; }
        if (plan2d(&plan, ny, nx, 0x6a /* CUFFT_D2Z */) != 0) { plan = -1; return false; }
        pnx = nx; pny = ny; pdev = dev;
        return true;
    }
};
CuFFT g_fft;
std::mutex g_fft_mutex;                      // one plan cache per process: tf_radial_spectrum holds it from plan lookup to exec
size_t sp_field_bytes(int nx, int ny) { return align_up((size_t)nx * ny * sizeof(double)); }
size_t sp_half_bytes(int nx, int ny) { return align_up((size_t)ny * (nx / 2 + 1) * 2 * sizeof(double)); }
}  // namespace

size_t tf_spectrum_workspace_bytes(int nx, int ny, int kmax)
{
    if (nx < 2 || ny < 2 || kmax < 0) return 0;
    const size_t nk = (size_t)kmax * kmax + 1;
    return 2 * sp_field_bytes(nx, ny) + sp_half_bytes(nx, ny) + align_up(nk * sizeof(double)) + align_up(nk * sizeof(unsigned long long));
}

tf_status tf_radial_spectrum(const double* h, int nx, int ny, double L, double H0, double sigma, int kmax, double* q,
                             double* zeta, long long* count, int cap, int* nk_out, void* dev_ws, void* cuda_stream)
{
    if (nx < 2 || ny < 2 || kmax < 0 || cap < 0) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_radial_spectrum: bad shape, kmax or cap");
    if ((long long)nx * ny >= (1LL << 31)) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_radial_spectrum: nx*ny must be < 2^31");
    if (!(L > 0) || !std::isfinite(L) || !std::isfinite(H0) || !(sigma >= 0) || !std::isfinite(sigma))
        return fail(nullptr, TF_ERR_INVALID_ARG, "tf_radial_spectrum: need L > 0, sigma >= 0, finite H0");
    if (!h || !q || !zeta || !count || !nk_out || !dev_ws) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_radial_spectrum: NULL pointer");
    if (kmax > 20000) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_radial_spectrum: kmax <= 20000");
    SpWeights W;
    W.r = sigma > 0 ? (int)std::ceil(3.0 * sigma) : 0;
    if (W.r > SP_MAXW) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_radial_spectrum: ceil(3 sigma) must be <= 64");
    {
        double sum = 0.0;
        for (int a = 0; a <= 2 * W.r; ++a) { const double m = a - W.r; W.w[a] = W.r ? std::exp(-m * m / (2.0 * sigma * sigma)) : 1.0; sum += W.w[a]; }
        for (int a = 0; a <= 2 * W.r; ++a) W.w[a] /= sum;
    }
    std::lock_guard<std::mutex> fft_lock(g_fft_mutex);
    if (!g_fft.load()) return fail(nullptr, TF_ERR_UNSUPPORTED, "tf_radial_spectrum: libcufft.so.11 not found");
    if (!g_fft.get_plan(nx, ny)) return fail(nullptr, TF_ERR_CUDA, "tf_radial_spectrum: cufftPlan2d failed");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t n = (size_t)nx * ny, nk = (size_t)kmax * kmax + 1;
    char* ws = (char*)dev_ws;
    double* A = (double*)ws;
    double* B = (double*)(ws + sp_field_bytes(nx, ny));
    double2* Z = (double2*)(ws + 2 * sp_field_bytes(nx, ny));
    double* sums = (double*)((char*)Z + sp_half_bytes(nx, ny));
    unsigned long long* cnts = (unsigned long long*)((char*)sums + align_up(nk * sizeof(double)));
    TF_CUDA(nullptr, cudaMemsetAsync(sums, 0, align_up(nk * sizeof(double)) + nk * sizeof(unsigned long long), st));
    const unsigned gl = (unsigned)std::min<size_t>((n + SP_THREADS - 1) / SP_THREADS, (size_t)num_sms() * 16);
    const dim3 g2((unsigned)((nx + SP_THREADS - 1) / SP_THREADS), (unsigned)ny);
    if (g2.y > 65535u) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_radial_spectrum: ny must be <= 65535");
    sp_subtract_kernel<<<gl, SP_THREADS, 0, st>>>(n, h, H0, A);
    if (g_fft.set_stream(g_fft.plan, st) != 0 || g_fft.exec_d2z(g_fft.plan, A, Z) != 0)
        return fail(nullptr, TF_ERR_CUDA, "tf_radial_spectrum: cufftExecD2Z failed");
    sp_magnitude_kernel<<<g2, SP_THREADS, 0, st>>>(nx, ny, Z, A);
    const double* smooth = A;
    if (W.r > 0) {
        sp_gauss_kernel<true><<<g2, SP_THREADS, 0, st>>>(nx, ny, A, B, W);
        sp_gauss_kernel<false><<<g2, SP_THREADS, 0, st>>>(nx, ny, B, A, W);
    }
    sp_radial_kernel<<<g2, SP_THREADS, 0, st>>>(nx, ny, smooth, (long long)kmax * kmax, sums, cnts);
    count_launch(W.r > 0 ? 5 : 3);
    TF_CUDA(nullptr, cudaGetLastError());
    std::vector<double> hs(nk);
    std::vector<unsigned long long> hc(nk);
    TF_CUDA(nullptr, cudaMemcpyAsync(hs.data(), sums, nk * sizeof(double), cudaMemcpyDeviceToHost, st));
    TF_CUDA(nullptr, cudaMemcpyAsync(hc.data(), cnts, nk * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    TF_CUDA(nullptr, cudaStreamSynchronize(st));
    int m = 0;
    const double PI2 = 6.283185307179586476925286766559;
    for (size_t k = 0; k < nk; ++k) {
        if (!hc[k]) continue;
        if (m < cap) { q[m] = PI2 * std::sqrt((double)k) / L; zeta[m] = hs[k] / (double)hc[k]; count[m] = (long long)hc[k]; }
        ++m;
    }
    *nk_out = m;
    return TF_OK;
}

// ---- App. B steps 5-6 and the maxima: host-side 1-D post-processing of the radial spectrum
tf_status tf_radial_peaks(const double* q, const double* zeta, int nk, int per_interval, int ngrid, double* qgrid,
                          double* zsmooth, double* peak_q, double* peak_z, int peak_cap, int* npeaks)
{
    if (!q || !zeta || nk < 2 || per_interval < 2 || ngrid < 8 || peak_cap < 0 || (peak_cap > 0 && (!peak_q || !peak_z)) || !npeaks)
        return fail(nullptr, TF_ERR_INVALID_ARG, "tf_radial_peaks: bad arguments");
    // points with q > 0, ascending
    std::vector<double> x, y;
    for (int i = 0; i < nk; ++i) {
        if (!std::isfinite(q[i]) || !std::isfinite(zeta[i])) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_radial_peaks: non-finite input");
        if (i > 0 && !(q[i] > q[i - 1])) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_radial_peaks: q must be strictly ascending");
        if (q[i] > 0.0) { x.push_back(q[i]); y.push_back(zeta[i]); }
    }
    const int n = (int)x.size();
    if (n < per_interval) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_radial_peaks: fewer points than one interval");
    // (B.2) knots: every interval holds per_interval points, the last one what is left; a_0 = 0 at q = 0
    std::vector<double> ks(1, 0.0);
    for (int i = per_interval - 1; i < n; i += per_interval) ks.push_back(x[i]);
    if (ks.back() < x[n - 1]) ks.push_back(x[n - 1]);
    const int K = (int)ks.size() - 1;
    // normal equations of the hat functions of knots 1..K: symmetric positive definite, tridiagonal
    std::vector<double> d(K, 0.0), u(K, 0.0), r(K, 0.0), a(K + 1, 0.0);
    int k = 0;
    for (int i = 0; i < n; ++i) {
        while (k < K - 1 && x[i] > ks[k + 1]) ++k;               // interval [ks[k], ks[k+1]] containing x[i]
        const double sft = (x[i] - ks[k]) / (ks[k + 1] - ks[k]);
        if (k >= 1) { d[k - 1] += (1.0 - sft) * (1.0 - sft); u[k - 1] += (1.0 - sft) * sft; r[k - 1] += (1.0 - sft) * y[i]; }
        d[k] += sft * sft;
        r[k] += sft * y[i];
    }
    for (int j = 1; j < K; ++j) {                                // Thomas on the symmetric system (sub-diagonal = u)
        const double m = u[j - 1] / d[j - 1];
        d[j] -= m * u[j - 1];
        r[j] -= m * r[j - 1];
    }
    if (!(d[K - 1] > 0.0)) return fail(nullptr, TF_ERR_INVALID_ARG, "tf_radial_peaks: singular fit");
    a[K] = r[K - 1] / d[K - 1];
    for (int j = K - 2; j >= 0; --j) a[j + 1] = (r[j] - u[j] * a[j + 2]) / d[j];
    // 400-point grid on [0, q_K], evaluate, (B.3) moving average with P = 3, 2, 1 (window cut at the ends)
    std::vector<double> g(ngrid), f(ngrid), t(ngrid), df(ngrid);
    const double h = ks[K] / (ngrid - 1);
    k = 0;
    for (int i = 0; i < ngrid; ++i) {
        g[i] = i == ngrid - 1 ? ks[K] : i * h;
        while (k < K - 1 && g[i] > ks[k + 1]) ++k;
        const double sft = (g[i] - ks[k]) / (ks[k + 1] - ks[k]);
        f[i] = a[k] + sft * (a[k + 1] - a[k]);
    }
    for (int P = 3; P >= 1; --P) {
        for (int i = 0; i < ngrid; ++i) {
            const int lo = std::max(0, i - P), hi = std::min(ngrid - 1, i + P);
            double sum = 0.0;
            for (int j = lo; j <= hi; ++j) sum += f[j];
            t[i] = sum / (hi - lo + 1);
        }
        f.swap(t);
    }
    // maxima: second-order differences, roots of the derivative by sign change + linear interpolation
    for (int i = 1; i < ngrid - 1; ++i) df[i] = (f[i + 1] - f[i - 1]) / (2.0 * h);
    df[0] = (-3.0 * f[0] + 4.0 * f[1] - f[2]) / (2.0 * h);
    df[ngrid - 1] = (3.0 * f[ngrid - 1] - 4.0 * f[ngrid - 2] + f[ngrid - 3]) / (2.0 * h);
    int np = 0;
    for (int i = 0; i < ngrid - 1; ++i) {
        if (df[i] > 0.0 && df[i + 1] <= 0.0) {
            const double tt = df[i] / (df[i] - df[i + 1]);
            int c = tt < 0.5 ? i : i + 1;
            c = std::min(std::max(c, 1), ngrid - 2);
            if (f[c + 1] - 2.0 * f[c] + f[c - 1] < 0.0) {
                if (np < peak_cap) { peak_q[np] = g[i] + tt * h; peak_z[np] = f[i] + tt * (f[i + 1] - f[i]); }
                ++np;
            }
        }
    }
    *npeaks = np;
    if (qgrid) std::copy(g.begin(), g.end(), qgrid);
    if (zsmooth) std::copy(f.begin(), f.end(), zsmooth);
    return TF_OK;
}

const char* tf_last_error(const tf_ctx* c) { return c ? c->err.c_str() : g_err.c_str(); }

unsigned long long tf_kernel_launches(void) { return g_launches.load(); }

}  // extern "C"
