// uc_kernels.cuh -- sm_100a kernels of the restarted PDHG hot path.
//
// Everything here works in the PERMUTED, SCALED index spaces built by uc_format.hpp.  One thread
// owns one row of the sliced-ELL part (a warp owns a slice, so matrix loads are lane-consecutive:
// 128 B of column indices + 256 B of values per warp per step); a row of the long tail is owned by
// one warp.  No atomics touch floating-point data: every reduction is block partial -> final sum by
// the last block to finish (ticket counter).
//
// Arithmetic follows DESIGN.md R3..R11 operation by operation, in the order of the sequential
// statement of the method, because the adaptive step rule makes the trajectory exponentially
// sensitive to rounding: row sums run left to right in the caller's CSR
// order with separately rounded multiply and add (this file is compiled with -fmad=false), rows of
// the long tail included; every long reduction is carried in double-double (uc_dd.cuh) so that its
// rounded value does not depend on the summation order.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <math.h>
#include <stddef.h>
#include <assert.h>
#include "../../include/uc_pdhg.h"
#include "../../include/uc_pdhg_hooks.h"
#include "uc_dd.cuh"
#include "uc_format.hpp"

namespace ucpdhg {

constexpr int kBlock = 256;          // threads per block of every row-parallel kernel
constexpr int kWarps = kBlock / 32;  // = slices per block
constexpr int kFinalBlock = 1024;    // threads of the single-block finalisers
#ifndef UC_CHECK_MINB
#define UC_CHECK_MINB 3
#endif
constexpr int kCheckMinBlocks = UC_CHECK_MINB;   // resident blocks per SM the check kernels are compiled for

struct KktT { double rp2_s, rd2_s, rp2_u, rd2_u, pobj, dobj; };

// status record written by the device into mapped pinned host memory at every check
struct HostStatus {
    int32_t done, status, ret_avg, have_avg;
    int64_t k, accepted, restarts, nchk;
    double rel_kkt, rel_rp, rel_rd, rel_gap, pobj, dobj, eta, omega;
};

// device-resident control block: all step-size / primal-weight / restart scalars live here so that
// the captured graph is static (SURVEY.md hard part 4)
struct Ctrl {
    // ---- the first 48 bytes are what every CTA of an attempt kernel needs before it may touch the iterate: they
    // are fetched with three 16-byte loads in ONE round trip (load_hot), on the critical path of every attempt
    double eta, omega, eta_prev, w;
    int cur;            // which of the two x / y buffers holds the current iterate
    int pending;        // 1: the current iterate has not been added to the weighted sums yet (weight eta_prev)
    int done, status;
    // ----
    double mu_prev;
    long long k, t0, accepted, restarts, limit, nchk;
    int ret_avg, have_avg, restart_kind, cand_avg, fixed, pad0;
    KktT Tr, Tcur, Tavg;
    double eps_abs, eps_rel, beta_s, beta_n, beta_a, smoothing, norm_q, norm_c;
    unsigned int ticket_b, pad1, pad2, pad3;
    const double2* powtab;     // [limit] entry k-1 = {(k+1)^-0.6, (k+1)^-0.3} for attempt k (R5)
    uc_attempt_record* att; long long att_cap;
    uc_check_record* chk; long long chk_cap;
    const int* host_stop;      // mapped host flag: (solve generation << 3) | UC_CANCELLED or UC_TIME_LIMIT; 0 = none
    int gen, pad4;             // generation of the solve in flight: a stop request of another generation is stale
    HostStatus* host_status;   // mapped host record
};

struct CtrlHot { double eta, omega, eta_prev, w; int cur, pending, done, status; };
static_assert(offsetof(Ctrl, cur) == 32 && offsetof(Ctrl, status) == 44, "Ctrl hot block layout");
__device__ __forceinline__ CtrlHot load_hot(const Ctrl* ctl) {       // L2 reads (the previous kernel wrote them)
    const double2 a = __ldcg(reinterpret_cast<const double2*>(ctl)), b = __ldcg(reinterpret_cast<const double2*>(ctl) + 1);
    const int4 f = __ldcg(reinterpret_cast<const int4*>(ctl) + 2);
    return CtrlHot{a.x, a.y, b.x, b.y, f.x, f.y, f.z, f.w};
}

struct Sell {
    const long long* sp;   // slice pointers [nslices+1]
    const int* col;        // 32-bit column indices of the WIDE slices (NULL if every slice is narrow)
    const unsigned short* col16;   // 16-bit offsets from cbase[slice] of the NARROW slices (NULL if every slice is wide)
    const int* cbase;      // [nslices] >= 0: narrow slice, its smallest column index; -1: wide slice   (uc_format.hpp)
    double* val;
    long long nshort;      // rows in the sliced part
    int nslices;
    int nblk;              // blocks covering the sliced part = ceil(nslices / kWarps)
    const long long* lp;   // long-tail CSR pointers [nlong+1]
    const int* lcol;
    double* lval;
    int nlong;
    int nlblk;             // blocks covering the long tail = ceil(nlong / kWarps); they come FIRST in the grid
    int grid;              // nlblk + nblk, at least 1
    const StepDesc* steps;  // [steps_per_warp][sched_warps] schedule of the persistent attempt kernels (uc_attempt.cuh)
    int steps_per_warp, sched_warps;
    long long nslots, ncols;   // stored slots of the sliced part; length of the vector the column indices address
    int cta_warps;             // consumer warps per CTA of the attempt kernel that runs this schedule (+ 1 long-row warp)
};
// -DUC_DEBUG_BOUNDS: every address the attempt pipelines derive from a step descriptor or a stored column index is
// checked on the device (compute-sanitizer is not available on every GPU pool; this build is the substitute and is run
// through the GPU parity tests once per change of the pipelines, profiles/).
#ifdef UC_DEBUG_BOUNDS
#define UC_BOUNDS_ASSERT(cond) assert(cond)
#else
#define UC_BOUNDS_ASSERT(cond) do { } while (0)
#endif

struct Vecs {
    long long n, m;
    double* x[2]; double* y[2];
    double2* xg;                 // {xbar, dx} of the attempt in flight, gathered by the K pass
    double* xsum; double* ysum;  // eta-weighted sums (R6)
    double* xr; double* yr;      // restart point (R11)
    const double *c, *l, *u, *q; // scaled data
    const unsigned char* isG;
    const double *Dr, *Dc;
    dd* partA;                   // [gridPA]     sum dx^2            (one per CTA of the persistent primal kernel)
    dd* partB;                   // [2][gridPB]  sum dy^2, sum dy * (K dx)
    dd* partD;                   // [8][gridA]   check, dual side
    dd* partP;                   // [6][gridB]   check, primal side
    dd* partR;                   // [2][gridR]   restart distances
    int gridA, gridB, gridR;     // grids of the check kernels (persistent: grid-stride over the layout's blocks) and of
                                 // the one-thread-per-element restart / flush kernels
    int gridPA, gridPB;          // persistent grids of the two attempt kernels
#ifdef UC_TIMELINE
    unsigned long long* tl;      // [grid][kTlWarps][kTlMarks] globaltimer marks of the kernel being launched (measurement build only)
#endif
};
// -DUC_TIMELINE (measurement build, uc_pdhg_timeline): every warp of the attempt kernels records when it entered the
// kernel, when its grid dependency resolved, when it finished its steps and when it left.
constexpr int kTlWarps = 32, kTlMarks = 8;
#ifdef UC_TIMELINE
__device__ __forceinline__ unsigned long long tl_now() { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
#define UC_TL_MARK(V, i)                                                                                               \
    do { if ((V).tl && (threadIdx.x & 31) == 0)                                                                        \
        (V).tl[((size_t)blockIdx.x * kTlWarps + (threadIdx.x >> 5)) * kTlMarks + (i)] = tl_now(); } while (0)
#else
#define UC_TL_MARK(V, i) do { } while (0)
#endif

// ------------------------------------------------------------------------------------------ loads
__device__ __forceinline__ double ld_stream(const double* p) {   // read-once data: keep it out of L1
    double v; asm("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(p)); return v;
}
__device__ __forceinline__ int ld_stream(const int* p) {
    int v; asm("ld.global.nc.L1::no_allocate.s32 %0, [%1];" : "=r"(v) : "l"(p)); return v;
}
__device__ __forceinline__ int ld_stream(const unsigned short* p) {
    unsigned short v; asm("ld.global.nc.L1::no_allocate.u16 %0, [%1];" : "=h"(v) : "l"(p)); return (int)v;
}
__device__ __forceinline__ int ld_flag(const int* p) { return *(const volatile int*)p; }

__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
// s + p(lane 0) + p(lane 1) + ... + p(lane 31), added in that order; same result in every lane
__device__ __forceinline__ double warp_seq_add(double s, double p) {
#pragma unroll
    for (int l = 0; l < 32; ++l) s = __dadd_rn(s, __shfl_sync(0xffffffffu, p, l));
    return s;
}
__device__ __forceinline__ dd warp_sum_dd(dd v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        dd t;
        t.hi = __shfl_xor_sync(0xffffffffu, v.hi, o);
        t.lo = __shfl_xor_sync(0xffffffffu, v.lo, o);
        v = dd_add(v, t);
    }
    return v;
}

// block-wide double-double sums of NV values (each thread contributes one double-double per value);
// result valid in thread 0.  red: NV * 32 dd of shared memory.  Two stages, both warp-parallel: every warp
// reduces its own NV values by shuffles, then warp q (mod #warps) reduces the per-warp results of value q.
template <int NV>
__device__ __forceinline__ void block_sum_dd(dd (&v)[NV], dd* red) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int q = 0; q < NV; ++q) {
        v[q] = warp_sum_dd(v[q]);
        if (lane == 0) red[q * 32 + warp] = v[q];
    }
    __syncthreads();
    for (int q = warp; q < NV; q += nw) {
        dd t = lane < nw ? red[q * 32 + lane] : dd{0.0, 0.0};
        t = warp_sum_dd(t);
        if (lane == 0) red[q * 32] = t;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int q = 0; q < NV; ++q) v[q] = red[q * 32];
    }
    __syncthreads();
}

// The same sums when only warp 0 needs them (the attempt kernels: this is the serial tail of every attempt).  Every warp
// reduces its own values by shuffles (the NV chains interleave), parks them in shared memory and ARRIVES at named
// barrier 1 -- it does not wait and is free to leave the kernel; warp 0 waits for all arrivals and adds the per-warp
// results.  Returns true in warp 0 (result in every lane of it), false elsewhere.  red: NV * 32 dd.
template <int NV>
__device__ __forceinline__ void warp_sum_dd_n(dd (&v)[NV]) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int q = 0; q < NV; ++q) {
            dd t;
            t.hi = __shfl_xor_sync(0xffffffffu, v[q].hi, o);
            t.lo = __shfl_xor_sync(0xffffffffu, v[q].lo, o);
            v[q] = dd_acc(v[q], t);                         // cascaded: see uc_dd.cuh
        }
    }
}
template <int NV>
__device__ __forceinline__ bool block_sum_dd_warp0(dd (&v)[NV], dd* red) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    warp_sum_dd_n<NV>(v);
    if (lane == 0) {
#pragma unroll
        for (int q = 0; q < NV; ++q) red[q * 32 + warp] = v[q];
    }
    if (warp != 0) { asm volatile("bar.arrive 1, %0;" ::"r"(nw * 32) : "memory"); return false; }
    asm volatile("bar.sync 1, %0;" ::"r"(nw * 32) : "memory");
#pragma unroll
    for (int q = 0; q < NV; ++q) v[q] = lane < nw ? red[q * 32 + lane] : dd{0.0, 0.0};
    warp_sum_dd_n<NV>(v);
    return true;
}

// double-double sums of NV partial arrays (part + q * stride, `count` entries each) by one block, in one pass;
// results valid in thread 0
template <int NV>
__device__ __forceinline__ void final_sums(const dd* part, long long stride, int count, dd (&v)[NV], dd* red) {
#pragma unroll
    for (int q = 0; q < NV; ++q) v[q] = dd{0.0, 0.0};
    for (int i = threadIdx.x; i < count; i += blockDim.x) {
#pragma unroll
        for (int q = 0; q < NV; ++q) {
            dd t; t.hi = __ldcg(&part[q * stride + i].hi); t.lo = __ldcg(&part[q * stride + i].lo);
            v[q] = dd_add(v[q], t);
        }
    }
    block_sum_dd<NV>(v, red);
}

// --------------------------------------------------------------------------- row ownership
// Grid layout of every row-parallel kernel: blocks [0, nlblk) own the long tail (one warp per row;
// they start first so that their sequential sums hide behind the sliced part), blocks
// [nlblk, nlblk + nblk) own the sliced part (one thread per row).
struct RowId { long long row; int slice; int lrow; bool owner; };
// vb: the (virtual) block of the layout this thread block is working on -- blockIdx.x for the one-block-per-256-rows
// kernels, a grid-stride counter for the check kernels
__device__ __forceinline__ RowId my_row(const Sell& A, int vb) {
    RowId r; r.row = -1; r.slice = -1; r.lrow = -1; r.owner = false;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (vb >= A.nlblk) {
        long long j = (long long)(vb - A.nlblk) * kBlock + threadIdx.x;
        int s = (int)(j >> 5);
        if (s < A.nslices) { r.slice = s; r.row = j; r.owner = j < A.nshort; }
    } else {
        int lr = vb * kWarps + warp;
        if (lr < A.nlong) { r.lrow = lr; r.row = A.nshort + lr; r.owner = (lane == 0); }
    }
    return r;
}
__device__ __forceinline__ RowId my_row(const Sell& A) { return my_row(A, (int)blockIdx.x); }

// --------------------------------------------------------------------------- SpMV row traversals
// s[q] += sum_t val_t * g_t[q] over the entries of the row, left to right, multiply and add rounded
// separately.  `gather(col, g)` fills g[0..NV) for a column.  Padding slots hold (col 0, val 0) and
// add +0.0.  Sliced row: one thread, four entries' loads in flight per step.
// column index stored at slot p of a slice whose base is cb (cb < 0: wide slice)
__device__ __forceinline__ int sell_col(const Sell& A, int cb, long long p) {
    return cb >= 0 ? cb + ld_stream(A.col16 + p) : ld_stream(A.col + p);
}
template <int NV, class G>
__device__ __forceinline__ void sell_row(const Sell& A, int slice, int lane, double (&s)[NV], G gather) {
    long long p = __ldg(A.sp + slice) + lane;
    const long long e = __ldg(A.sp + slice + 1);
    const int cb = __ldg(A.cbase + slice);
    for (; p + 96 < e; p += 128) {
        int c[4]; double v[4]; double g[4][NV];
#pragma unroll
        for (int u = 0; u < 4; ++u) { c[u] = sell_col(A, cb, p + 32 * u); v[u] = ld_stream(A.val + p + 32 * u); }
#pragma unroll
        for (int u = 0; u < 4; ++u) gather(c[u], g[u]);
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int q = 0; q < NV; ++q) s[q] = __dadd_rn(s[q], __dmul_rn(v[u], g[u][q]));
    }
    for (; p < e; p += 32) {
        int c = sell_col(A, cb, p); double v = ld_stream(A.val + p); double g[NV];
        gather(c, g);
#pragma unroll
        for (int q = 0; q < NV; ++q) s[q] = __dadd_rn(s[q], __dmul_rn(v, g[q]));
    }
}
// Long-tail row r: the warp forms 32 products at a time (coalesced loads), then adds them in
// entry order; the sums end up in every lane.
// Memory latency, not the add chain, is what a long row costs (25 dependent round trips for 800 entries
// if taken 32 at a time), so entries are taken 128 at a time and the (col, val) loads of the next batch
// are in flight while the current batch is gathered and summed.
template <int NV, class G>
__device__ __forceinline__ void long_row(const Sell& A, int r, int lane, double (&s)[NV], G gather) {
    constexpr int U = 4;
    const long long b = __ldg(A.lp + r), e = __ldg(A.lp + r + 1);
    int cn[U]; double vn[U];
    auto load_cv = [&](long long p0) {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const long long p = p0 + 32 * u + lane;
            cn[u] = 0; vn[u] = 0.0;
            if (p < e) { cn[u] = ld_stream(A.lcol + p); vn[u] = ld_stream(A.lval + p); }
        }
    };
    load_cv(b);
    for (long long p0 = b; p0 < e; p0 += 32 * U) {
        double prod[U][NV];
#pragma unroll
        for (int u = 0; u < U; ++u) {                 // padding lanes gather column 0 and multiply by 0
            double g[NV];
            gather(cn[u], g);
#pragma unroll
            for (int q = 0; q < NV; ++q) prod[u][q] = g[q];
        }
        double v[U];
#pragma unroll
        for (int u = 0; u < U; ++u) v[u] = vn[u];
        if (p0 + 32 * U < e) load_cv(p0 + 32 * U);
#pragma unroll
        for (int u = 0; u < U; ++u)
#pragma unroll
            for (int q = 0; q < NV; ++q) prod[u][q] = (p0 + 32 * u + lane < e) ? __dmul_rn(v[u], prod[u][q]) : 0.0;
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if (p0 + 32 * u >= e) break;              // warp-uniform: whole chunk beyond the row end
#pragma unroll
            for (int q = 0; q < NV; ++q) s[q] = warp_seq_add(s[q], prod[u][q]);
        }
    }
}
template <int NV, class G>
__device__ __forceinline__ void row_dot(const Sell& A, const RowId& r, int lane, double (&s)[NV], G gather) {
    if (r.slice >= 0) sell_row<NV>(A, r.slice, lane, s, gather);
    else long_row<NV>(A, r.lrow, lane, s, gather);
}

// --------------------------------------------------------------------------- A11 check, dual side
// per variable j (row of K~'), for z in {current, average}: rho = c - K~'y, lambda, r_d, c.x, bound
// terms of the dual objective (R9).  partD rows: [rd2_s, rd2_u, pobj, dbound] x {cur, avg}.
// flush != 0 (the periodic check): the pending term of R6 (eta_prev * current iterate, deferred by the attempt
// kernels) is applied here instead of in a pass of its own: this kernel adds it on the fly to the y-sums it gathers
// (k_check_primal, which runs next, writes them back) and writes the flushed x-sums of its own rows back.
__global__ void __launch_bounds__(kBlock, kCheckMinBlocks) k_check_dual(Sell KT, Vecs V, Ctrl* ctl, int flush) {
    __shared__ dd red[8 * 32];
    if (ld_flag(&ctl->done)) return;
    const int cur = ctl->cur;
    const bool pend = flush && ctl->pending; const double e = ctl->eta_prev;
    const double w = ctl->w; const bool avg = w > 0.0;
    const double* __restrict__ ycur = V.y[cur];
    const double* __restrict__ ysum = V.ysum;
    const int lane = threadIdx.x & 31;
    dd acc[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) acc[q] = dd{0.0, 0.0};
    for (int vb = blockIdx.x; vb < KT.grid; vb += gridDim.x) {      // persistent blocks: ONE block reduction per block
        const RowId r = my_row(KT, vb);
        if (r.row < 0) continue;
        double g[2] = {0.0, 0.0};
        if (avg) row_dot<2>(KT, r, lane, g, [&](int c, double (&o)[2]) { o[0] = ycur[c]; o[1] = (pend ? ysum[c] + e * o[0] : ysum[c]) / w; });
        else { double g1[1] = {0.0}; row_dot<1>(KT, r, lane, g1, [&](int c, double (&o)[1]) { o[0] = ycur[c]; }); g[0] = g1[0]; }
        if (r.owner) {
            const long long j = r.row;
            const double cj = V.c[j], lj = V.l[j], uj = V.u[j], dc = V.Dc[j];
            const bool lfin = isfinite(lj), ufin = isfinite(uj);
            const double xc = V.x[cur][j];
            double xs = V.xsum[j];
            if (pend) { xs = xs + e * xc; V.xsum[j] = xs; }
#pragma unroll
            for (int z = 0; z < 2; ++z) {
                if (z == 1 && !avg) break;
                const double xj = z ? xs / w : xc;
                const double rj = cj - g[z];
                double lam = 0.0;
                if (rj > 0.0 && lfin) lam = rj;
                if (rj < 0.0 && ufin) lam = rj;
                const double rd = rj - lam;
                acc[4 * z + 0] = dd_add_d(acc[4 * z + 0], rd * rd);
                acc[4 * z + 1] = dd_add_d(acc[4 * z + 1], (dc * rd) * (dc * rd));
                acc[4 * z + 2] = dd_add_d(acc[4 * z + 2], cj * xj);
                acc[4 * z + 3] = dd_add_d(acc[4 * z + 3], lam > 0.0 ? lj * lam : (lam < 0.0 ? uj * lam : 0.0));
            }
        }
    }
    block_sum_dd<8>(acc, red);
    if (threadIdx.x == 0)
        for (int q = 0; q < 8; ++q) V.partD[(long long)q * V.gridA + blockIdx.x] = acc[q];
}

// --------------------------------------------------------------------------- A11 check, primal side
// per row i of K~: a = K~x - q, r_p, q.y (R9).  partP rows: [rp2_s, rp2_u, qy] x {cur, avg}.
// flush != 0: the x-sums it gathers were flushed by k_check_dual just before; it flushes the y-sums of its own rows.
__global__ void __launch_bounds__(kBlock, kCheckMinBlocks) k_check_primal(Sell K, Vecs V, Ctrl* ctl, int flush) {
    __shared__ dd red[6 * 32];
    if (ld_flag(&ctl->done)) return;
    const int cur = ctl->cur;
    const bool pend = flush && ctl->pending; const double e = ctl->eta_prev;
    const double w = ctl->w; const bool avg = w > 0.0;
    const double* __restrict__ xcur = V.x[cur];
    const double* __restrict__ xsum = V.xsum;
    const int lane = threadIdx.x & 31;
    dd acc[6];
#pragma unroll
    for (int q = 0; q < 6; ++q) acc[q] = dd{0.0, 0.0};
    for (int vb = blockIdx.x; vb < K.grid; vb += gridDim.x) {       // persistent blocks: ONE block reduction per block
        const RowId r = my_row(K, vb);
        if (r.row < 0) continue;
        double a[2] = {0.0, 0.0};
        if (avg) row_dot<2>(K, r, lane, a, [&](int c, double (&o)[2]) { o[0] = xcur[c]; o[1] = xsum[c] / w; });
        else { double a1[1] = {0.0}; row_dot<1>(K, r, lane, a1, [&](int c, double (&o)[1]) { o[0] = xcur[c]; }); a[0] = a1[0]; }
        if (r.owner) {
            const long long i = r.row;
            const double qi = V.q[i], dr = V.Dr[i]; const int isg = V.isG[i];
            const double yc = V.y[cur][i];
            double ys = V.ysum[i];
            if (pend) { ys = ys + e * yc; V.ysum[i] = ys; }
#pragma unroll
            for (int z = 0; z < 2; ++z) {
                if (z == 1 && !avg) break;
                const double ai = a[z] - qi;
                const double yi = z ? ys / w : yc;
                const double rp = isg ? (ai < 0.0 ? ai : 0.0) : ai;
                acc[3 * z + 0] = dd_add_d(acc[3 * z + 0], rp * rp);
                acc[3 * z + 1] = dd_add_d(acc[3 * z + 1], (dr * rp) * (dr * rp));
                acc[3 * z + 2] = dd_add_d(acc[3 * z + 2], qi * yi);
            }
        }
    }
    block_sum_dd<6>(acc, red);
    if (threadIdx.x == 0)
        for (int q = 0; q < 6; ++q) V.partP[(long long)q * V.gridB + blockIdx.x] = acc[q];
}

__device__ __forceinline__ double kkt_omega(const KktT& t, double w) {
    const double g = t.pobj - t.dobj;
    return sqrt(w * w * t.rp2_s + t.rd2_s / (w * w) + g * g);
}
__device__ __forceinline__ void rel_terms(const Ctrl* c, const KktT& t, double& rp, double& rd, double& gap) {
    rp = sqrt(t.rp2_u) / (1.0 + c->norm_q);
    rd = sqrt(t.rd2_u) / (1.0 + c->norm_c);
    gap = fabs(t.pobj - t.dobj) / (1.0 + fabs(t.pobj) + fabs(t.dobj));
}
__device__ __forceinline__ double rel_kkt(const Ctrl* c, const KktT& t) {
    double a, b, g; rel_terms(c, t, a, b, g);
    const double r = a > b ? a : b;
    return r > g ? r : g;
}
__device__ __forceinline__ bool converged(const Ctrl* c, const KktT& t) {
    return sqrt(t.rp2_u) <= c->eps_abs + c->eps_rel * c->norm_q && sqrt(t.rd2_u) <= c->eps_abs + c->eps_rel * c->norm_c &&
           fabs(t.pobj - t.dobj) <= c->eps_abs + c->eps_rel * (fabs(t.pobj) + fabs(t.dobj));
}
__device__ __forceinline__ void publish(Ctrl* c, const KktT& t) {
    HostStatus s;
    s.done = c->done; s.status = c->status; s.ret_avg = c->ret_avg; s.have_avg = c->have_avg;
    s.k = c->k; s.accepted = c->accepted; s.restarts = c->restarts; s.nchk = c->nchk;
    rel_terms(c, t, s.rel_rp, s.rel_rd, s.rel_gap);
    s.rel_kkt = rel_kkt(c, t);
    s.pobj = t.pobj; s.dobj = t.dobj; s.eta = c->eta; s.omega = c->omega;
    *c->host_status = s;
    __threadfence_system();
}

// modes of k_check_finalize
enum { kModeInit = 0,    // z^0: store the KKT components of the restart point (R2)
       kModeCheck = 1,   // R8..R12: termination, candidate, restart decision
       kModeReport = 2   // fixed-iteration end: only report the current iterate's KKT terms (R14)
};

// A11 end + A12 decision + A13: single block.
__global__ void __launch_bounds__(kFinalBlock) k_check_finalize(Vecs V, Ctrl* ctl, int mode) {
    __shared__ dd red[8 * 32];
    if (ld_flag(&ctl->done)) return;
    dd T[14];
    {
        dd a[8], b[6];
        final_sums<8>(V.partD, V.gridA, V.gridA, a, red);
        final_sums<6>(V.partP, V.gridB, V.gridB, b, red);
        if (threadIdx.x != 0) return;
#pragma unroll
        for (int q = 0; q < 8; ++q) T[q] = a[q];
#pragma unroll
        for (int q = 0; q < 6; ++q) T[8 + q] = b[q];
    }
    const bool have_avg = ctl->w > 0.0;
    KktT Tc, Ta;
    Tc.rd2_s = dd_round(T[0]); Tc.rd2_u = dd_round(T[1]); Tc.pobj = dd_round(T[2]);
    Tc.rp2_s = dd_round(T[8]); Tc.rp2_u = dd_round(T[9]); Tc.dobj = dd_round(dd_add(T[10], T[3]));
    Ta = Tc;
    if (have_avg) {
        Ta.rd2_s = dd_round(T[4]); Ta.rd2_u = dd_round(T[5]); Ta.pobj = dd_round(T[6]);
        Ta.rp2_s = dd_round(T[11]); Ta.rp2_u = dd_round(T[12]); Ta.dobj = dd_round(dd_add(T[13], T[7]));
    }
    ctl->Tcur = Tc;
    if (mode == kModeInit) { ctl->Tr = Tc; ctl->Tavg = Tc; return; }
    if (mode == kModeReport) { ctl->ret_avg = 0; ctl->status = UC_ITERATION_LIMIT; ctl->done = 1; publish(ctl, Tc); return; }
    if (have_avg) ctl->Tavg = Ta;       // otherwise the previous average terms stay, as in the sequential statement
    ctl->have_avg = have_avg;
    ctl->pending = 0;                   // the two check kernels have applied it
    const long long k = ctl->k;
    const double omega = ctl->omega;
    const double rk_cur = rel_kkt(ctl, Tc), rk_avg = have_avg ? rel_kkt(ctl, Ta) : INFINITY;
    uc_check_record rec;
    rec.k = k; rec.restart_kind = 0; rec.candidate = 0; rec.omega_after = omega; rec.mu_c = 0.0; rec.mu_r = 0.0;
    rec.relkkt_cur = rk_cur; rec.relkkt_avg = rk_avg;
    int status = -1, ret_avg = 0;
    if (!isfinite(rk_cur)) status = UC_NUMERICAL_ERROR;
    else if (!ctl->fixed) {                                        // R12
        if (have_avg && converged(ctl, Ta)) { status = UC_OPTIMAL; ret_avg = 1; }
        else if (converged(ctl, Tc)) { status = UC_OPTIMAL; ret_avg = 0; }
    }
    if (status < 0) {
        const int stop = *(const volatile int*)ctl->host_stop;    // cancel / time limit from the host, for THIS solve
        if ((stop >> 3) == ctl->gen && (stop & 7)) status = stop & 7;
        else if (k >= ctl->limit) status = UC_ITERATION_LIMIT;
        if (status >= 0 && !ctl->fixed) ret_avg = have_avg && rk_avg < rk_cur;    // best of cur / avg
    }
    int kind = 0;
    if (status < 0) {                                              // R10
        const int cand_avg = have_avg && (kkt_omega(Ta, omega) < kkt_omega(Tc, omega));
        const KktT& Tk = cand_avg ? Ta : Tc;
        const double mu_c = kkt_omega(Tk, omega), mu_r = kkt_omega(ctl->Tr, omega);
        const long long t = k - ctl->t0;
        if (mu_c <= ctl->beta_s * mu_r) kind = 1;
        else if (mu_c <= ctl->beta_n * mu_r && mu_c > ctl->mu_prev) kind = 2;
        else if ((double)t >= ctl->beta_a * (double)k) kind = 3;
        rec.candidate = cand_avg; rec.mu_c = mu_c; rec.mu_r = mu_r; rec.restart_kind = kind;
        if (kind) {
            ctl->cand_avg = cand_avg; ctl->Tr = Tk; ctl->t0 = k; ctl->mu_prev = INFINITY; ctl->restarts += 1;
        } else ctl->mu_prev = mu_c;
    }
    ctl->restart_kind = kind;
    if (ctl->chk && ctl->nchk < ctl->chk_cap) ctl->chk[ctl->nchk] = rec;
    ctl->nchk += 1;
    if (status >= 0) { ctl->status = status; ctl->ret_avg = ret_avg; ctl->done = 1; }
    publish(ctl, (status >= 0 && ret_avg) ? Ta : Tc);
}

// --------------------------------------------------------------------------- A12 restart, vectors
// z <- candidate, z_r <- candidate, sums <- 0, partial ||x_c - x_r||^2 and ||y_c - y_r||^2   (R11)
__global__ void __launch_bounds__(kBlock) k_restart_vec(Vecs V, Ctrl* ctl) {
    __shared__ dd red[64];
    if (ld_flag(&ctl->done) || !ctl->restart_kind) return;
    const int cur = ctl->cur, ca = ctl->cand_avg; const double w = ctl->w;
    long long t = (long long)blockIdx.x * kBlock + threadIdx.x;
    dd acc[2] = {dd{0.0, 0.0}, dd{0.0, 0.0}};
    if (t < V.n) {
        const double xc = ca ? V.xsum[t] / w : V.x[cur][t];
        const double d = xc - V.xr[t]; acc[0].hi = d * d;
        V.x[cur][t] = xc; V.xr[t] = xc; V.xsum[t] = 0.0;
    } else if (t - V.n < V.m) {
        t -= V.n;
        const double yc = ca ? V.ysum[t] / w : V.y[cur][t];
        const double d = yc - V.yr[t]; acc[1].hi = d * d;
        V.y[cur][t] = yc; V.yr[t] = yc; V.ysum[t] = 0.0;
    }
    block_sum_dd<2>(acc, red);
    if (threadIdx.x == 0) { V.partR[blockIdx.x] = acc[0]; V.partR[V.gridR + blockIdx.x] = acc[1]; }
}
// A12 restart, scalars: primal weight (R11), w <- 0
__global__ void __launch_bounds__(kFinalBlock) k_restart_finalize(Vecs V, Ctrl* ctl) {
    __shared__ dd red[2 * 32];
    if (ld_flag(&ctl->done) || !ctl->restart_kind) return;
    dd sxy[2];
    final_sums<2>(V.partR, V.gridR, V.gridR, sxy, red);
    if (threadIdx.x != 0) return;
    const double Dx = sqrt(dd_round(sxy[0])), Dy = sqrt(dd_round(sxy[1]));
    if (Dx > 1e-10 && Dy > 1e-10) {
        const double th = ctl->smoothing;
        ctl->omega = exp_rounded(th * log_rounded(Dy / Dx) + (1.0 - th) * log_rounded(ctl->omega));
    }
    ctl->w = 0.0; ctl->pending = 0; ctl->restart_kind = 0;
    if (ctl->chk && ctl->nchk - 1 < ctl->chk_cap) ctl->chk[ctl->nchk - 1].omega_after = ctl->omega;
    ctl->host_status->omega = ctl->omega;
    __threadfence_system();
}

// --------------------------------------------------------------------------- R2 initial point
// x = clamp(Dc * x0 or 0, l, u), y = proj_Y(Dr * y0 or 0); sums <- 0; restart point <- z^0.
// x0 / y0 are device arrays in the ORIGINAL order (nullable); perm: new -> old.
__global__ void __launch_bounds__(kBlock) k_init_point(Vecs V, const double* x0, const double* y0,
                                                       const long long* perm_c, const long long* perm_r) {
    long long t = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (t < V.n) {
        double v = x0 ? x0[perm_c[t]] * V.Dc[t] : 0.0;
        const double lj = V.l[t], uj = V.u[t];
        v = v < lj ? lj : (v > uj ? uj : v);
        V.x[0][t] = v; V.x[1][t] = v; V.xr[t] = v; V.xsum[t] = 0.0; V.xg[t] = make_double2(v, 0.0);
    } else if (t - V.n < V.m) {
        t -= V.n;
        double v = y0 ? y0[perm_r[t]] * V.Dr[t] : 0.0;
        if (V.isG[t] && v < 0.0) v = 0.0;
        V.y[0][t] = v; V.y[1][t] = v; V.yr[t] = v; V.ysum[t] = 0.0;
    }
}

// --------------------------------------------------------------------------- A14 unscale + un-permute
__global__ void __launch_bounds__(kBlock) k_output(Vecs V, const Ctrl* ctl, double* x_out, double* y_out,
                                                   const long long* perm_c, const long long* perm_r) {
    const int cur = ctl->cur, ra = ctl->ret_avg; const double w = ctl->w;
    long long t = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (t < V.n) {
        if (x_out) x_out[perm_c[t]] = (ra ? V.xsum[t] / w : V.x[cur][t]) / V.Dc[t];
    } else if (t - V.n < V.m) {
        t -= V.n;
        if (y_out) y_out[perm_r[t]] = (ra ? V.ysum[t] / w : V.y[cur][t]) / V.Dr[t];
    }
}

// ============================================================================ preconditioning (R1)
// A2 / A3: out[row] = sqrt(stat) with stat = max |v| (mode 0), sum |v| (mode 1) or sum |v|^p (mode 2),
// summed left to right; an empty row gives 1.
__global__ void __launch_bounds__(kBlock) k_row_stat(Sell A, int mode, double p, double* out) {
    const int lane = threadIdx.x & 31;
    const RowId r = my_row(A);
    if (r.row < 0) return;
    double s = 0.0;
    auto term = [&](double v) { double a = fabs(v); return mode == 2 ? (a > 0.0 ? pow(a, p) : 0.0) : a; };
    if (r.slice >= 0) {
        for (long long q = A.sp[r.slice] + lane; q < A.sp[r.slice + 1]; q += 32) {
            double a = term(A.val[q]);
            s = (mode == 0) ? fmax(s, a) : s + a;
        }
    } else {
        const long long b = A.lp[r.lrow], e = A.lp[r.lrow + 1];
        for (long long q0 = b; q0 < e; q0 += 32) {
            double a = (q0 + lane < e) ? term(A.lval[q0 + lane]) : 0.0;
            s = (mode == 0) ? fmax(s, warp_max(a)) : warp_seq_add(s, a);
        }
    }
    if (r.owner) out[r.row] = s > 0.0 ? sqrt(s) : 1.0;
}
// K~_ij <- K~_ij / (r_i * s_j): `own` is indexed by this layout's rows, `other` by its columns.  The
// product own*other is the same floating-point number in both layouts, so K~ and K~' stay bit-equal.
__global__ void __launch_bounds__(kBlock) k_scale_matrix(Sell A, const double* own, const double* other) {
    const int lane = threadIdx.x & 31;
    const RowId r = my_row(A);
    if (r.row < 0) return;
    if (r.slice >= 0) {
        const double o = r.owner ? own[r.row] : 1.0;
        const int cb = A.cbase[r.slice];
        for (long long q = A.sp[r.slice] + lane; q < A.sp[r.slice + 1]; q += 32) A.val[q] = A.val[q] / (o * other[sell_col(A, cb, q)]);
    } else {
        const double o = own[r.row];
        for (long long q = A.lp[r.lrow] + lane; q < A.lp[r.lrow + 1]; q += 32) A.lval[q] = A.lval[q] / (o * other[A.lcol[q]]);
    }
}
__global__ void k_vec_mul(double* d, const double* f, long long n) {
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n) d[t] *= f[t];
}
__global__ void k_vec_fill(double* d, double v, long long n) {
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n) d[t] = v;
}
// A4: scaled data.  b, c, l, u are device copies in the ORIGINAL order.
__global__ void __launch_bounds__(kBlock) k_scale_problem(long long n, long long m, const double* b, const double* c,
                                                          const double* l, const double* u, const char* sense,
                                                          const long long* perm_c, const long long* perm_r,
                                                          const double* Dr, const double* Dc, double* qs, double* cs,
                                                          double* ls, double* us, unsigned char* isG) {
    long long t = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (t < n) {
        const long long o = perm_c[t];
        cs[t] = c[o] / Dc[t];
        ls[t] = (l[o] <= -1e20) ? -INFINITY : l[o] * Dc[t];       // R13
        us[t] = (u[o] >= 1e20) ? INFINITY : u[o] * Dc[t];
    } else if (t - n < m) {
        t -= n;
        const long long o = perm_r[t];
        qs[t] = b[o] / Dr[t];
        isG[t] = sense[o] == 'G';
    }
}
__global__ void __launch_bounds__(kBlock) k_scale_bounds(long long n, const double* l, const double* u,
                                                         const long long* perm_c, const double* Dc, double* ls, double* us) {
    long long t = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (t < n) {
        const long long o = perm_c[t];
        ls[t] = (l[o] <= -1e20) ? -INFINITY : l[o] * Dc[t];
        us[t] = (u[o] >= 1e20) ? INFINITY : u[o] * Dc[t];
    }
}

__global__ void __launch_bounds__(kBlock) k_scale_cost(long long n, const double* c, const long long* perm_c, const double* Dc, double* cs) {
    long long t = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (t < n) cs[t] = c[perm_c[t]] / Dc[t];
}

// two-stage reductions for the one-time scalars of R2 / R9: op 0 = sum of squares (double-double),
// op 1 = max |v|
__global__ void __launch_bounds__(kBlock) k_reduce(const double* v, long long n, int op, dd* part) {
    __shared__ dd red[32];
    dd a[1] = {dd{0.0, 0.0}};
    double mx = 0.0;
    for (long long t = (long long)blockIdx.x * kBlock + threadIdx.x; t < n; t += (long long)gridDim.x * kBlock) {
        const double x = v[t];
        if (op) mx = fmax(mx, fabs(x)); else a[0] = dd_add_d(a[0], x * x);
    }
    if (op) {
        mx = warp_max(mx);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5].hi = mx;
        __syncthreads();
        if (threadIdx.x == 0) { for (int w = 1; w < kWarps; ++w) mx = fmax(mx, red[w].hi); part[blockIdx.x] = dd{mx, 0.0}; }
    } else {
        block_sum_dd<1>(a, red);
        if (threadIdx.x == 0) part[blockIdx.x] = a[0];
    }
}
__global__ void k_reduce_final(const dd* part, int count, int op, double* out) {     // one warp
    if (blockIdx.x != 0 || threadIdx.x >= 32) return;
    dd a = dd{0.0, 0.0};
    for (int i = threadIdx.x; i < count; i += 32) { if (op) a.hi = fmax(a.hi, part[i].hi); else a = dd_add(a, part[i]); }
    if (op) a.hi = warp_max(a.hi); else a = warp_sum_dd(a);
    if (threadIdx.x == 0) *out = dd_round(a);
}

// plain SpMV with the solver's traversal (test hook uc_lp_spmv)
__global__ void __launch_bounds__(kBlock) k_spmv(Sell A, const double* vec, double* out) {
    const int lane = threadIdx.x & 31;
    const RowId r = my_row(A);
    if (r.row < 0) return;
    double s[1] = {0.0};
    row_dot<1>(A, r, lane, s, [&](int c, double (&o)[1]) { o[0] = __ldg(vec + c); });
    if (r.owner) out[r.row] = s[0];
}
__global__ void k_gather(const double* src, const long long* perm, long long n, double* dst) {   // dst[new] = src[old]
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n) dst[t] = src[perm[t]];
}
__global__ void k_scatter(const double* src, const long long* perm, long long n, double* dst) {  // dst[old] = src[new]
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n) dst[perm[t]] = src[t];
}

}  // namespace ucpdhg
