// uc_attempt.cuh -- the two kernels of one PDHG attempt, sm_100a.
//
//   k_primal  (A5+A6+A10): g = K~'y ; x' = clamp(x - (eta/omega)(c - g), l, u) ; xbar = 2x' - x ;
//                          partial sum (x'-x)^2 ; deferred xsum += eta_prev x              (R3, R6)
//   k_dual    (A7+A8+A9+A10): r = K~ xbar ; y' = proj_Y(y + eta omega (q - r)) ; partial sums dy^2 and
//                          dy.(K~ dx) ; the last CTA finishes the three reductions and runs the
//                          step-size rule and the accept test                              (R3..R5)
//
// Both are HBM-bound streams (0.16 flop/B), so the design question is only how to keep ~45 KB per SM in
// flight with 3.4 entries per row.  Answer: persistent, warp-specialised CTAs, two per SM, each with
//   * one PRODUCER warp: for every tile (<= 8 slices = 256 rows, <= kCap stored entries) it issues 1-D
//     TMA bulk copies (cp.async.bulk ... mbarrier::complete_tx) of everything the tile streams -- the
//     column indices and values of its slices (one contiguous span of the sliced-ELL arrays) and the
//     256-row segments of the per-row vectors -- into a ring of kStages shared-memory stages, up to
//     kStages tiles ahead of the consumers;
//   * kCons CONSUMER warps: warp w owns slice w of the tile, one thread per row; it waits on the
//     stage's full-barrier, reads its operands from shared memory, gathers the other vector
//     (y, or the pair {xbar, dx}) from L2 with up to four loads in flight, forms the row sum left to
//     right, applies the update, stores coalesced, and releases the stage;
//   * one LONG-ROW warp: rows longer than the sliced-ELL threshold (the T reserve rows of the UC LP),
//     one row at a time, concurrently with the tile pipeline.
// Tiles are dealt round-robin (tile = blockIdx.x + i * gridDim.x).  Every thread keeps its
// double-double partial sums in registers across all its tiles; there is ONE block reduction per
// kernel, then one partial per CTA, and the last CTA to finish (ticket) adds the <= 2 * #SM partials.
//
// Arithmetic is unchanged from the sequential statement: row sums left to right in CSR order, multiply
// and add rounded separately (-fmad=false), long reductions in double-double (order-independent once
// rounded), see DESIGN.md "Numerics".
#pragma once
#include "uc_kernels.cuh"

namespace ucpdhg {

constexpr int kCons = 8;                       // consumer warps per CTA = slices per tile
constexpr int kAttemptThreads = (kCons + 2) * 32;   // + producer warp + long-row warp
constexpr int kStages = 3;                     // shared-memory stages per CTA
constexpr int kCap = 2048;                     // stored matrix entries one stage can hold
constexpr int kTileRows = kCons * 32;
constexpr int kCtasPerSm = 2;

// ------------------------------------------------------------------------------------------ PTX
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// 1-D TMA bulk copy global -> shared, completion counted in bytes on `bar`.  dst, src and bytes are
// multiples of 16.
__device__ __forceinline__ void tma_load(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fence_barrier_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

// ------------------------------------------------------------------------------------------ stage
struct StageHdr {
    long long span_base;     // first stored entry of the tile in the sliced-ELL arrays
    int first_slice, nslices, staged, pad;
    int woff[kCons + 1];     // entry offset of each slice inside the span
    int pad2;
};
static_assert(sizeof(StageHdr) == 64, "StageHdr layout");

template <int NVEC, bool BYTEVEC>
struct StageT {
    StageHdr hdr;
    int col[kCap];
    double val[kCap];
    double vec[NVEC][kTileRows];
    unsigned char bvec[BYTEVEC ? kTileRows : 16];
};
template <int NVEC, bool BYTEVEC>
struct PipeT {
    StageT<NVEC, BYTEVEC> st[kStages];
    uint64_t full[kStages], empty[kStages];
    dd red[2 * 32];
    int is_last;
};
using PrimalPipe = PipeT<5, false>;   // x, c, l, u, xsum
using DualPipe = PipeT<3, true>;      // y, q, ysum + isG

// ------------------------------------------------------------------------------------------ producer
// One warp.  For tile i of this CTA: wait until the consumers have released stage i % kStages, write the
// tile header, arm the full-barrier with the byte count and issue the bulk copies.  `vec_copies(stage,
// row0, rows, bar)` issues the per-row vector copies and returns their byte count.  The tile's slice
// pointers are loaded one tile ahead so that their latency hides behind the wait.
template <class Pipe, class VC>
__device__ __forceinline__ void producer_loop(const Sell& A, Pipe& P, int lane, VC vec_copies) {
    int t = blockIdx.x;
    int fs = 0, ns = 0; long long spv = 0;
    auto fetch = [&](int tile) {
        fs = __ldg(A.tile_ptr + tile); ns = __ldg(A.tile_ptr + tile + 1) - fs;
        spv = (lane <= ns) ? __ldg(A.sp + fs + lane) : 0;
    };
    if (t < A.ntiles) fetch(t);
    for (int i = 0; t < A.ntiles; ++i, t += gridDim.x) {
        const int s = i % kStages;
        const uint32_t ph = (uint32_t)(i / kStages) & 1u;
        const int cfs = fs, cns = ns; const long long cspv = spv;
        if (t + (int)gridDim.x < A.ntiles) fetch(t + gridDim.x);
        mbar_wait(&P.empty[s], ph ^ 1u);
        auto& S = P.st[s];
        const long long base = __shfl_sync(0xffffffffu, cspv, 0);
        const int span = (int)(__shfl_sync(0xffffffffu, cspv, cns) - base);
        const int staged = span <= kCap;
        if (lane <= cns) S.hdr.woff[lane] = (int)(cspv - base);
        if (lane == 0) { S.hdr.span_base = base; S.hdr.first_slice = cfs; S.hdr.nslices = cns; S.hdr.staged = staged; }
        __syncwarp();
        if (lane == 0) {
            const long long row0 = 32LL * cfs; const int rows = 32 * cns;
            uint32_t bytes = vec_copies(S, row0, rows, (uint64_t*)nullptr);       // count only
            if (staged) bytes += 12u * (uint32_t)span;
            mbar_expect_tx(&P.full[s], bytes);
            vec_copies(S, row0, rows, &P.full[s]);
            if (staged && span > 0) {
                tma_load(S.col, A.col + base, 4u * (uint32_t)span, &P.full[s]);
                tma_load(S.val, A.val + base, 8u * (uint32_t)span, &P.full[s]);
            }
        }
        __syncwarp();
    }
}

template <class Pipe>
__device__ __forceinline__ void pipe_init(Pipe& P) {
    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) { mbar_init(&P.full[s], 1); mbar_init(&P.empty[s], kCons); }
        fence_barrier_init();
    }
    __syncthreads();
}

// Row sum of one sliced-ELL row from (colp, valp) -- either the shared-memory stage or, for a tile that
// did not fit a stage, global memory -- entries t*32+lane, t = 0..width-1, left to right.  Four gathers
// are in flight at a time; slots past the width are not added.
template <int NV, class CP, class VP, class G>
__device__ __forceinline__ void slice_row(CP colp, VP valp, int width, int lane, double (&s)[NV], G gather) {
    for (int t = 0; t < width; t += 4) {
        int c[4]; double v[4]; double g[4][NV];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const bool ok = t + u < width;
            c[u] = ok ? colp[(t + u) * 32 + lane] : 0;
            v[u] = ok ? valp[(t + u) * 32 + lane] : 0.0;
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) gather(c[u], g[u]);
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (t + u < width) {
#pragma unroll
                for (int q = 0; q < NV; ++q) s[q] = __dadd_rn(s[q], __dmul_rn(v[u], g[u][q]));
            }
    }
}

// ----------------------------------------------------------------- A5+A6 (+A10): primal kernel
// One row j of K~' (= variable j): given g = (K~'y)_j, the R3 update and the R6 deferred average.
struct PrimalRow { double x, c, l, u, xs; };
__device__ __forceinline__ double primal_update(const Vecs& V, double* __restrict__ xnext, long long j, const PrimalRow& r,
                                                double g, double tau, int pend, double eta_prev) {
    if (pend) V.xsum[j] = r.xs + eta_prev * r.x;
    const double v = r.x - tau * (r.c - g);
    const double xn = v < r.l ? r.l : (v > r.u ? r.u : v);
    const double xb = 2.0 * xn - r.x;
    const double dx = xn - r.x;
    xnext[j] = xn;
    V.xg[j] = make_double2(xb, dx);
    return dx * dx;
}

__global__ void __launch_bounds__(kAttemptThreads, kCtasPerSm) k_primal(Sell KT, Vecs V, Ctrl* ctl) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    PrimalPipe& P = *reinterpret_cast<PrimalPipe*>(smem_raw);
    if (ld_flag(&ctl->done)) return;
    const int cur = ctl->cur, pend = ctl->pending;
    const double eta_prev = ctl->eta_prev, tau = ctl->eta / ctl->omega;
    const double* __restrict__ xcur = V.x[cur];
    const double* __restrict__ ycur = V.y[cur];
    double* __restrict__ xnext = V.x[cur ^ 1];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    pipe_init(P);
    dd acc[1] = {dd{0.0, 0.0}};

    if (warp == kCons) {                                   // ---- producer
        producer_loop(KT, P, lane, [&](auto& S, long long row0, int rows, uint64_t* bar) -> uint32_t {
            const uint32_t b = 8u * (uint32_t)rows;
            if (bar) {
                tma_load(S.vec[0], xcur + row0, b, bar);
                tma_load(S.vec[1], V.c + row0, b, bar);
                tma_load(S.vec[2], V.l + row0, b, bar);
                tma_load(S.vec[3], V.u + row0, b, bar);
                if (pend) tma_load(S.vec[4], V.xsum + row0, b, bar);
            }
            return (pend ? 5u : 4u) * b;
        });
    } else if (warp == kCons + 1) {                        // ---- long rows, one per pass
        for (int r = blockIdx.x; r < KT.nlong; r += gridDim.x) {
            const long long j = KT.nshort + r;
            PrimalRow pr{0.0, 0.0, 0.0, 0.0, 0.0};
            if (lane == 0) { pr.x = xcur[j]; pr.c = V.c[j]; pr.l = V.l[j]; pr.u = V.u[j]; if (pend) pr.xs = V.xsum[j]; }
            double g[1] = {0.0};
            long_row<1>(KT, r, lane, g, [&](int c, double (&o)[1]) { o[0] = __ldg(ycur + c); });
            if (lane == 0) acc[0] = dd_add_d(acc[0], primal_update(V, xnext, j, pr, g[0], tau, pend, eta_prev));
        }
    } else {                                               // ---- consumers: warp w owns slice w of each tile
        int t = blockIdx.x;
        for (int i = 0; t < KT.ntiles; ++i, t += gridDim.x) {
            const int s = i % kStages;
            mbar_wait(&P.full[s], (uint32_t)(i / kStages) & 1u);
            auto& S = P.st[s];
            if (warp < S.hdr.nslices) {
                const long long j = 32LL * (S.hdr.first_slice + warp) + lane;
                const int r = warp * 32 + lane;
                const int off = S.hdr.woff[warp], width = (S.hdr.woff[warp + 1] - off) >> 5;
                PrimalRow pr{S.vec[0][r], S.vec[1][r], S.vec[2][r], S.vec[3][r], pend ? S.vec[4][r] : 0.0};
                double g[1] = {0.0};
                auto gather = [&](int c, double (&o)[1]) { o[0] = __ldg(ycur + c); };
                if (S.hdr.staged) slice_row<1>(S.col + off, S.val + off, width, lane, g, gather);
                else slice_row<1>(KT.col + S.hdr.span_base + off, (const double*)KT.val + S.hdr.span_base + off, width, lane, g, gather);
                __syncwarp();
                if (lane == 0) mbar_arrive(&P.empty[s]);
                if (j < KT.nshort) acc[0] = dd_add_d(acc[0], primal_update(V, xnext, j, pr, g[0], tau, pend, eta_prev));
            } else {
                __syncwarp();
                if (lane == 0) mbar_arrive(&P.empty[s]);
            }
        }
    }
    block_sum_dd<1>(acc, P.red);
    if (threadIdx.x == 0) V.partA[blockIdx.x] = acc[0];
}

// ------------------------------------------------------------ A7+A8+A9 (+A10): dual kernel
struct DualRow { double y, q, ys; int isg; };
// kx[0] = (K~ xbar)_i, kx[1] = (K~ dx)_i.  Returns dy; the caller accumulates dy^2 and dy * kx[1].
__device__ __forceinline__ double dual_update(const Vecs& V, double* __restrict__ ynext, long long i, const DualRow& r,
                                              const double (&kx)[2], double sig, int pend, double eta_prev) {
    if (pend) V.ysum[i] = r.ys + eta_prev * r.y;
    const double v = r.y + sig * (r.q - kx[0]);
    const double yn = (r.isg && v < 0.0) ? 0.0 : v;
    ynext[i] = yn;
    return yn - r.y;
}

__global__ void __launch_bounds__(kAttemptThreads, kCtasPerSm) k_dual(Sell K, Vecs V, Ctrl* ctl) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    DualPipe& P = *reinterpret_cast<DualPipe*>(smem_raw);
    if (ld_flag(&ctl->done)) return;
    const int cur = ctl->cur, pend = ctl->pending;
    const double eta_prev = ctl->eta_prev, sig = ctl->eta * ctl->omega;
    const double* __restrict__ ycur = V.y[cur];
    double* __restrict__ ynext = V.y[cur ^ 1];
    const double2* __restrict__ xg = V.xg;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    pipe_init(P);
    dd acc[2] = {dd{0.0, 0.0}, dd{0.0, 0.0}};
    auto gather = [&](int c, double (&o)[2]) { const double2 t = __ldg(xg + c); o[0] = t.x; o[1] = t.y; };

    if (warp == kCons) {                                   // ---- producer
        producer_loop(K, P, lane, [&](auto& S, long long row0, int rows, uint64_t* bar) -> uint32_t {
            const uint32_t b = 8u * (uint32_t)rows;
            if (bar) {
                tma_load(S.vec[0], ycur + row0, b, bar);
                tma_load(S.vec[1], V.q + row0, b, bar);
                if (pend) tma_load(S.vec[2], V.ysum + row0, b, bar);
                tma_load(S.bvec, V.isG + row0, (uint32_t)rows, bar);
            }
            return (pend ? 3u : 2u) * b + (uint32_t)rows;
        });
    } else if (warp == kCons + 1) {                        // ---- long rows
        for (int r = blockIdx.x; r < K.nlong; r += gridDim.x) {
            const long long i = K.nshort + r;
            DualRow dr{0.0, 0.0, 0.0, 0};
            if (lane == 0) { dr.y = ycur[i]; dr.q = V.q[i]; dr.isg = V.isG[i]; if (pend) dr.ys = V.ysum[i]; }
            double kx[2] = {0.0, 0.0};
            long_row<2>(K, r, lane, kx, gather);
            if (lane == 0) {
                const double dy = dual_update(V, ynext, i, dr, kx, sig, pend, eta_prev);
                acc[0] = dd_add_d(acc[0], dy * dy); acc[1] = dd_add_d(acc[1], dy * kx[1]);
            }
        }
    } else {                                               // ---- consumers
        int t = blockIdx.x;
        for (int it = 0; t < K.ntiles; ++it, t += gridDim.x) {
            const int s = it % kStages;
            mbar_wait(&P.full[s], (uint32_t)(it / kStages) & 1u);
            auto& S = P.st[s];
            if (warp < S.hdr.nslices) {
                const long long i = 32LL * (S.hdr.first_slice + warp) + lane;
                const int r = warp * 32 + lane;
                const int off = S.hdr.woff[warp], width = (S.hdr.woff[warp + 1] - off) >> 5;
                DualRow dr{S.vec[0][r], S.vec[1][r], pend ? S.vec[2][r] : 0.0, (int)S.bvec[r]};
                double kx[2] = {0.0, 0.0};
                if (S.hdr.staged) slice_row<2>(S.col + off, S.val + off, width, lane, kx, gather);
                else slice_row<2>(K.col + S.hdr.span_base + off, (const double*)K.val + S.hdr.span_base + off, width, lane, kx, gather);
                __syncwarp();
                if (lane == 0) mbar_arrive(&P.empty[s]);
                if (i < K.nshort) {
                    const double dy = dual_update(V, ynext, i, dr, kx, sig, pend, eta_prev);
                    acc[0] = dd_add_d(acc[0], dy * dy); acc[1] = dd_add_d(acc[1], dy * kx[1]);
                }
            } else {
                __syncwarp();
                if (lane == 0) mbar_arrive(&P.empty[s]);
            }
        }
    }
    block_sum_dd<2>(acc, P.red);
    if (threadIdx.x == 0) { V.partB[blockIdx.x] = acc[0]; V.partB[V.gridPB + blockIdx.x] = acc[1]; }
    // ---- A9: the last CTA finishes the reductions and runs the step-size rule (R5)
    if (threadIdx.x == 0) {
        __threadfence();
        P.is_last = (atomicAdd(&ctl->ticket_b, 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (!P.is_last) return;
    const dd sdx = final_sum(V.partA, V.gridPA, P.red);
    const dd sdy = final_sum(V.partB, V.gridPB, P.red);
    const dd sin_ = final_sum(V.partB + V.gridPB, V.gridPB, P.red);
    if (threadIdx.x != 0) return;
    ctl->ticket_b = 0;
    const double dx2 = dd_round(sdx), dy2 = dd_round(sdy), inter = fabs(dd_round(sin_));
    const double eta = ctl->eta, omega = ctl->omega;
    const long long k = ctl->k + 1;
    const double N = omega * dx2 + dy2 / omega;
    const double eta_bar = (inter > 0.0) ? N / (2.0 * inter) : INFINITY;
    const double2 pw = ctl->powtab[k - 1];                   // {(k+1)^-0.6, (k+1)^-0.3}
    const double grow = (1.0 + pw.x) * eta;
    const double eta_next = isinf(eta_bar) ? grow : fmin((1.0 - pw.y) * eta_bar, grow);
    const int accept = eta <= eta_bar;
    if (ctl->att && k - 1 < ctl->att_cap) {
        uc_attempt_record rec;
        rec.eta_used = eta; rec.eta_bar = eta_bar; rec.eta_next = eta_next;
        rec.dx2 = dx2; rec.dy2 = dy2; rec.inter = inter; rec.accepted = accept; rec.pad_ = 0;
        ctl->att[k - 1] = rec;
    }
    if (accept) { ctl->cur = cur ^ 1; ctl->pending = 1; ctl->eta_prev = eta; ctl->w += eta; ctl->accepted += 1; }
    else ctl->pending = 0;
    ctl->eta = eta_next;
    ctl->k = k;
    if (!isfinite(eta_next) || !(eta_next > 0.0)) { ctl->status = UC_NUMERICAL_ERROR; ctl->done = 1; }
}

}  // namespace ucpdhg
