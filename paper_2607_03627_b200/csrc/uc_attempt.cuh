// uc_attempt.cuh -- the two kernels of one PDHG attempt, sm_100a.
//
//   k_primal  (A5+A6+A10): g = K~'y ; x' = clamp(x - (eta/omega)(c - g), l, u) ; xbar = 2x' - x ;
//                          partial sum (x'-x)^2 ; deferred xsum += eta_prev x              (R3, R6)
//   k_dual    (A7+A8+A9+A10): r = K~ xbar ; y' = proj_Y(y + eta omega (q - r)) ; partial sums dy^2 and
//                          dy.(K~ dx) ; the last CTA finishes the three reductions and runs the
//                          step-size rule and the accept test                              (R3..R5)
//
// Both stream rows with ~3.4 entries (0.16 flop/B), each entry needing an irregular 8/16-byte gather.  What bounds them
// is not DRAM and not instruction issue but the path between L2 and the SMs: every gather that misses L1 is its own L2
// request for a 32-byte sector (profiles/r02a: 5,900 B/cycle of L2 sectors chip-wide against a ~6,300 B/cycle ceiling,
// DRAM at 42-54 %; 17 % fewer instructions changed nothing).  What was measured on B200 (profiles/):
//   * a 1-D TMA bulk copy (cp.async.bulk) costs its issuing thread ~160 cycles whatever its size -- right for
//     16 KB tiles, hopeless for the 2 KB vector segments and ~1 KB value chunks this path is made of;
//   * a coalesced cp.async (LDGSTS.128) costs ~8 cycles and holds no register while in flight;
//   * an asynchronous copy whose shared-memory destination is not aligned like its global source fetches every global
//     sector twice (hence the 128-byte data slots);
//   * a gather that allocates in L1 (cp.async.ca) pays off once a CTA sweeps a CONTIGUOUS range of rows: neighbouring
//     rows gather from the same few blocks of the vector (uc_format.hpp build_schedule).
// Hence: persistent CTAs (one per SM) of up to 15 CONSUMER warps, every one of which runs its own three-stage software
// pipeline on its own shared-memory data slots, with NO block-level synchronisation inside the loop.  The unit of work
// is a STEP (uc_format.hpp): up to kChunkT entries per row of one slice (32 rows, one per lane).  In the iteration
// that computes step j a warp also issues
//     A(j + DB + 2): plain loads of the step's column indices into REGISTERS (2 or 4 bytes per lane and entry)
//     B(j + DB):     cp.async of the step's matrix values, of the 32-row segments of the per-row vectors (last step of a
//                    slice only) and, with the indices A brought in, one 8/16-byte cp.async per stored entry e:
//                    gv[e] <- src[col[e]]  (the entry of y, or of the pair {xbar, dx}, that e multiplies)  -> data slots
//     C(j):          everything read from shared memory: row sums left to right, update, coalesced stores.
// One cp.async group is committed per step; cp.async.wait_group DB + __syncwarp is the only wait.  A slice wider than
// kChunkT is a run of consecutive steps whose row sums stay in registers.  The schedule (a contiguous range of slices
// per CTA, dealt inside the CTA to the least-loaded warp, built at create time) is static, so a solve is reproducible bit
// for bit.  One extra warp per CTA takes the rows longer than the sliced-ELL threshold (the T reserve rows of the UC
// LP), one row at a time, concurrently.
// L2 policy: streamed-once data is loaded (cp.async.cg / ld.global.nc.L1::no_allocate) and stored evict_first; the
// gathered vectors (y', {xbar, dx}) are stored evict_last so that the gathers of the NEXT kernel hit in the 126 MB L2.
// Every thread keeps its double-double partial sums in registers across all its steps; there is ONE block reduction
// per kernel, then one partial per CTA; warp 0 of the last CTA to finish (ticket) adds the <= #SM partials with
// shuffles only and runs the step rule on scalars parked in shared memory while the kernel started (the serial tail
// of every attempt: DESIGN.md section 7, profiles/r02c_timeline.md).
//
// Arithmetic is unchanged from the sequential statement: row sums left to right in CSR order, multiply
// and add rounded separately (-fmad=false), long reductions in double-double (order-independent once
// rounded), see DESIGN.md "Numerics".
#pragma once
#include "uc_kernels.cuh"

namespace ucpdhg {

// build-time tunables (-DUC_...): the defaults are the measured optimum on config 3 (profiles/)
#ifndef UC_PRIMAL_WARPS
#define UC_PRIMAL_WARPS 15     // consumer warps per CTA of k_primal
#endif
#ifndef UC_DUAL_WARPS
#define UC_DUAL_WARPS 15       // consumer warps per CTA of k_dual
#endif
#ifndef UC_CTAS_PER_SM
#define UC_CTAS_PER_SM 1
#endif
#ifndef UC_DB
#define UC_DB 1
#endif
#ifndef UC_MIN_WARPS
#define UC_MIN_WARPS 4
#endif
// consumer warps per CTA: the most a CTA may have (the rings of that many are laid out in shared memory).  A handle
// launches fewer when its LP has fewer than #SM x that many slices (uc_lp_create: attempt_shape), down to kMinWarps: on
// small LPs a warp has one slice or none, and every extra warp only lengthens the block barrier of the serial tail.
constexpr int kPrimalWarps = UC_PRIMAL_WARPS, kDualWarps = UC_DUAL_WARPS, kMinWarps = UC_MIN_WARPS;
constexpr int kCtasPerSm = UC_CTAS_PER_SM;
constexpr int kPrimalThreads = (kPrimalWarps + 1) * 32, kDualThreads = (kDualWarps + 1) * 32;   // + long-row warp
// pipeline depth, per kernel: the data copies (values, vectors, gathers) run DB steps ahead of the compute (DB + 1 data
// slots; 1 or 3), the index loads DB + 2 steps ahead.  DB = 3 was measured slower: it takes the L1 the gathers live on.
#ifndef UC_PRIMAL_DB
#define UC_PRIMAL_DB UC_DB
#endif
#ifndef UC_DUAL_DB
#define UC_DUAL_DB UC_DB
#endif
constexpr int kChunkE = kChunkT * 32;          // stored entries per step

// ------------------------------------------------------------------------------------------ PTX
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
// L2 eviction policies (createpolicy): streamed-once data leaves L2 first, gathered vectors last
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t p; asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p)); return p;
}
__device__ __forceinline__ uint64_t policy_evict_last() {
    uint64_t p; asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p)); return p;
}
// asynchronous global -> shared copies (LDGSTS): no destination register; completion per thread, by group.
// 16-byte streaming copy, L1 bypass, evict_first in L2
__device__ __forceinline__ void cp_stream16(void* dst, const void* src, uint64_t pol) {
    asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" ::"r"(smem_u32(dst)), "l"(src), "l"(pol) : "memory");
}
// 8 / 16-byte gather
__device__ __forceinline__ void cp_gather(double* dst, const double* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_gather(double2* dst, const double2* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");   // L1 bypass: measured faster
}
// Predicated forms: the comparison `a < b` becomes a predicate on the copy itself.  The conditions below are warp-uniform
// functions of the step descriptor, but the compiler cannot know that (the descriptor comes out of a shuffle), so an
// `if` around a copy costs a BSSY / BRA / BSYNC triple; the loop is bound by instruction issue latency at 4 warps per
// scheduler (profiles/r02a), so every instruction on a warp's dependent chain counts.
__device__ __forceinline__ void cp_stream16_lt(int a, int b, void* dst, const void* src, uint64_t pol) {
    asm volatile("{\n\t.reg .pred q;\n\tsetp.lt.s32 q, %0, %1;\n\t@q cp.async.cg.shared.global.L2::cache_hint [%2], [%3], 16, %4;\n\t}"
                 ::"r"(a), "r"(b), "r"(smem_u32(dst)), "l"(src), "l"(pol) : "memory");
}
__device__ __forceinline__ void cp_gather_lt(int a, int b, double* dst, const double* src) {
    asm volatile("{\n\t.reg .pred q;\n\tsetp.lt.s32 q, %0, %1;\n\t@q cp.async.ca.shared.global [%2], [%3], 8;\n\t}"
                 ::"r"(a), "r"(b), "r"(smem_u32(dst)), "l"(src) : "memory");
}
#ifndef UC_DUAL_GATHER
#define UC_DUAL_GATHER "ca"
#endif
__device__ __forceinline__ void cp_gather_lt(int a, int b, double2* dst, const double2* src) {
    asm volatile("{\n\t.reg .pred q;\n\tsetp.lt.s32 q, %0, %1;\n\t@q cp.async." UC_DUAL_GATHER ".shared.global [%2], [%3], 16;\n\t}"
                 ::"r"(a), "r"(b), "r"(smem_u32(dst)), "l"(src) : "memory");
}
// column index of a stored entry, straight into a register (streamed once: no L1 allocation), only if a < b; `v` keeps
// its old value otherwise (never used: the gather it would feed carries the same predicate)
__device__ __forceinline__ void ld_index_lt(int a, int b, int& v, const unsigned short* p) {
    // a 16-bit load may name a 32-bit destination (zero-extended): one predicated LDG, nothing that depends on it here
    asm("{\n\t.reg .pred q;\n\tsetp.lt.s32 q, %1, %2;\n\t@q ld.global.nc.L1::no_allocate.u16 %0, [%3];\n\t}"
        : "+r"(v) : "r"(a), "r"(b), "l"(p));
}
__device__ __forceinline__ void ld_index_lt(int a, int b, int& v, const int* p) {
    asm("{\n\t.reg .pred q;\n\tsetp.lt.s32 q, %1, %2;\n\t@q ld.global.nc.L1::no_allocate.s32 %0, [%3];\n\t}"
        : "+r"(v) : "r"(a), "r"(b), "l"(p));
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void st_hint(double* p, double v, uint64_t pol) {
    asm volatile("st.global.L2::cache_hint.f64 [%0], %1, %2;" ::"l"(p), "d"(v), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_hint(double2* p, double2 v, uint64_t pol) {
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}
struct Policies { uint64_t first, last; };

// ------------------------------------------------------------------------------------------ per-warp rings
// GT: what one entry gathers -- double (y) or double2 ({xbar, dx}).  Everything in here is private to ONE warp.
// A slot is a multiple of 128 bytes: an asynchronous copy whose shared-memory destination is not aligned like its global
// source (16 bytes off, as the second slot of the primal ring was) is split at the shared-memory sector boundaries and
// fetches every 32-byte global sector TWICE (profiles/r02b: 2.2 M of 6.6 M L2 sectors of the streamed data per launch).
template <int NVEC, bool BYTEVEC, class GT>
struct alignas(128) DataSlot {
    double val[kChunkE];
    GT gv[kChunkE];              // gv[e] = gathered vector entry for stored entry e
    double vec[NVEC][32];        // 32-row segments of the per-row vectors (last step of a slice only)
    unsigned char bvec[BYTEVEC ? 32 : 16];
};
// DB = how many steps the data copies run ahead of the compute: 1 (two slots) or 3 (four slots); the slot of step s
// is s & (kSlots - 1), a compile-time constant in the loop below (unrolled by four)
template <int NVEC, bool BYTEVEC, class GT, int DB>
struct WarpRing {
    static_assert(DB == 1 || DB == 3, "data ring: 2 or 4 slots");
    static constexpr int kDB = DB, kSlots = DB + 1;
    DataSlot<NVEC, BYTEVEC, GT> data[kSlots];
};
template <int NVEC, bool BYTEVEC, class GT, int WARPS, int DB>
struct SmemT {
    WarpRing<NVEC, BYTEVEC, GT, DB> w[WARPS];
    dd red[2 * 32];
};
using PrimalSmem = SmemT<5, false, double, kPrimalWarps, UC_PRIMAL_DB>;   // x, c, l, u, xsum ; gathers y
using DualSmem = SmemT<3, true, double2, kDualWarps, UC_DUAL_DB>;         // y, q, ysum + isG ; gathers {xbar, dx}
constexpr size_t kPrimalSmemBytes = sizeof(PrimalSmem), kDualSmemBytes = sizeof(DualSmem);
static_assert(kCtasPerSm * (kPrimalSmemBytes + 1024) <= 228 * 1024 && kCtasPerSm * (kDualSmemBytes + 1024) <= 228 * 1024,
              "the CTAs of either attempt kernel must fit the shared memory of one SM");

// Calls f(std::integral_constant<int, nt>) for nt = 1..kChunkT (nothing for nt = 0).  nt is warp-uniform, so
// the branch does not diverge and each case is straight-line code without predicated-off instructions.
template <int N> struct IntC { static constexpr int value = N; };
template <class F>
__device__ __forceinline__ void dispatch_nt(int nt, F f) {
    static_assert(kChunkT == 4, "dispatch_nt covers 1..4");
    switch (nt) {
        case 1: f(IntC<1>{}); break;
        case 2: f(IntC<2>{}); break;
        case 3: f(IntC<3>{}); break;
        case 4: f(IntC<4>{}); break;
        default: break;
    }
}

// ------------------------------------------------------------------------------------------ the pipeline
// Runs the steps of consumer warp `gw` (of A.sched_warps) through a three-stage software pipeline.  In the iteration
// that computes step j the warp also issues
//     A(j + DB + 2): plain loads of the step's column indices into REGISTERS (coalesced, 2 or 4 bytes per lane and
//                    entry; they are consumed two iterations later, so their latency is off the dependent chain)
//     B(j + DB):     cp.async of the step's matrix values, of the 32-row segments of the per-row vectors (last step
//                    of a slice only) and one 8/16-byte cp.async per stored entry, gv[e] <- src[col[e]]  -> data ring
//     C(j):          everything read from shared memory: row sums left to right, update, coalesced stores.
//   issue_vecs(slot, row0, last01)  issues the cp.async copies of the 32-row vector segments of a slice
//   compute(slot, info, row0)       consumes one step from shared memory
// The loop is unrolled by four with every ring slot and queue position a compile-time constant: the kernel is bound by
// instruction issue latency (4 warps per scheduler, each a long dependent chain), so the bookkeeping of a step --
// queue rotation, slot wrap-around, address arithmetic -- was as expensive as its arithmetic before (profiles/r02a:
// 252 SASS instructions per step, 19 of them register moves at the loop head).
// The schedule is read 32 steps at a time (lane l holds step 32 b + l of the warp; the next batch is loaded one batch
// ahead) and handed from stage to stage in registers.
// dep_ready() is called once, just before the first B stage: everything before it (schedule loads, the first index
// loads) touches only data that no kernel writes, so it overlaps the tail of the previous kernel (programmatic
// dependent launch); it returns false if the solve is already over.
template <class Ring, class GT, class FD, class FV, class FC>
__device__ __forceinline__ bool warp_pipeline(const Sell& A, Ring& R, int gw, int lane, const GT* const& gsrc,
                                              uint64_t pol_first, FD dep_ready, FV issue_vecs, FC compute) {
    constexpr int DB = Ring::kDB, NS = Ring::kSlots, DA = DB + 2;
    int J = A.steps_per_warp;                                      // shrinks to this warp's own count at its end marker
    const long long GW = A.sched_warps;
    auto load_desc = [&](int k) -> int4 {
        return k < J ? __ldg(reinterpret_cast<const int4*>(A.steps + (long long)k * GW + gw)) : make_int4(0, 0, -1, 0);
    };
    int4 dcur = load_desc(lane), dnxt = load_desc(32 + lane);
    // A -> B, position = step & 3: descriptor fields and the column indices of the lane's entries
    int q_info[4] = {0, 0, 0, 0}, q_row[4] = {0, 0, 0, 0}, q_cb[4] = {-1, -1, -1, -1}, q_idx[4][kChunkT];
    unsigned q_eb[4] = {0u, 0u, 0u, 0u};
#pragma unroll
    for (int q = 0; q < 4; ++q)
#pragma unroll
        for (int t = 0; t < kChunkT; ++t) q_idx[q][t] = 0;
    // B -> C, position = data slot
    int c_info[NS], c_row[NS];
#pragma unroll
    for (int q = 0; q < NS; ++q) { c_info[q] = 0; c_row[q] = 0; }

    // one iteration; P = j & 3 at compile time; PRO: prologue (no compute, stages of negative steps skipped)
    auto body = [&](auto Pc, auto PROc, const int j) {
        constexpr int P = decltype(Pc)::value;
        constexpr bool PRO = decltype(PROc)::value != 0;
        // ---- A: column indices of step sa = j + DA
        const int sa = j + DA;
        if (!PRO || sa >= 0) {
            constexpr int qa = (P + DA) & 3;
            if constexpr (qa == 0 && !PRO) {                      // sa is a multiple of 4 here: a batch may begin
                if ((sa & 31) == 0) { dcur = dnxt; dnxt = load_desc(sa + 32 + lane); }
            }
            const int src_lane = sa & 31;
            const unsigned w0 = (unsigned)__shfl_sync(0xffffffffu, dcur.x, src_lane);
            const int row_a = __shfl_sync(0xffffffffu, dcur.y, src_lane);
            const int cb_a = __shfl_sync(0xffffffffu, dcur.z, src_lane);   // >= 0: 16-bit offsets from cb_a (uc_format.hpp)
            const int info_a = (int)(w0 >> 26), nt = info_a & 7;
            const unsigned eb32 = w0 & 0x3ffffffu;                          // first stored entry of the step / 32
            if (info_a & kStepEnd) J = min(J, sa);
            q_info[qa] = info_a; q_row[qa] = row_a; q_cb[qa] = cb_a < 0 ? 0 : cb_a; q_eb[qa] = eb32;
            const long long e0 = ((long long)eb32 << 5) + lane;
            UC_BOUNDS_ASSERT(nt <= kChunkT && ((long long)eb32 << 5) + 32LL * nt <= A.nslots && row_a >= 0 && row_a <= A.nshort + 31 && (row_a & 31) == 0);
            UC_BOUNDS_ASSERT(nt == 0 || (cb_a >= 0 ? A.col16 != nullptr : A.col != nullptr));
            if (cb_a >= 0) {
                const unsigned short* p = A.col16 + e0;
#pragma unroll
                for (int t = 0; t < kChunkT; ++t) ld_index_lt(t, nt, q_idx[qa][t], p + 32 * t);
            } else {
                const int* p = A.col + e0;
#pragma unroll
                for (int t = 0; t < kChunkT; ++t) ld_index_lt(t, nt, q_idx[qa][t], p + 32 * t);
            }
        }
        // ---- B: values, vectors and gathers of step sb = j + DB
        const int sb = j + DB;
        if (!PRO || sb >= 0) {
            constexpr int qb = (P + DB) & 3, db = (P + DB) & (NS - 1);
            const int info_b = q_info[qb], row_b = q_row[qb], nt = info_b & 7;
            auto& D = R.data[db];
            const double* vsrc = A.val + ((long long)q_eb[qb] << 5);
#pragma unroll
            for (int k = 0; k < kChunkT / 2; ++k) {
                const int p = k * 32 + lane;                       // 16-byte piece of the value chunk
                cp_stream16_lt(p, nt * 16, &D.val[p * 2], vsrc + p * 2, pol_first);
            }
            issue_vecs(D, row_b, (info_b >> 4) & 1);               // kStepLast
            const GT* gs = gsrc + q_cb[qb];
#pragma unroll
            for (int t = 0; t < kChunkT; ++t) {
                UC_BOUNDS_ASSERT(t >= nt || (q_cb[qb] + q_idx[qb][t] >= 0 && (long long)q_cb[qb] + q_idx[qb][t] < A.ncols));
                cp_gather_lt(t, nt, &D.gv[t * 32 + lane], gs + q_idx[qb][t]);
            }
            c_info[db] = info_b; c_row[db] = row_b;
            cp_commit();
        }
        // ---- C: step j
        if constexpr (!PRO) {
            constexpr int dc = P & (NS - 1);
            cp_wait<DB>();
            __syncwarp();                                          // the copies of every lane are visible to the warp
            if (c_info[dc]) compute(R.data[dc], c_info[dc], c_row[dc]);
            __syncwarp();                                          // the slot is rewritten by the next iteration's copies
        }
    };
    static_assert(kStepLast == 16, "issue_vecs takes bit 4 of the step info");
    constexpr int kPro = (DA + 3) & ~3;                            // prologue iterations (a multiple of four)
    bool live = true;
#pragma unroll
    for (int i = 0; i < kPro; ++i) {
        const int j = i - kPro;
        if (j == -DB) { live = dep_ready(); if (!live) break; }
        switch (i & 3) {
            case 0: body(IntC<0>{}, IntC<1>{}, j); break;
            case 1: body(IntC<1>{}, IntC<1>{}, j); break;
            case 2: body(IntC<2>{}, IntC<1>{}, j); break;
            default: body(IntC<3>{}, IntC<1>{}, j); break;
        }
    }
    if (!live) { cp_wait<0>(); return false; }
    for (int j = 0; j < J; j += 4) {
        body(IntC<0>{}, IntC<0>{}, j);
        body(IntC<1>{}, IntC<0>{}, j + 1);
        body(IntC<2>{}, IntC<0>{}, j + 2);
        body(IntC<3>{}, IntC<0>{}, j + 3);
    }
    cp_wait<0>();
    return true;
}

// Programmatic dependent launch (PDL): the next kernel in the stream may start its prologue as soon as every
// CTA of this one has passed grid_launch_dependents(); grid_dependency_wait() returns once the previous kernel
// has completed and its writes are visible.
__device__ __forceinline__ void grid_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void grid_dependency_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// Row sum contribution of one step: entries t*32+lane of the slot, t = 0..nt-1, left to right.
template <int NV, class GT>
__device__ __forceinline__ void step_sum(const double* valp, const GT* gvp, int nt, int lane, double (&s)[NV]) {
    dispatch_nt(nt, [&](auto n) {
        constexpr int N = decltype(n)::value;
        double v[N]; GT g[N];
#pragma unroll
        for (int t = 0; t < N; ++t) { v[t] = valp[t * 32 + lane]; g[t] = gvp[t * 32 + lane]; }
#pragma unroll
        for (int t = 0; t < N; ++t) {
            if constexpr (NV == 1) s[0] = __dadd_rn(s[0], __dmul_rn(v[t], g[t]));
            else { s[0] = __dadd_rn(s[0], __dmul_rn(v[t], g[t].x)); s[1] = __dadd_rn(s[1], __dmul_rn(v[t], g[t].y)); }
        }
    });
}

// ----------------------------------------------------------------- A5+A6 (+A10): primal kernel
// One row j of K~' (= variable j): given g = (K~'y)_j, the R3 update and the R6 deferred average.
struct PrimalRow { double x, c, l, u, xs; };
__device__ __forceinline__ double primal_update(const Vecs& V, double* __restrict__ xnext, long long j, const PrimalRow& r,
                                                double g, double tau, int pend, double eta_prev, const Policies& pol) {
    if (pend) st_hint(V.xsum + j, r.xs + eta_prev * r.x, pol.first);
    const double v = r.x - tau * (r.c - g);
    const double xn = v < r.l ? r.l : (v > r.u ? r.u : v);
    const double xb = 2.0 * xn - r.x;
    const double dx = xn - r.x;
    st_hint(xnext + j, xn, pol.first);
    st_hint(V.xg + j, make_double2(xb, dx), pol.last);      // gathered by the next k_dual: keep it in L2
    return dx * dx;
}

__global__ void __launch_bounds__(kPrimalThreads, kCtasPerSm) k_primal(Sell KT, Vecs V, Ctrl* ctl) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    PrimalSmem& P = *reinterpret_cast<PrimalSmem*>(smem_raw);
    dd* const red = P.red;
    UC_TL_MARK(V, 0);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    dd acc[1] = {dd{0.0, 0.0}};
    const Policies pol{policy_evict_first(), policy_evict_last()};
    // everything below is set by dep_ready(), i.e. read after the previous kernel has completed
    int pend = 0; double eta_prev = 0.0, tau = 0.0;
    const double* xcur = nullptr; const double* ycur = nullptr; double* xnext = nullptr;
    const double* vsrc[3]; int voff[3]; int vkey[3];   // this lane's share of a slice's vector segments: piece k covers
                                                       // vector v = 2k + lane/16, doubles off, off+1; vkey 0: copy it
    auto dep_ready = [&]() -> bool {
        grid_dependency_wait();
        // only now may the next k_dual start: the k_dual before this kernel has completed, so the control block it left
        // is final and the next k_dual may read it BEFORE its own dependency (this kernel) resolves
        grid_launch_dependents();
        UC_TL_MARK(V, 1);
        const CtrlHot h = load_hot(ctl);
        if (h.done) return false;
        const int cur = h.cur;
        pend = h.pending; eta_prev = h.eta_prev; tau = h.eta / h.omega;
        xcur = V.x[cur]; ycur = V.y[cur]; xnext = V.x[cur ^ 1];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const int v = 2 * k + (lane >> 4), off = (lane & 15) * 2;
            vsrc[k] = (v == 0 ? xcur : v == 1 ? V.c : v == 2 ? V.l : v == 3 ? V.u : V.xsum) + off;
            voff[k] = v * 32 + off; vkey[k] = (v < 4 || (v == 4 && pend)) ? 0 : 1;
        }
        return true;
    };

    if (warp == KT.cta_warps) {                               // ---- long rows, one per pass
        if (!dep_ready()) return;
        for (int r = blockIdx.x; r < KT.nlong; r += gridDim.x) {
            const long long j = KT.nshort + r;
            PrimalRow pr{0.0, 0.0, 0.0, 0.0, 0.0};
            if (lane == 0) { pr.x = xcur[j]; pr.c = V.c[j]; pr.l = V.l[j]; pr.u = V.u[j]; if (pend) pr.xs = V.xsum[j]; }
            double g[1] = {0.0};
            long_row<1>(KT, r, lane, g, [&](int c, double (&o)[1]) { o[0] = __ldg(ycur + c); });
            if (lane == 0) acc[0] = dd_add_d(acc[0], primal_update(V, xnext, j, pr, g[0], tau, pend, eta_prev, pol));
        }
    } else {                                               // ---- consumer warps
        double g[1] = {0.0};
        const bool live = warp_pipeline(KT, P.w[warp], (int)blockIdx.x * KT.cta_warps + warp, lane, ycur, pol.first, dep_ready,
            [&](auto& D, int row0, int last01) {           // x, c, l, u (, xsum): 16 pieces of 16 bytes each
#pragma unroll
                for (int k = 0; k < 3; ++k) cp_stream16_lt(vkey[k], last01, &D.vec[0][0] + voff[k], vsrc[k] + row0, pol.first);
            },
            [&](auto& D, int info, int row0) {
                if (info & kStepFirst) g[0] = 0.0;
                step_sum<1>(D.val, D.gv, info & 7, lane, g);
                if (info & kStepLast) {
                    const long long j = (long long)row0 + lane;
                    if (j < KT.nshort) {
                        const PrimalRow pr{D.vec[0][lane], D.vec[1][lane], D.vec[2][lane], D.vec[3][lane], pend ? D.vec[4][lane] : 0.0};
                        acc[0] = dd_add_d(acc[0], primal_update(V, xnext, j, pr, g[0], tau, pend, eta_prev, pol));
                    }
                }
            });
        if (!live) return;
    }
    UC_TL_MARK(V, 2);
    if (!block_sum_dd_warp0<1>(acc, red)) return;           // the other warps leave; warp 0 finishes the CTA's partial
    if (lane == 0) V.partA[blockIdx.x] = acc[0];
    UC_TL_MARK(V, 3);
}

// ------------------------------------------------------------ A7+A8+A9 (+A10): dual kernel
struct DualRow { double y, q, ys; int isg; };
// kx[0] = (K~ xbar)_i, kx[1] = (K~ dx)_i.  Returns dy; the caller accumulates dy^2 and dy * kx[1].
__device__ __forceinline__ double dual_update(const Vecs& V, double* __restrict__ ynext, long long i, const DualRow& r,
                                              const double (&kx)[2], double sig, int pend, double eta_prev, const Policies& pol) {
    if (pend) st_hint(V.ysum + i, r.ys + eta_prev * r.y, pol.first);
    const double v = r.y + sig * (r.q - kx[0]);
    const double yn = (r.isg && v < 0.0) ? 0.0 : v;
    st_hint(ynext + i, yn, pol.last);                       // gathered by the next k_primal: keep it in L2
    return yn - r.y;
}

__global__ void __launch_bounds__(kDualThreads, kCtasPerSm) k_dual(Sell K, Vecs V, Ctrl* ctl) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    DualSmem& P = *reinterpret_cast<DualSmem*>(smem_raw);
    dd* const red = P.red;
    grid_launch_dependents();
    UC_TL_MARK(V, 0);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    dd acc[2] = {dd{0.0, 0.0}, dd{0.0, 0.0}};
    const Policies pol{policy_evict_first(), policy_evict_last()};
    const double2* xg = V.xg;
    int cur = 0, pend = 0; double eta_prev = 0.0, sig = 0.0;
    const double* ycur = nullptr; double* ynext = nullptr;
    const double* vsrc[2]; int voff[2]; int vkey[2];   // this lane's share of a slice's vector segments (vkey 0: copy it)
    const int bkey = (lane == 16 || lane == 17) ? 0 : 1;
    // inputs of the step rule (A9), fetched by one thread of every CTA while the kernel starts and parked in shared
    // memory: whichever CTA finishes last then runs the rule without a single cold load on the critical path of the
    // whole solve
    struct RuleIn { double eta, omega, w; long long k, acc, cap; double2 pw; uc_attempt_record* att; };
    __shared__ RuleIn rule_in;
    // The control block is read HERE, before the dependency on k_primal resolves: k_primal does not write it, and the
    // k_dual that did has completed (k_primal lets this kernel start only after its own dependency resolved).  One L2
    // round trip less on the serial path of every attempt.
    const CtrlHot h = load_hot(ctl);
    cur = h.cur; pend = h.pending; eta_prev = h.eta_prev; sig = h.eta * h.omega;
    if (threadIdx.x == K.cta_warps * 32 && !h.done) {      // the long-row warp: its dependent loads delay no slice
        RuleIn r;
        r.eta = h.eta; r.omega = h.omega; r.w = h.w; r.k = ctl->k; r.acc = ctl->accepted;
        r.att = ctl->att; r.cap = ctl->att_cap; r.pw = ctl->powtab[r.k];     // {(k+1)^-0.6, (k+1)^-0.3} of attempt k = r.k + 1
        rule_in = r;
    }
    ycur = V.y[cur]; ynext = V.y[cur ^ 1];
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        const int v = 2 * k + (lane >> 4), off = (lane & 15) * 2;
        vsrc[k] = (v == 0 ? ycur : v == 1 ? V.q : V.ysum) + off;
        voff[k] = v * 32 + off; vkey[k] = (v < 2 || (v == 2 && pend)) ? 0 : 1;
    }
    const bool solve_over = h.done != 0;
    auto dep_ready = [&]() -> bool {
        grid_dependency_wait();
        UC_TL_MARK(V, 1);
        return !solve_over;
    };

    if (warp == K.cta_warps) {                              // ---- long rows
        if (!dep_ready()) return;
        auto gather = [&](int c, double (&o)[2]) { const double2 t = __ldg(xg + c); o[0] = t.x; o[1] = t.y; };
        for (int r = blockIdx.x; r < K.nlong; r += gridDim.x) {
            const long long i = K.nshort + r;
            DualRow dr{0.0, 0.0, 0.0, 0};
            if (lane == 0) { dr.y = ycur[i]; dr.q = V.q[i]; dr.isg = V.isG[i]; if (pend) dr.ys = V.ysum[i]; }
            double kx[2] = {0.0, 0.0};
            long_row<2>(K, r, lane, kx, gather);
            if (lane == 0) {
                const double dy = dual_update(V, ynext, i, dr, kx, sig, pend, eta_prev, pol);
                acc[0] = dd_add_d(acc[0], dy * dy); acc[1] = dd_add_d(acc[1], dy * kx[1]);
            }
        }
    } else {                                               // ---- consumer warps
        double kx[2] = {0.0, 0.0};
        const bool live = warp_pipeline(K, P.w[warp], (int)blockIdx.x * K.cta_warps + warp, lane, xg, pol.first, dep_ready,
            [&](auto& D, int row0, int last01) {           // y, q (, ysum): 16 pieces each; isG: 2 pieces
#pragma unroll
                for (int k = 0; k < 2; ++k) cp_stream16_lt(vkey[k], last01, &D.vec[0][0] + voff[k], vsrc[k] + row0, pol.first);
                cp_stream16_lt(bkey, last01, &D.bvec[(lane & 1) * 16], V.isG + row0 + (lane & 1) * 16, pol.first);
            },
            [&](auto& D, int info, int row0) {
                if (info & kStepFirst) { kx[0] = 0.0; kx[1] = 0.0; }
                step_sum<2>(D.val, D.gv, info & 7, lane, kx);
                if (info & kStepLast) {
                    const long long i = (long long)row0 + lane;
                    if (i < K.nshort) {
                        const DualRow dr{D.vec[0][lane], D.vec[1][lane], pend ? D.vec[2][lane] : 0.0, (int)D.bvec[lane]};
                        const double dy = dual_update(V, ynext, i, dr, kx, sig, pend, eta_prev, pol);
                        acc[0] = dd_add_d(acc[0], dy * dy); acc[1] = dd_add_d(acc[1], dy * kx[1]);
                    }
                }
            });
        if (!live) return;
    }
    UC_TL_MARK(V, 2);
    // ---- A9: the last CTA finishes the reductions and runs the step-size rule (R5).  This is the serial tail of
    // every attempt (timeline of profiles/r02b: 6.7 us of 85 on config 3 before this form), so it is ONE warp, with every
    // wait it contains taken once: the other warps only arrive at the block barrier and leave; the CTA's partials are
    // published by the release half of the ticket (no separate fence); the last CTA's warp fetches all partials of all
    // CTAs in one round trip before it adds any; no cold load: the rule's inputs were parked in shared memory.
    if (!block_sum_dd_warp0<2>(acc, red)) return;
    UC_TL_MARK(V, 3);
    unsigned last = 0;
    if (lane == 0) {
        V.partB[blockIdx.x] = acc[0]; V.partB[V.gridPB + blockIdx.x] = acc[1];
        unsigned old;
        asm volatile("atom.add.acq_rel.gpu.global.u32 %0, [%1], 1;" : "=r"(old) : "l"(&ctl->ticket_b) : "memory");
        last = old == gridDim.x - 1;
    }
    UC_TL_MARK(V, 4);
    if (!__shfl_sync(0xffffffffu, last, 0)) return;
    dd s3[3] = {dd{0.0, 0.0}, dd{0.0, 0.0}, dd{0.0, 0.0}};
    {
        constexpr int U = 5;                              // 5 x 32 >= the 148 CTAs of a B200: one batch, one round trip
        const double2* pa = reinterpret_cast<const double2*>(V.partA);
        const double2* pb = reinterpret_cast<const double2*>(V.partB);
        const int ga = V.gridPA, gb = V.gridPB, gmax = ga > gb ? ga : gb;
        for (int base = 0; base < gmax; base += 32 * U) {
            double2 ta[U], tb[U], tc[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int i = base + u * 32 + lane;
                ta[u] = i < ga ? __ldcg(pa + i) : make_double2(0.0, 0.0);
                tb[u] = i < gb ? __ldcg(pb + i) : make_double2(0.0, 0.0);
                tc[u] = i < gb ? __ldcg(pb + gb + i) : make_double2(0.0, 0.0);
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                s3[0] = dd_acc(s3[0], dd{ta[u].x, ta[u].y});
                s3[1] = dd_acc(s3[1], dd{tb[u].x, tb[u].y});
                s3[2] = dd_acc(s3[2], dd{tc[u].x, tc[u].y});
            }
        }
    }
    UC_TL_MARK(V, 5);
    warp_sum_dd_n<3>(s3);
    UC_TL_MARK(V, 6);
    if (lane != 0) return;
    ctl->ticket_b = 0;
    const double dx2 = dd_round(s3[0]), dy2 = dd_round(s3[1]), inter = fabs(dd_round(s3[2]));
    const double r_eta = rule_in.eta, r_omega = rule_in.omega, r_w = rule_in.w;      // written before the block sum's barriers
    const long long r_k = rule_in.k, r_acc = rule_in.acc, r_cap = rule_in.cap;
    const double2 r_pw = rule_in.pw; uc_attempt_record* const r_att = rule_in.att;
    const double eta = r_eta, omega = r_omega;
    const long long k = r_k + 1;
    const double N = omega * dx2 + dy2 / omega;
    const double eta_bar = (inter > 0.0) ? N / (2.0 * inter) : INFINITY;
    const double2 pw = r_pw;
    const double grow = (1.0 + pw.x) * eta;
    const double eta_next = isinf(eta_bar) ? grow : fmin((1.0 - pw.y) * eta_bar, grow);
    const int accept = eta <= eta_bar;
    if (r_att && k - 1 < r_cap) {
        uc_attempt_record rec;
        rec.eta_used = eta; rec.eta_bar = eta_bar; rec.eta_next = eta_next;
        rec.dx2 = dx2; rec.dy2 = dy2; rec.inter = inter; rec.accepted = accept; rec.pad_ = 0;
        r_att[k - 1] = rec;
    }
    if (accept) { ctl->cur = cur ^ 1; ctl->pending = 1; ctl->eta_prev = eta; ctl->w = r_w + eta; ctl->accepted = r_acc + 1; }
    else ctl->pending = 0;
    ctl->eta = eta_next;
    ctl->k = k;
    if (!isfinite(eta_next) || !(eta_next > 0.0)) { ctl->status = UC_NUMERICAL_ERROR; ctl->done = 1; }
    UC_TL_MARK(V, 3);                        // the warp that ran the step rule: when the attempt was decided
}

}  // namespace ucpdhg
