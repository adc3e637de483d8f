// uc_format.hpp -- host-side ingest: validation, transpose and the sliced-ELL layout.
//
// Layout ("SELL-32 + long tail"):
//   rows are relabelled  new -> old  by `perm`:  rows with at most `long_thr` entries come first,
//   taken in the caller's order in windows of `window` rows and sorted by length inside each window
//   (stable counting sort), so that 32 consecutive rows -- one slice, one warp -- have (nearly) equal
//   length; rows longer than `long_thr` follow and are stored as plain CSR (one warp per row).
//   Slice s holds rows 32s..32s+31 column-major: slot(base_s + t*32 + lane) = t-th entry of row
//   32s+lane, padded with (col 0, val 0) up to the slice width, so lane-consecutive loads coalesce.
// The relabelling is internal: both matrices, all vectors and both diagonal scalings live in the
// permuted index spaces; results are un-permuted on the way out.
#pragma once
#include <cstdint>
#include <string>
#include <vector>
#include <algorithm>
#include <queue>
#include <functional>
#include <utility>
#include <thread>
#include <cmath>
#include <climits>

namespace ucpdhg {

// One step of the warp-private pipelines of the persistent attempt kernels (uc_attempt.cuh): a chunk of at
// most kChunkT entries per row of one slice.  A slice wider than kChunkT is a run of consecutive steps of
// the same warp, the row sums carried in registers from one to the next.  16 bytes.
constexpr int kChunkT = 4;
struct StepDesc {
    uint32_t w0;       // bits 0-25: (first stored entry of the chunk in the sliced-ELL arrays) / 32; bits 26-31: info
    int32_t row0;      // first row of the slice
    int32_t cbase;     // >= 0: the slice's column indices are stored as 16-bit offsets from cbase; -1: as 32-bit indices
    int32_t pad_;
};
// info: bits 0-2 entries per row in this chunk (0 = padding step: nothing to do)
constexpr int kStepFirst = 8;    // first chunk of its slice
constexpr int kStepLast = 16;    // last chunk of its slice (the update is applied)
constexpr int kStepEnd = 32;     // the warp has no further steps (set on its first padding step)
static_assert(sizeof(StepDesc) == 16, "StepDesc layout");

// f(begin, end) over [0, n) on up to 8 host threads (uc_lp_create is a one-time cost, but it is inside the
// end-to-end time: the layouts of a 6M-entry matrix take ~0.5 s on one core)
template <class F>
inline void parallel_ranges(int64_t n, int64_t grain, F f) {
    unsigned hw = std::thread::hardware_concurrency();
    int64_t nt = std::max<int64_t>(1, std::min<int64_t>(std::min<int64_t>(hw ? hw : 1, 8), n / std::max<int64_t>(grain, 1)));
    if (nt <= 1) { f((int64_t)0, n); return; }
    std::vector<std::thread> th;
    const int64_t per = (n + nt - 1) / nt;
    for (int64_t t = 0; t < nt; ++t) {
        const int64_t b = t * per, e = std::min(n, b + per);
        if (b < e) th.emplace_back([=] { f(b, e); });
    }
    for (auto& x : th) x.join();
}

struct HostSell {
    int64_t nrows = 0, nshort = 0, nlong = 0, nslices = 0;
    std::vector<int64_t> slice_ptr;   // [nslices+1]
    std::vector<int32_t> col;         // [slots]  column indices (the reference; uploaded only if some slice is wide)
    std::vector<uint16_t> col16;      // [slots]  16-bit offsets from cbase[slice] (uploaded only if some slice is narrow)
    std::vector<int32_t> cbase;       // [nslices] smallest column index of a narrow slice, -1 for a wide one
    int64_t narrow_slots = 0;         // stored slots (incl. padding) of the narrow slices
    std::vector<int32_t> rlen;        // [nshort] entries of each row of the sliced part
    std::vector<double> val;          // [slots]
    std::vector<int64_t> src;         // [slots]  caller's CSR position of the slot, -1 = padding (only if asked for)
    std::vector<int64_t> lptr;        // [nlong+1]
    std::vector<int32_t> lcol;
    std::vector<double> lval;
    std::vector<int64_t> lsrc;
    std::vector<StepDesc> steps;      // [steps_per_warp][sched_warps] schedule of the persistent attempt kernels
    int64_t steps_per_warp = 0, sched_warps = 0;
};

// Static schedule of the persistent attempt kernels for `ctas` CTAs of `warps_per_cta` consumer warps.
//   1. The slices are cut into `ctas` CONTIGUOUS ranges of (nearly) equal estimated cost, one per CTA: the gathers of
//      neighbouring rows fall into the same few blocks of the gathered vector (in a UC LP: the rows / variables of one
//      period), so a CTA that sweeps a contiguous range finds most gathered sectors in ITS L1 -- the attempt kernels
//      are bound by L2 sector throughput (~6300 B/cycle chip-wide), of which scattered 8/16-byte gathers, each pulling
//      a 32-byte sector, were half (profiles/r02b).
//   2. Inside its range a CTA deals the slices, in ascending order, to its warp with the least estimated work so far
//      (ties: lowest warp), so that its warps finish together while, at any moment, they work on neighbouring slices
//      (one shared working set in L1).
// The estimate (7 per step + 1.3 per entry per row + 4 for the step that applies the update, in units of ~100 cycles) was
// fitted in round 1 to per-warp cycle counters of a scratch build that is not in this tree; what IS reproducible is its
// result: the spread of the warps' busy times that python -m paper_2607_03627_b200.timeline prints (profiles/).  A warp takes its slices in ascending order, each as
// ceil(width / kChunkT) steps.  Stored step-major, steps[j * warps + w] with w = cta * warps_per_cta + warp, padded with
// empty steps to the longest warp, so that step j of all warps is one coalesced read.  The assignment is fixed at
// create time: solves are reproducible bit for bit.
inline int64_t slice_cost(int64_t wd) {
    const int64_t nch = std::max<int64_t>(1, (wd + kChunkT - 1) / kChunkT);
    return 70 * nch + 13 * wd + 40;
}
inline void build_schedule(HostSell& S, int64_t ctas, int64_t warps_per_cta) {
    if (ctas < 1) ctas = 1;
    if (warps_per_cta < 1) warps_per_cta = 1;
    const int64_t warps = ctas * warps_per_cta;
    S.sched_warps = warps;
    std::vector<int32_t> owner((size_t)S.nslices);
    std::vector<int64_t> count((size_t)warps, 0);
    {
        std::vector<int64_t> wd((size_t)S.nslices);
        int64_t total = 0;
        for (int64_t s = 0; s < S.nslices; ++s) { wd[(size_t)s] = (S.slice_ptr[(size_t)s + 1] - S.slice_ptr[(size_t)s]) / 32; total += slice_cost(wd[(size_t)s]); }
        typedef std::pair<int64_t, int64_t> Load;                    // (work so far, warp)
        int64_t s = 0, done = 0;
        for (int64_t c = 0; c < ctas; ++c) {
            // range of CTA c: up to the slice where the running cost passes (c + 1) / ctas of the total
            const int64_t target = (total * (c + 1)) / ctas;
            std::priority_queue<Load, std::vector<Load>, std::greater<Load>> heap;
            for (int64_t w = 0; w < warps_per_cta; ++w) heap.push(Load(0, c * warps_per_cta + w));
            while (s < S.nslices && (c == ctas - 1 || done + slice_cost(wd[(size_t)s]) / 2 <= target)) {
                Load l = heap.top(); heap.pop();
                owner[(size_t)s] = (int32_t)l.second;
                l.first += slice_cost(wd[(size_t)s]);
                done += slice_cost(wd[(size_t)s]);
                count[(size_t)l.second] += std::max<int64_t>(1, (wd[(size_t)s] + kChunkT - 1) / kChunkT);
                heap.push(l);
                ++s;
            }
        }
    }
    int64_t J = 0;
    for (int64_t c : count) J = std::max(J, c);
    S.steps_per_warp = J;
    S.steps.assign((size_t)(J * warps), StepDesc{0u, 0, -1, 0});
    std::fill(count.begin(), count.end(), 0);
    for (int64_t s = 0; s < S.nslices; ++s) {
        const int64_t wd = (S.slice_ptr[(size_t)s + 1] - S.slice_ptr[(size_t)s]) / 32;
        const int64_t nch = std::max<int64_t>(1, (wd + kChunkT - 1) / kChunkT);
        const int64_t w = owner[(size_t)s];
        for (int64_t c = 0; c < nch; ++c) {
            StepDesc d;
            const int64_t nt = std::min<int64_t>(kChunkT, wd - kChunkT * c);
            const uint32_t info = (uint32_t)std::max<int64_t>(nt, 0) | (c == 0 ? kStepFirst : 0) | (c == nch - 1 ? kStepLast : 0);
            d.w0 = (uint32_t)((S.slice_ptr[(size_t)s] + 32 * kChunkT * c) >> 5) | (info << 26);   // slots < 2^31 (checked at create)
            d.row0 = (int32_t)(32 * s);
            d.cbase = S.cbase.empty() ? -1 : S.cbase[(size_t)s]; d.pad_ = 0;
            S.steps[(size_t)(count[(size_t)w]++ * warps + w)] = d;
        }
    }
    for (int64_t w = 0; w < warps; ++w)
        if (count[(size_t)w] < J) S.steps[(size_t)(count[(size_t)w] * warps + w)].w0 = (uint32_t)kStepEnd << 26;
}

// new -> old permutation: short rows in length-sorted windows, long rows last.
inline void build_perm(const std::vector<int64_t>& len, int64_t window, int64_t long_thr,
                       std::vector<int64_t>& perm, std::vector<int64_t>& inv, int64_t& nshort) {
    const int64_t N = (int64_t)len.size();
    perm.clear(); perm.reserve(N);
    std::vector<int64_t> longs, win;
    std::vector<int64_t> cnt((size_t)long_thr + 2);
    win.reserve((size_t)window);
    auto flush = [&]() {
        std::fill(cnt.begin(), cnt.end(), 0);
        for (int64_t r : win) cnt[(size_t)len[r] + 1]++;
        for (size_t k = 1; k < cnt.size(); ++k) cnt[k] += cnt[k - 1];
        size_t base = perm.size();
        perm.resize(base + win.size());
        for (int64_t r : win) perm[base + (size_t)cnt[(size_t)len[r]]++] = r;
        win.clear();
    };
    for (int64_t r = 0; r < N; ++r) {
        if (len[r] > long_thr) { longs.push_back(r); continue; }
        win.push_back(r);
        if ((int64_t)win.size() == window) flush();
    }
    if (!win.empty()) flush();
    nshort = (int64_t)perm.size();
    perm.insert(perm.end(), longs.begin(), longs.end());
    inv.assign((size_t)N, 0);
    for (int64_t k = 0; k < N; ++k) inv[(size_t)perm[k]] = k;
}

// CSR (ptr, idx, val, optional src positions) with rows relabelled by perm and column indices by
// inv_other -> SELL + long tail.
inline void build_sell(int64_t nrows, const int64_t* ptr, const int32_t* idx, const double* val, const int64_t* srcpos,
                       const std::vector<int64_t>& perm, int64_t nshort, const std::vector<int64_t>& inv_other,
                       bool want_src, HostSell& S) {
    S.nrows = nrows; S.nshort = nshort; S.nlong = nrows - nshort;
    S.nslices = (nshort + 31) / 32;
    S.slice_ptr.assign((size_t)S.nslices + 1, 0);
    parallel_ranges(S.nslices, 1024, [&](int64_t sb, int64_t se) {
        for (int64_t s = sb; s < se; ++s) {
            int64_t w = 0;
            for (int64_t r = 32 * s; r < std::min<int64_t>(32 * s + 32, nshort); ++r) {
                int64_t o = perm[(size_t)r];
                w = std::max(w, ptr[o + 1] - ptr[o]);
            }
            S.slice_ptr[(size_t)s + 1] = 32 * w;
        }
    });
    for (int64_t s = 0; s < S.nslices; ++s) S.slice_ptr[(size_t)s + 1] += S.slice_ptr[(size_t)s];
    const int64_t slots = S.slice_ptr[(size_t)S.nslices];
    S.col.assign((size_t)slots, 0); S.val.assign((size_t)slots, 0.0);
    if (want_src) S.src.assign((size_t)slots, -1);
    S.rlen.assign((size_t)nshort, 0);
    parallel_ranges(nshort, 32768, [&](int64_t rb, int64_t re) {
        for (int64_t r = rb; r < re; ++r) {
            int64_t o = perm[(size_t)r], s = r >> 5, lane = r & 31, base = S.slice_ptr[(size_t)s];
            S.rlen[(size_t)r] = (int32_t)(ptr[o + 1] - ptr[o]);
            for (int64_t p = ptr[o], t = 0; p < ptr[o + 1]; ++p, ++t) {
                size_t k = (size_t)(base + t * 32 + lane);
                S.col[k] = (int32_t)inv_other[(size_t)idx[p]];
                S.val[k] = val[p];
                if (want_src) S.src[k] = srcpos ? srcpos[p] : p;
            }
        }
    });
    S.lptr.assign((size_t)S.nlong + 1, 0);
    for (int64_t r = 0; r < S.nlong; ++r) {
        int64_t o = perm[(size_t)(nshort + r)];
        S.lptr[(size_t)r + 1] = S.lptr[(size_t)r] + (ptr[o + 1] - ptr[o]);
    }
    const int64_t lnnz = S.lptr[(size_t)S.nlong];
    S.lcol.resize((size_t)lnnz); S.lval.resize((size_t)lnnz);
    if (want_src) S.lsrc.resize((size_t)lnnz);
    for (int64_t r = 0; r < S.nlong; ++r) {
        int64_t o = perm[(size_t)(nshort + r)], k = S.lptr[(size_t)r];
        for (int64_t p = ptr[o]; p < ptr[o + 1]; ++p, ++k) {
            S.lcol[(size_t)k] = (int32_t)inv_other[(size_t)idx[p]];
            S.lval[(size_t)k] = val[p];
            if (want_src) S.lsrc[(size_t)k] = srcpos ? srcpos[p] : p;
        }
    }
}

// Byte reduction ("16-bit column deltas within slices"): a slice whose column indices span less
// than 2^16 is NARROW -- its indices are stored as 16-bit offsets from the slice's smallest column index (cbase), 2 bytes
// per stored entry instead of 4.  In a UC LP the rows of one period touch the variables of that period and the one
// before (and the other way round for K'), so every slice of configs 0-3 is narrow; uniformly random columns (the
// roofline sweep) make every slice wide and nothing changes for them.  Integer work: decoding gives back the
// 32-bit index bit for bit.  Padding slots of a narrow slice decode to cbase (value 0.0, as before).
inline void compress_columns(HostSell& S, bool enable) {
    S.cbase.assign((size_t)S.nslices, -1);
    S.col16.clear(); S.narrow_slots = 0;
    if (!enable || S.nslices == 0) return;
    std::vector<int64_t> narrow_of((size_t)S.nslices, 0);
    parallel_ranges(S.nslices, 2048, [&](int64_t sb, int64_t se) {
        for (int64_t s = sb; s < se; ++s) {
            const int64_t b = S.slice_ptr[(size_t)s], e = S.slice_ptr[(size_t)s + 1];
            int32_t lo = INT32_MAX, hi = -1;
            for (int64_t lane = 0; lane < 32 && 32 * s + lane < S.nshort; ++lane)
                for (int64_t t = 0; t < S.rlen[(size_t)(32 * s + lane)]; ++t) {
                    const int32_t c = S.col[(size_t)(b + 32 * t + lane)];
                    lo = std::min(lo, c); hi = std::max(hi, c);
                }
            if (hi < 0) { lo = 0; hi = 0; }                       // a slice of empty rows
            if ((int64_t)hi - lo <= 65535) { S.cbase[(size_t)s] = lo; narrow_of[(size_t)s] = e - b; }
        }
    });
    for (int64_t v : narrow_of) S.narrow_slots += v;
    if (S.narrow_slots == 0) return;
    S.col16.assign(S.col.size(), 0);
    parallel_ranges(S.nslices, 2048, [&](int64_t sb, int64_t se) {
        for (int64_t s = sb; s < se; ++s) {
            const int32_t cb = S.cbase[(size_t)s];
            if (cb < 0) continue;
            const int64_t b = S.slice_ptr[(size_t)s];
            for (int64_t lane = 0; lane < 32 && 32 * s + lane < S.nshort; ++lane)
                for (int64_t t = 0; t < S.rlen[(size_t)(32 * s + lane)]; ++t) {
                    const size_t k = (size_t)(b + 32 * t + lane);
                    S.col16[k] = (uint16_t)(S.col[k] - cb);                 // padding slots keep offset 0
                }
        }
    });
}


// Validate the caller's CSR (A0) and return "" or the reason it is rejected.  Two parts: validate_args looks at the
// sizes and pointers only (what must hold before any array is read or copied); validate_entries scans the arrays
// (uc_lp_create runs it on a helper thread while the arrays are being copied to the device, and waits for it before
// the first kernel reads them).
inline std::string validate_args(int64_t m, int64_t n, int64_t nnz, const int64_t* row_ptr, const int32_t* col_idx,
                                 const double* val, const char* sense, const double* b, const double* c,
                                 const double* l, const double* u) {
    if (m < 0 || n < 0 || nnz < 0) return "negative size";
    if (!row_ptr) return "row_ptr is NULL";
    if (m > 2000000000LL || n > 2000000000LL || nnz > 2000000000LL) return "size exceeds the int32 index range of the layout";
    if (row_ptr[0] != 0 || row_ptr[m] != nnz) return "row_ptr[0] != 0 or row_ptr[m] != nnz";
    if (nnz > 0 && (!col_idx || !val)) return "col_idx / val is NULL";
    if ((m > 0 && (!sense || !b)) || (n > 0 && (!c || !l || !u))) return "a vector argument is NULL";
    return "";
}
inline std::string validate_entries(int64_t m, int64_t n, int64_t nnz, const int64_t* row_ptr, const int32_t* col_idx,
                                    const double* val, const char* sense, const double* b, const double* c,
                                    const double* l, const double* u) {
    for (int64_t i = 0; i < m; ++i)
        if (row_ptr[i + 1] < row_ptr[i] || row_ptr[i + 1] > nnz) return "row_ptr is not monotone";
    // rows are checked in parallel ranges, each with its own duplicate-detection stamps; the reported reason is
    // that of the first range (in row order) that found one
    const int kMaxRanges = 8;
    std::vector<std::string> why_r((size_t)kMaxRanges);
    const int64_t per = (m + kMaxRanges - 1) / kMaxRanges;
    parallel_ranges(kMaxRanges, 1, [&](int64_t tb, int64_t te) {
        std::vector<int64_t> stamp((size_t)std::max<int64_t>(n, 1), -1);
        for (int64_t t = tb; t < te; ++t) {
            const char* bad = nullptr;
            for (int64_t i = t * per; i < std::min(m, (t + 1) * per) && !bad; ++i) {
                if (sense[i] != 'E' && sense[i] != 'G') { bad = "sense must be 'E' or 'G'"; break; }
                if (!std::isfinite(b[i])) { bad = "b has a non-finite entry"; break; }
                for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) {
                    int64_t j = col_idx[p];
                    if (j < 0 || j >= n) { bad = "column index out of range"; break; }
                    if (stamp[(size_t)j] == i) { bad = "duplicate entry within a row"; break; }
                    stamp[(size_t)j] = i;
                    if (!std::isfinite(val[p])) { bad = "val has a non-finite entry"; break; }
                }
            }
            if (bad) why_r[(size_t)t] = bad;
        }
    });
    for (const std::string& w : why_r) if (!w.empty()) return w;
    for (int64_t j = 0; j < n; ++j) {
        if (!std::isfinite(c[j])) return "c has a non-finite entry";
        if (std::isnan(l[j]) || std::isnan(u[j])) return "a bound is NaN";
        if (l[j] > u[j]) return "l > u";
    }
    return "";
}
inline std::string validate_csr(int64_t m, int64_t n, int64_t nnz, const int64_t* row_ptr, const int32_t* col_idx,
                                const double* val, const char* sense, const double* b, const double* c,
                                const double* l, const double* u) {
    std::string why = validate_args(m, n, nnz, row_ptr, col_idx, val, sense, b, c, l, u);
    return why.empty() ? validate_entries(m, n, nnz, row_ptr, col_idx, val, sense, b, c, l, u) : why;
}

// A1 in three pieces, so that the caller can overlap them (and the upload of K) on two threads:
//   build_perms  row / column lengths and both permutations (cheap; fixes the slice counts)
//   build_K      the SELL layout of K
//   build_KT     explicit transpose (counting sort by column, stable in the row index) + the SELL layout of K'
struct HostProblem {
    int64_t m = 0, n = 0, nnz = 0;
    std::vector<int64_t> perm_r, inv_r, perm_c, inv_c;   // new -> old, old -> new
    std::vector<int64_t> lenc;                           // entries per column
    int64_t nshort_r = 0, nshort_c = 0;                  // rows / columns in the sliced parts
    HostSell K, KT;
};
inline void build_perms(int64_t m, int64_t n, int64_t nnz, const int64_t* row_ptr, const int32_t* col_idx,
                        int64_t window, int64_t long_thr, HostProblem& P) {
    P.m = m; P.n = n; P.nnz = nnz;
    std::vector<int64_t> lenr((size_t)m);
    P.lenc.assign((size_t)n, 0);
    for (int64_t i = 0; i < m; ++i) lenr[(size_t)i] = row_ptr[i + 1] - row_ptr[i];
    for (int64_t p = 0; p < nnz; ++p) P.lenc[(size_t)col_idx[p]]++;
    std::thread t([&] { build_perm(lenr, window, long_thr, P.perm_r, P.inv_r, P.nshort_r); });
    build_perm(P.lenc, window, long_thr, P.perm_c, P.inv_c, P.nshort_c);
    t.join();
}
inline void build_K(const int64_t* row_ptr, const int32_t* col_idx, const double* val, bool want_src, HostProblem& P) {
    build_sell(P.m, row_ptr, col_idx, val, nullptr, P.perm_r, P.nshort_r, P.inv_c, want_src, P.K);
}
inline void build_KT(const int64_t* row_ptr, const int32_t* col_idx, const double* val, bool want_src, HostProblem& P) {
    const int64_t m = P.m, n = P.n, nnz = P.nnz;
    std::vector<int64_t> tptr((size_t)n + 1, 0), tsrc(want_src ? (size_t)nnz : 0);
    std::vector<int32_t> tidx((size_t)nnz);
    std::vector<double> tval((size_t)nnz);
    for (int64_t j = 0; j < n; ++j) tptr[(size_t)j + 1] = tptr[(size_t)j] + P.lenc[(size_t)j];
    // counting sort by column, stable in the row index; each thread owns a range of columns, scans every entry and
    // scatters only its own (its slice of the fill pointers stays in cache)
    parallel_ranges(n, 65536, [&](int64_t jb, int64_t je) {
        std::vector<int64_t> fill(tptr.begin() + jb, tptr.begin() + je);
        for (int64_t i = 0; i < m; ++i)
            for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) {
                const int64_t j = col_idx[p];
                if (j < jb || j >= je) continue;
                const int64_t k = fill[(size_t)(j - jb)]++;
                tidx[(size_t)k] = (int32_t)i; tval[(size_t)k] = val[p];
                if (want_src) tsrc[(size_t)k] = p;
            }
    });
    build_sell(n, tptr.data(), tidx.data(), tval.data(), want_src ? tsrc.data() : nullptr, P.perm_c, P.nshort_c, P.inv_r, want_src, P.KT);
}


}  // namespace ucpdhg
