// uc_ingest.cuh -- ingest step A1 on the DEVICE: from the caller's CSR, copied to the device
// once, build the row / column permutations, the explicit transpose and both sliced-ELL layouts with the 16-bit
// column offsets, as kernels.  Everything here is integer work and reproduces uc_format.hpp (the host builders, kept
// as the checker: uc_host_layout_selftest and uc_lp_compare_layout) bit for bit:
//   * permutation: rows with at most `thr` entries first, in windows of `window` rows of the caller's order, each
//     window stably sorted by length; the longer rows after them in the caller's order.  One stable radix sort of
//     (window * (thr + 1) + length) over the short rows gives exactly that order.
//   * transpose: a stable radix sort of the entries by column index keeps, inside a column, the caller's row order --
//     the order the sequential statement's column scatter produces and bit parity of the row sums depends on.
//   * layouts: one thread per (relabelled) row fills its slots  slot(base_s + t * 32 + lane) ; one warp per long row.
// The sorts and prefix sums are CUB device primitives (part of the CUDA toolkit, used like a library routine; one-time
// set-up, not the iteration path).  The attempt schedule (a sequential least-loaded assignment over ~10^5 slices,
// uc_format.hpp build_schedule) stays on the host: it needs only the slice widths and bases, which are copied back.
#pragma once
#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>
#include <cub/device/device_reduce.cuh>
#include "uc_kernels.cuh"

namespace ucpdhg {

constexpr int kIngestBlock = 256;

// ---- lengths
__global__ void k_ing_row_len(const long long* __restrict__ ptr, long long m, int* __restrict__ len) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < m) len[i] = (int)(ptr[i + 1] - ptr[i]);
}
__global__ void k_ing_col_count(const int* __restrict__ col, long long nnz, int* __restrict__ cnt) {
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p < nnz) atomicAdd(cnt + col[p], 1);
}
// row of every entry: the largest i with ptr[i] <= p
__global__ void k_ing_row_ids(const long long* __restrict__ ptr, long long m, long long nnz, int* __restrict__ rowid) {
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= nnz) return;
    long long lo = 0, hi = m;                  // invariant: ptr[lo] <= p < ptr[hi]
    while (hi - lo > 1) { const long long mid = (lo + hi) >> 1; if (ptr[mid] <= p) lo = mid; else hi = mid; }
    rowid[p] = (int)lo;
}

__global__ void k_ing_widen(const int* __restrict__ in, long long* __restrict__ out, long long count) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < count) out[i] = in[i];
}
__global__ void k_ing_iota(int* __restrict__ out, long long count) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < count) out[i] = (int)i;
}

// ---- permutation
__global__ void k_ing_short_flag(const int* __restrict__ len, long long N, int thr, int* __restrict__ flag) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) flag[i] = len[i] <= thr;
}
// rank[i] = short rows before i (exclusive scan of the flags).  Short row i: key / value of the sort; long row i: its
// final place.
__global__ void k_ing_perm_keys(const int* __restrict__ len, const int* __restrict__ rank, long long N, int thr, long long window,
                                long long nshort, unsigned long long* __restrict__ keys, int* __restrict__ vals, long long* __restrict__ perm) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const long long k = rank[i];
    if (len[i] <= thr) { keys[k] = (unsigned long long)(k / window) * (unsigned long long)(thr + 1) + (unsigned long long)len[i]; vals[k] = (int)i; }
    else perm[nshort + (i - k)] = i;
}
__global__ void k_ing_perm_finish(const int* __restrict__ sorted, long long nshort, long long N, long long* __restrict__ perm, long long* __restrict__ inv) {
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    long long o;
    if (k < nshort) { o = sorted[k]; perm[k] = o; } else o = perm[k];
    inv[o] = k;
}

// ---- slice widths and long-row lengths
__global__ void k_ing_slice_width(const int* __restrict__ len, const long long* __restrict__ perm, long long nshort, long long nslices,
                                  long long* __restrict__ slots) {
    const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= nslices) return;
    int w = 0;
    for (long long r = 32 * s; r < 32 * s + 32 && r < nshort; ++r) w = max(w, len[perm[r]]);
    slots[s] = 32LL * w;
}
__global__ void k_ing_long_len(const int* __restrict__ len, const long long* __restrict__ perm, long long nshort, long long nlong, long long* __restrict__ out) {
    const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (r < nlong) out[r] = len[perm[nshort + r]];
}
// exclusive scan results have no total at the end: sp[count] = sp[count-1] + last
__global__ void k_ing_close_scan(long long* sp, const long long* last_in, long long count) {
    if (threadIdx.x == 0 && blockIdx.x == 0) sp[count] = count > 0 ? sp[count - 1] + last_in[count - 1] : 0;
}

// ---- layout fill.  Source of row o's t-th entry:
//   K  (order == nullptr): p = ptr[o] + t, column col[p]
//   K' (order != nullptr): p = order[ptr[o] + t] (ptr = column pointers, order = entries sorted by column), "column" rowid[p]
struct FillSrc { const long long* ptr; const int* order; const int* idx; const double* val; };
__device__ __forceinline__ long long fill_pos(const FillSrc& S, long long o, long long t) {
    const long long q = S.ptr[o] + t;
    return S.order ? (long long)S.order[q] : q;
}
__global__ void k_ing_fill_sell(FillSrc S, const long long* __restrict__ perm, const long long* __restrict__ inv_other, long long nshort,
                                const long long* __restrict__ sp, int* __restrict__ col, double* __restrict__ val, long long* __restrict__ src) {
    const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= nshort) return;
    const long long o = perm[r], base = sp[r >> 5] + (r & 31);
    const int len = (int)(S.ptr[o + 1] - S.ptr[o]);
    for (int t = 0; t < len; ++t) {
        const long long p = fill_pos(S, o, t), k = base + 32LL * t;
        col[k] = (int)inv_other[S.idx[p]];
        val[k] = S.val[p];
        if (src) src[k] = p;
    }
}
__global__ void k_ing_fill_long(FillSrc S, const long long* __restrict__ perm, const long long* __restrict__ inv_other, long long nshort, long long nlong,
                                const long long* __restrict__ lptr, int* __restrict__ lcol, double* __restrict__ lval, long long* __restrict__ lsrc) {
    const long long w = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (w >= nlong) return;
    const long long o = perm[nshort + w], b = lptr[w];
    const long long len = S.ptr[o + 1] - S.ptr[o];
    for (long long t = lane; t < len; t += 32) {
        const long long p = fill_pos(S, o, t);
        lcol[b + t] = (int)inv_other[S.idx[p]];
        lval[b + t] = S.val[p];
        if (lsrc) lsrc[b + t] = p;
    }
}

// ---- 16-bit column offsets (uc_format.hpp compress_columns): one warp per slice
__global__ void k_ing_slice_base(const int* __restrict__ len, const long long* __restrict__ perm, long long nshort, long long nslices,
                                 const long long* __restrict__ sp, const int* __restrict__ col, int enable, int* __restrict__ cbase,
                                 long long* __restrict__ narrow_of) {
    const long long s = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (s >= nslices) return;
    const long long r = 32 * s + lane, b = sp[s];
    int lo = INT_MAX, hi = -1;
    if (r < nshort) {
        const int l = len[perm[r]];
        for (int t = 0; t < l; ++t) { const int c = col[b + 32LL * t + lane]; lo = min(lo, c); hi = max(hi, c); }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o)); hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o)); }
    if (hi < 0) { lo = 0; hi = 0; }
    const bool narrow = enable && (long long)hi - lo <= 65535;
    if (lane == 0) { cbase[s] = narrow ? lo : -1; narrow_of[s] = narrow ? sp[s + 1] - b : 0; }
}
__global__ void k_ing_col16(const int* __restrict__ len, const long long* __restrict__ perm, long long nshort, long long nslices,
                            const long long* __restrict__ sp, const int* __restrict__ col, const int* __restrict__ cbase,
                            unsigned short* __restrict__ col16) {
    const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= nshort) return;
    const long long s = r >> 5;
    const int cb = cbase[s];
    if (cb < 0) return;
    const long long b = sp[s] + (r & 31);
    const int l = len[perm[r]];
    for (int t = 0; t < l; ++t) col16[b + 32LL * t] = (unsigned short)(col[b + 32LL * t] - cb);      // padding slots keep offset 0
}

inline int ing_grid(long long n, int per = kIngestBlock) { return (int)std::max<long long>(1, (n + per - 1) / per); }
inline int bits_for(unsigned long long maxval) { int b = 1; while (b < 64 && (maxval >> b) != 0) ++b; return b; }

}  // namespace ucpdhg
