// uc_pdhg.cu -- the C ABI of include/uc_pdhg.h: handle, ingest, preconditioning driver, the
// CUDA-graph iteration loop, cancel, output.  All arithmetic of the method runs in the kernels of
// uc_kernels.cuh; the host only marshals, launches and polls.  There is no CPU fallback.
#include <atomic>
#include <chrono>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <exception>
#include <limits>
#include <mutex>
#include <thread>
#include <new>
#include <string>
#include <vector>

#include "uc_format.hpp"
#include "uc_kernels.cuh"
#include "uc_attempt.cuh"
#include "uc_ingest.cuh"

using namespace ucpdhg;

namespace {

thread_local std::string g_err;

int fail(int code, const std::string& msg) { g_err = msg; return code; }

struct CudaFail { cudaError_t e; const char* what; };
struct TooLarge { const char* what; };                            // a size limit of the layout, not an allocation failure
#define CK(call)                                                 \
    do {                                                         \
        cudaError_t e__ = (call);                                \
        if (e__ != cudaSuccess) throw CudaFail{e__, #call};      \
    } while (0)

// code of a standard exception caught at the ABI: allocation failures keep UC_ERR_NOMEM, everything else (std::system_error
// of a helper thread, std::length_error, ...) is an internal failure with its own code
int std_code(const std::exception& e) {
    return (dynamic_cast<const std::bad_alloc*>(&e) || dynamic_cast<const std::bad_array_new_length*>(&e)) ? UC_ERR_NOMEM : UC_ERR_INTERNAL;
}

double now_s() {
    return std::chrono::duration<double>(std::chrono::steady_clock::now().time_since_epoch()).count();
}
inline int cdiv(long long a, long long b) { return (int)((a + b - 1) / b); }

}  // namespace

struct uc_lp {
    int device = 0;
    cudaStream_t own_stream = nullptr;
    int64_t m = 0, n = 0, nnz = 0;
    uc_lp_options opt{};
    std::vector<void*> allocs;
    size_t device_bytes = 0;
    // permutations (device, new -> old)
    long long *perm_r = nullptr, *perm_c = nullptr;
    Sell K{}, KT{};
    Vecs V{};
    Ctrl* ctl = nullptr;
    double *Dr = nullptr, *Dc = nullptr;   // writable aliases of V.Dr / V.Dc
    // device staging of the host-buffer entry point (uc_pdhg_solve): results before they go to the caller's buffers, and a
    // warm start after it came from them.  Owned by the handle: no cudaMalloc / cudaFree on the solve path (they
    // synchronise the device and were seen to stall for hundreds of ms now and then).
    double *stage_x = nullptr, *stage_y = nullptr, *stage_x0 = nullptr, *stage_y0 = nullptr;
    // scratch of uc_lp_update_bounds / uc_lp_update_objective, allocated by the first such call and kept: re-solve loops
    // call them once per node, and a cudaMalloc / cudaFree pair per call stalls the device (see above).  The n-vectors of
    // those calls are stage_x (always there) and stage_x0 (allocated on first need); nothing else uses them while the
    // handle's busy flag is held.
    dd* upd_part = nullptr; double* upd_scal = nullptr;
    double *qs = nullptr, *cs = nullptr, *ls = nullptr, *us = nullptr;
    unsigned char* isG = nullptr;
    // host <-> device mailboxes (pinned, mapped)
    HostStatus* h_status = nullptr; HostStatus* d_status = nullptr;
    int* h_stop = nullptr; int* d_stop = nullptr;
    // cancel protocol (uc_pdhg_cancel): `state` = (generation << 1) | busy, changed only by solve entry / exit.  A
    // cancel that finds a solve in flight stamps the stop flag with THAT solve's generation (a later solve ignores
    // it); a cancel that finds the handle idle is kept for the next solve (cancel_requested).
    std::atomic<int> cancel_requested{0};
    std::atomic<unsigned> state{0};
    std::atomic<int> busy{0};
    // one-time scalars
    double eta0 = 1.0, omega0 = 1.0, norm_b = 0.0, norm_c = 0.0, norm_qs = 0.0;   // norm_qs: scaled ||q~|| (omega0 of R2)
    double precondition_seconds = 0.0, create_seconds = 0.0;
    int64_t k_slots = 0, kt_slots = 0, k_long_nnz = 0, kt_long_nnz = 0, k_narrow = 0, kt_narrow = 0;
    // step-rule factors {(k+1)^-0.6, (k+1)^-0.3}, k = 1.. (R5): a constant schedule, tabulated once
    double2* powtab = nullptr;
    long long powtab_len = 0;
    // graph cache
    cudaGraphExec_t exec = nullptr;
    int graph_ce = 0;
    int graph_nodes = 0;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    cudaEvent_t ev_t0 = nullptr, ev_t1 = nullptr;
    // source maps for uc_lp_get_scaled_values (only with keep_source_map)
    std::vector<int64_t> k_src, k_lsrc, kt_src, kt_lsrc;

    // every array gets one slice (32 elements) of zeroed slack: the bulk copies of the attempt kernels read
    // whole 32-row segments, and the last slice of the sliced part may be ragged.  Zeroing is ordered on the handle's
    // stream, like everything else uc_lp_create does on the device.  With an arena reserved (the fixed set of vectors:
    // one cudaMalloc instead of ~25) arrays are carved out of it.
    std::mutex alloc_mutex;                // the host-ingest path uploads the two layouts from two threads
    char* arena = nullptr; size_t arena_cap = 0, arena_used = 0;
    void reserve_arena(size_t bytes) {
        void* p = nullptr;
        cudaError_t e = cudaMalloc(&p, bytes);
        if (e != cudaSuccess) throw CudaFail{e, "cudaMalloc"};
        if (cudaMemsetAsync(p, 0, bytes, own_stream) != cudaSuccess) throw CudaFail{cudaGetLastError(), "cudaMemsetAsync"};
        std::lock_guard<std::mutex> g(alloc_mutex);
        allocs.push_back(p); device_bytes += bytes;
        arena = (char*)p; arena_cap = bytes; arena_used = 0;
    }
    template <class T>
    T* dalloc(size_t count) {
        void* p = nullptr;
        size_t bytes = (((count + 32) * sizeof(T) + 255) / 256) * 256;
        {
            std::lock_guard<std::mutex> g(alloc_mutex);
            if (arena && arena_used + bytes <= arena_cap) { p = arena + arena_used; arena_used += bytes; return (T*)p; }
        }
        cudaError_t e = cudaMalloc(&p, bytes);
        if (e != cudaSuccess) throw CudaFail{e, "cudaMalloc"};
        {
            std::lock_guard<std::mutex> g(alloc_mutex);
            allocs.push_back(p);
            device_bytes += bytes;
        }
        if (cudaMemsetAsync(p, 0, bytes, own_stream) != cudaSuccess) throw CudaFail{cudaGetLastError(), "cudaMemsetAsync"};
        return (T*)p;
    }
    void dfree(void* p) {
        if (!p) return;
        std::lock_guard<std::mutex> g(alloc_mutex);
        for (auto& q : allocs) if (q == p) { cudaFree(p); q = nullptr; return; }
    }
    template <class T>
    T* upload(const std::vector<T>& h) {
        T* d = dalloc<T>(h.size());
        if (!h.empty()) {
            CK(cudaMemcpyAsync(d, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice, own_stream));
            CK(cudaStreamSynchronize(own_stream));           // the source is pageable host memory of the caller's frame
        }
        return d;
    }
};

namespace {

struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev) { cudaGetDevice(&prev); if (prev != dev) cudaSetDevice(dev); else prev = -1; }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

Sell upload_sell(uc_lp* lp, const HostSell& H) {
    Sell S{};
    static_assert(sizeof(long long) == sizeof(int64_t), "int64 layout");
    S.sp = (const long long*)lp->upload(H.slice_ptr);
    // column indices: only the representation(s) that some slice uses (uc_format.hpp compress_columns)
    const int64_t slots = (int64_t)H.col.size();
    S.col = H.narrow_slots < slots ? lp->upload(H.col) : nullptr;
    S.col16 = H.narrow_slots > 0 ? lp->upload(H.col16) : nullptr;
    S.cbase = lp->upload(H.cbase);
    S.val = lp->upload(H.val);
    S.nshort = H.nshort; S.nslices = (int)H.nslices; S.nblk = cdiv(H.nslices, kWarps);
    S.lp = (const long long*)lp->upload(H.lptr);
    S.lcol = lp->upload(H.lcol);
    S.lval = lp->upload(H.lval);
    S.nlong = (int)H.nlong;
    S.nlblk = cdiv(H.nlong, kWarps);
    S.grid = S.nlblk + S.nblk;
    if (S.grid < 1) S.grid = 1;
    S.steps = lp->upload(H.steps);
    S.steps_per_warp = (int)H.steps_per_warp; S.sched_warps = (int)H.sched_warps;
    S.nslots = slots;
    return S;
}


// ------------------------------------------------------------------------------------------ A1 on the device
// Temporary device memory of uc_lp_create: one allocation, bump-allocated, released when create returns.
struct TempArena {
    // One block, bump-allocated.  The block is kept in a per-device cache of this process when uc_lp_create returns (up to
    // kScratchKeep bytes; a larger one is freed) and reused by the next uc_lp_create: cudaMalloc / cudaFree of ~1 GB
    // synchronise the device and were seen to stall for 0.1-0.6 s now and then -- more than the whole of uc_lp_create.
    // (A stream-ordered pool was measured too: its first ~1 GB allocation costs 0.35 s.)
    static constexpr size_t kScratchKeep = (size_t)2 << 30;
    struct Cache { std::mutex mu; std::vector<void*> base; std::vector<size_t> cap; std::vector<char> busy; };
    static Cache& cache() { static Cache c; return c; }
    char* base = nullptr; size_t cap = 0, used = 0; int dev = -1; bool cached = false;
    // set by uc_lp_create after its last stream synchronisation: nothing enqueued can still touch the block.  On every
    // other way out (an exception, a validation failure after the copies were enqueued) copies and ingest kernels may
    // still be running, on the handle's stream or the upload thread's, and the handle's stream may already be destroyed:
    // the destructor then waits for the whole device before the block can be handed to the next uc_lp_create or freed.
    bool quiesced = false;
    ~TempArena() {
        if (!base) return;
        if (!quiesced) cudaDeviceSynchronize();          // the creating thread still has the arena's device current
        Cache& C = cache();
        std::lock_guard<std::mutex> g(C.mu);
        if (cached) { C.busy[(size_t)dev] = 0; return; }                     // back to the cache
        if (cap <= kScratchKeep && !C.busy[(size_t)dev]) {                   // becomes the cache (the smaller old one goes)
            if (C.base[(size_t)dev]) cudaFree(C.base[(size_t)dev]);
            C.base[(size_t)dev] = base; C.cap[(size_t)dev] = cap;
        } else cudaFree(base);
    }
    // bytes the cache holds for `device` right now (in use by a running uc_lp_create or not)
    static size_t cached_bytes(int device) {
        Cache& C = cache();
        std::lock_guard<std::mutex> g(C.mu);
        return device >= 0 && device < (int)C.base.size() && C.base[(size_t)device] ? C.cap[(size_t)device] : 0;
    }
    // free the cached block of `device` (-1: of every device) unless a uc_lp_create is using it; returns the bytes freed
    static size_t release(int device) {
        Cache& C = cache();
        std::lock_guard<std::mutex> g(C.mu);
        size_t freed = 0;
        int prev = -1; cudaGetDevice(&prev);
        for (int d = 0; d < (int)C.base.size(); ++d) {
            if ((device >= 0 && d != device) || !C.base[(size_t)d] || C.busy[(size_t)d]) continue;
            cudaSetDevice(d);
            cudaFree(C.base[(size_t)d]);
            freed += C.cap[(size_t)d]; C.base[(size_t)d] = nullptr; C.cap[(size_t)d] = 0;
        }
        if (prev >= 0) cudaSetDevice(prev);
        return freed;
    }
    void reserve(size_t bytes, int device) {
        dev = device;
        Cache& C = cache();
        {
            std::lock_guard<std::mutex> g(C.mu);
            if ((int)C.base.size() <= dev) { C.base.resize((size_t)dev + 1, nullptr); C.cap.resize((size_t)dev + 1, 0); C.busy.resize((size_t)dev + 1, 0); }
            if (!C.busy[(size_t)dev] && C.base[(size_t)dev] && C.cap[(size_t)dev] >= bytes) {
                base = (char*)C.base[(size_t)dev]; cap = C.cap[(size_t)dev]; C.busy[(size_t)dev] = 1; cached = true;
                return;
            }
        }
        CK(cudaMalloc((void**)&base, bytes)); cap = bytes;
    }
    template <class T> T* get(size_t count) {
        const size_t bytes = ((count * sizeof(T) + 255) / 256 + 1) * 256;
        if (used + bytes > cap) throw CudaFail{cudaErrorMemoryAllocation, "temporary arena of uc_lp_create"};
        T* p = (T*)(base + used); used += bytes; return p;
    }
};
struct DevCsr { long long* ptr = nullptr; int* col = nullptr; double* val = nullptr; };   // the caller's CSR on the device
struct DevPerm { long long* perm = nullptr; long long* inv = nullptr; long long nshort = 0; };

long long d2h_ll(const long long* d, cudaStream_t st) {
    long long h = 0;
    CK(cudaMemcpyAsync(&h, d, sizeof h, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return h;
}
// new -> old permutation of N rows with lengths len (uc_format.hpp build_perm), its inverse, and the short-row count
DevPerm device_perm(uc_lp* lp, TempArena& T, const int* len, long long N, int thr, long long window, cudaStream_t st) {
    DevPerm P;
    P.perm = lp->dalloc<long long>((size_t)N); P.inv = T.get<long long>((size_t)N + 1);
    if (N == 0) return P;
    int* flag = T.get<int>((size_t)N); int* rank = T.get<int>((size_t)N + 1);
    k_ing_short_flag<<<ing_grid(N), kIngestBlock, 0, st>>>(len, N, thr, flag);
    size_t bytes = 0;
    CK(cub::DeviceScan::ExclusiveSum(nullptr, bytes, flag, rank, N, st));
    void* tmp = T.get<char>(bytes);
    CK(cub::DeviceScan::ExclusiveSum(tmp, bytes, flag, rank, N, st));
    int h_rank = 0, h_flag = 0;
    CK(cudaMemcpyAsync(&h_rank, rank + (N - 1), sizeof(int), cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(&h_flag, flag + (N - 1), sizeof(int), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    P.nshort = (long long)h_rank + h_flag;
    unsigned long long *k0 = T.get<unsigned long long>((size_t)P.nshort + 1), *k1 = T.get<unsigned long long>((size_t)P.nshort + 1);
    int *v0 = T.get<int>((size_t)P.nshort + 1), *v1 = T.get<int>((size_t)P.nshort + 1);
    k_ing_perm_keys<<<ing_grid(N), kIngestBlock, 0, st>>>(len, rank, N, thr, window, P.nshort, k0, v0, P.perm);
    if (P.nshort > 0) {
        const unsigned long long maxkey = (unsigned long long)((P.nshort - 1) / window) * (unsigned long long)(thr + 1) + (unsigned long long)thr;
        const int end_bit = bits_for(maxkey);
        CK(cub::DeviceRadixSort::SortPairs(nullptr, bytes, k0, k1, v0, v1, P.nshort, 0, end_bit, st));
        tmp = T.get<char>(bytes);
        CK(cub::DeviceRadixSort::SortPairs(tmp, bytes, k0, k1, v0, v1, P.nshort, 0, end_bit, st));    // stable
    }
    k_ing_perm_finish<<<ing_grid(N), kIngestBlock, 0, st>>>(v1, P.nshort, N, P.perm, P.inv);
    return P;
}
// One side (K or K'): slice pointers, sliced-ELL arrays, long tail, 16-bit offsets, schedule.  Returns the device
// layout; fills the counters of the handle through the out parameters.
struct SideStats { int64_t slots = 0, long_nnz = 0, narrow = 0; };
Sell device_side(uc_lp* lp, TempArena& T, const FillSrc& S, const int* len, long long N, const DevPerm& P, const long long* inv_other,
                 bool compress, bool want_src, int ctas, int warps_per_cta, cudaStream_t st, SideStats& stats,
                 std::vector<int64_t>* h_src, std::vector<int64_t>* h_lsrc) {
    Sell A{};
    const long long nshort = P.nshort, nlong = N - nshort, nslices = (nshort + 31) / 32;
    // slice pointers
    long long* slots = T.get<long long>((size_t)nslices + 1);
    long long* sp = lp->dalloc<long long>((size_t)nslices + 1);
    if (nslices) k_ing_slice_width<<<ing_grid(nslices), kIngestBlock, 0, st>>>(len, P.perm, nshort, nslices, slots);
    size_t bytes = 0; void* tmp = nullptr;
    if (nslices) {
        CK(cub::DeviceScan::ExclusiveSum(nullptr, bytes, slots, sp, nslices, st));
        tmp = T.get<char>(bytes);
        CK(cub::DeviceScan::ExclusiveSum(tmp, bytes, slots, sp, nslices, st));
    }
    k_ing_close_scan<<<1, 32, 0, st>>>(sp, slots, nslices);
    // long tail pointers
    long long* llen = T.get<long long>((size_t)nlong + 1);
    long long* lptr = lp->dalloc<long long>((size_t)nlong + 1);
    if (nlong) {
        k_ing_long_len<<<ing_grid(nlong), kIngestBlock, 0, st>>>(len, P.perm, nshort, nlong, llen);
        CK(cub::DeviceScan::ExclusiveSum(nullptr, bytes, llen, lptr, nlong, st));
        tmp = T.get<char>(bytes);
        CK(cub::DeviceScan::ExclusiveSum(tmp, bytes, llen, lptr, nlong, st));
    }
    k_ing_close_scan<<<1, 32, 0, st>>>(lptr, llen, nlong);
    const long long nslots = d2h_ll(sp + nslices, st), lnnz = d2h_ll(lptr + nlong, st);
    if (nslots >= (1LL << 31)) throw TooLarge{"more than 2^31 stored slots in one sliced-ELL layout (step descriptors address entries / 32 in 26 bits)"};
    stats.slots = nslots; stats.long_nnz = lnnz;
    // arrays (zeroed by dalloc: padding slots are (col 0, val 0.0))
    int* col = lp->dalloc<int>((size_t)nslots);
    double* val = lp->dalloc<double>((size_t)nslots);
    int* lcol = lp->dalloc<int>((size_t)lnnz);
    double* lval = lp->dalloc<double>((size_t)lnnz);
    long long *src = nullptr, *lsrc = nullptr;
    if (want_src) {
        src = T.get<long long>((size_t)nslots + 1); lsrc = T.get<long long>((size_t)lnnz + 1);
        CK(cudaMemsetAsync(src, 0xff, sizeof(long long) * (size_t)nslots, st));             // -1 = padding
    }
    if (nshort) k_ing_fill_sell<<<ing_grid(nshort), kIngestBlock, 0, st>>>(S, P.perm, inv_other, nshort, sp, col, val, src);
    if (nlong) k_ing_fill_long<<<ing_grid(nlong * 32), kIngestBlock, 0, st>>>(S, P.perm, inv_other, nshort, nlong, lptr, lcol, lval, lsrc);
    // 16-bit offsets
    int* cbase = lp->dalloc<int>((size_t)nslices);
    long long* narrow_of = T.get<long long>((size_t)nslices + 1);
    long long* narrow_sum = T.get<long long>(1);
    unsigned short* col16 = nullptr;
    long long narrow = 0;
    if (nslices) {
        k_ing_slice_base<<<ing_grid(nslices * 32), kIngestBlock, 0, st>>>(len, P.perm, nshort, nslices, sp, col, compress ? 1 : 0, cbase, narrow_of);
        CK(cub::DeviceReduce::Sum(nullptr, bytes, narrow_of, narrow_sum, nslices, st));
        tmp = T.get<char>(bytes);
        CK(cub::DeviceReduce::Sum(tmp, bytes, narrow_of, narrow_sum, nslices, st));
        narrow = d2h_ll(narrow_sum, st);
        if (narrow > 0) {
            col16 = lp->dalloc<unsigned short>((size_t)nslots);
            k_ing_col16<<<ing_grid(nshort), kIngestBlock, 0, st>>>(len, P.perm, nshort, nslices, sp, col, cbase, col16);
        }
    }
    stats.narrow = narrow;
    // schedule on the host from the slice bases and the per-slice index bases
    HostSell H;
    H.nslices = nslices; H.nshort = nshort; H.nlong = nlong; H.nrows = N;
    H.slice_ptr.assign((size_t)nslices + 1, 0); H.cbase.assign((size_t)nslices, -1);
    CK(cudaMemcpyAsync(H.slice_ptr.data(), sp, sizeof(long long) * (size_t)(nslices + 1), cudaMemcpyDeviceToHost, st));
    if (nslices) CK(cudaMemcpyAsync(H.cbase.data(), cbase, sizeof(int) * (size_t)nslices, cudaMemcpyDeviceToHost, st));
    if (want_src) {
        h_src->resize((size_t)nslots); h_lsrc->resize((size_t)lnnz);
        if (nslots) CK(cudaMemcpyAsync(h_src->data(), src, sizeof(long long) * (size_t)nslots, cudaMemcpyDeviceToHost, st));
        if (lnnz) CK(cudaMemcpyAsync(h_lsrc->data(), lsrc, sizeof(long long) * (size_t)lnnz, cudaMemcpyDeviceToHost, st));
    }
    CK(cudaStreamSynchronize(st));
    build_schedule(H, ctas, warps_per_cta);
    A.sp = sp; A.col = col; A.col16 = col16; A.cbase = cbase; A.val = val;
    A.nshort = nshort; A.nslices = (int)nslices; A.nblk = cdiv(nslices, kWarps);
    A.lp = lptr; A.lcol = lcol; A.lval = lval; A.nlong = (int)nlong; A.nlblk = cdiv(nlong, kWarps);
    A.grid = std::max(1, A.nlblk + A.nblk);
    A.steps = lp->upload(H.steps);
    A.steps_per_warp = (int)H.steps_per_warp; A.sched_warps = (int)H.sched_warps;
    A.nslots = nslots;
    if (narrow == nslots && nslots > 0) { lp->dfree(col); A.col = nullptr; }            // every slice is narrow: the 32-bit copy is not kept
    return A;
}

// two-stage reduction of a device array into one device double (op 0: sum of squares, 1: max |v|); stream-ordered, no sync
void reduce_to_dev(const double* v, long long count, int op, dd* part, double* out_dev, cudaStream_t st) {
    int blocks = count > 0 ? (int)std::min<long long>(1024, (count + kBlock - 1) / kBlock) : 1;
    k_reduce<<<blocks, kBlock, 0, st>>>(v, count, op, part);
    k_reduce_final<<<1, 32, 0, st>>>(part, blocks, op, out_dev);
}
// two-stage reduction of a device array to one host double (op 0: sum of squares, 1: max |v|)
double reduce_to_host(uc_lp* lp, const double* v, long long count, int op, dd* part, double* out_dev, cudaStream_t st) {
    int blocks = count > 0 ? std::min<long long>(1024, (count + kBlock - 1) / kBlock) : 1;
    k_reduce<<<blocks, kBlock, 0, st>>>(v, count, op, part);
    k_reduce_final<<<1, 32, 0, st>>>(part, blocks, op, out_dev);
    double h = 0.0;
    CK(cudaMemcpyAsync(&h, out_dev, sizeof(double), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    (void)lp;
    return h;
}

// R1: Ruiz x ruiz_iters, then Pock-Chambolle(alpha); accumulates Dr, Dc; scales both layouts.
void precondition(uc_lp* lp, cudaStream_t st, double* r, double* s) {      // r[m], s[n]: scratch of the caller
    const long long m = lp->m, n = lp->n;
    k_vec_fill<<<cdiv(std::max<long long>(m, 1), 256), 256, 0, st>>>(lp->Dr, 1.0, m);
    k_vec_fill<<<cdiv(std::max<long long>(n, 1), 256), 256, 0, st>>>(lp->Dc, 1.0, n);
    const double alpha = lp->opt.pc_alpha;
    const int passes = lp->opt.ruiz_iters + (alpha > 0.0 ? 1 : 0);
    for (int pass = 0; pass < passes; ++pass) {
        const bool ruiz = pass < lp->opt.ruiz_iters;
        int mode_r = ruiz ? 0 : (alpha == 1.0 ? 1 : 2), mode_c = mode_r;
        double p_r = 2.0 - alpha, p_c = alpha;
        k_row_stat<<<lp->K.grid, kBlock, 0, st>>>(lp->K, mode_r, p_r, r);
        k_row_stat<<<lp->KT.grid, kBlock, 0, st>>>(lp->KT, mode_c, p_c, s);
        k_scale_matrix<<<lp->K.grid, kBlock, 0, st>>>(lp->K, r, s);
        k_scale_matrix<<<lp->KT.grid, kBlock, 0, st>>>(lp->KT, s, r);
        k_vec_mul<<<cdiv(std::max<long long>(m, 1), 256), 256, 0, st>>>(lp->Dr, r, m);
        k_vec_mul<<<cdiv(std::max<long long>(n, 1), 256), 256, 0, st>>>(lp->Dc, s, n);
    }
    CK(cudaGetLastError());
}

// The factors of the step rule depend on the attempt counter only.  They are tabulated on the host with
// the C library's pow (correctly rounded in all but freak cases), because one ulp in eta is amplified
// exponentially by the adaptive rule and CUDA's pow is only 2-ulp accurate.
// The table covers the attempts the device can reach before the host looks again, not iter_limit: it starts at
// kPowtabStart entries and the launch loop doubles it ahead of the attempt counter (grow_powtab), so a huge
// iteration limit costs nothing up front and a cancel is never stuck behind table building.
constexpr long long kPowtabStart = 1 << 18;
void fill_powtab(std::vector<double2>& h, long long from, long long to) {     // entries for attempts from+1 .. to
    h.resize((size_t)(to - from));
    for (long long k = from + 1; k <= to; ++k) h[(size_t)(k - from - 1)] = make_double2(std::pow((double)(k + 1), -0.6), std::pow((double)(k + 1), -0.3));
}
void ensure_powtab(uc_lp* lp, long long need) {
    need = std::max<long long>(need, 4096);
    if (need <= lp->powtab_len) return;
    std::vector<double2> h;
    fill_powtab(h, 0, need);
    if (lp->powtab) { cudaFree(lp->powtab); lp->powtab = nullptr; lp->powtab_len = 0; }
    CK(cudaMalloc((void**)&lp->powtab, sizeof(double2) * (size_t)need));
    CK(cudaMemcpy(lp->powtab, h.data(), sizeof(double2) * (size_t)need, cudaMemcpyHostToDevice));
    lp->powtab_len = need;
}
// Grow the table to at least `need` entries while a solve is in flight on `st`: the new table is complete before
// the pointer in Ctrl is switched (stream-ordered, i.e. between two graph launches); the old table is kept in
// `retired` until the solve has drained the stream.
void grow_powtab(uc_lp* lp, long long need, long long limit, cudaStream_t st, std::vector<double2*>& retired) {
    if (need <= lp->powtab_len) return;
    const long long len = std::min<long long>(limit, std::max<long long>(need, 2 * lp->powtab_len));
    std::vector<double2> h;
    fill_powtab(h, lp->powtab_len, len);
    double2* nt = nullptr;
    CK(cudaMalloc((void**)&nt, sizeof(double2) * (size_t)len));
    CK(cudaMemcpyAsync(nt, lp->powtab, sizeof(double2) * (size_t)lp->powtab_len, cudaMemcpyDeviceToDevice, st));
    CK(cudaMemcpyAsync(nt + lp->powtab_len, h.data(), sizeof(double2) * h.size(), cudaMemcpyHostToDevice, st));
    CK(cudaStreamSynchronize(st));                    // `h` is pageable and goes out of scope; the loop keeps 2 launches queued
    retired.push_back(lp->powtab);
    lp->powtab = nt; lp->powtab_len = len;
    CK(cudaMemcpyAsync(&lp->ctl->powtab, &lp->powtab, sizeof(double2*), cudaMemcpyHostToDevice, st));
}

// The two attempt kernels are launched with programmatic stream serialization (PDL): a kernel's prologue
// (schedule loads, first index copies) overlaps the tail of the kernel before it; the kernel itself waits
// (griddepcontrol.wait) before it reads anything a previous kernel wrote.  Captured into the graph as
// programmatic dependency edges.
template <class Kern>
void launch_pdl(Kern kern, int grid, int threads, size_t smem, cudaStream_t st, const Sell& A, const Vecs& V, Ctrl* ctl) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)threads); cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    CK(cudaLaunchKernelEx(&cfg, kern, A, V, ctl));
}
// Both attempt kernels ask for the SAME amount of dynamic shared memory, so that an SM never changes its L1 / shared
// memory split between them (the two alternate ~20,000 times per second)
#ifdef UC_SMEM_REQUEST
constexpr size_t kAttemptSmemBytes = UC_SMEM_REQUEST;
#else
constexpr size_t kAttemptSmemBytes = kPrimalSmemBytes > kDualSmemBytes ? kPrimalSmemBytes : kDualSmemBytes;
#endif
static_assert(kAttemptSmemBytes >= kPrimalSmemBytes && kAttemptSmemBytes >= kDualSmemBytes, "shared memory request");
void launch_primal(uc_lp* lp, cudaStream_t st) { launch_pdl(k_primal, lp->V.gridPA, (lp->KT.cta_warps + 1) * 32, kAttemptSmemBytes, st, lp->KT, lp->V, lp->ctl); }
void launch_dual(uc_lp* lp, cudaStream_t st) { launch_pdl(k_dual, lp->V.gridPB, (lp->K.cta_warps + 1) * 32, kAttemptSmemBytes, st, lp->K, lp->V, lp->ctl); }
void launch_attempt(uc_lp* lp, cudaStream_t st) { launch_primal(lp, st); launch_dual(lp, st); }
void launch_kkt(uc_lp* lp, cudaStream_t st, int mode) {
    const int flush = mode == kModeCheck;        // the periodic check also applies the pending average term (R6)
    k_check_dual<<<lp->V.gridA, kBlock, 0, st>>>(lp->KT, lp->V, lp->ctl, flush);
    k_check_primal<<<lp->V.gridB, kBlock, 0, st>>>(lp->K, lp->V, lp->ctl, flush);
    k_check_finalize<<<1, kFinalBlock, 0, st>>>(lp->V, lp->ctl, mode);
}
void launch_check(uc_lp* lp, cudaStream_t st) {
    launch_kkt(lp, st, kModeCheck);
    k_restart_vec<<<lp->V.gridR, kBlock, 0, st>>>(lp->V, lp->ctl);
    k_restart_finalize<<<1, kFinalBlock, 0, st>>>(lp->V, lp->ctl);
}
constexpr int kCheckLaunches = 5;

// R2: control block, initial point, KKT components of the restart point z^0 (4 launches); synchronises `st`.
void start_run(uc_lp* lp, const uc_pdhg_params& prm, cudaStream_t st, long long limit, bool fixed,
               const double* dx0, const double* dy0, uc_attempt_record* d_att, uc_check_record* d_chk) {
    ensure_powtab(lp, std::min<long long>(limit, kPowtabStart));
    Ctrl h{};
    h.eta = prm.eta0 > 0.0 ? prm.eta0 : lp->eta0;                  // R2b: state carried over from an earlier solve, else R2
    h.omega = prm.omega0 > 0.0 ? prm.omega0 : lp->omega0;
    h.eta_prev = 0.0; h.w = 0.0; h.mu_prev = INFINITY;
    h.limit = limit; h.fixed = fixed ? 1 : 0; h.status = UC_ITERATION_LIMIT;
    h.eps_abs = prm.eps_abs; h.eps_rel = prm.eps_rel; h.beta_s = prm.beta_sufficient; h.beta_n = prm.beta_necessary;
    h.beta_a = prm.beta_artificial; h.smoothing = prm.weight_smoothing; h.norm_q = lp->norm_b; h.norm_c = lp->norm_c;
    h.att = d_att; h.att_cap = d_att ? prm.attempt_trace_cap : 0; h.chk = d_chk; h.chk_cap = d_chk ? prm.check_trace_cap : 0;
    h.host_stop = lp->d_stop; h.host_status = lp->d_status; h.powtab = lp->powtab;
    h.gen = (int)((lp->state.load() >> 1) & 0x0fffffffu);
    CK(cudaMemcpyAsync(lp->ctl, &h, sizeof(Ctrl), cudaMemcpyHostToDevice, st));
    k_init_point<<<lp->V.gridR, kBlock, 0, st>>>(lp->V, dx0, dy0, lp->perm_c, lp->perm_r);
    launch_kkt(lp, st, kModeInit);
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(st));                     // the pageable Ctrl copy and any staged warm start are consumed
}


// capture `ce` attempts + one check into an executable graph (A15)
void build_graph(uc_lp* lp, int ce) {
    if (lp->exec && lp->graph_ce == ce) return;
    if (lp->exec) { cudaGraphExecDestroy(lp->exec); lp->exec = nullptr; }
    cudaGraph_t g = nullptr;
    CK(cudaStreamBeginCapture(lp->own_stream, cudaStreamCaptureModeThreadLocal));
    for (int i = 0; i < ce; ++i) launch_attempt(lp, lp->own_stream);
    launch_check(lp, lp->own_stream);
    CK(cudaStreamEndCapture(lp->own_stream, &g));
    CK(cudaGraphInstantiate(&lp->exec, g, 0));
    CK(cudaGraphDestroy(g));
    lp->graph_ce = ce;
    lp->graph_nodes = 2 * ce + kCheckLaunches;
}

void destroy_impl(uc_lp* lp) {
    if (!lp) return;
    cudaSetDevice(lp->device);
    if (lp->exec) cudaGraphExecDestroy(lp->exec);
    for (auto& e : lp->ev) if (e) cudaEventDestroy(e);
    if (lp->ev_t0) cudaEventDestroy(lp->ev_t0);
    if (lp->ev_t1) cudaEventDestroy(lp->ev_t1);
    for (void* p : lp->allocs) if (p) cudaFree(p);
    if (lp->powtab) cudaFree(lp->powtab);
    if (lp->h_status) cudaFreeHost(lp->h_status);        // one allocation: the stop flag lives behind the status record
    if (lp->own_stream) cudaStreamDestroy(lp->own_stream);
    delete lp;
}

int64_t bytes_per_attempt(const uc_lp* lp) {
    // what one attempt streams in THIS layout: matrix slots (8 B value + 4 B index, or 2 B index in a narrow
    // slice; padding included), step descriptors (16 B per scheduled step, padding steps included), and per variable 8 (x) + 24 (c,l,u) + 16 (xsum r/w) + 8 (x') + 16 ({xbar,dx}) + 16
    // (gather of the pair) = 88 B, per row 8 (y) + 8 (q) + 1 (sense) + 16 (ysum r/w) + 8 (y') + 8 (gather) = 49 B
    return 12 * (lp->k_slots + lp->kt_slots + lp->k_long_nnz + lp->kt_long_nnz) - 2 * (lp->k_narrow + lp->kt_narrow) +
           16 * ((int64_t)lp->K.steps_per_warp * lp->K.sched_warps + (int64_t)lp->KT.steps_per_warp * lp->KT.sched_warps) +
           88 * lp->n + 49 * lp->m;
}

}  // namespace

// ================================================================================== C ABI
extern "C" {

const char* uc_last_error(void) { return g_err.c_str(); }


// Host-only check of A0/A1 (no device): builds the permutations, both SELL-32 layouts and both attempt schedules
// exactly as uc_lp_create does and verifies them against the caller's CSR.  Returns UC_OK or UC_ERR_INVALID with
// the first violated property in uc_last_error().
int uc_host_layout_selftest(int64_t m, int64_t n, int64_t nnz, const int64_t* row_ptr, const int32_t* col_idx, const double* val,
                            int32_t sell_window, int32_t long_row_threshold, int32_t sched_ctas, int32_t warps_per_cta) {
    if (m < 0 || n < 0 || nnz < 0 || !row_ptr || sell_window < 32 || long_row_threshold < 1 || sched_ctas < 1 || warps_per_cta < 1)
        return fail(UC_ERR_INVALID, "bad argument");
    try {
    HostProblem P;
    build_perms(m, n, nnz, row_ptr, col_idx, sell_window, long_row_threshold, P);
    build_K(row_ptr, col_idx, val, true, P);
    build_KT(row_ptr, col_idx, val, true, P);
    compress_columns(P.K, true);
    compress_columns(P.KT, true);
    build_schedule(P.K, sched_ctas, warps_per_cta);
    build_schedule(P.KT, sched_ctas, warps_per_cta);
    auto bad = [&](const std::string& what) { return fail(UC_ERR_INVALID, what); };
    // ---- permutations: bijections, rows with <= threshold entries first, the others last in the caller's order
    auto check_perm = [&](const std::vector<int64_t>& perm, const std::vector<int64_t>& inv, int64_t N, int64_t nshort,
                          const std::vector<int64_t>& len) -> const char* {
        if ((int64_t)perm.size() != N || (int64_t)inv.size() != N) return "permutation size";
        std::vector<char> seen((size_t)N, 0);
        for (int64_t k = 0; k < N; ++k) {
            const int64_t o = perm[(size_t)k];
            if (o < 0 || o >= N || seen[(size_t)o]) return "not a permutation";
            seen[(size_t)o] = 1;
            if (inv[(size_t)o] != k) return "inverse permutation";
            if ((k < nshort) != (len[(size_t)o] <= long_row_threshold)) return "short / long split";
            if (k > nshort && perm[(size_t)k - 1] > o) return "long rows out of order";
        }
        return nullptr;
    };
    std::vector<int64_t> lenr((size_t)m);
    for (int64_t i = 0; i < m; ++i) lenr[(size_t)i] = row_ptr[i + 1] - row_ptr[i];
    if (const char* w = check_perm(P.perm_r, P.inv_r, m, P.nshort_r, lenr)) return bad(std::string("rows: ") + w);
    if (const char* w = check_perm(P.perm_c, P.inv_c, n, P.nshort_c, P.lenc)) return bad(std::string("columns: ") + w);
    // ---- expected K' rows: for column j the entries (i, K_ij) in ascending caller row order (what the sequential
    // statement's column scatter produces)
    std::vector<std::vector<std::pair<int64_t, int64_t>>> cols((size_t)n);       // (row, CSR position)
    for (int64_t i = 0; i < m; ++i)
        for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) cols[(size_t)col_idx[p]].push_back({i, p});
    // ---- layouts: every stored entry is the caller's entry, in the caller's order, relabelled; padding is (0, 0.0)
    auto check_sell = [&](const HostSell& S, bool transposed) -> std::string {
        const std::vector<int64_t>& perm = transposed ? P.perm_c : P.perm_r;
        const std::vector<int64_t>& inv_other = transposed ? P.inv_r : P.inv_c;
        const int64_t N = transposed ? n : m;
        if (S.nrows != N || S.nshort + S.nlong != N || S.nslices != (S.nshort + 31) / 32) return "counts";
        auto row_len = [&](int64_t o) { return transposed ? (int64_t)cols[(size_t)o].size() : row_ptr[o + 1] - row_ptr[o]; };
        auto entry = [&](int64_t o, int64_t t, int64_t& c_new, double& v, int64_t& pos) {
            if (transposed) { pos = cols[(size_t)o][(size_t)t].second; c_new = inv_other[(size_t)cols[(size_t)o][(size_t)t].first]; }
            else { pos = row_ptr[o] + t; c_new = inv_other[(size_t)col_idx[pos]]; }
            v = val[pos];
        };
        for (int64_t s = 0; s < S.nslices; ++s) {
            int64_t w = 0;
            for (int64_t r = 32 * s; r < std::min<int64_t>(32 * s + 32, S.nshort); ++r) w = std::max(w, row_len(perm[(size_t)r]));
            if (S.slice_ptr[(size_t)s + 1] - S.slice_ptr[(size_t)s] != 32 * w) return "slice width";
            for (int64_t lane = 0; lane < 32; ++lane) {
                const int64_t r = 32 * s + lane;
                const int64_t len = r < S.nshort ? row_len(perm[(size_t)r]) : 0;
                for (int64_t t = 0; t < w; ++t) {
                    const size_t k = (size_t)(S.slice_ptr[(size_t)s] + 32 * t + lane);
                    if (t < len) {
                        int64_t c_new, pos; double v;
                        entry(perm[(size_t)r], t, c_new, v, pos);
                        if (S.col[k] != (int32_t)c_new || std::memcmp(&S.val[k], &v, sizeof v) != 0 || S.src[k] != pos) return "stored entry";
                    } else if (S.col[k] != 0 || S.val[k] != 0.0 || S.src[k] != -1) return "padding slot";
                }
            }
        }
        for (int64_t r = 0; r < S.nlong; ++r) {
            const int64_t o = perm[(size_t)(S.nshort + r)];
            if (S.lptr[(size_t)r + 1] - S.lptr[(size_t)r] != row_len(o)) return "long row length";
            for (int64_t t = 0; t < row_len(o); ++t) {
                int64_t c_new, pos; double v;
                entry(o, t, c_new, v, pos);
                const size_t k = (size_t)(S.lptr[(size_t)r] + t);
                if (S.lcol[k] != (int32_t)c_new || std::memcmp(&S.lval[k], &v, sizeof v) != 0 || S.lsrc[k] != pos) return "long row entry";
            }
        }
        // ---- 16-bit column offsets: a narrow slice decodes to the 32-bit indices bit for bit, its span fits 16 bits,
        // and a slice is wide only if its span does not fit
        if ((int64_t)S.cbase.size() != S.nslices) return "cbase size";
        for (int64_t s = 0; s < S.nslices; ++s) {
            const int32_t cb = S.cbase[(size_t)s];
            int32_t lo = INT32_MAX, hi = -1;
            for (int64_t lane = 0; lane < 32 && 32 * s + lane < S.nshort; ++lane) {
                const int64_t len = row_len(perm[(size_t)(32 * s + lane)]);
                for (int64_t t = 0; t < len; ++t) {
                    const size_t k = (size_t)(S.slice_ptr[(size_t)s] + 32 * t + lane);
                    lo = std::min(lo, S.col[k]); hi = std::max(hi, S.col[k]);
                    if (cb >= 0 && cb + (int32_t)S.col16[k] != S.col[k]) return "16-bit column offset does not decode to the index";
                }
            }
            if (hi >= 0) {
                if (cb >= 0 && (cb != lo || hi - lo > 65535)) return "narrow slice base / span";
                if (cb < 0 && (int64_t)hi - lo <= 65535) return "a slice that fits 16 bits is stored wide";
            }
        }
        // ---- schedule: every slice exactly once, as consecutive chunks of one warp, flags and offsets right
        const int64_t W = S.sched_warps, J = S.steps_per_warp;
        if ((int64_t)S.steps.size() != W * J) return "schedule size";
        std::vector<int> done((size_t)S.nslices, 0);
        for (int64_t wq = 0; wq < W; ++wq) {
            bool ended = false; int64_t prev_slice = -1;
            for (int64_t j = 0; j < J; ) {
                const StepDesc d = S.steps[(size_t)(j * W + wq)];
                const uint32_t info = d.w0 >> 26;
                if (ended) { if (d.w0 != 0 || d.row0 != 0 || d.cbase != -1) return "step after the end marker"; ++j; continue; }
                if (info & kStepEnd) { if ((info & 31) != 0) return "end marker carries work"; ended = true; ++j; continue; }
                if (!(info & kStepFirst) || d.row0 % 32) return "slice does not start with its first chunk";
                const int64_t sl = d.row0 / 32;
                if (sl < 0 || sl >= S.nslices || done[(size_t)sl]++) return "slice scheduled twice or out of range";
                if (sl <= prev_slice) return "a warp's slices are not ascending";
                prev_slice = sl;
                const int64_t wd = (S.slice_ptr[(size_t)sl + 1] - S.slice_ptr[(size_t)sl]) / 32;
                const int64_t nch = std::max<int64_t>(1, (wd + kChunkT - 1) / kChunkT);
                for (int64_t c = 0; c < nch; ++c, ++j) {
                    if (j >= J) return "slice cut off by the end of the schedule";
                    const StepDesc e = S.steps[(size_t)(j * W + wq)];
                    const uint32_t ei = e.w0 >> 26;
                    const int64_t nt = std::max<int64_t>(0, std::min<int64_t>(kChunkT, wd - kChunkT * c));
                    if (e.row0 != d.row0 || e.cbase != S.cbase[(size_t)sl] || (int64_t)(ei & 7) != nt || ((ei & kStepFirst) != 0) != (c == 0) ||
                        ((ei & kStepLast) != 0) != (c == nch - 1) || (ei & kStepEnd) ||
                        ((int64_t)(e.w0 & 0x3ffffffu) << 5) != S.slice_ptr[(size_t)sl] + 32 * kChunkT * c)
                        return "chunk descriptor";
                }
            }
            if (!ended && J > 0) {                       // a warp without end marker must own the full J steps
                const uint32_t li = S.steps[(size_t)((J - 1) * W + wq)].w0 >> 26;
                if (!(li & kStepLast)) return "last step of a full warp is not a last chunk";
            }
        }
        for (int64_t sl = 0; sl < S.nslices; ++sl) if (done[(size_t)sl] != 1) return "slice not scheduled";
        // ---- a CTA owns one contiguous range of slices, ranges in CTA order
        if (W != (int64_t)sched_ctas * warps_per_cta) return "schedule width";
        int64_t prev_hi = -1;
        for (int64_t c = 0; c < sched_ctas; ++c) {
            int64_t lo = S.nslices, hi = -1, cnt = 0;
            for (int64_t wq = c * warps_per_cta; wq < (c + 1) * warps_per_cta; ++wq)
                for (int64_t j = 0; j < J; ++j) {
                    const StepDesc d = S.steps[(size_t)(j * W + wq)];
                    if (!((d.w0 >> 26) & kStepFirst)) continue;
                    const int64_t sl = d.row0 / 32;
                    lo = std::min(lo, sl); hi = std::max(hi, sl); ++cnt;
                }
            if (cnt == 0) continue;
            if (hi - lo + 1 != cnt) return "the slices of a CTA are not one contiguous range";
            if (lo != prev_hi + 1) return "CTA ranges out of order";
            prev_hi = hi;
        }
        return "";
    };
    std::string w = check_sell(P.K, false);
    if (!w.empty()) return bad("K layout: " + w);
    w = check_sell(P.KT, true);
    if (!w.empty()) return bad("K' layout: " + w);
    } catch (const std::exception& e) {                        // nothing may unwind through the C ABI
        return fail(std_code(e), std::string("uc_host_layout_selftest: ") + e.what());
    }
    return UC_OK;
}

double uc_host_log_rounded(double a) { return log_rounded(a); }
double uc_host_exp_rounded(double x) { return exp_rounded(x); }

void uc_lp_default_options(uc_lp_options* o) {
    if (!o) return;
    o->device = -1; o->ruiz_iters = 10; o->pc_alpha = 1.0; o->sell_window = 4096; o->long_row_threshold = 32;
    o->keep_source_map = 0; o->index_compression = 1; o->host_ingest = 0; o->max_ctas = 0;
}

void uc_pdhg_default_params(uc_pdhg_params* p) {
    if (!p) return;
    std::memset(p, 0, sizeof *p);
    p->iter_limit = 100000; p->eps_rel = 1e-4; p->eps_abs = 1e-4;
    p->time_limit_s = std::numeric_limits<double>::infinity();
    p->check_every = 64; p->fixed_iterations = 0;
    p->beta_sufficient = 0.2; p->beta_necessary = 0.8; p->beta_artificial = 0.36; p->weight_smoothing = 0.5;
}

int uc_lp_create(int64_t m, int64_t n, int64_t nnz, const int64_t* row_ptr, const int32_t* col_idx, const double* val,
                 const char* sense, const double* b, const double* c, const double* l, const double* u,
                 const uc_lp_options* opt_in, uc_lp** out) {
    if (!out) return fail(UC_ERR_INVALID, "out is NULL");
    *out = nullptr;
    const double t_create = now_s();
    uc_lp_options opt;
    uc_lp_default_options(&opt);
    if (opt_in) opt = *opt_in;
    if (opt.ruiz_iters < 0 || opt.pc_alpha < 0.0 || opt.pc_alpha > 2.0 || opt.sell_window < 32 || opt.long_row_threshold < 1 || opt.max_ctas < 0)
        return fail(UC_ERR_INVALID, "bad uc_lp_options");
    const bool tim = std::getenv("UC_CREATE_TIMING") != nullptr;
    double tph = now_s();
    auto phase = [&](const char* what) { if (tim) { double t = now_s(); std::fprintf(stderr, "  create: %-28s %7.2f ms\n", what, (t - tph) * 1e3); tph = t; } };
    std::string why = validate_args(m, n, nnz, row_ptr, col_idx, val, sense, b, c, l, u);
    if (!why.empty()) return fail(UC_ERR_INVALID, why);
    // A0: the arrays are scanned on a helper thread while this thread copies them to the device; no kernel reads them
    // before the verdict is in (join_validation), and bad input is still rejected when there is no device at all
    std::string why_entries;
    std::thread validator([&] {
        try { why_entries = validate_entries(m, n, nnz, row_ptr, col_idx, val, sense, b, c, l, u); }
        catch (...) { why_entries = "host allocation failed during validation"; }
    });
    bool validated = false;
    auto join_validation = [&]() { if (!validated) { validator.join(); validated = true; } return why_entries.empty(); };

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        if (!join_validation()) return fail(UC_ERR_INVALID, why_entries);
        return fail(UC_ERR_CUDA, "no CUDA device: this library has no CPU path");
    }
    int dev = opt.device;
    if (dev < 0 && cudaGetDevice(&dev) != cudaSuccess) { join_validation(); return fail(UC_ERR_CUDA, "cudaGetDevice failed"); }
    if (dev >= ndev) { join_validation(); return fail(UC_ERR_INVALID, "device ordinal out of range"); }

    uc_lp* lp = nullptr;
    try {
        lp = new uc_lp();
        lp->device = dev; lp->m = m; lp->n = n; lp->nnz = nnz; lp->opt = opt;
        DeviceGuard guard(dev);
        CK(cudaStreamCreateWithFlags(&lp->own_stream, cudaStreamNonBlocking));
        for (auto& e : lp->ev) CK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        CK(cudaEventCreate(&lp->ev_t0)); CK(cudaEventCreate(&lp->ev_t1));
        cudaStream_t st = lp->own_stream;

        const bool want_src = opt.keep_source_map != 0;
        int sms = 0, warpsPA = kPrimalWarps, warpsPB = kDualWarps;
        CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        // persistent grids of the attempt kernels: kCtasPerSm CTAs per SM, never more CTAs than work, and no more
        // consumer warps per CTA than the slices need (at least kMinWarps, at most the compiled maximum)
        auto attempt_shape = [&](int64_t nshort, int64_t nlong, int max_warps, int& grid, int& warps) {
            int64_t cap = (int64_t)kCtasPerSm * std::max(sms, 1);
            if (opt.max_ctas > 0) cap = std::min<int64_t>(cap, opt.max_ctas);
            const int64_t slices = (nshort + 31) / 32;
            warps = (int)std::max<int64_t>(std::min<int64_t>(kMinWarps, max_warps), std::min<int64_t>(max_warps, (slices + cap - 1) / cap));
            grid = (int)std::max<int64_t>(1, std::min<int64_t>(cap, std::max<int64_t>((slices + warps - 1) / warps, nlong)));
        };
        auto attempt_grids = [&](int64_t nshort_r, int64_t nshort_c, int& gridPA, int& gridPB) {
            attempt_shape(nshort_c, n - nshort_c, kPrimalWarps, gridPA, warpsPA);
            attempt_shape(nshort_r, m - nshort_r, kDualWarps, gridPB, warpsPB);
        };
        int gridPA = 1, gridPB = 1;
        // temporaries of this call: the data vectors in the caller's order, and (device ingest) the caller's CSR with
        // everything the ingest kernels and sorts need
        TempArena T;
        {
            const size_t vec_bytes = (size_t)8 * (size_t)(2 * m + 4 * n) + (size_t)m + 12 * 512 + sizeof(dd) * 1024 + 4096;
            const size_t src_bytes = want_src ? 16 * ((size_t)nnz + 32 * (size_t)(m + n) / 32 + 1024) * 3 : 0;
            const size_t ingest_bytes = opt.host_ingest ? 0 : (size_t)(8 * (m + 1) + 44 * nnz + 28 * n + 4 * m + 44 * (m + n)) +
                                        ((size_t)(m + n) / 32 + 2) * 40 + src_bytes + 256 * 64 + ((size_t)64 << 20);
            T.reserve(vec_bytes + ingest_bytes, dev);
        }
        TempArena& TV = T;
        double* db = TV.get<double>((size_t)m + 1); double* dc = TV.get<double>((size_t)n + 1);
        double* dl = TV.get<double>((size_t)n + 1); double* du = TV.get<double>((size_t)n + 1);
        char* dsense = TV.get<char>((size_t)m + 1);
        dd* part = TV.get<dd>(1024); double* scal = TV.get<double>(8);
        double* rscr = TV.get<double>((size_t)m + 1); double* sscr = TV.get<double>((size_t)n + 1);      // Ruiz / Pock-Chambolle factors of a pass
        cudaError_t vec_err = cudaSuccess;
        std::thread vec_up([&] {
            cudaSetDevice(dev);
            cudaStream_t s2 = nullptr;
            vec_err = cudaStreamCreateWithFlags(&s2, cudaStreamNonBlocking);
            auto up = [&](void* d, const void* h, size_t bytes) { if (vec_err == cudaSuccess && bytes) vec_err = cudaMemcpyAsync(d, h, bytes, cudaMemcpyHostToDevice, s2); };
            up(db, b, sizeof(double) * (size_t)m); up(dc, c, sizeof(double) * (size_t)n);
            up(dl, l, sizeof(double) * (size_t)n); up(du, u, sizeof(double) * (size_t)n); up(dsense, sense, (size_t)m);
            if (vec_err == cudaSuccess) vec_err = cudaStreamSynchronize(s2);
            if (s2) cudaStreamDestroy(s2);
        });
        struct Joiner { std::thread& t; ~Joiner() { if (t.joinable()) t.join(); } } vec_joiner{vec_up};
        phase("stream/events");
        if (!opt.host_ingest) {
            // ---- A1 on the device (uc_ingest.cuh): one copy of the caller's CSR, then kernels
            long long* d_ptr = T.get<long long>((size_t)m + 1);
            int* d_col = T.get<int>((size_t)nnz + 1);
            double* d_val = T.get<double>((size_t)nnz + 1);
            CK(cudaMemcpyAsync(d_ptr, row_ptr, sizeof(long long) * (size_t)(m + 1), cudaMemcpyHostToDevice, st));
            if (nnz) {
                CK(cudaMemcpyAsync(d_col, col_idx, sizeof(int) * (size_t)nnz, cudaMemcpyHostToDevice, st));
                CK(cudaMemcpyAsync(d_val, val, sizeof(double) * (size_t)nnz, cudaMemcpyHostToDevice, st));
            }
            phase("H2D of the CSR");
            if (!join_validation()) { destroy_impl(lp); return fail(UC_ERR_INVALID, why_entries); }
            phase("validation verdict");
            int* lenr = T.get<int>((size_t)m + 1); int* lenc = T.get<int>((size_t)n + 1);
            int* rowid = T.get<int>((size_t)nnz + 1);
            CK(cudaMemsetAsync(lenc, 0, sizeof(int) * (size_t)(n + 1), st));
            if (m) k_ing_row_len<<<ing_grid(m), kIngestBlock, 0, st>>>(d_ptr, m, lenr);
            if (nnz) {
                k_ing_col_count<<<ing_grid(nnz), kIngestBlock, 0, st>>>(d_col, nnz, lenc);
                k_ing_row_ids<<<ing_grid(nnz), kIngestBlock, 0, st>>>(d_ptr, m, nnz, rowid);
            }
            DevPerm Pr = device_perm(lp, T, lenr, m, opt.long_row_threshold, opt.sell_window, st);
            DevPerm Pc = device_perm(lp, T, lenc, n, opt.long_row_threshold, opt.sell_window, st);
            attempt_grids(Pr.nshort, Pc.nshort, gridPA, gridPB);
            // explicit transpose: column pointers + the entries in (column, caller's row) order
            long long* tptr = T.get<long long>((size_t)n + 2);
            int* order = T.get<int>((size_t)nnz + 1);
            {
                long long* wide = T.get<long long>((size_t)n + 1);
                size_t bytes = 0; void* tmp = nullptr;
                if (n) {
                    k_ing_widen<<<ing_grid(n), kIngestBlock, 0, st>>>(lenc, wide, n);
                    CK(cub::DeviceScan::ExclusiveSum(nullptr, bytes, wide, tptr, n, st));
                    tmp = T.get<char>(bytes);
                    CK(cub::DeviceScan::ExclusiveSum(tmp, bytes, wide, tptr, n, st));
                }
                k_ing_close_scan<<<1, 32, 0, st>>>(tptr, wide, n);
                if (nnz) {
                    unsigned* k0 = reinterpret_cast<unsigned*>(d_col);                     // column indices are >= 0
                    unsigned* k1 = T.get<unsigned>((size_t)nnz + 1);
                    int* v0 = T.get<int>((size_t)nnz + 1);
                    k_ing_iota<<<ing_grid(nnz), kIngestBlock, 0, st>>>(v0, nnz);
                    const int end_bit = bits_for((unsigned long long)std::max<int64_t>(n - 1, 1));
                    CK(cub::DeviceRadixSort::SortPairs(nullptr, bytes, k0, k1, v0, order, nnz, 0, end_bit, st));
                    tmp = T.get<char>(bytes);
                    CK(cub::DeviceRadixSort::SortPairs(tmp, bytes, k0, k1, v0, order, nnz, 0, end_bit, st));   // stable: rows ascend inside a column
                }
            }
            SideStats sk, skt;
            lp->K = device_side(lp, T, FillSrc{d_ptr, nullptr, d_col, d_val}, lenr, m, Pr, Pc.inv, opt.index_compression != 0, want_src,
                                gridPB, warpsPB, st, sk, &lp->k_src, &lp->k_lsrc);
            lp->KT = device_side(lp, T, FillSrc{tptr, order, rowid, d_val}, lenc, n, Pc, Pr.inv, opt.index_compression != 0, want_src,
                                 gridPA, warpsPA, st, skt, &lp->kt_src, &lp->kt_lsrc);
            lp->k_slots = sk.slots; lp->kt_slots = skt.slots; lp->k_long_nnz = sk.long_nnz; lp->kt_long_nnz = skt.long_nnz;
            lp->k_narrow = sk.narrow; lp->kt_narrow = skt.narrow;
            lp->perm_r = Pr.perm; lp->perm_c = Pc.perm;
            phase("device ingest");
        } else {
        // ---- A1 on the host (uc_format.hpp; the checker's builders): layouts on up to 8 threads, then uploaded.  The K
        // side (layout, schedule, upload) runs on a helper thread while this thread transposes and builds the K' side.
        if (!join_validation()) { destroy_impl(lp); return fail(UC_ERR_INVALID, why_entries); }
        HostProblem P;
        build_perms(m, n, nnz, row_ptr, col_idx, opt.sell_window, opt.long_row_threshold, P);
        phase("perms");
        attempt_grids(P.nshort_r, P.nshort_c, gridPA, gridPB);
        std::exception_ptr k_side_error;
        std::thread k_side([&] {
            try {
                cudaSetDevice(dev);
                build_K(row_ptr, col_idx, val, want_src, P);
                if (P.K.col.size() >= (size_t)1 << 31) throw TooLarge{"more than 2^31 stored slots in one sliced-ELL layout"};
                compress_columns(P.K, opt.index_compression != 0);
                build_schedule(P.K, gridPB, warpsPB);
                lp->K = upload_sell(lp, P.K);
            } catch (...) { k_side_error = std::current_exception(); }
        });
        try {
            build_KT(row_ptr, col_idx, val, want_src, P);
            phase("build_KT");
            if (P.KT.col.size() >= (size_t)1 << 31) throw TooLarge{"more than 2^31 stored slots in one sliced-ELL layout"};
            compress_columns(P.KT, opt.index_compression != 0);
            phase("compress KT");
            build_schedule(P.KT, gridPA, warpsPA);
            phase("schedule KT");
            lp->KT = upload_sell(lp, P.KT);
            phase("upload KT");
        } catch (...) { k_side.join(); throw; }
        k_side.join();
        phase("join K side");
        if (k_side_error) std::rethrow_exception(k_side_error);
        lp->k_slots = (int64_t)P.K.col.size(); lp->kt_slots = (int64_t)P.KT.col.size();
        lp->k_long_nnz = (int64_t)P.K.lcol.size(); lp->kt_long_nnz = (int64_t)P.KT.lcol.size();
        lp->k_narrow = P.K.narrow_slots; lp->kt_narrow = P.KT.narrow_slots;
        lp->perm_r = (long long*)lp->upload(P.perm_r);
        lp->perm_c = (long long*)lp->upload(P.perm_c);
        if (opt.keep_source_map) { lp->k_src = std::move(P.K.src); lp->k_lsrc = std::move(P.K.lsrc); lp->kt_src = std::move(P.KT.src); lp->kt_lsrc = std::move(P.KT.lsrc); }

        }
        lp->K.ncols = n; lp->KT.ncols = m; lp->K.cta_warps = warpsPB; lp->KT.cta_warps = warpsPA;
        Vecs& V = lp->V;
        V.n = n; V.m = m;
        lp->reserve_arena((size_t)(13 * 8 + 16) * (size_t)(n + 64) + (size_t)(9 * 8 + 1) * (size_t)(m + 64) + ((size_t)1 << 20));   // incl. the four staging vectors
        for (int i = 0; i < 2; ++i) { V.x[i] = lp->dalloc<double>((size_t)n); V.y[i] = lp->dalloc<double>((size_t)m); }
        V.xg = lp->dalloc<double2>((size_t)n);
        V.xsum = lp->dalloc<double>((size_t)n); V.ysum = lp->dalloc<double>((size_t)m);
        V.xr = lp->dalloc<double>((size_t)n); V.yr = lp->dalloc<double>((size_t)m);
        lp->stage_x = lp->dalloc<double>((size_t)n); lp->stage_y = lp->dalloc<double>((size_t)m);
        lp->cs = lp->dalloc<double>((size_t)n); lp->ls = lp->dalloc<double>((size_t)n); lp->us = lp->dalloc<double>((size_t)n);
        lp->qs = lp->dalloc<double>((size_t)m); lp->isG = lp->dalloc<unsigned char>((size_t)m);
        lp->Dr = lp->dalloc<double>((size_t)m); lp->Dc = lp->dalloc<double>((size_t)n);
        V.c = lp->cs; V.l = lp->ls; V.u = lp->us; V.q = lp->qs; V.isG = lp->isG; V.Dr = lp->Dr; V.Dc = lp->Dc;
        V.gridR = std::max(1, cdiv(n + m, kBlock));
        {   // check kernels: persistent blocks, kCheckMinBlocks per SM, grid-stride over the layout's 256-row blocks
            int sms = 0;
            CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
            const int cap = kCheckMinBlocks * std::max(opt.max_ctas > 0 ? std::min(sms, opt.max_ctas) : sms, 1);
            V.gridA = std::max(1, std::min(cap, lp->KT.grid)); V.gridB = std::max(1, std::min(cap, lp->K.grid));
        }
        V.gridPA = gridPA; V.gridPB = gridPB;
        CK(cudaFuncSetAttribute(k_primal, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kAttemptSmemBytes));
        CK(cudaFuncSetAttribute(k_dual, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kAttemptSmemBytes));
        V.partA = lp->dalloc<dd>((size_t)V.gridPA);
        V.partB = lp->dalloc<dd>((size_t)2 * V.gridPB);
        V.partD = lp->dalloc<dd>((size_t)8 * V.gridA);
        V.partP = lp->dalloc<dd>((size_t)6 * V.gridB);
        V.partR = lp->dalloc<dd>((size_t)2 * V.gridR);
        lp->ctl = lp->dalloc<Ctrl>(1);
        CK(cudaMemsetAsync(lp->ctl, 0, sizeof(Ctrl), st));
        // the two host <-> device mailboxes share ONE mapped pinned allocation (the status record, then the stop flag on
        // its own 128-byte line): pinned allocations and their release are slow, synchronising driver calls
        static_assert(sizeof(HostStatus) <= 128, "mailbox layout");
        CK(cudaHostAlloc((void**)&lp->h_status, 256, cudaHostAllocMapped));
        lp->h_stop = reinterpret_cast<int*>(reinterpret_cast<char*>(lp->h_status) + 128);
        std::memset(lp->h_status, 0, 256);
        CK(cudaHostGetDevicePointer((void**)&lp->d_status, lp->h_status, 0));
        CK(cudaHostGetDevicePointer((void**)&lp->d_stop, lp->h_stop, 0));

        vec_up.join();
        if (vec_err != cudaSuccess) throw CudaFail{vec_err, "upload of b, c, l, u, sense"};
        phase("vectors alloc + upload");
        // unscaled norms for R9 (before anything is scaled); A2, A3: preconditioning; A4: scaled data and the initial
        // scalars of R2.  The six scalars come back in ONE copy.
        reduce_to_dev(db, m, 0, part, scal + 0, st);
        reduce_to_dev(dc, n, 0, part, scal + 1, st);
        CK(cudaEventRecord(lp->ev_t0, st));
        precondition(lp, st, rscr, sscr);
        k_scale_problem<<<V.gridR, kBlock, 0, st>>>(n, m, db, dc, dl, du, dsense, lp->perm_c, lp->perm_r, lp->Dr, lp->Dc,
                                                    lp->qs, lp->cs, lp->ls, lp->us, lp->isG);
        CK(cudaGetLastError());
        reduce_to_dev(lp->K.val, lp->k_slots, 1, part, scal + 2, st);
        reduce_to_dev(lp->K.lval, lp->k_long_nnz, 1, part, scal + 3, st);
        reduce_to_dev(lp->cs, n, 0, part, scal + 4, st);
        reduce_to_dev(lp->qs, m, 0, part, scal + 5, st);
        CK(cudaEventRecord(lp->ev_t1, st));
        double hs[6];
        CK(cudaMemcpyAsync(hs, scal, sizeof hs, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        T.quiesced = true;                               // last use of the temporary arena (scal, part) is done
        float ms = 0.f; CK(cudaEventElapsedTime(&ms, lp->ev_t0, lp->ev_t1));
        lp->precondition_seconds = ms * 1e-3;
        lp->norm_b = std::sqrt(hs[0]); lp->norm_c = std::sqrt(hs[1]);
        const double kmax = std::max(hs[2], hs[3]), ncs = std::sqrt(hs[4]), nqs = std::sqrt(hs[5]);
        lp->eta0 = kmax > 0.0 ? 1.0 / kmax : 1.0;
        lp->omega0 = (ncs > 1e-10 && nqs > 1e-10) ? ncs / nqs : 1.0;
        lp->norm_qs = nqs;
        phase("precondition + scalars");
        lp->create_seconds = now_s() - t_create;
    } catch (const CudaFail& f) {
        std::string msg = std::string(f.what) + ": " + cudaGetErrorString(f.e);
        int code = (f.e == cudaErrorMemoryAllocation) ? UC_ERR_NOMEM : UC_ERR_CUDA;
        join_validation();
        destroy_impl(lp);
        return fail(code, msg);
    } catch (const TooLarge& t) {
        join_validation();
        destroy_impl(lp);
        return fail(UC_ERR_INVALID, t.what);
    } catch (const std::bad_alloc&) {
        join_validation();
        destroy_impl(lp);
        return fail(UC_ERR_NOMEM, "host allocation failed");
    } catch (const std::exception& e) {                       // std::system_error of a helper thread, std::length_error, ...
        join_validation();
        destroy_impl(lp);
        return fail(std_code(e), std::string("uc_lp_create: ") + e.what());
    }
    join_validation();
    *out = lp;
    return UC_OK;
}

void uc_lp_destroy(uc_lp* lp) { destroy_impl(lp); }

int uc_release_scratch(int32_t device, int64_t* bytes_released) {
    if (device < -1) return fail(UC_ERR_INVALID, "uc_release_scratch: device must be an ordinal or -1");
    const size_t freed = TempArena::release(device);
    if (bytes_released) *bytes_released = (int64_t)freed;
    return UC_OK;
}

int uc_lp_update_bounds(uc_lp* lp, const double* l_new, const double* u_new) {
    if (!lp || (lp->n > 0 && (!l_new || !u_new))) return fail(UC_ERR_INVALID, "NULL argument");
    for (int64_t j = 0; j < lp->n; ++j)
        if (std::isnan(l_new[j]) || std::isnan(u_new[j]) || l_new[j] > u_new[j]) return fail(UC_ERR_INVALID, "bad bound");
    int expected = 0;
    if (!lp->busy.compare_exchange_strong(expected, 1)) return fail(UC_ERR_BUSY, "a solve is running on this handle");
    int rc = UC_OK;
    try {
        DeviceGuard guard(lp->device);
        if (!lp->stage_x0) lp->stage_x0 = lp->dalloc<double>((size_t)lp->n);          // first use on this handle; kept
        double *dl = lp->stage_x, *du = lp->stage_x0;
        // on the handle's stream (a non-blocking one: a copy on the legacy stream would not be ordered before the kernel,
        // nor after the zero-fill of a fresh stage_x0)
        if (lp->n) {
            CK(cudaMemcpyAsync(dl, l_new, sizeof(double) * (size_t)lp->n, cudaMemcpyHostToDevice, lp->own_stream));
            CK(cudaMemcpyAsync(du, u_new, sizeof(double) * (size_t)lp->n, cudaMemcpyHostToDevice, lp->own_stream));
        }
        k_scale_bounds<<<std::max(1, cdiv(lp->n, kBlock)), kBlock, 0, lp->own_stream>>>(lp->n, dl, du, lp->perm_c, lp->Dc, lp->ls, lp->us);
        CK(cudaGetLastError());
        CK(cudaStreamSynchronize(lp->own_stream));
    } catch (const CudaFail& f) {
        rc = fail(UC_ERR_CUDA, std::string(f.what) + ": " + cudaGetErrorString(f.e));
    }
    lp->busy.store(0);
    return rc;
}

int uc_lp_update_objective(uc_lp* lp, const double* c_new) {
    if (!lp || (lp->n > 0 && !c_new)) return fail(UC_ERR_INVALID, "NULL argument");
    for (int64_t j = 0; j < lp->n; ++j)
        if (!std::isfinite(c_new[j])) return fail(UC_ERR_INVALID, "c has a non-finite entry");
    int expected = 0;
    if (!lp->busy.compare_exchange_strong(expected, 1)) return fail(UC_ERR_BUSY, "a solve is running on this handle");
    int rc = UC_OK;
    try {
        DeviceGuard guard(lp->device);
        cudaStream_t st = lp->own_stream;
        if (!lp->upd_part) { lp->upd_part = lp->dalloc<dd>(1024); lp->upd_scal = lp->dalloc<double>(8); }   // first call on this handle; kept
        double* dc = lp->stage_x; dd* part = lp->upd_part; double* scal = lp->upd_scal;
        if (lp->n) CK(cudaMemcpyAsync(dc, c_new, sizeof(double) * (size_t)lp->n, cudaMemcpyHostToDevice, st));
        lp->norm_c = std::sqrt(reduce_to_host(lp, dc, lp->n, 0, part, scal, st));            // unscaled ||c|| of R9
        k_scale_cost<<<std::max(1, cdiv(lp->n, kBlock)), kBlock, 0, st>>>(lp->n, dc, lp->perm_c, lp->Dc, lp->cs);
        CK(cudaGetLastError());
        const double ncs = std::sqrt(reduce_to_host(lp, lp->cs, lp->n, 0, part, scal, st));   // R2: omega0 = ||c~|| / ||q~||
        lp->omega0 = (ncs > 1e-10 && lp->norm_qs > 1e-10) ? ncs / lp->norm_qs : 1.0;
    } catch (const CudaFail& f) {
        rc = fail(UC_ERR_CUDA, std::string(f.what) + ": " + cudaGetErrorString(f.e));
    }
    lp->busy.store(0);
    return rc;
}

int uc_pdhg_cancel(uc_lp* lp) {
    if (!lp) return fail(UC_ERR_INVALID, "handle is NULL");
    const unsigned st = lp->state.load();
    if ((st & 1u) && lp->h_stop) __atomic_store_n(lp->h_stop, (int)(((st >> 1) & 0x0fffffffu) << 3) | UC_CANCELLED, __ATOMIC_SEQ_CST);
    else lp->cancel_requested.store(1);
    return UC_OK;
}

int uc_pdhg_cancel_clear(uc_lp* lp, int32_t* was_pending) {
    if (!lp) return fail(UC_ERR_INVALID, "handle is NULL");
    const int had = lp->cancel_requested.exchange(0);
    if (was_pending) *was_pending = had;
    return UC_OK;
}

static int solve_impl(uc_lp* lp, const uc_pdhg_params* pin, double* x_out, double* y_out, uc_pdhg_result* res, bool dev_io) {
    if (!lp || !res) return fail(UC_ERR_INVALID, "handle or result is NULL");
    uc_pdhg_params prm;
    uc_pdhg_default_params(&prm);
    if (pin) prm = *pin;
    if (prm.check_every <= 0 || prm.iter_limit < 0 || prm.fixed_iterations < 0 || !(prm.eps_rel >= 0.0) || !(prm.eps_abs >= 0.0) ||
        prm.attempt_trace_cap < 0 || prm.check_trace_cap < 0 || !(prm.eta0 >= 0.0) || !(prm.omega0 >= 0.0) ||
        !std::isfinite(prm.eta0) || !std::isfinite(prm.omega0))
        return fail(UC_ERR_INVALID, "bad uc_pdhg_params");
    int expected = 0;
    if (!lp->busy.compare_exchange_strong(expected, 1)) return fail(UC_ERR_BUSY, "a solve is already running on this handle");
    std::memset(res, 0, sizeof *res);
    const double t_wall = now_s();
    int rc = UC_OK;
    bool in_flight = false;
    uc_attempt_record* d_att = nullptr; uc_check_record* d_chk = nullptr;
    try {
        DeviceGuard guard(lp->device);
        cudaStream_t st = prm.stream ? (cudaStream_t)prm.stream : lp->own_stream;
        const long long n = lp->n, m = lp->m;
        const bool fixed = prm.fixed_iterations > 0;
        const long long limit = fixed ? prm.fixed_iterations : prm.iter_limit;
        const int ce = prm.check_every;

        // a cancel that arrived while the handle was idle is honoured here (PAPER.md l.80-85 race): nothing runs,
        // x_out / y_out are left untouched
        if (lp->cancel_requested.exchange(0)) {
            res->status = UC_CANCELLED;
            res->solve_seconds = now_s() - t_wall;
            lp->busy.store(0);
            return UC_OK;
        }
        // from here on uc_pdhg_cancel stamps the stop flag with this solve's generation
        const unsigned gen = ((lp->state.load() >> 1) + 1u) & 0x0fffffffu;
        lp->state.store((gen << 1) | 1u);
        in_flight = true;
        const int my_cancel = (int)(gen << 3) | UC_CANCELLED, my_timeout = (int)(gen << 3) | UC_TIME_LIMIT;
        std::memset(lp->h_status, 0, sizeof(HostStatus));

        // warm start
        const double *dx0 = nullptr, *dy0 = nullptr;
        if (prm.x0) {
            if (dev_io) dx0 = prm.x0;
            else {
                if (!lp->stage_x0) lp->stage_x0 = lp->dalloc<double>((size_t)n);      // first warm start on this handle; kept
                CK(cudaMemcpyAsync(lp->stage_x0, prm.x0, sizeof(double) * (size_t)n, cudaMemcpyHostToDevice, st)); dx0 = lp->stage_x0;
            }
        }
        if (prm.y0) {
            if (dev_io) dy0 = prm.y0;
            else {
                if (!lp->stage_y0) lp->stage_y0 = lp->dalloc<double>((size_t)m);
                CK(cudaMemcpyAsync(lp->stage_y0, prm.y0, sizeof(double) * (size_t)m, cudaMemcpyHostToDevice, st)); dy0 = lp->stage_y0;
            }
        }
        if (prm.attempt_trace && prm.attempt_trace_cap > 0) CK(cudaMalloc((void**)&d_att, sizeof(uc_attempt_record) * (size_t)prm.attempt_trace_cap));
        if (prm.check_trace && prm.check_trace_cap > 0) CK(cudaMalloc((void**)&d_chk, sizeof(uc_check_record) * (size_t)prm.check_trace_cap));

        int64_t launches = 0;
        start_run(lp, prm, st, limit, fixed, dx0, dy0, d_att, d_chk);
        launches += 4;
        build_graph(lp, ce);

        // ---- the loop: one graph launch = `ce` attempts + one check; two launches kept in flight
        CK(cudaEventRecord(lp->ev_t0, st));
        const long long nblocks = limit / ce, rem = limit % ce;
        const int depth = 2;
        bool done = false;
        long long b = 0;
        std::vector<double2*> retired_powtabs;
        for (; b < nblocks && !done; ++b) {
            if ((b + 8) * ce > lp->powtab_len && lp->powtab_len < limit) grow_powtab(lp, std::min<long long>(limit, (b + 8) * ce), limit, st, retired_powtabs);
            CK(cudaGraphLaunch(lp->exec, st));
            launches += lp->graph_nodes;
            CK(cudaEventRecord(lp->ev[b % depth], st));
            if (b >= depth - 1) {
                CK(cudaEventSynchronize(lp->ev[(b - depth + 1) % depth]));
                if (((volatile HostStatus*)lp->h_status)->done) done = true;
                // a cancel that saw the handle idle just as this solve started
                if (!done && lp->cancel_requested.exchange(0)) __atomic_store_n(lp->h_stop, my_cancel, __ATOMIC_SEQ_CST);
                if (!done && now_s() - t_wall > prm.time_limit_s) {      // never overwrites a cancel of this solve
                    int cur = __atomic_load_n(lp->h_stop, __ATOMIC_SEQ_CST);
                    if (cur != my_cancel) __atomic_compare_exchange_n(lp->h_stop, &cur, my_timeout, false, __ATOMIC_SEQ_CST, __ATOMIC_SEQ_CST);
                }
            }
        }
        CK(cudaStreamSynchronize(st));
        done = ((volatile HostStatus*)lp->h_status)->done != 0;
        if (!done && rem > 0) {
            grow_powtab(lp, limit, limit, st, retired_powtabs);
            for (long long r = 0; r < rem; ++r) launch_attempt(lp, st);
            launches += 2 * rem;
            if (!fixed) { launch_check(lp, st); launches += kCheckLaunches; }
            CK(cudaStreamSynchronize(st));
            done = ((volatile HostStatus*)lp->h_status)->done != 0;
        }
        CK(cudaEventRecord(lp->ev_t1, st));
        for (double2* t : retired_powtabs) cudaFree(t);     // the stream has drained: nobody reads the old tables
        if (!done) {                                       // fixed-iteration end (R14) or iter_limit = 0: report only
            launch_kkt(lp, st, kModeReport);
            launches += 3;
        }
        // ---- A14: unscale, un-permute, hand back
        double* ox = x_out; double* oy = y_out;
        if (!dev_io) {
            if (x_out) ox = lp->stage_x;
            if (y_out) oy = lp->stage_y;
        }
        if (ox || oy) { k_output<<<lp->V.gridR, kBlock, 0, st>>>(lp->V, lp->ctl, ox, oy, lp->perm_c, lp->perm_r); launches += 1; }
        CK(cudaGetLastError());
        if (!dev_io) {
            if (x_out && n) CK(cudaMemcpyAsync(x_out, ox, sizeof(double) * (size_t)n, cudaMemcpyDeviceToHost, st));
            if (y_out && m) CK(cudaMemcpyAsync(y_out, oy, sizeof(double) * (size_t)m, cudaMemcpyDeviceToHost, st));
        }
        Ctrl hc;
        CK(cudaMemcpyAsync(&hc, lp->ctl, sizeof(Ctrl), cudaMemcpyDeviceToHost, st));
        if (d_att) { long long cnt = std::min<long long>(prm.attempt_trace_cap, limit); if (cnt > 0) CK(cudaMemcpyAsync(prm.attempt_trace, d_att, sizeof(uc_attempt_record) * (size_t)cnt, cudaMemcpyDeviceToHost, st)); }
        if (d_chk) CK(cudaMemcpyAsync(prm.check_trace, d_chk, sizeof(uc_check_record) * (size_t)prm.check_trace_cap, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        float ms = 0.f; CK(cudaEventElapsedTime(&ms, lp->ev_t0, lp->ev_t1));

        const HostStatus hs = *lp->h_status;
        res->status = hc.status; res->returned_average = hc.ret_avg;
        res->iterations = hc.k; res->accepted = hc.accepted; res->restarts = hc.restarts;
        res->rel_kkt = hs.rel_kkt; res->rel_primal_res = hs.rel_rp; res->rel_dual_res = hs.rel_rd; res->rel_gap = hs.rel_gap;
        res->primal_obj = hs.pobj; res->dual_obj = hs.dobj; res->eta = hc.eta; res->omega = hc.omega;
        res->loop_seconds = ms * 1e-3;
        res->attempt_records = hc.k; res->check_records = hc.nchk;
        res->kernel_launches = launches;
    } catch (const CudaFail& f) {
        rc = fail((f.e == cudaErrorMemoryAllocation) ? UC_ERR_NOMEM : UC_ERR_CUDA, std::string(f.what) + ": " + cudaGetErrorString(f.e));
    } catch (const std::exception& e) {                        // nothing may unwind through the C ABI
        rc = fail(std_code(e), std::string("uc_pdhg_solve: ") + e.what());
    }
    if (d_att) cudaFree(d_att);
    if (d_chk) cudaFree(d_chk);
    res->solve_seconds = now_s() - t_wall;
    if (in_flight) {
        // the solve is over: a cancel stamped with its generation is stale from now on (it cannot leak into the next
        // solve), and one that slipped into cancel_requested while it was starting is consumed with it
        lp->state.store(lp->state.load() & ~1u);
        lp->cancel_requested.store(0);
    }
    lp->busy.store(0);
    return rc;
}

int uc_pdhg_solve(uc_lp* lp, const uc_pdhg_params* p, double* x_out, double* y_out, uc_pdhg_result* res) {
    return solve_impl(lp, p, x_out, y_out, res, false);
}
int uc_pdhg_solve_device(uc_lp* lp, const uc_pdhg_params* p, double* x_out, double* y_out, uc_pdhg_result* res) {
    return solve_impl(lp, p, x_out, y_out, res, true);
}

int uc_pdhg_solve_batch(uc_lp* const* handles, int32_t count, const uc_pdhg_params* params, double* const* x_out,
                        double* const* y_out, uc_pdhg_result* results, int32_t max_concurrent) {
    if (count < 0 || (count > 0 && (!handles || !results))) return fail(UC_ERR_INVALID, "bad argument");
    if (params && (params->stream || params->x0 || params->y0 || params->attempt_trace || params->check_trace))
        return fail(UC_ERR_INVALID, "uc_pdhg_solve_batch: stream, warm start and trace fields must be NULL (they are per solve)");
    for (int32_t i = 0; i < count; ++i) {
        if (!handles[i]) return fail(UC_ERR_INVALID, "a handle is NULL");
        for (int32_t j = 0; j < i; ++j) if (handles[j] == handles[i]) return fail(UC_ERR_INVALID, "the same handle appears twice");
    }
    const int workers = std::max(1, std::min<int>(count, max_concurrent > 0 ? max_concurrent : 16));
    std::atomic<int32_t> next{0};
    std::vector<int> rcs((size_t)count, UC_OK);
    std::vector<std::string> errs((size_t)count);
    auto work = [&]() {
        for (;;) {
            const int32_t i = next.fetch_add(1);
            if (i >= count) return;
            rcs[(size_t)i] = solve_impl(handles[i], params, x_out ? x_out[i] : nullptr, y_out ? y_out[i] : nullptr, &results[i], false);
            if (rcs[(size_t)i] != UC_OK) errs[(size_t)i] = g_err;       // thread-local text of the worker
        }
    };
    // Workers are joined on every way out of this scope: a std::thread that is destroyed while joinable ends the process,
    // and nothing may unwind through the C ABI.  If a worker cannot be started (std::system_error), the ones that did start
    // and the calling thread drain the queue between them.
    struct Pool { std::vector<std::thread> th; ~Pool() { for (auto& t : th) if (t.joinable()) t.join(); } };
    std::string spawn_err; int spawn_code = UC_ERR_INTERNAL;
    {
        Pool pool;
        try {
            pool.th.reserve((size_t)workers);
            for (int w = 1; w < workers; ++w) pool.th.emplace_back(work);
        } catch (const std::exception&) { /* fewer workers than asked for */ }
        try { work(); } catch (const std::exception& e) { spawn_err = e.what(); spawn_code = std_code(e); next.store(count); }
    }
    if (!spawn_err.empty()) return fail(spawn_code, "uc_pdhg_solve_batch: " + spawn_err);
    for (int32_t i = 0; i < count; ++i)
        if (rcs[(size_t)i] != UC_OK) return fail(rcs[(size_t)i], "solve " + std::to_string(i) + ": " + errs[(size_t)i]);
    return UC_OK;
}

int uc_pdhg_time_kernels(uc_lp* lp, void* stream, int32_t attempts, double* primal_ms, double* dual_ms) {
    if (!lp || attempts <= 0 || !primal_ms || !dual_ms) return fail(UC_ERR_INVALID, "bad argument");
    int expected = 0;
    if (!lp->busy.compare_exchange_strong(expected, 1)) return fail(UC_ERR_BUSY, "a solve is running on this handle");
    int rc = UC_OK;
    std::vector<cudaEvent_t> ev;
    try {
        DeviceGuard guard(lp->device);
        cudaStream_t st = stream ? (cudaStream_t)stream : lp->own_stream;
        uc_pdhg_params prm; uc_pdhg_default_params(&prm);
        const int warm = 8;
        ensure_powtab(lp, (long long)attempts + warm);      // start_run only sizes the table for the launch loop of a solve
        start_run(lp, prm, st, (long long)attempts + warm, true, nullptr, nullptr, nullptr, nullptr);
        for (int i = 0; i < warm; ++i) launch_attempt(lp, st);
        ev.resize((size_t)2 * attempts + 1);
        for (auto& e : ev) CK(cudaEventCreate(&e));
        CK(cudaEventRecord(ev[0], st));
        for (int i = 0; i < attempts; ++i) {
            launch_primal(lp, st);
            CK(cudaEventRecord(ev[(size_t)2 * i + 1], st));
            launch_dual(lp, st);
            CK(cudaEventRecord(ev[(size_t)2 * i + 2], st));
        }
        CK(cudaStreamSynchronize(st));
        double a = 0.0, b = 0.0;
        for (int i = 0; i < attempts; ++i) {
            float ms = 0.f;
            CK(cudaEventElapsedTime(&ms, ev[(size_t)2 * i], ev[(size_t)2 * i + 1])); a += ms;
            CK(cudaEventElapsedTime(&ms, ev[(size_t)2 * i + 1], ev[(size_t)2 * i + 2])); b += ms;
        }
        *primal_ms = a / attempts; *dual_ms = b / attempts;
    } catch (const CudaFail& f) {
        rc = fail(UC_ERR_CUDA, std::string(f.what) + ": " + cudaGetErrorString(f.e));
    }
    for (auto& e : ev) if (e) cudaEventDestroy(e);
    lp->busy.store(0);
    return rc;
}

int uc_pdhg_timeline(uc_lp* lp, void* stream, int32_t attempts, uint64_t* out, int64_t cap, int32_t* grid_primal, int32_t* grid_dual) {
#ifndef UC_TIMELINE
    (void)lp; (void)stream; (void)attempts; (void)out; (void)cap; (void)grid_primal; (void)grid_dual;
    return fail(UC_ERR_INVALID, "this library was built without -DUC_TIMELINE");
#else
    if (!lp || attempts <= 0 || !out || !grid_primal || !grid_dual) return fail(UC_ERR_INVALID, "bad argument");
    const int64_t need = (int64_t)(lp->V.gridPA + lp->V.gridPB) * kTlWarps * kTlMarks;
    if (cap < need) return fail(UC_ERR_INVALID, "timeline buffer too small: need " + std::to_string(need) + " entries");
    int expected = 0;
    if (!lp->busy.compare_exchange_strong(expected, 1)) return fail(UC_ERR_BUSY, "a solve is running on this handle");
    int rc = UC_OK;
    unsigned long long* d = nullptr;
    try {
        DeviceGuard guard(lp->device);
        cudaStream_t st = stream ? (cudaStream_t)stream : lp->own_stream;
        uc_pdhg_params prm; uc_pdhg_default_params(&prm);
        CK(cudaMalloc((void**)&d, sizeof(unsigned long long) * (size_t)need));
        CK(cudaMemset(d, 0, sizeof(unsigned long long) * (size_t)need));
        ensure_powtab(lp, (long long)attempts);
        start_run(lp, prm, st, (long long)attempts, true, nullptr, nullptr, nullptr, nullptr);
        // the marks of the LAST attempt survive; the dual block starts after the primal block
        for (int i = 0; i < attempts; ++i) {
            const bool last = i == attempts - 1;
            lp->V.tl = last ? d : nullptr;
            launch_primal(lp, st);
            lp->V.tl = last ? d + (size_t)lp->V.gridPA * kTlWarps * kTlMarks : nullptr;
            launch_dual(lp, st);
        }
        lp->V.tl = nullptr;
        CK(cudaMemcpyAsync(out, d, sizeof(unsigned long long) * (size_t)need, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        *grid_primal = lp->V.gridPA; *grid_dual = lp->V.gridPB;
    } catch (const CudaFail& f) {
        rc = fail(UC_ERR_CUDA, std::string(f.what) + ": " + cudaGetErrorString(f.e));
    }
    if (d) cudaFree(d);
    lp->busy.store(0);
    return rc;
#endif
}

int uc_lp_get_info(const uc_lp* lp, uc_lp_info* info) {
    if (!lp || !info) return fail(UC_ERR_INVALID, "NULL argument");
    std::memset(info, 0, sizeof *info);
    info->m = lp->m; info->n = lp->n; info->nnz = lp->nnz;
    info->k_sell_slots = lp->k_slots; info->kt_sell_slots = lp->kt_slots;
    info->k_long_rows = lp->K.nlong; info->kt_long_rows = lp->KT.nlong;
    info->k_long_nnz = lp->k_long_nnz; info->kt_long_nnz = lp->kt_long_nnz;
    info->device_bytes = (int64_t)lp->device_bytes;
    info->precondition_seconds = lp->precondition_seconds; info->create_seconds = lp->create_seconds;
    info->eta0 = lp->eta0; info->omega0 = lp->omega0; info->norm_b = lp->norm_b; info->norm_c = lp->norm_c;
    info->bytes_per_attempt = bytes_per_attempt(lp);
    info->k_narrow_slots = lp->k_narrow; info->kt_narrow_slots = lp->kt_narrow;
    info->scratch_cached_bytes = (int64_t)TempArena::cached_bytes(lp->device);
    return UC_OK;
}

// Test hook for A1: rebuild the permutations, both layouts and both schedules with the HOST builders (uc_format.hpp, the
// code uc_host_layout_selftest checks against the caller's CSR) and compare them bit for bit with what the handle holds
// on the device.  The matrix values are compared only if the handle was created without preconditioning (ruiz_iters = 0,
// pc_alpha = 0), since uc_lp_create scales them in place.
int uc_lp_compare_layout(uc_lp* lp, int64_t m, int64_t n, int64_t nnz, const int64_t* row_ptr, const int32_t* col_idx, const double* val) {
    if (!lp || !row_ptr || m != lp->m || n != lp->n || nnz != lp->nnz) return fail(UC_ERR_INVALID, "bad argument");
    try {
        DeviceGuard guard(lp->device);
        HostProblem P;
        build_perms(m, n, nnz, row_ptr, col_idx, lp->opt.sell_window, lp->opt.long_row_threshold, P);
        build_K(row_ptr, col_idx, val, false, P);
        build_KT(row_ptr, col_idx, val, false, P);
        compress_columns(P.K, lp->opt.index_compression != 0);
        compress_columns(P.KT, lp->opt.index_compression != 0);
        build_schedule(P.K, lp->V.gridPB, lp->K.cta_warps);
        build_schedule(P.KT, lp->V.gridPA, lp->KT.cta_warps);
        const bool scaled = lp->opt.ruiz_iters > 0 || lp->opt.pc_alpha > 0.0;
        std::string why;
        auto same = [&](const char* what, const void* dev, const void* host, size_t bytes) {
            if (!why.empty() || bytes == 0) return;
            if (!dev) { why = std::string(what) + ": missing on the device"; return; }
            std::vector<char> t(bytes);
            CK(cudaMemcpy(t.data(), dev, bytes, cudaMemcpyDeviceToHost));
            if (std::memcmp(t.data(), host, bytes) != 0) {
                size_t k = 0; while (k < bytes && t[k] == ((const char*)host)[k]) ++k;
                why = std::string(what) + ": differs at byte " + std::to_string(k);
            }
        };
        same("row permutation", lp->perm_r, P.perm_r.data(), sizeof(int64_t) * (size_t)m);
        same("column permutation", lp->perm_c, P.perm_c.data(), sizeof(int64_t) * (size_t)n);
        auto side = [&](const char* name, const Sell& D, const HostSell& H) {
            const std::string nm(name);
            if (!why.empty()) return;
            if (D.nshort != H.nshort || D.nslices != H.nslices || D.nlong != H.nlong) { why = nm + ": counts"; return; }
            if (D.steps_per_warp != H.steps_per_warp || D.sched_warps != H.sched_warps) { why = nm + ": schedule shape"; return; }
            const size_t slots = H.col.size();
            same((nm + " slice pointers").c_str(), D.sp, H.slice_ptr.data(), sizeof(int64_t) * H.slice_ptr.size());
            same((nm + " slice index bases").c_str(), D.cbase, H.cbase.data(), sizeof(int32_t) * H.cbase.size());
            if ((size_t)H.narrow_slots < slots) same((nm + " 32-bit column indices").c_str(), D.col, H.col.data(), sizeof(int32_t) * slots);
            else if (D.col && slots) why = nm + ": 32-bit column indices kept although every slice is narrow";
            if (H.narrow_slots > 0) same((nm + " 16-bit column offsets").c_str(), D.col16, H.col16.data(), sizeof(uint16_t) * slots);
            else if (D.col16) why = nm + ": 16-bit offsets present although no slice is narrow";
            if (!scaled) same((nm + " values").c_str(), D.val, H.val.data(), sizeof(double) * slots);
            same((nm + " long-row pointers").c_str(), D.lp, H.lptr.data(), sizeof(int64_t) * H.lptr.size());
            same((nm + " long-row columns").c_str(), D.lcol, H.lcol.data(), sizeof(int32_t) * H.lcol.size());
            if (!scaled) same((nm + " long-row values").c_str(), D.lval, H.lval.data(), sizeof(double) * H.lval.size());
            same((nm + " schedule").c_str(), D.steps, H.steps.data(), sizeof(StepDesc) * H.steps.size());
        };
        side("K", lp->K, P.K);
        side("K'", lp->KT, P.KT);
        if (lp->k_slots != (int64_t)P.K.col.size() || lp->kt_slots != (int64_t)P.KT.col.size() || lp->k_narrow != P.K.narrow_slots ||
            lp->kt_narrow != P.KT.narrow_slots || lp->k_long_nnz != (int64_t)P.K.lcol.size() || lp->kt_long_nnz != (int64_t)P.KT.lcol.size())
            if (why.empty()) why = "slot / narrow / long-row counters";
        if (!why.empty()) return fail(UC_ERR_INVALID, why);
    } catch (const CudaFail& f) {
        return fail(UC_ERR_CUDA, std::string(f.what) + ": " + cudaGetErrorString(f.e));
    } catch (const std::exception& e) {
        return fail(std_code(e), e.what());
    }
    return UC_OK;
}

int uc_lp_get_scaling(uc_lp* lp, double* Dr_out, double* Dc_out) {
    if (!lp) return fail(UC_ERR_INVALID, "handle is NULL");
    try {
        DeviceGuard guard(lp->device);
        std::vector<double> t;
        if (Dr_out) {
            t.resize((size_t)lp->m);
            if (lp->m) CK(cudaMemcpy(t.data(), lp->Dr, sizeof(double) * (size_t)lp->m, cudaMemcpyDeviceToHost));
            std::vector<long long> pr((size_t)lp->m);
            if (lp->m) CK(cudaMemcpy(pr.data(), lp->perm_r, sizeof(long long) * (size_t)lp->m, cudaMemcpyDeviceToHost));
            for (int64_t k = 0; k < lp->m; ++k) Dr_out[pr[(size_t)k]] = t[(size_t)k];
        }
        if (Dc_out) {
            t.resize((size_t)lp->n);
            if (lp->n) CK(cudaMemcpy(t.data(), lp->Dc, sizeof(double) * (size_t)lp->n, cudaMemcpyDeviceToHost));
            std::vector<long long> pc((size_t)lp->n);
            if (lp->n) CK(cudaMemcpy(pc.data(), lp->perm_c, sizeof(long long) * (size_t)lp->n, cudaMemcpyDeviceToHost));
            for (int64_t k = 0; k < lp->n; ++k) Dc_out[pc[(size_t)k]] = t[(size_t)k];
        }
    } catch (const CudaFail& f) {
        return fail(UC_ERR_CUDA, std::string(f.what) + ": " + cudaGetErrorString(f.e));
    } catch (const std::exception& e) {                        // nothing may unwind through the C ABI
        return fail(std_code(e), e.what());
    }
    return UC_OK;
}

int uc_lp_get_scaled_values(uc_lp* lp, int32_t from_transpose, double* val_out) {
    if (!lp || (lp->nnz > 0 && !val_out)) return fail(UC_ERR_INVALID, "NULL argument");
    if (!lp->opt.keep_source_map) return fail(UC_ERR_INVALID, "handle was created without keep_source_map");
    try {
        DeviceGuard guard(lp->device);
        const Sell& S = from_transpose ? lp->KT : lp->K;
        const std::vector<int64_t>& src = from_transpose ? lp->kt_src : lp->k_src;
        const std::vector<int64_t>& lsrc = from_transpose ? lp->kt_lsrc : lp->k_lsrc;
        std::vector<double> t(src.size());
        if (!t.empty()) CK(cudaMemcpy(t.data(), S.val, sizeof(double) * t.size(), cudaMemcpyDeviceToHost));
        for (size_t k = 0; k < src.size(); ++k) if (src[k] >= 0) val_out[src[k]] = t[k];
        t.resize(lsrc.size());
        if (!t.empty()) CK(cudaMemcpy(t.data(), S.lval, sizeof(double) * t.size(), cudaMemcpyDeviceToHost));
        for (size_t k = 0; k < lsrc.size(); ++k) val_out[lsrc[k]] = t[k];
    } catch (const CudaFail& f) {
        return fail(UC_ERR_CUDA, std::string(f.what) + ": " + cudaGetErrorString(f.e));
    } catch (const std::exception& e) {                        // nothing may unwind through the C ABI
        return fail(std_code(e), e.what());
    }
    return UC_OK;
}

int uc_lp_spmv(uc_lp* lp, int32_t transpose, const double* v, double* out) {
    if (!lp || !v || !out) return fail(UC_ERR_INVALID, "NULL argument");
    int expected = 0;
    if (!lp->busy.compare_exchange_strong(expected, 1)) return fail(UC_ERR_BUSY, "a solve is running on this handle");
    int rc = UC_OK;
    double *din = nullptr, *dperm = nullptr, *dres = nullptr, *dout = nullptr;
    try {
        DeviceGuard guard(lp->device);
        const long long nin = transpose ? lp->m : lp->n, nout = transpose ? lp->n : lp->m;
        const long long* pin = transpose ? lp->perm_r : lp->perm_c;
        const long long* pout = transpose ? lp->perm_c : lp->perm_r;
        const Sell& S = transpose ? lp->KT : lp->K;
        cudaStream_t st = lp->own_stream;
        CK(cudaMalloc((void**)&din, sizeof(double) * (size_t)std::max<long long>(nin, 1)));
        CK(cudaMalloc((void**)&dperm, sizeof(double) * (size_t)std::max<long long>(nin, 1)));
        CK(cudaMalloc((void**)&dres, sizeof(double) * (size_t)std::max<long long>(nout, 1)));
        CK(cudaMalloc((void**)&dout, sizeof(double) * (size_t)std::max<long long>(nout, 1)));
        if (nin) CK(cudaMemcpyAsync(din, v, sizeof(double) * (size_t)nin, cudaMemcpyHostToDevice, st));
        k_gather<<<std::max(1, cdiv(nin, 256)), 256, 0, st>>>(din, pin, nin, dperm);
        k_spmv<<<S.grid, kBlock, 0, st>>>(S, dperm, dres);
        k_scatter<<<std::max(1, cdiv(nout, 256)), 256, 0, st>>>(dres, pout, nout, dout);
        CK(cudaGetLastError());
        if (nout) CK(cudaMemcpyAsync(out, dout, sizeof(double) * (size_t)nout, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
    } catch (const CudaFail& f) {
        rc = fail(UC_ERR_CUDA, std::string(f.what) + ": " + cudaGetErrorString(f.e));
    }
    if (din) cudaFree(din);
    if (dperm) cudaFree(dperm);
    if (dres) cudaFree(dres);
    if (dout) cudaFree(dout);
    lp->busy.store(0);
    return rc;
}

}  // extern "C"

// --------------------------------------------------------------------------------- uc_lp_spmv_static (include/uc_pdhg.h)
// The same three kernels as uc_lp_spmv (k_gather -> k_spmv -> k_scatter), for callers that may not allocate device memory:
// the permuted input and the permuted result, which uc_lp_spmv puts into two cudaMalloc'ed buffers, live in this fixed
// array instead.  It is part of the library image: every device that loads libuc_pdhg.so holds these
// UC_SPMV_STATIC_MAX_DOUBLES * 8 bytes (2 MiB) until the process exits, whether the entry point is ever called or not.
// One array per device, shared by every handle, stream and thread: see the header for what that means for callers.
static __device__ __align__(256) double g_spmv_static_scratch[UC_SPMV_STATIC_MAX_DOUBLES];

namespace {

constexpr int kStaticMaxDevices = 64;
std::mutex g_spmv_static_mu;
double* g_spmv_static_addr[kStaticMaxDevices] = {};   // device address of the array, per device; nullptr = not looked up yet

// In host code `g_spmv_static_scratch` is only the host-side shadow of the symbol: its address means nothing to a kernel.
// The device address is asked for once per device, with that device current (the array exists once per device).
// Returns cudaSuccess and the address, or the error of the lookup (nothing is cached then: the next call tries again).
cudaError_t spmv_static_scratch(int device, double** out) {
    std::lock_guard<std::mutex> g(g_spmv_static_mu);
    if (!g_spmv_static_addr[device]) {
        void* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, g_spmv_static_scratch);
        if (e != cudaSuccess) return e;
        g_spmv_static_addr[device] = (double*)p;
    }
    *out = g_spmv_static_addr[device];
    return cudaSuccess;
}

}  // namespace

extern "C" int uc_lp_spmv_static(uc_lp* lp, int32_t transpose, const double* v_device, double* out_device, void* stream) {
    if (!lp) return fail(UC_ERR_INVALID, "handle is NULL");
    const long long nin = transpose ? lp->m : lp->n, nout = transpose ? lp->n : lp->m;
    if ((nin > 0 && !v_device) || (nout > 0 && !out_device)) return fail(UC_ERR_INVALID, "NULL argument");
    // each of the two scratch vectors starts on a 256-byte boundary of the array
    const long long nin_pad = (nin + 31) / 32 * 32, nout_pad = (nout + 31) / 32 * 32;
    if (nin_pad + nout_pad > (long long)UC_SPMV_STATIC_MAX_DOUBLES)
        return fail(UC_ERR_INVALID, "uc_lp_spmv_static: m + n = " + std::to_string(nin + nout) + " (each rounded up to a multiple of 32) exceeds the "
                    "fixed scratch of UC_SPMV_STATIC_MAX_DOUBLES = " + std::to_string((long long)UC_SPMV_STATIC_MAX_DOUBLES) +
                    " doubles; use uc_lp_spmv, which allocates what it needs");
    if (lp->device < 0 || lp->device >= kStaticMaxDevices) return fail(UC_ERR_INVALID, "uc_lp_spmv_static: device ordinal above 63");
    int expected = 0;
    if (!lp->busy.compare_exchange_strong(expected, 1)) return fail(UC_ERR_BUSY, "a solve is running on this handle");
    int rc = UC_OK;
    {
        DeviceGuard guard(lp->device);
        double* scratch = nullptr;
        cudaError_t e = spmv_static_scratch(lp->device, &scratch);
        if (e != cudaSuccess) rc = fail(UC_ERR_CUDA, std::string("cudaGetSymbolAddress(g_spmv_static_scratch): ") + cudaGetErrorString(e));
        else {
            const long long* pin = transpose ? lp->perm_r : lp->perm_c;
            const long long* pout = transpose ? lp->perm_c : lp->perm_r;
            const Sell& S = transpose ? lp->KT : lp->K;
            cudaStream_t st = stream ? (cudaStream_t)stream : lp->own_stream;
            double* dperm = scratch;               // v in the layout's column order, nin entries
            double* dres = scratch + nin_pad;      // the product in the layout's row order, nout entries
            // Nothing here has to start at zero: k_gather writes all nin entries of dperm before k_spmv reads them, k_spmv
            // writes all nout entries of dres (rows without entries store 0.0) before k_scatter reads them, and neither
            // kernel reads past nin / nout.  What an earlier call left in the array is never looked at.
            k_gather<<<std::max(1, cdiv(nin, 256)), 256, 0, st>>>(v_device, pin, nin, dperm);
            k_spmv<<<S.grid, kBlock, 0, st>>>(S, dperm, dres);
            k_scatter<<<std::max(1, cdiv(nout, 256)), 256, 0, st>>>(dres, pout, nout, out_device);
            e = cudaGetLastError();
            if (e != cudaSuccess) rc = fail(UC_ERR_CUDA, std::string("uc_lp_spmv_static launch: ") + cudaGetErrorString(e));
        }
    }
    lp->busy.store(0);
    return rc;
}
