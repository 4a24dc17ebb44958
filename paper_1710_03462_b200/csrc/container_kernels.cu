// container_kernels.cu -- NEXT-3: container operations on the device.
//   * removal of the particles flagged in a kill mask, applied to EVERY component array:
//       SWAP_LAST  the paper's default "overwrite the removed element with the last one", in place
//                  and unordered, applied to a set in the usual forward loop that re-examines the slot it just filled
//                  (Q20).  In parallel that is: m = n - #killed; the k-th flagged slot below m (ascending)
//                  receives the k-th surviving particle at or above m counted from the END.  Only those rows move.
//       STABLE     order-preserving stream compaction into a second container (dst[rank(i)] = src[i]).
//     Both are deterministic: every destination is a pure function of the mask (prefix sums, no arrival-order
//     atomics).
//   * gather of arbitrary rows into packed AoS records -- the bulk form of getElement(i);
//     push_back of AoS records is soax_aos_to_soa at an offset (api.cu).
// Tiles of 4096 mask bytes; element e of a tile is handled by thread e % 512 in round e / 512, so that every array
// access of a warp is to 32 consecutive elements; in-tile ranks come from warp ballots and a 128-segment scan.
#include "common.cuh"
#include "ops.hpp"
#include "tma.cuh"

namespace soax {

constexpr int kCThreads = 512;
constexpr int kCItems = 8;
constexpr int kCTile = kCThreads * kCItems;  // 4096
constexpr int kCSegs = kCTile / 32;          // 128 warp-sized segments per tile

// ---- pass 1: flagged bytes per tile ---------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) kill_count_kernel(const uint8_t* __restrict__ kill, int64_t n, uint32_t* __restrict__ tile_count) {
    __shared__ uint32_t sm[8];
    const int64_t t0 = (int64_t)blockIdx.x * kCTile;
    uint32_t c = 0;
    if (t0 + kCTile <= n && (reinterpret_cast<uintptr_t>(kill) & 15) == 0) {
        const uint4 v = reinterpret_cast<const uint4*>(kill + t0)[threadIdx.x];  // 16 mask bytes per thread
        const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int b = 0; b < 4; ++b) c += ((w[i] >> (8 * b)) & 0xffu) != 0;
    } else {
        for (int i = threadIdx.x; i < kCTile; i += 256)
            if (t0 + i < n) c += kill[t0 + i] != 0;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) c += __shfl_down_sync(0xffffffffu, c, o);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = c;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t s = 0;
        for (int w = 0; w < 8; ++w) s += sm[w];
        tile_count[blockIdx.x] = s;
    }
}

// ---- pass 2 (one CTA): exclusive scan of the tile counts in place; info[0] = K = #flagged, info[1] = h = #flagged
// below m = n - K (the holes of SWAP_LAST) ------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024) kill_scan_kernel(uint32_t* __restrict__ tile_count, int64_t ntiles, const uint8_t* __restrict__ kill,
                                                         int64_t n, uint64_t* __restrict__ info) {
    __shared__ uint32_t warp_sum[32];
    __shared__ uint32_t carry_sm;
    __shared__ uint32_t cnt_sm;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) { carry_sm = 0; cnt_sm = 0; }
    __syncthreads();
    for (int64_t base = 0; base < ntiles; base += 1024) {
        const int64_t i = base + threadIdx.x;
        const uint32_t x = i < ntiles ? tile_count[i] : 0u;
        uint32_t inc = x;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += y;
        }
        if (lane == 31) warp_sum[warp] = inc;
        __syncthreads();
        if (warp == 0) {
            const uint32_t w = warp_sum[lane];
            uint32_t winc = w;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t y = __shfl_up_sync(0xffffffffu, winc, o);
                if (lane >= o) winc += y;
            }
            warp_sum[lane] = winc - w;
        }
        __syncthreads();
        const uint32_t carry = carry_sm;
        if (i < ntiles) tile_count[i] = carry + warp_sum[warp] + inc - x;
        __syncthreads();
        if (threadIdx.x == 1023) carry_sm = carry + warp_sum[warp] + inc;
        __syncthreads();
    }
    const uint64_t K = carry_sm;
    const int64_t m = n - (int64_t)K;
    // flagged below m: the exclusive prefix of m's tile plus the flagged bytes of that tile before m
    const int64_t tm = m / kCTile;
    uint32_t c = 0;
    for (int64_t e = tm * kCTile + threadIdx.x; e < m; e += 1024) c += kill[e] != 0;
    if (c) atomicAdd(&cnt_sm, c);  // integer: order does not matter
    __syncthreads();
    if (threadIdx.x == 0) {
        info[0] = K;
        info[1] = (tm < ntiles ? tile_count[tm] : (uint32_t)K) + cnt_sm;
    }
}

// ---- in-tile exclusive rank of the flagged elements -------------------------------------------------------------------
// flag[k] belongs to element k*512 + tid of the tile.  Returns in rank[k] the number of flagged elements of the tile
// with a smaller element index.  seg: >= kCSegs + 32 words of shared memory.
__device__ __forceinline__ void tile_rank(const bool (&flag)[kCItems], uint32_t (&rank)[kCItems], uint32_t* seg) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t lt = (1u << lane) - 1u;
    uint32_t bal[kCItems];
#pragma unroll
    for (int k = 0; k < kCItems; ++k) {
        bal[k] = __ballot_sync(0xffffffffu, flag[k]);
        if (lane == 0) seg[k * (kCThreads / 32) + warp] = __popc(bal[k]);  // segment index = element index / 32
    }
    __syncthreads();
    if (threadIdx.x < kCSegs) {  // exclusive scan of the 128 segment counts by the first four warps
        const uint32_t x = seg[threadIdx.x];
        uint32_t inc = x;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += y;
        }
        seg[threadIdx.x] = inc - x;
        if (lane == 31) seg[kCSegs + warp] = inc;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kCItems; ++k) {
        const int s = k * (kCThreads / 32) + warp;
        uint32_t before = seg[s];
        for (int w = 0; w < (s >> 5); ++w) before += seg[kCSegs + w];
        rank[k] = before + __popc(bal[k] & lt);
    }
    __syncthreads();  // seg may be reused by the caller
}

// ---- SWAP_LAST: the slots to fill (flagged, below m) and the rows that fill them (surviving, at or above m) -----------
__global__ void __launch_bounds__(kCThreads) holes_movers_kernel(const uint8_t* __restrict__ kill, int64_t n, const uint64_t* __restrict__ info,
                                                                 const uint32_t* __restrict__ tile_prefix, uint32_t* __restrict__ holes,
                                                                 uint32_t* __restrict__ movers) {
    const int64_t m = n - (int64_t)info[0];  // survivors; read from the device so that the host need not wait for it
    const uint32_t h = (uint32_t)info[1];
    if (h == 0) return;                      // nothing flagged below m: truncation alone removes them
    __shared__ uint32_t seg[kCSegs + 32];
    const int64_t t0 = (int64_t)blockIdx.x * kCTile;
    bool flag[kCItems];
    uint32_t rank[kCItems];
#pragma unroll
    for (int k = 0; k < kCItems; ++k) {
        const int64_t e = t0 + k * kCThreads + threadIdx.x;
        flag[k] = e < n && kill[e] != 0;
    }
    tile_rank(flag, rank, seg);
    const uint32_t before = tile_prefix[blockIdx.x];
#pragma unroll
    for (int k = 0; k < kCItems; ++k) {
        const int64_t e = t0 + k * kCThreads + threadIdx.x;
        if (e >= n) continue;
        const uint32_t ks = before + rank[k];  // flagged elements with a smaller index
        if (flag[k]) {
            if (e < m) holes[ks] = (uint32_t)e;
        } else if (e >= m) {
            movers[h - 1u - ((uint32_t)(e - m) - (ks - h))] = (uint32_t)e;  // survivors in [m, e), counted from the end
        }
    }
}

template <class L>
__global__ void __launch_bounds__(256) move_rows_kernel(Ptrs<L::ncomp> a, const uint32_t* __restrict__ holes, const uint32_t* __restrict__ movers,
                                                        const uint64_t* __restrict__ info) {
    const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= (uint32_t)info[1]) return;  // the grid is sized for the worst case n / 2: surplus CTAs leave at once
    const uint32_t to = holes[k], from = movers[k];
    for_each_comp<L>([&](auto ci) {
        constexpr int C = decltype(ci)::value;
        comp_ptr<L, C>(a)[to] = comp_ptr<L, C>(a)[from];
    });
}

// ---- STABLE: dst[i - #flagged before i] = src[i] for every surviving i, every component array ---------------------------
template <class L>
__global__ void __launch_bounds__(kCThreads) compact_kernel(Ptrs<L::ncomp> src, Ptrs<L::ncomp> dst, const uint8_t* __restrict__ kill, int64_t n,
                                                            const uint32_t* __restrict__ tile_prefix, int64_t dst_capacity) {
    __shared__ uint32_t seg[kCSegs + 32];
    const int64_t t0 = (int64_t)blockIdx.x * kCTile;
    bool flag[kCItems];
    uint32_t rank[kCItems];
#pragma unroll
    for (int k = 0; k < kCItems; ++k) {
        const int64_t e = t0 + k * kCThreads + threadIdx.x;
        flag[k] = e < n && kill[e] != 0;
    }
    tile_rank(flag, rank, seg);
    const int64_t before = tile_prefix[blockIdx.x];
    int64_t dest[kCItems];
#pragma unroll
    for (int k = 0; k < kCItems; ++k) {
        const int64_t e = t0 + k * kCThreads + threadIdx.x;
        dest[k] = (e < n && !flag[k]) ? e - before - rank[k] : -1;
        if (dest[k] >= dst_capacity) dest[k] = -1;  // too small a destination is reported by the host (ALLOC); never write past it
    }
    for_each_comp<L>([&](auto ci) {
        constexpr int C = decltype(ci)::value;
        using T = typename L::template comp_type<C>;
        const T* s = comp_ptr<L, C>(src);
        T* d = comp_ptr<L, C>(dst);
        T v[kCItems];
#pragma unroll
        for (int k = 0; k < kCItems; ++k)
            if (dest[k] >= 0) v[k] = s[t0 + k * kCThreads + threadIdx.x];
#pragma unroll
        for (int k = 0; k < kCItems; ++k)
            if (dest[k] >= 0) d[dest[k]] = v[k];
    });
}

// ---- bulk getElement: rows idx[0..m) as packed AoS records ----------------------------------------------------------------
constexpr int kGTile = 256;
template <class L>
__global__ void __launch_bounds__(kGTile) gather_rows_kernel(Ptrs<L::ncomp> a, const uint32_t* __restrict__ idx, int64_t m, unsigned char* aos) {
    constexpr int S = L::aos_stride;
    extern __shared__ __align__(128) unsigned char sm[];
    const int64_t ntiles = (m + kGTile - 1) / kGTile;
    for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const int64_t t0 = t * kGTile;
        const int cnt = (int)(m - t0 < kGTile ? m - t0 : kGTile);
        if ((int)threadIdx.x < cnt) {
            const uint32_t row = idx[t0 + threadIdx.x];
            unsigned char* rec = sm + threadIdx.x * S;
            for_each_comp<L>([&](auto ci) {  // byte images: the record is packed, fields may be misaligned (Q1)
                constexpr int C = decltype(ci)::value;
                using T = typename L::template comp_type<C>;
                const T v = comp_ptr<L, C>(a)[row];
                memcpy(rec + L::aos_offset(C), &v, sizeof(T));
            });
        }
        __syncthreads();
        if (cnt == kGTile) {  // a full tile leaves as one bulk store
            fence_async_smem();
            __syncthreads();
            if (threadIdx.x == 0) {
                bulk_s2g(aos + t0 * S, sm, kGTile * S);
                bulk_commit();
                bulk_wait_read();
            }
        } else {
            for (int o = threadIdx.x; o < cnt * S; o += kGTile) aos[t0 * S + o] = sm[o];
        }
        __syncthreads();
    }
}

// ---- host side ----------------------------------------------------------------------------------------------------------------
struct RemovePlan {
    int64_t ntiles;
    size_t tile_count, info, holes, movers, total;
    explicit RemovePlan(int64_t n) {
        ntiles = (n + kCTile - 1) / kCTile;
        if (ntiles < 1) ntiles = 1;
        size_t o = 0;
        auto take = [&](size_t bytes) { size_t at = o; o += align_up(bytes ? bytes : 1, kAlign); return at; };
        tile_count = take((size_t)ntiles * 4);
        info = take(2 * sizeof(uint64_t));
        holes = take(((size_t)n / 2 + 1) * 4);  // #holes = #movers <= min(K, n - K) <= n / 2
        movers = take(((size_t)n / 2 + 1) * 4);
        total = o;
    }
};
size_t remove_scratch_bytes(int64_t n) { return RemovePlan(n).total; }

template <class L>
int remove_entry(void* const* src, void* const* dst, const uint8_t* kill, int64_t n, int mode, void* scratch, int64_t* host_new_n,
                 int64_t dst_capacity, cudaStream_t st) {
    if (n == 0) { *host_new_n = 0; return SOAX_OK; }
    const RemovePlan plan(n);
    char* sc = static_cast<char*>(scratch);
    uint32_t* tile_count = reinterpret_cast<uint32_t*>(sc + plan.tile_count);
    uint64_t* info = reinterpret_cast<uint64_t*>(sc + plan.info);
    uint32_t* holes = reinterpret_cast<uint32_t*>(sc + plan.holes);
    uint32_t* movers = reinterpret_cast<uint32_t*>(sc + plan.movers);
    kill_count_kernel<<<(unsigned)plan.ntiles, 256, 0, st>>>(kill, n, tile_count);
    SOAX_TRY(launched());
    kill_scan_kernel<<<1, 1024, 0, st>>>(tile_count, plan.ntiles, kill, n, info);
    SOAX_TRY(launched());
    // Nothing below waits for the count: the kernels read it from `info` on the device, and the one synchronisation
    // of this call (the host needs the new size for the handle) comes after everything has been enqueued.
    uint64_t host_info[2] = {0, 0};
    SOAX_CUDA(cudaMemcpyAsync(host_info, info, sizeof host_info, cudaMemcpyDeviceToHost, st));
    if (mode == SOAX_REMOVE_SWAP_LAST) {
        holes_movers_kernel<<<(unsigned)plan.ntiles, kCThreads, 0, st>>>(kill, n, info, tile_count, holes, movers);
        SOAX_TRY(launched());
        const unsigned blocks = (unsigned)((n / 2 + 255) / 256);  // #holes <= n / 2
        move_rows_kernel<L><<<blocks < 1 ? 1 : blocks, 256, 0, st>>>(make_ptrs<L>(src), holes, movers, info);
        SOAX_TRY(launched());
    } else {
        compact_kernel<L><<<(unsigned)plan.ntiles, kCThreads, 0, st>>>(make_ptrs<L>(src), make_ptrs<L>(dst), kill, n, tile_count, dst_capacity);
        SOAX_TRY(launched());
    }
    SOAX_CUDA(cudaStreamSynchronize(st));
    const int64_t m = n - (int64_t)host_info[0];
    *host_new_n = m;
    if (mode == SOAX_REMOVE_STABLE && m > dst_capacity) return SOAX_ERR_ALLOC;
    return SOAX_OK;
}

template <class L>
int gather_rows_entry(void* const* comps, const uint32_t* idx, int64_t m, void* aos, cudaStream_t st) {
    if (m == 0) return SOAX_OK;
    constexpr int smem = kGTile * L::aos_stride;
    const int64_t ntiles = (m + kGTile - 1) / kGTile;
    const int64_t cap = (int64_t)kSMs * 8;
    gather_rows_kernel<L><<<(unsigned)(ntiles < cap ? ntiles : cap), kGTile, smem, st>>>(make_ptrs<L>(comps), idx, m, static_cast<unsigned char*>(aos));
    return launched();
}

#define X(L)                                                                                                                  \
    template int remove_entry<L>(void* const*, void* const*, const uint8_t*, int64_t, int, void*, int64_t*, int64_t, cudaStream_t); \
    template int gather_rows_entry<L>(void* const*, const uint32_t*, int64_t, void*, cudaStream_t);
SOAX_FOR_EACH_LAYOUT(X)
#undef X

}  // namespace soax
