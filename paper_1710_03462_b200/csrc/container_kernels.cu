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
// Mask bytes are counted per SEGMENT of 256 (one warp's worth: 8 rounds of 32 lanes) and per tile of 16 segments; a
// one-CTA scan turns the tile counts into prefixes.  The stable compaction takes a tile per CTA through a TMA ring and writes
// 16-byte vectors (compact_ring_kernel); the in-place removal ranks holes and movers per warp-owned segment without shared
// memory or CTA barriers and then moves one row per thread.
#include <mutex>

#include "common.cuh"
#include "ops.hpp"
#include "tma.cuh"

namespace soax {

constexpr int kSeg = 256;                    // mask bytes per segment = elements per warp
constexpr int kSegRounds = kSeg / 32;        // 8
constexpr int kCTile = 4096;                 // mask bytes per tile (count kernel CTA)
constexpr int kSegsPerTile = kCTile / kSeg;  // 16

// ---- pass 1: flagged bytes per segment and per tile ----------------------------------------------------------------
// thread t owns mask bytes [16 t, 16 t + 16) of the tile; 16 consecutive threads cover one segment
// `flip` = 1 (SOAX_REMOVE_KEEP_FLAGGED): the mask marks the particles to KEEP; a row is removed iff (byte != 0) != flip.
__global__ void __launch_bounds__(256) kill_count_kernel(const uint8_t* __restrict__ kill, int64_t n, uint32_t flip, uint32_t* __restrict__ tile_count,
                                                         uint32_t* __restrict__ seg_count) {
    __shared__ uint32_t sm[8];
    const int64_t b0 = (int64_t)blockIdx.x * kCTile + 16 * threadIdx.x;
    uint32_t c = 0;
    if (b0 + 16 <= n && (reinterpret_cast<uintptr_t>(kill) & 15) == 0) {
        const uint4 v = *reinterpret_cast<const uint4*>(kill + b0);
        const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int b = 0; b < 4; ++b) c += (uint32_t)(((w[i] >> (8 * b)) & 0xffu) != 0) ^ flip;
    } else {
        for (int i = 0; i < 16; ++i)
            if (b0 + i < n) c += (uint32_t)(kill[b0 + i] != 0) ^ flip;
    }
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);  // sum over the 16 threads of a segment
    if ((threadIdx.x & 15) == 0) seg_count[(int64_t)blockIdx.x * kSegsPerTile + (threadIdx.x >> 4)] = c;
    c += __shfl_xor_sync(0xffffffffu, c, 16);  // both segments of the warp
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = c;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t t = 0;
        for (int w = 0; w < 8; ++w) t += sm[w];
        tile_count[blockIdx.x] = t;
    }
}

// ---- pass 2 (one CTA): exclusive scan of the tile counts in place; info[0] = K = #flagged, info[1] = h = #flagged
// below m = n - K (the holes of SWAP_LAST) ------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024) kill_scan_kernel(uint32_t* __restrict__ tile_count, int64_t ntiles, const uint8_t* __restrict__ kill,
                                                         int64_t n, uint32_t flip, uint64_t* __restrict__ info, int64_t* __restrict__ host_count) {
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
    for (int64_t e = tm * kCTile + threadIdx.x; e < m; e += 1024) c += (uint32_t)(kill[e] != 0) ^ flip;
    if (c) atomicAdd(&cnt_sm, c);  // integer: order does not matter
    __syncthreads();
    if (threadIdx.x == 0) {
        info[0] = K;
        info[1] = (tm < ntiles ? tile_count[tm] : (uint32_t)K) + cnt_sm;
        info[2] = (uint64_t)m;  // the survivor count
        *host_count = m;        // mapped pinned host memory owned by the handle: the host reads it after the count event
        __threadfence_system();
    }
}

// ---- per-warp ranking of one segment ----------------------------------------------------------------------------------
// Element k*32 + lane of segment `seg` (k = 0..7).  Returns the ballots of the flagged elements and `before` = number
// of flagged elements in front of the segment.
struct SegRank {
    uint32_t bal[kSegRounds];
    uint32_t before;
};
__device__ __forceinline__ SegRank seg_rank(const uint8_t* __restrict__ kill, int64_t n, uint32_t flip, int64_t seg,
                                            const uint32_t* __restrict__ tile_prefix, const uint32_t* __restrict__ seg_count) {
    const int lane = threadIdx.x & 31;
    SegRank r;
    const int64_t e0 = seg * kSeg + lane;
    uint8_t f[kSegRounds];
#pragma unroll
    for (int k = 0; k < kSegRounds; ++k) f[k] = e0 + k * 32 < n ? (uint8_t)((uint32_t)(kill[e0 + k * 32] != 0) ^ flip) : (uint8_t)0;
    const int64_t tile = seg / kSegsPerTile;
    const int s_in = (int)(seg % kSegsPerTile);
    uint32_t c = lane < s_in ? seg_count[tile * kSegsPerTile + lane] : 0u;  // counts of the segments before this one
#pragma unroll
    for (int o = 8; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    r.before = tile_prefix[tile] + __shfl_sync(0xffffffffu, c, 0);
#pragma unroll
    for (int k = 0; k < kSegRounds; ++k) r.bal[k] = __ballot_sync(0xffffffffu, f[k] != 0);
    return r;
}

// ---- SWAP_LAST: the slots to fill (flagged, below m) and the rows that fill them (surviving, at or above m) -----------
__global__ void __launch_bounds__(256) holes_movers_kernel(const uint8_t* __restrict__ kill, int64_t n, uint32_t flip, const uint64_t* __restrict__ info,
                                                           const uint32_t* __restrict__ tile_prefix, const uint32_t* __restrict__ seg_count,
                                                           uint32_t* __restrict__ holes, uint32_t* __restrict__ movers) {
    const int64_t m = n - (int64_t)info[0];  // survivors; read from the device so that the host need not wait for it
    const uint32_t h = (uint32_t)info[1];
    if (h == 0) return;                      // nothing flagged below m: truncation alone removes them
    const int64_t seg = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (seg * kSeg >= n) return;
    const int lane = threadIdx.x & 31;
    const uint32_t lt = (1u << lane) - 1u;
    const SegRank r = seg_rank(kill, n, flip, seg, tile_prefix, seg_count);
    uint32_t run = r.before;
#pragma unroll
    for (int k = 0; k < kSegRounds; ++k) {
        const int64_t e = seg * kSeg + k * 32 + lane;
        const uint32_t ks = run + __popc(r.bal[k] & lt);  // flagged elements with a smaller index
        run += __popc(r.bal[k]);
        if (e >= n) continue;
        if (r.bal[k] >> lane & 1u) {
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
    // all loads, then all stores: interleaved, every load would have to wait for the store before it (same arrays)
    constexpr int kGroup = 16;
    constexpr int kGroups = (L::ncomp + kGroup - 1) / kGroup;
    for_each_int<kGroups>([&](auto gi) {
        constexpr int G0 = decltype(gi)::value * kGroup;
        constexpr int GN = L::ncomp - G0 < kGroup ? L::ncomp - G0 : kGroup;
        CompRegs<L, G0, 1, std::make_integer_sequence<int, GN>> v;
        for_each_int<GN>([&](auto ci) {
            constexpr int C = G0 + decltype(ci)::value;
            v.template get<C>()[0] = comp_ptr<L, C>(a)[from];
        });
        for_each_int<GN>([&](auto ci) {
            constexpr int C = G0 + decltype(ci)::value;
            comp_ptr<L, C>(a)[to] = v.template get<C>()[0];
        });
    });
}

// ---- STABLE: dst[i - #flagged before i] = src[i] for every surviving i, every component array ---------------------------
// One CTA per tile of 4096 source rows (the tile of the count pass, so tile_prefix[tile] = flagged rows before it).  Thread t
// owns rows [8 t, 8 t + 8): a block scan of the survivor counts gives every survivor its slot in the tile's compacted run, and
// `inv` (slot -> source row) is built once.  Then every component array of the tile arrives by ONE bulk asynchronous copy (TMA)
// into a 3-stage ring, and the compacted run leaves as 16-BYTE VECTOR STORES: the run is contiguous in dst, so after at most 3
// (4-byte types) head elements every thread writes 4 consecutive elements (2 of 8 bytes, 16 of 1 byte) at a 16-byte aligned
// address -- 16 sectors per store request instead of the ~5 of a warp that writes 29 survivors one element per lane.
constexpr int kCompThreads = 512;
constexpr int kCompItems = kCTile / kCompThreads;  // 8 rows per thread
constexpr int kCompStages = 3;
constexpr int kCompStageBytes = kCTile * 8;
constexpr int kCompSmem = kCompStages * kCompStageBytes + kCTile * 2 /*inv*/ + 32 * 4 /*scan*/ + 64 /*mbarriers*/;

template <class L>
__global__ void __launch_bounds__(kCompThreads, 2) compact_ring_kernel(Ptrs<L::ncomp> src, Ptrs<L::ncomp> dst, const uint8_t* __restrict__ kill, int64_t n,
                                                                      uint32_t flip, const uint32_t* __restrict__ tile_prefix, int64_t dst_capacity) {
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char* ring = smem;
    uint16_t* inv = reinterpret_cast<uint16_t*>(smem + kCompStages * kCompStageBytes);
    uint32_t* scan_sm = reinterpret_cast<uint32_t*>(smem + kCompStages * kCompStageBytes + kCTile * 2);
    uint64_t* full = reinterpret_cast<uint64_t*>(scan_sm + 32);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t tile0 = (int64_t)blockIdx.x * kCTile;
    const int cnt = (int)(n - tile0 < kCTile ? n - tile0 : kCTile);
    const bool bulk = cnt == kCTile;
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kCompStages; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    auto fill = [&](auto ci) {  // start bringing component C of the tile into stage C % 3 (nothing past the last component)
        constexpr int C = decltype(ci)::value;
        if constexpr (C < L::ncomp) {
            using T = typename L::template comp_type<C>;
            unsigned char* sb = ring + (C % kCompStages) * kCompStageBytes;
            const T* g = comp_ptr<L, C>(src) + tile0;
            if (bulk) {
                if (tid == 0) {
                    mbar_expect_tx(&full[C % kCompStages], kCTile * (uint32_t)sizeof(T));
                    bulk_g2s(sb, g, kCTile * (uint32_t)sizeof(T), &full[C % kCompStages]);
                }
            } else {
                for (int i = tid; i < cnt; i += kCompThreads) reinterpret_cast<T*>(sb)[i] = g[i];
            }
        }
    };
    fill(std::integral_constant<int, 0>{});
    fill(std::integral_constant<int, 1>{});
    fill(std::integral_constant<int, 2>{});

    // ---- survivors of this thread's 8 rows, block scan, inv ------------------------------------------------------------------
    uint32_t alive = 0;  // bit i: row 8 t + i survives
    {
        const int64_t r0 = tile0 + (int64_t)tid * kCompItems;
        if (r0 + kCompItems <= n && (reinterpret_cast<uintptr_t>(kill + r0) & 7) == 0) {
            const uint2 m = *reinterpret_cast<const uint2*>(kill + r0);
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                alive |= ((uint32_t)(((m.x >> (8 * i)) & 0xffu) == 0) ^ flip) << i;
                alive |= ((uint32_t)(((m.y >> (8 * i)) & 0xffu) == 0) ^ flip) << (4 + i);
            }
        } else {
#pragma unroll
            for (int i = 0; i < kCompItems; ++i)
                if (r0 + i < n) alive |= ((uint32_t)(kill[r0 + i] == 0) ^ flip) << i;
        }
    }
    const uint32_t mine = __popc(alive);
    uint32_t inc = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += y;
    }
    if (lane == 31) scan_sm[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        const uint32_t w = lane < kCompThreads / 32 ? scan_sm[lane] : 0u;
        uint32_t winc = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += y;
        }
        scan_sm[lane] = winc - w;
        if (lane == 31) scan_sm[31] = winc;  // (lanes >= 16 hold the total as well: kCompThreads / 32 = 16 warps)
    }
    __syncthreads();
    uint32_t slot = scan_sm[warp] + inc - mine;
    const uint32_t total = scan_sm[31];
#pragma unroll
    for (int i = 0; i < kCompItems; ++i)
        if (alive >> i & 1u) inv[slot++] = (uint16_t)(tid * kCompItems + i);
    __syncthreads();

    // ---- the compacted run of the tile: dst slots [d0, d0 + S) -----------------------------------------------------------------
    const int64_t d0 = tile0 - (int64_t)tile_prefix[blockIdx.x];
    // too small a destination is reported through the count (Q25); never write past it
    const int S = (int)(dst_capacity > d0 ? (dst_capacity - d0 < (int64_t)total ? dst_capacity - d0 : (int64_t)total) : 0);
    for_each_comp<L>([&](auto ci) {
        constexpr int C = decltype(ci)::value;
        using T = typename L::template comp_type<C>;
        constexpr int V = 16 / (int)sizeof(T);  // elements per 16-byte store
        if (bulk) mbar_wait(&full[C % kCompStages], (C / kCompStages) & 1);
        else __syncthreads();
        const T* sb = reinterpret_cast<const T*>(ring + (C % kCompStages) * kCompStageBytes);
        T* out = comp_ptr<L, C>(dst) + d0;
        const int head = (int)((V - (d0 & (V - 1))) & (V - 1)) < S ? (int)((V - (d0 & (V - 1))) & (V - 1)) : S;
        const int ngroups = (S - head) / V;
        for (int g = tid; g < ngroups; g += kCompThreads) {
            const int j0 = head + g * V;
            struct alignas(16) Pack { T v[V]; } p;
#pragma unroll
            for (int i = 0; i < V; ++i) p.v[i] = sb[inv[j0 + i]];
            *reinterpret_cast<Pack*>(out + j0) = p;  // 16-byte aligned: (d0 + head) is a multiple of V and the array base of 256
        }
        const int tail0 = head + ngroups * V;
        if (tid < head) out[tid] = sb[inv[tid]];
        if (tid < S - tail0) out[tail0 + tid] = sb[inv[tail0 + tid]];
        // The stores come BEFORE the barrier: they consume the loaded values, so every read of the stage has completed when
        // its thread arrives and the bulk copy that refills the stage cannot overtake them (see bin_kernels.cu).
        __syncthreads();
        fill(std::integral_constant<int, C + kCompStages>{});
    });
}

// ---- bulk getElement: rows idx[0..m) as packed AoS records ----------------------------------------------------------------
constexpr int kGTile = 256;
template <class L>
__global__ void __launch_bounds__(kGTile) gather_rows_kernel(Ptrs<L::ncomp> a, int64_t n, const uint32_t* __restrict__ idx, int64_t m, unsigned char* aos) {
    constexpr int S = L::aos_stride;
    extern __shared__ __align__(128) unsigned char sm[];
    const int64_t ntiles = (m + kGTile - 1) / kGTile;
    for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const int64_t t0 = t * kGTile;
        const int cnt = (int)(m - t0 < kGTile ? m - t0 : kGTile);
        if ((int)threadIdx.x < cnt) {
            const uint32_t row = idx[t0 + threadIdx.x];
            unsigned char* rec = sm + threadIdx.x * S;
            if ((int64_t)row >= n) {  // out of range: never dereferenced, the record is zero bytes
                for (int b = 0; b < S; ++b) rec[b] = 0;
            } else {
            // all the (random) loads of a group of components first, then the stores into the packed record, whose
            // fields may be misaligned (Q1): byte images
            constexpr int kGroup = 16;
            constexpr int kGroups = (L::ncomp + kGroup - 1) / kGroup;
            for_each_int<kGroups>([&](auto gi) {
                constexpr int G0 = decltype(gi)::value * kGroup;
                constexpr int GN = L::ncomp - G0 < kGroup ? L::ncomp - G0 : kGroup;
                CompRegs<L, G0, 1, std::make_integer_sequence<int, GN>> v;
                for_each_int<GN>([&](auto ci) {
                    constexpr int C = G0 + decltype(ci)::value;
                    v.template get<C>()[0] = comp_ptr<L, C>(a)[row];
                });
                for_each_int<GN>([&](auto ci) {
                    constexpr int C = G0 + decltype(ci)::value;
                    using T = typename L::template comp_type<C>;
                    memcpy(rec + L::aos_offset(C), v.template get<C>(), sizeof(T));
                });
            });
            }
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
    size_t tile_count, seg_count, info, holes, movers, total;
    explicit RemovePlan(int64_t n) {
        ntiles = (n + kCTile - 1) / kCTile;
        if (ntiles < 1) ntiles = 1;
        size_t o = 0;
        auto take = [&](size_t bytes) { size_t at = o; o += align_up(bytes ? bytes : 1, kAlign); return at; };
        tile_count = take((size_t)ntiles * 4);
        seg_count = take((size_t)ntiles * kSegsPerTile * 4);
        info = take(3 * sizeof(uint64_t));
        holes = take(((size_t)n / 2 + 1) * 4);  // #holes = #movers <= min(K, n - K) <= n / 2
        movers = take(((size_t)n / 2 + 1) * 4);
        total = o;
    }
};
size_t remove_scratch_bytes(int64_t n) { return RemovePlan(n).total; }

template <class L>
int remove_entry(void* const* src, void* const* dst, const uint8_t* kill, int64_t n, int mode, void* scratch,
                 int64_t dst_capacity, int64_t* pin_n, int64_t* host_new_n, cudaEvent_t count_ready, cudaStream_t st) {
    const RemovePlan plan(n);
    char* sc = static_cast<char*>(scratch);
    uint32_t* tile_count = reinterpret_cast<uint32_t*>(sc + plan.tile_count);
    uint32_t* seg_count = reinterpret_cast<uint32_t*>(sc + plan.seg_count);
    uint64_t* info = reinterpret_cast<uint64_t*>(sc + plan.info);
    uint32_t* holes = reinterpret_cast<uint32_t*>(sc + plan.holes);
    uint32_t* movers = reinterpret_cast<uint32_t*>(sc + plan.movers);
    const uint32_t flip = (mode & SOAX_REMOVE_KEEP_FLAGGED) ? 1u : 0u;
    mode &= ~SOAX_REMOVE_KEEP_FLAGGED;
    kill_count_kernel<<<(unsigned)plan.ntiles, 256, 0, st>>>(kill, n, flip, tile_count, seg_count);
    const unsigned seg_blocks = (unsigned)(((n + kSeg - 1) / kSeg + 7) / 8);  // 8 warps = 8 segments per CTA
    SOAX_TRY(launched());
    kill_scan_kernel<<<1, 1024, 0, st>>>(tile_count, plan.ntiles, kill, n, flip, info, pin_n);
    SOAX_TRY(launched());
    // Nothing waits for the count, neither here nor on the device: the data kernels read it from `info`, and the scan
    // kernel itself stores it into the handle's mapped pinned word (no copy node in the stream); `count_ready` lets the
    // handle pick it up later.
    // The caller's own word is the one thing that goes through a copy node; from pageable memory that copy blocks the host
    // until both count kernels have run (soax.h says so).
    if (host_new_n) SOAX_CUDA(cudaMemcpyAsync(host_new_n, info + 2, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    SOAX_CUDA(cudaEventRecord(count_ready, st));
    if (mode == SOAX_REMOVE_SWAP_LAST) {
        holes_movers_kernel<<<seg_blocks, 256, 0, st>>>(kill, n, flip, info, tile_count, seg_count, holes, movers);
        SOAX_TRY(launched());
        const unsigned blocks = (unsigned)((n / 2 + 255) / 256);  // #holes <= n / 2
        move_rows_kernel<L><<<blocks < 1 ? 1 : blocks, 256, 0, st>>>(make_ptrs<L>(src), holes, movers, info);
        SOAX_TRY(launched());
    } else {
        SOAX_CUDA(cudaFuncSetAttribute(compact_ring_kernel<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, kCompSmem));
        compact_ring_kernel<L><<<(unsigned)plan.ntiles, kCompThreads, kCompSmem, st>>>(make_ptrs<L>(src), make_ptrs<L>(dst), kill, n, flip, tile_count, dst_capacity);
        SOAX_TRY(launched());
    }
    return SOAX_OK;
}

template <class L>
int gather_rows_entry(void* const* comps, int64_t n, const uint32_t* idx, int64_t m, void* aos, cudaStream_t st) {
    if (m == 0) return SOAX_OK;
    constexpr int smem = kGTile * L::aos_stride;
    const int64_t ntiles = (m + kGTile - 1) / kGTile;
    const int64_t cap = (int64_t)kSMs * 8;
    gather_rows_kernel<L><<<(unsigned)(ntiles < cap ? ntiles : cap), kGTile, smem, st>>>(make_ptrs<L>(comps), n, idx, m, static_cast<unsigned char*>(aos));
    return launched();
}

// ---- stable removal without a scratch buffer from the caller (soax_remove_stable_noalloc) -------------------------------------
// The per-tile and per-segment counts of the mask and the three result words of the scan are the only scratch the stable
// compaction needs (68 bytes per tile of 4096 rows; holes and movers belong to SWAP_LAST only).  For callers that have no
// way of providing device memory for them, that scratch lives HERE, in an array that is part of the library image: every
// GPU that loads libsoax.so holds these kStaticScratchBytes (about 0.27 MB) until the process exits.  Layout of the array
// (every piece 256-byte aligned): tile counts for kNoAllocMaxN rows | segment counts | info[3].
constexpr int64_t kNoAllocMaxN = (int64_t)1 << 24;                    // SOAX_NOALLOC_MAX_N of soax.h
constexpr size_t kStaticTiles = (size_t)(kNoAllocMaxN / kCTile);      // 4096
constexpr size_t kStaticTileOff = 0;
constexpr size_t kStaticSegOff = kStaticTileOff + kStaticTiles * 4;                  // 16 KB of tile counts before it
constexpr size_t kStaticInfoOff = kStaticSegOff + kStaticTiles * kSegsPerTile * 4;   // 256 KB of segment counts before it
constexpr size_t kStaticScratchBytes = kStaticInfoOff + kAlign;
static_assert(kStaticSegOff % kAlign == 0 && kStaticInfoOff % kAlign == 0, "pieces of the static scratch start on 256-byte boundaries");
static_assert(SOAX_NOALLOC_MAX_N == kNoAllocMaxN, "soax.h states the limit this array was sized for");
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

// In HOST code the name g_static_scratch is only a handle for the runtime, not an address a kernel could use: the device
// address has to be asked for, per device, with that device current.  Done once per device, at the first call there.
constexpr int kMaxDevices = 64;
static std::mutex g_static_mu;
static unsigned char* g_static_ptr[kMaxDevices] = {};

static int static_scratch(unsigned char** out) {
    int dev = -1;
    SOAX_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return SOAX_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[dev]) {
        void* p = nullptr;
        SOAX_CUDA(cudaGetSymbolAddress(&p, g_static_scratch));  // the copy of the array that lives on the current device
        if (!p) return SOAX_ERR_CUDA;
        g_static_ptr[dev] = static_cast<unsigned char*>(p);
    }
    *out = g_static_ptr[dev];
    return SOAX_OK;
}

// The same three kernels, in the same order and launch shapes, as the STABLE branch of remove_entry; only where the counts
// live differs, and the survivor count goes to the caller's device word instead of a pinned word of the handle (creating
// that word and its event would allocate).  Nothing in the array has to start at zero: kill_count_kernel writes the count
// of every tile and of every segment of [0, n) before anything reads them, the scan writes info, and entries past this
// call's tiles -- left over from an earlier, larger call -- are never read.
template <class L>
int remove_stable_noalloc_entry(void* const* src, void* const* dst, const uint8_t* kill, int64_t n, uint32_t flip, int64_t dst_capacity,
                                int64_t* dev_new_n, cudaStream_t st) {
    if (n > kNoAllocMaxN) return SOAX_ERR_TOO_LARGE;
    unsigned char* sc = nullptr;
    SOAX_TRY(static_scratch(&sc));
    uint32_t* tile_count = reinterpret_cast<uint32_t*>(sc + kStaticTileOff);
    uint32_t* seg_count = reinterpret_cast<uint32_t*>(sc + kStaticSegOff);
    uint64_t* info = reinterpret_cast<uint64_t*>(sc + kStaticInfoOff);
    const int64_t ntiles = (n + kCTile - 1) / kCTile;
    kill_count_kernel<<<(unsigned)ntiles, 256, 0, st>>>(kill, n, flip, tile_count, seg_count);
    SOAX_TRY(launched());
    kill_scan_kernel<<<1, 1024, 0, st>>>(tile_count, ntiles, kill, n, flip, info, dev_new_n);
    SOAX_TRY(launched());
    SOAX_CUDA(cudaFuncSetAttribute(compact_ring_kernel<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, kCompSmem));
    compact_ring_kernel<L><<<(unsigned)ntiles, kCompThreads, kCompSmem, st>>>(make_ptrs<L>(src), make_ptrs<L>(dst), kill, n, flip, tile_count, dst_capacity);
    return launched();
}

#define X(L)                                                                                                                  \
    template int remove_stable_noalloc_entry<L>(void* const*, void* const*, const uint8_t*, int64_t, uint32_t, int64_t, int64_t*, cudaStream_t); \
    template int remove_entry<L>(void* const*, void* const*, const uint8_t*, int64_t, int, void*, int64_t, int64_t*, int64_t*, cudaEvent_t, cudaStream_t); \
    template int gather_rows_entry<L>(void* const*, int64_t, const uint32_t*, int64_t, void*, cudaStream_t);
SOAX_FOR_EACH_LAYOUT(X)
#undef X

}  // namespace soax
