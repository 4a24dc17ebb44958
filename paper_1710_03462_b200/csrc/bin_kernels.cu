// bin_kernels.cu -- a10..a14: PIC-style cell binning with a STABLE counting-sort permutation of every field
// array (BASELINE.json config 5).
//
// Design.  The 3*log2(G)-bit cell key is sorted by a least-significant-digit counting sort whose
// digits are as wide as 9 bits (G = 64: 18 bits = TWO passes of 512 bins), and the WHOLE RECORD travels with its key
// through the passes together with its source index, so `perm` falls out as the carried index and no random gather
// of the field arrays is ever made (a per-array gather would read one 32-byte sector per 4- or 8-byte item).
//   cell_hist   [drift +] cell index [+ kinetic energy] and the first digit's per-tile histogram     36 B read, 4 B written
//   colscan_*   exclusive scan of the [tile][digit] table in digit-major order                      (small)
//   scatter     every array of the tile (keys, carried indices, each component array) arrives in shared memory as ONE
//               bulk asynchronous copy (TMA) into a 3-stage ring; stable in-tile ranks come from warp ballots and
//               per-warp running counters; output slot j reads ring[inv[j]] and writes its global slot, consecutive
//               threads writing consecutive slots of a bin's run.  The first pass applies the requested DRIFT to the
//               positions on their way through the ring (src is never written).
//   tile_hist   per-tile histogram of the next digit (later passes)                                  4 B read
//   cell_bounds counts / offsets from the sorted keys by binary search per cell                      (small)
// A 512-bin pass leaves runs of only ~8 elements per tile and bin, whose ragged ends are partial 32-byte sectors; the
// L2 turns a partial-sector write into a DRAM read-modify-write unless the rest of the sector arrives within about a
// microsecond (measured, profiles/r2_bin_study.md).  Wide-digit passes are therefore launched in THREAD-BLOCK CLUSTERS
// of 4 CTAs that own neighbouring tiles and meet at a cluster barrier before every array's stores: the four pieces of
// a bin's run reach the L2 together and merge into full sectors.
// Every step is a pure function of the data (no arrival-order atomics decide a position), so the result is the
// unique stable permutation for ANY particle distribution, and bit-identical from run to run.
#include <type_traits>

#include "common.cuh"
#include "ops.hpp"
#include "tma.cuh"

namespace soax {

int sum_partials(const double* partial, int m, double* out, cudaStream_t st);  // reduce_kernels.cu

constexpr int kRadixBits = 9;
constexpr int kRadix = 1 << kRadixBits;        // at most 512 bins per pass
#ifndef SOAX_SORT_THREADS
#define SOAX_SORT_THREADS 512
#endif
constexpr int kSortThreads = SOAX_SORT_THREADS;  // 16 warps
constexpr int kItems = 8;                      // keys per thread
constexpr int kTileN = kSortThreads * kItems;  // 4096 particles per tile
constexpr int kWarps = kSortThreads / 32;
constexpr int kScanRows = 64;                  // tiles per column-scan chunk
constexpr int kCellThreads = 256;

// ---- pass 0: [drift +] cell index [+ kinetic energy] + first-digit histogram, one CTA per tile --------------------
// src is read only: with DRIFT the key is the cell of the DRIFTED position, which the first scatter pass recomputes
// with the same fma while it moves the position arrays (same operands, same operation: same bits).
template <class L, bool DRIFT, bool KE, int P>
__device__ __forceinline__ double cell_group(const Ptrs<L::ncomp>& a, int64_t i0, uint32_t* cell, double dt, double G,
                                             int gmax, int log2g, uint32_t mask, uint32_t* h) {
    using V = typename L::template type_of<vel_tag>;
    Vec<double, P> x[3];
    Vec<V, P> v[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) x[d] = ld_vec<double, P>(field_ptr<L, pos_tag>(a, d) + i0);
    if constexpr (DRIFT || KE) {
#pragma unroll
        for (int d = 0; d < 3; ++d) v[d] = ld_vec<V, P>(field_ptr<L, vel_tag>(a, d) + i0);
    }
    if constexpr (DRIFT) {
#pragma unroll
        for (int d = 0; d < 3; ++d)
#pragma unroll
            for (int j = 0; j < P; ++j) x[d].v[j] = drift1<V>(dt, v[d].v[j], x[d].v[j]);
    }
    Vec<uint32_t, P> c;
    double e = 0.0;
#pragma unroll
    for (int j = 0; j < P; ++j) {
        c.v[j] = cell_of(x[0].v[j], x[1].v[j], x[2].v[j], G, gmax, log2g);
        atomicAdd(&h[c.v[j] & mask], 1u);
        if constexpr (KE)
            e += energy1<false>((double)v[0].v[j], (double)v[1].v[j], (double)v[2].v[j], 0.0, 0.0, 0.0, 0.0, 0.0);
    }
    st_vec<uint32_t, P>(cell + i0, c);
    return e;
}

template <class L, bool DRIFT, bool KE>
__global__ void __launch_bounds__(kCellThreads) cell_hist_kernel(Ptrs<L::ncomp> a, int64_t n, uint32_t* cell, double dt, int log2g,
                                                                 uint32_t mask, uint32_t* __restrict__ hist, double* ke_partial) {
    constexpr int P = 4;
    __shared__ double sm[32];
    __shared__ uint32_t h[kRadix];
    for (int i = threadIdx.x; i < kRadix; i += kCellThreads) h[i] = 0;
    __syncthreads();
    const double G = (double)(1 << log2g);
    const int gmax = (1 << log2g) - 1;
    const int64_t tile0 = (int64_t)blockIdx.x * kTileN;
    double e = 0.0;
    if (tile0 + kTileN <= n) {
#pragma unroll
        for (int it = 0; it < kTileN / (kCellThreads * P); ++it)
            e += cell_group<L, DRIFT, KE, P>(a, tile0 + (int64_t)(it * kCellThreads + threadIdx.x) * P, cell, dt, G, gmax, log2g, mask, h);
    } else {
        for (int64_t i = tile0 + threadIdx.x; i < n; i += kCellThreads)
            e += cell_group<L, DRIFT, KE, 1>(a, i, cell, dt, G, gmax, log2g, mask, h);
    }
    __syncthreads();
    for (int i = threadIdx.x; i <= (int)mask; i += kCellThreads) hist[(int64_t)blockIdx.x * (mask + 1) + i] = h[i];
    if constexpr (KE) {
        e = block_sum(e, sm);
        if (threadIdx.x == 0) ke_partial[blockIdx.x] = e;
    }
}

// ---- per-tile digit histogram (passes after the first) -----------------------------------------------------------
__global__ void __launch_bounds__(kSortThreads) tile_hist_kernel(const uint32_t* __restrict__ keys, int64_t n, int shift, uint32_t mask,
                                                                 uint32_t* __restrict__ hist) {
    __shared__ uint32_t h[kRadix];
    if (threadIdx.x < kRadix) h[threadIdx.x] = 0;
    __syncthreads();
    const int64_t tile0 = (int64_t)blockIdx.x * kTileN;
    if (tile0 + kTileN <= n) {  // full tile: two 128-bit loads per thread (the histogram does not care about order)
        const uint4* k4 = reinterpret_cast<const uint4*>(keys + tile0);
        const uint4 a = k4[threadIdx.x], b = k4[threadIdx.x + kSortThreads];
        const uint32_t w[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
#pragma unroll
        for (int k = 0; k < 8; ++k) atomicAdd(&h[(w[k] >> shift) & mask], 1u);
    } else {
#pragma unroll
        for (int k = 0; k < kItems; ++k) {
            const int64_t e = tile0 + k * kSortThreads + threadIdx.x;
            if (e < n) atomicAdd(&h[(keys[e] >> shift) & mask], 1u);
        }
    }
    __syncthreads();
    if (threadIdx.x <= mask) hist[(int64_t)blockIdx.x * (mask + 1) + threadIdx.x] = h[threadIdx.x];  // row of mask+1 bins
}

// ---- exclusive scan of hist[tile][digit] in (digit-major, tile-minor) order ----------------------------------------
// phase 1: column sums of each chunk of kScanRows tiles.  Loads are issued in batches of 16 independent rows so
// that the table streams at memory speed instead of one dependent round trip per row.
constexpr int kScanBatch = 16;
__global__ void __launch_bounds__(kRadix) colscan_reduce_kernel(const uint32_t* __restrict__ hist, int ntiles, int nb,
                                                                uint32_t* __restrict__ partial) {
    const int r0 = blockIdx.x * kScanRows, r1 = min(r0 + kScanRows, ntiles);
    if ((int)threadIdx.x >= nb) return;
    uint32_t s = 0;
    for (int r = r0; r < r1; r += kScanBatch) {
        uint32_t v[kScanBatch];
#pragma unroll
        for (int u = 0; u < kScanBatch; ++u) v[u] = r + u < r1 ? hist[(int64_t)(r + u) * nb + threadIdx.x] : 0u;
#pragma unroll
        for (int u = 0; u < kScanBatch; ++u) s += v[u];
    }
    partial[(int64_t)blockIdx.x * nb + threadIdx.x] = s;
}
// exclusive scan of one value per thread over a CTA of kRadix threads
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t x, uint32_t* sm /* >= 32 */) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t inc = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += y;
    }
    if (lane == 31) sm[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        uint32_t w = lane < (int)(blockDim.x >> 5) ? sm[lane] : 0, winc = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += y;
        }
        sm[lane] = winc - w;
    }
    __syncthreads();
    return inc - x + sm[warp];
}
// phase 2 (one CTA): per digit, exclusive scan of the chunk sums over chunks; then exclusive scan of the digit
// totals over digits -> dbase[digit]
__global__ void __launch_bounds__(kRadix) colscan_top_kernel(uint32_t* __restrict__ partial, int nchunks, int nb,
                                                             uint32_t* __restrict__ dbase) {
    __shared__ uint32_t sm[32];
    const bool on = (int)threadIdx.x < nb;  // blockDim = max(32, nb): idle lanes still take part in the scan
    uint32_t run = 0;
    for (int c = 0; on && c < nchunks; c += kScanBatch) {
        uint32_t v[kScanBatch];
#pragma unroll
        for (int u = 0; u < kScanBatch; ++u) v[u] = c + u < nchunks ? partial[(int64_t)(c + u) * nb + threadIdx.x] : 0u;
#pragma unroll
        for (int u = 0; u < kScanBatch; ++u) {
            if (c + u < nchunks) partial[(int64_t)(c + u) * nb + threadIdx.x] = run;
            run += v[u];
        }
    }
    const uint32_t ex = block_excl_scan(run, sm);
    if (on) dbase[threadIdx.x] = ex;
}
// phase 3: hist[tile][digit] <- global offset of the first item of (digit, tile)
__global__ void __launch_bounds__(kRadix) colscan_apply_kernel(uint32_t* __restrict__ hist, int ntiles, int nb,
                                                               const uint32_t* __restrict__ partial,
                                                               const uint32_t* __restrict__ dbase) {
    const int r0 = blockIdx.x * kScanRows, r1 = min(r0 + kScanRows, ntiles);
    if ((int)threadIdx.x >= nb) return;
    uint32_t run = dbase[threadIdx.x] + partial[(int64_t)blockIdx.x * nb + threadIdx.x];
    for (int r = r0; r < r1; r += kScanBatch) {
        uint32_t v[kScanBatch];
#pragma unroll
        for (int u = 0; u < kScanBatch; ++u) v[u] = r + u < r1 ? hist[(int64_t)(r + u) * nb + threadIdx.x] : 0u;
#pragma unroll
        for (int u = 0; u < kScanBatch; ++u) {
            if (r + u < r1) hist[(int64_t)(r + u) * nb + threadIdx.x] = run;
            run += v[u];
        }
    }
}

// ---- the order in which the arrays of a tile pass through the 3-stage ring, fixed at compile time -------------------
// Array ids: 0 = keys, 1 = carried source indices (HAS_IDX), then the component arrays.  Arrays are LOADED in `load`
// order and MOVED (written to their destination) in `move` order; the two differ only under DRIFT, where the position
// component c needs the velocity component c in shared memory at the same time: vel_c is loaded just before pos_c and
// moved just after it.  Load k >= 3 goes into the stage freed by move k - 3.
constexpr int kRingStages = 3;
template <class L, bool HAS_IDX, bool DRIFT>
struct RingPlan {
    static constexpr int kFirstComp = HAS_IDX ? 2 : 1;
    static constexpr int kArrays = kFirstComp + L::ncomp;
    int load[kArrays] = {}, move[kArrays] = {}, stage[kArrays] = {}, parity[kArrays] = {}, partner[kArrays] = {};
    constexpr RingPlan() {
        int nl = 0, nm = 0;
        for (int a = 0; a < kFirstComp; ++a) { load[nl++] = a; move[nm++] = a; }
        bool used[L::ncomp > 0 ? L::ncomp : 1] = {};
        for (int a = 0; a < kArrays; ++a) partner[a] = -1;
        if constexpr (DRIFT) {
            constexpr int P0 = L::template begin_of<pos_tag>, V0 = L::template begin_of<vel_tag>;
            for (int c = 0; c < 3; ++c) {
                load[nl++] = kFirstComp + V0 + c; load[nl++] = kFirstComp + P0 + c;
                move[nm++] = kFirstComp + P0 + c; move[nm++] = kFirstComp + V0 + c;
                partner[kFirstComp + P0 + c] = kFirstComp + V0 + c;
                used[P0 + c] = used[V0 + c] = true;
            }
        }
        for (int c = 0; c < L::ncomp; ++c)
            if (!used[c]) { load[nl++] = kFirstComp + c; move[nm++] = kFirstComp + c; }
        int uses[kRingStages] = {};
        for (int k = 0; k < kArrays; ++k) {
            const int s = k < kRingStages ? k : stage[move[k - kRingStages]];
            stage[load[k]] = s;
            parity[load[k]] = uses[s] & 1;
            ++uses[s];
        }
    }
};

// Time-synchronisation of the CTAs of a thread-block cluster (no memory ordering needed: it only makes the CTAs that
// own neighbouring tiles write the pieces of a bin's run at the same moment, so that the L2 merges them into full sectors).
__device__ __forceinline__ void cluster_sync_relaxed() {
    asm volatile("barrier.cluster.arrive.relaxed.aligned;\n\tbarrier.cluster.wait.aligned;" ::: "memory");
}

// Pacing of the scatter stores (measured, profiles/r2_bin_study.md): a thread has kItems stores per array; issued back to
// back they reach the L2 out of step with the stores of the neighbouring CTAs that complete the same sectors.  Between
// two stores of a thread the CTA (pace_sync 1) or the whole cluster (2, the default with clusters) therefore meets at a
// barrier, so that at any moment the cluster writes ONE window of ~64 neighbouring bins; a sleep of a few tens of
// nanoseconds can be added for studies.
__device__ __forceinline__ void pace(int k, int pace_sync, int pace_ns) {
    if (k == 0) return;
    if (pace_sync == 1) __syncthreads();
    if (pace_sync == 2) cluster_sync_relaxed();
    if (pace_ns) __nanosleep(pace_ns);
}

// ---- stable scatter of one tile through the TMA ring ----------------------------------------------------------------
// 64 registers/thread and ~106 KB of shared memory let two CTAs share an SM: one ranks while the other streams.
constexpr int kStageBytes = kTileN * 8;  // one array of the tile at 8 bytes per element
constexpr int kRingSmem = kRingStages * kStageBytes + kTileN * 2 /*inv*/ + kRadix * 4 /*delta*/ + 32 * 4 /*scan*/ + 64 /*mbarriers*/;
static_assert(kWarps * kRadix * 4 <= kStageBytes, "the per-warp counters alias ring stage 1");

struct ScatterArgs {
    const uint32_t* key_in; uint32_t* key_out;   // key_out may be null (last pass when no counts are wanted)
    const uint32_t* idx_in; uint32_t* idx_out;   // idx_out may be null (no permutation wanted)
    const uint32_t* base;                        // [tile][nb] global slot of the first item of (digit, tile)
    int64_t n; int shift; uint32_t mask; int nbits; int ntiles; int csync; double dt; int pace_sync, pace_ns;
};

template <class L, bool HAS_IDX, bool DRIFT>
__global__ void __launch_bounds__(kSortThreads, 1024 / kSortThreads) scatter_ring_kernel(Ptrs<L::ncomp> src, Ptrs<L::ncomp> dst, ScatterArgs g) {
    static_assert(!(HAS_IDX && DRIFT), "the drift is applied in the first pass, which generates the indices");
    using Plan = RingPlan<L, HAS_IDX, DRIFT>;
    constexpr Plan plan{};
    constexpr int kFirstComp = Plan::kFirstComp, kArrays = Plan::kArrays;
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char* ring = smem;
    uint16_t* inv = reinterpret_cast<uint16_t*>(smem + kRingStages * kStageBytes);
    uint32_t* delta = reinterpret_cast<uint32_t*>(smem + kRingStages * kStageBytes + kTileN * 2);
    uint32_t* scan_sm = delta + kRadix;
    uint64_t* full = reinterpret_cast<uint64_t*>(scan_sm + 32);
    uint32_t* wcnt = reinterpret_cast<uint32_t*>(ring + kStageBytes);  // aliases stage 1 until the ranking is done

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t n = g.n, tile0 = (int64_t)blockIdx.x * kTileN;
    const int shift = g.shift;
    const uint32_t mask = g.mask;
    const int cnt = n - tile0 < kTileN ? (n > tile0 ? (int)(n - tile0) : 0) : kTileN;  // 0: padding CTA of a cluster launch
    const bool bulk = cnt == kTileN;  // CTA-uniform: the ragged last tile is filled by ordinary loads instead

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kRingStages; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    // fill(stage, array): start bringing `cnt` elements of an array into a ring stage.  Called by ALL threads at
    // CTA-uniform points, after a __syncthreads() that retired every reader of the stage.
    auto fill = [&](int stage, const auto* gp) {
        using T = std::remove_cv_t<std::remove_pointer_t<decltype(gp)>>;
        unsigned char* sb = ring + stage * kStageBytes;
        if (bulk) {
            if (tid == 0) {
                mbar_expect_tx(&full[stage], kTileN * (uint32_t)sizeof(T));
                bulk_g2s(sb, gp + tile0, kTileN * (uint32_t)sizeof(T), &full[stage]);
            }
        } else {
            T* s = reinterpret_cast<T*>(sb);
            for (int i = tid; i < cnt; i += kSortThreads) s[i] = gp[tile0 + i];
        }
    };
    // ready(stage, parity): the array requested by the matching fill() is in shared memory
    auto ready = [&](int stage, uint32_t parity) {
        if (bulk) mbar_wait(&full[stage], parity);
        else __syncthreads();
    };
    // fill_load<k>(): issue the k-th load of the plan (nothing if the plan has fewer arrays)
    auto fill_load = [&](auto ki) {
        constexpr int k = decltype(ki)::value;
        if constexpr (k < kArrays) {
            constexpr int a = plan.load[k];
            if constexpr (a == 0) fill(plan.stage[a], g.key_in);
            else if constexpr (HAS_IDX && a == 1) fill(plan.stage[a], g.idx_in);
            else fill(plan.stage[a], comp_ptr<L, a - kFirstComp>(src));
        }
    };
    static_assert(plan.load[0] == 0 && plan.move[0] == 0 && plan.stage[0] == 0, "the keys lead");
    for (int i = tid; i < kWarps * kRadix; i += kSortThreads) wcnt[i] = 0;
    const uint32_t my_base = (tid <= (int)mask && (int)blockIdx.x < g.ntiles ? g.base[(int64_t)blockIdx.x * (mask + 1) + tid] : 0u);  // consumed after the ranking
    __syncthreads();  // barriers initialised, counters zeroed

    // Stage 1 is the counters for now, so start with loads 0 and 2.
    fill_load(std::integral_constant<int, 0>{});
    fill_load(std::integral_constant<int, 2>{});

    // ---- ranking: warp w owns elements [256 w, 256 w + 256) of the tile, 8 rounds of 32 in element order -------
    ready(0, 0);
    const uint32_t* keybuf = reinterpret_cast<const uint32_t*>(ring);
    const int e0 = warp * (32 * kItems) + lane;
    uint32_t lpos[kItems];
    uint32_t* mycnt = wcnt + warp * kRadix;
    const uint32_t lt = (1u << lane) - 1u;
    uint32_t peers[kItems];
#pragma unroll
    for (int k = 0; k < kItems; ++k) {  // lanes holding the same digit, from one ballot per digit bit (no MATCH: its cost grows with the number of distinct values)
        const int e = e0 + k * 32;
        const bool valid = e < cnt;
        const uint32_t d = valid ? (keybuf[e] >> shift) & mask : 0u;
        uint32_t m = __ballot_sync(0xffffffffu, valid);
#pragma unroll
        for (int b = 0; b < kRadixBits; ++b) {
            if (b >= g.nbits) break;  // warp-uniform: as many ballots as the digit has bits
            const bool bit = (d >> b) & 1u;
            const uint32_t bal = __ballot_sync(0xffffffffu, bit);
            m &= bit ? bal : ~bal;
        }
        peers[k] = valid ? m : 0u;
        lpos[k] = d;
    }
#pragma unroll
    for (int k = 0; k < kItems; ++k) {
        const uint32_t d = lpos[k];
        const uint32_t old = mycnt[d];
        lpos[k] = old + __popc(peers[k] & lt);
        __syncwarp();
        if (peers[k] != 0u && lane == 31 - __clz(peers[k])) mycnt[d] = old + __popc(peers[k]);
        __syncwarp();
    }
    __syncthreads();
    {   // digit d = tid: tile total -> first slot of the bin in tile-sorted order -> per-warp first slots
        uint32_t total = 0;
        if (tid < kRadix) {
#pragma unroll
            for (int w = 0; w < kWarps; ++w) total += wcnt[w * kRadix + tid];
        }
        uint32_t run = block_excl_scan(total, scan_sm);
        if (tid < kRadix) {
            delta[tid] = my_base - run;
#pragma unroll
            for (int w = 0; w < kWarps; ++w) {
                const uint32_t c = wcnt[w * kRadix + tid];
                wcnt[w * kRadix + tid] = run;
                run += c;
            }
        }
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kItems; ++k) {
        const int e = e0 + k * 32;
        if (e < cnt) inv[lpos[k] + mycnt[(keybuf[e] >> shift) & mask]] = (uint16_t)e;
    }
    fence_async_smem();  // the counters (generic-proxy writes) are about to be overwritten by a bulk copy
    __syncthreads();     // inv complete, counters dead: stage 1 joins the ring
    fill_load(std::integral_constant<int, 1>{});

    // ---- output slots: thread t owns slots t, t + 512, ... of the tile-sorted order, so that in its k-th store the whole CTA
    // (and, in step with it, the other CTAs of the cluster) writes ONE window of 512 consecutive slots = the runs of ~64
    // neighbouring bins.  Few runs open at a time is what lets the L2 merge their pieces: giving every warp its own 256
    // consecutive slots instead (16 windows open per CTA) was measured 25 % slower (profiles/r2_bin_study.md).
#define SLOT(k) (tid + (k) * kSortThreads)
    uint32_t gdest[kItems], srcp[kItems / 2];  // source elements packed two per register
    {
        uint32_t kv[kItems];
#pragma unroll
        for (int k = 0; k < kItems; ++k) {
            const int j = SLOT(k);
            uint32_t s = 0;
            kv[k] = 0;
            gdest[k] = 0;
            if (j < cnt) {
                s = inv[j];
                kv[k] = keybuf[s];
                gdest[k] = delta[(kv[k] >> shift) & mask] + (uint32_t)j;
            }
            if (k & 1) srcp[k >> 1] |= s << 16; else srcp[k >> 1] = s;
        }
        if (g.csync) cluster_sync_relaxed();
        if (g.key_out) {
#pragma unroll
            for (int k = 0; k < kItems; ++k) {
                pace(k, g.pace_sync, g.pace_ns);
                if (SLOT(k) < cnt) g.key_out[gdest[k]] = kv[k];
            }
        }
        if constexpr (!HAS_IDX) {
            if (g.idx_out) {
                if (g.csync && g.key_out) cluster_sync_relaxed();
#pragma unroll
                for (int k = 0; k < kItems; ++k) {
                    pace(k, g.pace_sync, g.pace_ns);
                    if (SLOT(k) < cnt) g.idx_out[gdest[k]] = (uint32_t)(tile0 + ((srcp[k >> 1] >> ((k & 1) * 16)) & 0xffffu));
                }
            }
        }
    }
    // gdest depends on every key read of this thread, and gdest is consumed by stores or kept live below: the reads of
    // stage 0 have completed before the barrier (see the note in move()).
    __syncthreads();  // the keys have been read: stage 0 is free
    fill_load(std::integral_constant<int, kRingStages>{});

    // move<m>(): write the m-th array of the move order to its destination, then refill its stage with load m + 3
    auto move = [&](auto mi) {
        constexpr int m = decltype(mi)::value;
        constexpr int a = plan.move[m];
        constexpr int p = plan.partner[a];
        auto body = [&](const auto* tp, auto* gout) {
            using T = std::remove_cv_t<std::remove_pointer_t<decltype(tp)>>;
            ready(plan.stage[a], plan.parity[a]);
            const T* sb = reinterpret_cast<const T*>(ring + plan.stage[a] * kStageBytes);
            T v[kItems];
            if constexpr (p >= 0) {  // DRIFT: this is a position component; its velocity component is in another stage
                using V = typename L::template comp_type<(p >= 0 ? p - kFirstComp : 0)>;
                ready(plan.stage[p >= 0 ? p : 0], plan.parity[p >= 0 ? p : 0]);
                const V* vb = reinterpret_cast<const V*>(ring + plan.stage[p >= 0 ? p : 0] * kStageBytes);
#pragma unroll
                for (int k = 0; k < kItems; ++k) {
                    const uint32_t s = (srcp[k >> 1] >> ((k & 1) * 16)) & 0xffffu;
                    if (SLOT(k) < cnt) v[k] = drift1<V>(g.dt, vb[s], sb[s]);
                }
            } else {
#pragma unroll
                for (int k = 0; k < kItems; ++k) {
                    const uint32_t s = (srcp[k >> 1] >> ((k & 1) * 16)) & 0xffffu;
                    if (SLOT(k) < cnt) v[k] = sb[s];
                }
            }
            if (g.csync) cluster_sync_relaxed();
            // The stores come BEFORE the barrier on purpose: they consume the loaded values, so every shared-memory read
            // of this stage has completed when its thread arrives.  A barrier alone does not order reads that are still
            // in flight in the generic proxy against the bulk copy (async proxy) that refills the stage.
#pragma unroll
            for (int k = 0; k < kItems; ++k) {
                pace(k, g.pace_sync, g.pace_ns);
                if (SLOT(k) < cnt) gout[gdest[k]] = v[k];
            }
            __syncthreads();  // the stage can take the next load
            fill_load(std::integral_constant<int, m + kRingStages>{});
        };
        if constexpr (HAS_IDX && a == 1) body(g.idx_in, g.idx_out);
        else body(comp_ptr<L, (a >= kFirstComp ? a - kFirstComp : 0)>(src), comp_ptr<L, (a >= kFirstComp ? a - kFirstComp : 0)>(dst));
    };
    for_each_int<kArrays - 1>([&](auto i) { move(std::integral_constant<int, decltype(i)::value + 1>{}); });
#undef SLOT
}

// ---- counts / offsets from the sorted keys: off[c] = first sorted slot whose key is >= c (binary search) -------------
__global__ void __launch_bounds__(256) cell_bounds_kernel(const uint32_t* __restrict__ sorted, int64_t n, uint32_t ncell,
                                                          uint32_t* __restrict__ counts, uint32_t* __restrict__ offsets) {
    __shared__ uint32_t off[257];
    auto lower_bound = [&](uint32_t c) {
        int64_t lo = 0, hi = n;
        while (lo < hi) {
            const int64_t mid = (lo + hi) >> 1;
            if (sorted[mid] < c) lo = mid + 1; else hi = mid;
        }
        return (uint32_t)lo;
    };
    const uint32_t c = blockIdx.x * 256u + threadIdx.x;
    off[threadIdx.x] = c <= ncell ? lower_bound(c) : (uint32_t)n;
    if (threadIdx.x == 0) off[256] = c + 256u <= ncell ? lower_bound(c + 256u) : (uint32_t)n;
    __syncthreads();
    if (c < ncell) {
        if (counts) counts[c] = off[threadIdx.x + 1] - off[threadIdx.x];
        if (offsets) offsets[c] = off[threadIdx.x];
    }
}

// ---- host side: scratch plan and the pipeline -------------------------------------------------------------------------
struct PassPlan {
    int npass, width[18];
    PassPlan(int log2g, int bits_override) {
        const int bits = 3 * log2g;
        const int w = bits_override > 0 ? bits_override : kRadixBits;
        npass = bits == 0 ? 1 : (bits + w - 1) / w;
        int shift = 0;
        for (int p = 0; p < npass; ++p) {  // balanced digit widths
            width[p] = bits == 0 ? 0 : (bits - shift + (npass - p) - 1) / (npass - p);
            shift += width[p];
        }
    }
};

template <class L>
struct BinPlan {
    size_t key0, key1, idx1, idx3, slab, hist, partial, dbase, ke, total;
    int64_t ntiles, nchunks;
    size_t comp_off[L::ncomp];
    BinPlan(int64_t n, int npass) {
        ntiles = (n + kTileN - 1) / kTileN;
        if (ntiles < 1) ntiles = 1;
        nchunks = (ntiles + kScanRows - 1) / kScanRows;
        size_t o = 0;
        auto take = [&](size_t bytes) { size_t at = o; o += align_up(bytes ? bytes : 1, kAlign); return at; };
        key0 = take((size_t)n * 4);
        key1 = take((size_t)n * 4);
        idx1 = take(npass >= 2 ? (size_t)n * 4 : 0);
        idx3 = take(npass >= 3 ? (size_t)n * 4 : 0);
        slab = o;
        for (int c = 0; c < L::ncomp; ++c) comp_off[c] = take(npass >= 2 ? (size_t)n * L::comp_size(c) : 0);
        hist = take((size_t)ntiles * kRadix * 4);
        partial = take((size_t)nchunks * kRadix * 4);
        dbase = take(kRadix * 4);
        ke = take((size_t)ntiles * sizeof(double));
        total = o;
    }
};

template <class L>
size_t bin_scratch_bytes(int64_t n, int log2g) {
    if constexpr (!L::template has_as<pos_tag, double, 3>()) return 0;
    else return BinPlan<L>(n, PassPlan(log2g, g_tune.bin_bits).npass).total;
}

template <class K>
int launch_scatter(K kernel, int cluster, unsigned ntiles, cudaStream_t st, const void* src, const void* dst, const ScatterArgs& g) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((ntiles + cluster - 1) / cluster * cluster);  // padding CTAs own no tile but join the cluster barriers
    cfg.blockDim = dim3(kSortThreads);
    cfg.dynamicSmemBytes = kRingSmem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = cluster; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = cluster > 1 ? 1 : 0;
    void* args[] = {const_cast<void*>(src), const_cast<void*>(dst), const_cast<ScatterArgs*>(&g)};
    SOAX_CUDA(cudaLaunchKernelExC(&cfg, reinterpret_cast<const void*>(kernel), args));
    return launched();
}

template <class L>
int bin_permute_entry(const BinArgs& a, cudaStream_t st) {
    constexpr bool has_pos = L::template has_as<pos_tag, double, 3>();
    constexpr bool has_vel = L::template has_as<vel_tag, float, 3>() || L::template has_as<vel_tag, double, 3>();
    if constexpr (!has_pos) {
        return SOAX_ERR_UNSUPPORTED;
    } else {
        const int64_t n = a.n;
        const uint32_t ncell = 1u << (3 * a.log2g);
        const bool drift = a.drift_dt != 0.0, ke = a.kinetic != nullptr;
        if ((drift || ke) && !has_vel) return SOAX_ERR_UNSUPPORTED;
        if (n == 0) {
            if (a.counts) SOAX_CUDA(cudaMemsetAsync(a.counts, 0, (size_t)ncell * 4, st));
            if (a.offsets) SOAX_CUDA(cudaMemsetAsync(a.offsets, 0, (size_t)ncell * 4, st));
            if (ke) SOAX_CUDA(cudaMemsetAsync(a.kinetic, 0, sizeof(double), st));
            return SOAX_OK;
        }
        const PassPlan pp(a.log2g, g_tune.bin_bits);
        const int npass = pp.npass;
        const BinPlan<L> plan(n, npass);
        if (a.scratch_bytes < plan.total) return SOAX_ERR_ALLOC;
        char* sc = static_cast<char*>(a.scratch);
        uint32_t* keys[2] = {reinterpret_cast<uint32_t*>(sc + plan.key0), reinterpret_cast<uint32_t*>(sc + plan.key1)};
        uint32_t* idxs[2] = {reinterpret_cast<uint32_t*>(sc + plan.idx1), reinterpret_cast<uint32_t*>(sc + plan.idx3)};
        uint32_t* hist = reinterpret_cast<uint32_t*>(sc + plan.hist);
        uint32_t* partial = reinterpret_cast<uint32_t*>(sc + plan.partial);
        uint32_t* dbase = reinterpret_cast<uint32_t*>(sc + plan.dbase);
        double* kep = reinterpret_cast<double*>(sc + plan.ke);
        const Ptrs<L::ncomp> src = make_ptrs<L>(a.src), dst = make_ptrs<L>(a.dst);
        Ptrs<L::ncomp> tmp;
        for (int c = 0; c < L::ncomp; ++c) tmp.p[c] = sc + plan.comp_off[c];
        const unsigned ntiles = (unsigned)plan.ntiles, nchunks = (unsigned)plan.nchunks;
        const bool want_sorted_keys = a.counts || a.offsets;

        // The function attributes are per device: set them on every call (cheap) rather than once per process.
        for (const void* f : {(const void*)scatter_ring_kernel<L, false, false>, (const void*)scatter_ring_kernel<L, true, false>,
                              (const void*)scatter_ring_kernel<L, false, has_vel>}) {
            SOAX_CUDA(cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, kRingSmem));
            SOAX_CUDA(cudaFuncSetAttribute(f, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
        }

        // Least-significant-digit passes over the 3*log2g key bits.
        int shift = 0;
        for (int pass = 0; pass < npass; ++pass) {
            const bool last = pass == npass - 1;
            const int w = pp.width[pass];
            const uint32_t mask = (1u << w) - 1u;
            const int nb = (int)mask + 1, scan_threads = nb < 32 ? 32 : nb;  // the table is [tile][nb]
            const uint32_t* kin = keys[pass & 1];
            if (pass == 0) {  // [drift +] cell index [+ KE] + first-digit histogram; src is read only
                if constexpr (has_vel) {
                    if (drift && ke) cell_hist_kernel<L, true, true><<<ntiles, kCellThreads, 0, st>>>(src, n, keys[0], a.drift_dt, a.log2g, mask, hist, kep);
                    else if (drift) cell_hist_kernel<L, true, false><<<ntiles, kCellThreads, 0, st>>>(src, n, keys[0], a.drift_dt, a.log2g, mask, hist, kep);
                    else if (ke) cell_hist_kernel<L, false, true><<<ntiles, kCellThreads, 0, st>>>(src, n, keys[0], a.drift_dt, a.log2g, mask, hist, kep);
                    else cell_hist_kernel<L, false, false><<<ntiles, kCellThreads, 0, st>>>(src, n, keys[0], a.drift_dt, a.log2g, mask, hist, kep);
                } else {
                    cell_hist_kernel<L, false, false><<<ntiles, kCellThreads, 0, st>>>(src, n, keys[0], a.drift_dt, a.log2g, mask, hist, kep);
                }
                SOAX_TRY(launched());
                if (ke) SOAX_TRY(sum_partials(kep, (int)ntiles, a.kinetic, st));
            } else {
                tile_hist_kernel<<<ntiles, kSortThreads, 0, st>>>(kin, n, shift, mask, hist);
                SOAX_TRY(launched());
            }
            colscan_reduce_kernel<<<nchunks, scan_threads, 0, st>>>(hist, (int)ntiles, nb, partial);
            SOAX_TRY(launched());
            colscan_top_kernel<<<1, scan_threads, 0, st>>>(partial, (int)nchunks, nb, dbase);
            SOAX_TRY(launched());
            colscan_apply_kernel<<<nchunks, scan_threads, 0, st>>>(hist, (int)ntiles, nb, partial, dbase);
            SOAX_TRY(launched());

            // the last pass writes dst; before it the records alternate between the scratch slab and dst
            const bool to_dst = ((npass - 1 - pass) & 1) == 0;
            const Ptrs<L::ncomp>& from = pass == 0 ? src : (to_dst ? tmp : dst);
            const Ptrs<L::ncomp>& to = to_dst ? dst : tmp;
            ScatterArgs g{};
            g.key_in = kin;
            g.key_out = (!last || want_sorted_keys) ? keys[(pass + 1) & 1] : nullptr;  // sorted keys end in keys[npass & 1]
            g.idx_in = pass == 0 || !a.perm ? nullptr : idxs[(pass - 1) & 1];
            g.idx_out = !a.perm ? nullptr : (last ? a.perm : idxs[pass & 1]);
            g.base = hist; g.n = n; g.shift = shift; g.mask = mask; g.nbits = w; g.ntiles = (int)ntiles; g.dt = a.drift_dt; 
            // Short runs (wide digits) need the neighbouring tiles' pieces to reach the L2 together: clusters + barrier.
            const int want_cluster = g_tune.bin_cluster > 0 ? g_tune.bin_cluster : 4;
            const int cluster = (g_tune.bin_cluster > 0 || w >= 8) ? want_cluster : 1;
            g.csync = cluster > 1 && g_tune.bin_csync != 0;
            g.pace_sync = g_tune.bin_pace >= 0 ? (g_tune.bin_pace >> 12) & 3 : (cluster > 1 ? 2 : 0);
            if (g.pace_sync == 2 && cluster == 1) g.pace_sync = 1;
            g.pace_ns = g_tune.bin_pace >= 0 ? g_tune.bin_pace & 0xfff : 0;
            if (pass == 0) {
                if constexpr (has_vel) {
                    if (drift) SOAX_TRY(launch_scatter(scatter_ring_kernel<L, false, true>, cluster, ntiles, st, &from, &to, g));
                    else SOAX_TRY(launch_scatter(scatter_ring_kernel<L, false, false>, cluster, ntiles, st, &from, &to, g));
                } else {
                    SOAX_TRY(launch_scatter(scatter_ring_kernel<L, false, false>, cluster, ntiles, st, &from, &to, g));
                }
            } else if (a.perm) {
                SOAX_TRY(launch_scatter(scatter_ring_kernel<L, true, false>, cluster, ntiles, st, &from, &to, g));
            } else {
                SOAX_TRY(launch_scatter(scatter_ring_kernel<L, false, false>, cluster, ntiles, st, &from, &to, g));
            }
            shift += w;
        }
        if (want_sorted_keys) {
            cell_bounds_kernel<<<ncell / 256 + 1, 256, 0, st>>>(keys[npass & 1], n, ncell, a.counts, a.offsets);
            SOAX_TRY(launched());
        }
        return SOAX_OK;
    }
}

#define X(L)                                                               \
    template int bin_permute_entry<L>(const BinArgs&, cudaStream_t);      \
    template size_t bin_scratch_bytes<L>(int64_t, int);
SOAX_FOR_EACH_LAYOUT(X)
#undef X

}  // namespace soax
