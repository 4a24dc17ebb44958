// bin_kernels.cu -- a10..a14: PIC-style cell binning with a STABLE counting-sort permutation of every field
// array (BASELINE.json config 5).
//
// Design: the 18-bit cell key is sorted by a two-pass least-significant-digit counting
// sort with 9-bit digits (512 bins per pass), and the WHOLE RECORD travels with its key through both passes
// together with its source index, so `perm` falls out as the carried index and no random gather of the field
// arrays is ever made (a per-array gather would read one 32-byte sector per 4- or 8-byte item).  Each pass:
//   tile_hist   per-tile digit histogram (tiles of kTileN consecutive particles)            4 B/particle read
//   colscan_*   exclusive scan of the [tile][digit] table in digit-major order              (small)
//   scatter     stable in-tile ranks (warp match + per-warp running counters), then every component array is
//               moved src[i] -> dst[base[tile][digit] + rank]
// Every step is a pure function of the data (no arrival-order atomics decide a position), so the result is the
// unique stable permutation for ANY particle distribution, and bit-identical from run to run.
// counts / offsets come from the sorted keys by boundary detection.
#include "common.cuh"
#include "ops.hpp"
#include "tma.cuh"

namespace soax {

int sum_partials(const double* partial, int m, double* out, cudaStream_t st);  // reduce_kernels.cu

constexpr int kRadixBits = 9;
constexpr int kRadix = 1 << kRadixBits;        // 512 bins per pass
constexpr int kSortThreads = 512;              // 16 warps
constexpr int kItems = 8;                      // keys per thread
constexpr int kTileN = kSortThreads * kItems;  // 4096 particles per tile
constexpr int kWarps = kSortThreads / 32;
constexpr int kScanRows = 64;                  // tiles per column-scan chunk

// ---- pass 0: [drift +] cell index [+ kinetic energy], P = 4 particles per thread, fixed grid -------------------
template <class L, bool DRIFT, bool KE, int P>
__device__ __forceinline__ double cell_group(const Ptrs<L::ncomp>& a, int64_t i0, uint32_t* cell, double dt, double G,
                                             int gmax, int log2g) {
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
        for (int d = 0; d < 3; ++d) {
#pragma unroll
            for (int j = 0; j < P; ++j) x[d].v[j] = drift1<V>(dt, v[d].v[j], x[d].v[j]);
            st_vec<double, P>(field_ptr<L, pos_tag>(a, d) + i0, x[d]);
        }
    }
    Vec<uint32_t, P> c;
    double e = 0.0;
#pragma unroll
    for (int j = 0; j < P; ++j) {
        c.v[j] = cell_of(x[0].v[j], x[1].v[j], x[2].v[j], G, gmax, log2g);
        if constexpr (KE)
            e += energy1<false>((double)v[0].v[j], (double)v[1].v[j], (double)v[2].v[j], 0.0, 0.0, 0.0, 0.0, 0.0);
    }
    st_vec<uint32_t, P>(cell + i0, c);
    return e;
}

template <class L, bool DRIFT, bool KE>
__global__ void __launch_bounds__(256) cell_kernel(Ptrs<L::ncomp> a, int64_t n, uint32_t* cell, double dt, int log2g,
                                                   double* ke_partial) {
    constexpr int P = 4;
    __shared__ double sm[32];
    const double G = (double)(1 << log2g);
    const int gmax = (1 << log2g) - 1;
    const int64_t ngroups = n / P;
    const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    double e = 0.0;
    for (int64_t g = tid; g < ngroups; g += stride) e += cell_group<L, DRIFT, KE, P>(a, g * P, cell, dt, G, gmax, log2g);
    const int64_t t = ngroups * P + tid;
    if (t < n) e += cell_group<L, DRIFT, KE, 1>(a, t, cell, dt, G, gmax, log2g);
    if constexpr (KE) {
        e = block_sum(e, sm);
        if (threadIdx.x == 0) ke_partial[blockIdx.x] = e;
    }
}

// ---- per-tile digit histogram -------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kSortThreads) tile_hist_kernel(const uint32_t* __restrict__ keys, int64_t n, int shift, uint32_t mask,
                                                                 uint32_t* __restrict__ hist) {
    __shared__ uint32_t h[kRadix];
    h[threadIdx.x] = 0;
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

// ---- stable scatter of one tile: keys, source indices and EVERY component array ------------------------------------
template <class L>
__global__ void __launch_bounds__(kSortThreads) scatter_kernel(Ptrs<L::ncomp> src, Ptrs<L::ncomp> dst,
                                                               const uint32_t* __restrict__ key_in, uint32_t* __restrict__ key_out,
                                                               const uint32_t* __restrict__ idx_in, uint32_t* __restrict__ idx_out,
                                                               const uint32_t* __restrict__ base, int64_t n, int shift, uint32_t mask) {
    __shared__ uint32_t wcnt[kWarps * kRadix];  // per-warp running digit counters, then per-warp global bases
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < kWarps * kRadix; i += kSortThreads) wcnt[i] = 0;
    __syncthreads();

    // warp w owns the 32*kItems consecutive particles starting at tile0 + w*32*kItems; round k covers 32 of them
    const int64_t e0 = (int64_t)blockIdx.x * kTileN + warp * (32 * kItems) + lane;
    uint32_t key[kItems], dest[kItems];
    uint32_t* mycnt = wcnt + warp * kRadix;
    const uint32_t lt = (1u << lane) - 1u;
#pragma unroll
    for (int k = 0; k < kItems; ++k) {
        const int64_t e = e0 + k * 32;
        const bool valid = e < n;
        key[k] = valid ? key_in[e] : 0u;
        const uint32_t d = (key[k] >> shift) & mask;
        const uint32_t peers = __match_any_sync(0xffffffffu, valid ? d : (0x10000u | lane));
        const uint32_t old = mycnt[d];
        dest[k] = old + __popc(peers & lt);  // rank among the warp's earlier particles with this digit
        __syncwarp();
        if (valid && lane == 31 - __clz(peers)) mycnt[d] = old + __popc(peers);
        __syncwarp();
    }
    __syncthreads();
    // digit d (one thread each): turn the per-warp counts into global bases, warps in order
    {
        uint32_t run = (threadIdx.x <= mask ? base[(int64_t)blockIdx.x * (mask + 1) + threadIdx.x] : 0u);
#pragma unroll
        for (int w = 0; w < kWarps; ++w) {
            const uint32_t c = wcnt[w * kRadix + threadIdx.x];
            wcnt[w * kRadix + threadIdx.x] = run;
            run += c;
        }
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kItems; ++k) dest[k] += mycnt[(key[k] >> shift) & mask];

#pragma unroll
    for (int k = 0; k < kItems; ++k) {
        const int64_t e = e0 + k * 32;
        if (e < n) {
            key_out[dest[k]] = key[k];
            idx_out[dest[k]] = idx_in ? idx_in[e] : (uint32_t)e;
        }
    }
    for_each_comp<L>([&](auto ci) {
        constexpr int C = decltype(ci)::value;
        using T = typename L::template comp_type<C>;
        const T* s = comp_ptr<L, C>(src);
        T* t = comp_ptr<L, C>(dst);
        T val[kItems];
#pragma unroll
        for (int k = 0; k < kItems; ++k) {
            const int64_t e = e0 + k * 32;
            if (e < n) val[k] = s[e];
        }
#pragma unroll
        for (int k = 0; k < kItems; ++k) {
            const int64_t e = e0 + k * 32;
            if (e < n) t[dest[k]] = val[k];
        }
    });
}

// ---- stable scatter, shared-memory staged: the tile is first sorted INSIDE shared memory, so that consecutive
// threads then write consecutive slots of each bin's run and every run leaves the SM as a few full sectors
// (the direct kernel above sends 32 different sectors per warp store).  One staging buffer (8 bytes per slot)
// is reused for the key array, the index array and each component array in turn; it aliases the per-warp
// counters, which are dead once every particle knows its slot.
template <class T>
__device__ __forceinline__ void stage_move(const T* __restrict__ s, T* __restrict__ t, unsigned char* buf, int64_t e0, int64_t n,
                                           int cnt, const uint32_t (&lpos)[kItems], const uint32_t (&gdest)[kItems]) {
    T* sm = reinterpret_cast<T*>(buf);
    T val[kItems];
#pragma unroll
    for (int k = 0; k < kItems; ++k) {
        const int64_t e = e0 + k * 32;
        if (e < n) val[k] = s[e];
    }
    __syncthreads();  // the previous array has been read out of the buffer
#pragma unroll
    for (int k = 0; k < kItems; ++k)
        if (e0 + k * 32 < n) sm[lpos[k]] = val[k];
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kItems; ++k) {
        const int j = threadIdx.x + k * kSortThreads;
        if (j < cnt) t[gdest[k]] = sm[j];
    }
}

template <class L>
__global__ void __launch_bounds__(kSortThreads) scatter_staged_kernel(Ptrs<L::ncomp> src, Ptrs<L::ncomp> dst,
                                                                      const uint32_t* __restrict__ key_in, uint32_t* __restrict__ key_out,
                                                                      const uint32_t* __restrict__ idx_in, uint32_t* __restrict__ idx_out,
                                                                      const uint32_t* __restrict__ base, int64_t n, int shift, uint32_t mask) {
    __shared__ __align__(16) unsigned char buf[kWarps * kRadix * 4 > kTileN * 8 ? kWarps * kRadix * 4 : kTileN * 8];
    __shared__ uint32_t delta[kRadix];  // global slot of a bin's first item minus its first slot inside the sorted tile
    __shared__ uint32_t scan_sm[32];
    uint32_t* wcnt = reinterpret_cast<uint32_t*>(buf);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < kWarps * kRadix; i += kSortThreads) wcnt[i] = 0;
    __syncthreads();

    const int64_t tile0 = (int64_t)blockIdx.x * kTileN;
    const int cnt = (int)(n - tile0 < kTileN ? n - tile0 : kTileN);
    const int64_t e0 = tile0 + warp * (32 * kItems) + lane;
    uint32_t key[kItems], lpos[kItems], gdest[kItems];
    uint32_t* mycnt = wcnt + warp * kRadix;
    const uint32_t lt = (1u << lane) - 1u;
#pragma unroll
    for (int k = 0; k < kItems; ++k) {
        const int64_t e = e0 + k * 32;
        const bool valid = e < n;
        key[k] = valid ? key_in[e] : 0u;
        const uint32_t d = (key[k] >> shift) & mask;
        const uint32_t peers = __match_any_sync(0xffffffffu, valid ? d : (0x10000u | lane));
        const uint32_t old = mycnt[d];
        lpos[k] = old + __popc(peers & lt);
        __syncwarp();
        if (valid && lane == 31 - __clz(peers)) mycnt[d] = old + __popc(peers);
        __syncwarp();
    }
    __syncthreads();
    {   // digit d = threadIdx.x: tile total -> first slot of the bin inside the sorted tile -> per-warp first slots
        uint32_t total = 0;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) total += wcnt[w * kRadix + threadIdx.x];
        uint32_t run = block_excl_scan(total, scan_sm);
        delta[threadIdx.x] = (threadIdx.x <= mask ? base[(int64_t)blockIdx.x * (mask + 1) + threadIdx.x] : 0u) - run;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) {
            const uint32_t c = wcnt[w * kRadix + threadIdx.x];
            wcnt[w * kRadix + threadIdx.x] = run;
            run += c;
        }
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < kItems; ++k) lpos[k] += mycnt[(key[k] >> shift) & mask];
    __syncthreads();  // the counters are dead from here on: `buf` becomes the staging buffer

    // keys first: the sorted keys tell every output slot j which bin (hence which global run) it belongs to
    {
        uint32_t* sm = reinterpret_cast<uint32_t*>(buf);
#pragma unroll
        for (int k = 0; k < kItems; ++k)
            if (e0 + k * 32 < n) sm[lpos[k]] = key[k];
        __syncthreads();
#pragma unroll
        for (int k = 0; k < kItems; ++k) {
            const int j = threadIdx.x + k * kSortThreads;
            if (j < cnt) {
                const uint32_t kj = sm[j];
                gdest[k] = delta[(kj >> shift) & mask] + (uint32_t)j;
                key_out[gdest[k]] = kj;
            }
        }
    }
    // source indices (generated in the first pass, carried in the second): perm falls out of the last pass
    {
        uint32_t* sm = reinterpret_cast<uint32_t*>(buf);
        uint32_t val[kItems];
#pragma unroll
        for (int k = 0; k < kItems; ++k) {
            const int64_t e = e0 + k * 32;
            if (e < n) val[k] = idx_in ? idx_in[e] : (uint32_t)e;
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < kItems; ++k)
            if (e0 + k * 32 < n) sm[lpos[k]] = val[k];
        __syncthreads();
#pragma unroll
        for (int k = 0; k < kItems; ++k) {
            const int j = threadIdx.x + k * kSortThreads;
            if (j < cnt) idx_out[gdest[k]] = sm[j];
        }
    }
    for_each_comp<L>([&](auto ci) {
        constexpr int C = decltype(ci)::value;
        stage_move(comp_ptr<L, C>(src), comp_ptr<L, C>(dst), buf, e0, n, cnt, lpos, gdest);
    });
}

// ---- stable scatter, TMA ring (default): every array of the tile (keys, carried source indices, each component
// array) arrives in shared memory as ONE 1-D bulk asynchronous copy (cp.async.bulk -> UBLKCP) into a 3-stage
// ring, so the loads of the next arrays are in flight while the current one is being written out; nothing passes
// through registers on the way in.  The tile is never physically sorted in shared memory: after the ranking
// every output slot j knows its source element inv[j] (the inverse of the in-tile stable permutation), reads
// ring[inv[j]] and writes it to its global slot, consecutive threads writing consecutive slots of a bin's run.
// 64 registers/thread and ~106 KB of shared memory let two CTAs share an SM: one ranks while the other streams.
constexpr int kRingStages = 3;
constexpr int kStageBytes = kTileN * 8;  // one array of the tile at 8 bytes per element
constexpr int kRingSmem = kRingStages * kStageBytes + kTileN * 2 /*inv*/ + kRadix * 4 /*delta*/ + 32 * 4 /*scan*/ + 64 /*mbarriers*/;
static_assert(kWarps * kRadix * 4 <= kStageBytes, "the per-warp counters alias ring stage 1");

template <class L, bool HAS_IDX>
__global__ void __launch_bounds__(kSortThreads, 2) scatter_ring_kernel(Ptrs<L::ncomp> src, Ptrs<L::ncomp> dst,
                                                                      const uint32_t* __restrict__ key_in, uint32_t* __restrict__ key_out,
                                                                      const uint32_t* __restrict__ idx_in, uint32_t* __restrict__ idx_out,
                                                                      const uint32_t* __restrict__ base, int64_t n, int shift, uint32_t mask) {
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char* ring = smem;
    uint16_t* inv = reinterpret_cast<uint16_t*>(smem + kRingStages * kStageBytes);
    uint32_t* delta = reinterpret_cast<uint32_t*>(smem + kRingStages * kStageBytes + kTileN * 2);
    uint32_t* scan_sm = delta + kRadix;
    uint64_t* full = reinterpret_cast<uint64_t*>(scan_sm + 32);
    uint32_t* wcnt = reinterpret_cast<uint32_t*>(ring + kStageBytes);  // aliases stage 1 until the ranking is done

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t tile0 = (int64_t)blockIdx.x * kTileN;
    const int cnt = (int)(n - tile0 < kTileN ? n - tile0 : kTileN);
    const bool bulk = cnt == kTileN;  // CTA-uniform: the ragged last tile is filled by ordinary loads instead

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kRingStages; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    // fill(stage, array): start bringing `cnt` elements of an array into a ring stage.  Called by ALL threads at
    // CTA-uniform points, after a __syncthreads() that retired every reader of the stage.
    auto fill = [&](int stage, const auto* g) {
        using T = std::remove_cv_t<std::remove_pointer_t<decltype(g)>>;
        unsigned char* sb = ring + stage * kStageBytes;
        if (bulk) {
            if (tid == 0) {
                mbar_expect_tx(&full[stage], kTileN * (uint32_t)sizeof(T));
                bulk_g2s(sb, g + tile0, kTileN * (uint32_t)sizeof(T), &full[stage]);
            }
        } else {
            T* s = reinterpret_cast<T*>(sb);
            for (int i = tid; i < cnt; i += kSortThreads) s[i] = g[tile0 + i];
        }
    };
    // ready(stage, parity): the array requested by the matching fill() is in shared memory
    auto ready = [&](int stage, uint32_t parity) {
        if (bulk) mbar_wait(&full[stage], parity);
        else __syncthreads();
    };
    for (int i = tid; i < kWarps * kRadix; i += kSortThreads) wcnt[i] = 0;
    const uint32_t my_base = (tid <= (int)mask ? base[(int64_t)blockIdx.x * (mask + 1) + tid] : 0u);  // issued now, consumed after the ranking
    __syncthreads();  // barriers initialised, counters zeroed

    // sequence of arrays moved by this CTA: 0 = keys, [1 = carried indices,] then the components; array a uses
    // ring stage a % 3 for the (a / 3)-th time.  Stage 1 is the counters for now, so start with arrays 0 and 2.
    constexpr int kFirstComp = HAS_IDX ? 2 : 1;
    constexpr int kArrays = kFirstComp + L::ncomp;
    auto fill_array = [&](auto ai) {  // ai: integral_constant<int, a>
        constexpr int a = decltype(ai)::value;
        if constexpr (a >= kArrays) {
        } else if constexpr (a == 0) {
            fill(0, key_in);
        } else if constexpr (HAS_IDX && a == 1) {
            fill(1, idx_in);
        } else {
            constexpr int C = a - kFirstComp;
            fill(a % kRingStages, comp_ptr<L, C>(src));
        }
    };
    fill_array(std::integral_constant<int, 0>{});
    fill_array(std::integral_constant<int, 2>{});

    // ---- ranking: warp w owns elements [256 w, 256 w + 256) of the tile, 8 rounds of 32 in element order -------
    ready(0, 0);
    const uint32_t* keybuf = reinterpret_cast<const uint32_t*>(ring);
    const int e0 = warp * (32 * kItems) + lane;
    uint32_t lpos[kItems];
    uint32_t* mycnt = wcnt + warp * kRadix;
    const uint32_t lt = (1u << lane) - 1u;
    uint32_t peers[kItems];
#pragma unroll
    for (int k = 0; k < kItems; ++k) {  // lanes holding the same digit, from kRadixBits ballots (no MATCH: its cost grows with the number of distinct values)
        const int e = e0 + k * 32;
        const bool valid = e < cnt;
        const uint32_t d = valid ? (keybuf[e] >> shift) & mask : 0u;
        uint32_t m = __ballot_sync(0xffffffffu, valid);
#pragma unroll
        for (int b = 0; b < kRadixBits; ++b) {
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
#pragma unroll
        for (int w = 0; w < kWarps; ++w) total += wcnt[w * kRadix + tid];
        uint32_t run = block_excl_scan(total, scan_sm);
        delta[tid] = my_base - run;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) {
            const uint32_t c = wcnt[w * kRadix + tid];
            wcnt[w * kRadix + tid] = run;
            run += c;
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
    fill_array(std::integral_constant<int, 1>{});

    // ---- output slots: thread t owns slots t, t + 512, ... of the tile-sorted order --------------------------------
    uint32_t gdest[kItems], srcp[kItems / 2];  // source elements packed two per register
#pragma unroll
    for (int k = 0; k < kItems; ++k) {
        const int j = tid + k * kSortThreads;
        uint32_t s = 0;
        if (j < cnt) {
            s = inv[j];
            const uint32_t kj = keybuf[s];
            gdest[k] = delta[(kj >> shift) & mask] + (uint32_t)j;
            key_out[gdest[k]] = kj;
            if constexpr (!HAS_IDX) idx_out[gdest[k]] = (uint32_t)(tile0 + s);
        }
        if (k & 1) srcp[k >> 1] |= s << 16; else srcp[k >> 1] = s;
    }
    __syncthreads();  // the keys have been read: stage 0 is free
    fill_array(std::integral_constant<int, 3>{});

    auto move_array = [&](auto ai, const auto* /*type tag*/ tp, auto* gout) {
        constexpr int a = decltype(ai)::value;
        using T = std::remove_cv_t<std::remove_pointer_t<decltype(tp)>>;
        ready(a % kRingStages, (a / kRingStages) & 1);
        const T* sb = reinterpret_cast<const T*>(ring + (a % kRingStages) * kStageBytes);
        T v[kItems];
#pragma unroll
        for (int k = 0; k < kItems; ++k) {
            const uint32_t s = (srcp[k >> 1] >> ((k & 1) * 16)) & 0xffffu;
            if (tid + k * kSortThreads < cnt) v[k] = sb[s];
        }
        // The stores come BEFORE the barrier on purpose: they consume the loaded values, so every shared-memory
        // read of this stage has completed when its thread arrives.  A barrier alone does not order reads that are
        // still in flight in the generic proxy against the bulk copy (async proxy) that refills the stage.
#pragma unroll
        for (int k = 0; k < kItems; ++k)
            if (tid + k * kSortThreads < cnt) gout[gdest[k]] = v[k];
        __syncthreads();  // the stage can take the array three places ahead
        fill_array(std::integral_constant<int, a + kRingStages>{});
    };
    if constexpr (HAS_IDX) move_array(std::integral_constant<int, 1>{}, idx_in, idx_out);
    for_each_comp<L>([&](auto ci) {
        constexpr int C = decltype(ci)::value;
        move_array(std::integral_constant<int, kFirstComp + C>{}, comp_ptr<L, C>(src), comp_ptr<L, C>(dst));
    });
}

// ---- counts / offsets from the sorted keys --------------------------------------------------------------------------
// off[c] = first sorted slot whose key is >= c, for c = 0..ncell (off[ncell] = n)
__global__ void __launch_bounds__(256) boundaries_kernel(const uint32_t* __restrict__ sorted, int64_t n, uint32_t ncell,
                                                         uint32_t* __restrict__ off) {
    // four consecutive sorted keys per thread (one 128-bit load) plus the key before them
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t ngroups = (n + 3) / 4;
    for (int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; g < ngroups; g += stride) {
        const int64_t j0 = g * 4;
        uint32_t k[4];
        if (j0 + 4 <= n) {
            const uint4 v = *reinterpret_cast<const uint4*>(sorted + j0);
            k[0] = v.x; k[1] = v.y; k[2] = v.z; k[3] = v.w;
        } else {
#pragma unroll
            for (int i = 0; i < 4; ++i) k[i] = j0 + i < n ? sorted[j0 + i] : 0u;
        }
        uint32_t first = j0 == 0 ? 0u : sorted[j0 - 1] + 1u;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int64_t j = j0 + i;
            if (j >= n) break;
            for (uint32_t c = first; c <= k[i]; ++c) off[c] = (uint32_t)j;
            first = k[i] + 1u;
            if (j == n - 1)
                for (uint32_t c = k[i] + 1u; c <= ncell; ++c) off[c] = (uint32_t)n;
        }
    }
}
__global__ void __launch_bounds__(256) counts_kernel(const uint32_t* __restrict__ off, uint32_t ncell, uint32_t* counts,
                                                     uint32_t* offsets) {
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c < ncell) {
        if (counts) counts[c] = off[c + 1] - off[c];
        if (offsets) offsets[c] = off[c];
    }
}

// ---- host side: scratch plan and the pipeline -------------------------------------------------------------------------
template <class L>
struct BinPlan {
    size_t key0, key1, idx1, idx2, idx3, slab, hist, partial, dbase, off, ke, total;
    int64_t ntiles, nchunks;
    size_t comp_off[L::ncomp];
    BinPlan(int64_t n, int log2g) {
        ntiles = (n + kTileN - 1) / kTileN;
        if (ntiles < 1) ntiles = 1;
        nchunks = (ntiles + kScanRows - 1) / kScanRows;
        const size_t ncell = (size_t)1 << (3 * log2g);
        size_t o = 0;
        auto take = [&](size_t bytes) { size_t at = o; o += align_up(bytes ? bytes : 1, kAlign); return at; };
        key0 = take((size_t)n * 4);
        key1 = take((size_t)n * 4);
        idx1 = take((size_t)n * 4);
        idx2 = take((size_t)n * 4);
        idx3 = take((size_t)n * 4);
        slab = o;
        for (int c = 0; c < L::ncomp; ++c) comp_off[c] = take((size_t)n * L::comp_size(c));
        hist = take((size_t)ntiles * kRadix * 4);
        partial = take((size_t)nchunks * kRadix * 4);
        dbase = take(kRadix * 4);
        off = take((ncell + 1) * 4);
        ke = take(kEnergyScratchBytes);
        total = o;
    }
};

template <class L>
size_t bin_scratch_bytes(int64_t n, int log2g) {
    if constexpr (!L::template has_as<pos_tag, double, 3>()) return 0;
    else return BinPlan<L>(n, log2g).total;
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
        const BinPlan<L> plan(n, a.log2g);
        char* sc = static_cast<char*>(a.scratch);
        uint32_t* key0 = reinterpret_cast<uint32_t*>(sc + plan.key0);
        uint32_t* key1 = reinterpret_cast<uint32_t*>(sc + plan.key1);
        uint32_t* idx1 = reinterpret_cast<uint32_t*>(sc + plan.idx1);
        uint32_t* idx2 = a.perm ? a.perm : reinterpret_cast<uint32_t*>(sc + plan.idx2);
        uint32_t* idx3 = reinterpret_cast<uint32_t*>(sc + plan.idx3);
        uint32_t* hist = reinterpret_cast<uint32_t*>(sc + plan.hist);
        uint32_t* partial = reinterpret_cast<uint32_t*>(sc + plan.partial);
        uint32_t* dbase = reinterpret_cast<uint32_t*>(sc + plan.dbase);
        uint32_t* off = reinterpret_cast<uint32_t*>(sc + plan.off);
        double* kep = reinterpret_cast<double*>(sc + plan.ke);
        const Ptrs<L::ncomp> src = make_ptrs<L>(a.src), dst = make_ptrs<L>(a.dst);
        Ptrs<L::ncomp> tmp;
        for (int c = 0; c < L::ncomp; ++c) tmp.p[c] = sc + plan.comp_off[c];

        // pass 0: [drift +] cell index [+ KE]
        if constexpr (has_vel) {
            if (drift && ke) cell_kernel<L, true, true><<<kEnergyBlocks, 256, 0, st>>>(src, n, key0, a.drift_dt, a.log2g, kep);
            else if (drift) cell_kernel<L, true, false><<<kEnergyBlocks, 256, 0, st>>>(src, n, key0, a.drift_dt, a.log2g, kep);
            else if (ke) cell_kernel<L, false, true><<<kEnergyBlocks, 256, 0, st>>>(src, n, key0, a.drift_dt, a.log2g, kep);
            else cell_kernel<L, false, false><<<kEnergyBlocks, 256, 0, st>>>(src, n, key0, a.drift_dt, a.log2g, kep);
        } else {
            cell_kernel<L, false, false><<<kEnergyBlocks, 256, 0, st>>>(src, n, key0, a.drift_dt, a.log2g, kep);
        }
        SOAX_TRY(launched());
        if (ke) SOAX_TRY(sum_partials(kep, kEnergyBlocks, a.kinetic, st));

        static const bool ring_ready = [] {
            return cudaFuncSetAttribute(scatter_ring_kernel<L, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kRingSmem) == cudaSuccess &&
                   cudaFuncSetAttribute(scatter_ring_kernel<L, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kRingSmem) == cudaSuccess;
        }();
        if (!ring_ready) return cuda_fail(cudaGetLastError());
        // Least-significant-digit passes over the 3*log2g key bits.  Digit width is a measured trade (profiles/): a pass
        // with 512 bins leaves runs of ~8 elements whose ragged ends cost partial-sector read-modify-writes in L2
        // (5.0 ms per pass at 2^27), a pass with 64 bins leaves runs of ~64 (2.2 ms), so three 6-bit passes beat two
        // 9-bit passes.  soax_tune("bin_bits") overrides the width.
        const int bits = 3 * a.log2g;
        const int width = g_tune.bin_bits > 0 ? g_tune.bin_bits : 6;
        const int npass = bits == 0 ? 1 : (bits + width - 1) / width;
        const unsigned ntiles = (unsigned)plan.ntiles, nchunks = (unsigned)plan.nchunks;
        uint32_t* keys[2] = {key0, key1};
        uint32_t* idxs[2] = {idx1, idx3};
        int shift = 0;
        for (int pass = 0; pass < npass; ++pass) {
            const bool last = pass == npass - 1;
            const int w = (bits - shift + (npass - pass) - 1) / (npass - pass);  // balanced digit widths
            const uint32_t mask = (1u << w) - 1u;
            const uint32_t* kin = keys[pass & 1];
            uint32_t* kout = keys[(pass + 1) & 1];  // sorted keys end in keys[npass & 1]
            const uint32_t* iin = pass == 0 ? nullptr : idxs[(pass - 1) & 1];
            uint32_t* iout = last ? idx2 : idxs[pass & 1];
            // the last pass writes dst; before it the records alternate between the scratch slab and dst
            const bool to_dst = ((npass - 1 - pass) & 1) == 0;
            const Ptrs<L::ncomp>& from = pass == 0 ? src : (to_dst ? tmp : dst);
            const Ptrs<L::ncomp>& to = to_dst ? dst : tmp;
            tile_hist_kernel<<<ntiles, kSortThreads, 0, st>>>(kin, n, shift, mask, hist);
            SOAX_TRY(launched());
            const int nb = (int)mask + 1, scan_threads = nb < 32 ? 32 : nb;  // the table is [tile][nb]
            colscan_reduce_kernel<<<nchunks, scan_threads, 0, st>>>(hist, (int)ntiles, nb, partial);
            SOAX_TRY(launched());
            colscan_top_kernel<<<1, scan_threads, 0, st>>>(partial, (int)nchunks, nb, dbase);
            SOAX_TRY(launched());
            colscan_apply_kernel<<<nchunks, scan_threads, 0, st>>>(hist, (int)ntiles, nb, partial, dbase);
            SOAX_TRY(launched());
            if (g_tune.bin_stage == 2) {
                if (pass == 0) scatter_ring_kernel<L, false><<<ntiles, kSortThreads, kRingSmem, st>>>(from, to, kin, kout, iin, iout, hist, n, shift, mask);
                else scatter_ring_kernel<L, true><<<ntiles, kSortThreads, kRingSmem, st>>>(from, to, kin, kout, iin, iout, hist, n, shift, mask);
            } else if (g_tune.bin_stage == 1)
                scatter_staged_kernel<L><<<ntiles, kSortThreads, 0, st>>>(from, to, kin, kout, iin, iout, hist, n, shift, mask);
            else
                scatter_kernel<L><<<ntiles, kSortThreads, 0, st>>>(from, to, kin, kout, iin, iout, hist, n, shift, mask);
            SOAX_TRY(launched());
            shift += w;
        }
        if (a.counts || a.offsets) {
            const uint32_t* sorted = keys[npass & 1];
            boundaries_kernel<<<kSMs * 8, 256, 0, st>>>(sorted, n, ncell, off);
            SOAX_TRY(launched());
            counts_kernel<<<(ncell + 255) / 256, 256, 0, st>>>(off, ncell, a.counts, a.offsets);
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
