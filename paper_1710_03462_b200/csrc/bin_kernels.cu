// bin_kernels.cu -- a10..a14: PIC-style cell binning with a STABLE counting-sort permutation of every field
// array (BASELINE.json config 5).
//
// Design.  The 3*log2(G)-bit cell key is sorted by a least-significant-digit counting sort whose
// digits are as wide as 9 bits (G = 64: 18 bits = TWO passes of 512 bins), and the WHOLE RECORD travels with its key
// through the passes together with its source index, so `perm` falls out as the carried index and no random gather
// of the field arrays is ever made (a per-array gather would read one 32-byte sector per 4- or 8-byte item).
//   cell_hist   [drift +] cell index [+ kinetic energy] and the first digit's per-tile histogram     36 B read, 4 B written
//   colscan_*   exclusive scan of the [tile][digit] table in digit-major order                      (small)
//   scatter     every UNIT of the tile (the key + carried index, each 8-byte component, each PAIR of 4-byte components)
//               arrives in shared memory by bulk asynchronous copy (TMA) into a 3-stage ring; stable in-tile ranks come
//               from warp ballots and per-warp running counters; output slot j reads ring[inv[j]] and writes its global
//               slot, consecutive threads writing consecutive slots of a bin's run.  Between the passes the records live
//               in a PAIRED scratch format (4-byte arrays two by two as 8-byte elements: 6 streams instead of 9 for R1);
//               the first pass reads the caller's SoA and applies the requested DRIFT to the positions on their way
//               through the ring (src is never written), the last pass writes the caller's SoA.
//   tile_hist   per-tile histogram of the next digit (later passes)                                  4 B read
//   cell_bounds counts / offsets from the sorted positions by binary search per cell                 (small)
// A 512-bin pass leaves runs of only ~8 elements per tile and bin, whose ragged ends are partial 32-byte sectors.  The L2
// keeps a partly written sector until its other half arrives only while FEW are open (a few MB; an unsynchronised pass holds
// ~1.8 M of them open and pays a DRAM read-modify-write for most), and DRAM reaches its copy rate only for contiguous pieces
// of 256 bytes and more (both measured: profiles/r2_mem_probes.md).  Wide-digit passes are therefore launched in THREAD-BLOCK
// CLUSTERS of 4 CTAs that own neighbouring tiles and meet at a cluster barrier before every array's stores: the four pieces
// of a bin's run reach the L2 together, merge into full sectors, and leave for DRAM as one 256-byte piece.
// Every step is a pure function of the data (no arrival-order atomics decide a position), so the result is the
// unique stable permutation for ANY particle distribution, and bit-identical from run to run.
#include <cstdio>
#include <cstdlib>
#include <type_traits>
#include <vector>

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
// `stride` = 1: plain keys; 2: the (key, index) pairs of the paired format (the key is the first word of each pair).
__global__ void __launch_bounds__(kSortThreads) tile_hist_kernel(const uint32_t* __restrict__ keys, int stride, int64_t n, int shift, uint32_t mask,
                                                                 uint32_t* __restrict__ hist) {
    __shared__ uint32_t h[kRadix];
    for (int i = threadIdx.x; i < kRadix; i += kSortThreads) h[i] = 0;
    __syncthreads();
    const int64_t tile0 = (int64_t)blockIdx.x * kTileN;
    if (tile0 + kTileN <= n && stride == 1) {  // full tile: two 128-bit loads per thread (the histogram does not care about order)
        const uint4* k4 = reinterpret_cast<const uint4*>(keys + tile0);
        const uint4 a = k4[threadIdx.x], b = k4[threadIdx.x + kSortThreads];
        const uint32_t w[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
#pragma unroll
        for (int k = 0; k < 8; ++k) atomicAdd(&h[(w[k] >> shift) & mask], 1u);
    } else if (tile0 + kTileN <= n) {  // full tile of pairs: four 128-bit loads per thread, the keys are words 0 and 2
        const uint4* k4 = reinterpret_cast<const uint4*>(keys + 2 * tile0);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const uint4 a = k4[threadIdx.x + q * kSortThreads];
            atomicAdd(&h[(a.x >> shift) & mask], 1u);
            atomicAdd(&h[(a.z >> shift) & mask], 1u);
        }
    } else {
#pragma unroll
        for (int k = 0; k < kItems; ++k) {
            const int64_t e = tile0 + k * kSortThreads + threadIdx.x;
            if (e < n) atomicAdd(&h[(keys[e * stride] >> shift) & mask], 1u);
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i <= (int)mask; i += kSortThreads) hist[(int64_t)blockIdx.x * (mask + 1) + i] = h[i];  // row of mask+1 bins
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

// ---- units: what moves through the ring as ONE element stream ---------------------------------------------------------------
// Between the passes the records live in a PAIRED format of this file's own choosing: 4-byte arrays travel two by two as
// 8-byte elements -- (key, carried source index), and the 4-byte components in declaration order, e.g. R1: (id, vel0),
// (vel1, vel2) -- so that a tile of R1 is 6 element streams instead of 9: a third fewer array moves (each costs a dozen
// barriers) and a third fewer ragged run ends.  Unit 0 is the key [+ index]; a unit is a single component (any size) or a
// pair of 4-byte components.  The first pass reads plain SoA (a pair = two bulk copies into the two halves of a stage) and
// the last pass writes plain SoA (a pair = two 4-byte stores), so the format never leaves the scratch buffer.
template <class L, bool HAS_IDX>
struct Units {
    static constexpr int kMax = 1 + L::ncomp;
    int n = 1;
    int a[kMax] = {}, b[kMax] = {}, bytes[kMax] = {};       // components of the unit (b = -1: single), element bytes when paired
    int unit_of[L::ncomp > 0 ? L::ncomp : 1] = {}, half_of[L::ncomp > 0 ? L::ncomp : 1] = {};
    constexpr Units() {
        a[0] = b[0] = -1;
        bytes[0] = HAS_IDX ? 8 : 4;
        int open = -1;  // a 4-byte single still waiting for a partner
        for (int c = 0; c < L::ncomp; ++c) {
            if (L::comp_size(c) == 4 && open >= 0) {
                b[open] = c; bytes[open] = 8; unit_of[c] = open; half_of[c] = 1; open = -1;
            } else {
                const int u = n++;
                a[u] = c; b[u] = -1; bytes[u] = L::comp_size(c); unit_of[c] = u; half_of[c] = 0;
                if (L::comp_size(c) == 4) open = u;
            }
        }
    }
};

// ---- the order in which the units of a tile pass through the 3-stage ring, fixed at compile time ---------------------------
// Units are LOADED in `load` order and MOVED (written to their destination) in `move` order; the two differ only under DRIFT,
// where the position component c needs the unit that holds the velocity component c in shared memory at the same time: that
// unit is loaded before pos_c and moved after the last position component that needs it.  Load k >= 3 goes into the stage
// freed by move k - 3; the constructor checks that every unit a move needs has been requested by then.
constexpr int kRingStages = 3;

// Study builds (-DSOAX_SCATTER_TRACE, see build.py): thread 0 of every CTA stamps the phases of its tile with %globaltimer; with
// SOAX_TRACE=<prefix> in the environment the first launches of the scatter write <prefix>_<n>.bin ([CTA][64] uint64 nanoseconds).
// Compiled out of the shipped library.
#ifdef SOAX_SCATTER_TRACE
__device__ unsigned long long* g_trace = nullptr;
#define TR(i) do { if (g_trace && threadIdx.x == 0) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); g_trace[(size_t)blockIdx.x * 64 + (i)] = t_; } } while (0)
#else
#define TR(i) do { } while (0)
#endif
template <class L, bool HAS_IDX, bool DRIFT>
struct RingPlan {
    using U = Units<L, HAS_IDX>;
    static constexpr int kMaxUnits = U::kMax;
    int nu = 0;
    int load[kMaxUnits] = {}, move[kMaxUnits] = {}, stage[kMaxUnits] = {}, parity[kMaxUnits] = {};
    int partner[kMaxUnits] = {}, partner_half[kMaxUnits] = {};  // by unit: the unit (and half) holding the velocity of a position unit
    bool ok = true;
    constexpr RingPlan() {
        constexpr U units{};
        nu = units.n;
        int nl = 0, nm = 0;
        bool loaded[kMaxUnits] = {}, moved[kMaxUnits] = {};
        for (int u = 0; u < kMaxUnits; ++u) partner[u] = -1;
        load[nl++] = 0; move[nm++] = 0; loaded[0] = moved[0] = true;
        if constexpr (DRIFT) {
            constexpr int P0 = L::template begin_of<pos_tag>, V0 = L::template begin_of<vel_tag>;
            for (int c = 0; c < 3; ++c) {
                const int up = units.unit_of[P0 + c], uv = units.unit_of[V0 + c];
                partner[up] = uv; partner_half[up] = units.half_of[V0 + c];
                if (!loaded[uv]) { load[nl++] = uv; loaded[uv] = true; }
                load[nl++] = up; loaded[up] = true;
                move[nm++] = up; moved[up] = true;
                bool needed_later = false;
                for (int c2 = c + 1; c2 < 3; ++c2) needed_later |= units.unit_of[V0 + c2] == uv;
                if (!needed_later && !moved[uv]) { move[nm++] = uv; moved[uv] = true; }
            }
        }
        for (int u = 1; u < nu; ++u) {
            if (!loaded[u]) load[nl++] = u;
            if (!moved[u]) move[nm++] = u;
        }
        int uses[kRingStages] = {}, load_index[kMaxUnits] = {};
        for (int k = 0; k < nu; ++k) {
            const int s = k < kRingStages ? k : stage[move[k - kRingStages]];
            stage[load[k]] = s;
            parity[load[k]] = uses[s] & 1;
            load_index[load[k]] = k;
            ++uses[s];
        }
        for (int m = 0; m < nu; ++m) {  // everything move m reads was requested no later than after move m - 1
            const int u = move[m];
            ok &= load_index[u] <= m + kRingStages - 1;
            if (partner[u] >= 0) {
                ok &= load_index[partner[u]] <= m + kRingStages - 1;
                bool partner_still_there = true;  // the partner's stage is freed by the partner's own move, which must come later
                for (int m2 = 0; m2 < m; ++m2) partner_still_there &= move[m2] != partner[u];
                ok &= partner_still_there;
            }
        }
    }
};

// Time-synchronisation of the CTAs of a thread-block cluster (no memory ordering needed: it only makes the CTAs that
// own neighbouring tiles write the pieces of a bin's run at the same moment, so that the L2 merges them into full sectors
// while few partly written sectors are open: profiles/r2_mem_probes.md).
__device__ __forceinline__ void cluster_sync_relaxed() {
    asm volatile("barrier.cluster.arrive.relaxed.aligned;\n\tbarrier.cluster.wait.aligned;" ::: "memory");
}

// Pacing of the scatter stores (measured, profiles/r2_bin_study.md): a thread has kItems stores per unit; issued back to
// back they reach the L2 out of step with the stores of the neighbouring CTAs that complete the same sectors.  Between
// two stores of a thread the CTA (pace_sync 1) or the whole cluster (2, the default with clusters) therefore meets at a
// barrier, so that at any moment the cluster writes ONE window of ~64 neighbouring bins; a sleep of a few tens of
// nanoseconds can be added for studies.
__device__ __forceinline__ void pace(int k, int pace_sync, int pace_ns, int pace_every = 1) {
    if (k == 0 || (k % pace_every) != 0) return;
    if (pace_sync == 1) __syncthreads();
    if (pace_sync == 2) cluster_sync_relaxed();
    if (pace_ns) __nanosleep(pace_ns);
}

// ---- stable scatter of one tile through the TMA ring ----------------------------------------------------------------
// 64 registers/thread and ~106 KB of shared memory let two CTAs share an SM: one ranks while the other streams.
constexpr int kStageBytes = kTileN * 8;  // one unit of the tile at 8 bytes per element
constexpr int kRingSmem = kRingStages * kStageBytes + kTileN * 2 /*inv*/ + kRadix * 4 /*delta*/ + 32 * 4 /*scan*/ + 64 /*mbarriers*/;
static_assert(kWarps * kRadix * 4 <= kStageBytes, "the per-warp counters alias ring stage 1");

template <int N>
struct UnitPtrs {
    void* p[N];
};

struct ScatterArgs {
    const uint32_t* key_in;   // IN = SoA (first pass): the cell keys made by cell_hist_kernel
    uint32_t* idx_out;        // OUT = SoA (last pass): the permutation (HAS_IDX)
    const uint32_t* base;     // [tile][nb] global slot of the first item of (digit, tile)
    int64_t n; int shift; uint32_t mask; int nbits; int ntiles; int csync; double dt; int pace_sync, pace_ns, pace_every;
};

// IN_PAIRED / OUT_PAIRED: the format on either side (false = plain SoA: src in the first pass, dst in the last).
template <class L, bool HAS_IDX, bool IN_PAIRED, bool OUT_PAIRED, bool DRIFT>
__global__ void __launch_bounds__(kSortThreads, 1024 / kSortThreads)
scatter_ring_kernel(Ptrs<L::ncomp> soa_in, Ptrs<L::ncomp> soa_out, UnitPtrs<1 + L::ncomp> pin, UnitPtrs<1 + L::ncomp> pout, ScatterArgs g) {
    static_assert(!(DRIFT && IN_PAIRED), "the drift is applied in the first pass, which reads the caller's SoA");
    using Plan = RingPlan<L, HAS_IDX, DRIFT>;
    constexpr Plan plan{};
    constexpr Units<L, HAS_IDX> units{};
    static_assert(plan.ok, "the ring plan does not keep a velocity unit resident while its position component moves");
    constexpr int kUnits = units.n;
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

    TR(0);
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kRingStages; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    // copy(stage, byte offset in the stage, global array, element bytes): bring `cnt` elements of one array into a ring stage.
    // Called by ALL threads at CTA-uniform points, after a __syncthreads() that retired every reader of the stage.
    auto copy = [&](int stage, int at, const void* gp, int esize) {
        unsigned char* sb = ring + stage * kStageBytes + at;
        const unsigned char* gb = static_cast<const unsigned char*>(gp) + tile0 * esize;
        if (bulk) {
            if (tid == 0) bulk_g2s(sb, gb, (uint32_t)(kTileN * esize), &full[stage]);
        } else if (esize == 8) {
            for (int i = tid; i < cnt; i += kSortThreads) reinterpret_cast<uint64_t*>(sb)[i] = reinterpret_cast<const uint64_t*>(gb)[i];
        } else if (esize == 4) {
            for (int i = tid; i < cnt; i += kSortThreads) reinterpret_cast<uint32_t*>(sb)[i] = reinterpret_cast<const uint32_t*>(gb)[i];
        } else {
            for (int i = tid; i < cnt * esize; i += kSortThreads) sb[i] = gb[i];
        }
    };
    // ready(stage, parity): the unit requested by the matching fill is in shared memory
    auto ready = [&](int stage, uint32_t parity) {
        if (bulk) mbar_wait(&full[stage], parity);
        else __syncthreads();
    };
    // fill_load<k>(): issue the k-th load of the plan (nothing if the plan has fewer units)
    auto fill_load = [&](auto ki) {
        constexpr int k = decltype(ki)::value;
        if constexpr (k < kUnits) {
            constexpr int u = plan.load[k];
            constexpr int st = plan.stage[u];
            constexpr int ua = units.a[u], ub = units.b[u], ubytes = units.bytes[u];  // (constant-evaluated: `units` is not captured)
            if constexpr (IN_PAIRED) {
                if (bulk && tid == 0) mbar_expect_tx(&full[st], (uint32_t)(kTileN * ubytes));
                copy(st, 0, pin.p[u], ubytes);
            } else if constexpr (u == 0) {
                if (bulk && tid == 0) mbar_expect_tx(&full[st], (uint32_t)(kTileN * 4));
                copy(st, 0, g.key_in, 4);
            } else if constexpr (ub < 0) {
                if (bulk && tid == 0) mbar_expect_tx(&full[st], (uint32_t)(kTileN * ubytes));
                copy(st, 0, soa_in.p[ua], ubytes);
            } else {  // a pair read from plain SoA: two copies into the two halves of the stage
                if (bulk && tid == 0) mbar_expect_tx(&full[st], (uint32_t)(kTileN * 8));
                copy(st, 0, soa_in.p[ua], 4);
                copy(st, kTileN * 4, soa_in.p[ub], 4);
            }
        }
    };
    // halves of a pair unit in its stage: interleaved (lo, hi) when it arrived paired, two half-stages when it came from SoA
    auto pair_at = [&](const unsigned char* sb, uint32_t s) -> uint2 {
        if constexpr (IN_PAIRED) return reinterpret_cast<const uint2*>(sb)[s];
        else return make_uint2(reinterpret_cast<const uint32_t*>(sb)[s], reinterpret_cast<const uint32_t*>(sb)[kTileN + s]);
    };
    constexpr bool kKeyIsPair = IN_PAIRED && HAS_IDX;  // unit 0 in shared memory: (key, idx) pairs, else plain keys
    auto key_at = [&](uint32_t e) -> uint32_t {
        if constexpr (kKeyIsPair) return reinterpret_cast<const uint2*>(ring)[e].x;
        else return reinterpret_cast<const uint32_t*>(ring)[e];
    };
    static_assert(plan.load[0] == 0 && plan.move[0] == 0 && plan.stage[0] == 0, "the keys lead");
    // Stage 1 is the counters for now, so start with loads 0 and 2 -- at once: thread 0 has initialised the barriers it arms
    // (program order + the init fence), and the latency of the keys' copy hides behind the set-up below.
    fill_load(std::integral_constant<int, 0>{});
    fill_load(std::integral_constant<int, 2>{});
    for (int i = tid; i < kWarps * kRadix; i += kSortThreads) wcnt[i] = 0;
    constexpr int kBinsPerThread = kRadix / kSortThreads > 0 ? kRadix / kSortThreads : 1;  // thread t owns bins [t B, t B + B)
    uint32_t my_base[kBinsPerThread];  // consumed after the ranking
#pragma unroll
    for (int i = 0; i < kBinsPerThread; ++i) {
        const int b = tid * kBinsPerThread + i;
        my_base[i] = (b <= (int)mask && (int)blockIdx.x < g.ntiles ? g.base[(int64_t)blockIdx.x * (mask + 1) + b] : 0u);
    }
    __syncthreads();  // barriers initialised, counters zeroed

    // ---- ranking: warp w owns elements [256 w, 256 w + 256) of the tile, 8 rounds of 32 in element order -------
    TR(1);
    ready(0, 0);
    TR(2);
    const int e0 = warp * (32 * kItems) + lane;
    uint32_t lpos[kItems];
    uint32_t* mycnt = wcnt + warp * kRadix;
    const uint32_t lt = (1u << lane) - 1u;
    uint32_t peers[kItems];
#pragma unroll
    for (int k = 0; k < kItems; ++k) {  // lanes holding the same digit, from one ballot per digit bit (MATCH costs twice as much; an atomicOr into a per-warp mask table the same: profiles/r2_scatter_trace.md)
        const int e = e0 + k * 32;
        const bool valid = e < cnt;
        const uint32_t d = valid ? (key_at(e) >> shift) & mask : 0u;
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
    TR(40);
#pragma unroll
    for (int k = 0; k < kItems; ++k) {
        const uint32_t d = lpos[k];
        const uint32_t old = mycnt[d];
        lpos[k] = old + __popc(peers[k] & lt);
        __syncwarp();
        if (peers[k] != 0u && lane == 31 - __clz(peers[k])) mycnt[d] = old + __popc(peers[k]);
        __syncwarp();
    }
    TR(41);
    __syncthreads();
    TR(42);
    {   // bins of this thread: tile totals -> first slot of each bin in tile-sorted order -> per-warp first slots
        uint32_t tot[kBinsPerThread], sum = 0;
#pragma unroll
        for (int i = 0; i < kBinsPerThread; ++i) {
            const int b = tid * kBinsPerThread + i;
            tot[i] = 0;
            if (b < kRadix) {
#pragma unroll
                for (int w = 0; w < kWarps; ++w) tot[i] += wcnt[w * kRadix + b];
            }
            sum += tot[i];
        }
        uint32_t run = block_excl_scan(sum, scan_sm);
#pragma unroll
        for (int i = 0; i < kBinsPerThread; ++i) {
            const int b = tid * kBinsPerThread + i;
            if (b < kRadix) {
                delta[b] = my_base[i] - run;
#pragma unroll
                for (int w = 0; w < kWarps; ++w) {
                    const uint32_t c = wcnt[w * kRadix + b];
                    wcnt[w * kRadix + b] = run;
                    run += c;
                }
            }
        }
    }
    TR(43);
    __syncthreads();
    TR(44);
#pragma unroll
    for (int k = 0; k < kItems; ++k) {
        const int e = e0 + k * 32;
        if (e < cnt) inv[lpos[k] + mycnt[(key_at(e) >> shift) & mask]] = (uint16_t)e;
    }
    TR(45);
    fence_async_smem();  // the counters (generic-proxy writes) are about to be overwritten by a bulk copy
    __syncthreads();     // inv complete, counters dead: stage 1 joins the ring
    fill_load(std::integral_constant<int, 1>{});
    TR(3);

    // ---- output slots: thread t owns slots t, t + 512, ... of the tile-sorted order, so that in its k-th store the whole CTA
    // (and, in step with it, the other CTAs of the cluster) writes ONE window of 512 consecutive slots = the runs of ~64
    // neighbouring bins.  Few runs open at a time is what lets the L2 merge their pieces: giving every warp its own 256
    // consecutive slots instead (16 windows open per CTA) was measured 25 % slower (profiles/r2_bin_study.md).
#define SLOT(k) (tid + (k) * kSortThreads)
#define SRC(k) ((srcp[(k) >> 1] >> (((k) & 1) * 16)) & 0xffffu)
    uint32_t gdest[kItems], srcp[kItems / 2];  // source elements packed two per register
    {   // unit 0: the key [and the source index: generated in the first pass, carried afterwards]
        uint32_t kv[kItems], iv[kItems];
#pragma unroll
        for (int k = 0; k < kItems; ++k) {
            const int j = SLOT(k);
            uint32_t s = 0;
            kv[k] = iv[k] = gdest[k] = 0;
            if (j < cnt) {
                s = inv[j];
                if constexpr (kKeyIsPair) {
                    const uint2 p = reinterpret_cast<const uint2*>(ring)[s];
                    kv[k] = p.x; iv[k] = p.y;
                } else {
                    kv[k] = key_at(s);
                    iv[k] = (uint32_t)(tile0 + s);
                }
                gdest[k] = delta[(kv[k] >> shift) & mask] + (uint32_t)j;
            }
            if (k & 1) srcp[k >> 1] |= s << 16; else srcp[k >> 1] = s;
        }
        TR(4);
        if (g.csync) cluster_sync_relaxed();
        TR(5);
        // The stores come BEFORE the barrier on purpose: they consume the loaded values, so every shared-memory read of this
        // stage has completed when its thread arrives.  A barrier alone does not order reads that are still in flight in the
        // generic proxy against the bulk copy (async proxy) that refills the stage.
        if constexpr (OUT_PAIRED) {
#pragma unroll
            for (int k = 0; k < kItems; ++k) {
                pace(k, g.pace_sync, g.pace_ns, g.pace_every);
                if (SLOT(k) < cnt) {
                    if constexpr (HAS_IDX) static_cast<uint2*>(pout.p[0])[gdest[k]] = make_uint2(kv[k], iv[k]);
                    else static_cast<uint32_t*>(pout.p[0])[gdest[k]] = kv[k];
                }
            }
        } else {
            if constexpr (HAS_IDX) {  // the last pass writes no keys: counts / offsets come from the sorted positions
#pragma unroll
                for (int k = 0; k < kItems; ++k) {
                    pace(k, g.pace_sync, g.pace_ns, g.pace_every);
                    if (SLOT(k) < cnt) g.idx_out[gdest[k]] = iv[k];
                }
            }
        }
    }
    TR(6);
    __syncthreads();  // the keys have been read: stage 0 is free
    TR(7);
    fill_load(std::integral_constant<int, kRingStages>{});

    // move<m>(): write the m-th unit of the move order to its destination, then refill its stage with load m + 3
    auto move = [&](auto mi) {
        constexpr int m = decltype(mi)::value;
        constexpr int u = plan.move[m];
        constexpr int p = plan.partner[u];
        constexpr int ca = units.a[u] >= 0 ? units.a[u] : 0, cb = units.b[u] >= 0 ? units.b[u] : 0;
        constexpr bool is_pair = units.b[u] >= 0;
        constexpr int st = plan.stage[u], par = plan.parity[u];
        TR(8 + 6 * (m - 1) + 0);
        ready(st, par);
        TR(8 + 6 * (m - 1) + 1);
        const unsigned char* sb = ring + st * kStageBytes;
        if constexpr (is_pair) {  // a pair of 4-byte components
            uint2 v[kItems];
#pragma unroll
            for (int k = 0; k < kItems; ++k)
                if (SLOT(k) < cnt) v[k] = pair_at(sb, SRC(k));
            TR(8 + 6 * (m - 1) + 2);
            if (g.csync) cluster_sync_relaxed();
            TR(8 + 6 * (m - 1) + 3);
#pragma unroll
            for (int k = 0; k < kItems; ++k) {
                pace(k, g.pace_sync, g.pace_ns, g.pace_every);
                if (SLOT(k) < cnt) {
                    if constexpr (OUT_PAIRED) {
                        static_cast<uint2*>(pout.p[u])[gdest[k]] = v[k];
                    } else {
                        static_cast<uint32_t*>(soa_out.p[ca])[gdest[k]] = v[k].x;
                        static_cast<uint32_t*>(soa_out.p[cb])[gdest[k]] = v[k].y;
                    }
                    (void)cb;
                }
            }
        } else {
            using T = typename L::template comp_type<ca>;
            const T* tb = reinterpret_cast<const T*>(sb);
            T v[kItems];
            if constexpr (p >= 0) {  // DRIFT: a position component; its velocity component sits in another unit's stage
                constexpr int pu = p >= 0 ? p : 0;
                constexpr int pst = plan.stage[pu], ppar = plan.parity[pu];
                constexpr int voff = units.b[pu] >= 0 ? plan.partner_half[u] * kTileN : 0;  // second half of a pair's stage
                using V = typename L::template type_of<vel_tag>;
                ready(pst, ppar);
                const V* vb = reinterpret_cast<const V*>(ring + pst * kStageBytes) + voff;
#pragma unroll
                for (int k = 0; k < kItems; ++k) {
                    const uint32_t s = SRC(k);
                    if (SLOT(k) < cnt) v[k] = drift1<V>(g.dt, vb[s], tb[s]);
                }
            } else {
#pragma unroll
                for (int k = 0; k < kItems; ++k)
                    if (SLOT(k) < cnt) v[k] = tb[SRC(k)];
            }
            TR(8 + 6 * (m - 1) + 2);
            if (g.csync) cluster_sync_relaxed();
            TR(8 + 6 * (m - 1) + 3);
            T* gout = OUT_PAIRED ? static_cast<T*>(pout.p[u]) : static_cast<T*>(soa_out.p[ca]);
#pragma unroll
            for (int k = 0; k < kItems; ++k) {
                pace(k, g.pace_sync, g.pace_ns, g.pace_every);
                if (SLOT(k) < cnt) gout[gdest[k]] = v[k];
            }
        }
        TR(8 + 6 * (m - 1) + 4);
        __syncthreads();  // every read of the stage has been consumed by a store: it can take the next load
        TR(8 + 6 * (m - 1) + 5);
        fill_load(std::integral_constant<int, m + kRingStages>{});
    };
    for_each_int<kUnits - 1>([&](auto i) { move(std::integral_constant<int, decltype(i)::value + 1>{}); });
#undef SLOT
#undef SRC
}

// ---- counts / offsets from the SORTED POSITIONS: off[c] = first slot of dst whose cell is >= c (binary search) -------------
// The last pass writes no key array at all: the cell of a sorted particle is recomputed from its (drifted) position, which
// is exact (a10 is a pure function of the position).  262 144 cells x 27 probes x 3 loads: far cheaper than writing and
// re-reading 4 bytes per particle.
__global__ void __launch_bounds__(256) cell_bounds_kernel(const double* __restrict__ x0, const double* __restrict__ x1, const double* __restrict__ x2,
                                                          int64_t n, int log2g, uint32_t* __restrict__ counts, uint32_t* __restrict__ offsets) {
    __shared__ uint32_t off[257];
    const uint32_t ncell = 1u << (3 * log2g);
    const double G = (double)(1 << log2g);
    const int gmax = (1 << log2g) - 1;
    auto lower_bound = [&](uint32_t c) {
        int64_t lo = 0, hi = n;
        while (lo < hi) {
            const int64_t mid = (lo + hi) >> 1;
            if (cell_of(x0[mid], x1[mid], x2[mid], G, gmax, log2g) < c) lo = mid + 1; else hi = mid;
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

// Scratch: the cell keys made by cell_hist_kernel, one buffer in the
// PAIRED format per intermediate result that is alive at a time (one for two passes, two to ping-pong between for more),
// and the small tables.  The unit arrays are sized for the units WITH a carried index (the larger of the two unit lists).
// IN PLACE (soax_bin_permute_inplace, two passes): the sorted set returns to src and the second container is only a work
// area, so the intermediate's 8-byte single units live in the work container's own component arrays and its first 4-byte
// array holds the cell keys; only unit 0 (key, carried index) and the PAIRS of 4-byte components need scratch.
template <class L>
constexpr bool unit_in_work(int u) {  // in-place: does unit u of the intermediate live in the work container?
    constexpr Units<L, true> units{};
    return u >= 1 && u < units.n && units.b[u] < 0 && units.bytes[u] == 8;
}
template <class L>
constexpr int key_comp_in_work() {  // in-place: the work container's array that holds the cell keys (-1: scratch)
    for (int c = 0; c < L::ncomp; ++c)
        if (L::comp_size(c) == 4) return c;
    return -1;
}
template <class L>
struct BinPlan {
    static constexpr int kU = 1 + L::ncomp;
    size_t key0, hist, partial, dbase, ke, total;
    size_t unit_off[2][kU];
    int64_t ntiles, nchunks;
    BinPlan(int64_t n, int npass, bool inplace) {
        constexpr Units<L, true> units{};
        ntiles = (n + kTileN - 1) / kTileN;
        if (ntiles < 1) ntiles = 1;
        nchunks = (ntiles + kScanRows - 1) / kScanRows;
        size_t o = 0;
        auto take = [&](size_t bytes) { size_t at = o; o += align_up(bytes ? bytes : 1, kAlign); return at; };
        // with two or more passes the keys live in dst (see bin_permute_entry); in place: in the work container's first 4-byte array
        key0 = take((inplace ? key_comp_in_work<L>() >= 0 : npass >= 2) ? 0 : (size_t)n * 4);
        for (int b = 0; b < 2; ++b)
            for (int u = 0; u < kU; ++u) {
                bool here = b < npass - 1 && u < units.n;
                if (inplace) here = here && !unit_in_work<L>(u);
                unit_off[b][u] = take(here ? (size_t)n * units.bytes[u] : 0);
            }
        hist = take((size_t)ntiles * kRadix * 4);
        partial = take((size_t)nchunks * kRadix * 4);
        dbase = take(kRadix * 4);
        ke = take((size_t)ntiles * sizeof(double));
        total = o;
    }
};

template <class L>
size_t bin_scratch_bytes(int64_t n, int log2g, bool inplace) {
    if constexpr (!L::template has_as<pos_tag, double, 3>()) return 0;
    else {
        const int npass = PassPlan(log2g, g_tune.bin_bits).npass;
        if (inplace && npass != 2) return 0;
        return BinPlan<L>(n, npass, inplace).total;
    }
}

template <class L, bool HAS_IDX, bool IN_PAIRED, bool OUT_PAIRED, bool DRIFT>
int launch_scatter(int cluster, unsigned ntiles, cudaStream_t st, const Ptrs<L::ncomp>& soa_in, const Ptrs<L::ncomp>& soa_out,
                   const UnitPtrs<1 + L::ncomp>& pin, const UnitPtrs<1 + L::ncomp>& pout, const ScatterArgs& g) {
    auto kernel = scatter_ring_kernel<L, HAS_IDX, IN_PAIRED, OUT_PAIRED, DRIFT>;
    // The function attributes are per device: set them on every call (cheap) rather than once per process.
    SOAX_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kRingSmem));
    SOAX_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
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
#ifdef SOAX_SCATTER_TRACE
    static int trace_no = 0;  // per instantiation: <prefix>_<in paired><out paired>_<n>.bin
    const char* tp = getenv("SOAX_TRACE");
    if (tp && (trace_no >= 2 || 1 + L::ncomp > 9)) tp = nullptr;  // trace slots exist for up to 8 moves
    unsigned long long* tbuf = nullptr;
    if (tp) {
        SOAX_CUDA(cudaMalloc(&tbuf, (size_t)cfg.gridDim.x * 64 * 8));
        SOAX_CUDA(cudaMemset(tbuf, 0, (size_t)cfg.gridDim.x * 64 * 8));
        SOAX_CUDA(cudaMemcpyToSymbol(g_trace, &tbuf, sizeof(tbuf)));
    }
#endif
    SOAX_CUDA(cudaLaunchKernelEx(&cfg, kernel, soa_in, soa_out, pin, pout, g));
#ifdef SOAX_SCATTER_TRACE
    if (tp) {
        SOAX_CUDA(cudaDeviceSynchronize());
        std::vector<unsigned long long> h((size_t)cfg.gridDim.x * 64);
        SOAX_CUDA(cudaMemcpy(h.data(), tbuf, h.size() * 8, cudaMemcpyDeviceToHost));
        char name[512];
        std::snprintf(name, sizeof name, "%s_%d%d_%d.bin", tp, (int)IN_PAIRED, (int)OUT_PAIRED, trace_no++);
        if (FILE* f = std::fopen(name, "wb")) {
            std::fwrite(h.data(), 8, h.size(), f);
            std::fclose(f);
        }
        SOAX_CUDA(cudaFree(tbuf));
        tbuf = nullptr;
        SOAX_CUDA(cudaMemcpyToSymbol(g_trace, &tbuf, sizeof(tbuf)));
    }
#endif
    return launched();
}

// one pass: the format on either side follows from its position; the drift belongs to the first pass
template <class L, bool HAS_IDX>
int scatter_pass(bool first, bool last, bool drift, int cluster, unsigned ntiles, cudaStream_t st, const Ptrs<L::ncomp>& src,
                 const Ptrs<L::ncomp>& dst, const UnitPtrs<1 + L::ncomp>& pin, const UnitPtrs<1 + L::ncomp>& pout, const ScatterArgs& g) {
    constexpr bool has_vel = L::template has_as<vel_tag, float, 3>() || L::template has_as<vel_tag, double, 3>();
    if (first && last) {
        if constexpr (has_vel) { if (drift) return launch_scatter<L, HAS_IDX, false, false, true>(cluster, ntiles, st, src, dst, pin, pout, g); }
        return launch_scatter<L, HAS_IDX, false, false, false>(cluster, ntiles, st, src, dst, pin, pout, g);
    }
    if (first) {
        if constexpr (has_vel) { if (drift) return launch_scatter<L, HAS_IDX, false, true, true>(cluster, ntiles, st, src, dst, pin, pout, g); }
        return launch_scatter<L, HAS_IDX, false, true, false>(cluster, ntiles, st, src, dst, pin, pout, g);
    }
    if (last) return launch_scatter<L, HAS_IDX, true, false, false>(cluster, ntiles, st, src, dst, pin, pout, g);
    return launch_scatter<L, HAS_IDX, true, true, false>(cluster, ntiles, st, src, dst, pin, pout, g);
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
        if (a.inplace && npass != 2) return SOAX_ERR_UNSUPPORTED;  // the set returns to src after an even number of passes
        const BinPlan<L> plan(n, npass, a.inplace);
        if (a.scratch_bytes < plan.total) return SOAX_ERR_ALLOC;
        char* sc = static_cast<char*>(a.scratch);
        // The cell keys are dead once the first pass has read them, and dst is not written before the last pass: with two
        // or more passes the keys live in dst's own memory (its first component array of >= 4 bytes per element).  In place
        // dst is the work container, whose 8-byte arrays hold intermediate units: the keys take its first 4-byte array.
        uint32_t* key0 = reinterpret_cast<uint32_t*>(sc + plan.key0);
        if (a.inplace) {
            if constexpr (key_comp_in_work<L>() >= 0) key0 = static_cast<uint32_t*>(a.dst[key_comp_in_work<L>()]);
        } else if (npass >= 2) {
            for (int c = 0; c < L::ncomp; ++c)
                if (L::comp_size(c) >= 4) { key0 = static_cast<uint32_t*>(a.dst[c]); break; }
        }
        uint32_t* hist = reinterpret_cast<uint32_t*>(sc + plan.hist);
        uint32_t* partial = reinterpret_cast<uint32_t*>(sc + plan.partial);
        uint32_t* dbase = reinterpret_cast<uint32_t*>(sc + plan.dbase);
        double* kep = reinterpret_cast<double*>(sc + plan.ke);
        // in place the last pass writes the caller's src again (nothing reads src after the first pass)
        const Ptrs<L::ncomp> src = make_ptrs<L>(a.src), dst = make_ptrs<L>(a.inplace ? a.src : a.dst);
        UnitPtrs<1 + L::ncomp> buf[2];
        for (int b = 0; b < 2; ++b)
            for (int u = 0; u < 1 + L::ncomp; ++u) buf[b].p[u] = sc + plan.unit_off[b][u];
        if (a.inplace) {
            constexpr Units<L, true> units{};
            for_each_int<1 + L::ncomp>([&](auto ui) {
                constexpr int u = decltype(ui)::value;
                if constexpr (unit_in_work<L>(u)) buf[0].p[u] = a.dst[units.a[u]];
            });
        }
        const unsigned ntiles = (unsigned)plan.ntiles, nchunks = (unsigned)plan.nchunks;
        const bool has_idx = a.perm != nullptr;

        // Least-significant-digit passes over the 3*log2g key bits.
        int shift = 0;
        for (int pass = 0; pass < npass; ++pass) {
            const bool first = pass == 0, last = pass == npass - 1;
            const int w = pp.width[pass];
            const uint32_t mask = (1u << w) - 1u;
            const int nb = (int)mask + 1, scan_threads = nb < 32 ? 32 : nb;  // the table is [tile][nb]
            const UnitPtrs<1 + L::ncomp>& pin = buf[(pass + 1) & 1];   // written by the pass before
            const UnitPtrs<1 + L::ncomp>& pout = buf[pass & 1];
            if (first) {  // [drift +] cell index [+ KE] + first-digit histogram; src is read only
                if constexpr (has_vel) {
                    if (drift && ke) cell_hist_kernel<L, true, true><<<ntiles, kCellThreads, 0, st>>>(src, n, key0, a.drift_dt, a.log2g, mask, hist, kep);
                    else if (drift) cell_hist_kernel<L, true, false><<<ntiles, kCellThreads, 0, st>>>(src, n, key0, a.drift_dt, a.log2g, mask, hist, kep);
                    else if (ke) cell_hist_kernel<L, false, true><<<ntiles, kCellThreads, 0, st>>>(src, n, key0, a.drift_dt, a.log2g, mask, hist, kep);
                    else cell_hist_kernel<L, false, false><<<ntiles, kCellThreads, 0, st>>>(src, n, key0, a.drift_dt, a.log2g, mask, hist, kep);
                } else {
                    cell_hist_kernel<L, false, false><<<ntiles, kCellThreads, 0, st>>>(src, n, key0, a.drift_dt, a.log2g, mask, hist, kep);
                }
                SOAX_TRY(launched());
                if (ke) SOAX_TRY(sum_partials(kep, (int)ntiles, a.kinetic, st));
            } else {  // the keys of the pass before: unit 0 of the paired buffer, every second word if an index travels along
                tile_hist_kernel<<<ntiles, kSortThreads, 0, st>>>(static_cast<const uint32_t*>(pin.p[0]), has_idx ? 2 : 1, n, shift, mask, hist);
                SOAX_TRY(launched());
            }
            colscan_reduce_kernel<<<nchunks, scan_threads, 0, st>>>(hist, (int)ntiles, nb, partial);
            SOAX_TRY(launched());
            colscan_top_kernel<<<1, scan_threads, 0, st>>>(partial, (int)nchunks, nb, dbase);
            SOAX_TRY(launched());
            colscan_apply_kernel<<<nchunks, scan_threads, 0, st>>>(hist, (int)ntiles, nb, partial, dbase);
            SOAX_TRY(launched());

            ScatterArgs g{};
            g.key_in = key0;
            g.idx_out = a.perm;
            g.base = hist; g.n = n; g.shift = shift; g.mask = mask; g.nbits = w; g.ntiles = (int)ntiles; g.dt = a.drift_dt;
            // Short runs (wide digits) need the neighbouring tiles' pieces to reach the L2 together: clusters + barriers.
            const int want_cluster = g_tune.bin_cluster > 0 ? g_tune.bin_cluster : 4;
            const int cluster = (g_tune.bin_cluster > 0 || w >= 8) ? want_cluster : 1;
            g.csync = cluster > 1 && g_tune.bin_csync != 0;
            g.pace_sync = g_tune.bin_pace >= 0 ? (g_tune.bin_pace >> 12) & 3 : (cluster > 1 ? 2 : 0);
            if (g.pace_sync == 2 && cluster == 1) g.pace_sync = 1;
            g.pace_ns = g_tune.bin_pace >= 0 ? g_tune.bin_pace & 0xfff : 0;
            g.pace_every = g_tune.bin_pace_every > 0 ? g_tune.bin_pace_every : (g.pace_sync == 2 ? 2 : 1);  // measured: a cluster barrier every second store
            if (has_idx) SOAX_TRY((scatter_pass<L, true>(first, last, drift, cluster, ntiles, st, src, dst, pin, pout, g)));
            else SOAX_TRY((scatter_pass<L, false>(first, last, drift, cluster, ntiles, st, src, dst, pin, pout, g)));
            shift += w;
        }
        if (a.counts || a.offsets) {
            cell_bounds_kernel<<<ncell / 256 + 1, 256, 0, st>>>(field_ptr<L, pos_tag>(dst, 0), field_ptr<L, pos_tag>(dst, 1), field_ptr<L, pos_tag>(dst, 2), n,
                                                                 a.log2g, a.counts, a.offsets);
            SOAX_TRY(launched());
        }
        return SOAX_OK;
    }
}

#define X(L)                                                               \
    template int bin_permute_entry<L>(const BinArgs&, cudaStream_t);      \
    template size_t bin_scratch_bytes<L>(int64_t, int, bool);
SOAX_FOR_EACH_LAYOUT(X)
#undef X

}  // namespace soax
