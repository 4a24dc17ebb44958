// aos_kernels.cu -- a5, a6, a7: everything that touches the Array-of-Structures image of a layout.
//   * step_aos variant 0: the paper's AoS GPU kernel (K5): one thread per record, each field read
//     and written in place with the stride of the record between neighbouring lanes (uncoalesced by design);
//     it is the in-library baseline the SoA kernels are compared against (config 3).
//   * step_aos variant 1: best effort on the same data: whole tiles of records are staged through shared memory
//     with bulk asynchronous copies (TMA, UBLKCP), updated there, and written back in one piece.
//   * aos_to_soa / soa_to_aos: the AoS side of a tile moves as ONE contiguous bulk copy global<->shared; the
//     SoA side is read/written with fully coalesced per-component accesses.
// The packed record (Q1) puts R1's doubles at offset 4 mod 8, so fields are accessed in pieces of the largest
// power of two that divides both the stride and the field offset (4 bytes for R1, 1 byte for R2's 89-byte
// record).
#include "common.cuh"
#include "ops.hpp"
#include "tma.cuh"

namespace soax {

constexpr int cgcd(int a, int b) { return b == 0 ? a : cgcd(b, a % b); }

// Load / store a T at an address whose alignment is only known to be A bytes (A a power of two <= 16).
template <class T, int A>
__device__ __forceinline__ T ld_piecewise(const unsigned char* p) {
    if constexpr (A >= (int)sizeof(T)) {
        return *reinterpret_cast<const T*>(p);
    } else if constexpr (A >= 4) {
        static_assert(sizeof(T) == 8, "only 8-byte types are split into words");
        const uint32_t lo = *reinterpret_cast<const uint32_t*>(p), hi = *reinterpret_cast<const uint32_t*>(p + 4);
        const unsigned long long u = ((unsigned long long)hi << 32) | lo;
        T r;
        memcpy(&r, &u, 8);
        return r;
    } else {
        unsigned char b[sizeof(T)];
#pragma unroll
        for (int i = 0; i < (int)sizeof(T); ++i) b[i] = p[i];
        T r;
        memcpy(&r, b, sizeof(T));
        return r;
    }
}
template <class T, int A>
__device__ __forceinline__ void st_piecewise(unsigned char* p, T v) {
    if constexpr (A >= (int)sizeof(T)) {
        *reinterpret_cast<T*>(p) = v;
    } else if constexpr (A >= 4) {
        unsigned long long u;
        memcpy(&u, &v, 8);
        *reinterpret_cast<uint32_t*>(p) = (uint32_t)u;
        *reinterpret_cast<uint32_t*>(p + 4) = (uint32_t)(u >> 32);
    } else {
        unsigned char b[sizeof(T)];
        memcpy(b, &v, sizeof(T));
#pragma unroll
        for (int i = 0; i < (int)sizeof(T); ++i) p[i] = b[i];
    }
}
// alignment guaranteed for component C of a packed record whose array base is 16-byte aligned
template <class L, int C>
constexpr int comp_align() { return cgcd(16, cgcd(L::aos_stride, L::aos_offset(C))); }

template <class L, class Tag>
__device__ __forceinline__ typename L::template type_of<Tag> ld_field(const unsigned char* rec, int k) {
    using T = typename L::template type_of<Tag>;
    constexpr int c0 = L::template begin_of<Tag>;
    constexpr int A = cgcd(16, cgcd(L::aos_stride, cgcd(L::aos_offset(c0), (int)sizeof(T))));
    return ld_piecewise<T, A>(rec + L::aos_offset(c0) + k * (int)sizeof(T));
}
template <class L, class Tag>
__device__ __forceinline__ void st_field(unsigned char* rec, int k, typename L::template type_of<Tag> v) {
    using T = typename L::template type_of<Tag>;
    constexpr int c0 = L::template begin_of<Tag>;
    constexpr int A = cgcd(16, cgcd(L::aos_stride, cgcd(L::aos_offset(c0), (int)sizeof(T))));
    st_piecewise<T, A>(rec + L::aos_offset(c0) + k * (int)sizeof(T), v);
}

// The update of ONE record held at `rec` (global or shared memory): same operation sequence as the SoA kernels.
template <class L, int KIND>
__device__ __forceinline__ void step_record(unsigned char* rec, double dt, double k, double ctr) {
    using V = typename L::template type_of<vel_tag>;
    if constexpr (KIND == SOAX_STEP_EULER_NOWRAP) {
        // Eq. 1 as printed on the paper's own record (Listing 4): x_c += dt v_c, one
        // fma in the type of pos, no wrap; temp[SIZE] rides along untouched -- that is the whole point of Fig. 8.
        using X = typename L::template type_of<pos_tag>;
        const X dt_x = (X)dt;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const X x = ld_field<L, pos_tag>(rec, d);
            const V v = ld_field<L, vel_tag>(rec, d);
            st_field<L, pos_tag>(rec, d, fma_t(dt_x, (X)v, x));
        }
        return;
    }
    const V dt_v = (V)dt;  // (float)dt rounds to nearest: dt_f of the contract
    double x[3];
    V v[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) { x[d] = ld_field<L, pos_tag>(rec, d); v[d] = ld_field<L, vel_tag>(rec, d); }
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        if constexpr (KIND == SOAX_STEP_SYMPLECTIC_EULER_HARMONIC) v[d] = kick1<V>(dt_v, k, ctr, x[d], v[d]);
        x[d] = drift1<V>(dt, v[d], x[d]);
    }
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        if constexpr (KIND == SOAX_STEP_SYMPLECTIC_EULER_HARMONIC) st_field<L, vel_tag>(rec, d, v[d]);
        st_field<L, pos_tag>(rec, d, x[d]);
    }
}

// ---- a5 variant 0: thread per record, strided access -------------------------------------------
template <class L, int KIND>
__global__ void __launch_bounds__(1024) step_aos_direct_kernel(unsigned char* aos, int64_t n, double dt, double k, double ctr) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) step_record<L, KIND>(aos + i * L::aos_stride, dt, k, ctr);
}

// ---- tile staging shared by variant 1 and the transposes -------------------------------------------------------
constexpr int kTile = 256;  // records per tile = threads per CTA; kTile * stride is a multiple of 16 bytes

// copy A bytes (A a power of two <= 16) between addresses aligned to A
template <int A>
__device__ __forceinline__ void copy_piece(unsigned char* dst, const unsigned char* src) {
    if constexpr (A == 16) *reinterpret_cast<uint4*>(dst) = *reinterpret_cast<const uint4*>(src);
    else if constexpr (A == 8) *reinterpret_cast<uint2*>(dst) = *reinterpret_cast<const uint2*>(src);
    else if constexpr (A == 4) *reinterpret_cast<uint32_t*>(dst) = *reinterpret_cast<const uint32_t*>(src);
    else if constexpr (A == 2) *reinterpret_cast<uint16_t*>(dst) = *reinterpret_cast<const uint16_t*>(src);
    else *dst = *src;
}

// bring records [t0, t0 + cnt) into shared memory: one bulk copy for a full tile, piecewise copies for the tail
template <class L>
__device__ __forceinline__ void tile_load(unsigned char* sm, const unsigned char* aos, int64_t t0, int cnt, uint64_t* bar,
                                          uint32_t& phase) {
    constexpr int S = L::aos_stride;
    if (cnt == kTile) {
        if (threadIdx.x == 0) {
            mbar_expect_tx(bar, kTile * S);
            bulk_g2s(sm, aos + t0 * S, kTile * S, bar);
        }
        mbar_wait(bar, phase);
        phase ^= 1;
    } else {
        constexpr int A = cgcd(16, S);  // tail: copy in pieces the record size allows
        const unsigned char* g = aos + t0 * S;
        for (int o = threadIdx.x * A; o < cnt * S; o += blockDim.x * A) copy_piece<A>(sm + o, g + o);
        __syncthreads();
    }
}
// write records [t0, t0 + cnt) back from shared memory; all threads must have finished writing `sm`
template <class L>
__device__ __forceinline__ void tile_store(unsigned char* aos, const unsigned char* sm, int64_t t0, int cnt) {
    constexpr int S = L::aos_stride;
    if (cnt == kTile) {
        fence_async_smem();
        __syncthreads();
        if (threadIdx.x == 0) {
            bulk_s2g(aos + t0 * S, sm, kTile * S);
            bulk_commit();
            bulk_wait_read();  // the buffer is reused by the next tile
        }
        __syncthreads();
    } else {
        __syncthreads();
        constexpr int A = cgcd(16, S);
        unsigned char* g = aos + t0 * S;
        for (int o = threadIdx.x * A; o < cnt * S; o += blockDim.x * A) copy_piece<A>(g + o, sm + o);
        __syncthreads();
    }
}

// ---- a5 variant 1: records staged through shared memory --------------------------------------------------------
template <class L, int KIND>
__global__ void __launch_bounds__(kTile) step_aos_staged_kernel(unsigned char* aos, int64_t n, double dt, double k, double ctr) {
    extern __shared__ __align__(128) unsigned char sm[];
    __shared__ uint64_t bar;
    if (threadIdx.x == 0) { mbar_init(&bar, 1); mbar_fence_init(); }
    __syncthreads();
    uint32_t phase = 0;
    const int64_t ntiles = (n + kTile - 1) / kTile;
    for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const int64_t t0 = t * kTile;
        const int cnt = (int)(n - t0 < kTile ? n - t0 : kTile);
        tile_load<L>(sm, aos, t0, cnt, &bar, phase);
        if ((int)threadIdx.x < cnt) step_record<L, KIND>(sm + threadIdx.x * L::aos_stride, dt, k, ctr);
        tile_store<L>(aos, sm, t0, cnt);
    }
}

// ---- a6: AoS -> SoA ----------------------------------------------------------------------------------------------
template <class L>
__global__ void __launch_bounds__(kTile) aos_to_soa_kernel(Ptrs<L::ncomp> a, const unsigned char* aos, int64_t n) {
    extern __shared__ __align__(128) unsigned char sm[];
    __shared__ uint64_t bar;
    if (threadIdx.x == 0) { mbar_init(&bar, 1); mbar_fence_init(); }
    __syncthreads();
    uint32_t phase = 0;
    const int64_t ntiles = (n + kTile - 1) / kTile;
    for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const int64_t t0 = t * kTile;
        const int cnt = (int)(n - t0 < kTile ? n - t0 : kTile);
        tile_load<L>(sm, aos, t0, cnt, &bar, phase);
        if ((int)threadIdx.x < cnt) {
            const unsigned char* rec = sm + threadIdx.x * L::aos_stride;
            for_each_comp<L>([&](auto ci) {
                constexpr int C = decltype(ci)::value;
                using T = typename L::template comp_type<C>;
                comp_ptr<L, C>(a)[t0 + threadIdx.x] = ld_piecewise<T, comp_align<L, C>()>(rec + L::aos_offset(C));
            });
        }
        __syncthreads();  // everyone is done reading before the next bulk copy overwrites the tile
    }
}

// ---- a7: SoA -> AoS ----------------------------------------------------------------------------------------------
template <class L>
__global__ void __launch_bounds__(kTile) soa_to_aos_kernel(Ptrs<L::ncomp> a, unsigned char* aos, int64_t n) {
    extern __shared__ __align__(128) unsigned char sm[];
    const int64_t ntiles = (n + kTile - 1) / kTile;
    for (int64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const int64_t t0 = t * kTile;
        const int cnt = (int)(n - t0 < kTile ? n - t0 : kTile);
        if ((int)threadIdx.x < cnt) {
            unsigned char* rec = sm + threadIdx.x * L::aos_stride;
            for_each_comp<L>([&](auto ci) {
                constexpr int C = decltype(ci)::value;
                using T = typename L::template comp_type<C>;
                st_piecewise<T, comp_align<L, C>()>(rec + L::aos_offset(C), comp_ptr<L, C>(a)[t0 + threadIdx.x]);
            });
        }
        tile_store<L>(aos, sm, t0, cnt);
    }
}

// ---- a6 / a7, pipelined (default): a persistent CTA walks its tiles with a ring of NS shared-memory stages --------
// A stage holds R*kTile records.  AoS -> SoA: the bulk copy of the tile NS-1 places ahead is in flight while the
// current one is read out of shared memory (each thread takes records t, t+256, ... so that every warp reads
// neighbouring records -- 2-way bank conflicts at a 40-byte stride -- and writes 128/256 contiguous bytes per
// component array).  SoA -> AoS: all R*ncomp global loads of a thread are issued first (R*40 bytes in flight per
// thread for R1), then the records are assembled in the stage and leave as ONE bulk store whose read of shared
// memory overlaps the loads of the next tile.  Records behind the last full tile go straight between the two
// global images, piece by piece.
template <class L, int R, int NS> constexpr int ring_smem() { return NS * R * kTile * L::aos_stride + 64; }

template <class L>
__device__ __forceinline__ void tail_aos_to_soa(const Ptrs<L::ncomp>& a, const unsigned char* aos, int64_t from, int64_t n) {
    for (int64_t i = from + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const unsigned char* rec = aos + i * L::aos_stride;
        for_each_comp<L>([&](auto ci) {
            constexpr int C = decltype(ci)::value;
            using T = typename L::template comp_type<C>;
            comp_ptr<L, C>(a)[i] = ld_piecewise<T, comp_align<L, C>()>(rec + L::aos_offset(C));
        });
    }
}
template <class L>
__device__ __forceinline__ void tail_soa_to_aos(const Ptrs<L::ncomp>& a, unsigned char* aos, int64_t from, int64_t n) {
    for (int64_t i = from + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        unsigned char* rec = aos + i * L::aos_stride;
        for_each_comp<L>([&](auto ci) {
            constexpr int C = decltype(ci)::value;
            using T = typename L::template comp_type<C>;
            st_piecewise<T, comp_align<L, C>()>(rec + L::aos_offset(C), comp_ptr<L, C>(a)[i]);
        });
    }
}

template <class L, int R, int NS>
__global__ void __launch_bounds__(kTile) aos_to_soa_ring_kernel(Ptrs<L::ncomp> a, const unsigned char* aos, int64_t n) {
    constexpr int SB = R * kTile * L::aos_stride, TILE = R * kTile, S = L::aos_stride;
    extern __shared__ __align__(128) unsigned char sm[];
    uint64_t* full = reinterpret_cast<uint64_t*>(sm + NS * SB);
    const int tid = threadIdx.x;
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    const int64_t nfull = n / TILE;
    const int64_t mine = nfull > blockIdx.x ? (nfull - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;  // tiles of this CTA
    auto issue = [&](int64_t k) {  // thread 0: start the bulk copy of this CTA's k-th tile into stage k % NS
        const int64_t t = blockIdx.x + k * gridDim.x;
        mbar_expect_tx(&full[k % NS], SB);
        bulk_g2s(sm + (k % NS) * SB, aos + t * (int64_t)TILE * S, SB, &full[k % NS]);
    };
    if (tid == 0)
        for (int64_t k = 0; k < NS - 1 && k < mine; ++k) issue(k);
    for (int64_t k = 0; k < mine; ++k) {
        // stage (k-1) % NS was read in the previous iteration; its reads completed before the barrier that ended it
        if (tid == 0 && k + NS - 1 < mine) issue(k + NS - 1);
        mbar_wait(&full[k % NS], (uint32_t)((k / NS) & 1));
        const unsigned char* st = sm + (k % NS) * SB;
        const int64_t t0 = (blockIdx.x + k * gridDim.x) * (int64_t)TILE;
        for_each_comp<L>([&](auto ci) {
            constexpr int C = decltype(ci)::value;
            using T = typename L::template comp_type<C>;
            T v[R];
#pragma unroll
            for (int r = 0; r < R; ++r) v[r] = ld_piecewise<T, comp_align<L, C>()>(st + (tid + r * kTile) * S + L::aos_offset(C));
#pragma unroll
            for (int r = 0; r < R; ++r) comp_ptr<L, C>(a)[t0 + tid + r * kTile] = v[r];  // consumes the reads before the barrier
        });
        __syncthreads();
    }
    tail_aos_to_soa<L>(a, aos, nfull * TILE, n);
}

template <class L, int R, int NS>
__global__ void __launch_bounds__(kTile) soa_to_aos_ring_kernel(Ptrs<L::ncomp> a, unsigned char* aos, int64_t n) {
    constexpr int SB = R * kTile * L::aos_stride, TILE = R * kTile, S = L::aos_stride;
    extern __shared__ __align__(128) unsigned char sm[];
    const int tid = threadIdx.x;
    const int64_t nfull = n / TILE;
    const int64_t mine = nfull > blockIdx.x ? (nfull - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    for (int64_t k = 0; k < mine; ++k) {
        unsigned char* st = sm + (k % NS) * SB;
        const int64_t t0 = (blockIdx.x + k * gridDim.x) * (int64_t)TILE;
        // the bulk store that last read this stage was committed NS iterations ago: at most NS-1 younger ones may be pending
        if (tid == 0 && k >= NS) asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(NS - 1) : "memory");
        __syncthreads();
        // every global load of the thread is issued before the first shared-memory store; typed registers per component
        // (a common 64-bit image makes the compiler funnel the loads through one temporary and serialise them)
        constexpr int kGroup = 16;
        constexpr int kGroups = (L::ncomp + kGroup - 1) / kGroup;
        for_each_int<kGroups>([&](auto gi) {
            constexpr int G0 = decltype(gi)::value * kGroup;
            constexpr int GN = L::ncomp - G0 < kGroup ? L::ncomp - G0 : kGroup;
            CompRegs<L, G0, R, std::make_integer_sequence<int, GN>> v;
            for_each_int<GN>([&](auto ci) {
                constexpr int C = G0 + decltype(ci)::value;
#pragma unroll
                for (int r = 0; r < R; ++r) v.template get<C>()[r] = comp_ptr<L, C>(a)[t0 + tid + r * kTile];
            });
            for_each_int<GN>([&](auto ci) {
                constexpr int C = G0 + decltype(ci)::value;
                using T = typename L::template comp_type<C>;
#pragma unroll
                for (int r = 0; r < R; ++r)
                    st_piecewise<T, comp_align<L, C>()>(st + (tid + r * kTile) * S + L::aos_offset(C), v.template get<C>()[r]);
            });
        });
        fence_async_smem();
        __syncthreads();
        if (tid == 0) {
            bulk_s2g(aos + t0 * S, st, SB);
            bulk_commit();
        }
    }
    if (tid == 0) bulk_wait_read();  // shared memory must outlive the last bulk stores' reads
    tail_soa_to_aos<L>(a, aos, nfull * TILE, n);
}

// ---- host side -----------------------------------------------------------------------------------------------------
template <class L>
static unsigned tile_grid(int64_t n, int ctas_per_sm) {
    const int64_t ntiles = (n + kTile - 1) / kTile;
    const int64_t cap = (int64_t)kSMs * ctas_per_sm;
    return (unsigned)(ntiles < cap ? (ntiles < 1 ? 1 : ntiles) : cap);
}
template <class L>
constexpr int tile_ctas_per_sm() {
    constexpr int bytes = kTile * L::aos_stride + 64;
    constexpr int by_smem = (200 * 1024) / bytes;
    return by_smem < 8 ? (by_smem < 1 ? 1 : by_smem) : 8;  // 2048 threads / 256
}

template <class L, int KIND>
static int step_aos_kind(void* aos, int64_t n, const soax_step_params* p, int variant, cudaStream_t st) {
    constexpr bool wrapped = L::template has_as<pos_tag, double, 3>() &&
                             (L::template has_as<vel_tag, float, 3>() || L::template has_as<vel_tag, double, 3>());
    constexpr bool plain = (L::template has_as<pos_tag, double, 3>() || L::template has_as<pos_tag, float, 3>()) &&
                           (L::template has_as<vel_tag, float, 3>() || L::template has_as<vel_tag, double, 3>());
    constexpr bool ok = KIND == SOAX_STEP_EULER_NOWRAP ? plain : wrapped;
    if constexpr (!ok) {
        return SOAX_ERR_UNSUPPORTED;
    } else {
        unsigned char* base = static_cast<unsigned char*>(aos);
        if (variant == 0) {
            const int block = g_tune.aos_block;
            step_aos_direct_kernel<L, KIND><<<(unsigned)((n + block - 1) / block), block, 0, st>>>(base, n, p->dt, p->k, p->center);
        } else if (variant == 1) {
            constexpr int smem = kTile * L::aos_stride;
            step_aos_staged_kernel<L, KIND><<<tile_grid<L>(n, tile_ctas_per_sm<L>()), kTile, smem, st>>>(base, n, p->dt, p->k, p->center);
        } else {
            return SOAX_ERR_INVALID_ARG;
        }
        return launched();
    }
}

template <class L>
int step_aos_entry(void* aos, int64_t n, const soax_step_params* p, int variant, cudaStream_t st) {
    if (n == 0) return SOAX_OK;
    switch (p->kind) {
        case SOAX_STEP_DRIFT: return step_aos_kind<L, SOAX_STEP_DRIFT>(aos, n, p, variant, st);
        case SOAX_STEP_SYMPLECTIC_EULER_HARMONIC: return step_aos_kind<L, SOAX_STEP_SYMPLECTIC_EULER_HARMONIC>(aos, n, p, variant, st);
        case SOAX_STEP_EULER_NOWRAP: return step_aos_kind<L, SOAX_STEP_EULER_NOWRAP>(aos, n, p, variant, st);
        case SOAX_STEP_RK2_MIDPOINT_HARMONIC_MASKED: return SOAX_ERR_UNSUPPORTED;
        default: return SOAX_ERR_INVALID_ARG;
    }
}

template <class L, int R, int NS>
static unsigned ring_grid(int64_t n, int default_ctas) {
    constexpr int by_smem = (220 * 1024) / ring_smem<L, R, NS>();
    constexpr int per_sm = by_smem < 8 ? by_smem : 8;
    const int64_t ntiles = n / (R * kTile);
    const int want = g_tune.xpose_ctas > 0 ? g_tune.xpose_ctas : default_ctas;
    const int64_t cap = (int64_t)kSMs * (want < per_sm ? want : per_sm);
    return (unsigned)(ntiles < cap ? (ntiles < 1 ? 1 : ntiles) : cap);
}
template <class L, int R, int NS>
static int launch_a2s(void* const* comps, const void* aos, int64_t n, cudaStream_t st) {
    if constexpr (ring_smem<L, R, NS>() > 220 * 1024) return SOAX_ERR_UNSUPPORTED;
    else {
        SOAX_CUDA(cudaFuncSetAttribute(aos_to_soa_ring_kernel<L, R, NS>, cudaFuncAttributeMaxDynamicSharedMemorySize, ring_smem<L, R, NS>()));  // per device, cheap: set on every call
        aos_to_soa_ring_kernel<L, R, NS><<<ring_grid<L, R, NS>(n, 2), kTile, ring_smem<L, R, NS>(), st>>>(make_ptrs<L>(comps), static_cast<const unsigned char*>(aos), n);
        return launched();
    }
}
template <class L, int R, int NS>
static int launch_s2a(void* const* comps, void* aos, int64_t n, cudaStream_t st) {
    if constexpr (ring_smem<L, R, NS>() > 220 * 1024) return SOAX_ERR_UNSUPPORTED;
    else {
        SOAX_CUDA(cudaFuncSetAttribute(soa_to_aos_ring_kernel<L, R, NS>, cudaFuncAttributeMaxDynamicSharedMemorySize, ring_smem<L, R, NS>()));  // per device, cheap: set on every call
        soa_to_aos_ring_kernel<L, R, NS><<<ring_grid<L, R, NS>(n, 4), kTile, ring_smem<L, R, NS>(), st>>>(make_ptrs<L>(comps), static_cast<unsigned char*>(aos), n);
        return launched();
    }
}
// Measured on B200 (profiles/r2_sweeps.md, bench.py --sweeps): the shapes differ by a factor of three, and FEW resident CTAs
// win (the ring already keeps the copies in flight; more CTAs only thrash): AoS->SoA is best with 256 records per stage,
// two stages, two CTAs per SM (6.29 TB/s for R1); SoA->AoS with 512 records, one stage, four CTAs per SM (6.29 TB/s).
// soax_tune("xpose_r" / "xpose_ns" / "xpose_ctas") override both directions for sweeps.
#define SOAX_RING_SWITCH(FN, DEFAULT_R, DEFAULT_NS, ...)                                            \
    {                                                                                               \
        int r_ = g_tune.xpose_r > 0 ? g_tune.xpose_r : DEFAULT_R;                                   \
        const int ns_ = g_tune.xpose_ns > 0 ? g_tune.xpose_ns : DEFAULT_NS;                         \
        while (r_ > 1 && ns_ * r_ * kTile * L::aos_stride + 64 > 110 * 1024) r_ >>= 1; /* two CTAs per SM at least */ \
        switch (r_ * 10 + ns_) {                                                                    \
            case 11: return FN<L, 1, 1>(__VA_ARGS__); case 12: return FN<L, 1, 2>(__VA_ARGS__);     \
            case 21: return FN<L, 2, 1>(__VA_ARGS__); case 22: return FN<L, 2, 2>(__VA_ARGS__);     \
            case 41: return FN<L, 4, 1>(__VA_ARGS__); case 42: return FN<L, 4, 2>(__VA_ARGS__);     \
            default: return SOAX_ERR_INVALID_ARG;                                                   \
        }                                                                                           \
    }
template <class L>
int aos_to_soa_entry(void* const* comps, const void* aos, int64_t n, cudaStream_t st) {
    if (g_tune.xpose_ring) SOAX_RING_SWITCH(launch_a2s, 1, 2, comps, aos, n, st)
    constexpr int smem = kTile * L::aos_stride;
    aos_to_soa_kernel<L><<<tile_grid<L>(n, tile_ctas_per_sm<L>()), kTile, smem, st>>>(make_ptrs<L>(comps), static_cast<const unsigned char*>(aos), n);
    return launched();
}
template <class L>
int soa_to_aos_entry(void* const* comps, void* aos, int64_t n, cudaStream_t st) {
    if (g_tune.xpose_ring) SOAX_RING_SWITCH(launch_s2a, 2, 1, comps, aos, n, st)
    constexpr int smem = kTile * L::aos_stride;
    soa_to_aos_kernel<L><<<tile_grid<L>(n, tile_ctas_per_sm<L>()), kTile, smem, st>>>(make_ptrs<L>(comps), static_cast<unsigned char*>(aos), n);
    return launched();
}

// ---- NEXT-4: merge of sorted runs as a SEGMENTED GATHER of packed records into the component arrays -------------------------
// Output row j comes from input record seg_src[i] + (j - seg_dst[i]), i = the last segment with seg_dst[i] <= j.  A CTA owns
// kGatherRows consecutive output rows: two binary searches of the (cached) table bracket its segments, which are copied into
// shared memory once; every row then finds its segment by a short search there (the whole-table search per row of the first
// version cost 21 dependent loads at 2 M segments).  Consecutive rows of a segment read consecutive records, so the AoS side
// is read in whole sectors (through L1, like the thread-per-record AoS kernel), the SoA side is written coalesced.
constexpr int kGatherThreads = 256, kGatherRowsPerThread = 4, kGatherRows = kGatherThreads * kGatherRowsPerThread;
constexpr int kGatherCap = 2048;  // segments of a tile held in shared memory (empty segments count); more: whole-table search
// (Measured and dropped: copying the tile's records into shared memory in output order with 8-byte loads first and taking
// them apart there -- 0.44 ms against 0.31 at 2^24: the three phases of a CTA serialise and only three CTAs fit an SM.)
template <class L>
__global__ void __launch_bounds__(kGatherThreads) gather_segments_kernel(Ptrs<L::ncomp> dst, const unsigned char* __restrict__ aos,
                                                              const uint32_t* __restrict__ seg_dst, const uint32_t* __restrict__ seg_src,
                                                              int64_t nseg, int64_t n) {
    __shared__ uint32_t s_dst[kGatherCap], s_src[kGatherCap];
    __shared__ int64_t s_first, s_last;
    const int64_t j0 = (int64_t)blockIdx.x * kGatherRows;
    const int64_t j1 = j0 + kGatherRows < n ? j0 + kGatherRows : n;  // rows [j0, j1)
    auto last_le = [&](int64_t j) {  // index of the last segment with seg_dst <= j (segment 0 starts at row 0)
        int64_t lo = 0, hi = nseg;
        while (lo < hi) {
            const int64_t mid = (lo + hi) >> 1;
            if ((int64_t)seg_dst[mid] <= j) lo = mid + 1; else hi = mid;
        }
        return lo > 0 ? lo - 1 : 0;  // a table that does not start at row 0 is served from segment 0, not from index -1
    };
    if (threadIdx.x < 2) {
        const int64_t i = last_le(threadIdx.x == 0 ? j0 : j1 - 1);
        if (threadIdx.x == 0) s_first = i; else s_last = i;
    }
    __syncthreads();
    const int64_t first = s_first, count = s_last - s_first + 1;
    const bool tables = count <= kGatherCap;
    if (tables) {
        for (int i = threadIdx.x; i < (int)count; i += kGatherThreads) {
            s_dst[i] = seg_dst[first + i];
            s_src[i] = seg_src[first + i];
        }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < kGatherRowsPerThread; ++r) {
        const int64_t j = j0 + r * kGatherThreads + threadIdx.x;
        if (j >= j1) break;
        int64_t src_row;
        if (tables) {
            int lo = 0, hi = (int)count;
            while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if ((int64_t)s_dst[mid] <= j) lo = mid + 1; else hi = mid;
            }
            const int i = lo > 0 ? lo - 1 : 0;
            const int64_t off = j - (int64_t)s_dst[i];
            src_row = (int64_t)s_src[i] + (off > 0 ? off : 0);
        } else {
            const int64_t i = last_le(j);
            const int64_t off = j - (int64_t)seg_dst[i];
            src_row = (int64_t)seg_src[i] + (off > 0 ? off : 0);
        }
        const unsigned char* rec = aos + src_row * L::aos_stride;
        constexpr int kGroup = 16;
        constexpr int kGroups = (L::ncomp + kGroup - 1) / kGroup;
        for_each_int<kGroups>([&](auto gi) {
            constexpr int G0 = decltype(gi)::value * kGroup;
            constexpr int GN = L::ncomp - G0 < kGroup ? L::ncomp - G0 : kGroup;
            CompRegs<L, G0, 1, std::make_integer_sequence<int, GN>> v;
            for_each_int<GN>([&](auto ci) {
                constexpr int C = G0 + decltype(ci)::value;
                using T = typename L::template comp_type<C>;
                v.template get<C>()[0] = ld_piecewise<T, comp_align<L, C>()>(rec + L::aos_offset(C));
            });
            for_each_int<GN>([&](auto ci) {
                constexpr int C = G0 + decltype(ci)::value;
                comp_ptr<L, C>(dst)[j] = v.template get<C>()[0];
            });
        });
    }
}
template <class L>
int gather_segments_entry(void* const* comps, const void* aos, const uint32_t* seg_dst, const uint32_t* seg_src, int64_t nseg, int64_t n,
                          cudaStream_t st) {
    if (n == 0) return SOAX_OK;
    gather_segments_kernel<L><<<(unsigned)((n + kGatherRows - 1) / kGatherRows), kGatherThreads, 0, st>>>(
        make_ptrs<L>(comps), static_cast<const unsigned char*>(aos), seg_dst, seg_src, nseg, n);
    return launched();
}

#define X(L)                                                                                         \
    template int gather_segments_entry<L>(void* const*, const void*, const uint32_t*, const uint32_t*, int64_t, int64_t, cudaStream_t); \
    template int step_aos_entry<L>(void*, int64_t, const soax_step_params*, int, cudaStream_t);      \
    template int aos_to_soa_entry<L>(void* const*, const void*, int64_t, cudaStream_t);              \
    template int soa_to_aos_entry<L>(void* const*, void*, int64_t, cudaStream_t);
SOAX_FOR_EACH_LAYOUT(X)
#undef X

}  // namespace soax
