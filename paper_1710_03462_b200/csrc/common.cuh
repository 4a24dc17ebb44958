// common.cuh -- device helpers shared by the kernels: the arithmetic contract (wrap, explicit fma), vector
// memory access (128- and 256-bit per thread per field array) and launch bookkeeping.
// GPU side only: the oracle (oracle/) shares nothing with this file.
#pragma once
#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>

#include "layout.hpp"

namespace soax {

// ---- launch bookkeeping -------------------------------------------------------------------------------------
extern std::atomic<int64_t> g_launches;
extern thread_local int g_last_cuda_error;
inline int cuda_fail(cudaError_t e) { g_last_cuda_error = (int)e; return SOAX_ERR_CUDA; }
// after a <<<>>> launch: count it and pick up launch-configuration errors without synchronising
inline int launched() {
    g_launches.fetch_add(1, std::memory_order_relaxed);
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail(e); }
    return SOAX_OK;
}
#define SOAX_TRY(expr) do { int rc_ = (expr); if (rc_ != SOAX_OK) return rc_; } while (0)
#define SOAX_CUDA(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) return ::soax::cuda_fail(e_); } while (0)

constexpr int kSMs = 148;  // B200: 2 dies x 74 SMs; grids of persistent kernels are sized in multiples of this

// ---- arithmetic contract: compiled with -fmad=false, every fma below is explicit ----------------
// a3, Q3: wrap into [0,1): w = x - floor(x); a result of exactly 1.0 (x = -tiny) is mapped to 0.0.
// The fast path never calls floor(): for -1 <= x < 2 the floor is one of {-1, 0, 1}, and x - f == x + (-f)
// exactly in IEEE arithmetic, so adding {+1.0, +0.0, -1.0} performs the SAME rounded operation as the
// definition (including -0.0 + +0.0 = +0.0, which is what -0.0 - floor(-0.0) = -0.0 - (-0.0) gives).
__device__ __forceinline__ double wrap01(double x) {
    double w;
    if (x >= -1.0 && x < 2.0) {
        const double nf = x < 0.0 ? 1.0 : (x >= 1.0 ? -1.0 : 0.0);
        w = x + nf;
    } else {
        w = x - floor(x);  // also the NaN path (comparisons false): NaN propagates
    }
    return w >= 1.0 ? 0.0 : w;
}

// destination-type rule (Q2): an update is ONE fma in the type of the field being written
__device__ __forceinline__ double fma_t(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ float fma_t(float a, float b, float c) { return fmaf(a, b, c); }

// a2: DRIFT of one component. V = float (R1) or double (R2).
template <class V>
__device__ __forceinline__ double drift1(double dt, V vel, double pos) {
    return wrap01(fma(dt, (double)vel, pos));
}
// a4: symplectic-Euler kick of one component: F = (V)(-(k*(pos - ctr))); vel = fma_V((V)dt, F, vel).
template <class V>
__device__ __forceinline__ V kick1(V dt_v, double k, double ctr, double pos, V vel) {
    const V F = (V)(-(k * (pos - ctr)));
    return fma_t(dt_v, F, vel);
}
// a8: energy term of one particle (k*d*d potential only if HARMONIC).
template <bool HARMONIC>
__device__ __forceinline__ double energy1(double v0, double v1, double v2, double x0, double x1, double x2,
                                          double k, double ctr) {
    double q = v0 * v0;
    q = fma(v1, v1, q);
    q = fma(v2, v2, q);
    if (HARMONIC) {
        double d = x0 - ctr; q = fma(k * d, d, q);
        d = x1 - ctr;        q = fma(k * d, d, q);
        d = x2 - ctr;        q = fma(k * d, d, q);
    }
    return 0.5 * q;
}
// a10: cell index on a G^3 grid, G = 2^log2g a power of two so pos*G is exact (Q16); x slowest (Q11).
// Truncation toward zero; out-of-box positions (a precondition violation) are clamped into the grid.
__device__ __forceinline__ uint32_t cell_of(double x0, double x1, double x2, double G, int gmax, int log2g) {
    int i0 = min(max((int)(x0 * G), 0), gmax);
    int i1 = min(max((int)(x1 * G), 0), gmax);
    int i2 = min(max((int)(x2 * G), 0), gmax);
    return (uint32_t)((((i0 << log2g) | i1) << log2g) | i2);
}

// ---- vector access: P consecutive elements of one component array per thread --------------------------------
// sizeof(T)*P in {1,2,4,8,16,32,64}; 32 bytes = one LDG.E.256 / STG.E.256 (sm_100 and later only), 16 = .128,
// 64 = two 256-bit accesses.
template <class T, int P>
struct alignas(sizeof(T) * P > 32 ? 32 : sizeof(T) * P) Vec {
    T v[P];
};

// Streaming loads/stores: each element is touched exactly once per pass, so do not allocate in L1.
template <class T, int P>
__device__ __forceinline__ Vec<T, P> ld_vec(const T* p) {
    constexpr int B = sizeof(T) * P;
    Vec<T, P> r;
    if constexpr (B == 64) {
        uint32_t* w = reinterpret_cast<uint32_t*>(&r);
        asm volatile("ld.global.L1::no_allocate.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                     : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]), "=r"(w[4]), "=r"(w[5]), "=r"(w[6]), "=r"(w[7])
                     : "l"(p));
        asm volatile("ld.global.L1::no_allocate.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8+32];"
                     : "=r"(w[8]), "=r"(w[9]), "=r"(w[10]), "=r"(w[11]), "=r"(w[12]), "=r"(w[13]), "=r"(w[14]), "=r"(w[15])
                     : "l"(p));
    } else if constexpr (B == 32) {
        uint32_t* w = reinterpret_cast<uint32_t*>(&r);
        asm volatile("ld.global.L1::no_allocate.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                     : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]), "=r"(w[4]), "=r"(w[5]), "=r"(w[6]), "=r"(w[7])
                     : "l"(p));
    } else if constexpr (B == 16) {
        uint32_t* w = reinterpret_cast<uint32_t*>(&r);
        asm volatile("ld.global.L1::no_allocate.v4.b32 {%0,%1,%2,%3}, [%4];"
                     : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]) : "l"(p));
    } else if constexpr (B == 8) {
        uint32_t* w = reinterpret_cast<uint32_t*>(&r);
        asm volatile("ld.global.L1::no_allocate.v2.b32 {%0,%1}, [%2];" : "=r"(w[0]), "=r"(w[1]) : "l"(p));
    } else {
        r = *reinterpret_cast<const Vec<T, P>*>(p);
    }
    return r;
}
template <class T, int P>
__device__ __forceinline__ void st_vec(T* p, const Vec<T, P>& r) {
    constexpr int B = sizeof(T) * P;
    if constexpr (B == 64) {
        const uint32_t* w = reinterpret_cast<const uint32_t*>(&r);
        asm volatile("st.global.L1::no_allocate.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                     :: "l"(p), "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]), "r"(w[4]), "r"(w[5]), "r"(w[6]), "r"(w[7])
                     : "memory");
        asm volatile("st.global.L1::no_allocate.v8.b32 [%0+32], {%1,%2,%3,%4,%5,%6,%7,%8};"
                     :: "l"(p), "r"(w[8]), "r"(w[9]), "r"(w[10]), "r"(w[11]), "r"(w[12]), "r"(w[13]), "r"(w[14]), "r"(w[15])
                     : "memory");
    } else if constexpr (B == 32) {
        const uint32_t* w = reinterpret_cast<const uint32_t*>(&r);
        asm volatile("st.global.L1::no_allocate.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                     :: "l"(p), "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]), "r"(w[4]), "r"(w[5]), "r"(w[6]), "r"(w[7])
                     : "memory");
    } else if constexpr (B == 16) {
        const uint32_t* w = reinterpret_cast<const uint32_t*>(&r);
        asm volatile("st.global.L1::no_allocate.v4.b32 [%0], {%1,%2,%3,%4};"
                     :: "l"(p), "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]) : "memory");
    } else if constexpr (B == 8) {
        const uint32_t* w = reinterpret_cast<const uint32_t*>(&r);
        asm volatile("st.global.L1::no_allocate.v2.b32 [%0], {%1,%2};" :: "l"(p), "r"(w[0]), "r"(w[1]) : "memory");
    } else {
        *reinterpret_cast<Vec<T, P>*>(p) = r;
    }
}

// ---- warp / block reductions in double, fixed order (deterministic) ------------------------------------------
__device__ __forceinline__ double warp_sum(double x) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
    return x;  // lane 0 holds the sum
}
// Sum over the block; result valid in thread 0.  smem: >= 32 doubles.  All threads must call.
__device__ __forceinline__ double block_sum(double x, double* smem) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = (blockDim.x + 31) >> 5;
    x = warp_sum(x);
    __syncthreads();  // protect smem from a previous use
    if (lane == 0) smem[warp] = x;
    __syncthreads();
    if (warp == 0) {
        x = lane < nwarp ? smem[lane] : 0.0;
        x = warp_sum(x);
    }
    return x;
}

}  // namespace soax
