// rank_probe.cu -- cost of the stable in-warp ranking of the binning scatter (8 rounds of 32 nine-bit digits per warp, 16 warps
// per CTA, two CTAs per SM, running per-warp digit counters in shared memory) with three ways of finding the lanes that hold
// the same digit.  Stand-alone (`python bench.py --mem-probes` builds and runs it); one JSON line per variant.
//   ballots   one warp vote per digit bit (the shipped kernel)
//   match     __match_any_sync
//   atomic_or every lane ORs its bit into the digit's word of a per-warp mask table and reads the word back
//   floor     the loop around them alone (zeroing the tables, loading the keys, the CTA barriers)
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
constexpr int kItems = 8, kRadix = 512, kWarps = 16;

template <int MODE>
__global__ void __launch_bounds__(512, 2) rank_kernel(const uint32_t* __restrict__ keys, uint32_t* __restrict__ out, int iters) {
    __shared__ uint32_t wcnt[kWarps * kRadix];
    extern __shared__ uint32_t wmask[];  // atomic_or: kWarps * kRadix words
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    uint32_t* mycnt = wcnt + warp * kRadix;
    const uint32_t lt = (1u << lane) - 1u;
    uint32_t acc = 0;
    for (int it = 0; it < iters; ++it) {
        for (int i = tid; i < kWarps * kRadix; i += 512) wcnt[i] = 0;
        if (MODE == 2) for (int i = tid; i < kWarps * kRadix; i += 512) wmask[i] = 0u;
        __syncthreads();
        const uint32_t* kp = keys + ((size_t)blockIdx.x * iters + it) % 4096 * 4096 + warp * 256 + lane;
        uint32_t lpos[kItems], dig[kItems];
#pragma unroll
        for (int k = 0; k < kItems; ++k) dig[k] = kp[k * 32] & 511u;
        if (MODE == 3) {
#pragma unroll
            for (int k = 0; k < kItems; ++k) lpos[k] = dig[k];
        } else if (MODE == 2) {
            uint32_t* mymask = wmask + warp * kRadix;
#pragma unroll
            for (int k = 0; k < kItems; ++k) {
                const uint32_t d = dig[k];
                atomicOr(&mymask[d], 1u << lane);
                __syncwarp();
                const uint32_t m = mymask[d];
                const uint32_t old = mycnt[d];
                lpos[k] = old + __popc(m & lt);
                __syncwarp();
                if (lane == 31 - __clz(m)) { mycnt[d] = old + __popc(m); mymask[d] = 0u; }
                __syncwarp();
            }
        } else {
#pragma unroll
            for (int k = 0; k < kItems; ++k) {
                const uint32_t d = dig[k];
                uint32_t m = 0xffffffffu;
                if (MODE == 1) {
                    m = __match_any_sync(0xffffffffu, d);
                } else {
#pragma unroll
                    for (int b = 0; b < 9; ++b) {
                        const bool bit = (d >> b) & 1u;
                        const uint32_t bal = __ballot_sync(0xffffffffu, bit);
                        m &= bit ? bal : ~bal;
                    }
                }
                const uint32_t old = mycnt[d];
                lpos[k] = old + __popc(m & lt);
                __syncwarp();
                if (lane == 31 - __clz(m)) mycnt[d] = old + __popc(m);
                __syncwarp();
            }
        }
#pragma unroll
        for (int k = 0; k < kItems; ++k) acc += lpos[k] * (k + 1);
        __syncthreads();
    }
    out[(size_t)blockIdx.x * 512 + tid] = acc;
}

int main() {
    uint32_t *keys, *out;
    const size_t nk = 4096ull * 4096;
    if (cudaMalloc(&keys, nk * 4) != cudaSuccess || cudaMalloc(&out, 296 * 512 * 4) != cudaSuccess) { std::printf("{\"probe_error\": \"cudaMalloc\"}\n"); return 1; }
    uint32_t* h = new uint32_t[nk];
    uint64_t x = 88172645463325252ull;
    for (size_t i = 0; i < nk; ++i) { x ^= x << 13; x ^= x >> 7; x ^= x << 17; h[i] = (uint32_t)(x >> 20); }
    cudaMemcpy(keys, h, nk * 4, cudaMemcpyHostToDevice);
    const int iters = 200;
    const char* names[4] = {"ballots", "match", "atomic_or", "floor"};
    uint32_t* ref = new uint32_t[296 * 512];
    uint32_t* got = new uint32_t[296 * 512];
    cudaFuncSetAttribute(rank_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 32768);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    for (int mode = 0; mode < 4; ++mode) {
        for (int rep = 0; rep < 2; ++rep) {
            cudaEventRecord(e0);
            if (mode == 0) rank_kernel<0><<<296, 512>>>(keys, out, iters);
            if (mode == 1) rank_kernel<1><<<296, 512>>>(keys, out, iters);
            if (mode == 2) rank_kernel<2><<<296, 512, 32768>>>(keys, out, iters);
            if (mode == 3) rank_kernel<3><<<296, 512>>>(keys, out, iters);
            cudaEventRecord(e1); cudaEventSynchronize(e1);
        }
        float ms;
        cudaEventElapsedTime(&ms, e0, e1);
        cudaMemcpy(mode == 0 ? ref : got, out, 296 * 512 * 4, cudaMemcpyDeviceToHost);
        int same = 1;
        if (mode == 1 || mode == 2) for (int i = 0; i < 296 * 512; ++i) same &= got[i] == ref[i];
        std::printf("{\"probe\": \"rank\", \"variant\": \"%s\", \"us_per_tile_two_ctas_per_sm\": %.2f, \"ranks_equal_ballots\": %s, \"cuda_error\": %d}\n", names[mode],
                    ms * 1e3 / iters, mode == 3 ? "null" : (same ? "true" : "false"), (int)cudaGetLastError());
    }
    return 0;
}
