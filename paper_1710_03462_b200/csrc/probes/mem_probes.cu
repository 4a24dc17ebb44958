// mem_probes.cu -- two stand-alone measurements of the B200 memory system behind DESIGN.md's account of the binning scatter
// (why a 512-bin pass needs the pieces of a bin's run to reach the L2 together, and why wider pieces are faster).  Not part of
// libsoax.so: `python bench.py --mem-probes` compiles this file with nvcc and runs it; one JSON line per measurement.
//
//   partial   every 32-byte sector of a 1 GiB buffer is written in two halves by the same CTA, `delay_ns` apart, `S` sectors
//             at a time per CTA.  grid x S x 32 B = the volume of half-written sectors open at any moment.  Question: how
//             long / how many half-written sectors does the L2 hold before a sector costs a DRAM read-modify-write?
//             (DRAM bytes per launch come from `ncu --metrics dram__bytes_read.sum,dram__bytes_write.sum`; the time alone
//             already shows it: 0.35 ms when every sector is completed in the L2, 0.6 ms when none is.)
//   burst     a sequential read stream plus a write stream made of bursts of B bytes (full sectors) at pseudo-random
//             places of a 4 GiB buffer.  Question: how large must a contiguous piece be for DRAM to run at its copy rate?
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>

__global__ void __launch_bounds__(256) partial_kernel(ulonglong2* out, long long total_sectors, int S, int delay_ns, int second) {
    const long long nchunks = total_sectors / S;
    for (long long c = blockIdx.x; c < nchunks; c += gridDim.x) {
        ulonglong2* base = out + c * (long long)S * 2;
        for (int i = threadIdx.x; i < S; i += 256) base[2 * i] = make_ulonglong2(c, i);
        if (delay_ns > 0) {
            __syncthreads();
            const long long t0 = clock64();
            while (clock64() - t0 < (long long)delay_ns * 19 / 10) __nanosleep(100);  // ~1.9 GHz
            __syncthreads();
        }
        if (second)
            for (int i = threadIdx.x; i < S; i += 256) base[2 * i + 1] = make_ulonglong2(i, c);
    }
}

// item i (16 bytes) of burst b goes to burst slot perm(b): an odd multiplier modulo a power of two is a bijection
__global__ void __launch_bounds__(256) burst_kernel(const uint4* __restrict__ in, uint4* __restrict__ out, long long total16, int log2burst16,
                                                   int log2nbursts, int do_read) {
    const long long stride = (long long)gridDim.x * 256;
    for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < total16; i += stride) {
        const long long b = i >> log2burst16, r = i & ((1ll << log2burst16) - 1);
        const long long pb = (long long)(((unsigned long long)b * 0x9E3779B97F4A7C15ull + 12345ull) & ((1ull << log2nbursts) - 1ull));
        uint4 v = make_uint4((unsigned)i, 1u, 2u, 3u);
        if (do_read) v = in[i];
        out[(pb << log2burst16) + r] = v;
    }
}

#define CHECK(x)                                                                       \
    do {                                                                               \
        cudaError_t e_ = (x);                                                          \
        if (e_ != cudaSuccess) {                                                       \
            std::printf("{\"probe_error\": \"%s\"}\n", cudaGetErrorString(e_));        \
            return 1;                                                                  \
        }                                                                              \
    } while (0)

int main() {
    cudaEvent_t e0, e1;
    CHECK(cudaEventCreate(&e0));
    CHECK(cudaEventCreate(&e1));
    {   // ---- partial-sector probe
        const long long bytes = 1ll << 30;
        ulonglong2* d;
        CHECK(cudaMalloc(&d, bytes));
        CHECK(cudaMemset(d, 0, bytes));
        const long long total_sectors = bytes / 32;
        const int grid = 148 * 8;
        const int Ss[] = {64, 256, 1024, 4096};
        const int delays[] = {0, 300, 1000, 3000, 10000, 30000};
        for (int second = 1; second >= 0; --second)
            for (int S : Ss)
                for (int dl : delays) {
                    if (!second && dl) continue;
                    CHECK(cudaEventRecord(e0));
                    partial_kernel<<<grid, 256>>>(d, total_sectors, S, dl, second);
                    CHECK(cudaEventRecord(e1));
                    CHECK(cudaEventSynchronize(e1));
                    float ms;
                    CHECK(cudaEventElapsedTime(&ms, e0, e1));
                    std::printf("{\"probe\": \"partial\", \"second_half_written\": %d, \"sectors_per_cta_chunk\": %d, \"open_half_written_MB\": %.1f, "
                                "\"delay_ns\": %d, \"ms\": %.3f}\n", second, S, grid * (double)S * 32 / 1e6, dl, ms);
                }
        CHECK(cudaFree(d));
    }
    {   // ---- burst-size probe
        const long long bytes = 4ll << 30;
        uint4 *in, *out;
        CHECK(cudaMalloc(&in, bytes));
        CHECK(cudaMalloc(&out, bytes));
        CHECK(cudaMemset(in, 1, bytes));
        CHECK(cudaMemset(out, 0, bytes));
        const long long total16 = bytes / 16;  // 2^28 items
        for (int do_read = 1; do_read >= 0; --do_read)
            for (int lb = 1; lb <= 12; ++lb) {  // bursts of 32 B ... 64 KB
                float best = 1e9f;
                for (int rep = 0; rep < 3; ++rep) {
                    CHECK(cudaEventRecord(e0));
                    burst_kernel<<<148 * 16, 256>>>(in, out, total16, lb, 28 - lb, do_read);
                    CHECK(cudaEventRecord(e1));
                    CHECK(cudaEventSynchronize(e1));
                    float ms;
                    CHECK(cudaEventElapsedTime(&ms, e0, e1));
                    if (ms < best) best = ms;
                }
                std::printf("{\"probe\": \"burst\", \"sequential_read_stream\": %d, \"burst_bytes\": %d, \"ms\": %.3f, \"GBps\": %.0f}\n", do_read, 16 << lb, best,
                            (do_read ? 2.0 : 1.0) * bytes / best / 1e6);
            }
        CHECK(cudaFree(in));
        CHECK(cudaFree(out));
    }
    CHECK(cudaGetLastError());
    return 0;
}
