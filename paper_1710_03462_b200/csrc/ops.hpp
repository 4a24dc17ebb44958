// ops.hpp -- per-layout entry points.  Each family lives in its own .cu, is a template over the layout and is
// explicitly instantiated for every layout of SOAX_FOR_EACH_LAYOUT; registry.cu stores the instantiations'
// addresses in the layout descriptor ("a field-descriptor and layout registry that generates per-layout CUDA
// kernels from C++ templates").
#pragma once
#include <cuda_runtime.h>

#include "layout.hpp"

// The layouts compiled into the library.  Adding a layout = one line here (and a `using` in layout.hpp).
#define SOAX_FOR_EACH_LAYOUT(X) X(R1) X(R1R) X(R2) X(B6<0>) X(B6<8>) X(B6<16>) X(B6<32>)

namespace soax {

// Launch-shape knobs (soax_tune).  Defaults are the measured best on B200 (profiles/).
struct Tuning {
    int step_ppt = 4;       // particles per thread in the SoA step kernels: 1, 2 or 4
    int step_block = 256;   // threads per CTA
    int step_persist = 0;   // 0: one CTA per tile of work; k > 0: persistent grid of k CTAs per SM
    int step_graph = 1;     // 1: soax_step(nsteps >= 2) on a capturable stream replays a captured graph of nsteps launches
    int aos_block = 256;
    int xpose_ring = 1;     // 1: pipelined ring transposes (default), 0: one tile per CTA visit
    int xpose_r = 0, xpose_ns = 0, xpose_ctas = 0;  // ring shape override: 256*r records per stage, ns stages, CTAs per SM cap (0 = default)
    int bin_bits = 0;       // digit width of the counting-sort passes: 0 = default (9: two passes for G = 64), else 1..9
    int bin_cluster = 0;    // 0 = default (clusters of 4 CTAs for digits of 8 or 9 bits, none below); 1, 2, 4, 8, 16: forced
    int bin_pace_every = 0; // a pacing barrier every this many stores of a thread (0 = default: 2 for the cluster barrier, else 1)
    int bin_pace = -1;      // pacing of the scatter stores: -1 = default (cluster barrier with clusters); else bits 12-13 = 1: CTA barrier, 2: cluster barrier between a thread's stores; low 12 bits = nanoseconds of sleep
    int bin_csync = 1;      // with clusters: 1 = cluster barrier before every array's stores (default), 0 = none
};
extern Tuning g_tune;

template <class L> int step_entry(void* const* comps, int64_t n, const soax_step_params* p, cudaStream_t st);
template <class L> int step_aos_entry(void* aos, int64_t n, const soax_step_params* p, int variant, cudaStream_t st);
template <class L> int aos_to_soa_entry(void* const* comps, const void* aos, int64_t n, cudaStream_t st);
template <class L> int soa_to_aos_entry(void* const* comps, void* aos, int64_t n, cudaStream_t st);
template <class L> int gather_segments_entry(void* const* comps, const void* aos, const uint32_t* seg_dst, const uint32_t* seg_src, int64_t nseg,
                                             int64_t n, cudaStream_t st);
template <class L> int energy_entry(void* const* comps, int64_t n, int kind, double k, double ctr, void* scratch,
                                    double* out, cudaStream_t st);
struct BinArgs {
    void* const* src; void* const* dst; int64_t n; int log2g; double drift_dt;
    uint32_t* counts; uint32_t* offsets; uint32_t* perm; double* kinetic;
    void* scratch; size_t scratch_bytes;
    bool inplace;  // soax_bin_permute_inplace: `dst` is a WORK container; the sorted set returns to src
};
template <class L> int bin_permute_entry(const BinArgs& a, cudaStream_t st);
template <class L> size_t bin_scratch_bytes(int64_t n, int log2g, bool inplace);

// NEXT-3 (container_kernels.cu)
// Enqueues everything and returns: the scan kernel stores the survivor count straight into pin_n (MAPPED pinned host memory: no
// copy node), a cudaMemcpyAsync brings it to host_new_n if that is not null, and count_ready is recorded after both.
template <class L> int remove_entry(void* const* src, void* const* dst, const uint8_t* kill, int64_t n, int mode, void* scratch,
                                    int64_t dst_capacity, int64_t* pin_n, int64_t* host_new_n,
                                    cudaEvent_t count_ready, cudaStream_t st);
// The STABLE removal with its scratch in a file-scope device array of container_kernels.cu (soax_remove_stable_noalloc): no
// device, pinned or event allocation anywhere on the path; the survivor count goes to dev_new_n (device memory).
template <class L> int remove_stable_noalloc_entry(void* const* src, void* const* dst, const uint8_t* kill, int64_t n, uint32_t flip,
                                                   int64_t dst_capacity, int64_t* dev_new_n, cudaStream_t st);
template <class L> int gather_rows_entry(void* const* comps, int64_t n, const uint32_t* idx, int64_t m, void* aos, cudaStream_t st);
size_t remove_scratch_bytes(int64_t n);

constexpr int kEnergyBlocks = 1184;  // 148 SMs x 8 CTAs: fixed, so the reduction tree is fixed
constexpr size_t kEnergyScratchBytes = (size_t)kEnergyBlocks * sizeof(double);

template <class L> inline Ptrs<L::ncomp> make_ptrs(void* const* comps) {
    Ptrs<L::ncomp> a;
    for (int c = 0; c < L::ncomp; ++c) a.p[c] = comps[c];
    return a;
}

// byte size of the slab for `cap` particles: every component array starts on a 256-byte boundary
constexpr size_t kAlign = 256;
inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

}  // namespace soax
