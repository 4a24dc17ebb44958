// reduce_kernels.cu -- a8: energy reduction in double ("warp-shuffle plus block reductions in double").
// Pass 1: a FIXED grid of kEnergyBlocks CTAs; each thread sums the terms of its P-particle groups in
// grid-stride order, then warp shuffles + one shared-memory step give the CTA's partial.  Pass 2: one CTA sums
// the partials in a fixed order.  Grid, block and order never depend on the device or on timing, so the result
// is run-to-run deterministic (no floating-point atomics).  HBM-bound: 36 B/particle (KE+PE) or 12 (KE).
#include "common.cuh"
#include "ops.hpp"

namespace soax {

constexpr int kEnergyThreads = 256;

template <class L, bool HARMONIC, int P>
__device__ __forceinline__ double energy_group(const Ptrs<L::ncomp>& a, int64_t i0, double k, double ctr) {
    using V = typename L::template type_of<vel_tag>;
    Vec<V, P> v[3];
    Vec<double, P> x[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) v[d] = ld_vec<V, P>(field_ptr<L, vel_tag>(a, d) + i0);
    if constexpr (HARMONIC) {
#pragma unroll
        for (int d = 0; d < 3; ++d) x[d] = ld_vec<double, P>(field_ptr<L, pos_tag>(a, d) + i0);
    } else {
#pragma unroll
        for (int d = 0; d < 3; ++d)
#pragma unroll
            for (int j = 0; j < P; ++j) x[d].v[j] = 0.0;
    }
    double s = 0.0;
#pragma unroll
    for (int j = 0; j < P; ++j)
        s += energy1<HARMONIC>((double)v[0].v[j], (double)v[1].v[j], (double)v[2].v[j], x[0].v[j], x[1].v[j],
                               x[2].v[j], k, ctr);
    return s;
}

template <class L, bool HARMONIC>
__global__ void __launch_bounds__(kEnergyThreads) energy_partial_kernel(Ptrs<L::ncomp> a, int64_t n, double k,
                                                                        double ctr, double* partial) {
    constexpr int P = 4;
    __shared__ double sm[32];
    const int64_t ngroups = n / P;
    const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    double s = 0.0;
    for (int64_t g = tid; g < ngroups; g += stride) s += energy_group<L, HARMONIC, P>(a, g * P, k, ctr);
    const int64_t t = ngroups * P + tid;
    if (t < n) s += energy_group<L, HARMONIC, 1>(a, t, k, ctr);
    s = block_sum(s, sm);
    if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

// Sum `m` doubles in a fixed order with one CTA; writes *out.
__global__ void __launch_bounds__(1024) sum_partials_kernel(const double* partial, int m, double* out) {
    __shared__ double sm[32];
    double s = 0.0;
    for (int i = threadIdx.x; i < m; i += blockDim.x) s += partial[i];
    s = block_sum(s, sm);
    if (threadIdx.x == 0) *out = s;
}

int sum_partials(const double* partial, int m, double* out, cudaStream_t st) {
    sum_partials_kernel<<<1, 1024, 0, st>>>(partial, m, out);
    return launched();
}

template <class L>
int energy_entry(void* const* comps, int64_t n, int kind, double k, double ctr, void* scratch, double* out,
                 cudaStream_t st) {
    constexpr bool has_vel = L::template has_as<vel_tag, float, 3>() || L::template has_as<vel_tag, double, 3>();
    constexpr bool has_pos = L::template has_as<pos_tag, double, 3>();
    if constexpr (!has_vel) {
        return SOAX_ERR_UNSUPPORTED;
    } else {
        const Ptrs<L::ncomp> a = make_ptrs<L>(comps);
        double* partial = static_cast<double*>(scratch);
        if (kind == SOAX_ENERGY_KINETIC) {
            energy_partial_kernel<L, false><<<kEnergyBlocks, kEnergyThreads, 0, st>>>(a, n, k, ctr, partial);
        } else if (kind == SOAX_ENERGY_KINETIC_PLUS_HARMONIC) {
            if constexpr (!has_pos) return SOAX_ERR_UNSUPPORTED;
            else energy_partial_kernel<L, true><<<kEnergyBlocks, kEnergyThreads, 0, st>>>(a, n, k, ctr, partial);
        } else {
            return SOAX_ERR_INVALID_ARG;
        }
        SOAX_TRY(launched());
        return sum_partials(partial, kEnergyBlocks, out, st);
    }
}

#define X(L) template int energy_entry<L>(void* const*, int64_t, int, double, double, void*, double*, cudaStream_t);
SOAX_FOR_EACH_LAYOUT(X)
#undef X

}  // namespace soax
