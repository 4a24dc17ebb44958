// step_kernels.cu -- a2, a3, a4, a9: the SoA streaming integration steps (Eq. 1; K4 of the
// component inventory, re-designed: ONE fused launch updates every component of pos and vel, each thread owns P
// consecutive particles and touches every field array with one 256-bit (double, int64) / 128-bit (float) /
// 32-bit (uint8) access, instead of the paper's one launch per component with scalar 4-byte accesses,
// PAPER.md:231).  HBM-bound: no shared memory, no reuse, nothing for tensor cores to do.
#include "common.cuh"
#include "ops.hpp"

namespace soax {

struct StepK {
    double dt, k, ctr, hh;
    float dt_f;
    uint32_t mask;
};

// ---- one group of P consecutive particles starting at i0 (P = 1 serves the ragged tail) ---------------------
template <class L, int KIND, int P>
__device__ __forceinline__ void step_group(const Ptrs<L::ncomp>& a, int64_t i0, const StepK& c) {
    using X = typename L::template type_of<pos_tag>;
    using V = typename L::template type_of<vel_tag>;
    if constexpr (KIND == SOAX_STEP_DRIFT || KIND == SOAX_STEP_SYMPLECTIC_EULER_HARMONIC) {
        Vec<double, P> x[3];
        Vec<V, P> v[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) x[d] = ld_vec<double, P>(field_ptr<L, pos_tag>(a, d) + i0);
#pragma unroll
        for (int d = 0; d < 3; ++d) v[d] = ld_vec<V, P>(field_ptr<L, vel_tag>(a, d) + i0);
        const V dt_v = sizeof(V) == 4 ? (V)c.dt_f : (V)c.dt;
#pragma unroll
        for (int d = 0; d < 3; ++d)
#pragma unroll
            for (int j = 0; j < P; ++j) {
                if constexpr (KIND == SOAX_STEP_SYMPLECTIC_EULER_HARMONIC)
                    v[d].v[j] = kick1<V>(dt_v, c.k, c.ctr, x[d].v[j], v[d].v[j]);
                x[d].v[j] = drift1<V>(c.dt, v[d].v[j], x[d].v[j]);
            }
        if constexpr (KIND == SOAX_STEP_SYMPLECTIC_EULER_HARMONIC) {
#pragma unroll
            for (int d = 0; d < 3; ++d) st_vec<V, P>(field_ptr<L, vel_tag>(a, d) + i0, v[d]);
        }
#pragma unroll
        for (int d = 0; d < 3; ++d) st_vec<double, P>(field_ptr<L, pos_tag>(a, d) + i0, x[d]);
    } else if constexpr (KIND == SOAX_STEP_EULER_NOWRAP) {
        // Eq. 1 as printed: x_c += dt v_c, one fma in the type of pos, no wrap.
        Vec<X, P> x[3];
        Vec<V, P> v[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) x[d] = ld_vec<X, P>(field_ptr<L, pos_tag>(a, d) + i0);
#pragma unroll
        for (int d = 0; d < 3; ++d) v[d] = ld_vec<V, P>(field_ptr<L, vel_tag>(a, d) + i0);
        const X dt_x = sizeof(X) == 4 ? (X)c.dt_f : (X)c.dt;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
#pragma unroll
            for (int j = 0; j < P; ++j) x[d].v[j] = fma_t(dt_x, (X)v[d].v[j], x[d].v[j]);
            st_vec<X, P>(field_ptr<L, pos_tag>(a, d) + i0, x[d]);
        }
    } else {  // SOAX_STEP_RK2_MIDPOINT_HARMONIC_MASKED (a9): Q6 force on wrapped midpoint, Q7 acc = a2, Q8 w = k/m
        const Vec<uint8_t, P> fl = ld_vec<uint8_t, P>(field_ptr<L, flags_tag>(a, 0) + i0);
        bool act[P], any = false, all = true;
#pragma unroll
        for (int j = 0; j < P; ++j) { act[j] = (fl.v[j] & c.mask) != 0; any |= act[j]; all &= act[j]; }
        if (!any) return;  // unused fields cost nothing in an SoA
        const Vec<float, P> m = ld_vec<float, P>(field_ptr<L, mass_tag>(a, 0) + i0);
        Vec<double, P> x[3], v[3], ac[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) x[d] = ld_vec<double, P>(field_ptr<L, pos_tag>(a, d) + i0);
#pragma unroll
        for (int d = 0; d < 3; ++d) v[d] = ld_vec<double, P>(field_ptr<L, vel_tag>(a, d) + i0);
        if (!all) {  // inactive particles keep their acc bits: merge into the full-width store
#pragma unroll
            for (int d = 0; d < 3; ++d) ac[d] = ld_vec<double, P>(field_ptr<L, acc_tag>(a, d) + i0);
        }
#pragma unroll
        for (int j = 0; j < P; ++j) {
            if (!act[j]) continue;
            const double w = c.k / (double)m.v[j];
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                const double a1 = -(w * (x[d].v[j] - c.ctr));
                const double ph = wrap01(fma(c.hh, v[d].v[j], x[d].v[j]));
                const double vh = fma(c.hh, a1, v[d].v[j]);
                const double a2 = -(w * (ph - c.ctr));
                x[d].v[j] = wrap01(fma(c.dt, vh, x[d].v[j]));
                v[d].v[j] = fma(c.dt, a2, v[d].v[j]);
                ac[d].v[j] = a2;
            }
        }
#pragma unroll
        for (int d = 0; d < 3; ++d) st_vec<double, P>(field_ptr<L, pos_tag>(a, d) + i0, x[d]);
#pragma unroll
        for (int d = 0; d < 3; ++d) st_vec<double, P>(field_ptr<L, vel_tag>(a, d) + i0, v[d]);
#pragma unroll
        for (int d = 0; d < 3; ++d) st_vec<double, P>(field_ptr<L, acc_tag>(a, d) + i0, ac[d]);
    }
}

// Grid-stride over groups of P particles; the n % P tail particles are done one by one by the first threads
// of the grid ("split handling for odd tails").  One launch = one full pass over memory = one time step (Q14).
template <class L, int KIND, int P>
__global__ void __launch_bounds__(512) step_soa_kernel(Ptrs<L::ncomp> a, int64_t n, StepK c) {
    const int64_t ngroups = n / P;
    const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t g = tid; g < ngroups; g += stride) step_group<L, KIND, P>(a, g * P, c);
    if (P > 1) {
        const int64_t t = ngroups * P + tid;
        if (t < n) step_group<L, KIND, 1>(a, t, c);
    }
}

template <class L, int KIND>
constexpr bool step_supported() {
    if constexpr (KIND == SOAX_STEP_DRIFT || KIND == SOAX_STEP_SYMPLECTIC_EULER_HARMONIC)
        return L::template has_as<pos_tag, double, 3>() &&
               (L::template has_as<vel_tag, float, 3>() || L::template has_as<vel_tag, double, 3>());
    else if constexpr (KIND == SOAX_STEP_EULER_NOWRAP)
        return L::template has<pos_tag> && L::template has<vel_tag> && L::template field<(L::template find<pos_tag>() < 0 ? 0 : L::template find<pos_tag>())>::dim == 3 &&
               L::template field<(L::template find<vel_tag>() < 0 ? 0 : L::template find<vel_tag>())>::dim == 3 &&
               !std::is_integral<typename L::template type_of<pos_tag>>::value &&
               !std::is_integral<typename L::template type_of<vel_tag>>::value;
    else
        return L::template has_as<pos_tag, double, 3>() && L::template has_as<vel_tag, double, 3>() &&
               L::template has_as<acc_tag, double, 3>() && L::template has_as<mass_tag, float, 1>() &&
               L::template has_as<flags_tag, uint8_t, 1>();
}

template <class L, int KIND, int P>
static int launch_step(const Ptrs<L::ncomp>& a, int64_t n, const StepK& c, cudaStream_t st) {
    if (n == 0) return SOAX_OK;
    const int block = g_tune.step_block;
    const int64_t threads = (n / P > n % P ? n / P : n % P);
    int64_t blocks = (threads + block - 1) / block;
    if (g_tune.step_persist > 0 && blocks > (int64_t)kSMs * g_tune.step_persist) blocks = (int64_t)kSMs * g_tune.step_persist;
    if (blocks < 1) blocks = 1;
    step_soa_kernel<L, KIND, P><<<(unsigned)blocks, block, 0, st>>>(a, n, c);
    return launched();
}

template <class L, int KIND>
static int step_kind(const Ptrs<L::ncomp>& a, int64_t n, const StepK& c, cudaStream_t st) {
    if constexpr (!step_supported<L, KIND>()) {
        return SOAX_ERR_UNSUPPORTED;
    } else {
        switch (g_tune.step_ppt) {
            case 1: return launch_step<L, KIND, 1>(a, n, c, st);
            case 2: return launch_step<L, KIND, 2>(a, n, c, st);
            default: return launch_step<L, KIND, 4>(a, n, c, st);
        }
    }
}

template <class L>
int step_entry(void* const* comps, int64_t n, const soax_step_params* p, cudaStream_t st) {
    const Ptrs<L::ncomp> a = make_ptrs<L>(comps);
    StepK c;
    c.dt = p->dt; c.k = p->k; c.ctr = p->center; c.hh = 0.5 * p->dt; c.dt_f = (float)p->dt; c.mask = p->flag_mask;
    switch (p->kind) {
        case SOAX_STEP_DRIFT: return step_kind<L, SOAX_STEP_DRIFT>(a, n, c, st);
        case SOAX_STEP_SYMPLECTIC_EULER_HARMONIC: return step_kind<L, SOAX_STEP_SYMPLECTIC_EULER_HARMONIC>(a, n, c, st);
        case SOAX_STEP_RK2_MIDPOINT_HARMONIC_MASKED: return step_kind<L, SOAX_STEP_RK2_MIDPOINT_HARMONIC_MASKED>(a, n, c, st);
        case SOAX_STEP_EULER_NOWRAP: return step_kind<L, SOAX_STEP_EULER_NOWRAP>(a, n, c, st);
        default: return SOAX_ERR_INVALID_ARG;
    }
}

#define X(L) template int step_entry<L>(void* const*, int64_t, const soax_step_params*, cudaStream_t);
SOAX_FOR_EACH_LAYOUT(X)
#undef X

}  // namespace soax
