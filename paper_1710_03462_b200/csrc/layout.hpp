// layout.hpp -- compile-time field lists ("layouts") and the run-time descriptors generated from them.
//
// The paper builds its SoA from a std::tuple of attribute classes made by SOAX_ATTRIBUTE (PAPER.md:267-287,
// Listing 5) and walks that tuple with recursive templates (TupleDo).  Here the same
// idea is restated for CUDA: a Layout<Field<Tag,T,Dim>...> typelist; every kernel that must touch "each
// component array" (transposes, permutation, upload) is instantiated per layout and unrolls over the list
// at compile time with index sequences, so the generated code holds one straight-line access per array.
// Physics kernels look fields up BY TAG (pos, vel, ...) at compile time; a layout lacking a field simply
// does not instantiate that kernel and the C boundary answers SOAX_ERR_UNSUPPORTED.
#pragma once
#include <cstddef>
#include <cstdint>
#include <type_traits>
#include <utility>

#include "../../include/soax.h"

namespace soax {

// ---- attribute tags (the paper's attribute class names) ---------------------------------
struct id_tag     { static constexpr const char* name = "id"; };
struct pos_tag    { static constexpr const char* name = "pos"; };
struct vel_tag    { static constexpr const char* name = "vel"; };
struct acc_tag    { static constexpr const char* name = "acc"; };
struct mass_tag   { static constexpr const char* name = "mass"; };
struct charge_tag { static constexpr const char* name = "charge"; };
struct flags_tag  { static constexpr const char* name = "flags"; };
struct temp_tag   { static constexpr const char* name = "temp"; };

template <class T> struct dtype_of;
template <> struct dtype_of<int32_t> { static constexpr int value = SOAX_I32; };
template <> struct dtype_of<int64_t> { static constexpr int value = SOAX_I64; };
template <> struct dtype_of<uint8_t> { static constexpr int value = SOAX_U8; };
template <> struct dtype_of<float>   { static constexpr int value = SOAX_F32; };
template <> struct dtype_of<double>  { static constexpr int value = SOAX_F64; };

constexpr int dtype_size(int dt) { return dt == SOAX_I32 ? 4 : dt == SOAX_I64 ? 8 : dt == SOAX_U8 ? 1 : dt == SOAX_F32 ? 4 : dt == SOAX_F64 ? 8 : 0; }

template <class Tag, class T, int Dim>
struct Field {
    using tag = Tag;
    using type = T;
    static constexpr int dim = Dim;
    static_assert(Dim >= 1, "a field has at least one component");
};

constexpr int kMaxComp = 48;  // B6_32: 3 + 3 + 32 = 38 component arrays

// Kernel argument: one device pointer per component array, passed BY VALUE (the paper's deviceWrapper,
// PAPER.md:362-364, reduced to what it was for: raw pointers that can be copied into a kernel).
template <int NC>
struct Ptrs {
    void* p[NC];
};

namespace detail {
template <int I, class... Fs> struct nth;
template <class F, class... Fs> struct nth<0, F, Fs...> { using type = F; };
template <int I, class F, class... Fs> struct nth<I, F, Fs...> { using type = typename nth<I - 1, Fs...>::type; };
}  // namespace detail

template <class... Fs>
struct Layout {
    static constexpr int nfields = sizeof...(Fs);
    static constexpr int ncomp = (Fs::dim + ... + 0);
    static_assert(ncomp <= kMaxComp, "raise kMaxComp");
    template <int I> using field = typename detail::nth<I, Fs...>::type;

    // ---- field-level tables -----------------------------------------------------------------------------
    static constexpr int field_dim(int f) { int d[] = {Fs::dim...}; return d[f]; }
    static constexpr int field_size(int f) { int s[] = {(int)sizeof(typename Fs::type)...}; return s[f]; }
    static constexpr int field_dtype(int f) { int s[] = {dtype_of<typename Fs::type>::value...}; return s[f]; }
    static constexpr int field_begin(int f) { int b = 0; for (int i = 0; i < f; ++i) b += field_dim(i); return b; }

    // ---- component-level tables (component-major: posArr(0), posArr(1), posArr(2), ... PAPER.md:294) ------
    static constexpr int comp_field(int c) { int f = 0; while (c >= field_dim(f)) { c -= field_dim(f); ++f; } return f; }
    static constexpr int comp_size(int c) { return field_size(comp_field(c)); }
    static constexpr int comp_dtype(int c) { return field_dtype(comp_field(c)); }
    static constexpr int comp_in_field(int c) { return c - field_begin(comp_field(c)); }
    template <int C> using comp_type = typename field<comp_field(C)>::type;

    // ---- packed AoS image: declaration order, no padding (Q1) ---------------------------------------------
    static constexpr int aos_offset(int c) { int o = 0; for (int i = 0; i < c; ++i) o += comp_size(i); return o; }
    static constexpr int aos_stride = aos_offset(ncomp);
    static constexpr int soa_bytes = aos_stride;  // bytes per particle summed over the component arrays

    // ---- lookup by tag ------------------------------------------------------------------------------------
    template <class Tag> static constexpr int find() {
        bool m[] = {std::is_same<typename Fs::tag, Tag>::value...};
        for (int i = 0; i < nfields; ++i) if (m[i]) return i;
        return -1;
    }
    template <class Tag> static constexpr bool has = find<Tag>() >= 0;
    template <class Tag, class T, int Dim> static constexpr bool has_as() {
        constexpr int f = find<Tag>();
        if constexpr (f < 0) return false;
        else return std::is_same<typename field<f>::type, T>::value && field<f>::dim == Dim;
    }
    template <class Tag> static constexpr int begin_of = field_begin(find<Tag>() < 0 ? 0 : find<Tag>());
    template <class Tag> using type_of = typename field<(find<Tag>() < 0 ? 0 : find<Tag>())>::type;

    static const char* field_name(int f) { const char* n[] = {Fs::tag::name...}; return n[f]; }
};

// Typed pointer to component C of layout L.
template <class L, int C>
__host__ __device__ inline typename L::template comp_type<C>* comp_ptr(const Ptrs<L::ncomp>& a) {
    return static_cast<typename L::template comp_type<C>*>(a.p[C]);
}
// Typed pointer to component k of the field tagged Tag.
template <class L, class Tag>
__host__ __device__ inline typename L::template type_of<Tag>* field_ptr(const Ptrs<L::ncomp>& a, int k) {
    return static_cast<typename L::template type_of<Tag>*>(a.p[L::template begin_of<Tag> + k]);
}

// for_each_comp<L>(f): f(std::integral_constant<int, C>{}) for C = 0..ncomp-1, unrolled at compile time --
// the TupleDo recursion of PAPER.md:326-348 written with an index sequence.
template <class F, int... Cs>
__host__ __device__ inline void for_each_comp_impl(F&& f, std::integer_sequence<int, Cs...>) {
    (f(std::integral_constant<int, Cs>{}), ...);
}
template <class L, class F>
__host__ __device__ inline void for_each_comp(F&& f) {
    for_each_comp_impl(static_cast<F&&>(f), std::make_integer_sequence<int, L::ncomp>{});
}

// for_each_int<N>(f): f(std::integral_constant<int, I>{}) for I = 0..N-1.
template <int N, class F>
__host__ __device__ inline void for_each_int(F&& f) {
    for_each_comp_impl(static_cast<F&&>(f), std::make_integer_sequence<int, N>{});
}

// CompRegs<L, C0, N, integer_sequence<int, 0..M-1>>: N registers of the right type for each of the components C0..C0+M-1.
template <int C, class T, int N> struct CompSlot { T v[N]; };
template <class L, int C0, int N, class Seq> struct CompRegs;
template <class L, int C0, int N, int... Is>
struct CompRegs<L, C0, N, std::integer_sequence<int, Is...>> : CompSlot<C0 + Is, typename L::template comp_type<C0 + Is>, N>... {
    template <int C> __host__ __device__ typename L::template comp_type<C>* get() {
        return static_cast<CompSlot<C, typename L::template comp_type<C>, N>&>(*this).v;
    }
};

// ---- the layouts this library instantiates -----------------------------------------------------------------
// R1: the program summary's record: configs 1, 2, 3, 5.
using R1 = Layout<Field<id_tag, int32_t, 1>, Field<pos_tag, double, 3>, Field<vel_tag, float, 3>>;
// R1R: the same fields declared {pos; vel; id}: packed offsets 0 / 24 / 36, stride 40, every field naturally aligned --
// the sensitivity row of reading Q1 (what config 3's AoS kernels gain when the doubles are 8-byte aligned).
using R1R = Layout<Field<pos_tag, double, 3>, Field<vel_tag, float, 3>, Field<id_tag, int32_t, 1>>;
// R2: the wide heterogeneous record of BASELINE.json config 4.
using R2 = Layout<Field<id_tag, int64_t, 1>, Field<pos_tag, double, 3>, Field<vel_tag, double, 3>,
                  Field<acc_tag, double, 3>, Field<mass_tag, float, 1>, Field<charge_tag, float, 1>,
                  Field<flags_tag, uint8_t, 1>>;
// B6_S: the paper's benchmark particle, Listing 4: float x[3]; float v[3]; float temp[SIZE].
template <int S> struct B6_of { using type = Layout<Field<pos_tag, float, 3>, Field<vel_tag, float, 3>, Field<temp_tag, float, S>>; };
template <> struct B6_of<0> { using type = Layout<Field<pos_tag, float, 3>, Field<vel_tag, float, 3>>; };
template <int S> using B6 = typename B6_of<S>::type;

static_assert(R1::ncomp == 7 && R1::aos_stride == 40 && R1::aos_offset(1) == 4 && R1::aos_offset(4) == 28, "R1 (Q1)");
static_assert(R1R::aos_stride == 40 && R1R::aos_offset(3) == 24 && R1R::aos_offset(6) == 36, "R1R (Q1 sensitivity row)");
static_assert(R2::ncomp == 13 && R2::aos_stride == 89, "R2");
static_assert(B6<0>::aos_stride == 24 && B6<32>::aos_stride == 152, "PAPER.md:237: 24 bytes at SIZE=0");

}  // namespace soax
